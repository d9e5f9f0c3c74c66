// a5 + a6: Felsenstein pruning and the root / site-pattern log-likelihood reduction
// (Eq.(4): L_u(i) = [sum_j p_ij(v) L_v(j)] [sum_k p_ik(w) L_w(k)], post-order; tips are 0/1 vectors,
//  all-ones if missing; L72: sum_i L_root(i) pi_i, independent sites and rate categories aggregated).
//
// Layout in HBM: partials[internal node][category][pattern][state] fp64, scale_exp[internal node][pattern] int32.
// Nodes are processed level by level (one launch per post-order level, all launches in one CUDA graph); patterns are
// independent, so a level needs no inter-CTA synchronisation.  Rescaling (reading A12): every (node, pattern) is
// divided by 2^e with e = floor(log2(max over category and state)), which is exact in binary floating point; the
// exponents accumulate up the tree and re-enter at the root as e * ln 2.
//
//   prune4_kernel<C>   K == 4: one thread per pattern, all C categories in registers; child partials stream as
//                      256-bit loads (LDG.E.256), fully coalesced ([C][L][4] is pattern-contiguous per category),
//                      tips are read as one byte per pattern; one 256-bit store per category.  HBM-bound.
//   prune_generic_kernel  any K <= 64: one CTA per (node, tile of patterns); per category the two K x K matrices
//                      and the child tiles are staged in shared memory, DFMA mat-vec products.
//   root_site_kernel / final_sum_kernel  per-pattern ln-likelihood, deterministic two-stage weighted sum.
#include "epx_internal.h"

namespace {

struct __align__(32) double4a { double x, y, z, w; };

__device__ __forceinline__ double4a ld256(const double* p)
{
    double4a v;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void st256(double* p, double a, double b, double c, double d)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// exponent of a positive normal double, and the exact power of two 2^-e
__device__ __forceinline__ int exponent_of(double m) { return ((__double2hiint(m) >> 20) & 0x7ff) - 1023; }
__device__ __forceinline__ double pow2_neg(int e) { return __hiloint2double((1023 - e) << 20, 0); }

// ------------------------------------------------------------------------------------------------ K == 4
template <int C>
__global__ void __launch_bounds__(256) prune4_kernel(const PruneOp* __restrict__ ops, int tiles, int L,
    const double* __restrict__ P, const uint8_t* __restrict__ tips, double* __restrict__ partials,
    int32_t* __restrict__ scale_exp)
{
    __shared__ double Pm[2][C][16];
    const PruneOp op = ops[blockIdx.x / tiles];
    const int tid = threadIdx.x;
    const int p = (blockIdx.x % tiles) * 256 + tid;
    if (tid < 2 * C * 16) {
        int ch = tid / (C * 16), rem = tid % (C * 16);
        Pm[ch][rem / 16][rem % 16] = P[((size_t)op.child[ch] * C) * 16 + rem];
    }
    __syncthreads();
    if (p >= L) return;

    double f[2][C][4];
    int ex = 0;
#pragma unroll
    for (int ch = 0; ch < 2; ch++) {
        if (op.child_is_tip[ch]) {
            const int s = tips[(size_t)op.child[ch] * L + p];
#pragma unroll
            for (int c = 0; c < C; c++)
#pragma unroll
                for (int i = 0; i < 4; i++) f[ch][c][i] = (s < 4) ? Pm[ch][c][i * 4 + s] : 1.0;
        } else {
            const double* src = partials + ((size_t)op.cpidx[ch] * C * L + p) * 4;
            double4a v[C];
#pragma unroll
            for (int c = 0; c < C; c++) v[c] = ld256(src + (size_t)c * L * 4);
            ex += scale_exp[(size_t)op.cpidx[ch] * L + p];
#pragma unroll
            for (int c = 0; c < C; c++)
#pragma unroll
                for (int i = 0; i < 4; i++) {
                    const double* row = &Pm[ch][c][i * 4];
                    f[ch][c][i] = fma(row[3], v[c].w, fma(row[2], v[c].z, fma(row[1], v[c].y, row[0] * v[c].x)));
                }
        }
    }
    double m = 0.0;
#pragma unroll
    for (int c = 0; c < C; c++)
#pragma unroll
        for (int i = 0; i < 4; i++) {
            f[0][c][i] *= f[1][c][i];
            m = fmax(m, f[0][c][i]);
        }
    double sc = 1.0;
    if (m > 0.0 && m < 1.7e308) {
        const int e = exponent_of(m);
        if (e > -1000) { sc = pow2_neg(e); ex += e; }      // (sub)normal-range guard; never taken by real data
    }
    double* dst = partials + ((size_t)op.pidx * C * L + p) * 4;
#pragma unroll
    for (int c = 0; c < C; c++)
        st256(dst + (size_t)c * L * 4, f[0][c][0] * sc, f[0][c][1] * sc, f[0][c][2] * sc, f[0][c][3] * sc);
    scale_exp[(size_t)op.pidx * L + p] = ex;
}

// ------------------------------------------------------------------------------------------------ any K
constexpr int GT = 256;

__global__ void __launch_bounds__(GT) prune_generic_kernel(const PruneOp* __restrict__ ops, int tiles, int tile_p,
    int K, int C, int L, const double* __restrict__ P, const uint8_t* __restrict__ tips,
    double* __restrict__ partials, int32_t* __restrict__ scale_exp)
{
    extern __shared__ double sm[];
    const int KK = K * K;
    double* Pm = sm;                                  // [2][K*K]
    double* ch_t = Pm + 2 * (size_t)KK;               // [2][tile_p][K]
    double* out = ch_t + 2 * (size_t)tile_p * K;      // [C][tile_p][K]
    double* scl = out + (size_t)C * tile_p * K;       // [tile_p]
    int* st = reinterpret_cast<int*>(scl + tile_p);   // [2][tile_p] tip states
    const PruneOp op = ops[blockIdx.x / tiles];
    const int tid = threadIdx.x;
    const int p0 = (blockIdx.x % tiles) * tile_p;
    const int np = min(tile_p, L - p0);

    for (int ch = 0; ch < 2; ch++)
        if (op.child_is_tip[ch])
            for (int p = tid; p < np; p += GT) st[ch * tile_p + p] = tips[(size_t)op.child[ch] * L + p0 + p];

    for (int c = 0; c < C; c++) {
        __syncthreads();
        for (int ch = 0; ch < 2; ch++) {
            const double* src = P + ((size_t)op.child[ch] * C + c) * KK;
            for (int idx = tid; idx < KK; idx += GT) Pm[ch * KK + idx] = src[idx];
            if (!op.child_is_tip[ch]) {
                const double* cs = partials + (((size_t)op.cpidx[ch] * C + c) * L + p0) * K;
                for (int idx = tid; idx < np * K; idx += GT) ch_t[(size_t)ch * tile_p * K + idx] = cs[idx];
            }
        }
        __syncthreads();
        for (int idx = tid; idx < np * K; idx += GT) {
            const int p = idx / K, i = idx % K;
            double prod = 1.0;
            for (int ch = 0; ch < 2; ch++) {
                const double* row = Pm + ch * KK + i * K;
                double a;
                if (op.child_is_tip[ch]) {
                    const int s = st[ch * tile_p + p];
                    a = s < K ? row[s] : 1.0;
                } else {
                    const double* v = ch_t + ((size_t)ch * tile_p + p) * K;
                    a = 0.0;
                    for (int j = 0; j < K; j++) a = fma(row[j], v[j], a);
                }
                prod *= a;
            }
            out[((size_t)c * tile_p + p) * K + i] = prod;
        }
    }
    __syncthreads();
    // per-pattern maximum over (category, state): 8 lanes per pattern
    for (int pb = 0; pb < np; pb += GT / 8) {
        const int p = pb + tid / 8, sub = tid & 7;
        double m = 0.0;
        if (p < np)
            for (int c = 0; c < C; c++)
                for (int i = sub; i < K; i += 8) m = fmax(m, out[((size_t)c * tile_p + p) * K + i]);
        for (int o = 4; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (p < np && sub == 0) {
            int ex = 0;
            for (int ch = 0; ch < 2; ch++)
                if (!op.child_is_tip[ch]) ex += scale_exp[(size_t)op.cpidx[ch] * L + p0 + p];
            double sc = 1.0;
            if (m > 0.0 && m < 1.7e308) {
                const int e = exponent_of(m);
                if (e > -1000) { sc = pow2_neg(e); ex += e; }
            }
            scl[p] = sc;
            scale_exp[(size_t)op.pidx * L + p0 + p] = ex;
        }
    }
    __syncthreads();
    for (int c = 0; c < C; c++) {
        double* dst = partials + (((size_t)op.pidx * C + c) * L + p0) * K;
        for (int idx = tid; idx < np * K; idx += GT) dst[idx] = out[(size_t)c * tile_p * K + idx] * scl[idx / K];
    }
}

// ------------------------------------------------------------------------------------------------ a6
__global__ void __launch_bounds__(256) root_site_kernel(int K, int C, int L, int root_pidx, int root_node,
    const double* __restrict__ partials, const int32_t* __restrict__ scale_exp, const double* __restrict__ freqs,
    const int32_t* __restrict__ e_hi, const double* __restrict__ root_freqs, const double* __restrict__ weights,
    const double* __restrict__ pattern_wt, double* __restrict__ site_lnl, double* __restrict__ block_sums,
    int32_t* __restrict__ status)
{
    __shared__ double red[8];
    const int tid = threadIdx.x;
    const int p = blockIdx.x * 256 + tid;
    const double* rf = root_freqs ? root_freqs : freqs + (size_t)e_hi[root_node] * K;   // reading A9
    double contrib = 0.0;
    if (p < L) {
        double site = 0.0;
        for (int c = 0; c < C; c++) {
            const double* v = partials + (((size_t)root_pidx * C + c) * L + p) * K;
            double s = 0.0;
            for (int i = 0; i < K; i++) s = fma(rf[i], v[i], s);
            site = fma(weights[c], s, site);
        }
        if (!(site > 0.0) || !(site < 1.7e308)) atomicOr(status, EPX_ST_BAD_SITE);
        const double ln = log(site) + (double)scale_exp[(size_t)root_pidx * L + p] * 0.6931471805599453094;
        site_lnl[p] = ln;
        contrib = pattern_wt[p] * ln;
    }
    for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
    if ((tid & 31) == 0) red[tid >> 5] = contrib;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; w++) t += red[w];
        block_sums[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(256) final_sum_kernel(int n, const double* __restrict__ block_sums,
                                                        double* __restrict__ lnl)
{
    __shared__ double red[8];
    const int tid = threadIdx.x;
    double t = 0.0;
    for (int i = tid; i < n; i += 256) t += block_sums[i];
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if ((tid & 31) == 0) red[tid >> 5] = t;
    __syncthreads();
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; w++) s += red[w];
        *lnl = s;
    }
}

size_t generic_smem(int K, int C, int tile_p)
{
    return sizeof(double) * (2 * (size_t)K * K + 2 * (size_t)tile_p * K + (size_t)C * tile_p * K + tile_p) +
           sizeof(int) * 2 * tile_p;
}

template <int C>
void launch_prune4(const PruneOp* ops, int nops, int L, const DevBuffers& d, cudaStream_t s)
{
    const int tiles = (L + 255) / 256;
    prune4_kernel<C><<<nops * tiles, 256, 0, s>>>(ops, tiles, L, d.P, d.tips, d.partials, d.scale_exp);
}

}  // namespace

int prune_tile(int K, int C)
{
    int t = 32;
    while (t > 1 && generic_smem(K, C, t) > 200 * 1024) t >>= 1;
    return t;
}

int prune_init_attributes()
{
    return cudaFuncSetAttribute(prune_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) == cudaSuccess ? 0 : -1;
}

int launch_pruning(const epx_ctx* c, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    const int K = c->K, C = c->C, L = c->L;
    int launched = 0;
    const int n_levels = (int)c->level_off.size() - 1;
    for (int l = 0; l < n_levels; l++) {
        const int first = c->level_off[l], nops = c->level_off[l + 1] - first;
        if (nops == 0) continue;
        const PruneOp* ops = d.ops + first;
        if (K == 4 && c->prune_kernel != 1) {
            switch (C) {
                case 1: launch_prune4<1>(ops, nops, L, d, s); break;
                case 2: launch_prune4<2>(ops, nops, L, d, s); break;
                case 3: launch_prune4<3>(ops, nops, L, d, s); break;
                case 4: launch_prune4<4>(ops, nops, L, d, s); break;
                case 5: launch_prune4<5>(ops, nops, L, d, s); break;
                case 6: launch_prune4<6>(ops, nops, L, d, s); break;
                case 7: launch_prune4<7>(ops, nops, L, d, s); break;
                default: launch_prune4<8>(ops, nops, L, d, s); break;
            }
        } else {
            const int tile_p = prune_tile(K, C);
            const int tiles = (L + tile_p - 1) / tile_p;
            prune_generic_kernel<<<nops * tiles, GT, generic_smem(K, C, tile_p), s>>>(ops, tiles, tile_p, K, C, L, d.P,
                                                                                      d.tips, d.partials, d.scale_exp);
        }
        launched++;
    }
    return cudaGetLastError() == cudaSuccess ? launched : -1;
}

int launch_root_reduction(const epx_ctx* c, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    const int blocks = c->reduce_blocks;
    const int root_pidx = c->node_pidx[c->root];
    root_site_kernel<<<blocks, 256, 0, s>>>(c->K, c->C, c->L, root_pidx, c->root, d.partials, d.scale_exp, d.freqs,
                                            d.e_hi, c->has_root_freqs ? d.root_freqs : nullptr, d.weights,
                                            d.pattern_wt, d.site_lnl, d.block_sums, d.status);
    final_sum_kernel<<<1, 256, 0, s>>>(blocks, d.block_sums, d.lnl);
    return cudaGetLastError() == cudaSuccess ? 2 : -1;
}
