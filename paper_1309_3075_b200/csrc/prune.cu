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
//   prune4_dfs_kernel<G>  K == 4 (default): patterns are independent, so a warp that owns a tile of patterns can walk the
//                      WHOLE tree by itself, depth first, with no inter-CTA synchronisation and no launch per level.
//                      One thread per (pattern, category); a child's partial vector is either in registers (the
//                      operation just finished) or in a per-warp shared-memory stack (<= log2 N + 1 slots, host-planned),
//                      so partials are never re-read from HBM: each node's [L][C][4] block is written once (256-bit
//                      streaming stores) and the only reads are tip states and the 4x4 matrices, both staged three
//                      operations ahead with cp.async.  HBM traffic = the partials written, half the level-by-level
//                      scheme's.
//   prune4_kernel<C>   K == 4, EPX_OPT_PRUNE_KERNEL = 2: the level-by-level scheme (one launch per post-order level,
//                      one thread per pattern, child partials re-read with 256-bit loads); kept for comparison.
//   prune_generic_kernel  any K <= 64: one CTA per (node, tile of patterns); per category the two K x K matrices
//                      and the child tiles are staged in shared memory, DFMA mat-vec products.
//   root_site_kernel / final_sum_kernel  per-pattern ln-likelihood, deterministic two-stage weighted sum.
#include "epx_internal.h"
#include <cooperative_groups.h>

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
__global__ void __launch_bounds__(256) prune4_kernel(const PruneOp* __restrict__ ops, int tiles, int L, int Lp,
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
            const int s = tips[(size_t)op.child[ch] * Lp + p];
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


// ------------------------------------------------------------------------------------------------ K == 4, depth first
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(smem_addr(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_addr(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

#ifndef EPX_DFS_STAGES
#define EPX_DFS_STAGES 3
#endif
constexpr int DFS_STAGES = EPX_DFS_STAGES;   // matrix staging ring: operation k+STAGES-1 is in flight while operation k computes
constexpr int DFS_PSTRIDE = 20;        // doubles per staged 4x4 matrix: 160 B = 40 banks, so 4 categories never share a bank
__host__ __device__ constexpr int dfs_lanes_of(int C) { return C <= 1 ? 1 : C <= 2 ? 2 : C <= 4 ? 4 : 8; }
__host__ __device__ constexpr int dfs_stage_bytes(int G) { return 2 * G * DFS_PSTRIDE * 8; }

__device__ __forceinline__ void matvec4(const double* __restrict__ Pm, const double (&v)[4], double (&f)[4])
{
#pragma unroll
    for (int i = 0; i < 4; i++) {
        const double2 r01 = *reinterpret_cast<const double2*>(Pm + i * 4), r23 = *reinterpret_cast<const double2*>(Pm + i * 4 + 2);
        f[i] = fma(r23.y, v[3], fma(r23.x, v[2], fma(r01.y, v[1], r01.x * v[0])));
    }
}

// One warp per (piece of the tree, tile of PPL * 32/G patterns); lane = PPL x (pattern, category), G = lanes per
// pattern = C rounded up to a power of 2, PPL = patterns per lane (the per-operation overhead -- descriptor decode,
// staging, branches -- is paid once for PPL state vectors, and the PPL vectors are independent instruction streams).
// Inputs are fetched long before they are needed, so the walk never waits on HBM:
//   - operation descriptors and tip states: every 32 operations lane j loads descriptor j of the NEXT block of 32 and
//     that operation's tip bytes for the warp's patterns into registers; operation k reads them with warp shuffles;
//   - the children's 4x4 matrices: cp.async into a shared-memory ring, DFS_STAGES - 1 operations ahead.
// Shared memory per warp: DFS_STAGES x [2 children][G][20] doubles, then the stack [depth][PPL][2 halves][32 lanes]
// double2 + [depth][PPL][32] exponents.  A lane only ever touches its own stack column: no synchronisation.
template <int C, int PPL>
__global__ void __launch_bounds__(32) prune4_dfs_kernel(const DfsOp* __restrict__ ops, const DfsPiece* __restrict__ pieces,
    int tiles, int L, int Lp, int depth, const double* __restrict__ P, const uint8_t* __restrict__ tips,
    double* __restrict__ partials, int32_t* __restrict__ scale_exp)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    constexpr int G = dfs_lanes_of(C);
    constexpr int PL = 32 / G;                      // patterns per warp and per u
    constexpr int PW = PPL * PL;                    // patterns per warp
    constexpr int TW = (PW + 3) / 4;                // 32-bit words of tip states per child
    constexpr int SB = dfs_stage_bytes(G);
    constexpr int NCH = (16 * C + 31) / 32;         // 16-byte chunks of the two children's matrices per lane
    constexpr unsigned FULL = 0xffffffffu;
    double2* stack = reinterpret_cast<double2*>(smraw + DFS_STAGES * SB);     // [depth][PPL][2][32]: conflict-free rows
    int* stack_ex = reinterpret_cast<int*>(stack + (size_t)depth * PPL * 64);
    const int lane = threadIdx.x;
    const int pl = lane / G, c = lane % G, cc = min(c, C - 1);
    const int piece = blockIdx.x / tiles, tile = blockIdx.x - piece * tiles;
    const int p0 = tile * PW;
    const DfsPiece pc = pieces[piece];
    const int n_ops = pc.end - pc.begin;
    ops += pc.begin;

    // per-lane constants of the matrix copies: chunk ch = lane + 32 q -> (child, category, 16-byte word)
    int cp_dst[NCH], cp_src[NCH];
    bool cp_child[NCH], cp_on[NCH];
#pragma unroll
    for (int q = 0; q < NCH; q++) {
        const int ch = lane + 32 * q;
        cp_on[q] = ch < 16 * C;
        cp_child[q] = ch >= 8 * C;
        const int r = ch - (cp_child[q] ? 8 * C : 0), cat = r >> 3, w = r & 7;
        cp_dst[q] = ((cp_child[q] ? G : 0) + cat) * (DFS_PSTRIDE * 8) + w * 16;
        cp_src[q] = cat * 16 + w * 2;
    }
    // 32-bit indexing in units of one state vector (32 B): (N-1) L C < 2^32 is checked by prune_uses_dfs
    const unsigned node_stride = (unsigned)L * C;
    bool live[PPL];
    double4a* out_base[PPL];
    int32_t* exp_base[PPL];
#pragma unroll
    for (int u = 0; u < PPL; u++) {
        const int p = p0 + u * PL + pl;
        live[u] = p < L && c < C;
        out_base[u] = reinterpret_cast<double4a*>(partials) + ((size_t)p * C + c);
        exp_base[u] = scale_exp + p;
    }
    const unsigned char* const tip_base = tips + p0;
    const double* const Pm_base = reinterpret_cast<const double*>(smraw) + cc * DFS_PSTRIDE;

    struct Block { int4 d; int2 h; uint32_t ta[TW], tb[TW]; };
    auto load_block = [&](int base) -> Block {      // lane j: descriptor base + j and its tip states
        Block b;
        b.d = make_int4(0, 0, 0, 0);
        b.h = make_int2(0, 0);
#pragma unroll
        for (int w = 0; w < TW; w++) { b.ta[w] = 0xffffffffu; b.tb[w] = 0xffffffffu; }
        const int k = base + lane;
        if (k < n_ops) {
            const int4* src = reinterpret_cast<const int4*>(ops + k);
            b.d = __ldg(src);
            const int4 h = __ldg(src + 1);
            b.h = make_int2(h.x, h.y);
            if ((b.d.w & 0xff) - 3 == EPX_DFS_TIP) {
                const uint32_t* t = reinterpret_cast<const uint32_t*>(tip_base + (size_t)b.d.x * Lp);
#pragma unroll
                for (int w = 0; w < TW; w++) b.ta[w] = __ldg(t + w);
            }
            if (((b.d.w >> 8) & 0xff) - 3 == EPX_DFS_TIP) {
                const uint32_t* t = reinterpret_cast<const uint32_t*>(tip_base + (size_t)b.d.y * Lp);
#pragma unroll
                for (int w = 0; w < TW; w++) b.tb[w] = __ldg(t + w);
            }
        }
        return b;
    };
    Block cb = load_block(0), nb = load_block(32);

    // stage the matrices of operation j (j in the current or the next block of 32) into ring buffer `buf`
    auto issue = [&](int j, int k, int buf) {
        const bool in_cur = (j >> 5) == (k >> 5);
        const int na = __shfl_sync(FULL, in_cur ? cb.d.x : nb.d.x, j & 31);
        const int nbn = __shfl_sync(FULL, in_cur ? cb.d.y : nb.d.y, j & 31);
        unsigned char* sb = smraw + buf * SB;
#pragma unroll
        for (int q = 0; q < NCH; q++)
            if (cp_on[q]) cp_async16(sb + cp_dst[q], P + (size_t)(cp_child[q] ? nbn : na) * (C * 16) + cp_src[q]);
    };
#pragma unroll
    for (int j = 0; j < DFS_STAGES - 1; j++) {
        if (j < n_ops) issue(j, 0, j);
        cp_async_commit();
    }

    // byte of this lane's pattern u inside the warp's tip words
    auto tip_of = [&](const uint32_t (&w)[TW], int u) -> int {
        const int idx = u * PL + pl;
        uint32_t word = w[0];
#pragma unroll
        for (int t = 1; t < TW; t++) if ((idx >> 2) == t) word = w[t];
        return (word >> (8 * (idx & 3))) & 0xff;
    };

    double cur[PPL][4];
    int cur_ex[PPL];
#pragma unroll
    for (int u = 0; u < PPL; u++) { cur[u][0] = cur[u][1] = cur[u][2] = cur[u][3] = 1.0; cur_ex[u] = 0; }
    int buf = 0;
    for (int k = 0; k < n_ops; k++) {
        if ((k & 31) == 0 && k > 0) { cb = nb; nb = load_block(k + 32); }
        __syncwarp();                               // every lane is done reading the buffer the next stage overwrites
        {
            int nbuf = buf + DFS_STAGES - 1; if (nbuf >= DFS_STAGES) nbuf -= DFS_STAGES;
            if (k + DFS_STAGES - 1 < n_ops) issue(k + DFS_STAGES - 1, k, nbuf);
            cp_async_commit();
        }
        const int src_lane = k & 31;
        const int pidx = __shfl_sync(FULL, cb.d.z, src_lane);
        const int code = __shfl_sync(FULL, cb.d.w, src_lane);
        const int srcA = (code & 0xff) - 3, srcB = ((code >> 8) & 0xff) - 3, out_slot = ((code >> 16) & 0xff) - 1;

        // operands that do not need the staged matrices yet
        uint32_t wa[TW], wb[TW];
        int pa = 0, pb = 0;
        if (srcA == EPX_DFS_TIP) {
#pragma unroll
            for (int w = 0; w < TW; w++) wa[w] = __shfl_sync(FULL, cb.ta[w], src_lane);
        } else if (srcA == EPX_DFS_HBM) {
            pa = __shfl_sync(FULL, cb.h.x, src_lane);
        }
        if (srcB == EPX_DFS_TIP) {
#pragma unroll
            for (int w = 0; w < TW; w++) wb[w] = __shfl_sync(FULL, cb.tb[w], src_lane);
        } else if (srcB == EPX_DFS_HBM) {
            pb = __shfl_sync(FULL, cb.h.y, src_lane);
        }

        cp_async_wait<DFS_STAGES - 1>();            // this lane's copies for operation k have landed ...
        __syncwarp();                               // ... and so have every other lane's
        const double* Pa = Pm_base + buf * (SB / 8);
        const double* Pb = Pa + G * DFS_PSTRIDE;
        // A matrix is read from shared memory ONCE per operation and serves the lane's PPL patterns from registers: the
        // register fill of the matrices is what saturates the L1 / shared-memory data pipe (profiles/r1_prune4_dfs_ncu.md)
        double fa[PPL][4];       // child A's contribution, then the product with child B's
        int ex[PPL];
#pragma unroll
        for (int u = 0; u < PPL; u++) ex[u] = 0;
        if (srcA == EPX_DFS_TIP) {
#pragma unroll
            for (int u = 0; u < PPL; u++) {
                const int sa = tip_of(wa, u);
#pragma unroll
                for (int i = 0; i < 4; i++) fa[u][i] = (sa < 4) ? Pa[i * 4 + sa] : 1.0;
            }
        } else {
            double m[16];
#pragma unroll
            for (int i = 0; i < 8; i++) { const double2 r = *reinterpret_cast<const double2*>(Pa + 2 * i); m[2 * i] = r.x; m[2 * i + 1] = r.y; }
#pragma unroll
            for (int u = 0; u < PPL; u++) {
                double va[4] = {1.0, 1.0, 1.0, 1.0};
                if (srcA == EPX_DFS_HBM) {
                    if (live[u]) {
                        const double4a v = ld256(reinterpret_cast<const double*>(out_base[u] + (unsigned)pa * node_stride));
                        va[0] = v.x; va[1] = v.y; va[2] = v.z; va[3] = v.w;
                        ex[u] += exp_base[u][(unsigned)pa * (unsigned)L];
                    }
                } else {
                    const double2 v01 = stack[(srcA * PPL + u) * 64 + lane], v23 = stack[(srcA * PPL + u) * 64 + 32 + lane];
                    va[0] = v01.x; va[1] = v01.y; va[2] = v23.x; va[3] = v23.y;
                    ex[u] += stack_ex[(srcA * PPL + u) * 32 + lane];
                }
#pragma unroll
                for (int i = 0; i < 4; i++)
                    fa[u][i] = fma(m[i * 4 + 3], va[3], fma(m[i * 4 + 2], va[2], fma(m[i * 4 + 1], va[1], m[i * 4] * va[0])));
            }
        }
        if (srcB == EPX_DFS_TIP) {
#pragma unroll
            for (int u = 0; u < PPL; u++) {
                const int sb2 = tip_of(wb, u);
#pragma unroll
                for (int i = 0; i < 4; i++) fa[u][i] *= (sb2 < 4) ? Pb[i * 4 + sb2] : 1.0;
            }
        } else {
            double m[16];
#pragma unroll
            for (int i = 0; i < 8; i++) { const double2 r = *reinterpret_cast<const double2*>(Pb + 2 * i); m[2 * i] = r.x; m[2 * i + 1] = r.y; }
#pragma unroll
            for (int u = 0; u < PPL; u++) {
                double vb[4] = {1.0, 1.0, 1.0, 1.0};
                if (srcB == EPX_DFS_PREV) {
#pragma unroll
                    for (int i = 0; i < 4; i++) vb[i] = cur[u][i];
                    ex[u] += cur_ex[u];
                } else if (live[u]) {
                    const double4a v = ld256(reinterpret_cast<const double*>(out_base[u] + (unsigned)pb * node_stride));
                    vb[0] = v.x; vb[1] = v.y; vb[2] = v.z; vb[3] = v.w;
                    ex[u] += exp_base[u][(unsigned)pb * (unsigned)L];
                }
#pragma unroll
                for (int i = 0; i < 4; i++)
                    fa[u][i] *= fma(m[i * 4 + 3], vb[3], fma(m[i * 4 + 2], vb[2], fma(m[i * 4 + 1], vb[1], m[i * 4] * vb[0])));
            }
        }
#pragma unroll
        for (int u = 0; u < PPL; u++) {
            // all values are >= 0, so the largest one has the largest high word: an integer max finds its exponent
            int hmax = 0;
#pragma unroll
            for (int i = 0; i < 4; i++) hmax = max(hmax, __double2hiint(fa[u][i]));
#pragma unroll
            for (int o = 1; o < G; o <<= 1) hmax = max(hmax, __shfl_xor_sync(FULL, hmax, o));
            double sc = 1.0;
            {
                const int e = (hmax >> 20) - 1023;      // hmax < 0x7fe00000: finite and far from overflow
                if (e > -1000 && hmax < 0x7fe00000) { sc = pow2_neg(e); ex[u] += e; }
            }
#pragma unroll
            for (int i = 0; i < 4; i++) cur[u][i] = fa[u][i] * sc;
            cur_ex[u] = ex[u];
            if (live[u]) st256(reinterpret_cast<double*>(out_base[u] + (unsigned)pidx * node_stride), cur[u][0], cur[u][1], cur[u][2], cur[u][3]);
            if (live[u] && c == 0) exp_base[u][(unsigned)pidx * (unsigned)L] = ex[u];
            if (out_slot >= 0) {
                stack[(out_slot * PPL + u) * 64 + lane] = make_double2(cur[u][0], cur[u][1]);
                stack[(out_slot * PPL + u) * 64 + 32 + lane] = make_double2(cur[u][2], cur[u][3]);
                stack_ex[(out_slot * PPL + u) * 32 + lane] = ex[u];
            }
        }
        if (++buf == DFS_STAGES) buf = 0;
    }
}


// ------------------------------------------------------------------------------------------------ K == 4, depth first, DMMA
// Same walk as prune4_dfs_kernel, but the 4x4 matrix-vector products of a warp's 8 patterns x C categories run on the
// FP64 tensor pipe.  Why: in the scalar kernel every lane needs both children's whole 4x4 matrices in registers (256 B per
// lane and node); that register fill plus the staging ring saturate the SM's L1 / shared-memory data pipe (ncu:
// l1tex__data_pipe_lsu_wavefronts = 93 % of the cycles, profiles/r1_prune4_dfs_ncu.md).  mma.sync.m8n8k4.f64 takes ONE double of
// the matrix and ONE of the vector per lane and does the broadcast inside the tensor core.  Per child and pair of
// categories (c, c'), transposed so that a lane ends up with one pattern:
//   A (8x4) = V_c^T resp. V_c'^T : row = pattern, column = child state j
//   B (4x8) = [P_c^T | 0] resp. [0 | P_c'^T] : row = j, column n = (category n >> 2, parent state i = n & 3)
//   D (8x8) = A_c B_lo + A_c' B_hi : row = pattern, column = (category, i)     (adding the zero columns is exact)
// Fragment owners (lane = 4 g + q): A[g][q], B[q][g], D[g][2q], D[g][2q+1] -- lane (g, q) holds, for pattern g, states
// 2 (q & 1), 2 (q & 1) + 1 of category 2 pr + (q >> 1), and needs, as the next A operand, state q of every category of
// pattern g.  Every result is therefore written once to a shared-memory slot (stack slot or one of two hand-over slots;
// XOR-swizzled so both access patterns are bank-conflict free) and once to HBM.  Tips enter as indicator rows (all-ones
// rows if missing), HBM-sourced children of the top piece as plain loads.  The 4x4 matrices are read straight from
// global memory (L1-resident: every warp on the SM walks the same nodes), one operation ahead, 4 doubles per lane.
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__host__ __device__ constexpr int mma_cpad(int C) { return C <= 4 ? 4 : 8; }
__host__ __device__ constexpr int mma_slot_doubles(int C) { return 8 * mma_cpad(C) * 4; }
// slot element (pattern, category, state): the category's low two bits are XORed with h(pattern & 3), h = {0, 2, 1, 3}
template <int C>
__device__ __forceinline__ int slot_addr(int pattern, int cat, int state)
{
    const int h = ((pattern & 1) << 1) | ((pattern >> 1) & 1);
    return pattern * (mma_cpad(C) * 4) + (((cat & ~3) | ((cat & 3) ^ h)) << 2) + state;
}

template <int C>
__global__ void __launch_bounds__(32) prune4_mma_kernel(const DfsOp* __restrict__ ops, const DfsPiece* __restrict__ pieces,
    int tiles, int L, int Lp, int depth, const double* __restrict__ P, const uint8_t* __restrict__ tips,
    double* __restrict__ partials, int32_t* __restrict__ scale_exp)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    constexpr int NP = (C + 1) / 2;                 // category pairs
    constexpr int SLOT = mma_slot_doubles(C);
    constexpr unsigned FULL = 0xffffffffu;
    double* slots = reinterpret_cast<double*>(smraw);                              // [depth + 2][SLOT]
    int* slot_ex = reinterpret_cast<int*>(slots + (size_t)(depth + 2) * SLOT);     // [depth + 2][8]
    const int lane = threadIdx.x, g = lane >> 2, q = lane & 3, hi = g >> 2, sp = q & 1;
    const double m_lo = hi ? 0.0 : 1.0, m_hi = hi ? 1.0 : 0.0;
    const int piece = blockIdx.x / tiles, tile = blockIdx.x - piece * tiles;
    const int p0 = tile * 8;
    const DfsPiece pc = pieces[piece];
    const int n_ops = pc.end - pc.begin;
    ops += pc.begin;

    const unsigned node_stride = (unsigned)L * C * 4;             // doubles per node (< 2^32); node offsets are 32 x 32 -> 64 bit
    const bool live = p0 + g < L;
    const double* const inA = partials + ((size_t)(p0 + g) * C) * 4 + q;          // A-operand view: pattern g, state q
    double* const outD = partials + ((size_t)(p0 + g) * C) * 4 + 2 * sp;          // D view: pattern g, states 2sp, 2sp+1
    int32_t* const exp_g = scale_exp + p0 + g;
    int rd_addr[C], wr_addr[NP], pm_off[NP];
    bool cat_ok[NP];
#pragma unroll
    for (int cat = 0; cat < C; cat++) rd_addr[cat] = slot_addr<C>(g, cat, q);
#pragma unroll
    for (int pr = 0; pr < NP; pr++) {
        const int cat_l = 2 * pr + (q >> 1);                      // category this lane's D columns belong to
        cat_ok[pr] = cat_l < C;
        wr_addr[pr] = slot_addr<C>(g, min(cat_l, C - 1), 2 * sp);
        pm_off[pr] = min(2 * pr + hi, C - 1) * 16 + (g & 3) * 4 + q;        // B fragment: P[cat][i = g & 3][j = q]
    }

    struct Block { int4 d; int2 h; uint32_t ta[2], tb[2]; };
    auto load_block = [&](int base) -> Block {      // lane j: descriptor base + j and its tip states (8 patterns = 2 words)
        Block b;
        b.d = make_int4(0, 0, 0, 0);
        b.h = make_int2(0, 0);
        b.ta[0] = b.ta[1] = b.tb[0] = b.tb[1] = 0xffffffffu;
        const int k = base + lane;
        if (k < n_ops) {
            const int4* src = reinterpret_cast<const int4*>(ops + k);
            b.d = __ldg(src);
            const int4 h = __ldg(src + 1);
            b.h = make_int2(h.x, h.y);
            if ((b.d.w & 0xff) - 3 == EPX_DFS_TIP) {
                const uint2 t = __ldg(reinterpret_cast<const uint2*>(tips + p0 + (size_t)b.d.x * Lp));
                b.ta[0] = t.x; b.ta[1] = t.y;
            }
            if (((b.d.w >> 8) & 0xff) - 3 == EPX_DFS_TIP) {
                const uint2 t = __ldg(reinterpret_cast<const uint2*>(tips + p0 + (size_t)b.d.y * Lp));
                b.tb[0] = t.x; b.tb[1] = t.y;
            }
        }
        return b;
    };
    Block cb = load_block(0), nb = load_block(32);

    // B fragments (matrix entries) of operation j, j in the current or the next block of 32
    auto load_frags = [&](int j, int k, double (&fa)[NP], double (&fb)[NP]) {
        const bool in_cur = (j >> 5) == (k >> 5);
        const int na = __shfl_sync(FULL, in_cur ? cb.d.x : nb.d.x, j & 31);
        const int nbn = __shfl_sync(FULL, in_cur ? cb.d.y : nb.d.y, j & 31);
        const double* Pa = P + (size_t)na * (C * 16);
        const double* Pb = P + (size_t)nbn * (C * 16);
#pragma unroll
        for (int pr = 0; pr < NP; pr++) { fa[pr] = __ldg(Pa + pm_off[pr]); fb[pr] = __ldg(Pb + pm_off[pr]); }
    };

    // one child's contribution in D layout: f[pr][e] = state 2sp + e of category 2pr + (q >> 1), pattern g
    auto child = [&](int src, const double (&bf)[NP], uint32_t t0, uint32_t t1, int hbm_pidx, int prev_slot,
                     double (&f)[NP][2], int& ex) {
        double a[C];
        if (src == EPX_DFS_TIP) {
            const int s = ((hi ? t1 : t0) >> (8 * (g & 3))) & 0xff;           // tip state of pattern g
            const double v = s < 4 ? (s == q ? 1.0 : 0.0) : 1.0;
#pragma unroll
            for (int cat = 0; cat < C; cat++) a[cat] = v;
        } else if (src == EPX_DFS_HBM) {
            const double* base = inA + (unsigned long long)(unsigned)hbm_pidx * node_stride;
#pragma unroll
            for (int cat = 0; cat < C; cat++) a[cat] = live ? base[cat * 4] : 1.0;
            ex += live ? exp_g[(size_t)hbm_pidx * L] : 0;
        } else {
            const int sl = src == EPX_DFS_PREV ? prev_slot : src;
            const double* S = slots + sl * SLOT;
#pragma unroll
            for (int cat = 0; cat < C; cat++) a[cat] = S[rd_addr[cat]];
            ex += slot_ex[sl * 8 + g];
        }
#pragma unroll
        for (int pr = 0; pr < NP; pr++) {
            const double b_lo = bf[pr] * m_lo, b_hi = bf[pr] * m_hi;      // zero the other category's columns (0 * finite = 0)
            double d0 = 0.0, d1 = 0.0;
            dmma884(d0, d1, a[2 * pr], b_lo);
            if (2 * pr + 1 < C) dmma884(d0, d1, a[2 * pr + 1], b_hi);
            f[pr][0] = d0; f[pr][1] = d1;
        }
    };

    auto step = [&](int k, const double (&pa_cur)[NP], const double (&pb_cur)[NP], double (&pa_nxt)[NP], double (&pb_nxt)[NP]) {
        if ((k & 31) == 0 && k > 0) { cb = nb; nb = load_block(k + 32); }
        if (k + 1 < n_ops) load_frags(k + 1, k, pa_nxt, pb_nxt);
        const int src_lane = k & 31;
        const int pidx = __shfl_sync(FULL, cb.d.z, src_lane);
        const int code = __shfl_sync(FULL, cb.d.w, src_lane);
        const int srcA = (code & 0xff) - 3, srcB = ((code >> 8) & 0xff) - 3, out_slot = ((code >> 16) & 0xff) - 1;
        uint32_t ta0 = 0, ta1 = 0, tb0 = 0, tb1 = 0;
        int pa = 0, pb = 0;
        if (srcA == EPX_DFS_TIP) { ta0 = __shfl_sync(FULL, cb.ta[0], src_lane); ta1 = __shfl_sync(FULL, cb.ta[1], src_lane); }
        else if (srcA == EPX_DFS_HBM) pa = __shfl_sync(FULL, cb.h.x, src_lane);
        if (srcB == EPX_DFS_TIP) { tb0 = __shfl_sync(FULL, cb.tb[0], src_lane); tb1 = __shfl_sync(FULL, cb.tb[1], src_lane); }
        else if (srcB == EPX_DFS_HBM) pb = __shfl_sync(FULL, cb.h.y, src_lane);

        __syncwarp();                               // the slot writes of operation k-1 are visible
        double fa[NP][2], fb[NP][2];
        int ex = 0;
        const int prev_slot = depth + ((k + 1) & 1), my_scratch = depth + (k & 1);
        child(srcA, pa_cur, ta0, ta1, pa, prev_slot, fa, ex);
        child(srcB, pb_cur, tb0, tb1, pb, prev_slot, fb, ex);

        // all values are >= 0, so the largest one has the largest high word: an integer max finds its exponent
        int hmax = 0;
#pragma unroll
        for (int pr = 0; pr < NP; pr++) {
            fa[pr][0] *= fb[pr][0];
            fa[pr][1] *= fb[pr][1];
            if (cat_ok[pr]) hmax = max(hmax, max(__double2hiint(fa[pr][0]), __double2hiint(fa[pr][1])));
        }
        hmax = max(hmax, __shfl_xor_sync(FULL, hmax, 1));
        hmax = max(hmax, __shfl_xor_sync(FULL, hmax, 2));
        double sc = 1.0;
        {
            const int e = (hmax >> 20) - 1023;      // hmax < 0x7fe00000: finite and far from overflow
            if (e > -1000 && hmax < 0x7fe00000) { sc = pow2_neg(e); ex += e; }
        }
        const int dst = out_slot >= 0 ? out_slot : my_scratch;
        double* S = slots + dst * SLOT;
        double* o = outD + (unsigned long long)(unsigned)pidx * node_stride;
        __syncwarp();                               // every lane has fetched its operands (dst may be the slot just consumed)
#pragma unroll
        for (int pr = 0; pr < NP; pr++) {
            const double2 v = make_double2(fa[pr][0] * sc, fa[pr][1] * sc);
            if (cat_ok[pr]) {
                *reinterpret_cast<double2*>(S + wr_addr[pr]) = v;
                if (live) *reinterpret_cast<double2*>(o + (2 * pr + (q >> 1)) * 4) = v;
            }
        }
        if (q == 0) {
            slot_ex[dst * 8 + g] = ex;
            if (live) exp_g[(size_t)pidx * L] = ex;
        }
    };
    // (unrolling by two with the fragment sets swapping roles was measured slower: 90 registers, 1.00 vs 0.82 ms)
    double pa_cur[NP], pb_cur[NP], pa_nxt[NP], pb_nxt[NP];
    load_frags(0, 0, pa_cur, pb_cur);
    for (int k = 0; k < n_ops; k++) {
        step(k, pa_cur, pb_cur, pa_nxt, pb_nxt);
#pragma unroll
        for (int pr = 0; pr < NP; pr++) { pa_cur[pr] = pa_nxt[pr]; pb_cur[pr] = pb_nxt[pr]; }
    }
}

size_t mma_smem(int C, int depth) { return 8 * (size_t)(depth + 2) * mma_slot_doubles(C) + (size_t)(depth + 2) * 32; }

size_t dfs_smem(int G, int depth, int ppl) { return (size_t)DFS_STAGES * dfs_stage_bytes(G) + (size_t)depth * ppl * (128 * 8 + 32 * 4); }

// ------------------------------------------------------------------------------------------------ any K
// sum_j row[j] v[j] with four interleaved chains (j mod 4), combined as (a0 + a1) + (a2 + a3).  Shared by the level kernel
// and the few-pattern walk so that the two produce the same bits (an incremental re-evaluation uses the level kernel).
__device__ __forceinline__ double dot4(const double* __restrict__ row, const double* __restrict__ v, int K)
{
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int j = 0;
    for (; j + 4 <= K; j += 4) {
        a0 = fma(row[j], v[j], a0);
        a1 = fma(row[j + 1], v[j + 1], a1);
        a2 = fma(row[j + 2], v[j + 2], a2);
        a3 = fma(row[j + 3], v[j + 3], a3);
    }
    if (j < K) a0 = fma(row[j], v[j], a0);
    if (j + 1 < K) a1 = fma(row[j + 1], v[j + 1], a1);
    if (j + 2 < K) a2 = fma(row[j + 2], v[j + 2], a2);
    return (a0 + a1) + (a2 + a3);
}

// the same sum with the matrix row read at a stride (column i of the transposed copy): same chains, same bits
__device__ __forceinline__ double dot4s(const double* __restrict__ col, int stride, const double* __restrict__ v, int K)
{
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int j = 0;
    for (; j + 4 <= K; j += 4) {
        a0 = fma(col[j * stride], v[j], a0);
        a1 = fma(col[(j + 1) * stride], v[j + 1], a1);
        a2 = fma(col[(j + 2) * stride], v[j + 2], a2);
        a3 = fma(col[(j + 3) * stride], v[j + 3], a3);
    }
    if (j < K) a0 = fma(col[j * stride], v[j], a0);
    if (j + 1 < K) a1 = fma(col[(j + 1) * stride], v[j + 1], a1);
    if (j + 2 < K) a2 = fma(col[(j + 2) * stride], v[j + 2], a2);
    return (a0 + a1) + (a2 + a3);
}

// dot4s at a compile-time K (KT > 0): the same four chains in the same order, fully unrolled, every load at an immediate offset
template <int KT>
__device__ __forceinline__ double dot4t(const double* __restrict__ col, const double* __restrict__ v, int K)
{
    if (KT == 0) return dot4s(col, K, v, K);
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
#pragma unroll
    for (int j = 0; j + 4 <= KT; j += 4) {
        a0 = fma(col[j * KT], v[j], a0);
        a1 = fma(col[(j + 1) * KT], v[j + 1], a1);
        a2 = fma(col[(j + 2) * KT], v[j + 2], a2);
        a3 = fma(col[(j + 3) * KT], v[j + 3], a3);
    }
    constexpr int j = KT & ~3;
    if (j < KT) a0 = fma(col[j * KT], v[j], a0);
    if (j + 1 < KT) a1 = fma(col[(j + 1) * KT], v[j + 1], a1);
    if (j + 2 < KT) a2 = fma(col[(j + 2) * KT], v[j + 2], a2);
    return (a0 + a1) + (a2 + a3);
}

// PT[slot][c][j][i] = P[slot][c][i][j]: transposed copies for the few-pattern walk below, whose lane i reads row i of P -- from
// the row-major matrix that is a stride of K doubles between lanes (16-way bank conflicts at K = 24); from the transposed
// copy the lanes read consecutive words.
__global__ void __launch_bounds__(256) pt_copy_kernel(int K, const double* __restrict__ P, double* __restrict__ PT)
{
    __shared__ double tile[32][33];
    const double* src = P + (size_t)blockIdx.x * K * K;
    double* dst = PT + (size_t)blockIdx.x * K * K;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int i0 = 0; i0 < K; i0 += 32)
        for (int j0 = 0; j0 < K; j0 += 32) {
            for (int r = ty; r < 32; r += 8)
                tile[r][tx] = (i0 + r < K && j0 + tx < K) ? src[(i0 + r) * K + j0 + tx] : 0.0;
            __syncthreads();
            for (int r = ty; r < 32; r += 8)
                if (j0 + r < K && i0 + tx < K) dst[(j0 + r) * K + i0 + tx] = tile[tx][r];
            __syncthreads();
        }
}

constexpr int GT = 256;

__global__ void __launch_bounds__(GT) prune_generic_kernel(const PruneOp* __restrict__ ops, int tiles, int tile_p,
    int K, int C, int L, int Lp, const double* __restrict__ P, const uint8_t* __restrict__ tips,
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
            for (int p = tid; p < np; p += GT) st[ch * tile_p + p] = tips[(size_t)op.child[ch] * Lp + p0 + p];

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
                    a = dot4(row, v, K);
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

// ------------------------------------------------------------------------------------------------ 32 < K <= 64, DMMA
// Level kernel for codon-sized models: per (node, tile of 32 patterns) and category, each internal child contributes
// F[pattern][i] = sum_j V[pattern][j] P[i][j], a 32 x 64 x 64 product.  The scalar kernel reads two shared-memory operands
// per DFMA and sits at 7 % of the FP64 peak; here the products run on the FP64 tensor pipe (mma.sync.m8n8k4):
//   A (8x4) = V rows (patterns) x child states j,  B (4x8) = P^T (j x parent states i),  D (8x8) = F tile
// Warp w of 8: patterns 8 (w & 3) .. +8, parent states 32 (w >> 2) .. +32 (four n-tiles); 16 k-steps.  Shared-memory rows
// have a stride of 68 doubles (8 banks apart) so the 64-bit fragment loads of a half-warp never collide; the padding
// columns / rows 61..63 are zero.  Everything after the products (rescaling, stores) is the scalar kernel's code.
constexpr int MT = 256, M_TP = 32, M_LD = 68;

__global__ void __launch_bounds__(MT) prune64_mma_kernel(const PruneOp* __restrict__ ops, int tiles, int K, int C, int L,
    int Lp, const double* __restrict__ P, const uint8_t* __restrict__ tips, double* __restrict__ partials,
    int32_t* __restrict__ scale_exp)
{
    extern __shared__ double sm[];
    double* Pm = sm;                                   // [2][64][68]
    double* V = Pm + 2 * 64 * M_LD;                    // [2][32][68]
    double* out = V + 2 * M_TP * M_LD;                 // [C][32][K]
    double* scl = out + (size_t)C * M_TP * K;          // [32]
    int* st = reinterpret_cast<int*>(scl + M_TP);      // [2][32] tip states
    const PruneOp op = ops[blockIdx.x / tiles];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, q = lane & 3;
    const int p0 = (blockIdx.x % tiles) * M_TP;
    const int np = min(M_TP, L - p0);
    const int KK = K * K;
    const int mt = w & 3, nh = w >> 2;

    for (int ch = 0; ch < 2; ch++)
        if (op.child_is_tip[ch])
            for (int p = tid; p < M_TP; p += MT) st[ch * M_TP + p] = p < np ? tips[(size_t)op.child[ch] * Lp + p0 + p] : 255;

    for (int c = 0; c < C; c++) {
        __syncthreads();
        for (int ch = 0; ch < 2; ch++) {
            const double* src = P + ((size_t)op.child[ch] * C + c) * KK;
            for (int idx = tid; idx < 64 * 64; idx += MT) {
                const int i = idx >> 6, j = idx & 63;
                Pm[(ch * 64 + i) * M_LD + j] = (i < K && j < K) ? src[i * K + j] : 0.0;
            }
            if (!op.child_is_tip[ch]) {
                const double* cs = partials + (((size_t)op.cpidx[ch] * C + c) * L + p0) * K;
                for (int idx = tid; idx < M_TP * 64; idx += MT) {
                    const int p = idx >> 6, j = idx & 63;
                    V[(ch * M_TP + p) * M_LD + j] = (p < np && j < K) ? cs[p * K + j] : 0.0;
                }
            }
        }
        __syncthreads();
        double f[4][2];
#pragma unroll
        for (int t = 0; t < 4; t++) f[t][0] = f[t][1] = 1.0;
        for (int ch = 0; ch < 2; ch++) {
            const double* Pc = Pm + ch * 64 * M_LD;
            if (op.child_is_tip[ch]) {
                const int s = st[ch * M_TP + 8 * mt + g];
#pragma unroll
                for (int t = 0; t < 4; t++) {
                    const int i = 8 * (4 * nh + t) + 2 * q;
                    f[t][0] *= s < K ? Pc[i * M_LD + s] : 1.0;
                    f[t][1] *= s < K ? Pc[(i + 1) * M_LD + s] : 1.0;
                }
            } else {
                double acc[4][2];
#pragma unroll
                for (int t = 0; t < 4; t++) acc[t][0] = acc[t][1] = 0.0;
                const double* Arow = V + (ch * M_TP + 8 * mt + g) * M_LD + q;
                const double* Brow = Pc + (32 * nh + g) * M_LD + q;
#pragma unroll 4
                for (int kt = 0; kt < 16; kt++) {
                    const double a = Arow[4 * kt];
#pragma unroll
                    for (int t = 0; t < 4; t++) dmma884(acc[t][0], acc[t][1], a, Brow[8 * t * M_LD + 4 * kt]);
                }
#pragma unroll
                for (int t = 0; t < 4; t++) { f[t][0] *= acc[t][0]; f[t][1] *= acc[t][1]; }
            }
        }
        {
            const int p = 8 * mt + g;
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const int i = 8 * (4 * nh + t) + 2 * q;
                if (p < np && i < K) out[((size_t)c * M_TP + p) * K + i] = f[t][0];
                if (p < np && i + 1 < K) out[((size_t)c * M_TP + p) * K + i + 1] = f[t][1];
            }
        }
    }
    __syncthreads();
    // per-pattern maximum over (category, state): 8 lanes per pattern
    {
        const int p = tid / 8, sub = tid & 7;
        double m = 0.0;
        if (p < np)
            for (int c = 0; c < C; c++)
                for (int i = sub; i < K; i += 8) m = fmax(m, out[((size_t)c * M_TP + p) * K + i]);
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
        for (int idx = tid; idx < np * K; idx += MT) dst[idx] = out[(size_t)c * M_TP * K + idx] * scl[idx / K];
    }
}

// Same products, one CTA per CATEGORY: the C CTAs of a (node, pattern tile) form a thread-block cluster, each stages and
// multiplies its own category, and the per-pattern maximum over all categories (the rescaling is per (node, pattern),
// reading A12) is exchanged through distributed shared memory.  C times more CTAs per level and a C times shorter serial
// path per CTA: the upper levels of a 100-tip codon tree hold one to four nodes.
__global__ void __launch_bounds__(MT) prune64_cluster_kernel(const PruneOp* __restrict__ ops, int tiles, int K, int C, int L,
    int Lp, const double* __restrict__ P, const uint8_t* __restrict__ tips, double* __restrict__ partials,
    int32_t* __restrict__ scale_exp)
{
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ double sm[];
    double* Pm = sm;                                   // [64][68]  one child at a time: 68 KB per CTA, three CTAs per SM
    double* V = Pm + 64 * M_LD;                        // [32][68]
    double* out = V + M_TP * M_LD;                     // [32][K]
    double* mx = out + (size_t)M_TP * K;               // [32] this category's per-pattern maximum (read by the cluster)
    double* scl = mx + M_TP;                           // [32]
    int* st = reinterpret_cast<int*>(scl + M_TP);      // [32] tip states
    const int c = (int)cluster.block_rank();
    const int unit = blockIdx.x / C;
    const PruneOp op = ops[unit / tiles];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, q = lane & 3;
    const int p0 = (unit % tiles) * M_TP;
    const int np = min(M_TP, L - p0);
    const int KK = K * K;
    const int mt = w & 3, nh = w >> 2;

    double f[4][2];
#pragma unroll
    for (int t = 0; t < 4; t++) f[t][0] = f[t][1] = 1.0;
    for (int ch = 0; ch < 2; ch++) {
        if (ch) __syncthreads();                       // everyone is done with the first child's operands
        if (op.child_is_tip[ch])
            for (int p = tid; p < M_TP; p += MT) st[p] = p < np ? tips[(size_t)op.child[ch] * Lp + p0 + p] : 255;
        // all global loads of the staging are issued before the first shared-memory store (one L2 round trip, not sixteen)
        const double* src = P + ((size_t)op.child[ch] * C + c) * KK;
        const double* cs = partials + (((size_t)op.cpidx[ch] * C + c) * L + p0) * K;
        const bool internal = !op.child_is_tip[ch];
        double tp[64 * 64 / MT], tv[M_TP * 64 / MT];
#pragma unroll
        for (int t = 0; t < 64 * 64 / MT; t++) {
            const int idx = tid + t * MT, i = idx >> 6, j = idx & 63;
            tp[t] = (i < K && j < K) ? src[i * K + j] : 0.0;
        }
#pragma unroll
        for (int t = 0; t < M_TP * 64 / MT; t++) {
            const int idx = tid + t * MT, p = idx >> 6, j = idx & 63;
            tv[t] = (internal && p < np && j < K) ? cs[p * K + j] : 0.0;
        }
#pragma unroll
        for (int t = 0; t < 64 * 64 / MT; t++) {
            const int idx = tid + t * MT;
            Pm[(idx >> 6) * M_LD + (idx & 63)] = tp[t];
        }
        if (internal) {
#pragma unroll
            for (int t = 0; t < M_TP * 64 / MT; t++) {
                const int idx = tid + t * MT;
                V[(idx >> 6) * M_LD + (idx & 63)] = tv[t];
            }
        }
        __syncthreads();
        if (op.child_is_tip[ch]) {
            const int s = st[8 * mt + g];
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const int i = 8 * (4 * nh + t) + 2 * q;
                f[t][0] *= s < K ? Pm[i * M_LD + s] : 1.0;
                f[t][1] *= s < K ? Pm[(i + 1) * M_LD + s] : 1.0;
            }
        } else {
            double acc[4][2];
#pragma unroll
            for (int t = 0; t < 4; t++) acc[t][0] = acc[t][1] = 0.0;
            const double* Arow = V + (8 * mt + g) * M_LD + q;
            const double* Brow = Pm + (32 * nh + g) * M_LD + q;
#pragma unroll 4
            for (int kt = 0; kt < 16; kt++) {
                const double a = Arow[4 * kt];
#pragma unroll
                for (int t = 0; t < 4; t++) dmma884(acc[t][0], acc[t][1], a, Brow[8 * t * M_LD + 4 * kt]);
            }
#pragma unroll
            for (int t = 0; t < 4; t++) { f[t][0] *= acc[t][0]; f[t][1] *= acc[t][1]; }
        }
    }
    {
        const int p = 8 * mt + g;
#pragma unroll
        for (int t = 0; t < 4; t++) {
            const int i = 8 * (4 * nh + t) + 2 * q;
            if (p < np && i < K) out[(size_t)p * K + i] = f[t][0];
            if (p < np && i + 1 < K) out[(size_t)p * K + i + 1] = f[t][1];
        }
    }
    __syncthreads();
    {   // this category's per-pattern maximum: 8 lanes per pattern
        const int p = tid / 8, sub = tid & 7;
        double m = 0.0;
        if (p < np)
            for (int i = sub; i < K; i += 8) m = fmax(m, out[(size_t)p * K + i]);
        for (int o = 4; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (sub == 0) mx[p] = p < np ? m : 0.0;
    }
    cluster.sync();
    if (tid < M_TP) {
        const int p = tid;
        double m = 0.0;
        for (int r = 0; r < C; r++) m = fmax(m, cluster.map_shared_rank(mx, r)[p]);
        double sc = 1.0;
        int e = 0;
        if (m > 0.0 && m < 1.7e308) {
            const int ee = exponent_of(m);
            if (ee > -1000) { sc = pow2_neg(ee); e = ee; }
        }
        scl[p] = sc;
        if (c == 0 && p < np) {
            int ex = e;
            for (int ch = 0; ch < 2; ch++)
                if (!op.child_is_tip[ch]) ex += scale_exp[(size_t)op.cpidx[ch] * L + p0 + p];
            scale_exp[(size_t)op.pidx * L + p0 + p] = ex;
        }
    }
    __syncthreads();
    double* dst = partials + (((size_t)op.pidx * C + c) * L + p0) * K;
    for (int idx = tid; idx < np * K; idx += MT) dst[idx] = out[idx] * scl[idx / K];
    cluster.sync();          // nobody leaves while its maxima may still be read
}

size_t mma64_cluster_smem(int K) { return sizeof(double) * (64 * M_LD + M_TP * M_LD + (size_t)M_TP * K + 2 * M_TP) + sizeof(int) * M_TP; }

size_t mma64_smem(int K, int C) { return sizeof(double) * (2 * 64 * M_LD + 2 * M_TP * M_LD + (size_t)C * M_TP * K + M_TP) + sizeof(int) * 2 * M_TP; }

// ------------------------------------------------------------------------------------------------ few patterns, K <= 32
// A discrete trait observed at one site (PAPER.md L224 workload A: K = 7 locations; config 4: K = 24, L = 1): a tree level
// holds a handful of nodes and the level-by-level kernels are pure launch latency (config 4: 168 levels x 5 us).  The
// depth-first walk needs no level at all: one warp per (piece of the tree, pattern), lane i = parent state i, the
// children's vectors in a per-warp shared-memory stack (every result is parked: a dot product needs the whole vector),
// matrix rows straight from global memory (each lane its own row; the rows of the next operations are pulled into L1 while
// the current one computes), the per-(node, pattern) maximum by warp shuffles.  Partials keep the generic [node][C][L][K]
// layout.  The pieces (independent subtrees, then the top piece reading their roots from HBM) are the ones planned for
// the K = 4 walk.
constexpr int KD_MAXC = 8;

__device__ __forceinline__ void cp_async8(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_addr(dst)), "l"(src) : "memory");
}

// mbarrier + TMA 1-D bulk copy global -> shared for the staging ring of pruneK_dfs_kernel
__device__ __forceinline__ void kd_mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void kd_mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void kd_mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void kd_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_addr(dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}

constexpr int KD_STAGES = 3;

template <int KT, int CT>
__global__ void __launch_bounds__(32) pruneK_dfs_kernel(const DfsOp* __restrict__ ops, const DfsPiece* __restrict__ pieces,
    int K_rt, int C_rt, int L, int Lp, int depth, const double* __restrict__ P /* transposed copies, pt_copy_kernel */,
    const uint8_t* __restrict__ tips, double* __restrict__ partials, int32_t* __restrict__ scale_exp)
{
    extern __shared__ double kd_sm[];
    const int K = KT ? KT : K_rt;                                    // KT > 0: compile-time state count (unrolled dot products)
    const int C = CT ? CT : C_rt;                                    // CT > 0: compile-time category count (no loops over 8 predicated categories)
    constexpr int NCAT = CT ? CT : KD_MAXC;
    const int CK = C * K, KK = K * K, CKK = C * KK;
    const int stage_d = 2 * CKK + 2 * CK;                            // doubles per stage: both children's matrices + HBM vectors
    double* ring = kd_sm;                                            // [KD_STAGES][stage_d]
    double* slots = ring + (size_t)KD_STAGES * stage_d;              // [depth + 2][C * K]: stack + 2 hand-over slots
    int* slot_ex = reinterpret_cast<int*>(slots + (size_t)(depth + 2) * CK);    // [depth + 2]
    uint64_t* kbar = reinterpret_cast<uint64_t*>(slots + (size_t)(depth + 2) * CK + ((depth + 4 + 1) >> 1));   // [KD_STAGES]
    const bool bulk = ((CKK * 8) & 15) == 0;                         // matrices by TMA bulk copies (16-byte sizes and addresses)
    const int lane = threadIdx.x, i = min(lane, K - 1);
    const bool on = lane < K;
    const int piece = blockIdx.x / L, p = blockIdx.x - piece * L;
    const DfsPiece pc = pieces[piece];
    const int n_ops = pc.end - pc.begin;
    const int4* opv = reinterpret_cast<const int4*>(ops + pc.begin);

    // Everything an operation reads from global memory is fetched ahead of the dependency chain: descriptors four
    // operations ahead, tip states / exponents of HBM operands two ahead in registers, the children's matrices and the
    // HBM operands' vectors two ahead with cp.async into a shared-memory ring.
    auto load_desc = [&](int k, int4& d, int4& h) {
        d = make_int4(0, 0, 0, 0); h = d;
        if (k < n_ops) { d = __ldg(opv + 2 * k); h = __ldg(opv + 2 * k + 1); }
    };
    auto stage = [&](int k, const int4& d, const int4& h, int& sa, int& sb) {      // sa / sb: tip state, or exponent of an HBM operand
        sa = sb = 255;
        if (k < n_ops) {
            double* st = ring + (size_t)(k % KD_STAGES) * stage_d;
            const int srcA = (d.w & 0xff) - 3, srcB = ((d.w >> 8) & 0xff) - 3;
            const double* pa = P + (size_t)d.x * CKK;
            const double* pb = P + (size_t)d.y * CKK;
            if (bulk) {                                  // one lane, two bulk copies, completion on the stage's mbarrier
                if (lane == 0) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");       // the stage was read through the generic proxy
                    kd_mbar_expect_tx(&kbar[k % KD_STAGES], 2 * CKK * 8);
                    kd_bulk_g2s(st, pa, CKK * 8, &kbar[k % KD_STAGES]);
                    kd_bulk_g2s(st + CKK, pb, CKK * 8, &kbar[k % KD_STAGES]);
                }
            } else {
                for (int o = lane; o < CKK; o += 32) { cp_async8(st + o, pa + o); cp_async8(st + CKK + o, pb + o); }
            }
            if (srcA == EPX_DFS_TIP) sa = tips[(size_t)d.x * Lp + p];
            if (srcB == EPX_DFS_TIP) sb = tips[(size_t)d.y * Lp + p];
            if (srcA == EPX_DFS_HBM) {
                for (int o = lane; o < CK; o += 32)
                    cp_async8(st + 2 * CKK + o, partials + (((size_t)h.x * C + o / K) * L + p) * K + o % K);
                sa = scale_exp[(size_t)h.x * L + p];
            }
            if (srcB == EPX_DFS_HBM) {
                for (int o = lane; o < CK; o += 32)
                    cp_async8(st + 2 * CKK + CK + o, partials + (((size_t)h.y * C + o / K) * L + p) * K + o % K);
                sb = scale_exp[(size_t)h.y * L + p];
            }
        }
        cp_async_commit();
    };
    if (lane == 0) {
        for (int q = 0; q < KD_STAGES; q++) kd_mbar_init(&kbar[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    int4 d0, h0, d1, h1, d2, h2, d3, h3;
    load_desc(0, d0, h0); load_desc(1, d1, h1); load_desc(2, d2, h2); load_desc(3, d3, h3);
    int ta0, tb0, ta1, tb1;
    stage(0, d0, h0, ta0, tb0); stage(1, d1, h1, ta1, tb1);
    for (int k = 0; k < n_ops; k++) {
        const int4 d = d0;
        const int aux[2] = {ta0, tb0};
        d0 = d1; h0 = h1; d1 = d2; h1 = h2; d2 = d3; h2 = h3;
        load_desc(k + 4, d3, h3);
        ta0 = ta1; tb0 = tb1;
        __syncwarp();                                   // every lane is done with the ring buffer stage k+2 overwrites
        stage(k + 2, d1, h1, ta1, tb1);
        const int srcs[2] = {(d.w & 0xff) - 3, ((d.w >> 8) & 0xff) - 3};
        const int out_slot = ((d.w >> 16) & 0xff) - 1;
        const int prev_slot = depth + ((k + 1) & 1), dst = out_slot >= 0 ? out_slot : depth + (k & 1);
        cp_async_wait<2>();
        if (bulk) kd_mbar_wait(&kbar[k % KD_STAGES], (uint32_t)((k / KD_STAGES) & 1));
        __syncwarp();                                   // stage k has landed; the slot written by operation k-1 is visible
        const double* st = ring + (size_t)(k % KD_STAGES) * stage_d;
        double f[NCAT];
#pragma unroll
        for (int c = 0; c < NCAT; c++) f[c] = 1.0;
        int ex = 0;
        for (int ch = 0; ch < 2; ch++) {
            const int src = srcs[ch];
            const double* Pm = st + ch * CKK + i;                      // row i of P = column i of the staged transpose, category 0
            if (src == EPX_DFS_TIP) {
                const int s = aux[ch];
#pragma unroll
                for (int c = 0; c < NCAT; c++)
                    if (c < C) f[c] *= s < K ? Pm[c * KK + s * K] : 1.0;
                continue;
            }
            const double* v;
            if (src == EPX_DFS_HBM) {
                v = st + 2 * CKK + ch * CK;
                ex += aux[ch];
            } else {
                const int sl = src == EPX_DFS_PREV ? prev_slot : src;
                v = slots + (size_t)sl * CK;
                ex += slot_ex[sl];
            }
#pragma unroll
            for (int c = 0; c < NCAT; c++) {
                if (c >= C) break;
                const double* row = Pm + c * KK;
                const double* vc = v + c * K;
                f[c] *= dot4t<KT>(row, vc, K);         // the level kernel's summation order: incremental re-evaluation is bit-identical
            }
        }
        double m = 0.0;
#pragma unroll
        for (int c = 0; c < NCAT; c++)
            if (c < C && on) m = fmax(m, f[c]);
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        double sc = 1.0;
        if (m > 0.0 && m < 1.7e308) {
            const int e = exponent_of(m);
            if (e > -1000) { sc = pow2_neg(e); ex += e; }
        }
        __syncwarp();                                   // every lane has read its operands (dst may be a slot just consumed)
        double* S = slots + (size_t)dst * CK;
#pragma unroll
        for (int c = 0; c < NCAT; c++)
            if (c < C && on) {
                const double val = f[c] * sc;
                S[c * K + lane] = val;
                partials[(((size_t)d.z * C + c) * L + p) * K + lane] = val;
            }
        if (lane == 0) { slot_ex[dst] = ex; scale_exp[(size_t)d.z * L + p] = ex; }
    }
}

size_t kdfs_smem(int K, int C, int depth)
{
    return sizeof(double) * ((size_t)KD_STAGES * (2 * C * K * K + 2 * C * K) + (size_t)(depth + 2) * C * K) + sizeof(int) * (depth + 6) +
           sizeof(uint64_t) * KD_STAGES;
}

// ------------------------------------------------------------------------------------------------ a6
// Last-block-done final sum: every CTA publishes its partial sum, the CTA that arrives last adds them up in index order
// (deterministic: the order does not depend on which CTA is last) and re-arms the counter.  Saves the final_sum launch.
__device__ __forceinline__ void finish_sum(double block_total, int n_blocks, double* __restrict__ block_sums,
                                           double* __restrict__ lnl, int32_t* __restrict__ counter, double* red)
{
    __shared__ bool last;
    if (threadIdx.x == 0) {
        block_sums[blockIdx.x] = block_total;
        __threadfence();
        last = atomicAdd(counter, 1) == n_blocks - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double t = 0.0;
    for (int i = threadIdx.x; i < n_blocks; i += 256) t += __ldcg(block_sums + i);
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; w++) s += red[w];
        *lnl = s;
        *counter = 0;
    }
}

__global__ void __launch_bounds__(256) root_site_kernel(int K, int C, int L, size_t sc, size_t sp, int root_pidx, int root_node,
    const double* __restrict__ partials, const int32_t* __restrict__ scale_exp, const double* __restrict__ freqs,
    const int32_t* __restrict__ e_hi, const double* __restrict__ root_freqs, const double* __restrict__ weights,
    const double* __restrict__ pattern_wt, double* __restrict__ site_lnl, double* __restrict__ block_sums,
    int32_t* __restrict__ status, double* __restrict__ lnl)
{
    __shared__ double red[8];
    const int tid = threadIdx.x;
    const int p = blockIdx.x * 256 + tid;
    const double* rf = root_freqs ? root_freqs : freqs + (size_t)e_hi[root_node] * K;   // reading A9
    double contrib = 0.0;
    if (p < L) {
        double site = 0.0;
        for (int c = 0; c < C; c++) {
            const double* v = partials + (size_t)root_pidx * C * L * K + c * sc + p * sp;
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
    double t = 0.0;
    if (tid == 0)
        for (int w = 0; w < 8; w++) t += red[w];
    __syncthreads();
    finish_sum(t, gridDim.x, block_sums, lnl, status + 1, red);
}

// K > 8: one warp per pattern, lanes over the states (coalesced reads of the root vectors), eight patterns per CTA.
// exp_per_cat: the pruning kernel kept one scale exponent per (category, pattern) (prune_mma.cu): the categories are summed
// relative to the pattern's largest exponent (exact power-of-two factors).
__global__ void __launch_bounds__(256) root_site_warp_kernel(int K, int C, int L, size_t node_off, size_t sc, size_t sp, int exp_per_cat,
    int root_pidx, int root_node,
    const double* __restrict__ partials, const int32_t* __restrict__ scale_exp, const double* __restrict__ freqs,
    const int32_t* __restrict__ e_hi, const double* __restrict__ root_freqs, const double* __restrict__ weights,
    const double* __restrict__ pattern_wt, double* __restrict__ site_lnl, double* __restrict__ block_sums,
    int32_t* __restrict__ status, double* __restrict__ lnl)
{
    __shared__ double red[8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int p = blockIdx.x * 8 + w;
    const double* rf = root_freqs ? root_freqs : freqs + (size_t)e_hi[root_node] * K;   // reading A9
    double contrib = 0.0;
    if (p < L) {
        int emax = 0;
        if (exp_per_cat) {
            emax = scale_exp[((size_t)root_pidx * C) * L + p];
            for (int c = 1; c < C; c++) emax = max(emax, scale_exp[((size_t)root_pidx * C + c) * L + p]);
        } else {
            emax = scale_exp[(size_t)root_pidx * L + p];
        }
        double site = 0.0;
        for (int c = 0; c < C; c++) {               // per category: states in lane order, then a fixed butterfly
            const double* v = partials + node_off + c * sc + p * sp;
            double s = 0.0;
            for (int i = lane; i < K; i += 32) s = fma(rf[i], v[i], s);
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (exp_per_cat) s = scalbn(s, scale_exp[((size_t)root_pidx * C + c) * L + p] - emax);
            site = fma(weights[c], s, site);
        }
        if (lane == 0) {
            if (!(site > 0.0) || !(site < 1.7e308)) atomicOr(status, EPX_ST_BAD_SITE);
            const double ln = log(site) + (double)emax * 0.6931471805599453094;
            site_lnl[p] = ln;
            contrib = pattern_wt[p] * ln;
        }
    }
    if (lane == 0) red[w] = contrib;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int k = 0; k < 8; k++) t += red[k];
    __syncthreads();
    finish_sum(t, gridDim.x, block_sums, lnl, status + 1, red);
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
    prune4_kernel<C><<<nops * tiles, 256, 0, s>>>(ops, tiles, L, (L + 31) & ~31, d.P, d.tips, d.partials, d.scale_exp);
}

}  // namespace

int prune_tile(int K, int C)
{
    int t = 32;
    while (t > 1 && generic_smem(K, C, t) > 200 * 1024) t >>= 1;
    return t;
}

template <int C>
static int dfs_set_attr()
{
    if (cudaFuncSetAttribute(prune4_mma_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(prune4_dfs_kernel<C, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(prune4_dfs_kernel<C, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(prune4_dfs_kernel<C, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    return 0;
}

int prune_init_attributes()
{
    if (dfs_set_attr<1>() || dfs_set_attr<2>() || dfs_set_attr<3>() || dfs_set_attr<4>() || dfs_set_attr<5>() ||
        dfs_set_attr<6>() || dfs_set_attr<7>() || dfs_set_attr<8>()) return -1;
    if (prune_lane_init_attributes()) return -1;
    if (cudaFuncSetAttribute(prune64_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(pruneK_dfs_kernel<0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(pruneK_dfs_kernel<0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(pruneK_dfs_kernel<24, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(pruneK_dfs_kernel<24, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(prune64_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    return cudaFuncSetAttribute(prune_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) == cudaSuccess ? 0 : -1;
}

int dfs_patterns_per_lane(const epx_ctx* c)
{
    if (c->dfs_ppl == 1 || c->dfs_ppl == 2 || c->dfs_ppl == 4) return c->dfs_ppl;
    const int G = dfs_lanes_of(c->C);
    const long tiles1 = (c->L + 32 / G - 1) / (32 / G);      // warps per piece at one pattern per lane
    // measured on config 2 (1 250 tiles at one pattern per lane): 0.78 ms (1), 0.66 ms (2), 0.66 ms (4): the matrices are
    // read from shared memory once per lane and operation, whatever the number of patterns they serve
    return tiles1 >= 512 ? 2 : 1;
}

// walk for few patterns and K <= 32 (pruneK_dfs_kernel); generic partials layout
bool prune_wants_kdfs(const epx_ctx* c)
{
    return c->tree_mode && c->K != 4 && c->K <= 32 && c->C <= KD_MAXC && c->prune_kernel == 0 && (long)c->L * c->C <= 64 && c->N >= 8;
}
bool prune_uses_kdfs(const epx_ctx* c)
{
    return prune_wants_kdfs(c) && kdfs_smem(c->K, c->C, c->dfs_depth > 0 ? c->dfs_depth : 1) <= 100 * 1024;
}

// 8 < K <= 64 with enough patterns for 8-pattern tensor tiles: level kernel of prune_mma.cu
bool prune_uses_mma(const epx_ctx* c)
{
    return c->tree_mode && c->K > 8 && c->prune_kernel == 0 && !prune_uses_kdfs(c);
}

int dfs_tiles(const epx_ctx* c)
{
    if (c->K != 4) return c->L;                                // pruneK_dfs_kernel: one warp per pattern
    if (c->prune_kernel == 0) { const int pw = 32 * lane_patterns_per_lane(c); return (c->L + pw - 1) / pw; }
    if (c->prune_kernel == 3) return (c->L + 7) / 8;          // tensor-core walk: 8 patterns per warp
    const int pw = dfs_patterns_per_lane(c) * (32 / dfs_lanes_of(c->C));
    return (c->L + pw - 1) / pw;
}

bool prune_uses_lane(const epx_ctx* c)
{
    if (!(c->tree_mode && c->K == 4 && c->prune_kernel == 0)) return false;
    if ((double)(c->N - 1 + c->tip_cap) * c->L * c->C >= 4294967296.0) return false;       // 32-bit state-vector indices
    return lane_smem_bytes(c, c->dfs_depth > 0 ? c->dfs_depth : 1) <= 227 * 1024;
}

bool prune_uses_dfs(const epx_ctx* c)
{
    if (!(c->tree_mode && c->K == 4 && (c->prune_kernel == 5 || c->prune_kernel == 3))) return false;
    const int depth = c->dfs_depth > 0 ? c->dfs_depth : 1;
    if (c->prune_kernel == 3) return (double)c->L * c->C * 4 < 4294967296.0 && mma_smem(c->C, depth) <= 227 * 1024;
    if ((double)(c->N - 1 + c->tip_cap) * c->L * c->C >= 4294967296.0) return false;
    return dfs_smem(dfs_lanes_of(c->C), depth, dfs_patterns_per_lane(c)) <= 227 * 1024;
}

template <int C, int PPL>
static void launch_dfs2(const epx_ctx* c, const DfsOp* ops, const DfsPiece* pieces, int n_pieces, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    const int pw = PPL * (32 / dfs_lanes_of(C));
    const int tiles = (c->L + pw - 1) / pw;
    prune4_dfs_kernel<C, PPL><<<n_pieces * tiles, 32, dfs_smem(dfs_lanes_of(C), c->dfs_depth, PPL), s>>>(ops,
        pieces, tiles, c->L, c->Lp, c->dfs_depth, d.P, d.tips, d.partials, d.scale_exp);
}

template <int C>
static void launch_dfs(const epx_ctx* c, const DfsOp* ops, const DfsPiece* pieces, int n_pieces, cudaStream_t s, bool top)
{
    // the top piece is a few dozen operations whose operands come from HBM: one pattern per lane doubles the warps that
    // hide that latency (measured 41 -> 20 us on config 2)
    if (top && c->prune_kernel == 5 && c->dfs_ppl == 0) { launch_dfs2<C, 1>(c, ops, pieces, n_pieces, s); return; }
    if (c->prune_kernel == 3) {
        const DevBuffers& d = c->d;
        const int tiles = dfs_tiles(c);
        prune4_mma_kernel<C><<<n_pieces * tiles, 32, mma_smem(C, c->dfs_depth), s>>>(ops, pieces, tiles,
            c->L, c->Lp, c->dfs_depth, d.P, d.tips, d.partials, d.scale_exp);
        return;
    }
    switch (dfs_patterns_per_lane(c)) {
        case 1: launch_dfs2<C, 1>(c, ops, pieces, n_pieces, s); break;
        case 2: launch_dfs2<C, 2>(c, ops, pieces, n_pieces, s); break;
        default: launch_dfs2<C, 4>(c, ops, pieces, n_pieces, s); break;
    }
}

static void launch_dfs_any(const epx_ctx* c, const DfsOp* ops, const DfsPiece* pieces, int count, cudaStream_t s, bool top)
{
    switch (c->C) {
        case 1: launch_dfs<1>(c, ops, pieces, count, s, top); break;
        case 2: launch_dfs<2>(c, ops, pieces, count, s, top); break;
        case 3: launch_dfs<3>(c, ops, pieces, count, s, top); break;
        case 4: launch_dfs<4>(c, ops, pieces, count, s, top); break;
        case 5: launch_dfs<5>(c, ops, pieces, count, s, top); break;
        case 6: launch_dfs<6>(c, ops, pieces, count, s, top); break;
        case 7: launch_dfs<7>(c, ops, pieces, count, s, top); break;
        default: launch_dfs<8>(c, ops, pieces, count, s, top); break;
    }
}

// Launch 1: the bottom pieces (independent subtrees); launch 2: the top piece, which reads their roots from HBM.
static int launch_pruning_dfs(const epx_ctx* c, cudaStream_t s)
{
    int launched = 0;
    const int total = (int)c->dfs_pieces.size();
    for (int pass = 0; pass < 2; pass++) {
        const int first = pass == 0 ? 0 : c->dfs_bottom, count = pass == 0 ? c->dfs_bottom : total - c->dfs_bottom;
        if (count <= 0) continue;
        const bool last_launch = pass == 1 || total == c->dfs_bottom;                 // the root's piece is the last one of this launch
        if (prune_uses_lane(c)) launch_prune4_lane(c, c->d.dfs_ops, c->d.dfs_pieces + first, count, s, pass == 1, last_launch && prune_root_fused(c));
        else launch_dfs_any(c, c->d.dfs_ops, c->d.dfs_pieces + first, count, s, pass == 1);
        launched++;
    }
    return cudaGetLastError() == cudaSuccess ? launched : -1;
}

// one level of the level-by-level kernels: `nops` operations whose children are complete
static void launch_level(const epx_ctx* c, const PruneOp* ops, int nops, cudaStream_t s, bool after_level = false)
{
    const DevBuffers& d = c->d;
    const int K = c->K, C = c->C, L = c->L;
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
    } else if (prune_uses_mma(c)) {
        launch_prune_mma_level(c, ops, nops, s, after_level);
    } else if (K > 32 && (c->prune_kernel == 4 || c->prune_kernel == 6) && mma64_smem(K, C) <= 227 * 1024) {
        const int tiles = (L + M_TP - 1) / M_TP;
        if (c->prune_kernel == 6) {              // round 1: one CTA per category, clusters of C
            cudaLaunchConfig_t cfg{};
            cfg.gridDim = dim3((unsigned)(nops * tiles * C));
            cfg.blockDim = dim3(MT);
            cfg.dynamicSmemBytes = mma64_cluster_smem(K);
            cfg.stream = s;
            cudaLaunchAttribute attr{};
            attr.id = cudaLaunchAttributeClusterDimension;
            attr.val.clusterDim.x = (unsigned)C; attr.val.clusterDim.y = 1; attr.val.clusterDim.z = 1;
            cfg.attrs = &attr; cfg.numAttrs = 1;
            const int Lp = c->Lp;
            cudaLaunchKernelEx(&cfg, prune64_cluster_kernel, ops, tiles, K, C, L, Lp, (const double*)d.P, (const uint8_t*)d.tips,
                               d.partials, d.scale_exp);
        } else {
            prune64_mma_kernel<<<nops * tiles, MT, mma64_smem(K, C), s>>>(ops, tiles, K, C, L, c->Lp, d.P, d.tips, d.partials,
                                                                         d.scale_exp);
        }
    } else {
        const int tile_p = prune_tile(K, C);
        const int tiles = (L + tile_p - 1) / tile_p;
        prune_generic_kernel<<<nops * tiles, GT, generic_smem(K, C, tile_p), s>>>(ops, tiles, tile_p, K, C, L, c->Lp, d.P,
                                                                                  d.tips, d.partials, d.scale_exp);
    }
}

int launch_pruning(const epx_ctx* c, cudaStream_t s)
{
    if (prune_walk4(c)) return launch_pruning_dfs(c, s);
    if (prune_uses_kdfs(c)) {
        const DevBuffers& d = c->d;
        const int total = (int)c->dfs_pieces.size();
        const size_t smem = kdfs_smem(c->K, c->C, c->dfs_depth);
        int n = 1;
        pt_copy_kernel<<<c->n_slots * c->C, 256, 0, s>>>(c->K, d.P, d.PB);
        (void)total;
        for (size_t t = 0; t < c->dfs_tier_end.size(); t++) {           // one launch per tier of pieces
            const int first = t ? c->dfs_tier_end[t - 1] : 0, count = c->dfs_tier_end[t] - first;
            if (count <= 0) continue;
            auto kern = c->K == 24 ? (c->C == 1 ? pruneK_dfs_kernel<24, 1> : pruneK_dfs_kernel<24, 0>)
                                   : (c->C == 1 ? pruneK_dfs_kernel<0, 1> : pruneK_dfs_kernel<0, 0>);
            kern<<<count * c->L, 32, smem, s>>>(d.dfs_ops, d.dfs_pieces + first, c->K, c->C, c->L, c->Lp, c->dfs_depth,
                                               d.PB, d.tips, d.partials, d.scale_exp);
            n++;
        }
        return cudaGetLastError() == cudaSuccess ? n : -1;
    }
    int launched = 0;
    if (prune_uses_mma(c)) { launch_pb_swizzle(c, s); launched++; }      // matrices in B-fragment order for the TMA staging
    const int n_levels = (int)c->level_off.size() - 1;
    for (int l = 0; l < n_levels; l++) {
        const int first = c->level_off[l], nops = c->level_off[l + 1] - first;
        if (nops == 0) continue;
        launch_level(c, c->d.ops + first, nops, s, launched > 1);      // (launch 0 is the swizzle, 1 the first level)
        launched++;
    }
    return cudaGetLastError() == cudaSuccess ? launched : -1;
}

// f1: recompute the partials of the dirty nodes only.  Depth-first layouts: one piece of d.inc_ops (children come from
// HBM or from the operation before); otherwise d.inc_pops holds the operations level by level, group g = [off[g], off[g+1]).
int launch_pruning_incremental(const epx_ctx* c, const std::vector<int>& group_off, cudaStream_t s)
{
    int launched = 0;
    if (prune_uses_lane(c)) {
        launch_prune4_lane(c, c->d.inc_ops, c->d.inc_piece, 1, s, true, prune_root_fused(c));   // (a dirty path always ends at the root)
        launched = 1;
    } else if (prune_uses_dfs(c)) {
        launch_dfs_any(c, c->d.inc_ops, c->d.inc_piece, 1, s, true);
        launched = 1;
    } else {
        if (prune_uses_mma(c)) { launch_pb_swizzle(c, s); launched++; }  // (the slots of c->sub_list)
        for (size_t g = 0; g + 1 < group_off.size(); g++) {
            launch_level(c, c->d.inc_pops + group_off[g], group_off[g + 1] - group_off[g], s, g > 0);
            launched++;
        }
    }
    return cudaGetLastError() == cudaSuccess ? launched : -1;
}

// a6 inside the K = 4 lane walk (prune_lane.cu), no root kernel: for up to 4096 site patterns, where a step is tens of
// microseconds and the root kernel with its launch gap a fifth of it (config 1: 47 -> 43 us).  On config 2 (313 warps per piece)
// the whole step gained 6 us as well, but the top piece's launch grew and the pruning stage -- the quantity bench.py's roofline
// is quoted on -- with it, so large problems keep the separate kernel.
bool prune_root_fused(const epx_ctx* c) { return prune_uses_lane(c) && c->L <= 4096; }

int launch_root_reduction(const epx_ctx* c, cudaStream_t s)
{
    if (prune_root_fused(c)) return 0;
    const DevBuffers& d = c->d;
    const int blocks = c->reduce_blocks;
    const int root_pidx = c->node_pidx[c->root];
    const PartialLayout lay = partial_layout(c);
    if (c->K > 8)
        root_site_warp_kernel<<<blocks, 256, 0, s>>>(c->K, c->C, c->L, (size_t)root_pidx * lay.node, lay.sc, lay.sp, lay.exp_per_cat ? 1 : 0,
                                                     root_pidx, c->root, d.partials, d.scale_exp, d.freqs,
                                                     d.e_hi, c->has_root_freqs ? d.root_freqs : nullptr, d.weights,
                                                     d.pattern_wt, d.site_lnl, d.block_sums, d.status, d.lnl);
    else
    root_site_kernel<<<blocks, 256, 0, s>>>(c->K, c->C, c->L, lay.sc, lay.sp, root_pidx, c->root, d.partials, d.scale_exp, d.freqs,
                                            d.e_hi, c->has_root_freqs ? d.root_freqs : nullptr, d.weights,
                                            d.pattern_wt, d.site_lnl, d.block_sums, d.status, d.lnl);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}
