// a3 + a4 fused, reversible path: segment exponentials and the ordered matrix-chain convolution
// (Eq.(3); L84-L109 Eq.(5)-(7), parent end = leftmost factor; L314-L323 App. A).
//
// The paper runs two kernels with intermediate buffers in global memory (UpdateTransitionMatrices, then
// ConvolveTransitionMatrices per boundary).  Here one kernel keeps the whole chain on chip and stays in the
// eigenbasis across epoch boundaries.  With S_e = Pi_e^{1/2} Q_e Pi_e^{-1/2} = U_e L_e U_e^T and segments
// s = 1..n (epochs e_1 > e_2 > ... > e_n, durations d_s, category rate r):
//   P = Pi_{e_1}^{-1/2} [ U_{e_1} D_1 W_{e_1} D_2 W_{e_2} ... D_n U_{e_n}^T ] Pi_{e_n}^{1/2},
//   D_s = exp(L_{e_s} r d_s),   W_e = U_e^T diag(sqrt(pi_e/pi_{e-1})) U_{e-1}   (prep_kernel)
// i.e. n dense products per (branch, category) instead of the 3n-1 of exp-then-convolve.  Algebraically identical
// to Eq. (7); the flop count reported by bench.py is the executed one.
//
// Three kernels:
//   chain_rows_kernel<4>  K == 4: one thread per (slot, category, row) keeps its row of the chain in registers
//   chain_generic_kernel  any K <= 64: one CTA per (slot, category), operands staged in shared memory, DFMA
//   chain_dmma64_kernel   32 < K <= 64: one CTA per (slot, 4 categories); 256x64 accumulator in registers,
//                         mma.sync m8n8k4 f64 (DMMA) tiles, B operands pre-swizzled in fragment order and staged by
//                         TMA bulk copies (cp.async.bulk + mbarrier) into a double-buffered shared-memory ring
#include "epx_internal.h"
#include "seg_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ K == 4
template <int K>
__global__ void __launch_bounds__(256) chain_rows_kernel(int n_slots, int C, const int32_t* __restrict__ list,
    int M, const double* __restrict__ tau, const int32_t* __restrict__ parent, const double* __restrict__ height,
    const double* __restrict__ child_h, const double* __restrict__ parent_h, const double* __restrict__ brate,
    const double* __restrict__ rates, const double* __restrict__ lam, const double* __restrict__ U,
    const double* __restrict__ W, const double* __restrict__ sp, const double* __restrict__ isp,
    double* __restrict__ P, int32_t* __restrict__ status, int staged, const int32_t* __restrict__ n_dev)
{
    if (n_dev) n_slots = *n_dev;                 // incremental graph: fixed grid, the slot count lives on the device
    // The per-epoch inputs (boundaries, eigenvalues, eigenvectors, sqrt(pi)) are a few KB: one cooperative copy into shared
    // memory replaces the chains of dependent global loads of the boundary search and of every segment.
    extern __shared__ double cs[];
    if (staged) {
        double* s_tau = cs; double* s_lam = s_tau + (M - 1); double* s_U = s_lam + M * K; double* s_sp = s_U + M * K * K; double* s_isp = s_sp + M * K;
        for (int t = threadIdx.x; t < M - 1; t += blockDim.x) s_tau[t] = tau[t];
        for (int t = threadIdx.x; t < M * K; t += blockDim.x) { s_lam[t] = lam[t]; s_sp[t] = sp[t]; s_isp[t] = isp[t]; }
        for (int t = threadIdx.x; t < M * K * K; t += blockDim.x) s_U[t] = U[t];
        __syncthreads();
        tau = s_tau; lam = s_lam; U = s_U; sp = s_sp; isp = s_isp;
    }
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)n_slots * C * K) return;
    const int i = (int)(idx % K);
    const int c = (int)((idx / K) % C);
    const int bi = (int)(idx / ((long long)K * C));
    const int b = list ? list[bi] : bi;            // f1: only the listed slots
    double* out = P + (((size_t)b * C + c) * K + i) * K;
    // The branch is segmented HERE (a1's expressions: same epochs, same durations bit for bit), so this kernel depends on the
    // eigensystems only and the segmenter kernels -- whose arrays remain API outputs -- run beside it in the graph.
    double hc, hp;
    epxseg::branch_ends(b, parent, height, child_h, parent_h, hc, hp);
    const int e_lo = epxseg::count_less(tau, M - 1, hc, true), e_hi = epxseg::count_less(tau, M - 1, hp, false);
    const int n = (hp > hc) ? (e_hi - e_lo + 1) : 0;
    if (n == 0) {
#pragma unroll
        for (int j = 0; j < K; j++) out[j] = (i == j) ? 1.0 : 0.0;
        return;
    }
    const double rv = brate ? brate[b] : 1.0;
    const double r = rates[c];
    double upper = hp;
    // Deviation form: the thread carries a = (row i of the running product) - e_i and multiplies by
    //   P_s = I + Pi^{-1/2} U expm1(L r d) U^T Pi^{1/2}
    // segment by segment.  On a short segment every entry of P_s - I is O(r d) and is computed to a few ulp of ITSELF
    // (U exp(L t) U^T instead leaves the orthogonality residual of U, ~1e-16 absolute, on off-diagonal entries of
    // 1e-6 .. 1e-9: the 1e-12 bound on P holds either way, but a cherry's partial is a product of two such entries and
    // config 2's per-node partials drifted to 1e-10 relative).  Same algebra as Eq. (7); W is not needed.
    double a[K];
#pragma unroll
    for (int j = 0; j < K; j++) a[j] = 0.0;
    for (int s = 0; s < n; s++) {
        const int e = e_hi - s;
        const double lower = (s == n - 1) ? hc : tau[e - 1];
        const double rd = r * (brate ? (upper - lower) * rv : upper - lower);
        upper = lower;
        const double* Ue = U + (size_t)e * K * K;
        double z[K];
        const double si = isp[e * K + i];
#pragma unroll
        for (int k = 0; k < K; k++) z[k] = si * Ue[i * K + k];
        if (s > 0) {
#pragma unroll
            for (int j = 0; j < K; j++) {
                const double aj = a[j] * isp[e * K + j];
#pragma unroll
                for (int k = 0; k < K; k++) z[k] = fma(aj, Ue[j * K + k], z[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < K; k++) z[k] *= expm1(lam[e * K + k] * rd);
#pragma unroll
        for (int j = 0; j < K; j++) {
            double t = 0.0;
#pragma unroll
            for (int k = 0; k < K; k++) t = fma(z[k], Ue[j * K + k], t);
            a[j] = fma(t, sp[e * K + j], a[j]);
        }
    }
    bool bad = false;
#pragma unroll
    for (int j = 0; j < K; j++) {
        const double v = (i == j ? 1.0 : 0.0) + a[j];
        bad |= !isfinite(v);
        out[j] = fmax(v, 0.0);      // reading A18: rounding can leave -1e-17; P is a probability
    }
    if (bad) atomicOr(status, EPX_ST_NONFINITE_P);
}

// ------------------------------------------------------------------------------------------------ any K
constexpr int GT = 256;

__global__ void __launch_bounds__(GT) chain_generic_kernel(int K, int Kp, int C, const int32_t* __restrict__ order,
    const int32_t* __restrict__ n_seg, const int32_t* __restrict__ seg_off, const int32_t* __restrict__ seg_epoch,
    const double* __restrict__ seg_dur, const double* __restrict__ rates, const double* __restrict__ lam,
    const double* __restrict__ U, const double* __restrict__ W, const double* __restrict__ sp,
    const double* __restrict__ isp, double* __restrict__ P, int32_t* __restrict__ status)
{
    extern __shared__ double sm[];
    const int ld = Kp + 1;
    double* X = sm;                       // [Kp][ld]
    double* Y = X + (size_t)Kp * ld;      // [Kp][ld]
    double* B = Y + (size_t)Kp * ld;      // [Kp][Kp]  right-hand operand
    double* D = B + (size_t)Kp * Kp;      // [Kp]
    const int tid = threadIdx.x;
    const int b = order[blockIdx.x / C], c = blockIdx.x % C;
    double* out = P + ((size_t)b * C + c) * K * K;
    const int n = n_seg[b];
    if (n == 0) {
        for (int idx = tid; idx < K * K; idx += GT) out[idx] = (idx / K == idx % K) ? 1.0 : 0.0;
        return;
    }
    const int off = seg_off[b];
    const double r = rates[c];
    const int e_hi = seg_epoch[off];
    int e = e_hi;
    if (tid < Kp) D[tid] = exp(lam[e * Kp + tid] * r * seg_dur[off]);
    __syncthreads();
    for (int idx = tid; idx < Kp * Kp; idx += GT) {
        int i = idx / Kp, k = idx % Kp;
        X[i * ld + k] = U[(size_t)e * Kp * Kp + idx] * D[k];
    }
    for (int s = 1; s <= n; s++) {
        const bool last = (s == n);
        __syncthreads();
        if (!last) {
            const double* Wm = W + (size_t)e * Kp * Kp;
            for (int idx = tid; idx < Kp * Kp; idx += GT) B[idx] = Wm[idx];
            e = seg_epoch[off + s];
            if (tid < Kp) D[tid] = exp(lam[e * Kp + tid] * r * seg_dur[off + s]);
        } else {
            const double* Ue = U + (size_t)e * Kp * Kp;   // B = U_e^T
            for (int idx = tid; idx < Kp * Kp; idx += GT) { int j = idx / Kp, k = idx % Kp; B[k * Kp + j] = Ue[idx]; }
            if (tid < Kp) D[tid] = sp[e * Kp + tid];
        }
        __syncthreads();
        for (int idx = tid; idx < Kp * Kp; idx += GT) {
            int i = idx / Kp, j = idx % Kp;
            double a = 0.0;
            for (int k = 0; k < Kp; k++) a = fma(X[i * ld + k], B[k * Kp + j], a);
            Y[i * ld + j] = a * D[j];
        }
        double* t = X; X = Y; Y = t;
    }
    __syncthreads();
    bool bad = false;
    for (int idx = tid; idx < K * K; idx += GT) {
        int i = idx / K, j = idx % K;
        double v = isp[e_hi * Kp + i] * X[i * ld + j];
        bad |= !isfinite(v);
        out[idx] = fmax(v, 0.0);
    }
    if (bad) atomicOr(status, EPX_ST_NONFINITE_P);
}

// ------------------------------------------------------------------------------------------------ 32 < K <= 64, DMMA
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "DONE:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// TMA 1-D bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

constexpr int FRAG_DOUBLES = 4096;      // one 64x64 operand in fragment order

// NCAT categories per CTA, WPC warps per category (a warp owns 64 / WPC rows of the running product).
//   <1, 4>: 128 threads for ONE category (default): 32 accumulator registers per lane, no spill, three CTAs per SM; the only
//           layout that can take a per-category operand (the cached products of consecutive full epochs).
//   <2, 2>: round 1's layout (EPX_OPT_CHAIN_KERNEL = 2): one staged operand serves two categories, 64 accumulator registers
//           per lane (255 registers, 72 B spilled), two CTAs per SM.
template <int NCAT>
struct DmmaSmemT {
    double B[2][FRAG_DOUBLES];          // TMA destination ring (2 x 32 KB)
    double D[2][NCAT][64];              // exp(lambda r d) per stage / category
    uint64_t bar[2];
};

// index of the cached product of the full epochs a, a-1, ..., b  (1 <= b <= a <= M-2)
__host__ __device__ inline int epoch_pair_index(int a, int b) { return (a - 1) * a / 2 + (b - 1); }

// acc (MTW m-tiles x 8 n-tiles of C fragments) <- (acc * diag(D)) * B, B in fragment order in shared memory
template <int MTW>
__device__ __forceinline__ void dmma_stage(double (&acc)[MTW][8][2], const double2* __restrict__ Bs, const double2* __restrict__ Ds,
                                           int lane, int q)
{
#pragma unroll
    for (int mp = 0; mp < MTW / 2; mp++) {
        double a[2][8][2];
#pragma unroll
        for (int kt = 0; kt < 8; kt++) {
            const double2 dv = Ds[kt * 4 + q];       // D[8kt + 2q], D[8kt + 2q + 1]
#pragma unroll
            for (int mi = 0; mi < 2; mi++) {
                a[mi][kt][0] = acc[2 * mp + mi][kt][0] * dv.x;
                a[mi][kt][1] = acc[2 * mp + mi][kt][1] * dv.y;
                acc[2 * mp + mi][kt][0] = 0.0;
                acc[2 * mp + mi][kt][1] = 0.0;
            }
        }
#pragma unroll
        for (int kt = 0; kt < 8; kt++)
#pragma unroll
            for (int nt = 0; nt < 8; nt++) {
                const double2 bv = Bs[(kt * 8 + nt) * 32 + lane];
                // h outer, mi inner: two other DMMAs sit between the two that update the same accumulator tile
#pragma unroll
                for (int h = 0; h < 2; h++)
#pragma unroll
                    for (int mi = 0; mi < 2; mi++)
                        dmma884(acc[2 * mp + mi][nt][0], acc[2 * mp + mi][nt][1], a[mi][kt][h], h ? bv.y : bv.x);
            }
    }
}

template <int NCAT, int WPC>
__global__ void __launch_bounds__(32 * WPC * NCAT, NCAT == 2 ? 2 : 3) chain_dmma64_kernel(int K, int C, int M,
    const int32_t* __restrict__ order,
    const int32_t* __restrict__ n_seg, const int32_t* __restrict__ seg_off, const int32_t* __restrict__ seg_epoch,
    const double* __restrict__ seg_dur, const double* __restrict__ rates, const double* __restrict__ lam,
    const double* __restrict__ WB, const double* __restrict__ UTB, const double* __restrict__ GB, const double* __restrict__ sp,
    const double* __restrict__ isp, double* __restrict__ P, int32_t* __restrict__ status)
{
    constexpr int DT = 32 * WPC * NCAT, MTW = 8 / WPC;
    extern __shared__ __align__(128) unsigned char smraw[];
    DmmaSmemT<NCAT>& sm = *reinterpret_cast<DmmaSmemT<NCAT>*>(smraw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int ncg = (C + NCAT - 1) / NCAT;
    const int b = order[blockIdx.x / ncg], cg = blockIdx.x % ncg;
    const int wc = w / WPC, rb = w % WPC;          // category of the CTA this warp serves, its block of 8 * MTW rows
    const int c = cg * NCAT + wc;
    const bool active = c < C;
    const int n = n_seg[b];
    if (n == 0) {
        for (int cc = cg * NCAT; cc < min(C, cg * NCAT + NCAT); cc++) {
            double* out = P + ((size_t)b * C + cc) * K * K;
            for (int idx = tid; idx < K * K; idx += DT) out[idx] = (idx / K == idx % K) ? 1.0 : 0.0;
        }
        return;
    }
    const int off = seg_off[b];
    const int e_hi = seg_epoch[off], e_lo = seg_epoch[off + n - 1];
    // f1: a chain over >= 2 full epochs multiplies by their cached product instead (one operand per category: NCAT == 1)
    const bool cached = NCAT == 1 && GB != nullptr && n >= 4;
    const int ns = cached ? 3 : n;                 // products of this chain

    // stage t: B operand = WB[epoch_t] for a boundary epoch_t -> epoch_t - 1, U^T of e_lo for the last; with the cache the
    // middle stage is the product of the full epochs e_hi - 1 .. e_lo + 1 (already scaled: its D is 1)
    auto stage_src = [&](int t) -> const double* {
        if (cached)
            return t == 0 ? WB + (size_t)e_hi * FRAG_DOUBLES
                 : t == 1 ? GB + ((size_t)epoch_pair_index(e_hi - 1, e_lo + 1) * C + cg) * FRAG_DOUBLES
                          : UTB + (size_t)e_lo * FRAG_DOUBLES;
        return (t < n - 1) ? WB + (size_t)seg_epoch[off + t] * FRAG_DOUBLES : UTB + (size_t)e_lo * FRAG_DOUBLES;
    };
    auto fill_D = [&](int t) {     // one value per thread: category tid>>6, eigen index tid&63
        if (tid >= 64 * NCAT) return;
        const int cc = cg * NCAT + (tid >> 6), k = tid & 63;
        const double r = cc < C ? rates[cc] : 0.0;
        const int s = cached ? (t == 0 ? 0 : n - 1) : t;
        sm.D[t & 1][tid >> 6][k] = (cached && t == 1) ? 1.0 : exp(lam[seg_epoch[off + s] * 64 + k] * (r * seg_dur[off + s]));
    };
    if (tid == 0) {
        mbar_init(&sm.bar[0], 1);
        mbar_init(&sm.bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&sm.bar[0], FRAG_DOUBLES * 8);
        bulk_g2s(sm.B[0], stage_src(0), FRAG_DOUBLES * 8, &sm.bar[0]);
    }
    fill_D(0);

    // accumulator = the warp's slab of the running product, as MTW (m) x 8 (n) C-fragments.
    // Start: rows of U_{e_hi}; U^T in B-fragment order doubles as U in A-fragment order (same index map).
    double acc[MTW][8][2];
    {
        const double2* src = reinterpret_cast<const double2*>(UTB + (size_t)e_hi * FRAG_DOUBLES);
#pragma unroll
        for (int mt = 0; mt < MTW; mt++)
#pragma unroll
            for (int kt = 0; kt < 8; kt++) {
                double2 v = __ldg(&src[(kt * 8 + (MTW * rb + mt)) * 32 + lane]);
                acc[mt][kt][0] = v.x;
                acc[mt][kt][1] = v.y;
            }
    }
    __syncthreads();

    for (int t = 0; t < ns; t++) {
        const int st = t & 1;
        if (t + 1 < ns) {              // prefetch the next stage into the other buffer (freed at the end of t-1)
            if (tid == 0) {
                mbar_expect_tx(&sm.bar[st ^ 1], FRAG_DOUBLES * 8);
                bulk_g2s(sm.B[st ^ 1], stage_src(t + 1), FRAG_DOUBLES * 8, &sm.bar[st ^ 1]);
            }
            fill_D(t + 1);
        }
        mbar_wait(&sm.bar[st], (t >> 1) & 1);
        if (active)
            dmma_stage<MTW>(acc, reinterpret_cast<const double2*>(sm.B[st]), reinterpret_cast<const double2*>(sm.D[st][wc]), lane, q);
        __syncthreads();
    }

    if (!active) return;
    double* out = P + ((size_t)b * C + c) * K * K;
    bool bad = false;
#pragma unroll
    for (int mt = 0; mt < MTW; mt++) {
        const int i = 8 * MTW * rb + 8 * mt + g;
        if (i >= K) continue;
        const double si = isp[e_hi * 64 + i];
#pragma unroll
        for (int nt = 0; nt < 8; nt++)
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const int j = 8 * nt + 2 * q + h;
                if (j < K) {
                    double v = si * acc[mt][nt][h] * sp[e_lo * 64 + j];
                    bad |= !isfinite(v);
                    out[(size_t)i * K + j] = fmax(v, 0.0);
                }
            }
    }
    if (bad) atomicOr(status, EPX_ST_NONFINITE_P);
}

// f1, second half (the convolutions dominate when many branches cross many
// boundaries).  Products of consecutive FULL epochs do not depend on the branch:
//   G[a, b] = D_a W_a D_{a-1} W_{a-1} ... D_b W_b,   D_e = exp(Lambda_e r_c (tau_e - tau_{e-1})),   1 <= b <= a <= M-2
// maps the eigenbasis of epoch a to that of epoch b - 1.  One CTA per (a, pair of categories) accumulates G[a, a], G[a, a-1],
// ..., G[a, 1] with the chain kernel's own stage code, starting from the identity, and stores each in B-fragment order.
__global__ void __launch_bounds__(128, 2) epoch_product_table_kernel(int C, int M, const double* __restrict__ tau,
    const double* __restrict__ rates, const double* __restrict__ lam, const double* __restrict__ WB, double* __restrict__ GB)
{
    extern __shared__ __align__(128) unsigned char smraw[];
    DmmaSmemT<2>& sm = *reinterpret_cast<DmmaSmemT<2>*>(smraw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, q = lane & 3;
    const int ncg = (C + 1) / 2;
    const int a = 1 + blockIdx.x / ncg, cg = blockIdx.x % ncg;
    const int c = cg * 2 + (w >> 1), half = w & 1;
    const bool active = c < C;
    const int ns = a;                               // stages: epochs a, a-1, ..., 1
    auto fill_D = [&](int t) {
        const int cc = cg * 2 + (tid >> 6), k = tid & 63, e = a - t;
        const double r = cc < C ? rates[cc] : 0.0;
        sm.D[t & 1][tid >> 6][k] = exp(lam[e * 64 + k] * (r * (tau[e] - tau[e - 1])));
    };
    if (tid == 0) {
        mbar_init(&sm.bar[0], 1);
        mbar_init(&sm.bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&sm.bar[0], FRAG_DOUBLES * 8);
        bulk_g2s(sm.B[0], WB + (size_t)a * FRAG_DOUBLES, FRAG_DOUBLES * 8, &sm.bar[0]);
    }
    fill_D(0);
    double acc[4][8][2];                            // identity: row 32 half + 8 mt + g, columns 8 nt + 2 q + h
#pragma unroll
    for (int mt = 0; mt < 4; mt++)
#pragma unroll
        for (int nt = 0; nt < 8; nt++)
#pragma unroll
            for (int h = 0; h < 2; h++) acc[mt][nt][h] = (32 * half + 8 * mt + g == 8 * nt + 2 * q + h) ? 1.0 : 0.0;
    __syncthreads();
    for (int t = 0; t < ns; t++) {
        const int st = t & 1;
        if (t + 1 < ns) {
            if (tid == 0) {
                mbar_expect_tx(&sm.bar[st ^ 1], FRAG_DOUBLES * 8);
                bulk_g2s(sm.B[st ^ 1], WB + (size_t)(a - t - 1) * FRAG_DOUBLES, FRAG_DOUBLES * 8, &sm.bar[st ^ 1]);
            }
            fill_D(t + 1);
        }
        mbar_wait(&sm.bar[st], (t >> 1) & 1);
        if (active) {
            dmma_stage<4>(acc, reinterpret_cast<const double2*>(sm.B[st]), reinterpret_cast<const double2*>(sm.D[st][w >> 1]), lane, q);
            // G[a, a - t] in B-fragment order: element X[kappa][col] sits at ((kappa/8 * 8 + col/8) * 32 + 4 (col%8) + (kappa%8)/2) * 2 + kappa%2
            double* out = GB + ((size_t)epoch_pair_index(a, a - t) * C + c) * FRAG_DOUBLES;
#pragma unroll
            for (int mt = 0; mt < 4; mt++)
#pragma unroll
                for (int nt = 0; nt < 8; nt++)
#pragma unroll
                    for (int h = 0; h < 2; h++)
                        out[(((4 * half + mt) * 8 + nt) * 32 + 4 * (2 * q + h) + (g >> 1)) * 2 + (g & 1)] = acc[mt][nt][h];
        }
        __syncthreads();
    }
}

}  // namespace

int chain_init_attributes()
{
    if (cudaFuncSetAttribute(chain_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(chain_dmma64_kernel<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(DmmaSmemT<2>)) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(chain_dmma64_kernel<1, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(DmmaSmemT<1>)) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(epoch_product_table_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(DmmaSmemT<2>)) != cudaSuccess) return -1;
    return 0;
}

// f1: the chain kernels multiply by cached products of consecutive full epochs (option on, 64-padded reversible models,
// durations not rescaled per branch, at least two interior epochs)
bool chain_uses_epoch_products(const epx_ctx* c)
{
    return c->epoch_products && c->Kp == 64 && c->chain_kernel != 1 && !c->has_brates && c->M >= 4;
}

int launch_chain_reversible(const epx_ctx* c, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    const int K = c->K, Kp = c->Kp, C = c->C;
    // f1: an incremental call recomputes only the slots of c->sub_list (any order); a full call all of them, longest first
    const int n = c->sub_list ? c->sub_count : c->n_slots;
    const int32_t* order = c->sub_list ? c->sub_list : d.order;
    if (n == 0) return 0;
    if (K == 4 && c->chain_kernel != 1) {      // (EPX_OPT_CHAIN_KERNEL = 1 forces the generic kernel at K = 4 too)
        long long threads = (long long)n * C * 4;
        int blocks = (int)((threads + 255) / 256);
        const size_t stage_bytes = sizeof(double) * ((size_t)c->M - 1 + (size_t)c->M * (4 * 4 + 3 * 4));
        const int staged = stage_bytes <= 16 * 1024;
        chain_rows_kernel<4><<<c->sub_count_dev ? (EPX_INC_GRAPH_SLOTS * C * 4 + 255) / 256 : blocks, 256, staged ? stage_bytes : 0, s>>>(n, C, c->sub_list, c->M, d.tau, c->tree_mode ? d.parent : nullptr, d.height,
                                                    d.child_h, d.parent_h, c->has_brates ? d.brate : nullptr, d.rates,
                                                    d.lam, d.U, d.W, d.sp, d.isp, d.P, d.status, staged, c->sub_count_dev);
    } else if (Kp == 64 && c->chain_kernel != 1) {
        int launched = 0;
        if (chain_uses_epoch_products(c)) {
            // (an incremental call keeps the table: it depends on the boundaries, the models and the category rates only)
            if (!c->sub_list) {
                epoch_product_table_kernel<<<(c->M - 2) * ((C + 1) / 2), 128, sizeof(DmmaSmemT<2>), s>>>(C, c->M, d.tau, d.rates, d.lam,
                                                                                                       d.WB, d.GB);
                launched++;
            }
            chain_dmma64_kernel<1, 4><<<n * C, 128, sizeof(DmmaSmemT<1>), s>>>(K, C, c->M, order, d.n_seg, d.seg_off, d.seg_epoch,
                                                                               d.seg_dur, d.rates, d.lam, d.WB, d.UTB, d.GB, d.sp,
                                                                               d.isp, d.P, d.status);
        } else if (c->chain_kernel != 2) {       // default: one category per CTA, four warps of 16 rows (162 registers, no spill,
                                                 // three CTAs per SM: measured 4.74 ms on config 5 against 5.02 ms for <2, 2>)
            chain_dmma64_kernel<1, 4><<<n * C, 128, sizeof(DmmaSmemT<1>), s>>>(K, C, c->M, order, d.n_seg, d.seg_off, d.seg_epoch,
                                                                               d.seg_dur, d.rates, d.lam, d.WB, d.UTB, nullptr, d.sp,
                                                                               d.isp, d.P, d.status);
        } else {                                 // round 1's layout: two categories per CTA share one staged operand
            const int ncg = (C + 1) / 2;
            chain_dmma64_kernel<2, 2><<<n * ncg, 128, sizeof(DmmaSmemT<2>), s>>>(K, C, c->M, order, d.n_seg, d.seg_off, d.seg_epoch,
                                                                                 d.seg_dur, d.rates, d.lam, d.WB, d.UTB, nullptr,
                                                                                 d.sp, d.isp, d.P, d.status);
        }
        return cudaGetLastError() == cudaSuccess ? launched + 1 : -1;
    } else {
        size_t smem = sizeof(double) * (2 * (size_t)Kp * (Kp + 1) + (size_t)Kp * Kp + Kp);
        chain_generic_kernel<<<n * C, GT, smem, s>>>(K, Kp, C, order, d.n_seg, d.seg_off, d.seg_epoch, d.seg_dur,
                                                     d.rates, d.lam, d.U, d.W, d.sp, d.isp, d.P, d.status);
    }
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}
