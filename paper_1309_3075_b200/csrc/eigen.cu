// a2: per-epoch eigensystem of a reversible rate matrix (PAPER.md L58 detailed balance; L80, L314-L316: one
// decomposition per process, reused for every (rate, time)).
//
// With pi_i q_ij = pi_j q_ji the matrix S = Pi^{1/2} Q Pi^{-1/2} is symmetric, S = U Lambda U^T, and
//   exp(Q r d) = Pi^{-1/2} U exp(Lambda r d) U^T Pi^{1/2}.
// jacobi_kernel: one CTA per epoch, cyclic Jacobi with a round-robin parallel ordering (K/2 disjoint rotations per
// round, K-1 rounds per sweep) entirely in shared memory.
// prep_kernel: the epoch-to-epoch change of basis W_e = U_e^T diag(sqrt(pi_e / pi_{e-1})) U_{e-1} that lets the chain
// kernel stay in the eigenbasis across a boundary (one product per segment instead of three), plus copies of W and
// U^T in DMMA B-fragment order for the 64-wide tensor-core chain kernel.
#include "epx_internal.h"
#include <cstdio>
#include <type_traits>

namespace {

constexpr int JT_MAX = 1024;   // threads per CTA for K > 32 (one 2x2 block of S per thread and round); 256 otherwise

// Two-sided Jacobi, round-robin ordering: in one round the n/2 pivot pairs are disjoint, so S' = J^T S J splits into
// (n/2)^2 independent 2x2 blocks (rows of pair a, columns of pair b) that each depend on their own four entries and the
// two rotations only.  One thread per block applies the column and the row rotation in registers: two barriers per round
// instead of three, and 961 busy threads at K = 61.
__global__ void __launch_bounds__(JT_MAX) jacobi_kernel(int K, int Kp, const double* __restrict__ Qall,
                                                        const double* __restrict__ freqs, double* __restrict__ lam,
                                                        double* __restrict__ Uout, double* __restrict__ sp_out,
                                                        double* __restrict__ isp_out, int32_t* __restrict__ status,
                                                        int M, const int32_t* __restrict__ eproc)
{
    extern __shared__ double sm[];
    if (eproc[blockIdx.x] != (int)blockIdx.x) return;      // f2: this epoch shares the process of an earlier one
    const int JT = blockDim.x;
    const int ld = K | 1;                       // odd row stride: column walks are bank-conflict free
    double* S = sm;                             // [K][ld]
    double* V = S + (size_t)K * ld;             // [K][ld]
    double* rc = V + (size_t)K * ld;            // [K/2+1] cos
    double* rs = rc + (K / 2 + 1);              // [K/2+1] sin
    double* red = rs + (K / 2 + 1);             // [32] reduction scratch
    int* rp = (int*)(red + 32);                 // [K/2+1] p
    int* rq = rp + (K / 2 + 1);                 // [K/2+1] q (>= K: the dummy player of an odd K)
    __shared__ double s_off2, s_tot2;

    const int e = blockIdx.x, tid = threadIdx.x;
    const double* Q = Qall + (size_t)e * K * K;
    const double* pi = freqs + (size_t)e * K;

    for (int idx = tid; idx < K * K; idx += JT) {
        int i = idx / K, j = idx % K;
        double a = sqrt(pi[i]) * Q[i * K + j] / sqrt(pi[j]);
        double b = sqrt(pi[j]) * Q[j * K + i] / sqrt(pi[i]);
        S[i * ld + j] = 0.5 * (a + b);
        V[i * ld + j] = (i == j) ? 1.0 : 0.0;
    }
    __syncthreads();

    auto block_sum = [&](double v) -> double {
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((tid & 31) == 0) red[tid >> 5] = v;
        __syncthreads();
        double t = 0;
        for (int w = 0; w < JT / 32; w++) t += red[w];
        __syncthreads();
        return t;
    };
    {
        double t = 0;
        for (int idx = tid; idx < K * K; idx += JT) { double x = S[(idx / K) * ld + idx % K]; t += x * x; }
        t = block_sum(t);
        if (tid == 0) s_tot2 = t;
    }
    __syncthreads();

    const int n = (K + 1) & ~1;          // players (a dummy one if K is odd)
    const int npair = n / 2;
    const double eps = 2.220446049250313e-16;
    // item -> (pair a, pair b) and (pair, row) maps do not change from round to round
    const int blk_a = tid / npair, blk_b = tid - blk_a * npair;
    const int v_k = tid / K, v_i = tid - v_k * K;
    bool converged = false;
    for (int sweep = 0; sweep < 40 && !converged; sweep++) {
        for (int r = 0; r < n - 1; r++) {
            if (tid < npair) {
                int a, b;
                if (tid == 0) { a = n - 1; b = r; }
                else { a = (r + tid) % (n - 1); b = (r - tid + (n - 1)) % (n - 1); }
                int p = min(a, b), q = max(a, b);
                double c = 1.0, s = 0.0;
                if (q < K) {
                    const double apq = S[p * ld + q];
                    if (fabs(apq) > 1e-300) {
                        // t = tan of the rotation angle, the root of smaller magnitude of t^2 + 2 theta t - 1 = 0 with
                        // theta = d / h: t = sgn(d) h / (|d| + sqrt(d^2 + h^2)); one rsqrt per square root, one division
                        const double d = S[q * ld + q] - S[p * ld + p], h = 2.0 * apq;
                        const double r2 = fma(d, d, h * h);
                        const double r = r2 * rsqrt(r2);
                        const double t = (d < 0 ? -h : h) / (fabs(d) + r);
                        c = rsqrt(fma(t, t, 1.0));
                        s = t * c;
                    }
                }
                rp[tid] = p; rq[tid] = q; rc[tid] = c; rs[tid] = s;
            }
            __syncthreads();
            // S <- J^T S J, one 2x2 block per item
            for (int blk = tid; blk < npair * npair; blk += JT) {
                const int a = blk == tid ? blk_a : blk / npair, b = blk == tid ? blk_b : blk - a * npair;
                const int pa = rp[a], qa = rq[a], pb = rp[b], qb = rq[b];
                const double ca = rc[a], sa = rs[a], cb = rc[b], sb = rs[b];
                const bool ra = qa < K, cbv = qb < K;            // second row / column is a real index
                double x00 = S[pa * ld + pb];
                double x01 = cbv ? S[pa * ld + qb] : 0.0;
                double x10 = ra ? S[qa * ld + pb] : 0.0;
                double x11 = (ra && cbv) ? S[qa * ld + qb] : 0.0;
                // columns (pair b)
                double t00 = cb * x00 - sb * x01, t01 = sb * x00 + cb * x01;
                double t10 = cb * x10 - sb * x11, t11 = sb * x10 + cb * x11;
                // rows (pair a)
                double y00 = ca * t00 - sa * t10, y01 = ca * t01 - sa * t11;
                double y10 = sa * t00 + ca * t10, y11 = sa * t01 + ca * t11;
                if (a == b) { y01 = 0.0; y10 = 0.0; }            // the pivot pair is annihilated exactly
                S[pa * ld + pb] = y00;
                if (cbv) S[pa * ld + qb] = y01;
                if (ra) S[qa * ld + pb] = y10;
                if (ra && cbv) S[qa * ld + qb] = y11;
            }
            // V <- V J
            for (int idx = tid; idx < npair * K; idx += JT) {
                const int k = idx == tid ? v_k : idx / K, i = idx == tid ? v_i : idx - k * K, q = rq[k];
                if (q >= K) continue;
                const int p = rp[k];
                const double c = rc[k], s = rs[k];
                const double x = V[i * ld + p], y = V[i * ld + q];
                V[i * ld + p] = c * x - s * y;
                V[i * ld + q] = s * x + c * y;
            }
            __syncthreads();
        }
        double t = 0;
        for (int idx = tid; idx < K * K; idx += JT) {
            int i = idx / K, j = idx % K;
            if (i != j) { double x = S[i * ld + j]; t += x * x; }
        }
        t = block_sum(t);
        if (tid == 0) s_off2 = t;
        __syncthreads();
        converged = s_off2 <= 0.25 * eps * eps * s_tot2;
#ifdef EPX_DEBUG_JACOBI
        if (tid == 0) printf("epoch %d sweep %d off/tot %.3e\n", e, sweep, sqrt(s_off2 / s_tot2));
#endif
    }
    if (tid == 0 && !(s_off2 <= 1e-28 * s_tot2)) atomicOr(status, EPX_ST_JACOBI_NOCONV);

    for (int f = e; f < M; f++) {             // every epoch of this process gets the eigensystem
        if (eproc[f] != e) continue;
        double* U = Uout + (size_t)f * Kp * Kp;
        for (int idx = tid; idx < Kp * Kp; idx += JT) {
            int i = idx / Kp, j = idx % Kp;
            U[idx] = (i < K && j < K) ? V[i * ld + j] : 0.0;
        }
        for (int i = tid; i < Kp; i += JT) {
            lam[(size_t)f * Kp + i] = i < K ? S[i * ld + i] : 0.0;
            sp_out[(size_t)f * Kp + i] = i < K ? sqrt(pi[i]) : 0.0;
            isp_out[(size_t)f * Kp + i] = i < K ? 1.0 / sqrt(pi[i]) : 0.0;
        }
    }
}

// ------------------------------------------------------------------------------------------------ K <= 62: one barrier per round
// The same two-sided round-robin Jacobi, reorganised so that a round costs ONE barrier, no index arithmetic and conflict-free
// shared-memory traffic (the kernel above spends 221 instructions per warp and round, half of them on indices; its 16 CTAs
// were 15 % of config 5's step):
//   * the players of the tournament sit in two rows, tops T_0..T_{m-1} at positions 0..m-1 and bottoms B_0..B_{m-1} at
//     positions m..2m-1; pair k = (T_k, B_k).  S and V are stored in position order.  After a round the tournament rotates by
//     a FIXED permutation (T_0 stays, tops move right, bottoms move left, the ends change rows), so thread (a, b) always reads
//     the 2x2 block {a, m+a} x {b, m+b} at the same addresses of the current buffer and writes its rotated block to the same
//     four addresses of the other buffer (ping-pong): every address is a per-thread constant, and a warp's consecutive b are
//     consecutive words on the read AND on the write side (64-bit accesses, no bank conflicts -- a first version with the
//     pair in adjacent positions scattered its stores and was bound by shared-memory wavefronts, 2 130 per round).
//   * the same thread rotates V's block (rows a, m+a; columns of pair b) with the rotation of pair b it already holds.
//   * the rotation of a NEW pair j needs three entries of the updated matrix (two diagonal ones, the new pivot).  A spare
//     warp computes them directly from the OLD matrix and the OLD rotations (closed forms of the 2x2 updates) while the
//     other warps update S and V, so the next round's rotations are ready at the same barrier.
//   * an odd K gets a dummy player (position 2m-1) whose row and column stay zero (its rotations are the identity).
// After every sweep (n - 1 rounds) the players are back in their original positions, position = state index.
// Launders a per-thread constant through an empty asm: the compiler keeps it in a register instead of re-deriving it from
// special registers / the constant bank inside the round loops (S2R + LDC chains were ~200 cycles of every round).
#define JC_PIN(x) asm volatile("" : "+r"(x))

__device__ __forceinline__ int jac_newpos(int pos, int m)
{
    if (pos == 0 || m == 1) return pos;
    if (pos < m) return pos <= m - 2 ? pos + 1 : 2 * m - 1;      // tops move right, the last one drops to the bottom row
    return pos == m ? 1 : pos - 1;                               // bottoms move left, the first one rises to the top row
}

// 1/sqrt(x) and 1/x for normal x > 0: hardware seed (MUFU.RSQ64H / RCP64H, ~2^-22) + Newton-type corrections in FMAs.
// The rotation of the next round is the critical path of a round (one warp computes it while 31 update S and V), and
// CUDA's correctly-rounded rsqrt() / division are ~20 dependent instructions each.
__device__ __forceinline__ double fast_rsqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x * y, y, 1.0);                        // 1 - x y^2  ~ 2^-22
    return fma(y * e, fma(0.375, e, 0.5), y);                    // y (1 + e/2 + 3 e^2 / 8): error O(e^3) ~ 2^-66 + rounding
}
__device__ __forceinline__ double fast_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);                                            // 2^-44
    e = fma(-x, y, 1.0);
    return fma(y, e, y);                                         // 2^-88 + rounding
}

// Rotation (c, s) that annihilates the pivot apq of the pair with diagonal entries (spp, sqq).  t = tan of the angle, the root
// of smaller magnitude of t^2 + 2 theta t - 1 = 0 with theta = d / h.  t only has to be accurate enough to annihilate the pivot
// to rounding; c^2 + s^2 = 1 holds to rounding because c = rsqrt(1 + t^2) is accurate to ~1 ulp and s = t c.
__device__ __forceinline__ double2 jac_rotation(double spp, double sqq, double apq)
{
    const double d = sqq - spp, h = 2.0 * apq;
    const double r2 = fma(d, d, h * h);
    if (!(r2 > 1e-280) || !(fabs(apq) > 1e-300)) return make_double2(1.0, 0.0);
    const double r = r2 * fast_rsqrt(r2);
    const double t = (d < 0 ? -h : h) * fast_rcp(fabs(d) + r);
    const double c = fast_rsqrt(fma(t, t, 1.0));
    return make_double2(c, t * c);
}

__global__ void __launch_bounds__(1024) jacobi1_kernel(int K, int Kp, const double* __restrict__ Qall,
                                                       const double* __restrict__ freqs, double* __restrict__ lam,
                                                       double* __restrict__ Uout, double* __restrict__ sp_out,
                                                       double* __restrict__ isp_out, int32_t* __restrict__ status,
                                                       int M, const int32_t* __restrict__ eproc)
{
    extern __shared__ __align__(16) double sm[];
    if (eproc[blockIdx.x] != (int)blockIdx.x) return;   // f2: this epoch shares the process of an earlier one
    const int m = (K + 1) >> 1, n = 2 * m;              // pairs, players
    const int NB = blockDim.x - 32;                     // block threads; the last warp prepares the rotations
    const int nn = n * n, kn = K * n;
    double* const S0 = sm;                              // [2][n][n] ping-pong, position order
    double* const V0 = S0 + 2 * nn;                     // [2][K][n] ping-pong, columns in position order
    double2* const R0 = reinterpret_cast<double2*>(V0 + 2 * kn);                          // [2][m] (cos, sin)
    double* const red = reinterpret_cast<double*>(R0 + 2 * m);                            // [33]
    const int e = blockIdx.x, tid = threadIdx.x, T = blockDim.x;
    const double* Q = Qall + (size_t)e * K * K;
    const double* pi = freqs + (size_t)e * K;

    for (int idx = tid; idx < n * n; idx += T) {        // position = state index at the start of every sweep
        const int i = idx / n, j = idx - i * n;
        double v = 0.0;
        if (i < K && j < K) {
            const double a = sqrt(pi[i]) * Q[i * K + j] / sqrt(pi[j]);
            const double b = sqrt(pi[j]) * Q[j * K + i] / sqrt(pi[i]);
            v = 0.5 * (a + b);
        }
        S0[idx] = v;
    }
    for (int idx = tid; idx < K * n; idx += T) { const int i = idx / n, j = idx - i * n; V0[idx] = (i == j) ? 1.0 : 0.0; }
    __syncthreads();
    auto block_sum = [&](double v) -> double {          // all threads call
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((tid & 31) == 0) red[tid >> 5] = v;
        __syncthreads();
        double t = 0;
        for (int w = 0; w < T / 32; w++) t += red[w];
        __syncthreads();
        return t;
    };
    double tot2;
    {
        double t = 0;
        for (int idx = tid; idx < n * n; idx += T) { const double x = S0[idx]; t += x * x; }
        tot2 = block_sum(t);
    }

    // per-thread constants: block (a, b) = rows {a, m+a} x columns {b, m+b}
    const bool is_blk = tid < m * m;
    const int a = is_blk ? tid / m : 0, b = is_blk ? tid - a * m : 0;
    const int rt = a * n, rb = (m + a) * n, ct = b, cb = m + b;                           // read
    const int wrt = jac_newpos(a, m) * n, wrb = jac_newpos(m + a, m) * n;                 // write rows (S)
    const int wct = jac_newpos(b, m), wcb = jac_newpos(m + b, m);                         // write columns (S and V)
    const bool v0_on = is_blk && a < K, v1_on = is_blk && m + a < K;                      // V rows a and m + a
    // rotation warp, lane j < m: the players that form NEW pair j sit at old positions x (-> T_j) and y (-> B_j)
    const int j = tid - NB;
    const bool is_rot = j >= 0 && j < m;
    int x = 0, y = m;
    if (is_rot)
        for (int p = 0; p < n; p++) {
            const int q = jac_newpos(p, m);
            if (q == j) x = p;
            if (q == m + j) y = p;
        }
    const int ax = x % m, ay = y % m, px = x / m, py = y / m;

    if (is_rot) R0[j] = jac_rotation(S0[j * n + j], S0[(m + j) * n + m + j], S0[j * n + m + j]);
    __syncthreads();

    // (everything the round loop reads is pinned in a register: see JC_PIN)
    int p_rt = rt, p_rb = rb, p_ct = ct, p_cb = cb, p_wrt = wrt, p_wrb = wrb, p_wct = wct, p_wcb = wcb, p_a = a, p_b = b;
    int p_blk = is_blk, p_v0 = v0_on, p_v1 = v1_on, p_rot = is_rot, p_j = is_rot ? j : 0, p_rounds = n - 1, p_nn = nn, p_kn = kn, p_m = m;
    int i_app = ax * n + ax, i_apq = ax * n + m + ax, i_aqq = (m + ax) * n + m + ax, i_bpp = ay * n + ay, i_bpq = ay * n + m + ay,
        i_bqq = (m + ay) * n + m + ay, i_x00 = ax * n + ay, i_x01 = ax * n + m + ay, i_x10 = (m + ax) * n + ay, i_x11 = (m + ax) * n + m + ay;
    int p_ax = ax, p_ay = ay, p_px = px, p_py = py;
    JC_PIN(p_rt); JC_PIN(p_rb); JC_PIN(p_ct); JC_PIN(p_cb); JC_PIN(p_wrt); JC_PIN(p_wrb); JC_PIN(p_wct); JC_PIN(p_wcb); JC_PIN(p_a); JC_PIN(p_b);
    JC_PIN(p_blk); JC_PIN(p_v0); JC_PIN(p_v1); JC_PIN(p_rot); JC_PIN(p_j); JC_PIN(p_rounds); JC_PIN(p_nn); JC_PIN(p_kn); JC_PIN(p_m);
    JC_PIN(i_app); JC_PIN(i_apq); JC_PIN(i_aqq); JC_PIN(i_bpp); JC_PIN(i_bpq); JC_PIN(i_bqq); JC_PIN(i_x00); JC_PIN(i_x01); JC_PIN(i_x10); JC_PIN(i_x11);
    JC_PIN(p_ax); JC_PIN(p_ay); JC_PIN(p_px); JC_PIN(p_py);

    int cur = 0;
    bool converged = false;
    double off2 = 0.0;
    for (int sweep = 0; sweep < 40 && !converged; sweep++) {
        double my_off = 0.0;
        for (int r = 0; r < p_rounds; r++) {
            const double* S = S0 + cur * p_nn;
            double* Sn = S0 + (cur ^ 1) * p_nn;
            const double2* R = R0 + cur * p_m;
            if (p_blk) {
                const double2 ra = R[p_a], rbb = R[p_b];
                const double x00 = S[p_rt + p_ct], x01 = S[p_rt + p_cb], x10 = S[p_rb + p_ct], x11 = S[p_rb + p_cb];
                // columns (pair b), then rows (pair a): S <- J^T S J on this 2x2 block
                const double t00 = rbb.x * x00 - rbb.y * x01, t01 = rbb.y * x00 + rbb.x * x01;
                const double t10 = rbb.x * x10 - rbb.y * x11, t11 = rbb.y * x10 + rbb.x * x11;
                double y00 = ra.x * t00 - ra.y * t10, y01 = ra.x * t01 - ra.y * t11;
                double y10 = ra.y * t00 + ra.x * t10, y11 = ra.y * t01 + ra.x * t11;
                if (p_a == p_b) { y01 = 0.0; y10 = 0.0; }            // the pivot pair is annihilated exactly
                Sn[p_wrt + p_wct] = y00; Sn[p_wrt + p_wcb] = y01; Sn[p_wrb + p_wct] = y10; Sn[p_wrb + p_wcb] = y11;
                if (r == p_rounds - 1) my_off = p_a == p_b ? 0.0 : fma(y00, y00, fma(y01, y01, fma(y10, y10, y11 * y11)));
                // V <- V J: rows a and m + a, the columns of pair b
                const double* V = V0 + cur * p_kn;
                double* Vn = V0 + (cur ^ 1) * p_kn;
                if (p_v0) {
                    const double v0 = V[p_rt + p_ct], v1 = V[p_rt + p_cb];
                    Vn[p_rt + p_wct] = rbb.x * v0 - rbb.y * v1;
                    Vn[p_rt + p_wcb] = rbb.y * v0 + rbb.x * v1;
                }
                if (p_v1) {
                    const double v0 = V[p_rb + p_ct], v1 = V[p_rb + p_cb];
                    Vn[p_rb + p_wct] = rbb.x * v0 - rbb.y * v1;
                    Vn[p_rb + p_wcb] = rbb.y * v0 + rbb.x * v1;
                }
            } else if (p_rot) {
                double2 nr = make_double2(1.0, 0.0);
                if (p_ax != p_ay) {
                    const double2 ra = R[p_ax], rbb = R[p_ay];
                    const double app = S[i_app], apq = S[i_apq], aqq = S[i_aqq];
                    const double bpp = S[i_bpp], bpq = S[i_bpq], bqq = S[i_bqq];
                    const double x00 = S[i_x00], x01 = S[i_x01], x10 = S[i_x10], x11 = S[i_x11];
                    // the player's updated diagonal entry: (J^T S J)_pp = c^2 Spp - 2 c s Spq + s^2 Sqq, _qq = s^2 Spp + 2 c s Spq + c^2 Sqq
                    const double ca2 = ra.x * ra.x, sa2 = ra.y * ra.y, csa = 2.0 * ra.x * ra.y;
                    const double cb2 = rbb.x * rbb.x, sb2 = rbb.y * rbb.y, csb = 2.0 * rbb.x * rbb.y;
                    const double dx = p_px ? fma(sa2, app, fma(csa, apq, ca2 * aqq)) : fma(ca2, app, fma(-csa, apq, sa2 * aqq));
                    const double dy = p_py ? fma(sb2, bpp, fma(csb, bpq, cb2 * bqq)) : fma(cb2, bpp, fma(-csb, bpq, sb2 * bqq));
                    // the new pivot = entry (px, py) of the updated block (ax, ay)
                    const double t0 = p_py ? rbb.y * x00 + rbb.x * x01 : rbb.x * x00 - rbb.y * x01;
                    const double t1 = p_py ? rbb.y * x10 + rbb.x * x11 : rbb.x * x10 - rbb.y * x11;
                    const double piv = p_px ? ra.y * t0 + ra.x * t1 : ra.x * t0 - ra.y * t1;
                    nr = jac_rotation(dx, dy, piv);
                }
                R0[(cur ^ 1) * p_m + p_j] = nr;
            }
            __syncthreads();
            cur ^= 1;
        }
        off2 = block_sum(my_off);
        converged = off2 <= 0.25 * 2.220446049250313e-16 * 2.220446049250313e-16 * tot2;
    }
    if (tid == 0 && !(off2 <= 1e-28 * tot2)) atomicOr(status, EPX_ST_JACOBI_NOCONV);

    const double* S = S0 + cur * nn;
    const double* V = V0 + cur * kn;
    for (int f = e; f < M; f++) {             // every epoch of this process gets the eigensystem
        if (eproc[f] != e) continue;
        double* U = Uout + (size_t)f * Kp * Kp;
        for (int idx = tid; idx < Kp * Kp; idx += T) {
            const int i = idx / Kp, jj = idx % Kp;
            U[idx] = (i < K && jj < K) ? V[i * n + jj] : 0.0;
        }
        for (int i = tid; i < Kp; i += T) {
            lam[(size_t)f * Kp + i] = i < K ? S[i * n + i] : 0.0;
            sp_out[(size_t)f * Kp + i] = i < K ? sqrt(pi[i]) : 0.0;
            isp_out[(size_t)f * Kp + i] = i < K ? 1.0 / sqrt(pi[i]) : 0.0;
        }
    }
}

// ------------------------------------------------------------------------------------------------ 32 < K <= 62: a cluster per process
// jacobi1_kernel is bound by the shared-memory bandwidth of ONE SM per process (config 5: 16 of 148 SMs busy for 0.52 ms, a
// serial prefix of the chain kernel).  Here a thread-block cluster of 1 + NV CTAs shares a process:
//   * CTA 0 owns S and is the only one on the critical path.  S is symmetric, so it keeps the entries (p, q) with p <= q only
//     and runs one thread per block (a, b) with a <= b: 496 threads instead of 961, half the shared-memory traffic.  As in
//     jacobi1_kernel every address is a per-thread constant (positions are fixed, the players rotate), the buffers ping-pong
//     and a round costs one CTA barrier; the row stride is odd so that the transposed accesses are conflict free.
//   * V <- V J touches V's rows independently and never feeds back into S: CTAs 1..NV own K / NV rows of V each and apply the
//     rotations CTA 0's rotation warp pushes into a ring in THEIR shared memory (st.async: a 16-byte store whose
//     completion is counted on the V CTA's mbarrier -- no fence anywhere in the iteration).  They run behind CTA 0 at their own pace; the ring's flow control (a progress word each V CTA stores
//     back) never stalls CTA 0 in practice because a V CTA has less work per round.  After every sweep CTA 0 sends its
//     verdict (converged or not); a sweep's rounds are the only thing the V CTAs wait for.
// No cluster barrier inside the iteration (one at the start, one at the end).
__device__ __forceinline__ uint32_t jc_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t jc_mapa(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// 16 bytes into a peer's shared memory, completion counted on the peer's mbarrier (no fence: the store and its
// complete_tx are ordered by the hardware, the consumer's try_wait makes the data visible)
__device__ __forceinline__ void jc_st_async2(uint32_t addr, double2 v, uint32_t mbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];"
                 ::"r"(addr), "d"(v.x), "d"(v.y), "r"(mbar) : "memory");
}
// progress words: relaxed cluster-scope accesses (no MEMBAR.GPU / CCTL.IVALL, which release / acquire at cluster scope cost).
// They carry no data: a V CTA posts a round after its CTA barrier, when every load of the ring slot has been consumed.
__device__ __forceinline__ void jc_st_relaxed_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.relaxed.cluster.shared::cluster.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t jc_ld_relaxed_u32(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.relaxed.cluster.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(jc_smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t jc_ld_relaxed_u32a(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.relaxed.cluster.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void jc_mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(jc_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void jc_mbar_expect(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(jc_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void jc_mbar_wait(uint64_t* bar, uint32_t parity)
{
    const uint32_t addr = jc_smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void jc_cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// shared-memory accesses at a 32-bit shared address + compile-time byte offset (the generic pointers of a cluster launch make
// the compiler rebuild the shared window base from SR_CgaCtaId inside the loop)
template <int OFF> __device__ __forceinline__ double jc_lds(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(a), "n"(OFF) : "memory");
    return v;
}
template <int OFF> __device__ __forceinline__ double2 jc_lds2(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(v.x), "=d"(v.y) : "r"(a), "n"(OFF) : "memory");
    return v;
}
template <int OFF> __device__ __forceinline__ void jc_sts(uint32_t a, double v)
{
    asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(a), "n"(OFF), "d"(v) : "memory");
}
template <int OFF> __device__ __forceinline__ void jc_sts2(uint32_t a, double2 v)
{
    asm volatile("st.shared.v2.f64 [%0+%1], {%2, %3};" ::"r"(a), "n"(OFF), "d"(v.x), "d"(v.y) : "memory");
}

constexpr int JSV_NS = 8;          // ring slots of rotations in a V CTA
constexpr int JSV_SBUF = 62 * 62;  // doubles per ping-pong buffer of S / of a V CTA's rows (compile-time: the buffer switch is an immediate offset)
constexpr int JSV_RBUF = 32;       // rotations per ping-pong buffer

struct JsvHeader {                 // at the start of every CTA's dynamic shared memory (same offsets: mapa)
    uint64_t full[JSV_NS];         // V CTAs: slot filled (the V CTA's own arrive + 16 m bytes stored by CTA 0's rotation lanes)
    uint32_t vprog[8];             // CTA 0: rounds V CTA v has finished
    uint32_t verdict;              // V CTAs: 2 * (sweeps decided) + converged
    uint32_t pad[7];
};

template <int NV>
__global__ void __launch_bounds__(704) jacobi_sv_kernel(int K, int Kp, const double* __restrict__ Qall,
                                                         const double* __restrict__ freqs, double* __restrict__ lam,
                                                         double* __restrict__ Uout, double* __restrict__ sp_out,
                                                         double* __restrict__ isp_out, int32_t* __restrict__ status,
                                                         int M, const int32_t* __restrict__ eproc)
{
    extern __shared__ __align__(16) double sm[];
    constexpr int G = NV + 1, NS = JSV_NS;
    const int e = blockIdx.x / G;                       // the whole cluster serves (or skips) one process
    if (eproc[e] != e) return;
    uint32_t g;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(g));
    const int m = (K + 1) >> 1, n = 2 * m;
    const int tid = threadIdx.x, T = blockDim.x;
    JsvHeader* const hd = reinterpret_cast<JsvHeader*>(sm);
    double2* const ring = reinterpret_cast<double2*>(hd + 1);                             // [NS][m] (V CTAs)
    double* const body = reinterpret_cast<double*>(ring + NS * m);
    const double* Q = Qall + (size_t)e * K * K;
    const double* pi = freqs + (size_t)e * K;

    if (tid == 0) {
        for (int q = 0; q < NS; q++) { jc_mbar_init(&hd->full[q], 1); if (g != 0) jc_mbar_expect(&hd->full[q], 16u * (uint32_t)m); }
        for (int q = 0; q < 8; q++) hd->vprog[q] = 0;
        hd->verdict = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    if (g == 0) {
        // ------------------------------------------------------------------------------------------ CTA 0: S and the rotations
        const int ld = n;                   // even stride: the rotation lanes' diagonal walks (stride ld + 1) are conflict free
        double* const S0 = body;                                                          // [2][JSV_SBUF] = [2][n][ld], entries p <= q
        double2* const R0 = reinterpret_cast<double2*>(S0 + 2 * JSV_SBUF);                // [2][JSV_RBUF] (cos, sin)
        double* const red = reinterpret_cast<double*>(R0 + 2 * JSV_RBUF);                 // [33]
        auto sidx = [&](int p, int q) { return min(p, q) * ld + max(p, q); };
        for (int idx = tid; idx < n * n; idx += T) {    // position = state index at the start of every sweep
            const int i = idx / n, j = idx - i * n;
            if (i > j) continue;
            double v = 0.0;
            if (i < K && j < K) {
                const double a = sqrt(pi[i]) * Q[i * K + j] / sqrt(pi[j]);
                const double b = sqrt(pi[j]) * Q[j * K + i] / sqrt(pi[i]);
                v = 0.5 * (a + b);
            }
            S0[i * ld + j] = v;
        }
        __syncthreads();
        auto block_sum = [&](double v) -> double {      // all threads call
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if ((tid & 31) == 0) red[tid >> 5] = v;
            __syncthreads();
            double t = 0;
            for (int w = 0; w < T / 32; w++) t += red[w];
            __syncthreads();
            return t;
        };
        double tot2;
        {
            double t = 0;
            for (int idx = tid; idx < n * n; idx += T) {
                const int i = idx / n, j = idx - i * n;
                if (i <= j) { const double x = S0[i * ld + j]; t += i == j ? x * x : 2.0 * x * x; }
            }
            tot2 = block_sum(t);
        }
        // per-thread constants: block (a, b), a <= b = rows {a, m+a} x columns {b, m+b}; row a of the triangle has m - a blocks
        // Warp w runs on scheduler w % 4.  The rotations are the serial chain of a round (~25 dependent fp64 operations),
        // so the rotation warp (warp 3) gets a scheduler and its fp64 lanes to itself: the block threads use the warps
        // with w % 4 != 3 only, the other warps of scheduler 3 idle at the barrier.
        const int nblk = m * (m + 1) / 2;
        const int wid = tid >> 5;
        const int bt = (wid & 3) == 3 ? -1 : ((wid - (wid >> 2)) << 5) + (tid & 31);
        const bool is_blk = bt >= 0 && bt < nblk;
        int a = 0, b = 0;
        if (is_blk) {
            int rem = bt;
            while (rem >= m - a) { rem -= m - a; a++; }
            b = a + rem;
        }
        const bool diag = a == b;
        const int r00 = sidx(a, b), r01 = sidx(a, m + b), r10 = sidx(m + a, b), r11 = sidx(m + a, m + b);
        const int pt = jac_newpos(a, m), pb = jac_newpos(m + a, m), qt = jac_newpos(b, m), qb = jac_newpos(m + b, m);
        const int w00 = sidx(pt, qt), w01 = sidx(pt, qb), w10 = sidx(pb, qt), w11 = sidx(pb, qb);
        // rotation warp, lane j < m: the players that form NEW pair j sit at old positions x (-> T_j) and y (-> B_j)
        const int j = tid - 96;
        const bool is_rot = j >= 0 && j < m;
        int x = 0, y = m;
        if (is_rot)
            for (int p = 0; p < n; p++) {
                const int q = jac_newpos(p, m);
                if (q == j) x = p;
                if (q == m + j) y = p;
            }
        const int ax = x % m, ay = y % m, px = x / m, py = y / m;
        const int i_app = sidx(ax, ax), i_apq = sidx(ax, m + ax), i_aqq = sidx(m + ax, m + ax);
        const int i_bpp = sidx(ay, ay), i_bpq = sidx(ay, m + ay), i_bqq = sidx(m + ay, m + ay);
        // block (ax, ay) by position (sidx picks the stored copy of a symmetric entry)
        const int i_x00 = sidx(ax, ay), i_x01 = sidx(ax, m + ay), i_x10 = sidx(m + ax, ay), i_x11 = sidx(m + ax, m + ay);
        const uint32_t ring_u32 = jc_smem_u32(ring), full_u32 = jc_smem_u32(&hd->full[0]), vprog_u32 = jc_smem_u32(&hd->vprog[0]);
        uint32_t ring_v[NV], full_v[NV];
#pragma unroll
        for (int v = 0; v < NV; v++) { ring_v[v] = jc_mapa(ring_u32, v + 1); full_v[v] = jc_mapa(full_u32, v + 1); }
        auto push0 = [&](double2 nr) {                  // the first rotations (round 0): every slot is free
#pragma unroll
            for (int v = 0; v < NV; v++) jc_st_async2(ring_v[v] + 16u * (uint32_t)j, nr, full_v[v]);
        };
        jc_cluster_barrier();                           // every CTA of the cluster is running, its barriers initialised
        if (is_rot) {
            const double2 nr = jac_rotation(S0[sidx(j, j)], S0[sidx(m + j, m + j)], S0[sidx(j, m + j)]);
            R0[j] = nr;
            push0(nr);
        }
        __syncthreads();

        // Per-thread base pointers; the buffer of a round is a compile-time offset (the round body is instantiated for both
        // parities), so a round is loads / stores at register + immediate and no address arithmetic: the block warps issue
        // 27 instructions per round instead of 58, and the rotation lanes' operand loads leave at once.
        const uint32_t s_u32 = jc_smem_u32(S0), r_u32 = jc_smem_u32(R0);
        uint32_t p00 = s_u32 + 8 * r00, p01 = s_u32 + 8 * r01, p10 = s_u32 + 8 * r10, p11 = s_u32 + 8 * r11;
        uint32_t q00 = s_u32 + 8 * w00, q01 = s_u32 + 8 * w01, q10 = s_u32 + 8 * w10, q11 = s_u32 + 8 * w11;
        uint32_t Ra = r_u32 + 16 * a, Rb = r_u32 + 16 * b;
        uint32_t o_app = s_u32 + 8 * i_app, o_apq = s_u32 + 8 * i_apq, o_aqq = s_u32 + 8 * i_aqq, o_bpp = s_u32 + 8 * i_bpp,
                 o_bpq = s_u32 + 8 * i_bpq, o_bqq = s_u32 + 8 * i_bqq, o_x00 = s_u32 + 8 * i_x00, o_x01 = s_u32 + 8 * i_x01,
                 o_x10 = s_u32 + 8 * i_x10, o_x11 = s_u32 + 8 * i_x11;
        uint32_t Rax = r_u32 + 16 * ax, Ray = r_u32 + 16 * ay, Rj = r_u32 + 16 * (is_rot ? j : 0);
        JC_PIN(p00); JC_PIN(p01); JC_PIN(p10); JC_PIN(p11); JC_PIN(q00); JC_PIN(q01); JC_PIN(q10); JC_PIN(q11); JC_PIN(Ra); JC_PIN(Rb);
        JC_PIN(o_app); JC_PIN(o_apq); JC_PIN(o_aqq); JC_PIN(o_bpp); JC_PIN(o_bpq); JC_PIN(o_bqq);
        JC_PIN(o_x00); JC_PIN(o_x01); JC_PIN(o_x10); JC_PIN(o_x11); JC_PIN(Rax); JC_PIN(Ray); JC_PIN(Rj);
        int f_blk = is_blk, f_diag = diag, f_rot = is_rot, f_px = px, f_py = py, f_axy = ax != ay, rounds = n - 1;
        JC_PIN(f_blk); JC_PIN(f_diag); JC_PIN(f_rot); JC_PIN(f_px); JC_PIN(f_py); JC_PIN(f_axy); JC_PIN(rounds);
        uint32_t vprog_a = vprog_u32, ring_lane[NV], full_a[NV], slot_stride = 16u * (uint32_t)m;
#pragma unroll
        for (int v = 0; v < NV; v++) { ring_lane[v] = ring_v[v] + 16u * (uint32_t)(is_rot ? j : 0); full_a[v] = full_v[v]; JC_PIN(ring_lane[v]); JC_PIN(full_a[v]); }
        JC_PIN(vprog_a); JC_PIN(slot_stride);
        auto push = [&](int t, double2 nr, const uint32_t* seen) {   // rotation lane: rotation j of global round t to every V CTA
            const uint32_t slot = (uint32_t)t % NS;
#pragma unroll
            for (int v = 0; v < NV; v++) {
                if ((int)seen[v] < t + 1 - NS)
                    while ((int)jc_ld_relaxed_u32a(vprog_a + 4 * v) < t + 1 - NS) { }     // slot free (never waits in practice)
                jc_st_async2(ring_lane[v] + slot * slot_stride, nr, full_a[v] + 8u * slot);
            }
        };
        // Warp-specialised rounds: the block warps and the rotation warp run their own small loops (each scheduler's
        // instruction cache holds one of them) and meet at a named barrier that only they join; the other warps of
        // scheduler 3 sleep until the end of the sweep.
        const int nbw = (nblk + 31) >> 5;                                   // block warps
        const bool blk_warp = (wid & 3) != 3 && (wid - (wid >> 2)) < nbw;
        const bool rot_warp = wid == 3;
        int nbar = 32 * (nbw + 1);
        JC_PIN(nbar);
        auto round_barrier = [&]() { asm volatile("bar.sync 1, %0;" ::"r"(nbar) : "memory"); };
        int t = 0;
        double my_off = 0.0;
        auto blk_round = [&](auto CURC, bool last) {
            constexpr int CUR = decltype(CURC)::value, SO = 8 * CUR * JSV_SBUF, SN = 8 * (CUR ^ 1) * JSV_SBUF, RO = 16 * CUR * JSV_RBUF;
            if (f_blk) {
                const double2 ra = jc_lds2<RO>(Ra), rbb = jc_lds2<RO>(Rb);
                const double x00 = jc_lds<SO>(p00), x01 = jc_lds<SO>(p01), x10 = jc_lds<SO>(p10), x11 = jc_lds<SO>(p11);
                // columns (pair b), then rows (pair a): S <- J^T S J on this 2x2 block
                const double t00 = rbb.x * x00 - rbb.y * x01, t01 = rbb.y * x00 + rbb.x * x01;
                const double t10 = rbb.x * x10 - rbb.y * x11, t11 = rbb.y * x10 + rbb.x * x11;
                const double y00 = ra.x * t00 - ra.y * t10, y01 = ra.x * t01 - ra.y * t11;
                const double y10 = ra.y * t00 + ra.x * t10, y11 = ra.y * t01 + ra.x * t11;
                // (the rotated pivot of a diagonal block is stored as computed, not forced to zero: the iteration stays an
                // orthogonal similarity to rounding)
                jc_sts<SN>(q00, y00); jc_sts<SN>(q01, y01); jc_sts<SN>(q11, y11);
                if (!f_diag) jc_sts<SN>(q10, y10);                    // (a diagonal block's w10 is its w01)
                if (last) my_off = f_diag ? 2.0 * y01 * y01 : 2.0 * fma(y00, y00, fma(y01, y01, fma(y10, y10, y11 * y11)));
            }
            round_barrier();
        };
        auto rot_round = [&](auto CURC) {
            constexpr int CUR = decltype(CURC)::value, SO = 8 * CUR * JSV_SBUF, RO = 16 * CUR * JSV_RBUF, RN = 16 * (CUR ^ 1) * JSV_RBUF;
            if (f_rot) {
                double2 nr = make_double2(1.0, 0.0);
                uint32_t seen[NV];                           // the V CTAs' progress, read beside the operands
#pragma unroll
                for (int v = 0; v < NV; v++) seen[v] = jc_ld_relaxed_u32a(vprog_a + 4 * v);
                if (f_axy) {
                    const double2 ra = jc_lds2<RO>(Rax), rbb = jc_lds2<RO>(Ray);
                    const double app = jc_lds<SO>(o_app), apq = jc_lds<SO>(o_apq), aqq = jc_lds<SO>(o_aqq);
                    const double bpp = jc_lds<SO>(o_bpp), bpq = jc_lds<SO>(o_bpq), bqq = jc_lds<SO>(o_bqq);
                    const double x00 = jc_lds<SO>(o_x00), x01 = jc_lds<SO>(o_x01), x10 = jc_lds<SO>(o_x10), x11 = jc_lds<SO>(o_x11);
                    // the player's updated diagonal entry: (J^T S J)_pp = c^2 Spp - 2 c s Spq + s^2 Sqq, _qq = s^2 Spp + 2 c s Spq + c^2 Sqq
                    const double ca2 = ra.x * ra.x, sa2 = ra.y * ra.y, csa = 2.0 * ra.x * ra.y;
                    const double cb2 = rbb.x * rbb.x, sb2 = rbb.y * rbb.y, csb = 2.0 * rbb.x * rbb.y;
                    const double dx = f_px ? fma(sa2, app, fma(csa, apq, ca2 * aqq)) : fma(ca2, app, fma(-csa, apq, sa2 * aqq));
                    const double dy = f_py ? fma(sb2, bpp, fma(csb, bpq, cb2 * bqq)) : fma(cb2, bpp, fma(-csb, bpq, sb2 * bqq));
                    // the new pivot = entry (px, py) of the updated block (ax, ay)
                    const double t0 = f_py ? rbb.y * x00 + rbb.x * x01 : rbb.x * x00 - rbb.y * x01;
                    const double t1 = f_py ? rbb.y * x10 + rbb.x * x11 : rbb.x * x10 - rbb.y * x11;
                    const double piv = f_px ? ra.y * t0 + ra.x * t1 : ra.x * t0 - ra.y * t1;
                    nr = jac_rotation(dx, dy, piv);
                }
                jc_sts2<RN>(Rj, nr);
                push(t + 1, nr, seen);
            }
            round_barrier();
        };
        int cur = 0;
        bool converged = false;
        double off2 = 0.0;
        for (int sweep = 0; sweep < 40 && !converged; sweep++) {
            if (blk_warp) {
                for (int r = 0; r < rounds; r++) {
                    if (((cur + r) & 1) == 0) blk_round(std::integral_constant<int, 0>{}, r == rounds - 1);
                    else blk_round(std::integral_constant<int, 1>{}, r == rounds - 1);
                }
            } else if (rot_warp) {
                for (int r = 0; r < rounds; r++, t++) {
                    if (((cur + r) & 1) == 0) rot_round(std::integral_constant<int, 0>{});
                    else rot_round(std::integral_constant<int, 1>{});
                }
            }
            cur = (cur + n - 1) & 1;
            off2 = block_sum(my_off);
            converged = off2 <= 0.25 * 2.220446049250313e-16 * 2.220446049250313e-16 * tot2;
            if (tid < NV) jc_st_relaxed_u32(jc_mapa(jc_smem_u32(&hd->verdict), tid + 1), 2u * (uint32_t)(sweep + 1) + (converged || sweep == 39 ? 1u : 0u));
        }
        if (tid == 0 && !(off2 <= 1e-28 * tot2)) atomicOr(status, EPX_ST_JACOBI_NOCONV);
        const double* S = S0 + cur * JSV_SBUF;
        for (int f = e; f < M; f++) {             // every epoch of this process gets the eigensystem
            if (eproc[f] != e) continue;
            for (int i = tid; i < Kp; i += T) {
                lam[(size_t)f * Kp + i] = i < K ? S[i * ld + i] : 0.0;
                sp_out[(size_t)f * Kp + i] = i < K ? sqrt(pi[i]) : 0.0;
                isp_out[(size_t)f * Kp + i] = i < K ? 1.0 / sqrt(pi[i]) : 0.0;
            }
            double* U = Uout + (size_t)f * Kp * Kp;
            for (int idx = K * Kp + tid; idx < Kp * Kp; idx += T) U[idx] = 0.0;          // padding rows
        }
    } else {
        // ------------------------------------------------------------------------------------------ CTAs 1..NV: rows of V
        const int rv = (K + NV - 1) / NV, i_lo = ((int)g - 1) * rv, rcnt = max(0, min(rv, K - i_lo));
        double* const V0 = body;                                                          // [2][JSV_SBUF] = [2][rv][n], columns in position order
        const int vn = rv * n;
        for (int idx = tid; idx < vn; idx += T) { const int i = idx / n, jj = idx - i * n; V0[idx] = (i_lo + i == jj) ? 1.0 : 0.0; }
        const bool is_v = tid < rcnt * m;
        const int il = is_v ? tid / m : 0, b = is_v ? tid % m : 0;
        const double *vr0 = V0 + il * n + b, *vr1 = V0 + il * n + m + b;
        double *vw0 = V0 + il * n + jac_newpos(b, m), *vw1 = V0 + il * n + jac_newpos(m + b, m);
        const uint32_t vprog_remote = jc_mapa(jc_smem_u32(&hd->vprog[g - 1]), 0);
        jc_cluster_barrier();
        __syncthreads();
        int cur = 0, t = 0;
        auto round = [&](auto CURC) {
            constexpr int CUR = decltype(CURC)::value, VO = CUR * JSV_SBUF, VN = (CUR ^ 1) * JSV_SBUF;
            const int slot = t % NS;
            jc_mbar_wait(&hd->full[slot], (uint32_t)((t / NS) & 1));
            if (is_v) {
                const double2 rbb = ring[slot * m + b];
                const double v0 = vr0[VO], v1 = vr1[VO];
                vw0[VN] = rbb.x * v0 - rbb.y * v1;
                vw1[VN] = rbb.y * v0 + rbb.x * v1;
            }
            __syncthreads();
            if (tid == 0) {
                jc_mbar_expect(&hd->full[slot], 16u * (uint32_t)m);          // arm the slot for round t + NS ...
                jc_st_relaxed_u32(vprog_remote, (uint32_t)(t + 1));          // ... and hand it back to CTA 0
            }
        };
        bool done = false;
        for (int sweep = 0; !done; sweep++) {
            for (int r = 0; r < n - 1; r++, t++) {
                if (cur == 0) round(std::integral_constant<int, 0>{});
                else round(std::integral_constant<int, 1>{});
                cur ^= 1;
            }
            uint32_t vd;
            while (((vd = jc_ld_relaxed_u32(&hd->verdict)) >> 1) <= (uint32_t)sweep) { }
            done = vd & 1u;
        }
        const double* V = V0 + cur * JSV_SBUF;
        for (int f = e; f < M; f++) {
            if (eproc[f] != e) continue;
            double* U = Uout + (size_t)f * Kp * Kp;
            for (int idx = tid; idx < rcnt * Kp; idx += T) {
                const int i = idx / Kp, jj = idx - i * Kp;
                U[(size_t)(i_lo + i) * Kp + jj] = jj < K ? V[i * n + jj] : 0.0;
            }
        }
    }
    jc_cluster_barrier();                               // nobody leaves while a peer may still store into its shared memory
}

size_t jacobi_sv_smem(int K, int NV)
{
    const size_t m = (K + 1) / 2, n = 2 * m, rv = (K + NV - 1) / NV;
    const size_t s_cta = sizeof(double) * (2 * JSV_SBUF + 4 * JSV_RBUF + 34);
    const size_t v_cta = sizeof(double) * (JSV_SBUF + rv * n);
    const size_t need = sizeof(JsvHeader) + 16 * JSV_NS * m + (s_cta > v_cta ? s_cta : v_cta) + 16;
    // more than half of an SM's shared memory: the CTAs of a cluster must sit on different SMs (a V CTA beside CTA 0 would
    // take the issue slots and shared-memory bandwidth the split is there to free)
    return need > 120 * 1024 ? need : 120 * 1024;
}

// ------------------------------------------------------------------------------------------------ K == 4: one warp, no shared memory
// The 4-state models sit on the critical path of every nucleotide evaluation (a3 / a4 wait for them; 13 us in jacobi1_kernel:
// 20 rounds of a CTA barrier and a rotation chain through shared memory).  Here a warp holds everything in registers: lane
// 4 i + j of the lower half owns S[i][j], of the upper half V[i][j].  The three rounds of a sweep pair index t with t ^ 1, t ^ 2,
// t ^ 3, so a partner row / column is the lane with those bits flipped: a round is 6 shuffles for the two rotations (every lane
// computes both), 3 for the 2x2 update and a dozen fp64 operations; no barrier anywhere.
__global__ void __launch_bounds__(32) jacobi4_kernel(const double* __restrict__ Qall, const double* __restrict__ freqs,
                                                     double* __restrict__ lam, double* __restrict__ Uout, double* __restrict__ sp_out,
                                                     double* __restrict__ isp_out, int32_t* __restrict__ status, int M,
                                                     const int32_t* __restrict__ eproc)
{
    constexpr unsigned FULL = 0xffffffffu;
    const int e = blockIdx.x;
    if (eproc[e] != e) return;                          // f2: this epoch shares the process of an earlier one
    const int lane = threadIdx.x, i = (lane >> 2) & 3, j = lane & 3;
    const bool is_s = lane < 16;
    const double* Q = Qall + (size_t)e * 16;
    const double* pi = freqs + (size_t)e * 4;
    double x;
    {
        const double si = sqrt(pi[i]), sj = sqrt(pi[j]);
        const double a = si * Q[i * 4 + j] / sj, b = sj * Q[j * 4 + i] / si;
        x = is_s ? 0.5 * (a + b) : (i == j ? 1.0 : 0.0);
    }
    auto warp_sum = [&](double v) { for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o); return v; };
    const double tot2 = warp_sum(is_s ? x * x : 0.0);
    double off2 = 0.0;
    bool converged = false;
    for (int sweep = 0; sweep < 40 && !converged; sweep++) {
#pragma unroll
        for (int m = 1; m <= 3; m++) {                  // pairs (t, t ^ m); p = the smaller index
            const int ip = i ^ m, jp = j ^ m;
            const int pi_ = min(i, ip), qi = max(i, ip), pj = min(j, jp), qj = max(j, jp);
            // the two rotations this lane needs, from the S half (every lane computes them: no broadcast step)
            const double2 ri = jac_rotation(__shfl_sync(FULL, x, 5 * pi_), __shfl_sync(FULL, x, 5 * qi), __shfl_sync(FULL, x, 4 * pi_ + qi));
            const double2 rj = jac_rotation(__shfl_sync(FULL, x, 5 * pj), __shfl_sync(FULL, x, 5 * qj), __shfl_sync(FULL, x, 4 * pj + qj));
            const double xj = __shfl_xor_sync(FULL, x, m);           // same row, partner column
            const double xi = __shfl_xor_sync(FULL, x, m << 2);      // partner row, same column
            const double xij = __shfl_xor_sync(FULL, x, m | (m << 2));
            // new column p = c col_p - s col_q, new column q = s col_p + c col_q (and the same for rows): S <- J^T S J, V <- V J
            const double bj = j < jp ? -rj.y : rj.y, bi = i < ip ? -ri.y : ri.y;
            const double row_own = fma(bj, xj, rj.x * x), row_par = fma(bj, xij, rj.x * xi);
            x = is_s ? fma(bi, row_par, ri.x * row_own) : row_own;
        }
        off2 = warp_sum(is_s && i != j ? x * x : 0.0);
        converged = off2 <= 0.25 * 2.220446049250313e-16 * 2.220446049250313e-16 * tot2;
    }
    if (lane == 0 && !(off2 <= 1e-28 * tot2)) atomicOr(status, EPX_ST_JACOBI_NOCONV);
    for (int f = e; f < M; f++) {                       // every epoch of this process gets the eigensystem (Kp == K == 4)
        if (eproc[f] != e) continue;
        if (!is_s) Uout[(size_t)f * 16 + 4 * i + j] = x;
        else if (i == j) lam[(size_t)f * 4 + i] = x;
        if (lane < 4) { sp_out[(size_t)f * 4 + lane] = sqrt(pi[lane]); isp_out[(size_t)f * 4 + lane] = 1.0 / sqrt(pi[lane]); }
    }
}

size_t jacobi1_smem(int K)
{
    const size_t m = (K + 1) / 2, n = 2 * m;
    return sizeof(double) * (2 * n * n + 2 * (size_t)K * n + 4 * m + 34) + 16;
}

constexpr int JT = 256;   // threads per CTA of the prep kernels

// W_e[a][b] = sum_k U_e[k][a] * sqrt(pi_e[k] / pi_{e-1}[k]) * U_{e-1}[k][b]   (e >= 1)
// Fragment order (lane = 4g + q of an m8n8k4 DMMA; the contraction index of k-step (kt,h) at position q is
// kappa = 8kt + 2q + h, i.e. exactly the column a C-fragment register h of accumulator tile kt holds):
//   XB[((kt*8 + nt)*32 + lane)*2 + h] = X[kappa][8nt + g]
__global__ void __launch_bounds__(JT) prep_kernel(int Kp, const double* __restrict__ U, const double* __restrict__ sp,
                                                  const double* __restrict__ isp, double* __restrict__ W,
                                                  double* __restrict__ WB, double* __restrict__ UTB)
{
    const int e = blockIdx.x, tid = threadIdx.x;
    const double* Ue = U + (size_t)e * Kp * Kp;
    double* We = W + (size_t)e * Kp * Kp;
    if (e >= 1 && Kp <= 32) {
        // both operands staged in shared memory once (the loop below was a chain of dependent global loads: 19 us for K = 20)
        __shared__ double ue[32 * 33], um[32 * 32];
        const double* Um = U + (size_t)(e - 1) * Kp * Kp;
        const double* spe = sp + (size_t)e * Kp;
        const double* ispm = isp + (size_t)(e - 1) * Kp;
        for (int idx = tid; idx < Kp * Kp; idx += JT) {
            const int k = idx / Kp, a = idx % Kp;
            ue[a * 33 + k] = Ue[idx] * (spe[k] * ispm[k]);      // transposed: thread (a, b) walks its row
            um[idx] = Um[idx];
        }
        __syncthreads();
        for (int idx = tid; idx < Kp * Kp; idx += JT) {
            const int a = idx / Kp, b = idx % Kp;
            double acc = 0.0;
            for (int k = 0; k < Kp; k++) acc = fma(ue[a * 33 + k], um[k * Kp + b], acc);
            We[idx] = acc;
        }
    } else if (e >= 1) {
        const double* Um = U + (size_t)(e - 1) * Kp * Kp;
        const double* spe = sp + (size_t)e * Kp;
        const double* ispm = isp + (size_t)(e - 1) * Kp;
        for (int idx = tid; idx < Kp * Kp; idx += JT) {
            int a = idx / Kp, b = idx % Kp;
            double acc = 0.0;
            for (int k = 0; k < Kp; k++) acc = fma(Ue[k * Kp + a] * (spe[k] * ispm[k]), Um[k * Kp + b], acc);
            We[idx] = acc;
        }
    } else {
        for (int idx = tid; idx < Kp * Kp; idx += JT) We[idx] = 0.0;
    }
    if (Kp != 64) return;
    __syncthreads();   // We written by this CTA is read back below
    double* WBe = WB + (size_t)e * 4096;
    double* UTBe = UTB + (size_t)e * 4096;
    for (int idx = tid; idx < 4096; idx += JT) {
        int h = idx & 1, lane = (idx >> 1) & 31, nt = (idx >> 6) & 7, kt = idx >> 9;
        int g = lane >> 2, q = lane & 3;
        int kappa = 8 * kt + 2 * q + h, col = 8 * nt + g;
        WBe[idx] = We[kappa * 64 + col];
        UTBe[idx] = Ue[col * 64 + kappa];      // U^T[kappa][col]
    }
}


// 64-padded models: grid (M, 8), CTA (e, y) computes rows 8y .. 8y+7 of W_e and writes W, WB and UTB directly.
__global__ void __launch_bounds__(JT) prep64_kernel(const double* __restrict__ U, const double* __restrict__ sp,
                                                    const double* __restrict__ isp, double* __restrict__ W,
                                                    double* __restrict__ WB, double* __restrict__ UTB)
{
    __shared__ double ue[64][8];      // U_e[k][a0 + j] * sqrt(pi_e[k] / pi_{e-1}[k])
    const int e = blockIdx.x, a0 = blockIdx.y * 8, tid = threadIdx.x;
    const double* Ue = U + (size_t)e * 4096;
    const int b = tid & 63, ar = tid >> 6;
    double acc[2] = {0.0, 0.0};
    if (e >= 1) {
        const double* Um = U + (size_t)(e - 1) * 4096;
        for (int idx = tid; idx < 512; idx += JT) {
            const int k = idx >> 3, j = idx & 7;
            ue[k][j] = Ue[k * 64 + a0 + j] * (sp[(size_t)e * 64 + k] * isp[(size_t)(e - 1) * 64 + k]);
        }
        __syncthreads();
#pragma unroll 8
        for (int k = 0; k < 64; k++) {
            const double um = Um[k * 64 + b];
            acc[0] = fma(ue[k][ar], um, acc[0]);
            acc[1] = fma(ue[k][ar + 4], um, acc[1]);
        }
    }
#pragma unroll
    for (int h2 = 0; h2 < 2; h2++) {
        const int a = a0 + ar + 4 * h2;                 // row (contraction index kappa of the B fragment), column b
        const int kt = a >> 3, q = (a & 7) >> 1, h = a & 1, nt = b >> 3, g = b & 7;
        const int idx = ((kt * 8 + nt) * 32 + 4 * g + q) * 2 + h;
        W[(size_t)e * 4096 + a * 64 + b] = acc[h2];
        WB[(size_t)e * 4096 + idx] = acc[h2];
        UTB[(size_t)e * 4096 + idx] = Ue[b * 64 + a];   // U^T[a][b]
    }
}

}  // namespace

int eigen_init_attributes()
{
    if (cudaFuncSetAttribute(jacobi1_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)jacobi1_smem(62)) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(jacobi_sv_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)jacobi_sv_smem(62, 3)) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(jacobi_sv_kernel<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)jacobi_sv_smem(62, 7)) != cudaSuccess) return -1;
    return cudaFuncSetAttribute(jacobi_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024) == cudaSuccess ? 0 : -1;
}

int launch_eigensystems(const epx_ctx* c, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    const int K = c->K, Kp = c->Kp;
    const int ld = K | 1;
    size_t smem = sizeof(double) * (2 * (size_t)K * ld + 2 * (K / 2 + 1) + 32) + sizeof(int) * 2 * (K / 2 + 1);
    const int jk = c->jacobi_kernel;           // 0 auto, 1 round-1 kernel, 2 one CTA per process, 14 / 18 clusters of 4 / 8
    if (K == 4 && jk == 0) {                   // one warp per process, everything in registers
        jacobi4_kernel<<<c->M, 32, 0, s>>>(d.Q, d.freqs, d.lam, d.U, d.sp, d.isp, d.status, c->M, d.eproc);
        if (c->chain_kernel == 0) return cudaGetLastError() == cudaSuccess ? 1 : -1;      // chain_rows_kernel<4> needs no W
        prep_kernel<<<c->M, JT, 0, s>>>(Kp, d.U, d.sp, d.isp, d.W, d.WB, d.UTB);
        return cudaGetLastError() == cudaSuccess ? 2 : -1;
    }
    const int G = (jk == 14 || jk == 18) ? jk - 10 : (jk == 0 && K > 32 && K <= 62) ? 4 : 1;
    if (K <= 62 && K >= 16 && G > 1) {
        const int m = (K + 1) / 2, NV = G - 1, rv = (K + NV - 1) / NV;
        int warps = 4, bw = (m * (m + 1) / 2 + 31) / 32;   // CTA 0: block warps w % 4 != 3, the rotation warp is warp 3
        while (warps - warps / 4 < bw) warps++;
        warps = max(warps, (rv * m + 31) / 32);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(c->M * G)); cfg.blockDim = dim3((unsigned)(32 * warps));
        cfg.dynamicSmemBytes = jacobi_sv_smem(K, NV); cfg.stream = s;
        cudaLaunchAttribute attr;
        attr.id = cudaLaunchAttributeClusterDimension;
        attr.val.clusterDim.x = (unsigned)G; attr.val.clusterDim.y = 1; attr.val.clusterDim.z = 1;
        cfg.attrs = &attr; cfg.numAttrs = 1;
        auto kern = G == 4 ? jacobi_sv_kernel<3> : jacobi_sv_kernel<7>;
        cudaLaunchKernelEx(&cfg, kern, K, Kp, (const double*)d.Q, (const double*)d.freqs, d.lam, d.U, d.sp, d.isp, d.status, c->M,
                           (const int32_t*)d.eproc);
    } else if (K <= 62 && jk != 1) {
        const int m = (K + 1) / 2;
        jacobi1_kernel<<<c->M, ((m * m + 31) & ~31) + 32, jacobi1_smem(K), s>>>(K, Kp, d.Q, d.freqs, d.lam, d.U, d.sp, d.isp, d.status, c->M, d.eproc);
    } else {
        jacobi_kernel<<<c->M, K > 32 ? JT_MAX : 256, smem, s>>>(K, Kp, d.Q, d.freqs, d.lam, d.U, d.sp, d.isp, d.status, c->M, d.eproc);
    }
    if (Kp == 64) prep64_kernel<<<dim3(c->M, 8), JT, 0, s>>>(d.U, d.sp, d.isp, d.W, d.WB, d.UTB);
    else prep_kernel<<<c->M, JT, 0, s>>>(Kp, d.U, d.sp, d.isp, d.W, d.WB, d.UTB);
    return cudaGetLastError() == cudaSuccess ? 2 : -1;
}
