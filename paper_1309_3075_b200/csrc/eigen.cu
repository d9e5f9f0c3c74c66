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

namespace {

constexpr int JT_MAX = 1024;   // threads per CTA for K > 32 (one 2x2 block of S per thread and round); 256 otherwise

// Two-sided Jacobi, round-robin ordering: in one round the n/2 pivot pairs are disjoint, so S' = J^T S J splits into
// (n/2)^2 independent 2x2 blocks (rows of pair a, columns of pair b) that each depend on their own four entries and the
// two rotations only.  One thread per block applies the column and the row rotation in registers: two barriers per round
// instead of three, and 961 busy threads at K = 61.
__global__ void __launch_bounds__(JT_MAX) jacobi_kernel(int K, int Kp, const double* __restrict__ Qall,
                                                        const double* __restrict__ freqs, double* __restrict__ lam,
                                                        double* __restrict__ Uout, double* __restrict__ sp_out,
                                                        double* __restrict__ isp_out, int32_t* __restrict__ status)
{
    extern __shared__ double sm[];
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

    double* U = Uout + (size_t)e * Kp * Kp;
    for (int idx = tid; idx < Kp * Kp; idx += JT) {
        int i = idx / Kp, j = idx % Kp;
        U[idx] = (i < K && j < K) ? V[i * ld + j] : 0.0;
    }
    for (int i = tid; i < Kp; i += JT) {
        lam[(size_t)e * Kp + i] = i < K ? S[i * ld + i] : 0.0;
        sp_out[(size_t)e * Kp + i] = i < K ? sqrt(pi[i]) : 0.0;
        isp_out[(size_t)e * Kp + i] = i < K ? 1.0 / sqrt(pi[i]) : 0.0;
    }
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
    if (e >= 1) {
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
    return cudaFuncSetAttribute(jacobi_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024) == cudaSuccess ? 0 : -1;
}

int launch_eigensystems(const epx_ctx* c, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    const int K = c->K, Kp = c->Kp;
    const int ld = K | 1;
    size_t smem = sizeof(double) * (2 * (size_t)K * ld + 2 * (K / 2 + 1) + 32) + sizeof(int) * 2 * (K / 2 + 1);
    jacobi_kernel<<<c->M, K > 32 ? JT_MAX : 256, smem, s>>>(K, Kp, d.Q, d.freqs, d.lam, d.U, d.sp, d.isp, d.status);
    if (Kp == 64) prep64_kernel<<<dim3(c->M, 8), JT, 0, s>>>(d.U, d.sp, d.isp, d.W, d.WB, d.UTB);
    else prep_kernel<<<c->M, JT, 0, s>>>(Kp, d.U, d.sp, d.isp, d.W, d.WB, d.UTB);
    return cudaGetLastError() == cudaSuccess ? 2 : -1;
}
