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

namespace {

constexpr int JT = 256;   // threads per CTA

__global__ void __launch_bounds__(JT) jacobi_kernel(int K, int Kp, const double* __restrict__ Qall,
                                                    const double* __restrict__ freqs, double* __restrict__ lam,
                                                    double* __restrict__ Uout, double* __restrict__ sp_out,
                                                    double* __restrict__ isp_out, int32_t* __restrict__ status)
{
    extern __shared__ double sm[];
    const int ld = K | 1;                       // odd row stride: column walks are bank-conflict free
    double* S = sm;                             // [K][ld]
    double* V = S + (size_t)K * ld;             // [K][ld]
    double* rc = V + (size_t)K * ld;            // [K/2+1] cos
    double* rs = rc + (K / 2 + 1);              // [K/2+1] sin
    double* red = rs + (K / 2 + 1);             // [JT/32] reduction scratch
    int* rp = (int*)(red + JT / 32);            // [K/2+1] p
    int* rq = rp + (K / 2 + 1);                 // [K/2+1] q
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
                    double apq = S[p * ld + q];
                    if (fabs(apq) > 1e-300) {
                        double theta = (S[q * ld + q] - S[p * ld + p]) / (2.0 * apq);
                        double t = 1.0 / (fabs(theta) + sqrt(theta * theta + 1.0));
                        if (theta < 0) t = -t;
                        c = 1.0 / sqrt(t * t + 1.0);
                        s = t * c;
                    }
                } else {
                    p = -1;
                }
                rp[tid] = p; rq[tid] = q; rc[tid] = c; rs[tid] = s;
            }
            __syncthreads();
            // columns: S <- S J, V <- V J
            for (int idx = tid; idx < npair * K; idx += JT) {
                int k = idx / K, i = idx % K, p = rp[k];
                if (p < 0) continue;
                int q = rq[k];
                double c = rc[k], s = rs[k];
                double x = S[i * ld + p], y = S[i * ld + q];
                S[i * ld + p] = c * x - s * y;
                S[i * ld + q] = s * x + c * y;
                x = V[i * ld + p]; y = V[i * ld + q];
                V[i * ld + p] = c * x - s * y;
                V[i * ld + q] = s * x + c * y;
            }
            __syncthreads();
            // rows: S <- J^T S ; the pivot pair is annihilated exactly
            for (int idx = tid; idx < npair * K; idx += JT) {
                int k = idx / K, j = idx % K, p = rp[k];
                if (p < 0) continue;
                int q = rq[k];
                double c = rc[k], s = rs[k];
                double x = S[p * ld + j], y = S[q * ld + j];
                double xp = c * x - s * y, yq = s * x + c * y;
                if (j == q) xp = 0.0;
                if (j == p) yq = 0.0;
                S[p * ld + j] = xp;
                S[q * ld + j] = yq;
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
    size_t smem = sizeof(double) * (2 * (size_t)K * ld + 2 * (K / 2 + 1) + JT / 32) + sizeof(int) * 2 * (K / 2 + 1);
    jacobi_kernel<<<c->M, JT, smem, s>>>(K, Kp, d.Q, d.freqs, d.lam, d.U, d.sp, d.isp, d.status);
    prep_kernel<<<c->M, JT, 0, s>>>(Kp, d.U, d.sp, d.isp, d.W, d.WB, d.UTB);
    return cudaGetLastError() == cudaSuccess ? 2 : -1;
}
