// a2' + a3 + a4, asymmetric path: exp(Q_e r d) by [13/13] Pade scaling-and-squaring, chained per branch
// (P(t) = exp(tQ), citing Moler & Van Loan for its numerical evaluation; L84-L109 Eq.(5)-(7)).
// The paper only ever says "eigen decomposition" and is silent on asymmetric Q with complex spectra (reading A13);
// Pade needs no spectrum.  Textbook method (Higham 2005): A <- A / 2^s with ||A||_1 / 2^s <= theta_13,
//   U = A [A6 (b13 A6 + b11 A4 + b9 A2) + b7 A6 + b5 A4 + b3 A2 + b1 I]
//   V =    A6 (b12 A6 + b10 A4 + b8 A2) + b6 A6 + b4 A4 + b2 A2 + b0 I
//   (V - U) R = (V + U)   (Gauss-Jordan, partial pivoting), then R <- R^2 s times.
//
// pade_full_epoch_kernel: one CTA per (interior epoch, category): E = exp(Q_e r_c (tau_e - tau_{e-1})), the factor
//   every branch that spans the whole epoch uses (a2').
// pade_chain_kernel: one CTA per (slot, category): first and last segment by Pade, interior segments from the
//   full-epoch table, product accumulated left to right (parent end first) in shared memory; P written once.
#include "epx_internal.h"

namespace {

constexpr int PT_MAX = 512;  // threads per CTA: 512 for K > 32 (a 61 x 61 product is 8 row tiles x 2 groups of 4 column tiles = one
                             // item per warp; config 3 chain 0.264 -> 0.224 ms), 256 otherwise (K = 24 is barrier-bound in the
                             // Gauss-Jordan sweep: 512 threads measured 0.81 ms against 0.33 ms on config 4)
__host__ __device__ inline int pade_threads(int K) { return K > 32 ? 512 : 128; }

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// C = A B for dense K x K matrices in shared memory (row stride K).  The K^3 products of the scaling-and-squaring
// exponentials are where this file spends its time; they run on the FP64 tensor pipe: warp w owns the 8-row tiles w,
// w + 8, ..., all column tiles of a row tile accumulate in registers, fragments outside the matrix are zero.
template <int PT>
__device__ __forceinline__ void mm(int K, const double* __restrict__ A, const double* __restrict__ B,
                                   double* __restrict__ Cm)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, q = lane & 3;
    // Which matrix rows / columns form an 8-wide tile is free (the same map on the A rows, the B columns and the D entries).
    // Odd K (row stride odd): tile t of a 16-group takes {0, 4, 8, 12, 1, 5, 9, 13} + 2 (t & 1), so the half-warp that makes
    // one shared-memory wavefront (rows / columns g = 0..3 or 4..7, k = q) hits 16 different 8-byte banks; with consecutive rows
    // the stride-61 walks of the codon models were 2-way conflicts on every operand load (l1tex 84 %, the limiter of the kernel).
    const bool perm = K & 1;
    const int nt_n = perm ? 2 * ((K + 15) >> 4) : (K + 7) >> 3, nk = (K + 3) >> 2, ngrp = (nt_n + 3) >> 2;
    auto index = [&](int t, int gg) { return perm ? 16 * (t >> 1) + 2 * (t & 1) + 4 * (gg & 3) + (gg >> 2) : 8 * t + gg; };
    for (int item = w; item < nt_n * ngrp; item += PT / 32) {      // item = (row tile, group of four column tiles)
        const int mt = item / ngrp, n0 = 4 * (item - mt * ngrp);
        const int row = index(mt, g);
        const bool row_ok = row < K;
        {
            double acc[4][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
            int colB[4];
#pragma unroll
            for (int t = 0; t < 4; t++) colB[t] = index(n0 + t, g);
            // (operands outside the matrix: the load is unconditional at a clamped index and the VALUE is selected -- a guarded
            //  load may compile to a branch, and mma.sync needs the whole warp converged)
            const double* Arow = A + min(row, K - 1) * K;
            int colC[4];
#pragma unroll
            for (int t = 0; t < 4; t++) colC[t] = min(colB[t], K - 1);
            for (int kt = 0; kt < nk; kt++) {
                const int k = 4 * kt + q, kc = min(k, K - 1);
                const bool k_ok = k < K;
                const double av = Arow[kc];
                const double a = (row_ok && k_ok) ? av : 0.0;
                const double* Bk = B + kc * K;
#pragma unroll
                for (int t = 0; t < 4; t++) {
                    const double bv = Bk[colC[t]];
                    const double b = (k_ok && colB[t] < K) ? bv : 0.0;
                    dmma884(acc[t][0], acc[t][1], a, b);
                }
            }
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const int c0 = index(n0 + t, 2 * q), c1 = index(n0 + t, 2 * q + 1);
                if (row_ok && c0 < K) Cm[row * K + c0] = acc[t][0];
                if (row_ok && c1 < K) Cm[row * K + c1] = acc[t][1];
            }
        }
    }
    __syncthreads();
}

struct PadeBufs {
    double *A, *A2, *A4, *A6, *T1, *T2, *col;
    double* red;   // [PT_MAX/32 + 2]
};

// In: b.A holds the (unscaled) matrix.  Returns the buffer (b.T1 or b.T2) that holds exp(A).  All threads call.
template <int PT>
__device__ double* pade13(int K, PadeBufs& b, int32_t* status)
{
    const double c[14] = {64764752532480000.0, 32382376266240000.0, 7771770303897600.0, 1187353796428800.0,
                          129060195264000.0, 10559470521600.0, 670442572800.0, 33522128640.0, 1323241920.0,
                          40840800.0, 960960.0, 16380.0, 182.0, 1.0};
    const int tid = threadIdx.x, KK = K * K;
    // ||A||_1 = max column sum
    double m = 0.0;
    for (int j = tid; j < K; j += PT) {
        double s = 0.0;
        for (int i = 0; i < K; i++) s += fabs(b.A[i * K + j]);
        m = fmax(m, s);
    }
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((tid & 31) == 0) b.red[tid >> 5] = m;
    __syncthreads();
    double nrm = 0.0;
    for (int w = 0; w < PT / 32; w++) nrm = fmax(nrm, b.red[w]);
    int s = 0;
    if (nrm > 5.371920351148152) s = max(0, (int)ceil(log2(nrm / 5.371920351148152)));
    if (!(nrm < 1e300)) { s = 0; if (tid == 0) atomicOr(status, EPX_ST_NONFINITE_P); }
    const double sc = ldexp(1.0, -s);
    __syncthreads();
    for (int idx = tid; idx < KK; idx += PT) b.A[idx] *= sc;
    __syncthreads();
    mm<PT>(K, b.A, b.A, b.A2);
    mm<PT>(K, b.A2, b.A2, b.A4);
    mm<PT>(K, b.A4, b.A2, b.A6);
    for (int idx = tid; idx < KK; idx += PT) b.T1[idx] = c[13] * b.A6[idx] + c[11] * b.A4[idx] + c[9] * b.A2[idx];
    __syncthreads();
    mm<PT>(K, b.A6, b.T1, b.T2);
    for (int idx = tid; idx < KK; idx += PT) {
        double d = (idx / K == idx % K) ? c[1] : 0.0;
        b.T2[idx] += c[7] * b.A6[idx] + c[5] * b.A4[idx] + c[3] * b.A2[idx] + d;
    }
    __syncthreads();
    mm<PT>(K, b.A, b.T2, b.T1);                                 // T1 = U
    for (int idx = tid; idx < KK; idx += PT) b.T2[idx] = c[12] * b.A6[idx] + c[10] * b.A4[idx] + c[8] * b.A2[idx];
    __syncthreads();
    mm<PT>(K, b.A6, b.T2, b.A);                                 // A = A6 * (...)
    for (int idx = tid; idx < KK; idx += PT) {
        double d = (idx / K == idx % K) ? c[0] : 0.0;
        double v = b.A[idx] + c[6] * b.A6[idx] + c[4] * b.A4[idx] + c[2] * b.A2[idx] + d;   // V
        double u = b.T1[idx];
        b.A2[idx] = v - u;                                  // left-hand side
        b.T1[idx] = v + u;                                  // right-hand side, becomes R
    }
    __syncthreads();
    // Gauss-Jordan with partial pivoting on [A2 | T1].  Thread (r0, j) owns column j of the augmented matrix for the rows
    // r0, r0 + nr, ...: no index arithmetic inside the sweep (the K = 24 case is bound by instruction issue and barriers).
    double* Lh = b.A2;
    double* Rh = b.T1;
    int* piv = reinterpret_cast<int*>(b.red + PT_MAX / 32);
    double* prow = b.col + K;                          // [2K] the scaled pivot row
    const int K2 = 2 * K, nr = PT / K2, r0 = tid / K2, j = tid - r0 * K2;
    const bool on = nr > 0 ? r0 < nr : tid < K2;       // (a CTA narrower than 2K columns is not launched: PT >= 256 >= 2K)
    double* const Mj = j < K ? Lh + j : Rh + (j - K);  // column j, row stride K
    for (int k = 0; k < K; k++) {
        if (tid < 32) {
            double best = -1.0; int bi = k;
            for (int i = k + tid; i < K; i += 32) { double v = fabs(Lh[i * K + k]); if (v > best) { best = v; bi = i; } }
            for (int o = 16; o > 0; o >>= 1) {
                double ob = __shfl_xor_sync(0xffffffffu, best, o);
                int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
            }
            if (tid == 0) {
                *piv = bi;
                if (!(best > 0.0)) atomicOr(status, EPX_ST_PADE_SINGULAR);
            }
        }
        __syncthreads();
        const int p = *piv;
        if (p != k) {                                  // (uniform)
            if (tid < K2) { const double t = Mj[k * K]; Mj[k * K] = Mj[p * K]; Mj[p * K] = t; }
            __syncthreads();
        }
        const double pinv = 1.0 / Lh[k * K + k];
        if (tid < K) b.col[tid] = (tid == k) ? 0.0 : Lh[tid * K + k];
        if (tid < K2) prow[tid] = Mj[k * K] * pinv;
        __syncthreads();
        if (on) {
            const double pk = prow[j];
            for (int i = r0; i < K; i += nr) Mj[i * K] = (i == k) ? pk : fma(-b.col[i], pk, Mj[i * K]);
        }
        __syncthreads();
    }
    double* R = b.T1;
    double* O = b.T2;
    for (int q = 0; q < s; q++) {
        mm<PT>(K, R, R, O);
        double* t = R; R = O; O = t;
    }
    return R;
}

// Componentwise-accurate alternative (reading A21 in DESIGN.md): exp(A) = e^{-mu} exp(A + mu I), mu = max_i |A_ii|.
// A + mu I is entrywise non-negative, its Taylor series (exp(tQ) = sum_j (tQ)^j / j!) has only
// non-negative terms, and squaring a non-negative matrix adds non-negative numbers: no cancellation anywhere, so
// every entry of the result -- including the ones that vanish like t^g for states g substitutions apart -- carries
// a relative error of a few hundred ulp.  Pade and the eigen path only bound the ABSOLUTE error (~1e-14), which a
// likelihood over short branches and distant tip states (codon data) amplifies without limit.
//   M = (A + mu I) / 2^s, ||M||_inf = mu / 2^s <= 1;  degree-16 Taylor by Paterson-Stockmeyer (powers M^2..M^4, three
//   Horner steps: 6 products);  R = e^{-mu/2^s} * poly(M) (stochastic);  R <- R^2 s times.
// In: b.A holds A.  Returns the buffer that holds exp(A).  All threads call.
template <int PT>
__device__ double* expm_shifted_taylor(int K, PadeBufs& b, int32_t* status)
{
    const double c[17] = {1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320,
                          1.0 / 362880, 1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0,
                          1.0 / 87178291200.0, 1.0 / 1307674368000.0, 1.0 / 20922789888000.0};
    const int tid = threadIdx.x, KK = K * K;
    double m = 0.0;
    for (int i = tid; i < K; i += PT) m = fmax(m, -b.A[i * K + i]);
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((tid & 31) == 0) b.red[tid >> 5] = m;
    __syncthreads();
    double mu = 0.0;
    for (int w = 0; w < PT / 32; w++) mu = fmax(mu, b.red[w]);
    int s = 0;
    if (mu > 1.0) s = (int)ceil(log2(mu));
    if (!(mu < 1e300)) { s = 0; if (tid == 0) atomicOr(status, EPX_ST_NONFINITE_P); }
    const double sc = ldexp(1.0, -s);
    __syncthreads();
    double* M1 = b.A; double* M2 = b.A2; double* M3 = b.A4; double* M4 = b.A6;
    for (int idx = tid; idx < KK; idx += PT) {
        double v = M1[idx];
        if (idx / K == idx % K) v = fmax(v + mu, 0.0);
        M1[idx] = v * sc;
    }
    __syncthreads();
    mm<PT>(K, M1, M1, M2);
    mm<PT>(K, M2, M1, M3);
    mm<PT>(K, M2, M2, M4);
    auto block = [&](int k, int idx) -> double {   // B_k = c[4k] I + c[4k+1] M + c[4k+2] M^2 + c[4k+3] M^3
        double d = (idx / K == idx % K) ? c[4 * k] : 0.0;
        return d + c[4 * k + 1] * M1[idx] + c[4 * k + 2] * M2[idx] + c[4 * k + 3] * M3[idx];
    };
    double* R = b.T1;
    double* O = b.T2;
    for (int idx = tid; idx < KK; idx += PT) R[idx] = block(3, idx) + c[16] * M4[idx];
    __syncthreads();
    for (int k = 2; k >= 0; k--) {
        mm<PT>(K, R, M4, O);
        for (int idx = tid; idx < KK; idx += PT) O[idx] += block(k, idx);
        __syncthreads();
        double* t = R; R = O; O = t;
    }
    const double damp = exp(-mu * sc);
    for (int idx = tid; idx < KK; idx += PT) R[idx] *= damp;
    __syncthreads();
    for (int q = 0; q < s; q++) {
        mm<PT>(K, R, R, O);
        double* t = R; R = O; O = t;
    }
    return R;
}

template <int METHOD, int PT>
__device__ __forceinline__ double* expm_dense(int K, PadeBufs& b, int32_t* status)
{
    return METHOD == 0 ? pade13<PT>(K, b, status) : expm_shifted_taylor<PT>(K, b, status);
}

__device__ __forceinline__ void carve(int K, double* sm, PadeBufs& b, double*& acc)
{
    const size_t KK = (size_t)K * K;
    b.A = sm; b.A2 = sm + KK; b.A4 = sm + 2 * KK; b.A6 = sm + 3 * KK; b.T1 = sm + 4 * KK; b.T2 = sm + 5 * KK;
    acc = sm + 6 * KK;
    b.col = sm + 7 * KK;          // [K] pivot column + [2K] scaled pivot row
    b.red = b.col + 3 * K;
}

template <int METHOD, int PT, int KT>
__global__ void __launch_bounds__(PT) pade_full_epoch_kernel(int K_rt, int M, int C, const double* __restrict__ Q,
    const double* __restrict__ tau, const double* __restrict__ rates, double* __restrict__ Efull,
    int32_t* __restrict__ status, const int32_t* __restrict__ fproc)
{
    extern __shared__ double sm[];
    const int K = KT ? KT : K_rt;          // KT > 0: compile-time state count (full tiles, unrolled products and sweeps)
    PadeBufs b; double* acc;
    carve(K, sm, b, acc);
    const int e = 1 + blockIdx.x / C, c = blockIdx.x % C;    // interior epochs 1 .. M-2
    if (fproc[e] != e) return;                               // f2: same process and duration as an earlier epoch
    const double scale = rates[c] * (tau[e] - tau[e - 1]);
    const double* Qe = Q + (size_t)e * K * K;
    for (int idx = threadIdx.x; idx < K * K; idx += PT) b.A[idx] = Qe[idx] * scale;
    __syncthreads();
    double* R = expm_dense<METHOD, PT>(K, b, status);
    for (int f = e; f <= M - 2; f++) {                       // every epoch that shares this entry
        if (fproc[f] != e) continue;
        double* out = Efull + ((size_t)f * C + c) * K * K;
        for (int idx = threadIdx.x; idx < K * K; idx += PT) out[idx] = R[idx];
    }
}

template <int METHOD, int PT, int KT>
__global__ void __launch_bounds__(PT) pade_chain_kernel(int K_rt, int C, int use_table, const int32_t* __restrict__ order,
    const int32_t* __restrict__ n_seg, const int32_t* __restrict__ seg_off, const int32_t* __restrict__ seg_epoch,
    const double* __restrict__ seg_dur, const double* __restrict__ rates, const double* __restrict__ Q,
    const double* __restrict__ Efull, double* __restrict__ P, int32_t* __restrict__ status)
{
    extern __shared__ double sm[];
    const int K = KT ? KT : K_rt;
    PadeBufs b; double* acc;
    carve(K, sm, b, acc);
    const int tid = threadIdx.x, KK = K * K;
    const int slot = order[blockIdx.x / C], c = blockIdx.x % C;
    double* out = P + ((size_t)slot * C + c) * KK;
    const int n = n_seg[slot];
    if (n == 0) {
        for (int idx = tid; idx < KK; idx += PT) out[idx] = (idx / K == idx % K) ? 1.0 : 0.0;
        return;
    }
    const int off = seg_off[slot];
    const double r = rates[c];
    double* cur = nullptr;           // running product (nullptr = identity so far)
    for (int s = 0; s < n; s++) {
        const int e = seg_epoch[off + s];
        double* E;
        if (use_table && s > 0 && s < n - 1) {    // the branch spans the whole of epoch e at rate r_c: table lookup
            const double* src = Efull + ((size_t)e * C + c) * KK;
            for (int idx = tid; idx < KK; idx += PT) b.T1[idx] = src[idx];
            __syncthreads();
            E = b.T1;
        } else {
            const double scale = r * seg_dur[off + s];
            const double* Qe = Q + (size_t)e * KK;
            for (int idx = tid; idx < KK; idx += PT) b.A[idx] = Qe[idx] * scale;
            __syncthreads();
            E = expm_dense<METHOD, PT>(K, b, status);
        }
        if (!cur) {
            for (int idx = tid; idx < KK; idx += PT) acc[idx] = E[idx];
            __syncthreads();
            cur = acc;
        } else {
            mm<PT>(K, cur, E, b.A);      // b.A is free once E is known; the old product buffer becomes the new b.A
            double* t = cur; cur = b.A; b.A = t;
        }
    }
    bool bad = false;
    for (int idx = tid; idx < KK; idx += PT) {
        double v = cur[idx];
        bad |= !isfinite(v);
        out[idx] = fmax(v, 0.0);
    }
    if (bad) atomicOr(status, EPX_ST_NONFINITE_P);
}

}  // namespace

size_t pade_smem_bytes(int K)
{
    return sizeof(double) * (7 * (size_t)K * K + 3 * K + PT_MAX / 32 + 2);
}

template <int METHOD, int PT, int KT>
static int pade_attr()
{
    if (cudaFuncSetAttribute(pade_full_epoch_kernel<METHOD, PT, KT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(pade_chain_kernel<METHOD, PT, KT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -1;
    return 0;
}

int pade_init_attributes()
{
    return pade_attr<0, 128, 0>() | pade_attr<0, 128, 24>() | pade_attr<0, 512, 0>() | pade_attr<1, 128, 0>() | pade_attr<1, 512, 0>() | pade_attr<1, 512, 61>();
}

template <int METHOD, int PT, int KT = 0>
static int launch_dense(const epx_ctx* c, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    const int K = c->K, C = c->C, M = c->M;
    const size_t smem = pade_smem_bytes(K);
    int launched = 0;
    const int use_table = c->has_brates ? 0 : 1;     // with branch rates an interior segment lasts r_v * (tau_e - tau_{e-1})
    const int n = c->sub_list ? c->sub_count : c->n_slots;          // f1: only the listed slots; the full-epoch table
    const int32_t* order = c->sub_list ? c->sub_list : d.order;      // depends on tau, Q and the rates only and is kept
    if (n == 0) return 0;
    if (M >= 3 && use_table && !c->sub_list) {
        pade_full_epoch_kernel<METHOD, PT, KT><<<(M - 2) * C, PT, smem, s>>>(K, M, C, d.Q, d.tau, d.rates, d.Efull, d.status, d.fproc);
        launched++;
    }
    pade_chain_kernel<METHOD, PT, KT><<<n * C, PT, smem, s>>>(K, C, use_table, order, d.n_seg, d.seg_off, d.seg_epoch, d.seg_dur,
                                                           d.rates, d.Q, d.Efull, d.P, d.status);
    launched++;
    return cudaGetLastError() == cudaSuccess ? launched : -1;
}

int launch_pade_chain(const epx_ctx* c, cudaStream_t s)
{
    if (c->K == 24) return launch_dense<0, 128, 24>(c, s);       // the trait-model size of config 4 at compile time
    return pade_threads(c->K) == 512 ? launch_dense<0, 512>(c, s) : launch_dense<0, 128>(c, s);
}
int launch_taylor_chain(const epx_ctx* c, cudaStream_t s)
{
    if (c->K == 61) return launch_dense<1, 512, 61>(c, s);       // the codon models of config 3 at compile time
    return pade_threads(c->K) == 512 ? launch_dense<1, 512>(c, s) : launch_dense<1, 128>(c, s);
}
