// a5 for 8 < K <= 64 (amino-acid and codon models): level-by-level Felsenstein pruning on the FP64 tensor pipe
// (Eq.(4): L_u(i) = [sum_j p_ij(v) L_v(j)] [sum_k p_ik(w) L_w(k)]; cost O(K^2 N C L), L72).
//
// Per (node, category) an internal child contributes F[pattern][i] = sum_j V[pattern][j] P[i][j]: an L x KP x KP product with
// the SAME KP x KP matrix for all L patterns (KP = K rounded up to 8).  One CTA = (node, category, chunk of patterns):
//   * the child's matrix is staged ONCE per CTA by a TMA bulk copy (cp.async.bulk + mbarrier) from a copy that
//     pb_swizzle_kernel keeps in mma.m8n8k4 B-fragment order (PB), so the inner loop reads it with conflict-free 64-bit
//     shared-memory loads -- round 1's kernel staged 61 x 61 doubles with strided 8-byte loads per 32 patterns and spent its
//     time there (profiles/r1_other_configs_ncu.md: DMMA pipe 21-27 % busy);
//   * a warp owns 8 patterns; lane (g, q) = pattern g and S = KP / 4 of its states, VW (4, or 2 if S is odd-ish) at a time:
//     element e of lane q is state st(q, e) = (e / VW) 4 VW + q VW + e % VW, so the 4 lanes of a pattern read / write 4 VW
//     CONTIGUOUS doubles per instruction (a full 128-byte line with 256-bit accesses).  The contraction index of k-step kt
//     at position q is state st(q, kt) and column 2 q + h of n-tile nt is state st(q, 2 nt + h): a lane's A operand (child
//     vector) AND its D fragment (result) are the same S elements, so vectors go from global memory to the tensor pipe and
//     back with no shared-memory round trip.  (A first version gave a lane S contiguous states: every 128-bit load of a
//     warp then touched 32 different lines and the kernel was bound by L1 tag lookups, l1tex 85 % busy.)
//   * tip children are gathers P[i][state] from the row-major matrix (no product, no staging).
// Rescaling (reading A12) is per (node, CATEGORY, pattern) here -- a category is a CTA of its own, and a power-of-two factor
// per category is as exact as one per pattern; the root reduction and epx_get_partials fold the C exponents together.
// Partials layout of these contexts: [node][C][L][KP] (padding states are 0), scale_exp[node][C][L].
#include "prune_common.cuh"

using namespace epxdev;

namespace {

constexpr int MMA_T = 256;        // 8 warps x 8 patterns = 64 patterns per pass over the chunk

template <int KP>
struct Frag {
    static constexpr int S = KP / 4, NT = KP / 8, KT = KP / 4, MAT = KP * KP;
    static constexpr int VW = (S % 4 == 0) ? 4 : 2;          // doubles per vector access
    static constexpr int NC = S / VW;                        // vector accesses per lane and state vector
    __host__ __device__ static constexpr int st(int q, int e) { return (e / VW) * 4 * VW + q * VW + e % VW; }
};

// Internal nodes' slots: PB[slot][c][(kt * NT + nt) * 32 + 4 g + q] = P[i][j],  j = st(q, kt) (contraction),
//                                                                    i = st(g >> 1, 2 nt + (g & 1))   (B-fragment order)
template <int KP>
__global__ void __launch_bounds__(256) pb_swizzle_kernel(int K, int C, int n_tips, const uint8_t* __restrict__ tip_vec,
                                                         const int32_t* __restrict__ list, const double* __restrict__ P,
                                                         double* __restrict__ PB)
{
    using F = Frag<KP>;
    constexpr int NT = F::NT;
    const int slot = list ? list[blockIdx.x / C] : blockIdx.x / C, c = blockIdx.x % C;
    const double* src = P + ((size_t)slot * C + c) * K * K;
    double* dst = PB + ((size_t)slot * C + c) * KP * KP;
    if (slot < n_tips && !tip_vec[slot]) {           // (a tip with a partial vector is multiplied like an internal child)
        __shared__ double tile[32][33];
        for (int s0 = 0; s0 < KP; s0 += 32)
            for (int i0 = 0; i0 < KP; i0 += 32) {
                const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
                for (int r = ty; r < 32; r += 8) {      // read P[i0 + r][s0 + tx] (coalesced along s)
                    const int i = i0 + r, sidx = s0 + tx;
                    tile[r][tx] = (i < K && sidx < K) ? src[i * K + sidx] : 0.0;
                }
                __syncthreads();
                for (int r = ty; r < 32; r += 8) {      // write PT[s0 + r][i0 + tx] (coalesced along i)
                    const int sidx = s0 + r, i = i0 + tx;
                    if (sidx < KP && i < KP) dst[sidx * KP + i] = tile[tx][r];
                }
                __syncthreads();
            }
        return;
    }
    for (int idx = threadIdx.x; idx < KP * KP; idx += 256) {
        const int lane = idx & 31, t = idx >> 5, nt = t % NT, kt = t / NT;
        const int g = lane >> 2, q = lane & 3;
        const int j = F::st(q, kt), i = F::st(g >> 1, 2 * nt + (g & 1));
        dst[idx] = (i < K && j < K) ? src[i * K + j] : 0.0;
    }
}

template <int KP>
__global__ void __launch_bounds__(MMA_T, KP > 48 ? 2 : 3) prune_mma_kernel(const PruneOp* __restrict__ ops, int chunks, int chunk_p, int K, int C,
    int L, int Lp, const double* __restrict__ PB, const uint8_t* __restrict__ tips,
    double* __restrict__ partials, int32_t* __restrict__ scale_exp)
{
    using F = Frag<KP>;
    constexpr int S = F::S, NT = F::NT, KT = F::KT, MAT = F::MAT, VW = F::VW, NC = F::NC;
    extern __shared__ __align__(128) unsigned char smraw[];
    double* Bs = reinterpret_cast<double*>(smraw);                      // [2][KP * KP] fragment-ordered child matrices
    uint64_t* bar = reinterpret_cast<uint64_t*>(Bs + 2 * MAT);          // [2]
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, q = lane & 3;
    const int chunk = blockIdx.x % chunks, unit = blockIdx.x / chunks;
    const int c = unit % C;
    const PruneOp op = ops[unit / C];
    const int p_begin = chunk * chunk_p, p_end = min(L, p_begin + chunk_p);

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
        for (int ch = 0; ch < 2; ch++)
            if (!op.child_is_tip[ch]) {
                mbar_expect_tx(&bar[ch], MAT * 8);
                bulk_g2s(Bs + ch * MAT, PB + ((size_t)op.child[ch] * C + c) * MAT, MAT * 8, &bar[ch]);
            }
    }
    __syncthreads();                                                    // the barriers are initialised
    // Programmatic dependent launch: a level's CTAs become resident, initialise their barriers and stage their matrices (PB
    // is complete before the first level starts) while the level below is still running, and wait HERE for its partials.
    // The trigger comes after the wait, so by induction every earlier level is complete when a CTA passes this point.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const size_t LK = (size_t)L * KP;
    for (int p8 = p_begin + 8 * w; p8 < p_end; p8 += 8 * (MMA_T / 32)) {
        const int p = p8 + g;
        const bool live = p < p_end;
        // both children's operands are requested before the first product starts: an internal child's vector (S contiguous
        // states of pattern g), or for a tip child the column its state selects = a row of the transposed copy
        double a[2][S];
        int ex = 0, tip_s[2] = {0, 0};
#pragma unroll
        for (int ch = 0; ch < 2; ch++) {
            const double* v;
            if (op.child_is_tip[ch]) {
                const int s = live ? tips[(size_t)op.child[ch] * Lp + p] : 255;
                tip_s[ch] = s;
                v = PB + ((size_t)op.child[ch] * C + c) * MAT + (size_t)min(s, K - 1) * KP + q * VW;
            } else {
                v = partials + ((size_t)op.cpidx[ch] * C + c) * LK + (size_t)(live ? p : p_begin) * KP + q * VW;
                if (live) ex += scale_exp[((size_t)op.cpidx[ch] * C + c) * L + p];
            }
#pragma unroll
            for (int m = 0; m < NC; m++) {
                if (VW == 4) {
                    const double4a r = ld256(v + m * 16);
                    a[ch][4 * m] = r.x; a[ch][4 * m + 1] = r.y; a[ch][4 * m + 2] = r.z; a[ch][4 * m + 3] = r.w;
                } else {
                    const double2 r = *reinterpret_cast<const double2*>(v + m * 8);
                    a[ch][2 * m] = r.x; a[ch][2 * m + 1] = r.y;
                }
            }
        }
        double f[S];
#pragma unroll
        for (int ch = 0; ch < 2; ch++) {
            if (op.child_is_tip[ch]) {
#pragma unroll
                for (int k = 0; k < S; k++) {
                    const double t = tip_s[ch] < K ? a[ch][k] : (F::st(q, k) < K ? 1.0 : 0.0);     // missing state: all ones
                    f[k] = ch ? f[k] * t : t;
                }
            } else {
                double acc[NT][2];
#pragma unroll
                for (int nt = 0; nt < NT; nt++) acc[nt][0] = acc[nt][1] = 0.0;
                mbar_wait(&bar[ch], 0);
                const double* Bc = Bs + ch * MAT + lane;
#pragma unroll
                for (int kt = 0; kt < KT; kt++)
#pragma unroll
                    for (int nt = 0; nt < NT; nt++) dmma884(acc[nt][0], acc[nt][1], a[ch][kt], Bc[(kt * NT + nt) * 32]);
#pragma unroll
                for (int nt = 0; nt < NT; nt++) {
                    f[2 * nt] = ch ? f[2 * nt] * acc[nt][0] : acc[nt][0];
                    f[2 * nt + 1] = ch ? f[2 * nt + 1] * acc[nt][1] : acc[nt][1];
                }
            }
        }
        // all values are >= 0: the largest has the largest high word; 4 lanes hold a pattern's K states
        int hmax = 0;
#pragma unroll
        for (int k = 0; k < S; k++) hmax = max(hmax, __double2hiint(f[k]));
        hmax = max(hmax, __shfl_xor_sync(0xffffffffu, hmax, 1));
        hmax = max(hmax, __shfl_xor_sync(0xffffffffu, hmax, 2));
        double sc = 1.0;
        {
            const int e = (hmax >> 20) - 1023;
            if (e > -1000 && hmax < 0x7fe00000) { sc = pow2_neg(e); ex += e; }
        }
        if (live) {
            double* dst = partials + ((size_t)op.pidx * C + c) * LK + (size_t)p * KP + q * VW;
#pragma unroll
            for (int m = 0; m < NC; m++) {
                if (VW == 4) st256(dst + m * 16, f[4 * m] * sc, f[4 * m + 1] * sc, f[4 * m + 2] * sc, f[4 * m + 3] * sc);
                else *reinterpret_cast<double2*>(dst + m * 8) = make_double2(f[2 * m] * sc, f[2 * m + 1] * sc);
            }
            if (q == 0) scale_exp[((size_t)op.pidx * C + c) * L + p] = ex;
        }
    }
}

template <int KP>
size_t mma_smem() { return (size_t)2 * KP * KP * 8 + 16; }

template <int KP>
int mma_attr()
{
    return cudaFuncSetAttribute(prune_mma_kernel<KP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mma_smem<KP>()) == cudaSuccess ? 0 : -1;
}

template <int KP>
void mma_launch(const epx_ctx* c, const PruneOp* ops, int nops, cudaStream_t s, bool pdl)
{
    const DevBuffers& d = c->d;
    const int chunk_p = prune_mma_chunk(c, nops), chunks = (c->L + chunk_p - 1) / chunk_p;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(nops * c->C * chunks));
    cfg.blockDim = dim3(MMA_T);
    cfg.dynamicSmemBytes = mma_smem<KP>();
    cfg.stream = s;
    cudaLaunchAttribute attr{};
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &attr; cfg.numAttrs = pdl ? 1 : 0;          // (the level below is an mma level too: it triggers early)
    cudaLaunchKernelEx(&cfg, prune_mma_kernel<KP>, ops, chunks, chunk_p, c->K, c->C, c->L, c->Lp, (const double*)d.PB,
                       (const uint8_t*)d.tips, d.partials, d.scale_exp);
}

template <int KP>
void swz_launch(const epx_ctx* c, cudaStream_t s)
{
    const int n = c->sub_list ? c->sub_count : c->n_slots;
    if (n > 0) pb_swizzle_kernel<KP><<<n * c->C, 256, 0, s>>>(c->K, c->C, c->N, c->d.tip_vec, c->sub_list, c->d.P, c->d.PB);
}

}  // namespace

// Site patterns per CTA for a level of `nops` operations: 64 (one 8-pattern tile per warp) unless the level then has more
// than ~4 waves of CTAs, where a CTA loops over 128 or 256 patterns with its staged matrices.
int prune_mma_chunk(const epx_ctx* c, int nops)
{
    if (c->mma_chunk > 0) return (c->mma_chunk + 7) & ~7;
    const long ctas64 = (long)nops * c->C * ((c->L + 63) / 64);
    return ctas64 > 8 * 296 ? 256 : ctas64 > 4 * 296 ? 128 : 64;
}

int prune_mma_init_attributes()
{
    return mma_attr<16>() | mma_attr<24>() | mma_attr<32>() | mma_attr<40>() | mma_attr<48>() | mma_attr<56>() | mma_attr<64>();
}

// One post-order level: `nops` operations whose children are complete.
void launch_prune_mma_level(const epx_ctx* c, const PruneOp* ops, int nops, cudaStream_t s, bool pdl)
{
    switch (prune_kp(c)) {
        case 16: mma_launch<16>(c, ops, nops, s, pdl); break;
        case 24: mma_launch<24>(c, ops, nops, s, pdl); break;
        case 32: mma_launch<32>(c, ops, nops, s, pdl); break;
        case 40: mma_launch<40>(c, ops, nops, s, pdl); break;
        case 48: mma_launch<48>(c, ops, nops, s, pdl); break;
        case 56: mma_launch<56>(c, ops, nops, s, pdl); break;
        default: mma_launch<64>(c, ops, nops, s, pdl); break;
    }
}

// Fragment-ordered copies of the branch matrices (all slots, or the slots of c->sub_list for an incremental call).
void launch_pb_swizzle(const epx_ctx* c, cudaStream_t s)
{
    switch (prune_kp(c)) {
        case 16: swz_launch<16>(c, s); break;
        case 24: swz_launch<24>(c, s); break;
        case 32: swz_launch<32>(c, s); break;
        case 40: swz_launch<40>(c, s); break;
        case 48: swz_launch<48>(c, s); break;
        case 56: swz_launch<56>(c, s); break;
        default: swz_launch<64>(c, s); break;
    }
}
