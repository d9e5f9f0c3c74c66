// a5, K == 4 (default): depth-first Felsenstein pruning, one LANE per site pattern
// (Eq.(4): L_u(i) = [sum_j p_ij(v) L_v(j)] [sum_k p_ik(w) L_w(k)], post-order; L72: patterns are independent).
//
// Why another walk kernel: prune4_dfs_kernel (prune.cu) puts a (pattern, category) on a lane, so the 4 categories of a warp
// read 4 different 4x4 matrices and every LDS.128 of a matrix costs 4 shared-memory wavefronts; ncu showed that kernel bound
// by the SM's L1 / shared-memory data pipe (88 % busy), not by HBM (profiles/r1_prune4_dfs_ncu.md).  Here a lane owns a whole
// pattern -- all C categories in registers -- so
//   * every matrix entry is read at ONE address by the whole warp (a broadcast: one wavefront per LDS.128, 32 patterns served),
//   * the per-(node, pattern) maximum over (category, state) of the rescaling (reading A12) needs no shuffle at all,
//   * the partials go to HBM in the generic layout [node][C][L][4]: per category a warp stores 32 consecutive 32-byte state
//     vectors = 1 KB contiguous per st.global.v4.f64.
// The walk itself is the host-planned one of build_plan(): pieces of the tree (independent subtrees, then the top piece),
// a child's vector handed over in registers or parked in a per-warp shared-memory stack, so partials are written once and
// never read back.  Inputs are fetched ahead of the dependency chain: operation descriptors 32 at a time into registers
// (one per lane, read by shuffle); the two children's matrices (2 x C x 128 B) and, for tip children, the warp's 32 x PPL tip
// states with cp.async into a ring LN_STAGES - 1 operations ahead.  HB = true (top piece, incremental re-evaluation: most
// operands are partials written by another launch) also streams those operands and their exponents through the ring.
#include "prune_common.cuh"

using namespace epxdev;

namespace {

constexpr int LN_STAGES = 4;

__host__ __device__ constexpr int ln_stage_bytes(int C, int PPL, bool HB)
{
    return 2 * C * 128 + 2 * 32 * PPL + (HB ? 2 * PPL * (C * 1024 + 128) : 0);
}
size_t ln_smem(int C, int PPL, bool HB, int depth)
{
    return (size_t)LN_STAGES * ln_stage_bytes(C, PPL, HB) + (size_t)depth * PPL * (C * 1024 + 128);
}

// a6 inside the walk: the warps of the piece that ends at the root also reduce their patterns (PAPER.md L72:
// l_p = sum_c w_c sum_i pi_i L_root(i), logL = sum_p wt_p ln l_p) -- the root's vectors are still in registers, and the
// separate root kernel (9 us + a launch gap, a fifth of config 1's step) disappears.  site_lnl == nullptr: not fused.
struct LaneRoot {
    const double *freqs, *root_freqs, *weights, *pattern_wt, *tau, *height;
    double *site_lnl, *block_sums, *lnl;
    int32_t* status;         // [0] status word, [1] arrival counter
    int root_node, M;
};

template <int C, int PPL, bool HB>
__global__ void __launch_bounds__(32) prune4_lane_kernel(const DfsOp* __restrict__ ops, const DfsPiece* __restrict__ pieces,
    int tiles, int L, int Lp, int depth, const double* __restrict__ P, const uint8_t* __restrict__ tips,
    double* __restrict__ partials, int32_t* __restrict__ scale_exp, const LaneRoot root)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    constexpr int PW = 32 * PPL;                    // patterns per warp
    constexpr int MB = 2 * C * 128;                 // ring stage: both children's matrices [2][C][16] f64 ...
    constexpr int TB = 2 * PW;                      // ... tip states of the warp's patterns [2][PW] u8 ...
    constexpr int VB = HB ? 2 * PPL * C * 1024 : 0; // ... HBM operands [2][PPL][C][2 halves][32 lanes] double2 ...
    constexpr int SB = ln_stage_bytes(C, PPL, HB);  // ... and their exponents [2][PPL][32] i32
    constexpr int NCH = (16 * C + 31) / 32;         // 16-byte chunks of the two matrices per lane
    constexpr unsigned FULL = 0xffffffffu;
    double2* stack = reinterpret_cast<double2*>(smraw + LN_STAGES * SB);                    // [depth][PPL][C][2][32]
    int* stack_ex = reinterpret_cast<int*>(stack + (size_t)depth * PPL * C * 64);           // [depth][PPL][32]
    const int lane = threadIdx.x;
    const int piece = blockIdx.x / tiles, tile = blockIdx.x - piece * tiles;
    const int p0 = tile * PW;
    const DfsPiece pc = pieces[piece];
    const int n_ops = pc.end - pc.begin;
    ops += pc.begin;
    // a6 (fused): the root's frequency vector is located and the pattern weights are requested NOW, so that the walk hides the
    // chain of dependent loads (boundary search) that would otherwise sit at the tail of the kernel
    const bool do_root = root.site_lnl != nullptr && piece == (int)(gridDim.x / tiles) - 1;
    const double* rf = nullptr;
    if (do_root) {
        rf = root.root_freqs;
        if (!rf) {                                       // reading A9: the epoch that holds the root, #{k : tau_k < h_root}
            const double h = root.height[root.root_node];
            int lo = 0, hi = root.M - 1;
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (root.tau[mid] < h) lo = mid + 1; else hi = mid; }
            rf = root.freqs + (size_t)lo * 4;
        }
        asm volatile("prefetch.global.L1 [%0];" ::"l"(rf));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(root.weights));
        if (p0 + lane < L) asm volatile("prefetch.global.L1 [%0];" ::"l"(root.pattern_wt + p0 + lane));
    }

    // 32-bit indexing in units of one state vector (32 B): (N-1 + tip blocks) C L < 2^32 is checked by prune_uses_dfs
    const unsigned uL = (unsigned)L, node_stride = uL * C;
    bool live[PPL];
    unsigned pat[PPL];
#pragma unroll
    for (int u = 0; u < PPL; u++) { pat[u] = (unsigned)(p0 + u * 32 + lane); live[u] = pat[u] < uL; }
    double4a* const vec = reinterpret_cast<double4a*>(partials);
    const unsigned char* const tip_base = tips + p0;

    struct Block { int4 d; int2 h; };
    auto load_block = [&](int base) -> Block {      // lane j: descriptor base + j
        Block b;
        b.d = make_int4(0, 0, 0, 0);
        b.h = make_int2(0, 0);
        const int k = base + lane;
        if (k < n_ops) {
            const int4* src = reinterpret_cast<const int4*>(ops + k);
            b.d = __ldg(src);
            const int4 h = __ldg(src + 1);
            b.h = make_int2(h.x, h.y);
        }
        return b;
    };
    Block cb = load_block(0), nb = load_block(32);

    // stage everything operation j (in the current or the next block of 32) reads from global memory into ring buffer `buf`
    auto issue = [&](int j, int k, int buf) {
        const bool in_cur = (j >> 5) == (k >> 5);
        const int na = __shfl_sync(FULL, in_cur ? cb.d.x : nb.d.x, j & 31);
        const int nbn = __shfl_sync(FULL, in_cur ? cb.d.y : nb.d.y, j & 31);
        const int code = __shfl_sync(FULL, in_cur ? cb.d.w : nb.d.w, j & 31);
        const int srcA = (code & 0xff) - 3, srcB = ((code >> 8) & 0xff) - 3;
        unsigned char* sb = smraw + buf * SB;
#pragma unroll
        for (int q = 0; q < NCH; q++) {
            const int ch = lane + 32 * q;
            if (ch < 16 * C) {
                const bool second = ch >= 8 * C;
                cp_async16(sb + ch * 16, P + (size_t)(second ? nbn : na) * (C * 16) + (ch - (second ? 8 * C : 0)) * 2);
            }
        }
        if (lane < 4 * PPL) {                       // tip states: 16 patterns per copy
            const bool second = lane >= 2 * PPL;
            const int w = lane - (second ? 2 * PPL : 0);
            if ((second ? srcB : srcA) == EPX_DFS_TIP && p0 + 16 * w < Lp)
                cp_async16(sb + MB + (second ? PW : 0) + 16 * w, tip_base + (size_t)(second ? nbn : na) * Lp + 16 * w);
        }
        if (HB) {
            const int pa = __shfl_sync(FULL, in_cur ? cb.h.x : nb.h.x, j & 31);
            const int pb = __shfl_sync(FULL, in_cur ? cb.h.y : nb.h.y, j & 31);
#pragma unroll
            for (int h = 0; h < 2; h++) {
                if ((h ? srcB : srcA) != EPX_DFS_HBM || (code & (h ? EPX_DFS_LATE_B : EPX_DFS_LATE_A))) continue;
                const unsigned node = (unsigned)(h ? pb : pa);
#pragma unroll
                for (int u = 0; u < PPL; u++) {
                    if (!live[u]) continue;
                    unsigned char* dst = sb + MB + TB + ((h * PPL + u) * C) * 1024 + lane * 16;
#pragma unroll
                    for (int c = 0; c < C; c++) {
                        const double* src = reinterpret_cast<const double*>(vec + (node * node_stride + c * uL + pat[u]));
                        cp_async16(dst + c * 1024, src);
                        cp_async16(dst + c * 1024 + 512, src + 2);
                    }
                    cp_async4(sb + MB + TB + VB + ((h * PPL + u) * 32 + lane) * 4, scale_exp + (size_t)node * uL + pat[u]);
                }
            }
        }
    };
#pragma unroll
    for (int j = 0; j < LN_STAGES - 1; j++) {
        if (j < n_ops) issue(j, 0, j);
        cp_async_commit();
    }

    double cur[PPL][C][4];                          // result of the previous operation (hand-over to its parent)
    int cur_ex[PPL];
#pragma unroll
    for (int u = 0; u < PPL; u++) {
        cur_ex[u] = 0;
#pragma unroll
        for (int c = 0; c < C; c++) cur[u][c][0] = cur[u][c][1] = cur[u][c][2] = cur[u][c][3] = 1.0;
    }
    int buf = 0;
    for (int k = 0; k < n_ops; k++) {
        if ((k & 31) == 0 && k > 0) { cb = nb; nb = load_block(k + 32); }
        __syncwarp();                               // every lane is done reading the buffer the next stage overwrites
        {
            int nbuf = buf + LN_STAGES - 1; if (nbuf >= LN_STAGES) nbuf -= LN_STAGES;
            if (k + LN_STAGES - 1 < n_ops) issue(k + LN_STAGES - 1, k, nbuf);
            cp_async_commit();
        }
        const int src_lane = k & 31;
        const unsigned pidx = (unsigned)__shfl_sync(FULL, cb.d.z, src_lane);
        const int code = __shfl_sync(FULL, cb.d.w, src_lane);
        const int srcA = (code & 0xff) - 3, srcB = ((code >> 8) & 0xff) - 3, out_slot = ((code >> 16) & 0xff) - 1;
        unsigned pa = 0, pb = 0;
        if (srcA == EPX_DFS_HBM) pa = (unsigned)__shfl_sync(FULL, cb.h.x, src_lane);
        if (srcB == EPX_DFS_HBM) pb = (unsigned)__shfl_sync(FULL, cb.h.y, src_lane);

        cp_async_wait<LN_STAGES - 1>();             // this lane's copies for operation k have landed ...
        __syncwarp();                               // ... and so have every other lane's
        const unsigned char* sb = smraw + buf * SB;
        const double* Pa = reinterpret_cast<const double*>(sb);
        const double* Pb = Pa + C * 16;

        double f[PPL][C][4];
        int ex[PPL];
#pragma unroll
        for (int u = 0; u < PPL; u++) ex[u] = 0;
        // one child's contribution: f = (first ? 1 : f) * (P v) -- the same expression tree as prune4_dfs_kernel, bit for bit
        auto child = [&](const int src, const double* __restrict__ Pm, const int h, const unsigned hp, const bool first) {
            const bool ring = HB && !(code & (h ? EPX_DFS_LATE_B : EPX_DFS_LATE_A));      // HBM operand prefetched into the ring
            if (src == EPX_DFS_TIP) {
#pragma unroll
                for (int u = 0; u < PPL; u++) {
                    const int s = sb[MB + h * PW + u * 32 + lane];
#pragma unroll
                    for (int c = 0; c < C; c++)
#pragma unroll
                        for (int i = 0; i < 4; i++) {
                            const double t = (s < 4) ? Pm[c * 16 + i * 4 + s] : 1.0;
                            f[u][c][i] = first ? t : f[u][c][i] * t;
                        }
                }
                return;
            }
#pragma unroll
            for (int u = 0; u < PPL; u++) {
                if (src == EPX_DFS_PREV) ex[u] += cur_ex[u];
                else if (src == EPX_DFS_HBM) {
                    if (ring) ex[u] += *reinterpret_cast<const int*>(sb + MB + TB + VB + ((h * PPL + u) * 32 + lane) * 4);
                    else if (live[u]) ex[u] += scale_exp[(size_t)hp * uL + pat[u]];
                } else ex[u] += stack_ex[(src * PPL + u) * 32 + lane];
            }
#pragma unroll
            for (int c = 0; c < C; c++) {
                double m[16];                       // broadcast reads: the whole warp reads the same 16-byte word
#pragma unroll
                for (int i = 0; i < 8; i++) { const double2 r = *reinterpret_cast<const double2*>(Pm + c * 16 + 2 * i); m[2 * i] = r.x; m[2 * i + 1] = r.y; }
#pragma unroll
                for (int u = 0; u < PPL; u++) {
                    double v[4];
                    if (src == EPX_DFS_PREV) {
#pragma unroll
                        for (int i = 0; i < 4; i++) v[i] = cur[u][c][i];
                    } else if (src == EPX_DFS_HBM) {
                        if (ring) {
                            const double2* r = reinterpret_cast<const double2*>(sb + MB + TB + ((h * PPL + u) * C + c) * 1024) + lane;
                            const double2 v01 = r[0], v23 = r[32];
                            v[0] = v01.x; v[1] = v01.y; v[2] = v23.x; v[3] = v23.y;
                        } else {
                            v[0] = v[1] = v[2] = v[3] = 1.0;
                            if (live[u]) {
                                const double4a t = ld256(reinterpret_cast<const double*>(vec + (hp * node_stride + c * uL + pat[u])));
                                v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
                            }
                        }
                    } else {
                        const double2* r = stack + ((src * PPL + u) * C + c) * 64 + lane;
                        const double2 v01 = r[0], v23 = r[32];
                        v[0] = v01.x; v[1] = v01.y; v[2] = v23.x; v[3] = v23.y;
                    }
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        const double t = fma(m[i * 4 + 3], v[3], fma(m[i * 4 + 2], v[2], fma(m[i * 4 + 1], v[1], m[i * 4] * v[0])));
                        f[u][c][i] = first ? t : f[u][c][i] * t;
                    }
                }
            }
        };
        child(srcA, Pa, 0, pa, true);
        child(srcB, Pb, 1, pb, false);

#pragma unroll
        for (int u = 0; u < PPL; u++) {
            // all values are >= 0, so the largest one has the largest high word: an integer max finds its exponent
            int hmax = 0;
#pragma unroll
            for (int c = 0; c < C; c++)
#pragma unroll
                for (int i = 0; i < 4; i++) hmax = max(hmax, __double2hiint(f[u][c][i]));
            double sc = 1.0;
            {
                const int e = (hmax >> 20) - 1023;      // hmax < 0x7fe00000: finite and far from overflow
                if (e > -1000 && hmax < 0x7fe00000) { sc = pow2_neg(e); ex[u] += e; }
            }
            cur_ex[u] = ex[u];
#pragma unroll
            for (int c = 0; c < C; c++) {
#pragma unroll
                for (int i = 0; i < 4; i++) cur[u][c][i] = f[u][c][i] * sc;
                if (live[u])
                    st256(reinterpret_cast<double*>(vec + (pidx * node_stride + c * uL + pat[u])), cur[u][c][0], cur[u][c][1],
                          cur[u][c][2], cur[u][c][3]);
                if (out_slot >= 0) {
                    double2* w = stack + ((out_slot * PPL + u) * C + c) * 64 + lane;
                    w[0] = make_double2(cur[u][c][0], cur[u][c][1]);
                    w[32] = make_double2(cur[u][c][2], cur[u][c][3]);
                }
            }
            if (live[u]) scale_exp[(size_t)pidx * uL + pat[u]] = ex[u];
            if (out_slot >= 0) stack_ex[(out_slot * PPL + u) * 32 + lane] = ex[u];
        }
        if (++buf == LN_STAGES) buf = 0;
    }
    if (!do_root) return;
    // ---- a6 for this warp's patterns: `cur` is the root's (rescaled) vector set, cur_ex its exponent.  The expressions per
    // pattern are those of root_site_kernel (same site log-likelihoods bit for bit); the weighted sum is taken per warp, then
    // over the warps in index order by whichever warp arrives last.
    double contrib = 0.0;
#pragma unroll
    for (int u = 0; u < PPL; u++) {
        if (!live[u]) continue;
        double site = 0.0;
#pragma unroll
        for (int c = 0; c < C; c++) {
            double sacc = 0.0;
#pragma unroll
            for (int i = 0; i < 4; i++) sacc = fma(rf[i], cur[u][c][i], sacc);
            site = fma(root.weights[c], sacc, site);
        }
        if (!(site > 0.0) || !(site < 1.7e308)) atomicOr(root.status, EPX_ST_BAD_SITE);
        const double ln = log(site) + (double)cur_ex[u] * 0.6931471805599453094;
        root.site_lnl[pat[u]] = ln;
        contrib += root.pattern_wt[pat[u]] * ln;
    }
    for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(FULL, contrib, o);
    int last = 0;
    if (lane == 0) {
        root.block_sums[tile] = contrib;
        __threadfence();
        last = atomicAdd(root.status + 1, 1) == tiles - 1;
    }
    last = __shfl_sync(FULL, last, 0);
    if (!last) return;
    __threadfence();
    double t = 0.0;
    for (int i0 = 0; i0 < tiles; i0 += 128) {            // four loads in flight per lane; the order of the sum is fixed by the indices
        double v[4];
#pragma unroll
        for (int q = 0; q < 4; q++) { const int i = i0 + 32 * q + lane; v[q] = i < tiles ? __ldcg(root.block_sums + i) : 0.0; }
#pragma unroll
        for (int q = 0; q < 4; q++) t += v[q];
    }
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(FULL, t, o);
    if (lane == 0) { *root.lnl = t; root.status[1] = 0; }
}

template <int C, int PPL, bool HB>
int ln_attr()
{
    return cudaFuncSetAttribute(prune4_lane_kernel<C, PPL, HB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) ==
           cudaSuccess ? 0 : -1;
}
template <int C>
int ln_attr_c() { return ln_attr<C, 1, false>() | ln_attr<C, 2, false>() | ln_attr<C, 1, true>(); }

template <int C, int PPL, bool HB>
void ln_launch(const epx_ctx* c, const DfsOp* ops, const DfsPiece* pieces, int n_pieces, cudaStream_t s, bool with_root)
{
    const DevBuffers& d = c->d;
    const int tiles = (c->L + 32 * PPL - 1) / (32 * PPL);
    LaneRoot root{};
    if (with_root) {
        root.freqs = d.freqs; root.root_freqs = c->has_root_freqs ? d.root_freqs : nullptr; root.weights = d.weights;
        root.pattern_wt = d.pattern_wt; root.tau = d.tau; root.height = d.height; root.site_lnl = d.site_lnl;
        root.block_sums = d.block_sums; root.lnl = d.lnl; root.status = d.status; root.root_node = c->root; root.M = c->M;
    }
    prune4_lane_kernel<C, PPL, HB><<<n_pieces * tiles, 32, ln_smem(C, PPL, HB, c->dfs_depth), s>>>(ops, pieces, tiles, c->L, c->Lp,
        c->dfs_depth, d.P, d.tips, d.partials, d.scale_exp, root);
}

template <int C>
void ln_launch_c(const epx_ctx* c, const DfsOp* ops, const DfsPiece* pieces, int n_pieces, cudaStream_t s, bool hbm_operands, bool with_root)
{
    if (hbm_operands) { ln_launch<C, 1, true>(c, ops, pieces, n_pieces, s, with_root); return; }
    if (lane_patterns_per_lane(c) == 2) ln_launch<C, 2, false>(c, ops, pieces, n_pieces, s, with_root);
    else ln_launch<C, 1, false>(c, ops, pieces, n_pieces, s, with_root);
}

}  // namespace

int lane_patterns_per_lane(const epx_ctx* c)
{
    if (c->dfs_ppl == 1 || c->dfs_ppl == 2) return c->dfs_ppl;
    return 1;
}

size_t lane_smem_bytes(const epx_ctx* c, int depth)
{
    return std::max(ln_smem(c->C, lane_patterns_per_lane(c), false, depth), ln_smem(c->C, 1, true, depth));
}

int prune_lane_init_attributes()
{
    return ln_attr_c<1>() | ln_attr_c<2>() | ln_attr_c<3>() | ln_attr_c<4>() | ln_attr_c<5>() | ln_attr_c<6>() | ln_attr_c<7>() |
           ln_attr_c<8>();
}

// `hbm_operands`: the piece reads most of its operands from partials written by an earlier launch (top piece, incremental
// re-evaluation): one pattern per lane, operands streamed through the staging ring.
void launch_prune4_lane(const epx_ctx* c, const DfsOp* ops, const DfsPiece* pieces, int n_pieces, cudaStream_t s, bool hbm_operands,
                        bool with_root)
{
    switch (c->C) {
        case 1: ln_launch_c<1>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
        case 2: ln_launch_c<2>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
        case 3: ln_launch_c<3>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
        case 4: ln_launch_c<4>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
        case 5: ln_launch_c<5>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
        case 6: ln_launch_c<6>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
        case 7: ln_launch_c<7>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
        default: ln_launch_c<8>(c, ops, pieces, n_pieces, s, hbm_operands, with_root); break;
    }
}
