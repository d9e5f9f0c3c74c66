// C-ABI boundary and host orchestration of libepx (include/epx.h).  The host side validates inputs, owns the plan
// (post-order levels, buffer offsets inside the caller's workspace), uploads inputs, and enqueues the kernels of
// segmenter.cu / eigen.cu / chain.cu / pade.cu / prune.cu on the caller's stream (replayed from a CUDA graph when the
// stream is not the legacy default stream).  No arithmetic of the method runs on the host.
#include "../../include/epx.h"
#include "epx_internal.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <condition_variable>
#include <functional>
#include <mutex>
#include <thread>
#include <pthread.h>
#if defined(__SSE2__)
#include <emmintrin.h>
#endif

namespace {

int fail(epx_ctx* c, int code, const char* fmt, ...) __attribute__((format(printf, 3, 4)));
int fail(epx_ctx* c, int code, const char* fmt, ...)
{
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    return code;
}

#define CUDA_TRY(c, call)                                                                         \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess) return fail((c), EPX_E_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// Carve the workspace.  With base == nullptr only the total size is computed.
size_t plan_workspace(const epx_ctx* c, char* base, DevBuffers* d)
{
    size_t off = 0;
    auto take = [&](size_t bytes) -> char* {
        char* p = base ? base + off : nullptr;
        off += align_up(bytes ? bytes : 1);
        return p;
    };
    const size_t K = c->K, M = c->M, C = c->C, N = c->N, L = c->L, Kp = c->Kp, S = c->n_slots;
    DevBuffers t{};
    t.tau = (double*)take(8 * (M - 1));
    t.Q = (double*)take(8 * M * K * K);
    t.freqs = (double*)take(8 * M * K);
    t.rates = (double*)take(8 * C);
    t.weights = (double*)take(8 * C);
    t.root_freqs = (double*)take(8 * K);
    t.eproc = (int32_t*)take(4 * M);
    t.fproc = (int32_t*)take(4 * M);
    if (c->tree_mode) {
        t.parent = (int32_t*)take(4 * S);
        t.height = (double*)take(8 * S);
        t.tips = (uint8_t*)take(N * (size_t)c->Lp);
        t.pattern_wt = (double*)take(8 * L);
        t.tip_vec = (uint8_t*)take(N);
        t.ops = (PruneOp*)take(sizeof(PruneOp) * (N - 1));
        t.dfs_ops = (DfsOp*)take(sizeof(DfsOp) * (N - 1));
        t.dfs_pieces = (DfsPiece*)take(sizeof(DfsPiece) * (N - 1));
    } else {
        t.child_h = (double*)take(8 * S);
        t.parent_h = (double*)take(8 * S);
    }
    t.brate = (double*)take(8 * S);
    t.n_seg = (int32_t*)take(4 * S);
    t.e_hi = (int32_t*)take(4 * S);
    t.seg_off = (int32_t*)take(4 * (S + 1));
    t.seg_epoch = (int32_t*)take(4 * S * M);
    t.seg_dur = (double*)take(8 * S * M);
    t.order = (int32_t*)take(4 * S);
    t.lam = (double*)take(8 * M * Kp);
    t.U = (double*)take(8 * M * Kp * Kp);
    t.W = (double*)take(8 * M * Kp * Kp);
    t.sp = (double*)take(8 * M * Kp);
    t.isp = (double*)take(8 * M * Kp);
    t.WB = (double*)take(Kp == 64 ? 8 * M * 4096 : 0);
    t.UTB = (double*)take(Kp == 64 ? 8 * M * 4096 : 0);
    t.GB = (double*)take(Kp == 64 && M >= 4 ? 8 * ((M - 2) * (M - 1) / 2) * C * 4096 : 0);
    t.Efull = (double*)take(8 * M * C * K * K);
    t.P = (double*)take(8 * S * C * K * K);
    if (c->tree_mode) {
        // sized for every layout an option can select later: states padded to 8 and one exponent per category when K > 8
        const size_t Kalloc = K > 8 ? (size_t)prune_kp(c) : K;
        t.PB = (double*)take(K != 4 ? 8 * S * C * Kalloc * Kalloc : 0);     // fragment-ordered / transposed copies of P
        t.partials = (double*)take(8 * (N - 1 + (size_t)c->tip_cap) * C * L * Kalloc);
        t.scale_exp = (int32_t*)take(4 * (N - 1 + (size_t)c->tip_cap) * L * (K > 8 ? C : 1));
        t.site_lnl = (double*)take(8 * L);
        t.block_sums = (double*)take(8 * ((L + 7) / 8));
    }
    // one block: the piece of an incremental walk (8 B), the number of listed slots (4 B, read by the incremental graph's chain
    // kernel), 4 B of padding, the slot list -- so that a move uploads them with ONE copy
    {
        unsigned char* hdr = (unsigned char*)take(16 + 4 * S);
        t.inc_piece = (DfsPiece*)hdr;
        t.inc_slots = (int32_t*)(hdr ? hdr + 16 : nullptr);
    }
    if (c->tree_mode) {
        t.inc_ops = (DfsOp*)take(sizeof(DfsOp) * (N - 1));
        t.inc_pops = (PruneOp*)take(sizeof(PruneOp) * (N - 1));
    }
    t.lnl = (double*)take(8);
    t.status = (int32_t*)take(8);      // [0] status word, [1] arrival counter of the root reduction
    if (d) *d = t;
    return off;
}

void drop_graphs(epx_ctx* c)
{
    c->inc_valid = false;      // whatever invalidates the graphs also invalidates an incremental continuation
    c->tipp_dirty = true;      // ... and may change the partials layout the tip blocks were written in
    if (c->graph_mat) { cudaGraphExecDestroy(c->graph_mat); c->graph_mat = nullptr; }
    if (c->graph_inc) { cudaGraphExecDestroy(c->graph_inc); c->graph_inc = nullptr; }
    if (c->graph_lik) { cudaGraphExecDestroy(c->graph_lik); c->graph_lik = nullptr; }
}

// Post-order plan: level(tip) = 0, level(u) = 1 + max(level(children)); ops sorted by level.
int build_plan(epx_ctx* c)
{
    const int n = c->n_nodes, N = c->N;
    std::vector<int> left(n, -1), right(n, -1), level(n, 0);
    int root = -1, roots = 0;
    for (int i = 0; i < n; i++) {
        int p = c->parent[i];
        if (p < 0) { root = i; roots++; continue; }
        if (p >= n || p < N || p == i) return fail(c, EPX_E_TREE, "node %d: parent %d is not an internal node", i, p);
        if (c->height[p] < c->height[i]) return fail(c, EPX_E_TREE, "node %d is above its parent %d", i, p);
        if (left[p] < 0) left[p] = i;
        else if (right[p] < 0) right[p] = i;
        else return fail(c, EPX_E_TREE, "node %d has more than two children", p);
    }
    if (roots != 1) return fail(c, EPX_E_TREE, "%d roots (need exactly one)", roots);
    for (int i = 0; i < n; i++) {
        if (!std::isfinite(c->height[i])) return fail(c, EPX_E_TREE, "height[%d] is not finite", i);
        if (i < N ? (left[i] >= 0) : (right[i] < 0)) return fail(c, EPX_E_TREE, "node %d: not bifurcating / tip with children", i);
    }
    // iterative post-order from the root (also proves every node is reachable, i.e. no cycle)
    std::vector<int> stack{root}, order;
    order.reserve(n);
    while (!stack.empty()) {
        int u = stack.back(); stack.pop_back();
        order.push_back(u);
        if (left[u] >= 0) { stack.push_back(left[u]); stack.push_back(right[u]); }
    }
    if ((int)order.size() != n) return fail(c, EPX_E_TREE, "tree is not connected (cycle)");
    int max_level = 0;
    for (int k = n - 1; k >= 0; k--) {
        int u = order[k];
        if (left[u] >= 0) level[u] = 1 + std::max(level[left[u]], level[right[u]]);
        max_level = std::max(max_level, level[u]);
    }
    std::vector<int> internal;
    for (int i = 0; i < n; i++) if (left[i] >= 0) internal.push_back(i);
    std::stable_sort(internal.begin(), internal.end(), [&](int a, int b) { return level[a] < level[b]; });
    c->node_pidx.assign(n, -1);
    for (size_t k = 0; k < internal.size(); k++) c->node_pidx[internal[k]] = (int)k;
    if (c->tip_slot.empty()) c->tip_slot.assign(N, -1);
    for (int t = 0; t < N; t++)
        if (c->tip_slot[t] >= 0) c->node_pidx[t] = (N - 1) + c->tip_slot[t];      // its block of 0/1 (or weighted) partials
    c->ops.resize(internal.size());
    c->level_off.assign(max_level + 1, 0);
    for (size_t k = 0; k < internal.size(); k++) {
        int u = internal[k];
        PruneOp& op = c->ops[k];
        op.node = u;
        op.pidx = (int)k;
        op.child[0] = left[u];
        op.child[1] = right[u];
        for (int h = 0; h < 2; h++) {
            op.child_is_tip[h] = op.child[h] < N && c->tip_slot[op.child[h]] < 0;
            op.cpidx[h] = c->node_pidx[op.child[h]];
        }
        c->level_off[level[u]]++;      // count per level (levels 1..max_level)
    }
    // level_off[l] currently holds the count of level l (index 0 unused = 0): turn into offsets over levels 1..max
    std::vector<int> offs(max_level + 1, 0);
    for (int l = 1; l <= max_level; l++) offs[l] = offs[l - 1] + c->level_off[l];
    c->level_off = offs;               // ops of level l (1-based) are [offs[l-1], offs[l])
    c->root = root;
    c->node_level = level;
    c->node_left = left;
    c->node_right = right;

    // Depth-first post-order walk for prune4_dfs_kernel.  Every internal node becomes one DfsOp; the child visited
    // SECOND hands its result over in registers, the child visited FIRST parks its result in a stack slot.  Visiting
    // the subtree that needs more slots first (Sethi-Ullman) keeps the stack at <= log2(N) + 1 slots.
    // One warp walks one piece for one tile of patterns.  With few patterns a single walk of the whole tree leaves the
    // SMs short of warps, so the tree is cut into independent subtrees (bottom pieces, one launch) and the part above
    // them (top piece, a second launch that reads the bottom pieces' root partials from HBM).
    std::vector<int> size(n, 0), need(n, 0);
    for (int k = n - 1; k >= 0; k--) {
        int u = order[k];
        if (left[u] >= 0) size[u] = 1 + size[left[u]] + size[right[u]];
    }
    std::vector<char> is_cut(n, 0);           // roots of the bottom pieces
    std::vector<int> cuts;
    {
        const long tiles = dfs_tiles(c);
        // pieces wanted (< 8 = no cut): 4 x the number needed for 24 warps per SM; measured on config 2 (625 tiles):
        // 12 -> 0.69 ms, 24 -> 0.68 ms, 48 -> 0.70 ms, 64 -> 0.73 ms
        // lane-per-pattern walk (K == 4 default; ~10 one-warp CTAs per SM): ~5 000 warps in flight keep the store stream
        // saturated; measured on config 2 (313 tiles): 8 -> 0.520 ms, 12 -> 0.486, 16 -> 0.483, 24 -> 0.485, 48 -> 0.501
        const long auto_want = prune_uses_lane(c) ? std::min<long>(64, (5000 + tiles - 1) / tiles)
                                                  : std::min<long>(64, 4 * ((148L * 24 + tiles - 1) / tiles));
        const long want = c->dfs_want > 0 ? c->dfs_want : auto_want;
        std::vector<int> heap{root};          // max-heap on subtree size
        auto cmp = [&](int x, int y) { return size[x] < size[y]; };
        const long min_cut = c->dfs_want > 0 ? 2 : 8;
        while (want >= min_cut && (long)heap.size() + (long)cuts.size() < want) {
            std::pop_heap(heap.begin(), heap.end(), cmp);
            int u = heap.back(); heap.pop_back();
            if (size[u] <= 8) { heap.push_back(u); std::push_heap(heap.begin(), heap.end(), cmp); break; }
            for (int ch : {left[u], right[u]})
                if (left[ch] >= 0) {
                    if (size[ch] <= 8) cuts.push_back(ch);
                    else { heap.push_back(ch); std::push_heap(heap.begin(), heap.end(), cmp); }
                }
            if (heap.empty()) break;
        }
        if (!(heap.size() == 1 && heap[0] == root && cuts.empty())) for (int u : heap) cuts.push_back(u);
        else cuts.push_back(root);
        std::sort(cuts.begin(), cuts.end(), [&](int x, int y) { return size[x] != size[y] ? size[x] > size[y] : x < y; });
        for (int u : cuts) is_cut[u] = 1;
    }
    const bool has_top = !(cuts.size() == 1 && cuts[0] == root);
    // Tiers of pieces, one launch each: the bottom pieces, then what reads their roots from HBM, and so on.
    std::vector<std::vector<int>> tier_roots;
    tier_roots.push_back(cuts);
    if (has_top) tier_roots.push_back({root});
    // Few-pattern walk (K != 4, one warp per pattern) on a DEEP tree: the time is the chain of dependent operations, largest
    // bottom piece + top piece (322 of config 4's 1499).  Level bands cut that chain to about the depth of the tree: a piece =
    // a connected set of nodes whose level (height above the tips in operations) falls into one band, bands widening
    // like (k / T)^2.5 towards the root (the upper tree is a caterpillar: a band of width w there is a chain of ~w operations,
    // while near the tips many small subtrees run side by side).  Config 4: 6 bands, 186 dependent operations.
    if (prune_wants_kdfs(c) && c->dfs_want == 0 && max_level >= 48) {
        const int T = std::min(8, std::max(3, (max_level + 14) / 28));
        std::vector<int> th(T);
        for (int k = 0; k < T; k++) th[k] = std::max(k + 1, (int)std::lround(max_level * std::pow((k + 1.0) / T, 2.5)));    // (exponents 1.5 .. 3 measured: 2.5 gives the shortest chain on config 4)
        th[T - 1] = max_level;
        std::vector<int> band(n, -1);
        for (int u : internal) { int k = 0; while (level[u] > th[k]) k++; band[u] = k; }
        std::fill(is_cut.begin(), is_cut.end(), 0);
        tier_roots.assign(T, {});
        std::vector<int> comp(n, 0);              // operations of the piece below (and including) u
        for (int k = n - 1; k >= 0; k--) {
            const int u = order[k];
            if (left[u] < 0) continue;
            comp[u] = 1;
            for (int ch : {left[u], right[u]}) if (left[ch] >= 0 && band[ch] == band[u]) comp[u] += comp[ch];
        }
        for (int u : internal)
            if (c->parent[u] < 0 || band[c->parent[u]] != band[u]) { tier_roots[band[u]].push_back(u); is_cut[u] = 1; }
        for (auto& r : tier_roots) std::sort(r.begin(), r.end(), [&](int x, int y) { return comp[x] != comp[y] ? comp[x] > comp[y] : x < y; });
        tier_roots.erase(std::remove_if(tier_roots.begin(), tier_roots.end(), [](const std::vector<int>& r) { return r.empty(); }), tier_roots.end());
    }
    // kind of a child as seen from the piece being walked: 0 tip, 1 internal (walk into it), 2 root of a bottom piece
    // (a tip with a partial vector is read from HBM like the root of another piece)
    // (a piece never contains the root of another piece except as an operand: inside a bottom piece there is none)
    auto kind = [&](int v, bool) { return left[v] < 0 ? (c->tip_slot[v] >= 0 ? 2 : 0) : is_cut[v] ? 2 : 1; };
    for (int k = n - 1; k >= 0; k--) {         // stack slots a walk of u's piece needs (Sethi-Ullman), children before parents
        int u = order[k];
        if (left[u] < 0) continue;
        int ka = kind(left[u], true), kb = kind(right[u], true);
        int na = ka == 1 ? need[left[u]] : 0, nb = kb == 1 ? need[right[u]] : 0;
        if (ka == 1 && kb == 1) need[u] = std::max(std::max(na, nb), std::min(na, nb) + 1);
        else need[u] = std::max(1, std::max(na, nb));
    }
    struct Frame { int u, first, second, stage, slot; };
    std::vector<Frame> fr;
    std::vector<int> free_slots;
    int high = 0;
    c->dfs_ops.clear();
    c->dfs_ops.reserve(internal.size());
    c->dfs_pieces.clear();
    auto walk = [&](int piece_root, bool top) {
        const int begin = (int)c->dfs_ops.size();
        free_slots.clear();
        int next_slot = 0;
        auto push_node = [&](int u) {
            int a = left[u], b = right[u];
            bool ia = kind(a, top) == 1, ib = kind(b, top) == 1;
            // first = the walked child with the larger need (or the leaf when only one child is walked)
            if ((ia && ib && need[b] > need[a]) || (ia && !ib)) std::swap(a, b);
            fr.push_back({u, a, b, 0, -1});
        };
        push_node(piece_root);
        while (!fr.empty()) {
            const size_t topi = fr.size() - 1;
            Frame f = fr[topi];
            const int k1 = kind(f.first, top), k2 = kind(f.second, top);
            if (f.stage == 0) {
                fr[topi].stage = 1;
                if (k1 == 1) { push_node(f.first); continue; }
                f.stage = 1;
            }
            if (f.stage == 1) {
                if (k1 == 1) {     // the op just emitted is `first`: park its result
                    int s;
                    if (!free_slots.empty()) { s = free_slots.back(); free_slots.pop_back(); }
                    else s = next_slot++;
                    c->dfs_ops.back().code |= (s + 1) << 16;
                    fr[topi].slot = f.slot = s;
                }
                fr[topi].stage = 2;
                if (k2 == 1) { push_node(f.second); continue; }
            }
            DfsOp op{};
            op.a = f.first; op.b = f.second; op.pidx = c->node_pidx[f.u];
            const int srcA = k1 == 1 ? f.slot : k1 == 2 ? EPX_DFS_HBM : EPX_DFS_TIP;
            const int srcB = k2 == 1 ? EPX_DFS_PREV : k2 == 2 ? EPX_DFS_HBM : EPX_DFS_TIP;
            op.pa = k1 == 2 ? c->node_pidx[f.first] : 0;
            op.pb = k2 == 2 ? c->node_pidx[f.second] : 0;
            op.code = (srcA + 3) | ((srcB + 3) << 8);
            if (f.slot >= 0) free_slots.push_back(f.slot);
            c->dfs_ops.push_back(op);
            fr.pop_back();
        }
        high = std::max(high, next_slot);
        c->dfs_pieces.push_back({begin, (int)c->dfs_ops.size()});
    };
    c->dfs_tier_end.clear();
    for (const auto& roots : tier_roots) {
        for (int u : roots) walk(u, true);
        c->dfs_tier_end.push_back((int)c->dfs_pieces.size());
    }
    c->dfs_bottom = c->dfs_tier_end[0];
    c->dfs_depth = std::max(high, 1);
    if (high > 250) return fail(c, EPX_E_TREE, "tree needs %d pruning stack slots (limit 250)", high);
    return EPX_OK;
}

}  // namespace

extern "C" {

int epx_create(epx_ctx** out, int K, int M, int C, int N_tips, int L, int device)
{
    if (!out) return EPX_E_ARG;
    *out = nullptr;
    if (K < 2 || K > EPX_MAX_K || M < 1 || M > EPX_MAX_M || C < 1 || C > EPX_MAX_C) return EPX_E_ARG;
    if (N_tips != 0 && (N_tips < 2 || L < 1)) return EPX_E_ARG;
    if (device < 0) return EPX_E_ARG;
    epx_ctx* c = new (std::nothrow) epx_ctx();
    if (!c) return EPX_E_ARG;
    c->K = K; c->M = M; c->C = C; c->N = N_tips; c->L = N_tips ? L : 0; c->device = device;
    c->Kp = K <= 4 ? K : (K <= 32 ? (K + 7) & ~7 : 64);
    c->tree_mode = N_tips > 0;
    c->n_nodes = c->tree_mode ? 2 * N_tips - 1 : 0;
    c->n_slots = c->n_nodes;
    c->Q.assign((size_t)M * K * K, 0.0);
    c->freqs.assign((size_t)M * K, 0.0);
    c->model_set.assign(M, 0);
    c->model_sparse.assign(M, 0);
    if (c->tree_mode) {
        c->Lp = (L + 31) & ~31;
        c->pattern_wt.assign(L, 1.0);
        c->wt_dirty = true;
        c->reduce_blocks = K > 8 ? (L + 7) / 8 : (L + 255) / 256;       // K > 8: one warp per pattern (root_site_warp_kernel)
    }
    if (M == 1) { c->has_tau = true; }
    *out = c;
    return EPX_OK;
}

void epx_destroy(epx_ctx* c)
{
    if (!c) return;
    drop_graphs(c);
    for (cudaEvent_t e : c->ev) if (e) cudaEventDestroy(e);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->ev_seg) cudaEventDestroy(c->ev_seg);
    if (c->side) cudaStreamDestroy(c->side);
    if (c->tips) { if (c->tips_pinned) cudaFreeHost(c->tips); else free(c->tips); }
    delete c;
}

const char* epx_last_error(const epx_ctx* c) { return c ? c->err.c_str() : "null ctx"; }

int epx_workspace_bytes(const epx_ctx* c, size_t* bytes)
{
    if (!c || !bytes) return EPX_E_ARG;
    if (!c->tree_mode && !c->has_branches) return EPX_E_STATE;
    *bytes = plan_workspace(c, nullptr, nullptr);
    return EPX_OK;
}

int epx_bind(epx_ctx* c, void* ws, size_t bytes, void* stream)
{
    if (!c || !ws) return EPX_E_ARG;
    if (!c->tree_mode && !c->has_branches) return fail(c, EPX_E_STATE, "branch-list mode: call epx_set_branches before epx_bind");
    if ((uintptr_t)ws & 255) return fail(c, EPX_E_WORKSPACE, "workspace must be 256-byte aligned");
    size_t need = plan_workspace(c, nullptr, nullptr);
    if (bytes < need) return fail(c, EPX_E_WORKSPACE, "workspace has %zu bytes, %zu needed", bytes, need);
    CUDA_TRY(c, cudaSetDevice(c->device));
    cudaPointerAttributes attr{};
    CUDA_TRY(c, cudaPointerGetAttributes(&attr, ws));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return fail(c, EPX_E_WORKSPACE, "workspace is not device memory");
    if (chain_init_attributes() || pade_init_attributes() || eigen_init_attributes() || prune_init_attributes() ||
        prune_mma_init_attributes())
        return fail(c, EPX_E_CUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(cudaGetLastError()));
    drop_graphs(c);
    plan_workspace(c, (char*)ws, &c->d);
    c->ws = ws; c->ws_bytes = bytes; c->stream = (cudaStream_t)stream; c->bound = true;
    c->tau_dirty = c->model_dirty = c->rates_dirty = c->tree_dirty = c->branches_dirty = c->tips_dirty = c->wt_dirty =
        c->rootf_dirty = c->brates_dirty = true;
    c->have_result = false;
    return EPX_OK;
}

int epx_set_option(epx_ctx* c, int option, int value)
{
    if (!c) return EPX_E_ARG;
    switch (option) {
        case 1: c->chain_kernel = value; break;
        case 2: c->use_graph = value; break;
        case 3:
            c->prune_kernel = value;
            if (c->has_tree) { int rc = build_plan(c); if (rc) return rc; c->tree_dirty = true; }   // pieces depend on the kernel's tile
            break;
        case 4: if (value < 0 || value > 2) return fail(c, EPX_E_ARG, "exp method %d", value); c->exp_method = value; break;
        case 5: c->stage_events = value ? 1 : 0; break;
        case 6:
            if (value != 0 && value != 1 && value != 2 && value != 4) return fail(c, EPX_E_ARG, "patterns per lane %d", value);
            c->dfs_ppl = value;
            if (c->has_tree) { int rc = build_plan(c); if (rc) return rc; c->tree_dirty = true; }
            break;
        case 11: c->epoch_products = value ? 1 : 0; break;
        case 10: c->dedup = value ? 1 : 0; c->model_dirty = true; break;
        case 9:
            if (value != 0 && value != 1 && value != 2 && value != 14 && value != 18) return fail(c, EPX_E_ARG, "jacobi kernel %d", value);
            
            c->jacobi_kernel = value;
            break;
        case 8:
            if (value < 0 || value > (1 << 20)) return fail(c, EPX_E_ARG, "chunk %d", value);
            c->mma_chunk = value;
            break;
        case 7:
            if (value < 0 || value > 4096) return fail(c, EPX_E_ARG, "pieces %d", value);
            c->dfs_want = value;
            if (c->has_tree) { int rc = build_plan(c); if (rc) return rc; c->tree_dirty = true; }
            break;
        default: return fail(c, EPX_E_ARG, "unknown option %d", option);
    }
    drop_graphs(c);
    return EPX_OK;
}

int epx_set_epoch_boundaries(epx_ctx* c, const double* tau)
{
    if (!c) return EPX_E_ARG;
    if (c->M == 1) { c->has_tau = true; return EPX_OK; }
    if (!tau) return fail(c, EPX_E_ARG, "tau is NULL");
    for (int k = 0; k < c->M - 1; k++) {
        if (!std::isfinite(tau[k])) return fail(c, EPX_E_ARG, "tau[%d] is not finite", k);
        if (k && !(tau[k] > tau[k - 1])) return fail(c, EPX_E_ARG, "tau must be strictly increasing (index %d)", k);
    }
    c->tau.assign(tau, tau + c->M - 1);
    c->has_tau = true; c->tau_dirty = true;
    return EPX_OK;
}

int epx_set_epoch_model(epx_ctx* c, int epoch, const double* Q, const double* freqs, int reversible)
{
    if (!c || !Q || !freqs) return EPX_E_ARG;
    if (epoch < 0 || epoch >= c->M) return fail(c, EPX_E_ARG, "epoch %d out of range", epoch);
    const int K = c->K;
    double maxdiag = 0.0;
    for (int i = 0; i < K; i++) maxdiag = std::max(maxdiag, std::fabs(Q[i * K + i]));
    long double fs = 0;
    for (int i = 0; i < K; i++) {
        long double s = 0;
        for (int j = 0; j < K; j++) {
            double q = Q[i * K + j];
            if (!std::isfinite(q)) return fail(c, EPX_E_MODEL, "Q[%d][%d] is not finite", i, j);
            if (i != j && q < 0) return fail(c, EPX_E_MODEL, "Q[%d][%d] < 0", i, j);
            s += q;
        }
        if (std::fabs((double)s) > 1e-9 * maxdiag) return fail(c, EPX_E_MODEL, "row %d of Q sums to %g", i, (double)s);
        if (!(freqs[i] >= 0)) return fail(c, EPX_E_MODEL, "freqs[%d] < 0 or NaN", i);
        fs += freqs[i];
    }
    if (std::fabs((double)(fs - 1)) > 1e-9) return fail(c, EPX_E_MODEL, "freqs sum to %.12g", (double)fs);
    if (reversible) {
        double maxflux = 0.0;
        for (int i = 0; i < K; i++) {
            if (!(freqs[i] > 0)) return fail(c, EPX_E_MODEL, "reversible model needs freqs[%d] > 0", i);
            for (int j = 0; j < K; j++) if (i != j) maxflux = std::max(maxflux, freqs[i] * Q[i * K + j]);
        }
        for (int i = 0; i < K; i++)
            for (int j = i + 1; j < K; j++)
                if (std::fabs(freqs[i] * Q[i * K + j] - freqs[j] * Q[j * K + i]) > 1e-9 * maxflux)
                    return fail(c, EPX_E_MODEL, "detailed balance violated at (%d,%d)", i, j);
    }
    int flag = reversible ? 1 : 0;
    if (c->reversible >= 0 && c->reversible != flag) {
        bool others = false;
        for (int e = 0; e < c->M; e++) if (e != epoch && c->model_set[e]) others = true;
        if (others) return fail(c, EPX_E_MODEL, "all epochs of a ctx must share the reversible flag");
    }
    if (c->reversible != flag) drop_graphs(c);
    c->reversible = flag;
    std::copy(Q, Q + K * K, c->Q.begin() + (size_t)epoch * K * K);
    std::copy(freqs, freqs + K, c->freqs.begin() + (size_t)epoch * K);
    c->model_set[epoch] = 1;
    {
        const bool was = c->use_taylor();
        char sparse = 0;
        for (int i = 0; i < K; i++)
            for (int j = 0; j < K; j++) if (i != j && Q[i * K + j] == 0.0) sparse = 1;
        c->model_sparse[epoch] = sparse;
        if (was != c->use_taylor()) drop_graphs(c);
    }
    c->model_dirty = true;
    return EPX_OK;
}

int epx_set_category_rates(epx_ctx* c, const double* rates, const double* weights)
{
    if (!c || !rates || !weights) return EPX_E_ARG;
    long double ws = 0;
    for (int k = 0; k < c->C; k++) {
        if (!(rates[k] >= 0) || !std::isfinite(rates[k])) return fail(c, EPX_E_ARG, "rates[%d] must be finite and >= 0", k);
        if (!(weights[k] >= 0)) return fail(c, EPX_E_ARG, "weights[%d] < 0 or NaN", k);
        ws += weights[k];
    }
    if (std::fabs((double)(ws - 1)) > 1e-9) return fail(c, EPX_E_ARG, "category weights sum to %.12g", (double)ws);
    c->rates.assign(rates, rates + c->C);
    c->weights.assign(weights, weights + c->C);
    c->has_rates = true; c->rates_dirty = true;
    return EPX_OK;
}

int epx_set_tree(epx_ctx* c, const int32_t* parent, const double* height)
{
    if (!c || !parent || !height) return EPX_E_ARG;
    if (!c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in branch-list mode");
    if (c->has_tree && (int)c->parent.size() == c->n_nodes && std::memcmp(c->parent.data(), parent, sizeof(int32_t) * c->n_nodes) == 0) {
        // Same topology (an MCMC chain mostly moves heights): the pruning plans, the launch shapes and the CUDA graphs depend
        // on the topology only, so only the heights are validated and replaced (the plans cost 0.2 ms for 2 000 tips).
        for (int i = 0; i < c->n_nodes; i++) {
            if (!std::isfinite(height[i])) return fail(c, EPX_E_TREE, "height[%d] is not finite", i);
            const int p = parent[i];
            if (p >= 0 && height[p] < height[i]) return fail(c, EPX_E_TREE, "node %d is above its parent %d", i, p);
        }
        c->height.assign(height, height + c->n_nodes);
        c->heights_dirty = true;
        c->inc_valid = false;              // every branch may have changed: the next evaluation is a full one
        c->dirty_nodes.clear();
        return EPX_OK;
    }
    std::vector<int32_t> old_parent = c->parent;
    c->parent.assign(parent, parent + c->n_nodes);
    c->height.assign(height, height + c->n_nodes);
    int rc = build_plan(c);
    if (rc != EPX_OK) { c->has_tree = false; return rc; }
    if (old_parent != c->parent) drop_graphs(c);      // launch shapes depend on the topology only
    c->has_tree = true; c->tree_dirty = true;
    c->dirty_nodes.clear();
    return EPX_OK;
}

int epx_set_node_heights(epx_ctx* c, int n, const int32_t* nodes, const double* heights)
{
    if (!c || n < 0 || (n > 0 && (!nodes || !heights))) return EPX_E_ARG;
    if (!c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in branch-list mode");
    if (!c->has_tree) return fail(c, EPX_E_STATE, "epx_set_tree has not been called");
    std::vector<double> old(n);
    for (int k = 0; k < n; k++) {
        if (nodes[k] < 0 || nodes[k] >= c->n_nodes) return fail(c, EPX_E_ARG, "node %d out of range", nodes[k]);
        if (!std::isfinite(heights[k])) return fail(c, EPX_E_ARG, "height of node %d is not finite", nodes[k]);
    }
    for (int k = 0; k < n; k++) { old[k] = c->height[nodes[k]]; c->height[nodes[k]] = heights[k]; }
    for (int k = 0; k < n; k++) {          // the order of parents and children must survive the move
        const int u = nodes[k], p = c->parent[u];
        bool ok = p < 0 || c->height[p] >= c->height[u];
        if (c->node_left[u] >= 0) ok = ok && c->height[u] >= c->height[c->node_left[u]] && c->height[u] >= c->height[c->node_right[u]];
        if (!ok) {
            for (int j = n - 1; j >= 0; j--) c->height[nodes[j]] = old[j];
            return fail(c, EPX_E_TREE, "node %d would leave the interval between its children and its parent", u);
        }
    }
    c->dirty_nodes.insert(c->dirty_nodes.end(), nodes, nodes + n);
    c->heights_dirty = true;
    return EPX_OK;
}

int epx_set_branches(epx_ctx* c, int n_br, const double* child_height, const double* parent_height)
{
    if (!c || !child_height || !parent_height || n_br < 1) return EPX_E_ARG;
    if (c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in tree mode");
    if (c->bound && n_br != c->n_slots) return fail(c, EPX_E_STATE, "n_br cannot change after epx_bind");
    for (int b = 0; b < n_br; b++) {
        if (!std::isfinite(child_height[b]) || !std::isfinite(parent_height[b]) || parent_height[b] < child_height[b])
            return fail(c, EPX_E_ARG, "branch %d: need finite parent_height >= child_height", b);
    }
    c->child_h.assign(child_height, child_height + n_br);
    c->parent_h.assign(parent_height, parent_height + n_br);
    c->n_slots = n_br;
    c->has_branches = true; c->branches_dirty = true;
    return EPX_OK;
}

int epx_set_branch_rates(epx_ctx* c, const double* rates)
{
    if (!c) return EPX_E_ARG;
    const bool had = c->has_brates;
    if (!rates) {
        c->has_brates = false;
    } else {
        if (!c->tree_mode && !c->has_branches) return fail(c, EPX_E_STATE, "branch-list mode: call epx_set_branches first");
        for (int b = 0; b < c->n_slots; b++)
            if (!std::isfinite(rates[b]) || rates[b] < 0) return fail(c, EPX_E_ARG, "branch rate %d must be finite and >= 0", b);
        c->brates.assign(rates, rates + c->n_slots);
        c->has_brates = true; c->brates_dirty = true;
    }
    if (had != c->has_brates) drop_graphs(c);     // kernel arguments (rate pointer, full-epoch table use) change
    return EPX_OK;
}

// Host worker threads for the tip-state repacking, created once per process and parked on a condition variable (spawning
// 15 threads per call cost ~0.4 ms of a 1.4 ms call).  Never destroyed: the threads are detached and the object is leaked on
// purpose, so there is no destruction-order hazard at exit; a forked child starts a fresh pool.
namespace {
struct HostPool {
    std::mutex mu, busy;
    std::condition_variable cv, cv_done;
    std::function<void()> job;
    int want = 0, started = 0, finished = 0, nthreads = 0;
    unsigned long long gen = 0;
    HostPool()
    {
        nthreads = (int)std::min<size_t>(15, std::max(1u, std::thread::hardware_concurrency()) - 1);
        for (int i = 0; i < nthreads; i++) std::thread([this] { loop(); }).detach();
    }
    void loop()
    {
        unsigned long long seen = 0;
        std::unique_lock<std::mutex> lk(mu);
        for (;;) {
            cv.wait(lk, [&] { return gen != seen; });
            seen = gen;
            if (started >= want) continue;
            started++;
            lk.unlock();
            job();
            lk.lock();
            if (++finished == want) cv_done.notify_all();
        }
    }
    // `k` workers run fn once each while the caller goes on; finish() waits for them.  One job at a time per process.
    void start(int k, std::function<void()> fn)
    {
        busy.lock();
        std::lock_guard<std::mutex> lk(mu);
        job = std::move(fn); want = std::min(k, nthreads); started = finished = 0; gen++;
        cv.notify_all();
    }
    void finish()
    {
        {
            std::unique_lock<std::mutex> lk(mu);
            cv_done.wait(lk, [&] { return finished == want; });
            job = nullptr;
        }
        busy.unlock();
    }
};
HostPool* g_pool = nullptr;
std::mutex g_pool_mu;             // guards g_pool
std::once_flag g_pool_fork;
// fork(): only the forking thread exists in the child, so a pool mutex that some other thread held at that moment would stay
// locked there for ever (the child's first epx_set_tip_states would hang).  The prepare handler therefore takes all three locks
// (in the order start() takes them: g_pool_mu, busy, mu -- an in-flight repacking job is waited for), both sides release them
// again, and the child drops the pool (its worker threads do not exist there; a fresh one is made on first use).
void pool_fork_prepare()
{
    g_pool_mu.lock();
    if (g_pool) { g_pool->busy.lock(); g_pool->mu.lock(); }
}
void pool_fork_parent()
{
    if (g_pool) { g_pool->mu.unlock(); g_pool->busy.unlock(); }
    g_pool_mu.unlock();
}
void pool_fork_child()
{
    if (g_pool) { g_pool->mu.unlock(); g_pool->busy.unlock(); }
    g_pool = nullptr;             // (the old object is leaked on purpose: its condition variables belong to threads that are gone)
    g_pool_mu.unlock();
}
HostPool& host_pool()
{
    std::call_once(g_pool_fork, [] { pthread_atfork(pool_fork_prepare, pool_fork_parent, pool_fork_child); });
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (!g_pool) g_pool = new HostPool();
    return *g_pool;
}
}  // namespace

// Repack tip states (int32 or bytes) into the padded byte rows of the page-locked staging buffer.  Integer repacking,
// split over host threads; no arithmetic of the method.
extern "C++" {
template <typename T>
static int set_tips_impl(epx_ctx* c, const T* states)
{
    if (!c || !states) return EPX_E_ARG;
    if (!c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in branch-list mode");
    const size_t L = (size_t)c->L, Lp = (size_t)c->Lp, N = (size_t)c->N;
    if (!c->tips) {
        // page-locked staging buffer: the upload is then a plain DMA that overlaps the host work of the next setters
        void* ptr = nullptr;
        if (cudaSetDevice(c->device) == cudaSuccess && cudaHostAlloc(&ptr, N * Lp, cudaHostAllocDefault) == cudaSuccess) {
            c->tips = (uint8_t*)ptr; c->tips_pinned = true;
        } else {
            cudaGetLastError();
            c->tips = (uint8_t*)malloc(N * Lp);
            if (!c->tips) return fail(c, EPX_E_ARG, "out of host memory for %zu tip states", N * Lp);
        }
    } else if (c->bound) {
        // an earlier upload may still be reading the staging buffer
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    }
    const unsigned K = (unsigned)c->K;
    uint8_t* const base = c->tips;
    // rows [t0, t1): everything the inner loops read is a by-value local (a byte store may alias any object in memory, so
    // values reached through a closure or the ctx would be re-read every iteration and the loops would not vectorise)
    auto convert_rows = [](const T* states, uint8_t* base, size_t L, size_t Lp, unsigned K, size_t t0, size_t t1) {
        for (size_t t = t0; t < t1; t++) {
            const T* __restrict__ src = states + t * L;
            uint8_t* __restrict__ dst = base + t * Lp;
            if (sizeof(T) == 1) {
                const uint8_t k8 = (uint8_t)K;                // K <= 64
                const uint8_t* __restrict__ s8 = reinterpret_cast<const uint8_t*>(src);
                size_t p = 0;
#if defined(__SSE2__)
                // Streaming (non-temporal) stores: the staging buffer is only read by the DMA engine, and lines left dirty in
                // the caches of six cores halved the host -> device rate (20 MB: 0.8 - 1.0 ms against 0.4 ms).  Rows of the
                // page-locked buffer start on 32-byte boundaries (Lp is a multiple of 32).
                if ((reinterpret_cast<uintptr_t>(dst) & 15) == 0) {
                    const __m128i kv = _mm_set1_epi8((char)k8);
                    for (; p + 16 <= L; p += 16) {
                        const __m128i v = _mm_loadu_si128(reinterpret_cast<const __m128i*>(s8 + p));
                        const __m128i ge = _mm_cmpeq_epi8(_mm_max_epu8(v, kv), v);          // v >= K (unsigned): 0xff
                        _mm_stream_si128(reinterpret_cast<__m128i*>(dst + p), _mm_or_si128(v, ge));
                    }
                }
#endif
                for (; p < L; p++) dst[p] = (uint8_t)(s8[p] | (uint8_t)(0 - (uint8_t)(s8[p] >= k8)));   // byte-wide
            } else {
                const uint32_t* __restrict__ s32 = reinterpret_cast<const uint32_t*>(src);
                size_t p = 0;
#if defined(__SSE2__)
                if ((reinterpret_cast<uintptr_t>(dst) & 15) == 0) {         // 16 states per streamed store (see the byte form)
                    const __m128i bias = _mm_set1_epi32((int)0x80000000u), kk = _mm_set1_epi32((int)(K ^ 0x80000000u));
                    const __m128i miss = _mm_set1_epi32(255);
                    for (; p + 16 <= L; p += 16) {
                        __m128i r[4];
                        for (int q = 0; q < 4; q++) {
                            const __m128i u = _mm_loadu_si128(reinterpret_cast<const __m128i*>(s32 + p + 4 * q));
                            const __m128i lt = _mm_cmplt_epi32(_mm_xor_si128(u, bias), kk);              // u < K, unsigned
                            r[q] = _mm_or_si128(_mm_and_si128(lt, u), _mm_andnot_si128(lt, miss));
                        }
                        _mm_stream_si128(reinterpret_cast<__m128i*>(dst + p),
                                         _mm_packus_epi16(_mm_packs_epi32(r[0], r[1]), _mm_packs_epi32(r[2], r[3])));
                    }
                }
#endif
                for (; p < L; p++) {
                    const uint32_t s = s32[p];                // negative int32 -> huge -> missing
                    dst[p] = (uint8_t)(s < K ? s : 255u);
                }
            }
            for (size_t p = L; p < Lp; p++) dst[p] = 255;
        }
#if defined(__SSE2__)
        _mm_sfence();                                         // the streamed rows are globally visible before the chunk is reported
#endif
    };
    // measured on a 16-core host: bytes -> bytes saturates the memory system at 5-6 threads (more are slower), the int32 form
    // reads four times as much and keeps gaining up to 16
    const size_t max_nt = sizeof(T) == 1 ? 6 : 16;
    const size_t nthreads = std::min<size_t>(std::min<size_t>(max_nt, std::max(1u, std::thread::hardware_concurrency())), (N * L) >> 21);
    if (nthreads <= 1) {
        convert_rows(states, base, L, Lp, K, 0, N);
    } else if (!(c->bound && c->tips_pinned)) {
        HostPool& pool = host_pool();
        const size_t nw = std::min<size_t>(nthreads, (size_t)pool.nthreads + 1);
        std::atomic<size_t> share{1};
        pool.start((int)nw - 1, [&] {
            const size_t w = share.fetch_add(1);
            convert_rows(states, base, L, Lp, K, N * w / nw, N * (w + 1) / nw);
        });
        convert_rows(states, base, L, Lp, K, 0, N / nw);            // the calling thread takes the first share
        pool.finish();
    } else {
        // Bound ctx: the host -> device copy is pipelined with the repacking.  Workers take chunks of rows in order; the
        // calling thread enqueues the copy of chunk k on the ctx's stream as soon as chunk k is complete, so the DMA of one
        // chunk runs while the next ones are still being repacked (page-locked source, stream-ordered after the last
        // evaluation that read the tips).
        CUDA_TRY(c, cudaSetDevice(c->device));
        const size_t nchunks = std::min<size_t>(N, 4 * nthreads);
        // copies of >= 4 MB: a host -> device copy has tens of microseconds of fixed cost (64 copies of 0.3 MB took 1.6 ms
        // where 5 of 4 MB take 0.5)
        const size_t per_copy = std::max<size_t>(1, std::min(nchunks, ((size_t)4 << 20) * nchunks / (N * Lp) + 1));
        std::atomic<size_t> next{0};
        std::vector<std::atomic<int>> done(nchunks);
        for (auto& f : done) f.store(0, std::memory_order_relaxed);
        auto worker = [&]() {
            for (size_t k; (k = next.fetch_add(1)) < nchunks;) {
                convert_rows(states, base, L, Lp, K, N * k / nchunks, N * (k + 1) / nchunks);
                done[k].store(1, std::memory_order_release);
            }
        };
        HostPool& pool = host_pool();
        pool.start((int)nthreads - 1, worker);

        if (pool.nthreads == 0) worker();
        cudaError_t err = cudaSuccess;
        for (size_t k0 = 0; k0 < nchunks; k0 += per_copy) {
            const size_t k1 = std::min(nchunks, k0 + per_copy);
            for (size_t k = k0; k < k1; k++)
                while (!done[k].load(std::memory_order_acquire)) std::this_thread::yield();
            const size_t r0 = N * k0 / nchunks, r1 = N * k1 / nchunks;
            if (err == cudaSuccess)
                err = cudaMemcpyAsync(c->d.tips + r0 * Lp, base + r0 * Lp, (r1 - r0) * Lp, cudaMemcpyHostToDevice, c->stream);
        }
        pool.finish();
        if (err != cudaSuccess) return fail(c, EPX_E_CUDA, "cudaMemcpyAsync (tip states): %s", cudaGetErrorString(err));
        c->has_tips = true; c->tips_dirty = false;     // already on its way to the device
        c->inc_valid = false;
        return EPX_OK;
    }
    c->has_tips = true; c->tips_dirty = true;
    return EPX_OK;
}
}  // extern "C++"

int epx_set_tip_states(epx_ctx* c, const int32_t* states) { return set_tips_impl(c, states); }
int epx_set_tip_states_u8(epx_ctx* c, const uint8_t* states) { return set_tips_impl(c, states); }

int epx_reserve_tip_partials(epx_ctx* c, int max_tips)
{
    if (!c || max_tips < 0) return EPX_E_ARG;
    if (!c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in branch-list mode");
    if (c->bound) return fail(c, EPX_E_STATE, "epx_reserve_tip_partials must precede epx_bind");
    for (int slot : c->tip_slot)
        if (slot >= 0) return fail(c, EPX_E_STATE, "a tip still carries a vector: epx_set_tip_partials(tip, NULL) first");
    if (max_tips > c->N) max_tips = c->N;
    c->tip_cap = max_tips;
    c->tip_slot.assign(c->N, -1);
    c->tip_part.assign((size_t)max_tips * c->L * c->K, 0.0);
    c->slot_free.clear();
    for (int s = max_tips - 1; s >= 0; s--) c->slot_free.push_back(s);
    return EPX_OK;
}

int epx_set_tip_partials(epx_ctx* c, int tip, const double* partials)
{
    if (!c) return EPX_E_ARG;
    if (!c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in branch-list mode");
    if (tip < 0 || tip >= c->N) return fail(c, EPX_E_ARG, "tip %d out of range", tip);
    if (c->tip_slot.empty()) c->tip_slot.assign(c->N, -1);
    const size_t LK = (size_t)c->L * c->K;
    int slot = c->tip_slot[tip];
    if (!partials) {                                    // back to the tip's state
        if (slot < 0) return EPX_OK;
        c->slot_free.push_back(slot);
        c->tip_slot[tip] = -1;
    } else {
        for (size_t i = 0; i < LK; i++)
            if (!(partials[i] >= 0) || !std::isfinite(partials[i])) return fail(c, EPX_E_ARG, "tip partial %zu must be finite and >= 0", i);
        if (slot < 0) {
            if (c->slot_free.empty()) return fail(c, EPX_E_STATE, "no tip-partial block left: epx_reserve_tip_partials(%d)", c->tip_cap);
            slot = c->slot_free.back(); c->slot_free.pop_back();
            c->tip_slot[tip] = slot;
        } else {
            std::copy(partials, partials + LK, c->tip_part.begin() + (size_t)slot * LK);
            c->tipp_dirty = true; c->inc_valid = false;
            return EPX_OK;                              // same plan, new values
        }
        std::copy(partials, partials + LK, c->tip_part.begin() + (size_t)slot * LK);
    }
    drop_graphs(c);                                     // the plans change: this tip is now read as a vector / as a state
    if (c->has_tree) { int rc = build_plan(c); if (rc) return rc; c->tree_dirty = true; }
    return EPX_OK;
}

int epx_set_pattern_weights(epx_ctx* c, const double* wt)
{
    if (!c) return EPX_E_ARG;
    if (!c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in branch-list mode");
    if (wt) {
        for (int p = 0; p < c->L; p++) if (!std::isfinite(wt[p])) return fail(c, EPX_E_ARG, "wt[%d] is not finite", p);
        c->pattern_wt.assign(wt, wt + c->L);
    } else {
        c->pattern_wt.assign(c->L, 1.0);
    }
    c->wt_dirty = true;
    return EPX_OK;
}

int epx_set_root_frequencies(epx_ctx* c, const double* freqs)
{
    if (!c) return EPX_E_ARG;
    if (!c->tree_mode) return fail(c, EPX_E_STATE, "ctx is in branch-list mode");
    bool had = c->has_root_freqs;
    if (freqs) {
        long double s = 0;
        for (int i = 0; i < c->K; i++) { if (!(freqs[i] >= 0)) return fail(c, EPX_E_ARG, "root freqs[%d] < 0 or NaN", i); s += freqs[i]; }
        if (std::fabs((double)(s - 1)) > 1e-9) return fail(c, EPX_E_ARG, "root freqs sum to %.12g", (double)s);
        c->root_freqs.assign(freqs, freqs + c->K);
        c->has_root_freqs = true; c->rootf_dirty = true;
    } else {
        c->has_root_freqs = false;
    }
    if (had != c->has_root_freqs) drop_graphs(c);
    return EPX_OK;
}

}  // extern "C"

#include "api_compute.inc"
