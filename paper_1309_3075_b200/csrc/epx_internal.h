// Internal declarations shared by the CUDA translation units of libepx (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <algorithm>
#include <string>
#include <vector>

#define EPX_MAX_K 64
#define EPX_MAX_C 8
#define EPX_MAX_M 4096
#define EPX_INC_GRAPH_SLOTS 64     // matrix slots an incremental call may touch and still replay its CUDA graph
#define EPX_SORT_BINS 64 /* counting-sort bins for n_seg (n_seg >= 63 share the top bin) */

// Device-side status word bits (written by kernels, read back by the *log_likelihood calls).
enum : int {
    EPX_ST_JACOBI_NOCONV = 1,
    EPX_ST_NONFINITE_P = 2,
    EPX_ST_BAD_SITE = 4,
    EPX_ST_PADE_SINGULAR = 8,
};

// One pruning operation: an internal node and its two children (children sorted by label).
struct PruneOp {
    int node;
    int child[2];
    int child_is_tip[2];
    int pidx;        // index of `node` in the internal-partials array
    int cpidx[2];    // same for internal children (unused for tips)
};

// One operation of the depth-first pruning walk (prune4_dfs_kernel): node = product of its FIRST child (a) and its
// SECOND child (b).  code = (srcA+3) | (srcB+3) << 8 | (out_slot+1) << 16 with
//   src: -3 partials of another piece, read from HBM (pa / pb = its index in the partials array)
//        -2 tip   -1 result of the previous operation, still in registers (second child only)
//        >= 0 shared-memory stack slot (first child only)
//   out_slot: -1 = consumed by the next operation or by another launch; else the stack slot the result is parked in.
struct __align__(16) DfsOp {
    int32_t a, b;        // child node ids (matrix slot, tip row)
    int32_t pidx;        // this node's index in the partials array
    int32_t code;
    int32_t pa, pb;      // partials index of an HBM-sourced child
    int32_t pad0, pad1;
};
// bits 24 / 25 of code: the HBM operand a / b is written earlier in the SAME launch (incremental pieces): load it when the
// operation runs, never ahead of time
#define EPX_DFS_LATE_A (1 << 24)
#define EPX_DFS_LATE_B (1 << 25)
#define EPX_DFS_HBM (-3)
#define EPX_DFS_TIP (-2)
#define EPX_DFS_PREV (-1)
// A piece of the tree walked by one warp per pattern tile: operations [begin, end) of the DfsOp array.
struct DfsPiece { int32_t begin, end; };

// All device pointers, carved out of the caller's workspace by plan_workspace().
struct DevBuffers {
    // inputs
    double* tau;          // [M-1]
    double* Q;            // [M][K][K]
    double* freqs;        // [M][K]
    double* rates;        // [C]
    double* weights;      // [C]
    double* root_freqs;   // [K] (valid iff has_root_freqs)
    int32_t* eproc;       // [M] f2: first epoch with the same (Q, freqs) -- the process phi_m of PAPER.md L78; eproc[e] <= e
    int32_t* fproc;       // [M] first interior epoch with the same process AND the same duration tau_e - tau_{e-1} (full-epoch table)
    int32_t* parent;      // [n_nodes] tree mode
    double* height;       // [n_nodes] tree mode
    double* child_h;      // [n_br] branch-list mode
    double* parent_h;     // [n_br] branch-list mode
    double* brate;        // [n_slots] branch rate scalars (valid iff has_brates)
    uint8_t* tips;        // [N][Lp] 0..K-1, 255 = missing; rows padded to Lp = L rounded up to 32
    double* pattern_wt;   // [L]
    uint8_t* tip_vec;     // [N] 1 = the tip carries a partial vector (f3) and is read like an internal child
    PruneOp* ops;         // [N-1] sorted by level
    DfsOp* dfs_ops;       // [N-1] depth-first post-order (K == 4 pruning walk), piece after piece
    DfsPiece* dfs_pieces; // [<= N-1] op ranges of the pieces: bottom pieces (largest first), then the top piece
    // a1
    int32_t* n_seg;       // [n_br]
    int32_t* e_hi;        // [n_br] epoch of the parent end
    int32_t* seg_off;     // [n_br+1]
    int32_t* seg_epoch;   // [n_br*M] capacity
    double* seg_dur;      // [n_br*M] capacity
    int32_t* order;       // [n_br] slots sorted by n_seg, longest first
    // a2 (reversible): all with row stride Kp
    double* lam;          // [M][Kp]
    double* U;            // [M][Kp][Kp] eigenvectors of S = Pi^1/2 Q Pi^-1/2 (columns), zero padded
    double* W;            // [M][Kp][Kp] W[e] = U_e^T diag(sqrt(pi_e/pi_{e-1})) U_{e-1}, e >= 1
    double* sp;           // [M][Kp] sqrt(pi)
    double* isp;          // [M][Kp] 1/sqrt(pi)
    double* WB;           // [M][64*64] W in DMMA B-fragment order   (Kp == 64 only)
    double* UTB;          // [M][64*64] U^T in DMMA B-fragment order == U in A-fragment order (Kp == 64 only)
    double* GB;           // [(M-2)(M-1)/2][C][64*64] f1: products of consecutive full epochs, B-fragment order (Kp == 64 only)
    // a2' (asymmetric)
    double* Efull;        // [M][C][K][K] exp(Q_e r_c (tau_e - tau_{e-1})) for interior epochs 1..M-2
    // a3/a4 output
    double* P;            // [n_slots][C][K][K]
    double* PB;           // [n_slots][C][KP*KP] the same matrices in mma.m8n8k4 B-fragment order (tree mode, K > 8; prune_mma.cu)
    // a5
    double* partials;     // [N-1][C][L][K] internal nodes only, in op order
    int32_t* scale_exp;   // [N-1][L]
    // a6
    double* site_lnl;     // [L]
    double* block_sums;   // [reduce blocks]
    double* lnl;          // [1]
    int32_t* status;      // [1]
    // f1 incremental re-evaluation (lists rebuilt by every epx_log_likelihood_incremental call)
    int32_t* inc_slots;   // [n_slots] matrix slots to recompute
    DfsOp* inc_ops;       // [N-1] K == 4: the dirty nodes as one depth-first piece (children read from HBM or handed over)
    DfsPiece* inc_piece;  // [1]
    PruneOp* inc_pops;    // [N-1] other K: the dirty nodes' level-kernel operations, level by level
};

struct epx_ctx {
    int K = 0, M = 0, C = 0, N = 0, L = 0, device = 0;
    int Kp = 0;            // padded K used by the eigen buffers
    int n_nodes = 0;       // 2N-1 (tree mode)
    int n_slots = 0;       // matrix slots: n_nodes (tree mode) or n_br
    bool tree_mode = false;
    int reversible = -1;   // -1 unset, else the common flag of all epochs
    int chain_kernel = 0;  // EPX_OPT_CHAIN_KERNEL: 0 auto, 1 force the generic shared-memory kernel
    int use_graph = 1;     // EPX_OPT_USE_GRAPH
    int prune_kernel = 0;  // EPX_OPT_PRUNE_KERNEL: 0 auto, 1 force the generic shared-memory kernel
    int dfs_ppl = 0;       // EPX_OPT_DFS_PPL: patterns per lane of the depth-first pruning walk (0 auto, 1, 2, 4)
    int dfs_want = 0;      // EPX_OPT_DFS_PIECES: pieces the tree is cut into for the depth-first walks (0 auto)
    int epoch_products = 0; // EPX_OPT_EPOCH_PRODUCTS: 1 = chains over >= 2 full epochs use their cached product (f1); 0 (default) off
    int dedup = 1;         // EPX_OPT_SHARE_PROCESSES: 1 (default) one eigensystem / table entry per distinct process, 0 one per epoch
    std::vector<int32_t> eproc, fproc;   // host copies of the maps above (rebuilt when a model or a boundary changes)
    int jacobi_kernel = 0; // EPX_OPT_JACOBI_KERNEL: 0 auto, 1 round 1 kernel, 2 one CTA per process, 12 / 14 / 18 clusters of 2 / 4 / 8
    int mma_chunk = 0;     // EPX_OPT_MMA_CHUNK: site patterns per CTA of the tensor-pipe level kernel (0 auto)
    int exp_method = 0;    // EPX_OPT_EXP_METHOD: 0 auto, 1 spectral (Jacobi / Pade), 2 componentwise (shifted Taylor)
    std::vector<char> model_sparse;   // per epoch: Q has a structural zero off the diagonal

    // host copies of the inputs (uploaded lazily; *_dirty = needs upload)
    std::vector<double> tau, Q, freqs, rates, weights, root_freqs, height, child_h, parent_h, pattern_wt, brates;
    bool has_brates = false, brates_dirty = false;
    std::vector<int32_t> parent;
    uint8_t* tips = nullptr;           // [N][Lp] host staging of the tip states, page-locked (DMA source); see epx_set_tip_states
    bool tips_pinned = false;
    std::vector<char> model_set;
    bool has_tau = false, has_rates = false, has_tree = false, has_branches = false, has_tips = false,
         has_root_freqs = false;
    bool tau_dirty = false, model_dirty = false, rates_dirty = false, tree_dirty = false, branches_dirty = false,
         tips_dirty = false, wt_dirty = false, rootf_dirty = false;

    // plan (host): pruning ops sorted by level
    std::vector<PruneOp> ops;
    std::vector<int> level_off;        // ops[level_off[l] .. level_off[l+1]) form level l
    std::vector<int> node_pidx;        // node -> index in partials (internal) or -1
    std::vector<int> node_level;       // post-order level of every node (tips 0)
    std::vector<int> node_left, node_right;   // children (-1 for tips)
    // f1: nodes whose height changed since the last evaluation (epx_set_node_heights), and whether the device still
    // holds a complete evaluation of the current inputs that an incremental call can build on
    std::vector<int> dirty_nodes;
    bool inc_valid = false, heights_dirty = false;
    bool last_status_ok = false;        // device status word of the last evaluation was read and was 0
    bool status_known = false;          // ... was read at all (an enqueue without a fetch leaves it unknown)
    // f3: tips with a partial-likelihood vector instead of a state (partially observed).  Such a tip gets a
    // block in the partials array (index N-1 + slot, exponents 0) and enters the pruning plans like an internal child.
    int tip_cap = 0;                    // blocks reserved by epx_reserve_tip_partials (before epx_bind)
    std::vector<int> tip_slot;          // [N] slot of a tip, -1 = plain state
    std::vector<double> tip_part;       // [tip_cap][L][K] host copies
    std::vector<int> slot_free;         // free slots
    bool tipp_dirty = false;
    const int32_t* sub_list = nullptr;  // when set, the chain launchers recompute only these slots ...
    int sub_count = 0;                  // ... this many
    std::vector<DfsOp> dfs_ops;        // depth-first post-order walk with its stack-slot allocation
    std::vector<DfsPiece> dfs_pieces;  // bottom pieces (independent subtrees, largest first), then the top piece if any
    int dfs_bottom = 0;                // number of bottom pieces (launch 1); the rest (0 or 1) is launch 2
    std::vector<int> dfs_tier_end;     // pieces up to and including tier t (one launch per tier; K = 4 walks: at most two tiers)
    int dfs_depth = 0;                 // stack slots the walk needs
    int Lp = 0;                        // L rounded up to a multiple of 32 (row stride of the tip-state array)
    int root = -1;
    int reduce_blocks = 0;

    // binding
    void* ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    bool bound = false;
    DevBuffers d{};

    // CUDA graphs (only with a non-default stream)
    cudaGraphExec_t graph_mat = nullptr, graph_lik = nullptr, graph_inc = nullptr;   // graph_inc: an incremental call at K = 4 (fixed launch shapes)
    long long graph_inc_nodes = 0;
    const int32_t* sub_count_dev = nullptr;   // when set (incremental graph): the chain kernel reads the number of listed slots from here
    long long graph_mat_nodes = 0, graph_lik_nodes = 0;
    bool graphs_valid = false;

    // EPX_OPT_STAGE_EVENTS: ev[0] before the first stage, ev[k+1] after stage k (created lazily, destroyed with the ctx)
    int stage_events = 0;
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int stage_launches_mat[5] = {0, 0, 0, 0, 0}, stage_launches_lik[5] = {0, 0, 0, 0, 0};
    int graph_lik_launches[5] = {0, 0, 0, 0, 0}, graph_inc_launches[5] = {0, 0, 0, 0, 0};   // per-stage counts of the captured sequences
    bool capturing = false;   // enqueue_kernels is running under stream capture
    // graph mode only: a1 (segmenter) and a2 (eigensystems) are independent and run as two branches of the graph
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_seg = nullptr;

    long long launches = 0;
    bool have_result = false;
    bool have_lik = false;   // the last compute call included a5/a6
    std::string err;

    // a3 method of the next compute call (reading A21): the componentwise-accurate exponential serves likelihoods
    // over reversible models with structural zeros (codon models); everything else takes the spectral path.
    bool use_taylor() const
    {
        if (exp_method == 1) return false;
        if (exp_method == 2) return true;
        if (!tree_mode || reversible != 1) return false;
        for (char z : model_sparse) if (z) return true;
        return false;
    }
};

// ---- kernel launchers (each enqueues on `s`, returns the number of kernels launched, or -1 and sets the CUDA error)
int launch_segmenter(const epx_ctx* c, cudaStream_t s);
int launch_eigensystems(const epx_ctx* c, cudaStream_t s);
int launch_chain_reversible(const epx_ctx* c, cudaStream_t s);
bool chain_uses_epoch_products(const epx_ctx* c);
int launch_pade_chain(const epx_ctx* c, cudaStream_t s);
int launch_taylor_chain(const epx_ctx* c, cudaStream_t s);   // same kernels, shifted non-negative Taylor exponential
int launch_pruning(const epx_ctx* c, cudaStream_t s);
int launch_pruning_incremental(const epx_ctx* c, const std::vector<int>& group_off, cudaStream_t s);
int launch_root_reduction(const epx_ctx* c, cudaStream_t s);
size_t pade_smem_bytes(int K);
int chain_init_attributes();
int pade_init_attributes();
int eigen_init_attributes();
int prune_init_attributes();
int prune_tile(int K, int C);   // patterns per CTA of the generic pruning kernel
int dfs_tiles(const epx_ctx* c);         // warps per piece of the depth-first walk
bool prune_wants_kdfs(const epx_ctx* c); // the same without the shared-memory check (which needs the plan)
bool prune_uses_kdfs(const epx_ctx* c);  // K != 4 depth-first walk for few patterns (generic partials layout)
bool prune_uses_lane(const epx_ctx* c);  // K == 4 depth-first walk, one lane per pattern (default; generic partials layout)
bool prune_uses_dfs(const epx_ctx* c);   // K == 4 depth-first walk, lane = (pattern, category): partials are laid out [node][L][C][4]
inline bool prune_walk4(const epx_ctx* c) { return prune_uses_lane(c) || prune_uses_dfs(c); }   // any K == 4 walk (DfsOp plans)
// prune_lane.cu
int lane_patterns_per_lane(const epx_ctx* c);
size_t lane_smem_bytes(const epx_ctx* c, int depth);
int prune_lane_init_attributes();
void launch_prune4_lane(const epx_ctx* c, const DfsOp* ops, const DfsPiece* pieces, int n_pieces, cudaStream_t s, bool hbm_operands,
                        bool with_root = false);   // with_root: the LAST piece ends at the root; its warps also do a6
bool prune_root_fused(const epx_ctx* c);   // a6 runs inside the K = 4 lane walk (no root kernel)
// prune_mma.cu: level kernel on the FP64 tensor pipe for 8 < K <= 64
inline int prune_kp(const epx_ctx* c) { return (c->K + 7) & ~7; }
bool prune_uses_mma(const epx_ctx* c);
int prune_mma_chunk(const epx_ctx* c, int nops);
int prune_mma_init_attributes();
void launch_prune_mma_level(const epx_ctx* c, const PruneOp* ops, int nops, cudaStream_t s, bool pdl);
void launch_pb_swizzle(const epx_ctx* c, cudaStream_t s);

// Where the pruning kernels of this ctx keep partials and scale exponents.  Element (node block n, category c, pattern p,
// state i) sits at n * node + c * sc + p * sp + i; its exponent at (n * C + c) * L + p if exp_per_cat, else at n * L + p.
struct PartialLayout { size_t node, sc, sp; int ks; bool exp_per_cat; };
inline PartialLayout partial_layout(const epx_ctx* c)
{
    PartialLayout l;
    const size_t K = c->K, C = c->C, L = c->L;
    if (prune_uses_mma(c)) { const size_t KP = prune_kp(c); l = {C * L * KP, L * KP, KP, (int)KP, true}; }
    else if (prune_uses_dfs(c)) l = {C * L * K, K, C * K, (int)K, false};
    else l = {C * L * K, L * K, K, (int)K, false};
    return l;
}
