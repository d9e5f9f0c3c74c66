/*
 * epx.h -- C-ABI boundary of the B200-native epoch-substitution-model hot path (arxiv 1309.3075).
 *
 * What the library computes (citations are PAPER.md lines; "A<n>" are the readings listed in DESIGN.md):
 *   a1  branch -> ordered (epoch, duration) segments, parent end first        L78 (change-point process), L117 (weights)
 *   a2  per-epoch eigensystem of a reversible Q (symmetrised Jacobi)          L58 (detailed balance), L80, L314-L316
 *   a2' Pade [13/13] scaling-and-squaring for an asymmetric Q                 L48 (exp(tQ), Moler & Van Loan)
 *   a3  segment transition matrices exp(Q_e * r_c * d)                        L58-L60 Eq.(3)
 *   a4  ordered chain product P_b = prod_k exp(Q_k r_c t_k), parent end first L84-L109 Eq.(5)-(7) (A2)
 *   a5  Felsenstein pruning of partial likelihoods, post-order                L64-L72 Eq.(4)
 *   a6  root / category / site-pattern aggregation into log-likelihoods       L72
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  fp64 throughout.
 *
 * Conventions
 *   - Time is HEIGHT, measured backwards from the most recent tip (A1).  Epoch e in 0..M-1 covers heights
 *     [tau[e-1], tau[e]) with tau[-1] = -inf and tau[M-1] = +inf; `tau` holds the M-1 finite boundaries, so
 *     epoch 0 is the most recent one and the leftmost factor of P_b is the OLDEST epoch on the branch.
 *   - Matrices are row-major K x K, P[i][j] = Pr(child-end state j | parent-end state i).
 *   - Every call returns 0 (EPX_OK) or a negative error code; nothing throws, aborts or prints.
 *     epx_last_error(ctx) is a ctx-owned NUL-terminated message, valid until the next call on that ctx.
 *   - All `const T*` inputs below are HOST pointers and are copied during the call (caller keeps ownership).
 *   - Device memory and the stream are OWNED BY THE CALLER and borrowed: the library allocates no device
 *     memory.  `dev_workspace` must stay alive and untouched while the ctx is bound to it.
 *   - A ctx is not thread-safe; distinct ctxs are independent.
 *   - Nothing is cached between compute calls: every epx_update_matrices / epx_*log_likelihood call re-runs
 *     all of its steps on the device.  Setters only re-upload the array they set.  The one exception is asked for by
 *     name: epx_log_likelihood_incremental reuses the matrices and partials of the previous evaluation that a node move
 *     cannot have changed.
 */
#ifndef EPX_H
#define EPX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct epx_ctx epx_ctx; /* opaque; created / destroyed by the library */

enum {
    EPX_OK = 0,
    EPX_E_ARG = -1,       /* NULL / out-of-range argument */
    EPX_E_STATE = -2,     /* a required setter or epx_bind has not been called, or wrong mode */
    EPX_E_TREE = -3,      /* not a strictly bifurcating rooted tree with tips 0..N-1, or a child above its parent */
    EPX_E_MODEL = -4,     /* Q rows do not sum to 0, negative off-diagonal, freqs not a distribution, reversible flag violated */
    EPX_E_WORKSPACE = -5, /* workspace too small or misaligned (256 B) */
    EPX_E_CUDA = -6,      /* a CUDA runtime call failed (message holds cudaGetErrorString) */
    EPX_E_NUMERIC = -7    /* Jacobi did not converge / non-finite matrix / a site likelihood <= 0 */
};

/* Limits of this build: 2 <= K <= 64, 1 <= M <= 4096, 1 <= C <= 8, N_tips == 0 or >= 2, L >= 1 when N_tips > 0. */

/* Create a context for K states, M epochs, C rate categories, N_tips tips (0 = branch-list mode: matrices only,
 * no tree / likelihood; "matrix convolution" workload) and L site patterns on CUDA device `device`. */
int epx_create(epx_ctx** out, int K, int M, int C, int N_tips, int L, int device);
void epx_destroy(epx_ctx* ctx);

/* Bytes of device workspace the ctx needs.  Tree mode: valid right after create.  Branch-list mode: after
 * epx_set_branches (the size depends on n_br). */
int epx_workspace_bytes(const epx_ctx* ctx, size_t* bytes);

/* Borrow `bytes` of DEVICE memory (256-byte aligned) and a cudaStream_t (may be 0 = legacy default stream; CUDA
 * graphs are only used with a non-default stream).  All kernels and copies of this ctx are ordered on that stream.
 * Inputs set before or after bind are uploaded lazily by the next compute call. */
int epx_bind(epx_ctx* ctx, void* dev_workspace, size_t bytes, void* cuda_stream);

/* ---- model inputs (PAPER.md L46 Q, L58 pi, L72 categories, L78 epochs) ---- */
/* tau: M-1 finite, strictly increasing boundary heights (NULL allowed iff M == 1). */
int epx_set_epoch_boundaries(epx_ctx* ctx, const double* tau);
/* Q: K*K row-major including the diagonal, used as given (not normalised, A7/A8); |sum_j Q_ij| <= 1e-9 max|Q_ii|,
 * off-diagonals >= 0.  freqs: K, >= 0, sum 1.  reversible = 1 selects the Jacobi path and requires pi_i > 0 and
 * |pi_i q_ij - pi_j q_ji| <= 1e-9 max|pi q|; 0 selects Pade.  All epochs of a ctx must use the same flag. */
int epx_set_epoch_model(epx_ctx* ctx, int epoch, const double* Q, const double* freqs, int reversible);
/* Shared processes (S processes Q_s, M epochs, phi_m in 1..S picks the process active in epoch m; L193, L203:
 * 13-14 epochs alternating 2 or 4 matrices).  Models are set per epoch; epochs whose Q and freqs are bit-identical are
 * detected and share ONE eigensystem (and one full-epoch exponential per distinct duration on the Pade path).  This call
 * reports the detected map: phi[e] in 0..*n_processes-1, numbered by first appearance (phi: M entries).  Needs every epoch
 * model set.  Sharing never changes results (EPX_OPT_SHARE_PROCESSES = 0 computes one per epoch: bit-identical). */
int epx_epoch_processes(epx_ctx* ctx, int32_t* phi, int* n_processes);
/* rates: C, >= 0 (the r_c of Eq. 3, A6).  weights: C, >= 0, sum 1. */
int epx_set_category_rates(epx_ctx* ctx, const double* rates, const double* weights);

/* ---- tree mode (N tips, 2N-1 nodes, bifurcating) ---- */
/* parent: 2N-1 entries, tips are 0..N-1, the root has -1.  height: 2N-1, height[parent] >= height[child].
 * EPX_E_TREE on anything else.  A call whose parent array equals the current one only validates and replaces the heights (the
 * pruning plans and launch graphs depend on the topology alone) and, if it fails, leaves the current tree in place; a new
 * topology that fails validation leaves the context without a tree. */
int epx_set_tree(epx_ctx* ctx, const int32_t* parent, const double* height);
/* states: [N][L] row-major; 0..K-1 = observed state, anything else = missing (all-ones tip vector, A10).  Large inputs
 * (>= 4 M states) are repacked by a process-wide pool of host threads that serves ONE call at a time: tip-state setters of
 * different contexts or threads queue behind each other for that part.  The pool survives fork() (the child starts its own). */
int epx_set_tip_states(epx_ctx* ctx, const int32_t* states);
/* The same from bytes ([N][L] row-major; 0..K-1 = observed state, anything else, e.g. 255, = missing): a quarter of the
 * host memory traffic of the int32 form -- sequence data are bytes to begin with. */
int epx_set_tip_states_u8(epx_ctx* ctx, const uint8_t* states);
/* Partially observed tips (tip vectors are "0 or 1 depending on whether trait i is (partially) observed").
 * epx_reserve_tip_partials: how many tips may carry a vector at the same time (each costs one block of partials,
 * C*L*K doubles, in the workspace); call before epx_workspace_bytes / epx_bind.  Default 0.
 * epx_set_tip_partials: tip `tip` is described by partials[L][K] (>= 0, finite: 0/1 for an ambiguity set, any weights in
 * general) instead of its state; NULL returns it to its state from epx_set_tip_states.  The same vector serves every
 * rate category. */
int epx_reserve_tip_partials(epx_ctx* ctx, int max_tips);
int epx_set_tip_partials(epx_ctx* ctx, int tip, const double* partials);
/* wt: L pattern weights (a weight w == the pattern repeated w times), or NULL = all 1. */
int epx_set_pattern_weights(epx_ctx* ctx, const double* wt);
/* freqs: K root distribution, or NULL (default) = the freqs of the root's epoch (A9).  The root's epoch follows the
 * parent-end rule of a branch (A3): e = #{k : tau[k] < height[root]}.  A root exactly ON a boundary tau[k] therefore takes
 * the YOUNGER epoch k (the process everything below it evolved under), although as a child end that height would open
 * epoch k+1: the half-open intervals [tau[e-1], tau[e]) above describe child ends; parent ends (and the root) use
 * (tau[e-1], tau[e]]. */
int epx_set_root_frequencies(epx_ctx* ctx, const double* freqs);

/* ---- branch-list mode ---- */
/* n_br branches given by their two end heights, parent_height[b] >= child_height[b]. */
int epx_set_branches(epx_ctx* ctx, int n_br, const double* child_height, const double* parent_height);

/* ---- optional: per-branch rate scalars r_v (relaxed clocks; the rate is constant along a branch) ----
 * rates: one per matrix slot (tree mode: 2N-1 entries indexed by node, the root's entry is ignored; branch-list mode: n_br
 * entries), finite and >= 0, or NULL = all 1 (the default).  The effective rate of a segment is r_v * r_c (reading A6), so
 * P_b = prod_k exp(Q_k r_v r_c t_k); epx_get_segments then reports durations already multiplied by r_v.  Branch-list
 * mode: call after epx_set_branches. */
int epx_set_branch_rates(epx_ctx* ctx, const double* rates);

/* ---- compute ---- */
/* a1..a4, enqueued on the stream, does not synchronise.  Matrix slot = node index (tree mode; the root's slot
 * holds the identity) or branch index. */
int epx_update_matrices(epx_ctx* ctx);
/* a1..a6, enqueued on the stream, does not synchronise (tree mode only). */
int epx_enqueue_log_likelihood(epx_ctx* ctx);
/* a1..a6, then synchronises the stream and writes the total log-likelihood to *logL (host). EPX_E_NUMERIC if a
 * device-side numeric check failed (*logL is still written). */
int epx_log_likelihood(epx_ctx* ctx, double* logL);
/* Synchronise and fetch the result of the last enqueue (same checks as epx_log_likelihood). */
int epx_fetch_log_likelihood(epx_ctx* ctx, double* logL);

/* Many independent instances (eight patients, one codon model each): the same as
 * epx_log_likelihood on each of the n contexts, but every context's work is enqueued (on the stream it was bound with) before
 * the first result is fetched, so the kernel sequences of contexts bound to DIFFERENT streams overlap on the device; contexts
 * that share a stream run one after the other.  logL: n host doubles.  rc: n per-context return codes, or NULL.  Returns
 * EPX_OK or the first non-zero code; the other contexts are still evaluated.  Results are bit-identical to single calls. */
int epx_log_likelihood_batch(epx_ctx* const* ctxs, int n, double* logL, int* rc);

/* ---- incremental re-evaluation (an MCMC step re-dispatches only what its proposal
 * touches) ----
 * epx_set_node_heights: move `n` nodes (node ids, new heights) without changing the topology; every moved node must stay
 * between its children and its parent (EPX_E_TREE otherwise, nothing is changed).  Cheaper than epx_set_tree: no plan is
 * rebuilt, and the moved nodes are remembered.
 * epx_log_likelihood_incremental: like epx_log_likelihood, but when the device still holds a complete evaluation of the
 * current inputs and only node heights moved since, it recomputes just the matrices of the moved nodes' branches and of
 * their children's branches, and the partials of the moved nodes and their ancestors.  The result is bit-identical to a
 * full evaluation.  In every other situation it is a full evaluation. */
int epx_set_node_heights(epx_ctx* ctx, int n, const int32_t* nodes, const double* heights);
int epx_log_likelihood_incremental(epx_ctx* ctx, double* logL);

/* ---- read-back (each synchronises the stream; results of the LAST compute call) ---- */
/* Segment list of matrix slot `slot`: *n_seg entries, parent end first; epoch/dur hold at least M entries. */
int epx_get_segments(epx_ctx* ctx, int slot, int* n_seg, int32_t* epoch, double* dur);
/* One K*K matrix (host, row-major). */
int epx_get_matrix(epx_ctx* ctx, int slot, int category, double* out);
/* Borrowed DEVICE pointer to all matrices, [slot][C][K][K] row-major fp64, valid while bound. */
int epx_matrices_device(epx_ctx* ctx, const double** dptr);
/* Partials of `node` as [C][L][K] (host) and the per-pattern power-of-two exponents scale_exp[L]:
 * true partial = out * 2^scale_exp (A12).  Tips return their 0/1 vectors and zero exponents. */
int epx_get_partials(epx_ctx* ctx, int node, double* out, int32_t* scale_exp);
/* Per-pattern log-likelihoods ln l_p (unweighted), L entries (host). */
int epx_get_site_log_likelihoods(epx_ctx* ctx, double* out);

/* ---- introspection ---- */
/* Number of kernel launches (graph nodes count individually) the ctx has enqueued since create. */
int epx_launch_count(const epx_ctx* ctx, long long* n);
const char* epx_last_error(const epx_ctx* ctx);

/* Stages of a compute call, in enqueue order. */
enum {
    EPX_STAGE_SEGMENT = 0, /* a1 */
    EPX_STAGE_EIGEN = 1,   /* a2 Jacobi + change-of-basis prep (0 launches on the Pade / Taylor paths).  When the call is
                              replayed from a CUDA graph a2 runs as a second branch beside a1 (they are independent) and
                              this stage's time is only what a1 did not hide */
    EPX_STAGE_CHAIN = 2,   /* a2' + a3 + a4 */
    EPX_STAGE_PRUNE = 3,   /* a5, one launch per post-order level */
    EPX_STAGE_ROOT = 4,    /* a6 */
    EPX_N_STAGES = 5
};
/* With EPX_OPT_STAGE_EVENTS = 1 every compute call -- epx_log_likelihood_incremental included (its a2 stage is empty: the
 * eigensystems are reused) -- records a CUDA event on the stream before the first stage and
 * after each stage (inside the CUDA graph when one is used).  This call synchronises the stream and writes the device
 * time of each stage of the LAST compute call to ms[EPX_N_STAGES] and the number of kernels each stage launched to
 * launches[EPX_N_STAGES] (either may be NULL).  Stages the call did not run report 0 ms / 0 launches.
 * K == 4 on the eigensystem path with a non-default stream: the segmenter runs on a second stream beside a2..a5 (the chain
 * kernel segments its own branches), so EPX_STAGE_SEGMENT reports ~0 ms with its launches counted -- its time is hidden, not
 * measured, and these stage times are not comparable with a run where a1 sits in front (EPX_OPT_USE_GRAPH = 0).
 * EPX_E_STATE if the option is off or nothing has run. */
int epx_get_stage_ms(epx_ctx* ctx, float* ms, int* launches);

/* Measured fp64 peak on `device`: kind 0 = DFMA (plain FP64 FMA pipe), kind 1 = DMMA (mma.sync m8n8k4 f64).
 * Runs a register-only kernel for about `ms_target` ms on `cuda_stream` and writes TFLOP/s (2 flop per FMA) to
 * *tflops (host).  `dev_scratch` is >= 8 bytes of caller-owned DEVICE memory (never written in practice; it keeps the
 * compiler from deleting the arithmetic).  Synchronises the stream. */
int epx_measure_fp64_peak(int device, int kind, double ms_target, void* dev_scratch, void* cuda_stream, double* tflops);

/* ---- a1 alone, for callers that may not allocate device memory (PAPER.md L78 change-point process, L117 the epochs a
 * branch spans; readings A1-A3) ----
 * Everything above borrows a workspace that somebody had to allocate.  Some callers cannot: a routine that runs inside
 * another program's sampling loop under that program's fixed GPU memory budget, a callback on a path where cudaMalloc's
 * device-wide synchronisation would stall other streams, a plug-in whose host hands it input and output buffers from its own
 * arena and nothing more.  For them this one call splits a branch list into its per-epoch segments using only the buffers it
 * is given: its intermediates (segment counts, parent-end epochs, a sort order; 12 bytes per branch) live in an array that
 * is part of the library's device image -- 384 KiB on every GPU that loads the library, until the process exits.  The call
 * makes no cudaMalloc / cudaFree and uses no allocating library routine.
 *
 *   device            CUDA device the pointers and the stream belong to; made current for the call, the previous one restored.
 *   n_br              0 .. EPX_STATIC_MAX_BRANCHES branches.  More is refused with EPX_E_WORKSPACE and a message naming the
 *                     limit (split the list, or use a bound context: epx_set_branches + epx_update_matrices).
 *   M, dev_tau        M epochs (1 .. 4096) and their M-1 finite, strictly increasing boundary heights (DEVICE; may be NULL iff
 *                     M == 1).  Not validated: the caller vouches for the order, as it does for the heights.
 *   dev_child_height, dev_parent_height   [n_br] DEVICE, parent >= child (a branch of length 0 gets no segment).
 *   dev_seg_off       [n_br + 1] DEVICE out: CSR offsets; dev_seg_off[n_br] = total number of segments.
 *   dev_seg_epoch, dev_seg_dur, cap       DEVICE out with room for `cap` segments each: branch b's segments sit at
 *                     [seg_off[b], seg_off[b+1]), parent end first (epoch numbers descending), unscaled durations -- the
 *                     values epx_get_all_segments returns for the same branches, bit for bit.  Segments at positions >= cap are
 *                     not stored (check dev_seg_off[n_br] <= cap; n_br * M always suffices).  May be NULL iff cap == 0.
 *   cuda_stream       the three kernels are enqueued here; the call does not synchronise.  Inputs, outputs and the stream stay
 *                     the caller's.
 *   errbuf, errbuf_len   optional host buffer for a NUL-terminated message when the return code is not EPX_OK (there is no ctx
 *                     to keep it); may be NULL / 0.
 *
 * First call on a device: looks up where that device keeps the built-in array (cudaGetSymbolAddress) and remembers it; this may
 * make the CUDA runtime load the library's device code.  Make that first call during start-up, before the stream is put under
 * stream capture.  Later calls on the same device only launch kernels.
 * Sharing: every call on a device uses the same array, and the array keeps the previous call's contents.  Each call overwrites
 * the part it reads before reading it, so calls that follow one another on the GPU (same stream, or ordered by events) are
 * independent; two calls whose kernels can overlap on the GPU (different streams, different host threads) race on the array
 * and may both return wrong segments.  Thread-safe on the host side otherwise.
 * Returns EPX_OK, EPX_E_ARG (NULL pointer, range), EPX_E_WORKSPACE (n_br over the limit) or EPX_E_CUDA. */
#define EPX_STATIC_MAX_BRANCHES 32768
int epx_segment_branches_static(int device, int n_br, int M, const double* dev_tau, const double* dev_child_height,
                                const double* dev_parent_height, int32_t* dev_seg_off, int32_t* dev_seg_epoch,
                                double* dev_seg_dur, int cap, void* cuda_stream, char* errbuf, size_t errbuf_len);

/* ---- tuning / test hooks (options 1-3, 6-8, 10 have no effect on results; 9 and 11 only within rounding) ---- */
enum {
    EPX_OPT_CHAIN_KERNEL = 1, /* 0 auto (default); 1 force the generic shared-memory chain kernel; 2 (32 < K <= 64) round 1's
                                 tensor-pipe layout, two categories per CTA, instead of one category per CTA (four warps of 16 rows) */
    EPX_OPT_USE_GRAPH = 2,    /* 1 (default) replay the kernel sequence from a CUDA graph on non-default streams; 0 launch directly */
    EPX_OPT_PRUNE_KERNEL = 3, /* 0 auto (default).  K == 4: depth-first walk, one lane per site pattern, partials never
                                 re-read from HBM.  8 < K <= 64: level kernel on the FP64 tensor pipe, matrices staged by TMA in
                                 fragment order (few patterns and K <= 32: a depth-first walk instead).  Other K: generic.
                                 1 force the generic shared-memory level kernel; 2 (K == 4) the level-by-level register kernel;
                                 3 (K == 4) the depth-first walk with the 4x4 products on the FP64 tensor pipe; 5 (K == 4) round
                                 1's walk with one lane per (pattern, category); 4 / 6 (32 < K <= 64) round 1's tensor-pipe level
                                 kernels (one CTA per (node, tile) looping over the categories / a cluster of one CTA per
                                 category).  2-6 are kept for comparison */
    EPX_OPT_EXP_METHOD = 4,   /* a3 method.  1 spectral: Jacobi eigensystem (reversible) / Pade 13 (asymmetric), absolute
                                 error ~1e-14 per entry.  2 componentwise: shifted non-negative Taylor scaling-and-squaring,
                                 every entry to a few hundred ulp RELATIVE, ~8 dense products per segment.  0 auto (default):
                                 2 for tree-mode (likelihood) contexts whose reversible Q have structural zeros (codon
                                 models: entries of P that vanish like t^2, t^3 decide the likelihood of short branches),
                                 else 1.  This one DOES change results, within the tolerances above (A21). */
    EPX_OPT_STAGE_EVENTS = 5, /* 1 record per-stage CUDA events for epx_get_stage_ms; 0 (default) none */
    EPX_OPT_DFS_PPL = 6,      /* K == 4 depth-first pruning: site patterns per lane, 1, 2 or 4 (4: kernel 5 only); 0 (default) auto */
    EPX_OPT_DFS_PIECES = 7,   /* depth-first pruning: number of pieces the tree is cut into (independent subtrees walked by
                                 different warps + the part above them); 0 (default) auto */
    EPX_OPT_MMA_CHUNK = 8,    /* 8 < K <= 64 tensor-pipe level kernel: site patterns per CTA (rounded up to 8); 0 (default) auto */
    EPX_OPT_JACOBI_KERNEL = 9, /* a2: 0 (default) auto: K == 4 one warp per process (everything in registers); 32 < K <= 62 a
                                 thread-block cluster of 4 CTAs per process (S in one CTA, V's rows in the three others, rotations
                                 streamed through distributed shared memory); otherwise one CTA per process with one barrier per
                                 round.  2 one CTA per process for any K <= 62; 14 / 18 clusters of 4 / 8 CTAs (16 <= K <= 62);
                                 1 round 1's two-barrier kernel.  All meet the same bounds; their bits differ */
    EPX_OPT_SHARE_PROCESSES = 10, /* 1 (default) one eigensystem / full-epoch exponential per distinct process (epx_epoch_processes);
                                 0 one per epoch */
    EPX_OPT_EPOCH_PRODUCTS = 11 /* SURVEY.md 8(f) f1.  0 (default): every branch multiplies its whole chain, one product per
                                 segment.  1 (reversible models with 32 < K <= 64, M >= 4, no branch rates): the products of
                                 consecutive full epochs, D_a W_a ... D_b W_b per category, are tabulated once per call
                                 ((M-2)(M-1)/2 C matrices) and a branch that crosses >= 2 full epochs does 3 products
                                 whatever its length.  Same P within rounding (the association order changes) */
};
int epx_set_option(epx_ctx* ctx, int option, int value);
/* Device status word of the last compute call (0 = all numeric checks passed); synchronises. */
int epx_status(epx_ctx* ctx, int* status);
/* Whole CSR segment list of the last compute call: seg_off[n_slots+1], epoch/dur with capacity `cap` entries. */
int epx_get_all_segments(epx_ctx* ctx, int32_t* seg_off, int32_t* epoch, double* dur, int cap);
/* Number of post-order levels of the tree (= pruning launches per likelihood call of the level kernels). */
int epx_tree_levels(const epx_ctx* ctx, int* n_levels);
/* Shape of the pruning plan of the current tree (host integers; tree mode, after epx_set_tree; EPX_E_STATE otherwise):
 * info[0] post-order levels; [1] pruning operations (internal nodes); [2] 1 if this ctx prunes with a depth-first walk
 * (pieces of the tree walked by independent warps), 0 if level by level; [3] bottom pieces (independent subtrees, one
 * launch); [4] operations of the largest bottom piece; [5] operations above the bottom pieces that depend on each other:
 * the top piece (second launch; 0 = none), or, when a deep tree is cut into several tiers of pieces (few-pattern walk: level
 * bands, one launch per tier), the sum over the higher tiers of their largest piece; [6] stack slots a walk needs;
 * [7] pruning kernel launches per full evaluation.  [4] + [5] is the dependent-operation chain that bounds the walk when
 * there are few site patterns (PAPER.md L224 workload A, config 4). */
int epx_plan_info(const epx_ctx* ctx, int32_t info[8]);

#ifdef __cplusplus
}
#endif
#endif /* EPX_H */
