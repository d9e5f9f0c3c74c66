/*
 * CPU ORACLE for the epoch substitution model hot path  --  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load
 * or call this file.  It shares no code, header, table or helper with the CUDA product under
 * paper_1309_3075_b200/ and neither includes the other.
 *
 * It is the plain definition of what the path computes, written out slowly, in the paper's order:
 *   O2  segmentation of a branch at the epoch boundaries       PAPER.md:L78 (change-point process), L117 (weights)
 *   O3  exp(A) by its power series, scaled and squared          PAPER.md:L48  P(t)=exp(tQ)=sum_j (tQ)^j/j!
 *   O3' exp(Qt) by uniformisation (second, independent method)  same definition, all terms non-negative
 *   O4  ordered chain product, parent end first                 PAPER.md:L92-L106 Eq.(5)-(7) (reading A2 in DESIGN.md)
 *   O5  Felsenstein pruning by naive recursion, no rescaling    PAPER.md:L64-L72 Eq.(4)
 *   O6  root / site / category aggregation
 * None of it is an approximation scheme of its own: P and logL are unique real numbers and every routine
 * here converges to them to rounding.  Compiled twice from this one source:
 *   -DORC_LONG_DOUBLE : REAL = 80-bit long double (64-bit mantissa)  -> the parity referee
 *   (default)         : REAL = double                                -> the timed CPU baseline ("as it stands")
 *   -DORC_QUAD        : REAL = __float128 (113-bit mantissa)         -> pins the referee's own rounding, nothing else
 * Pins (tests/test_oracle_pins.py): JC69 closed form, K-state equal-input multi-epoch closed form (fixes the
 * product ORDER), row sums, homogeneous collapse, redundant boundaries, scipy.linalg.expm, Taylor vs
 * uniformisation, detailed balance / stationarity, brute-force enumeration of ancestral states, two-tip
 * closed form, all-missing tips, pattern-weight and category invariances; the root-epoch rule of reading A9
 * (orc_epoch_of_parent_end) by hand-stated epochs -- inside an epoch, above the last boundary, exactly on a
 * boundary -- and by two-tip likelihoods evaluated with the frequencies of the epoch named by hand.  Nothing is
 * "parity unpinned".
 *
 * Height convention: time runs backwards from the most recent tip; epoch e (0 = most recent) covers heights
 * [tau[e-1], tau[e]) with tau[-1] = -inf and tau[M-1] = +inf; `tau` holds the M-1 finite boundaries.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <float.h>

#if defined(ORC_QUAD)
/* Third build, same source: REAL = IEEE binary128 (113-bit mantissa, libquadmath).  It exists for ONE pin (last
 * row of the pin table; the series definition of exp at PAPER.md:L48): the long-double referee's own rounding error, measured
 * against 49 more bits, must sit far inside the 1e-12 / 1e-9 parity gates.  Not used by any parity test or bench leg. */
#include <quadmath.h>
typedef __float128 REAL;
#define R_EPS FLT128_EPSILON
#define R_LOG logq
#define R_EXP expq
#define R_FABS fabsq
#define R_LDEXP ldexpq
#elif defined(ORC_LONG_DOUBLE)
typedef long double REAL;
#define R_EPS LDBL_EPSILON
#define R_LOG logl
#define R_EXP expl
#define R_FABS fabsl
#define R_LDEXP ldexpl
#else
typedef double REAL;
#define R_EPS DBL_EPSILON
#define R_LOG log
#define R_EXP exp
#define R_FABS fabs
#define R_LDEXP ldexp
#endif

int orc_real_bytes(void) { return (int)sizeof(REAL); }
/* REAL -> long double, element by element (a rounding for the binary128 build, a copy or a widening otherwise): how the
 * Python front-end reads results of a build whose REAL numpy cannot represent.  No arithmetic of the method. */
void orc_real_to_ld(size_t n, const REAL *in, long double *out) { for (size_t i = 0; i < n; i++) out[i] = (long double)in[i]; }

/* ---------------------------------------------------------------- O2: segmentation */
/* Walk the boundaries linearly from the parent height down to the child height. Emits (epoch, duration) with
 * duration > 0 only, parent end first (so epochs strictly decrease by 1). Returns the number of segments
 * written, or -1 if `cap` is too small. Zero-length branch => 0 segments (P = I). */
static int segment_one(double h_child, double h_parent, int M, const double *tau, int *epoch, double *dur, int cap)
{
    int e = M - 1, n = 0;
    while (e > 0 && tau[e - 1] >= h_parent) e--;          /* epoch holding the parent end: #{k: tau_k < h_parent} */
    double upper = h_parent;
    for (;;) {
        int last = (e == 0) || (tau[e - 1] <= h_child);   /* child end lies in this epoch */
        double lower = last ? h_child : tau[e - 1];
        REAL d = (REAL)upper - (REAL)lower;
        if (d > 0) {
            if (n >= cap) return -1;
            epoch[n] = e;
            dur[n] = (double)d;
            n++;
        }
        if (last) break;
        upper = tau[e - 1];
        e--;
    }
    return n;
}

int orc_segments(int n_br, const double *child_h, const double *parent_h, int M, const double *tau,
                 int *seg_off, int *seg_epoch, double *seg_dur, int cap)
{
    int total = 0;
    seg_off[0] = 0;
    for (int b = 0; b < n_br; b++) {
        int n = segment_one(child_h[b], parent_h[b], M, tau, seg_epoch + total, seg_dur + total, cap - total);
        if (n < 0) return -1;
        total += n;
        seg_off[b + 1] = total;
    }
    return total;
}

/* epoch containing the root: #{k : tau_k < h_root}  (reading A9: the parent-end rule of A3, so a root exactly on a
 * boundary takes the YOUNGER epoch -- everything below it evolved under that process).  Pinned by
 * tests/test_oracle_pins.py::test_root_epoch_selection_hand_stated and ::test_two_tip_likelihood_uses_the_root_epochs_frequencies. */
int orc_epoch_of_parent_end(double h, int M, const double *tau)
{
    int e = 0;
    for (int k = 0; k < M - 1; k++) if (tau[k] < h) e++;
    return e;
}

/* ---------------------------------------------------------------- dense helpers: naive triple loop */
static void matmul(int K, const REAL *A, const REAL *B, REAL *C)
{
    for (int i = 0; i < K; i++)
        for (int j = 0; j < K; j++) {
            REAL s = 0;
            for (int k = 0; k < K; k++) s += A[i * K + k] * B[k * K + j];
            C[i * K + j] = s;
        }
}

static REAL norm_inf(int K, const REAL *A)
{
    REAL m = 0;
    for (int i = 0; i < K; i++) {
        REAL s = 0;
        for (int j = 0; j < K; j++) s += R_FABS(A[i * K + j]);
        if (s > m) m = s;
    }
    return m;
}

/* ---------------------------------------------------------------- O3: exp(A) = sum_j A^j / j! */
/* A is scaled by 2^-s so that ||A/2^s||_inf <= 1/2, the series is summed term by term until the term's
 * inf-norm drops below eps/64, and the result is squared s times (exp(A) = exp(A/2^s)^(2^s)). */
void orc_expm_taylor(int K, const REAL *A, REAL *out)
{
    size_t n = (size_t)K * K;
    REAL *S = malloc(n * sizeof(REAL)), *T = malloc(n * sizeof(REAL)), *U = malloc(n * sizeof(REAL));
    REAL nrm = norm_inf(K, A);
    int s = 0;
    while (R_LDEXP(nrm, -s) > (REAL)0.5) s++;
    for (size_t i = 0; i < n; i++) S[i] = R_LDEXP(A[i], -s);
    for (size_t i = 0; i < n; i++) { out[i] = 0; T[i] = 0; }
    for (int i = 0; i < K; i++) { out[i * K + i] = 1; T[i * K + i] = 1; }   /* j = 0 term: I */
    for (int j = 1; j < 200; j++) {
        matmul(K, T, S, U);                                               /* T <- T * S / j  = S^j / j! */
        for (size_t i = 0; i < n; i++) { T[i] = U[i] / (REAL)j; out[i] += T[i]; }
        if (norm_inf(K, T) < R_EPS / 64) break;
    }
    for (int q = 0; q < s; q++) {
        matmul(K, out, out, U);
        memcpy(out, U, n * sizeof(REAL));
    }
    free(S); free(T); free(U);
}

/* ---------------------------------------------------------------- O3': uniformisation */
/* exp(A) for a rate matrix A (non-negative off-diagonal, rows sum to 0): with mu = max_i |a_ii| and the
 * stochastic matrix R = I + A/mu,  exp(A) = sum_n e^{-mu} mu^n / n! * R^n.  Every term is non-negative.
 * Returns the number of terms used, or -1 if it did not converge in `max_terms`. */
int orc_expm_uniformisation(int K, const REAL *A, REAL *out, int max_terms)
{
    size_t n = (size_t)K * K;
    REAL mu = 0;
    for (int i = 0; i < K; i++) if (-A[i * K + i] > mu) mu = -A[i * K + i];
    for (size_t i = 0; i < n; i++) out[i] = 0;
    if (mu == 0) { for (int i = 0; i < K; i++) out[i * K + i] = 1; return 0; }
    REAL *R = malloc(n * sizeof(REAL)), *Rn = malloc(n * sizeof(REAL)), *U = malloc(n * sizeof(REAL));
    for (size_t i = 0; i < n; i++) R[i] = A[i] / mu;
    for (int i = 0; i < K; i++) R[i * K + i] += 1;
    for (size_t i = 0; i < n; i++) Rn[i] = 0;
    for (int i = 0; i < K; i++) Rn[i * K + i] = 1;
    REAL w = R_EXP(-mu), cum = 0;
    int it = -1;
    for (int k = 0; k < max_terms; k++) {
        for (size_t i = 0; i < n; i++) out[i] += w * Rn[i];
        cum += w;
        if ((REAL)k > mu && w < R_EPS / 1024) { it = k + 1; break; }
        matmul(K, Rn, R, U);
        memcpy(Rn, U, n * sizeof(REAL));
        w = w * mu / (REAL)(k + 1);
    }
    free(R); free(Rn); free(U);
    (void)cum;
    return it;
}

/* ---------------------------------------------------------------- O3+O4: branch matrices  (Eq. 3, 5-7) */
/* P[b][c] = prod over the branch's segments, parent end first, of exp(Q[epoch] * r_c * duration).
 * A branch with no segment gets the identity. Q is given in double (the caller's bits) and widened. */
int orc_branch_matrices(int K, int M, int C, const double *Q, const double *rates, int n_br, const int *seg_off,
                        const int *seg_epoch, const double *seg_dur, REAL *P)
{
    size_t n = (size_t)K * K;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < n_br; b++) {
        REAL *A = malloc(n * sizeof(REAL)), *E = malloc(n * sizeof(REAL)), *T = malloc(n * sizeof(REAL));
        for (int c = 0; c < C; c++) {
            REAL *Pb = P + ((size_t)b * C + c) * n;
            for (size_t i = 0; i < n; i++) Pb[i] = 0;
            for (int i = 0; i < K; i++) Pb[i * K + i] = 1;
            for (int s = seg_off[b]; s < seg_off[b + 1]; s++) {
                int e = seg_epoch[s];
                if (e < 0 || e >= M) {
#pragma omp atomic write
                    bad = 1;
                    continue;
                }
                REAL scale = (REAL)rates[c] * (REAL)seg_dur[s];
                for (size_t i = 0; i < n; i++) A[i] = (REAL)Q[(size_t)e * n + i] * scale;
                orc_expm_taylor(K, A, E);
                matmul(K, Pb, E, T);                                   /* parent end is the leftmost factor */
                memcpy(Pb, T, n * sizeof(REAL));
            }
        }
        free(A); free(E); free(T);
    }
    return bad ? -1 : 0;
}

/* ---------------------------------------------------------------- O5: pruning by naive recursion (Eq. 4) */
typedef struct {
    int K, C, N, L;
    const int *left, *right;     /* children, -1 for tips */
    const REAL *P;               /* [node][C][K][K], row = parent-end state */
    const int *tips;             /* [N][L] */
    const double *tip_partials;  /* optional [N][L][K]: tip vectors of partially observed tips */
    const unsigned char *tip_has;/* optional [N]: 1 = use tip_partials for this tip */
    REAL *partials;              /* optional [node][C][L][K] */
} prune_ctx;

static void partial(const prune_ctx *x, int node, int p, int c, REAL *out)
{
    int K = x->K;
    if (x->left[node] < 0 && x->tip_has && x->tip_has[node]) {           /* partially observed tip: its given vector (L72) */
        for (int i = 0; i < K; i++) out[i] = (REAL)x->tip_partials[((size_t)node * x->L + p) * K + i];
    } else if (x->left[node] < 0) {                                      /* tip: 0/1 indicator, all-ones if missing (L72) */
        int s = x->tips[(size_t)node * x->L + p];
        for (int i = 0; i < K; i++) out[i] = (s >= 0 && s < K) ? (i == s ? 1 : 0) : 1;
    } else {
        int v = x->left[node], w = x->right[node];
        REAL *Lv = malloc(2 * (size_t)K * sizeof(REAL)), *Lw = Lv + K;
        partial(x, v, p, c, Lv);
        partial(x, w, p, c, Lw);
        const REAL *Pv = x->P + ((size_t)v * x->C + c) * K * K;
        const REAL *Pw = x->P + ((size_t)w * x->C + c) * K * K;
        for (int i = 0; i < K; i++) {
            REAL a = 0, b = 0;
            for (int j = 0; j < K; j++) a += Pv[i * K + j] * Lv[j];
            for (int k = 0; k < K; k++) b += Pw[i * K + k] * Lw[k];
            out[i] = a * b;
        }
        free(Lv);
    }
    if (x->partials)
        memcpy(x->partials + (((size_t)node * x->C + c) * x->L + p) * K, out, (size_t)K * sizeof(REAL));
}

/* ---------------------------------------------------------------- O6: root, sites, categories (L72) */
/* site_lnl[p] = ln sum_c w_c sum_i pi_i L_root,c,p(i);  *lnl = sum_p wt_p site_lnl[p]  (Kahan-summed).
 * Returns 0, -2 for a malformed tree, -3 if some site likelihood is not a positive normal number. */
int orc_log_likelihood_tp(int K, int C, int N, int L, const int *parent, const REAL *P, const int *tips,
                          const double *root_freqs, const double *cat_weights, const double *pattern_wt,
                          REAL *site_lnl, REAL *lnl, REAL *partials, const double *tip_partials,
                          const unsigned char *tip_has);

int orc_log_likelihood(int K, int C, int N, int L, const int *parent, const REAL *P, const int *tips,
                       const double *root_freqs, const double *cat_weights, const double *pattern_wt,
                       REAL *site_lnl, REAL *lnl, REAL *partials)
{
    return orc_log_likelihood_tp(K, C, N, L, parent, P, tips, root_freqs, cat_weights, pattern_wt, site_lnl, lnl, partials,
                                 NULL, NULL);
}

/* The same with tip vectors for some tips: tip_has[t] = 1 => tip t's partial likelihoods are tip_partials[t][p][0..K-1]
 * ("0 or 1 depending on whether trait i is (partially) observed") instead of the indicator of its state. */
int orc_log_likelihood_tp(int K, int C, int N, int L, const int *parent, const REAL *P, const int *tips,
                          const double *root_freqs, const double *cat_weights, const double *pattern_wt,
                          REAL *site_lnl, REAL *lnl, REAL *partials, const double *tip_partials,
                          const unsigned char *tip_has)
{
    int n_nodes = 2 * N - 1, root = -1;
    int *left = malloc(sizeof(int) * n_nodes), *right = malloc(sizeof(int) * n_nodes);
    for (int i = 0; i < n_nodes; i++) left[i] = right[i] = -1;
    int ok = 1;
    for (int i = 0; i < n_nodes; i++) {
        int p = parent[i];
        if (p < 0) { if (root >= 0) ok = 0; root = i; continue; }
        if (p >= n_nodes || p < N) { ok = 0; continue; }
        if (left[p] < 0) left[p] = i; else if (right[p] < 0) right[p] = i; else ok = 0;
    }
    for (int i = N; i < n_nodes && ok; i++) if (left[i] < 0 || right[i] < 0) ok = 0;
    if (!ok || root < 0) { free(left); free(right); return -2; }

    prune_ctx x = { K, C, N, L, left, right, P, tips, tip_partials, tip_has, partials };
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 8)
    for (int p = 0; p < L; p++) {
        REAL *Lr = malloc((size_t)K * sizeof(REAL));
        REAL site = 0;
        for (int c = 0; c < C; c++) {
            partial(&x, root, p, c, Lr);
            REAL s = 0;
            for (int i = 0; i < K; i++) s += (REAL)root_freqs[i] * Lr[i];
            site += (REAL)cat_weights[c] * s;
        }
        free(Lr);
#ifdef ORC_LONG_DOUBLE
        if (!(site >= LDBL_MIN) || site != site) {        /* not a positive normal number */
#else
        if (!(site >= DBL_MIN) || site != site) {
#endif
#pragma omp atomic write
            bad = 1;
        }
        site_lnl[p] = R_LOG(site);
    }
    REAL sum = 0, comp = 0;                                              /* Kahan */
    for (int p = 0; p < L; p++) {
        REAL y = (REAL)(pattern_wt ? pattern_wt[p] : 1.0) * site_lnl[p] - comp;
        REAL t = sum + y;
        comp = (t - sum) - y;
        sum = t;
    }
    *lnl = sum;
    free(left); free(right);
    return bad ? -3 : 0;
}

/* ---------------------------------------------------------------- O1: the validation rules */
/* 0 ok; -4: a row of Q does not sum to 0, a negative off-diagonal, freqs not a distribution, or (reversible)
 * detailed balance pi_i q_ij = pi_j q_ji violated / some pi_i <= 0. */
int orc_validate_model(int K, const double *Q, const double *freqs, int reversible)
{
    REAL maxdiag = 0, maxflux = 0, fs = 0;
    for (int i = 0; i < K; i++) if (R_FABS((REAL)Q[i * K + i]) > maxdiag) maxdiag = R_FABS((REAL)Q[i * K + i]);
    for (int i = 0; i < K; i++) {
        REAL s = 0;
        for (int j = 0; j < K; j++) {
            if (!isfinite(Q[i * K + j])) return -4;
            s += (REAL)Q[i * K + j];
            if (i != j && Q[i * K + j] < 0) return -4;
        }
        if (R_FABS(s) > (REAL)1e-9 * maxdiag) return -4;
        if (!(freqs[i] >= 0)) return -4;
        fs += (REAL)freqs[i];
    }
    if (R_FABS(fs - 1) > (REAL)1e-9) return -4;
    if (reversible) {
        for (int i = 0; i < K; i++) {
            if (!(freqs[i] > 0)) return -4;
            for (int j = 0; j < K; j++) {
                REAL f = (REAL)freqs[i] * (REAL)Q[i * K + j];
                if (i != j && f > maxflux) maxflux = f;
            }
        }
        for (int i = 0; i < K; i++)
            for (int j = i + 1; j < K; j++)
                if (R_FABS((REAL)freqs[i] * Q[i * K + j] - (REAL)freqs[j] * Q[j * K + i]) > (REAL)1e-9 * maxflux) return -4;
    }
    return 0;
}

/* 0 ok; -3: not a strictly bifurcating rooted tree with tips 0..N-1, or a child above its parent. */
int orc_validate_tree(int N, const int *parent, const double *height)
{
    int n_nodes = 2 * N - 1, roots = 0;
    if (N < 2) return -3;
    int *deg = calloc(n_nodes, sizeof(int));
    int ok = 1;
    for (int i = 0; i < n_nodes && ok; i++) {
        int p = parent[i];
        if (!isfinite(height[i])) ok = 0;
        if (p < 0) { roots++; continue; }
        if (p >= n_nodes || p < N || p == i) { ok = 0; break; }
        if (height[p] < height[i]) ok = 0;
        deg[p]++;
    }
    if (roots != 1) ok = 0;
    for (int i = 0; i < n_nodes && ok; i++) if (deg[i] != (i < N ? 0 : 2)) ok = 0;
    /* acyclic: walking up from every node must reach the root in < n_nodes steps */
    for (int i = 0; i < n_nodes && ok; i++) {
        int u = i, steps = 0;
        while (parent[u] >= 0 && steps <= n_nodes) { u = parent[u]; steps++; }
        if (steps > n_nodes) ok = 0;
    }
    free(deg);
    return ok ? 0 : -3;
}
