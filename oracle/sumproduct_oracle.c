/*
 * ORACLE -- test infrastructure, NOT product code.
 *
 * A plain, slow, obviously-correct CPU implementation of what the hot path computes: flooding-schedule
 * Sum-Product belief-propagation decoding (Algorithm 1, "P:340-367") of a
 * quasi-cyclic LDPC code (lifting rule P:324) in the syndrome form H x = s named by BASELINE.json's north_star.
 * With s = 0 it is exactly the paper's Algorithm 1.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this library.
 * It shares no code, header, table or constant with the CUDA path (paper_1702_07740_b200/csrc/) and neither
 * includes the other.
 *
 * What it does, in the paper's order and notation, on the EXPLICIT sparse H (no use of the circulant structure
 * beyond building H, no blocking, no fusion, no reordering):
 *   Step 1      Q_v = llr[v] (fp32 input widened exactly);  L_vc <- Q_v on every edge.
 *   for t = 1..max_iter
 *     Step 2 for every check c and every v in N(c), by DIRECT EXCLUSION over v' in N(c)\v:
 *                          S = sum Phi(|L_v'c|),  sgn = (-1)^{s_c} * prod sgn(L_v'c),
 *                          m_cv = sgn * min(Phi(S), msg_max),   Phi(x) = -ln tanh(x/2) = log1p(2/expm1(x))
 *     Step 3 L_v  = Q_v + sum_{c in M(v)} m_cv            (stored edge order = increasing check index)
 *                        L_vc = Q_v + sum_{c' in M(v)\c} m_c'v         (direct exclusion, same order)
 *     Step 4 xhat_v = 0 if L_v >= 0 else 1;  if early_stop and H xhat = s (mod 2): iters = t, stop.
 *   Step 5 is the identity in syndrome form (no parity bits are discarded; P:367 is caller-side slicing).
 * Readings where the paper is silent (DESIGN.md §"Readings"): S1 syndrome sign, S2 msg_max clamp on |m_cv| only
 * (default 30.0), S3 sgn(x) = -1 iff x < 0 (so -0.0 and +0.0 are +), S4 tie L_v = 0 -> bit 0, S5 check every
 * iteration, S6 iters = first passing t else max_iter, S7 outputs of the last executed iteration, S9 H is m x n with
 * rows = checks, S10 shift p: check R*Z+r -- variable C*Z+((r+p) mod Z).
 *
 * Pins (tests/, -m "not gpu"): brute-force bitwise MAP on cycle-free codes (n <= 20), closed forms of degree-2/3
 * checks, Phi values and involution, syndrome<->codeword equivalence, syndrome invariant against an independent
 * dense mat-vec, noiseless limit, degree-1 invariant, lifting rule against np.roll of the identity, frame
 * independence.  See tests/test_oracle_pins.py.
 *
 * The arithmetic type is `double` (the definition).  A `float` instantiation of the same text exists as a
 * DIAGNOSTIC only (it shows the fp32 rounding-noise floor next to "GPU vs oracle64").
 */
#include <math.h>
#include <omp.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------------------------ */
/* Explicit sparse H from (base_shifts, Z), by the printed lifting rule.                                 */
/* ------------------------------------------------------------------------------------------------------------ */
typedef struct {
    int64_t n, m, E;
    int64_t *row_ptr;   /* [m+1]  edges of check c are row_ptr[c] .. row_ptr[c+1]-1, variables increasing in C   */
    int64_t *edge_var;  /* [E]    variable of edge e                                                            */
    int64_t *col_ptr;   /* [n+1]  edges of variable v, in increasing check index                                 */
    int64_t *col_edge;  /* [E]    edge ids                                                                       */
} sparse_h;

static void free_h(sparse_h *h) {
    free(h->row_ptr); free(h->edge_var); free(h->col_ptr); free(h->col_edge);
}

static int build_h(const int32_t *base, int mb, int nb, int Z, sparse_h *h) {
    memset(h, 0, sizeof(*h));
    h->n = (int64_t)nb * Z;
    h->m = (int64_t)mb * Z;
    int64_t nnz_base = 0;
    for (int i = 0; i < mb * nb; ++i) {
        if (base[i] < -1 || base[i] >= Z) return -1;
        if (base[i] >= 0) ++nnz_base;
    }
    h->E = nnz_base * Z;
    h->row_ptr = calloc((size_t)h->m + 1, sizeof(int64_t));
    h->edge_var = calloc((size_t)h->E + 1, sizeof(int64_t));
    h->col_ptr = calloc((size_t)h->n + 1, sizeof(int64_t));
    h->col_edge = calloc((size_t)h->E + 1, sizeof(int64_t));
    if (!h->row_ptr || !h->edge_var || !h->col_ptr || !h->col_edge) { free_h(h); return -2; }
    /* rows: check c = R*Z + r is connected, for every non-zero block (R,C) with shift p, to v = C*Z + (r+p) mod Z */
    int64_t e = 0;
    for (int R = 0; R < mb; ++R)
        for (int r = 0; r < Z; ++r) {
            h->row_ptr[(int64_t)R * Z + r] = e;
            for (int C = 0; C < nb; ++C) {
                int p = base[R * nb + C];
                if (p >= 0) h->edge_var[e++] = (int64_t)C * Z + (r + p) % Z;
            }
        }
    h->row_ptr[h->m] = e;
    /* columns: counting sort of the edges by variable; scanning edges in increasing e keeps checks increasing */
    for (int64_t k = 0; k < h->E; ++k) h->col_ptr[h->edge_var[k] + 1]++;
    for (int64_t v = 0; v < h->n; ++v) h->col_ptr[v + 1] += h->col_ptr[v];
    int64_t *fill = calloc((size_t)h->n + 1, sizeof(int64_t));
    if (!fill) { free_h(h); return -2; }
    for (int64_t k = 0; k < h->E; ++k) {
        int64_t v = h->edge_var[k];
        h->col_edge[h->col_ptr[v] + fill[v]++] = k;
    }
    free(fill);
    return 0;
}

/* The same H from the non-zero blocks only: block (brow[k], bcol[k]) = identity shifted right by bshift[k].
 * Entries may come in any order; inside a check the edges are stored by increasing base column, as in build_h.
 * A repeated (row, col) pair is rejected (a block is one circulant). */
typedef struct { int32_t r, c, p; } base_entry;
static int cmp_entry(const void *a, const void *b) {
    const base_entry *x = a, *y = b;
    if (x->r != y->r) return x->r < y->r ? -1 : 1;
    if (x->c != y->c) return x->c < y->c ? -1 : 1;
    return 0;
}
static int build_h_sparse(const int32_t *brow, const int32_t *bcol, const int32_t *bshift, int64_t nnz_base,
                          int mb, int nb, int Z, sparse_h *h) {
    memset(h, 0, sizeof(*h));
    h->n = (int64_t)nb * Z;
    h->m = (int64_t)mb * Z;
    h->E = nnz_base * Z;
    base_entry *ent = malloc(sizeof(base_entry) * (size_t)(nnz_base + 1));
    int64_t *first = calloc((size_t)mb + 1, sizeof(int64_t));      /* entries of base row R: first[R] .. first[R+1]-1 */
    if (!ent || !first) { free(ent); free(first); return -2; }
    for (int64_t k = 0; k < nnz_base; ++k) {
        if (brow[k] < 0 || brow[k] >= mb || bcol[k] < 0 || bcol[k] >= nb || bshift[k] < 0 || bshift[k] >= Z) {
            free(ent); free(first); return -1;
        }
        ent[k].r = brow[k]; ent[k].c = bcol[k]; ent[k].p = bshift[k];
    }
    qsort(ent, (size_t)nnz_base, sizeof(base_entry), cmp_entry);
    for (int64_t k = 1; k < nnz_base; ++k)
        if (ent[k].r == ent[k - 1].r && ent[k].c == ent[k - 1].c) { free(ent); free(first); return -1; }
    for (int64_t k = 0; k < nnz_base; ++k) first[ent[k].r + 1]++;
    for (int R = 0; R < mb; ++R) first[R + 1] += first[R];
    h->row_ptr = calloc((size_t)h->m + 1, sizeof(int64_t));
    h->edge_var = calloc((size_t)h->E + 1, sizeof(int64_t));
    h->col_ptr = calloc((size_t)h->n + 1, sizeof(int64_t));
    h->col_edge = calloc((size_t)h->E + 1, sizeof(int64_t));
    int64_t *fill = calloc((size_t)h->n + 1, sizeof(int64_t));
    if (!h->row_ptr || !h->edge_var || !h->col_ptr || !h->col_edge || !fill) {
        free_h(h); free(ent); free(first); free(fill); return -2;
    }
    int64_t e = 0;
    for (int R = 0; R < mb; ++R)
        for (int r = 0; r < Z; ++r) {
            h->row_ptr[(int64_t)R * Z + r] = e;
            for (int64_t k = first[R]; k < first[R + 1]; ++k)
                h->edge_var[e++] = (int64_t)ent[k].c * Z + (r + ent[k].p) % Z;
        }
    h->row_ptr[h->m] = e;
    for (int64_t k = 0; k < h->E; ++k) h->col_ptr[h->edge_var[k] + 1]++;
    for (int64_t v = 0; v < h->n; ++v) h->col_ptr[v + 1] += h->col_ptr[v];
    for (int64_t k = 0; k < h->E; ++k) {
        int64_t v = h->edge_var[k];
        h->col_edge[h->col_ptr[v] + fill[v]++] = k;
    }
    free(fill); free(ent); free(first);
    return 0;
}

/* COO dump of H for the lifting-rule pin (P9). rows/cols have room for nnz_base*Z entries. Returns E or <0. */
int64_t oracle_build_h_coo(const int32_t *base, int mb, int nb, int Z, int64_t *rows, int64_t *cols) {
    sparse_h h;
    if (build_h(base, mb, nb, Z, &h) != 0) return -1;
    for (int64_t c = 0; c < h.m; ++c)
        for (int64_t e = h.row_ptr[c]; e < h.row_ptr[c + 1]; ++e) { rows[e] = c; cols[e] = h.edge_var[e]; }
    int64_t E = h.E;
    free_h(&h);
    return E;
}

/* H xhat = s (mod 2)?  (P:363 generalised to a syndrome, S1) */
static int syndrome_ok(const sparse_h *h, const uint8_t *xhat, const uint8_t *s) {
    for (int64_t c = 0; c < h->m; ++c) {
        int parity = 0;
        for (int64_t e = h->row_ptr[c]; e < h->row_ptr[c + 1]; ++e) parity ^= xhat[h->edge_var[e]] & 1;
        if (parity != (s[c] & 1)) return 0;
    }
    return 1;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* Algorithm 1, instantiated for double (the definition) and float (diagnostic).                                 */
/* ------------------------------------------------------------------------------------------------------------ */
#define REAL double
#define PHI(x) log1p(2.0 / expm1(x))
#define FABS(x) fabs(x)
#define DECODE_FRAME decode_frame_f64
#include "sumproduct_core.inc"
#undef REAL
#undef PHI
#undef FABS
#undef DECODE_FRAME

#define REAL float
#define PHI(x) log1pf(2.0f / expm1f(x))
#define FABS(x) fabsf(x)
#define DECODE_FRAME decode_frame_f32
#include "sumproduct_core.inc"
#undef REAL
#undef PHI
#undef FABS
#undef DECODE_FRAME

double oracle_phi(double x) { return log1p(2.0 / expm1(x)); }

/*
 * All pointers are HOST pointers, frame-major contiguous:
 *   llr float[n_frames][n], syndrome uint8[n_frames][m], hard uint8[n_frames][n], iters int32[n_frames],
 *   pass uint8[n_frames], posterior double[n_frames][n] (may be NULL),
 *   msg_cv double[n_frames][E] (may be NULL): the CN->VN messages m_cv of the last executed iteration in
 *   check-major edge order (the order of oracle_build_h_coo).
 * precision: 64 = double (definition), 32 = float diagnostic (outputs still widened to double).
 * check_from: the early-termination test (early_stop != 0) runs at iterations t >= check_from only (the
 * paper enables it after the expected iteration count); 1 = every iteration.
 * Frames are independent and run one per OpenMP thread (n_threads <= 0: the OpenMP default).  Returns 0, or <0 on bad arguments / allocation failure.
 */
static int decode_frames(sparse_h *hp, const float *llr, const uint8_t *syndrome, int n_frames, int max_iter,
                         int early_stop, int check_from, double msg_max, int precision, int n_threads,
                         uint8_t *hard, int32_t *iters, uint8_t *pass, double *posterior, double *msg_cv);

int oracle_decode_from(const int32_t *base, int mb, int nb, int Z,
                       const float *llr, const uint8_t *syndrome, int n_frames, int max_iter, int early_stop,
                       int check_from, double msg_max, int precision, int n_threads,
                       uint8_t *hard, int32_t *iters, uint8_t *pass, double *posterior, double *msg_cv) {
    if (!base || !llr || !syndrome || !hard || !iters || !pass) return -1;
    if (mb <= 0 || nb <= 0 || Z <= 0 || n_frames < 0 || max_iter < 0) return -1;
    if (precision != 64 && precision != 32) return -1;
    sparse_h h;
    int rc = build_h(base, mb, nb, Z, &h);
    if (rc != 0) return rc;
    return decode_frames(&h, llr, syndrome, n_frames, max_iter, early_stop, check_from, msg_max, precision, n_threads,
                         hard, iters, pass, posterior, msg_cv);
}

/* The same decode with H given by its non-zero blocks (build_h_sparse). */
int oracle_decode_sparse(const int32_t *brow, const int32_t *bcol, const int32_t *bshift, int64_t nnz_base,
                         int mb, int nb, int Z,
                         const float *llr, const uint8_t *syndrome, int n_frames, int max_iter, int early_stop,
                         int check_from, double msg_max, int precision, int n_threads,
                         uint8_t *hard, int32_t *iters, uint8_t *pass, double *posterior, double *msg_cv) {
    if (!llr || !syndrome || !hard || !iters || !pass || nnz_base < 0) return -1;
    if (nnz_base > 0 && (!brow || !bcol || !bshift)) return -1;
    if (mb <= 0 || nb <= 0 || Z <= 0 || n_frames < 0 || max_iter < 0) return -1;
    if (precision != 64 && precision != 32) return -1;
    sparse_h h;
    int rc = build_h_sparse(brow, bcol, bshift, nnz_base, mb, nb, Z, &h);
    if (rc != 0) return rc;
    return decode_frames(&h, llr, syndrome, n_frames, max_iter, early_stop, check_from, msg_max, precision, n_threads,
                         hard, iters, pass, posterior, msg_cv);
}

/* s = H x (mod 2) for n_frames words with H given by its non-zero blocks: an independent product for the harness of
 * large base graphs (x uint8 [n_frames][n] -> s uint8 [n_frames][m]). */
int oracle_syndrome_sparse(const int32_t *brow, const int32_t *bcol, const int32_t *bshift, int64_t nnz_base,
                           int mb, int nb, int Z, const uint8_t *x, int n_frames, uint8_t *s) {
    if (!x || !s || mb <= 0 || nb <= 0 || Z <= 0 || n_frames < 0 || nnz_base < 0) return -1;
    const int64_t n = (int64_t)nb * Z, m = (int64_t)mb * Z;
    memset(s, 0, (size_t)(m * n_frames));
    for (int64_t k = 0; k < nnz_base; ++k) {
        if (brow[k] < 0 || brow[k] >= mb || bcol[k] < 0 || bcol[k] >= nb || bshift[k] < 0 || bshift[k] >= Z) return -1;
        for (int f = 0; f < n_frames; ++f)
            for (int r = 0; r < Z; ++r)
                s[f * m + (int64_t)brow[k] * Z + r] ^= x[f * n + (int64_t)bcol[k] * Z + (r + bshift[k]) % Z] & 1;
    }
    return 0;
}

static int decode_frames(sparse_h *hp, const float *llr, const uint8_t *syndrome, int n_frames, int max_iter,
                         int early_stop, int check_from, double msg_max, int precision, int n_threads,
                         uint8_t *hard, int32_t *iters, uint8_t *pass, double *posterior, double *msg_cv) {
    sparse_h h = *hp;
    int fail = 0;
    const int nt = n_threads > 0 ? n_threads : omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
    for (int f = 0; f < n_frames; ++f) {
        const float *q = llr + (int64_t)f * h.n;
        const uint8_t *s = syndrome + (int64_t)f * h.m;
        double *post = posterior ? posterior + (int64_t)f * h.n : NULL;
        double *mo = msg_cv ? msg_cv + (int64_t)f * h.E : NULL;
        int r = (precision == 64)
            ? decode_frame_f64(&h, q, s, max_iter, early_stop, check_from, msg_max, hard + (int64_t)f * h.n, iters + f, pass + f, post, mo)
            : decode_frame_f32(&h, q, s, max_iter, early_stop, check_from, msg_max, hard + (int64_t)f * h.n, iters + f, pass + f, post, mo);
        if (r != 0) {
#pragma omp atomic write
            fail = 1;
        }
    }
    free_h(&h);
    return fail ? -2 : 0;
}

/* The early-termination test at every iteration (reading S5). */
int oracle_decode(const int32_t *base, int mb, int nb, int Z,
                  const float *llr, const uint8_t *syndrome, int n_frames, int max_iter, int early_stop,
                  double msg_max, int precision, int n_threads,
                  uint8_t *hard, int32_t *iters, uint8_t *pass, double *posterior, double *msg_cv) {
    return oracle_decode_from(base, mb, nb, Z, llr, syndrome, n_frames, max_iter, early_stop, 1, msg_max, precision,
                              n_threads, hard, iters, pass, posterior, msg_cv);
}
