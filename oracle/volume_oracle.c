/* Volume oracle: the same definitions as oracle/kripke_oracle.py, in plain C, for the sizes the
 * Python oracle cannot reach.  TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may load it.  It shares no source, header, table
 * or helper with paper_2606_15437_b200/ (the CUDA path).
 *
 * It is deliberately plain: a world set is an array of n bytes (0/1), a relation is an n x n byte
 * matrix, a valuation is one byte array per variable.  No truth set is ever packed into an integer
 * and no connective is a bit operation; bits are read only to decode the indices f and v.
 *   - satisfaction of each connective: PAPER.md:38-40 (section 2), evaluated bottom-up in the order
 *     of the postfix program (each subformula's truth array is computed once per model);
 *   - box: true at w iff every u with R[w][u] has x[u];  dia: some u with R[w][u] has x[u];
 *   - refuted iff the truth array is not all ones;
 *   - classes by first-order definitions; enumeration order = ascending f;
 *   - outputs: Algorithm 1's FAIL / FIRST under DESIGN.md readings R6-R8:
 *     refuting (frame, valuation) models, refuting frames, lexicographically first (f, v) and the
 *     least falsifying world;
 *   - pair path: worlds where exactly one of phi, psi holds.
 * Index conventions (readings R2, R3): R[w][u] = bit (w*n+u) of f; V_i[w] = bit (i*n+w) of v.
 * Pinned by tests/test_oracle_pins.py against closed forms and against the Python oracle.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MAXN 6
#define MAXVARS 4
#define MAXDEPTH 64
#define NO_WITNESS UINT64_MAX

enum { OP_TOP = 0x00, OP_BOT = 0x01, OP_VAR0 = 0x10, OP_NOT = 0x20, OP_BOX = 0x21, OP_DIA = 0x22,
       OP_AND = 0x30, OP_OR = 0x31, OP_IMP = 0x32 };
enum { CLS_K = 0, CLS_T = 1, CLS_S4 = 2, CLS_S5 = 3 };

typedef unsigned char u8;

static void decode_frame(int n, uint64_t f, u8 R[MAXN][MAXN]) {
    for (int w = 0; w < n; ++w)
        for (int u = 0; u < n; ++u) R[w][u] = (u8)((f >> (w * n + u)) & 1u);
}

static void decode_valuation(int n, int k, uint64_t v, u8 V[MAXVARS][MAXN]) {
    for (int i = 0; i < k; ++i)
        for (int w = 0; w < n; ++w) V[i][w] = (u8)((v >> (i * n + w)) & 1u);
}

/* Truth array of the formula on the model (n, R, V).  Returns 0, or -1 if malformed.
 * (Inlined into eval_program below once per value of n, so the loops over worlds have constant
 * trip counts; the body is the same for every n.) */
static inline __attribute__((always_inline)) int eval_program_n(
        const u8 *code, uint32_t len, const int n, u8 R[MAXN][MAXN], u8 V[MAXVARS][MAXN], u8 out[MAXN]) {
    u8 st[MAXDEPTH][MAXN];
    int sp = 0;
    for (uint32_t pc = 0; pc < len; ++pc) {
        u8 c = code[pc];
        if (c == OP_TOP || c == OP_BOT || (c >= OP_VAR0 && c < OP_VAR0 + MAXVARS)) {
            if (sp >= MAXDEPTH) return -1;
            for (int w = 0; w < n; ++w)
                st[sp][w] = (c == OP_TOP) ? 1 : (c == OP_BOT) ? 0 : V[c - OP_VAR0][w];
            ++sp;
        } else if (c == OP_NOT) {
            if (sp < 1) return -1;
            for (int w = 0; w < n; ++w) st[sp - 1][w] = !st[sp - 1][w];
        } else if (c == OP_BOX || c == OP_DIA) {
            if (sp < 1) return -1;
            u8 r[MAXN];
            for (int w = 0; w < n; ++w) {
                int all = 1, some = 0;
                for (int u = 0; u < n; ++u)
                    if (R[w][u]) {
                        if (st[sp - 1][u]) some = 1; else all = 0;
                    }
                r[w] = (u8)((c == OP_BOX) ? all : some);
            }
            memcpy(st[sp - 1], r, (size_t)n);
        } else if (c == OP_AND || c == OP_OR || c == OP_IMP) {
            if (sp < 2) return -1;
            for (int w = 0; w < n; ++w) {
                int x = st[sp - 2][w], y = st[sp - 1][w];
                st[sp - 2][w] = (u8)((c == OP_AND) ? (x && y) : (c == OP_OR) ? (x || y) : (!x || y));
            }
            --sp;
        } else {
            return -1;
        }
    }
    if (sp != 1) return -1;
    memcpy(out, st[0], (size_t)n);
    return 0;
}

static int eval_program(const u8 *code, uint32_t len, int n, u8 R[MAXN][MAXN], u8 V[MAXVARS][MAXN],
                        u8 out[MAXN]) {
    switch (n) {
    case 1: return eval_program_n(code, len, 1, R, V, out);
    case 2: return eval_program_n(code, len, 2, R, V, out);
    case 3: return eval_program_n(code, len, 3, R, V, out);
    case 4: return eval_program_n(code, len, 4, R, V, out);
    case 5: return eval_program_n(code, len, 5, R, V, out);
    case 6: return eval_program_n(code, len, 6, R, V, out);
    }
    return -1;
}

/* ---- first-order frame conditions (PAPER.md:42 and Table 9) ---- */
enum { COND_REFLEXIVE = 0, COND_TRANSITIVE = 1, COND_SYMMETRIC = 2, COND_SERIAL = 3,
       COND_EUCLIDEAN = 4, COND_PARTFUNC = 5, COND_DENSE = 6, COND_CONFLUENT = 7 };

static int holds(int n, u8 R[MAXN][MAXN], int cond) {
    switch (cond) {
    case COND_REFLEXIVE:
        for (int w = 0; w < n; ++w) if (!R[w][w]) return 0;
        return 1;
    case COND_TRANSITIVE:
        for (int w = 0; w < n; ++w) for (int u = 0; u < n; ++u) for (int t = 0; t < n; ++t)
            if (R[w][u] && R[u][t] && !R[w][t]) return 0;
        return 1;
    case COND_SYMMETRIC:
        for (int w = 0; w < n; ++w) for (int u = 0; u < n; ++u)
            if (R[w][u] && !R[u][w]) return 0;
        return 1;
    case COND_SERIAL:
        for (int w = 0; w < n; ++w) {
            int any = 0;
            for (int u = 0; u < n; ++u) any |= R[w][u];
            if (!any) return 0;
        }
        return 1;
    case COND_EUCLIDEAN:   /* wRu and wRt imply uRt */
        for (int w = 0; w < n; ++w) for (int u = 0; u < n; ++u) for (int t = 0; t < n; ++t)
            if (R[w][u] && R[w][t] && !R[u][t]) return 0;
        return 1;
    case COND_PARTFUNC:    /* wRu and wRt imply u = t */
        for (int w = 0; w < n; ++w) for (int u = 0; u < n; ++u) for (int t = 0; t < n; ++t)
            if (R[w][u] && R[w][t] && u != t) return 0;
        return 1;
    case COND_DENSE:       /* wRt implies some u with wRu and uRt */
        for (int w = 0; w < n; ++w) for (int t = 0; t < n; ++t)
            if (R[w][t]) {
                int any = 0;
                for (int u = 0; u < n; ++u) any |= (R[w][u] && R[u][t]);
                if (!any) return 0;
            }
        return 1;
    case COND_CONFLUENT:   /* wRu and wRt imply some z with uRz and tRz */
        for (int w = 0; w < n; ++w) for (int u = 0; u < n; ++u) for (int t = 0; t < n; ++t)
            if (R[w][u] && R[w][t]) {
                int any = 0;
                for (int z = 0; z < n; ++z) any |= (R[u][z] && R[t][z]);
                if (!any) return 0;
            }
        return 1;
    }
    return 0;
}

static int in_class(int n, u8 R[MAXN][MAXN], int cls) {
    if (cls == CLS_K) return 1;
    if (!holds(n, R, COND_REFLEXIVE)) return 0;
    if (cls == CLS_T) return 1;
    if (!holds(n, R, COND_TRANSITIVE)) return 0;
    if (cls == CLS_S4) return 1;
    return holds(n, R, COND_SYMMETRIC);
}

/* Number of labelled n-world frames satisfying one condition (all 2^(n*n) scanned). */
uint64_t kov_count_condition(int n, int cond) {
    if (n < 1 || n > 5) return 0;
    uint64_t total = 1ull << (n * n), count = 0;
#pragma omp parallel for reduction(+ : count) schedule(static)
    for (uint64_t f = 0; f < total; ++f) {
        u8 R[MAXN][MAXN];
        decode_frame(n, f, R);
        count += (uint64_t)holds(n, R, cond);
    }
    return count;
}

/* For each frame f of n worlds: out[f] = 1 iff the condition holds (n <= 4 is the intended use). */
int kov_condition_bitmap(int n, int cond, u8 *out) {
    if (n < 1 || n > 5) return -1;
    uint64_t total = 1ull << (n * n);
    for (uint64_t f = 0; f < total; ++f) {
        u8 R[MAXN][MAXN];
        decode_frame(n, f, R);
        out[f] = (u8)holds(n, R, cond);
    }
    return 0;
}

/* Ascending K-indices of the class members.  Returns the count (writes at most cap of them; pass
 * out = NULL to count only).  n <= 5: the whole K range is scanned, nothing clever. */
int64_t kov_class_frames(int n, int cls, uint64_t *out, uint64_t cap) {
    if (n < 1 || n > 5 || cls < 0 || cls > 3) return -1;
    uint64_t total = 1ull << (n * n), count = 0;
    for (uint64_t f = 0; f < total; ++f) {
        u8 R[MAXN][MAXN];
        decode_frame(n, f, R);
        if (in_class(n, R, cls)) {
            if (out && count < cap) out[count] = f;
            ++count;
        }
    }
    return (int64_t)count;
}

/* Truth array of one formula on one model; 0 on success. */
int kov_truth(const u8 *code, uint32_t len, int n, uint64_t f, int k, uint64_t v, u8 *truth_out) {
    if (n < 1 || n > MAXN || k < 0 || k > MAXVARS) return -1;
    u8 R[MAXN][MAXN], V[MAXVARS][MAXN];
    decode_frame(n, f, R);
    decode_valuation(n, k, v, V);
    return eval_program(code, len, n, R, V, truth_out);
}

typedef struct {
    uint64_t pos;      /* position in the frame list (NO_WITNESS if none) */
    uint64_t v;
    uint32_t w;
} first_t;

/* Census of B formulas (or P pairs if pairs != NULL) over an explicit list of frames.
 *   frames[i]  K-index of the i-th frame; weights[i] (or NULL = 1) multiplies its contribution to
 *              both counts (used for isomorphism-orbit counting, where the list holds one
 *              representative per orbit and the weight is the orbit size).
 *   outputs    per formula / pair: refuting (distinguishing) models, frames, first (f, v, w) in
 *              list order, wit_f = UINT64_MAX if none.
 * Returns 0, or -1 on a malformed program / bad argument. */
int kov_census_list(const u8 *code, const uint32_t *offs, uint32_t B,
                    const uint32_t *pairs, uint32_t P,
                    int n, int k, const uint64_t *frames, const uint64_t *weights, uint64_t nframes,
                    uint64_t *models_out, uint64_t *frames_out,
                    uint64_t *wit_f, uint32_t *wit_v, uint32_t *wit_w, int nthreads) {
    if (n < 1 || n > MAXN || k < 0 || k > MAXVARS || k * n > 30) return -1;
    const uint32_t Q = pairs ? P : B;     /* number of output records */
    const uint64_t nval = 1ull << (k * n);
    int bad = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    uint64_t *acc_m = calloc((size_t)nthreads * Q, sizeof(uint64_t));
    uint64_t *acc_f = calloc((size_t)nthreads * Q, sizeof(uint64_t));
    first_t *first = malloc((size_t)nthreads * Q * sizeof(first_t));
    /* every valuation decoded once: vtab[v] is the k x n byte matrix of valuation index v */
    u8 (*vtab)[MAXVARS][MAXN] = malloc((size_t)nval * sizeof(*vtab));
    if (!acc_m || !acc_f || !first || !vtab) return -1;
    for (size_t i = 0; i < (size_t)nthreads * Q; ++i) first[i].pos = NO_WITNESS;
    for (uint64_t v = 0; v < nval; ++v) decode_valuation(n, k, v, vtab[v]);

#pragma omp parallel num_threads(nthreads)
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        uint64_t *am = acc_m + (size_t)tid * Q, *af = acc_f + (size_t)tid * Q;
        first_t *fi = first + (size_t)tid * Q;
#pragma omp for schedule(dynamic, 4)
        for (uint64_t pos = 0; pos < nframes; ++pos) {
            u8 R[MAXN][MAXN];
            decode_frame(n, frames[pos], R);
            uint64_t wgt = weights ? weights[pos] : 1;
            for (uint32_t q = 0; q < Q; ++q) {
                uint32_t a = pairs ? pairs[2 * q] : q, b = pairs ? pairs[2 * q + 1] : q;
                int hit = 0;
                for (uint64_t v = 0; v < nval; ++v) {
                    u8 ta[MAXN], tb[MAXN];
                    int fail_world = -1;
                    if (eval_program(code + offs[a], offs[a + 1] - offs[a], n, R, vtab[v], ta)) bad = 1;
                    if (pairs) {      /* least world where exactly one of the two formulas holds */
                        if (eval_program(code + offs[b], offs[b + 1] - offs[b], n, R, vtab[v], tb)) bad = 1;
                        for (int w = 0; w < n; ++w)
                            if ((ta[w] != 0) != (tb[w] != 0)) { fail_world = w; break; }
                    } else {          /* least world outside the truth set */
                        for (int w = 0; w < n; ++w)
                            if (!ta[w]) { fail_world = w; break; }
                    }
                    if (fail_world >= 0) {
                        am[q] += wgt;
                        hit = 1;
                        if (pos < fi[q].pos) { fi[q].pos = pos; fi[q].v = v; fi[q].w = (uint32_t)fail_world; }
                    }
                }
                if (hit) af[q] += wgt;
            }
        }
    }
    for (uint32_t q = 0; q < Q; ++q) {
        uint64_t m = 0, fr = 0;
        first_t best; best.pos = NO_WITNESS; best.v = 0; best.w = 0;
        for (int t = 0; t < nthreads; ++t) {
            m += acc_m[(size_t)t * Q + q];
            fr += acc_f[(size_t)t * Q + q];
            if (first[(size_t)t * Q + q].pos < best.pos) best = first[(size_t)t * Q + q];
        }
        models_out[q] = m;
        frames_out[q] = fr;
        wit_f[q] = (best.pos == NO_WITNESS) ? NO_WITNESS : frames[best.pos];
        wit_v[q] = (uint32_t)best.v;
        wit_w[q] = best.w;
    }
    free(acc_m); free(acc_f); free(first); free(vtab);
    return bad ? -1 : 0;
}

int kov_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Semantic signature of each formula: two independent 64-bit hashes of the sequence of its truth
 * arrays over every model (frame, valuation) of 1..max_n worlds, in ascending (n, f, v) order.
 * Two formulas get the same signature iff (up to a 2^-128 hash collision) their truth sets agree
 * on every model of <= max_n worlds - the equivalence PAPER.md:143 dedups the corpus by.
 * The hashes only compress the comparison; they are no part of the semantics. */
int kov_signatures(const u8 *code, const uint32_t *offs, uint32_t B, int max_n, int k,
                   uint64_t *sig_a, uint64_t *sig_b) {
    if (max_n < 1 || max_n > 4 || k < 0 || k > MAXVARS) return -1;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64)
    for (uint32_t b = 0; b < B; ++b) {
        uint64_t ha = 1469598103934665603ull, hb = 0x9E3779B97F4A7C15ull;
        for (int n = 1; n <= max_n; ++n) {
            uint64_t nfr = 1ull << (n * n), nval = 1ull << (k * n);
            for (uint64_t f = 0; f < nfr; ++f) {
                u8 R[MAXN][MAXN], V[MAXVARS][MAXN], t[MAXN];
                decode_frame(n, f, R);
                for (uint64_t v = 0; v < nval; ++v) {
                    decode_valuation(n, k, v, V);
                    if (eval_program(code + offs[b], offs[b + 1] - offs[b], n, R, V, t)) bad = 1;
                    for (int w = 0; w < n; ++w) {
                        ha = (ha ^ (uint64_t)(t[w] + 1)) * 1099511628211ull;
                        hb = (hb + (uint64_t)(t[w] + 1)) * 0xD6E8FEB86659FD93ull;
                        hb ^= hb >> 29;
                    }
                }
            }
        }
        sig_a[b] = ha;
        sig_b[b] = hb;
    }
    return bad ? -1 : 0;
}

/* ---- isomorphism orbits of labelled frames (relabelling invariance) ----
 * A permutation pi of the worlds maps the relation R to {(pi(w), pi(u)) : (w,u) in R}.  Counts of
 * refuting models / frames of a fixed formula are equal on isomorphic frames (rename the worlds in
 * the valuation as well), so a full-class-K count equals the sum over orbit representatives of
 * orbit size x the representative's count.  A frame is its orbit's representative iff no image is
 * smaller than it; the orbit size is the number of distinct images.  Plain enumeration of all n!
 * permutations, nothing clever. */
static uint64_t apply_perm(int n, const int *pi, uint64_t f) {
    uint64_t g = 0;
    for (int w = 0; w < n; ++w)
        for (int u = 0; u < n; ++u)
            if ((f >> (w * n + u)) & 1u) g |= 1ull << (pi[w] * n + pi[u]);
    return g;
}

static int next_perm(int n, int *p) {           /* lexicographic successor; 0 when done */
    int i = n - 2;
    while (i >= 0 && p[i] > p[i + 1]) --i;
    if (i < 0) return 0;
    int j = n - 1;
    while (p[j] < p[i]) --j;
    int t = p[i]; p[i] = p[j]; p[j] = t;
    for (int a = i + 1, b = n - 1; a < b; ++a, --b) { t = p[a]; p[a] = p[b]; p[b] = t; }
    return 1;
}

/* Writes the ascending orbit representatives of all n-world frames and their orbit sizes; returns
 * the number of orbits (or -1).  Pass reps = NULL to count only. */
int64_t kov_orbits(int n, uint64_t *reps, uint64_t *sizes, uint64_t cap) {
    if (n < 1 || n > 5) return -1;
    int nperm = 1;
    for (int i = 2; i <= n; ++i) nperm *= i;
    int (*perms)[MAXN] = malloc((size_t)nperm * sizeof(*perms));
    int p[MAXN];
    for (int i = 0; i < n; ++i) p[i] = i;
    int c = 0;
    do { memcpy(perms[c++], p, sizeof(p)); } while (next_perm(n, p));
    uint64_t total = 1ull << (n * n);
    u8 *is_rep = calloc(total, 1);
#pragma omp parallel for schedule(dynamic, 4096)
    for (uint64_t f = 0; f < total; ++f) {
        int rep = 1;
        for (int i = 0; i < nperm && rep; ++i)
            if (apply_perm(n, perms[i], f) < f) rep = 0;
        is_rep[f] = (u8)rep;
    }
    uint64_t count = 0;
    for (uint64_t f = 0; f < total; ++f) {
        if (!is_rep[f]) continue;
        if (reps && count < cap) {
            uint64_t img[120];
            for (int i = 0; i < nperm; ++i) img[i] = apply_perm(n, perms[i], f);
            uint64_t distinct = 0;
            for (int i = 0; i < nperm; ++i) {
                int seen = 0;
                for (int j = 0; j < i; ++j) if (img[j] == img[i]) { seen = 1; break; }
                distinct += !seen;
            }
            reps[count] = f;
            sizes[count] = distinct;
        }
        ++count;
    }
    free(is_rep); free(perms);
    return (int64_t)count;
}

/* ---- explicit frame lists, up to 16 worlds (PAPER.md:183-185 templates, :192 synthesized relations) ----
 * The same definitions once more, with the relation given as an n x n byte matrix per frame instead
 * of an index, and arrays sized for 16 worlds.  rel[(j*n + w)*n + u] != 0 iff frame j has w -> u. */
#define BIGN 16

static int eval_program_big(const u8 *code, uint32_t len, int n, const u8 *R /* n*n */,
                            u8 V[MAXVARS][BIGN], u8 out[BIGN]) {
    u8 st[MAXDEPTH][BIGN];
    int sp = 0;
    for (uint32_t pc = 0; pc < len; ++pc) {
        u8 c = code[pc];
        if (c == OP_TOP || c == OP_BOT || (c >= OP_VAR0 && c < OP_VAR0 + MAXVARS)) {
            if (sp >= MAXDEPTH) return -1;
            for (int w = 0; w < n; ++w)
                st[sp][w] = (c == OP_TOP) ? 1 : (c == OP_BOT) ? 0 : V[c - OP_VAR0][w];
            ++sp;
        } else if (c == OP_NOT) {
            if (sp < 1) return -1;
            for (int w = 0; w < n; ++w) st[sp - 1][w] = !st[sp - 1][w];
        } else if (c == OP_BOX || c == OP_DIA) {
            if (sp < 1) return -1;
            u8 r[BIGN];
            for (int w = 0; w < n; ++w) {
                int all = 1, some = 0;            /* box: every successor; dia: some successor */
                for (int u = 0; u < n; ++u)
                    if (R[w * n + u]) {
                        if (st[sp - 1][u]) some = 1; else all = 0;
                    }
                r[w] = (u8)((c == OP_BOX) ? all : some);
            }
            memcpy(st[sp - 1], r, (size_t)n);
        } else if (c == OP_AND || c == OP_OR || c == OP_IMP) {
            if (sp < 2) return -1;
            for (int w = 0; w < n; ++w) {
                int x = st[sp - 2][w], y = st[sp - 1][w];
                st[sp - 2][w] = (u8)((c == OP_AND) ? (x && y) : (c == OP_OR) ? (x || y) : (!x || y));
            }
            --sp;
        } else {
            return -1;
        }
    }
    if (sp != 1) return -1;
    memcpy(out, st[0], (size_t)n);
    return 0;
}

/* Census of B formulas (or P pairs) over the explicit frames rel[0..nframes) and all 2^(k*n)
 * valuations.  Outputs as kov_census_list; the witness frame is the POSITION in the list. */
int kov_census_relations(const u8 *code, const uint32_t *offs, uint32_t B,
                         const uint32_t *pairs, uint32_t P, int n, int k,
                         const u8 *rel, uint64_t nframes,
                         uint64_t *models_out, uint64_t *frames_out,
                         uint64_t *wit_f, uint32_t *wit_v, uint32_t *wit_w, int nthreads) {
    if (n < 1 || n > BIGN || k < 0 || k > MAXVARS || k * n > 24) return -1;
    const uint32_t Q = pairs ? P : B;
    const uint64_t nval = 1ull << (k * n);
    int bad = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    uint64_t *acc_m = calloc((size_t)nthreads * Q, sizeof(uint64_t));
    uint64_t *acc_f = calloc((size_t)nthreads * Q, sizeof(uint64_t));
    first_t *first = malloc((size_t)nthreads * Q * sizeof(first_t));
    if (!acc_m || !acc_f || !first) return -1;
    for (size_t i = 0; i < (size_t)nthreads * Q; ++i) first[i].pos = NO_WITNESS;

#pragma omp parallel num_threads(nthreads)
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        uint64_t *am = acc_m + (size_t)tid * Q, *af = acc_f + (size_t)tid * Q;
        first_t *fi = first + (size_t)tid * Q;
#pragma omp for schedule(dynamic, 4)
        for (uint64_t pos = 0; pos < nframes; ++pos) {
            const u8 *R = rel + (size_t)pos * n * n;
            for (uint32_t q = 0; q < Q; ++q) {
                uint32_t a = pairs ? pairs[2 * q] : q, b = pairs ? pairs[2 * q + 1] : q;
                int hit = 0;
                for (uint64_t v = 0; v < nval; ++v) {
                    u8 V[MAXVARS][BIGN], ta[BIGN], tb[BIGN];
                    for (int i = 0; i < k; ++i)
                        for (int w = 0; w < n; ++w) V[i][w] = (u8)((v >> (i * n + w)) & 1u);
                    int fail_world = -1;
                    if (eval_program_big(code + offs[a], offs[a + 1] - offs[a], n, R, V, ta)) bad = 1;
                    if (pairs) {
                        if (eval_program_big(code + offs[b], offs[b + 1] - offs[b], n, R, V, tb)) bad = 1;
                        for (int w = 0; w < n; ++w)
                            if ((ta[w] != 0) != (tb[w] != 0)) { fail_world = w; break; }
                    } else {
                        for (int w = 0; w < n; ++w)
                            if (!ta[w]) { fail_world = w; break; }
                    }
                    if (fail_world >= 0) {
                        am[q] += 1;
                        hit = 1;
                        if (pos < fi[q].pos) { fi[q].pos = pos; fi[q].v = v; fi[q].w = (uint32_t)fail_world; }
                    }
                }
                if (hit) af[q] += 1;
            }
        }
    }
    for (uint32_t q = 0; q < Q; ++q) {
        uint64_t m = 0, fr = 0;
        first_t best; best.pos = NO_WITNESS; best.v = 0; best.w = 0;
        for (int t = 0; t < nthreads; ++t) {
            m += acc_m[(size_t)t * Q + q];
            fr += acc_f[(size_t)t * Q + q];
            if (first[(size_t)t * Q + q].pos < best.pos) best = first[(size_t)t * Q + q];
        }
        models_out[q] = m;
        frames_out[q] = fr;
        wit_f[q] = best.pos;
        wit_v[q] = (uint32_t)best.v;
        wit_w[q] = best.w;
    }
    free(acc_m); free(acc_f); free(first);
    return bad ? -1 : 0;
}

/* ---- frame validity per frame ("valid on a frame"; PAPER.md:358-380 correspondence) ----
 * out[b * nframes + i] = 1 iff formula b is valid on frame frames[i]: no valuation of the k variables
 * and no world falsify it.  Same plain evaluation as kov_census_list. */
int kov_validity_list(const u8 *code, const uint32_t *offs, uint32_t B, int n, int k,
                      const uint64_t *frames, uint64_t nframes, u8 *out, int nthreads) {
    if (n < 1 || n > MAXN || k < 0 || k > MAXVARS || k * n > 30) return -1;
    const uint64_t nval = 1ull << (k * n);
    int bad = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 16)
    for (uint64_t i = 0; i < nframes; ++i) {
        u8 R[MAXN][MAXN], V[MAXVARS][MAXN], t[MAXN];
        decode_frame(n, frames[i], R);
        for (uint32_t b = 0; b < B; ++b) {
            int valid = 1;
            for (uint64_t v = 0; v < nval && valid; ++v) {
                decode_valuation(n, k, v, V);
                if (eval_program(code + offs[b], offs[b + 1] - offs[b], n, R, V, t)) bad = 1;
                for (int w = 0; w < n; ++w)
                    if (!t[w]) valid = 0;
            }
            out[(size_t)b * nframes + i] = (u8)valid;
        }
    }
    return bad ? -1 : 0;
}

/* ---- failure densities ("D_ij = the fraction of valuation-world pairs on which formula i
 * fails on frame j") ----  out[b * nframes + j] = #{(v, w) : world w is outside the truth set of formula b
 * under valuation v on frame j}; the density is that count divided by 2^(k*n) * n. */
int kov_failure_counts(const u8 *code, const uint32_t *offs, uint32_t B, int n, int k,
                       const uint64_t *frames, uint64_t nframes, uint32_t *out, int nthreads) {
    if (n < 1 || n > MAXN || k < 0 || k > MAXVARS || k * n > 24) return -1;
    const uint64_t nval = 1ull << (k * n);
    int bad = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 16)
    for (uint64_t j = 0; j < nframes; ++j) {
        u8 R[MAXN][MAXN], V[MAXVARS][MAXN], t[MAXN];
        decode_frame(n, frames[j], R);
        for (uint32_t b = 0; b < B; ++b) {
            uint32_t cnt = 0;
            for (uint64_t v = 0; v < nval; ++v) {
                decode_valuation(n, k, v, V);
                if (eval_program(code + offs[b], offs[b + 1] - offs[b], n, R, V, t)) bad = 1;
                for (int w = 0; w < n; ++w) cnt += !t[w];
            }
            out[(size_t)b * nframes + j] = cnt;
        }
    }
    return bad ? -1 : 0;
}

/* The same over explicit relations rel[nframes][n][n] (n <= 16). */
int kov_failure_counts_relations(const u8 *code, const uint32_t *offs, uint32_t B, int n, int k,
                                 const u8 *rel, uint64_t nframes, uint32_t *out, int nthreads) {
    if (n < 1 || n > BIGN || k < 0 || k > MAXVARS || k * n > 24) return -1;
    const uint64_t nval = 1ull << (k * n);
    int bad = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 16)
    for (uint64_t j = 0; j < nframes; ++j) {
        const u8 *R = rel + (size_t)j * n * n;
        for (uint32_t b = 0; b < B; ++b) {
            uint32_t cnt = 0;
            for (uint64_t v = 0; v < nval; ++v) {
                u8 V[MAXVARS][BIGN], t[BIGN];
                for (int i = 0; i < k; ++i)
                    for (int w = 0; w < n; ++w) V[i][w] = (u8)((v >> (i * n + w)) & 1u);
                if (eval_program_big(code + offs[b], offs[b + 1] - offs[b], n, R, V, t)) bad = 1;
                for (int w = 0; w < n; ++w) cnt += !t[w];
            }
            out[(size_t)b * nframes + j] = cnt;
        }
    }
    return bad ? -1 : 0;
}
