/*
 * ORACLE, tier 1 (TEST INFRASTRUCTURE ONLY — the product never links, loads or
 * calls this file; only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs do).
 *
 * A plain matrix-free CPU restatement of the paper's own CPU comparator
 * (sequential, same algorithm including eq. 13, H_up / H_dn in
 * CSR, double precision), used where the definitional tier 0
 * (oracle/hubbard_def.py) is too slow: full-vector H*v and Lanczos on the
 * larger configurations.  It carries no authority of its own: every routine
 * here is checked against tier 0 on small sectors (tests/test_oracle_pins.py).
 *
 * Independent of the CUDA library: own enumeration (scan of all 2^N_s numbers,
 * PAPER.md:63-67), own rank (binary search in that sorted list), own signs
 * (two-step second-quantisation rule: c_j then c+_i, each with the parity of
 * the operators standing to its left in the string of eq. 4, PAPER.md:41-47 —
 * NOT the "electrons hopped over" shortcut of PAPER.md:99-104, so that the two
 * rules check each other).
 *
 * Everything is fp64.  OpenMP is used only to spread rows of H*v over host
 * cores for the timed CPU baseline; n_threads = 1 is the paper's sequential
 * comparator.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static int popc(uint32_t x) { return __builtin_popcount(x); }

/* Ascending list of all n_sites-bit numbers with n_el bits set.
 * Returns the count; writes at most cap entries. */
int64_t ref_basis(int n_sites, int n_el, uint32_t *out, int64_t cap)
{
    int64_t n = 0;
    uint64_t lim = 1ull << n_sites;
    for (uint64_t s = 0; s < lim; ++s) {
        if (popc((uint32_t)s) == n_el) {
            if (n < cap) out[n] = (uint32_t)s;
            ++n;
        }
    }
    return n;
}

static int64_t find_state(const uint32_t *states, int64_t n, uint32_t s)
{
    int64_t lo = 0, hi = n - 1;
    while (lo <= hi) {
        int64_t mid = (lo + hi) / 2;
        if (states[mid] == s) return mid;
        if (states[mid] < s) lo = mid + 1; else hi = mid - 1;
    }
    return -1;
}

/* Parity of the creation operators standing to the LEFT of (spin, site) in the
 * canonical string of eq. (4): same-spin operators on lower sites, plus — for a
 * down operator — all n_left up operators. */
static int left_parity(uint32_t bits, int site, int n_left)
{
    uint32_t below = bits & ((site == 0) ? 0u : (0xffffffffu >> (32 - site)));
    return (popc(below) + n_left) & 1;
}

typedef struct { int64_t col; double val; } entry_t;

static int cmp_entry(const void *a, const void *b)
{
    int64_t ca = ((const entry_t *)a)->col, cb = ((const entry_t *)b)->col;
    return (ca > cb) - (ca < cb);
}

/* Per-spin hopping matrix (eq. 14) in CSR, row = target
 * state, entries sorted by column, duplicates merged, exact zeros dropped.
 * n_left = number of other-spin operators standing left of this spin's
 * operators (0 for up, N_up for down).  `rowptr` has n+1 entries; `cols`/`vals`
 * have room for cap entries.  Returns nnz, or -1 if cap is too small. */
int64_t ref_hops_csr(int n_sites, int n_el, int n_left, const int32_t *bonds, int n_bonds, double t,
                     const uint32_t *states, int64_t n, int64_t *rowptr, int32_t *cols, double *vals,
                     int64_t cap)
{
    entry_t *tmp = (entry_t *)malloc(sizeof(entry_t) * (size_t)(4 * n_bonds + 4));
    int64_t nnz = 0;
    (void)n_sites; (void)n_el;
    for (int64_t r = 0; r < n; ++r) {
        /* row r of a real symmetric matrix = column r: apply H_hop to |r>. */
        uint32_t s = states[r];
        int cnt = 0;
        for (int b = 0; b < n_bonds; ++b) {
            for (int dir = 0; dir < 2; ++dir) {
                int src = dir ? bonds[2 * b] : bonds[2 * b + 1];
                int dst = dir ? bonds[2 * b + 1] : bonds[2 * b];
                if (!((s >> src) & 1u)) continue;          /* c_src |..> = 0 */
                int p1 = left_parity(s, src, n_left);
                uint32_t s1 = s & ~(1u << src);
                if ((s1 >> dst) & 1u) continue;            /* (c+)^2 = 0 */
                int p2 = left_parity(s1, dst, n_left);
                uint32_t s2 = s1 | (1u << dst);
                tmp[cnt].col = find_state(states, n, s2);
                tmp[cnt].val = ((p1 + p2) & 1) ? t : -t;   /* -t * (-1)^(p1+p2) */
                ++cnt;
            }
        }
        qsort(tmp, (size_t)cnt, sizeof(entry_t), cmp_entry);
        rowptr[r] = nnz;
        for (int k = 0; k < cnt;) {
            int64_t c = tmp[k].col;
            double v = 0.0;
            while (k < cnt && tmp[k].col == c) v += tmp[k++].val;
            if (v != 0.0) {
                if (nnz >= cap) { free(tmp); return -1; }
                cols[nnz] = (int32_t)c;
                vals[nnz] = v;
                ++nnz;
            }
        }
    }
    rowptr[n] = nnz;
    free(tmp);
    return nnz;
}

/* y = H x, matrix-free (PAPER.md:236-336 restated for one CPU thread per row
 * of V): up term eq. 15, down term eq. 16, on-the-fly diagonal Algorithm 4.
 * x, y: dim_up*dim_dn doubles, J = i_up*dim_dn + i_dn (eq. 7). */
void ref_apply(int64_t dim_up, int64_t dim_dn, const uint32_t *st_up, const uint32_t *st_dn,
               const int64_t *rp_up, const int32_t *cj_up, const double *cv_up,
               const int64_t *rp_dn, const int32_t *cj_dn, const double *cv_dn,
               double U, const double *x, double *y, int n_threads)
{
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t a = 0; a < dim_up; ++a) {
        double *ya = y + a * dim_dn;
        const double *xa = x + a * dim_dn;
        uint32_t sa = st_up[a];
        for (int64_t b = 0; b < dim_dn; ++b) {
            double sum = 0.0;
            for (int64_t k = rp_dn[b]; k < rp_dn[b + 1]; ++k) sum += cv_dn[k] * xa[cj_dn[k]];
            sum += U * (double)popc(sa & st_dn[b]) * xa[b];
            ya[b] = sum;
        }
        for (int64_t k = rp_up[a]; k < rp_up[a + 1]; ++k) {
            const double *xr = x + (int64_t)cj_up[k] * dim_dn;
            double v = cv_up[k];
            for (int64_t b = 0; b < dim_dn; ++b) ya[b] += v * xr[b];
        }
    }
}

static double dot(const double *a, const double *b, int64_t n)
{
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) s += a[i] * b[i];
    return s;
}

/* The paper's CPU comparator: Algorithm 1 with the
 * two-vector update of eq. 13.  f (in: start vector, need
 * not be normalised) and g are caller-provided work vectors of length dim; a
 * third scratch vector h holds H f_j (the CPU code has no fused kernel).
 * alpha[j-1] = a_j, beta[j-1] = b_{j+1}.  Returns the number of iterations done
 * (breakdown rule: DESIGN.md reading Q11). */
int ref_lanczos(int64_t dim_up, int64_t dim_dn, const uint32_t *st_up, const uint32_t *st_dn,
                const int64_t *rp_up, const int32_t *cj_up, const double *cv_up,
                const int64_t *rp_dn, const int32_t *cj_dn, const double *cv_dn,
                double U, double *f, double *g, double *h, int m, double tau,
                double *alpha, double *beta, int n_threads)
{
    int64_t dim = dim_up * dim_dn;
    double nrm = sqrt(dot(f, f, dim));
    for (int64_t i = 0; i < dim; ++i) { f[i] /= nrm; g[i] = 0.0; }   /* f_1, f_0 = 0 */
    double b = 0.0, amax = 0.0;
    double *fj = f, *fp = g;
    int done = 0;
    for (int j = 0; j < m; ++j) {
        ref_apply(dim_up, dim_dn, st_up, st_dn, rp_up, cj_up, cv_up, rp_dn, cj_dn, cv_dn, U, fj, h, n_threads);
        for (int64_t i = 0; i < dim; ++i) fp[i] = -b * fp[i];        /* eq. 13  */
        for (int64_t i = 0; i < dim; ++i) fp[i] = fp[i] + h[i];      /* eq. 13' : fp is now q_j */
        double a = dot(fp, fj, dim);                                 /* line 5 */
        for (int64_t i = 0; i < dim; ++i) fp[i] -= a * fj[i];        /* line 6 */
        double bn = sqrt(dot(fp, fp, dim));                          /* line 7 */
        alpha[j] = a; beta[j] = bn; done = j + 1;
        if (fabs(a) > amax) amax = fabs(a);
        if (!(bn > tau * (amax > 1.0 ? amax : 1.0)) || !isfinite(bn)) break;  /* lines 8-10 */
        for (int64_t i = 0; i < dim; ++i) fp[i] /= bn;               /* line 11 */
        double *tmpp = fj; fj = fp; fp = tmpp;
        b = bn;
    }
    return done;
}

int ref_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
