/*
 * hec_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU
 * oracle for the batched naive Hasse-Weil count of arXiv 1805.11991 (M. Raum).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this file.  It shares NO code, header, table or
 * constant generator with the CUDA path under paper_1805_11991_b200/csrc/.
 *
 * What it computes -- the plain definition (section 1.1):
 *   for f = sum_{n=0}^{2g+2} c_n X^n over F_q (q = p^r, p odd) and E = F_{q^k},
 *     N_k = #C_f(E) = r0(f,E) + 2 rsq(f,E) + (1 + chi_E(f(inf))),  f(inf) := c_{2g+2}
 *   r0  = #{x in E : f(x) = 0}
 *   rsq = #{x in E : f(x) a NONZERO square in E}      (reading G3 in DESIGN.md:
 *         PAPER.md:47 omits "nonzero"; Algorithm 1's else-if, PAPER.md:145-147,
 *         confirms it)
 *   1 + chi_E(c) = 1 if c = 0, 2 if c is a nonzero square in E, 0 otherwise.
 *   squarefree = [deg gcd(f, f') = 0] over F_q.
 *
 * How (section 2.2 -- the representation the paper calls
 * "inherently slow"; NO Zech/log/antilog tables anywhere in this file):
 *   E = F_p[t]/(P_E), P_E = lexicographically smallest monic IRREDUCIBLE of
 *   degree r*k (need not be primitive -- N_k does not depend on it).
 *   Elements are digit vectors over F_p; multiplication is the schoolbook
 *   product followed by reduction modulo P_E; f(x) by Horner (Algorithm 1
 *   line 8) at every x in E; squareness by Euler's criterion
 *   y^((#E-1)/2) = 1.
 *
 * Meaning of the input integers (reading G7 in DESIGN.md): an F_q element is
 * the integer sum a_i p^i  <->  sum a_i T^i in F_p[T]/(R_q), little-endian
 * base-p digits, R_q = lexicographically smallest monic
 * PRIMITIVE polynomial of degree r (order the tuple (a_{r-1},...,a_0)).
 * F_q sits inside E by T -> rho, rho any root of R_q in E found by exhaustive
 * search (N_k is the same for every root).
 *
 * Every exported function is pinned by tests/test_oracle_pins.py
 * (-m "not gpu").  No function here is "parity unpinned".
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXN 12            /* largest extension degree r*k over F_p */
#define ORC_MAXDEG 64          /* largest polynomial degree 2g+2 */

typedef struct { uint32_t d[ORC_MAXN]; } elt;            /* digits, d[i] multiplies t^i */
typedef struct { uint32_t p, n; uint32_t mod[ORC_MAXN + 1]; } ring;  /* F_p[t]/(mod), mod monic of degree n */

/* ---------------------------------------------------------------- F_p[t]/(mod) */

static elt elt_zero(void) { elt z; memset(&z, 0, sizeof z); return z; }
static elt elt_one(void) { elt z = elt_zero(); z.d[0] = 1; return z; }

static int elt_is_zero(const ring *R, const elt *a) {
    for (uint32_t i = 0; i < R->n; i++) if (a->d[i]) return 0;
    return 1;
}
static int elt_eq(const ring *R, const elt *a, const elt *b) {
    for (uint32_t i = 0; i < R->n; i++) if (a->d[i] != b->d[i]) return 0;
    return 1;
}
static elt elt_add(const ring *R, const elt *a, const elt *b) {
    elt c = elt_zero();
    for (uint32_t i = 0; i < R->n; i++) c.d[i] = (a->d[i] + b->d[i]) % R->p;
    return c;
}
/* schoolbook product, then reduction modulo the monic modulus */
static elt elt_mul(const ring *R, const elt *a, const elt *b) {
    uint64_t w[2 * ORC_MAXN];
    uint32_t n = R->n, p = R->p;
    for (uint32_t i = 0; i < 2 * n; i++) w[i] = 0;
    for (uint32_t i = 0; i < n; i++)
        for (uint32_t j = 0; j < n; j++)
            w[i + j] += (uint64_t)a->d[i] * b->d[j];
    for (uint32_t i = 0; i < 2 * n; i++) w[i] %= p;
    /* t^m = -(mod[n-1] t^{m-1} + ... + mod[0] t^{m-n}) for m >= n */
    for (uint32_t m = 2 * n - 2; m >= n && m < 2 * n; m--) {
        uint64_t top = w[m];
        if (!top) continue;
        w[m] = 0;
        for (uint32_t i = 0; i < n; i++) {
            uint64_t sub = (top * R->mod[i]) % p;
            w[m - n + i] = (w[m - n + i] + p - sub) % p;
        }
    }
    elt c = elt_zero();
    for (uint32_t i = 0; i < n; i++) c.d[i] = (uint32_t)w[i];
    return c;
}
static elt elt_pow(const ring *R, elt a, uint64_t e) {
    elt r = elt_one();
    while (e) {
        if (e & 1) r = elt_mul(R, &r, &a);
        a = elt_mul(R, &a, &a);
        e >>= 1;
    }
    return r;
}
static uint64_t ring_size(const ring *R) {
    uint64_t Q = 1;
    for (uint32_t i = 0; i < R->n; i++) Q *= R->p;
    return Q;
}
/* integer e in [0, p^n) -> element with little-endian base-p digits */
static elt elt_from_int(const ring *R, uint64_t e) {
    elt a = elt_zero();
    for (uint32_t i = 0; i < R->n; i++) { a.d[i] = (uint32_t)(e % R->p); e /= R->p; }
    return a;
}

/* ---------------------------------------------- irreducible / primitive moduli */

/* does the monic polynomial b (degree db >= 1) divide the monic a (degree da)? */
static int poly_divides(uint32_t p, const uint32_t *a, uint32_t da, const uint32_t *b, uint32_t db) {
    uint32_t w[ORC_MAXN + 1];
    for (uint32_t i = 0; i <= da; i++) w[i] = a[i];
    for (uint32_t m = da; m >= db && m <= da; m--) {
        uint32_t top = w[m];
        if (!top) continue;
        for (uint32_t i = 0; i <= db; i++)
            w[m - db + i] = (uint32_t)((w[m - db + i] + (uint64_t)(p - top) * b[i]) % p);
    }
    for (uint32_t i = 0; i < db; i++) if (w[i]) return 0;
    return 1;
}
/* brute force: no monic divisor of degree 1 .. n/2 */
static int poly_is_irreducible(uint32_t p, uint32_t n, const uint32_t *mod) {
    for (uint32_t db = 1; 2 * db <= n; db++) {
        uint64_t cnt = 1;
        for (uint32_t i = 0; i < db; i++) cnt *= p;
        for (uint64_t e = 0; e < cnt; e++) {
            uint32_t b[ORC_MAXN + 1];
            uint64_t v = e;
            for (uint32_t i = 0; i < db; i++) { b[i] = (uint32_t)(v % p); v /= p; }
            b[db] = 1;
            if (poly_divides(p, mod, n, b, db)) return 0;
        }
    }
    return 1;
}
/* candidate number e in lexicographic order of (a_{n-1}, ..., a_0): a_0 is the
 * fastest-running digit, so counting e = sum a_i p^i upwards IS that order. */
static void modulus_from_index(uint32_t p, uint32_t n, uint64_t e, uint32_t *mod) {
    for (uint32_t i = 0; i < n; i++) { mod[i] = (uint32_t)(e % p); e /= p; }
    mod[n] = 1;
}
/* brute force: t, t^2, ... first returns to 1 at exponent exactly p^n - 1 */
static int modulus_is_primitive(uint32_t p, uint32_t n, const uint32_t *mod) {
    ring R; R.p = p; R.n = n; memcpy(R.mod, mod, (n + 1) * sizeof(uint32_t));
    if (mod[0] == 0) return 0;
    uint64_t Q = ring_size(&R);
    elt t = elt_zero();
    if (n == 1) t.d[0] = (p - mod[0]) % p; else t.d[1] = 1;
    elt one = elt_one(), y = t;
    for (uint64_t j = 1; j < Q - 1; j++) {
        if (elt_eq(&R, &y, &one)) return 0;
        y = elt_mul(&R, &y, &t);
    }
    return elt_eq(&R, &y, &one);
}

/* Exported: lexicographically smallest monic irreducible of degree n over F_p. */
int orc_smallest_irreducible(uint32_t p, uint32_t n, uint32_t *out_mod) {
    if (n < 1 || n > ORC_MAXN) return -1;
    uint64_t cnt = 1;
    for (uint32_t i = 0; i < n; i++) cnt *= p;
    for (uint64_t e = 0; e < cnt; e++) {
        uint32_t mod[ORC_MAXN + 1];
        modulus_from_index(p, n, e, mod);
        if (n == 1 || poly_is_irreducible(p, n, mod)) {
            memcpy(out_mod, mod, (n + 1) * sizeof(uint32_t));
            return 0;
        }
    }
    return -2;
}
/* Exported: lexicographically smallest monic PRIMITIVE polynomial (reading G7). */
int orc_smallest_primitive(uint32_t p, uint32_t n, uint32_t *out_mod) {
    if (n < 1 || n > ORC_MAXN) return -1;
    uint64_t cnt = 1;
    for (uint32_t i = 0; i < n; i++) cnt *= p;
    for (uint64_t e = 0; e < cnt; e++) {
        uint32_t mod[ORC_MAXN + 1];
        modulus_from_index(p, n, e, mod);
        if (modulus_is_primitive(p, n, mod)) {
            memcpy(out_mod, mod, (n + 1) * sizeof(uint32_t));
            return 0;
        }
    }
    return -2;
}
/* Exported: is this monic modulus primitive (brute-force order of t)? */
int orc_is_primitive(uint32_t p, uint32_t n, const uint32_t *mod) {
    if (n < 1 || n > ORC_MAXN) return -1;
    return modulus_is_primitive(p, n, mod);
}
/* Exported: product of two encoded elements in F_p[t]/(mod); used by the
 * not-gpu tests to check the LIBRARY's antilog/Zech tables against polynomial
 * arithmetic (the oracle itself never builds such tables). */
int64_t orc_mul_encoded(uint32_t p, uint32_t n, const uint32_t *mod, uint64_t a, uint64_t b) {
    if (n < 1 || n > ORC_MAXN) return -1;
    ring R; R.p = p; R.n = n; memcpy(R.mod, mod, (n + 1) * sizeof(uint32_t));
    elt ea = elt_from_int(&R, a), eb = elt_from_int(&R, b);
    elt c = elt_mul(&R, &ea, &eb);
    uint64_t v = 0;
    for (uint32_t i = n; i-- > 0;) v = v * p + c.d[i];
    return (int64_t)v;
}

/* --------------------------------------------------- F_q inside E = F_{q^k} */

typedef struct {
    ring E;               /* F_p[t]/(P_E), degree r*k */
    uint64_t Q;           /* #E */
    uint32_t q;
    elt *iota;            /* iota[c] = image of the F_q element encoded c */
} ext_field;

/* R_q(y) for y in E, R_q monic of degree r with F_p coefficients */
static elt eval_Rq(const ring *E, const uint32_t *Rq, uint32_t r, const elt *y) {
    elt acc = elt_one();                         /* leading coefficient 1 */
    for (uint32_t i = r; i-- > 0;) {
        acc = elt_mul(E, &acc, y);
        acc.d[0] = (acc.d[0] + Rq[i]) % E->p;
    }
    return acc;
}
static int ext_field_init(ext_field *F, uint32_t p, uint32_t r, uint32_t k) {
    uint32_t n = r * k;
    if (n > ORC_MAXN) return -1;
    F->E.p = p; F->E.n = n;
    if (orc_smallest_irreducible(p, n, F->E.mod)) return -2;
    F->Q = ring_size(&F->E);
    uint32_t q = 1;
    for (uint32_t i = 0; i < r; i++) q *= p;
    F->q = q;
    F->iota = (elt *)malloc((size_t)q * sizeof(elt));
    if (!F->iota) return -3;
    if (r == 1) {                                /* prime q: the residue is the constant polynomial */
        for (uint32_t c = 0; c < q; c++) { F->iota[c] = elt_zero(); F->iota[c].d[0] = c; }
        return 0;
    }
    uint32_t Rq[ORC_MAXN + 1];
    if (orc_smallest_primitive(p, r, Rq)) return -4;
    /* exhaustive search for a root rho of R_q in E */
    elt rho = elt_zero(); int found = 0;
    for (uint64_t e = 0; e < F->Q && !found; e++) {
        elt y = elt_from_int(&F->E, e);
        elt v = eval_Rq(&F->E, Rq, r, &y);
        if (elt_is_zero(&F->E, &v)) { rho = y; found = 1; }
    }
    if (!found) return -5;
    /* iota(sum a_i T^i) = sum a_i rho^i */
    for (uint32_t c = 0; c < q; c++) {
        elt acc = elt_zero(), pw = elt_one();
        uint32_t v = c;
        for (uint32_t i = 0; i < r; i++) {
            uint32_t a = v % p; v /= p;
            for (uint32_t j = 0; j < n; j++)
                acc.d[j] = (uint32_t)((acc.d[j] + (uint64_t)a * pw.d[j]) % p);
            pw = elt_mul(&F->E, &pw, &rho);
        }
        F->iota[c] = acc;
    }
    return 0;
}
static void ext_field_free(ext_field *F) { free(F->iota); F->iota = NULL; }

/* 1 + chi_E(y): 1 if y = 0, 2 if y a nonzero square (Euler), else 0 */
static uint32_t one_plus_chi(const ext_field *F, const elt *y) {
    if (elt_is_zero(&F->E, y)) return 1;
    elt e = elt_pow(&F->E, *y, (F->Q - 1) / 2);
    elt one = elt_one();
    return elt_eq(&F->E, &e, &one) ? 2u : 0u;
}

/* N_k for one curve: coefficient row c[0..2g+2] (encoded F_q elements). */
static uint32_t count_points(const ext_field *F, const uint16_t *c, uint32_t ncoef) {
    uint32_t N = 0;
    for (uint64_t e = 0; e < F->Q; e++) {
        elt x = elt_from_int(&F->E, e);
        elt acc = F->iota[c[ncoef - 1]];
        for (uint32_t i = ncoef - 1; i-- > 0;) {   /* Horner, Algorithm 1 line 8 */
            acc = elt_mul(&F->E, &acc, &x);
            acc = elt_add(&F->E, &acc, &F->iota[c[i]]);
        }
        N += one_plus_chi(F, &acc);                /* 1 for a zero, 2 for a nonzero square */
    }
    N += one_plus_chi(F, &F->iota[c[ncoef - 1]]);  /* points at infinity, f(inf) = c_{2g+2} */
    return N;
}

/* r0_k = #{x in F_{q^k} : f(x) = 0}, the affine zeros only: the input of "compute lambda from r0"
 * (Algorithm 1 line 18). */
static uint32_t count_roots(const ext_field *F, const uint16_t *c, uint32_t ncoef) {
    uint32_t N = 0;
    for (uint64_t e = 0; e < F->Q; e++) {
        elt x = elt_from_int(&F->E, e);
        elt acc = F->iota[c[ncoef - 1]];
        for (uint32_t i = ncoef - 1; i-- > 0;) {
            acc = elt_mul(&F->E, &acc, &x);
            acc = elt_add(&F->E, &acc, &F->iota[c[i]]);
        }
        N += (uint32_t)elt_is_zero(&F->E, &acc);
    }
    return N;
}

/* ------------------------------------------------- squarefree: gcd(f, f') over F_q */

typedef struct { int deg; elt c[ORC_MAXDEG + 1]; } fpoly;   /* deg = -1 for the zero polynomial */

static void fpoly_trim(const ring *K, fpoly *a) {
    while (a->deg >= 0 && elt_is_zero(K, &a->c[a->deg])) a->deg--;
}
/* a mod b, b nonzero */
static fpoly fpoly_rem(const ring *K, uint64_t q, fpoly a, const fpoly *b) {
    elt inv = elt_pow(K, b->c[b->deg], q - 2);
    while (a.deg >= b->deg) {
        elt f = elt_mul(K, &a.c[a.deg], &inv);
        int s = a.deg - b->deg;
        for (int i = 0; i <= b->deg; i++) {
            elt t = elt_mul(K, &f, &b->c[i]);
            for (uint32_t j = 0; j < K->n; j++)
                a.c[s + i].d[j] = (a.c[s + i].d[j] + K->p - t.d[j]) % K->p;
        }
        fpoly_trim(K, &a);
    }
    return a;
}
static int is_squarefree(const ring *K, uint64_t q, const uint16_t *c, uint32_t ncoef) {
    fpoly f, df;
    f.deg = (int)ncoef - 1;
    for (uint32_t i = 0; i < ncoef; i++) f.c[i] = elt_from_int(K, c[i]);
    fpoly_trim(K, &f);
    df.deg = f.deg - 1;
    for (int i = 1; i <= f.deg; i++) {              /* (i mod p) * c_i */
        uint32_t m = (uint32_t)i % K->p;
        for (uint32_t j = 0; j < K->n; j++)
            df.c[i - 1].d[j] = (uint32_t)(((uint64_t)f.c[i].d[j] * m) % K->p);
        for (uint32_t j = K->n; j < ORC_MAXN; j++) df.c[i - 1].d[j] = 0;
    }
    fpoly_trim(K, &df);
    /* Euclid; gcd(f, 0) = f (reading G14: f' = 0 means f is a p-th power) */
    fpoly a = f, b = df;
    while (b.deg >= 0) {
        fpoly r = fpoly_rem(K, q, a, &b);
        a = b; b = r;
    }
    return a.deg == 0;
}

/* ------------------------------------------------------------------ batch entry */

/*
 * coeffs[n][2g+3] row-major, coeffs[i][j] = coefficient of X^j (encoded F_q
 * element, < q).  out_counts[n][width] = (N_1..N_width); out_squarefree[n] in {0,1}
 * (may be NULL).  k_lo..k_hi (1-based, inclusive) selects which N_k are
 * computed (others are left untouched) so that tests can bound the cost.
 * Returns 0, or <0: -10 bad field, -11 coefficient >= q, -12 degree < 2g+1
 * (reading G13), -13 bad k range.  *threads_used reports OpenMP threads.
 */
int orc_count_range(uint32_t p, uint32_t r, uint32_t g, const uint16_t *coeffs, size_t n,
                    uint32_t k_lo, uint32_t k_hi, uint32_t width, uint32_t *out_counts,
                    uint8_t *out_squarefree, int nthreads, int *threads_used) {
    /* width = number of columns of out_counts; width > g lets a test ask for N_k beyond
     * the genus (the formula of PAPER.md:41 holds for every extension E). */
    if (p < 3 || r < 1 || g < 1 || 2 * g + 2 > ORC_MAXDEG) return -10;
    if (k_lo < 1 || k_hi > width || width >= ORC_MAXDEG || k_lo > k_hi + 1) return -13;
    uint32_t ncoef = 2 * g + 3;
    uint32_t q = 1;
    for (uint32_t i = 0; i < r; i++) q *= p;
    for (size_t i = 0; i < n; i++) {
        const uint16_t *c = coeffs + i * ncoef;
        for (uint32_t j = 0; j < ncoef; j++) if (c[j] >= q) return -11;
        if (c[ncoef - 1] == 0 && c[ncoef - 2] == 0) return -12;
    }
    ext_field F[ORC_MAXDEG];
    for (uint32_t k = k_lo; k <= k_hi; k++)
        if (ext_field_init(&F[k], p, r, k)) return -10;
    ring K; K.p = p; K.n = r;
    if (orc_smallest_primitive(p, r, K.mod)) return -10;
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#endif
    (void)nthreads;
#pragma omp parallel for schedule(dynamic, 1)
    for (long long i = 0; i < (long long)n; i++) {
        const uint16_t *c = coeffs + (size_t)i * ncoef;
        for (uint32_t k = k_lo; k <= k_hi; k++)
            out_counts[(size_t)i * width + (k - 1)] = count_points(&F[k], c, ncoef);
        if (out_squarefree) out_squarefree[i] = (uint8_t)is_squarefree(&K, q, c, ncoef);
    }
    for (uint32_t k = k_lo; k <= k_hi; k++) ext_field_free(&F[k]);
    if (threads_used) *threads_used = used;
    return 0;
}

/* out_roots[n][width], columns k_lo-1 .. k_hi-1: r0_k of every row (same argument rules as orc_count_range). */
int orc_roots_range(uint32_t p, uint32_t r, uint32_t g, const uint16_t *coeffs, size_t n,
                    uint32_t k_lo, uint32_t k_hi, uint32_t width, uint32_t *out_roots, int nthreads) {
    if (p < 3 || r < 1 || g < 1 || 2 * g + 2 > ORC_MAXDEG) return -10;
    if (k_lo < 1 || k_hi > width || width >= ORC_MAXDEG || k_lo > k_hi + 1) return -13;
    uint32_t ncoef = 2 * g + 3;
    uint32_t q = 1;
    for (uint32_t i = 0; i < r; i++) q *= p;
    for (size_t i = 0; i < n; i++) {
        const uint16_t *c = coeffs + i * ncoef;
        for (uint32_t j = 0; j < ncoef; j++) if (c[j] >= q) return -11;
        if (c[ncoef - 1] == 0 && c[ncoef - 2] == 0) return -12;
    }
    ext_field F[ORC_MAXDEG];
    for (uint32_t k = k_lo; k <= k_hi; k++)
        if (ext_field_init(&F[k], p, r, k)) return -10;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    (void)nthreads;
#pragma omp parallel for schedule(dynamic, 1)
    for (long long i = 0; i < (long long)n; i++) {
        const uint16_t *c = coeffs + (size_t)i * ncoef;
        for (uint32_t k = k_lo; k <= k_hi; k++)
            out_roots[(size_t)i * width + (k - 1)] = count_roots(&F[k], c, ncoef);
    }
    for (uint32_t k = k_lo; k <= k_hi; k++) ext_field_free(&F[k]);
    return 0;
}

int orc_count(uint32_t p, uint32_t r, uint32_t g, const uint16_t *coeffs, size_t n,
              uint32_t *out_counts, uint8_t *out_squarefree, int nthreads, int *threads_used) {
    return orc_count_range(p, r, g, coeffs, n, 1, g, g, out_counts, out_squarefree, nthreads, threads_used);
}
