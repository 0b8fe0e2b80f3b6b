/*
 * hec.h -- C ABI of libhec: batched naive Hasse-Weil point counts of hyperelliptic
 * curves y^2 = f(x) over small finite fields in Zech-logarithm representation
 * (arXiv 1805.11991, M. Raum; citations are /root/reference/PAPER.md:<line>).
 *
 * Conventions shared by every call
 *   - extern "C", plain pointers and sizes, no exceptions or aborts cross the ABI.
 *   - Every int-returning call returns HEC_OK (0) or a negative hec_status;
 *     hec_last_error() returns a thread-local, NUL-terminated description of the
 *     last failure on the calling thread (valid until the next failing call).
 *   - "host or device" pointers are classified with cudaPointerGetAttributes.  All
 *     array arguments of one call must live on the same side.  Device work is
 *     enqueued on the stream given to hec_set_stream (default: the legacy default
 *     stream) and the call returns after that work has completed (it synchronises
 *     the stream, because the status code depends on device-side validation).
 *   - The caller owns every buffer it passes in; the library owns hec_field handles
 *     and its internal per-(q,g) device plans (released by hec_shutdown).
 *   - ONE GPU PER PROCESS: the library's state (table plans, staging buffers, the
 *     histogram pool) lives on the CUDA device that is current at the first call that
 *     touches the device.  A later call with another current device fails with
 *     HEC_ERR_INVALID_ARG; hec_shutdown() releases everything, after which the next
 *     call binds to the device current then.
 *   - An F_q element (q = p^r, p an odd prime) is the integer sum a_i p^i, which
 *     stands for sum a_i T^i in F_p[T]/(R_q) (little-endian base-p digits,
 *     PAPER.md:199); R_q is the lexicographically smallest monic primitive
 *     polynomial of degree r over F_p, ordering the tuple (a_{r-1}, ..., a_0)
 *     (reading G7).  For prime q this is the plain residue.
 */
#ifndef HEC_H
#define HEC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum hec_status {
    HEC_OK = 0,
    HEC_ERR_INVALID_FIELD = -1,   /* p not an odd prime, r or k < 1, q^k above HEC_MAX_FIELD_SIZE */
    HEC_ERR_INVALID_ARG = -2,     /* NULL pointer, g < 1, g above HEC_MAX_GENUS, mixed host/device pointers */
    HEC_ERR_COEFF_RANGE = -3,     /* some coefficient >= q; hec_last_error_index() = first offending row */
    HEC_ERR_DEGREE = -4,          /* some row has c[2g+2] = c[2g+1] = 0 (degree < 2g+1) */
    HEC_ERR_CAPACITY = -5,        /* hec_histogram: cap < number of distinct tuples (*out_m is still set);
                                     hec_histogram_static: also n above HEC_HISTOGRAM_STATIC_MAX_ROWS */
    HEC_ERR_UNSUPPORTED = -6,     /* hec_histogram: the tuple does not pack into 64 bits */
    HEC_ERR_CUDA = -7,            /* a CUDA runtime call failed, or no device is present */
    HEC_ERR_NOMEM = -8
} hec_status;

#define HEC_MAX_FIELD_SIZE (1u << 26)   /* largest supported q^k */
#define HEC_MAX_GENUS 5u

const char *hec_last_error(void);
/* Row index attached to the last HEC_ERR_COEFF_RANGE / HEC_ERR_DEGREE on this thread, else (size_t)-1. */
size_t hec_last_error_index(void);

/* ------------------------------------------------------------------------------------------------
 * hec_build_field -- section 2.3 and 3.1-3.2.
 *
 * Builds F_{q^k}, q = p^r, entirely on the host (no CUDA call): picks the lexicographically
 * smallest monic primitive polynomial P of degree n = r*k over F_p (reading G7), takes alpha = t as
 * the generator g_q of PAPER.md:203, and tabulates
 *   antilog[i] = encoding of alpha^i                       0 <= i <= Q-2
 *   log[e]     = i with antilog[i] = e, log[0] = Q-1        0 <= e <= Q-1     (encoding (3.1))
 *   zech[i]    = m(i) with alpha^m(i) = 1 + alpha^i, or Q-1 if 1 + alpha^i = 0   (table (3.2))
 *   embed[c]   = log of the image in F_{q^k} of the F_q element encoded c, embed[0] = Q-1
 *                (F_q -> F_{q^k} sends T to rho = alpha^(s (Q-1)/(q-1)), s the smallest unit mod q-1
 *                 with R_q(rho) = 0; reading G6: NOT simply c's log times (Q-1)/(q-1))
 * Returns NULL on failure (hec_last_error says why).  The handle is immutable and may be shared
 * between threads; release it with hec_free_field.
 */
typedef struct hec_field hec_field;
hec_field *hec_build_field(uint32_t p, uint32_t r, uint32_t k);
void hec_free_field(hec_field *F);

/* hec_build_field_device -- the same field, with the tables built by CUDA kernels (the "tables" column of the
 * paper's Table 1: the precomputation that dominates a single large-p curve).
 * The modulus is found on the host by order tests (t^(Q-1) = 1, t^((Q-1)/l) != 1 for every prime l | Q-1); the
 * antilog / log / Zech tables are computed on the current device and stream (hec_set_stream) and copied into the
 * handle, so every accessor above works unchanged.  The result equals hec_build_field(p, r, k) entry for entry.
 * Needs a CUDA device (NULL + HEC_ERR_CUDA message otherwise; no host fallback) and p < 65536.
 * hec_count builds its own fields this way when q^k > 65536. */
hec_field *hec_build_field_device(uint32_t p, uint32_t r, uint32_t k);

/* Read-only accessors (paper's conventions: logs in [0, Q-2], zero <-> Q-1).  The out arrays are HOST
 * arrays owned by the caller with the stated number of elements.  A NULL field returns 0 / does nothing. */
uint32_t hec_field_p(const hec_field *F);
uint32_t hec_field_degree(const hec_field *F);                 /* n = r*k */
uint32_t hec_field_q(const hec_field *F);                      /* size of the base field */
uint32_t hec_field_Q(const hec_field *F);                      /* size of the field, q^k */
uint32_t hec_field_embed_unit(const hec_field *F);             /* s above (1 when k = 1) */
void hec_field_modulus(const hec_field *F, uint32_t *out);     /* n+1 coefficients a_0..a_{n-1}, 1 */
void hec_field_antilog(const hec_field *F, uint32_t *out);     /* Q-1 entries */
void hec_field_log(const hec_field *F, uint32_t *out);         /* Q entries */
void hec_field_zech(const hec_field *F, uint32_t *out);        /* Q-1 entries */
void hec_field_embed(const hec_field *F, uint32_t *out);       /* q entries */

/* ------------------------------------------------------------------------------------------------
 * hec_count -- Algorithm 1 lines 6-14 for a whole batch of curves, plus the
 * points at infinity and x = 0 and the squarefree filter.
 *
 *   coeffs[n][2g+3]   row-major uint16, coeffs[i][j] = coefficient of X^j of curve i (F_q encoding above)
 *   out_counts[n][g]  uint32, row i = (N_1 .. N_g), N_k = #C_f(F_{q^k})
 *                       = #{x: f(x)=0} + 2 #{x: f(x) a nonzero square} + (1 if c_{2g+2}=0;
 *                         2 if c_{2g+2} a nonzero square in F_{q^k}; else 0)
 *   out_squarefree[n] uint8 in {0,1}: deg gcd(f, f') = 0 over F_q; may be NULL
 * N_k is computed by the same formula whether or not f is squarefree (reading G12).
 * Pointers: all host or all device.  Host pointers: the library stages the batch through its own
 * device buffers; from 2^20 rows on, in four chunks through two internal copy streams, so that the H2D copy of
 * chunk i+1 and the D2H copies of chunk i-1 run under the kernels of chunk i (pinned host memory overlaps;
 * pageable memory is staged by the driver and is merely slower).  n = 0 is a no-op.
 * Errors: HEC_ERR_INVALID_FIELD (q not an odd prime power below 65536, q^g too large),
 * HEC_ERR_INVALID_ARG, HEC_ERR_COEFF_RANGE, HEC_ERR_DEGREE (outputs are unspecified after these
 * two), HEC_ERR_CUDA, HEC_ERR_NOMEM.
 */
int hec_count(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n,
              uint32_t *out_counts, uint8_t *out_squarefree);

/* ------------------------------------------------------------------------------------------------
 * hec_histogram -- the multiplicity map of eq. (1.2) / Algorithm 1 line 20
 * in its reduced form: unweighted, keyed by the tuple (N_1..N_g) only.
 *
 *   counts[n][g]      uint32 rows (typically hec_count's output)
 *   mask[n]           uint8 or NULL; rows with mask 0 are skipped (the paper counts squarefree f only)
 *   out_tuples[cap][g], out_mult[cap]   distinct rows in ASCENDING LEXICOGRAPHIC order + multiplicities
 *   *out_m            number of distinct rows (HOST pointer, always written on HEC_OK / HEC_ERR_CAPACITY)
 * Two-call pattern: if cap < *out_m nothing is written to out_tuples/out_mult and HEC_ERR_CAPACITY is
 * returned; out_tuples/out_mult may be NULL when cap = 0.  counts/mask/out_tuples/out_mult: all host or
 * all device.  Sum of out_mult = number of unmasked rows.  HEC_ERR_UNSUPPORTED if the per-column
 * ranges (max - min) need more than 64 bits in total.
 */
int hec_histogram(const uint32_t *counts, const uint8_t *mask, size_t n, uint32_t g,
                  uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m);

/*
 * hec_count_histogram -- one pass of the whole hot path in ONE call: hec_count followed by hec_histogram of the rows
 * with a nonzero squarefree flag (of every row when out_squarefree is NULL).  Arguments as in hec_count and
 * hec_histogram (same capacity protocol: on HEC_ERR_CAPACITY out_counts / out_squarefree are complete and only the
 * histogram has to be repeated, e.g. with hec_histogram).  All array pointers host or all device.  With host
 * pointers the counts never make the round trip: the histogram runs on the device copies while the last D2H copies
 * of the counts are still in flight, and only the distinct tuples come back.
 */
int hec_count_histogram(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t *out_counts,
                        uint8_t *out_squarefree, uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m);

/*
 * hec_histogram_merge -- the one exchange step of the multi-GPU path: merges partial
 * histograms.  in_tuples[n][g] with multiplicities in_mult[n] (tuples may repeat, e.g. the concatenation of
 * several ranks' hec_histogram outputs; entries with multiplicity 0 are ignored) -> distinct tuples in
 * ascending lexicographic order with summed multiplicities.  Same pointer, capacity and error rules as
 * hec_histogram.
 */
int hec_histogram_merge(const uint32_t *in_tuples, const uint64_t *in_mult, size_t n, uint32_t g,
                        uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m);

/*
 * hec_histogram_static -- hec_histogram (same map, eq. (1.2) / Algorithm 1 line 20; same output order)
 * for callers that must not allocate device memory.  hec_histogram takes its hash table and sort buffers from a pool
 * that calls cudaMalloc when it has to grow.  That is no good in a process where another component (a tensor
 * framework's caching allocator, a serving engine) has already claimed almost all device memory -- the allocation
 * fails or takes memory that was promised elsewhere -- nor where the device-wide synchronisation inside cudaMalloc /
 * cudaFree would stall streams that do not belong to this library.  This entry point calls no cudaMalloc, cudaFree or
 * other allocating routine, on any call: all of its scratch lives in one fixed array inside the library's device image
 * (about 8.07 MiB; every GPU on which the process uses CUDA with libhec loaded carries it until the process exits).
 *
 *   n <= HEC_HISTOGRAM_STATIC_MAX_ROWS (2^17 rows), else HEC_ERR_CAPACITY with a message that names the limit
 *       (*out_m = 0; nothing is computed).  Larger batches: call per slice, then hec_histogram_merge where allowed.
 *   counts[n][g], mask[n] (or NULL), out_tuples[cap][g], out_mult[cap]: DEVICE pointers, owned by the caller (host arrays
 *       would need a staging allocation and are refused with HEC_ERR_INVALID_ARG); *out_m: host pointer.
 *   Capacity protocol, output order and the remaining errors as in hec_histogram.
 * Set-up: the first call on a device looks up the array's device address (cudaGetSymbolAddress, with that device
 * current) and the SM count and keeps them; make that first call ahead of any stream capture.  It does not bind the
 * library to a device and needs no other libhec call before it.
 * Sharing: every call on a device uses the same array, which still holds what the previous call left there (the call
 * resets what it needs).  Two calls whose device work overlaps -- different streams (hec_set_stream), different host
 * threads -- race on it and give garbage; run them one after the other.  Work is enqueued on the hec_set_stream stream
 * and the call returns after synchronising that stream.
 */
#define HEC_HISTOGRAM_STATIC_MAX_ROWS 131072
int hec_histogram_static(const uint32_t *counts, const uint8_t *mask, size_t n, uint32_t g,
                         uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m);

/* ------------------------------------------------------------------------------------------------
 * Algorithm 1 around the hot path, without the partition lambda: SURVEY.md 8(f) NEXT-1.
 *
 * hec_reduced_total / hec_reduced_rows -- the reduced polynomials P~'_d(F_q) of sections 1.2-1.3,
 * BEFORE the squarefree filter, generated by a kernel from their index (no input in HBM), d = 2g+1 or 2g+2.
 * A stratum fixes the coefficients at and above `top` and normalises the support below `top` by X -> aX, f -> f/e^2:
 *   p not dividing d: one stratum, c_{d-1} = 0 by the shift X -> X - c_{d-1}/(d c_d), top = d-1, group order q(q-1)^2;
 *   p | d (reading G19: the printed set, misses every polynomial with c_{d-1} = 0 != c_{d-2}):
 *       stratum c_{d-1} != 0: c_{d-2} = 0 by the shift (as printed), top = d-2, c_{d-1} = 1..q-1, group order q(q-1)^2;
 *       stratum c_{d-1} = 0:  no shift (a shift cannot change c_{d-1}), top = d-1, group {(a,0,e)} of order (q-1)^2.
 * Inside a stratum (c_d = 1..q-1 throughout):
 *   family A0   .. + 1                                                        mult |group| / (2(q-1))
 *   family A1   .. + X   (if 1 < top)                                         mult |group| / (2(q-1))   (reading G18: the
 *               printed set omits the support {d, 1}; without it the map misses these curves)
 *   families B(i,j), 1 <= i < top, 0 <= j < i:  .. + X^i + c_j X^j + c_{j-1} X^{j-1} + .. + c_0,
 *               c_j = alpha^s, s < gamma = gcd(q-1, i-j), c_{j-1}..c_0 in F_q    mult |group| / (2 gamma)
 *   (reading G9: i and j are the two LARGEST indices below top with nonzero coefficient).
 * Index order: strata as listed; A0, A1, then B(i,j) with j fastest; inside a family
 *   (((c_d - 1) n1 + (c_{d-1} - 1)) gamma + s) q^j + sum_{l<j} c_l q^l   (n1 = q-1 in the stratum c_{d-1} != 0, else the
 *   c_{d-1} term is absent).
 *   out_coeffs[n][2g+3] uint16 (layout of hec_count), out_mult[n] uint64 = mult(f); both host or both device.
 * Errors: HEC_ERR_INVALID_ARG (d, index range), HEC_ERR_UNSUPPORTED (more than 2^64 polynomials), HEC_ERR_CUDA.
 *
 * hec_curve_map -- N_{g,d}: for every reduced f (in chunks of 2^24 rows, hec_set_map_chunk_rows: rows kernel -> hec_count -> weighted
 * histogram of the squarefree rows), add mult(f) at (N_1..N_g) and at the tuple of the quadratic twist n f
 * (Algorithm 1 lines 19-21; reading G8: N_k -> 2 q^k + 2 - N_k for odd k, N_k for even k).  The result equals
 * #{f squarefree of degree d over F_q with that tuple} (eq. (1.2) without lambda).  Output as for hec_histogram:
 * ascending lexicographic tuples, uint64 weights, two-call capacity protocol (*out_m always set).
 */
/* ------------------------------------------------------------------------------------------------
 * lambda(f): SURVEY.md 8(f) NEXT-3 (Algorithm 1 line 18: "compute lambda from r0 if
 * possible; otherwise by factoring").
 *
 * hec_count_ex = hec_count plus two optional outputs (same pointer rules; NULL = not wanted):
 *   out_roots[n][g]  uint32  r0_k = #{x in F_{q^k} : f(x) = 0}, the affine zeros
 *   out_lambda[n]    uint8   index (hec_lambda_partitions) of the factorisation type of f over F_q: the partition
 *                            of 2g+2 into the degrees of the irreducible factors, for degree 2g+1 amended by a summand 1
 *                            (PAPER.md:61); 0xFF when f is not squarefree.
 * How: r0_k = sum_{e | k} e n_e (n_e = number of irreducible factors of degree e), so Moebius inversion gives n_e for
 * e <= g; the rest of the degree is one irreducible factor, except when it is 2g+2 (no factor of degree <= g): then
 * Stickelberger's theorem decides between "irreducible" and "two factors of degree g+1" by the quadratic character
 * of disc(f), which the squarefree kernel's Euclid run on (f, f') yields for free -- no factoring is ever needed.
 *
 * hec_lambda_partitions: the partitions of 2g+2 as multiplicity vectors (n_1 .. n_{2g+2}), out_parts[count][2g+2],
 * in ascending lexicographic order of that vector; the row number is the lambda index.  Two-call capacity protocol.
 * Host pointers only; needs no device.
 *
 * hec_curve_map_lambda: hec_curve_map with the full key of the paper's map (1.2), PAPER.md:63-67:
 * out_keys[m][g+1] = (N_1 .. N_g, lambda index); g <= HEC_MAX_GENUS - 1.
 */
int hec_count_ex(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t *out_counts, uint8_t *out_squarefree,
                 uint32_t *out_roots, uint8_t *out_lambda);
int hec_lambda_partitions(uint32_t g, uint8_t *out_parts, size_t cap, size_t *out_count);
int hec_curve_map_lambda(uint32_t q, uint32_t g, uint32_t d, uint32_t *out_keys, uint64_t *out_weights, size_t cap, size_t *out_m);

int hec_reduced_total(uint32_t q, uint32_t g, uint32_t d, uint64_t *out_total);
int hec_reduced_rows(uint32_t q, uint32_t g, uint32_t d, uint64_t first, size_t n, uint16_t *out_coeffs, uint64_t *out_mult);
int hec_curve_map(uint32_t q, uint32_t g, uint32_t d, uint32_t *out_tuples, uint64_t *out_weights, size_t cap, size_t *out_m);
/* Algorithm 1 in full (line 2: "for d in {2g+1, 2g+2}"): the merge of the maps of both degrees, N_{g,q}.
 * With lambda the two degrees stay apart where their types differ (degree 2g+1 carries the extra summand 1). */
int hec_curve_map_all(uint32_t q, uint32_t g, int with_lambda, uint32_t *out_keys, uint64_t *out_weights, size_t cap, size_t *out_m);
/* The multi-GPU form: the contribution of the reduced polynomials with index in [first, first + n) --
 * their tuples AND their twists' -- so that the map is the hec_histogram_merge of the ranks' outputs over a partition of
 * [0, hec_reduced_total).  with_lambda != 0: keys have g+1 columns as in hec_curve_map_lambda. */
int hec_curve_map_range(uint32_t q, uint32_t g, uint32_t d, uint64_t first, uint64_t n, int with_lambda, uint32_t *out_keys,
                        uint64_t *out_weights, size_t cap, size_t *out_m);
/* Rows per chunk of hec_curve_map / hec_curve_map_lambda (default 2^24; device memory per chunk is about 90 B per row). */
int hec_set_map_chunk_rows(size_t rows);

/* ------------------------------------------------------------------------------------------------
 * Execution control and instrumentation (used by the tests, bench.py and the ncu runs).
 */
/* cudaStream_t (as void*) on which later calls enqueue their device work; NULL = default stream. */
int hec_set_stream(void *cuda_stream);

typedef enum hec_regime {
    HEC_REGIME_AUTO = 0,       /* per field: full table in shared memory if it fits (Horner: extended 16-bit table; radix:
                                  2x16-bit pair table), else a half table (Z(-n) = Z(n) - n; 32-bit, else 16+8-bit / 16+1-bit
                                  planes) in shared memory if it fits, else the L2-resident table */
    HEC_REGIME_SMEM = 1,       /* force the full shared-memory table for the largest field (HEC_ERR_INVALID_ARG
                                  when it cannot fit) */
    HEC_REGIME_L2 = 2,         /* force the L2-resident (global memory, 32-bit words) table for the largest field */
    HEC_REGIME_SMEM_HALF = 3   /* force the shared-memory half table for the largest field (HEC_ERR_INVALID_ARG when
                                  it cannot fit or the field has fewer than 2^13 elements) */
} hec_regime;
int hec_set_regime(int regime);

/* Evaluation scheme of hec_count (results are identical; f is evaluated at every x either way). */
typedef enum hec_eval {
    HEC_EVAL_AUTO = 0,         /* radix-R split (not in the paper): with R in {2, 4, 8} the largest power of two dividing
                                  q^k - 1 (capped per table layout), f(X) = sum_{r<R} X^r F_r(X^R): the R points x zeta^j of a
                                  coset of the R-th roots of unity share the R Horner chains F_r(x^R) and are combined by an
                                  R-point butterfly network of Zech additions, one table entry serving a + w b and a - w b
                                  (about 5x fewer lookups at degree 10).  Tables: pairs (Z[n], Z[n + M/2]) or half tables. */
    HEC_EVAL_HORNER = 1,       /* the paper's scheme (Algorithm 1 line 8): one Horner chain per x */
    HEC_EVAL_RADIX2 = 2,       /* as AUTO with R capped at 2 / 4 / 8 (tuning and tests); no loop runs above the cap: the
                                  R = 16 monomial-class loop for rows of 9..16 coefficients is AUTO's alone */
    HEC_EVAL_RADIX4 = 4,
    HEC_EVAL_RADIX8 = 8,
    HEC_EVAL_ORBIT = 16        /* as AUTO, but one representative per Frobenius orbit of x (f(x^q) = f(x)^q for f over F_q),
                                  each count weighted by the orbit length: the same N_k from about 1/k of the evaluations
                                  (not the paper's "every x" loop, so never the default) */
} hec_eval;
int hec_set_eval(int eval);

/* Statistics of the last hec_count of the process (the library state is ONE process-global object behind a mutex,
 * not per thread: with several host threads this is whichever hec_count finished last): device time of the count kernel(s) and
 * of the squarefree kernel (CUDA events on the launch stream, ms), number of kernel launches (one count
 * launch per group of fields whose tables share one shared-memory image, plus the squarefree kernel), the
 * regime used for the largest field (hec_regime) and its table layout -- Horner kernel: 0 global 32-bit
 * extended, 1 shared 16-bit extended, 2 shared 32-bit half, 3 shared 16+8-bit half; radix kernel: 4 shared
 * 2x16-bit pairs, 5 shared 32-bit half, 6 shared 16+1-bit half, 7 global 2x32-bit pairs --, the largest
 * dynamic shared memory per CTA, grid and block size of the last count launch, independent x (Horner) or
 * cosets (radix) per lane per pass, and the radix of every field. */
typedef struct hec_count_stats {
    float count_kernel_ms;     /* chunks == 1: the count launch(es) alone.  chunks > 1 (host-pointer calls from 2^20 rows on): from
                                  the first chunk's launch to the end of the last chunk's count kernel, which includes the
                                  waits for the H2D copies and the squarefree kernels of the earlier chunks -- a span, not a
                                  kernel time; time kernels on device-resident inputs */
    float squarefree_kernel_ms;/* chunks > 1: the last chunk's squarefree kernel only */
    uint32_t launches;
    uint32_t regime;
    uint32_t smem_bytes;
    uint32_t grid;
    uint32_t block;
    uint32_t chains_per_lane;
    uint32_t table_mode;
    uint32_t radix_fields;     /* nibble k-1: radix R used for N_k (0: one Horner chain per x) */
    uint32_t splits;           /* warps per curve: 1 for batches; > 1 when a small batch (down to a single curve) is spread
                                  over the whole GPU, each warp taking a slice of the x range of every field */
    uint32_t fast_fields;      /* bit k-1: field k carried fast tables or a parity table (hec_set_fast_tables) */
    uint32_t chunks;           /* host-pointer calls: number of row chunks pipelined through the copy streams (1: none) */
} hec_count_stats;
int hec_last_count_stats(hec_count_stats *out);

/* Shift pre-pass of the radix evaluation (on by default; hec_set_shift(0) turns it off -- tests run both).
 * N_k(f) = N_k(f(X + t)) for every t in F_q: x -> x + t permutes each F_{q^k}, and the leading coefficient (points at
 * infinity), the root counts and the factorisation type do not change.  The radix-R evaluation takes its straight-line
 * network only when every residue class of exponents mod R holds a nonzero coefficient; before counting, hec_count
 * therefore replaces each row that has an empty class mod R (R = the radix of the largest field, when it is 4 or 8 and the
 * rows have at least R coefficients) by the first f(X + alpha^s), s = 0 .. 7, without one.  The squarefree flag and lambda
 * are computed from the original rows.
 * hec_shift_rows exposes that pre-pass: out_coeffs[n][2g+3] = the rows hec_count evaluates (coeffs itself where no
 * pre-pass applies); both host or both device pointers. */
int hec_set_shift(int on);
int hec_shift_rows(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint16_t *out_coeffs);

/* Fast tables of the radix evaluation (on by default; hec_set_fast_tables(0) turns them off -- tests run both, the counts
 * are identical).  A shared-memory field stored as pairs (Z[n], Z[n + M/2]) also gets, when the launch's shared memory has
 * room, (i) a copy of Z transposed by residue mod R, T[c][j] = Z[c + R j], which serves the first lookup of every
 * residue-class chain of Algorithm 1 line 8 -- there lane l reads Z[delta + R (n0 + l)], R words apart in the
 * plain table (an R-way bank conflict) and consecutive entries of one row of T -- and (ii) e n mod M for the lanes' first
 * cosets and the step 64 e mod M, e = 0 .. 2g+2, so that the per-curve set-up needs no modular reduction.  A top field stored as a
 * half table (Z[0 .. M/2]) gets (iii) a packed parity table, 2 bits per n (parity of Z[n], of Z[n + M/2]), which the last stage of
 * the evaluation -- it only classifies, PAPER.md:145-147 -- reads instead of the two or three loads of a pair.  With these tables, rows
 * whose coefficients up to the degree are all nonzero run loops specialised on "one term per residue class" (at most 8 coefficients
 * and 8 | M, or at most 16 and 16 | M; the shift pre-pass then asks for every coefficient to be nonzero).
 * hec_count_stats.fast_fields: bit k-1 set iff field k carried such tables in the last call.  Takes effect on the next plan build
 * for a (q, g) (the setting is part of the plan key). */
int hec_set_fast_tables(int on);

/* Representation independence ("rerun with another primitive polynomial -- every N_k identical").
 * v = 0 (default): the library's own fields F_{q^k} are built on the lexicographically smallest primitive polynomial
 * (reading G7); v > 0: on the (v+1)-th smallest, i.e. another generator alpha, other log / Zech / embedding tables.
 * Every output of hec_count / hec_count_ex / hec_curve_map must be unchanged.  F_q itself (k = 1) keeps its smallest
 * polynomial: for q = p^r, r > 1 it fixes the encoding of the inputs, and the reduced polynomials of Algorithm 1 are
 * defined through its generator.  hec_build_field / hec_build_field_device always return the smallest.
 * Drops the cached plans; v <= 16.  The setting is checked when a field is built: if F_{q^k} has no more than v primitive
 * polynomials of its degree (F_9 has two), the next hec_count fails with HEC_ERR_INVALID_FIELD and a message that names
 * the variant.  hec_shutdown() puts the setting back to 0. */
int hec_set_field_variant(uint32_t v);

/* Total number of kernels launched by this library since load (bench.py's gpu_launches). */
uint64_t hec_launch_count(void);

/*
 * Gather micro-benchmark for the lookup ceilings: every lane follows a dependent chain
 * idx <- table[idx] + warp-uniform offset + lane term (the count kernel's inner step) through a table of
 * `entries` uniformly random entries of `entry_bytes` (2 or 4) bytes; with 2-byte entries and more than
 * 65536 + 256 entries the uniform offset rotates so that the whole footprint is touched.  where = 0: shared memory; 1: global memory through L1 (ld.global.nc);
 * 2: global memory bypassing L1 (ld.global.cg).  Runs `lookups_per_lane` dependent lookups on each of
 * `chains` independent chains per lane with one CTA of `block` threads per SM times `ctas_per_sm`,
 * and writes lookups per second and the kernel time.  Table contents are seeded.
 */
int hec_gather_bench(int where, uint32_t entries, uint32_t entry_bytes, uint32_t block, uint32_t ctas_per_sm,
                     uint32_t chains, uint32_t lookups_per_lane, double *out_lookups_per_s, float *out_ms);

/* Release cached fields, device plans, staging buffers, the histogram pool and the internal streams and events; the next
 * call binds to the device that is current then.  Two settings are tied to what is released and go back to their
 * defaults: the stream (hec_set_stream: a stream of the old device is not a valid handle on another one) becomes the
 * default stream, the field variant becomes 0.  hec_set_regime / hec_set_eval / hec_set_shift / hec_set_fast_tables /
 * hec_set_map_chunk_rows persist.  The fixed scratch array of hec_histogram_static is not released (it is part of the
 * module image). */
void hec_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* HEC_H */
