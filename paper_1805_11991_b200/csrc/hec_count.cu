// hec_count / hec_count_ex: host side (plan builder, staging, error reporting) and the small per-curve kernels
// (squarefree flag + lambda, shift pre-pass).  The count kernels themselves are in hec_count_kernels.cuh.
#include "hec_count_kernels.cuh"

uint64_t hec_launch_counter::value = 0;
void hec_histogram_release_pool();

namespace {

// --------------------------------------------------------------------------------------------
// a6: squarefree flag, deg gcd(f, f') = 0 over F_q, one thread per curve, Euclid's
// algorithm with F_q elements as logs (zero = M) and the k = 1 Zech table (addition law of reading G5).
// --------------------------------------------------------------------------------------------
constexpr int kSqMaxCoef = 2 * HEC_MAX_GENUS + 3;

struct FqLog {
    uint32_t M;
    const uint32_t *zech;
    __device__ __forceinline__ uint32_t mul(uint32_t a, uint32_t b) const {
        if (a == M || b == M) return M;
        uint32_t s = a + b;
        return s >= M ? s - M : s;
    }
    __device__ __forceinline__ uint32_t inv(uint32_t a) const { return a == 0 ? 0 : M - a; }
    __device__ __forceinline__ uint32_t neg(uint32_t a) const {
        if (a == M) return M;
        uint32_t s = a + (M >> 1);                    // -1 = alpha^{M/2}
        return s >= M ? s - M : s;
    }
    __device__ __forceinline__ uint32_t add(uint32_t a, uint32_t b) const {
        if (a == M) return b;
        if (b == M) return a;
        uint32_t d = b >= a ? b - a : b + M - a;
        uint32_t z = __ldg(zech + d);
        if (z == M) return M;
        uint32_t s = a + z;
        return s >= M ? s - M : s;
    }
};

__global__ void __launch_bounds__(256) hec_squarefree_kernel(const HecSquarefreeParams P) {
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const FqLog K{P.M, P.zech};
    const uint32_t ZERO = P.M;
    uint32_t a[kSqMaxCoef], b[kSqMaxCoef];
    int da = -1, db = -1;
    const uint16_t *row = P.coeffs + i * P.ncoef;
    bool ok = true;
    for (uint32_t j = 0; j < P.ncoef; j++) {
        const uint32_t cj = row[j];
        if (cj >= P.q) { ok = false; break; }
        const uint32_t l = cj ? __ldg(P.emb + cj) : ZERO;
        a[j] = l;
        if (l != ZERO) da = (int)j;
        // derivative: (j mod p) * c_j, the integer j mod p being the prime-field element encoded j mod p
        if (j >= 1) {
            const uint32_t jm = j % P.p;
            const uint32_t lj = jm ? __ldg(P.emb + jm) : ZERO;
            const uint32_t t = K.mul(l, lj);
            b[j - 1] = t;
            if (t != ZERO) db = (int)j - 1;
        }
    }
    if (!ok || da < (int)P.ncoef - 2) {                              // reported by the count kernel
        if (P.out) P.out[i] = 0;
        if (P.out_lambda) P.out_lambda[i] = 0xFF;
        return;
    }
    // Euclid: gcd(f, 0) = f (reading G14).  Alongside, the parity of log Res(f, f') (the quadratic character of the
    // resultant: Res(A, B) = (-1)^{deg A deg B} lc(B)^{deg A - deg R} Res(B, R) for R = A mod B, Res(A, b) = b^{deg A}),
    // needed by lambda below.
    const int d = da, d1 = db;
    const uint32_t lcf = a[da];
    const uint32_t par_m1 = (P.M >> 1) & 1u;                         // -1 = alpha^{M/2}
    uint32_t par = 0;
    while (db >= 0) {
        const int m = da, nn = db;
        const uint32_t lb = b[db];
        // a <- a mod b
        const uint32_t binv = K.inv(b[db]);
        while (da >= db) {
            const uint32_t fac = K.neg(K.mul(a[da], binv));
            const int s = da - db;
            for (int t = 0; t < db; t++) a[s + t] = K.add(a[s + t], K.mul(fac, b[t]));
            a[da] = ZERO;
            while (da >= 0 && a[da] == ZERO) da--;
        }
        if (nn == 0) par ^= (uint32_t)m & lb & 1u;
        else if (da >= 0) par ^= (((uint32_t)(m * nn) & 1u) & par_m1) ^ ((uint32_t)(m - da) & lb & 1u);
        // swap (a, b)
        for (int t = 0; t < (int)kSqMaxCoef; t++) { const uint32_t x = a[t]; a[t] = b[t]; b[t] = x; }
        const int td = da; da = db; db = td;
    }
    const bool squarefree = da == 0;
    if (P.out) P.out[i] = squarefree ? 1 : 0;
    if (!P.out_lambda) return;
    if (!squarefree) { P.out_lambda[i] = 0xFF; return; }
    // lambda(f) (Algorithm 1 line 18: "from r0 if possible; otherwise by factoring").  An irreducible factor
    // of degree e has its e roots in F_{q^k} iff e | k, so r0_k = sum_{e | k} e n_e and Moebius inversion gives n_e for
    // e <= g.  The rest of the degree is ONE irreducible factor unless it is 2g+2 (no factor of degree <= g at all): then
    // f is irreducible or a product of two irreducibles of degree g+1, and Stickelberger's theorem decides without
    // factoring: the number of irreducible factors is congruent to deg f mod 2 iff disc(f) is a square, where
    // disc(f) = (-1)^{d(d-1)/2} lc(f)^{-(d + deg f')} Res(f, f') up to squares.
    const uint32_t *r0 = P.roots + i * P.g;
    int ne[kSqMaxCoef];
    for (int e = 0; e < (int)kSqMaxCoef; e++) ne[e] = 0;
    int rest = d;
    for (int e = 1; e <= (int)P.g; e++) {
        const int sub = e == 1 ? 0 : (e == 4 ? (int)r0[1] : (int)r0[0]);     // e = 2, 3, 5: r0_e - r0_1; e = 4: r0_4 - r0_2
        ne[e] = ((int)r0[e - 1] - sub) / e;
        rest -= e * ne[e];
    }
    if (rest == 2 * (int)P.g + 2) {
        const uint32_t par_disc = par ^ (((uint32_t)(d * (d - 1) / 2) & 1u) & par_m1) ^ ((uint32_t)(d + d1) & lcf & 1u);
        if (par_disc == 0) ne[P.g + 1] = 2; else ne[rest] = 1;
    } else if (rest > 0) {
        ne[rest] = 1;
    }
    if (d == 2 * (int)P.g + 1) ne[1]++;                              // an additional summand 1
    unsigned long long code = 0;
    for (int e = 1; e <= 2 * (int)P.g + 2; e++) code |= (unsigned long long)ne[e] << (4 * (e - 1));
    uint32_t idx = 0xFE;                                             // never left: every type is in the table
    for (uint32_t t = 0; t < P.n_parts; t++)
        if (P.part_codes[t] == code) { idx = t; break; }
    P.out_lambda[i] = (uint8_t)idx;
}

// --------------------------------------------------------------------------------------------
// Pre-pass of the radix evaluation (not in the paper): N_k(f) = N_k(f(X + t)) for t in F_q -- x -> x + t permutes every
// F_{q^k}, the leading coefficient and hence the points at infinity are unchanged, and so are the root counts.  A row
// with an EMPTY residue class mod R (it would fall back to a smaller radix, hec_radix.cuh) is replaced by the first
// shift f(X + alpha^s), s = 0, 1, .., that has every class non-empty (Taylor shift by repeated synthetic division, O(d^2)
// Zech additions in F_q); rows that are fine, invalid, or have no such shift among the first kShiftTries are copied.
// One thread per curve; the squarefree / lambda kernel keeps reading the original rows.
// --------------------------------------------------------------------------------------------
constexpr int kShiftTries = 8;

__global__ void __launch_bounds__(256) hec_shift_kernel(const HecShiftParams P) {
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const FqLog K{P.M, P.zech};
    const uint32_t ZERO = P.M;
    const uint16_t *row = P.coeffs + i * P.ncoef;
    uint16_t *out = P.out + i * P.ncoef;
    uint32_t c[kSqMaxCoef], a[kSqMaxCoef], b[kSqMaxCoef];
    uint32_t nz = 0;
    bool ok = true;
    int d = -1;
    for (uint32_t j = 0; j < P.ncoef; j++) {
        c[j] = row[j];
        if (c[j] >= P.q) ok = false;
        if (c[j]) { nz |= 1u << j; d = (int)j; }
    }
    auto all_present = [&](uint32_t mask) {
        if (P.dense) return d >= 0 && (mask & ((2u << d) - 1u)) == (2u << d) - 1u;
        uint32_t m = mask;
        for (uint32_t s = P.R; s < P.ncoef; s += P.R) m |= mask >> s;
        return (m & ((1u << P.R) - 1u)) == (1u << P.R) - 1u;
    };
    bool done = !ok || d < (int)P.ncoef - 2 || (!P.dense && d + 1 < (int)P.R) || all_present(nz);
    if (!done) {
        for (int j = 0; j <= d; j++) a[j] = c[j] ? __ldg(P.emb + c[j]) : ZERO;
        for (int s = 0; s < kShiftTries && s < (int)P.M && !done; s++) {
            for (int j = 0; j <= d; j++) b[j] = a[j];
            for (int lo = 0; lo < d; lo++)                     // f(X + t): d rounds of b_j += t b_{j+1}, j = d-1 .. lo
                for (int j = d - 1; j >= lo; j--) b[j] = K.add(b[j], K.mul((uint32_t)s, b[j + 1]));
            uint32_t m = 0;
            for (int j = 0; j <= d; j++) m |= (b[j] != ZERO ? 1u : 0u) << j;
            if (all_present(m)) {
                for (int j = 0; j <= d; j++) c[j] = b[j] == ZERO ? 0u : __ldg(P.antilog + b[j]);
                done = true;
            }
        }
    }
    for (uint32_t j = 0; j < P.ncoef; j++) out[j] = (uint16_t)c[j];
}

LibState g_state;

int ensure_device(LibState &S) {
    if (S.device_ready) {                         // one GPU per process (hec.h): plans, staging buffers and pools live on S.device
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess || cur != S.device) {
            cudaGetLastError();
            HEC_FAIL(HEC_ERR_INVALID_ARG, "libhec is bound to the CUDA device that was current at its first call (one GPU per process); "
                                          "call hec_shutdown() before switching devices");
        }
        return HEC_OK;
    }
    int dev = 0, cnt = 0;
    if (cudaGetDeviceCount(&cnt) != cudaSuccess || cnt == 0) {
        cudaGetLastError();
        HEC_FAIL(HEC_ERR_CUDA, "no CUDA device present: libhec has no CPU fallback");
    }
    HEC_CUDA_OK(cudaGetDevice(&dev));
    HEC_CUDA_OK(cudaDeviceGetAttribute(&S.sm_count, cudaDevAttrMultiProcessorCount, dev));
    HEC_CUDA_OK(cudaDeviceGetAttribute(&S.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    for (auto &e : S.ev) HEC_CUDA_OK(cudaEventCreate(&e));
    for (auto &e : S.ev_chunk) HEC_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    HEC_CUDA_OK(cudaStreamCreateWithFlags(&S.copy_in, cudaStreamNonBlocking));
    HEC_CUDA_OK(cudaStreamCreateWithFlags(&S.copy_out, cudaStreamNonBlocking));
    S.device = dev;
    S.device_ready = true;
    hec_allow_device_field_build(true);          // fields above 2^16 elements are now built by hec_field_device.cu
    return HEC_OK;
}

uint32_t align16(uint32_t x) { return (x + 15u) & ~15u; }

hec_table_geom table_geom(uint32_t M, uint32_t D, uint32_t U) {
    hec_table_geom t;
    t.M = M;
    uint32_t lanes = std::min<uint32_t>(32u * U, M);
    t.padl = (D * lanes + 2u) & ~1u;
    t.lmax = M + t.padl;            // M even, padl even
    t.entries = 2u * t.lmax + M;
    return t;
}

template <typename T>
void fill_extended(const hec_field &F, const hec_table_geom &t, T *out) {
    const uint32_t M = t.M, Z0 = M + t.lmax;
    uint32_t n = 0;
    for (uint32_t i = 0; i < Z0; i++) {
        const uint32_t z = F.zech[n];
        out[i] = (T)(z == M ? Z0 : z);
        if (++n == M) n = 0;
    }
    for (uint32_t i = Z0; i < t.entries; i++) out[i] = (T)0u;
}

// Half table (kernel comment "Half tables"): entry b in [0, h] holds Z(h - b) - h, entry h + 1 holds -h
// ("the accumulator was zero": the new relative log is log 1 = 0); Z(h) = "1 + alpha^h = 0" is the sentinel.
uint32_t half_entries(uint32_t M) { return (M >> 1) + 2u; }
void fill_half32(const hec_field &F, uint32_t M, int32_t *out) {
    const uint32_t h = M >> 1;
    for (uint32_t b = 0; b <= h; b++) {
        const uint32_t z = F.zech[h - b];
        out[b] = z == M ? INT32_MIN : 4 * ((int32_t)z - (int32_t)h);
    }
    out[h + 1] = -4 * (int32_t)h;
}
void fill_half24(const hec_field &F, uint32_t M, uint16_t *lo, int8_t *hi) {
    const uint32_t h = M >> 1;
    for (uint32_t b = 0; b <= h + 1; b++) {
        const uint32_t z = b <= h ? F.zech[h - b] : 0u;
        const int32_t w = (int32_t)z - (int32_t)h;
        lo[b] = z == M ? 0 : (uint16_t)((uint32_t)w & 0xFFFFu);
        hi[b] = z == M ? (int8_t)-128 : (int8_t)(w >> 16);
    }
}

// Tables of the radix evaluation (hec_radix.cuh "Table policies").  A vanishing sum (the paper's sentinel,
// PAPER.md:254) is stored as 0, a value Z never takes otherwise.
uint32_t zech0(const hec_field &F, uint32_t M, uint32_t n) { const uint32_t z = F.zech[n]; return z == M ? 0u : z; }
void fill_pair16(const hec_field &F, uint32_t M, uint32_t *out) {
    const uint32_t h = M >> 1;
    for (uint32_t n = 0; n < M; n++) out[n] = zech0(F, M, n) | (zech0(F, M, n + h >= M ? n + h - M : n + h) << 16);
}
void fill_gpair64(const hec_field &F, uint32_t M, uint32_t *out) {
    const uint32_t h = M >> 1;
    for (uint32_t n = 0; n < M; n++) { out[2 * n] = zech0(F, M, n); out[2 * n + 1] = zech0(F, M, n + h >= M ? n + h - M : n + h); }
}
void fill_rhalf32(const hec_field &F, uint32_t M, uint32_t *out) {
    for (uint32_t i = 0; i <= (M >> 1); i++) out[i] = zech0(F, M, i);
}
void fill_rhalf17(const hec_field &F, uint32_t M, uint16_t *lo, uint8_t *bits) {
    const uint32_t h = M >> 1;
    for (uint32_t i = 0; i <= h; i++) {
        lo[i] = (uint16_t)(zech0(F, M, i) & 0xFFFFu);
        bits[i] = (uint8_t)(((zech0(F, M, i) >> 16) & 1u) | (((zech0(F, M, h - i) >> 16) & 1u) << 1));
    }
}

// Fast tables of a PAIR16 field (hec_radix.cuh: radix_fast_x): lanepow[e][lane] = (e lane mod M) | (e (lane + 32) mod M) << 16
// and stepe[e] = (64 e mod M) in both halves for e = 0 .. D, then the transposed Zech table, R rows of S + 64 16-bit
// entries, T[c][j] = Z[c + R (j mod S)], S = M / R, each row padded to a multiple of 4 bytes.
uint32_t fast_row_bytes(uint32_t M, uint32_t R) { return (2u * (M / R + 64u) + 3u) & ~3u; }
uint32_t fast_head_bytes(uint32_t D) { return (D + 1u) * 128u + (((D + 1u) * 4u + 15u) & ~15u); }
uint32_t fast_bytes(uint32_t M, uint32_t R, uint32_t D) { return align16(fast_head_bytes(D) + R * fast_row_bytes(M, R)); }
void fill_fast_tables(const hec_field &F, uint32_t M, uint32_t R, uint32_t D, uint8_t *out) {
    uint32_t *lanepow = reinterpret_cast<uint32_t *>(out), *stepe = lanepow + (D + 1u) * 32u;
    for (uint32_t e = 0; e <= D; e++) {
        for (uint32_t l = 0; l < 32u; l++) lanepow[e * 32u + l] = (e * l) % M | ((e * (l + 32u)) % M) << 16;
        stepe[e] = ((64u * e) % M) * 0x10001u;
    }
    const uint32_t S = M / R, rowB = fast_row_bytes(M, R);
    for (uint32_t c = 0; c < R; c++) {
        uint16_t *row = reinterpret_cast<uint16_t *>(out + fast_head_bytes(D) + c * rowB);
        for (uint32_t j = 0; j < S + 64u; j++) row[j] = (uint16_t)zech0(F, M, c + R * (j % S));
    }
}

// Packed parity table of a field (hec_radix.cuh: network_mono): entry n = parity(Z[n]) | parity(Z[n + M/2]) << 1, four per byte.
uint32_t parity_table_bytes(uint32_t M) { return align16((M + 3u) / 4u); }
void fill_parity_table(const hec_field &F, uint32_t M, uint8_t *out) {
    const uint32_t h = M >> 1;
    std::fill(out, out + parity_table_bytes(M), (uint8_t)0);
    for (uint32_t n = 0; n < M; n++) {
        const uint32_t bits = (zech0(F, M, n) & 1u) | ((zech0(F, M, n + h >= M ? n + h - M : n + h) & 1u) << 1);
        out[n >> 2] |= (uint8_t)(bits << ((n & 3u) * 2u));
    }
}

// Smallest field for which the half-table step is valid: the lane term must stay below h (kernel comment).
constexpr uint32_t kHalfMinM = 1u << 13;
constexpr uint32_t kHalf24MaxM = 1u << 22;      // |Z - h| < 127 * 65536
constexpr uint32_t kRadixScratchBytes = kWarps * hec_radix::kScratchWords * 4u;

// Radix of one field: the largest R in {2, 4, 8} with R | M, capped by the evaluation scheme.  Measured on B200
// (profiles/): with a pair table one entry serves both butterfly outputs, so R = 8 wins; with a half table a
// pair costs two (three) loads and R = 4 is the better trade for the short chains of genus 2.
uint32_t pick_radix(uint32_t M, int eval, int mode, uint32_t g) {
    uint32_t cap = eval == HEC_EVAL_RADIX2 ? 2u : eval == HEC_EVAL_RADIX4 ? 4u : 8u;
    if ((eval == HEC_EVAL_AUTO || eval == HEC_EVAL_ORBIT) && mode == HEC_TAB_RHALF32 && g <= 2) cap = 4u;
    uint32_t R = 2;
    while (R < cap && M % (2u * R) == 0) R *= 2u;
    return R;
}

int build_plan(LibState &S, uint32_t q, uint32_t g, int regime, int eval, DevicePlan **out) {
    const bool radix = eval != HEC_EVAL_HORNER;
    auto key = std::make_tuple(q, g, regime, eval | (S.fast_enabled ? 0x100 : 0));
    auto it = S.plans.find(key);
    if (it != S.plans.end()) { *out = it->second.get(); return HEC_OK; }

    uint32_t p, r;
    if (!hec_factor_q(q, &p, &r)) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q must be an odd prime power below 65536");
    uint64_t Qg = 1;
    for (uint32_t i = 0; i < g; i++) { Qg *= q; if (Qg > HEC_MAX_FIELD_SIZE) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q^g exceeds HEC_MAX_FIELD_SIZE (2^26)"); }

    std::unique_ptr<DevicePlan> plan(new DevicePlan);
    plan->q = q; plan->g = g; plan->p = p; plan->r = r; plan->radix = radix;
    const uint32_t D = 2 * g + 2;
    const uint32_t U = (uint32_t)plan->U;
    const uint32_t budget = (uint32_t)S.smem_optin - 1024u - (radix ? kRadixScratchBytes : 0u);
    const int base_mode = radix ? HEC_TAB_PAIR16 : HEC_TAB_EXT16;      // layout of the fields below the top of a launch
    const int global_mode = radix ? HEC_TAB_GPAIR64 : HEC_TAB_GLOBAL32;

    std::vector<const hec_field *> fields(g);
    std::vector<hec_table_geom> geom(g);
    for (uint32_t k = 1; k <= g; k++) {
        fields[k - 1] = hec_cached_field(p, r, k);
        if (!fields[k - 1]) return HEC_ERR_INVALID_FIELD;
        geom[k - 1] = table_geom(fields[k - 1]->Q - 1, D, U);
    }
    // ---- table mode of every field and the grouping into launches (one shared-memory image per launch)
    auto mode_bytes = [&](uint32_t k, int mode) -> uint32_t {      // 0: the layout cannot hold this field
        const hec_table_geom &t = geom[k - 1];
        const uint32_t M = t.M;
        uint64_t b = 0;
        switch (mode) {
            case HEC_TAB_EXT16:
                if ((uint64_t)t.lmax + t.M > 65535u) return 0;           // Z0 = M + LP must fit 16 bits
                b = (uint64_t)t.entries * 2u;
                break;
            case HEC_TAB_HALF32:
            case HEC_TAB_HALF24: {
                if (M < kHalfMinM || (mode == HEC_TAB_HALF24 && M >= kHalf24MaxM)) return 0;
                const uint64_t e = half_entries(M);
                b = mode == HEC_TAB_HALF32 ? e * 4u : (uint64_t)align16((uint32_t)(e * 2u)) + e;
                break;
            }
            case HEC_TAB_PAIR16:
                if (M > 32768u) return 0;                                 // both halves of a packed value stay below 2 M <= 65536
                b = (uint64_t)M * 4u;
                break;
            case HEC_TAB_SPAIR16:
                if (M <= 32768u || M >= 65536u) return 0;                 // below: PAIR16 with packed arithmetic; above: 17-bit values
                b = (uint64_t)M * 4u;
                break;
            case HEC_TAB_RHALF32:
                b = ((uint64_t)(M >> 1) + 1u) * 4u;
                break;
            case HEC_TAB_RHALF17:
                if (M >= (1u << 17)) return 0;
                b = (uint64_t)align16(((M >> 1) + 1u) * 2u) + (M >> 1) + 1u;
                break;
            default:
                return 1u;                                                // global tables take no shared memory
        }
        return b <= budget ? align16((uint32_t)b) : 0;
    };
    std::vector<int> mode(g, base_mode);
    std::vector<uint32_t> bytes(g, 0);
    for (uint32_t k = 1; k <= g; k++) {
        const bool top = k == g;
        int m = -1;
        uint32_t b = 0;
        auto try_mode = [&](int cand) {
            if (m >= 0) return;
            const uint32_t cb = mode_bytes(k, cand);
            if (cb) { m = cand; b = cand == global_mode ? 0u : cb; }
        };
        const int half_a = radix ? HEC_TAB_RHALF32 : HEC_TAB_HALF32, half_b = radix ? HEC_TAB_RHALF17 : HEC_TAB_HALF24;
        if (top && regime == HEC_REGIME_L2) {
            try_mode(global_mode);
        } else if (top && regime == HEC_REGIME_SMEM) {
            try_mode(base_mode);
            if (radix) try_mode(HEC_TAB_SPAIR16);
            if (m < 0) HEC_FAIL(HEC_ERR_INVALID_ARG, "HEC_REGIME_SMEM: the full Zech table of the largest field does not fit shared memory");
        } else if (top && regime == HEC_REGIME_SMEM_HALF) {
            if (geom[k - 1].M >= kHalfMinM) { try_mode(half_a); try_mode(half_b); }
            if (m < 0) HEC_FAIL(HEC_ERR_INVALID_ARG, "HEC_REGIME_SMEM_HALF: the half table of the largest field does not fit shared memory (or the field is below 2^13 elements)");
        } else {
            try_mode(base_mode);
            if (radix && top) try_mode(HEC_TAB_SPAIR16);                  // one load per pair where a half table needs two and a fold
            try_mode(half_a);
            try_mode(half_b);
            try_mode(global_mode);
        }
        mode[k - 1] = m;
        bytes[k - 1] = b;
    }
    plan->top_mode = mode[g - 1];
    // fast tables (radix_fast_x) for the PAIR16 fields, the largest field first, as long as one launch still holds everything
    std::vector<uint32_t> radix_of(g, 0), fastb(g, 0);
    for (uint32_t k = 1; k <= g; k++) radix_of[k - 1] = radix ? pick_radix(geom[k - 1].M, eval, mode[k - 1], g) : 0u;
    // Packed parity table of the top field (half-table layouts: the classifying last stage reads it instead of the pair), if it fits.
    // With it, dense rows run the monomial-class loop (radix_mono_x).
    uint32_t ptb = 0, mono_r = 0;
    if (radix && S.fast_enabled && (mode[g - 1] == HEC_TAB_RHALF32 || mode[g - 1] == HEC_TAB_RHALF17)) {
        uint64_t total = parity_table_bytes(geom[g - 1].M);
        for (uint32_t k = 1; k <= g; k++) total += bytes[k - 1];
        if (total <= budget) {
            ptb = parity_table_bytes(geom[g - 1].M);
            // monomial classes (radix_mono_x): R = 8 for at most 8 coefficients, R = 16 for 9 .. 16, where R | M
            const uint32_t Rm = D + 1 <= 8 ? 8u : 16u;
            // (an explicit HEC_EVAL_RADIX8 request stays a pure radix-8 run: the R = 16 loop is AUTO's alone)
            if ((eval == HEC_EVAL_AUTO || (eval == HEC_EVAL_RADIX8 && Rm == 8u)) && D + 1 <= 16 && geom[g - 1].M % Rm == 0 && geom[g - 1].M >= 4096u) {
                mono_r = Rm;
                if (Rm == 8u) radix_of[g - 1] = 8u;      // rows that do not qualify run the general loops at R <= 8 either way
            }
        }
    }
    if (radix && S.fast_enabled && mode[g - 1] == HEC_TAB_SPAIR16 && (eval == HEC_EVAL_AUTO || eval == HEC_EVAL_RADIX8) && D + 1 <= 16) {
        const uint32_t Rm = D + 1 <= 8 ? 8u : 16u;
        if (geom[g - 1].M % Rm == 0 && (eval == HEC_EVAL_AUTO || Rm == 8u)) mono_r = Rm;   // the pair table serves the last stage too
    }
    if (radix && S.fast_enabled) {
        uint64_t total = ptb;
        for (uint32_t k = 1; k <= g; k++) total += bytes[k - 1];
        for (uint32_t k = g; k >= 1; k--) {
            if (mode[k - 1] != HEC_TAB_PAIR16) continue;
            const uint32_t fb = fast_bytes(geom[k - 1].M, radix_of[k - 1], D);
            if (total + fb > budget) continue;
            total += fb;
            fastb[k - 1] = fb;
        }
    }
    struct Group { uint32_t k_lo, k_hi, smem; };
    std::vector<Group> groups;
    {
        Group cur{1, 0, 0};
        for (uint32_t k = 1; k <= g; k++) {
            const uint32_t extra = fastb[k - 1] + (k == g ? ptb : 0u);
            if (cur.k_hi >= cur.k_lo && cur.smem + bytes[k - 1] + extra > budget) { groups.push_back(cur); cur = Group{k, 0, 0}; }
            cur.k_hi = k;
            cur.smem += bytes[k - 1] + extra;
            if (mode[k - 1] != base_mode) { groups.push_back(cur); cur = Group{k + 1, 0, 0}; }   // only the top of a launch may differ
        }
        if (cur.k_hi >= cur.k_lo) groups.push_back(cur);
    }

    // ---- one device allocation: [launch blobs][global tables][embed tables][squarefree tables]
    std::vector<uint8_t> host;
    auto reserve = [&](size_t nbytes) { size_t o = host.size(); host.resize(o + ((nbytes + 255) & ~(size_t)255)); return o; };
    std::vector<size_t> blob_off(groups.size()), gtab_off(g, 0), emb_off(g, 0);
    for (size_t gi = 0; gi < groups.size(); gi++) {
        const Group &G = groups[gi];
        blob_off[gi] = reserve(std::max<uint32_t>(G.smem, 16u));
        uint32_t so = 0;
        for (uint32_t k = G.k_lo; k <= G.k_hi; k++) {
            const hec_table_geom &t = geom[k - 1];
            HecFieldDev &fd = plan->f[k - 1];
            fd.M = t.M; fd.mode = (uint32_t)mode[k - 1]; fd.z0 = t.M + t.lmax; fd.rcpM = (uint32_t)((1ull << 32) / t.M);
            fd.lane_cap = std::min<uint32_t>(32u * U, t.M);
            fd.smem_off = so; fd.smem_off2 = 0; fd.gtab = nullptr;
            fd.radix = radix_of[k - 1];
            fd.fast_off = 0; fd.fast_row = 0; fd.pt_off = 0; fd.mono_r = (k == g) ? mono_r : 0u;
            uint8_t *dst = host.data() + blob_off[gi] + so;
            switch (mode[k - 1]) {
                case HEC_TAB_EXT16:
                    fill_extended<uint16_t>(*fields[k - 1], t, reinterpret_cast<uint16_t *>(dst));
                    break;
                case HEC_TAB_HALF32:
                    fill_half32(*fields[k - 1], t.M, reinterpret_cast<int32_t *>(dst));
                    break;
                case HEC_TAB_HALF24: {
                    const uint32_t lo_bytes = align16(half_entries(t.M) * 2u);
                    fd.smem_off2 = so + lo_bytes;
                    fill_half24(*fields[k - 1], t.M, reinterpret_cast<uint16_t *>(dst), reinterpret_cast<int8_t *>(dst + lo_bytes));
                    break;
                }
                case HEC_TAB_SPAIR16:
                    fill_pair16(*fields[k - 1], t.M, reinterpret_cast<uint32_t *>(dst));
                    break;
                case HEC_TAB_PAIR16:
                    fill_pair16(*fields[k - 1], t.M, reinterpret_cast<uint32_t *>(dst));
                    if (fastb[k - 1]) {
                        fd.fast_off = so + bytes[k - 1];
                        fd.fast_row = fast_row_bytes(t.M, fd.radix);
                        fill_fast_tables(*fields[k - 1], t.M, fd.radix, D, dst + bytes[k - 1]);
                    }
                    break;
                case HEC_TAB_RHALF32:
                    fill_rhalf32(*fields[k - 1], t.M, reinterpret_cast<uint32_t *>(dst));
                    if (k == g && ptb) {
                        fd.pt_off = so + bytes[k - 1];
                        fill_parity_table(*fields[k - 1], t.M, dst + bytes[k - 1]);
                    }
                    break;
                case HEC_TAB_RHALF17: {
                    const uint32_t lo_bytes = align16(((t.M >> 1) + 1u) * 2u);
                    fd.smem_off2 = so + lo_bytes;
                    fill_rhalf17(*fields[k - 1], t.M, reinterpret_cast<uint16_t *>(dst), dst + lo_bytes);
                    if (k == g && ptb) {
                        fd.pt_off = so + bytes[k - 1];
                        fill_parity_table(*fields[k - 1], t.M, dst + bytes[k - 1]);
                    }
                    break;
                }
                default:
                    break;
            }
            so += bytes[k - 1] + fastb[k - 1] + (k == g ? ptb : 0u);
        }
    }
    for (uint32_t k = 1; k <= g; k++) {
        const hec_table_geom &t = geom[k - 1];
        if (mode[k - 1] == HEC_TAB_GLOBAL32) {
            gtab_off[k - 1] = reserve((size_t)t.entries * 4u);
            fill_extended<uint32_t>(*fields[k - 1], t, reinterpret_cast<uint32_t *>(host.data() + gtab_off[k - 1]));
        } else if (mode[k - 1] == HEC_TAB_GPAIR64) {
            gtab_off[k - 1] = reserve((size_t)t.M * 8u);
            fill_gpair64(*fields[k - 1], t.M, reinterpret_cast<uint32_t *>(host.data() + gtab_off[k - 1]));
        }
        emb_off[k - 1] = reserve((size_t)q * 4u);
        uint32_t *e = reinterpret_cast<uint32_t *>(host.data() + emb_off[k - 1]);
        for (uint32_t c = 0; c < q; c++) e[c] = fields[k - 1]->embed[c] == t.M ? HEC_LOG_ZERO : fields[k - 1]->embed[c];
    }
    // HEC_EVAL_ORBIT: per field and R' in {2, 4, 8} with R' | R, one coset index per orbit of n -> q n on Z/(M/R'),
    // packed n | (orbit length << 28) (hec_radix.cuh: radix_orbit_x)
    std::vector<std::array<size_t, 3>> orb_off(g, std::array<size_t, 3>{0, 0, 0});
    std::vector<std::array<uint32_t, 3>> orb_cnt(g, std::array<uint32_t, 3>{0, 0, 0});
    if (eval == HEC_EVAL_ORBIT) {
        for (uint32_t k = 1; k <= g; k++) {
            const uint32_t M = geom[k - 1].M, Rk = plan->f[k - 1].radix;
            for (uint32_t t = 0, Rp = 2; t < 3 && Rp <= Rk; t++, Rp *= 2) {
                const uint32_t Sp = M / Rp;
                if (Sp >= (1u << 28)) HEC_FAIL(HEC_ERR_UNSUPPORTED, "HEC_EVAL_ORBIT: field too large");
                std::vector<bool> seen(Sp, false);
                std::vector<uint32_t> reps;
                for (uint32_t n = 0; n < Sp; n++) {
                    if (seen[n]) continue;
                    uint32_t len = 0, m = n;
                    do { seen[m] = true; m = (uint32_t)(((uint64_t)m * q) % Sp); len++; } while (m != n);
                    reps.push_back(n | (len << 28));
                }
                orb_off[k - 1][t] = reserve(reps.size() * 4u);
                orb_cnt[k - 1][t] = (uint32_t)reps.size();
                std::copy(reps.begin(), reps.end(), reinterpret_cast<uint32_t *>(host.data() + orb_off[k - 1][t]));
            }
        }
    }
    const std::vector<std::vector<uint8_t>> parts = hec_partitions_of(2 * g + 2);
    const size_t part_off = reserve(parts.size() * 8u);
    for (size_t t = 0; t < parts.size(); t++) {
        unsigned long long code = 0;
        for (size_t e = 0; e < parts[t].size(); e++) code |= (unsigned long long)parts[t][e] << (4 * e);
        reinterpret_cast<unsigned long long *>(host.data() + part_off)[t] = code;
    }
    const size_t sqa_off = reserve((size_t)(q - 1) * 4u);
    std::copy(fields[0]->antilog.begin(), fields[0]->antilog.end(), reinterpret_cast<uint32_t *>(host.data() + sqa_off));
    const size_t sqz_off = reserve((size_t)(q - 1) * 4u);
    std::copy(fields[0]->zech.begin(), fields[0]->zech.end(), reinterpret_cast<uint32_t *>(host.data() + sqz_off));

    HEC_CUDA_OK(cudaMalloc(&plan->d_blob, host.size()));
    HEC_CUDA_OK(cudaMemcpy(plan->d_blob, host.data(), host.size(), cudaMemcpyHostToDevice));
    HEC_CUDA_OK(cudaMalloc((void **)&plan->d_err, 2 * sizeof(unsigned long long)));
    const uint8_t *base = static_cast<const uint8_t *>(plan->d_blob);
    for (size_t gi = 0; gi < groups.size(); gi++) {
        LaunchPlan L;
        L.k_lo = groups[gi].k_lo; L.k_hi = groups[gi].k_hi;
        L.top_mode = mode[L.k_hi - 1];
        L.blob = reinterpret_cast<const uint4 *>(base + blob_off[gi]);
        L.blob_bytes = align16(groups[gi].smem);
        L.smem_bytes = std::max<uint32_t>(L.blob_bytes, 16u) + (radix ? kRadixScratchBytes : 0u);
        plan->launches.push_back(L);
    }
    for (uint32_t k = 1; k <= g; k++) {
        const bool glob = mode[k - 1] == HEC_TAB_GLOBAL32 || mode[k - 1] == HEC_TAB_GPAIR64;
        plan->f[k - 1].gtab = glob ? reinterpret_cast<const uint32_t *>(base + gtab_off[k - 1]) : nullptr;
        plan->f[k - 1].emb = reinterpret_cast<const uint32_t *>(base + emb_off[k - 1]);
        for (int t = 0; t < 3; t++) {
            plan->f[k - 1].orb_fast = (eval == HEC_EVAL_ORBIT && mode[k - 1] == HEC_TAB_PAIR16 && S.fast_enabled) ? 1u : 0u;
            plan->f[k - 1].n_orb[t] = orb_cnt[k - 1][t];
            plan->f[k - 1].orb[t] = orb_cnt[k - 1][t] ? reinterpret_cast<const uint32_t *>(base + orb_off[k - 1][t]) : nullptr;
        }
    }
    plan->sq_zech = reinterpret_cast<const uint32_t *>(base + sqz_off);
    plan->sq_emb = plan->f[0].emb;
    plan->sq_antilog = reinterpret_cast<const uint32_t *>(base + sqa_off);
    // the shift pre-pass pays where the dominant (largest) field has R >= 4 and the rows have at least R coefficients
    plan->shift_R = (radix && plan->f[g - 1].radix >= 4u && 2 * g + 2 >= plan->f[g - 1].radix) ? plan->f[g - 1].radix : 0u;
    // monomial classes (radix_mono_x / radix_mono8_packed_x): every coefficient up to the degree nonzero
    // (not below 2048 elements: there the pre-pass costs more than the rows it moves onto the monomial loop save -- q = 25, g = 2:
    // 0.23 ms of pre-pass against a 1.4 ms count kernel; rows with a zero coefficient then take radix_fast_x at R = 4)
    plan->shift_dense = mono_r != 0 || (radix && D + 1 <= 8 && plan->f[g - 1].radix == 8u && plan->f[g - 1].fast_off != 0 &&
                                        geom[g - 1].M >= 2048u);
    if (plan->shift_dense) plan->shift_R = 8u;
    plan->d_part_codes = reinterpret_cast<const unsigned long long *>(base + part_off);
    plan->n_parts = (uint32_t)parts.size();

    *out = plan.get();
    S.plans[key] = std::move(plan);
    return HEC_OK;
}

// rows -> rows with every residue class mod plan.shift_R non-empty where a shift achieves it; into `out` or S.d_shift
int run_shift(LibState &S, const DevicePlan &plan, const uint16_t *d_rows, size_t n, uint16_t *d_out) {
    const uint32_t ncoef = 2 * plan.g + 3;
    const size_t bytes = n * ncoef * sizeof(uint16_t);
    if (!d_out) {
        if (bytes > S.shift_bytes) {
            if (S.d_shift) cudaFree(S.d_shift);
            S.d_shift = nullptr; S.shift_bytes = 0;
            if (cudaMalloc(&S.d_shift, bytes) != cudaSuccess) { cudaGetLastError(); HEC_FAIL(HEC_ERR_NOMEM, "cannot allocate the shifted-row buffer"); }
            S.shift_bytes = bytes;
        }
        d_out = static_cast<uint16_t *>(S.d_shift);
    }
    HecShiftParams H;
    H.coeffs = d_rows; H.out = d_out; H.n = n; H.q = plan.q; H.M = plan.q - 1; H.ncoef = ncoef;
    H.R = plan.shift_R ? plan.shift_R : 2u;
    H.dense = plan.shift_dense ? 1u : 0u;
    H.zech = plan.sq_zech; H.emb = plan.sq_emb; H.antilog = plan.sq_antilog;
    hec_shift_kernel<<<(unsigned)((n + 255) / 256), 256, 0, S.stream>>>(H);
    hec_launch_counter::value++;
    S.stats.launches++;
    HEC_CUDA_OK(cudaGetLastError());
    return HEC_OK;
}

bool is_device_pointer(const void *p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

// Shared with the other translation units.
// Partitions of `total` as multiplicity vectors (n_1 .. n_total) in ascending lexicographic order of that vector: the
// index order of the lambda codes (hec.h).
std::vector<std::vector<uint8_t>> hec_partitions_of(uint32_t total) {
    std::vector<std::vector<uint8_t>> res;
    std::vector<uint8_t> acc(total, 0);
    struct Rec {
        static void go(uint32_t e, uint32_t left, uint32_t total, std::vector<uint8_t> &acc, std::vector<std::vector<uint8_t>> &res) {
            if (e > total) { if (left == 0) res.push_back(acc); return; }
            for (uint32_t m = 0; m * e <= left; m++) { acc[e - 1] = (uint8_t)m; go(e + 1, left - m * e, total, acc, res); }
            acc[e - 1] = 0;
        }
    };
    Rec::go(1, total, total, acc, res);
    std::sort(res.begin(), res.end());
    return res;
}
cudaStream_t hec_current_stream() { return g_state.stream; }
int hec_ensure_device(int *sm_count, int *smem_optin) {
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    int rc = ensure_device(g_state);
    if (rc) return rc;
    if (sm_count) *sm_count = g_state.sm_count;
    if (smem_optin) *smem_optin = g_state.smem_optin;
    return HEC_OK;
}
bool hec_is_device_pointer(const void *p) { return is_device_pointer(p); }

extern "C" {

int hec_set_stream(void *cuda_stream) {
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    g_state.stream = static_cast<cudaStream_t>(cuda_stream);
    return HEC_OK;
}

int hec_set_regime(int regime) {
    if (regime < HEC_REGIME_AUTO || regime > HEC_REGIME_SMEM_HALF) HEC_FAIL(HEC_ERR_INVALID_ARG, "unknown regime");
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    g_state.regime = regime;
    return HEC_OK;
}

int hec_set_eval(int eval) {
    if (eval != HEC_EVAL_AUTO && eval != HEC_EVAL_HORNER && eval != HEC_EVAL_RADIX2 && eval != HEC_EVAL_RADIX4 && eval != HEC_EVAL_RADIX8 && eval != HEC_EVAL_ORBIT) HEC_FAIL(HEC_ERR_INVALID_ARG, "unknown evaluation scheme");
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    g_state.eval = eval;
    return HEC_OK;
}

int hec_last_count_stats(hec_count_stats *out) {
    if (!out) HEC_FAIL(HEC_ERR_INVALID_ARG, "out is NULL");
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    *out = g_state.stats;
    return HEC_OK;
}

uint64_t hec_launch_count(void) { return hec_launch_counter::value; }

int hec_count(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t *out_counts, uint8_t *out_squarefree) {
    return hec_count_ex(q, g, coeffs, n, out_counts, out_squarefree, nullptr, nullptr);
}

}  // extern "C"

namespace {

// Host buffers: rows in chunks through three streams -- H2D of chunk i+1 and D2H of chunk i-1 run under the kernels of
// chunk i (pinned host memory; pageable memory is staged by the driver and still correct).  Below this many rows one chunk.
constexpr size_t kPipelineMinRows = (size_t)1 << 20;
constexpr int kPipelineChunks = 4;

// hec_count_ex.  keep_device (host-pointer calls of hec_count_histogram): do not wait for the D2H copies; return the device
// copies of the counts and the flags (valid until the next call) so that the histogram can start under those copies, and
// leave the status check to finish_count().
struct CountTail {
    DevicePlan *plan = nullptr;
    unsigned long long err[2] = {~0ull, ~0ull};
    bool pending = false;          // D2H copies in flight on S.copy_out
    const uint32_t *d_counts = nullptr;
    const uint8_t *d_sf = nullptr;
};

int finish_count(LibState &S, CountTail &T) {
    const cudaError_t e_out = T.pending ? cudaStreamSynchronize(S.copy_out) : cudaSuccess;
    T.pending = false;
    const cudaError_t e_main = cudaStreamSynchronize(S.stream);   // waited for even when the copy stream failed
    if (e_out != cudaSuccess || e_main != cudaSuccess) {
        cudaGetLastError();
        hec_set_error(HEC_ERR_CUDA, std::string("hec_count: ") + cudaGetErrorString(e_out != cudaSuccess ? e_out : e_main));
        return HEC_ERR_CUDA;
    }
    cudaEventElapsedTime(&S.stats.count_kernel_ms, S.ev[0], S.ev[1]);
    cudaEventElapsedTime(&S.stats.squarefree_kernel_ms, S.ev[1], S.ev[2]);
    if (T.err[0] != ~0ull) {
        hec_set_error(HEC_ERR_COEFF_RANGE, "a coefficient is >= q", (size_t)T.err[0]);
        return HEC_ERR_COEFF_RANGE;
    }
    if (T.err[1] != ~0ull) {
        hec_set_error(HEC_ERR_DEGREE, "a row has c[2g+2] = c[2g+1] = 0 (degree < 2g+1)", (size_t)T.err[1]);
        return HEC_ERR_DEGREE;
    }
    return HEC_OK;
}

// Error exits of count_impl: copies of earlier chunks may still be running on the copy streams into the caller's host
// buffers and the staging buffer.  Unless disarmed, the guard waits for all three streams, so that after a failing
// call the caller may free or reuse its buffers.
struct DrainOnError {
    LibState &S;
    bool armed = true;
    explicit DrainOnError(LibState &s) : S(s) {}
    ~DrainOnError() {
        if (!armed) return;
        if (S.copy_in) cudaStreamSynchronize(S.copy_in);
        if (S.copy_out) cudaStreamSynchronize(S.copy_out);
        cudaStreamSynchronize(S.stream);
        cudaGetLastError();
    }
};

int count_impl(LibState &S, uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t *out_counts, uint8_t *out_squarefree,
               uint32_t *out_roots, uint8_t *out_lambda, bool keep_device, CountTail &T) {
    uint32_t p, r;
    hec_factor_q(q, &p, &r);
    const bool dev_in = is_device_pointer(coeffs), dev_out = is_device_pointer(out_counts);
    const bool dev_sf = out_squarefree ? is_device_pointer(out_squarefree) : dev_out;
    const bool dev_r0 = out_roots ? is_device_pointer(out_roots) : dev_out;
    const bool dev_lam = out_lambda ? is_device_pointer(out_lambda) : dev_out;
    if (dev_in != dev_out || dev_sf != dev_out || dev_r0 != dev_out || dev_lam != dev_out)
        HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs/out_counts/out_squarefree/out_roots/out_lambda must all be host or all device pointers");

    DevicePlan *plan = nullptr;
    int rc = build_plan(S, q, g, S.regime, S.eval, &plan);
    if (rc) return rc;
    T.plan = plan;

    const size_t ncoef = 2 * (size_t)g + 3;
    const size_t in_bytes = n * ncoef * sizeof(uint16_t), cnt_bytes = n * g * sizeof(uint32_t), sf_bytes = out_squarefree ? n : 0;
    const uint16_t *d_coeffs = coeffs;
    uint32_t *d_counts = out_counts;
    uint8_t *d_sf = out_squarefree;
    uint32_t *d_r0 = out_roots;
    uint8_t *d_lam = out_lambda;
    const bool need_r0 = out_roots || out_lambda;              // lambda is computed from r0 (Algorithm 1 line 18)
    const size_t lam_bytes = out_lambda ? n : 0;
    if (!dev_in || (need_r0 && !out_roots)) {
        const size_t a = dev_in ? 0 : (in_bytes + 255) & ~(size_t)255, b = dev_in ? 0 : (cnt_bytes + 255) & ~(size_t)255;
        const size_t c = dev_in ? 0 : (sf_bytes + 255) & ~(size_t)255;
        const size_t r0b = (!need_r0 || (dev_in && out_roots)) ? 0 : (cnt_bytes + 255) & ~(size_t)255;
        const size_t need = a + b + c + r0b + (dev_in ? 0 : lam_bytes);
        if (need > S.stage_bytes) {
            if (S.d_stage) cudaFree(S.d_stage);
            S.d_stage = nullptr; S.stage_bytes = 0;
            if (cudaMalloc(&S.d_stage, need) != cudaSuccess) { cudaGetLastError(); HEC_FAIL(HEC_ERR_NOMEM, "cannot allocate device staging buffers"); }
            S.stage_bytes = need;
        }
        uint8_t *base = static_cast<uint8_t *>(S.d_stage);
        if (!dev_in) {
            d_coeffs = reinterpret_cast<const uint16_t *>(base);
            d_counts = reinterpret_cast<uint32_t *>(base + a);
            d_sf = out_squarefree ? base + a + b : nullptr;
            d_lam = out_lambda ? base + a + b + c + r0b : nullptr;
        }
        if (r0b) d_r0 = reinterpret_cast<uint32_t *>(base + a + b + c);
    }
    T.d_counts = d_counts;
    T.d_sf = d_sf;

    static const unsigned long long kNoErr[2] = {~0ull, ~0ull};
    HEC_CUDA_OK(cudaMemcpyAsync(plan->d_err, kNoErr, sizeof kNoErr, cudaMemcpyHostToDevice, S.stream));

    HecCountParams P;
    P.q = q; P.blob = nullptr; P.blob_bytes = 0; P.err = plan->d_err; P.k_lo = 1; P.k_hi = g; P.scratch_off = 0;
    // Small batches (down to the single curve of the paper's Table 1): spread every curve over
    // `splits` warps so that the whole GPU works on it; each warp takes a slice of the cosets of every field.
    P.splits = 1;
    if (plan->radix) {
        const unsigned long long warps = (unsigned long long)S.sm_count * kWarps;
        const uint32_t Mtop = plan->f[g - 1].M;
        if (n < 2 * warps && Mtop >= 4096u) {
            const unsigned long long want = (2 * warps + n - 1) / n;
            P.splits = (uint32_t)std::max<unsigned long long>(1, std::min<unsigned long long>(want, Mtop / 2048u));
        }
    }
    if (P.splits > 1) {
        HEC_CUDA_OK(cudaMemsetAsync(d_counts, 0, cnt_bytes, S.stream));
        if (need_r0) HEC_CUDA_OK(cudaMemsetAsync(d_r0, 0, cnt_bytes, S.stream));
    }
    for (uint32_t k = 0; k < HEC_MAX_GENUS; k++) P.f[k] = plan->f[k < g ? k : 0];

    S.stats = hec_count_stats{};
    S.stats.table_mode = (uint32_t)plan->top_mode;
    S.stats.regime = (plan->top_mode == HEC_TAB_EXT16 || plan->top_mode == HEC_TAB_PAIR16 || plan->top_mode == HEC_TAB_SPAIR16) ? HEC_REGIME_SMEM
                     : (plan->top_mode == HEC_TAB_GLOBAL32 || plan->top_mode == HEC_TAB_GPAIR64) ? HEC_REGIME_L2 : HEC_REGIME_SMEM_HALF;
    S.stats.splits = P.splits;

    const bool shift = plan->shift_R && S.shift_enabled;
    if (shift) {                                               // the whole batch's shifted rows live in S.d_shift
        if (in_bytes > S.shift_bytes) {
            if (S.d_shift) cudaFree(S.d_shift);
            S.d_shift = nullptr; S.shift_bytes = 0;
            if (cudaMalloc(&S.d_shift, in_bytes) != cudaSuccess) { cudaGetLastError(); HEC_FAIL(HEC_ERR_NOMEM, "cannot allocate the shifted-row buffer"); }
            S.shift_bytes = in_bytes;
        }
    }
    const int chunks = (!dev_in && n >= kPipelineMinRows) ? kPipelineChunks : 1;
    S.stats.chunks = (uint32_t)chunks;
    if (chunks > 1) {                                          // the copy streams start after whatever precedes on S.stream
        HEC_CUDA_OK(cudaEventRecord(S.ev_chunk[0], S.stream));
        HEC_CUDA_OK(cudaStreamWaitEvent(S.copy_in, S.ev_chunk[0], 0));
        HEC_CUDA_OK(cudaStreamWaitEvent(S.copy_out, S.ev_chunk[0], 0));
    }
    HEC_CUDA_OK(cudaEventRecord(S.ev[0], S.stream));
    DrainOnError drain(S);
    for (int c = 0; c < chunks; c++) {
        const size_t lo = n * (size_t)c / chunks, hi = n * (size_t)(c + 1) / chunks, nc = hi - lo;
        if (nc == 0) continue;
        cudaStream_t s_in = chunks > 1 ? S.copy_in : S.stream, s_out = chunks > 1 ? S.copy_out : S.stream;
        if (!dev_in) {
            HEC_CUDA_OK(cudaMemcpyAsync(const_cast<uint16_t *>(d_coeffs) + lo * ncoef, coeffs + lo * ncoef, nc * ncoef * sizeof(uint16_t),
                                        cudaMemcpyHostToDevice, s_in));
            if (chunks > 1) {
                HEC_CUDA_OK(cudaEventRecord(S.ev_chunk[1 + 2 * c], s_in));
                HEC_CUDA_OK(cudaStreamWaitEvent(S.stream, S.ev_chunk[1 + 2 * c], 0));
            }
        }
        P.coeffs = d_coeffs + lo * ncoef; P.out = d_counts + lo * g; P.out_r0 = need_r0 ? d_r0 + lo * g : nullptr; P.n = nc; P.row0 = lo;
        if (shift) {                                           // pre-pass: no empty residue class mod R (hec_shift_kernel)
            uint16_t *d_sh = static_cast<uint16_t *>(S.d_shift) + lo * ncoef;
            if ((rc = run_shift(S, *plan, P.coeffs, nc, d_sh))) return rc;
            P.coeffs = d_sh;
        }
        switch (g) {
            case 1: rc = hec_launch_count_g1(S, *plan, P); break;
            case 2: rc = hec_launch_count_g2(S, *plan, P); break;
            case 3: rc = hec_launch_count_g3(S, *plan, P); break;
            case 4: rc = hec_launch_count_g4(S, *plan, P); break;
            default: rc = hec_launch_count_g5(S, *plan, P); break;
        }
        if (rc) return rc;
        if (c == chunks - 1) HEC_CUDA_OK(cudaEventRecord(S.ev[1], S.stream));
        if (d_sf || d_lam) {
            HecSquarefreeParams Q;
            Q.coeffs = d_coeffs + lo * ncoef; Q.out = d_sf ? d_sf + lo : nullptr; Q.n = nc; Q.p = p; Q.q = q; Q.M = q - 1; Q.ncoef = (uint32_t)ncoef;
            Q.zech = plan->sq_zech; Q.emb = plan->sq_emb;
            Q.roots = d_lam ? d_r0 + lo * g : nullptr; Q.out_lambda = d_lam ? d_lam + lo : nullptr;
            Q.part_codes = plan->d_part_codes; Q.n_parts = plan->n_parts; Q.g = g;
            const unsigned long long blocks = (nc + 255) / 256;
            hec_squarefree_kernel<<<(unsigned)blocks, 256, 0, S.stream>>>(Q);
            hec_launch_counter::value++;
            S.stats.launches++;
            HEC_CUDA_OK(cudaGetLastError());
        }
        if (!dev_in) {
            if (chunks > 1) {
                HEC_CUDA_OK(cudaEventRecord(S.ev_chunk[2 + 2 * c], S.stream));
                HEC_CUDA_OK(cudaStreamWaitEvent(s_out, S.ev_chunk[2 + 2 * c], 0));
            }
            HEC_CUDA_OK(cudaMemcpyAsync(out_counts + lo * g, d_counts + lo * g, nc * g * sizeof(uint32_t), cudaMemcpyDeviceToHost, s_out));
            if (out_squarefree) HEC_CUDA_OK(cudaMemcpyAsync(out_squarefree + lo, d_sf + lo, nc, cudaMemcpyDeviceToHost, s_out));
            if (out_roots) HEC_CUDA_OK(cudaMemcpyAsync(out_roots + lo * g, d_r0 + lo * g, nc * g * sizeof(uint32_t), cudaMemcpyDeviceToHost, s_out));
            if (out_lambda) HEC_CUDA_OK(cudaMemcpyAsync(out_lambda + lo, d_lam + lo, nc, cudaMemcpyDeviceToHost, s_out));
        }
    }
    HEC_CUDA_OK(cudaEventRecord(S.ev[2], S.stream));
    HEC_CUDA_OK(cudaMemcpyAsync(T.err, plan->d_err, sizeof T.err, cudaMemcpyDeviceToHost, S.stream));
    T.pending = chunks > 1;
    drain.armed = false;                                       // from here on finish_count waits for the copies
    if (keep_device) return HEC_OK;
    return finish_count(S, T);
}

int check_count_args(uint32_t q, uint32_t g) {
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    uint32_t p, r;
    if (!hec_factor_q(q, &p, &r)) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q must be an odd prime power below 65536");
    uint64_t Qg = 1;
    for (uint32_t i = 0; i < g; i++) { Qg *= q; if (Qg > HEC_MAX_FIELD_SIZE) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q^g exceeds HEC_MAX_FIELD_SIZE (2^26)"); }
    return HEC_OK;
}

}  // namespace

int hec_histogram_mixed(const uint32_t *counts, const uint8_t *mask, size_t n, uint32_t g, uint32_t *out_tuples, uint64_t *out_mult,
                        size_t cap, size_t *out_m);

extern "C" {

int hec_count_ex(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t *out_counts, uint8_t *out_squarefree,
                 uint32_t *out_roots, uint8_t *out_lambda) {
    int rc = check_count_args(q, g);
    if (rc) return rc;
    if (n == 0) return HEC_OK;
    if (!coeffs || !out_counts) HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs and out_counts must not be NULL");
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    LibState &S = g_state;
    if ((rc = ensure_device(S))) return rc;
    CountTail T;
    return count_impl(S, q, g, coeffs, n, out_counts, out_squarefree, out_roots, out_lambda, false, T);
}

int hec_count_histogram(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t *out_counts, uint8_t *out_squarefree,
                        uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m) {
    int rc = check_count_args(q, g);
    if (rc) return rc;
    if (!out_m) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_m must not be NULL");
    *out_m = 0;
    if (n == 0) return HEC_OK;
    if (!coeffs || !out_counts) HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs and out_counts must not be NULL");
    if (cap > 0 && (!out_tuples || !out_mult)) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_tuples/out_mult must not be NULL when cap > 0");
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    LibState &S = g_state;
    if ((rc = ensure_device(S))) return rc;
    const bool dev = is_device_pointer(coeffs);
    if (cap > 0 && (is_device_pointer(out_tuples) != dev || is_device_pointer(out_mult) != dev))
        HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs/out_counts/out_squarefree/out_tuples/out_mult must all be host or all device pointers");
    CountTail T;
    if ((rc = count_impl(S, q, g, coeffs, n, out_counts, out_squarefree, nullptr, nullptr, true, T))) return rc;
    // the histogram reads the device copies (for host callers: while the last D2H copies of the counts are still running)
    const hec_count_stats keep = S.stats;
    const int hrc = hec_histogram_mixed(T.d_counts, T.d_sf, n, g, out_tuples, out_mult, cap, out_m);
    S.stats = keep;
    rc = finish_count(S, T);
    return rc ? rc : hrc;
}

int hec_set_field_variant(uint32_t v) {
    if (v > 16u) HEC_FAIL(HEC_ERR_INVALID_ARG, "variant must be at most 16");
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    hec_set_field_variant_impl(v);
    g_state.plans.clear();                        // plans hold tables of the previous representation
    return HEC_OK;
}

int hec_set_fast_tables(int on) {
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    g_state.fast_enabled = on != 0;
    return HEC_OK;
}

int hec_set_shift(int on) {
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    g_state.shift_enabled = on != 0;
    return HEC_OK;
}

int hec_shift_rows(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint16_t *out_coeffs) {
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    if (n == 0) return HEC_OK;
    if (!coeffs || !out_coeffs) HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs and out_coeffs must not be NULL");
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    LibState &S = g_state;
    int rc = ensure_device(S);
    if (rc) return rc;
    const bool dev = is_device_pointer(coeffs);
    if (is_device_pointer(out_coeffs) != dev) HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs/out_coeffs must both be host or both device pointers");
    DevicePlan *plan = nullptr;
    if ((rc = build_plan(S, q, g, S.regime, S.eval, &plan))) return rc;
    const size_t bytes = n * (2 * (size_t)g + 3) * sizeof(uint16_t);
    if (!plan->shift_R) {                                      // no pre-pass for this plan: the rows pass through
        HEC_CUDA_OK(cudaMemcpyAsync(out_coeffs, coeffs, bytes, cudaMemcpyDefault, S.stream));
        HEC_CUDA_OK(cudaStreamSynchronize(S.stream));
        return HEC_OK;
    }
    void *d_in = nullptr;
    cudaError_t ce = cudaSuccess;
    if (!dev) {
        if (cudaMalloc(&d_in, bytes) != cudaSuccess) { cudaGetLastError(); HEC_FAIL(HEC_ERR_NOMEM, "cannot allocate device rows"); }
        ce = cudaMemcpyAsync(d_in, coeffs, bytes, cudaMemcpyHostToDevice, S.stream);
    }
    if (ce == cudaSuccess) rc = run_shift(S, *plan, dev ? coeffs : static_cast<const uint16_t *>(d_in), n, dev ? out_coeffs : nullptr);
    if (ce == cudaSuccess && rc == HEC_OK && !dev) ce = cudaMemcpyAsync(out_coeffs, S.d_shift, bytes, cudaMemcpyDeviceToHost, S.stream);
    const cudaError_t se = cudaStreamSynchronize(S.stream);    // always: nothing may still run when d_in is freed
    if (ce == cudaSuccess) ce = se;
    if (d_in) cudaFree(d_in);
    if (rc) return rc;
    if (ce != cudaSuccess) { cudaGetLastError(); hec_set_error(HEC_ERR_CUDA, std::string("hec_shift_rows: ") + cudaGetErrorString(ce)); return HEC_ERR_CUDA; }
    return HEC_OK;
}

int hec_lambda_partitions(uint32_t g, uint8_t *out_parts, size_t cap, size_t *out_count) {
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    if (!out_count) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_count must not be NULL");
    const std::vector<std::vector<uint8_t>> parts = hec_partitions_of(2 * g + 2);
    *out_count = parts.size();
    if (cap < parts.size()) HEC_FAIL(HEC_ERR_CAPACITY, "hec_lambda_partitions: cap is smaller than the number of partitions");
    if (!out_parts) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_parts must not be NULL");
    for (size_t t = 0; t < parts.size(); t++) std::copy(parts[t].begin(), parts[t].end(), out_parts + t * (2 * g + 2));
    return HEC_OK;
}

void hec_shutdown(void) {
    std::lock_guard<std::recursive_mutex> lock(g_state.mu);
    g_state.plans.clear();
    if (g_state.d_stage) { cudaFree(g_state.d_stage); g_state.d_stage = nullptr; g_state.stage_bytes = 0; }
    if (g_state.d_shift) { cudaFree(g_state.d_shift); g_state.d_shift = nullptr; g_state.shift_bytes = 0; }
    hec_histogram_release_pool();
    hec_clear_field_cache();
    for (auto &e : g_state.ev) if (e) { cudaEventDestroy(e); e = nullptr; }
    for (auto &e : g_state.ev_chunk) if (e) { cudaEventDestroy(e); e = nullptr; }
    if (g_state.copy_in) { cudaStreamDestroy(g_state.copy_in); g_state.copy_in = nullptr; }
    if (g_state.copy_out) { cudaStreamDestroy(g_state.copy_out); g_state.copy_out = nullptr; }
    g_state.device_ready = false;                 // the next call binds to the device current then
    // Settings that belong to the released device or representation go back to their defaults: a stream of the old device
    // is an invalid handle on the next one, and plans of another field variant are gone with the plans.
    g_state.stream = nullptr;
    hec_set_field_variant_impl(0);
}

}  // extern "C"
