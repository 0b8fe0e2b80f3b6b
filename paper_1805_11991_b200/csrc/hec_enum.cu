// Algorithm 1 of the paper around the hot path, without lambda:
//   hec_reduced_total / hec_reduced_rows   the reduced polynomials P~'_d(F_q) of sections 1.2-1.3,
//                                          generated on the device from their index, with mult(f);
//   hec_curve_map                          for every reduced f: (N_1..N_g) by hec_count, squarefree filter, then
//                                          "increment N at the tuple and at the tuple of the quadratic twist by mult(f)"
//                                          (Algorithm 1 lines 19-21) as a weighted device histogram.
// Readings: G9 (i, j are the two largest indices below d with nonzero coefficient), G8 (the
// twist is n f, n a non-square: N_k -> 2 q^k + 2 - N_k for odd k, N_k for even k), G18 (the family c_d X^d + X, which
// the printed set omits), G19 (only p not dividing d: the printed set for p | d is incomplete).
//
// Index order of P~'_d (before the squarefree filter), families one after the other.  A "stratum" fixes the coefficients
// at and above `top` and normalises the support below `top`:
//   p not dividing d:  one stratum, top = d-1 (c_{d-1} = 0 by the shift), group order |G| = q (q-1)^2
//   p | d (reading G19): first the stratum c_{d-1} != 0 (c_{d-2} = 0 by the shift, top = d-2, c_{d-1} = 1 .. q-1, |G|),
//                        then the stratum c_{d-1} = 0 (no shift, top = d-1, group {(a, 0, e)} of order (q-1)^2)
// and inside a stratum
//   A0   .. + 1                                                                         mult |group| / (2 (q-1))
//   A1   .. + X           (only if 1 < top; reading G18)                                mult |group| / (2 (q-1))
//   B(i,j), i = 1 .. top-1, j = 0 .. i-1 (j fastest):  .. + X^i + c_j X^j + (c_{j-1} .. c_0 free)
//        c_j = alpha^s, s = 0 .. gamma-1, gamma = gcd(q-1, i-j)  (alpha^0 .. alpha^{gamma-1} represent F_q^x / F_q^{x (i-j)})
//        mult |group| / (2 gamma)
//   index inside a family = (((c_d - 1) n1 + (c_{d-1} - 1)) gamma + s) q^j + sum_{l<j} c_l q^l, n1 = q-1 in the stratum
//   c_{d-1} != 0 (else n1 = 1 and the c_{d-1} term is absent); A0, A1: gamma = 1, j = 0.
#include <cuda_runtime.h>

#include <algorithm>
#include <numeric>
#include <vector>

#include "hec_device.cuh"

cudaStream_t hec_current_stream();
int hec_ensure_device(int *sm_count, int *smem_optin);
bool hec_is_device_pointer(const void *p);
int hec_histogram_weighted(const uint32_t *counts, const uint8_t *mask, const uint64_t *weights, size_t n, uint32_t g,
                           uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m);

namespace {

unsigned long long g_map_chunk_rows = 1ull << 24;   // hec_set_map_chunk_rows

struct Family {
    unsigned long long first;      // index of the family's first polynomial
    unsigned long long qj;         // q^j
    unsigned long long mult;
    uint32_t i, j, gamma;          // A0: i = 0, A1: i = 1, both with j = 0xFFFFFFFF
    uint32_t n1;                   // number of values of c_{d-1}: q-1 (stratum c_{d-1} != 0) or 1 (c_{d-1} = 0)
};

struct EnumParams {
    const Family *fam;             // device copy of the family table
    uint32_t nfam, q, d, ncoef;
    unsigned long long total;
    const uint32_t *antilog;       // F_q: alpha^s in the integer encoding, s < 16 (device)
};

__global__ void __launch_bounds__(256) reduced_rows_kernel(const __grid_constant__ EnumParams E, unsigned long long first,
                                                           unsigned long long n, uint16_t *__restrict__ rows,
                                                           unsigned long long *__restrict__ mult) {
    for (unsigned long long r = blockIdx.x * 256ull + threadIdx.x; r < n; r += gridDim.x * 256ull) {
        const unsigned long long idx = first + r;
        uint32_t lo = 0, hi = E.nfam - 1;                 // last family with fam.first <= idx
        while (lo < hi) {
            const uint32_t mid = (lo + hi + 1) >> 1;
            if (E.fam[mid].first <= idx) lo = mid; else hi = mid - 1;
        }
        const Family &F = E.fam[lo];
        unsigned long long t = idx - F.first;
        uint16_t c[2 * HEC_MAX_GENUS + 3];
#pragma unroll
        for (int l = 0; l < 2 * (int)HEC_MAX_GENUS + 3; l++) c[l] = 0;
        if (F.j == 0xFFFFFFFFu) {
            c[F.i] = 1;
        } else {
            unsigned long long low = t % F.qj;
            t /= F.qj;
            const uint32_t s = (uint32_t)(t % F.gamma);
            t /= F.gamma;
            for (uint32_t l = 0; l < F.j; l++) { c[l] = (uint16_t)(low % E.q); low /= E.q; }
            c[F.j] = (uint16_t)E.antilog[s];
            c[F.i] = 1;
        }
        if (F.n1 > 1u) { c[E.d - 1] = (uint16_t)(t % F.n1 + 1u); t /= F.n1; }
        c[E.d] = (uint16_t)(t + 1u);
        for (uint32_t l = 0; l < E.ncoef; l++) rows[r * E.ncoef + l] = c[l];
        mult[r] = F.mult;
    }
}

// tuples[m + r] = twist of tuples[r] (reading G8), weights copied.  Rows have `cols` >= g columns; columns beyond g
// (the lambda index: n f factors like f) are copied.
__global__ void __launch_bounds__(256) twist_kernel(uint32_t *tuples, unsigned long long *w, unsigned long long m, uint32_t g,
                                                    uint32_t cols, uint32_t q) {
    for (unsigned long long r = blockIdx.x * 256ull + threadIdx.x; r < m; r += gridDim.x * 256ull) {
        unsigned long long qk = 1;
        for (uint32_t k = 1; k <= cols; k++) {
            qk *= q;
            const uint32_t v = tuples[r * cols + k - 1];
            tuples[(m + r) * cols + k - 1] = (k <= g && (k & 1u)) ? (uint32_t)(2 * qk + 2 - v) : v;
        }
        w[m + r] = w[r];
    }
}

// keys[r] = (N_1 .. N_g, lambda index): the key of the paper's map (1.2).
__global__ void __launch_bounds__(256) append_lambda_kernel(const uint32_t *counts, const uint8_t *lam, unsigned long long n,
                                                            uint32_t g, uint32_t *keys) {
    for (unsigned long long r = blockIdx.x * 256ull + threadIdx.x; r < n; r += gridDim.x * 256ull) {
        for (uint32_t k = 0; k < g; k++) keys[r * (g + 1) + k] = counts[r * g + k];
        keys[r * (g + 1) + g] = lam[r];
    }
}

int build_families(uint32_t q, uint32_t g, uint32_t d, EnumParams &E, std::vector<Family> &fam) {
    uint32_t p, r;
    if (!hec_factor_q(q, &p, &r)) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q must be an odd prime power below 65536");
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    if (d != 2 * g + 1 && d != 2 * g + 2) HEC_FAIL(HEC_ERR_INVALID_ARG, "d must be 2g+1 or 2g+2");
    E.q = q; E.d = d; E.ncoef = 2 * g + 3; E.antilog = nullptr; E.fam = nullptr;
    fam.clear();
    unsigned long long at = 0;
    const unsigned long long Q = q;
    bool overflow = false;
    auto stratum = [&](uint32_t top, uint32_t n1, unsigned long long group) {
        auto push = [&](uint32_t i, uint32_t j, uint32_t gamma, unsigned long long qj) {
            Family F;
            F.first = at; F.qj = qj; F.mult = group / (2ull * (j == 0xFFFFFFFFu ? Q - 1 : gamma)); F.i = i; F.j = j; F.gamma = gamma; F.n1 = n1;
            const unsigned long long per = (Q - 1) * n1 * gamma;
            if (qj > (~0ull - at) / per) overflow = true;
            at += per * qj;
            fam.push_back(F);
        };
        push(0, 0xFFFFFFFFu, 1, 1);
        if (top > 1) push(1, 0xFFFFFFFFu, 1, 1);
        for (uint32_t i = 1; i < top; i++) {
            unsigned long long qj = 1;
            for (uint32_t j = 0; j < i; j++) {
                push(i, j, std::gcd(q - 1, i - j), qj);
                qj *= Q;
            }
        }
    };
    if (d % p) {
        stratum(d - 1, 1, Q * (Q - 1) * (Q - 1));
    } else {
        stratum(d - 2, q - 1, Q * (Q - 1) * (Q - 1));
        stratum(d - 1, 1, (Q - 1) * (Q - 1));
    }
    if (overflow) HEC_FAIL(HEC_ERR_UNSUPPORTED, "the number of reduced polynomials exceeds 2^64");
    E.nfam = (uint32_t)fam.size();
    E.total = at;
    return HEC_OK;
}

}  // namespace

namespace {

struct Scratch {          // plain device buffer, freed on scope exit
    void *p = nullptr;
    ~Scratch() { if (p) cudaFree(p); }
    int alloc(size_t bytes) {
        if (cudaMalloc(&p, std::max<size_t>(bytes, 16)) != cudaSuccess) { cudaGetLastError(); p = nullptr; HEC_FAIL(HEC_ERR_NOMEM, "hec_enum: cudaMalloc failed"); }
        return HEC_OK;
    }
};

// alpha^0 .. alpha^15 of F_q (gamma <= d - 2 <= 10 entries are ever read) and the family table, on the device
int upload_tables(uint32_t q, const std::vector<Family> &fam, Scratch &buf, EnumParams &E) {
    uint32_t p, r;
    hec_factor_q(q, &p, &r);
    const hec_field *Fq = hec_cached_field(p, r, 1);
    if (!Fq) return HEC_ERR_INVALID_FIELD;
    std::vector<uint8_t> h(64 + fam.size() * sizeof(Family));
    uint32_t *gen = reinterpret_cast<uint32_t *>(h.data());
    for (uint32_t s = 0; s < 16; s++) gen[s] = Fq->antilog[s % (q - 1)];
    std::copy(fam.begin(), fam.end(), reinterpret_cast<Family *>(h.data() + 64));
    int rc = buf.alloc(h.size());
    if (rc) return rc;
    HEC_CUDA_OK(cudaMemcpyAsync(buf.p, h.data(), h.size(), cudaMemcpyHostToDevice, hec_current_stream()));
    HEC_CUDA_OK(cudaStreamSynchronize(hec_current_stream()));      // h is a local buffer
    E.antilog = static_cast<const uint32_t *>(buf.p);
    E.fam = reinterpret_cast<const Family *>(static_cast<const uint8_t *>(buf.p) + 64);
    return HEC_OK;
}

int launch_rows(const EnumParams &E, unsigned long long first, size_t n, uint16_t *d_rows, unsigned long long *d_mult, int sms) {
    const unsigned grid = (unsigned)std::min<unsigned long long>((n + 255) / 256, (unsigned long long)sms * 8);
    reduced_rows_kernel<<<grid, 256, 0, hec_current_stream()>>>(E, first, n, d_rows, d_mult);
    hec_launch_counter::value++;
    HEC_CUDA_OK(cudaGetLastError());
    return HEC_OK;
}

}  // namespace

extern "C" {

int hec_reduced_total(uint32_t q, uint32_t g, uint32_t d, uint64_t *out_total) {
    if (!out_total) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_total must not be NULL");
    EnumParams E;
    std::vector<Family> fam;
    int rc = build_families(q, g, d, E, fam);
    if (rc) return rc;
    *out_total = E.total;
    return HEC_OK;
}

int hec_reduced_rows(uint32_t q, uint32_t g, uint32_t d, uint64_t first, size_t n, uint16_t *out_coeffs, uint64_t *out_mult) {
    EnumParams E;
    std::vector<Family> fam;
    int rc = build_families(q, g, d, E, fam);
    if (rc) return rc;
    if (first > E.total || n > E.total - first) HEC_FAIL(HEC_ERR_INVALID_ARG, "index range exceeds hec_reduced_total");
    if (n == 0) return HEC_OK;
    if (!out_coeffs || !out_mult) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_coeffs and out_mult must not be NULL");
    int sms = 0;
    if ((rc = hec_ensure_device(&sms, nullptr))) return rc;
    const bool dev = hec_is_device_pointer(out_coeffs);
    if (hec_is_device_pointer(out_mult) != dev) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_coeffs/out_mult must both be host or both device pointers");
    Scratch gen, rows, mult;
    if ((rc = upload_tables(q, fam, gen, E))) return rc;
    uint16_t *d_rows = out_coeffs;
    unsigned long long *d_mult = reinterpret_cast<unsigned long long *>(out_mult);
    const size_t row_bytes = n * E.ncoef * sizeof(uint16_t);
    if (!dev) {
        if ((rc = rows.alloc(row_bytes)) || (rc = mult.alloc(n * 8))) return rc;
        d_rows = static_cast<uint16_t *>(rows.p);
        d_mult = static_cast<unsigned long long *>(mult.p);
    }
    if ((rc = launch_rows(E, first, n, d_rows, d_mult, sms))) return rc;
    cudaStream_t st = hec_current_stream();
    if (!dev) {
        HEC_CUDA_OK(cudaMemcpyAsync(out_coeffs, d_rows, row_bytes, cudaMemcpyDeviceToHost, st));
        HEC_CUDA_OK(cudaMemcpyAsync(out_mult, d_mult, n * 8, cudaMemcpyDeviceToHost, st));
    }
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    return HEC_OK;
}

// keep_t / keep_w (internal callers): hand the final device buffers over instead of copying them out.
static int curve_map_impl(uint32_t q, uint32_t g, uint32_t d, bool with_lambda, uint64_t range_first, uint64_t range_n, bool whole,
                          uint32_t *out_tuples, uint64_t *out_weights, size_t cap, size_t *out_m,
                          Scratch *keep_t = nullptr, Scratch *keep_w = nullptr) {
    if (!out_m) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_m must not be NULL");
    *out_m = 0;
    if (cap > 0 && (!out_tuples || !out_weights)) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_tuples/out_weights must not be NULL when cap > 0");
    EnumParams E;
    std::vector<Family> fam;
    int rc = build_families(q, g, d, E, fam);
    if (rc) return rc;
    if (with_lambda && g + 1 > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_UNSUPPORTED, "hec_curve_map_lambda: g + 1 key columns exceed the histogram's limit");
    int sms = 0;
    if ((rc = hec_ensure_device(&sms, nullptr))) return rc;
    cudaStream_t st = hec_current_stream();
    Scratch gen;
    if ((rc = upload_tables(q, fam, gen, E))) return rc;
    const uint32_t cols = with_lambda ? g + 1 : g;             // key columns

    if (whole) { range_first = 0; range_n = E.total; }
    if (range_first > E.total || range_n > E.total - range_first) HEC_FAIL(HEC_ERR_INVALID_ARG, "index range exceeds hec_reduced_total");
    if (range_n == 0) return HEC_OK;
    const unsigned long long range_end = range_first + range_n;
    const size_t chunk = (size_t)std::min<unsigned long long>(range_n, g_map_chunk_rows);
    Scratch rows, mult, counts, flags, lam, keys, part_t, part_w, acc_t, acc_w, cat_t, cat_w;
    if ((rc = rows.alloc(chunk * E.ncoef * 2)) || (rc = mult.alloc(chunk * 8)) || (rc = counts.alloc(chunk * g * 4)) ||
        (rc = flags.alloc(chunk)) || (rc = part_t.alloc(chunk * cols * 4)) || (rc = part_w.alloc(chunk * 8))) return rc;
    if (with_lambda && ((rc = lam.alloc(chunk)) || (rc = keys.alloc(chunk * cols * 4)))) return rc;
    size_t acc_m = 0, acc_cap = 0;
    auto grow = [&](Scratch &t, Scratch &w, size_t &have, size_t need) -> int {
        if (need <= have) return HEC_OK;
        Scratch nt, nw;
        int e;
        const size_t want = std::max(need, 2 * have);
        if ((e = nt.alloc(want * cols * 4)) || (e = nw.alloc(want * 8))) return e;
        std::swap(t.p, nt.p); std::swap(w.p, nw.p);      // callers never need the old contents
        have = want;
        return HEC_OK;
    };
    size_t cat_cap = 0;
    for (unsigned long long first = range_first; first < range_end; first += chunk) {
        const size_t n = (size_t)std::min<unsigned long long>(chunk, range_end - first);
        if ((rc = launch_rows(E, first, n, static_cast<uint16_t *>(rows.p), static_cast<unsigned long long *>(mult.p), sms))) return rc;
        // Algorithm 1 lines 6-18 for the chunk, then the weighted histogram of its squarefree rows (line 20)
        if ((rc = hec_count_ex(q, g, static_cast<const uint16_t *>(rows.p), n, static_cast<uint32_t *>(counts.p),
                               static_cast<uint8_t *>(flags.p), nullptr, with_lambda ? static_cast<uint8_t *>(lam.p) : nullptr))) return rc;
        const uint32_t *key_rows = static_cast<const uint32_t *>(counts.p);
        if (with_lambda) {
            append_lambda_kernel<<<(unsigned)std::min<size_t>((n + 255) / 256, (size_t)sms * 8), 256, 0, st>>>(
                static_cast<const uint32_t *>(counts.p), static_cast<const uint8_t *>(lam.p), n, g, static_cast<uint32_t *>(keys.p));
            hec_launch_counter::value++;
            HEC_CUDA_OK(cudaGetLastError());
            key_rows = static_cast<const uint32_t *>(keys.p);
        }
        size_t m = 0;
        if ((rc = hec_histogram_weighted(key_rows, static_cast<const uint8_t *>(flags.p),
                                         static_cast<const uint64_t *>(mult.p), n, cols, static_cast<uint32_t *>(part_t.p),
                                         static_cast<uint64_t *>(part_w.p), chunk, &m))) return rc;
        if (m == 0) continue;
        // running map <- merge(running map, chunk's map)
        if ((rc = grow(cat_t, cat_w, cat_cap, acc_m + m))) return rc;
        if (acc_m) {
            HEC_CUDA_OK(cudaMemcpyAsync(cat_t.p, acc_t.p, acc_m * cols * 4, cudaMemcpyDeviceToDevice, st));
            HEC_CUDA_OK(cudaMemcpyAsync(cat_w.p, acc_w.p, acc_m * 8, cudaMemcpyDeviceToDevice, st));
        }
        HEC_CUDA_OK(cudaMemcpyAsync(static_cast<uint32_t *>(cat_t.p) + acc_m * cols, part_t.p, m * cols * 4, cudaMemcpyDeviceToDevice, st));
        HEC_CUDA_OK(cudaMemcpyAsync(static_cast<uint64_t *>(cat_w.p) + acc_m, part_w.p, m * 8, cudaMemcpyDeviceToDevice, st));
        if ((rc = grow(acc_t, acc_w, acc_cap, acc_m + m))) return rc;
        size_t merged = 0;
        if ((rc = hec_histogram_weighted(static_cast<const uint32_t *>(cat_t.p), nullptr, static_cast<const uint64_t *>(cat_w.p), acc_m + m, cols,
                                         static_cast<uint32_t *>(acc_t.p), static_cast<uint64_t *>(acc_w.p), acc_cap, &merged))) return rc;
        acc_m = merged;
    }
    if (acc_m == 0) return HEC_OK;
    // line 21: the same weight at the tuple of the quadratic twist (reading G8)
    if ((rc = grow(cat_t, cat_w, cat_cap, 2 * acc_m))) return rc;
    HEC_CUDA_OK(cudaMemcpyAsync(cat_t.p, acc_t.p, acc_m * cols * 4, cudaMemcpyDeviceToDevice, st));
    HEC_CUDA_OK(cudaMemcpyAsync(cat_w.p, acc_w.p, acc_m * 8, cudaMemcpyDeviceToDevice, st));
    twist_kernel<<<(unsigned)std::min<size_t>((acc_m + 255) / 256, (size_t)sms * 8), 256, 0, st>>>(
        static_cast<uint32_t *>(cat_t.p), static_cast<unsigned long long *>(cat_w.p), acc_m, g, cols, q);
    hec_launch_counter::value++;
    HEC_CUDA_OK(cudaGetLastError());
    Scratch fin_t, fin_w;
    if ((rc = fin_t.alloc(2 * acc_m * cols * 4)) || (rc = fin_w.alloc(2 * acc_m * 8))) return rc;
    size_t fin_m = 0;
    if ((rc = hec_histogram_weighted(static_cast<const uint32_t *>(cat_t.p), nullptr, static_cast<const uint64_t *>(cat_w.p), 2 * acc_m, cols,
                                     static_cast<uint32_t *>(fin_t.p), static_cast<uint64_t *>(fin_w.p), 2 * acc_m, &fin_m))) return rc;
    *out_m = fin_m;
    if (keep_t && keep_w) { std::swap(keep_t->p, fin_t.p); std::swap(keep_w->p, fin_w.p); return HEC_OK; }
    if (cap < fin_m) HEC_FAIL(HEC_ERR_CAPACITY, "hec_curve_map: cap is smaller than the number of distinct tuples");
    const bool dev = hec_is_device_pointer(out_tuples);
    if (hec_is_device_pointer(out_weights) != dev) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_tuples/out_weights must both be host or both device pointers");
    const cudaMemcpyKind kind = dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    HEC_CUDA_OK(cudaMemcpyAsync(out_tuples, fin_t.p, fin_m * cols * 4, kind, st));
    HEC_CUDA_OK(cudaMemcpyAsync(out_weights, fin_w.p, fin_m * 8, kind, st));
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    return HEC_OK;
}

int hec_set_map_chunk_rows(size_t rows) {
    if (rows < 1024 || rows > (1ull << 28)) HEC_FAIL(HEC_ERR_INVALID_ARG, "chunk rows must be in [2^10, 2^28]");
    g_map_chunk_rows = rows;
    return HEC_OK;
}

int hec_curve_map(uint32_t q, uint32_t g, uint32_t d, uint32_t *out_tuples, uint64_t *out_weights, size_t cap, size_t *out_m) {
    return curve_map_impl(q, g, d, false, 0, 0, true, out_tuples, out_weights, cap, out_m);
}

int hec_curve_map_lambda(uint32_t q, uint32_t g, uint32_t d, uint32_t *out_keys, uint64_t *out_weights, size_t cap, size_t *out_m) {
    return curve_map_impl(q, g, d, true, 0, 0, true, out_keys, out_weights, cap, out_m);
}

// Algorithm 1 in full (line 2: "for d in {2g+1, 2g+2}"): the maps of both degrees merged.
int hec_curve_map_all(uint32_t q, uint32_t g, int with_lambda, uint32_t *out_keys, uint64_t *out_weights, size_t cap, size_t *out_m) {
    if (!out_m) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_m must not be NULL");
    *out_m = 0;
    if (cap > 0 && (!out_keys || !out_weights)) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_keys/out_weights must not be NULL when cap > 0");
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    const uint32_t cols = with_lambda ? g + 1 : g;
    int rc;
    size_t m[2] = {0, 0};
    Scratch t[2], w[2];
    for (int s = 0; s < 2; s++) {
        const uint32_t d = 2 * g + 1 + (uint32_t)s;
        if ((rc = curve_map_impl(q, g, d, with_lambda != 0, 0, 0, true, nullptr, nullptr, 0, &m[s], &t[s], &w[s]))) return rc;
    }
    const size_t total = m[0] + m[1];
    if (total == 0) return HEC_OK;
    cudaStream_t st = hec_current_stream();
    Scratch cat_t, cat_w, fin_t, fin_w;
    if ((rc = cat_t.alloc(total * cols * 4)) || (rc = cat_w.alloc(total * 8)) || (rc = fin_t.alloc(total * cols * 4)) || (rc = fin_w.alloc(total * 8))) return rc;
    size_t at = 0;
    for (int s = 0; s < 2; s++) {
        if (!m[s]) continue;
        HEC_CUDA_OK(cudaMemcpyAsync(static_cast<uint32_t *>(cat_t.p) + at * cols, t[s].p, m[s] * cols * 4, cudaMemcpyDeviceToDevice, st));
        HEC_CUDA_OK(cudaMemcpyAsync(static_cast<uint64_t *>(cat_w.p) + at, w[s].p, m[s] * 8, cudaMemcpyDeviceToDevice, st));
        at += m[s];
    }
    size_t fin_m = 0;
    if ((rc = hec_histogram_weighted(static_cast<const uint32_t *>(cat_t.p), nullptr, static_cast<const uint64_t *>(cat_w.p), total, cols,
                                     static_cast<uint32_t *>(fin_t.p), static_cast<uint64_t *>(fin_w.p), total, &fin_m))) return rc;
    *out_m = fin_m;
    if (cap < fin_m) HEC_FAIL(HEC_ERR_CAPACITY, "hec_curve_map_all: cap is smaller than the number of distinct keys");
    const bool dev = hec_is_device_pointer(out_keys);
    if (hec_is_device_pointer(out_weights) != dev) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_keys/out_weights must both be host or both device pointers");
    const cudaMemcpyKind kind = dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    HEC_CUDA_OK(cudaMemcpyAsync(out_keys, fin_t.p, fin_m * cols * 4, kind, st));
    HEC_CUDA_OK(cudaMemcpyAsync(out_weights, fin_w.p, fin_m * 8, kind, st));
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    return HEC_OK;
}

int hec_curve_map_range(uint32_t q, uint32_t g, uint32_t d, uint64_t first, uint64_t n, int with_lambda, uint32_t *out_keys,
                        uint64_t *out_weights, size_t cap, size_t *out_m) {
    return curve_map_impl(q, g, d, with_lambda != 0, first, n, false, out_keys, out_weights, cap, out_m);
}

}  // extern "C"
