// hec_build_field: host-side construction of F_{q^k} in Zech-logarithm form.
// PAPER.md:203-221 (section 2.3: generator, Zech logarithm m(k)), PAPER.md:247-255 (section 3.1-3.2:
// encoding (3.1) with the zero element at q-1, table (3.2)).  The paper obtains generator and tables
// from FLINT; here the generator is t modulo the lexicographically smallest primitive
// polynomial (reading G7) and the tables come from one walk through the powers of t.
#include <algorithm>
#include <atomic>
#include <map>
#include <memory>
#include <mutex>
#include <tuple>

#include "hec_internal.h"

namespace {

thread_local std::string g_err_msg;
thread_local size_t g_err_index = (size_t)-1;

bool is_odd_prime(uint32_t p) {
    if (p < 3 || p % 2 == 0) return false;
    for (uint32_t d = 3; (uint64_t)d * d <= p; d += 2)
        if (p % d == 0) return false;
    return true;
}

// Elements are integers sum a_i p^i; Digits is the unpacked little-endian digit vector.
struct Ring {
    uint32_t p, n;
    std::vector<uint32_t> mod;   // n+1, monic
    std::vector<uint32_t> pw;    // p^i
};

void unpack(const Ring &R, uint32_t e, uint32_t *d) {
    for (uint32_t i = 0; i < R.n; i++) { d[i] = e % R.p; e /= R.p; }
}
uint32_t pack(const Ring &R, const uint32_t *d) {
    uint32_t e = 0;
    for (uint32_t i = R.n; i-- > 0;) e = e * R.p + d[i];
    return e;
}
// e * t mod P: shift the digits up and fold the overflow digit back with t^n = -(a_{n-1} t^{n-1} + .. + a_0)
uint32_t mul_by_t(const Ring &R, uint32_t e) {
    uint32_t d[32], s[32];
    unpack(R, e, d);
    uint32_t top = d[R.n - 1];
    s[0] = 0;
    for (uint32_t i = 1; i < R.n; i++) s[i] = d[i - 1];
    if (top)
        for (uint32_t i = 0; i < R.n; i++)
            s[i] = (uint32_t)((s[i] + (uint64_t)(R.p - top) * R.mod[i]) % R.p);
    return pack(R, s);
}
uint32_t add_enc(const Ring &R, uint32_t a, uint32_t b) {
    uint32_t da[32], db[32];
    unpack(R, a, da); unpack(R, b, db);
    for (uint32_t i = 0; i < R.n; i++) da[i] = (da[i] + db[i]) % R.p;
    return pack(R, da);
}
uint32_t scale_enc(const Ring &R, uint32_t a, uint32_t c) {   // c in F_p
    uint32_t da[32];
    unpack(R, a, da);
    for (uint32_t i = 0; i < R.n; i++) da[i] = (uint32_t)(((uint64_t)da[i] * c) % R.p);
    return pack(R, da);
}

// Walk 1, t, t^2, ...; P is primitive iff the walk first returns to 1 after exactly Q-1 steps.
// On success antilog holds the Q-1 powers.
bool walk_powers(const Ring &R, uint32_t Q, std::vector<uint32_t> &antilog) {
    if (R.mod[0] == 0) return false;
    antilog.resize(Q - 1);
    uint32_t e = 1;
    for (uint32_t i = 0; i < Q - 1; i++) {
        if (i > 0 && e == 1) return false;
        antilog[i] = e;
        e = mul_by_t(R, e);
    }
    return e == 1;
}

std::mutex g_cache_mutex;
std::atomic<bool> g_device_build{false};
std::atomic<uint32_t> g_variant{0};          // hec_set_field_variant: which primitive polynomial the library's own fields use
std::map<std::tuple<uint32_t, uint32_t, uint32_t, uint32_t>, std::unique_ptr<hec_field>> g_cache;

// skip: take the (skip+1)-th lexicographically smallest primitive polynomial (0: the smallest, reading G7)
hec_field *build_field_impl(uint32_t p, uint32_t r, uint32_t k, uint32_t skip = 0) {
    if (!is_odd_prime(p)) { hec_set_error(HEC_ERR_INVALID_FIELD, "p must be an odd prime"); return nullptr; }
    if (r < 1 || k < 1) { hec_set_error(HEC_ERR_INVALID_FIELD, "r and k must be >= 1"); return nullptr; }
    uint64_t q64 = 1, Q64 = 1;
    for (uint32_t i = 0; i < r; i++) { q64 *= p; if (q64 > HEC_MAX_FIELD_SIZE) break; }
    for (uint32_t i = 0; i < r * k && Q64 <= HEC_MAX_FIELD_SIZE; i++) Q64 *= p;
    if (q64 > HEC_MAX_FIELD_SIZE || Q64 > HEC_MAX_FIELD_SIZE) {
        hec_set_error(HEC_ERR_INVALID_FIELD, "q^k exceeds HEC_MAX_FIELD_SIZE (2^26)");
        return nullptr;
    }
    std::unique_ptr<hec_field> F(new hec_field);
    F->p = p; F->r = r; F->k = k; F->n = r * k;
    F->q = (uint32_t)q64; F->Q = (uint32_t)Q64;
    const uint32_t n = F->n, Q = F->Q, M = Q - 1;

    Ring R;
    R.p = p; R.n = n; R.mod.assign(n + 1, 0); R.mod[n] = 1;
    R.pw.assign(n + 1, 1);
    for (uint32_t i = 1; i <= n; i++) R.pw[i] = R.pw[i - 1] * p;

    // lexicographic order of (a_{n-1}, .., a_0): a_0 runs fastest, i.e. count e = sum a_i p^i upwards
    bool found = false;
    uint32_t seen = 0;
    for (uint32_t e = 1; e < Q && !found; e++) {
        unpack(R, e, R.mod.data());
        R.mod[n] = 1;
        if (n == 1) {
            // degree 1: t = -a_0 as an element of F_p; walk the powers of that residue
            uint32_t gen = (p - R.mod[0]) % p;
            if (gen == 0) continue;
            F->antilog.assign(M, 0);
            uint32_t x = 1; bool ok = true;
            for (uint32_t i = 0; i < M; i++) {
                if (i > 0 && x == 1) { ok = false; break; }
                F->antilog[i] = x;
                x = (uint32_t)(((uint64_t)x * gen) % p);
            }
            found = ok && x == 1;
        } else {
            found = walk_powers(R, Q, F->antilog);
        }
        if (found && seen < skip) { seen++; found = false; }
    }
    if (!found) {
        if (skip) hec_set_error(HEC_ERR_INVALID_FIELD, "hec_set_field_variant: variant " + std::to_string(skip) + " exceeds the number of primitive polynomials of this field (" + std::to_string(seen) + " of that degree)");
        else hec_set_error(HEC_ERR_INVALID_FIELD, "no primitive polynomial found");
        return nullptr;
    }
    F->modulus = R.mod;

    F->log.assign(Q, M);                       // log[0] = Q-1 (encoding (3.1))
    for (uint32_t i = 0; i < M; i++) F->log[F->antilog[i]] = i;
    F->zech.assign(M, M);
    for (uint32_t i = 0; i < M; i++) {
        uint32_t e = F->antilog[i];
        uint32_t d0 = e % p;
        uint32_t e1 = e - d0 + (d0 + 1) % p;   // 1 + alpha^i
        F->zech[i] = F->log[e1];               // Q-1 when 1 + alpha^i = 0 (table (3.2))
    }

    // embedding of F_q (reading G6)
    F->embed.assign(F->q, M);
    F->embed_unit = 1;
    if (r == 1) {
        for (uint32_t c = 1; c < p; c++) F->embed[c] = F->log[c];          // constants
    } else if (k == 1) {
        for (uint32_t c = 1; c < F->q; c++) F->embed[c] = F->log[c];       // same modulus R_q
    } else {
        const hec_field *Fq = hec_cached_field(p, r, 1);
        if (!Fq) return nullptr;
        const std::vector<uint32_t> &Rq = Fq->modulus;                      // degree r
        const uint32_t Mq = F->q - 1, step = M / Mq;
        uint32_t rho_log = M;
        for (uint32_t s = 1; s < Mq; s++) {                                 // q >= 9 here, so Mq >= 8
            if (std::__gcd(s, Mq) != 1) continue;
            uint64_t lr = ((uint64_t)s * step) % M;                         // candidate rho = alpha^(s*step)
            uint32_t acc = 0;                                               // R_q(rho)
            for (uint32_t i = 0; i <= r; i++)
                if (Rq[i]) acc = add_enc(R, acc, scale_enc(R, F->antilog[(lr * i) % M], Rq[i]));
            if (acc == 0) { rho_log = (uint32_t)lr; F->embed_unit = s; break; }
        }
        if (rho_log == M) { hec_set_error(HEC_ERR_INVALID_FIELD, "no root of R_q found in F_{q^k}"); return nullptr; }
        for (uint32_t c = 1; c < F->q; c++) {
            uint32_t acc = 0, v = c;
            for (uint32_t i = 0; i < r; i++) {
                uint32_t a = v % p; v /= p;
                if (a) acc = add_enc(R, acc, scale_enc(R, F->antilog[((uint64_t)rho_log * i) % M], a));
            }
            F->embed[c] = F->log[acc];
        }
    }
    return F.release();
}

}  // namespace

void hec_set_error(int code, const std::string &msg, size_t index) {
    (void)code;
    g_err_msg = msg;
    g_err_index = index;
}

bool hec_factor_q(uint32_t q, uint32_t *p_out, uint32_t *r_out) {
    if (q < 3 || q >= 65536) return false;
    for (uint32_t p = 3; p <= q; p += 2) {
        if (q % p) continue;
        if (!is_odd_prime(p)) return false;
        uint32_t v = q, r = 0;
        while (v % p == 0) { v /= p; r++; }
        if (v != 1) return false;
        *p_out = p; *r_out = r;
        return true;
    }
    return false;
}

const hec_field *hec_cached_field(uint32_t p, uint32_t r, uint32_t k) {
    // F_q itself keeps the smallest polynomial: for q = p^r, r > 1 it fixes the encoding of the inputs (hec.h), and the
    // reduced polynomials of Algorithm 1 are defined through its generator (hec_enum.cu)
    const uint32_t skip = k == 1 ? 0u : g_variant.load();
    {
        std::lock_guard<std::mutex> lock(g_cache_mutex);
        auto it = g_cache.find(std::make_tuple(p, r, k, skip));
        if (it != g_cache.end()) return it->second.get();
    }
    uint64_t Q = 1;
    for (uint32_t i = 0; i < r * k && Q <= HEC_MAX_FIELD_SIZE; i++) Q *= p;
    const bool on_device = g_device_build.load() && Q > kDeviceBuildMinQ && Q <= HEC_MAX_FIELD_SIZE && p < 65536;
    hec_field *F = on_device ? hec_build_field_device_impl(p, r, k, skip) : build_field_impl(p, r, k, skip);   // may recurse into the cache for (p, r, 1)
    if (!F) return nullptr;
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    auto &slot = g_cache[std::make_tuple(p, r, k, skip)];
    if (slot) { delete F; return slot.get(); }
    slot.reset(F);
    return F;
}

void hec_allow_device_field_build(bool on) { g_device_build.store(on); }
void hec_set_field_variant_impl(uint32_t v) { g_variant.store(v); }

void hec_clear_field_cache() {
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    g_cache.clear();
}

extern "C" {

const char *hec_last_error(void) { return g_err_msg.c_str(); }
size_t hec_last_error_index(void) { return g_err_index; }

hec_field *hec_build_field(uint32_t p, uint32_t r, uint32_t k) { return build_field_impl(p, r, k); }
void hec_free_field(hec_field *F) { delete F; }

uint32_t hec_field_p(const hec_field *F) { return F ? F->p : 0; }
uint32_t hec_field_degree(const hec_field *F) { return F ? F->n : 0; }
uint32_t hec_field_q(const hec_field *F) { return F ? F->q : 0; }
uint32_t hec_field_Q(const hec_field *F) { return F ? F->Q : 0; }
uint32_t hec_field_embed_unit(const hec_field *F) { return F ? F->embed_unit : 0; }
void hec_field_modulus(const hec_field *F, uint32_t *out) { if (F && out) std::copy(F->modulus.begin(), F->modulus.end(), out); }
void hec_field_antilog(const hec_field *F, uint32_t *out) { if (F && out) std::copy(F->antilog.begin(), F->antilog.end(), out); }
void hec_field_log(const hec_field *F, uint32_t *out) { if (F && out) std::copy(F->log.begin(), F->log.end(), out); }
void hec_field_zech(const hec_field *F, uint32_t *out) { if (F && out) std::copy(F->zech.begin(), F->zech.end(), out); }
void hec_field_embed(const hec_field *F, uint32_t *out) { if (F && out) std::copy(F->embed.begin(), F->embed.end(), out); }

}  // extern "C"
