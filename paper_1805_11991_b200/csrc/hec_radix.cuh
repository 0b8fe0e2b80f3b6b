// Radix-R evaluation of f at every x of F_{q^k}^x (not in the paper, which runs one
// Horner chain per x: Algorithm 1 line 8).  f is still evaluated at EVERY x (Algorithm 1 line 7,
// PAPER.md:141); the points are only grouped so that they share work.
//
// M = q^k - 1 is even, so for R in {2, 4, 8} with R | M the R-th roots of unity zeta^j = alpha^{j M/R} lie in the
// field.  Split f(X) = sum_{r<R} X^r F_r(X^R) and put G_r(x) = x^r F_r(x^R).  The R points of the coset
// x mu_R share the R values G_r:
//     f(zeta^j x) = sum_r zeta^{jr} G_r(x)                     (an R-point DFT of (G_r) in Zech arithmetic)
// * G_r: one relative Horner chain in x^R per residue class (hec_count.cu header): #terms - #classes lookups
//   per coset instead of R * deg f.
// * DFT: log2 R stages of R/2 butterflies (a, b) -> (a + w b, a - w b).  In Zech form (reading G5)
//     a + w b = a (1 + w b / a) -> log a + Z[n],   a - w b -> log a + Z[n + M/2],   n = log b - log a + log w
//   (-1 = alpha^{M/2}), so ONE table entry holding the pair (Z[n], Z[n + M/2]) serves both outputs.
//   Decimation in frequency with the output twiddles deferred: value i carries a pending factor zeta^{pend[i]}
//   that only enters the NEXT butterfly's log w, so no log is ever adjusted by itself.
// * The last stage only classifies (zero / parity of the log, reading G4): parity(log a + Z) = parity(log a) ^ parity(Z).
//
// Zero handling without a branch or a select in the hot loop: the tables store 0
// ("multiply by 1") where 1 + alpha^n = 0, so the fast path stays well formed; a running minimum over the
// looked-up values (Z is never 0 otherwise) flags every coset in which some intermediate or final value
// vanished.  Flagged cosets (about 1e-4 of the points) are queued per warp in shared memory and re-evaluated
// 32 at a time by exact_coset(), a plain scalar Zech evaluation that treats the zero element explicitly.
// Classes without any nonzero coefficient (G_r = 0 identically) are warp-uniform and take uniform branches.
//
// Two arithmetics: ArScalar (one coset per 32-bit register) for any table policy, and ArPacked (two cosets
// per register in 16-bit halves, VIADD.16x2 / VIADDMNMX.U16x2 / VIMNMX3.U16x2) for 16-bit fields with 2 M <= 65536.
#pragma once

#include <cstdint>

namespace hec_radix {

constexpr uint32_t kZero = 0x40000000u;      // "the element is zero" in the exact path (any value >= M)
constexpr int kQueueCap = 96;                // flagged cosets per warp: < 32 pending + <= 64 new per pass
constexpr int kScratchWords = 16 + kQueueCap;   // per warp: logs of the coefficients + queue

__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
    uint32_t r;
    asm("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(addr));
    return r;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) {
    uint16_t r;
    asm("ld.shared.u16 %0, [%1];" : "=h"(r) : "r"(addr));
    return r;
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
    uint32_t r;
    asm("ld.shared.u8 %0, [%1];" : "=r"(r) : "r"(addr));
    return r;
}

// ---------------------------------------------------------------------------------------------------------
// Table policies.  pair(n): (Z[n], Z[n + h]) for n in [0, M), h = M/2; single(n): Z[n].  Where the sum is
// zero (n = h for the first, n = 0 for the second) the returned value is unspecified-but-in-range: callers
// test n.  pair_word (PairS16 only): both values in one 32-bit word, 0 where the sum is zero.
// ---------------------------------------------------------------------------------------------------------

// Byte addresses tb + 4 lo16(n2) and tb + 4 hi16(n2) of the entries of a packed pair of indices: mask / shift and
// one LEA each (written as mad.lo so that ptxas does not fold the scaling into a shift + mask + add: 4 instead of
// 6 instructions per packed lookup).
__device__ __forceinline__ void packed_addr(uint32_t tb, uint32_t n2, uint32_t &a0, uint32_t &a1) {
    asm("{.reg .u32 t;\n\tand.b32 t, %2, 0xffff;\n\tmad.lo.u32 %0, t, 4, %3;\n\tshr.u32 t, %2, 16;\n\tmad.lo.u32 %1, t, 4, %3;}"
        : "=r"(a0), "=r"(a1) : "r"(n2), "r"(tb));
}

// PAIR16: shared memory, M 32-bit entries, lo16 = Z[n], hi16 = Z[n + h]  (M <= 32768).
struct PairS16 {
    static constexpr bool kParity = false;
    uint32_t tb;                                             // shared byte address of entry 0
    __device__ __forceinline__ uint32_t pair_word(uint32_t n) const { return lds_u32(tb + 4u * n); }
    __device__ __forceinline__ void pair(uint32_t n, uint32_t, uint32_t, uint32_t &za, uint32_t &zs) const {
        const uint32_t w = pair_word(n);
        za = w & 0xFFFFu;
        zs = w >> 16;
    }
    __device__ __forceinline__ uint32_t single(uint32_t n, uint32_t, uint32_t) const { return lds_u16(tb + 4u * n); }
};

// RHALF32: shared memory, HT[i] = Z[i] for 0 <= i <= h (HT[h] = 0), 32-bit entries.  Z(-m) = Z(m) - m (reading
// G16) gives Z[i + h] = HT[h - i] + i + h (mod M) for 0 <= i < h, so with i = n mod h the pair is
// (HT[i], HT[h - i] + i + h), swapped when n >= h.
// PT: the field also carries a packed parity table (tp: its shared byte address; 2 bits per n: parity of Z[n], of Z[n + h]; four
// entries per byte), which the classifying last stage of the network reads instead of the pair (one load instead of two / three).
template <bool PT>
struct HalfS32T {
    static constexpr bool kParity = PT;
    uint32_t tb, tbh;                                        // shared byte addresses of HT[0] and HT[h]
    uint32_t tp;
    __device__ __forceinline__ void pair(uint32_t n, uint32_t M, uint32_t h, uint32_t &za, uint32_t &zs) const {
        const uint32_t i = min(n, n - h);
        const uint32_t t1 = lds_u32(tb + 4u * i);
        uint32_t t2 = lds_u32(tbh - 4u * i) + i + h;
        t2 = min(t2, t2 - M);
        const bool sw = n >= h;
        za = sw ? t2 : t1;
        zs = sw ? t1 : t2;
    }
    __device__ __forceinline__ uint32_t single(uint32_t n, uint32_t M, uint32_t h) const {
        const uint32_t i = min(n, M - n);
        const uint32_t t = lds_u32(tb + 4u * i);
        const uint32_t u = t + n;
        return n > h ? min(u, u - M) : t;
    }
};

// RHALF17: as RHALF32 for M < 2^17: a 16-bit plane with the low halves of HT[0..h] and a byte plane whose
// entry i holds bit 16 of HT[i] (bit 0) and of HT[h - i] (bit 1): three loads per pair.
using HalfS32 = HalfS32T<false>;

template <bool PT>
struct HalfS17T {
    static constexpr bool kParity = PT;
    uint32_t tb, tbh, bb;                                    // 16-bit plane: HT[0], HT[h]; byte plane
    uint32_t tp;
    __device__ __forceinline__ void pair(uint32_t n, uint32_t M, uint32_t h, uint32_t &za, uint32_t &zs) const {
        const uint32_t i = min(n, n - h);
        const uint32_t l1 = lds_u16(tb + 2u * i), l2 = lds_u16(tbh - 2u * i), b = lds_u8(bb + i);
        const uint32_t t1 = l1 + ((b & 1u) << 16);
        uint32_t t2 = l2 + ((b & 2u) << 15) + i + h;
        t2 = min(t2, t2 - M);
        const bool sw = n >= h;
        za = sw ? t2 : t1;
        zs = sw ? t1 : t2;
    }
    __device__ __forceinline__ uint32_t single(uint32_t n, uint32_t M, uint32_t h) const {
        const uint32_t i = min(n, M - n);
        const uint32_t t = lds_u16(tb + 2u * i) + ((lds_u8(bb + i) & 1u) << 16);
        const uint32_t u = t + n;
        return n > h ? min(u, u - M) : t;
    }
};

using HalfS17 = HalfS17T<false>;

// GPAIR64: global memory (L1/L2-resident regime), M entries (Z[n], Z[n + h]) as uint2.
struct PairG64 {
    static constexpr bool kParity = false;
    const uint2 *t;
    __device__ __forceinline__ void pair(uint32_t n, uint32_t, uint32_t, uint32_t &za, uint32_t &zs) const {
        const uint2 w = __ldg(t + n);
        za = w.x;
        zs = w.y;
    }
    __device__ __forceinline__ uint32_t single(uint32_t n, uint32_t, uint32_t) const { return __ldg(&t[n].x); }
};

// ---------------------------------------------------------------------------------------------------------
// Arithmetics of the fast path.  A value V holds LANES logs in [0, M).
// ---------------------------------------------------------------------------------------------------------
struct ArScalar {
    static constexpr int LANES = 1;
    uint32_t M, h;
    __device__ __forceinline__ ArScalar(uint32_t M_) : M(M_), h(M_ >> 1) {}
    __device__ __forceinline__ uint32_t rep(uint32_t c) const { return c; }
    __device__ __forceinline__ uint32_t wrap(uint32_t x) const { return min(x, x - M); }              // [0, 2M) -> [0, M)
    __device__ __forceinline__ uint32_t subm(uint32_t b, uint32_t a) const { return wrap(b + M - a); }
    __device__ __forceinline__ uint32_t mn_init() const { return 0xFFFFFFFFu; }
    template <typename Pol>
    __device__ __forceinline__ void lookup_pair(const Pol &pol, uint32_t n, uint32_t &za, uint32_t &zs, uint32_t &mn) const {
        pol.pair(n, M, h, za, zs);
        mn = min(mn, min(n, n - h));                          // 0 iff n in {0, h}: one of the two sums vanished
    }
    template <typename Pol>
    __device__ __forceinline__ uint32_t lookup_single(const Pol &pol, uint32_t n, uint32_t &mn) const {
        mn = min(mn, n ^ h);
        return pol.single(n, M, h);
    }
    __device__ __forceinline__ uint32_t parity2(uint32_t a, uint32_t za, uint32_t zs) const { return ((a ^ za) & 1u) + ((a ^ zs) & 1u); }
    __device__ __forceinline__ uint32_t parity1(uint32_t a) const { return a & 1u; }
    // number of odd logs among a + Z[n], a + Z[n + h] from the packed parity table at tp; a zero sum is n = 0 or n = h
    __device__ __forceinline__ uint32_t parity_lookup(uint32_t tp, uint32_t a, uint32_t n, uint32_t &mn) const {
        mn = min(mn, min(n, n - h));
        const uint32_t p = lds_u8(tp + (n >> 2)) >> ((n & 3u) << 1);
        return ((a ^ p) & 1u) + ((a ^ (p >> 1)) & 1u);
    }
    __device__ __forceinline__ bool flagged(uint32_t mn, int) const { return mn == 0u; }
    __device__ __forceinline__ uint32_t keep(uint32_t v, bool k0, bool) const { return k0 ? v : 0u; }
    __device__ __forceinline__ uint32_t total(uint32_t v) const { return v; }
    __device__ __forceinline__ uint32_t join(uint32_t a, uint32_t) const { return a; }
    __device__ __forceinline__ uint32_t weighted(uint32_t v, uint32_t w0, uint32_t) const { return v * w0; }
};

struct ArPacked {
    static constexpr int LANES = 2;
    uint32_t M2, nM2, h2;
    __device__ __forceinline__ ArPacked(uint32_t M_) : M2(M_ * 0x10001u), nM2(((0x10000u - M_) & 0xFFFFu) * 0x10001u), h2((M_ >> 1) * 0x10001u) {}
    __device__ __forceinline__ uint32_t rep(uint32_t c) const { return c * 0x10001u; }
    __device__ __forceinline__ uint32_t wrap(uint32_t x) const { return __viaddmin_u16x2(x, nM2, x); }
    __device__ __forceinline__ uint32_t subm(uint32_t b, uint32_t a) const { return wrap(b + M2 - a); }   // halves stay in (0, 2M): no borrow
    __device__ __forceinline__ uint32_t mn_init() const { return 0xFFFFFFFFu; }
    __device__ __forceinline__ void lookup_pair(const PairS16 &pol, uint32_t n, uint32_t &za, uint32_t &zs, uint32_t &mn) const {
        uint32_t a0, a1;
        packed_addr(pol.tb, n, a0, a1);
        const uint32_t w0 = lds_u32(a0), w1 = lds_u32(a1);
        za = __byte_perm(w0, w1, 0x5410);
        zs = __byte_perm(w0, w1, 0x7632);
        mn = __vimin3_u16x2(mn, za, zs);                      // a stored 0 marks a vanished sum (per coset: per half)
    }
    __device__ __forceinline__ uint32_t lookup_single(const PairS16 &pol, uint32_t n, uint32_t &mn) const {
        uint32_t a0, a1;
        packed_addr(pol.tb, n, a0, a1);
        const uint32_t z0 = lds_u16(a0), z1 = lds_u16(a1);
        const uint32_t z = __byte_perm(z0, z1, 0x5410);
        mn = __vminu2(mn, z);
        return z;
    }
    __device__ __forceinline__ uint32_t parity2(uint32_t a, uint32_t za, uint32_t zs) const {
        return ((a ^ za) & 0x10001u) + ((a ^ zs) & 0x10001u);
    }
    __device__ __forceinline__ uint32_t parity1(uint32_t a) const { return a & 0x10001u; }
    __device__ __forceinline__ bool flagged(uint32_t mn, int c) const { return c ? (mn >> 16) == 0u : (mn & 0xFFFFu) == 0u; }
    __device__ __forceinline__ uint32_t keep(uint32_t v, bool k0, bool k1) const { return v & ((k0 ? 0xFFFFu : 0u) | (k1 ? 0xFFFF0000u : 0u)); }
    __device__ __forceinline__ uint32_t total(uint32_t v) const { return (v & 0xFFFFu) + (v >> 16); }
    __device__ __forceinline__ uint32_t join(uint32_t a, uint32_t b) const { return a | (b << 16); }
    __device__ __forceinline__ uint32_t weighted(uint32_t v, uint32_t w0, uint32_t w1) const { return (v & 0xFFFFu) * w0 + (((v >> 16) * w1) << 16); }
};

// ---------------------------------------------------------------------------------------------------------
// Exact evaluation of one coset (the rare path).  lc[i] = log of c_i in this field (entries with bit i of nz
// clear are not read).  Returns (#nonzero values << 16) | #nonzero values with odd log among f(zeta^j x), j < R.
// ---------------------------------------------------------------------------------------------------------
template <int D, int R, typename Pol>
__device__ __noinline__ uint32_t exact_coset(const Pol pol, const uint32_t M, const uint32_t nz, const volatile uint32_t *lc, const uint32_t n) {
    const uint32_t h = M >> 1, unit = M / R;
    auto wrap = [M](uint32_t x) { return min(x, x - M); };
    uint32_t v[R];
    int pend[R];
    for (int r = 0; r < R; r++) {
        uint32_t acc = kZero;
        for (int i = r + R * ((D - r) / R); i >= r; i -= R) {
            if (acc < M) acc = wrap(acc + R * n);                          // acc * x^R;  R n < M
            if ((nz >> i) & 1u) {                                          // acc + c_i
                const uint32_t b = lc[i];
                if (acc >= M) {
                    acc = b;
                } else {
                    const uint32_t dd = wrap(b + M - acc);
                    acc = dd == h ? kZero : wrap(acc + pol.single(dd, M, h));
                }
            }
        }
        if (acc < M) acc = wrap(acc + r * n);                              // G_r = x^r F_r(x^R);  r n < M
        v[r] = acc;
        pend[r] = 0;
    }
    for (int H = R / 2; H >= 1; H >>= 1)
        for (int blk = 0; blk < R; blk += 2 * H)
            for (int j = 0; j < H; j++) {
                const int i1 = blk + j, i2 = i1 + H;
                const uint32_t off = (uint32_t)((pend[i2] - pend[i1]) & (R - 1)) * unit;
                pend[i2] = (pend[i1] + j * (R / (2 * H))) & (R - 1);
                const uint32_t a = v[i1], b = v[i2];
                uint32_t s, d;
                if (a < M && b < M) {
                    const uint32_t dd = wrap(wrap(b + M - a) + off);
                    uint32_t za, zs;
                    pol.pair(dd, M, h, za, zs);
                    s = dd == h ? kZero : wrap(a + za);
                    d = dd == 0 ? kZero : wrap(a + zs);
                } else if (a < M) {
                    s = a; d = a;
                } else if (b < M) {
                    s = wrap(b + off);
                    d = wrap(s + h);
                } else {
                    s = kZero; d = kZero;
                }
                v[i1] = s;
                v[i2] = d;
            }
    uint32_t res = 0;
    for (int i = 0; i < R; i++)
        if (v[i] < M) res += 0x10000u + (v[i] & 1u);                       // every final pending twiddle is zeta^0
    return res;
}

// ---------------------------------------------------------------------------------------------------------
// Exact evaluation of the queued cosets, one POINT per lane (radix_all_x / radix_fast_x; the orbit scheme keeps
// exact_coset for its weights).  Each group of R lanes takes one queued coset n and lane j of the group evaluates f at
// x = zeta^j alpha^n by the plain Horner rule of Algorithm 1 line 8 in Zech form with the zero element
// handled explicitly: 32 / R cosets per round with every lane busy, where exact_coset walked the
// whole butterfly network in one lane per coset (measured on config 4: 10 % of all issued instructions, with
// 3 of 32 lanes active).  Adds to this lane's nz_exact / odd_exact (the caller sums over the warp anyway).
// ---------------------------------------------------------------------------------------------------------
// f(x) at ONE point x = alpha^lx, lx < M, by the Horner rule in Zech form; returns the log of the value or kZero.
// Straight-line: the term tests are warp-uniform, the zero element is carried as a predicate.
template <int D, typename Pol>
__device__ __forceinline__ uint32_t horner_point(const Pol &pol, const uint32_t M, const uint32_t nz, const volatile uint32_t *sc,
                                                 const uint32_t lx) {
    const uint32_t h = M >> 1;
    auto wrap = [M](uint32_t x) { return min(x, x - M); };
    uint32_t acc = 0;
    bool zero = true;
#pragma unroll
    for (int i = D; i >= 0; i--) {
        acc = wrap(acc + lx);                                              // acc * x (kept in range also while zero)
        if ((nz >> i) & 1u) {                                              // acc + c_i
            const uint32_t b = sc[i];
            const uint32_t dd = wrap(b + M - acc);
            const uint32_t s = wrap(acc + pol.single(dd, M, h));
            const bool cancel = !zero && dd == h;
            acc = zero ? b : s;
            zero = cancel;
        }
    }
    return zero ? kZero : acc;
}

// WEIGHTED (orbit scheme): a queue entry is n | (orbit length << 28) and every count is multiplied by the orbit length.
template <int D, int R, typename Pol, bool WEIGHTED = false>
__device__ __noinline__ void exact_queue(const Pol pol, const uint32_t M, const uint32_t nz, const volatile uint32_t *sc,
                                         const uint32_t qn, const uint32_t lane, uint32_t &nz_exact, uint32_t &odd_exact) {
    constexpr uint32_t LG = R == 16 ? 4u : R == 8 ? 3u : R == 4 ? 2u : 1u;
    const uint32_t S = M >> LG;
    const uint32_t j = lane & (uint32_t)(R - 1), slot = lane >> LG;
    for (uint32_t q0 = 0; q0 < qn; q0 += 32u / R) {
        const uint32_t qi = min(q0 + slot, qn - 1u);                       // idle slots repeat the last coset (not counted)
        const uint32_t e = sc[16 + qi];
        const uint32_t n = WEIGHTED ? (e & 0x0FFFFFFFu) : e, w = WEIGHTED ? (e >> 28) : 1u;
        const uint32_t acc = horner_point<D>(pol, M, nz, sc, n + j * S);   // log x < M
        if (q0 + slot < qn && acc < M) { nz_exact += w; odd_exact += w * (acc & 1u); }
    }
}

// Every x != 0 of a tiny field (M <= 64) by horner_point, one point per lane: there the coset machinery costs more than
// it saves (for q = 13, k = 1 every coset holds an intermediate zero and is re-evaluated anyway).  Returns this lane's
// (#{x: f(x) a nonzero square}, #{x: f(x) = 0}).
template <int D, typename Pol>
__device__ __noinline__ uint2 direct_all_x(const Pol pol, const uint32_t M, const uint32_t lane, const uint32_t nz, const uint32_t lcj,
                                           volatile uint32_t *scratch) {
    __syncwarp();
    if (lane <= (uint32_t)D) scratch[lane] = lcj;
    __syncwarp();
    uint32_t n_sq = 0, n_zero = 0;
    for (uint32_t base = 0; base < M; base += 32u) {
        const uint32_t lx = min(base + lane, M - 1u);
        const uint32_t acc = horner_point<D>(pol, M, nz, scratch, lx);
        if (base + lane < M) {
            n_zero += acc >= M ? 1u : 0u;
            n_sq += (acc < M && !(acc & 1u)) ? 1u : 0u;
        }
    }
    __syncwarp();
    return make_uint2(n_sq, n_zero);
}

// ---------------------------------------------------------------------------------------------------------
// The butterfly network of the fast path on LANES cosets at once.  present: bit r set iff G_r is not
// identically zero (warp-uniform; some G_r is present because the leading coefficient is nonzero, so no final
// value is identically zero).  Adds to ps the number of odd logs among the values (per lane of V) and folds the
// zero indicator of every lookup into mn.
// ---------------------------------------------------------------------------------------------------------
template <int R, bool ALL, typename Ar, typename Pol>
__device__ __forceinline__ void network(const Ar &ar, const Pol &pol, const uint32_t unit, uint32_t present,
                                        uint32_t (&v)[R], uint32_t &ps, uint32_t &mn) {
    int pend[R];
#pragma unroll
    for (int i = 0; i < R; i++) pend[i] = 0;
#pragma unroll
    for (int H = R / 2; H >= 1; H >>= 1) {
#pragma unroll
        for (int blk = 0; blk < R; blk += 2 * H) {
#pragma unroll
            for (int j = 0; j < H; j++) {
                const int i1 = blk + j, i2 = i1 + H;
                const int oe = (pend[i2] - pend[i1]) & (R - 1);
                pend[i2] = (pend[i1] + j * (R / (2 * H))) & (R - 1);
                const bool pa = ALL || ((present >> i1) & 1u), pb = ALL || ((present >> i2) & 1u);
                if (pa && pb) {
                    uint32_t n = ar.subm(v[i2], v[i1]);
                    if (oe) n = ar.wrap(n + ar.rep((uint32_t)oe * unit));
                    const uint32_t a = v[i1];
                    if constexpr (Pol::kParity) {
                        if (H == 1) {
                            ps += ar.parity_lookup(pol.tp, a, n, mn);
                        } else {
                            uint32_t za, zs;
                            ar.lookup_pair(pol, n, za, zs, mn);
                            v[i1] = ar.wrap(a + za);
                            v[i2] = ar.wrap(a + zs);
                        }
                    } else {
                        uint32_t za, zs;
                        ar.lookup_pair(pol, n, za, zs, mn);
                        if (H > 1) {
                            v[i1] = ar.wrap(a + za);
                            v[i2] = ar.wrap(a + zs);
                        } else {
                            ps += ar.parity2(a, za, zs);
                        }
                    }
                } else if (pa) {                                           // b = 0: both outputs are a
                    if (H > 1) v[i2] = v[i1];
                    else ps += 2u * ar.parity1(v[i1]);
                } else if (pb) {                                           // a = 0: w b and -w b
                    uint32_t t = v[i2];
                    if (oe) t = ar.wrap(t + ar.rep((uint32_t)oe * unit));
                    const uint32_t u = ar.wrap(t + ar.rep(unit * (R / 2)));
                    if (H > 1) { v[i1] = t; v[i2] = u; }
                    else ps += ar.parity1(t) + ar.parity1(u);
                }
                if (!ALL && (pa || pb)) present |= (1u << i1) | (1u << i2);
            }
        }
    }
}

// Bit r of the result is set iff residue class r mod R holds a nonzero coefficient (nz: bit i set iff c_i != 0).
template <int D, int R>
__device__ __forceinline__ bool all_classes_present(const uint32_t nz) {
    if (D + 1 < R) return false;
    uint32_t m = nz;
#pragma unroll
    for (int s = R; s <= D; s += R) m |= nz >> s;
    return (m & ((1u << R) - 1u)) == (1u << R) - 1u;
}

// ---------------------------------------------------------------------------------------------------------
// All x in F_{q^k}^x for one curve, one warp.  lcj: lane j holds the log of c_j in this field (any value when
// c_j = 0), nz: bit j set iff c_j != 0, scratch: kScratchWords words of shared memory owned by this warp.
// Returns this lane's share of n_zero = #{x != 0: f(x) = 0} and n_sq = #{x != 0: f(x) a nonzero square}, over the
// cosets of part `part` of `splits` (splits = 1: all of them; splits > 1 spreads one curve over many warps, the
// single-curve / small-batch mode of SURVEY.md 8(f) NEXT-2).
// ALL: the caller guarantees that every residue class mod R holds a nonzero coefficient (the straight-line
// network); otherwise the network takes warp-uniform branches around the absent classes.
// ---------------------------------------------------------------------------------------------------------
// Not inlined (as radix_fast_x): the loop wants all 64 registers; the kernel's per-curve state is saved around the call.
template <int D, int R, bool ALL, typename Ar, typename Pol>
__device__ __noinline__ uint2 radix_all_x(const Pol pol, const uint32_t M, const uint32_t rcpM, const uint32_t lane,
                                          const uint32_t nz, const uint32_t lcj, volatile uint32_t *scratch,
                                          const uint32_t part, const uint32_t splits) {
    uint32_t n_sq, n_zero;
    constexpr int L = Ar::LANES;
    constexpr int NT = D + 1 > R ? D + 1 - R : 0;      // terms 0 .. NT-1 can continue a chain
    constexpr int NTA = NT > 0 ? NT : 1;
    const Ar ar(M);
    const uint32_t S = M / R, unit = S;
    auto mod = [M, rcpM](uint32_t x) {                 // x mod M for any 32-bit x
        const uint32_t r = x - __umulhi(x, rcpM) * M;
        return r >= M ? r - M : r;
    };

    // this warp's share of the cosets: [c_lo, c_hi), part `part` of `splits` equal chunks (a multiple of 32 L cosets)
    uint32_t c_lo = 0, c_hi = S;
    if (splits > 1u) {
        const uint32_t chunk = ((S + splits - 1u) / splits + 32u * L - 1u) / (32u * L) * (32u * L);
        c_lo = min(S, part * chunk);
        c_hi = min(S, c_lo + chunk);
    }
    if (c_lo >= c_hi) return make_uint2(0u, 0u);       // warp-uniform

    __syncwarp();
    if (lane <= (uint32_t)D) scratch[lane] = lcj;
    __syncwarp();

    // ---- per-curve structure (warp-uniform) and this lane's chain offsets for its first cosets
    uint32_t n0[L];
#pragma unroll
    for (int c = 0; c < L; c++) n0[c] = c_lo + lane + 32u * c < c_hi ? c_lo + lane + 32u * c : 0u;
    const uint32_t step = mod(32u * L);
    uint32_t ul[NTA], inc[NTA], kc[R], kinc[R];
    uint32_t cm = 0, present = 0;
    uint32_t last_lc[R], last_e[R];
#pragma unroll
    for (int r = 0; r < R; r++) { last_lc[r] = 0; last_e[r] = 0; }
#pragma unroll
    for (int i = D; i >= 0; i--) {
        const int r = i % R;
        const uint32_t lci = __shfl_sync(0xffffffffu, lcj, i);
        if (i < NT) { ul[i] = 0; inc[i] = 0; }
        if (nz & (1u << i)) {
            if (i < NT && (present & (1u << r))) {
                const uint32_t m = last_e[r] - (uint32_t)i;
                const uint32_t delta = last_lc[r] >= lci ? last_lc[r] - lci : last_lc[r] + M - lci;
                uint32_t t[2] = {0, 0};
#pragma unroll
                for (int c = 0; c < L; c++) t[c] = mod(delta + m * n0[c]);
                ul[i] = ar.join(t[0], t[1]);
                inc[i] = ar.rep(mod(m * step));
                cm |= 1u << i;
            }
            present |= 1u << r;
            last_lc[r] = lci;
            last_e[r] = (uint32_t)i;
        }
    }
#pragma unroll
    for (int r = 0; r < R; r++) {                      // log G_r = W_r + K_r(n), K_r(n) = log c_{e_T} + e_T n
        uint32_t t[2] = {0, 0};
#pragma unroll
        for (int c = 0; c < L; c++) t[c] = mod(last_lc[r] + last_e[r] * n0[c]);
        kc[r] = ar.join(t[0], t[1]);
        kinc[r] = ar.rep(mod(last_e[r] * step));
    }

    uint32_t acc = 0, odd_fast = 0, passes = 0, pushed = 0, qn = 0, nz_exact = 0, odd_exact = 0;
    auto drain = [&]() { exact_queue<D, R>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact); };
    for (uint32_t base = c_lo; base < c_hi; base += 32u * L) {
        uint32_t v[R];
        uint32_t mn = ar.mn_init();
#pragma unroll
        for (int r = 0; r < R; r++) {
            uint32_t w = 0;
            bool chained = false;
#pragma unroll
            for (int i = NT - 1; i >= 0; i--) {
                if (i % R != r) continue;
                if (cm & (1u << i)) {
                    const uint32_t n = chained ? ar.wrap(w + ul[i]) : ul[i];
                    w = ar.lookup_single(pol, n, mn);
                    ul[i] = ar.wrap(ul[i] + inc[i]);
                    chained = true;
                }
            }
            v[r] = chained ? ar.wrap(w + kc[r]) : kc[r];
            kc[r] = ar.wrap(kc[r] + kinc[r]);
        }
        uint32_t ps = 0;
        network<R, ALL>(ar, pol, unit, present, v, ps, mn);
        bool valid[2] = {false, false}, flag[2] = {false, false};
        bool any_flag = false;
#pragma unroll
        for (int c = 0; c < L; c++) {
            valid[c] = base + lane + 32u * c < c_hi;
            flag[c] = valid[c] && ar.flagged(mn, c);
            any_flag |= flag[c];
        }
        if (__any_sync(0xffffffffu, any_flag)) {       // rare: queue the flagged cosets for exact evaluation
#pragma unroll
            for (int c = 0; c < L; c++) {
                const uint32_t bal = __ballot_sync(0xffffffffu, flag[c]);
                if (flag[c]) {
                    scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = base + lane + 32u * c;
                    pushed++;
                }
                qn += __popc(bal);
            }
            __syncwarp();
            if (qn >= 32u) {
                drain();
                qn = 0;
                __syncwarp();
            }
        }
        acc += ar.keep(ps, valid[0] && !flag[0], valid[1] && !flag[1]);
        if ((++passes & 1023u) == 0u) { odd_fast += ar.total(acc); acc = 0; }      // <= R per lane of V per pass
    }
    odd_fast += ar.total(acc);
    drain();
    __syncwarp();
    uint32_t n_valid = 0;                              // cosets of this lane
#pragma unroll
    for (int c = 0; c < L; c++) {
        const uint32_t first = c_lo + lane + 32u * c;
        if (first < c_hi) n_valid += (c_hi - first + 32u * L - 1u) / (32u * L);
    }
    const uint32_t n_nz = (n_valid - pushed) * R + nz_exact;        // every value of an unflagged coset is nonzero
    const uint32_t n_odd = odd_fast + odd_exact;
    n_zero = n_valid * R - n_nz;
    n_sq = n_nz - n_odd;
    return make_uint2(n_sq, n_zero);
}

// ---------------------------------------------------------------------------------------------------------
// The batch loop for PAIR16 fields (packed arithmetic, one warp per curve, every coset of the field, every residue
// class mod R non-empty with R the field's radix): radix_all_x<D, R, true, ArPacked> with three changes, all measured
// on config 4 (profiles/r01f_ncu_full_c4_radix_first1M.md -> profiles/r02*):
//  * Chain-start lookups.  The first link of the class-r chain reads Z[delta + R n] (the two top terms of the class
//    are R apart): lanes hold consecutive n, so in the pair table the 32 addresses are R words apart -- an R-way bank
//    conflict on every such load (4.04 wavefronts per request against 3.53 for a random gather).  R | M, so
//    delta + R n = c + R ((a + n) mod S) with c = delta mod R, a = delta div R warp-uniform: a transposed copy of Z,
//    T[c][j] = Z[c + R (j mod S)] for j < S + 64 (16-bit entries, rows padded by one pass so that a row never wraps
//    inside a pass), turns them into two conflict-free loads of consecutive entries at a warp-uniform offset.
//    Links that are not of this kind (later links of a chain, top terms 2R or more apart) keep the pair table.
//  * Per-curve set-up without modular reductions: e n mod M for the lane's first cosets (n = lane, lane + 32) and the
//    per-pass step 64 e mod M depend on the field only, so the host tabulates them (lanepow, stepe) for e = 0 .. D.
//  * Validity of the lane's cosets and the zero queue are only looked at in the last pass or after a zero was seen.
// Layout of the field's fast tables at shared byte address ft: [lanepow: (D+1) x 32 words][stepe: D+1 words, padded to
// 16 bytes][T: R rows of rowB bytes]; built by the host (hec_count.cu: fill_fast_tables).
// ---------------------------------------------------------------------------------------------------------
template <int D>
__host__ __device__ constexpr uint32_t fast_tables_head_bytes() { return (uint32_t)(D + 1) * 128u + (((uint32_t)(D + 1) * 4u + 15u) & ~15u); }

// Not inlined on purpose: the loop needs every one of the 64 registers a thread of a 1024-thread CTA can have (8 values,
// 8 + 8 class offsets and steps, the chain state); as a function of its own the kernel's per-curve state is saved around
// the call once per field instead of competing with the loop (inlined, ptxas re-derived constants inside the loop).
template <int D, int R>
__device__ __noinline__ uint2 radix_fast_x(const PairS16 pol, const uint32_t ft, const uint32_t rowB, const uint32_t M,
                                           const uint32_t lane, const uint32_t nz, const uint32_t lcj,
                                           volatile uint32_t *scratch) {
    uint32_t n_sq, n_zero;
    constexpr int NT = D + 1 > R ? D + 1 - R : 0;
    constexpr int NTA = NT > 0 ? NT : 1;
    constexpr uint32_t LG = R == 8 ? 3u : R == 4 ? 2u : 1u;
    const ArPacked ar(M);
    const uint32_t S = M >> LG, unit = S;
    const uint32_t tLP = ft + 4u * lane, tSE = ft + (uint32_t)(D + 1) * 128u, tT = ft + fast_tables_head_bytes<D>() + 2u * lane;

    __syncwarp();
    if (lane <= (uint32_t)D) scratch[lane] = lcj;
    __syncwarp();

    // ---- per-curve structure (warp-uniform masks; per-lane offsets from the field's tables)
    // link i (a nonzero term that continues the chain of its class):
    //   ct bit i: transposed kind, ca[i] = byte offset 2 ((a + base) mod S) (uniform), cb[i] = T + row c + 2 lane
    //   cm bit i: pair-table kind, ca[i] = packed index offsets of the lane's two cosets, cb[i] = their step per pass
    uint32_t ca[NTA], cb[NTA], kc[R], kinc[R];
    uint32_t cm = 0, ct = 0, present = 0, linked = 0;
    uint32_t last_lc[R], last_e[R];
#pragma unroll
    for (int r = 0; r < R; r++) { last_lc[r] = 0; last_e[r] = 0; }
#pragma unroll
    for (int i = D; i >= 0; i--) {
        const int r = i % R;
        const uint32_t lci = __shfl_sync(0xffffffffu, lcj, i);
        if (i < NT) { ca[i] = 0; cb[i] = 0; }
        if (nz & (1u << i)) {
            if (i < NT && (present & (1u << r))) {
                const uint32_t m = last_e[r] - (uint32_t)i;
                const uint32_t delta = last_lc[r] >= lci ? last_lc[r] - lci : last_lc[r] + M - lci;
                if (m == (uint32_t)R && !(linked & (1u << r))) {
                    ca[i] = 2u * (delta >> LG);
                    cb[i] = tT + (delta & (uint32_t)(R - 1)) * rowB;
                    ct |= 1u << i;
                } else {
                    ca[i] = ar.wrap(ar.rep(delta) + lds_u32(tLP + m * 128u));
                    cb[i] = lds_u32(tSE + 4u * m);
                    cm |= 1u << i;
                }
                linked |= 1u << r;
            }
            present |= 1u << r;
            last_lc[r] = lci;
            last_e[r] = (uint32_t)i;
        }
    }
#pragma unroll
    for (int r = 0; r < R; r++) {                      // log G_r = W_r + K_r(n), K_r(n) = log c_{e_T} + e_T n
        kc[r] = ar.wrap(ar.rep(last_lc[r]) + lds_u32(tLP + last_e[r] * 128u));
        kinc[r] = lds_u32(tSE + 4u * last_e[r]);
    }

    uint32_t acc = 0, pushed = 0, qn = 0, nz_exact = 0, odd_exact = 0;
    auto drain = [&]() { exact_queue<D, R>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact); };
    const uint32_t twoS = 2u * S;
    for (uint32_t base = 0; base < S; base += 64u) {
        uint32_t v[R];
        uint32_t mn = ar.mn_init();
#pragma unroll
        for (int r = 0; r < R; r++) {
            uint32_t w = 0;
            bool chained = false;
#pragma unroll
            for (int i = NT - 1; i >= 0; i--) {
                if (i % R != r) continue;
                // a term with no second term of its class above it (i + 2R > D) can only be a first link, R below the top term
                const bool only_t = i + 2 * R > D;
                if (ct & (1u << i)) {                  // always the first link of its chain
                    const uint32_t a0 = cb[i] + ca[i];
                    const uint32_t z0 = lds_u16(a0), z1 = lds_u16(a0 + 64u);
                    w = __byte_perm(z0, z1, 0x5410);
                    mn = __vminu2(mn, w);
                    const uint32_t nx = ca[i] + 128u;
                    ca[i] = min(nx, nx - twoS);
                    chained = true;
                } else if (!only_t && (cm & (1u << i))) {
                    const uint32_t n = chained ? ar.wrap(w + ca[i]) : ca[i];
                    w = ar.lookup_single(pol, n, mn);
                    ca[i] = ar.wrap(ca[i] + cb[i]);
                    chained = true;
                }
            }
            v[r] = chained ? ar.wrap(w + kc[r]) : kc[r];
            kc[r] = ar.wrap(kc[r] + kinc[r]);
        }
        uint32_t ps = 0;
        network<R, true>(ar, pol, unit, present, v, ps, mn);
        const bool zany = ((mn - 0x10001u) & ~mn & 0x80008000u) != 0u;   // some half of mn is 0 (halves are < 2^15 or 0xFFFF)
        if (__any_sync(0xffffffffu, zany) || base + 64u > S) {           // rare: a zero somewhere, or the ragged last pass
            const bool z0 = (mn & 0xFFFFu) == 0u, z1 = (mn >> 16) == 0u;
            const bool valid0 = base + lane < S, valid1 = base + lane + 32u < S;
            const bool flag0 = valid0 && z0, flag1 = valid1 && z1;
            if (__any_sync(0xffffffffu, flag0 || flag1)) {               // queue the flagged cosets for exact evaluation
                uint32_t bal = __ballot_sync(0xffffffffu, flag0);
                if (flag0) { scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = base + lane; pushed++; }
                qn += __popc(bal);
                bal = __ballot_sync(0xffffffffu, flag1);
                if (flag1) { scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = base + lane + 32u; pushed++; }
                qn += __popc(bal);
                __syncwarp();
                if (qn >= 32u) {
                    drain();
                    qn = 0;
                    __syncwarp();
                }
            }
            ps = ar.keep(ps, valid0 && !flag0, valid1 && !flag1);
        }
        acc += ps;                                     // <= R per half and pass, at most S / 64 + 1 <= 257 passes: no carry
    }
    const uint32_t odd_fast = ar.total(acc);
    drain();
    __syncwarp();
    uint32_t n_valid = 0;                              // cosets of this lane
    if (lane < S) n_valid += (S - lane + 63u) / 64u;
    if (lane + 32u < S) n_valid += (S - lane - 32u + 63u) / 64u;
    const uint32_t n_nz = (n_valid - pushed) * R + nz_exact;            // every value of an unflagged coset is nonzero
    const uint32_t n_odd = odd_fast + odd_exact;
    n_zero = n_valid * R - n_nz;
    n_sq = n_nz - n_odd;
    return make_uint2(n_sq, n_zero);
}

// ---------------------------------------------------------------------------------------------------------
// Monomial classes (genus <= 2 on a field with 8 | M, i.e. every F_{q^2}: D + 1 <= 8 terms, at most one per residue
// class mod 8): G_r = c_r x^r needs no chain at all, so the 8 points of a coset cost the butterflies only -- NP - 4 + 8
// pair lookups for NP = deg f + 1 nonzero coefficients against 3 chain + 4 pair lookups per FOUR points at R = 4.  The
// network is specialised at compile time on the present classes 0 .. NP-1 (the shift pre-pass makes every coefficient
// up to the degree nonzero).  For the half-table layout, where a pair costs two loads and a fold, the LAST stage -- which
// only classifies -- reads a 2-bit entry (parity of Z[n], parity of Z[n + M/2]) from a packed parity table instead
// (tp: its shared byte address, four entries per byte); zero sums are seen from n itself (n = 0 or M/2).
// One coset per lane and pass (scalar arithmetic: these fields have more than 2^16 elements).
// ---------------------------------------------------------------------------------------------------------
template <int R, int NP, bool PT, typename Ar, typename Pol>
__device__ __forceinline__ void network_mono(const Ar &ar, const Pol &pol, const uint32_t tp, const uint32_t unit,
                                             uint32_t (&v)[R], uint32_t &ps, uint32_t &mn) {
    int pend[R];
    bool pres[R];
#pragma unroll
    for (int i = 0; i < R; i++) { pend[i] = 0; pres[i] = i < NP; }
#pragma unroll
    for (int H = R / 2; H >= 1; H >>= 1) {
#pragma unroll
        for (int blk = 0; blk < R; blk += 2 * H) {
#pragma unroll
            for (int j = 0; j < H; j++) {
                const int i1 = blk + j, i2 = i1 + H;
                const int oe = (pend[i2] - pend[i1]) & (R - 1);
                pend[i2] = (pend[i1] + j * (R / (2 * H))) & (R - 1);
                const bool pa = pres[i1], pb = pres[i2];              // compile-time after unrolling
                if (pa && pb) {
                    uint32_t n = ar.subm(v[i2], v[i1]);
                    if (oe) n = ar.wrap(n + ar.rep((uint32_t)oe * unit));
                    const uint32_t a = v[i1];
                    if (H > 1 || !PT) {
                        uint32_t za, zs;
                        ar.lookup_pair(pol, n, za, zs, mn);
                        if (H > 1) {
                            v[i1] = ar.wrap(a + za);
                            v[i2] = ar.wrap(a + zs);
                        } else {
                            ps += ar.parity2(a, za, zs);
                        }
                    } else {
                        if constexpr (PT) ps += ar.parity_lookup(tp, a, n, mn);     // scalar arithmetic only
                    }
                } else if (pa) {                                      // b = 0: both outputs are a
                    if (H > 1) v[i2] = v[i1];
                    else ps += 2u * ar.parity1(v[i1]);
                } else if (pb) {                                      // a = 0: w b and -w b
                    uint32_t t = v[i2];
                    if (oe) t = ar.wrap(t + ar.rep((uint32_t)oe * unit));
                    const uint32_t u = ar.wrap(t + ar.rep(unit * (R / 2)));
                    if (H > 1) { v[i1] = t; v[i2] = u; }
                    else ps += ar.parity1(t) + ar.parity1(u);
                }
                if (pa || pb) { pres[i1] = true; pres[i2] = true; }
            }
        }
    }
}

// R = 8 for at most 8 coefficients (genus <= 2), R = 16 for at most 16 (genus 3 .. 6 on fields with 16 | M, e.g. 49^3 - 1:
// 9 coefficients, one butterfly with both inputs in the first stage, 24 in the other three, the last 8 from the parity table).
template <int D, int R, int NP, bool PT, typename Pol>
__device__ __noinline__ uint2 radix_mono_x(const Pol pol, const uint32_t tp, const uint32_t M, const uint32_t lane,
                                           const uint32_t nz, const uint32_t lcj, volatile uint32_t *scratch) {
    static_assert((R == 8 || R == 16) && NP <= R && NP >= R / 2, "monomial classes: one term per class, classes 0 .. NP-1");
    constexpr uint32_t LG = R == 16 ? 4u : 3u;
    const ArScalar ar(M);
    const uint32_t S = M >> LG, unit = S;

    __syncwarp();
    if (lane <= (uint32_t)D) scratch[lane] = lcj;
    __syncwarp();
    uint32_t kc[NP];                                   // log G_r = log c_r + r n for this lane's coset n = base + lane
#pragma unroll
    for (int r = 0; r < NP; r++) kc[r] = ar.wrap(__shfl_sync(0xffffffffu, lcj, r) + (uint32_t)r * lane);     // r lane < 16 * 32 <= M

    uint32_t acc = 0, pushed = 0, qn = 0, nz_exact = 0, odd_exact = 0;
    for (uint32_t base = 0; base < S; base += 32u) {
        uint32_t v[R];
        uint32_t mn = ar.mn_init(), ps = 0;
#pragma unroll
        for (int r = 0; r < R; r++) v[r] = r < NP ? kc[r] : 0u;
#pragma unroll
        for (int r = 1; r < NP; r++) kc[r] = ar.wrap(kc[r] + 32u * (uint32_t)r);
        network_mono<R, NP, PT>(ar, pol, tp, unit, v, ps, mn);
        const bool z = mn == 0u;
        if (__any_sync(0xffffffffu, z) || base + 32u > S) {              // rare: a zero somewhere, or the ragged last pass
            const bool valid = base + lane < S, flag = valid && z;
            const uint32_t bal = __ballot_sync(0xffffffffu, flag);
            if (bal) {
                if (flag) { scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = base + lane; pushed++; }
                qn += __popc(bal);
                __syncwarp();
                if (qn >= 32u) {
                    exact_queue<D, R>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact);
                    qn = 0;
                    __syncwarp();
                }
            }
            ps = (valid && !flag) ? ps : 0u;
        }
        acc += ps;
    }
    exact_queue<D, R>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact);
    __syncwarp();
    const uint32_t n_valid = lane < S ? (S - lane + 31u) / 32u : 0u;
    const uint32_t n_nz = (n_valid - pushed) * R + nz_exact;            // every value of an unflagged coset is nonzero
    const uint32_t n_zero = n_valid * R - n_nz;
    return make_uint2(n_nz - (acc + odd_exact), n_zero);
}

// The same for PAIR16 fields (genus <= 2, q^2 <= 32768: most of the paper's genus-2 range): packed arithmetic, two cosets per
// lane and pass; the lanes' first offsets and the per-pass steps come from the field's fast tables (radix_fast_x).
template <int D, int NP>
__device__ __noinline__ uint2 radix_mono8_packed_x(const PairS16 pol, const uint32_t ft, const uint32_t M, const uint32_t lane,
                                                   const uint32_t nz, const uint32_t lcj, volatile uint32_t *scratch) {
    constexpr int R = 8;
    static_assert(NP <= R && NP >= R / 2, "monomial classes: one term per class, classes 0 .. NP-1");
    const ArPacked ar(M);
    const uint32_t S = M >> 3, unit = S;
    const uint32_t tLP = ft + 4u * lane, tSE = ft + (uint32_t)(D + 1) * 128u;

    __syncwarp();
    if (lane <= (uint32_t)D) scratch[lane] = lcj;
    __syncwarp();
    uint32_t kc[NP], kinc[NP];
#pragma unroll
    for (int r = 0; r < NP; r++) {
        kc[r] = ar.wrap(ar.rep(__shfl_sync(0xffffffffu, lcj, r)) + lds_u32(tLP + (uint32_t)r * 128u));
        kinc[r] = lds_u32(tSE + 4u * (uint32_t)r);
    }
    uint32_t acc = 0, pushed = 0, qn = 0, nz_exact = 0, odd_exact = 0;
    for (uint32_t base = 0; base < S; base += 64u) {
        uint32_t v[R];
        uint32_t mn = ar.mn_init(), ps = 0;
#pragma unroll
        for (int r = 0; r < R; r++) v[r] = r < NP ? kc[r] : 0u;
#pragma unroll
        for (int r = 1; r < NP; r++) kc[r] = ar.wrap(kc[r] + kinc[r]);
        network_mono<R, NP, false>(ar, pol, 0u, unit, v, ps, mn);
        const bool zany = ((mn - 0x10001u) & ~mn & 0x80008000u) != 0u;
        if (__any_sync(0xffffffffu, zany) || base + 64u > S) {
            const bool z0 = (mn & 0xFFFFu) == 0u, z1 = (mn >> 16) == 0u;
            const bool valid0 = base + lane < S, valid1 = base + lane + 32u < S;
            const bool flag0 = valid0 && z0, flag1 = valid1 && z1;
            if (__any_sync(0xffffffffu, flag0 || flag1)) {
                uint32_t bal = __ballot_sync(0xffffffffu, flag0);
                if (flag0) { scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = base + lane; pushed++; }
                qn += __popc(bal);
                bal = __ballot_sync(0xffffffffu, flag1);
                if (flag1) { scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = base + lane + 32u; pushed++; }
                qn += __popc(bal);
                __syncwarp();
                if (qn >= 32u) {
                    exact_queue<D, R>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact);
                    qn = 0;
                    __syncwarp();
                }
            }
            ps = ar.keep(ps, valid0 && !flag0, valid1 && !flag1);
        }
        acc += ps;                                     // <= 8 per half and pass, at most 65 passes: no carry
    }
    exact_queue<D, R>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact);
    __syncwarp();
    uint32_t n_valid = 0;
    if (lane < S) n_valid += (S - lane + 63u) / 64u;
    if (lane + 32u < S) n_valid += (S - lane - 32u + 63u) / 64u;
    const uint32_t n_nz = (n_valid - pushed) * R + nz_exact;
    const uint32_t n_zero = n_valid * R - n_nz;
    return make_uint2(n_nz - (ar.total(acc) + odd_exact), n_zero);
}

// ---------------------------------------------------------------------------------------------------------
// The same, over ONE representative per Frobenius orbit of cosets (HEC_EVAL_ORBIT; not in the
// paper).  f has coefficients in F_q, so f(x^q) = f(x)^q: x and x^q give values that vanish together and are squares
// together.  On logs x -> x^q is n -> q n mod M; it permutes the cosets of mu_R (q is odd, R a power of two), acting on
// the coset index n in Z/(M/R) as multiplication by q, and the R values of coset q n are the q-th powers of those of
// coset n.  reps[t] = n | (orbit length << 28) lists one coset per orbit (built by the host, hec_count.cu); every
// count of a representative is weighted by its orbit length, so the result is the count over EVERY x, but only about
// 1/k of the points are evaluated.  The chain offsets can no longer advance by a constant per pass: each is
// (delta + m n) mod M, one multiply-high reduction per term and coset.
// ---------------------------------------------------------------------------------------------------------
template <int D, int R, bool ALL, typename Ar, typename Pol>
__device__ __noinline__ uint2 radix_orbit_x(const Pol pol, const uint32_t M, const uint32_t rcpM, const uint32_t lane,
                                            const uint32_t nz, const uint32_t lcj, volatile uint32_t *scratch,
                                            const uint32_t *__restrict__ reps, const uint32_t n_reps) {
    uint32_t n_sq, n_zero;
    constexpr int L = Ar::LANES;
    constexpr int NT = D + 1 > R ? D + 1 - R : 0;
    constexpr int NTA = NT > 0 ? NT : 1;
    const Ar ar(M);
    const uint32_t unit = M / R;
    auto mod = [M, rcpM](uint32_t x) {
        const uint32_t r = x - __umulhi(x, rcpM) * M;
        return r >= M ? r - M : r;
    };
    if (n_reps == 0u) return make_uint2(0u, 0u);

    __syncwarp();
    if (lane <= (uint32_t)D) scratch[lane] = lcj;
    __syncwarp();

    uint32_t dl[NTA], mm[NTA];
    uint32_t cm = 0, present = 0;
    uint32_t last_lc[R], last_e[R];
#pragma unroll
    for (int r = 0; r < R; r++) { last_lc[r] = 0; last_e[r] = 0; }
#pragma unroll
    for (int i = D; i >= 0; i--) {
        const int r = i % R;
        const uint32_t lci = __shfl_sync(0xffffffffu, lcj, i);
        if (i < NT) { dl[i] = 0; mm[i] = 0; }
        if (nz & (1u << i)) {
            if (i < NT && (present & (1u << r))) {
                mm[i] = last_e[r] - (uint32_t)i;
                dl[i] = last_lc[r] >= lci ? last_lc[r] - lci : last_lc[r] + M - lci;
                cm |= 1u << i;
            }
            present |= 1u << r;
            last_lc[r] = lci;
            last_e[r] = (uint32_t)i;
        }
    }

    uint32_t acc = 0, odd_fast = 0, passes = 0, qn = 0, nz_exact = 0, odd_exact = 0, w_ok = 0, w_flagged = 0;
    auto drain = [&]() {
        for (uint32_t j = lane; j < qn; j += 32u) {
            const uint32_t e = scratch[16 + j];
            const uint32_t res = exact_coset<D, R>(pol, M, nz, scratch, e & 0x0FFFFFFFu);
            nz_exact += (e >> 28) * (res >> 16);
            odd_exact += (e >> 28) * (res & 0xFFFFu);
        }
    };
    for (uint32_t base = 0; base < n_reps; base += 32u * L) {
        uint32_t nn[2] = {0, 0}, ww[2] = {0, 0};
#pragma unroll
        for (int c = 0; c < L; c++) {
            const uint32_t idx = base + lane + 32u * c;
            const uint32_t e = idx < n_reps ? __ldg(reps + idx) : 0u;     // weight 0: an invalid slot contributes nothing
            nn[c] = e & 0x0FFFFFFFu;
            ww[c] = e >> 28;
        }
        uint32_t v[R];
        uint32_t mn = ar.mn_init();
#pragma unroll
        for (int r = 0; r < R; r++) {
            uint32_t w = 0;
            bool chained = false;
#pragma unroll
            for (int i = NT - 1; i >= 0; i--) {
                if (i % R != r) continue;
                if (cm & (1u << i)) {
                    uint32_t t[2] = {0, 0};
#pragma unroll
                    for (int c = 0; c < L; c++) t[c] = mod(dl[i] + mm[i] * nn[c]);
                    const uint32_t ul = ar.join(t[0], t[1]);
                    const uint32_t n = chained ? ar.wrap(w + ul) : ul;
                    w = ar.lookup_single(pol, n, mn);
                    chained = true;
                }
            }
            uint32_t t[2] = {0, 0};
#pragma unroll
            for (int c = 0; c < L; c++) t[c] = mod(last_lc[r] + last_e[r] * nn[c]);
            const uint32_t kc = ar.join(t[0], t[1]);
            v[r] = chained ? ar.wrap(w + kc) : kc;
        }
        uint32_t ps = 0;
        network<R, ALL>(ar, pol, unit, present, v, ps, mn);
        bool flag[2] = {false, false};
        bool any_flag = false;
#pragma unroll
        for (int c = 0; c < L; c++) {
            flag[c] = ww[c] != 0u && ar.flagged(mn, c);
            any_flag |= flag[c];
        }
        if (__any_sync(0xffffffffu, any_flag)) {
#pragma unroll
            for (int c = 0; c < L; c++) {
                const uint32_t bal = __ballot_sync(0xffffffffu, flag[c]);
                if (flag[c]) {
                    scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = nn[c] | (ww[c] << 28);
                    w_flagged += ww[c];
                    ww[c] = 0u;
                }
                qn += __popc(bal);
            }
            __syncwarp();
            if (qn >= 32u) {
                drain();
                qn = 0;
                __syncwarp();
            }
        }
        acc += ar.weighted(ps, ww[0], ww[1]);           // <= R * k <= 40 per lane of V per pass
        w_ok += ww[0] + ww[1];
        if ((++passes & 1023u) == 0u) { odd_fast += ar.total(acc); acc = 0; }
    }
    odd_fast += ar.total(acc);
    drain();
    __syncwarp();
    const uint32_t n_nz = w_ok * R + nz_exact;          // every value of an unflagged coset is nonzero
    n_zero = w_flagged * R - nz_exact;
    n_sq = n_nz - (odd_fast + odd_exact);
    return make_uint2(n_sq, n_zero);
}

// ---------------------------------------------------------------------------------------------------------
// radix_orbit_x for PAIR16 fields, R in {4, 8}, every class non-empty (HEC_EVAL_ORBIT, round 2).  The offsets e n mod M
// of a representative n are built by repeated addition, n, 2n, .., Dn (one packed add + wrap each), instead of one
// multiply-high reduction per term and coset, and flagged cosets are re-evaluated one point per lane (exact_queue).
// Links whose exponent gap exceeds 2R (possible from D >= 3R on) are left to radix_orbit_x.
// ---------------------------------------------------------------------------------------------------------
template <int D, int R>
__device__ __noinline__ uint2 radix_orbit_fast_x(const PairS16 pol, const uint32_t M, const uint32_t rcpM, const uint32_t lane,
                                                 const uint32_t nz, const uint32_t lcj, volatile uint32_t *scratch,
                                                 const uint32_t *__restrict__ reps, const uint32_t n_reps) {
    constexpr int NT = D + 1 > R ? D + 1 - R : 0;
    constexpr int NTA = NT > 0 ? NT : 1;
    const ArPacked ar(M);
    const uint32_t unit = M / R;
    if (n_reps == 0u) return make_uint2(0u, 0u);

    uint32_t dl[NTA];                                  // chain links: rep(delta)
    uint32_t cm = 0, far = 0, present = 0, topmask = 0;   // far: links whose gap is 2R; topmask: bit e set iff e is the top exponent of its class
    bool ok = true;
    uint32_t last_lc[R], last_e[R];
#pragma unroll
    for (int r = 0; r < R; r++) { last_lc[r] = 0; last_e[r] = 0; }
#pragma unroll
    for (int i = D; i >= 0; i--) {
        const int r = i % R;
        const uint32_t lci = __shfl_sync(0xffffffffu, lcj, i);
        if (i < NT) dl[i] = 0;
        if (nz & (1u << i)) {
            if (i < NT && (present & (1u << r))) {
                const uint32_t m = last_e[r] - (uint32_t)i;
                dl[i] = ar.rep(last_lc[r] >= lci ? last_lc[r] - lci : last_lc[r] + M - lci);
                cm |= 1u << i;
                if (m == 2u * R) far |= 1u << i;
                else if (m != (uint32_t)R) ok = false;
            }
            present |= 1u << r;
            last_lc[r] = lci;
            last_e[r] = (uint32_t)i;
        }
    }
    if (!ok) return radix_orbit_x<D, R, true, ArPacked>(pol, M, rcpM, lane, nz, lcj, scratch, reps, n_reps);
#pragma unroll
    for (int r = 0; r < R; r++) { topmask |= 1u << last_e[r]; last_lc[r] = ar.rep(last_lc[r]); }

    __syncwarp();
    if (lane <= (uint32_t)D) scratch[lane] = lcj;
    __syncwarp();

    uint32_t acc = 0, qn = 0, nz_exact = 0, odd_exact = 0, w_ok = 0, w_flagged = 0;
    for (uint32_t base = 0; base < n_reps; base += 64u) {
        const uint32_t i0 = base + lane, i1 = i0 + 32u;
        const uint32_t e0 = i0 < n_reps ? __ldg(reps + i0) : 0u, e1 = i1 < n_reps ? __ldg(reps + i1) : 0u;   // weight 0: an invalid slot
        uint32_t w0 = e0 >> 28, w1 = e1 >> 28;
        const uint32_t nn = (e0 & 0xFFFFu) | (e1 << 16);                 // coset indices are below M / R <= 2^13
        // kn[r] = last_e[r] n mod M; pR = R n, p2R = 2R n
        uint32_t kn[R], pR = 0, p2R = 0, cur = 0;
#pragma unroll
        for (int r = 0; r < R; r++) kn[r] = 0;
#pragma unroll
        for (int e = 1; e <= D; e++) {
            cur = e == 1 ? nn : ar.wrap(cur + nn);
            if (e == R) pR = cur;
            if (e == 2 * R) p2R = cur;
            if (topmask & (1u << e)) kn[e % R] = cur;                    // warp-uniform
        }
        uint32_t v[R];
        uint32_t mn = ar.mn_init();
#pragma unroll
        for (int r = 0; r < R; r++) {
            uint32_t w = 0;
            bool chained = false;
#pragma unroll
            for (int i = NT - 1; i >= 0; i--) {
                if (i % R != r) continue;
                if (cm & (1u << i)) {
                    const uint32_t ul = ar.wrap(dl[i] + ((2 * R <= D && (far & (1u << i))) ? p2R : pR));
                    const uint32_t n = chained ? ar.wrap(w + ul) : ul;
                    w = ar.lookup_single(pol, n, mn);
                    chained = true;
                }
            }
            const uint32_t kc = ar.wrap(last_lc[r] + kn[r]);
            v[r] = chained ? ar.wrap(w + kc) : kc;
        }
        uint32_t ps = 0;
        network<R, true>(ar, pol, unit, present, v, ps, mn);
        const bool f0 = w0 != 0u && ar.flagged(mn, 0), f1 = w1 != 0u && ar.flagged(mn, 1);
        if (__any_sync(0xffffffffu, f0 || f1)) {
            uint32_t bal = __ballot_sync(0xffffffffu, f0);
            if (f0) { scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = e0; w_flagged += w0; w0 = 0u; }
            qn += __popc(bal);
            bal = __ballot_sync(0xffffffffu, f1);
            if (f1) { scratch[16 + qn + __popc(bal & ((1u << lane) - 1u))] = e1; w_flagged += w1; w1 = 0u; }
            qn += __popc(bal);
            __syncwarp();
            if (qn >= 32u) {
                exact_queue<D, R, PairS16, true>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact);
                qn = 0;
                __syncwarp();
            }
        }
        acc += (ps & 0xFFFFu) * w0 + (ps >> 16) * w1;  // <= 8 * 4 per pass: a plain 32-bit sum
        w_ok += w0 + w1;
    }
    exact_queue<D, R, PairS16, true>(pol, M, nz, scratch, qn, lane, nz_exact, odd_exact);
    __syncwarp();
    const uint32_t n_nz = w_ok * R + nz_exact;          // every value of an unflagged coset is nonzero
    // nz_exact / odd_exact are spread over the lanes by point, w_flagged by coset: only the warp sums are meaningful, and
    // n_zero = sum(w_flagged) R - sum(nz_exact) may be "negative" in one lane (mod 2^32 the warp sum is right)
    return make_uint2(n_nz - (acc + odd_exact), w_flagged * R - nz_exact);
}

}  // namespace hec_radix
