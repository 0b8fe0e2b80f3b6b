// hec_count: Algorithm 1 lines 6-14 for a batch of curves, in Zech-logarithm
// representation, one warp per curve with x strided across lanes.
//
// Horner in "relative" form.  Write f = sum_j c_{e_j} x^{e_j} over its nonzero terms e_1 = d > e_2 > ..,
// A_1 = c_{e_1}, A_j = A_{j-1} x^{m_j} + c_{e_j}, m_j = e_{j-1} - e_j.  With W_j = log(1 + A_{j-1} x^{m_j} / c_{e_j})
// the addition law (reading G5) alpha^i + alpha^j = alpha^{i + Z(j - i)} gives
//     W_j = Z[ W_{j-1} + m_j log x + (log c_{e_{j-1}} - log c_{e_j}) ]          (indices mod M = q^k - 1)
// so one Horner step is ONE table lookup plus one add: the multiplication by x and the
// coefficient are folded into the index.  The table is tabulated over an extended index range (the idea of
// PAPER.md:272, taken further) so that neither the modular reduction (the paper's exp_red_table,
// PAPER.md:252, 263) nor the zero tests cost an instruction: see hec_device.cuh.
//
// This header holds the count kernels and their launchers; it is compiled once per genus (hec_count_g<G>.cu, so that the
// template instantiations build in parallel) and included by hec_count.cu for the host-side plan and state types.
#pragma once

#include <algorithm>
#include <array>
#include <map>
#include <memory>
#include <mutex>
#include <tuple>
#include <type_traits>
#include <vector>

#include "hec_device.cuh"
#include "hec_radix.cuh"

#ifndef HEC_THREADS
#define HEC_THREADS 1024
#endif
constexpr int kThreads = HEC_THREADS;  // one CTA per SM, 32 warps, one curve per warp
constexpr int kWarps = kThreads / 32;
constexpr uint32_t kDirectMaxM = 64;   // fields with at most this many nonzero elements skip the coset split (hec_radix.cuh: direct_all_x)

// --------------------------------------------------------------------------------------------
// host side: per-(q, g) device plan and the library state (one per process and device, hec.h)
// --------------------------------------------------------------------------------------------
struct LaunchPlan {
    uint32_t k_lo = 1, k_hi = 1;
    int top_mode = HEC_TAB_EXT16;
    const uint4 *blob = nullptr;      // device image of this launch's shared-memory tables
    uint32_t blob_bytes = 0;          // multiple of 16
    uint32_t smem_bytes = 16;         // dynamic shared memory of the launch (blob + radix scratch)
};

struct DevicePlan {
    uint32_t q = 0, g = 0, p = 0, r = 0;
    bool radix = false;               // tables of the radix-R evaluation (hec_radix.cuh) or of the Horner kernel
    int top_mode = HEC_TAB_EXT16;     // table mode of the largest field
    int U = 4;
    void *d_blob = nullptr;           // all device tables in one allocation
    HecFieldDev f[HEC_MAX_GENUS];
    std::vector<LaunchPlan> launches;
    // squarefree
    const uint32_t *sq_zech = nullptr, *sq_emb = nullptr, *sq_antilog = nullptr;
    uint32_t shift_R = 0;             // hec_shift_kernel's target radix (0: no pre-pass for this plan)
    bool shift_dense = false;         // the pre-pass asks for every coefficient up to the degree to be nonzero
    const unsigned long long *d_part_codes = nullptr;   // lambda: packed partitions of 2g+2 in index order
    uint32_t n_parts = 0;
    unsigned long long *d_err = nullptr;
    ~DevicePlan() {
        if (d_blob) cudaFree(d_blob);
        if (d_err) cudaFree(d_err);
    }
};

struct LibState {
    std::recursive_mutex mu;   // recursive: hec_count -> field cache -> hec_build_field_device -> hec_ensure_device
    cudaStream_t stream = nullptr;
    int regime = HEC_REGIME_AUTO;
    int eval = HEC_EVAL_AUTO;
    std::map<std::tuple<uint32_t, uint32_t, int, int>, std::unique_ptr<DevicePlan>> plans;
    hec_count_stats stats{};
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    // host-buffer pipeline of hec_count (hec_count.cu: count_impl): copy streams and per-chunk events
    cudaStream_t copy_in = nullptr, copy_out = nullptr;
    cudaEvent_t ev_chunk[16] = {};
    // staging buffers for host-pointer calls
    void *d_stage = nullptr;
    size_t stage_bytes = 0;
    // rows after the shift pre-pass (hec_shift_kernel)
    void *d_shift = nullptr;
    size_t shift_bytes = 0;
    bool shift_enabled = true;
    bool fast_enabled = true;  // fast tables of the PAIR16 fields (radix_fast_x); part of the plan key
    int sm_count = 0, smem_optin = 0;
    int device = -1;           // the CUDA device the state lives on: the one current at the first call
    bool device_ready = false;
};

// One entry per genus, each in its own translation unit (hec_count_g<G>.cu): all count launches of one plan.
int hec_launch_count_g1(LibState &S, const DevicePlan &plan, HecCountParams P);
int hec_launch_count_g2(LibState &S, const DevicePlan &plan, HecCountParams P);
int hec_launch_count_g3(LibState &S, const DevicePlan &plan, HecCountParams P);
int hec_launch_count_g4(LibState &S, const DevicePlan &plan, HecCountParams P);
int hec_launch_count_g5(LibState &S, const DevicePlan &plan, HecCountParams P);

#ifdef HEC_COUNT_GENUS   // the kernels are only compiled in the per-genus translation units
namespace {


__device__ __forceinline__ uint32_t mod_once(uint32_t x, uint32_t M, uint32_t rcp) {
    // x mod M for any 32-bit x: the quotient estimate is at most one too small
    uint32_t r = x - __umulhi(x, rcp) * M;
    return r >= M ? r - M : r;
}

// ---------------------------------------------------------------------------------------------------------
// Table policies.  A policy turns the chain state v and the per-lane offset u (= uniform part + lane term,
// both in units of SC) into the next state with ONE pass through the Zech table; DESIGN.md "Table layouts".
//
// Extended tables (EXT16 in shared memory, GLOBAL32 in global memory): the state is the stored table value,
// a log W in [0, M) or Z0 = M + LP ("the element is zero"), LP = M + PADL.  The table is tabulated over
// idx = v + u, u in [0, LP):  idx in [0, M + LP) -> Zech of idx mod M (Z0 where 1 + alpha^idx = 0);
// idx in [Z0, Z0 + LP) -> 0 (the accumulator was zero: acc x^m + c = c, W = log 1 = 0).  So v + u never
// needs a reduction modulo M and the zero state is absorbed by the table itself.
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) {
    uint16_t r;
    asm("ld.shared.u16 %0, [%1];" : "=h"(r) : "r"(addr));
    return r;
}

// EXT16: 16-bit entries in shared memory.  Offsets are in bytes (SC = 2) and carry the table's shared-memory
// address, so a chain step is one shift-add and one LDS.
struct ExtTableS16 {
    static constexpr uint32_t SC = 2;
    uint32_t tb;          // shared-memory byte address of entry 0
    uint32_t M, Z0;
    __device__ __forceinline__ uint32_t init() const { return 0u; }                        // W_1 = log 1 = 0
    __device__ __forceinline__ uint32_t ub_init(uint32_t delta) const { return tb + 2u * delta; }
    __device__ __forceinline__ uint32_t ub_next(uint32_t ub, uint32_t inc) const {         // inc = 2 * (increment mod M)
        const uint32_t nx = ub + inc;
        return nx >= tb + 2u * M ? nx - 2u * M : nx;
    }
    __device__ __forceinline__ uint32_t step(uint32_t v, uint32_t u) const { return lds_u16(2u * v + u); }
    __device__ __forceinline__ uint32_t ld(uint32_t idx) const { return lds_u16(2u * idx + tb); }
    __device__ __forceinline__ bool zero(uint32_t v) const { return v >= M; }
    __device__ __forceinline__ uint32_t odd(uint32_t v) const { return v & 1u; }
};

// GLOBAL32: 32-bit entries in global memory, read through L1 (the L2-resident regime).
struct ExtTableG32 {
    static constexpr uint32_t SC = 1;
    const uint32_t *t;
    uint32_t M, Z0;
    __device__ __forceinline__ uint32_t init() const { return 0u; }
    __device__ __forceinline__ uint32_t ub_init(uint32_t delta) const { return delta; }    // delta in [0, M)
    __device__ __forceinline__ uint32_t ub_next(uint32_t ub, uint32_t inc) const {
        const uint32_t nx = ub + inc;
        return nx >= M ? nx - M : nx;
    }
    __device__ __forceinline__ uint32_t ld(uint32_t idx) const { return __ldg(t + idx); }
    __device__ __forceinline__ uint32_t step(uint32_t v, uint32_t u) const { return ld(v + u); }
    __device__ __forceinline__ bool zero(uint32_t v) const { return v >= M; }
    __device__ __forceinline__ uint32_t odd(uint32_t v) const { return v & 1u; }
};

// Half tables in shared memory, for fields whose extended table does not fit.  With h = M/2 and
// Z(-n) = Z(n) - n (mod M) only Z(0..h) is stored.  All quantities are byte offsets (units of SC):
//   x = v + u  is congruent to  n + h  with n the Zech argument;  v in [-hs, Ms), u in [-hs, hs + pad)
//   y = x mod Ms        three candidates x + Ms, x, x - Ms, unsigned minimum (fused add+min, VIADDMNMX)
//   b = min(y, Ms - y)  = SC (h - |d|), d = y/SC - h the signed residue of n nearest to 0; clamped to lims
//   table[b] = SC (Z(h - b/SC) - h);   v' = table[b] + min(y, hs) = SC (Z(|d|) + min(d, 0)) = SC Z(n)
// Zero handling without a branch: Z(h) (b = 0) is stored as a huge sentinel; a sentinel
// state makes x, y and Ms - y huge, so b clamps to lims, whose entry -hs gives v' = -hs + hs = 0 = log 1.
template <int BYTES>
struct HalfTable {
    static constexpr uint32_t SC = BYTES == 4 ? 4u : 2u;
    const char *lo, *hi;
    uint32_t M, Ms, hs, lims;
    __device__ __forceinline__ uint32_t init() const { return 0u; }
    __device__ __forceinline__ uint32_t ub_init(uint32_t delta) const {                    // (delta + h) mod M in [-h, h)
        const uint32_t h = M >> 1;
        uint32_t e = delta + h;
        e = e >= M ? e - M : e;
        const int32_t r = e >= h ? (int32_t)e - (int32_t)M : (int32_t)e;
        return (uint32_t)(r * (int32_t)SC);
    }
    __device__ __forceinline__ uint32_t ub_next(uint32_t ub, uint32_t inc) const {
        const int32_t nx = (int32_t)ub + (int32_t)inc;
        return (uint32_t)(nx >= (int32_t)hs ? nx - (int32_t)Ms : nx);
    }
    __device__ __forceinline__ uint32_t step(uint32_t v, uint32_t u) const {
        const uint32_t x = v + u;
        const uint32_t y = min(min(x + Ms, x), x - Ms);
        const uint32_t b = min(min(y, Ms - y), lims);
        const uint32_t mn = min(y, hs);
        if constexpr (BYTES == 4) {
            return *reinterpret_cast<const uint32_t *>(lo + b) + mn;
        } else {
            const uint32_t l = *reinterpret_cast<const uint16_t *>(lo + b);
            const int32_t h8 = *reinterpret_cast<const int8_t *>(hi + (b >> 1));
            return l * 2u + mn + (uint32_t)(h8 * 131072);
        }
    }
    __device__ __forceinline__ bool zero(uint32_t v) const { return (int32_t)v < -(1 << 22); }
    __device__ __forceinline__ uint32_t odd(uint32_t v) const { return (v / SC) & 1u; }    // M is even
};

// All x in F_{q^k}^x for one curve: returns this lane's share of
//   n_zero = #{x != 0 : f(x) = 0},  n_odd = #{x != 0 : f(x) != 0 and W_T odd}         (reading G3)
// Per-term uniform state: ub[i] = (delta_i + m_i * base) mod M, advanced by inc[i] per batch of 32*U points.
template <int D, int U, typename Pol>
__device__ __forceinline__ void horner_all_x(const Pol pol, const uint32_t M, const uint32_t lane, const uint32_t lane_cap,
                                             const uint32_t nzmask, const uint32_t (&delta)[D], const uint32_t (&incr)[D],
                                             const uint32_t (&gap)[D], uint32_t &n_odd, uint32_t &n_zero) {
    uint32_t lterm[U], ub[D], inc[D];
#pragma unroll
    for (int u = 0; u < U; u++) {
        const uint32_t l = lane + 32u * u;
        lterm[u] = (l < lane_cap ? l : 0u) * Pol::SC;
    }
#pragma unroll
    for (int i = 0; i < D; i++) {
        ub[i] = pol.ub_init(delta[i]);
        inc[i] = incr[i] * Pol::SC;
    }
    n_odd = 0;
    n_zero = 0;
    for (uint32_t base = 0; base < M; base += 32u * U) {
        uint32_t v[U];
#pragma unroll
        for (int u = 0; u < U; u++) v[u] = pol.init();
#pragma unroll
        for (int i = D - 1; i >= 0; i--) {
            if (nzmask & (1u << i)) {                             // warp-uniform: c_i != 0
                const uint32_t ubi = ub[i];
                const uint32_t m = gap[i];
#pragma unroll
                for (int u = 0; u < U; u++) v[u] = pol.step(v[u], ubi + m * lterm[u]);
                ub[i] = pol.ub_next(ubi, inc[i]);
            }
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            const bool valid = base + lane + 32u * u < M;
            const bool z = pol.zero(v[u]);
            n_odd += (valid && !z) ? pol.odd(v[u]) : 0u;
            n_zero += (valid && z) ? 1u : 0u;
        }
    }
}

// One launch computes N_k for k_lo <= k <= k_hi with one Horner chain per x (Algorithm 1 line 8):
// the paper's evaluation scheme (HEC_EVAL_HORNER).  Fields below k_hi use EXT16 tables; field k_hi uses TOP.
template <int G, int U, int TOP>
__global__ void __launch_bounds__(kThreads, 1) hec_count_kernel(const __grid_constant__ HecCountParams P) {
    constexpr int D = 2 * G + 2;          // largest degree; coefficient slots 0..D
    constexpr int NC = D + 1;
    extern __shared__ uint4 smem_blob[];

    for (uint32_t i = threadIdx.x; i < P.blob_bytes / 16; i += blockDim.x) smem_blob[i] = P.blob[i];
    __syncthreads();

    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warp = threadIdx.x >> 5;
    const unsigned long long stride = (unsigned long long)gridDim.x * kWarps;
    const char *smem = reinterpret_cast<const char *>(smem_blob);
    const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem_blob);

    for (unsigned long long curve = (unsigned long long)blockIdx.x * kWarps + warp; curve < P.n; curve += stride) {
        // ---- a2: coefficient load (lane j holds c_j) and boundary checks (readings G13, hec.h)
        uint32_t cj = 0;
        if (lane < NC) cj = P.coeffs[curve * NC + lane];
        const bool bad_range = __any_sync(0xffffffffu, cj >= P.q);
        const uint32_t nz = __ballot_sync(0xffffffffu, cj != 0);          // bit j: c_j != 0
        const bool mine = lane + 1 >= P.k_lo && lane + 1 <= P.k_hi;
        if (bad_range || (nz >> (D - 1)) == 0) {
            if (lane == 0) atomicMin(&P.err[bad_range ? 0 : 1], curve + P.row0);
            if (mine) { P.out[curve * G + lane] = 0; if (P.out_r0) P.out_r0[curve * G + lane] = 0; }
            continue;
        }

        uint32_t my_count = 0, my_r0 = 0;   // lane k-1 keeps N_k and r0_k
#pragma unroll
        for (uint32_t k = 1; k <= (uint32_t)G; k++) {
            if (k < P.k_lo || k > P.k_hi) continue;
            const HecFieldDev &F = P.f[k - 1];
            const uint32_t M = F.M;
            // embed: log of c_j in F_{q^k} (reading G6)
            const uint32_t lcj = (lane < NC && cj != 0) ? __ldg(F.emb + cj) : HEC_LOG_ZERO;
            // ---- a3 + a4: f at every x != 0, classify, per-lane partial sums of
            //   n_zero = #{x != 0 : f(x) = 0},  n_sq = #{x != 0 : f(x) a nonzero square}      (reading G3)
            uint32_t n_zero, n_sq;
            {
                uint32_t delta[D], incr[D], gap[D];
                uint32_t nzmask = 0, prev_lc = 0, prev_e = 0;
                bool started = false;
#pragma unroll
                for (int i = D; i >= 0; i--) {
                    const uint32_t lci = __shfl_sync(0xffffffffu, lcj, i);
                    if (i < D) { delta[i] = 0; incr[i] = 0; gap[i] = 0; }
                    if (nz & (1u << i)) {
                        if (started && i < D) {
                            const uint32_t m = prev_e - (uint32_t)i;
                            gap[i] = m;
                            delta[i] = prev_lc >= lci ? prev_lc - lci : prev_lc + M - lci;
                            incr[i] = mod_once(m * (32u * U), M, F.rcpM);
                            nzmask |= 1u << i;
                        }
                        started = true;
                        prev_lc = lci;
                        prev_e = (uint32_t)i;
                    }
                }
                uint32_t n_odd;
                if (TOP == HEC_TAB_EXT16 || k < P.k_hi) {
                    const ExtTableS16 pol{smem_base + F.smem_off, M, F.z0};
                    horner_all_x<D, U>(pol, M, lane, F.lane_cap, nzmask, delta, incr, gap, n_odd, n_zero);
                } else if constexpr (TOP == HEC_TAB_GLOBAL32) {
                    const ExtTableG32 pol{F.gtab, M, F.z0};
                    horner_all_x<D, U>(pol, M, lane, F.lane_cap, nzmask, delta, incr, gap, n_odd, n_zero);
                } else if constexpr (TOP == HEC_TAB_HALF32) {
                    const HalfTable<4> pol{smem + F.smem_off, nullptr, M, 4u * M, 2u * M, 4u * ((M >> 1) + 1u)};
                    horner_all_x<D, U>(pol, M, lane, F.lane_cap, nzmask, delta, incr, gap, n_odd, n_zero);
                } else if constexpr (TOP == HEC_TAB_HALF24) {
                    const HalfTable<3> pol{smem + F.smem_off, smem + F.smem_off2, M, 2u * M, M, 2u * ((M >> 1) + 1u)};
                    horner_all_x<D, U>(pol, M, lane, F.lane_cap, nzmask, delta, incr, gap, n_odd, n_zero);
                }
                // f(x) = A_T x^{e_T}; log f = log c_{e_T} + W_T + e_T log x; a nonzero value is a square iff its log
                // is even (reading G4; M is even).  log x = base + lane + 32u has the parity of the lane.
                const uint32_t n_valid = (M + 31u - lane) >> 5;
                const uint32_t flip = (prev_lc ^ (prev_e & lane)) & 1u;
                n_sq = flip ? n_odd : n_valid - n_zero - n_odd;
            }
            const uint32_t r0 = __reduce_add_sync(0xffffffffu, n_zero);
            const uint32_t rsq = __reduce_add_sync(0xffffffffu, n_sq);
            // ---- a5: x = 0 (reading G15) and the points at infinity
            const uint32_t lc0 = __shfl_sync(0xffffffffu, lcj, 0);
            const uint32_t lcD = __shfl_sync(0xffffffffu, lcj, D);
            const uint32_t x0 = (nz & 1u) == 0 ? 1u : ((lc0 & 1u) ? 0u : 2u);
            const uint32_t inf = ((nz >> D) & 1u) == 0 ? 1u : ((lcD & 1u) ? 0u : 2u);
            const uint32_t Nk = r0 + 2u * rsq + x0 + inf;
            if (lane + 1 == k) { my_count = Nk; my_r0 = r0 + ((nz & 1u) ? 0u : 1u); }
        }
        if (mine) {
            P.out[curve * G + lane] = my_count;
            if (P.out_r0) P.out_r0[curve * G + lane] = my_r0;
        }
    }
}

// One launch of the radix-R evaluation (hec_radix.cuh; HEC_EVAL_AUTO) for k_lo <= k <= k_hi.  Fields below k_hi
// use PAIR16 tables with the packed 16x2 arithmetic; field k_hi uses TOP.  Same mapping as above: persistent
// CTAs, one warp per curve, the lanes stride the coset index n = log x < M / R.
// Per curve and field: the largest R' <= R (R = the field's radix, R' | R | M) for which every residue class
// mod R' holds a nonzero coefficient runs the straight-line network; the branchy general network is kept only
// for R = 2 (f even or odd in X, or D + 1 < R').  Measured (profiles/r01c_ncu_full_c4_radix.md): compiling the
// general network for R = 4, 8 made the loop body overflow the instruction caches (41 % no_instruction stalls).
// FAST (PAIR16 fields of the batch kernel): a field that carries fast tables runs radix_fast_x when every class mod its full
// radix is non-empty, which the shift pre-pass arranges for all but a few rows.
template <int D, typename Ar, bool ORBIT, bool FAST, typename Pol>
__device__ __forceinline__ void radix_dispatch(const HecFieldDev &F, const Pol pol, const uint32_t smem_base, const uint32_t lane,
                                               const uint32_t nz, const uint32_t lcj, volatile uint32_t *scratch, const uint32_t part,
                                               const uint32_t splits, uint32_t &n_sq, uint32_t &n_zero) {
    using namespace hec_radix;
    const uint32_t R = F.radix, M = F.M, rcpM = F.rcpM;
    if constexpr (std::is_same<Pol, PairS16>::value && std::is_same<Ar, ArPacked>::value) {
        if (M <= kDirectMaxM) {                       // tiny field: every point directly (splits: part 0 takes them all)
            uint2 res = make_uint2(0u, 0u);
            if (part == 0u) res = direct_all_x<D>(pol, M, lane, nz, lcj, scratch);
            n_sq = res.x; n_zero = res.y;
            return;
        }
    }
    if constexpr (FAST) {
        if (F.fast_off) {
            const uint32_t ft = smem_base + F.fast_off;
            if constexpr (D + 1 <= 8) {                   // monomial classes (genus <= 2): R = 8 without chains
                const uint32_t dense = (nz >> D) ? (1u << (D + 1)) - 1u : (1u << D) - 1u;
                if (R == 8 && nz == dense) {
                    const uint2 res = (nz >> D) ? radix_mono8_packed_x<D, D + 1>(pol, ft, M, lane, nz, lcj, scratch)
                                                : radix_mono8_packed_x<D, D>(pol, ft, M, lane, nz, lcj, scratch);
                    n_sq = res.x; n_zero = res.y;
                    return;
                }
            }
            if (R == 8) { if (all_classes_present<D, 8>(nz)) { const uint2 res = radix_fast_x<D, 8>(pol, ft, F.fast_row, M, lane, nz, lcj, scratch); n_sq = res.x; n_zero = res.y; return; } }
            else if (R == 4) { if (all_classes_present<D, 4>(nz)) { const uint2 res = radix_fast_x<D, 4>(pol, ft, F.fast_row, M, lane, nz, lcj, scratch); n_sq = res.x; n_zero = res.y; return; } }
            else if (all_classes_present<D, 2>(nz)) { const uint2 res = radix_fast_x<D, 2>(pol, ft, F.fast_row, M, lane, nz, lcj, scratch); n_sq = res.x; n_zero = res.y; return; }
        }
    }
    uint2 res;
    if constexpr (ORBIT && std::is_same<Pol, PairS16>::value && std::is_same<Ar, ArPacked>::value) {
        if (F.orb_fast) {                                 // every class present at R = 4 or 8: offsets by repeated addition
            if (R >= 8 && all_classes_present<D, 8>(nz)) { res = radix_orbit_fast_x<D, 8>(pol, M, rcpM, lane, nz, lcj, scratch, F.orb[2], F.n_orb[2]); n_sq = res.x; n_zero = res.y; return; }
            if (R >= 4 && all_classes_present<D, 4>(nz)) { res = radix_orbit_fast_x<D, 4>(pol, M, rcpM, lane, nz, lcj, scratch, F.orb[1], F.n_orb[1]); n_sq = res.x; n_zero = res.y; return; }
        }
    }
    if constexpr (ORBIT) {
        if (R >= 8 && all_classes_present<D, 8>(nz)) res = radix_orbit_x<D, 8, true, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, F.orb[2], F.n_orb[2]);
        else if (R >= 4 && all_classes_present<D, 4>(nz)) res = radix_orbit_x<D, 4, true, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, F.orb[1], F.n_orb[1]);
        else if (all_classes_present<D, 2>(nz)) res = radix_orbit_x<D, 2, true, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, F.orb[0], F.n_orb[0]);
        else res = radix_orbit_x<D, 2, false, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, F.orb[0], F.n_orb[0]);
    } else {
        if (R >= 8 && all_classes_present<D, 8>(nz)) res = radix_all_x<D, 8, true, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, part, splits);
        else if (R >= 4 && all_classes_present<D, 4>(nz)) res = radix_all_x<D, 4, true, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, part, splits);
        else if (all_classes_present<D, 2>(nz)) res = radix_all_x<D, 2, true, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, part, splits);
        else res = radix_all_x<D, 2, false, Ar>(pol, M, rcpM, lane, nz, lcj, scratch, part, splits);
    }
    n_sq = res.x;
    n_zero = res.y;
}

// Monomial classes on a half-table top field with a parity table (hec_radix.cuh: radix_mono_x): rows with every coefficient up to
// the degree nonzero, at R = 8 (at most 8 coefficients) or R = 16 (9 .. 16).  Returns false if the row or the field does not qualify.
template <int D, bool SPLIT, bool ORBIT, bool PT, typename Pol>
__device__ __forceinline__ bool mono_dispatch(const HecFieldDev &F, const Pol pol, const uint32_t smem_base, const uint32_t lane,
                                              const uint32_t nz, const uint32_t lcj, volatile uint32_t *scratch, uint32_t &n_sq, uint32_t &n_zero) {
    if constexpr (!SPLIT && !ORBIT && D + 1 <= 16) {
        const uint32_t dense = (nz >> D) ? (1u << (D + 1)) - 1u : (1u << D) - 1u;
        if (!F.mono_r || nz != dense) return false;
        constexpr int R = D + 1 <= 8 ? 8 : 16;
        if (F.mono_r != (uint32_t)R) return false;
        const uint32_t tp = smem_base + F.pt_off;
        const uint2 res = (nz >> D) ? hec_radix::radix_mono_x<D, R, D + 1, PT>(pol, tp, F.M, lane, nz, lcj, scratch)
                                    : hec_radix::radix_mono_x<D, R, D, PT>(pol, tp, F.M, lane, nz, lcj, scratch);
        n_sq = res.x; n_zero = res.y;
        return true;
    } else {
        return false;
    }
}

// SPLIT = false: one warp per curve (batches; P.splits == 1).  SPLIT = true: a separate instantiation for small batches,
// so that the batch kernel carries none of the split bookkeeping (measured: 610 -> 685 ms on config 4 when it did).
// ORBIT (HEC_EVAL_ORBIT, never with SPLIT): one representative per Frobenius orbit of cosets, hec_radix::radix_orbit_x.
template <int G, int TOP, bool SPLIT, bool ORBIT>
__global__ void __launch_bounds__(kThreads, 1) hec_count_radix_kernel(const __grid_constant__ HecCountParams P) {
    constexpr int D = 2 * G + 2;
    constexpr int NC = D + 1;
    extern __shared__ uint4 smem_blob[];

    for (uint32_t i = threadIdx.x; i < P.blob_bytes / 16; i += blockDim.x) smem_blob[i] = P.blob[i];
    __syncthreads();

    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warp = threadIdx.x >> 5;
    const unsigned long long stride = (unsigned long long)gridDim.x * kWarps;
    const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem_blob);
    volatile uint32_t *scratch = reinterpret_cast<volatile uint32_t *>(reinterpret_cast<char *>(smem_blob) + P.scratch_off) +
                                 warp * hec_radix::kScratchWords;

    // one work item = (curve, part): part `part` of P.splits slices of the coset range of every field
    const uint32_t splits = SPLIT ? P.splits : 1u;
    const unsigned long long items = P.n * splits;
    for (unsigned long long item = (unsigned long long)blockIdx.x * kWarps + warp; item < items; item += stride) {
        const unsigned long long curve = SPLIT ? item / splits : item;
        const uint32_t part = SPLIT ? (uint32_t)(item - curve * splits) : 0u;
        // ---- a2: coefficient load (lane j holds c_j) and boundary checks (readings G13, hec.h)
        uint32_t cj = 0;
        if (lane < NC) cj = P.coeffs[curve * NC + lane];
        const bool bad_range = __any_sync(0xffffffffu, cj >= P.q);
        const uint32_t nz = __ballot_sync(0xffffffffu, cj != 0);
        const bool mine = lane + 1 >= P.k_lo && lane + 1 <= P.k_hi;
        if (bad_range || (nz >> (D - 1)) == 0) {
            if (lane == 0) atomicMin(&P.err[bad_range ? 0 : 1], curve + P.row0);
            if (mine && !SPLIT) { P.out[curve * G + lane] = 0; if (P.out_r0) P.out_r0[curve * G + lane] = 0; }
            continue;
        }
        uint32_t my_count = 0, my_r0 = 0;   // lane k-1 keeps N_k and r0_k
#pragma unroll 1
        for (uint32_t k = P.k_lo; k <= P.k_hi; k++) {
            const HecFieldDev &F = P.f[k - 1];
            const uint32_t M = F.M;
            const uint32_t lcj = (lane < NC && cj != 0) ? __ldg(F.emb + cj) : 0u;     // reading G6
            // ---- a3 + a4 (reading G3)
            uint32_t n_zero, n_sq;
            if (TOP == HEC_TAB_PAIR16 || k < P.k_hi) {
                const hec_radix::PairS16 pol{smem_base + F.smem_off};
                radix_dispatch<D, hec_radix::ArPacked, ORBIT, !SPLIT && !ORBIT>(F, pol, smem_base, lane, nz, lcj, scratch, part, splits, n_sq, n_zero);
            } else if constexpr (TOP == HEC_TAB_RHALF32) {
                const hec_radix::HalfS32 pol{smem_base + F.smem_off, smem_base + F.smem_off + 4u * (M >> 1)};
                if (!mono_dispatch<D, SPLIT, ORBIT, true>(F, pol, smem_base, lane, nz, lcj, scratch, n_sq, n_zero)) {
                    if (F.pt_off) {                                       // parity table for the classifying last stage
                        const hec_radix::HalfS32T<true> polp{pol.tb, pol.tbh, smem_base + F.pt_off};
                        radix_dispatch<D, hec_radix::ArScalar, ORBIT, false>(F, polp, smem_base, lane, nz, lcj, scratch, part, splits, n_sq, n_zero);
                    } else {
                        radix_dispatch<D, hec_radix::ArScalar, ORBIT, false>(F, pol, smem_base, lane, nz, lcj, scratch, part, splits, n_sq, n_zero);
                    }
                }
            } else if constexpr (TOP == HEC_TAB_RHALF17) {
                const hec_radix::HalfS17 pol{smem_base + F.smem_off, smem_base + F.smem_off + 2u * (M >> 1), smem_base + F.smem_off2};
                if (!mono_dispatch<D, SPLIT, ORBIT, true>(F, pol, smem_base, lane, nz, lcj, scratch, n_sq, n_zero)) {
                    if (F.pt_off) {
                        const hec_radix::HalfS17T<true> polp{pol.tb, pol.tbh, pol.bb, smem_base + F.pt_off};
                        radix_dispatch<D, hec_radix::ArScalar, ORBIT, false>(F, polp, smem_base, lane, nz, lcj, scratch, part, splits, n_sq, n_zero);
                    } else {
                        radix_dispatch<D, hec_radix::ArScalar, ORBIT, false>(F, pol, smem_base, lane, nz, lcj, scratch, part, splits, n_sq, n_zero);
                    }
                }
            } else if constexpr (TOP == HEC_TAB_SPAIR16) {
                const hec_radix::PairS16 pol{smem_base + F.smem_off};
                if (!mono_dispatch<D, SPLIT, ORBIT, false>(F, pol, smem_base, lane, nz, lcj, scratch, n_sq, n_zero))
                    radix_dispatch<D, hec_radix::ArScalar, ORBIT, false>(F, pol, smem_base, lane, nz, lcj, scratch, part, splits, n_sq, n_zero);
            } else if constexpr (TOP == HEC_TAB_GPAIR64) {
                const hec_radix::PairG64 pol{reinterpret_cast<const uint2 *>(F.gtab)};
                radix_dispatch<D, hec_radix::ArScalar, ORBIT, false>(F, pol, smem_base, lane, nz, lcj, scratch, part, splits, n_sq, n_zero);
            }
            const uint32_t r0 = __reduce_add_sync(0xffffffffu, n_zero);
            const uint32_t rsq = __reduce_add_sync(0xffffffffu, n_sq);
            // ---- a5: x = 0 (reading G15) and the points at infinity
            const uint32_t lc0 = __shfl_sync(0xffffffffu, lcj, 0);
            const uint32_t lcD = __shfl_sync(0xffffffffu, lcj, D);
            const uint32_t x0 = (nz & 1u) == 0 ? 1u : ((lc0 & 1u) ? 0u : 2u);
            const uint32_t inf = ((nz >> D) & 1u) == 0 ? 1u : ((lcD & 1u) ? 0u : 2u);
            const uint32_t Nk = r0 + 2u * rsq + (part == 0u ? x0 + inf : 0u);
            if (lane + 1 == k) { my_count = Nk; my_r0 = r0 + ((part == 0u && !(nz & 1u)) ? 1u : 0u); }
        }
        if (mine) {
            if (!SPLIT) {
                P.out[curve * G + lane] = my_count;
                if (P.out_r0) P.out_r0[curve * G + lane] = my_r0;
            } else {
                if (my_count) atomicAdd(&P.out[curve * G + lane], my_count);
                if (P.out_r0 && my_r0) atomicAdd(&P.out_r0[curve * G + lane], my_r0);
            }
        }
    }
}

template <typename Kern>
int launch_kernel(LibState &S, Kern kern, const LaunchPlan &L, const HecCountParams &P, uint32_t chains) {
    HEC_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem_bytes));
    uint32_t grid = (uint32_t)std::min<unsigned long long>((P.n * P.splits + kWarps - 1) / kWarps, (unsigned long long)S.sm_count);
    if (grid == 0) grid = 1;
    kern<<<grid, kThreads, L.smem_bytes, S.stream>>>(P);
    hec_launch_counter::value++;
    S.stats.grid = grid;
    S.stats.block = kThreads;
    S.stats.chains_per_lane = chains;
    S.stats.smem_bytes = std::max(S.stats.smem_bytes, L.smem_bytes);
    S.stats.launches++;
    HEC_CUDA_OK(cudaGetLastError());
    return HEC_OK;
}

template <int G, int TOP>
int launch_radix(LibState &S, const LaunchPlan &L, const HecCountParams &P, uint32_t chains) {
    if (P.splits > 1u) return launch_kernel(S, hec_count_radix_kernel<G, TOP, true, false>, L, P, chains);
    if (P.f[L.k_hi - 1].orb[0]) return launch_kernel(S, hec_count_radix_kernel<G, TOP, false, true>, L, P, chains);
    return launch_kernel(S, hec_count_radix_kernel<G, TOP, false, false>, L, P, chains);
}

template <int G, int U>
int launch_count(LibState &S, const DevicePlan &plan, HecCountParams P) {
    for (const LaunchPlan &L : plan.launches) {
        P.blob = L.blob; P.blob_bytes = L.blob_bytes; P.k_lo = L.k_lo; P.k_hi = L.k_hi;
        P.scratch_off = std::max<uint32_t>(L.blob_bytes, 16u);
        int rc;
        switch (L.top_mode) {
            case HEC_TAB_GLOBAL32: rc = launch_kernel(S, hec_count_kernel<G, U, HEC_TAB_GLOBAL32>, L, P, U); break;
            case HEC_TAB_HALF32: rc = launch_kernel(S, hec_count_kernel<G, U, HEC_TAB_HALF32>, L, P, U); break;
            case HEC_TAB_HALF24: rc = launch_kernel(S, hec_count_kernel<G, U, HEC_TAB_HALF24>, L, P, U); break;
            case HEC_TAB_EXT16: rc = launch_kernel(S, hec_count_kernel<G, U, HEC_TAB_EXT16>, L, P, U); break;
            case HEC_TAB_PAIR16: rc = launch_radix<G, HEC_TAB_PAIR16>(S, L, P, 2); break;
            case HEC_TAB_SPAIR16: rc = launch_radix<G, HEC_TAB_SPAIR16>(S, L, P, 1); break;
            case HEC_TAB_RHALF32: rc = launch_radix<G, HEC_TAB_RHALF32>(S, L, P, 1); break;
            case HEC_TAB_RHALF17: rc = launch_radix<G, HEC_TAB_RHALF17>(S, L, P, 1); break;
            default: rc = launch_radix<G, HEC_TAB_GPAIR64>(S, L, P, 1); break;
        }
        if (rc) return rc;
        if (plan.radix)
            for (uint32_t k = L.k_lo; k <= L.k_hi; k++) {
                S.stats.radix_fields |= plan.f[k - 1].radix << (4u * (k - 1));
                if ((plan.f[k - 1].fast_off || plan.f[k - 1].pt_off || plan.f[k - 1].mono_r) && P.splits == 1u && !plan.f[k - 1].orb[0]) S.stats.fast_fields |= 1u << (k - 1);
            }
    }
    return HEC_OK;
}

}  // namespace
#endif  // HEC_COUNT_GENUS
