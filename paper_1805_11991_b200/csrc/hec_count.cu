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
#include <algorithm>
#include <map>
#include <memory>
#include <mutex>
#include <vector>

#include "hec_device.cuh"

uint64_t hec_launch_counter::value = 0;

namespace {

constexpr int kThreads = 1024;
constexpr int kWarps = kThreads / 32;

struct SmemTable16 {
    const uint16_t *t;
    __device__ __forceinline__ uint32_t operator()(uint32_t idx) const { return t[idx]; }
};
struct GlobalTable32 {
    const uint32_t *t;
    __device__ __forceinline__ uint32_t operator()(uint32_t idx) const { return __ldg(t + idx); }
};

__device__ __forceinline__ uint32_t mod_once(uint32_t x, uint32_t M, uint32_t rcp) {
    // x mod M for any 32-bit x: the quotient estimate is at most one too small
    uint32_t r = x - __umulhi(x, rcp) * M;
    return r >= M ? r - M : r;
}

// All x in F_{q^k}^x for one curve: returns in (r0, rsq) this lane's share of
//   r0 = #{x != 0 : f(x) = 0},  rsq = #{x != 0 : f(x) a nonzero square}        (reading G3)
// Per-term uniform state: ub[i] = (delta_i + m_i * base) mod M, advanced by inc[i] per batch of 32*U points.
template <int D, int U, typename Table>
__device__ __forceinline__ void horner_all_x(const Table tab, const uint32_t M, const uint32_t OFF,
                                             const uint32_t lane, const uint32_t lane_cap,
                                             uint32_t nzmask, uint32_t (&ub)[D], const uint32_t (&inc)[D],
                                             const uint32_t (&gap)[D], uint32_t &n_odd, uint32_t &n_zero) {
    uint32_t lterm[U];
#pragma unroll
    for (int u = 0; u < U; u++) {
        uint32_t l = lane + 32u * u;
        lterm[u] = l < lane_cap ? l : 0u;
    }
    n_odd = 0;
    n_zero = 0;
    for (uint32_t base = 0; base < M; base += 32u * U) {
        uint32_t v[U];
#pragma unroll
        for (int u = 0; u < U; u++) v[u] = OFF;                  // W_1 = log 1 = 0
#pragma unroll
        for (int i = D - 1; i >= 0; i--) {
            if (nzmask & (1u << i)) {                             // warp-uniform: c_i != 0
                const uint32_t ubi = ub[i];
                const uint32_t m = gap[i];
#pragma unroll
                for (int u = 0; u < U; u++) v[u] = tab(v[u] + ubi + m * lterm[u]);
                uint32_t nx = ubi + inc[i];
                ub[i] = nx >= M ? nx - M : nx;
            }
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            const bool valid = base + lane + 32u * u < M;
            n_odd += valid ? (v[u] & 1u) : 0u;
            n_zero += (valid && v[u] == 0u) ? 1u : 0u;
        }
    }
}

template <int G, int U>
__global__ void __launch_bounds__(kThreads, 1) hec_count_kernel(const __grid_constant__ HecCountParams P) {
    constexpr int D = 2 * G + 2;          // largest degree; coefficient slots 0..D
    constexpr int NC = D + 1;
    extern __shared__ uint4 smem_blob[];

    for (uint32_t i = threadIdx.x; i < P.blob_bytes / 16; i += blockDim.x) smem_blob[i] = P.blob[i];
    __syncthreads();

    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warp = threadIdx.x >> 5;
    const unsigned long long stride = (unsigned long long)gridDim.x * kWarps;

    for (unsigned long long curve = (unsigned long long)blockIdx.x * kWarps + warp; curve < P.n; curve += stride) {
        // ---- a2: coefficient load (lane j holds c_j) and boundary checks (readings G13, hec.h)
        uint32_t cj = 0;
        if (lane < NC) cj = P.coeffs[curve * NC + lane];
        const bool bad_range = __any_sync(0xffffffffu, cj >= P.q);
        const uint32_t top2 = __shfl_sync(0xffffffffu, cj, D) | __shfl_sync(0xffffffffu, cj, D - 1);
        if (bad_range || top2 == 0) {
            if (lane == 0) atomicMin(&P.err[bad_range ? 0 : 1], curve);
            if (lane < G) P.out[curve * G + lane] = 0;
            continue;
        }
        uint32_t c[NC];
#pragma unroll
        for (int i = 0; i < NC; i++) c[i] = __shfl_sync(0xffffffffu, cj, i);

        uint32_t my_count = 0;   // lane k-1 keeps N_k
#pragma unroll 1
        for (int k = 1; k <= G; k++) {
            const HecFieldDev &F = P.f[k - 1];
            const uint32_t M = F.M, OFF = F.off;
            // embed: log of c_j in F_{q^k} (reading G6)
            const uint32_t lcj = (lane < NC && cj != 0) ? __ldg(F.emb + cj) : HEC_LOG_ZERO;
            uint32_t ub[D], inc[D], gap[D];
            uint32_t nzmask = 0, prev_lc = 0, prev_e = 0;
            bool started = false;
#pragma unroll
            for (int i = D; i >= 0; i--) {
                const uint32_t lci = __shfl_sync(0xffffffffu, lcj, i);
                if (i < D) { ub[i] = 0; inc[i] = 0; gap[i] = 0; }
                if (c[i] != 0) {
                    if (started && i < D) {
                        const uint32_t m = prev_e - (uint32_t)i;
                        gap[i] = m;
                        ub[i] = prev_lc >= lci ? prev_lc - lci : prev_lc + M - lci;     // delta_i
                        inc[i] = mod_once(m * (32u * U), M, F.rcpM);
                        nzmask |= 1u << i;
                    }
                    started = true;
                    prev_lc = lci;
                    prev_e = (uint32_t)i;
                }
            }
            // ---- a3 + a4: Horner at every x != 0, classify, per-lane partial sums
            uint32_t n_odd, n_zero;
            if (F.in_smem) {
                SmemTable16 tab{reinterpret_cast<const uint16_t *>(reinterpret_cast<const char *>(smem_blob) + F.smem_off)};
                horner_all_x<D, U>(tab, M, OFF, lane, F.lane_cap, nzmask, ub, inc, gap, n_odd, n_zero);
            } else {
                GlobalTable32 tab{F.gtab};
                horner_all_x<D, U>(tab, M, OFF, lane, F.lane_cap, nzmask, ub, inc, gap, n_odd, n_zero);
            }
            // f(x) = A_T x^{e_T}; log f = log c_{e_T} + W_T + e_T log x; a nonzero value is a square iff its log
            // is even (reading G4; M and OFF are even).  log x = base + lane + 32u has the parity of the lane.
            const uint32_t n_valid = (M + 31u - lane) >> 5;
            const uint32_t flip = (prev_lc ^ (prev_e & lane)) & 1u;
            const uint32_t rsq_lane = flip ? n_odd : n_valid - n_zero - n_odd;
            const uint32_t r0 = __reduce_add_sync(0xffffffffu, n_zero);
            const uint32_t rsq = __reduce_add_sync(0xffffffffu, rsq_lane);
            // ---- a5: x = 0 (reading G15) and the points at infinity
            const uint32_t lc0 = __shfl_sync(0xffffffffu, lcj, 0);
            const uint32_t lcD = __shfl_sync(0xffffffffu, lcj, D);
            const uint32_t x0 = c[0] == 0 ? 1u : ((lc0 & 1u) ? 0u : 2u);
            const uint32_t inf = c[D] == 0 ? 1u : ((lcD & 1u) ? 0u : 2u);
            const uint32_t Nk = r0 + 2u * rsq + x0 + inf;
            if ((int)lane == k - 1) my_count = Nk;
        }
        if (lane < G) P.out[curve * G + lane] = my_count;
    }
}

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
    if (!ok || da < (int)P.ncoef - 2) { P.out[i] = 0; return; }     // reported by the count kernel
    // Euclid: gcd(f, 0) = f (reading G14)
    while (db >= 0) {
        // a <- a mod b
        const uint32_t binv = K.inv(b[db]);
        while (da >= db) {
            const uint32_t fac = K.neg(K.mul(a[da], binv));
            const int s = da - db;
            for (int t = 0; t < db; t++) a[s + t] = K.add(a[s + t], K.mul(fac, b[t]));
            a[da] = ZERO;
            while (da >= 0 && a[da] == ZERO) da--;
        }
        // swap (a, b)
        for (int t = 0; t < (int)kSqMaxCoef; t++) { const uint32_t x = a[t]; a[t] = b[t]; b[t] = x; }
        const int td = da; da = db; db = td;
    }
    P.out[i] = da == 0 ? 1 : 0;
}

// --------------------------------------------------------------------------------------------
// host side: per-(q, g) device plan
// --------------------------------------------------------------------------------------------
struct DevicePlan {
    uint32_t q = 0, g = 0, p = 0, r = 0;
    int regime = 0;               // regime actually used for the largest field
    int U = 4;
    uint32_t smem_bytes = 0;
    void *d_blob = nullptr;       // all device tables in one allocation
    HecFieldDev f[HEC_MAX_GENUS];
    const uint4 *blob = nullptr;
    uint32_t blob_bytes = 0;
    // squarefree
    const uint32_t *sq_zech = nullptr, *sq_emb = nullptr;
    unsigned long long *d_err = nullptr;
    ~DevicePlan() {
        if (d_blob) cudaFree(d_blob);
        if (d_err) cudaFree(d_err);
    }
};

struct LibState {
    std::mutex mu;
    cudaStream_t stream = nullptr;
    int regime = HEC_REGIME_AUTO;
    std::map<std::tuple<uint32_t, uint32_t, int>, std::unique_ptr<DevicePlan>> plans;
    hec_count_stats stats{};
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    // staging buffers for host-pointer calls
    void *d_stage = nullptr;
    size_t stage_bytes = 0;
    int sm_count = 0, smem_optin = 0;
    bool device_ready = false;
};
LibState g_state;

int ensure_device(LibState &S) {
    if (S.device_ready) return HEC_OK;
    int dev = 0, cnt = 0;
    if (cudaGetDeviceCount(&cnt) != cudaSuccess || cnt == 0) {
        cudaGetLastError();
        HEC_FAIL(HEC_ERR_CUDA, "no CUDA device present: libhec has no CPU fallback");
    }
    HEC_CUDA_OK(cudaGetDevice(&dev));
    HEC_CUDA_OK(cudaDeviceGetAttribute(&S.sm_count, cudaDevAttrMultiProcessorCount, dev));
    HEC_CUDA_OK(cudaDeviceGetAttribute(&S.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    for (auto &e : S.ev) HEC_CUDA_OK(cudaEventCreate(&e));
    S.device_ready = true;
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
    const uint32_t M = t.M, OFF = t.lmax;
    for (uint32_t i = 0; i < t.lmax; i++) out[i] = (T)OFF;
    uint32_t n = 0;
    for (uint32_t i = OFF; i < t.entries; i++) {
        const uint32_t z = F.zech[n];
        out[i] = (T)(z == M ? 0u : OFF + z);
        if (++n == M) n = 0;
    }
}

int build_plan(LibState &S, uint32_t q, uint32_t g, int regime, DevicePlan **out) {
    auto key = std::make_tuple(q, g, regime);
    auto it = S.plans.find(key);
    if (it != S.plans.end()) { *out = it->second.get(); return HEC_OK; }

    uint32_t p, r;
    if (!hec_factor_q(q, &p, &r)) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q must be an odd prime power below 65536");
    uint64_t Qg = 1;
    for (uint32_t i = 0; i < g; i++) { Qg *= q; if (Qg > HEC_MAX_FIELD_SIZE) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q^g exceeds HEC_MAX_FIELD_SIZE (2^26)"); }

    std::unique_ptr<DevicePlan> plan(new DevicePlan);
    plan->q = q; plan->g = g; plan->p = p; plan->r = r;
    const uint32_t D = 2 * g + 2;
    const uint32_t U = (uint32_t)plan->U;
    const uint32_t budget = (uint32_t)S.smem_optin - 1024u;

    std::vector<const hec_field *> fields(g);
    std::vector<hec_table_geom> geom(g);
    for (uint32_t k = 1; k <= g; k++) {
        fields[k - 1] = hec_cached_field(p, r, k);
        if (!fields[k - 1]) return HEC_ERR_INVALID_FIELD;
        geom[k - 1] = table_geom(fields[k - 1]->Q - 1, D, U);
    }
    // which tables live in shared memory (16-bit stored values must fit)
    std::vector<int> in_smem(g, 0);
    uint32_t smem_used = 0;
    for (uint32_t k = 1; k <= g; k++) {
        const hec_table_geom &t = geom[k - 1];
        const bool fits16 = (uint64_t)t.lmax + t.M <= 65536u;
        const uint32_t bytes = align16(t.entries * 2u);
        const bool force_l2 = regime == HEC_REGIME_L2 && k == g;
        if (fits16 && !force_l2 && smem_used + bytes <= budget) { in_smem[k - 1] = 1; smem_used += bytes; }
    }
    if (regime == HEC_REGIME_SMEM && !in_smem[g - 1])
        HEC_FAIL(HEC_ERR_INVALID_ARG, "HEC_REGIME_SMEM: the extended Zech table of the largest field does not fit shared memory");
    plan->regime = in_smem[g - 1] ? HEC_REGIME_SMEM : HEC_REGIME_L2;

    // one device allocation: [smem blob][global 32-bit tables][embed tables][squarefree tables]
    std::vector<uint8_t> host;
    auto reserve = [&](size_t bytes) { size_t o = host.size(); host.resize(o + ((bytes + 255) & ~(size_t)255)); return o; };
    const size_t blob_off = reserve(std::max<uint32_t>(smem_used, 16u));
    std::vector<size_t> gtab_off(g, 0), emb_off(g, 0);
    uint32_t so = 0;
    for (uint32_t k = 1; k <= g; k++) {
        const hec_table_geom &t = geom[k - 1];
        HecFieldDev &fd = plan->f[k - 1];
        fd.M = t.M; fd.off = t.lmax; fd.rcpM = (uint32_t)((1ull << 32) / t.M);
        fd.in_smem = (uint32_t)in_smem[k - 1];
        fd.lane_cap = std::min<uint32_t>(32u * U, t.M);
        fd.smem_off = 0;
        if (in_smem[k - 1]) {
            fd.smem_off = so;
            fill_extended<uint16_t>(*fields[k - 1], t, reinterpret_cast<uint16_t *>(host.data() + blob_off + so));
            so += align16(t.entries * 2u);
        } else {
            gtab_off[k - 1] = reserve((size_t)t.entries * 4u);
            fill_extended<uint32_t>(*fields[k - 1], t, reinterpret_cast<uint32_t *>(host.data() + gtab_off[k - 1]));
        }
        emb_off[k - 1] = reserve((size_t)q * 4u);
        uint32_t *e = reinterpret_cast<uint32_t *>(host.data() + emb_off[k - 1]);
        for (uint32_t c = 0; c < q; c++) e[c] = fields[k - 1]->embed[c] == t.M ? HEC_LOG_ZERO : fields[k - 1]->embed[c];
    }
    const size_t sqz_off = reserve((size_t)(q - 1) * 4u);
    std::copy(fields[0]->zech.begin(), fields[0]->zech.end(), reinterpret_cast<uint32_t *>(host.data() + sqz_off));

    HEC_CUDA_OK(cudaMalloc(&plan->d_blob, host.size()));
    HEC_CUDA_OK(cudaMemcpy(plan->d_blob, host.data(), host.size(), cudaMemcpyHostToDevice));
    HEC_CUDA_OK(cudaMalloc((void **)&plan->d_err, 2 * sizeof(unsigned long long)));
    const uint8_t *base = static_cast<const uint8_t *>(plan->d_blob);
    plan->blob = reinterpret_cast<const uint4 *>(base + blob_off);
    plan->blob_bytes = align16(smem_used);
    plan->smem_bytes = std::max<uint32_t>(align16(smem_used), 16u);
    for (uint32_t k = 1; k <= g; k++) {
        plan->f[k - 1].gtab = in_smem[k - 1] ? nullptr : reinterpret_cast<const uint32_t *>(base + gtab_off[k - 1]);
        plan->f[k - 1].emb = reinterpret_cast<const uint32_t *>(base + emb_off[k - 1]);
    }
    plan->sq_zech = reinterpret_cast<const uint32_t *>(base + sqz_off);
    plan->sq_emb = plan->f[0].emb;

    *out = plan.get();
    S.plans[key] = std::move(plan);
    return HEC_OK;
}

template <int G, int U>
int launch_count(LibState &S, const DevicePlan &plan, const HecCountParams &P) {
    auto kern = hec_count_kernel<G, U>;
    HEC_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes));
    const unsigned long long warps_needed = (P.n + 0ull);
    uint32_t grid = (uint32_t)std::min<unsigned long long>((warps_needed + kWarps - 1) / kWarps, (unsigned long long)S.sm_count);
    if (grid == 0) grid = 1;
    kern<<<grid, kThreads, plan.smem_bytes, S.stream>>>(P);
    hec_launch_counter::value++;
    S.stats.grid = grid;
    S.stats.block = kThreads;
    S.stats.chains_per_lane = U;
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
cudaStream_t hec_current_stream() { return g_state.stream; }
int hec_ensure_device(int *sm_count, int *smem_optin) {
    std::lock_guard<std::mutex> lock(g_state.mu);
    int rc = ensure_device(g_state);
    if (rc) return rc;
    if (sm_count) *sm_count = g_state.sm_count;
    if (smem_optin) *smem_optin = g_state.smem_optin;
    return HEC_OK;
}
bool hec_is_device_pointer(const void *p) { return is_device_pointer(p); }

extern "C" {

int hec_set_stream(void *cuda_stream) {
    std::lock_guard<std::mutex> lock(g_state.mu);
    g_state.stream = static_cast<cudaStream_t>(cuda_stream);
    return HEC_OK;
}

int hec_set_regime(int regime) {
    if (regime < HEC_REGIME_AUTO || regime > HEC_REGIME_L2) HEC_FAIL(HEC_ERR_INVALID_ARG, "unknown regime");
    std::lock_guard<std::mutex> lock(g_state.mu);
    g_state.regime = regime;
    return HEC_OK;
}

int hec_last_count_stats(hec_count_stats *out) {
    if (!out) HEC_FAIL(HEC_ERR_INVALID_ARG, "out is NULL");
    std::lock_guard<std::mutex> lock(g_state.mu);
    *out = g_state.stats;
    return HEC_OK;
}

uint64_t hec_launch_count(void) { return hec_launch_counter::value; }

int hec_count(uint32_t q, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t *out_counts, uint8_t *out_squarefree) {
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    uint32_t p, r;
    if (!hec_factor_q(q, &p, &r)) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q must be an odd prime power below 65536");
    {
        uint64_t Qg = 1;
        for (uint32_t i = 0; i < g; i++) { Qg *= q; if (Qg > HEC_MAX_FIELD_SIZE) HEC_FAIL(HEC_ERR_INVALID_FIELD, "q^g exceeds HEC_MAX_FIELD_SIZE (2^26)"); }
    }
    if (n == 0) return HEC_OK;
    if (!coeffs || !out_counts) HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs and out_counts must not be NULL");

    std::lock_guard<std::mutex> lock(g_state.mu);
    LibState &S = g_state;
    int rc = ensure_device(S);
    if (rc) return rc;
    const bool dev_in = is_device_pointer(coeffs), dev_out = is_device_pointer(out_counts);
    const bool dev_sf = out_squarefree ? is_device_pointer(out_squarefree) : dev_out;
    if (dev_in != dev_out || dev_sf != dev_out) HEC_FAIL(HEC_ERR_INVALID_ARG, "coeffs/out_counts/out_squarefree must all be host or all device pointers");

    DevicePlan *plan = nullptr;
    rc = build_plan(S, q, g, S.regime, &plan);
    if (rc) return rc;

    const size_t ncoef = 2 * (size_t)g + 3;
    const size_t in_bytes = n * ncoef * sizeof(uint16_t), cnt_bytes = n * g * sizeof(uint32_t), sf_bytes = out_squarefree ? n : 0;
    const uint16_t *d_coeffs = coeffs;
    uint32_t *d_counts = out_counts;
    uint8_t *d_sf = out_squarefree;
    if (!dev_in) {
        const size_t a = (in_bytes + 255) & ~(size_t)255, b = (cnt_bytes + 255) & ~(size_t)255;
        const size_t need = a + b + sf_bytes;
        if (need > S.stage_bytes) {
            if (S.d_stage) cudaFree(S.d_stage);
            S.d_stage = nullptr; S.stage_bytes = 0;
            if (cudaMalloc(&S.d_stage, need) != cudaSuccess) { cudaGetLastError(); HEC_FAIL(HEC_ERR_NOMEM, "cannot allocate device staging buffers"); }
            S.stage_bytes = need;
        }
        uint8_t *base = static_cast<uint8_t *>(S.d_stage);
        d_coeffs = reinterpret_cast<const uint16_t *>(base);
        d_counts = reinterpret_cast<uint32_t *>(base + a);
        d_sf = out_squarefree ? base + a + b : nullptr;
        HEC_CUDA_OK(cudaMemcpyAsync(base, coeffs, in_bytes, cudaMemcpyHostToDevice, S.stream));
    }

    static const unsigned long long kNoErr[2] = {~0ull, ~0ull};
    HEC_CUDA_OK(cudaMemcpyAsync(plan->d_err, kNoErr, sizeof kNoErr, cudaMemcpyHostToDevice, S.stream));

    HecCountParams P;
    P.coeffs = d_coeffs; P.out = d_counts; P.n = n; P.q = q;
    P.blob = plan->blob; P.blob_bytes = plan->blob_bytes; P.err = plan->d_err;
    for (uint32_t k = 0; k < HEC_MAX_GENUS; k++) P.f[k] = plan->f[k < g ? k : 0];

    S.stats = hec_count_stats{};
    S.stats.regime = (uint32_t)plan->regime;
    S.stats.smem_bytes = plan->smem_bytes;
    HEC_CUDA_OK(cudaEventRecord(S.ev[0], S.stream));
    switch (g) {
        case 1: rc = launch_count<1, 4>(S, *plan, P); break;
        case 2: rc = launch_count<2, 4>(S, *plan, P); break;
        case 3: rc = launch_count<3, 4>(S, *plan, P); break;
        case 4: rc = launch_count<4, 4>(S, *plan, P); break;
        default: rc = launch_count<5, 4>(S, *plan, P); break;
    }
    if (rc) return rc;
    HEC_CUDA_OK(cudaEventRecord(S.ev[1], S.stream));
    S.stats.launches = 1;
    if (d_sf) {
        HecSquarefreeParams Q;
        Q.coeffs = d_coeffs; Q.out = d_sf; Q.n = n; Q.p = p; Q.q = q; Q.M = q - 1; Q.ncoef = (uint32_t)ncoef;
        Q.zech = plan->sq_zech; Q.emb = plan->sq_emb;
        const unsigned long long blocks = (n + 255) / 256;
        hec_squarefree_kernel<<<(unsigned)blocks, 256, 0, S.stream>>>(Q);
        hec_launch_counter::value++;
        S.stats.launches = 2;
        HEC_CUDA_OK(cudaGetLastError());
    }
    HEC_CUDA_OK(cudaEventRecord(S.ev[2], S.stream));
    unsigned long long err[2];
    HEC_CUDA_OK(cudaMemcpyAsync(err, plan->d_err, sizeof err, cudaMemcpyDeviceToHost, S.stream));
    if (!dev_in) {
        HEC_CUDA_OK(cudaMemcpyAsync(out_counts, d_counts, cnt_bytes, cudaMemcpyDeviceToHost, S.stream));
        if (out_squarefree) HEC_CUDA_OK(cudaMemcpyAsync(out_squarefree, d_sf, sf_bytes, cudaMemcpyDeviceToHost, S.stream));
    }
    HEC_CUDA_OK(cudaStreamSynchronize(S.stream));
    cudaEventElapsedTime(&S.stats.count_kernel_ms, S.ev[0], S.ev[1]);
    cudaEventElapsedTime(&S.stats.squarefree_kernel_ms, S.ev[1], S.ev[2]);
    if (err[0] != ~0ull) {
        hec_set_error(HEC_ERR_COEFF_RANGE, "a coefficient is >= q", (size_t)err[0]);
        return HEC_ERR_COEFF_RANGE;
    }
    if (err[1] != ~0ull) {
        hec_set_error(HEC_ERR_DEGREE, "a row has c[2g+2] = c[2g+1] = 0 (degree < 2g+1)", (size_t)err[1]);
        return HEC_ERR_DEGREE;
    }
    return HEC_OK;
}

void hec_shutdown(void) {
    std::lock_guard<std::mutex> lock(g_state.mu);
    g_state.plans.clear();
    if (g_state.d_stage) { cudaFree(g_state.d_stage); g_state.d_stage = nullptr; g_state.stage_bytes = 0; }
    hec_clear_field_cache();
}

}  // extern "C"
