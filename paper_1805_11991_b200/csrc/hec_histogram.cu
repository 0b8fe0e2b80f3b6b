// hec_histogram: multiplicities of the tuples (N_1..N_g) -- the map N_{g,q} of eq. (1.2), PAPER.md:63-69,
// incremented at Algorithm 1 line 20, in its reduced form (unweighted, no lambda).
// The paper does this on the host; here: pack each row into a 64-bit key relative to the column minima,
// aggregate in a per-CTA shared-memory hash table (shared-memory atomics), merge into a global hash table,
// compact the occupied slots, LSD-radix-sort the distinct keys (ascending lexicographic order) and unpack.
#include <algorithm>
#include <map>
#include <mutex>
#include <vector>

#include "hec_device.cuh"

cudaStream_t hec_current_stream();
int hec_ensure_device(int *sm_count, int *smem_optin);
bool hec_is_device_pointer(const void *p);

namespace {

constexpr unsigned long long kEmpty = ~0ull;
constexpr int kSharedSlots = 2048;          // per-CTA table: 2048 x (8 B key + 8 B count) = 32 KB
constexpr int kSharedProbes = 8;

struct PackSpec {
    uint32_t g;
    uint32_t mn[HEC_MAX_GENUS];
    uint32_t shift[HEC_MAX_GENUS];
    uint32_t bits[HEC_MAX_GENUS];
};

__global__ void hist_minmax_kernel(const uint32_t *counts, const uint8_t *mask, const unsigned long long *weights,
                                   unsigned long long n, uint32_t g, uint32_t *mn, uint32_t *mx, unsigned long long *rows) {
    uint32_t lmn[HEC_MAX_GENUS], lmx[HEC_MAX_GENUS];
    for (uint32_t k = 0; k < g; k++) { lmn[k] = 0xFFFFFFFFu; lmx[k] = 0; }
    unsigned long long cnt = 0;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        if (mask && !mask[i]) continue;
        if (weights && weights[i] == 0) continue;
        cnt++;
        for (uint32_t k = 0; k < g; k++) {
            const uint32_t v = counts[i * g + k];
            lmn[k] = min(lmn[k], v);
            lmx[k] = max(lmx[k], v);
        }
    }
    for (uint32_t k = 0; k < g; k++) {
        const uint32_t a = __reduce_min_sync(0xffffffffu, lmn[k]);
        const uint32_t b = __reduce_max_sync(0xffffffffu, lmx[k]);
        if ((threadIdx.x & 31) == 0) { atomicMin(&mn[k], a); atomicMax(&mx[k], b); }
    }
    for (int o = 16; o; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(rows, cnt);
}

__device__ __forceinline__ unsigned long long hash64(unsigned long long x) {
    x ^= x >> 33; x *= 0xff51afd7ed558ccdull; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull; x ^= x >> 33;
    return x;
}

__device__ __forceinline__ void global_insert(unsigned long long *gkeys, unsigned long long *gcnt, unsigned long long capmask,
                                              unsigned long long key, unsigned long long cnt) {
    unsigned long long slot = hash64(key) & capmask;
    for (;;) {
        const unsigned long long prev = atomicCAS(&gkeys[slot], kEmpty, key);
        if (prev == kEmpty || prev == key) { atomicAdd(&gcnt[slot], cnt); return; }
        slot = (slot + 1) & capmask;
    }
}

__global__ void __launch_bounds__(512) hist_insert_kernel(const uint32_t *counts, const uint8_t *mask, const unsigned long long *weights,
                                                          unsigned long long n, PackSpec S, unsigned long long *gkeys,
                                                          unsigned long long *gcnt, unsigned long long capmask) {
    __shared__ unsigned long long skeys[kSharedSlots];
    __shared__ unsigned long long scnt[kSharedSlots];
    for (int i = threadIdx.x; i < kSharedSlots; i += blockDim.x) { skeys[i] = kEmpty; scnt[i] = 0; }
    __syncthreads();
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        if (mask && !mask[i]) continue;
        const unsigned long long w = weights ? weights[i] : 1ull;
        if (w == 0) continue;
        unsigned long long key = 0;
        for (uint32_t k = 0; k < S.g; k++) key |= (unsigned long long)(counts[i * S.g + k] - S.mn[k]) << S.shift[k];
        uint32_t slot = (uint32_t)hash64(key) & (kSharedSlots - 1);
        bool done = false;
        for (int probe = 0; probe < kSharedProbes && !done; probe++) {
            const unsigned long long prev = atomicCAS(&skeys[slot], kEmpty, key);
            if (prev == kEmpty || prev == key) { atomicAdd(&scnt[slot], w); done = true; }
            slot = (slot + 1) & (kSharedSlots - 1);
        }
        if (!done) global_insert(gkeys, gcnt, capmask, key, w);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kSharedSlots; i += blockDim.x)
        if (skeys[i] != kEmpty) global_insert(gkeys, gcnt, capmask, skeys[i], scnt[i]);
}

__global__ void hist_compact_kernel(const unsigned long long *gkeys, const unsigned long long *gcnt, unsigned long long cap,
                                    unsigned long long *okeys, unsigned long long *ocnt, unsigned long long *m) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < cap;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long key = gkeys[i];
        if (key == kEmpty) continue;
        const unsigned long long pos = atomicAdd(m, 1ull);      // ptxas aggregates per warp (REDUX + one atomic)
        okeys[pos] = key;
        ocnt[pos] = gcnt[i];
    }
}

// ---- LSD radix sort of (key, value) pairs, 8 bits per pass, stable ---------------------------------
constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kItemsPerWarp = 256;
constexpr int kTile = kSortWarps * kItemsPerWarp;   // 2048

__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(const unsigned long long *keys, unsigned long long m, uint32_t shift,
                                                                  uint32_t *hist, uint32_t nblocks) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const unsigned long long base = (unsigned long long)blockIdx.x * kTile;
    for (int j = threadIdx.x; j < kTile; j += kSortThreads) {
        const unsigned long long i = base + j;
        if (i < m) atomicAdd(&h[(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// exclusive scan of `len` counters in place, one block; every thread takes kScanItems consecutive counters per round
constexpr int kScanItems = 16;
__global__ void __launch_bounds__(1024) radix_scan_kernel(uint32_t *hist, unsigned long long len) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (unsigned long long base = 0; base < len; base += 1024ull * kScanItems) {
        const unsigned long long i0 = base + (unsigned long long)threadIdx.x * kScanItems;
        uint32_t v[kScanItems];
        uint32_t tsum = 0;
#pragma unroll
        for (int j = 0; j < kScanItems; j++) { v[j] = i0 + j < len ? hist[i0 + j] : 0u; tsum += v[j]; }
        uint32_t s = tsum;
        for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, s, o); if (lane >= (uint32_t)o) s += t; }
        if (lane == 31) wsum[warp] = s;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = wsum[lane];
            for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, w, o); if (lane >= (uint32_t)o) w += t; }
            wsum[lane] = w;
        }
        __syncthreads();
        const uint32_t carry = carry_s;
        uint32_t excl = carry + (warp ? wsum[warp - 1] : 0) + s - tsum;
#pragma unroll
        for (int j = 0; j < kScanItems; j++) { if (i0 + j < len) hist[i0 + j] = excl; excl += v[j]; }
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + wsum[31];
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kSortThreads) radix_scatter_kernel(const unsigned long long *keys, const unsigned long long *vals,
                                                                     unsigned long long *okeys, unsigned long long *ovals,
                                                                     unsigned long long m, uint32_t shift, const uint32_t *hist,
                                                                     uint32_t nblocks) {
    __shared__ uint32_t wcount[kSortWarps][256];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j = threadIdx.x; j < kSortWarps * 256; j += kSortThreads) (&wcount[0][0])[j] = 0;
    __syncthreads();
    constexpr int kRounds = kItemsPerWarp / 32;
    unsigned long long key[kRounds];
    uint32_t off[kRounds];
    const unsigned long long wbase = (unsigned long long)blockIdx.x * kTile + (unsigned long long)warp * kItemsPerWarp;
#pragma unroll
    for (int rd = 0; rd < kRounds; rd++) {
        const unsigned long long i = wbase + rd * 32 + lane;
        const bool valid = i < m;
        key[rd] = valid ? keys[i] : 0;
        const uint32_t digit = valid ? (uint32_t)((key[rd] >> shift) & 255u) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, digit);
        const uint32_t rank = __popc(peers & ((1u << lane) - 1u));
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (valid && (int)lane == leader) { old = wcount[warp][digit]; wcount[warp][digit] = old + __popc(peers); }
        old = __shfl_sync(0xffffffffu, old, leader);
        off[rd] = old + rank;
        __syncwarp();
    }
    __syncthreads();
    {
        const uint32_t d = threadIdx.x;                      // kSortThreads == 256 digits
        uint32_t running = hist[(size_t)d * nblocks + blockIdx.x];
        for (int w = 0; w < kSortWarps; w++) { const uint32_t t = wcount[w][d]; wcount[w][d] = running; running += t; }
    }
    __syncthreads();
#pragma unroll
    for (int rd = 0; rd < kRounds; rd++) {
        const unsigned long long i = wbase + rd * 32 + lane;
        if (i < m) {
            const uint32_t digit = (uint32_t)((key[rd] >> shift) & 255u);
            const unsigned long long pos = (unsigned long long)wcount[warp][digit] + off[rd];
            okeys[pos] = key[rd];
            ovals[pos] = vals[i];
        }
    }
}

__global__ void hist_unpack_kernel(const unsigned long long *keys, const unsigned long long *cnt, unsigned long long m, PackSpec S,
                                   uint32_t *out_tuples, unsigned long long *out_mult) {
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const unsigned long long key = keys[i];
    for (uint32_t k = 0; k < S.g; k++) {
        const unsigned long long msk = S.bits[k] >= 64 ? ~0ull : ((1ull << S.bits[k]) - 1ull);
        out_tuples[i * S.g + k] = S.mn[k] + (uint32_t)((key >> S.shift[k]) & msk);
    }
    out_mult[i] = cnt[i];
}

// Device scratch comes from a small caching pool (best fit, grow-only, released by hec_shutdown): a call needs up to
// ~1 GB of hash-table and sort buffers, and cudaMalloc/cudaFree of that size cost far more than the kernels.
struct Pool {
    std::mutex mu;
    std::vector<std::pair<void *, size_t>> idle;
    std::map<void *, size_t> live;
    int get(size_t bytes, void **out) {
        std::lock_guard<std::mutex> lock(mu);
        size_t best = idle.size();
        for (size_t i = 0; i < idle.size(); i++)
            if (idle[i].second >= bytes && idle[i].second <= 2 * bytes + (1u << 20) && (best == idle.size() || idle[i].second < idle[best].second)) best = i;
        if (best != idle.size()) {
            *out = idle[best].first;
            live[*out] = idle[best].second;
            idle.erase(idle.begin() + (long)best);
            return HEC_OK;
        }
        void *p = nullptr;
        if (cudaMalloc(&p, bytes) != cudaSuccess) {
            cudaGetLastError();
            for (auto &b : idle) cudaFree(b.first);          // drop the cache and retry once
            idle.clear();
            if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); HEC_FAIL(HEC_ERR_NOMEM, "device allocation failed in hec_histogram"); }
        }
        live[p] = bytes;
        *out = p;
        return HEC_OK;
    }
    void put(void *p) {
        std::lock_guard<std::mutex> lock(mu);
        auto it = live.find(p);
        if (it == live.end()) return;
        idle.emplace_back(p, it->second);
        live.erase(it);
    }
    void clear() {
        std::lock_guard<std::mutex> lock(mu);
        for (auto &b : idle) cudaFree(b.first);
        idle.clear();
    }
};
Pool g_pool;

struct DeviceBuf {
    void *p = nullptr;
    ~DeviceBuf() { if (p) g_pool.put(p); }
    int alloc(size_t bytes) { return g_pool.get(std::max<size_t>(bytes, 256), &p); }
};

}  // namespace

void hec_histogram_release_pool() { g_pool.clear(); }

// mixed: device inputs with outputs on either side (hec_count_histogram with host buffers: the counts are still on the device)
static int histogram_impl(const uint32_t *counts, const uint8_t *mask, const uint64_t *weights, size_t n, uint32_t g,
                          uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m, bool mixed = false) {
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    if (!out_m) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_m must not be NULL");
    *out_m = 0;
    if (n == 0) return HEC_OK;
    if (!counts) HEC_FAIL(HEC_ERR_INVALID_ARG, "counts must not be NULL");
    if (cap > 0 && (!out_tuples || !out_mult)) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_tuples/out_mult must not be NULL when cap > 0");
    int sms = 0;
    int rc = hec_ensure_device(&sms, nullptr);
    if (rc) return rc;
    cudaStream_t st = hec_current_stream();
    const bool dev = hec_is_device_pointer(counts);
    const bool dev_out = (mixed && cap > 0) ? hec_is_device_pointer(out_tuples) : dev;
    if ((mask && hec_is_device_pointer(mask) != dev) || (weights && hec_is_device_pointer(weights) != dev) || (cap > 0 && (hec_is_device_pointer(out_tuples) != dev_out || hec_is_device_pointer(out_mult) != dev_out)))
        HEC_FAIL(HEC_ERR_INVALID_ARG, "counts/mask/out_tuples/out_mult must all be host or all device pointers");

    DeviceBuf in_counts, in_mask, in_w;
    const uint32_t *d_counts = counts;
    const uint8_t *d_mask = mask;
    const unsigned long long *d_w = reinterpret_cast<const unsigned long long *>(weights);
    if (!dev) {
        if ((rc = in_counts.alloc(n * g * sizeof(uint32_t)))) return rc;
        HEC_CUDA_OK(cudaMemcpyAsync(in_counts.p, counts, n * g * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
        d_counts = static_cast<const uint32_t *>(in_counts.p);
        if (mask) {
            if ((rc = in_mask.alloc(n))) return rc;
            HEC_CUDA_OK(cudaMemcpyAsync(in_mask.p, mask, n, cudaMemcpyHostToDevice, st));
            d_mask = static_cast<const uint8_t *>(in_mask.p);
        }
        if (weights) {
            if ((rc = in_w.alloc(n * 8))) return rc;
            HEC_CUDA_OK(cudaMemcpyAsync(in_w.p, weights, n * 8, cudaMemcpyHostToDevice, st));
            d_w = static_cast<const unsigned long long *>(in_w.p);
        }
    }

    // 1. column ranges over the unmasked rows
    DeviceBuf scal;   // [mn g][mx g] u32, then rows u64, m u64
    if ((rc = scal.alloc(64 + 2 * sizeof(unsigned long long)))) return rc;
    uint32_t h_init[16];
    for (int i = 0; i < 8; i++) { h_init[i] = 0xFFFFFFFFu; h_init[8 + i] = 0; }
    unsigned long long h_zero[2] = {0, 0};
    uint32_t *d_mn = static_cast<uint32_t *>(scal.p), *d_mx = d_mn + 8;
    unsigned long long *d_rows = reinterpret_cast<unsigned long long *>(static_cast<char *>(scal.p) + 64), *d_m = d_rows + 1;
    HEC_CUDA_OK(cudaMemcpyAsync(d_mn, h_init, sizeof h_init, cudaMemcpyHostToDevice, st));
    HEC_CUDA_OK(cudaMemcpyAsync(d_rows, h_zero, sizeof h_zero, cudaMemcpyHostToDevice, st));
    const unsigned grid = (unsigned)std::min<unsigned long long>((n + 511) / 512, (unsigned long long)sms * 4);
    hist_minmax_kernel<<<grid, 512, 0, st>>>(d_counts, d_mask, d_w, n, g, d_mn, d_mx, d_rows);
    hec_launch_counter::value++;
    uint32_t h_mm[16];
    unsigned long long h_rows = 0;
    HEC_CUDA_OK(cudaMemcpyAsync(h_mm, d_mn, sizeof h_mm, cudaMemcpyDeviceToHost, st));
    HEC_CUDA_OK(cudaMemcpyAsync(&h_rows, d_rows, sizeof h_rows, cudaMemcpyDeviceToHost, st));
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    if (h_rows == 0) return HEC_OK;

    PackSpec S;
    S.g = g;
    uint32_t total_bits = 0;
    for (uint32_t k = 0; k < g; k++) {
        S.mn[k] = h_mm[k];
        const uint32_t range = h_mm[8 + k] - h_mm[k];
        uint32_t b = 0;
        while (b < 32 && (range >> b)) b++;
        S.bits[k] = b;
        total_bits += b;
    }
    if (total_bits > 63) HEC_FAIL(HEC_ERR_UNSUPPORTED, "tuple ranges need more than 63 bits");
    uint32_t sh = total_bits;
    for (uint32_t k = 0; k < g; k++) { sh -= S.bits[k]; S.shift[k] = sh; }     // N_1 most significant

    // 2. shared-memory hash -> global hash
    unsigned long long capslots = 1024;
    while (capslots < 2 * h_rows) capslots <<= 1;
    if (total_bits < 40) { unsigned long long dom = 1ull << total_bits; while (capslots / 2 >= 2 * dom && capslots > 1024) capslots >>= 1; }
    DeviceBuf gkeys, gcnt;
    if ((rc = gkeys.alloc(capslots * 8)) || (rc = gcnt.alloc(capslots * 8))) return rc;
    HEC_CUDA_OK(cudaMemsetAsync(gkeys.p, 0xFF, capslots * 8, st));
    HEC_CUDA_OK(cudaMemsetAsync(gcnt.p, 0, capslots * 8, st));
    hist_insert_kernel<<<(unsigned)std::min<unsigned long long>((n + 511) / 512, (unsigned long long)sms * 2), 512, 0, st>>>(
        d_counts, d_mask, d_w, n, S, static_cast<unsigned long long *>(gkeys.p), static_cast<unsigned long long *>(gcnt.p), capslots - 1);
    hec_launch_counter::value++;
    HEC_CUDA_OK(cudaGetLastError());

    // 3. compact
    const unsigned long long maxm = std::min<unsigned long long>(h_rows, capslots);
    DeviceBuf k0, v0, k1, v1;
    if ((rc = k0.alloc(maxm * 8)) || (rc = v0.alloc(maxm * 8))) return rc;
    hist_compact_kernel<<<(unsigned)std::min<unsigned long long>((capslots + 255) / 256, (unsigned long long)sms * 8), 256, 0, st>>>(
        static_cast<unsigned long long *>(gkeys.p), static_cast<unsigned long long *>(gcnt.p), capslots,
        static_cast<unsigned long long *>(k0.p), static_cast<unsigned long long *>(v0.p), d_m);
    hec_launch_counter::value++;
    unsigned long long m = 0;
    HEC_CUDA_OK(cudaMemcpyAsync(&m, d_m, sizeof m, cudaMemcpyDeviceToHost, st));
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    *out_m = (size_t)m;
    if (cap < m) HEC_FAIL(HEC_ERR_CAPACITY, "cap is smaller than the number of distinct tuples");

    // 4. sort the distinct keys
    unsigned long long *ka = static_cast<unsigned long long *>(k0.p), *va = static_cast<unsigned long long *>(v0.p);
    if (total_bits > 0 && m > 1) {
        if ((rc = k1.alloc(m * 8)) || (rc = v1.alloc(m * 8))) return rc;
        unsigned long long *kb = static_cast<unsigned long long *>(k1.p), *vb = static_cast<unsigned long long *>(v1.p);
        const uint32_t nblocks = (uint32_t)((m + kTile - 1) / kTile);
        DeviceBuf hist;
        if ((rc = hist.alloc((size_t)256 * nblocks * 4))) return rc;
        for (uint32_t shift = 0; shift < total_bits; shift += 8) {
            radix_hist_kernel<<<nblocks, kSortThreads, 0, st>>>(ka, m, shift, static_cast<uint32_t *>(hist.p), nblocks);
            radix_scan_kernel<<<1, 1024, 0, st>>>(static_cast<uint32_t *>(hist.p), (unsigned long long)256 * nblocks);
            radix_scatter_kernel<<<nblocks, kSortThreads, 0, st>>>(ka, va, kb, vb, m, shift, static_cast<const uint32_t *>(hist.p), nblocks);
            hec_launch_counter::value += 3;
            std::swap(ka, kb);
            std::swap(va, vb);
        }
        HEC_CUDA_OK(cudaGetLastError());
    }

    // 5. unpack
    DeviceBuf o_t, o_m;
    uint32_t *d_t = out_tuples;
    unsigned long long *d_mu = reinterpret_cast<unsigned long long *>(out_mult);
    if (!dev_out) {
        if ((rc = o_t.alloc(m * g * 4)) || (rc = o_m.alloc(m * 8))) return rc;
        d_t = static_cast<uint32_t *>(o_t.p);
        d_mu = static_cast<unsigned long long *>(o_m.p);
    }
    hist_unpack_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(ka, va, m, S, d_t, d_mu);
    hec_launch_counter::value++;
    HEC_CUDA_OK(cudaGetLastError());
    if (!dev_out) {
        HEC_CUDA_OK(cudaMemcpyAsync(out_tuples, d_t, m * g * 4, cudaMemcpyDeviceToHost, st));
        HEC_CUDA_OK(cudaMemcpyAsync(out_mult, d_mu, m * 8, cudaMemcpyDeviceToHost, st));
    }
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    return HEC_OK;
}

extern "C" int hec_histogram(const uint32_t *counts, const uint8_t *mask, size_t n, uint32_t g, uint32_t *out_tuples,
                             uint64_t *out_mult, size_t cap, size_t *out_m) {
    return histogram_impl(counts, mask, nullptr, n, g, out_tuples, out_mult, cap, out_m);
}

// hec_count.cu (hec_count_histogram): device counts / mask, outputs on the caller's side
int hec_histogram_mixed(const uint32_t *counts, const uint8_t *mask, size_t n, uint32_t g, uint32_t *out_tuples, uint64_t *out_mult,
                        size_t cap, size_t *out_m) {
    return histogram_impl(counts, mask, nullptr, n, g, out_tuples, out_mult, cap, out_m, true);
}

// hec_enum.cu: weighted histogram of the rows with a nonzero mask (Algorithm 1 line 20 for one chunk).
int hec_histogram_weighted(const uint32_t *counts, const uint8_t *mask, const uint64_t *weights, size_t n, uint32_t g,
                           uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m) {
    return histogram_impl(counts, mask, weights, n, g, out_tuples, out_mult, cap, out_m);
}

extern "C" int hec_histogram_merge(const uint32_t *in_tuples, const uint64_t *in_mult, size_t n, uint32_t g,
                                   uint32_t *out_tuples, uint64_t *out_mult, size_t cap, size_t *out_m) {
    if (n > 0 && !in_mult) HEC_FAIL(HEC_ERR_INVALID_ARG, "in_mult must not be NULL");
    return histogram_impl(in_tuples, nullptr, in_mult, n, g, out_tuples, out_mult, cap, out_m);
}

// ---- hec_histogram_static: the same pipeline with every scratch buffer inside one fixed array -----------------------
// For callers that must not touch the device allocator.  Two kinds turn up in practice: (1) a process whose device
// memory already belongs to someone else -- a tensor framework's caching allocator or a serving engine that grabbed
// nearly all of HBM at start-up -- where a cudaMalloc of hec_histogram's hash and sort buffers either fails or eats
// into a budget the caller was promised; (2) a caller in a section where the device-wide synchronisation that
// cudaMalloc / cudaFree imply would stall unrelated streams (a latency-bound serving loop next to this library).
// hec_histogram's pool (above) grows on demand, so neither can use it.  Here the scratch is a file-scope device array
// of fixed size: it is part of the module image, every GPU that loads libhec holds these 8.07 MiB from the first CUDA
// call of the process until exit, and no call allocates or frees anything.
//
// Layout (bytes), kStaticMaxRows = 2^17 rows:
//   [0, 256)              column minima / maxima (16 x u32), unmasked-row counter, distinct-tuple counter
//   gkeys, gcnt           global hash: 2 * kStaticMaxRows slots x 8 B each            2 MiB + 2 MiB
//   k0, v0, k1, v1        compacted (key, multiplicity) pairs + the sort's ping-pong copy, kStaticMaxRows x 8 B each   4 MiB
//   hist                  256 digit counters per 2048-key sort tile                   64 KiB
constexpr size_t kStaticMaxRows = HEC_HISTOGRAM_STATIC_MAX_ROWS;
constexpr size_t kStaticSlots = 2 * kStaticMaxRows;
constexpr size_t kStaticTiles = (kStaticMaxRows + kTile - 1) / kTile;
constexpr size_t kStaticOffKeys = 256;
constexpr size_t kStaticOffCnt = kStaticOffKeys + kStaticSlots * 8;
constexpr size_t kStaticOffSort = kStaticOffCnt + kStaticSlots * 8;
constexpr size_t kStaticOffHist = kStaticOffSort + 4 * kStaticMaxRows * 8;
constexpr size_t kStaticBytes = kStaticOffHist + 256 * kStaticTiles * 4;
static_assert(kStaticMaxRows % kTile == 0 && (kStaticSlots & (kStaticSlots - 1)) == 0, "scratch layout");

static __device__ __align__(256) unsigned char hec_static_scratch[kStaticBytes];

namespace {
// In host code `hec_static_scratch` is only the host-side shadow of the device symbol, not somewhere a kernel may
// write: the device address is asked for once per device (with that device current) and kept here.
constexpr int kMaxDevices = 64;
struct StaticScratch {
    std::mutex mu;
    unsigned char *base[kMaxDevices] = {};
    int sms[kMaxDevices] = {};
} g_static;

int static_scratch_for_current_device(unsigned char **base, int *sms) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        HEC_FAIL(HEC_ERR_CUDA, "hec_histogram_static: no CUDA device present (libhec has no CPU fallback)");
    }
    if (dev < 0 || dev >= kMaxDevices) HEC_FAIL(HEC_ERR_UNSUPPORTED, "hec_histogram_static: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_static.mu);
    if (!g_static.base[dev]) {
        void *p = nullptr;
        HEC_CUDA_OK(cudaGetSymbolAddress(&p, hec_static_scratch));
        int n = 0;
        HEC_CUDA_OK(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev));
        g_static.sms[dev] = n;
        g_static.base[dev] = static_cast<unsigned char *>(p);
    }
    *base = g_static.base[dev];
    *sms = g_static.sms[dev];
    return HEC_OK;
}
}  // namespace

extern "C" int hec_histogram_static(const uint32_t *counts, const uint8_t *mask, size_t n, uint32_t g, uint32_t *out_tuples,
                                    uint64_t *out_mult, size_t cap, size_t *out_m) {
    if (g < 1 || g > HEC_MAX_GENUS) HEC_FAIL(HEC_ERR_INVALID_ARG, "g must be in [1, HEC_MAX_GENUS]");
    if (!out_m) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_m must not be NULL");
    *out_m = 0;
    if (n > kStaticMaxRows)
        HEC_FAIL(HEC_ERR_CAPACITY, "hec_histogram_static: n = " + std::to_string(n) + " rows exceed the fixed scratch array's limit of " +
                                       std::to_string(kStaticMaxRows) + " (HEC_HISTOGRAM_STATIC_MAX_ROWS); split the batch and combine the parts with "
                                       "hec_histogram_merge, or use hec_histogram where allocating is allowed");
    if (n == 0) return HEC_OK;
    if (!counts) HEC_FAIL(HEC_ERR_INVALID_ARG, "counts must not be NULL");
    if (cap > 0 && (!out_tuples || !out_mult)) HEC_FAIL(HEC_ERR_INVALID_ARG, "out_tuples/out_mult must not be NULL when cap > 0");
    unsigned char *base = nullptr;
    int sms = 0;
    int rc = static_scratch_for_current_device(&base, &sms);
    if (rc) return rc;
    // host arrays would need a staging buffer on the device, i.e. an allocation
    if (!hec_is_device_pointer(counts) || (mask && !hec_is_device_pointer(mask)) ||
        (cap > 0 && (!hec_is_device_pointer(out_tuples) || !hec_is_device_pointer(out_mult))))
        HEC_FAIL(HEC_ERR_INVALID_ARG, "hec_histogram_static: counts/mask/out_tuples/out_mult must be device pointers (staging host arrays would allocate)");
    cudaStream_t st = hec_current_stream();

    uint32_t *d_mn = reinterpret_cast<uint32_t *>(base), *d_mx = d_mn + 8;
    unsigned long long *d_rows = reinterpret_cast<unsigned long long *>(base + 64), *d_m = d_rows + 1;
    unsigned long long *gkeys = reinterpret_cast<unsigned long long *>(base + kStaticOffKeys);
    unsigned long long *gcnt = reinterpret_cast<unsigned long long *>(base + kStaticOffCnt);
    unsigned long long *ka = reinterpret_cast<unsigned long long *>(base + kStaticOffSort), *va = ka + kStaticMaxRows;
    unsigned long long *kb = va + kStaticMaxRows, *vb = kb + kStaticMaxRows;
    uint32_t *hist = reinterpret_cast<uint32_t *>(base + kStaticOffHist);

    // The array still holds the previous call's data: everything a kernel reads before writing is reset here
    // (scalars now, the hash slots below once their number is known); the sort buffers and digit counters are
    // written in full before they are read.
    uint32_t h_init[16];
    for (int i = 0; i < 8; i++) { h_init[i] = 0xFFFFFFFFu; h_init[8 + i] = 0; }
    unsigned long long h_zero[2] = {0, 0};
    HEC_CUDA_OK(cudaMemcpyAsync(d_mn, h_init, sizeof h_init, cudaMemcpyHostToDevice, st));
    HEC_CUDA_OK(cudaMemcpyAsync(d_rows, h_zero, sizeof h_zero, cudaMemcpyHostToDevice, st));
    const unsigned long long nn = n;
    hist_minmax_kernel<<<(unsigned)std::min<unsigned long long>((nn + 511) / 512, (unsigned long long)sms * 4), 512, 0, st>>>(
        counts, mask, nullptr, nn, g, d_mn, d_mx, d_rows);
    hec_launch_counter::value++;
    uint32_t h_mm[16];
    unsigned long long h_rows = 0;
    HEC_CUDA_OK(cudaMemcpyAsync(h_mm, d_mn, sizeof h_mm, cudaMemcpyDeviceToHost, st));
    HEC_CUDA_OK(cudaMemcpyAsync(&h_rows, d_rows, sizeof h_rows, cudaMemcpyDeviceToHost, st));
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    if (h_rows == 0) return HEC_OK;

    PackSpec S;
    S.g = g;
    uint32_t total_bits = 0;
    for (uint32_t k = 0; k < g; k++) {
        S.mn[k] = h_mm[k];
        const uint32_t range = h_mm[8 + k] - h_mm[k];
        uint32_t b = 0;
        while (b < 32 && (range >> b)) b++;
        S.bits[k] = b;
        total_bits += b;
    }
    if (total_bits > 63) HEC_FAIL(HEC_ERR_UNSUPPORTED, "tuple ranges need more than 63 bits");
    uint32_t sh = total_bits;
    for (uint32_t k = 0; k < g; k++) { sh -= S.bits[k]; S.shift[k] = sh; }     // N_1 most significant

    unsigned long long capslots = 1024;
    while (capslots < 2 * h_rows) capslots <<= 1;                              // <= kStaticSlots since h_rows <= n
    HEC_CUDA_OK(cudaMemsetAsync(gkeys, 0xFF, capslots * 8, st));
    HEC_CUDA_OK(cudaMemsetAsync(gcnt, 0, capslots * 8, st));
    hist_insert_kernel<<<(unsigned)std::min<unsigned long long>((nn + 511) / 512, (unsigned long long)sms * 2), 512, 0, st>>>(
        counts, mask, nullptr, nn, S, gkeys, gcnt, capslots - 1);
    hist_compact_kernel<<<(unsigned)std::min<unsigned long long>((capslots + 255) / 256, (unsigned long long)sms * 8), 256, 0, st>>>(
        gkeys, gcnt, capslots, ka, va, d_m);
    hec_launch_counter::value += 2;
    unsigned long long m = 0;
    HEC_CUDA_OK(cudaMemcpyAsync(&m, d_m, sizeof m, cudaMemcpyDeviceToHost, st));
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    HEC_CUDA_OK(cudaGetLastError());
    *out_m = (size_t)m;
    if (cap < m) HEC_FAIL(HEC_ERR_CAPACITY, "cap is smaller than the number of distinct tuples");

    if (total_bits > 0 && m > 1) {
        const uint32_t nblocks = (uint32_t)((m + kTile - 1) / kTile);
        for (uint32_t shift = 0; shift < total_bits; shift += 8) {
            radix_hist_kernel<<<nblocks, kSortThreads, 0, st>>>(ka, m, shift, hist, nblocks);
            radix_scan_kernel<<<1, 1024, 0, st>>>(hist, (unsigned long long)256 * nblocks);
            radix_scatter_kernel<<<nblocks, kSortThreads, 0, st>>>(ka, va, kb, vb, m, shift, hist, nblocks);
            hec_launch_counter::value += 3;
            std::swap(ka, kb);
            std::swap(va, vb);
        }
    }
    hist_unpack_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(ka, va, m, S, out_tuples, reinterpret_cast<unsigned long long *>(out_mult));
    hec_launch_counter::value++;
    HEC_CUDA_OK(cudaGetLastError());
    HEC_CUDA_OK(cudaStreamSynchronize(st));
    return HEC_OK;
}
