// hec_gather_bench: random-access lookup ceilings.  The count kernel's inner step is
// "idx <- table[idx] + (uniform + lane term)" (hec_count.cu); this micro-benchmark runs exactly that dependent
// chain on a table of uniformly random entries, from shared memory, through L1, or from L2 only, so that
// the achieved lookup rate of the real kernel can be quoted against a MEASURED ceiling at equal footprint
// and entry width (the shared-memory figure also has a closed form: 32 banks / E[max bank load]).
#include <algorithm>
#include <vector>

#include "hec_device.cuh"

cudaStream_t hec_current_stream();
int hec_ensure_device(int *sm_count, int *smem_optin);

namespace {

template <typename T, int WHERE>
__device__ __forceinline__ uint32_t gather_load(const T *t, uint32_t idx) {
    if constexpr (WHERE == 2) {
        return (uint32_t)__ldcg(t + idx);
    } else if constexpr (WHERE == 1) {
        return (uint32_t)__ldg(t + idx);
    } else {
        return (uint32_t)t[idx];
    }
}

template <typename T, int WHERE, int U>
__global__ void __launch_bounds__(1024) gather_kernel(const T *table, uint32_t entries, uint32_t maxval, uint32_t steps, uint32_t *sink) {
    extern __shared__ uint4 gsm[];
    const T *tab = table;
    if constexpr (WHERE == 0) {
        const uint32_t n16 = (uint32_t)(((size_t)entries * sizeof(T) + 15) / 16);
        const uint4 *src = reinterpret_cast<const uint4 *>(table);
        for (uint32_t i = threadIdx.x; i < n16; i += blockDim.x) gsm[i] = src[i];
        __syncthreads();
        tab = reinterpret_cast<const T *>(gsm);
    }
    const uint32_t lane = threadIdx.x & 31u;
    uint32_t v[U], l[U];
#pragma unroll
    for (int u = 0; u < U; u++) { l[u] = lane + 32u * u; v[u] = (threadIdx.x * 2654435761u + blockIdx.x * 40503u + u * 977u) % maxval; }
    // like the count kernel: index = looked-up value + warp-uniform offset + lane term
    const uint32_t lim = entries - 256u - maxval + 1u;
    uint32_t ub = 0;
    for (uint32_t s = 0; s < steps; s++) {
#pragma unroll
        for (int u = 0; u < U; u++) v[u] = gather_load<T, WHERE>(tab, v[u] + ub + l[u]);
        ub += 7919u;
        if (ub >= lim) ub %= lim;
    }
    uint32_t acc = 0;
#pragma unroll
    for (int u = 0; u < U; u++) acc ^= v[u];
    if (acc == 0xFFFFFFFFu) sink[0] = acc;       // never true: values are < entries
}

template <typename T, int WHERE>
int run_gather(const T *d_table, uint32_t entries, uint32_t maxval, uint32_t block, uint32_t grid, uint32_t chains, uint32_t steps,
               size_t smem, uint32_t *d_sink, cudaStream_t st) {
    auto launch = [&](auto kern) -> int {
        if (smem) HEC_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<grid, block, smem, st>>>(d_table, entries, maxval, steps, d_sink);
        hec_launch_counter::value++;
        HEC_CUDA_OK(cudaGetLastError());
        return HEC_OK;
    };
    switch (chains) {
        case 1: return launch(gather_kernel<T, WHERE, 1>);
        case 2: return launch(gather_kernel<T, WHERE, 2>);
        case 4: return launch(gather_kernel<T, WHERE, 4>);
        case 8: return launch(gather_kernel<T, WHERE, 8>);
        default: HEC_FAIL(HEC_ERR_INVALID_ARG, "chains must be 1, 2, 4 or 8");
    }
}

template <typename T>
int gather_typed(int where, uint32_t entries, uint32_t block, uint32_t ctas_per_sm, uint32_t chains, uint32_t steps,
                 double *out_rate, float *out_ms) {
    int sms = 0, optin = 0;
    int rc = hec_ensure_device(&sms, &optin);
    if (rc) return rc;
    cudaStream_t st = hec_current_stream();
    // seeded table: values uniform in [0, maxval) so that value + uniform offset + lane term stays in range
    const uint32_t maxval = (uint32_t)std::min<uint64_t>(entries - 256u, sizeof(T) == 2 ? 65536u : 0xFFFFFFFFu);
    std::vector<T> host(entries);
    uint64_t s = 0x1805119900000000ull + entries;
    for (uint32_t i = 0; i < entries; i++) {
        s += 0x9E3779B97F4A7C15ull;
        uint64_t z = s;
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        z ^= z >> 31;
        host[i] = (T)(((z >> 32) * (uint64_t)maxval) >> 32);
    }
    const size_t bytes = ((size_t)entries * sizeof(T) + 15) & ~(size_t)15;
    size_t smem = 0;
    if (where == 0) {
        smem = bytes;
        if (smem * ctas_per_sm > (size_t)optin) HEC_FAIL(HEC_ERR_INVALID_ARG, "table does not fit shared memory");
    }
    T *d_table = nullptr;
    uint32_t *d_sink = nullptr;
    HEC_CUDA_OK(cudaMalloc((void **)&d_table, bytes));
    HEC_CUDA_OK(cudaMalloc((void **)&d_sink, 16));
    HEC_CUDA_OK(cudaMemcpy(d_table, host.data(), (size_t)entries * sizeof(T), cudaMemcpyHostToDevice));
    const uint32_t grid = (uint32_t)sms * ctas_per_sm;
    cudaEvent_t e0, e1;
    HEC_CUDA_OK(cudaEventCreate(&e0));
    HEC_CUDA_OK(cudaEventCreate(&e1));
    for (int rep = 0; rep < 2 && rc == HEC_OK; rep++) {         // rep 0 warms up
        HEC_CUDA_OK(cudaEventRecord(e0, st));
        if (where == 0) rc = run_gather<T, 0>(d_table, entries, maxval, block, grid, chains, steps, smem, d_sink, st);
        else if (where == 1) rc = run_gather<T, 1>(d_table, entries, maxval, block, grid, chains, steps, 0, d_sink, st);
        else rc = run_gather<T, 2>(d_table, entries, maxval, block, grid, chains, steps, 0, d_sink, st);
        HEC_CUDA_OK(cudaEventRecord(e1, st));
        HEC_CUDA_OK(cudaStreamSynchronize(st));
    }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_table);
    cudaFree(d_sink);
    if (rc) return rc;
    if (out_ms) *out_ms = ms;
    if (out_rate) *out_rate = (double)grid * block * chains * steps / (ms * 1e-3);
    return HEC_OK;
}

}  // namespace

extern "C" int hec_gather_bench(int where, uint32_t entries, uint32_t entry_bytes, uint32_t block, uint32_t ctas_per_sm,
                                uint32_t chains, uint32_t lookups_per_lane, double *out_lookups_per_s, float *out_ms) {
    if (where < 0 || where > 2) HEC_FAIL(HEC_ERR_INVALID_ARG, "where must be 0 (shared), 1 (L1) or 2 (L2)");
    if (entries < 512) HEC_FAIL(HEC_ERR_INVALID_ARG, "entries must be >= 512");
    if (block < 32 || block > 1024 || block % 32) HEC_FAIL(HEC_ERR_INVALID_ARG, "block must be a multiple of 32 in [32, 1024]");
    if (ctas_per_sm < 1 || ctas_per_sm > 32) HEC_FAIL(HEC_ERR_INVALID_ARG, "ctas_per_sm must be in [1, 32]");
    if (entry_bytes == 2) {
        return gather_typed<uint16_t>(where, entries, block, ctas_per_sm, chains, lookups_per_lane, out_lookups_per_s, out_ms);
    }
    if (entry_bytes == 4)
        return gather_typed<uint32_t>(where, entries, block, ctas_per_sm, chains, lookups_per_lane, out_lookups_per_s, out_ms);
    HEC_FAIL(HEC_ERR_INVALID_ARG, "entry_bytes must be 2 or 4");
}
