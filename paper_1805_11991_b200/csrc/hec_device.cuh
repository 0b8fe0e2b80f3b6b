// Device-side parameter blocks shared by the kernels and their host launchers (not part of the ABI).
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

#include "hec_internal.h"

#define HEC_CUDA_OK(call)                                                                      \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess) {                                                              \
            hec_set_error(HEC_ERR_CUDA, std::string(#call ": ") + cudaGetErrorString(e__));    \
            return HEC_ERR_CUDA;                                                               \
        }                                                                                      \
    } while (0)

constexpr uint32_t HEC_LOG_ZERO = 0xFFFFFFFFu;   // embed table entry of the zero coefficient (device side)

// One field F_{q^k} as the count kernel sees it.
struct HecFieldDev {
    uint32_t M;          // q^k - 1
    uint32_t off;        // OFF = LMAX = M + PADL (even)
    uint32_t rcpM;       // floor(2^32 / M), for x mod M with one correction step
    uint32_t in_smem;    // 1: 16-bit table in the shared-memory blob at smem_off; 0: 32-bit table gtab
    uint32_t smem_off;   // byte offset inside the blob (16-byte aligned)
    uint32_t lane_cap;   // lanes with lane + 32u >= lane_cap use lane term 0 (they are masked out anyway)
    const uint32_t *gtab;   // extended table, 32-bit entries, global memory (L2-resident regime)
    const uint32_t *emb;    // q entries: log in F_{q^k} of the embedded coefficient, HEC_LOG_ZERO for 0
};

struct HecCountParams {
    const uint16_t *coeffs;        // [n][2g+3]
    uint32_t *out;                 // [n][g]
    unsigned long long n;
    uint32_t q;
    uint32_t blob_bytes;           // multiple of 16
    const uint4 *blob;             // concatenated shared-memory tables
    unsigned long long *err;       // err[0] = first row with a coefficient >= q, err[1] = first row of degree < 2g+1
    HecFieldDev f[HEC_MAX_GENUS];
};

struct HecSquarefreeParams {
    const uint16_t *coeffs;
    uint8_t *out;
    unsigned long long n;
    uint32_t p, q, M;              // M = q - 1
    uint32_t ncoef;                // 2g+3
    const uint32_t *zech;          // M entries, paper's convention (sentinel M)
    const uint32_t *emb;           // q entries: log in F_q or HEC_LOG_ZERO
};
