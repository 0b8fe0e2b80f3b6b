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

// How the Zech table of one field is stored for the count kernel.
enum HecTableMode : uint32_t {
    HEC_TAB_GLOBAL32 = 0,   // extended table, 32-bit entries, global memory (L1/L2-resident regime)
    HEC_TAB_EXT16 = 1,      // extended table, 16-bit entries, shared memory
    HEC_TAB_HALF32 = 2,     // half table (Z(-n) = Z(n) - n), 32-bit entries, shared memory
    HEC_TAB_HALF24 = 3,     // half table, 16-bit low plane + signed 8-bit high plane, shared memory
    // tables of the radix-R evaluation (hec_radix.cuh): entries serve the pair (Z[n], Z[n + M/2])
    HEC_TAB_PAIR16 = 4,     // M 32-bit entries (Z[n] | Z[n + M/2] << 16), shared memory, M <= 32768
    HEC_TAB_RHALF32 = 5,    // Z[0 .. M/2], 32-bit entries, shared memory
    HEC_TAB_RHALF17 = 6,    // Z[0 .. M/2]: 16-bit plane + byte plane with bit 16 of entries i and M/2 - i, shared memory, M < 2^17
    HEC_TAB_GPAIR64 = 7,    // M entries (Z[n], Z[n + M/2]) as two 32-bit words, global memory (L1/L2-resident regime)
    HEC_TAB_SPAIR16 = 8     // PAIR16's entries for 32768 < M < 65536 (values still fit 16 bits): one coset per lane, 32-bit arithmetic
};

// One field F_{q^k} as the count kernel sees it.
struct HecFieldDev {
    uint32_t M;          // q^k - 1
    uint32_t mode;       // HecTableMode
    uint32_t z0;         // extended tables: Z0 = M + LP, the stored value of the zero element (LP = M + PADL)
    uint32_t rcpM;       // floor(2^32 / M), for x mod M with one correction step
    uint32_t smem_off;   // byte offset inside the launch's blob (16-byte aligned): table / low plane
    uint32_t smem_off2;  // HALF24: byte offset of the high plane
    uint32_t lane_cap;   // lanes with lane + 32u >= lane_cap use lane term 0 (they are masked out anyway)
    uint32_t radix;      // radix evaluation: R in {2, 4, 8}, the largest with R | M; 0 for the Horner tables
    uint32_t fast_off;   // PAIR16: byte offset inside the blob of the field's fast tables (hec_radix.cuh: radix_fast_x), 0: none
    uint32_t fast_row;   // bytes per row of the transposed Zech table inside them
    uint32_t pt_off;     // RHALF32 top field with monomial classes (hec_radix.cuh: radix_mono8_x): byte offset of the packed
                         // parity table (2 bits per n: parity of Z[n], of Z[n + M/2]; four entries per byte), 0: none
    const uint32_t *orb[3]; // HEC_EVAL_ORBIT: Frobenius-orbit representatives of the cosets of mu_R, R = 2, 4, 8 (hec_radix.cuh)
    uint32_t n_orb[3];
    uint32_t mono_r;        // half-table top field with a parity table: 8 or 16 if dense rows run radix_mono_x at that radix, else 0
    uint32_t orb_fast;      // HEC_EVAL_ORBIT: the field may run radix_orbit_fast_x (PAIR16 and hec_set_fast_tables on)
    const uint32_t *gtab;   // GLOBAL32: extended table in global memory; GPAIR64: the pair table
    const uint32_t *emb;    // q entries: log in F_{q^k} of the embedded coefficient, HEC_LOG_ZERO for 0
};

struct HecCountParams {
    const uint16_t *coeffs;        // [n][2g+3]
    uint32_t *out;                 // [n][g]
    unsigned long long n;
    uint32_t q;
    uint32_t blob_bytes;           // multiple of 16
    const uint4 *blob;             // this launch's concatenated shared-memory tables
    unsigned long long *err;       // err[0] = first row with a coefficient >= q, err[1] = first row of degree < 2g+1
    uint32_t k_lo, k_hi;           // this launch computes N_k for k_lo <= k <= k_hi; only field k_hi may differ from the
                                   // launch's base layout (EXT16 for the Horner kernel, PAIR16 for the radix kernel)
    uint32_t scratch_off;          // radix kernel: byte offset (after the blob) of the per-warp scratch words
    uint32_t *out_r0;              // [n][g] or NULL: r0_k = #{x in F_{q^k}: f(x) = 0}, the input of lambda
    uint32_t splits;               // radix kernel: warps per curve (>= 1); > 1: out is pre-zeroed and accumulated with atomics
    unsigned long long row0;       // index of this launch's first row in the caller's batch (error reporting)
    HecFieldDev f[HEC_MAX_GENUS];
};

// hec_shift_kernel (hec_count.cu): rows whose residue classes mod R are not all non-empty are replaced by f(X + t).
struct HecShiftParams {
    const uint16_t *coeffs;        // [n][ncoef]
    uint16_t *out;                 // [n][ncoef]
    unsigned long long n;
    uint32_t q, M;                 // M = q - 1
    uint32_t ncoef;                // 2g+3
    uint32_t R;                    // target radix (4 or 8)
    uint32_t dense;                // 1: a row qualifies only if EVERY coefficient up to its degree is nonzero (monomial classes)
    const uint32_t *zech;          // F_q: M entries, paper's convention (sentinel M)
    const uint32_t *emb;           // q entries: log in F_q or HEC_LOG_ZERO
    const uint32_t *antilog;       // M entries: alpha^i in the integer encoding
};

struct HecSquarefreeParams {
    const uint16_t *coeffs;
    uint8_t *out;
    unsigned long long n;
    uint32_t p, q, M;              // M = q - 1
    uint32_t ncoef;                // 2g+3
    const uint32_t *zech;          // M entries, paper's convention (sentinel M)
    const uint32_t *emb;           // q entries: log in F_q or HEC_LOG_ZERO
    // lambda(f) (Algorithm 1 line 18), all NULL / 0 when not requested
    const uint32_t *roots;         // [n][g] r0_k from the count kernel
    uint8_t *out_lambda;           // [n] index of the partition, 0xFF when f is not squarefree
    const unsigned long long *part_codes;   // n_parts packed multiplicity vectors (4 bits per part size), index order
    uint32_t n_parts, g;
};
