// Internal declarations shared by the translation units of libhec (not part of the ABI).
#pragma once

#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "hec.h"

// ---------------------------------------------------------------------------- errors
void hec_set_error(int code, const std::string &msg, size_t index = (size_t)-1);
#define HEC_FAIL(code, msg) do { hec_set_error((code), (msg)); return (code); } while (0)

// ---------------------------------------------------------------------------- fields (host)
// Paper's conventions: logs in [0, Q-2]; the zero element / "1 + alpha^i = 0" is Q-1.
struct hec_field {
    uint32_t p = 0, r = 0, k = 0, n = 0;   // n = r*k
    uint32_t q = 0, Q = 0;                  // base field size p^r, field size q^k
    uint32_t embed_unit = 1;                // s of hec.h
    std::vector<uint32_t> modulus;          // n+1 coefficients, monic
    std::vector<uint32_t> antilog;          // Q-1
    std::vector<uint32_t> log;              // Q
    std::vector<uint32_t> zech;             // Q-1
    std::vector<uint32_t> embed;            // q
};

// q = p^r with p an odd prime?  (q < 65536)
bool hec_factor_q(uint32_t q, uint32_t *p, uint32_t *r);
// Cached, library-owned fields used by hec_count (never freed before hec_shutdown).
const hec_field *hec_cached_field(uint32_t p, uint32_t r, uint32_t k);
void hec_clear_field_cache();
// Tables built on the device (hec_field_device.cu); same result as the host build.
hec_field *hec_build_field_device_impl(uint32_t p, uint32_t r, uint32_t k, uint32_t skip = 0);
// hec_set_field_variant: the library's own fields take the (v+1)-th smallest primitive polynomial (hec.h)
void hec_set_field_variant_impl(uint32_t v);
// hec_cached_field builds fields above this size on the device once hec_count has initialised one.
constexpr uint32_t kDeviceBuildMinQ = 1u << 16;
void hec_allow_device_field_build(bool on);

// ---------------------------------------------------------------------------- device side
// Geometry of one extended Zech table.  Stored value of a lookup result:
//   Z(n) in [0, M)   the log of 1 + alpha^n
//   Z0 = M + LP      the element is zero (1 + alpha^n = 0), LP = M + PADL
// Index space: idx = stored value + L, L in [0, LP).
//   idx in [0, M + LP)       -> stored Zech of idx mod M
//   idx in [Z0, Z0 + LP)     -> 0   (accumulator was zero: acc*x^m + c = c, i.e. W = log 1 = 0)
struct hec_table_geom {
    uint32_t M;        // Q - 1
    uint32_t padl;     // largest lane term m * (32 U - 1) + 1, rounded up to even
    uint32_t lmax;     // LP = M + padl
    uint32_t entries;  // 2 * lmax + M
};

std::vector<std::vector<uint8_t>> hec_partitions_of(uint32_t total);

struct hec_launch_counter { static uint64_t value; };
