// hec_build_field_device: the tables of F_{q^k} built on the GPU (the "tables" column
// of the paper's Table 1, PAPER.md:303, 313-326 -- 13.5 s on the paper's CPU at p = 3001 -- becomes kernels).
// Same definitions as hec_field.cpp (readings G6, G7), different construction:
//   host   smallest primitive polynomial by ORDER TESTS (t^M = 1 and t^(M/l) != 1 for every prime l | M, M = Q - 1;
//          such a modulus is irreducible, because in a quotient by a reducible polynomial the order of t is below M
//          or divisible by p), instead of walking all Q - 1 powers per candidate;
//   device antilog[i] = t^i: thread tau starts at t^tau (square and multiply) and strides by the constant t^T,
//          writing antilog and its inverse permutation log (coalesced in i);
//          zech[i] = log[antilog[i] + 1] (add one to digit 0; log[0] = Q - 1 is the sentinel of table (3.2));
//   host   embedding of F_q: root rho of R_q by polynomial arithmetic, logs from the device-built table.
// Elements are integers sum a_i p^i, on the device as digit vectors of N = r k digits.
#include <cuda_runtime.h>

#include <algorithm>
#include <memory>
#include <numeric>
#include <vector>

#include "hec_internal.h"

cudaStream_t hec_current_stream();
int hec_ensure_device(int *sm_count, int *smem_optin);

namespace {

constexpr int kMaxDigits = 16;      // p >= 3 and Q <= 2^26  =>  n <= 16

struct FieldParams {
    uint32_t p, n, M, rcp_p;
    uint32_t negmod[kMaxDigits];    // -a_i mod p of the monic modulus t^n + sum a_i t^i
    uint32_t stride_elem[kMaxDigits];   // digits of t^T, T = number of threads of the antilog kernel
};

__host__ __device__ __forceinline__ uint32_t modp(uint32_t x, uint32_t p, uint32_t rcp) {
#ifdef __CUDA_ARCH__
    uint32_t r = x - __umulhi(x, rcp) * p;
#else
    uint32_t r = x - (uint32_t)(((uint64_t)x * rcp) >> 32) * p;
#endif
    if (r >= p) r -= p;
    if (r >= p) r -= p;
    return r;
}

// out = a * t mod P
template <int N>
__host__ __device__ __forceinline__ void mul_by_t(const FieldParams &fp, uint32_t (&a)[N]) {
    const uint32_t top = a[N - 1];
#pragma unroll
    for (int i = N - 1; i > 0; i--) a[i] = modp(a[i - 1] + top * fp.negmod[i], fp.p, fp.rcp_p);
    a[0] = modp(top * fp.negmod[0], fp.p, fp.rcp_p);
}

// out = a * b mod P: schoolbook product (digits < p < 2^16, so every partial sum of N products, each reduced, stays
// below 2^21), then the top coefficients are folded down with t^n = sum negmod[i] t^i.
template <int N>
__host__ __device__ __forceinline__ void mul(const FieldParams &fp, const uint32_t (&a)[N], const uint32_t (&b)[N], uint32_t (&out)[N]) {
    uint32_t prod[2 * N - 1];
#pragma unroll
    for (int s = 0; s < 2 * N - 1; s++) {
        uint32_t acc = 0;
#pragma unroll
        for (int i = 0; i < N; i++) {
            const int j = s - i;
            if (j >= 0 && j < N) acc += modp(a[i] * b[j], fp.p, fp.rcp_p);
        }
        prod[s] = modp(acc, fp.p, fp.rcp_p);
    }
#pragma unroll
    for (int s = 2 * N - 2; s >= N; s--) {
        const uint32_t c = prod[s];
#pragma unroll
        for (int i = 0; i < N; i++) prod[s - N + i] = modp(prod[s - N + i] + c * fp.negmod[i], fp.p, fp.rcp_p);
    }
#pragma unroll
    for (int i = 0; i < N; i++) out[i] = prod[i];
}

template <int N>
__host__ __device__ __forceinline__ void power_of_t(const FieldParams &fp, uint64_t e, uint32_t (&x)[N]) {
#pragma unroll
    for (int i = 0; i < N; i++) x[i] = 0;
    x[0] = 1;
    if (e == 0) return;
    int top = 63;
    while (!((e >> top) & 1ull)) top--;
    for (int bit = top; bit >= 0; bit--) {
        uint32_t sq[N];
        mul<N>(fp, x, x, sq);
#pragma unroll
        for (int i = 0; i < N; i++) x[i] = sq[i];
        if ((e >> bit) & 1ull) mul_by_t<N>(fp, x);
    }
}

template <int N>
__host__ __device__ __forceinline__ uint32_t encode(const FieldParams &fp, const uint32_t (&x)[N]) {
    uint32_t e = 0;
#pragma unroll
    for (int i = N - 1; i >= 0; i--) e = e * fp.p + x[i];
    return e;
}

// antilog[i] = t^i (encoding (3.1)), log = its inverse, log[0] = M.
template <int N>
__global__ void __launch_bounds__(256) antilog_kernel(const FieldParams fp, uint32_t *__restrict__ antilog, uint32_t *__restrict__ log) {
    const uint32_t T = gridDim.x * blockDim.x;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid == 0) log[0] = fp.M;
    if (tid >= fp.M) return;
    uint32_t x[N], step[N];
    power_of_t<N>(fp, tid, x);
#pragma unroll
    for (int i = 0; i < N; i++) step[i] = fp.stride_elem[i];
    for (uint32_t i = tid; i < fp.M; i += T) {
        const uint32_t e = encode<N>(fp, x);
        antilog[i] = e;
        log[e] = i;
        uint32_t nx[N];
        mul<N>(fp, x, step, nx);
#pragma unroll
        for (int j = 0; j < N; j++) x[j] = nx[j];
    }
}

// zech[i] = log(1 + alpha^i): table (3.2); the sentinel M = Q - 1 marks 1 + alpha^i = 0.
__global__ void __launch_bounds__(256) zech_kernel(uint32_t p, uint32_t M, const uint32_t *__restrict__ antilog,
                                                   const uint32_t *__restrict__ log, uint32_t *__restrict__ zech) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        const uint32_t e = antilog[i];
        const uint32_t d0 = e % p;
        const uint32_t e1 = d0 + 1 == p ? e - d0 : e + 1;
        zech[i] = log[e1];
    }
}

template <int N>
void launch_antilog(const FieldParams &fp, uint32_t grid, uint32_t *antilog, uint32_t *log, cudaStream_t st) {
    antilog_kernel<N><<<grid, 256, 0, st>>>(fp, antilog, log);
}

// ---------------------------------------------------------------------------------------- host arithmetic
// Runtime-n versions of the same operations (the searches below are O(n^2 log Q) per candidate).
struct HostRing {
    uint32_t p, n;
    std::vector<uint32_t> negmod;
    using El = std::vector<uint32_t>;
    El one() const { El e(n, 0); e[0] = 1; return e; }
    El mul(const El &a, const El &b) const {
        std::vector<uint64_t> prod(2 * n - 1, 0);
        for (uint32_t i = 0; i < n; i++)
            for (uint32_t j = 0; j < n; j++) prod[i + j] = (prod[i + j] + (uint64_t)a[i] * b[j]) % p;
        for (uint32_t s = 2 * n - 2; s >= n && s < 2 * n; s--) {
            const uint64_t c = prod[s];
            for (uint32_t i = 0; i < n; i++) prod[s - n + i] = (prod[s - n + i] + c * negmod[i]) % p;
        }
        El out(n);
        for (uint32_t i = 0; i < n; i++) out[i] = (uint32_t)prod[i];
        return out;
    }
    El pow(El base, uint64_t e) const {
        El acc = one();
        while (e) {
            if (e & 1) acc = mul(acc, base);
            base = mul(base, base);
            e >>= 1;
        }
        return acc;
    }
    El t() const {
        if (n == 1) return El{negmod[0] % p};
        El e(n, 0); e[1] = 1; return e;
    }
    bool is_one(const El &a) const {
        if (a[0] != 1) return false;
        for (uint32_t i = 1; i < n; i++) if (a[i]) return false;
        return true;
    }
    uint32_t encode(const El &a) const { uint32_t e = 0; for (uint32_t i = n; i-- > 0;) e = e * p + a[i]; return e; }
};

std::vector<uint32_t> prime_factors(uint32_t m) {
    std::vector<uint32_t> f;
    for (uint32_t d = 2; (uint64_t)d * d <= m; d++)
        if (m % d == 0) { f.push_back(d); while (m % d == 0) m /= d; }
    if (m > 1) f.push_back(m);
    return f;
}

}  // namespace

// Device build of the field; same result as the host build (hec_field.cpp), bit for bit.
hec_field *hec_build_field_device_impl(uint32_t p, uint32_t r, uint32_t k, uint32_t skip) {
    if (p < 3 || p % 2 == 0) { hec_set_error(HEC_ERR_INVALID_FIELD, "p must be an odd prime"); return nullptr; }
    for (uint32_t d = 3; (uint64_t)d * d <= p; d += 2)
        if (p % d == 0) { hec_set_error(HEC_ERR_INVALID_FIELD, "p must be an odd prime"); return nullptr; }
    if (r < 1 || k < 1) { hec_set_error(HEC_ERR_INVALID_FIELD, "r and k must be >= 1"); return nullptr; }
    if (p >= 65536) { hec_set_error(HEC_ERR_INVALID_FIELD, "hec_build_field_device needs p < 65536"); return nullptr; }
    uint64_t q64 = 1, Q64 = 1;
    for (uint32_t i = 0; i < r && q64 <= HEC_MAX_FIELD_SIZE; i++) q64 *= p;
    for (uint32_t i = 0; i < r * k && Q64 <= HEC_MAX_FIELD_SIZE; i++) Q64 *= p;
    if (q64 > HEC_MAX_FIELD_SIZE || Q64 > HEC_MAX_FIELD_SIZE) {
        hec_set_error(HEC_ERR_INVALID_FIELD, "q^k exceeds HEC_MAX_FIELD_SIZE (2^26)");
        return nullptr;
    }
    int sms = 0, smem = 0;
    if (hec_ensure_device(&sms, &smem) != HEC_OK) return nullptr;

    std::unique_ptr<hec_field> F(new hec_field);
    F->p = p; F->r = r; F->k = k; F->n = r * k;
    F->q = (uint32_t)q64; F->Q = (uint32_t)Q64;
    const uint32_t n = F->n, Q = F->Q, M = Q - 1;

    // ---- smallest primitive polynomial (reading G7: order the tuple (a_{n-1}, .., a_0), i.e. count e upwards)
    const std::vector<uint32_t> ell = prime_factors(M);
    HostRing R{p, n, std::vector<uint32_t>(n, 0)};
    bool found = false;
    uint32_t seen = 0;
    std::vector<uint32_t> modulus(n + 1, 0);
    for (uint32_t e = 1; e < Q && !found; e++) {
        uint32_t v = e;
        for (uint32_t i = 0; i < n; i++) { modulus[i] = v % p; v /= p; }
        modulus[n] = 1;
        if (modulus[0] == 0) continue;
        for (uint32_t i = 0; i < n; i++) R.negmod[i] = (p - modulus[i]) % p;
        const HostRing::El t = R.t();
        if (!R.is_one(R.pow(t, M))) continue;
        bool prim = true;
        for (uint32_t l : ell)
            if (R.is_one(R.pow(t, M / l))) { prim = false; break; }
        found = prim;
        if (found && seen < skip) { seen++; found = false; }
    }
    if (!found) {
        if (skip) hec_set_error(HEC_ERR_INVALID_FIELD, "hec_set_field_variant: variant " + std::to_string(skip) + " exceeds the number of primitive polynomials of this field (" + std::to_string(seen) + " of that degree)");
        else hec_set_error(HEC_ERR_INVALID_FIELD, "no primitive polynomial found");
        return nullptr;
    }
    F->modulus = modulus;

    // ---- device tables
    cudaStream_t st = hec_current_stream();
    const uint32_t threads_wanted = std::min<uint32_t>(M, (uint32_t)sms * 2048u);
    const uint32_t grid = (threads_wanted + 255u) / 256u;
    const uint32_t T = grid * 256u;
    FieldParams fp{};
    fp.p = p; fp.n = n; fp.M = M; fp.rcp_p = (uint32_t)((1ull << 32) / p);
    for (uint32_t i = 0; i < n; i++) fp.negmod[i] = R.negmod[i];
    {
        const HostRing::El s = R.pow(R.t(), T % M);
        for (uint32_t i = 0; i < n; i++) fp.stride_elem[i] = s[i];
    }
    uint32_t *d_buf = nullptr;
    const size_t words = (size_t)M + Q + M;
    if (cudaMalloc(&d_buf, words * sizeof(uint32_t)) != cudaSuccess) {
        cudaGetLastError();
        hec_set_error(HEC_ERR_CUDA, "hec_build_field_device: cudaMalloc failed");
        return nullptr;
    }
    uint32_t *d_antilog = d_buf, *d_log = d_buf + M, *d_zech = d_log + Q;
    switch (n) {
#define HEC_CASE(N) case N: launch_antilog<N>(fp, grid, d_antilog, d_log, st); break;
        HEC_CASE(1) HEC_CASE(2) HEC_CASE(3) HEC_CASE(4) HEC_CASE(5) HEC_CASE(6) HEC_CASE(7) HEC_CASE(8)
        HEC_CASE(9) HEC_CASE(10) HEC_CASE(11) HEC_CASE(12) HEC_CASE(13) HEC_CASE(14) HEC_CASE(15) HEC_CASE(16)
#undef HEC_CASE
        default:
            cudaFree(d_buf);
            hec_set_error(HEC_ERR_INVALID_FIELD, "extension degree above 16");
            return nullptr;
    }
    hec_launch_counter::value++;
    zech_kernel<<<std::min<uint32_t>((M + 255u) / 256u, (uint32_t)sms * 8u), 256, 0, st>>>(p, M, d_antilog, d_log, d_zech);
    hec_launch_counter::value++;
    F->antilog.resize(M); F->log.resize(Q); F->zech.resize(M);
    cudaError_t ce = cudaMemcpyAsync(F->antilog.data(), d_antilog, (size_t)M * 4, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(F->log.data(), d_log, (size_t)Q * 4, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(F->zech.data(), d_zech, (size_t)M * 4, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    cudaFree(d_buf);
    if (ce != cudaSuccess) {
        cudaGetLastError();
        hec_set_error(HEC_ERR_CUDA, std::string("hec_build_field_device: ") + cudaGetErrorString(ce));
        return nullptr;
    }

    // ---- embedding of F_q (reading G6): rho = alpha^(s M/(q-1)) with R_q(rho) = 0, s the smallest such unit
    F->embed.assign(F->q, M);
    F->embed_unit = 1;
    if (r == 1 || k == 1) {
        for (uint32_t c = 1; c < F->q; c++) F->embed[c] = F->log[c];
    } else {
        const hec_field *Fq = hec_cached_field(p, r, 1);
        if (!Fq) return nullptr;
        const std::vector<uint32_t> &Rq = Fq->modulus;
        const uint32_t Mq = F->q - 1, step = M / Mq;
        const HostRing::El beta = R.pow(R.t(), step);
        HostRing::El rho;
        bool ok = false;
        for (uint32_t s = 1; s < Mq && !ok; s++) {
            if (std::gcd(s, Mq) != 1) continue;
            const HostRing::El cand = R.pow(beta, s);
            HostRing::El acc(n, 0), pw = R.one();
            for (uint32_t i = 0; i <= r; i++) {
                for (uint32_t j = 0; j < n; j++) acc[j] = (uint32_t)((acc[j] + (uint64_t)pw[j] * Rq[i]) % p);
                pw = R.mul(pw, cand);
            }
            if (std::all_of(acc.begin(), acc.end(), [](uint32_t v) { return v == 0; })) { rho = cand; F->embed_unit = s; ok = true; }
        }
        if (!ok) { hec_set_error(HEC_ERR_INVALID_FIELD, "no root of R_q found in F_{q^k}"); return nullptr; }
        std::vector<HostRing::El> rho_pw(r);
        rho_pw[0] = R.one();
        for (uint32_t i = 1; i < r; i++) rho_pw[i] = R.mul(rho_pw[i - 1], rho);
        for (uint32_t c = 1; c < F->q; c++) {
            HostRing::El acc(n, 0);
            uint32_t v = c;
            for (uint32_t i = 0; i < r; i++) {
                const uint32_t a = v % p; v /= p;
                for (uint32_t j = 0; j < n; j++) acc[j] = (uint32_t)((acc[j] + (uint64_t)rho_pw[i][j] * a) % p);
            }
            F->embed[c] = F->log[R.encode(acc)];
        }
    }
    return F.release();
}

extern "C" hec_field *hec_build_field_device(uint32_t p, uint32_t r, uint32_t k) { return hec_build_field_device_impl(p, r, k, 0); }
