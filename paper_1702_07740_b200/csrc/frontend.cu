// The steps either side of the decoder, C ABI in include/qcldpc.h:
//   k_llr_init     Step 1 of Algorithm 1: Q_v = 2 R_v / sigma^2_{N_v} with the per-symbol noise variance of the d = 1
//                  scheme (reading G5: squared norm by default, the printed norm on request) or of the d = 2 scheme
//                  (from the printed a_i, b_i).  Elementwise, HBM-bound: 8 bytes read + 4 written per symbol.
//   k_pack_bits    hard decisions (one byte per bit) -> bits, most significant first (reading G8); 64-bit loads, one
//                  multiply per output byte.
//   k_crc32_check  CRC-32 (IEEE 802.3, reading G7) of the message part of each frame against the stored CRC field
//                  (Fig. 7; N_CRC = 32).  One CTA per frame: every thread takes a contiguous chunk
//                  (table-driven, table built in shared memory), the chunk remainders are moved to their place by a
//                  multiplication with x^(8 * bytes behind the chunk) mod P in GF(2)[x] and XOR-reduced.
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/qcldpc.h"

namespace {

constexpr int kFrontThreads = 256;
constexpr uint32_t kCrcPolyReflected = 0xEDB88320u;   // x^32 + x^26 + ... + 1 with bit 31 = x^0, bit 0 = x^31

// sigma^2_N of one symbol (DIM 1) from its X; IEEE division and plain products: no fused or approximate arithmetic, so
// that X = 0 gives an infinite variance and Q = +-0 exactly as the definition says
template <int POW>
__device__ __forceinline__ float noise_var_d1(float x, float s2) {
    const float nrm = fabsf(x);
    return __fdiv_rn(s2, POW == 1 ? nrm : __fmul_rn(nrm, nrm));
}
// sigma^2_N of a pair (DIM 2): (a^2 + b^2) sigma^2_Z
__device__ __forceinline__ float noise_var_d2(float x1, float x2, float s2) {
    const float den = __fadd_rn(__fmul_rn(x1, x1), __fmul_rn(x2, x2));
    const float a = __fdiv_rn(__fadd_rn(x1, x2), den);
    const float b = __fdiv_rn(__fsub_rn(x2, x1), den);
    return __fmul_rn(__fadd_rn(__fmul_rn(a, a), __fmul_rn(b, b)), s2);
}
__device__ __forceinline__ float llr_of(float r, float s2n) { return __fdiv_rn(__fmul_rn(2.0f, r), s2n); }

// One thread = VEC consecutive symbols of frame blockIdx.y (VEC = 4: float4 accesses, n % 4 == 0 and 16-byte aligned
// rows; VEC = 2: scalar accesses, any n; a pair never straddles two threads).
template <int DIM, int POW, int VEC>
__global__ void __launch_bounds__(kFrontThreads) k_llr_init(const float* __restrict__ r, const float* __restrict__ x,
                                                            const float* __restrict__ sigma2_z, int64_t n,
                                                            float* __restrict__ q) {
    const int f = blockIdx.y;
    const float s2 = sigma2_z[f];
    const int64_t i0 = ((int64_t)blockIdx.x * kFrontThreads + threadIdx.x) * VEC;
    if (i0 >= n) return;
    const int64_t o = (int64_t)f * n + i0;
    float rv[VEC], xv[VEC], qv[VEC];
    if (VEC == 4) {
        const float4 r4 = *reinterpret_cast<const float4*>(r + o);
        rv[0] = r4.x; rv[1] = r4.y; rv[2] = r4.z; rv[3] = r4.w;
        if (DIM > 0) {
            const float4 x4 = *reinterpret_cast<const float4*>(x + o);
            xv[0] = x4.x; xv[1] = x4.y; xv[2] = x4.z; xv[3] = x4.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < VEC; ++k) {
            const bool in = i0 + k < n;
            rv[k] = in ? r[o + k] : 0.0f;
            xv[k] = (DIM > 0 && in) ? x[o + k] : 1.0f;
        }
    }
#pragma unroll
    for (int k = 0; k < VEC; k += 2) {
        if (DIM == 2) {
            const float s2n = noise_var_d2(xv[k], xv[k + 1], s2);
            qv[k] = llr_of(rv[k], s2n);
            qv[k + 1] = llr_of(rv[k + 1], s2n);
        } else {
#pragma unroll
            for (int j = k; j < k + 2; ++j) qv[j] = llr_of(rv[j], DIM == 0 ? s2 : noise_var_d1<POW>(xv[j], s2));
        }
    }
    if (VEC == 4) {
        *reinterpret_cast<float4*>(q + o) = make_float4(qv[0], qv[1], qv[2], qv[3]);
    } else {
#pragma unroll
        for (int k = 0; k < VEC; ++k)
            if (i0 + k < n) q[o + k] = qv[k];
    }
}

// One thread = one output byte = bits 8j .. 8j+7 of frame blockIdx.y.  FAST: rows of `hard` are 8-byte aligned, one
// 64-bit load; bit b of the byte group (little-endian byte b of the word) goes to bit 7 - b of the result: after
// masking bit 0 of every byte, the multiplication by 0x8040201008040201 moves byte b's bit to position 63 - b (the
// partial products land on distinct bit positions, so nothing carries) and the top byte is the packed value.
template <bool FAST>
__global__ void __launch_bounds__(kFrontThreads) k_pack_bits(const uint8_t* __restrict__ hard, int64_t n, int64_t n_bits,
                                                             int64_t n_bytes, uint8_t* __restrict__ packed) {
    const int f = blockIdx.y;
    const int64_t j = (int64_t)blockIdx.x * kFrontThreads + threadIdx.x;
    if (j >= n_bytes) return;
    const uint8_t* src = hard + (int64_t)f * n + 8 * j;
    unsigned v;
    if (FAST && 8 * j + 8 <= n_bits) {
        const unsigned long long w = *reinterpret_cast<const unsigned long long*>(src);
        v = (unsigned)(((w & 0x0101010101010101ull) * 0x8040201008040201ull) >> 56);
    } else {
        v = 0;
#pragma unroll
        for (int b = 0; b < 8; ++b)
            if (8 * j + b < n_bits) v |= (unsigned)(src[b] & 1u) << (7 - b);
    }
    packed[(int64_t)f * n_bytes + j] = (uint8_t)v;
}

// a(x) b(x) mod P in GF(2)[x], bit 31 = x^0 ... bit 0 = x^31 (the register order of the reflected CRC)
__device__ __forceinline__ uint32_t gf2_mulmod(uint32_t a, uint32_t b) {
    uint32_t p = 0;
#pragma unroll 4
    for (int i = 0; i < 32; ++i) {
        if (a & (0x80000000u >> i)) p ^= b;                       // coefficient of x^i of a
        b = (b >> 1) ^ ((b & 1u) ? kCrcPolyReflected : 0u);       // b <- b x mod P
    }
    return p;
}
// x^(8 m) mod P
__device__ __forceinline__ uint32_t gf2_xpow8(unsigned long long m) {
    uint32_t res = 0x80000000u, base = 0x00800000u;               // 1 and x^8
    while (m) {
        if (m & 1ull) res = gf2_mulmod(res, base);
        base = gf2_mulmod(base, base);
        m >>= 1;
    }
    return res;
}

__global__ void __launch_bounds__(kFrontThreads) k_crc32_check(const uint8_t* __restrict__ packed, int64_t stride,
                                                               int64_t n_msg, uint32_t* __restrict__ crc_out,
                                                               uint8_t* __restrict__ ok_out) {
    __shared__ uint32_t s_tab[256];
    __shared__ uint32_t s_red[kFrontThreads / 32];
    const int tid = threadIdx.x;
    const uint8_t* row = packed + (int64_t)blockIdx.x * stride;
    {
        uint32_t c = (uint32_t)tid;
#pragma unroll
        for (int k = 0; k < 8; ++k) c = (c >> 1) ^ ((c & 1u) ? kCrcPolyReflected : 0u);
        s_tab[tid] = c;
    }
    __syncthreads();
    // thread t: bytes [t * chunk, min((t + 1) * chunk, n_msg)); remainder of chunk(x) x^32, then x^(8 * bytes behind it)
    const int64_t chunk = (n_msg + kFrontThreads - 1) / kFrontThreads;
    const int64_t beg = min((int64_t)tid * chunk, n_msg), end = min(beg + chunk, n_msg);
    uint32_t c = 0;
    for (int64_t k = beg; k < end; ++k) c = s_tab[(c ^ row[k]) & 0xffu] ^ (c >> 8);
    uint32_t part = (end > beg) ? gf2_mulmod(c, gf2_xpow8((unsigned long long)(n_msg - end))) : 0u;
    if (tid == 0) part ^= gf2_mulmod(0xFFFFFFFFu, gf2_xpow8((unsigned long long)n_msg));   // the initial value
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part ^= __shfl_xor_sync(0xffffffffu, part, o);
    if ((tid & 31) == 0) s_red[tid >> 5] = part;
    __syncthreads();
    if (tid == 0) {
        uint32_t total = 0;
#pragma unroll
        for (int w = 0; w < kFrontThreads / 32; ++w) total ^= s_red[w];
        const uint32_t crc = total ^ 0xFFFFFFFFu;                                        // final XOR
        const uint32_t stored = ((uint32_t)row[n_msg] << 24) | ((uint32_t)row[n_msg + 1] << 16) |
                                ((uint32_t)row[n_msg + 2] << 8) | (uint32_t)row[n_msg + 3];
        if (crc_out) crc_out[blockIdx.x] = crc;
        if (ok_out) ok_out[blockIdx.x] = (crc == stored) ? 1 : 0;
    }
}

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

template <int DIM, int POW>
cudaError_t launch_llr(const float* r, const float* x, const float* s2, int n_frames, int64_t n, float* q,
                       cudaStream_t st) {
    const bool vec = n % 4 == 0 && aligned(r, 16) && aligned(q, 16) && (DIM == 0 || aligned(x, 16));
    const int per = vec ? 4 : 2;
    const int64_t threads = (n + per - 1) / per;
    const dim3 grid((unsigned)((threads + kFrontThreads - 1) / kFrontThreads), (unsigned)n_frames);
    if (vec) k_llr_init<DIM, POW, 4><<<grid, kFrontThreads, 0, st>>>(r, x, s2, n, q);
    else k_llr_init<DIM, POW, 2><<<grid, kFrontThreads, 0, st>>>(r, x, s2, n, q);
    return cudaGetLastError();
}

}  // namespace

extern "C" {

int qcldpc_llr_init(const float* d_r, const float* d_x, const float* d_sigma2_z, int n_frames, int64_t n, int dim,
                    int norm_power, float* d_llr, void* stream) {
    if (!d_r || !d_sigma2_z || !d_llr || n_frames <= 0 || n_frames > QCLDPC_MAX_FRAMES || n <= 0)
        return QCLDPC_ERR_BAD_ARGUMENT;
    if (dim < 0 || dim > 2 || (dim > 0 && !d_x) || (dim == 1 && norm_power != 1 && norm_power != 2) ||
        (dim == 2 && n % 2))
        return QCLDPC_ERR_BAD_ARGUMENT;
    if ((n + 1) / 2 > (int64_t)0x7fffffff * kFrontThreads) return QCLDPC_ERR_UNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    if (dim == 0) e = launch_llr<0, 2>(d_r, d_x, d_sigma2_z, n_frames, n, d_llr, st);
    else if (dim == 2) e = launch_llr<2, 2>(d_r, d_x, d_sigma2_z, n_frames, n, d_llr, st);
    else if (norm_power == 1) e = launch_llr<1, 1>(d_r, d_x, d_sigma2_z, n_frames, n, d_llr, st);
    else e = launch_llr<1, 2>(d_r, d_x, d_sigma2_z, n_frames, n, d_llr, st);
    return e == cudaSuccess ? QCLDPC_OK : QCLDPC_ERR_CUDA;
}

int qcldpc_pack_bits(const uint8_t* d_hard, int n_frames, int64_t n, int64_t n_bits, uint8_t* d_packed, void* stream) {
    if (!d_hard || n_frames <= 0 || n_frames > QCLDPC_MAX_FRAMES || n <= 0 || n_bits < 0 || n_bits > n)
        return QCLDPC_ERR_BAD_ARGUMENT;
    const int64_t n_bytes = (n_bits + 7) / 8;
    if (n_bytes == 0) return QCLDPC_OK;                          // nothing to write: d_packed may be NULL
    if (!d_packed) return QCLDPC_ERR_BAD_ARGUMENT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const dim3 grid((unsigned)((n_bytes + kFrontThreads - 1) / kFrontThreads), (unsigned)n_frames);
    if (n % 8 == 0 && aligned(d_hard, 8)) k_pack_bits<true><<<grid, kFrontThreads, 0, st>>>(d_hard, n, n_bits, n_bytes, d_packed);
    else k_pack_bits<false><<<grid, kFrontThreads, 0, st>>>(d_hard, n, n_bits, n_bytes, d_packed);
    return cudaGetLastError() == cudaSuccess ? QCLDPC_OK : QCLDPC_ERR_CUDA;
}

int qcldpc_crc32_check(const uint8_t* d_packed, int n_frames, int64_t stride_bytes, int64_t k_bits, uint32_t* d_crc,
                       uint8_t* d_ok, void* stream) {
    if (!d_packed || (!d_crc && !d_ok) || n_frames <= 0 || k_bits < 32 || k_bits % 8 || stride_bytes < k_bits / 8)
        return QCLDPC_ERR_BAD_ARGUMENT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    k_crc32_check<<<(unsigned)n_frames, kFrontThreads, 0, st>>>(d_packed, stride_bytes, (k_bits - 32) / 8, d_crc, d_ok);
    return cudaGetLastError() == cudaSuccess ? QCLDPC_OK : QCLDPC_ERR_CUDA;
}

}  // extern "C"
