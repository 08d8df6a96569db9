// Block floating-point codec of the paper's compressed ghost exchange (Fig. 3) for sm_100a.
// "Each GPU thread encodes or decodes a four-value block": four FP32 values <-> one N_bits = 4 n_bits bit word whose low 8
// bits hold the shared biased exponent and whose remaining bits hold four v_bits = n_bits - 2 bit two's-complement
// coefficients (q_0 lowest).  n_bits = 16: one 64-bit store per block; 12: three 16-bit stores; 10: five 8-bit stores
// ("no storage word is straddled by two blocks, and encoding requires no atomics").
// Own implementation: exponent from the FP32 bit pattern, scaling by an exactly constructed power of two in FP64,
// cvt.rni for round-to-nearest-even (readings B1-B5).  HBM-bound: 16 B in, n_bits/2 B out per block.
#include <cstdint>

#include "chfsi_internal.h"

namespace chfsi {

__device__ __forceinline__ double pow2d(int e) {           // 2^e, exact, -1022 <= e <= 1023
    return __longlong_as_double((long long)(e + 1023) << 52);
}

// one block: x[0..3] -> word
template <int NBITS>
__device__ __forceinline__ unsigned long long bfp_encode_block(float x0, float x1, float x2, float x3) {
    constexpr int V = NBITS - 2;
    const unsigned m0 = __float_as_uint(x0) & 0x7fffffffu, m1 = __float_as_uint(x1) & 0x7fffffffu;
    const unsigned m2 = __float_as_uint(x2) & 0x7fffffffu, m3 = __float_as_uint(x3) & 0x7fffffffu;
    const unsigned mx = max(max(m0, m1), max(m2, m3));      // the bit pattern of max |x_i| (ordering of finite FP32 = ordering of bits)
    if (mx == 0u) return 0ull;                              // all-zero block: zero exponent field
    // 2^(e_max-1) <= max|x| < 2^e_max  <=>  e_max = E - 126 for the biased exponent field E >= 1; subnormal maxima (E = 0) are
    // clamped to e_max = -126 (reading B3), which is E - 126 + 1, i.e. the stored exponent is max(E, 0) + 1 either way
    const int E = (int)(mx >> 23);
    const int e = E + 1;                                    // stored biased exponent e = e_max + 127, 1..255
    const int emax = e - 127;
    const double sc = pow2d(V - 1 - emax);                  // |exponent| <= 139: exact in FP64
    constexpr int HI = (1 << (V - 1)) - 1;
    int q0 = __double2int_rn((double)x0 * sc), q1 = __double2int_rn((double)x1 * sc);
    int q2 = __double2int_rn((double)x2 * sc), q3 = __double2int_rn((double)x3 * sc);
    q0 = min(q0, HI); q1 = min(q1, HI); q2 = min(q2, HI); q3 = min(q3, HI);   // "only the upper bound requires clamping"
    constexpr unsigned long long MASK = (1ull << V) - 1ull;
    return (unsigned long long)e | (((unsigned long long)q0 & MASK) << 8) | (((unsigned long long)q1 & MASK) << (8 + V)) |
           (((unsigned long long)q2 & MASK) << (8 + 2 * V)) | (((unsigned long long)q3 & MASK) << (8 + 3 * V));
}

template <int NBITS>
__device__ __forceinline__ void bfp_store_block(unsigned char* dst, long long b, unsigned long long w) {
    if (NBITS == 16) {
        reinterpret_cast<unsigned long long*>(dst)[b] = w;
    } else if (NBITS == 12) {
        unsigned short* p = reinterpret_cast<unsigned short*>(dst) + 3 * b;
        p[0] = (unsigned short)w; p[1] = (unsigned short)(w >> 16); p[2] = (unsigned short)(w >> 32);
    } else {
        unsigned char* p = dst + 5 * b;
        p[0] = (unsigned char)w; p[1] = (unsigned char)(w >> 8); p[2] = (unsigned char)(w >> 16);
        p[3] = (unsigned char)(w >> 24); p[4] = (unsigned char)(w >> 32);
    }
}

template <int NBITS>
__device__ __forceinline__ unsigned long long bfp_load_block(const unsigned char* src, long long b) {
    if (NBITS == 16) return reinterpret_cast<const unsigned long long*>(src)[b];
    if (NBITS == 12) {
        const unsigned short* p = reinterpret_cast<const unsigned short*>(src) + 3 * b;
        return (unsigned long long)p[0] | ((unsigned long long)p[1] << 16) | ((unsigned long long)p[2] << 32);
    }
    const unsigned char* p = src + 5 * b;
    return (unsigned long long)p[0] | ((unsigned long long)p[1] << 8) | ((unsigned long long)p[2] << 16) |
           ((unsigned long long)p[3] << 24) | ((unsigned long long)p[4] << 32);
}

template <int NBITS>
__device__ __forceinline__ void bfp_decode_block(unsigned long long w, float (&x)[4]) {
    constexpr int V = NBITS - 2;
    const int e = (int)(w & 0xffull);
    if (e == 0) { x[0] = x[1] = x[2] = x[3] = 0.0f; return; }
    const double sc = pow2d(e - 127 - V + 1);               // x~_i = q_i 2^(e_max - v_bits + 1), exact
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const unsigned uq = (unsigned)((w >> (8 + i * V)) & ((1ull << V) - 1ull));
        const int q = (int)(uq << (32 - V)) >> (32 - V);    // restore the dropped copies of the sign bit
        x[i] = (float)((double)q * sc);                     // exact: |q| <= 2^13 and the result is a FP32 number (maybe subnormal)
    }
}

template <int NBITS>
__global__ void __launch_bounds__(256) bfp_encode_kernel(const float4* __restrict__ src, long long nblocks, unsigned char* __restrict__ dst) {
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < nblocks; b += (long long)gridDim.x * blockDim.x) {
        const float4 v = __ldcs(src + b);
        bfp_store_block<NBITS>(dst, b, bfp_encode_block<NBITS>(v.x, v.y, v.z, v.w));
    }
}

template <int NBITS>
__global__ void __launch_bounds__(256) bfp_decode_kernel(const unsigned char* __restrict__ src, long long nblocks, float4* __restrict__ dst) {
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < nblocks; b += (long long)gridDim.x * blockDim.x) {
        float x[4];
        bfp_decode_block<NBITS>(bfp_load_block<NBITS>(src, b), x);
        __stcs(dst + b, make_float4(x[0], x[1], x[2], x[3]));
    }
}

// Ghost update, send side: gather the listed (node, spin) rows of a multivector and encode in the same pass.
// Message value index ((r nvec + v) 2 + ri); one block = the complex values v, v+1 of one row (nvec even).
template <int NBITS, typename T>
__global__ void __launch_bounds__(256) bfp_gather_encode_kernel(const T* __restrict__ X, long long ld, int nvec,
                                                                const long long* __restrict__ rows, long long nrows,
                                                                unsigned char* __restrict__ dst) {
    const int bpr = nvec / 2;                               // blocks per row
    const long long nblocks = nrows * bpr;
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < nblocks; b += (long long)gridDim.x * blockDim.x) {
        const long long r = b / bpr;
        const int v = 2 * (int)(b - r * bpr);
        const T* p = X + (__ldg(rows + r) * ld + v) * 2;
        float x0, x1, x2, x3;
        if (sizeof(T) == 8) {
            const double2 a = *reinterpret_cast<const double2*>(p), c = *reinterpret_cast<const double2*>(p + 2);
            x0 = (float)a.x; x1 = (float)a.y; x2 = (float)c.x; x3 = (float)c.y;      // cvt.rn.f32.f64
        } else {
            const float4 a = *reinterpret_cast<const float4*>(p);
            x0 = a.x; x1 = a.y; x2 = a.z; x3 = a.w;
        }
        bfp_store_block<NBITS>(dst, b, bfp_encode_block<NBITS>(x0, x1, x2, x3));
    }
}

// Ghost accumulation, receive side: decode and atomically scatter-add into the owned rows.
template <int NBITS, typename T>
__global__ void __launch_bounds__(256) bfp_decode_scatter_kernel(const unsigned char* __restrict__ src, const long long* __restrict__ rows,
                                                                 long long nrows, int nvec, T* __restrict__ Y, long long ld) {
    const int bpr = nvec / 2;
    const long long nblocks = nrows * bpr;
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < nblocks; b += (long long)gridDim.x * blockDim.x) {
        const long long r = b / bpr;
        const int v = 2 * (int)(b - r * bpr);
        float x[4];
        bfp_decode_block<NBITS>(bfp_load_block<NBITS>(src, b), x);
        T* p = Y + (__ldg(rows + r) * ld + v) * 2;
#pragma unroll
        for (int i = 0; i < 4; ++i) atomicAdd(p + i, (T)x[i]);
    }
}

static unsigned grid_for(long long nblocks) {
    long long g = (nblocks + 255) / 256;
    const long long cap = 148ll * 8 * 4;                    // a few waves of 8 CTAs per SM; grid-stride beyond
    return (unsigned)(g < 1 ? 1 : (g > cap ? cap : g));
}

}  // namespace chfsi

using namespace chfsi;

static chfsi_status bfp_fail(chfsi_status st, const char* msg) { set_error(msg); return st; }

#define BFP_DISPATCH(NB, CALL)                                      \
    switch (NB) {                                                   \
        case 16: { constexpr int NBITS = 16; CALL; break; }         \
        case 12: { constexpr int NBITS = 12; CALL; break; }         \
        default: { constexpr int NBITS = 10; CALL; break; }         \
    }

static chfsi_status bfp_done(const char* who) {
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string(who) + ": " + cudaGetErrorString(e)); return CHFSI_ECUDA; }
    count_launch();
    return CHFSI_OK;
}

extern "C" {

chfsi_status chfsi_bfp_stream_bytes(int nbits, long long n, size_t* bytes) {
    if (!bytes) return bfp_fail(CHFSI_EINVAL, "bfp_stream_bytes: NULL argument");
    if (nbits != 16 && nbits != 12 && nbits != 10) return bfp_fail(CHFSI_EINVAL, "bfp: n_bits must be 16, 12 or 10");
    if (n < 0 || n % 4 != 0) return bfp_fail(CHFSI_EINVAL, "bfp: the number of values must be a non-negative multiple of 4");
    *bytes = (size_t)(n / 4) * (size_t)(nbits / 2);
    return CHFSI_OK;
}

chfsi_status chfsi_bfp_encode(int nbits, const void* src, long long n, void* dst, void* cuda_stream) {
    size_t nb;
    chfsi_status st = chfsi_bfp_stream_bytes(nbits, n, &nb);
    if (st != CHFSI_OK) return st;
    if (n == 0) return CHFSI_OK;
    if (!src || !dst) return bfp_fail(CHFSI_EINVAL, "bfp_encode: NULL device pointer");
    if (((uintptr_t)src & 15) || ((uintptr_t)dst & 7)) return bfp_fail(CHFSI_EINVAL, "bfp_encode: src must be 16-byte and dst 8-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const long long nblk = n / 4;
    BFP_DISPATCH(nbits, (bfp_encode_kernel<NBITS><<<grid_for(nblk), 256, 0, s>>>(static_cast<const float4*>(src), nblk, static_cast<unsigned char*>(dst))));
    return bfp_done("bfp_encode");
}

chfsi_status chfsi_bfp_decode(int nbits, const void* src, long long n, void* dst, void* cuda_stream) {
    size_t nb;
    chfsi_status st = chfsi_bfp_stream_bytes(nbits, n, &nb);
    if (st != CHFSI_OK) return st;
    if (n == 0) return CHFSI_OK;
    if (!src || !dst) return bfp_fail(CHFSI_EINVAL, "bfp_decode: NULL device pointer");
    if (((uintptr_t)dst & 15) || ((uintptr_t)src & 7)) return bfp_fail(CHFSI_EINVAL, "bfp_decode: dst must be 16-byte and src 8-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const long long nblk = n / 4;
    BFP_DISPATCH(nbits, (bfp_decode_kernel<NBITS><<<grid_for(nblk), 256, 0, s>>>(static_cast<const unsigned char*>(src), nblk, static_cast<float4*>(dst))));
    return bfp_done("bfp_decode");
}

static chfsi_status bfp_ghost_check(int nbits, const void* X, long long ld, int nvec, const long long* rows, long long nrows,
                                    const void* stream_ptr, int elem_bytes, const char* who) {
    if (nbits != 16 && nbits != 12 && nbits != 10) return bfp_fail(CHFSI_EINVAL, "bfp: n_bits must be 16, 12 or 10");
    if (elem_bytes != 8 && elem_bytes != 16) return bfp_fail(CHFSI_EINVAL, "bfp: complex_bytes must be 8 (complex64) or 16 (complex128)");
    if (nvec < 2 || nvec % 2 != 0) return bfp_fail(CHFSI_EINVAL, "bfp: nvec must be even (whole four-value blocks per row, PAPER.md:224)");
    if (ld < nvec || ld % 2 != 0) return bfp_fail(CHFSI_EINVAL, "bfp: ld must be even and >= nvec");
    if (nrows < 0) return bfp_fail(CHFSI_EINVAL, "bfp: nrows < 0");
    if (nrows > 0 && (!X || !rows || !stream_ptr)) return bfp_fail(CHFSI_EINVAL, "bfp: NULL device pointer");
    if (((uintptr_t)X & 15) || ((uintptr_t)stream_ptr & 7)) return bfp_fail(CHFSI_EINVAL, "bfp: multivector must be 16-byte and stream 8-byte aligned");
    (void)who;
    return CHFSI_OK;
}

chfsi_status chfsi_bfp_gather_encode(int nbits, const void* X, int complex_bytes, long long ld, int nvec,
                                     const long long* rows, long long nrows, void* dst, void* cuda_stream) {
    chfsi_status st = bfp_ghost_check(nbits, X, ld, nvec, rows, nrows, dst, complex_bytes, "bfp_gather_encode");
    if (st != CHFSI_OK || nrows == 0) return st;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const long long nblk = nrows * (nvec / 2);
    if (complex_bytes == 16) {
        BFP_DISPATCH(nbits, (bfp_gather_encode_kernel<NBITS, double><<<grid_for(nblk), 256, 0, s>>>(static_cast<const double*>(X), ld, nvec, rows, nrows, static_cast<unsigned char*>(dst))));
    } else {
        BFP_DISPATCH(nbits, (bfp_gather_encode_kernel<NBITS, float><<<grid_for(nblk), 256, 0, s>>>(static_cast<const float*>(X), ld, nvec, rows, nrows, static_cast<unsigned char*>(dst))));
    }
    return bfp_done("bfp_gather_encode");
}

chfsi_status chfsi_bfp_decode_scatter_add(int nbits, const void* src, const long long* rows, long long nrows, int nvec,
                                          void* Y, int complex_bytes, long long ld, void* cuda_stream) {
    chfsi_status st = bfp_ghost_check(nbits, Y, ld, nvec, rows, nrows, src, complex_bytes, "bfp_decode_scatter_add");
    if (st != CHFSI_OK || nrows == 0) return st;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const long long nblk = nrows * (nvec / 2);
    if (complex_bytes == 16) {
        BFP_DISPATCH(nbits, (bfp_decode_scatter_kernel<NBITS, double><<<grid_for(nblk), 256, 0, s>>>(static_cast<const unsigned char*>(src), rows, nrows, nvec, static_cast<double*>(Y), ld)));
    } else {
        BFP_DISPATCH(nbits, (bfp_decode_scatter_kernel<NBITS, float><<<grid_for(nblk), 256, 0, s>>>(static_cast<const unsigned char*>(src), rows, nrows, nvec, static_cast<float*>(Y), ld)));
    }
    return bfp_done("bfp_decode_scatter_add");
}

}  // extern "C"
