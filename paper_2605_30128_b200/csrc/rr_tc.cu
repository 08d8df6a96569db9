// Rayleigh-Ritz subspace rotation on the 5th-generation tensor cores (tcgen05 + TMEM), sm_100a only.
//
//   Yout = Y Q_diag (FP64)  +  Y Q_non-diag (3xTF32 on tcgen05.mma.kind::tf32, FP32 accumulation in TMEM)
//
// PAPER.md:232 evaluates Y Q_non-diag "in FP32 arithmetic" and Y Q_diag in FP64.  Here the off-diagonal product runs as
// three TF32 tensor-core products per term (x = hi + lo, hi = tf32(x), lo = tf32(x - hi); lo*hi + hi*lo + hi*hi, FP32
// accumulation): 21 operand bits, FP32-level accuracy (reading R2), at the tensor pipe's rate instead of FFMA's.
//
// Real form of the complex product.  A row of Y is 2 nvec reals (re, im interleaved) = the K index k' = 2 i + c; an output
// row is 2 nvec reals, column j' = 2 j + d.  B[k'][j'] = Qre_ij (c == d), Qim_ij (c = 0, d = 1), -Qim_ij (c = 1, d = 0).
//
// One CTA = 128 rows x 256 real output columns (M = 128, N = 256: one accumulator of 256 TMEM columns), K in chunks of 32
// reals (128-byte rows, the 128-byte swizzle of the UMMA shared-memory layout).  Warp roles:
//   warps 0-3 : converters -- load the FP64 rows of Y, round to FP32, split into hi / lo, store the two A tiles in the
//               swizzled K-major layout (generic proxy -> fence.proxy.async -> mbarrier); afterwards the epilogue: TMEM ->
//               registers (tcgen05.ld 32x32b), + Y Q_diag in FP64, store complex128.
//   warp 4    : one lane streams the pre-split, pre-swizzled B tiles (hi, lo; 32 KB each, contiguous in the workspace) with
//               cp.async.bulk onto an mbarrier.
//   warp 5    : allocates TMEM; one lane issues the tcgen05.mma's (12 per chunk) and commits them to the stage's `empty`
//               barrier and, after the last chunk, to `acc_full`.
// Two shared-memory stages of 96 KB (A hi/lo 2 x 16 KB, B hi/lo 2 x 32 KB).
#include <algorithm>
#include <cstdint>
#include <mutex>
#include <string>

#include "chfsi_internal.h"
#include "tma_util.cuh"

namespace chfsi {

constexpr int TC_M = 128, TC_N = 256, TC_KC = 32, TC_STAGES = 2;
constexpr int TC_A_BYTES = TC_M * 128, TC_B_BYTES = TC_N * 128;
constexpr int TC_STAGE_BYTES = 2 * TC_A_BYTES + 2 * TC_B_BYTES;
constexpr int TC_SMEM = TC_STAGES * TC_STAGE_BYTES + 1024;      // + slack to align the tiles to 1024 bytes
constexpr int TC_CONV_WARPS = 8, TC_CONV_THREADS = 32 * TC_CONV_WARPS;        // converters; then 4 epilogue warps, loader, MMA
constexpr int TC_LOAD_WARP = TC_CONV_WARPS + 4, TC_MMA_WARP = TC_CONV_WARPS + 5;
constexpr int TC_THREADS = 32 * (TC_CONV_WARPS + 6);

__device__ __forceinline__ float tf32_rna(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

// UMMA shared-memory descriptor of a K-major tile with 128-byte rows and the 128-byte swizzle: 8-row groups are 1024 bytes
// apart (SBO), the leading-dimension offset is unused for swizzled K-major operands, version 1 (sm_100), layout type 2.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)(1024 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}

// instruction descriptor: D = F32 (bits 4-5 = 1), A = B = TF32 (bits 7-9, 10-12 = 2), both K-major, N / 8 at bit 17, M / 16 at bit 24
constexpr uint32_t TC_IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TC_N >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);

__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(TC_IDESC), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---- Q -> dq (FP64 diagonal) and the real-form off-diagonal B, split into TF32 hi / lo, in the layout the kernel's stages
//      hold: tile (nh, kc) = 256 rows (n) x 32 reals (k), 128-byte rows, 16-byte chunks XOR-swizzled by n % 8.
__global__ void rr_tc_split_q_kernel(const double2* __restrict__ Q, int nvec, int kchunks, int nhalves, double2* __restrict__ dq,
                                     float* __restrict__ Bhi, float* __restrict__ Blo) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)nhalves * kchunks * TC_N * TC_KC;
    if (idx < nvec) dq[idx] = Q[idx * nvec + idx];
    if (idx >= total) return;
    const int k = (int)(idx % TC_KC);
    const int n = (int)((idx / TC_KC) % TC_N);
    const long long tile = idx / (TC_KC * TC_N);
    const int kc = (int)(tile % kchunks), nh = (int)(tile / kchunks);
    const int kp = kc * TC_KC + k, jp = nh * TC_N + n;
    const int i = kp >> 1, c = kp & 1, j = jp >> 1, d = jp & 1;
    double v = 0.0;
    if (i < nvec && j < nvec && i != j) {
        const double2 q = Q[(long long)i * nvec + j];
        v = (c == d) ? q.x : (c == 0 ? q.y : -q.y);
    }
    const float xf = (float)v;
    const float hi = tf32_rna(xf), lo = tf32_rna(xf - hi);
    const long long off = (tile * TC_N + n) * TC_KC + ((((k >> 2) ^ (n & 7)) << 2) | (k & 3));
    Bhi[off] = hi;
    Blo[off] = lo;
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
          "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
          "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Persistent: grid = number of SMs; a CTA walks tiles blockIdx.x, blockIdx.x + gridDim.x, ... (tile = 128 rows x one column
// half; the halves of a row tile are consecutive tile numbers, so they run at the same time on neighbouring SMs and the
// second read of the rows hits L2).  Chunks are numbered g = 0, 1, ... across the tiles of the CTA; stage g % 2.
__global__ void __launch_bounds__(TC_THREADS, 1)
rr_rotate_tc_kernel(const double2* __restrict__ Y, long long ldy, const float* __restrict__ Bhi, const float* __restrict__ Blo,
                    const double2* __restrict__ dq, long long nrows, int nvec, int kchunks, int nhalves, long long ntiles,
                    double2* __restrict__ C, long long ldc) {
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t a_full[TC_STAGES], b_full[TC_STAGES], empty[TC_STAGES], acc_full, acc_empty;
    __shared__ uint32_t tmem_base_s;
    __shared__ float stash[4 * 32 * 33];                     // epilogue transpose, one 32 x 32 block (+ padding) per epilogue warp
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // tiles on 1024-byte boundaries
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const long long nchunks_total = my_tiles * kchunks;

    if (threadIdx.x == 0) {
        for (int s = 0; s < TC_STAGES; ++s) { mbar_init(&a_full[s], TC_CONV_THREADS); mbar_init(&b_full[s], 1); mbar_init(&empty[s], 1); }
        mbar_init(&acc_full, 1);
        mbar_init(&acc_empty, 128);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == TC_MMA_WARP) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(2 * TC_N) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tmem_base_s;

    if (warp < TC_CONV_WARPS) {
        // ============ converters: FP64 rows of Y -> FP32 -> TF32 hi / lo, swizzled K-major A tiles ============
        // 256 threads: 16 threads per row (one complex each), 16 rows per pass, 8 passes per chunk; the loads of the next two
        // chunks are in flight while a chunk is converted (64 KB per SM)
        constexpr int NP = TC_M / (TC_CONV_THREADS / 16);
        const int cpx = threadIdx.x & 15;
        const int rsub = threadIdx.x >> 4;
        double2 y0[NP], y1[NP], y2[NP];
        auto load_chunk = [&](long long g, double2 (&dst)[NP]) {
            const long long ti = g / kchunks;
            const int c = (int)(g - ti * kchunks);
            const long long tile = blockIdx.x + ti * gridDim.x;
            const long long m0 = (tile / nhalves) * TC_M;
            const int i = c * (TC_KC / 2) + cpx;
#pragma unroll
            for (int pass = 0; pass < NP; ++pass) {
                const long long r = m0 + pass * (TC_M / NP) + rsub;
                dst[pass] = make_double2(0.0, 0.0);
                if (g < nchunks_total && r < nrows && i < nvec) dst[pass] = __ldg(Y + r * ldy + i);
            }
        };
        load_chunk(0, y0);
        load_chunk(1, y1);
        for (long long g = 0; g < nchunks_total; ++g) {
            const int s = (int)(g & 1);
            load_chunk(g + 2, y2);
            if (g >= TC_STAGES) mbar_wait(&empty[s], (uint32_t)(((g >> 1) - 1) & 1));
            unsigned char* Ahi = smem + (size_t)s * TC_STAGE_BYTES;
            unsigned char* Alo = Ahi + TC_A_BYTES;
#pragma unroll
            for (int pass = 0; pass < NP; ++pass) {
                const int row = pass * (TC_M / NP) + rsub;
                const float xr = (float)y0[pass].x, xi = (float)y0[pass].y;
                // hi = x rounded to TF32, nearest-away, with two integer operations (half a TF32 ulp added to the magnitude bits, the low
                // 13 bits cleared: what cvt.rna.tf32.f32 returns for finite x, without its conversion-pipe slot); lo = x - hi is exact in
                // FP32 and goes to the tensor core as it is, which reads its upper 19 bits
                const float hr = __uint_as_float((__float_as_uint(xr) + 0x1000u) & 0xFFFFE000u);
                const float hi_ = __uint_as_float((__float_as_uint(xi) + 0x1000u) & 0xFFFFE000u);
                const float lr = xr - hr, li = xi - hi_;
                const uint32_t off = (uint32_t)row * 128u + ((uint32_t)((cpx >> 1) ^ (row & 7)) << 4) + (uint32_t)(cpx & 1) * 8u;
                *reinterpret_cast<float2*>(Ahi + off) = make_float2(hr, hi_);
                *reinterpret_cast<float2*>(Alo + off) = make_float2(lr, li);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy stores -> visible to the tensor core
            mbar_arrive(&a_full[s]);
#pragma unroll
            for (int pass = 0; pass < NP; ++pass) { y0[pass] = y1[pass]; y1[pass] = y2[pass]; }
        }
    } else if (warp < TC_CONV_WARPS + 4) {
        // ============ epilogue: TMEM -> registers, + Y Q_diag (FP64), store ============
        const int ew = warp - TC_CONV_WARPS;                 // = warp % 4: this warp reads TMEM lanes 32 ew ... 32 ew + 31
        const uint32_t tlane = tmem + ((uint32_t)(ew * 32) << 16);
        for (long long ti = 0; ti < my_tiles; ++ti) {
            const long long tile = blockIdx.x + ti * gridDim.x;
            const int nh = (int)(tile % nhalves);
            mbar_wait(&acc_full, (uint32_t)(ti & 1));
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            // tcgen05.ld hands a thread one ROW (32 columns of it).  Loads and stores of 32 rows x 16 bytes per instruction cost 32
            // LSU wavefronts each (measured: LSU data pipe 67 % busy, the epilogue's 16.7 us of wavefronts per tile were the kernel's
            // bottleneck), so the block is transposed through shared memory: afterwards a half-warp covers the 16 complex values
            // (256 bytes) of one row, for the loads of Y (diagonal term) and the stores alike -- 4 wavefronts per instruction.
            float* st = stash + ew * (32 * 33);
            const long long rbase = (tile / nhalves) * TC_M + ew * 32;
#pragma unroll 1
            for (int cb = 0; cb < TC_N / 32; ++cb) {
                const int j = nh * (TC_N / 2) + cb * 16 + (lane & 15);
                const bool jok = j < nvec;
                // the 16 values of Y this lane needs for the block (rows 2 it + lane / 16), all in flight before the TMEM reads
                double2 yv[16];
#pragma unroll
                for (int it = 0; it < 16; ++it) {
                    const long long r = rbase + it * 2 + (lane >> 4);
                    yv[it] = make_double2(0.0, 0.0);
                    if (r < nrows && jok) yv[it] = __ldg(Y + r * ldy + j);
                }
                const double2 d = jok ? dq[j] : make_double2(0.0, 0.0);
                {
                    uint32_t v[32], w[32];
                    tmem_ld32(tlane + (uint32_t)(cb * 32), v);
                    tmem_ld32(tlane + (uint32_t)(TC_N + cb * 32), w);
                    if (cb == TC_N / 32 - 1) {               // the accumulators are in registers: the next tile may overwrite them
                        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                        mbar_arrive(&acc_empty);
                    }
                    __syncwarp();                            // the previous block's reads of the stash are done
#pragma unroll
                    for (int q = 0; q < 32; ++q) st[lane * 33 + q] = __uint_as_float(v[q]) + __uint_as_float(w[q]);
                }
                __syncwarp();
#pragma unroll
                for (int it = 0; it < 16; ++it) {
                    const int rr = it * 2 + (lane >> 4);
                    const long long r = rbase + rr;
                    if (r < nrows && jok) {
                        const float are = st[rr * 33 + 2 * (lane & 15)], aim = st[rr * 33 + 2 * (lane & 15) + 1];
                        C[r * ldc + j] = make_double2(fma(yv[it].x, d.x, fma(-yv[it].y, d.y, (double)are)),      // Y Q_diag in FP64
                                                      fma(yv[it].x, d.y, fma(yv[it].y, d.x, (double)aim)));
                    }
                }
            }
        }
    } else if (warp == TC_LOAD_WARP) {
        // ============ B loader ============
        if (lane == 0) {
            for (long long g = 0; g < nchunks_total; ++g) {
                const int s = (int)(g & 1);
                const long long ti = g / kchunks;
                const int c = (int)(g - ti * kchunks);
                const int nh = (int)((blockIdx.x + ti * gridDim.x) % nhalves);
                if (g >= TC_STAGES) mbar_wait(&empty[s], (uint32_t)(((g >> 1) - 1) & 1));
                unsigned char* Bh = smem + (size_t)s * TC_STAGE_BYTES + 2 * TC_A_BYTES;
                const size_t off = ((size_t)nh * kchunks + c) * (TC_N * TC_KC);
                mbar_expect_tx(&b_full[s], 2 * TC_B_BYTES);
                bulk_load(Bh, Bhi + off, TC_B_BYTES, &b_full[s]);
                bulk_load(Bh + TC_B_BYTES, Blo + off, TC_B_BYTES, &b_full[s]);
            }
        }
    } else {
        // ============ MMA issuer ============
        if (lane == 0) {
            long long g = 0;
            for (long long ti = 0; ti < my_tiles; ++ti) {
                if (ti > 0) {                                               // the epilogue has read the previous tile's accumulators
                    mbar_wait(&acc_empty, (uint32_t)((ti - 1) & 1));
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                }
                for (int c = 0; c < kchunks; ++c, ++g) {
                    const int s = (int)(g & 1);
                    mbar_wait(&a_full[s], (uint32_t)((g >> 1) & 1));
                    mbar_wait(&b_full[s], (uint32_t)((g >> 1) & 1));
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t a_hi = smem_u32(smem + (size_t)s * TC_STAGE_BYTES), a_lo = a_hi + TC_A_BYTES;
                    const uint32_t b_hi = a_hi + 2 * TC_A_BYTES, b_lo = b_hi + TC_B_BYTES;
#pragma unroll
                    for (int ks = 0; ks < TC_KC / 8; ++ks) {               // K = 8 TF32 (32 bytes) per instruction
                        const uint64_t dah = umma_desc_sw128(a_hi + ks * 32), dal = umma_desc_sw128(a_lo + ks * 32);
                        const uint64_t dbh = umma_desc_sw128(b_hi + ks * 32), dbl = umma_desc_sw128(b_lo + ks * 32);
                        // two accumulators: the tensor core truncates when it adds into FP32, once per instruction, so the error
                        // grows with the number of instructions that hit an accumulator; the (small) cross terms get their own
                        umma_tf32(tmem + TC_N, dal, dbh, (c | ks) != 0 ? 1u : 0u);
                        umma_tf32(tmem + TC_N, dah, dbl, 1u);
                        umma_tf32(tmem, dah, dbh, (c | ks) != 0 ? 1u : 0u);
                    }
                    umma_commit(&empty[s]);                                  // frees the stage when these MMAs have read it
                }
                umma_commit(&acc_full);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == TC_MMA_WARP) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(2 * TC_N) : "memory");
}

// workspace: dq (nvec complex128, padded to 256 bytes) | B hi | B lo
size_t rr_tc_workspace_bytes(int nvec) {
    const size_t kchunks = (2 * (size_t)nvec + TC_KC - 1) / TC_KC, nhalves = (2 * (size_t)nvec + TC_N - 1) / TC_N;
    return (((size_t)nvec * 16 + 255) / 256) * 256 + 2 * nhalves * kchunks * TC_N * TC_KC * sizeof(float) + 256;
}

cudaError_t launch_rr_rotate_tc(long long nrows, int nvec, const void* Y, long long ldy, const void* Q, void* Yout, long long ldo,
                                void* work, cudaStream_t st) {
    const int kchunks = (2 * nvec + TC_KC - 1) / TC_KC, nhalves = (2 * nvec + TC_N - 1) / TC_N;
    double2* dq = static_cast<double2*>(work);
    float* Bhi = reinterpret_cast<float*>(static_cast<char*>(work) + (((size_t)nvec * 16 + 255) / 256) * 256);
    float* Blo = Bhi + (size_t)nhalves * kchunks * TC_N * TC_KC;
    const long long total = std::max<long long>((long long)nhalves * kchunks * TC_N * TC_KC, nvec);
    rr_tc_split_q_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(static_cast<const double2*>(Q), nvec, kchunks, nhalves, dq, Bhi, Blo);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    count_launch();
    if (nrows == 0) return cudaSuccess;
    static std::once_flag once[32];
    int dev = 0;
    cudaGetDevice(&dev);
    cudaError_t ae = cudaSuccess;
    std::call_once(once[dev & 31], [&] { ae = cudaFuncSetAttribute(rr_rotate_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM); });
    if (ae != cudaSuccess) return ae;
    int nsm = 0;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const long long ntiles = ((nrows + TC_M - 1) / TC_M) * nhalves;
    const unsigned grid = (unsigned)std::min<long long>(ntiles, nsm > 0 ? nsm : 148);
    rr_rotate_tc_kernel<<<grid, TC_THREADS, TC_SMEM, st>>>(static_cast<const double2*>(Y), ldy, Bhi, Blo, dq, nrows, nvec, kchunks,
                                                           nhalves, ntiles, static_cast<double2*>(Yout), ldo);
    e = cudaGetLastError();
    if (e == cudaSuccess) count_launch();
    return e;
}

}  // namespace chfsi
