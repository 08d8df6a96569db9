// Pipe-rate micro-benchmark ("FP64/FP32/TF32 peaks are not in MEASURED_PEAKS.json; the builder measures them
// with an FMA / MMA micro-benchmark in the same run").  Register-resident dependent-free chains, 16 warps per SM, one CTA per SM;
// timed with CUDA events.  Results in TFLOP/s (2 flop per FMA): DFMA, FFMA, mma.m8n8k4.f64, mma.m16n8k8.tf32.
#include <cstdint>

#include "chfsi_internal.h"

namespace chfsi {

__global__ void __launch_bounds__(512) peak_dfma(double* out, int iters) {
    double a = threadIdx.x * 1e-3, b = 1.0 + threadIdx.x * 1e-4, c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = fma(a, c[i], b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(512) peak_ffma(float* out, int iters) {
    float a = threadIdx.x * 1e-3f, b = 1.0f + threadIdx.x * 1e-4f, c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = fmaf(a, c[i], b);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(512) peak_dmma(double* out, int iters) {
    double a = threadIdx.x * 1e-3, b = 1.0 + threadIdx.x * 1e-4, c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = i; c[i][1] = -i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(512) peak_tf32(float* out, int iters) {
    unsigned a[4], b[2];
#pragma unroll
    for (int i = 0; i < 4; ++i) a[i] = __float_as_uint(1.0f + threadIdx.x * 1e-3f + i);
    b[0] = __float_as_uint(0.5f); b[1] = __float_as_uint(0.25f);
    float c[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) c[i][j] = i + j;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                         : "+f"(c[i][0]), "+f"(c[i][1]), "+f"(c[i][2]), "+f"(c[i][3])
                         : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += c[i][j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace chfsi

using namespace chfsi;

extern "C" chfsi_status chfsi_measure_pipe_peaks(int device, double* tflops) {
    if (!tflops) { set_error("measure_pipe_peaks: NULL output"); return CHFSI_EINVAL; }
    int prev = 0, nsm = 0;
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess ||
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) {
        set_error("measure_pipe_peaks: cannot select device"); return CHFSI_ECUDA;
    }
    void* buf = nullptr;
    if (cudaMalloc(&buf, (size_t)nsm * 512 * 8) != cudaSuccess) { cudaSetDevice(prev); set_error("measure_pipe_peaks: cudaMalloc"); return CHFSI_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 20000, th = 512;
    // FMAs per thread and iteration: 16 (dfma, ffma); per warp: 8 x 256 (dmma), 8 x 1024 (tf32 mma)
    const double fma_per_launch[4] = {(double)iters * 16 * th * nsm, (double)iters * 16 * th * nsm,
                                      (double)iters * 8 * 256 * (th / 32) * nsm, (double)iters * 8 * 1024 * (th / 32) * nsm};
    for (int k = 0; k < 4; ++k) {
        float best = 1e30f;
        for (int rep = 0; rep < 3; ++rep) {
            cudaEventRecord(e0);
            if (k == 0) peak_dfma<<<nsm, th>>>(static_cast<double*>(buf), iters);
            else if (k == 1) peak_ffma<<<nsm, th>>>(static_cast<float*>(buf), iters);
            else if (k == 2) peak_dmma<<<nsm, th>>>(static_cast<double*>(buf), iters);
            else peak_tf32<<<nsm, th>>>(static_cast<float*>(buf), iters);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;           // the first launch warms up
        }
        tflops[k] = 2.0 * fma_per_launch[k] / (best * 1e-3) / 1e12;
    }
    const cudaError_t err = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf); cudaSetDevice(prev);
    if (err != cudaSuccess) { set_error(std::string("measure_pipe_peaks: ") + cudaGetErrorString(err)); return CHFSI_ECUDA; }
    return CHFSI_OK;
}
