// Rayleigh-Ritz pieces around the filter (Algorithm 1 lines 6-8) for sm_100a:
//   chfsi_rr_project : S = A^H diag(m) B, the projections Y^H M Y and Y^H H Y (RR-Proj), FP64, Hermitian tiles only once
//   chfsi_rr_rotate  : Y Q = Y Q_diag (FP64) + Y Q_non-diag (FP32) (RR-SR), or all FP64
// Both are register-tiled complex GEMMs on the FMA pipes.  On the B200 the FP64 tensor path (mma.m8n8k4.f64) shares the
// DFMA pipe (measured: DMMA 63.8, DFMA 58.5 FMA/clk/SM, the two add up when mixed -- DESIGN.md 6.6), so the projection is
// bound by the same pipe either way; the FP32 rotation runs on FFMA so that it really is "FP32 arithmetic".
#include <cstdint>
#include <mutex>
#include <string>

#include "chfsi_internal.h"

namespace chfsi {

// ---- S += A^H diag(w) B over this CTA's slab of rows.  Tile 64 x 64 complex, 16 x 16 threads, 4 x 4 outputs per thread
//      (i = ty + 16 a, j = tx + 16 b); K-slabs of 8 rows, double buffered through registers.
constexpr int PT = 64, PK = 8;

__global__ void __launch_bounds__(256, 2) rr_project_kernel(const double2* __restrict__ A, long long lda, const double2* __restrict__ B,
                                                         long long ldb, long long nrows, int nvec, long long rows_per_cta,
                                                         const double* __restrict__ mass, int hermitian, double2* __restrict__ S) {
    const int ti = blockIdx.y, tj = blockIdx.x;
    if (hermitian && tj < ti) return;                       // the lower triangle is mirrored afterwards
    __shared__ double2 As[PK][PT], Bs[PK][PT];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const long long r0 = (long long)blockIdx.z * rows_per_cta;
    const long long r1 = r0 + rows_per_cta < nrows ? r0 + rows_per_cta : nrows;
    double sre[4][4], sim[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) { sre[a][b] = 0.0; sim[a][b] = 0.0; }
    // loader: thread -> (row k = tid / 32 and + 4... : 512 elements per operand per slab, 2 per thread
    const int lk = tid >> 6, lc = tid & 63;                 // rows lk and lk + 4 of the slab, column lc of the tile
    double2 ra[2], rb[2];
    auto fetch = [&](long long rs) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const long long r = rs + lk + 4 * h;
            const bool ok = r < r1;
            const int ci = ti * PT + lc, cj = tj * PT + lc;
            ra[h] = (ok && ci < nvec) ? __ldg(A + r * lda + ci) : make_double2(0.0, 0.0);
            double2 bv = (ok && cj < nvec) ? __ldg(B + r * ldb + cj) : make_double2(0.0, 0.0);
            const double w = ok ? (mass ? __ldg(mass + (r >> 1)) : 1.0) : 0.0;      // row 2 I + alpha carries m_I
            rb[h] = make_double2(bv.x * w, bv.y * w);
        }
    };
    fetch(r0);
    for (long long rs = r0; rs < r1; rs += PK) {
#pragma unroll
        for (int h = 0; h < 2; ++h) { As[lk + 4 * h][lc] = ra[h]; Bs[lk + 4 * h][lc] = rb[h]; }
        __syncthreads();
        if (rs + PK < r1) fetch(rs + PK);
#pragma unroll
        for (int k = 0; k < PK; ++k) {
            double2 a[4], b[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { a[q] = As[k][ty + 16 * q]; b[q] = Bs[k][tx + 16 * q]; }
#pragma unroll
            for (int ia = 0; ia < 4; ++ia)
#pragma unroll
                for (int ib = 0; ib < 4; ++ib) {
                    // conj(a) b = (ar br + ai bi) + i (ar bi - ai br)
                    sre[ia][ib] = fma(a[ia].x, b[ib].x, sre[ia][ib]);
                    sre[ia][ib] = fma(a[ia].y, b[ib].y, sre[ia][ib]);
                    sim[ia][ib] = fma(a[ia].x, b[ib].y, sim[ia][ib]);
                    sim[ia][ib] = fma(-a[ia].y, b[ib].x, sim[ia][ib]);
                }
        }
        __syncthreads();
    }
#pragma unroll
    for (int ia = 0; ia < 4; ++ia)
#pragma unroll
        for (int ib = 0; ib < 4; ++ib) {
            const int i = ti * PT + ty + 16 * ia, j = tj * PT + tx + 16 * ib;
            if (i < nvec && j < nvec && (!hermitian || j >= i)) {
                double* d = reinterpret_cast<double*>(S + (long long)i * nvec + j);
                atomicAdd(d, sre[ia][ib]);
                atomicAdd(d + 1, sim[ia][ib]);
            }
        }
}

// S[j][i] = conj(S[i][j]) for j > i; the diagonal is made exactly real
__global__ void rr_mirror_kernel(double2* S, int nvec) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)nvec * nvec) return;
    const int i = (int)(idx / nvec), j = (int)(idx % nvec);
    if (j > i) { const double2 v = S[idx]; S[(long long)j * nvec + i] = make_double2(v.x, -v.y); }
    else if (i == j) S[idx].y = 0.0;
}

// ---- rotation.  Q split: dq[j] = Q[j][j] (FP64); Qo = Q with a zero diagonal, in the arithmetic type TQ
template <typename TQ2>
__global__ void rr_split_q_kernel(const double2* __restrict__ Q, int nvec, double2* __restrict__ dq, TQ2* __restrict__ Qo) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)nvec * nvec) return;
    const int i = (int)(idx / nvec), j = (int)(idx % nvec);
    const double2 v = Q[idx];
    if (i == j) { dq[j] = v; Qo[idx].x = 0; Qo[idx].y = 0; }
    else { Qo[idx].x = (decltype(Qo[idx].x))v.x; Qo[idx].y = (decltype(Qo[idx].y))v.y; }
}

// C[r][j] = Y[r][j] dq[j] (FP64) + sum_i (TC)Y[r][i] Qo[i][j] (arithmetic and accumulation in TC).  Tile RT rows x 64 columns,
// 16 x 16 threads, RA x 4 outputs per thread (r = ty + 16 a, j = tx + 16 b); K-slabs of 8 columns of Y.
template <typename TC, typename TC2, int RA>
__global__ void __launch_bounds__(256, 2) rr_rotate_kernel(const double2* __restrict__ Y, long long ldy, const TC2* __restrict__ Qo,
                                                        const double2* __restrict__ dq, long long nrows, int nvec,
                                                        double2* __restrict__ C, long long ldc) {
    constexpr int RT = 16 * RA, KT = 8;
    __shared__ TC2 Ys[KT][RT + 1], Qs[KT][PT];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const long long rbase = (long long)blockIdx.x * RT;
    const int jbase = blockIdx.y * PT;
    TC cre[RA][4], cim[RA][4];
#pragma unroll
    for (int a = 0; a < RA; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) { cre[a][b] = 0; cim[a][b] = 0; }
    // loader: the Y tile is RT rows x 8 columns (a row's 8 columns are 128 contiguous bytes), the Q tile 8 x 64; both are
    // fetched into registers one slab ahead of the arithmetic and converted to TC on the way
    constexpr int NY = RT * KT / 256, NQ = KT * PT / 256;
    TC2 ry[NY], rq[NQ];
    auto fetch = [&](int i0) {
#pragma unroll
        for (int u = 0; u < NY; ++u) {
            const int e = tid + 256 * u, rr = e / KT, kk = e % KT;
            const long long r = rbase + rr;
            const double2 v = (r < nrows && i0 + kk < nvec) ? __ldg(Y + r * ldy + i0 + kk) : make_double2(0.0, 0.0);
            ry[u].x = (TC)v.x; ry[u].y = (TC)v.y;
        }
#pragma unroll
        for (int u = 0; u < NQ; ++u) {
            const int e = tid + 256 * u, kk = e / PT, jj = e % PT;
            TC2 z; z.x = 0; z.y = 0;
            rq[u] = (i0 + kk < nvec && jbase + jj < nvec) ? Qo[(long long)(i0 + kk) * nvec + jbase + jj] : z;
        }
    };
    fetch(0);
    for (int i0 = 0; i0 < nvec; i0 += KT) {
#pragma unroll
        for (int u = 0; u < NY; ++u) { const int e = tid + 256 * u; Ys[e % KT][e / KT] = ry[u]; }
#pragma unroll
        for (int u = 0; u < NQ; ++u) { const int e = tid + 256 * u; Qs[e / PT][e % PT] = rq[u]; }
        __syncthreads();
        if (i0 + KT < nvec) fetch(i0 + KT);
#pragma unroll
        for (int k = 0; k < KT; ++k) {
            TC2 y[RA], q[4];
#pragma unroll
            for (int a = 0; a < RA; ++a) y[a] = Ys[k][ty + 16 * a];
#pragma unroll
            for (int b = 0; b < 4; ++b) q[b] = Qs[k][tx + 16 * b];
#pragma unroll
            for (int a = 0; a < RA; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    cre[a][b] = fma(y[a].x, q[b].x, cre[a][b]);
                    cre[a][b] = fma(-y[a].y, q[b].y, cre[a][b]);
                    cim[a][b] = fma(y[a].x, q[b].y, cim[a][b]);
                    cim[a][b] = fma(y[a].y, q[b].x, cim[a][b]);
                }
        }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < RA; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const long long r = rbase + ty + 16 * a;
            const int j = jbase + tx + 16 * b;
            if (r < nrows && j < nvec) {
                const double2 yv = __ldg(Y + r * ldy + j), d = dq[j];      // Y Q_diag in FP64
                C[r * ldc + j] = make_double2(fma(yv.x, d.x, fma(-yv.y, d.y, (double)cre[a][b])),
                                              fma(yv.x, d.y, fma(yv.y, d.x, (double)cim[a][b])));
            }
        }
}

}  // namespace chfsi

using namespace chfsi;

static chfsi_status rr_fail(chfsi_status st, const char* msg) { set_error(msg); return st; }
static chfsi_status rr_cuda(cudaError_t e, const char* who) {
    if (e == cudaSuccess) return CHFSI_OK;
    set_error(std::string(who) + ": " + cudaGetErrorString(e));
    return CHFSI_ECUDA;
}

extern "C" {

chfsi_status chfsi_rr_project(const chfsi_mesh* mesh, long long nrows, int nvec, const void* A, long long lda, const void* B,
                              long long ldb, int use_mass, int hermitian, void* S, void* cuda_stream) {
    if (nvec < 1 || nrows < 0) return rr_fail(CHFSI_EINVAL, "rr_project: nvec must be >= 1 and nrows >= 0");
    if (!A || !B || !S) return rr_fail(CHFSI_EINVAL, "rr_project: NULL device pointer");
    if (lda < nvec || ldb < nvec) return rr_fail(CHFSI_EINVAL, "rr_project: leading dimension < nvec");
    if (((uintptr_t)A & 15) || ((uintptr_t)B & 15) || ((uintptr_t)S & 15)) return rr_fail(CHFSI_EINVAL, "rr_project: pointers must be 16-byte aligned");
    const double* mass = nullptr;
    if (use_mass) {
        if (!mesh) return rr_fail(CHFSI_EINVAL, "rr_project: the mass weighting needs a mesh");
        if (!mesh->dMass) return rr_fail(CHFSI_ESTATE, "rr_project: chfsi_ham_set has not been called (it builds the device mass)");
        if (nrows != 2 * mesh->nnodes) return rr_fail(CHFSI_EINVAL, "rr_project: with the mass weighting nrows must be 2 * nnodes");
        mass = mesh->dMass;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    chfsi_status rc = rr_cuda(cudaMemsetAsync(S, 0, (size_t)nvec * nvec * 16, st), "rr_project memset");
    if (rc != CHFSI_OK) return rc;
    count_launch();
    const int nt = (nvec + PT - 1) / PT;
    const long long tiles = hermitian ? (long long)nt * (nt + 1) / 2 : (long long)nt * nt;
    // split the rows so that the live tiles fill the GPU a few times over; slabs are multiples of PK rows
    long long nz = (8 * 148) / tiles;                      // live CTAs = a whole number of waves of 2 CTAs per SM (rounded down)
    if (nz < 1) nz = 1;
    if (nz > 65535) nz = 65535;
    long long rows_per = ((nrows + nz - 1) / nz + PK - 1) / PK * PK;
    if (rows_per < PK) rows_per = PK;
    nz = nrows > 0 ? (nrows + rows_per - 1) / rows_per : 0;
    if (nz > 0) {
        rr_project_kernel<<<dim3(nt, nt, (unsigned)nz), 256, 0, st>>>(static_cast<const double2*>(A), lda, static_cast<const double2*>(B), ldb,
                                                                      nrows, nvec, rows_per, mass, hermitian ? 1 : 0, static_cast<double2*>(S));
        rc = rr_cuda(cudaGetLastError(), "rr_project");
        if (rc != CHFSI_OK) return rc;
        count_launch();
    }
    if (hermitian) {
        const long long n2 = (long long)nvec * nvec;
        rr_mirror_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(static_cast<double2*>(S), nvec);
        rc = rr_cuda(cudaGetLastError(), "rr_project mirror");
        if (rc != CHFSI_OK) return rc;
        count_launch();
    }
    return CHFSI_OK;
}

chfsi_status chfsi_rr_rotate_workspace_bytes(int nvec, size_t* bytes) {
    if (!bytes || nvec < 1) return rr_fail(CHFSI_EINVAL, "rr_rotate_workspace_bytes: bad argument");
    *bytes = (size_t)nvec * nvec * 16 + (size_t)nvec * 16 + 512;
    if (rr_tc_workspace_bytes(nvec) > *bytes) *bytes = rr_tc_workspace_bytes(nvec);   // CHFSI_TF32X3 (rr_tc.cu)
    return CHFSI_OK;
}

chfsi_status chfsi_rr_rotate(chfsi_prec prec, long long nrows, int nvec, const void* Y, long long ldy, const void* Q, void* Yout,
                             long long ldo, void* work, size_t work_bytes, void* cuda_stream) {
    if (prec != CHFSI_FP64 && prec != CHFSI_FP32 && prec != CHFSI_TF32X3)
        return rr_fail(CHFSI_EUNSUPPORTED, "rr_rotate: prec must be CHFSI_FP64, CHFSI_FP32 (mixed, PAPER.md:232) or CHFSI_TF32X3 (mixed on tcgen05)");
    if (nvec < 1 || nrows < 0) return rr_fail(CHFSI_EINVAL, "rr_rotate: nvec must be >= 1 and nrows >= 0");
    if (!Y || !Q || !Yout || !work) return rr_fail(CHFSI_EINVAL, "rr_rotate: NULL device pointer");
    if (Y == Yout) return rr_fail(CHFSI_EINVAL, "rr_rotate: Y and Yout must be distinct buffers");
    if (ldy < nvec || ldo < nvec) return rr_fail(CHFSI_EINVAL, "rr_rotate: leading dimension < nvec");
    // what this precision needs (chfsi_rr_rotate_workspace_bytes returns the largest over the precisions)
    const size_t need = prec == CHFSI_TF32X3 ? rr_tc_workspace_bytes(nvec) : (size_t)nvec * nvec * 16 + (size_t)nvec * 16 + 512;
    if (work_bytes < need || ((uintptr_t)work & 255)) return rr_fail(CHFSI_EINVAL, "rr_rotate: work too small or not 256-byte aligned");
    if (((uintptr_t)Y & 15) || ((uintptr_t)Q & 15) || ((uintptr_t)Yout & 15)) return rr_fail(CHFSI_EINVAL, "rr_rotate: pointers must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (prec == CHFSI_TF32X3) {
        if (nrows >= (1ll << 31) * 128) return rr_fail(CHFSI_EINVAL, "rr_rotate: too many rows");
        return rr_cuda(launch_rr_rotate_tc(nrows, nvec, Y, ldy, Q, Yout, ldo, work, st), "rr_rotate (tcgen05)");
    }
    double2* dq = static_cast<double2*>(work);
    void* qo = static_cast<char*>(work) + (((size_t)nvec * 16 + 255) / 256) * 256;
    const long long n2 = (long long)nvec * nvec;
    const unsigned ncolt = (unsigned)((nvec + PT - 1) / PT);
    chfsi_status rc;
    if (prec == CHFSI_FP32) {
        rr_split_q_kernel<float2><<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(static_cast<const double2*>(Q), nvec, dq, static_cast<float2*>(qo));
        rc = rr_cuda(cudaGetLastError(), "rr_rotate split");
        if (rc != CHFSI_OK) return rc;
        count_launch();
        if (nrows > 0) {
            constexpr int RA = 8;
            rr_rotate_kernel<float, float2, RA><<<dim3((unsigned)((nrows + 16 * RA - 1) / (16 * RA)), ncolt), 256, 0, st>>>(
                static_cast<const double2*>(Y), ldy, static_cast<const float2*>(qo), dq, nrows, nvec, static_cast<double2*>(Yout), ldo);
        }
    } else {
        rr_split_q_kernel<double2><<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(static_cast<const double2*>(Q), nvec, dq, static_cast<double2*>(qo));
        rc = rr_cuda(cudaGetLastError(), "rr_rotate split");
        if (rc != CHFSI_OK) return rc;
        count_launch();
        if (nrows > 0) {
            constexpr int RA = 4;
            rr_rotate_kernel<double, double2, RA><<<dim3((unsigned)((nrows + 16 * RA - 1) / (16 * RA)), ncolt), 256, 0, st>>>(
                static_cast<const double2*>(Y), ldy, static_cast<const double2*>(qo), dq, nrows, nvec, static_cast<double2*>(Yout), ldo);
        }
    }
    rc = rr_cuda(cudaGetLastError(), "rr_rotate");
    if (rc != CHFSI_OK) return rc;
    count_launch();
    return CHFSI_OK;
}

}  // extern "C"

// ---- chfsi_rr_rotate_static: the rotation for callers that cannot allocate (CUDA graph capture, serving loops) ---------
// The split-Q scratch of chfsi_rr_rotate (dq + Q with a zero diagonal) lives in this file-scope device array instead of a
// caller buffer: kRrStaticBytes = what the FP64 and FP32 paths need at CHFSI_RR_STATIC_MAX_NVEC = 4,203,008 bytes, held by every
// GPU that loads the library until the process exits.  In host code the array's NAME is a host-side stand-in, not a device
// address; the device address is resolved once per device with cudaGetSymbolAddress (that device current) and cached.
constexpr size_t kRrStaticBytes = (size_t)CHFSI_RR_STATIC_MAX_NVEC * CHFSI_RR_STATIC_MAX_NVEC * 16 + (size_t)CHFSI_RR_STATIC_MAX_NVEC * 16 + 512;
static __device__ __align__(256) unsigned char g_rr_static_scratch[kRrStaticBytes];

constexpr int kRrMaxDevices = 64;
static std::mutex g_rr_static_mu;
static void* g_rr_static_ptr[kRrMaxDevices] = {};

// device address of g_rr_static_scratch on the current device (resolved on the first call per device)
static chfsi_status rr_static_scratch(void** out) {
    int dev = -1;
    chfsi_status rc = rr_cuda(cudaGetDevice(&dev), "rr_rotate_static: cudaGetDevice");
    if (rc != CHFSI_OK) return rc;
    if (dev < 0 || dev >= kRrMaxDevices) return rr_fail(CHFSI_EUNSUPPORTED, "rr_rotate_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lk(g_rr_static_mu);
    if (g_rr_static_ptr[dev] == nullptr) {
        void* p = nullptr;
        rc = rr_cuda(cudaGetSymbolAddress(&p, g_rr_static_scratch), "rr_rotate_static: cudaGetSymbolAddress");
        if (rc != CHFSI_OK) return rc;
        if (p == nullptr || ((uintptr_t)p & 255)) return rr_fail(CHFSI_ECUDA, "rr_rotate_static: scratch symbol has no 256-byte aligned device address");
        g_rr_static_ptr[dev] = p;
    }
    *out = g_rr_static_ptr[dev];
    return CHFSI_OK;
}

extern "C" chfsi_status chfsi_rr_rotate_static(chfsi_prec prec, long long nrows, int nvec, const void* Y, long long ldy, const void* Q,
                                               void* Yout, long long ldo, void* cuda_stream) {
    if (prec != CHFSI_FP64 && prec != CHFSI_FP32)
        return rr_fail(CHFSI_EUNSUPPORTED, "rr_rotate_static: prec must be CHFSI_FP64 or CHFSI_FP32 (the static scratch holds the split Q of those two paths only)");
    if (nvec > CHFSI_RR_STATIC_MAX_NVEC)
        return rr_fail(CHFSI_EINVAL, "rr_rotate_static: nvec exceeds CHFSI_RR_STATIC_MAX_NVEC (512), the size of the library's static "
                                     "scratch; use chfsi_rr_rotate with a caller workspace");
    void* work = nullptr;
    const chfsi_status rc = rr_static_scratch(&work);
    if (rc != CHFSI_OK) return rc;
    // Nothing in the scratch has to start at zero: rr_split_q_kernel overwrites dq[0, nvec) and all nvec^2 entries of Qo
    // (zero diagonal included) before rr_rotate_kernel reads them, on the same stream; the last call's contents beyond
    // that range are never read.  chfsi_rr_rotate itself allocates nothing (two kernel launches on `cuda_stream`).
    return chfsi_rr_rotate(prec, nrows, nvec, Y, ldy, Q, Yout, ldo, work, kRrStaticBytes, cuda_stream);
}
