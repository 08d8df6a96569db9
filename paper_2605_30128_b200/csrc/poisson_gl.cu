// The paper's Kx formulation: "extracts the FE cell-level nodal values ..., then performs six batched tensor
// contractions covering interpolation of nodal values to quadrature points, application of the per-cell Jacobian, and integration
// back to the nodal basis, and finally assembles the cell contributions back into the global output vector" -- with p + 1
// Gauss-Legendre points per direction.  Selected by chfsi_poisson_set_quadrature(mesh, 1); the default Poisson operator is the
// GLL-collocated Laplacian of the filter (reading P2).  One CTA = one cell x one 64-byte group of real columns (4 complex
// vectors of one spin row); the cell tile lives in shared memory, a thread owns whole lines of it (values stay in registers
// along the line, "hybrid register-shared memory strategy"); the last stage is fused with the assembly by RED
// (PAPER.md:192).  Not tuned like the filter's cell kernels: it exists so that the paper's operator is built and checked.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <utility>
#include <vector>

#include "chfsi_internal.h"

namespace chfsi {

constexpr int kCB = 8;          // real columns per CTA: 64 bytes of a (node, spin) row

// one 1-D pass over the tile T[n^3][kCB]: along direction dir (0 = x fastest), out = M v or M^T v, in place
template <int P, bool TRANS>
__device__ __forceinline__ void gl_pass(double* T, const double (*M)[kMaxN], int dir) {
    constexpr int n = P + 1;
    const int stride = dir == 0 ? 1 : dir == 1 ? n : n * n;
    for (int task = threadIdx.x; task < n * n * kCB; task += blockDim.x) {
        const int col = task % kCB, line = task / kCB;
        const int i1 = line % n, i2 = line / n;
        const int base = dir == 0 ? (i2 * n + i1) * n : dir == 1 ? i2 * n * n + i1 : i2 * n + i1;
        double v[n], o[n];
#pragma unroll
        for (int j = 0; j < n; ++j) v[j] = T[(base + j * stride) * kCB + col];
#pragma unroll
        for (int i = 0; i < n; ++i) {
            double acc = 0.0;
#pragma unroll
            for (int j = 0; j < n; ++j) acc = fma(TRANS ? M[j][i] : M[i][j], v[j], acc);
            o[i] = acc;
        }
#pragma unroll
        for (int i = 0; i < n; ++i) T[(base + i * stride) * kCB + col] = o[i];
    }
}

template <int P>
__global__ void __launch_bounds__(256) pois_kx_gl_kernel(const __grid_constant__ GlTables tb, const double* __restrict__ U, long long ldu,
                                                         double* __restrict__ W, long long ldw, int nvec, double cH) {
    constexpr int n = P + 1, n3 = n * n * n;
    extern __shared__ double sm[];
    double* T0 = sm;                    // nodal values -> values at the Gauss points
    double* T1 = sm + n3 * kCB;         // integrated gradient terms
    __shared__ double Bs[kMaxN][kMaxN], Ds[kMaxN][kMaxN];
    for (int i = threadIdx.x; i < kMaxN * kMaxN; i += blockDim.x) { Bs[i / kMaxN][i % kMaxN] = tb.Bm[i / kMaxN][i % kMaxN]; Ds[i / kMaxN][i % kMaxN] = tb.Dq[i / kMaxN][i % kMaxN]; }
    int e = blockIdx.x;
    const int ex = e % tb.nc[0]; e /= tb.nc[0];
    const int ey = e % tb.nc[1], ez = e / tb.nc[1];
    const int groups = (2 * nvec + kCB - 1) / kCB;             // 64-byte groups per (node, spin) row
    const int s = blockIdx.y / groups, pos0 = (blockIdx.y % groups) * kCB;
    // (i) extraction through the local-to-global map (periodic wrap)
    for (int idx = threadIdx.x; idx < n3 * kCB; idx += blockDim.x) {
        const int col = idx % kCB, node = idx / kCB;
        const int a = node % n, b = (node / n) % n, c = node / (n * n);
        int gx = ex * P + a, gy = ey * P + b, gz = ez * P + c;
        if (gx == tb.n1[0]) gx = 0;
        if (gy == tb.n1[1]) gy = 0;
        if (gz == tb.n1[2]) gz = 0;
        const long long I = ((long long)gz * tb.n1[1] + gy) * tb.n1[0] + gx;
        T0[idx] = pos0 + col < 2 * nvec ? U[(2 * I + s) * 2 * ldu + pos0 + col] : 0.0;
    }
    __syncthreads();
    // (ii) interpolation to the Gauss points: three contractions with the value matrix
    for (int d = 0; d < 3; ++d) { gl_pass<P, false>(T0, Bs, d); __syncthreads(); }
    // gradient at the Gauss points, Jacobian and quadrature weights, transposed gradient: per direction, line by line
    for (int d = 0; d < 3; ++d) {
        const int stride = d == 0 ? 1 : d == 1 ? n : n * n;
        for (int task = threadIdx.x; task < n * n * kCB; task += blockDim.x) {
            const int col = task % kCB, line = task / kCB;
            const int i1 = line % n, i2 = line / n;
            const int base = d == 0 ? (i2 * n + i1) * n : d == 1 ? i2 * n * n + i1 : i2 * n + i1;
            const double w2 = tb.wq[i1] * tb.wq[i2] * tb.coef[d];
            double v[n], g[n];
#pragma unroll
            for (int j = 0; j < n; ++j) v[j] = T0[(base + j * stride) * kCB + col];
#pragma unroll
            for (int q = 0; q < n; ++q) {
                double acc = 0.0;
#pragma unroll
                for (int j = 0; j < n; ++j) acc = fma(Ds[q][j], v[j], acc);
                g[q] = acc * tb.wq[q] * w2;
            }
#pragma unroll
            for (int j = 0; j < n; ++j) {
                double acc = 0.0;
#pragma unroll
                for (int q = 0; q < n; ++q) acc = fma(Ds[q][j], g[q], acc);
                double* t = T1 + (base + j * stride) * kCB + col;
                *t = d == 0 ? acc : *t + acc;
            }
        }
        __syncthreads();
    }
    // integration back to the nodal basis: three transposed contractions
    for (int d = 0; d < 3; ++d) { gl_pass<P, true>(T1, Bs, d); __syncthreads(); }
    // (iii) assembly
    for (int idx = threadIdx.x; idx < n3 * kCB; idx += blockDim.x) {
        const int col = idx % kCB, node = idx / kCB;
        if (pos0 + col >= 2 * nvec) continue;
        const int a = node % n, b = (node / n) % n, c = node / (n * n);
        int gx = ex * P + a, gy = ey * P + b, gz = ez * P + c;
        if (gx == tb.n1[0]) gx = 0;
        if (gy == tb.n1[1]) gy = 0;
        if (gz == tb.n1[2]) gz = 0;
        const long long I = ((long long)gz * tb.n1[1] + gy) * tb.n1[0] + gx;
        atomicAdd(W + (2 * I + s) * 2 * ldw + pos0 + col, cH * T1[idx]);
    }
}

// ---- host tables: Gauss-Legendre points by Newton on P_n, Lagrange basis on the GLL nodes evaluated at them
static void legendre_p(int nn, double x, double& Pn, double& dPn) {
    double p0 = 1.0, p1 = x;
    if (nn == 0) { Pn = 1.0; dPn = 0.0; return; }
    for (int k = 1; k < nn; ++k) { const double p2 = ((2 * k + 1) * x * p1 - k * p0) / (k + 1); p0 = p1; p1 = p2; }
    Pn = p1;
    dPn = nn * (x * p1 - p0) / (x * x - 1.0);
}

bool build_gl_tables(const chfsi_mesh* m, GlTables& tb, std::vector<double>* k1_out, std::vector<double>* m1_out) {
    const int p = m->p, n = p + 1;
    std::vector<double> xq(n), wq(n);
    for (int i = 0; i < n; ++i) {
        double x = -std::cos(3.14159265358979323846 * (i + 0.75) / (n + 0.5));
        for (int it = 0; it < 100; ++it) {
            double P, dP;
            legendre_p(n, x, P, dP);
            const double dx = P / dP;
            x -= dx;
            if (std::fabs(dx) < 1e-16) break;
        }
        double P, dP;
        legendre_p(n, x, P, dP);
        xq[i] = x; wq[i] = 2.0 / ((1.0 - x * x) * dP * dP);
    }
    std::memset(&tb, 0, sizeof(tb));
    std::vector<double> Bm(n * n), Gm(n * n);
    const std::vector<double>& xi = m->xi;
    for (int i = 0; i < n; ++i) {
        double den = 1.0;
        for (int j = 0; j < n; ++j) if (j != i) den *= xi[i] - xi[j];
        for (int q = 0; q < n; ++q) {
            double val = 1.0, der = 0.0;
            for (int j = 0; j < n; ++j) if (j != i) val *= xq[q] - xi[j];
            for (int k = 0; k < n; ++k) {
                if (k == i) continue;
                double t = 1.0;
                for (int j = 0; j < n; ++j) if (j != i && j != k) t *= xq[q] - xi[j];
                der += t;
            }
            Bm[q * n + i] = val / den; Gm[q * n + i] = der / den;
        }
    }
    // Dq = G B^-1 (Gauss-Jordan on the (n x n) value matrix)
    std::vector<double> A(Bm), Inv(n * n, 0.0);
    for (int i = 0; i < n; ++i) Inv[i * n + i] = 1.0;
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r) if (std::fabs(A[r * n + c]) > std::fabs(A[piv * n + c])) piv = r;
        if (std::fabs(A[piv * n + c]) < 1e-300) return false;
        for (int k = 0; k < n; ++k) { std::swap(A[c * n + k], A[piv * n + k]); std::swap(Inv[c * n + k], Inv[piv * n + k]); }
        const double d = 1.0 / A[c * n + c];
        for (int k = 0; k < n; ++k) { A[c * n + k] *= d; Inv[c * n + k] *= d; }
        for (int r = 0; r < n; ++r) {
            if (r == c) continue;
            const double f = A[r * n + c];
            for (int k = 0; k < n; ++k) { A[r * n + k] -= f * A[c * n + k]; Inv[r * n + k] -= f * Inv[c * n + k]; }
        }
    }
    for (int q = 0; q < n; ++q)
        for (int r = 0; r < n; ++r) {
            double acc = 0.0;
            for (int i = 0; i < n; ++i) acc += Gm[q * n + i] * Inv[i * n + r];
            tb.Dq[q][r] = acc;
            tb.Bm[q][r] = Bm[q * n + r];
        }
    const double hx = m->L[0] / m->nc[0], hy = m->L[1] / m->nc[1], hz = m->L[2] / m->nc[2];
    const double J = hx * hy * hz / 8.0;
    const double h[3] = {hx, hy, hz};
    for (int d = 0; d < 3; ++d) { tb.coef[d] = J * (2.0 / h[d]) * (2.0 / h[d]); tb.nc[d] = m->nc[d]; tb.n1[d] = m->mc.n1[d]; }
    for (int q = 0; q < n; ++q) tb.wq[q] = wq[q];
    if (k1_out && m1_out) {     // diagonals of the exact 1-D stiffness G^T W G and mass B^T W B
        k1_out->assign(n, 0.0); m1_out->assign(n, 0.0);
        for (int a = 0; a < n; ++a)
            for (int q = 0; q < n; ++q) { (*k1_out)[a] += wq[q] * Gm[q * n + a] * Gm[q * n + a]; (*m1_out)[a] += wq[q] * Bm[q * n + a] * Bm[q * n + a]; }
    }
    return true;
}

cudaError_t launch_kx_gl(const chfsi_mesh* m, const GlTables& tb, int nvec, const double* U, long long ldu, double* W, long long ldw,
                         double cH, cudaStream_t st) {
    const int n = m->p + 1;
    const size_t smem = (size_t)2 * n * n * n * kCB * sizeof(double);
    const int groups = (2 * nvec + kCB - 1) / kCB;
    const dim3 grid((unsigned)(m->nc[0] * m->nc[1] * m->nc[2]), (unsigned)(2 * groups));
#define GL_CASE(PP)                                                                                                        \
    case PP: {                                                                                                             \
        static bool done[32] = {false};                                                                                    \
        if (!done[m->device & 31]) {                                                                                       \
            cudaError_t e = cudaFuncSetAttribute(pois_kx_gl_kernel<PP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
            if (e != cudaSuccess) return e;                                                                                \
            done[m->device & 31] = true;                                                                                   \
        }                                                                                                                  \
        pois_kx_gl_kernel<PP><<<grid, 256, smem, st>>>(tb, U, ldu, W, ldw, nvec, cH);                                      \
        break;                                                                                                             \
    }
    switch (m->p) {
        GL_CASE(1) GL_CASE(2) GL_CASE(3) GL_CASE(4) GL_CASE(5) GL_CASE(6) GL_CASE(7) GL_CASE(8)
        default: return cudaErrorInvalidValue;
    }
#undef GL_CASE
    count_launch();
    return cudaGetLastError();
}

}  // namespace chfsi
