// Matrix-free Poisson solve (eq. 5-6; the Kx kernel and Algorithm 2) on sm_100a.
//
// B200-first shape of it: eq. 6 has one Poisson problem per atom, so the solver is *batched* -- the 4 nvec real columns of a
// spinor-layout block (re / im of both components of nvec complex vectors) are 4 nvec independent right-hand sides, each with
// its own alpha, beta and convergence flag.  The Kx kernel is the library's dominant cell kernel (TMA gather + sum-factorised
// Laplacian + RED assembly, cell_march.cu / cell_xyz.cu) run on a handle whose Hamiltonian is the bare Laplacian: K = 2 x
// (kinetic part), and its fused R-term gives the Chebyshev residual r - K z in the same pass.  The scalars of Algorithm 2 live
// on the device (no host round trip per iteration; the host only looks at the count of unconverged columns every
// `check_every` iterations), the two dot products of line 6 are one kernel, lines 4 and 9 are one pass each, and each
// Chebyshev step is [Kx with fused residual] + [one fused pass: diagonal scaling, direction rescaling, accumulation]
// (PAPER.md:195).  All FP64.
#include <cmath>
#include <cstdint>
#include <new>
#include <vector>

#include "chfsi_internal.h"

namespace chfsi {

// A block is [2 M rows][ld complex]; seen as doubles a (node, spin) row holds 2 nvec values.  Column id of (spin s, vector v,
// part ri): cid = (s nvec + v) 2 + ri = s * 2 nvec + pos, pos = 2 v + ri the position inside the row.
struct PScal {
    double *eta, *delta, *delta_new, *gamma, *alpha, *beta;   // [4 nvec] each
    int *active, *iters, *nactive;                            // [4 nvec], [4 nvec], [1]
};

// out1[cid] += sum_I a b ; out2[cid] += sum_I c d (out2 may be null).  grid.x: node chunks; block: one thread per double of
// a node's two rows (strided when 4 nvec > blockDim).
__global__ void __launch_bounds__(512) pois_dot_kernel(const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ c,
                                                       const double* __restrict__ d, long long ld, int nvec, long long nnodes,
                                                       long long nodes_per_block, double* __restrict__ out1, double* __restrict__ out2) {
    const long long I0 = (long long)blockIdx.x * nodes_per_block;
    const long long I1 = I0 + nodes_per_block < nnodes ? I0 + nodes_per_block : nnodes;
    for (int col = threadIdx.x; col < 4 * nvec; col += blockDim.x) {
        const int s = col / (2 * nvec), pos = col - s * 2 * nvec;
        double s1 = 0.0, s2 = 0.0;
        for (long long I = I0; I < I1; ++I) {
            const long long o = (2 * I + s) * 2 * ld + pos;
            s1 = fma(a[o], b[o], s1);
            if (out2) s2 = fma(c[o], d[o], s2);
        }
        atomicAdd(out1 + col, s1);
        if (out2) atomicAdd(out2 + col, s2);
    }
}

// Lines 3, 8, 10 of Algorithm 2 on the device.  stage 0: alpha = delta / eta (0 for finished columns).
// stage 1: beta = delta_new / delta, delta <- delta_new, active <- sqrt(gamma) >= tol, iteration counters.
__global__ void pois_scalar_kernel(PScal sc, int ncol, int stage, double tol) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncol) return;
    if (stage == 0) {
        sc.alpha[c] = (sc.active[c] && sc.eta[c] != 0.0) ? sc.delta[c] / sc.eta[c] : 0.0;
        sc.eta[c] = 0.0;
    } else {
        const int act = sc.active[c];
        sc.beta[c] = (act && sc.delta[c] != 0.0) ? sc.delta_new[c] / sc.delta[c] : 0.0;
        if (act) { sc.delta[c] = sc.delta_new[c]; sc.iters[c] += 1; }
        const int still = act && sqrt(sc.gamma[c]) >= tol;
        sc.active[c] = still;
        sc.delta_new[c] = 0.0;
        if (still) atomicAdd(sc.nactive, 1);
    }
}

// element-wise passes over a block; MODE selects the fused update
enum PoisPass : int {
    PP_XR = 0,      // line 4: x += alpha p, r += alpha w
    PP_P = 1,       // line 9: p = -z + beta p (finished columns keep p)
    PP_CHEB0 = 2,   // Chebyshev start: d = r / (theta kd), z = d
    PP_CHEB = 3,    // Chebyshev step:  d = c1 d + c2 t / kd, z += d       (t = r - K z from the Kx pass)
    PP_INIT = 4,    // r = -f, x = 0
    PP_SHIFT = 5    // x -= shift[cid]  (zero mass-weighted mean)
};

template <int MODE>
__global__ void __launch_bounds__(256) pois_pass_kernel(double* __restrict__ A, double* __restrict__ Bv, const double* __restrict__ Cv,
                                                        const double* __restrict__ Dv, long long lda, long long ldc, int nvec, long long nnodes,
                                                        const double* __restrict__ kd, const double* __restrict__ coef, const int* __restrict__ active,
                                                        double c1, double c2) {
    // one thread per double of a (node, spin) row; A, Bv have leading dimension lda, Cv, Dv ldc
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long per_row = 2ll * nvec;
    if (idx >= 2 * nnodes * per_row) return;
    const long long row = idx / per_row;
    const int pos = (int)(idx - row * per_row);
    const int cid = (int)(row & 1) * 2 * nvec + pos;
    const long long oa = row * 2 * lda + pos, oc = row * 2 * ldc + pos;
    if (MODE == PP_XR) {
        const double al = coef[cid];
        A[oa] = fma(al, Cv[oc], A[oa]);           // x += alpha p   (A = x, Cv = p)
        Bv[oc] = fma(al, Dv[oc], Bv[oc]);         // r += alpha w   (Bv = r, Dv = w)
    } else if (MODE == PP_P) {
        if (active[cid]) A[oa] = fma(coef[cid], A[oa], -Cv[oc]);      // A = p, Cv = z
    } else if (MODE == PP_CHEB0) {
        const double v = Cv[oc] / (c1 * kd[row >> 1]);                 // c1 = theta; Cv = r; A = d, Bv = z
        A[oa] = v; Bv[oa] = v;
    } else if (MODE == PP_CHEB) {
        const double v = fma(c1, A[oa], c2 * Cv[oc] / kd[row >> 1]);   // A = d, Bv = z, Cv = t
        A[oa] = v; Bv[oa] += v;
    } else if (MODE == PP_INIT) {
        A[oa] = 0.0;                              // A = x
        Bv[oc] = -Cv[oc];                         // Bv = r (ldc), Cv = f ... f uses ldc as well (see the driver)
    } else {
        A[oa] -= coef[cid];
    }
}

// sum_I m_I x_I per column (for the zero-mean shift): out[cid] += ...
__global__ void __launch_bounds__(512) pois_wsum_kernel(const double* __restrict__ x, long long ld, int nvec, long long nnodes, long long nodes_per_block,
                                                        const double* __restrict__ mass, double* __restrict__ out) {
    const long long I0 = (long long)blockIdx.x * nodes_per_block;
    const long long I1 = I0 + nodes_per_block < nnodes ? I0 + nodes_per_block : nnodes;
    for (int col = threadIdx.x; col < 4 * nvec; col += blockDim.x) {
        const int s = col / (2 * nvec), pos = col - s * 2 * nvec;
        double acc = 0.0;
        for (long long I = I0; I < I1; ++I) acc = fma(mass[I], x[(2 * I + s) * 2 * ld + pos], acc);
        atomicAdd(out + col, acc);
    }
}
__global__ void pois_shift_scalar_kernel(double* s, int ncol, double inv_total) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < ncol) s[c] *= inv_total;
}
__global__ void pois_fill_kernel(double* p, long long n, double v) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}
__global__ void pois_filli_kernel(int* p, int n, int v) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

}  // namespace chfsi

using namespace chfsi;

static chfsi_status pfail(chfsi_status st, const char* msg) { set_error(msg); return st; }
#define PCU(call)                                                                      \
    do {                                                                               \
        cudaError_t e_ = (call);                                                       \
        if (e_ != cudaSuccess) { set_error(std::string(#call) + ": " + cudaGetErrorString(e_)); return CHFSI_ECUDA; } \
    } while (0)

static size_t al256(size_t b) { return (b + 255) / 256 * 256; }

static chfsi_status poisson_check(const chfsi_mesh* m, int nvec, const char* who) {
    if (!m) return pfail(CHFSI_EINVAL, "poisson: mesh is NULL");
    if (!m->ham_set || !m->bare_laplacian || !m->dKdiag || (m->poisson_rule == 1 && (!m->gl || !m->dKdiagGL)))
        return pfail(CHFSI_ESTATE, "poisson: the handle's Hamiltonian must be the bare Laplacian (chfsi_ham_set with NULL fields and no atoms)");
    if (m->mc.has_phase) return pfail(CHFSI_EINVAL, "poisson: real periodic fields only (kfrac must be 0)");
    if (nvec < 1) return pfail(CHFSI_EINVAL, "poisson: nvec must be >= 1");
    (void)who;
    return CHFSI_OK;
}

// W (+)= cH * 2 * (kinetic part)(U) + cR R through the library's cell kernel
static chfsi_status kx_launch(const chfsi_mesh* m, int nvec, const double* U, long long ldu, double* W, long long ldw, double cH,
                              const double* R, long long ldr, const double* ones, cudaStream_t st) {
    if (m->poisson_rule == 1) {
        // the paper's Gauss-Legendre Kx (poisson_gl.cu): W (zeroed by the caller) = R + cH K U
        if (R) {
            PCU(cudaMemcpy2DAsync(W, (size_t)ldw * 16, R, (size_t)ldr * 16, (size_t)nvec * 16, (size_t)2 * m->nnodes, cudaMemcpyDeviceToDevice, st));
            count_launch();
        }
        const cudaError_t e = launch_kx_gl(m, *m->gl, nvec, U, ldu, W, ldw, cH, st);
        if (e != cudaSuccess) { set_error(std::string("poisson Kx (Gauss-Legendre): ") + cudaGetErrorString(e)); return CHFSI_ECUDA; }
        return CHFSI_OK;
    }
    CellArgs ca{};
    ca.in = U; ca.ld_in = ldu; ca.out = W; ca.ld_out = ldw;
    ca.R = R; ca.ld_R = ldr; ca.cin = nullptr; ca.cR = R ? ones : nullptr;
    ca.cH = 2.0 * cH; ca.nvec = nvec; ca.flags = 0;
    const cudaError_t e = launch_cell(m, CHFSI_FP64, ca, st);
    if (e != cudaSuccess) { set_error(std::string("poisson Kx: ") + cudaGetErrorString(e)); return CHFSI_ECUDA; }
    return CHFSI_OK;
}

extern "C" {

chfsi_status chfsi_poisson_kdiag(const chfsi_mesh* m, double* kdiag_host) {
    if (!m || !kdiag_host) return pfail(CHFSI_EINVAL, "poisson_kdiag: NULL argument");
    if (!m->dKdiag) return pfail(CHFSI_ESTATE, "poisson_kdiag: chfsi_ham_set has not been called");
    const double* src = m->poisson_rule == 1 ? m->dKdiagGL : m->dKdiag;
    if (!src) return pfail(CHFSI_ESTATE, "poisson_kdiag: no diagonal for the selected quadrature");
    PCU(cudaMemcpy(kdiag_host, src, (size_t)m->nnodes * sizeof(double), cudaMemcpyDeviceToHost));
    return CHFSI_OK;
}

chfsi_status chfsi_poisson_set_quadrature(chfsi_mesh* m, int rule) {
    if (!m) return pfail(CHFSI_EINVAL, "poisson_set_quadrature: mesh is NULL");
    if (rule != 0 && rule != 1) return pfail(CHFSI_EINVAL, "poisson_set_quadrature: rule must be 0 (GLL) or 1 (Gauss-Legendre)");
    if (rule == 1 && !m->gl) {
        if (m->nc[0] < 2 || m->nc[1] < 2 || m->nc[2] < 2) return pfail(CHFSI_EINVAL, "poisson_set_quadrature: needs at least two cells per direction");
        GlTables* tb = new (std::nothrow) GlTables;
        if (!tb) return pfail(CHFSI_ENOMEM, "poisson_set_quadrature: out of host memory");
        std::vector<double> k1, m1;
        if (!build_gl_tables(m, *tb, &k1, &m1)) { delete tb; return pfail(CHFSI_ECUDA, "poisson_set_quadrature: table construction failed"); }
        // diag(K): K_e = sum_d coef_d K1 (x) M1 (x) M1 is separable, so the assembled diagonal is a sum of products of assembled 1-D diagonals
        const int p = m->p;
        std::vector<double> ka[3], ma[3];
        for (int d = 0; d < 3; ++d) {
            const int n1 = m->mc.n1[d];
            ka[d].assign(n1, 0.0); ma[d].assign(n1, 0.0);
            for (int g = 0; g < n1; ++g) {
                const int a = g % p;
                ka[d][g] = k1[a] + (a == 0 ? k1[p] : 0.0);
                ma[d][g] = m1[a] + (a == 0 ? m1[p] : 0.0);
            }
        }
        std::vector<double> kd((size_t)m->nnodes);
        const int nx = m->mc.n1[0], ny = m->mc.n1[1], nz = m->mc.n1[2];
        for (int iz = 0; iz < nz; ++iz)
            for (int iy = 0; iy < ny; ++iy)
                for (int ix = 0; ix < nx; ++ix)
                    kd[((size_t)iz * ny + iy) * nx + ix] = tb->coef[0] * ka[0][ix] * ma[1][iy] * ma[2][iz] + tb->coef[1] * ma[0][ix] * ka[1][iy] * ma[2][iz] +
                                                          tb->coef[2] * ma[0][ix] * ma[1][iy] * ka[2][iz];
        int prev = 0;
        cudaGetDevice(&prev); cudaSetDevice(m->device);
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&m->dKdiagGL), kd.size() * sizeof(double));
        if (e == cudaSuccess) e = cudaMemcpy(m->dKdiagGL, kd.data(), kd.size() * sizeof(double), cudaMemcpyHostToDevice);
        cudaSetDevice(prev);
        if (e != cudaSuccess) { delete tb; set_error(std::string("poisson_set_quadrature: ") + cudaGetErrorString(e)); return CHFSI_ECUDA; }
        m->gl = tb;
    }
    m->poisson_rule = rule;
    return CHFSI_OK;
}

chfsi_status chfsi_poisson_apply_K(const chfsi_mesh* m, int nvec, const void* U, long long ldu, void* W, long long ldw, void* cuda_stream) {
    chfsi_status rc = poisson_check(m, nvec, "poisson_apply_K");
    if (rc != CHFSI_OK) return rc;
    if (!U || !W || U == W) return pfail(CHFSI_EINVAL, "poisson_apply_K: NULL or aliased device pointers");
    if (ldu < nvec || ldw < nvec) return pfail(CHFSI_EINVAL, "poisson_apply_K: leading dimension < nvec");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    PCU(cudaMemset2DAsync(W, (size_t)ldw * 16, 0, (size_t)nvec * 16, (size_t)2 * m->nnodes, st));
    count_launch();
    return kx_launch(m, nvec, static_cast<const double*>(U), ldu, static_cast<double*>(W), ldw, 1.0, nullptr, 0, nullptr, st);
}

chfsi_status chfsi_poisson_workspace_bytes(const chfsi_mesh* m, int nvec, size_t* bytes) {
    if (!m || !bytes || nvec < 1) return pfail(CHFSI_EINVAL, "poisson_workspace_bytes: bad argument");
    const size_t vec = al256((size_t)2 * m->nnodes * nvec * 16);
    *bytes = 5 * vec + al256((size_t)nvec * 8) + 8 * al256((size_t)4 * nvec * 8) + 256;
    return CHFSI_OK;
}

chfsi_status chfsi_poisson_pcg(const chfsi_mesh* m, int nvec, const void* F, long long ldf, void* X, long long ldx, int cheb_degree,
                               double lmin, double lmax, double tol, int maxit, int check_every, void* work, size_t work_bytes,
                               int* iters_host, double* resnorm_host, void* cuda_stream) {
    chfsi_status rc = poisson_check(m, nvec, "poisson_pcg");
    if (rc != CHFSI_OK) return rc;
    if (!F || !X || !work || F == X) return pfail(CHFSI_EINVAL, "poisson_pcg: NULL or aliased device pointers");
    if (ldf < nvec || ldx < nvec) return pfail(CHFSI_EINVAL, "poisson_pcg: leading dimension < nvec");
    if (cheb_degree < 1 || cheb_degree > 64) return pfail(CHFSI_EINVAL, "poisson_pcg: cheb_degree must be in 1..64");
    if (!(lmax > lmin) || !(lmin > 0.0)) return pfail(CHFSI_EINVAL, "poisson_pcg: need 0 < lmin < lmax");
    if (!(tol > 0.0) || maxit < 0 || check_every < 0) return pfail(CHFSI_EINVAL, "poisson_pcg: bad tol / maxit / check_every");
    size_t need = 0;
    chfsi_poisson_workspace_bytes(m, nvec, &need);
    if (work_bytes < need || ((uintptr_t)work & 255)) return pfail(CHFSI_EINVAL, "poisson_pcg: work too small or not 256-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const long long M = m->nnodes;
    const int ncol = 4 * nvec;
    const size_t vec = al256((size_t)2 * M * nvec * 16);
    char* wp = static_cast<char*>(work);
    double* r = reinterpret_cast<double*>(wp); wp += vec;        // all work vectors have ld = nvec
    double* p = reinterpret_cast<double*>(wp); wp += vec;
    double* w = reinterpret_cast<double*>(wp); wp += vec;        // also t = r - K z inside the preconditioner
    double* z = reinterpret_cast<double*>(wp); wp += vec;
    double* d = reinterpret_cast<double*>(wp); wp += vec;
    double* ones = reinterpret_cast<double*>(wp); wp += al256((size_t)nvec * 8);
    PScal sc;
    const size_t sb = al256((size_t)ncol * 8);
    sc.eta = reinterpret_cast<double*>(wp); wp += sb;
    sc.delta = reinterpret_cast<double*>(wp); wp += sb;
    sc.delta_new = reinterpret_cast<double*>(wp); wp += sb;
    sc.gamma = reinterpret_cast<double*>(wp); wp += sb;
    sc.alpha = reinterpret_cast<double*>(wp); wp += sb;
    sc.beta = reinterpret_cast<double*>(wp); wp += sb;
    sc.active = reinterpret_cast<int*>(wp); wp += sb;
    sc.iters = reinterpret_cast<int*>(wp); wp += sb;
    sc.nactive = reinterpret_cast<int*>(wp);
    double* x = static_cast<double*>(X);
    const double* f = static_cast<const double*>(F);
    const long long nelem = 2 * M * 2 * nvec;
    const unsigned gpass = (unsigned)((nelem + 255) / 256);
    const unsigned gsc = (unsigned)((ncol + 127) / 128);
    long long npb = (M + 148 * 8 - 1) / (148 * 8);
    if (npb < 1) npb = 1;
    const unsigned gdot = (unsigned)((M + npb - 1) / npb);
    const int tdot = ncol < 512 ? ((ncol + 31) / 32) * 32 : 512;
    const double theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin), sigma = theta / delta;
    const double* kdiag = m->poisson_rule == 1 ? m->dKdiagGL : m->dKdiag;

    // z = P^-1 r: Chebyshev-Jacobi, cheb_degree - 1 applications of K
    auto precondition = [&]() -> chfsi_status {
        pois_pass_kernel<PP_CHEB0><<<gpass, 256, 0, st>>>(d, z, r, nullptr, nvec, nvec, nvec, M, kdiag, nullptr, nullptr, theta, 0.0);
        count_launch();
        double rho = 1.0 / sigma;
        for (int k = 1; k < cheb_degree; ++k) {
            const double rho_new = 1.0 / (2.0 * sigma - rho);
            PCU(cudaMemsetAsync(w, 0, (size_t)2 * M * nvec * 16, st)); count_launch();
            chfsi_status s2 = kx_launch(m, nvec, z, nvec, w, nvec, -1.0, r, nvec, ones, st);      // t = r - K z in one pass
            if (s2 != CHFSI_OK) return s2;
            pois_pass_kernel<PP_CHEB><<<gpass, 256, 0, st>>>(d, z, w, nullptr, nvec, nvec, nvec, M, kdiag, nullptr, nullptr,
                                                              rho_new * rho, 2.0 * rho_new / delta);
            count_launch();
            rho = rho_new;
        }
        return CHFSI_OK;
    };

    pois_fill_kernel<<<(unsigned)((nvec + 127) / 128), 128, 0, st>>>(ones, nvec, 1.0);
    PCU(cudaMemsetAsync(sc.eta, 0, 6 * sb, st));                           // eta .. beta
    pois_filli_kernel<<<gsc, 128, 0, st>>>(sc.active, ncol, 1);
    PCU(cudaMemsetAsync(sc.iters, 0, sb, st));
    // x = 0, r = K x - f = -f  (f is read with its own leading dimension: strided copy first)
    PCU(cudaMemcpy2DAsync(w, (size_t)nvec * 16, f, (size_t)ldf * 16, (size_t)nvec * 16, (size_t)2 * M, cudaMemcpyDeviceToDevice, st));
    PCU(cudaMemset2DAsync(x, (size_t)ldx * 16, 0, (size_t)nvec * 16, (size_t)2 * M, st));
    pois_pass_kernel<PP_INIT><<<gpass, 256, 0, st>>>(d, r, w, nullptr, nvec, nvec, nvec, M, nullptr, nullptr, nullptr, 0.0, 0.0);   // d is scratch here
    count_launch(5);
    rc = precondition();
    if (rc != CHFSI_OK) return rc;
    // p = -z, delta = r . z, gamma = |r|^2, active = sqrt(gamma) >= tol
    PCU(cudaMemsetAsync(p, 0, (size_t)2 * M * nvec * 16, st));
    pois_pass_kernel<PP_P><<<gpass, 256, 0, st>>>(p, nullptr, z, nullptr, nvec, nvec, nvec, M, nullptr, sc.beta, sc.active, 0.0, 0.0);   // beta = 0
    pois_dot_kernel<<<gdot, tdot, 0, st>>>(r, z, r, r, nvec, nvec, M, npb, sc.delta, sc.gamma);
    PCU(cudaMemsetAsync(sc.nactive, 0, sizeof(int), st));
    // stage 1 with delta_new = 0 would clobber delta: seed delta_new = delta first
    PCU(cudaMemcpyAsync(sc.delta_new, sc.delta, (size_t)ncol * 8, cudaMemcpyDeviceToDevice, st));
    pois_scalar_kernel<<<gsc, 128, 0, st>>>(sc, ncol, 1, tol);
    PCU(cudaMemsetAsync(sc.iters, 0, sb, st));                             // the seeding pass is not an iteration
    count_launch(6);

    int it = 0, h_nactive = 1;
    for (; it < maxit; ++it) {
        if (check_every > 0 && it % check_every == 0) {
            PCU(cudaMemcpyAsync(&h_nactive, sc.nactive, sizeof(int), cudaMemcpyDeviceToHost, st));
            PCU(cudaStreamSynchronize(st));
            if (h_nactive == 0) break;
        }
        PCU(cudaMemsetAsync(w, 0, (size_t)2 * M * nvec * 16, st));
        rc = kx_launch(m, nvec, p, nvec, w, nvec, 1.0, nullptr, 0, nullptr, st);                    // 1: w = K p
        if (rc != CHFSI_OK) return rc;
        pois_dot_kernel<<<gdot, tdot, 0, st>>>(p, w, nullptr, nullptr, nvec, nvec, M, npb, sc.eta, nullptr);   // 2: eta = p . w
        pois_scalar_kernel<<<gsc, 128, 0, st>>>(sc, ncol, 0, tol);                                  // 3: alpha = delta / eta
        pois_pass_kernel<PP_XR><<<gpass, 256, 0, st>>>(x, r, p, w, ldx, nvec, nvec, M, nullptr, sc.alpha, nullptr, 0.0, 0.0);   // 4
        count_launch(4);
        rc = precondition();                                                                        // 5: z = P^-1 r
        if (rc != CHFSI_OK) return rc;
        PCU(cudaMemsetAsync(sc.gamma, 0, sb, st));
        PCU(cudaMemsetAsync(sc.nactive, 0, sizeof(int), st));
        pois_dot_kernel<<<gdot, tdot, 0, st>>>(r, z, r, r, nvec, nvec, M, npb, sc.delta_new, sc.gamma);    // 6: (delta_new, gamma)
        pois_scalar_kernel<<<gsc, 128, 0, st>>>(sc, ncol, 1, tol);                                  // 8, 10
        pois_pass_kernel<PP_P><<<gpass, 256, 0, st>>>(p, nullptr, z, nullptr, nvec, nvec, nvec, M, nullptr, sc.beta, sc.active, 0.0, 0.0);   // 9
        count_launch(5);
    }
    // zero mass-weighted mean (reading P1)
    PCU(cudaMemsetAsync(sc.eta, 0, sb, st));
    pois_wsum_kernel<<<gdot, tdot, 0, st>>>(x, ldx, nvec, M, npb, m->dMass, sc.eta);
    const double total = m->L[0] * m->L[1] * m->L[2];                      // sum of the node masses = the box volume
    pois_shift_scalar_kernel<<<gsc, 128, 0, st>>>(sc.eta, ncol, 1.0 / total);
    pois_pass_kernel<PP_SHIFT><<<gpass, 256, 0, st>>>(x, nullptr, nullptr, nullptr, ldx, nvec, nvec, M, nullptr, sc.eta, nullptr, 0.0, 0.0);
    count_launch(4);
    if (iters_host || resnorm_host) {
        std::vector<double> g((size_t)ncol);
        std::vector<int> iv((size_t)ncol);
        PCU(cudaMemcpyAsync(g.data(), sc.gamma, (size_t)ncol * 8, cudaMemcpyDeviceToHost, st));
        PCU(cudaMemcpyAsync(iv.data(), sc.iters, (size_t)ncol * 4, cudaMemcpyDeviceToHost, st));
        PCU(cudaStreamSynchronize(st));
        for (int c = 0; c < ncol; ++c) {
            if (iters_host) iters_host[c] = iv[(size_t)c];
            if (resnorm_host) resnorm_host[c] = std::sqrt(g[(size_t)c]);
        }
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("poisson_pcg: ") + cudaGetErrorString(e)); return CHFSI_ECUDA; }
    return CHFSI_OK;
}

}  // extern "C"
