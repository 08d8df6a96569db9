// Internal declarations of libchfsi (sm_100a).  Not part of the C ABI (include/chfsi.h).
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "chfsi.h"

namespace chfsi {

constexpr int kMaxN = 9;        // p + 1 <= 9  (p <= 8)
constexpr int kMaxProj = 16;    // projectors per atom

// Everything a kernel needs to know about the mesh; passed by value (__grid_constant__), so the
// 1-D matrices sit in the constant bank and become immediate operands of the unrolled FMAs.
struct MeshConst {
    int p, n;                   // degree, n = p + 1
    int nc[3];                  // cells per direction
    int n1[3];                  // nodes per direction
    int ncells;
    int has_phase;              // any kfrac != integer
    long long nnodes;
    double Kd[3][kMaxN][kMaxN]; // 0.5 * J * (2/h_d)^2 * Khat[i][a]   (kinetic 1/2 folded in)
    float  Kf[3][kMaxN][kMaxN];
    double w[kMaxN];            // GLL weights
    float  wf[kMaxN];
    double m1[3][kMaxN];        // assembled 1-D mass at cell-local index a: (h_d/2) * (w_a, doubled on faces)
    double im1[3][kMaxN];       // reciprocals
    double ph_re[3], ph_im[3];  // Bloch phases phi_d = exp(2 pi i kfrac_d)
    const double* V;            // node fields (device), never null after ham_set
    const double* Bx;
    const double* By;
    const double* Bz;
};

enum CellFlags : int {
    kScaleIn = 1,     // w = in / m      (Z-form of eq. 11: H D^-1 Z)
    kSoutInvM = 2,    // multiply H w by 1/m   (M^-1 H, eq. 10 and chfsi_apply_H)
    kMassIn = 4,      // the in-term carries m_I  (residual R = H X - M X Lambda)
};

// out += cH * s_out * H(s_in * in) + cin[v] * f * in + cR[v] * R      (accumulated with RED.ADD.F64)
struct CellArgs {
    const double* in;  long long ld_in;     // leading dimensions in complex elements
    double* out;       long long ld_out;
    const double* R;   long long ld_R;      // nullptr: no R term
    const double* cin;                      // [nvec] per-vector coefficient of the in-term (device)
    const double* cR;                       // [nvec] per-vector coefficient of the R-term (device) or nullptr
    double cH;
    int nvec;
    int flags;
    // FP32 product only: `in` is multiplied by this power of two (exactly, in FP64) before the cast to FP32 and the
    // FP32 result by its reciprocal after widening, so that the scaled iterates Z_k / s_k stay
    // inside the FP32 range at any degree.  1.0 (or 0 = unset) elsewhere.
    double in_scale;
    // FP32-stored multivectors (CHFSI_FP32_STORED): `in` and `out` are complex64 (leading dimensions still in
    // complex elements); R stays complex128.
    int store_f32;
};

// tables of the Gauss-Legendre form of the Poisson operator (poisson_gl.cu)
struct GlTables {
    double Bm[kMaxN][kMaxN];    // B[q][i]  = l_i(xq_q): nodal values -> Gauss points
    double Dq[kMaxN][kMaxN];    // Dq[q][r] = collocation derivative at the Gauss points (G B^-1)
    double wq[kMaxN];           // Gauss weights
    double coef[3];             // J (2/h_d)^2
    int nc[3], n1[3];
};

struct ProjItem { int atom; int start; int count; };   // a slice of an atom's support list

struct NonlocalDev {
    int natoms = 0;
    int nitems = 0;
    int max_nproj = 0;
    long long nnz = 0;                  // total support entries
    ProjItem* items = nullptr;          // [nitems]   slices of 8 support nodes
    int nitems_big = 0;
    int uniform_np = 0;                 // nproj if every atom has the same number of projectors, else 0
    ProjItem* items_big = nullptr;      // [nitems_big] slices of 32 support nodes (fast kernels)
    long long* supp_node = nullptr;     // [nnz]
    double* supp_mass = nullptr;        // [nnz] m_I of each support entry
    long long* p_off = nullptr;         // [natoms] offset (in complex elements) of atom's P block
    long long* s_off = nullptr;         // [natoms+1] support offsets
    int* nproj = nullptr;               // [natoms]
    long long* c_off = nullptr;         // [natoms] offset of atom's coefficient rows in Cbuf (units of rows)
    long long* d_off = nullptr;         // [natoms] offset of atom's D matrix (complex elements)
    double2* P64 = nullptr;             // complex128 projector values
    float2* P32 = nullptr;
    double2* D64 = nullptr;
    long long crows = 0;                // sum over atoms of 2*nproj  (rows of Cbuf)
};

struct ProjArgs {
    const void* in; long long ld_in;    // complex128, or complex64 when store_f32
    double* C;                          // [crows][nvec] complex128, zeroed by the driver
    int nvec;
    int mass_u;                         // 1: u = m_I * in (apply on X); 0: u = in (Z-form)
    double in_scale;                    // see CellArgs::in_scale (the back pass gets cH / in_scale)
    int store_f32;
};

struct BackArgs {
    const double* C;                    // projected coefficients
    double* G;                          // scratch for G = D C, same shape as C
    void* out; long long ld_out;        // complex128, or complex64 when store_f32
    double cH;
    int nvec;
    int sout_invm;                      // 1: s_out = 1/m  => m * (1/m) = 1 ; 0: factor m_I
    int store_f32;
};

}  // namespace chfsi

struct chfsi_mesh {
    int device = 0;
    int p = 0;
    int nc[3] = {0, 0, 0};
    double L[3] = {0, 0, 0};
    double kfrac[3] = {0, 0, 0};
    long long nnodes = 0;
    bool ham_set = false;
    int cell_kernel[5] = {0, 0, 0, 0, 0};   // per chfsi_prec: chfsi_cell_kernel choice (0 = default)
    chfsi::MeshConst mc;
    std::vector<double> xi, w;          // host GLL tables
    std::vector<double> m1h[3];         // host assembled 1-D mass per global line index
    double* dV = nullptr;
    double* dBx = nullptr;
    double* dBy = nullptr;
    double* dBz = nullptr;
    double* dF = nullptr;               // packed fields [M][4] = V+Bz, V-Bz, Bx, By (march kernel)
    float* dF32 = nullptr;              // the same rounded to FP32 (FP32-stored mode: its pointwise terms are FP32)
    double* dMass = nullptr;            // node masses m_I [M] (Rayleigh-Ritz projection, Poisson solver); built in chfsi_ham_set
    double* dKdiag = nullptr;           // diag(K) of the stiffness matrix K = 2 x kinetic part [M] (Poisson preconditioner); built in chfsi_ham_set
    double* dKdiagGL = nullptr;         // the same for the Gauss-Legendre form (chfsi_poisson_set_quadrature)
    int poisson_rule = 0;               // 0: GLL collocation (the filter's Laplacian, cell kernel); 1: Gauss-Legendre (the paper's Kx)
    chfsi::GlTables* gl = nullptr;      // host copy of the Gauss-Legendre tables
    bool bare_laplacian = false;        // the Hamiltonian set last has no local fields and no projectors (Poisson handle)
    chfsi::NonlocalDev nl;
    // profiling aid (chfsi_profile_enable / chfsi_profile_read)
    mutable bool prof_on = false;
    mutable std::vector<cudaEvent_t> prof_ev;      // start/stop pairs
    mutable double prof_bytes = 0.0;
    // low-priority side stream: the nonlocal term of a step runs beside the cell kernel and fills the SMs that
    // kernel's last wave leaves idle (created in chfsi_ham_set)
    mutable cudaStream_t side = nullptr;
    mutable cudaEvent_t ev_proj = nullptr, ev_back = nullptr;
    // pinned staging ring for the per-chunk coefficient program of chfsi_cheb_filter (allocated in chfsi_ham_set): the
    // asynchronous upload reads pinned memory owned by the mesh, never a pageable buffer of the caller's stack frame
    static constexpr int kStageSlots = 4;
    static constexpr int kStageLambda = 8192;          // vectors per chunk the ring is sized for
    mutable double* h_stage = nullptr;
    mutable size_t stage_slot_doubles = 0;
    mutable int stage_next = 0;
    mutable cudaEvent_t stage_ev[kStageSlots] = {nullptr, nullptr, nullptr, nullptr};
    mutable bool stage_used[kStageSlots] = {false, false, false, false};
};

namespace chfsi {
// launchers (kernels.cu)
cudaError_t launch_cell(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t s);
cudaError_t launch_proj(const chfsi_mesh* m, chfsi_prec prec, const ProjArgs& a, cudaStream_t s);
cudaError_t launch_back(const chfsi_mesh* m, chfsi_prec prec, const BackArgs& a, cudaStream_t s);
// out[row][v] = ca[v] * (inv_mass ? A/m : A) + cb[v] * B   (B, cb may be null); rows = 2*nnodes
cudaError_t launch_axpby(const chfsi_mesh* m, double* out, long long ldo, const void* A, long long lda, int a_f32,
                         const double* ca, int a_inv_mass, const double* B, long long ldb,
                         const double* cb, int nvec, cudaStream_t s);
// dst (complex64, ld = ldd) = (float) src (complex128, ld = lds): the FP32 copy of Zh_1 = R (CHFSI_FP32_STORED)
cudaError_t launch_cast32(const chfsi_mesh* m, void* dst, long long ldd, const double* src, long long lds, int nvec, cudaStream_t s);
// buf *= f (an exact power of two) on a multivector of nvec columns, ld = nvec (renormalisation of the scaled iterates)
cudaError_t launch_scale(const chfsi_mesh* m, void* buf, int f32, int nvec, double f, cudaStream_t s);
// Per-step coefficient rows.  For vector v with Ritz value lam and the running Lambda_k(v) = L:
//   cin[r][v] = cin0 + cinL * L + cinLam * lam ;  cR[r][v] = cR0 + cRL * L ;
//   then, if advance: L_next = al * lam * L - be * L - ga * L_prev   (Lambda_k recurrence)
struct CoefRow { double cin0, cinL, cinLam, cR0, cRL, al, be, ga, advance; };
// hdr (device): [q0, q1, nrows, pad] then nrows CoefRow, then lam[nvec]; L_0 = 1, L_1 = q0 + q1 * lam.
// table (device): row r = [cin(0..nvec-1), cR(0..nvec-1)]
cudaError_t launch_coef(const double* hdr, double* table, int nrows, int nvec, cudaStream_t s);
bool cell_supported(int p, chfsi_prec prec);
// z-marching TMA kernel (cell_march.cu)
bool march_supported(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a);
cudaError_t launch_cell_march(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t s);
// line-owned x/y/z TMA kernel (cell_xyz.cu)
bool xyz_supported(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a);
// Rayleigh-Ritz rotation on tcgen05 (rr_tc.cu): FP64 diagonal + 3xTF32 off-diagonal; work as laid out by rr_tc_workspace_bytes
size_t rr_tc_workspace_bytes(int nvec);
cudaError_t launch_rr_rotate_tc(long long nrows, int nvec, const void* Y, long long ldy, const void* Q, void* Yout, long long ldo,
                                void* work, cudaStream_t st);
cudaError_t launch_cell_xyz(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t s);
// tensor-core cell kernel (cell_mma.cu): mma.sync TF32 / 3xTF32 on complex64 storage, mma.sync FP64 on complex128 storage
bool mma_supported(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a);
cudaError_t launch_cell_mma(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t s);
// Gauss-Legendre form of the Poisson operator (poisson_gl.cu)
bool build_gl_tables(const chfsi_mesh* m, GlTables& tb, std::vector<double>* k1_out, std::vector<double>* m1_out);
cudaError_t launch_kx_gl(const chfsi_mesh* m, const GlTables& tb, int nvec, const double* U, long long ldu, double* W, long long ldw,
                         double cH, cudaStream_t st);
void set_error(const std::string& s);
void count_launch(int n = 1);
}  // namespace chfsi
