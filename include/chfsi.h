/* chfsi.h -- C ABI of the B200 (sm_100a) Chebyshev-filter hot path of R-ChFSI
 * (arxiv/paper_2605_30128; PAPER.md = the paper text; section/equation numbers are the paper's).
 *
 * The library applies  M^-1 H  matrix-free to blocks of complex two-component spinors on a
 * periodic, uniform, hexahedral, degree-p GLL spectral-element mesh, and runs the paper's
 * Chebyshev recurrences on top of it:
 *     H = -1/2 Laplacian + V I + B.sigma + H_nloc                  (eqs. 4, 7)
 *     discretised as in Sec. III-A (eq. 8) with GLL collocation, so that the
 *     mass matrix M is diagonal ("D" of PAPER.md:119; BASELINE.json north_star).
 *
 * Conventions common to every call
 *   - Every function returns a chfsi_status; none throws, aborts or prints.
 *     chfsi_last_error() returns a thread-local, human-readable description of the last failure.
 *   - "host" pointers are ordinary CPU memory, copied before the call returns (the caller keeps
 *     ownership).  "device" pointers are CUDA device memory of the mesh's device, owned by the
 *     caller (e.g. torch tensors); the library never frees or retains them.
 *   - Multivector layout ("M_{2I+alpha,2J+beta}"): complex128 interleaved (re,im),
 *     row = 2*I + alpha (node I, spin alpha in {0,1}), vectors fastest:
 *         X[(2*I + alpha) * ld + v],  0 <= v < nvec <= ld,   ld counted in complex elements.
 *     Node I = (iz*N1y + iy)*N1x + ix with N1d = ncd * p nodes per direction; node coordinates
 *     x = (e + (xi_a + 1)/2) * h  for cell e and GLL node xi_a, a = 0..p-1.
 *   - chfsi_apply_H and chfsi_cheb_filter allocate nothing, never synchronise the host with the
 *     device, and enqueue all work on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) -- except that the nonlocal term of a step may run on a
 *     low-priority stream owned by the mesh, forked from and joined back into `cuda_stream` inside
 *     the call, so that work queued on `cuda_stream` after the call still sees it complete.  Setup
 *     calls (mesh_create, ham_set, destroy) may allocate and synchronise.
 *   - A mesh handle is used from one host thread at a time (it owns that side stream, its events
 *     and the profiling state); different meshes are independent.
 *   - I/O multivectors are complex128 whatever `prec` is: FP64<->FP32 conversion is fused into the
 *     kernels' loads and stores (north_star item 5; PAPER.md:208 describes the FP32 operands).
 */
#ifndef CHFSI_H
#define CHFSI_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct chfsi_mesh chfsi_mesh;   /* opaque; owns all device-side operator data */

typedef enum {
    CHFSI_OK = 0,
    CHFSI_EINVAL = 1,        /* bad argument (see each call) */
    CHFSI_ENOMEM = 2,        /* host or device allocation failed */
    CHFSI_ECUDA = 3,         /* a CUDA runtime call failed; see chfsi_last_error() */
    CHFSI_ESTATE = 4,        /* call out of order (apply before ham_set) */
    CHFSI_EUNSUPPORTED = 5   /* no kernel instantiated for this p / precision */
} chfsi_status;

/* Precision of the H.X product inside the recurrence ("FP32 or TF32").
 * The recurrence itself, the residual R and Lambda_k are always FP64. */
typedef enum {
    CHFSI_FP64 = 0,          /* everything FP64 */
    CHFSI_FP32 = 1,          /* H.X product in FP32 on fl32(Z_k); Z_k, R, Lambda_k and the recurrence stored/combined in FP64 */
    CHFSI_TF32 = 2,          /* FP32-stored multivectors (as CHFSI_FP32_STORED) with the S2 cell contractions on TF32 tensor cores
                                ("TF32 tensor operations"): operands rounded cvt.rna.tf32.f32, FP32 accumulate;
                                pointwise terms, phases and the update stay FP32/FP64.  chfsi_cheb_filter, RESIDUAL, even p. */
    CHFSI_TF32X3 = 3,        /* the same with the hi/lo split of both operands and three tensor-core products per
                                contraction (small terms first): FP32-level accuracy on the tensor pipe */
    CHFSI_FP32_STORED = 4    /* the paper's layout: the multivectors Z_k themselves are complex64 inside the
                                filter ("extraction, scatter/gather, and assembly kernels ... operate on FP32 multivectors,
                                halving global memory traffic"), FP32 arithmetic; "only the eigenproblem residual R and the
                                eigenvalue recurrence Lambda_k are retained in FP64", as are S0 and the recover step S7.
                                chfsi_cheb_filter with CHFSI_RECUR_RESIDUAL and even p only (EUNSUPPORTED otherwise). */
} chfsi_prec;

/* Implementation of the dominant (cell) kernel, see chfsi_mesh_set_cell_kernel. */
typedef enum {
    CHFSI_CELL_DEFAULT = 0,  /* the library's choice for this precision and degree */
    CHFSI_CELL_XYZ = 1,      /* line-owned FMA kernel (cell_xyz.cu) */
    CHFSI_CELL_MARCH = 2,    /* plane-march FMA kernel (cell_march.cu), FP64 */
    CHFSI_CELL_MMA = 3       /* tensor-core kernel (cell_mma.cu): mma.sync FP64 / TF32 */
} chfsi_cell_kernel;

typedef enum {
    CHFSI_RECUR_STANDARD = 0,   /* eq. 10 */
    CHFSI_RECUR_RESIDUAL = 1    /* eq. 11, R-ChFSI */
} chfsi_recur;

/* ---- mesh -------------------------------------------------------------------------------
 * Periodic box [0,Lx)x[0,Ly)x[0,Lz) cut into ncx*ncy*ncz equal hexahedral cells, FE degree p on
 * GLL nodes.  kfrac (host, 3 doubles, may be NULL = Gamma) gives the Bloch vector
 * k_d = kfrac_d * 2 pi / L_d: psi(r + L_d e_d) = exp(2 pi i kfrac_d) psi(r); cell-local nodes
 * that wrap around the box carry that phase (the paper is silent on k-points; reading O4).
 * Builds the GLL tables, the diagonal mass m_I and its FP32 copy on `device`.
 * EINVAL: nc* < 1, L* <= 0, p < 1, out == NULL.  EUNSUPPORTED: p not in {1..8}.  ECUDA/ENOMEM. */
chfsi_status chfsi_mesh_create(int ncx, int ncy, int ncz, double Lx, double Ly, double Lz, int p,
                               const double* kfrac, int device, chfsi_mesh** out);
chfsi_status chfsi_mesh_destroy(chfsi_mesh* mesh);          /* NULL is allowed */
/* Selects which implementation of the cell kernel later calls use for precision `prec` (a plain argument, there is no
 * environment switch); every implementation computes the same operation to the precision's tolerance.  A choice that is
 * not built for the degree / precision / call falls back to the default at launch.  EINVAL: NULL mesh, bad enums. */
chfsi_status chfsi_mesh_set_cell_kernel(chfsi_mesh* mesh, chfsi_prec prec, chfsi_cell_kernel kernel);

/* Queries (host outputs).  nnodes = M = N1x*N1y*N1z.  xyz: M*3 doubles (x,y,z per node).
 * mass: M doubles, m_I = sum over the cells containing node I of w_a w_b w_c (hx hy hz / 8). */
chfsi_status chfsi_mesh_num_nodes(const chfsi_mesh* mesh, long long* nnodes);
chfsi_status chfsi_mesh_node_coords(const chfsi_mesh* mesh, double* xyz);
chfsi_status chfsi_mesh_mass(const chfsi_mesh* mesh, double* mass);

/* ---- Hamiltonian data -------------------------------------------------------------------
 * Local part (eq. 4; spin blocks of eq. 12, pointwise under GLL collocation):
 *   V, Bx, By, Bz: host, M doubles each (NULL = zero field): V_eff and B_xc at the nodes, Hartree.
 * Nonlocal part (eq. 7; cell-level projectors and SOC coefficient matrices of
 * PAPER.md:204):  H_nl = M P D P^H M,
 *   natoms >= 0; supp_off: host, natoms+1 offsets into supp_node; supp_node: host, node indices
 *   of each atom's support (each node at most once per atom); nproj: host, natoms projector
 *   counts (1..16); P_re / P_im: host, for atom a a row-major [n_supp_a][nproj_a] block, blocks
 *   concatenated in atom order (P_im NULL = real projectors); any Bloch phase exp(-i k.T) of a
 *   periodic image is already folded into P by the caller.
 *   D: host, per atom a Hermitian (2 nproj_a)^2 complex matrix, interleaved (re,im), row-major,
 *   row/column index 2*beta + s (projector beta, spin s); matrices concatenated in atom order.
 * FP32 copies of all operator data are made here ("single device-to-device cast").
 * May be called again to replace the Hamiltonian.  EINVAL: support node out of range, bad
 * offsets, nproj out of range, NULL where data is required. */
chfsi_status chfsi_ham_set(chfsi_mesh* mesh, const double* V, const double* Bx, const double* By,
                           const double* Bz, int natoms, const long long* supp_off,
                           const long long* supp_node, const int* nproj, const double* P_re,
                           const double* P_im, const double* D);

/* ---- workspace --------------------------------------------------------------------------
 * Bytes of device scratch `work` needed by chfsi_cheb_filter(prec, recur, chunk) (and, with
 * recur = CHFSI_RECUR_STANDARD, an upper bound for chfsi_apply_H with nvec <= chunk).
 * The pointer passed as `work` must be 256-byte aligned. */
chfsi_status chfsi_workspace_bytes(const chfsi_mesh* mesh, chfsi_prec prec, chfsi_recur recur,
                                   int chunk, size_t* bytes);

/* ---- Y = M^-1 H X  (one Hamiltonian-multivector product, then D^-1) -----
 * X, Y: device, complex128, distinct buffers, layout above with leading dimensions ldx, ldy.
 * prec FP32: X is rounded to FP32 on load, the cell Laplacian and the projector contractions run
 * in FP32, the result is widened on store.  EINVAL: nvec < 1, ld < nvec, NULL, work too small or
 * misaligned, X == Y.  ESTATE: before chfsi_ham_set. */
chfsi_status chfsi_apply_H(const chfsi_mesh* mesh, chfsi_prec prec, int nvec, const void* X,
                           long long ldx, void* Y, long long ldy, void* work, size_t work_bytes,
                           void* cuda_stream);

/* ---- Y = C_m(M^-1 H) X  (Chebyshev filter of degree m = `degree`) --------
 * a = lambda_T (lower edge of the damped interval), b = lambda_max, a0 = lambda_min:
 * c = (a+b)/2, e = (b-a)/2, sigma_1 = e/(a0-c), sigma_{k+1} = 1/(2/sigma_1 - sigma_k).
 * recur STANDARD: eq. 10, Y_0 = X, Y_1 = sigma_1 (M^-1 H - c) X / e; lambda_host is ignored.
 * recur RESIDUAL: eq. 11 with D = M: R = H X - M X Lambda in FP64, Z_0 = 0, Z_1 = sigma_1 R / e,
 *   Lambda_k by the same recurrence in FP64 (one device thread per vector), Y = D^-1 Z_m + X Lambda_m;
 *   lambda_host: host, nvec Ritz values (any finite numbers are legal: with D = M the exact
 *   result does not depend on them).  With prec FP32 only the product H D^-1 Z_k is inexact;
 *   R, Z_k, Lambda_k and the four-term combination stay FP64.
 * The output is Y_m after m applications of H (m = 1 returns Y_1).
 * chunk = N_b > 0: vectors are processed in blocks of N_b columns ("N_b
 * wavefunctions"), chunk = 0: all at once.  Y may alias X exactly (same pointer and ld).
 * EINVAL: degree < 1 or > 1024, b <= a, a0 >= a, nvec < 1, ld < nvec, chunk < 0, chunk % 4 != 0 when
 * 0 < chunk < nvec, NULL pointers, lambda_host NULL with RESIDUAL, work too small
 * or misaligned.  ESTATE: before chfsi_ham_set. */
chfsi_status chfsi_cheb_filter(const chfsi_mesh* mesh, chfsi_prec prec, chfsi_recur recur,
                               int degree, double a, double b, double a0, int nvec, int chunk,
                               const void* X, long long ldx, const double* lambda_host, void* Y,
                               long long ldy, void* work, size_t work_bytes, void* cuda_stream);

/* Number of kernel launches (and memset/memcpy nodes) enqueued by this thread's last successful
 * chfsi_apply_H / chfsi_cheb_filter call; used by bench.py for its `gpu_launches` claim. */
long long chfsi_last_launch_count(void);

/* ---- profiling aid (bench.py's roofline block) --------------------------------------------
 * While enabled, every launch of the dominant kernel (the cell kernel: gather + sum-factorised
 * Laplacian + fused assembly/pointwise/recurrence update) is bracketed by CUDA events on the stream
 * it is launched on.  chfsi_profile_read synchronises on those events, returns the summed duration
 * (ms), the number of launches and the summed ALGORITHMIC bytes of those launches -- per unit
 * (complex DoF x vector): 16 B for each multivector read (in; R when the step uses it) plus 32 B for
 * the read-modify-write of the accumulated output, i.e. 64 B for an eq. 11 step with k >= 2 and
 * 48 B for eq. 10 steps, the residual S0 and the first eq. 11 step -- and clears the record. */
chfsi_status chfsi_profile_enable(chfsi_mesh* mesh, int on);
chfsi_status chfsi_profile_read(chfsi_mesh* mesh, double* cell_ms, long long* cell_launches,
                                double* cell_alg_bytes);

/* ---- block floating-point codec of the compressed ghost exchange (Fig. 3) -----------------
 * Four FP32 values <-> one N_bits = 4 n_bits bit word, n_bits in {16, 12, 10}: bits 0..7 = shared biased exponent
 * e = e_max + 127 with 2^(e_max-1) <= max|x_i| < 2^e_max (0 flags an all-zero block; FP32-subnormal maxima use
 * e_max = -126), then four v_bits = n_bits - 2 bit two's-complement coefficients q_i = round(x_i 2^(v_bits-1-e_max))
 * (ties to even, clamped above at 2^(v_bits-1) - 1), q_0 lowest; decode x~_i = q_i 2^(e_max-v_bits+1), exact.
 * Stream layout: block b at byte offset b * n_bits / 2, little-endian ("a single uint64_t", "three uint16_t", "five
 * uint8_t"), no padding.  Inputs must be finite.  One thread per block; no atomics in
 * encode.  All pointers are device memory; work is enqueued on cuda_stream; nothing is allocated or synchronised.
 * EINVAL: n_bits not in {16,12,10}, n < 0 or n % 4 != 0, NULL pointers with n > 0, misaligned pointers (FP32 / multi-
 * vector side 16 B, stream side 8 B), nvec odd or ld odd or ld < nvec in the fused forms. */
chfsi_status chfsi_bfp_stream_bytes(int nbits, long long n, size_t* bytes);      /* n n_bits / 8 */
chfsi_status chfsi_bfp_encode(int nbits, const void* src_f32, long long n, void* dst_stream, void* cuda_stream);
chfsi_status chfsi_bfp_decode(int nbits, const void* src_stream, long long n, void* dst_f32, void* cuda_stream);
/* Fused forms.  rows: device, nrows (node, spin) row indices 2 I + alpha of the message, in order.
 * The message is the FP32 values (re, im interleaved, vectors fastest) of those rows, 2 nvec values per row.
 * gather_encode ("gathers the entries for each neighbour and encodes them in the same pass"): X is a complex128
 * (complex_bytes 16; rounded to FP32 first) or complex64 (complex_bytes 8) multivector with leading dimension ld.
 * decode_scatter_add ("decodes the data and atomically scatter-adds it to the corresponding owned entries"):
 * Y[row] += decoded values, by atomic adds in Y's precision; a row may be listed several times. */
chfsi_status chfsi_bfp_gather_encode(int nbits, const void* X, int complex_bytes, long long ld, int nvec,
                                     const long long* rows, long long nrows, void* dst_stream, void* cuda_stream);
chfsi_status chfsi_bfp_decode_scatter_add(int nbits, const void* src_stream, const long long* rows, long long nrows,
                                          int nvec, void* Y, int complex_bytes, long long ld, void* cuda_stream);

/* ---- Rayleigh-Ritz pieces around the filter (Algorithm 1 lines 6-8) -------------
 * chfsi_rr_project (RR-Proj): S = A^H diag(w) B, S: device, nvec x nvec complex128, row-major, overwritten.  A, B: device,
 *   complex128, nrows rows, leading dimensions lda, ldb.  use_mass != 0: w = the node masses (row 2 I + alpha carries m_I,
 *   nrows must be 2 * nnodes): with A = B = Y it is Y^H M Y, with B = M^-1 H Y (chfsi_apply_H) it is Y^H H Y; use_mass = 0:
 *   w = 1 and mesh may be NULL.  hermitian != 0: only the tiles on and above the diagonal are computed and the rest is
 *   mirrored (the caller asserts that the exact S is Hermitian); the diagonal is returned exactly real.  FP64.
 * chfsi_rr_rotate (RR-SR): Yout = Y Q.  prec CHFSI_FP32: the paper's mixed precision, "Y Q_non-diag is evaluated in FP32
 *   arithmetic, while Y Q_diag is computed in FP64" (Y and the off-diagonal of Q are rounded to complex64, products and
 *   accumulation in FP32, the result widened and added to Y Q_diag).  prec CHFSI_FP64: all FP64.  prec CHFSI_TF32X3: the
 *   same mixed form with the off-diagonal product on the tcgen05 tensor cores: both operands rounded to FP32 and split into
 *   two TF32 parts, three TF32 products per term, FP32 accumulation in tensor memory (FP32-level accuracy; DESIGN.md reading
 *   R2).  Q: device, nvec x nvec complex128, row-major.  Y and Yout must be distinct.  work: device scratch of
 *   chfsi_rr_rotate_workspace_bytes(nvec) (enough for every precision), 256-byte aligned.  Diagonalising the projected
 *   pencil (RR-diag, ELPA in the paper) is left to the caller.
 * EINVAL: bad sizes / leading dimensions / alignment / NULL; EUNSUPPORTED: other precisions. */
chfsi_status chfsi_rr_project(const chfsi_mesh* mesh, long long nrows, int nvec, const void* A, long long lda,
                              const void* B, long long ldb, int use_mass, int hermitian, void* S, void* cuda_stream);
chfsi_status chfsi_rr_rotate_workspace_bytes(int nvec, size_t* bytes);
chfsi_status chfsi_rr_rotate(chfsi_prec prec, long long nrows, int nvec, const void* Y, long long ldy, const void* Q,
                             void* Yout, long long ldo, void* work, size_t work_bytes, void* cuda_stream);

/* chfsi_rr_rotate_static: chfsi_rr_rotate (same operation, same arguments, layout and errors; prec CHFSI_FP64
 * or CHFSI_FP32 only, CHFSI_EUNSUPPORTED otherwise) for callers that cannot allocate device memory and have no workspace to pass: code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc.  The split-Q scratch is a static device array inside the library, 4,203,008 bytes
 * (what those two precisions need at CHFSI_RR_STATIC_MAX_NVEC), resident on every GPU that loads the library until the
 * process exits.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine): it launches the same
 * two kernels as chfsi_rr_rotate on `cuda_stream`.  nvec > CHFSI_RR_STATIC_MAX_NVEC: CHFSI_EINVAL (use chfsi_rr_rotate).
 * The device address of the array is resolved on the first call on each device (cudaGetSymbolAddress with that device
 * current; make that first call outside stream capture).  ALL calls on a device share the one array, which keeps the last
 * call's contents; every call rewrites the part it reads, so nothing needs clearing -- but two calls that overlap on the
 * GPU (different streams without an ordering, or two host threads) RACE on it: serialise them. */
#define CHFSI_RR_STATIC_MAX_NVEC 512
chfsi_status chfsi_rr_rotate_static(chfsi_prec prec, long long nrows, int nvec, const void* Y, long long ldy, const void* Q,
                                    void* Yout, long long ldo, void* cuda_stream);

/* ---- matrix-free Poisson solve (eq. 5-6; Kx kernel and Algorithm 2) -----
 * Solves K x = f for the stiffness matrix K of -laplace on the handle's periodic mesh (GLL quadrature: K = 2 x the kinetic
 * part of H; reading P2), batched: a spinor-layout block [2 M rows][ld complex128] holds 4 nvec independent real
 * right-hand sides, column id cid = (s nvec + v) 2 + ri for spin row s, vector v, real / imaginary part ri (eq. 6 has one
 * problem per atom).  The handle's Hamiltonian must be the bare Laplacian: chfsi_ham_set(mesh, NULL, NULL, NULL, NULL, 0, ...),
 * kfrac = 0 and at least two cells per direction (ESTATE / EINVAL otherwise).  K is singular (constants): every column of f
 * must sum to zero; x starts at 0 and is returned with zero mass-weighted mean.
 * chfsi_poisson_kdiag: diag(K), host output, M doubles (the Jacobi scaling; the caller estimates the spectral bounds of
 *   K_diag^-1 K with it, "a short Lanczos run on the scaled operator").
 * chfsi_poisson_apply_K: W = K U (the Kx kernel: gather + sum-factorised contractions + assembly in one launch).
 * chfsi_poisson_pcg: Algorithm 2 with the degree-`cheb_degree` Chebyshev-Jacobi preconditioner on [lmin, lmax] (cheb_degree - 1
 *   extra Kx per iteration); stops a column when sqrt(|r|^2) < tol (absolute) or after maxit iterations.  The scalars stay on
 *   the device; the host reads the number of unconverged columns every `check_every` iterations (0: never -- the call then
 *   runs maxit iterations without synchronising).  iters_host / resnorm_host (host, 4 nvec each, may be NULL; reading them
 *   synchronises): iterations taken and final residual norm per column.  work: chfsi_poisson_workspace_bytes, 256-byte aligned.
 *   FP64 throughout. */
/* chfsi_poisson_set_quadrature: rule 0 (default) = GLL collocation as above; rule 1 = the paper's Kx with p + 1 Gauss-Legendre points
 *   per direction ("six batched tensor contractions covering interpolation of nodal values to quadrature points, application of the
 *   per-cell Jacobian, and integration back"): a different, consistent-mass discretisation of the same operator; every
 *   chfsi_poisson_* call then uses it (its own Kx kernel, its own diag(K)).  Setup call (may allocate).  Needs >= 2 cells per direction. */
chfsi_status chfsi_poisson_set_quadrature(chfsi_mesh* mesh, int rule);
chfsi_status chfsi_poisson_kdiag(const chfsi_mesh* mesh, double* kdiag_host);
chfsi_status chfsi_poisson_apply_K(const chfsi_mesh* mesh, int nvec, const void* U, long long ldu, void* W, long long ldw,
                                   void* cuda_stream);
chfsi_status chfsi_poisson_workspace_bytes(const chfsi_mesh* mesh, int nvec, size_t* bytes);
chfsi_status chfsi_poisson_pcg(const chfsi_mesh* mesh, int nvec, const void* F, long long ldf, void* X, long long ldx,
                               int cheb_degree, double lmin, double lmax, double tol, int maxit, int check_every,
                               void* work, size_t work_bytes, int* iters_host, double* resnorm_host, void* cuda_stream);

/* ---- measurement aid: issue-rate peaks of the FMA and mma.sync pipes ------------------------------
 * Runs four register-resident micro-kernels on `device` (one 512-thread CTA per SM, a few milliseconds each, synchronises)
 * and returns TFLOP/s (2 flop per FMA) in tflops[0..3]: FP64 FMA, FP32 FMA, mma.m8n8k4.f64, mma.m16n8k8.tf32.  bench.py
 * reports them as the "alu" / tensor roofs of the kernels that are not HBM-bound.  EINVAL: NULL; ECUDA / ENOMEM. */
chfsi_status chfsi_measure_pipe_peaks(int device, double* tflops);

const char* chfsi_last_error(void);     /* thread-local; never NULL */
const char* chfsi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CHFSI_H */
