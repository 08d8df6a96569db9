"""CPU oracle for the Chebyshev-filter hot path of R-ChFSI (arxiv/paper_2605_30128).

TEST INFRASTRUCTURE ONLY.  Plain, slow, FP64/complex128 numpy.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this package.  It shares no code with the CUDA path (`paper_2605_30128_b200/csrc`)
and imports nothing from it; the seeded *input* generators live in
`paper_2605_30128_b200/inputs.py`, which holds none of the method's arithmetic.

What it computes, and the passage each function follows (PAPER.md = /root/reference/PAPER.md;
"§8(c) Xn" = SURVEY.md §8(c) reading Xn, restated in DESIGN.md §3):

  gll(), diff_matrix(), k1d()      GLL nodes/weights/derivative matrix, 1-D stiffness
                                   ("1D Lagrange polynomials of degree p on GLL
                                   nodes"; O1, O2)
  Mesh                             periodic uniform hex mesh, local-to-global map with Bloch
                                   phase ("local-to-global map"; O4)
  cell_stiffness_dense()           K_e as the explicit Kronecker sum (definition, O2)
  apply_cell_stiffness()           the same action as three 1-D contractions (PAPER.md:102
                                   "sequence of 1D contractions")
  apply_H()                        Y = H X by the paper's four stages:
                                   extraction, cell-level product with the spin blocks of
                                   eq. 12, assembly, nonlocal P D P^H (eq. 7)
  apply_MinvH()                    M^-1 H with the diagonal (GLL-collocated) mass M == D
                                   ("D is either a GLL-integrated or lumped
                                   mass matrix"; BASELINE.json north_star "M is the diagonal
                                   mass matrix")
  cheb_sigmas(), cheb_filter_standard()   eq. 10
  cheb_filter_residual()           eq. 11, Z_0=0, Z_1=sigma_1 R/e,
                                   Y_q = D^-1 Z_q + X Lambda_q
  lanczos_bounds()                 k-step Lanczos upper bound (§8(c) A4)
  rayleigh_ritz(), subspace_iteration()   Algorithm 1 lines 2-10
  dense_H()                        brute-force assembly for tiny meshes (pin P10)

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): P1-P12 of SURVEY.md §8(c); every
function above is pinned by at least one of them -- no function here is "parity unpinned".

Array layout: a multivector is numpy complex128 [M, 2, nvec] = (node I, spin alpha, vector),
C-contiguous, i.e. the C-ABI layout X[(2 I + alpha) ld + v] with ld = nvec (PAPER.md:92
"M_{2I+alpha,2J+beta}").  Node I = (iz N1y + iy) N1x + ix.
"""
from __future__ import annotations

import math

import numpy as np


# =========================================================================== O1: GLL basis
def legendre(p: int, x):
    """P_p(x) by the three-term recurrence (Bonnet)."""
    x = np.asarray(x, dtype=np.float64)
    p0 = np.ones_like(x)
    if p == 0:
        return p0
    p1 = x.copy()
    for n in range(1, p):
        p0, p1 = p1, ((2 * n + 1) * x * p1 - n * p0) / (n + 1)
    return p1


def gll(p: int):
    """Gauss-Lobatto-Legendre nodes xi_0=-1 < ... < xi_p=1 and weights.

    Interior nodes are the roots of P_p'(x); w_i = 2 / (p (p+1) P_p(xi_i)^2)  (O1).
    Roots by Newton on q(x) = P_p'(x) from Chebyshev-Gauss-Lobatto starting guesses, using
    (1-x^2) P_p'' = 2 x P_p' - p(p+1) P_p.
    """
    if p < 1:
        raise ValueError("p >= 1")
    x = -np.cos(math.pi * np.arange(p + 1) / p)
    xi = x[1:-1].copy()
    for _ in range(100):
        # P_p'(x) = p (P_{p-1} - x P_p) / (1 - x^2)
        Pp = legendre(p, xi)
        Pm = legendre(p - 1, xi)
        d1 = p * (Pm - xi * Pp) / (1.0 - xi * xi)
        d2 = (2.0 * xi * d1 - p * (p + 1) * Pp) / (1.0 - xi * xi)
        dx = d1 / d2
        xi = xi - dx
        if np.max(np.abs(dx), initial=0.0) < 1e-16:
            break
    nodes = np.concatenate([[-1.0], xi, [1.0]])
    nodes = 0.5 * (nodes - nodes[::-1])          # enforce exact antisymmetry
    w = 2.0 / (p * (p + 1) * legendre(p, nodes) ** 2)
    return nodes, w


def diff_matrix(x: np.ndarray) -> np.ndarray:
    """Lagrange derivative matrix Dm[q,i] = l_i'(x_q) (barycentric form; diagonal = -row sum)."""
    n = x.size
    c = np.array([np.prod([x[i] - x[k] for k in range(n) if k != i]) for i in range(n)])
    Dm = np.zeros((n, n))
    for q in range(n):
        for i in range(n):
            if i != q:
                Dm[q, i] = (c[q] / c[i]) / (x[q] - x[i])
        Dm[q, q] = -np.sum(Dm[q, :])
    return Dm


def k1d(p: int) -> np.ndarray:
    """Reference 1-D stiffness Khat = Dm^T diag(w) Dm on [-1,1] (exact: integrand degree 2p-2)."""
    x, w = gll(p)
    Dm = diff_matrix(x)
    return Dm.T @ (w[:, None] * Dm)


# =========================================================================== mesh (O3, O4)
class Mesh:
    """Periodic uniform hexahedral mesh of degree-p GLL spectral elements with a Bloch phase.

    ncell = (ncx,ncy,ncz), L = (Lx,Ly,Lz), kfrac: k_d = kfrac_d 2 pi / L_d.
    DoFs are psi at the nodes in [0,L)^3; psi(r + L_d e_d) = phi_d psi(r), phi_d = exp(2 pi i kfrac_d).
    """

    def __init__(self, ncell, L, p, kfrac=(0.0, 0.0, 0.0)):
        self.ncell = tuple(int(c) for c in (ncell if np.ndim(ncell) else (ncell,) * 3))
        self.L = tuple(float(l) for l in (L if np.ndim(L) else (L,) * 3))
        self.p = int(p)
        self.kfrac = tuple(float(k) for k in kfrac)
        self.n1 = tuple(c * self.p for c in self.ncell)              # nodes per direction
        self.h = tuple(l / c for l, c in zip(self.L, self.ncell))
        self.nnodes = self.n1[0] * self.n1[1] * self.n1[2]
        self.xi, self.w = gll(self.p)
        self.Khat = k1d(self.p)
        self.phi = tuple(complex(np.exp(2j * math.pi * k)) for k in self.kfrac)
        self._build_maps()

    # -- local-to-global map with the wrapped-node phase (O4)
    def _build_maps(self):
        p, n = self.p, self.p + 1
        ncx, ncy, ncz = self.ncell
        n1x, n1y, n1z = self.n1
        ncells = ncx * ncy * ncz
        self.cell_nodes = np.empty((ncells, n * n * n), dtype=np.int64)
        self.cell_phase = np.empty((ncells, n * n * n), dtype=np.complex128)
        e = 0
        for ez in range(ncz):
            for ey in range(ncy):
                for ex in range(ncx):
                    l = 0
                    for c in range(n):
                        gz = ez * p + c
                        wz = gz == n1z
                        for b in range(n):
                            gy = ey * p + b
                            wy = gy == n1y
                            for a in range(n):
                                gx = ex * p + a
                                wx = gx == n1x
                                I = ((0 if wz else gz) * n1y + (0 if wy else gy)) * n1x + (0 if wx else gx)
                                ph = 1.0 + 0.0j
                                if wx:
                                    ph *= self.phi[0]
                                if wy:
                                    ph *= self.phi[1]
                                if wz:
                                    ph *= self.phi[2]
                                self.cell_nodes[e, l] = I
                                self.cell_phase[e, l] = ph
                                l += 1
                    e += 1
        # cell-local quadrature weights w_a w_b w_c (hx/2)(hy/2)(hz/2), index (c,b,a), a fastest
        jac = (self.h[0] / 2) * (self.h[1] / 2) * (self.h[2] / 2)
        w = self.w
        self.wq = (w[:, None, None] * w[None, :, None] * w[None, None, :]).reshape(-1) * jac
        # diagonal mass m_I = sum over cells containing I of wq (O3); |phase| = 1 so M is real
        m = np.zeros(self.nnodes)
        for e in range(ncells):
            np.add.at(m, self.cell_nodes[e], self.wq)
        self.mass = m
        # with a single cell in some direction a cell lists a global node twice (its two faces coincide)
        self.cell_unique = min(self.ncell) > 1

    def node_coords(self) -> np.ndarray:
        """[M,3] coordinates, node I = (iz N1y + iy) N1x + ix, x = (e + (xi+1)/2) h."""
        def line(d):
            ref = (self.xi[:-1] + 1.0) * 0.5 * self.h[d]
            return (np.arange(self.ncell[d])[:, None] * self.h[d] + ref[None, :]).reshape(-1)
        x, y, z = line(0), line(1), line(2)
        zz, yy, xx = np.meshgrid(z, y, x, indexing="ij")
        return np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1)


# =========================================================================== O2: kinetic
def cell_stiffness_dense(mesh: Mesh) -> np.ndarray:
    """K_e = J [ (2/hx)^2 W(x)W(x)Khat_x + (2/hy)^2 W(x)Khat_y(x)W + (2/hz)^2 Khat_z(x)W(x)W ]  (O2).

    Written in storage order (c,b,a) with a (x) fastest: kron(z-factor, y-factor, x-factor).
    J = (hx/2)(hy/2)(hz/2); W = diag(w).
    """
    W = np.diag(mesh.w)
    K = mesh.Khat
    hx, hy, hz = mesh.h
    jac = (hx / 2) * (hy / 2) * (hz / 2)
    Kx = np.kron(W, np.kron(W, K)) * (2 / hx) ** 2
    Ky = np.kron(W, np.kron(K, W)) * (2 / hy) ** 2
    Kz = np.kron(K, np.kron(W, W)) * (2 / hz) ** 2
    return jac * (Kx + Ky + Kz)


def apply_cell_stiffness(mesh: Mesh, Xe: np.ndarray) -> np.ndarray:
    """K_e Xe for Xe [(p+1)^3, ncols] by three 1-D contractions."""
    n = mesh.p + 1
    w, K = mesh.w, mesh.Khat
    hx, hy, hz = mesh.h
    jac = (hx / 2) * (hy / 2) * (hz / 2)
    T = Xe.reshape(n, n, n, -1)                                   # [c,b,a,col]
    ww = w[:, None] * w[None, :]
    out = (2 / hx) ** 2 * np.einsum("ia,cbav->cbiv", K, T) * ww[:, :, None, None]
    out += (2 / hy) ** 2 * np.einsum("jb,cbav->cjav", K, T) * ww[:, None, :, None]
    out += (2 / hz) ** 2 * np.einsum("kc,cbav->kbav", K, T) * ww[None, :, :, None]
    return (jac * out).reshape(n * n * n, -1)


# =========================================================================== Hamiltonian
class Hamiltonian:
    """Operator data: local fields at the nodes and nonlocal projectors (inputs of chfsi_ham_set)."""

    def __init__(self, mesh: Mesh, V, Bx, By, Bz, supp_off=None, supp_node=None, nproj=None,
                 P=None, D=None):
        M = mesh.nnodes
        self.mesh = mesh
        self.V = np.zeros(M) if V is None else np.asarray(V, np.float64)
        self.Bx = np.zeros(M) if Bx is None else np.asarray(Bx, np.float64)
        self.By = np.zeros(M) if By is None else np.asarray(By, np.float64)
        self.Bz = np.zeros(M) if Bz is None else np.asarray(Bz, np.float64)
        self.atoms = []                                              # (nodes, P[nsupp,nproj], D[2np,2np])
        if supp_off is not None and len(supp_off) > 1:
            off = 0
            for a in range(len(supp_off) - 1):
                nodes = np.asarray(supp_node[supp_off[a]:supp_off[a + 1]], np.int64)
                npj = int(nproj[a])
                Pa = np.asarray(P[off:off + nodes.size * npj], np.complex128).reshape(nodes.size, npj)
                off += nodes.size * npj
                self.atoms.append((nodes, Pa, np.asarray(D[a], np.complex128)))


def apply_H(ham: Hamiltonian, X: np.ndarray, use_dense_cell=False) -> np.ndarray:
    """Y = H X for X [M,2,nvec] complex128, by the four stages of PAPER.md:204.

    (i)   extraction  X^(e) = R^(e) X  (index gather; wrapped nodes carry the Bloch phase, O4)
    (ii)  cell product with the spin blocks of eq. 12:
            Y_up = (H_scal + H_Bz) X_up + (H_Bx - i H_By) X_dn
            Y_dn = (H_Bx + i H_By) X_up + (H_scal - H_Bz) X_dn
          H_scal^(e) = 1/2 K_e + diag(wq V), H_Bd^(e) = diag(wq B_d)  (GLL collocation, O2/O3)
    (iii) assembly    Y += R^(e)^H Y^(e)  (index scatter-add, conjugate phase)
    (iv)  nonlocal    Y += M P_a D_a P_a^H M X  per atom (eq. 7; O5)
    """
    mesh = ham.mesh
    M, two, nvec = X.shape
    assert M == mesh.nnodes and two == 2
    Y = np.zeros_like(X, dtype=np.complex128)
    Ke = cell_stiffness_dense(mesh) if use_dense_cell else None
    n3 = (mesh.p + 1) ** 3
    for e in range(mesh.cell_nodes.shape[0]):
        idx = mesh.cell_nodes[e]
        ph = mesh.cell_phase[e]
        Xe = X[idx] * ph[:, None, None]                              # (i)  [n3,2,nvec]
        flat = np.ascontiguousarray(Xe).reshape(n3, 2 * nvec).view(np.float64)   # real batch columns
        if use_dense_cell:
            KX = Ke @ flat
        else:
            KX = apply_cell_stiffness(mesh, flat)
        KX = np.ascontiguousarray(KX).view(np.complex128).reshape(n3, 2, nvec)
        wV = (mesh.wq * ham.V[idx])[:, None]
        wBx = (mesh.wq * ham.Bx[idx])[:, None]
        wBy = (mesh.wq * ham.By[idx])[:, None]
        wBz = (mesh.wq * ham.Bz[idx])[:, None]
        up, dn = Xe[:, 0, :], Xe[:, 1, :]
        Ye = np.empty_like(Xe)
        Ye[:, 0, :] = 0.5 * KX[:, 0, :] + (wV + wBz) * up + (wBx - 1j * wBy) * dn     # (ii)
        Ye[:, 1, :] = 0.5 * KX[:, 1, :] + (wBx + 1j * wBy) * up + (wV - wBz) * dn
        if mesh.cell_unique:                                         # (iii) scatter-ADD
            Y[idx] += np.conj(ph)[:, None, None] * Ye
        else:                                                        # a direction with one cell: both faces are the
            np.add.at(Y, idx, np.conj(ph)[:, None, None] * Ye)      # same global node, contributions accumulate
    for nodes, Pa, Da in ham.atoms:                                  # (iv)
        npj = Pa.shape[1]
        mX = mesh.mass[nodes][:, None, None] * X[nodes]              # [ns,2,nvec]
        C = np.einsum("ib,isv->bsv", np.conj(Pa), mX)                # c_{beta,s,v}
        G = (Da @ C.reshape(2 * npj, nvec)).reshape(npj, 2, nvec)    # index 2 beta + s
        Y[nodes] += mesh.mass[nodes][:, None, None] * np.einsum("ib,bsv->isv", Pa, G)
    return Y


def apply_MinvH(ham: Hamiltonian, X: np.ndarray) -> np.ndarray:
    """M^-1 H X with diagonal M (chfsi_apply_H)."""
    return apply_H(ham, X) / ham.mesh.mass[:, None, None]


def dense_H(ham: Hamiltonian) -> np.ndarray:
    """Dense 2M x 2M matrix of H, row/col index 2I+alpha (tiny meshes only; pin P10)."""
    M = ham.mesh.nnodes
    n = 2 * M
    E = np.eye(n, dtype=np.complex128).reshape(M, 2, n)
    return apply_H(ham, E).reshape(n, n)


# =========================================================================== Chebyshev filter
def cheb_sigmas(degree: int, a: float, b: float, a0: float):
    """c, e, sigma_1..sigma_degree of PAPER.md:119 with a=lambda_T, b=lambda_max, a0=lambda_min.

    c=(b+a)/2, e=(b-a)/2 (reading G1), sigma_1 = e/(a0-c), sigma_{k+1} = 1/(2/sigma_1 - sigma_k).
    """
    c = 0.5 * (b + a)
    e = 0.5 * (b - a)
    sig = np.empty(degree + 1)
    sig[0] = np.nan
    sig[1] = e / (a0 - c)
    for k in range(1, degree):
        sig[k + 1] = 1.0 / (2.0 / sig[1] - sig[k])
    return c, e, sig


def cheb_filter_standard(ham: Hamiltonian, X, degree: int, a: float, b: float, a0: float):
    """Y_m = C_m(M^-1 H) X by eq. 10.  m applications of M^-1 H."""
    if degree < 1:
        raise ValueError("degree >= 1 (reading A11)")
    c, e, sig = cheb_sigmas(degree, a, b, a0)
    Yprev = X.copy()
    Y = (sig[1] / e) * (apply_MinvH(ham, X) - c * X)                 # Y_1
    for k in range(1, degree):
        Ynext = (2 * sig[k + 1] / e) * apply_MinvH(ham, Y) - (2 * sig[k + 1] * c / e) * Y \
            - (sig[k] * sig[k + 1]) * Yprev
        Yprev, Y = Y, Ynext
    return Y


def cheb_filter_residual(ham: Hamiltonian, X, lam, degree: int, a: float, b: float, a0: float):
    """R-ChFSI filter, eq. 11 with D == M (diagonal mass).

    R = H X - M X Lambda;  Z_0 = 0, Z_1 = sigma_1 R / e;  Lambda_0 = I, Lambda_1 = sigma_1 (Lambda - c)/e;
    Z_{k+1} = (2 s_{k+1}/e) H D^-1 Z_k - (2 s_{k+1} c/e) Z_k - s_k s_{k+1} Z_{k-1} + (2 s_{k+1}/e) R Lambda_k
    Lambda_k by the same three-term recurrence;  Y_m = D^-1 Z_m + X Lambda_m.
    """
    if degree < 1:
        raise ValueError("degree >= 1 (reading A11)")
    mesh = ham.mesh
    m = mesh.mass[:, None, None]
    lam = np.asarray(lam, np.float64)
    c, e, sig = cheb_sigmas(degree, a, b, a0)
    R = apply_H(ham, X) - m * X * lam[None, None, :]
    Zprev = np.zeros_like(X)
    Z = (sig[1] / e) * R
    Lprev = np.ones_like(lam)
    Lk = sig[1] * (lam - c) / e
    for k in range(1, degree):
        al = 2 * sig[k + 1] / e
        be = 2 * sig[k + 1] * c / e
        ga = sig[k] * sig[k + 1]
        Znext = al * apply_H(ham, Z / m) - be * Z - ga * Zprev + al * R * Lk[None, None, :]
        Lnext = al * lam * Lk - be * Lk - ga * Lprev
        Zprev, Z = Z, Znext
        Lprev, Lk = Lk, Lnext
    return Z / m + X * Lk[None, None, :]


# =========================================================================== harness pieces
def m_inner(mesh: Mesh, A, B):
    """A^H M B for multivectors [M,2,na], [M,2,nb] -> [na,nb]."""
    Mn = mesh.nnodes
    Af = A.reshape(2 * Mn, -1)
    Bf = (mesh.mass[:, None, None] * B).reshape(2 * Mn, -1)
    return Af.conj().T @ Bf


def lanczos_bounds(ham: Hamiltonian, v0: np.ndarray, steps: int = 10):
    """k-step Lanczos on M^-1 H in the M inner product (§8(c) A4).

    Returns (theta_min, theta_max + ||f_k||_M): a0 estimate and the safeguarded upper bound b
    of the method the paper cites for ChFSI (PAPER.md:112 [44]; "short Lanczos run" PAPER.md:193).
    """
    mesh = ham.mesh
    v = v0 / math.sqrt(m_inner(mesh, v0, v0)[0, 0].real)
    alphas, betas = [], []
    vprev = np.zeros_like(v)
    beta = 0.0
    for j in range(steps):
        f = apply_MinvH(ham, v) - beta * vprev
        alpha = m_inner(mesh, v, f)[0, 0].real
        f = f - alpha * v
        alphas.append(alpha)
        beta = math.sqrt(m_inner(mesh, f, f)[0, 0].real)
        if j < steps - 1:
            betas.append(beta)
            vprev, v = v, f / beta
    T = np.diag(alphas) + np.diag(betas, 1) + np.diag(betas, -1)
    th = np.linalg.eigvalsh(T)
    return float(th[0]), float(th[-1] + beta)


def rayleigh_ritz(ham: Hamiltonian, Y):
    """Alg. 1 lines 6-9: solve Y^H H Y Q = Y^H M Y Q Lambda, return (Y Q, Lambda)."""
    mesh = ham.mesh
    Mn, _, nv = Y.shape
    HY = apply_H(ham, Y)
    Hs = Y.reshape(2 * Mn, nv).conj().T @ HY.reshape(2 * Mn, nv)
    Ss = m_inner(mesh, Y, Y)
    Hs = 0.5 * (Hs + Hs.conj().T)
    Ss = 0.5 * (Ss + Ss.conj().T)
    Lc = np.linalg.cholesky(Ss)
    Li = np.linalg.inv(Lc)
    A = Li @ Hs @ Li.conj().T
    lam, U = np.linalg.eigh(0.5 * (A + A.conj().T))
    Q = Li.conj().T @ U
    Xn = (Y.reshape(2 * Mn, nv) @ Q).reshape(Mn, 2, nv)
    return Xn, lam


def residual_norms(ham: Hamiltonian, X, lam):
    """|| H x_j - eps_j M x_j ||_2 per column (Alg. 1 line 2; reading A12: 2-norm)."""
    R = apply_H(ham, X) - ham.mesh.mass[:, None, None] * X * np.asarray(lam)[None, None, :]
    return np.sqrt(np.sum(np.abs(R) ** 2, axis=(0, 1)))


def subspace_iteration(ham: Hamiltonian, X0, degree: int, b: float, passes: int, tol=1e-6,
                       n_check=None, filter_fn=None):
    """Algorithm 1: RR on X0, then [filter -> RR -> update bounds] passes.

    filter_fn(X, lam, degree, a, b, a0) -> Y defaults to the oracle's eq. 11.  Line 10:
    a0 <- lambda_1, a <- lambda_{N} (reading A5).  Returns (X, lam, history of max residual).
    """
    if filter_fn is None:
        filter_fn = lambda X, lam, m, a, bb, a0: cheb_filter_residual(ham, X, lam, m, a, bb, a0)
    X, lam = rayleigh_ritz(ham, X0)
    nv = X.shape[2]
    n_check = n_check or (3 * nv) // 4
    hist = []
    for _ in range(passes):
        res = residual_norms(ham, X, lam)
        xn = np.sqrt(np.real(np.diag(m_inner(ham.mesh, X, X))))
        hist.append(float(np.max(res[:n_check] / xn[:n_check])))
        if hist[-1] <= tol:
            break
        a0 = float(lam[0])
        a = float(lam[-1])
        Y = filter_fn(X, lam, degree, a, b, a0)
        X, lam = rayleigh_ritz(ham, Y)
    return X, lam, hist
