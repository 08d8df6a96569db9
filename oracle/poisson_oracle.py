"""CPU oracle for the matrix-free Poisson solve (arxiv/paper_2605_30128: eq. 5-6; the Kx kernel and
Algorithm 2).

TEST INFRASTRUCTURE ONLY (same rules as fe_oracle.py): only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
cpu_baseline / `--impl reference` legs may import it; it shares no code with the CUDA path and imports nothing from it.

What it computes, and the passage each function follows:

  gauss_legendre(), shape_tables()   Gauss-Legendre points / weights and the 1-D shape-function value and gradient matrices
                                     at them ("These matrices hold the shape function values and their gradients at the
                                     quadrature points")
  cell_stiffness_quad()              K_e[i][j] = int grad N_i . grad N_j over a cell by quadrature (reading P2): the plain
                                     definition of the stiffness matrix of -laplace (eq. 5), dense, for small p
  apply_K()                          w = K u by the paper's fused pipeline written out cell by cell: extraction, "six batched
                                     tensor contractions covering interpolation of nodal values to quadrature points,
                                     application of the per-cell Jacobian, and integration back to the nodal basis", assembly
                                     
  k_diag()                           diag(K), the Jacobi scaling of the preconditioner
  lanczos_bounds_scaled()            "The spectral bounds are estimated once per solve by a short Lanczos run on the scaled
                                     operator" K_diag^-1 K
  cheb_jacobi()                      z = P^-1 r = chi(K_diag^-1 K) K_diag^-1 r, chi a degree-m Chebyshev approximation of
                                     1/lambda: m - 1 applications of K
  pcg()                              Algorithm 2 line by line, in its sign convention r = K x - f

Readings where the paper is silent (P1-P5):
  P1  boundary conditions: the mesh of this build is periodic, so K has the constants as null space; the right-hand side
      must have zero sum (a neutral charge), the iteration starts from x = 0, and the returned potential is shifted to zero
      mass-weighted mean.
  P2  quadrature: the paper's Kx interpolates to Gauss-Legendre points; this build integrates every bilinear form on the
      p + 1 GLL nodes (north_star's collocation, D3), so that the Poisson operator is the same Laplacian as the
      filter's kinetic term (K = 2 x kinetic part of H).  Both rules integrate the 1-D stiffness exactly; they differ in the
      transverse 1-D mass factors (diagonal GLL weights against the exact, non-diagonal Gauss mass).  Every routine here
      takes rule = "gll" (the default, what the CUDA path computes) or "gl" (the paper's, kept for reference and pinned).
  P3  right-hand side: f_I = 4 pi m_I rho_I (GLL-collocated load, consistent with the diagonal mass of DESIGN.md D2).
  P4  Chebyshev preconditioner: the classical three-term Chebyshev iteration for K z = r with Jacobi scaling, started from
      z = 0, on [lmin, lmax]; lmax = the largest Ritz value of a 10-step Lanczos run plus its residual norm, lmin = lmax / 30
      (the smallest eigenvalue of a periodic Laplacian shrinks with the box; a fixed ratio keeps the polynomial a smoother,
      and chi(lambda) lambda stays in (0, 2) for every 0 < lambda <= lmax, so P^-1 is positive definite on the iterates).
  P5  several right-hand sides (eq. 6 has one per atom): columns are independent problems, each with its own alpha, beta
      and its own convergence test on sqrt(gamma) (absolute residual norm, "absolute residual tolerance").

Pins (tests/test_poisson_pins.py): the quadrature-point cell stiffness equals the Kronecker form (GLL rule: fe_oracle's
K_e; Gauss rule: exact 1-D stiffness (x) exact 1-D masses), apply_K equals the assembled dense K, K 1 = 0 and K is symmetric positive semidefinite, the
preconditioner equals the same polynomial evaluated through a dense eigendecomposition, PCG reaches the dense
pseudo-inverse solution, and the analytic periodic solution of a cosine charge is approached spectrally in p.
"""
from __future__ import annotations

import numpy as np

from . import fe_oracle as fo


def gauss_legendre(nq: int):
    """Gauss-Legendre points and weights on [-1, 1] (library routine; pinned by sum(w) = 2 and exactness tests)."""
    return np.polynomial.legendre.leggauss(nq)


def shape_tables(p: int, rule: str = "gll"):
    """B[q][i] = l_i(xq_q), G[q][i] = l_i'(xq_q) for the degree-p Lagrange basis on the GLL nodes, at the p + 1 points of
    the quadrature rule, and the rule's weights."""
    xi, wg = fo.gll(p)
    n = p + 1
    nq = n
    if rule == "gl":
        xq, wq = gauss_legendre(nq)
    elif rule == "gll":
        xq, wq = xi.copy(), wg.copy()
    else:
        raise ValueError("rule must be 'gll' or 'gl'")
    Bm = np.zeros((nq, n))
    Gm = np.zeros((nq, n))
    for i in range(n):
        others = [j for j in range(n) if j != i]
        den = np.prod([xi[i] - xi[j] for j in others])
        for q in range(nq):
            Bm[q, i] = np.prod([xq[q] - xi[j] for j in others]) / den
            Gm[q, i] = sum(np.prod([xq[q] - xi[j] for j in others if j != k]) for k in others) / den
    return Bm, Gm, wq


def cell_stiffness_quad(mesh, rule: str = "gll") -> np.ndarray:
    """Dense K_e by the definition: sum over quadrature points of w_q |J| grad N_i . grad N_j (storage order z, y, x)."""
    p, n = mesh.p, mesh.p + 1
    Bm, Gm, wq = shape_tables(p, rule)
    h = mesh.h
    J = h[0] * h[1] * h[2] / 8.0
    Ke = np.zeros((n ** 3, n ** 3))
    tabs = {0: (Gm, Bm, Bm), 1: (Bm, Gm, Bm), 2: (Bm, Bm, Gm)}            # direction of the derivative: x, y, z
    for d in range(3):
        Tx, Ty, Tz = tabs[d]
        # gradient component d of every basis function at every Gauss point: [qz, qy, qx, kz, ky, kx]
        Dd = np.einsum("ak,bj,ci->abckji", Tz, Ty, Tx).reshape(n ** 3, n ** 3) * (2.0 / h[d])
        W = np.einsum("a,b,c->abc", wq, wq, wq).ravel() * J
        Ke += Dd.T @ (W[:, None] * Dd)
    return Ke


def apply_K(mesh, u: np.ndarray, rule: str = "gll") -> np.ndarray:
    """w = K u for real u [M, ncols], by the fused pipeline of PAPER.md:188-192, cell by cell: extraction through the
    local-to-global map, interpolation to the quadrature points (three 1-D contractions with the value matrix), the gradient at
    those points, the Jacobian and quadrature weight, the transposed steps back to the nodal basis, assembly."""
    u = np.asarray(u, dtype=np.float64)
    if any(abs(ph - 1.0) > 0 for ph in mesh.phi):
        raise ValueError("the Poisson operator acts on real periodic fields: kfrac must be 0")
    p, n = mesh.p, mesh.p + 1
    Bm, Gm, wq = shape_tables(p, rule)
    Dq = Gm @ np.linalg.inv(Bm)                       # collocation derivative at the quadrature points
    h = mesh.h
    J = h[0] * h[1] * h[2] / 8.0
    W3 = np.einsum("a,b,c->abc", wq, wq, wq) * J
    out = np.zeros_like(u)
    nc = u.shape[1]
    fwd = ("cx,abxv->abcv", "bx,axcv->abcv", "ax,xbcv->abcv")          # derivative along x, y, z of [qz, qy, qx, col]
    bwd = ("xc,abxv->abcv", "xb,axcv->abcv", "xa,xbcv->abcv")          # the transposed contractions
    for e in range(mesh.cell_nodes.shape[0]):
        idx = mesh.cell_nodes[e]
        ue = u[idx].reshape(n, n, n, nc)                                                      # (i) extraction
        uq = np.einsum("ak,bj,ci,kjiv->abcv", Bm, Bm, Bm, ue)                                 # (ii) to the Gauss points
        acc = np.zeros_like(uq)
        for d in range(3):
            g = np.einsum(fwd[d], Dq, uq) * (2.0 / h[d])                                      # gradient component
            g = g * W3[..., None] * (2.0 / h[d])                                              # Jacobian and weights
            acc += np.einsum(bwd[d], Dq, g)                                                   # transposed derivative
        we = np.einsum("ak,bj,ci,abcv->kjiv", Bm, Bm, Bm, acc)                                # back to the nodal basis
        np.add.at(out, idx, we.reshape(n ** 3, nc))                                           # (iii) assembly
    return out


def k_diag(mesh, rule: str = "gll") -> np.ndarray:
    """diag(K) by assembling the diagonals of the cell stiffness."""
    Ke = np.diag(cell_stiffness_quad(mesh, rule))
    d = np.zeros(mesh.nnodes)
    for e in range(mesh.cell_nodes.shape[0]):
        np.add.at(d, mesh.cell_nodes[e], Ke)
    return d


def lanczos_bounds_scaled(mesh, kd: np.ndarray, start: np.ndarray, steps: int = 10, rule: str = "gll"):
    """Largest Ritz value (plus the residual norm) of K_diag^-1 K from a `steps`-step Lanczos run in the K_diag inner
    product; returns (lmin, lmax) with lmin = lmax / 30 (reading P4)."""
    v = start - np.sum(kd * start) / np.sum(kd)
    v = v / np.sqrt(np.sum(kd * v * v))
    vprev = np.zeros_like(v)
    alphas, betas, beta = [], [], 0.0
    for j in range(steps):
        f = apply_K(mesh, v[:, None], rule)[:, 0] / kd - beta * vprev
        alpha = float(np.sum(kd * v * f))
        f = f - alpha * v
        alphas.append(alpha)
        beta = float(np.sqrt(np.sum(kd * f * f)))
        if j < steps - 1:
            betas.append(beta)
            vprev, v = v, f / beta
    T = np.diag(alphas) + np.diag(betas, 1) + np.diag(betas, -1)
    lmax = float(np.linalg.eigvalsh(T)[-1] + beta)
    return lmax / 30.0, lmax


def cheb_jacobi(mesh, kd: np.ndarray, r: np.ndarray, m: int, lmin: float, lmax: float, rule: str = "gll") -> np.ndarray:
    """z = chi(K_diag^-1 K) K_diag^-1 r with the degree-m Chebyshev approximation of 1/lambda on [lmin, lmax]: the
    three-term Chebyshev iteration for K z = r from z = 0 (reading P4); m - 1 applications of K."""
    theta, delta = 0.5 * (lmax + lmin), 0.5 * (lmax - lmin)
    sigma = theta / delta
    rho = 1.0 / sigma
    d = (r / kd[:, None]) / theta
    z = d.copy()
    for _ in range(1, m):
        rho_new = 1.0 / (2.0 * sigma - rho)
        res = r - apply_K(mesh, z, rule)
        d = rho_new * rho * d + (2.0 * rho_new / delta) * (res / kd[:, None])
        z = z + d
        rho = rho_new
    return z


def pcg(mesh, f: np.ndarray, m: int, lmin: float, lmax: float, tol: float, maxit: int, rule: str = "gll"):
    """Algorithm 2 for every column of f [M, ncols] independently (reading P5).  Returns (x, iterations per
    column, final residual norms).  Notation of the paper: r = K x - f, delta = r . z, eta = p . w, gamma = |r|^2."""
    f = np.asarray(f, dtype=np.float64)
    kd = k_diag(mesh, rule)
    nc = f.shape[1]
    x = np.zeros_like(f)
    r = -f.copy()                                      # r = K x - f with x = 0
    z = cheb_jacobi(mesh, kd, r, m, lmin, lmax, rule)
    p = -z
    delta = np.sum(r * z, axis=0)
    gamma = np.sum(r * r, axis=0)
    iters = np.zeros(nc, dtype=np.int64)
    active = np.sqrt(gamma) >= tol
    for _ in range(maxit):
        if not active.any():
            break
        w = apply_K(mesh, p, rule)                                     # 1: Kx kernel
        eta = np.sum(p * w, axis=0)                                    # 2: dot kernel
        alpha = np.where(active, delta / np.where(eta != 0, eta, 1.0), 0.0)   # 3
        x += alpha * p                                                 # 4: fused update
        r += alpha * w
        z = cheb_jacobi(mesh, kd, r, m, lmin, lmax, rule)              # 5: Chebyshev preconditioner
        delta_new = np.sum(r * z, axis=0)                              # 6: fused dot
        gamma = np.where(active, np.sum(r * r, axis=0), gamma)
        beta = np.where(active, delta_new / np.where(delta != 0, delta, 1.0), 0.0)   # 8
        delta = np.where(active, delta_new, delta)
        p = np.where(active, -z + beta * p, p)                         # 9
        iters += active
        active = active & (np.sqrt(gamma) >= tol)                      # 10
    x -= np.sum(mesh.mass[:, None] * x, axis=0) / np.sum(mesh.mass)    # zero mass-weighted mean (reading P1)
    return x, iters, np.sqrt(gamma)
