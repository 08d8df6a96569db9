"""Pins of the Poisson oracle (oracle/poisson_oracle.py) against what the paper and the mathematics fix
(eq. 5; the Kx kernel and Algorithm 2).  CPU only."""
import numpy as np
import pytest

from oracle import fe_oracle as fo
from oracle import poisson_oracle as po


def _dense_K(mesh, rule="gll"):
    Ke = po.cell_stiffness_quad(mesh, rule)
    K = np.zeros((mesh.nnodes, mesh.nnodes))
    for e in range(mesh.cell_nodes.shape[0]):
        idx = mesh.cell_nodes[e]
        np.add.at(K, (idx[:, None], idx[None, :]), Ke)
    return K


@pytest.mark.parametrize("p,ncell,L", [(2, (2, 2, 2), (4.0, 4.0, 4.0)), (3, (2, 1, 3), (3.0, 2.0, 4.5)), (4, (1, 2, 2), (2.0, 5.0, 4.0))])
def test_quadrature_point_stiffness_equals_the_kronecker_forms(p, ncell, L):
    """The definition sum_q w_q J grad N_i . grad N_j (Lagrange product formulas evaluated at the quadrature points) against
    Kronecker forms built another way.  GLL rule: K_e = J sum_d (2/h_d)^2 Khat (x) W (x) W of fe_oracle (barycentric
    derivative matrix; pinned there by P1/P4).  Gauss rule: the same with the exact 1-D mass B^T W_q B in the transverse
    directions; both rules give the same exact 1-D stiffness (integrand of degree 2p - 2)."""
    mesh = fo.Mesh(ncell, L, p)
    Kk = fo.cell_stiffness_dense(mesh)
    assert np.abs(po.cell_stiffness_quad(mesh, "gll") - Kk).max() < 1e-12 * np.abs(Kk).max()
    Bm, Gm, wq = po.shape_tables(p, "gl")
    assert abs(wq.sum() - 2.0) < 1e-14
    K1 = Gm.T @ (wq[:, None] * Gm)
    M1 = Bm.T @ (wq[:, None] * Bm)
    assert np.abs(K1 - mesh.Khat).max() < 1e-12 * np.abs(mesh.Khat).max()
    exact_mass = np.array([[np.polynomial.legendre.leggauss(2 * p + 2)[1] @ (
        np.prod([(np.polynomial.legendre.leggauss(2 * p + 2)[0] - mesh.xi[k]) / (mesh.xi[i] - mesh.xi[k]) for k in range(p + 1) if k != i], axis=0) *
        np.prod([(np.polynomial.legendre.leggauss(2 * p + 2)[0] - mesh.xi[k]) / (mesh.xi[j] - mesh.xi[k]) for k in range(p + 1) if k != j], axis=0))
        for j in range(p + 1)] for i in range(p + 1)])
    assert np.abs(M1 - exact_mass).max() < 1e-13
    hx, hy, hz = mesh.h
    J = hx * hy * hz / 8
    Kg = J * ((2 / hx) ** 2 * np.kron(M1, np.kron(M1, K1)) + (2 / hy) ** 2 * np.kron(M1, np.kron(K1, M1)) + (2 / hz) ** 2 * np.kron(K1, np.kron(M1, M1)))
    assert np.abs(po.cell_stiffness_quad(mesh, "gl") - Kg).max() < 1e-12 * np.abs(Kg).max()


def test_apply_K_equals_the_assembled_matrix_and_has_the_constant_null_space():
    mesh = fo.Mesh((2, 3, 2), (4.0, 5.0, 3.0), 3)
    K = _dense_K(mesh)
    rng = np.random.default_rng(0)
    u = rng.standard_normal((mesh.nnodes, 3))
    w = po.apply_K(mesh, u)
    assert np.abs(w - K @ u).max() < 1e-11 * np.abs(w).max()
    assert np.abs(po.apply_K(mesh, np.ones((mesh.nnodes, 1)))).max() < 1e-11
    assert np.abs(K - K.T).max() < 1e-12 * np.abs(K).max()
    ev = np.linalg.eigvalsh(K)
    assert abs(ev[0]) < 1e-10 * ev[-1] and ev[1] > 1e-6 * ev[-1]
    assert np.abs(po.k_diag(mesh) - np.diag(K)).max() < 1e-12 * np.diag(K).max()
    Kgl = _dense_K(mesh, "gl")                                            # the paper's Gauss rule through the same pipeline
    assert np.abs(po.apply_K(mesh, u, "gl") - Kgl @ u).max() < 1e-11 * np.abs(w).max()
    assert np.abs(po.apply_K(mesh, np.ones((mesh.nnodes, 1)), "gl")).max() < 1e-11
    # K is twice the kinetic part of H (-1/2 laplace) of the filter's oracle
    ham = fo.Hamiltonian(mesh, None, None, None, None)
    X = np.zeros((mesh.nnodes, 2, 1), dtype=np.complex128); X[:, 0, 0] = u[:, 0]
    assert np.abs(2.0 * fo.apply_H(ham, X)[:, 0, 0].real - w[:, 0]).max() < 1e-11 * np.abs(w).max()


def test_chebyshev_jacobi_is_the_stated_polynomial():
    """P^-1 = chi(K_diag^-1 K) K_diag^-1 with 1 - lambda chi(lambda) = T_m((theta - lambda)/delta) / T_m(theta/delta): checked through
    the dense eigendecomposition of the symmetrised scaled operator."""
    mesh = fo.Mesh((2, 2, 2), (4.0, 4.0, 4.0), 2)
    K = _dense_K(mesh)
    kd = po.k_diag(mesh)
    lmin, lmax = 0.1, 2.2
    rng = np.random.default_rng(1)
    r = rng.standard_normal((mesh.nnodes, 2))
    S = K / np.sqrt(kd)[:, None] / np.sqrt(kd)[None, :]
    lam, V = np.linalg.eigh(S)
    theta, delta = 0.5 * (lmax + lmin), 0.5 * (lmax - lmin)
    for m in (1, 2, 5):
        Tm = np.polynomial.chebyshev.Chebyshev.basis(m)
        one_minus = Tm((theta - lam) / delta) / Tm(theta / delta)
        chi = np.where(np.abs(lam) > 1e-12, (1.0 - one_minus) / np.where(np.abs(lam) > 1e-12, lam, 1.0), m * 0 + _chi0(m, theta, delta))
        ref = (V * chi[None, :]) @ (V.T @ (r / np.sqrt(kd)[:, None])) / np.sqrt(kd)[:, None]
        z = po.cheb_jacobi(mesh, kd, r, m, lmin, lmax)
        assert np.abs(z - ref).max() < 1e-10 * np.abs(ref).max(), m


def _chi0(m, theta, delta):
    """chi(0) = lim (1 - T_m((theta - l)/delta)/T_m(sigma))/l = T_m'(sigma) / (delta T_m(sigma))."""
    Tm = np.polynomial.chebyshev.Chebyshev.basis(m)
    return Tm.deriv()(theta / delta) / (delta * Tm(theta / delta))


def test_pcg_reaches_the_pseudo_inverse_solution_and_preconditioning_cuts_iterations():
    mesh = fo.Mesh((2, 2, 3), (4.0, 4.0, 6.0), 3)
    K = _dense_K(mesh)
    rng = np.random.default_rng(2)
    f = rng.standard_normal((mesh.nnodes, 3))
    f -= f.mean(axis=0)                                                  # neutral: sum f = 0 (reading P1)
    kd = po.k_diag(mesh)
    lmin, lmax = po.lanczos_bounds_scaled(mesh, kd, rng.standard_normal(mesh.nnodes))
    ev = np.linalg.eigvalsh(K / np.sqrt(kd)[:, None] / np.sqrt(kd)[None, :])
    assert ev[-1] <= lmax <= 1.3 * ev[-1]
    xref = np.linalg.lstsq(K, f, rcond=None)[0]
    xref -= np.sum(mesh.mass[:, None] * xref, axis=0) / mesh.mass.sum()
    its = {}
    for m in (1, 3, 5):
        x, it, res = po.pcg(mesh, f, m, lmin, lmax, 1e-10, 500)
        assert (res < 1e-10).all()
        assert np.abs(x - xref).max() < 1e-8 * np.abs(xref).max()
        assert np.abs(K @ x - f).max() < 1e-8
        its[m] = it.max()
    assert its[5] < its[3] < its[1]


def test_pcg_with_the_gauss_rule_reaches_its_pseudo_inverse_solution():
    """The paper's Gauss-Legendre form through the same Algorithm 2 (rule = "gl" is only passed through to apply_K / k_diag)."""
    mesh = fo.Mesh((2, 2, 2), (4.0, 4.0, 5.0), 3)
    K = _dense_K(mesh, "gl")
    rng = np.random.default_rng(4)
    f = rng.standard_normal((mesh.nnodes, 2)); f -= f.mean(axis=0)
    kd = po.k_diag(mesh, "gl")
    assert np.abs(kd - np.diag(K)).max() < 1e-12 * kd.max()
    lmin, lmax = po.lanczos_bounds_scaled(mesh, kd, rng.standard_normal(mesh.nnodes), rule="gl")
    x, it, res = po.pcg(mesh, f, 3, lmin, lmax, 1e-10, 500, rule="gl")
    xref = np.linalg.lstsq(K, f, rcond=None)[0]
    xref -= np.sum(mesh.mass[:, None] * xref, axis=0) / mesh.mass.sum()
    assert (res < 1e-10).all() and np.abs(x - xref).max() < 1e-8 * np.abs(xref).max()


def test_cosine_charge_is_solved_spectrally():
    """-laplace V = 4 pi rho with rho = cos(2 pi x / Lx) cos(2 pi z / Lz) has V = 4 pi rho / |k|^2; the FE solution (load
    f = 4 pi m rho, reading P3) approaches it spectrally as p rises (same mesh family as pin P9 of the filter oracle)."""
    errs = []
    for p in (2, 4, 6):
        mesh = fo.Mesh((3, 2, 3), (4.0, 5.0, 6.0), p)
        xyz = mesh.node_coords()
        kx, kz = 2 * np.pi / 4.0, 2 * np.pi / 6.0
        rho = np.cos(kx * xyz[:, 0]) * np.cos(kz * xyz[:, 2])
        f = (4 * np.pi * mesh.mass * rho)[:, None]
        f -= f.mean(axis=0)
        kd = po.k_diag(mesh)
        lmin, lmax = po.lanczos_bounds_scaled(mesh, kd, np.random.default_rng(3).standard_normal(mesh.nnodes))
        x, it, res = po.pcg(mesh, f, 3, lmin, lmax, 1e-12, 2000)
        exact = 4 * np.pi * rho / (kx ** 2 + kz ** 2)
        errs.append(np.abs(x[:, 0] - exact).max() / np.abs(exact).max())
    assert errs[0] > 30 * errs[1] > 900 * errs[2] and errs[2] < 1e-6, errs
