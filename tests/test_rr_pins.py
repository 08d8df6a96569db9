"""Pins of the Rayleigh-Ritz oracle (oracle/rr_oracle.py) against what the paper and the mathematics fix
(Algorithm 1 lines 6-8).  CPU only."""
import numpy as np
import pytest

from oracle import fe_oracle as fo
from oracle import rr_oracle as ro
from paper_2605_30128_b200 import inputs as inp


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def test_project_against_its_triple_loop():
    rng = np.random.default_rng(0)
    A, B, w = _rand(rng, 7, 3), _rand(rng, 7, 3), rng.uniform(0.5, 2.0, 7)
    S = ro.rr_project(A, B, w)
    ref = np.zeros((3, 3), dtype=np.complex128)
    for i in range(3):
        for j in range(3):
            for r in range(7):
                ref[i, j] += np.conj(A[r, i]) * w[r] * B[r, j]
    assert np.allclose(S, ref, rtol=1e-14, atol=1e-14)
    assert np.allclose(ro.rr_project(A, B), A.conj().T @ B)
    SM = ro.rr_project(A, A, w)
    assert np.allclose(SM, SM.conj().T, atol=1e-14) and np.all(np.linalg.eigvalsh(SM) > 0)      # Y^H M Y: Hermitian, positive


def test_rayleigh_ritz_is_exact_on_an_invariant_subspace():
    """Alg. 1 lines 6-8: on a basis of an invariant subspace of (H, M) the projected pencil (Y^H H Y, Y^H M Y) has exactly the
    eigenvalues of that subspace, and rotating by the Ritz vectors gives M-orthonormal eigenvectors.  2x2x2 cells, p = 2."""
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, kfrac=(0.25, 0.0, 0.0), nvec=4, natoms=1, nproj=4)
    mesh = fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    ham = fo.Hamiltonian(mesh, hi.V, hi.Bx, hi.By, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj, hi.P, hi.D)
    H = fo.dense_H(ham)
    m2 = np.repeat(mesh.mass, 2)
    lam, V = np.linalg.eigh(H / np.sqrt(m2)[:, None] / np.sqrt(m2)[None, :])
    V = V / np.sqrt(m2)[:, None]                                       # M-orthonormal eigenvectors of H v = lam M v
    rng = np.random.default_rng(1)
    G = _rand(rng, 6, 6)
    Y = V[:, :6] @ G                                                   # a scrambled basis of the lowest 6-dimensional eigenspace
    Y3 = Y.reshape(mesh.nnodes, 2, 6)
    HY = fo.apply_MinvH(ham, Y3).reshape(-1, 6)                        # M^-1 H Y
    SH, SM = ro.rr_project(Y, HY, m2), ro.rr_project(Y, Y, m2)
    L = np.linalg.cholesky(SM)
    Li = np.linalg.inv(L)
    ev, Z = np.linalg.eigh(Li @ SH @ Li.conj().T)
    assert np.allclose(ev, lam[:6], rtol=0, atol=1e-10)
    Q = Li.conj().T @ Z
    Xn = ro.rr_rotate(Y, Q, mixed=False)
    assert np.allclose(ro.rr_project(Xn, Xn, m2), np.eye(6), atol=1e-10)
    assert np.allclose((H @ Xn), (m2[:, None] * Xn) * ev[None, :], atol=1e-8)


@pytest.mark.parametrize("mixed", [False, True])
def test_rotation_special_cases_are_exact(mixed):
    rng = np.random.default_rng(2)
    Y = _rand(rng, 50, 5)
    assert np.array_equal(ro.rr_rotate(Y, np.eye(5), mixed), Y)
    d = np.exp(1j * rng.uniform(0, 6.28, 5))
    assert np.allclose(ro.rr_rotate(Y, np.diag(d), mixed), Y * d[None, :], rtol=1e-15, atol=0)   # diagonal part is FP64 in both modes
    if not mixed:
        perm = [2, 0, 4, 1, 3]
        Pm = np.zeros((5, 5)); Pm[perm, range(5)] = 1.0
        assert np.array_equal(ro.rr_rotate(Y, Pm, mixed), Y[:, perm])


def test_mixed_precision_rotation_error_is_fp32_sized_and_off_diagonal_only():
    """only Y Q_non-diag is FP32.  Near convergence Q is close to diagonal, which is why the scheme is safe:
    the error scales with |Q_non-diag|."""
    rng = np.random.default_rng(3)
    n = 64
    Y = _rand(rng, 400, n)
    Hm = _rand(rng, n, n); Hm = Hm + Hm.conj().T
    _, U = np.linalg.eigh(Hm)                                          # a generic unitary
    for eps in (1.0, 1e-3):
        Qm = np.diag(np.diag(U)) + eps * (U - np.diag(np.diag(U)))
        exact = ro.rr_rotate(Y, Qm, mixed=False)
        got = ro.rr_rotate(Y, Qm, mixed=True)
        err = np.linalg.norm(got - exact) / np.linalg.norm(exact)
        off = np.linalg.norm(Y @ (Qm - np.diag(np.diag(Qm)))) / np.linalg.norm(exact)
        assert err < 1e-6 * max(off, 1e-12) * 50 and err > 0
    # unitary rotation of an orthonormal block stays orthonormal to FP32 level
    Yo, _ = np.linalg.qr(Y)
    R = ro.rr_rotate(Yo, U, mixed=True)
    assert np.abs(R.conj().T @ R - np.eye(n)).max() < 1e-5
