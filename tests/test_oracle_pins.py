"""Pins for the CPU oracle.  CPU only.

Each pin checks the oracle against something the paper or the mathematics fixes -- closed
forms, invariants, brute force, an independent formulation -- never against itself.
"""
import math
import os

import numpy as np
import pytest

from oracle import fe_oracle as fo
from paper_2605_30128_b200 import inputs as inp

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _ham(cfg, mesh, seed=0, **kw):
    hi = inp.make_hamiltonian(cfg, mesh.node_coords(), seed=seed, **kw)
    return fo.Hamiltonian(mesh, hi.V, hi.Bx, hi.By, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj,
                          hi.P, hi.D), hi


def _mesh(cfg):
    return fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac)


def _line_operator(ncell, L, p, kfrac):
    """Independent 1-D assembled periodic (Bloch-twisted) stiffness and mass: K1 [N1,N1], m1 [N1].

    No 3-D cells, no gather/scatter: element matrices (2/h) Khat and (h/2) w summed on a ring.
    """
    xi, w = fo.gll(p)
    Kh = fo.k1d(p)
    h = L / ncell
    n1 = ncell * p
    phi = np.exp(2j * math.pi * kfrac)
    K1 = np.zeros((n1, n1), dtype=np.complex128)
    m1 = np.zeros(n1)
    for e in range(ncell):
        for a in range(p + 1):
            ga = e * p + a
            pa = phi if ga == n1 else 1.0
            ga %= n1
            m1[ga] += w[a] * h / 2
            for b in range(p + 1):
                gb = e * p + b
                pb = phi if gb == n1 else 1.0
                gb %= n1
                K1[ga, gb] += np.conj(pa) * (2 / h) * Kh[a, b] * pb
    return K1, m1


# ------------------------------------------------------------------ P1
def test_p1_gll_closed_forms_golden():
    for line in open(os.path.join(GOLD, "gll_closed_forms.txt")):
        if line.startswith("#") or not line.strip():
            continue
        p, i, xe, we = line.split()
        x, w = fo.gll(int(p))
        assert abs(x[int(i)] - eval(xe, {"math": math})) < 1e-15
        assert abs(w[int(i)] - eval(we, {"math": math})) < 1e-15


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_p1_gll_and_stiffness_identities(p):
    x, w = fo.gll(p)
    assert abs(w.sum() - 2.0) < 1e-14
    assert np.all(np.diff(x) > 0) and x[0] == -1.0 and x[-1] == 1.0
    # GLL quadrature integrates degree <= 2p-1 exactly
    for d in range(2 * p):
        exact = 0.0 if d % 2 else 2.0 / (d + 1)
        assert abs(np.dot(w, x ** d) - exact) < 1e-13
    Dm = fo.diff_matrix(x)
    assert np.max(np.abs(Dm @ np.ones(p + 1))) < 1e-12
    # derivative exact on monomials up to degree p
    for d in range(1, p + 1):
        assert np.max(np.abs(Dm @ x ** d - d * x ** (d - 1))) < 1e-11
    K = fo.k1d(p)
    assert np.max(np.abs(K - K.T)) < 1e-13
    assert np.max(np.abs(K @ np.ones(p + 1))) < 1e-12
    assert np.max(np.abs(K - K[::-1, ::-1])) < 1e-12          # centrosymmetric
    # u^T K v = int u' v' for polynomials of degree <= p : u = x^a, v = x^b
    for a in range(1, p + 1):
        for b in range(1, p + 1):
            d = a + b - 2
            exact = 0.0 if d % 2 else a * b * 2.0 / (d + 1)
            assert abs((x ** a) @ K @ (x ** b) - exact) < 1e-11


# ------------------------------------------------------------------ P2
def test_p2_mass_sum_and_constant_nullspace():
    mesh = fo.Mesh((2, 3, 2), (3.0, 4.5, 2.0), 3)
    assert abs(mesh.mass.sum() - 3.0 * 4.5 * 2.0) < 1e-12
    ham = fo.Hamiltonian(mesh, None, None, None, None)
    one = np.ones((mesh.nnodes, 2, 1), dtype=np.complex128)
    assert np.max(np.abs(fo.apply_H(ham, one))) < 1e-12


def test_cell_stiffness_sumfact_equals_dense_kron():
    mesh = fo.Mesh((2, 2, 2), (2.0, 3.0, 5.0), 3)                # anisotropic h catches axis mix-ups
    rng = np.random.default_rng(5)
    Xe = rng.standard_normal(((mesh.p + 1) ** 3, 6))
    A = fo.cell_stiffness_dense(mesh) @ Xe
    B = fo.apply_cell_stiffness(mesh, Xe)
    assert np.max(np.abs(A - B)) < 1e-12 * np.max(np.abs(A))
    # the dense-cell route through apply_H agrees too
    ham = fo.Hamiltonian(mesh, None, None, None, None)
    X = inp.make_vectors(mesh.nnodes, 2, seed=3)
    assert np.max(np.abs(fo.apply_H(ham, X) - fo.apply_H(ham, X, use_dense_cell=True))) < 1e-11


# ------------------------------------------------------------------ P3
@pytest.mark.parametrize("kfrac", [(0.0, 0.0, 0.0), (0.25, 0.1, -0.3)])
def test_p3_hermiticity_all_terms(kfrac):
    cfg = inp.tiny_config(ncell=3, p=3, L=6.0, kfrac=kfrac, natoms=2, nproj=8)
    mesh = _mesh(cfg)
    ham, _ = _ham(cfg, mesh)
    assert len(ham.atoms) == 2 and ham.atoms[0][0].size > 10
    u = inp.make_vectors(mesh.nnodes, [0], seed=1)
    v = inp.make_vectors(mesh.nnodes, [1], seed=1)
    a = np.vdot(u, fo.apply_H(ham, v))
    b = np.conj(np.vdot(v, fo.apply_H(ham, u)))
    assert abs(a - b) < 1e-13 * abs(a)


# ------------------------------------------------------------------ P4
@pytest.mark.parametrize("nc", [(2, 3, 2), (1, 3, 2), (2, 1, 1), (1, 1, 1)])
@pytest.mark.parametrize("kfrac", [(0.0, 0.0, 0.0), (0.25, 0.1, 0.0)])
def test_p4_kronecker_line_operator_form(kfrac, nc):
    """M^-1 K = A_x (x) I (x) I + I (x) A_y (x) I + I (x) I (x) A_z, A_d = M1^-1 K1 assembled in 1-D.
    Single-cell directions included: there a cell's two faces are the same global node, so the assembly
    (PAPER.md:204 (iii)) has to accumulate both local contributions."""
    L, p = (2.0, 3.3, 1.7), 3
    mesh = fo.Mesh(nc, L, p, kfrac)
    ham = fo.Hamiltonian(mesh, None, None, None, None)
    X = inp.make_vectors(mesh.nnodes, 3, seed=2)
    ref = 2.0 * fo.apply_MinvH(ham, X)                            # H = K/2 here
    A = []
    for d in range(3):
        K1, m1 = _line_operator(nc[d], L[d], p, kfrac[d])
        A.append(K1 / m1[:, None])
    n1x, n1y, n1z = mesh.n1
    T = X.reshape(n1z, n1y, n1x, 2, 3)
    out = np.einsum("ia,zyasv->zyisv", A[0], T) + np.einsum("jb,zbxsv->zjxsv", A[1], T) \
        + np.einsum("kc,cyxsv->kyxsv", A[2], T)
    assert np.max(np.abs(out.reshape(X.shape) - ref)) < 1e-12 * np.max(np.abs(ref))


# ------------------------------------------------------------------ P5
@pytest.mark.parametrize("degree", [1, 2, 8, 20])
def test_p5_residual_recurrence_equals_standard_for_any_lambda(degree):
    cfg = inp.tiny_config(ncell=2, p=3, L=5.0, kfrac=(0.25, 0.0, 0.0), natoms=1, nproj=4, nvec=3)
    mesh = _mesh(cfg)
    ham, _ = _ham(cfg, mesh)
    X = inp.make_vectors(mesh.nnodes, 3, seed=0)
    a0, b = fo.lanczos_bounds(ham, inp.lanczos_start(mesh.nnodes), 10)
    a = a0 + 0.1 * (b - a0)
    Y10 = fo.cheb_filter_standard(ham, X, degree, a, b, a0)
    for lam in (np.array([0.3, -1.0, 7.0]), np.zeros(3)):
        Y11 = fo.cheb_filter_residual(ham, X, lam, degree, a, b, a0)
        assert np.linalg.norm(Y11 - Y10) < 1e-12 * np.linalg.norm(Y10)


# ------------------------------------------------------------------ P6 + P10 (brute force)
def _brute_force(ham):
    mesh = ham.mesh
    H = fo.dense_H(ham)
    assert np.max(np.abs(H - H.conj().T)) < 1e-12 * np.max(np.abs(H))
    msq = np.sqrt(np.repeat(mesh.mass, 2))
    A = H / msq[:, None] / msq[None, :]
    lam, V = np.linalg.eigh(0.5 * (A + A.conj().T))
    return lam, V, msq


def _cheb_T(m, t):
    t = np.asarray(t, dtype=np.float64)
    out = np.empty_like(t)
    ins = np.abs(t) <= 1
    out[ins] = np.cos(m * np.arccos(t[ins]))
    s = np.sign(t[~ins])
    out[~ins] = (s ** m) * np.cosh(m * np.arccosh(np.abs(t[~ins])))
    return out


@pytest.mark.parametrize("kfrac", [(0.0, 0.0, 0.0), (0.25, 0.0, 0.0)])
def test_p10_filter_equals_dense_polynomial_2x2x2_p2(kfrac):
    """north_star check (b): 2x2x2 cells, p=2: filter output vs C_m(M^-1 H) by dense eigendecomposition."""
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, kfrac=kfrac, natoms=1, nproj=4, nvec=5, degree=9)
    mesh = _mesh(cfg)
    assert mesh.nnodes == 64
    ham, _ = _ham(cfg, mesh)
    assert ham.atoms[0][0].size >= 8
    lam, V, msq = _brute_force(ham)
    b = lam[-1] + 0.5
    a0 = lam[0] - 0.1
    a = lam[len(lam) // 3]
    c, e = 0.5 * (a + b), 0.5 * (b - a)
    m = cfg.degree
    X = inp.make_vectors(64, 5, seed=0)
    Cm = _cheb_T(m, (lam - c) / e) / _cheb_T(m, np.array([(a0 - c) / e]))[0]
    Xf = X.reshape(128, 5)
    ref = (V * Cm[None, :]) @ (V.conj().T @ (msq[:, None] * Xf)) / msq[:, None]
    Y10 = fo.cheb_filter_standard(ham, X, m, a, b, a0).reshape(128, 5)
    rq = np.real(np.einsum("iv,iv->v", Xf.conj(), (fo.apply_H(ham, X)).reshape(128, 5))) / \
        np.real(np.einsum("iv,iv->v", Xf.conj(), (msq ** 2)[:, None] * Xf))
    Y11 = fo.cheb_filter_residual(ham, X, rq, m, a, b, a0).reshape(128, 5)
    assert np.linalg.norm(Y10 - ref) < 1e-11 * np.linalg.norm(ref)
    assert np.linalg.norm(Y11 - ref) < 1e-11 * np.linalg.norm(ref)


def test_p6_eigenvector_scaled_by_chebyshev_ratio_and_sigma_identity():
    """north_star check (a): an eigenvector of M^-1 H is scaled by T_m of its mapped eigenvalue."""
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, natoms=1, nproj=4)
    mesh = _mesh(cfg)
    ham, _ = _ham(cfg, mesh)
    lam, V, msq = _brute_force(ham)
    b, a0, a = lam[-1] + 1.0, lam[0], lam[20]
    c, e = 0.5 * (a + b), 0.5 * (b - a)
    for m in (1, 2, 7, 16):
        for j in (0, 5, 60, 127):
            v = (V[:, j] / msq).reshape(64, 2, 1)
            scale = _cheb_T(m, np.array([(lam[j] - c) / e]))[0] / _cheb_T(m, np.array([(a0 - c) / e]))[0]
            for Y in (fo.cheb_filter_standard(ham, v, m, a, b, a0),
                      fo.cheb_filter_residual(ham, v, np.array([lam[j] + 0.3]), m, a, b, a0)):
                assert np.linalg.norm(Y - scale * v) < 1e-10 * max(abs(scale), 1e-3) * np.linalg.norm(v)
    # sigma_{k+1} = T_k(t0) / T_{k+1}(t0), t0 = (a0-c)/e
    _, _, sig = fo.cheb_sigmas(12, a, b, a0)
    t0 = np.array([(a0 - c) / e])
    for k in range(0, 12):
        assert abs(sig[k + 1] - _cheb_T(k, t0)[0] / _cheb_T(k + 1, t0)[0]) < 1e-12 * abs(sig[k + 1])


# ------------------------------------------------------------------ P7, P8
def _free_1d(ncell, L, p, kfrac):
    K1, m1 = _line_operator(ncell, L, p, kfrac)
    A = K1 / np.sqrt(m1)[:, None] / np.sqrt(m1)[None, :]
    mu, W = np.linalg.eigh(0.5 * (A + A.conj().T))
    return mu, W / np.sqrt(m1)[:, None]


def test_p7_free_electron_spectrum_golden():
    for line in open(os.path.join(GOLD, "free_electron_lambda_max.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, nc, L, p, kx, what, val = line.split()
        mu_x, _ = _free_1d(int(nc), float(L), int(p), float(kx))
        mu_0, _ = _free_1d(int(nc), float(L), int(p), 0.0)
        got = 0.5 * (mu_x[-1] + 2 * mu_0[-1]) if what == "lambda_max" else 0.5 * (mu_x[0] + 2 * mu_0[0])
        assert abs(got - float(val)) < 2e-5 * max(1.0, abs(float(val))) if what == "lambda_max" \
            else abs(got - float(val)) < 1e-7


@pytest.mark.parametrize("kfrac", [(0.0, 0.0, 0.0), (0.25, 0.0, 0.4)])
def test_p7_p8_tensor_product_eigenvectors_with_constant_fields(kfrac):
    """Free-electron eigenpairs 1/2(mu_i+mu_j+mu_k), v_i(x)v_j(x)v_k(x)spinor; constant V0, B shift by V0 +- |B|."""
    nc, L, p = (2, 2, 3), (3.0, 2.5, 4.0), 3
    mesh = fo.Mesh(nc, L, p, kfrac)
    M = mesh.nnodes
    mus, Ws = zip(*[_free_1d(nc[d], L[d], p, kfrac[d]) for d in range(3)])
    V0, B = -0.7, np.array([0.3, -0.2, 0.5])
    ham = fo.Hamiltonian(mesh, np.full(M, V0), np.full(M, B[0]), np.full(M, B[1]), np.full(M, B[2]))
    sig = np.array([[B[2], B[0] - 1j * B[1]], [B[0] + 1j * B[1], -B[2]]])
    sv, su = np.linalg.eigh(sig)                                   # -|B|, +|B|
    assert abs(sv[1] - np.linalg.norm(B)) < 1e-14
    for (i, j, k) in [(0, 0, 0), (1, 2, 3), (5, 4, 8), (nc[0] * p - 1, nc[1] * p - 1, nc[2] * p - 1)]:
        v = np.einsum("z,y,x->zyx", Ws[2][:, k], Ws[1][:, j], Ws[0][:, i]).reshape(M)
        for s in range(2):
            X = (v[:, None] * su[None, :, s]).reshape(M, 2, 1)
            lam = 0.5 * (mus[0][i] + mus[1][j] + mus[2][k]) + V0 + sv[s]
            Y = fo.apply_MinvH(ham, X)
            assert np.linalg.norm(Y - lam * X) < 1e-11 * max(1.0, abs(lam)) * np.linalg.norm(X)


# ------------------------------------------------------------------ P9
def test_p9_plane_wave_convergence_golden():
    """north_star check (c): discrete eigenvalue -> (2 pi n / L)^2 spectrally as p rises (from below)."""
    errs = {}
    for p in (2, 4, 6, 8):
        mu, _ = _free_1d(4, 7.0, p, 0.0)
        errs[p] = (mu[1] - (2 * math.pi / 7.0) ** 2) / (2 * math.pi / 7.0) ** 2
    assert abs(errs[2]) > abs(errs[4]) > abs(errs[6]) and abs(errs[8]) < 1e-11
    for line in open(os.path.join(GOLD, "planewave_rel_error.txt")):
        if line.startswith("#") or not line.strip():
            continue
        p, val = line.split()
        p, val = int(p), float(val)
        if p <= 6:
            assert abs(errs[p] - val) < 0.06 * abs(val)            # printed to 2 digits
    # with a Bloch twist: mu_min -> k^2
    k = 0.25 * 2 * math.pi / 7.0
    mu, _ = _free_1d(4, 7.0, 6, 0.25)
    assert abs(mu[0] - k * k) < 1e-10


# ------------------------------------------------------------------ P11
def test_p11_integer_kfrac_is_gamma():
    cfg0 = inp.tiny_config(ncell=2, p=3, L=5.0, kfrac=(0, 0, 0), natoms=1, nproj=4)
    cfg1 = inp.tiny_config(ncell=2, p=3, L=5.0, kfrac=(1.0, -2.0, 3.0), natoms=1, nproj=4)
    m0, m1 = _mesh(cfg0), _mesh(cfg1)
    h0, _ = _ham(cfg0, m0)
    h1, _ = _ham(cfg1, m1)
    X = inp.make_vectors(m0.nnodes, 2)
    A, B = fo.apply_MinvH(h0, X), fo.apply_MinvH(h1, X)
    assert np.max(np.abs(A - B)) < 1e-11 * np.max(np.abs(A))


def test_p11_translation_invariance_pins_projector_phase():
    """Shifting atoms and fields by one cell length leaves the spectrum unchanged at k != 0,
    also when the support crosses the periodic boundary; the opposite phase sign breaks it."""
    import dataclasses
    cfg = inp.tiny_config(ncell=3, p=2, L=6.0, kfrac=(0.25, 0.0, 0.0), natoms=1, nproj=4, ngauss=1)
    mesh = _mesh(cfg)
    xyz = mesh.node_coords()
    h = cfg.L / cfg.ncell

    def spectrum(atom, centre, flip=False):
        V, Bx, By, Bz = inp.local_fields(cfg, xyz, centre[None, :])
        # B rotates with x: make it translation-covariant by zeroing it (only V and P are shifted)
        so, sn, npj, P = inp.projector_tables(cfg, xyz, atom[None, :])
        if flip:
            P = np.conj(P)                                         # opposite phase sign (P real x phase)
        D = inp.soc_couplings(cfg)
        ham = fo.Hamiltonian(mesh, V, None, None, None, so, sn, npj, P, D)
        H = fo.dense_H(ham)
        msq = np.sqrt(np.repeat(mesh.mass, 2))
        return np.linalg.eigvalsh(H / msq[:, None] / msq[None, :]), so[-1]

    atom = np.array([4.6, 2.9, 3.1])                               # support (cutoff 2) crosses x = L when shifted
    centre = np.array([1.0, 2.0, 3.0])
    shift = np.array([h, 0.0, 0.0])
    s0, n0 = spectrum(atom, centre)
    s1, n1 = spectrum(np.mod(atom + shift, cfg.L), np.mod(centre + shift, cfg.L))
    assert n0 == n1 and n0 > 20
    assert np.max(np.abs(s0 - s1)) < 1e-11
    f0, _ = spectrum(atom, centre, flip=True)
    f1, _ = spectrum(np.mod(atom + shift, cfg.L), np.mod(centre + shift, cfg.L), flip=True)
    assert np.max(np.abs(f0 - f1)) > 1e-4


def test_p11_scalar_coupling_decouples_spins():
    cfg = inp.tiny_config(ncell=2, p=3, L=5.0, natoms=1, nproj=4)
    mesh = _mesh(cfg)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    D = 0.37 * np.eye(8, dtype=np.complex128)[None]
    ham = fo.Hamiltonian(mesh, hi.V, None, None, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj, hi.P, D)
    X = inp.make_vectors(mesh.nnodes, 2)
    X[:, 1, :] = 0
    Y = fo.apply_H(ham, X)
    assert np.max(np.abs(Y[:, 1, :])) == 0.0 and np.max(np.abs(Y[:, 0, :])) > 0


# ------------------------------------------------------------------ P12
def test_p12_column_independence():
    cfg = inp.tiny_config(ncell=2, p=3, L=5.0, kfrac=(0.25, 0, 0), natoms=1, nproj=8, nvec=6)
    mesh = _mesh(cfg)
    ham, _ = _ham(cfg, mesh)
    X = inp.make_vectors(mesh.nnodes, 6)
    lam = np.linspace(-1, 2, 6)
    a0, b = fo.lanczos_bounds(ham, inp.lanczos_start(mesh.nnodes), 8)
    a = a0 + 0.1 * (b - a0)
    Y = fo.cheb_filter_residual(ham, X, lam, 7, a, b, a0)
    Ys = fo.cheb_filter_residual(ham, X[:, :, [4, 1]], lam[[4, 1]], 7, a, b, a0)
    assert np.linalg.norm(Y[:, :, [4, 1]] - Ys) < 1e-13 * np.linalg.norm(Ys)
    assert np.array_equal(inp.make_vectors(mesh.nnodes, [4, 1]), X[:, :, [4, 1]])


# ------------------------------------------------------------------ Lanczos / RR
def test_lanczos_bound_brackets_spectrum_and_rr_recovers_eigenvalues():
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, natoms=1, nproj=4)
    mesh = _mesh(cfg)
    ham, _ = _ham(cfg, mesh)
    lam, V, msq = _brute_force(ham)
    a0, b = fo.lanczos_bounds(ham, inp.lanczos_start(mesh.nnodes), 10)
    assert b >= lam[-1] and a0 >= lam[0] - 1e-9 and a0 < lam[-1]
    # free electron check of the bound against the exact lambda_max (P7)
    hf = fo.Hamiltonian(mesh, None, None, None, None)
    mu, _ = _free_1d(2, 4.0, 2, 0.0)
    _, bf = fo.lanczos_bounds(hf, inp.lanczos_start(mesh.nnodes), 10)
    assert bf >= 1.5 * mu[-1] - 1e-9
    # Algorithm 1 converges to the dense eigenvalues
    X0 = inp.make_vectors(mesh.nnodes, 12, seed=4)
    X, ritz, hist = fo.subspace_iteration(ham, X0, degree=12, b=b, passes=40, tol=1e-9, n_check=8)
    assert hist[-1] <= 1e-9
    assert np.max(np.abs(ritz[:8] - lam[:8])) < 1e-9


# ------------------------------------------------------------------ nonlocal block, element by element
def test_nonlocal_block_elementwise_definition():
    """H_nl[(I,s),(J,s')] = m_I m_J sum_{b,b'} P[I,b] D[2b+s, 2b'+s'] conj(P[J,b'])  (eq. 7, O5),
    written as scalar loops: pins the orientation of D_a and the 2 beta + s index convention."""
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, kfrac=(0.25, 0.0, 0.0), natoms=1, nproj=4)
    mesh = _mesh(cfg)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    ham = fo.Hamiltonian(mesh, None, None, None, None, hi.supp_off, hi.supp_node, hi.nproj, hi.P, hi.D)
    ham0 = fo.Hamiltonian(mesh, None, None, None, None)
    Hnl = fo.dense_H(ham) - fo.dense_H(ham0)
    nodes = hi.supp_node
    P = hi.P.reshape(nodes.size, 4)
    D = hi.D[0]
    assert np.max(np.abs(D - D.T)) > 1e-2                          # D is genuinely complex Hermitian
    ref = np.zeros_like(Hnl)
    m = mesh.mass
    for ii, I in enumerate(nodes):
        for jj, J in enumerate(nodes):
            for s in range(2):
                for t in range(2):
                    acc = 0.0
                    for b in range(4):
                        for bp in range(4):
                            acc += P[ii, b] * D[2 * b + s, 2 * bp + t] * np.conj(P[jj, bp])
                    ref[2 * I + s, 2 * J + t] = m[I] * m[J] * acc
    assert np.max(np.abs(Hnl - ref)) < 1e-13 * np.max(np.abs(ref))


# ------------------------------------------------------------------ pointwise local fields (eq. 12, O3)
@pytest.mark.parametrize("nc,L,p,kfrac", [((3, 3, 3), (6.0, 6.0, 6.0), 3, (0.0, 0.0, 0.0)),
                                          ((1, 3, 2), (2.0, 4.5, 3.0), 4, (0.25, 0.1, 0.0)),
                                          ((2, 1, 1), (3.0, 2.0, 2.5), 2, (0.0, 0.0, 0.3))])
def test_local_fields_act_pointwise_with_eq12_spin_blocks(nc, L, p, kfrac):
    """With seeded NON-constant V, B and no projectors,  M^-1 H x - M^-1 H_0 x  (H_0: zero fields) must equal
    [[V+Bz, Bx - i By], [Bx + i By, V - Bz]]_I x_I  node by node (eq. 12 spin blocks, pointwise
    under GLL collocation, reading O3).  Pins WHICH node's field value stage (ii) of apply_H uses (a field
    taken at a permuted node survives every constant-field pin and Hermiticity), and, on the meshes with a
    single cell in a direction, the duplicate scatter of the potential term (np.add.at branch)."""
    mesh = fo.Mesh(nc, L, p, kfrac)
    rng = np.random.default_rng(77)
    M = mesh.nnodes
    V, Bx, By, Bz = (rng.uniform(-1.0, 1.0, M) for _ in range(4))
    ham = fo.Hamiltonian(mesh, V, Bx, By, Bz)
    ham0 = fo.Hamiltonian(mesh, None, None, None, None)
    X = inp.make_vectors(M, 3, seed=9)
    got = fo.apply_MinvH(ham, X) - fo.apply_MinvH(ham0, X)
    up, dn = X[:, 0, :], X[:, 1, :]
    ref = np.empty_like(X)
    ref[:, 0, :] = (V + Bz)[:, None] * up + (Bx - 1j * By)[:, None] * dn
    ref[:, 1, :] = (Bx + 1j * By)[:, None] * up + (V - Bz)[:, None] * dn
    scale = np.max(np.abs(fo.apply_MinvH(ham0, X)))               # the difference cancels the kinetic term
    assert np.max(np.abs(got - ref)) < 1e-13 * scale
    # each field separately, so that a swap of two fields cannot cancel
    for k, name in enumerate(["V", "Bx", "By", "Bz"]):
        f = [None] * 4
        f[k] = (V, Bx, By, Bz)[k]
        hk = fo.Hamiltonian(mesh, *f)
        gk = fo.apply_MinvH(hk, X) - fo.apply_MinvH(ham0, X)
        fk = f[k][:, None]
        rk = np.empty_like(X)
        if name == "V":
            rk[:, 0, :], rk[:, 1, :] = fk * up, fk * dn
        elif name == "Bx":
            rk[:, 0, :], rk[:, 1, :] = fk * dn, fk * up
        elif name == "By":
            rk[:, 0, :], rk[:, 1, :] = -1j * fk * dn, 1j * fk * up
        else:
            rk[:, 0, :], rk[:, 1, :] = fk * up, -fk * dn
        assert np.max(np.abs(gk - rk)) < 1e-13 * scale, name


# ------------------------------------------------------------------ node coordinates (PAPER.md:92 GLL nodes)
def test_node_coords_closed_forms_and_quadrature_exactness():
    """Mesh.node_coords: (i) closed forms -- p = 2: offsets {0, h/2}; p = 4: {0, h(1 - sqrt(3/7))/2, h/2,
    h(1 + sqrt(3/7))/2} (the P1 golden nodes mapped to a cell); (ii) node ordering I = (iz N1y + iy) N1x + ix;
    (iii) with the diagonal mass as weights the nodes integrate monomials of degree <= 2p-1 per direction
    exactly:  sum_I m_I x_I^a y_I^b z_I^c = Lx^(a+1)/(a+1) ...  -- false for uniformly spaced nodes."""
    m2 = fo.Mesh((2, 1, 1), (3.0, 1.0, 1.0), 2)
    xyz = m2.node_coords()
    assert xyz.shape == (m2.nnodes, 3)
    assert np.allclose(xyz[:4, 0], [0.0, 0.75, 1.5, 2.25], atol=1e-15)        # h = 1.5: {0, h/2} per cell
    m4 = fo.Mesh((1, 2, 1), (1.0, 4.0, 1.0), 4)
    xyz = m4.node_coords()
    h = 2.0
    r = math.sqrt(3.0 / 7.0)
    ref = np.array([0.0, h * (1 - r) / 2, h / 2, h * (1 + r) / 2])
    ys = xyz[::4, 1][:8]                                                       # x fastest: stride N1x = 4 walks y
    assert np.allclose(ys, np.concatenate([ref, h + ref]), atol=1e-15)
    # ordering: x fastest, then y, then z
    mesh = fo.Mesh((2, 3, 2), (3.0, 4.5, 2.0), 3)
    xyz = mesh.node_coords()
    n1x, n1y, n1z = mesh.n1
    g = xyz.reshape(n1z, n1y, n1x, 3)
    assert np.all(np.diff(g[0, 0, :, 0]) > 0) and np.all(g[:, :, 0, 0] == 0.0)
    assert np.all(np.diff(g[0, :, 0, 1]) > 0) and np.all(g[:, 0, :, 1] == 0.0)
    assert np.all(np.diff(g[:, 0, 0, 2]) > 0) and np.all(g[0, :, :, 2] == 0.0)
    # quadrature exactness with m_I (degree <= 2p-1 = 5 per direction).  The mesh is periodic (the node at x = L
    # is the node at x = 0), so the test functions vanish at both ends: f_a(t) = t^a (L - t), a >= 1.
    Ls = mesh.L

    def f(t, a, Ld):
        return t ** a * (Ld - t)

    def f_int(a, Ld):
        return Ld ** (a + 2) / (a + 1) - Ld ** (a + 2) / (a + 2)

    for (a, b, c) in [(1, 1, 1), (4, 1, 1), (1, 4, 1), (1, 1, 4), (2, 3, 1), (4, 4, 4), (3, 1, 2)]:
        got = np.sum(mesh.mass * f(xyz[:, 0], a, Ls[0]) * f(xyz[:, 1], b, Ls[1]) * f(xyz[:, 2], c, Ls[2]))
        exact = f_int(a, Ls[0]) * f_int(b, Ls[1]) * f_int(c, Ls[2])
        assert abs(got - exact) < 1e-12 * exact, (a, b, c)
    # ... and NOT beyond: degree 2p = 6 in one direction is not integrated exactly by (p+1)-point GLL
    got = np.sum(mesh.mass * f(xyz[:, 0], 5, Ls[0]) * f(xyz[:, 1], 1, Ls[1]) * f(xyz[:, 2], 1, Ls[2]))
    exact = f_int(5, Ls[0]) * f_int(1, Ls[1]) * f_int(1, Ls[2])
    assert abs(got - exact) > 1e-7 * exact


# ------------------------------------------------------------------ Algorithm 1 line 10
def test_algorithm1_line10_bounds_update():
    """Alg. 1 line 10: after each RR the filter is called with lambda_min <- lowest Ritz value,
    lambda_T <- highest Ritz value of the block, lambda_max fixed.  Recorded through the filter_fn hook."""
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, natoms=1, nproj=4)
    mesh = _mesh(cfg)
    ham, _ = _ham(cfg, mesh)
    lam_exact, _, _ = _brute_force(ham)
    calls = []

    def spy(X, lam, m, a, bb, a0):
        calls.append((np.array(lam), a, bb, a0))
        return fo.cheb_filter_residual(ham, X, lam, m, a, bb, a0)

    X0 = inp.make_vectors(mesh.nnodes, 6, seed=4)
    b = lam_exact[-1] + 1.0
    fo.subspace_iteration(ham, X0, degree=6, b=b, passes=3, tol=0.0, filter_fn=spy)
    assert len(calls) == 3
    for lam, a, bb, a0 in calls:
        assert bb == b
        assert a0 == lam[0] == np.min(lam)                 # lambda_min <- lambda_1
        assert a == lam[-1] == np.max(lam)                 # lambda_T  <- lambda_N
    # Ritz values decrease monotonically towards the exact ones from above
    assert calls[2][0][0] <= calls[0][0][0] + 1e-12 and calls[2][0][0] >= lam_exact[0] - 1e-10
