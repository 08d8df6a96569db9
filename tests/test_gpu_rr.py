"""Parity of the CUDA Rayleigh-Ritz pieces (through the C ABI) against the CPU oracle.  `-m gpu`.

Tolerances: the projection is FP64 with a different summation order than the oracle's matmul (split rows, REDs): relative
Frobenius 1e-12.  The mixed-precision rotation is FP32 in its off-diagonal part on both sides, in different summation orders:
relative Frobenius 1e-5 (north_star's FP32-inexact bar) and, as a property, within the FP32 bound of the exact FP64 product;
the FP64 rotation: 1e-13.  The tcgen05 rotation (CHFSI_TF32X3: FP64 diagonal + 3xTF32 off-diagonal, FP32 accumulation in tensor
memory) is held to the same two bars as the FP32 one (measured 1e-7 ... 1.3e-6 on these cases).  Several row tiles, both column
halves, ragged K chunks and ragged rows are covered by the sizes below and by test_rotate_tcgen05_tiles."""
import numpy as np
import pytest

from paper_2605_30128_b200 import inputs as inp
from test_gpu_parity import Problem, env, relerr  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ro():
    from oracle import rr_oracle
    return rr_oracle


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@pytest.mark.parametrize("nrows,nvec,ld", [(1000, 5, 5), (4099, 70, 72), (20000, 130, 130), (7, 64, 64)])
def test_project_plain(env, ro, nrows, nvec, ld):
    """No mass weighting, general (non-Hermitian) and Hermitian forms; ragged tiles, several row slabs, ld > nvec."""
    torch, _, B = env
    rng = np.random.default_rng(nrows)
    A, Bm = _rand(rng, nrows, ld), _rand(rng, nrows, ld)
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(Bm).cuda()
    S = torch.full((nvec, nvec), float("nan"), dtype=torch.complex128, device="cuda")
    B.chfsi_rr_project(None, Ad[:, :nvec], Bd[:, :nvec], S, use_mass=False, hermitian=False)
    assert relerr(S.cpu().numpy(), ro.rr_project(A[:, :nvec], Bm[:, :nvec])) < 1e-12
    B.chfsi_rr_project(None, Ad[:, :nvec], Ad[:, :nvec], S, use_mass=False, hermitian=True)
    Sh = S.cpu().numpy()
    assert relerr(Sh, ro.rr_project(A[:, :nvec], A[:, :nvec])) < 1e-12
    assert np.array_equal(Sh, Sh.conj().T) and not np.diag(Sh).imag.any()


def test_project_with_mass_on_a_mesh_and_rr_eigenvalues(env, ro):
    """Y^H M Y and Y^H H Y on a Bloch mesh with all terms on (H Y from chfsi_apply_H), against the oracle's projection of the
    oracle's H Y; then the whole Rayleigh-Ritz step (project, diagonalise on the host, rotate) against LAPACK on the dense pencil."""
    torch, fo, B = env
    cfg = inp.tiny_config(ncell=(3, 2, 2), p=4, L=(6.0, 4.0, 4.0), kfrac=(0.25, 0.0, 0.1), nvec=24, natoms=2, nproj=8, ngauss=3)
    pb = Problem(env, cfg)
    try:
        Y = inp.make_vectors(cfg.nnodes, 24)
        m2 = np.repeat(pb.omesh.mass, 2)
        HY = fo.apply_MinvH(pb.oham, Y)
        Yd = torch.from_numpy(Y).cuda()
        HYd = torch.empty_like(Yd)
        B.chfsi_apply_H(pb.gmesh, B.FP64, Yd, HYd, pb.work(B.FP64, B.RECUR_STANDARD, 24))
        SM = torch.empty((24, 24), dtype=torch.complex128, device="cuda")
        SH = torch.empty_like(SM)
        B.chfsi_rr_project(pb.gmesh, Yd, Yd, SM)
        B.chfsi_rr_project(pb.gmesh, Yd, HYd, SH)
        Yf, HYf = Y.reshape(-1, 24), HY.reshape(-1, 24)
        assert relerr(SM.cpu().numpy(), ro.rr_project(Yf, Yf, m2)) < 1e-12
        assert relerr(SH.cpu().numpy(), ro.rr_project(Yf, HYf, m2)) < 1e-12
        # Rayleigh-Ritz: eigenvalues of the projected pencil = those of the oracle's projected pencil; rotation gives M-orthonormal Ritz vectors
        SMh, SHh = SM.cpu().numpy(), SH.cpu().numpy()
        L = np.linalg.cholesky(SMh); Li = np.linalg.inv(L)
        ev, Z = np.linalg.eigh(Li @ SHh @ Li.conj().T)
        So, Ho = ro.rr_project(Yf, Yf, m2), ro.rr_project(Yf, HYf, m2)
        Lo = np.linalg.inv(np.linalg.cholesky(So))
        assert np.abs(ev - np.linalg.eigvalsh(Lo @ Ho @ Lo.conj().T)).max() < 1e-10
        Q = Li.conj().T @ Z
        Qd = torch.from_numpy(Q).cuda()
        work = torch.empty(B.chfsi_rr_rotate_workspace_bytes(24), dtype=torch.uint8, device="cuda")
        for prec, mixed, tol in [(B.FP64, False, 1e-13), (B.FP32, True, 1e-5), (B.TF32X3, True, 1e-5)]:
            Xd = torch.full_like(Yd, float("nan"))
            B.chfsi_rr_rotate(prec, Yd, Qd, Xd, work)
            X = Xd.cpu().numpy().reshape(-1, 24)
            assert relerr(X, ro.rr_rotate(Yf, Q, mixed)) < tol
            G = ro.rr_project(X, X, m2)
            assert np.abs(G - np.eye(24)).max() < (1e-10 if not mixed else 1e-4)
    finally:
        pb.close()


@pytest.mark.parametrize("nrows,nvec,ld", [(300, 6, 8), (5000, 100, 100), (130, 257, 260)])
def test_rotate_fp64_and_mixed(env, ro, nrows, nvec, ld):
    torch, _, B = env
    rng = np.random.default_rng(nvec)
    Y = _rand(rng, nrows, ld)
    Hm = _rand(rng, nvec, nvec); Hm = Hm + Hm.conj().T
    _, U = np.linalg.eigh(Hm)
    near = np.diag(np.diag(U)) + 1e-3 * (U - np.diag(np.diag(U)))       # near convergence Q is close to diagonal
    work = torch.empty(B.chfsi_rr_rotate_workspace_bytes(nvec), dtype=torch.uint8, device="cuda")
    Yd = torch.from_numpy(Y).cuda()
    for Q in (U, near, np.eye(nvec, dtype=np.complex128)):
        Qd = torch.from_numpy(np.ascontiguousarray(Q)).cuda()
        exact = ro.rr_rotate(Y[:, :nvec], Q, mixed=False)
        for prec, mixed, tol in [(B.FP64, False, 1e-13), (B.FP32, True, 1e-5), (B.TF32X3, True, 1e-5)]:
            out = torch.full((nrows, ld), float("nan"), dtype=torch.complex128, device="cuda")
            B.chfsi_rr_rotate(prec, Yd[:, :nvec], Qd, out[:, :nvec], work)
            got = out.cpu().numpy()[:, :nvec]
            assert relerr(got, ro.rr_rotate(Y[:, :nvec], Q, mixed)) < tol
            off = np.linalg.norm(Y[:, :nvec] @ (Q - np.diag(np.diag(Q)))) / np.linalg.norm(exact)
            assert relerr(got, exact) <= (1e-13 if not mixed else 1e-6 * (off + 1e-9) * 50)   # FP32 error scales with |Q_non-diag|
            if ld > nvec:
                assert np.isnan(out.cpu().numpy()[:, nvec:]).all()                            # padding columns untouched
    with pytest.raises(B.ChfsiError):
        B.chfsi_rr_rotate(B.FP64, Yd[:, :nvec], Qd, Yd[:, :nvec], work)                      # in place is refused
    with pytest.raises(B.ChfsiError):
        B.chfsi_rr_rotate(B.TF32, Yd[:, :nvec], Qd, out[:, :nvec], work)


@pytest.mark.parametrize("nrows,nvec", [(1, 1), (127, 15), (129, 16), (1000, 128), (385, 129), (2500, 300), (200, 1024)])
def test_rotate_tcgen05_tiles(env, ro, nrows, nvec):
    """The tcgen05 rotation across its tile boundaries: 1 / 2 / 3 / 8 column tiles of 128 vectors, ragged 16-vector K chunks, ragged
    128-row tiles; against the oracle's mixed product and the exact FP64 one, elementwise as well as in norm."""
    torch, _, B = env
    rng = np.random.default_rng(1000 * nvec + nrows)
    Y = _rand(rng, nrows, nvec)
    Q = _rand(rng, nvec, nvec) / np.sqrt(nvec)
    work = torch.empty(B.chfsi_rr_rotate_workspace_bytes(nvec), dtype=torch.uint8, device="cuda")
    out = torch.full((nrows, nvec), float("nan"), dtype=torch.complex128, device="cuda")
    B.chfsi_rr_rotate(B.TF32X3, torch.from_numpy(Y).cuda(), torch.from_numpy(Q).cuda(), out, work)
    got = out.cpu().numpy()
    exact = Y @ Q
    assert np.isfinite(got).all()
    assert relerr(got, ro.rr_rotate(Y, Q, True)) < 1e-5 and relerr(got, exact) < 1e-5
    assert np.abs(got - exact).max() < 1e-4 * np.abs(exact).max()


def test_project_full_size_block_properties(env, ro):
    """configs[1]'s block (221,184 rows x 128 vectors) in the launch configuration bench.py times: sampled entries of
    Y^H M Y against the oracle's column dot products, Hermitian symmetry, positive diagonal."""
    torch, fo, B = env
    cfg = inp.CONFIGS[1]
    mesh = B.chfsi_mesh_create(cfg.ncell, cfg.L, cfg.p, cfg.kfrac, 0)
    B.chfsi_ham_set(mesh, None, None, None, None)                       # builds the device mass (bare Laplacian)
    try:
        cols = [0, 1, 63, 64, 127]
        Yc = inp.make_vectors(cfg.nnodes, cols)
        Yd = torch.zeros((cfg.nnodes, 2, 128), dtype=torch.complex128, device="cuda")
        g = torch.Generator(device="cuda"); g.manual_seed(5)
        torch.view_as_real(Yd)[...] = torch.rand((cfg.nnodes, 2, 128, 2), generator=g, device="cuda", dtype=torch.float64) - 0.5
        Yd[:, :, cols] = torch.from_numpy(Yc).cuda()
        S = torch.empty((128, 128), dtype=torch.complex128, device="cuda")
        B.chfsi_rr_project(mesh, Yd, Yd, S)
        Sh = S.cpu().numpy()
        m2 = np.repeat(fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac).mass, 2)
        ref = ro.rr_project(Yc.reshape(-1, len(cols)), Yc.reshape(-1, len(cols)), m2)
        assert relerr(Sh[np.ix_(cols, cols)], ref) < 1e-12
        assert np.array_equal(Sh, Sh.conj().T) and (np.diag(Sh).real > 0).all()
    finally:
        B.chfsi_mesh_destroy(mesh)
