"""Parity of the CUDA Poisson path (Kx kernel, Chebyshev-Jacobi preconditioner, batched Algorithm 2; through the C ABI)
against the CPU oracle.  `-m gpu`.  FP64: apply_K 1e-13 relative; PCG solutions agree to the solver
tolerance (both sides iterate to an absolute residual 1e-10)."""
import numpy as np
import pytest

from test_gpu_parity import env, relerr  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def po():
    from oracle import poisson_oracle
    return poisson_oracle


def _block(cols, nnodes, nvec):
    """real columns [M, 4 nvec] (cid = (s nvec + v) 2 + ri) -> complex block [M, 2, nvec]"""
    c = cols.reshape(nnodes, 2, nvec, 2)
    return np.ascontiguousarray(c[..., 0] + 1j * c[..., 1])


def _cols(block):
    nn, _, nv = block.shape
    return np.stack([block.real, block.imag], axis=-1).reshape(nn, 4 * nv)


def _handle(B, ncell, L, p):
    mesh = B.chfsi_mesh_create(ncell, L, p, (0.0, 0.0, 0.0), 0)
    B.chfsi_ham_set(mesh, None, None, None, None)
    return mesh


def _lanczos(torch, B, mesh, kd_d, nnodes, steps=10, seed=0):
    """Harness side of PAPER.md:195: largest Ritz value + residual norm of K_diag^-1 K in the K_diag inner product, one column."""
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    v = torch.zeros((nnodes, 2, 1), dtype=torch.complex128, device="cuda")
    v[:, 0, 0] = torch.randn(nnodes, generator=g, device="cuda", dtype=torch.float64)
    col = lambda t: t[:, 0, 0].real
    x = col(v); x = x - (kd_d * x).sum() / kd_d.sum(); x = x / torch.sqrt((kd_d * x * x).sum())
    xprev = torch.zeros_like(x); beta = 0.0; al, be = [], []
    w = torch.empty_like(v)
    for j in range(steps):
        v.zero_(); v[:, 0, 0] = x
        B.chfsi_poisson_apply_K(mesh, v, w)
        f = col(w) / kd_d - beta * xprev
        a = float((kd_d * x * f).sum()); f = f - a * x; al.append(a)
        beta = float(torch.sqrt((kd_d * f * f).sum()))
        if j < steps - 1:
            be.append(beta); xprev, x = x, f / beta
    T = np.diag(al) + np.diag(be, 1) + np.diag(be, -1)
    lmax = float(np.linalg.eigvalsh(T)[-1] + beta)
    return lmax / 30.0, lmax


@pytest.mark.parametrize("p,ncell,L,nvec", [(2, (3, 2, 2), (3.0, 2.0, 2.5), 3), (4, (2, 3, 2), (4.0, 5.0, 3.0), 5),
                                            (6, (2, 2, 2), (4.0, 4.0, 4.0), 8), (8, (2, 2, 3), (4.0, 4.0, 6.0), 4)])
def test_apply_K_and_kdiag_match_the_oracle(env, po, p, ncell, L, nvec):
    torch, fo, B = env
    omesh = fo.Mesh(ncell, L, p)
    mesh = _handle(B, ncell, L, p)
    try:
        rng = np.random.default_rng(p)
        u = rng.standard_normal((omesh.nnodes, 4 * nvec))
        ref = po.apply_K(omesh, u)
        Ud = torch.from_numpy(_block(u, omesh.nnodes, nvec)).cuda()
        Wd = torch.full_like(Ud, float("nan"))
        B.chfsi_poisson_apply_K(mesh, Ud, Wd)
        got = _cols(Wd.cpu().numpy())
        assert relerr(got, ref) < 1e-13 and np.abs(got - ref).max() < 1e-12 * np.abs(ref).max()
        kd = B.chfsi_poisson_kdiag(mesh)
        kdo = po.k_diag(omesh)
        assert np.abs(kd - kdo).max() < 1e-13 * kdo.max()
    finally:
        B.chfsi_mesh_destroy(mesh)


@pytest.mark.parametrize("p,ncell,L,nvec,m", [(4, (2, 2, 3), (4.0, 4.0, 6.0), 2, 3), (6, (2, 2, 2), (4.0, 5.0, 4.0), 3, 5), (2, (3, 3, 2), (3.0, 3.0, 2.0), 1, 1)])
def test_pcg_matches_the_oracle(env, po, p, ncell, L, nvec, m):
    """Batched Algorithm 2: every real column is its own problem (different right-hand sides, one of them zero); same bounds
    on both sides.  Solutions agree to the solver tolerance, iteration counts within one (different summation orders)."""
    torch, fo, B = env
    omesh = fo.Mesh(ncell, L, p)
    mesh = _handle(B, ncell, L, p)
    try:
        rng = np.random.default_rng(10 + p)
        f = rng.standard_normal((omesh.nnodes, 4 * nvec)) * omesh.mass[:, None]
        f[:, 1] = 0.0                                                   # a zero right-hand side converges at once
        f -= f.mean(axis=0)
        kd = B.chfsi_poisson_kdiag(mesh)
        lmin, lmax = po.lanczos_bounds_scaled(omesh, kd, rng.standard_normal(omesh.nnodes))
        xo, ito, reso = po.pcg(omesh, f, m, lmin, lmax, 1e-10, 400)
        Fd = torch.from_numpy(_block(f, omesh.nnodes, nvec)).cuda()
        Xd = torch.full_like(Fd, float("nan"))
        work = torch.empty(B.chfsi_poisson_workspace_bytes(mesh, nvec), dtype=torch.uint8, device="cuda")
        it, res = B.chfsi_poisson_pcg(mesh, Fd, Xd, m, lmin, lmax, 1e-10, 400, work, check_every=5)
        x = _cols(Xd.cpu().numpy())
        assert (res.reshape(-1) < 1e-10).all() and it.reshape(-1)[1] == 0
        assert np.abs(it.reshape(-1) - ito).max() <= 1, (it.reshape(-1), ito)
        assert np.abs(x - xo).max() < 1e-8 * np.abs(xo).max()
        assert np.abs(po.apply_K(omesh, x) - f).max() < 1e-8           # it solves the oracle's system
        # never synchronising (check_every = 0) gives the same answer: finished columns freeze
        Xd2 = torch.full_like(Fd, float("nan"))
        B.chfsi_poisson_pcg(mesh, Fd, Xd2, m, lmin, lmax, 1e-10, int(it.max()) + 3, work, check_every=0, want_stats=False)
        assert np.abs(_cols(Xd2.cpu().numpy()) - x).max() < 1e-12 * np.abs(x).max()
    finally:
        B.chfsi_mesh_destroy(mesh)


@pytest.mark.parametrize("p,ncell,L,nvec", [(2, (3, 2, 2), (3.0, 2.0, 2.5), 3), (3, (2, 2, 2), (4.0, 4.0, 4.0), 2), (6, (2, 2, 2), (4.0, 5.0, 4.0), 5),
                                            (8, (2, 2, 2), (4.0, 4.0, 6.0), 4)])
def test_gauss_legendre_kx_and_pcg_match_the_oracle(env, po, p, ncell, L, nvec):
    """chfsi_poisson_set_quadrature(mesh, 1): the paper's Kx (interpolation to p + 1 Gauss points, Jacobian, integration back)
    against the oracle's rule = "gl" pipeline, its diag(K), and Algorithm 2 on top of it; then back to the default rule."""
    torch, fo, B = env
    omesh = fo.Mesh(ncell, L, p)
    mesh = _handle(B, ncell, L, p)
    try:
        B.chfsi_poisson_set_quadrature(mesh, 1)
        rng = np.random.default_rng(20 + p)
        u = rng.standard_normal((omesh.nnodes, 4 * nvec))
        ref = po.apply_K(omesh, u, "gl")
        Ud = torch.from_numpy(_block(u, omesh.nnodes, nvec)).cuda()
        Wd = torch.full_like(Ud, float("nan"))
        B.chfsi_poisson_apply_K(mesh, Ud, Wd)
        got = _cols(Wd.cpu().numpy())
        assert relerr(got, ref) < 1e-13 and np.abs(got - ref).max() < 1e-12 * np.abs(ref).max()
        kd = B.chfsi_poisson_kdiag(mesh)
        kdo = po.k_diag(omesh, "gl")
        assert np.abs(kd - kdo).max() < 1e-13 * kdo.max()
        if p <= 6:
            f = rng.standard_normal((omesh.nnodes, 4 * nvec)) * omesh.mass[:, None]
            f -= f.mean(axis=0)
            lmin, lmax = po.lanczos_bounds_scaled(omesh, kd, rng.standard_normal(omesh.nnodes), rule="gl")
            xo, ito, _ = po.pcg(omesh, f, 3, lmin, lmax, 1e-10, 400, rule="gl")
            Fd = torch.from_numpy(_block(f, omesh.nnodes, nvec)).cuda()
            Xd = torch.full_like(Fd, float("nan"))
            work = torch.empty(B.chfsi_poisson_workspace_bytes(mesh, nvec), dtype=torch.uint8, device="cuda")
            it, res = B.chfsi_poisson_pcg(mesh, Fd, Xd, 3, lmin, lmax, 1e-10, 400, work)
            x = _cols(Xd.cpu().numpy())
            assert (res < 1e-10).all() and np.abs(it.reshape(-1) - ito).max() <= 1
            assert np.abs(x - xo).max() < 1e-8 * np.abs(xo).max()
        B.chfsi_poisson_set_quadrature(mesh, 0)
        B.chfsi_poisson_apply_K(mesh, Ud, Wd)
        assert relerr(_cols(Wd.cpu().numpy()), po.apply_K(omesh, u)) < 1e-13
    finally:
        B.chfsi_mesh_destroy(mesh)


def test_cosine_charges_at_config1_size_and_error_codes(env, po):
    """configs[1]'s mesh (8^3 cells, p = 6, 110,592 nodes), 16 right-hand sides = 16 different plane-wave charges
    rho = cos(k . r): V = 4 pi rho / |k|^2 analytically; bounds from the harness-side Lanczos run."""
    torch, fo, B = env
    from paper_2605_30128_b200 import inputs as inp
    cfg = inp.CONFIGS[1]
    mesh = _handle(B, cfg.ncell, cfg.L, cfg.p)
    try:
        xyz = B.chfsi_mesh_node_coords(mesh)
        mass = B.chfsi_mesh_mass(mesh)
        nn, nvec = xyz.shape[0], 4
        ks = [(i % 3 + 1, (i // 3) % 2, (i // 6) % 3) for i in range(16)]
        rho = np.stack([np.cos(2 * np.pi / cfg.L * (k[0] * xyz[:, 0] + k[1] * xyz[:, 1] + k[2] * xyz[:, 2])) for k in ks], axis=1)
        k2 = np.array([(2 * np.pi / cfg.L) ** 2 * (k[0] ** 2 + k[1] ** 2 + k[2] ** 2) for k in ks])
        f = 4 * np.pi * mass[:, None] * rho
        f -= f.mean(axis=0)
        kd_d = torch.from_numpy(B.chfsi_poisson_kdiag(mesh)).cuda()
        lmin, lmax = _lanczos(torch, B, mesh, kd_d, nn)
        Fd = torch.from_numpy(_block(f, nn, nvec)).cuda()
        Xd = torch.empty_like(Fd)
        work = torch.empty(B.chfsi_poisson_workspace_bytes(mesh, nvec), dtype=torch.uint8, device="cuda")
        it, res = B.chfsi_poisson_pcg(mesh, Fd, Xd, 5, lmin, lmax, 1e-10, 500, work)
        x = _cols(Xd.cpu().numpy())
        exact = 4 * np.pi * rho / k2[None, :]
        err = np.abs(x - exact).max(axis=0) / np.abs(exact).max(axis=0)
        print("PCG iterations per column:", it.reshape(-1), " max rel. error vs analytic:", err.max())
        # discretisation error: 1e-10 at one wavelength per box, 1e-6 at three (2.7 cells per wavelength, p = 6)
        assert (res < 1e-10).all() and it.max() < 200 and err.max() < 2e-6 and err[0] < 1e-9
        # error behaviour: a handle with a potential is refused, so are Bloch meshes and bad bounds
        with pytest.raises(B.ChfsiError):
            B.chfsi_poisson_pcg(mesh, Fd, Xd, 5, lmax, lmin, 1e-10, 10, work)
        with pytest.raises(B.ChfsiError):
            B.chfsi_poisson_pcg(mesh, Fd, Fd, 5, lmin, lmax, 1e-10, 10, work)
        B.chfsi_ham_set(mesh, np.zeros(nn), None, None, None)
        with pytest.raises(B.ChfsiError):
            B.chfsi_poisson_apply_K(mesh, Fd, Xd)
    finally:
        B.chfsi_mesh_destroy(mesh)
