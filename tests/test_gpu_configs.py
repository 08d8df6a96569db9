"""BASELINE.json configs[2..4] at FULL size, in the launch configuration bench.py times, against the CPU oracle
on sampled columns (columns are independent), plus the eigenvalue criterion of
north_star (FP32-inexact filter: converged eigenvalues within 1e-8 Ha of the FP64 reference).  `-m gpu`.

Large blocks are never generated on the host: the sampled columns are the config's seeded columns
(`inputs.make_vectors`, seed 0) placed at chosen positions of the device block; every other column is filled
on the device (its values are irrelevant to the sampled outputs, its presence gives the timed launch shape).
"""
import os
import sys

import numpy as np
import pytest

from paper_2605_30128_b200 import inputs as inp

sys.path.insert(0, os.path.dirname(__file__))
from test_gpu_parity import Problem, relerr, TOL64, TOL32, TOL32S  # noqa: E402
TOL_TF32 = 5e-3   # single-pass TF32 per filter call; the eigenvalue criterion is what it is held to

pytestmark = pytest.mark.gpu


def check(out, ref, tol, what=""):
    """Relative Frobenius error (north_star's tolerance) AND the largest elementwise error, relative to the largest
    entry of the reference, held to 10x the same bar: a single wrong node cannot hide in the norm."""
    fro = relerr(out, ref)
    emax = float(np.max(np.abs(out - ref)) / np.max(np.abs(ref)))
    print(f"    {what}: rel. Frobenius {fro:.3e}, max elementwise {emax:.3e} (tol {tol:g})")
    assert fro < tol and emax < 10 * tol, (what, fro, emax)
    return fro


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import fe_oracle as fo
    from paper_2605_30128_b200 import binding as B
    B.lib()
    return torch, fo, B


class BigCase:
    """One mesh + Hamiltonian at a config's full size; oracle result of `ncols` seeded columns computed once."""

    def __init__(self, env, cfg, seeded_cols):
        torch, fo, B = env
        self.env, self.cfg = env, cfg
        self.pb = Problem(env, cfg)
        self.cols = list(seeded_cols)
        self.Xs = inp.make_vectors(cfg.nnodes, self.cols, seed=0)
        self.a, self.b, self.a0 = self.pb.bounds(10)
        self.lam_s = self.pb.rayleigh(self.Xs)
        self.ref = fo.cheb_filter_residual(self.pb.oham, self.Xs, self.lam_s, cfg.degree, self.a, self.b, self.a0)

    def close(self):
        self.pb.close()

    def run(self, nvec, positions, prec, chunk=0, ncols=None):
        """Filter an nvec-column device block whose columns `positions` hold the (first ncols of the) seeded sample;
        return those columns."""
        torch, fo, B = self.env
        cfg, pb = self.cfg, self.pb
        g = torch.Generator(device="cuda"); g.manual_seed(99)
        X = torch.empty((cfg.nnodes, 2, nvec), dtype=torch.complex128, device="cuda")
        Xr = torch.view_as_real(X)
        for j0 in range(0, nvec, 64):                      # filled in slabs: no full-size temporaries
            j1 = min(nvec, j0 + 64)
            Xr[:, :, j0:j1, :] = torch.rand((cfg.nnodes, 2, j1 - j0, 2), generator=g, device="cuda",
                                            dtype=torch.float64) * 2 - 1
        lam = np.zeros(nvec)
        for k, pos in enumerate(positions):
            X[:, :, pos] = torch.from_numpy(np.ascontiguousarray(self.Xs[:, :, k])).cuda()
            lam[pos] = self.lam_s[k]
        nb = chunk if chunk else nvec
        work = pb.work(prec, B.RECUR_RESIDUAL, nb)
        B.chfsi_cheb_filter(pb.gmesh, prec, B.RECUR_RESIDUAL, cfg.degree, self.a, self.b, self.a0, X, lam, X, work,
                            chunk=chunk)                   # in place (Y aliases X): halves the footprint
        torch.cuda.synchronize()
        out = np.stack([X[:, :, pos].cpu().numpy() for pos in positions], axis=2)
        del X, Xr, work
        torch.cuda.empty_cache()
        return out


C2_COLS = [0, 7, 8, 31, 32, 100, 170, 255, 256, 300, 341, 400, 448, 480, 510, 511]     # 16 seeded columns of configs[2]


@pytest.fixture(scope="module")
def case_c2(env):
    c = BigCase(env, inp.CONFIGS[2], C2_COLS)
    yield c
    c.close()


def test_config2_full_size_fp32_product(case_c2, env):
    """configs[2]: 16^3 cells, p=6, 512 vectors, degree 24: FP32 product inside eq. 11, FP32-stored multivectors, and the
    FP64 path, each against the FP64 oracle on 16 sampled columns."""
    _, _, B = env
    e32 = check(case_c2.run(512, C2_COLS, B.FP32), case_c2.ref, TOL32, "c2 fp32 product")
    assert e32 > 1e-10
    e32s = check(case_c2.run(512, C2_COLS, B.FP32_STORED), case_c2.ref, TOL32S, "c2 fp32 stored")
    assert e32s > 1e-10
    check(case_c2.run(512, C2_COLS, B.FP64), case_c2.ref, TOL64, "c2 fp64")


@pytest.mark.parametrize("nvec", [64, 128, 256, 1024])
def test_config4_sweep_nvec_and_precision(case_c2, env, nvec):
    """configs[4]: config 2's mesh, N_vec in {64,...,1024} x {FP64, FP32 product, FP32 stored, 3xTF32, TF32} (512 is the
    test above).  1024 vectors run in chunks of 256 so the workspace fits."""
    torch, _, B = env
    pos = [0, nvec // 3, nvec // 2 + 1, nvec - 1]
    chunk = 256 if nvec > 512 else 0
    ref4 = case_c2.ref[:, :, :4]                       # the first four seeded columns, placed at `pos`
    for prec, tol, name in [(B.FP64, TOL64, "fp64"), (B.FP32, TOL32, "fp32"), (B.FP32_STORED, TOL32S, "fp32s"),
                            (B.TF32X3, TOL32, "tf32x3"), (B.TF32, TOL_TF32, "tf32")]:
        check(case_c2.run(nvec, pos, prec, chunk=chunk, ncols=4), ref4, tol, f"c4 nvec={nvec} {name}")


def test_config3_full_size_p8_bloch_chunked(env):
    """configs[3]: 12^3 cells, p=8, k = (0.25,0,0) 2 pi/L, 216 atoms, 1024 vectors in chunks of 256, degree 30;
    sampled columns sit on both sides of a chunk edge; FP64 and FP32-inexact."""
    _, _, B = env
    case = BigCase(env, inp.CONFIGS[3], [0, 255, 256, 1023])
    try:
        pos = [0, 255, 256, 1023]
        check(case.run(1024, pos, B.FP64, chunk=256), case.ref, TOL64, "c3 fp64")
        e32 = check(case.run(1024, pos, B.FP32, chunk=256), case.ref, TOL32, "c3 fp32 product")
        e32s = check(case.run(1024, pos, B.FP32_STORED, chunk=256), case.ref, TOL32S, "c3 fp32 stored")
        assert e32 > 1e-10 and e32s > 1e-10
    finally:
        case.close()


# ------------------------------------------------------------------------------- eigenvalue criterion
def _converge(pb, X0, degree, b, prec, tol, n_check, max_passes, lib_rr=None):
    X, lam, hist = pb.subspace_iteration(X0, degree, b, max_passes, tol=tol, n_check=n_check, prec=prec, lib_rr=lib_rr)
    return lam, hist


def test_eigenvalues_fp32_filter_vs_dense_oracle(env):
    """north_star: with the FP32-inexact product the converged eigenvalues agree with the FP64 oracle within
    1e-8 Ha.  Oracle = LAPACK eigenvalues of the oracle's dense (H, M) on a 3^3-cell p=4 Bloch mesh with all
    terms on; GPU = Algorithm 1 driven by the host harness (RR in FP64, filter in FP32 / FP64)."""
    torch, fo, B = env
    from paper_2605_30128_b200.harness import GpuProblem
    cfg = inp.tiny_config(ncell=3, p=4, L=6.0, kfrac=(0.25, 0, 0), nvec=24, natoms=2, nproj=8, ngauss=3, degree=12)
    mesh = fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    ham = fo.Hamiltonian(mesh, hi.V, hi.Bx, hi.By, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj, hi.P, hi.D)
    H = fo.dense_H(ham)
    ms = np.repeat(mesh.mass, 2) ** -0.5
    exact = np.linalg.eigvalsh(ms[:, None] * H * ms[None, :])
    pb = GpuProblem(cfg, ham=hi)
    try:
        _, b = pb.lanczos_bounds(10)
        X0 = torch.from_numpy(inp.make_vectors(cfg.nnodes, cfg.nvec, seed=0)).cuda()
        n_check = 18
        # every inexact mode, incl. single-pass TF32 (its per-call error is 1e-3: what it is held to is this), and
        # the library's own Rayleigh-Ritz kernels with the paper's mixed-precision rotation
        for prec, lib_rr in ((B.FP32, None), (B.FP64, None), (B.FP32_STORED, None), (B.TF32X3, None), (B.TF32, None),
                             (B.FP64, B.FP64), (B.TF32, B.FP32), (B.FP32_STORED, B.TF32X3)):   # TF32X3 rotation = tcgen05 (rr_tc.cu)
            lam, hist = _converge(pb, X0, cfg.degree, b, prec, 1e-6, n_check, 200, lib_rr=lib_rr)
            assert hist[-1] <= 1e-6, (prec, lib_rr, hist[-5:])
            err = np.max(np.abs(lam[:n_check] - exact[:n_check]))
            print(f"prec {prec} lib_rr {lib_rr}: {len(hist)} passes, max eigenvalue error {err:.2e} Ha")
            assert err < 1e-8, (prec, lib_rr, err)
    finally:
        pb.close()


def test_eigenvalues_config2_mesh_fp32_vs_exact_free_electron_spectrum(env):
    """configs[2]'s mesh at full size (16^3 cells, p=6, 1.77M complex DoF), FP32 product, degree 24: with V = B = 0
    and no projectors the spectrum of M^-1 H is exactly 1/2 (mu_i + mu_j + mu_k), mu from the oracle-side 1-D
    problem; the harness-converged eigenvalues must match it within 1e-8 Ha."""
    torch, fo, B = env
    from paper_2605_30128_b200.harness import GpuProblem
    from test_oracle_pins import _free_1d
    cfg = inp.CONFIGS[2]
    mu, _ = _free_1d(cfg.ncell, cfg.L, cfg.p, 0.0)
    low = np.sort(mu)[:8]
    exact = np.sort(np.repeat(0.5 * (low[:, None, None] + low[None, :, None] + low[None, None, :]).ravel(), 2))
    from paper_2605_30128_b200 import binding as Bb
    m = Bb.chfsi_mesh_create(cfg.ncell, cfg.L, cfg.p, cfg.kfrac, 0)
    xyz = Bb.chfsi_mesh_node_coords(m)
    Bb.chfsi_mesh_destroy(m)
    hi = inp.make_hamiltonian(cfg, xyz, with_local=False, with_nonlocal=False)
    pb = GpuProblem(cfg, ham=hi)
    try:
        _, b = pb.lanczos_bounds(10)
        nvec, n_check = 64, 38                              # 38 = the three lowest shells (2 + 12 + 24)
        X0 = torch.from_numpy(inp.make_vectors(cfg.nnodes, nvec, seed=0)).cuda()
        lam, hist = _converge(pb, X0, cfg.degree, b, B.FP32, 3e-6, n_check, 150)
        assert hist[-1] <= 3e-6, hist[-5:]
        err = np.max(np.abs(lam[:n_check] - exact[:n_check]))
        assert err < 1e-8, err
    finally:
        pb.close()


def test_eigenvalues_config2_full_hamiltonian_vs_oracle_rayleigh_quotients(case_c2, env):
    """configs[2]'s full Hamiltonian at full size, oracle-referenced: Algorithm 1 is driven with the
    FP32-stored filter until the lowest states converge; the converged vectors then go to the HOST and the ORACLE's M^-1 H is
    applied to them once (0.2 s per column).  The eigenvalue the GPU path reports must equal the oracle's Rayleigh quotient of
    that vector within 1e-8 Ha, and the oracle's own residual of the pair must be small -- i.e. the GPU path has converged to
    eigenpairs of the oracle's operator, not of its own."""
    torch, fo, B = env
    from paper_2605_30128_b200.harness import GpuProblem
    cfg = inp.CONFIGS[2]
    pb = GpuProblem(cfg, ham=case_c2.pb.hi)
    try:
        _, b = pb.lanczos_bounds(10)
        nvec, n_check = 64, 32
        X0 = torch.from_numpy(inp.make_vectors(cfg.nnodes, nvec, seed=0)).cuda()
        X, lam, hist = pb.subspace_iteration(X0, cfg.degree, b, 150, tol=3e-6, n_check=n_check, prec=B.FP32_STORED)
        assert hist[-1] <= 3e-6, hist[-3:]
        ks = [0, 1, 2, 5, 17, 31]
        xs = np.stack([X[:, :, k].cpu().numpy() for k in ks], axis=2)                  # (nnodes, 2, 6)
        hx = fo.apply_MinvH(case_c2.pb.oham, xs)
        m = case_c2.pb.omesh.mass[:, None, None]
        for i, k in enumerate(ks):
            x, h = xs[:, :, i:i + 1], hx[:, :, i:i + 1]
            nrm = float(np.sum(m * np.abs(x) ** 2))
            rq = float(np.real(np.sum(m * np.conj(x) * h)) / nrm)
            res = float(np.sqrt(np.sum(m * np.abs(h - rq * x) ** 2) / nrm))
            print(f"c2 state {k}: GPU eigenvalue {lam[k]:.12f}, oracle Rayleigh quotient {rq:.12f}, oracle residual {res:.2e}")
            assert abs(rq - lam[k]) < 1e-8, (k, rq, lam[k])
            assert res < 2e-5, (k, res)
    finally:
        pb.close()


def test_eigenvalues_config2_fp32_vs_fp64_filter(env):
    """configs[2]'s Hamiltonian at full size, 64-vector block: the eigenvalues reached with the inexact filters (FP32
    product, FP32-stored, single-pass TF32) agree within 1e-8 Ha with those reached with the FP64 filter (itself held to
    1e-11 per call above).  An oracle-side subspace iteration at this size (~3.5 s per column and filter call on the
    host) is out of reach of a test; the oracle-referenced eigenvalue checks are the dense pencil above and the exact
    free-electron spectrum on this mesh."""
    torch, fo, B = env
    from paper_2605_30128_b200.harness import GpuProblem
    cfg = inp.CONFIGS[2]
    pb = GpuProblem(cfg)
    try:
        _, b = pb.lanczos_bounds(10)
        nvec, n_check = 64, 32
        X0 = torch.from_numpy(inp.make_vectors(cfg.nnodes, nvec, seed=0)).cuda()
        l64, h64 = _converge(pb, X0, cfg.degree, b, B.FP64, 3e-6, n_check, 150)
        assert h64[-1] <= 3e-6, h64[-3:]
        for prec in (B.FP32, B.FP32_STORED, B.TF32):
            lx, hx = _converge(pb, X0, cfg.degree, b, prec, 3e-6, n_check, 150)
            assert hx[-1] <= 3e-6, (prec, hx[-3:])
            err = np.max(np.abs(lx[:n_check] - l64[:n_check]))
            print(f"c2 prec {prec}: {len(hx)} passes (FP64: {len(h64)}), max eigenvalue difference {err:.2e} Ha")
            assert err < 1e-8, (prec, err)
    finally:
        pb.close()
