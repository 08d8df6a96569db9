"""Host-side harness around the C-ABI library: problem setup, Lanczos bounds, Rayleigh-Ritz and the
subspace-iteration loop of Algorithm 1.  NOT part of the library (BASELINE.json
north_star: "a host-side test harness that does Rayleigh-Ritz and is not part of the library").

Every Hamiltonian product goes through `chfsi_apply_H` / `chfsi_cheb_filter`; torch does the dense
subspace algebra (inner products, Cholesky, eigh) in FP64 on the GPU.
"""
from __future__ import annotations

import math

import numpy as np

from . import binding as B
from . import inputs as inp


class GpuProblem:
    """A mesh + Hamiltonian living in the library, with a cached workspace."""

    def __init__(self, cfg: inp.Config, seed: int = 0, device: int = 0, ham: inp.HamInputs | None = None):
        import torch
        self.torch = torch
        self.cfg = cfg
        self.device = device
        self.mesh = B.chfsi_mesh_create(cfg.ncell, cfg.L, cfg.p, cfg.kfrac, device)
        self.nnodes = B.chfsi_mesh_num_nodes(self.mesh)
        self.xyz = B.chfsi_mesh_node_coords(self.mesh)
        self.mass_h = B.chfsi_mesh_mass(self.mesh)
        self.mass = torch.from_numpy(self.mass_h).to(f"cuda:{device}")
        self.ham = ham if ham is not None else inp.make_hamiltonian(cfg, self.xyz, seed=seed)
        h = self.ham
        if len(h.supp_off) > 1:
            B.chfsi_ham_set(self.mesh, h.V, h.Bx, h.By, h.Bz, h.supp_off, h.supp_node, h.nproj, h.P, h.D)
        else:
            B.chfsi_ham_set(self.mesh, h.V, h.Bx, h.By, h.Bz)
        self._work = {}

    def close(self):
        if self.mesh is not None:
            B.chfsi_mesh_destroy(self.mesh)
            self.mesh = None
        self._work = {}

    def work(self, prec, recur, chunk):
        key = (prec, recur, chunk)
        if key not in self._work:
            n = B.chfsi_workspace_bytes(self.mesh, prec, recur, chunk)
            self._work[key] = self.torch.empty(n, dtype=self.torch.uint8, device=f"cuda:{self.device}")
        return self._work[key]

    # -- library calls
    def apply_MinvH(self, X, prec=B.FP64):
        Y = self.torch.empty_like(X)
        B.chfsi_apply_H(self.mesh, prec, X, Y, self.work(prec, B.RECUR_STANDARD, X.shape[-1]))
        return Y

    def cheb_filter(self, X, lam, degree, a, b, a0, prec=B.FP64, recur=B.RECUR_RESIDUAL, chunk=0, Y=None):
        Y = self.torch.empty_like(X) if Y is None else Y
        nb = chunk if chunk else X.shape[-1]
        B.chfsi_cheb_filter(self.mesh, prec, recur, degree, a, b, a0, X, lam, Y, self.work(prec, recur, nb),
                            chunk=chunk)
        return Y

    # -- dense subspace algebra (torch, FP64)
    def m_inner(self, A, Bm):
        M2 = 2 * self.nnodes
        return A.reshape(M2, -1).conj().T @ (self.mass[:, None, None] * Bm).reshape(M2, -1)

    def rayleigh_quotients(self, X, block=32):
        """x^H H x / x^H M x per column, in column blocks so that large multivectors need no full-size temporaries."""
        out = []
        for j0 in range(0, X.shape[-1], block):
            Xb = X[:, :, j0:j0 + block].contiguous()
            HX = self.apply_MinvH(Xb)
            mX = self.mass[:, None, None] * Xb
            num = (mX.conj() * HX).sum(dim=(0, 1)).real
            den = (mX.conj() * Xb).sum(dim=(0, 1)).real
            out.append((num / den).cpu().numpy())
            del HX, mX
        return np.concatenate(out)

    def lanczos_bounds(self, steps=10, seed=0):
        """(a0, b): lowest Ritz value and the safeguarded upper bound theta_max + ||f||_M."""
        t = self.torch
        v = t.from_numpy(inp.lanczos_start(self.nnodes, seed)).to(self.mass.device)
        v = v / math.sqrt(self.m_inner(v, v)[0, 0].real.item())
        alphas, betas = [], []
        vprev = t.zeros_like(v)
        beta = 0.0
        for j in range(steps):
            f = self.apply_MinvH(v) - beta * vprev
            alpha = self.m_inner(v, f)[0, 0].real.item()
            f = f - alpha * v
            alphas.append(alpha)
            beta = math.sqrt(self.m_inner(f, f)[0, 0].real.item())
            if j < steps - 1:
                betas.append(beta)
                vprev, v = v, f / beta
        T = np.diag(alphas) + np.diag(betas, 1) + np.diag(betas, -1)
        th = np.linalg.eigvalsh(T)
        return float(th[0]), float(th[-1] + beta)

    def rayleigh_ritz(self, Y, lib_rr=None):
        """Alg. 1 lines 6-9: Y^H H Y Q = Y^H M Y Q Lambda; returns (Y Q, Lambda).  lib_rr = None: projection and rotation
        with torch dense algebra; lib_rr = B.FP64 / B.FP32 / B.TF32X3: with the library's chfsi_rr_project and chfsi_rr_rotate (FP32 =
        the paper's FP64-diagonal + FP32-off-diagonal rotation; TF32X3 = the same on tcgen05, 3xTF32 off-diagonal).  The small dense eigenproblem stays in torch."""
        t = self.torch
        M2 = 2 * self.nnodes
        nv = Y.shape[-1]
        if lib_rr is not None:
            Yc = Y.contiguous()
            HYm = self.apply_MinvH(Yc)
            Hs = t.empty((nv, nv), dtype=t.complex128, device=Y.device)
            Ss = t.empty_like(Hs)
            B.chfsi_rr_project(self.mesh, Yc, HYm, Hs)
            B.chfsi_rr_project(self.mesh, Yc, Yc, Ss)
            del HYm
        else:
            HY = self.mass[:, None, None] * self.apply_MinvH(Y)
            Hs = Y.reshape(M2, nv).conj().T @ HY.reshape(M2, nv)
            Ss = self.m_inner(Y, Y)
        Hs = 0.5 * (Hs + Hs.conj().T)
        Ss = 0.5 * (Ss + Ss.conj().T)
        Lc = t.linalg.cholesky(Ss)
        A = t.linalg.solve_triangular(Lc, Hs, upper=False)
        A = t.linalg.solve_triangular(Lc, A.conj().T, upper=False).conj().T
        lam, U = t.linalg.eigh(0.5 * (A + A.conj().T))
        Q = t.linalg.solve_triangular(Lc.conj().T, U, upper=True)
        if lib_rr is not None:
            Xn = t.empty_like(Yc)
            wk = t.empty(B.chfsi_rr_rotate_workspace_bytes(nv), dtype=t.uint8, device=Y.device)
            B.chfsi_rr_rotate(lib_rr, Yc, Q.contiguous(), Xn, wk)
            return Xn, lam.cpu().numpy()
        Xn = (Y.reshape(M2, nv) @ Q).reshape(self.nnodes, 2, nv).contiguous()
        return Xn, lam.cpu().numpy()

    def residual_norms(self, X, lam):
        t = self.torch
        lam_d = t.from_numpy(np.asarray(lam)).to(X.device)
        R = self.mass[:, None, None] * (self.apply_MinvH(X) - X * lam_d[None, None, :])
        return t.sqrt((R.abs() ** 2).sum(dim=(0, 1))).cpu().numpy()

    def subspace_iteration(self, X0, degree, b, passes, tol=1e-6, n_check=None, prec=B.FP64,
                           recur=B.RECUR_RESIDUAL, chunk=0, lib_rr=None):
        """Algorithm 1 with the GPU filter in `prec`; RR and residuals in FP64 (lib_rr: see rayleigh_ritz).  Returns (X, lam, hist)."""
        X, lam = self.rayleigh_ritz(X0, lib_rr)
        nv = X.shape[-1]
        n_check = n_check or (3 * nv) // 4
        hist = []
        for _ in range(passes):
            res = self.residual_norms(X, lam)
            xn = np.sqrt(np.real(np.diag(self.m_inner(X, X).cpu().numpy())))
            hist.append(float(np.max(res[:n_check] / xn[:n_check])))
            if hist[-1] <= tol:
                break
            Y = self.cheb_filter(X, lam, degree, float(lam[-1]), b, float(lam[0]), prec, recur, chunk)
            X, lam = self.rayleigh_ritz(Y, lib_rr)
        return X, lam, hist
