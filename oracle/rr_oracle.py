"""CPU oracle for the Rayleigh-Ritz pieces around the filter (arxiv/paper_2605_30128, Sec. III-B 4, PAPER.md:228-234;
Algorithm 1 lines 6-8).

TEST INFRASTRUCTURE ONLY (same rules as fe_oracle.py): only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
cpu_baseline / `--impl reference` legs may import it; it shares no code with the CUDA path and imports nothing from it.

Both operations have a plain definition, so the oracle is that definition written out with numpy:

  rr_project(A, B, w)      RR-Proj, PAPER.md:228 (i) "projecting the FE-discretized Hamiltonian (H) and overlap (M) matrices
                           onto the Chebyshev filtered subspace": S = A^H diag(w) B, an N x N complex matrix.  With A = Y,
                           w = the node masses (row 2I + alpha carries m_I), B = Y it is Y^H M Y; with B = M^-1 H Y it is
                           Y^H H Y (M is diagonal here, D2).  FP64.
  rr_rotate(Y, Q, mixed)   RR-SR: "the subspace rotation Y_q Q is decomposed as Y_q Q = Y_q Q_diag +
                           Y_q Q_non-diag ... Y_q Q_non-diag is evaluated in FP32 arithmetic, while Y_q Q_diag is computed
                           in FP64 arithmetic."  mixed=False: the plain FP64 product.  mixed=True: step by step as stated --
                           Q_diag = diag(diag(Q)) applied in complex128; Y and Q_non-diag rounded to complex64, multiplied
                           and accumulated in complex64, widened, added.

Reading R1: "FP32 arithmetic" for the off-diagonal product means FP32 operands and FP32 accumulation
(the paper names no split or compensated scheme); the result is stored in FP64.  The order of the FP32 accumulation is
not fixed by the paper: comparisons against the CUDA path are tolerance based (FP32 level), never bitwise.

Pins (tests/test_rr_pins.py): the projection against its triple loop on tiny inputs, Hermitian symmetry of Y^H M Y,
Rayleigh-Ritz exactness on an invariant subspace (the projected pencil reproduces the dense eigenvalues), rotation by the
identity / by a phased permutation is exact in both modes, a unitary rotation of an M-orthonormal block stays
M-orthonormal, and the mixed-precision error obeys the FP32 bound while the diagonal part is exact to FP64.
"""
from __future__ import annotations

import numpy as np


def rr_project(A: np.ndarray, B: np.ndarray, w=None) -> np.ndarray:
    """S = A^H diag(w) B.  A, B: complex128 [rows, N]; w: float64 [rows] or None (= ones)."""
    A = np.asarray(A, dtype=np.complex128)
    B = np.asarray(B, dtype=np.complex128)
    if w is not None:
        B = np.asarray(w, dtype=np.float64)[:, None] * B
    return A.conj().T @ B


def rr_rotate(Y: np.ndarray, Q: np.ndarray, mixed: bool) -> np.ndarray:
    """Y Q.  Y: complex128 [rows, N], Q: complex128 [N, N]."""
    Y = np.asarray(Y, dtype=np.complex128)
    Q = np.asarray(Q, dtype=np.complex128)
    if not mixed:
        return Y @ Q
    d = np.diag(Q).copy()
    Qoff = Q - np.diag(d)
    out = Y * d[None, :]                                              # Y Q_diag in FP64
    off = Y.astype(np.complex64) @ Qoff.astype(np.complex64)           # Y Q_non-diag in FP32
    return out + off.astype(np.complex128)
