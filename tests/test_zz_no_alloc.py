"""chfsi_rr_rotate_static -- the rotation Yout = Y Q on the library's static device scratch, for callers that
cannot allocate -- against the existing path chfsi_rr_rotate (caller workspace), on two calls in a row.  `-m gpu`.

Collected last on purpose (file name): the suite runs with `pytest -x`.  Self-contained: it passes alone in a fresh process
and after the other tests (the static scratch keeps whatever the previous call left; every call rewrites what it reads).

Tolerances are those of tests/test_gpu_rr.py (FP64 rotation 1e-13, mixed FP64-diagonal + FP32-off-diagonal rotation 1e-5,
relative Frobenius); the two entry points launch the same kernels on the same operands, so the outputs are in fact equal."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2605_30128_b200 import binding as B
    B.lib()                                     # fails loudly if the extension is missing
    return torch, B


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _relerr(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def _unitary(rng, n):
    q, _ = np.linalg.qr(_rand(rng, n, n))
    return np.ascontiguousarray(q)


def test_rotate_static_matches_workspace_path_on_two_calls_in_a_row(env):
    torch, B = env
    rng = np.random.default_rng(20260530)
    # first call: a large block that fills most of the scratch; second call: a smaller nvec with ld > nvec, so that the
    # scratch still holds the first call's Q beyond what the second call rewrites
    cases = [(3001, 300, 300), (777, 70, 72)]
    for prec, tol in [(B.FP64, 1e-13), (B.FP32, 1e-5)]:
        for nrows, nvec, ld in cases:
            Y = _rand(rng, nrows, ld)
            Q = _unitary(rng, nvec)
            Yd, Qd = torch.from_numpy(Y).cuda(), torch.from_numpy(Q).cuda()
            work = torch.empty(B.chfsi_rr_rotate_workspace_bytes(nvec), dtype=torch.uint8, device="cuda")
            ref = torch.full((nrows, ld), float("nan"), dtype=torch.complex128, device="cuda")
            B.chfsi_rr_rotate(prec, Yd[:, :nvec], Qd, ref[:, :nvec], work)
            out = torch.full((nrows, ld), float("nan"), dtype=torch.complex128, device="cuda")
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            B.chfsi_rr_rotate_static(prec, Yd[:, :nvec], Qd, out[:, :nvec])
            torch.cuda.synchronize()
            free1 = torch.cuda.mem_get_info()[0]
            got, want = out.cpu().numpy(), ref.cpu().numpy()
            assert np.isfinite(got[:, :nvec]).all()
            assert _relerr(got[:, :nvec], want[:, :nvec]) < tol
            assert np.abs(got[:, :nvec] - want[:, :nvec]).max() <= tol * np.abs(want[:, :nvec]).max()
            # and against the plain definition (FP64 matmul on the host), so that a wrong scratch address cannot pass
            # by corrupting both paths alike
            exact = Y[:, :nvec] @ Q
            assert _relerr(got[:, :nvec], exact) < (1e-13 if prec == B.FP64 else 1e-5)
            if ld > nvec:
                assert np.isnan(got[:, nvec:]).all()                    # padding columns untouched
            if (nrows, nvec, ld) == cases[-1]:
                # second call in a row (every kernel of this precision is loaded by now): no device memory was taken
                assert free1 >= free0


def test_rotate_static_rejects_sizes_beyond_the_static_scratch(env):
    torch, B = env
    assert B.RR_STATIC_MAX_NVEC == 512
    n = B.RR_STATIC_MAX_NVEC + 1
    Y = torch.zeros((8, n), dtype=torch.complex128, device="cuda")
    Q = torch.eye(n, dtype=torch.complex128, device="cuda")
    out = torch.full((8, n), float("nan"), dtype=torch.complex128, device="cuda")
    with pytest.raises(B.ChfsiError) as ei:
        B.chfsi_rr_rotate_static(B.FP64, Y, Q, out)
    assert ei.value.status == B.EINVAL and "CHFSI_RR_STATIC_MAX_NVEC" in str(ei.value)
    torch.cuda.synchronize()
    assert torch.isnan(out.real).all()                                  # nothing was launched, nothing written
    # the largest admitted size runs and is right
    n = B.RR_STATIC_MAX_NVEC
    rng = np.random.default_rng(7)
    Yh, Qh = _rand(rng, 40, n), _unitary(rng, n)
    out = torch.empty((40, n), dtype=torch.complex128, device="cuda")
    B.chfsi_rr_rotate_static(B.FP64, torch.from_numpy(Yh).cuda(), torch.from_numpy(Qh).cuda(), out)
    assert _relerr(out.cpu().numpy(), Yh @ Qh) < 1e-13
