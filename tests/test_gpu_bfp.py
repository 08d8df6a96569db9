"""Parity of the CUDA BFP codec (through the C ABI) against the CPU oracle: byte-exact streams, bit-exact decoded values
(PAPER.md:216-226).  `-m gpu`."""
import numpy as np
import pytest

from paper_2605_30128_b200 import inputs as inp

pytestmark = pytest.mark.gpu
RATES = (16, 12, 10)


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import bfp_oracle as bo
    from paper_2605_30128_b200 import binding as B
    B.lib()
    return torch, bo, B


def _gpu_encode(env, x, nbits):
    torch, bo, B = env
    xd = torch.from_numpy(x).cuda()
    out = torch.full((B.chfsi_bfp_stream_bytes(nbits, x.size) + 8,), 0xAB, dtype=torch.uint8, device="cuda")
    B.chfsi_bfp_encode(nbits, xd, out)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    assert (o[-8:] == 0xAB).all()                       # nothing written past the stream
    return o[:-8]


@pytest.mark.parametrize("nbits", RATES)
def test_encode_decode_byte_exact(env, nbits):
    """Several CTAs and a ragged tail: 4 * (3 * 256 + 17) values."""
    torch, bo, B = env
    x = inp.make_ghost_values(4 * (3 * 256 + 17), seed=1)
    ref = bo.bfp_encode(x, nbits)
    got = _gpu_encode(env, x, nbits)
    assert np.array_equal(got, ref)
    yd = torch.empty(x.size, dtype=torch.float32, device="cuda")
    B.chfsi_bfp_decode(nbits, torch.from_numpy(ref).cuda(), yd)
    y = yd.cpu().numpy()
    assert np.array_equal(y.view(np.uint32), bo.bfp_decode(ref, x.size, nbits).view(np.uint32))


@pytest.mark.parametrize("nbits", RATES)
def test_edge_blocks(env, nbits):
    """Zero blocks, signed zeros, FP32 subnormal maxima, the largest finite value, ties, the clamp, a single block."""
    torch, bo, B = env
    v = nbits - 2
    blocks = [
        [0.0, 0.0, 0.0, 0.0], [-0.0, 0.0, -0.0, 0.0],
        [float.fromhex("0x1p-130"), 0.0, float.fromhex("-0x1p-140"), float.fromhex("0x1p-149")],
        [float.fromhex("0x1.fffffep+127"), float.fromhex("-0x1p+127"), 0.0, float.fromhex("0x1p+100")],
        [1.0 - 2.0 ** -20, -1.0 + 2.0 ** -20, 0.5 * 2.0 ** (1 - v), 1.5 * 2.0 ** (1 - v)],
        [float.fromhex("0x1p-126"), float.fromhex("-0x1.8p-127"), 0.0, 0.0],
        [-1.0, 1.0, -0.75, 0.75],
    ]
    x = np.array(blocks, dtype=np.float32).ravel()
    assert np.array_equal(_gpu_encode(env, x, nbits), bo.bfp_encode(x, nbits))
    one = np.array(blocks[4], dtype=np.float32)
    assert np.array_equal(_gpu_encode(env, one, nbits), bo.bfp_encode(one, nbits))
    # n = 0 is a no-op; n % 4 != 0 and a bad rate are refused
    empty = torch.empty(0, dtype=torch.float32, device="cuda")
    B.chfsi_bfp_encode(nbits, empty, torch.empty(0, dtype=torch.uint8, device="cuda"))
    with pytest.raises(B.ChfsiError):
        B.chfsi_bfp_stream_bytes(nbits, 6)
    with pytest.raises(B.ChfsiError):
        B.chfsi_bfp_stream_bytes(14, 8)


@pytest.mark.parametrize("nbits", RATES)
@pytest.mark.parametrize("cdtype", ["complex128", "complex64"])
def test_fused_ghost_exchange(env, nbits, cdtype):
    """gather+encode and decode+scatter-add on a face slab of a multivector: the x = 0 face rows of a
    6 x 5 x 4-node block with 12 vectors, ld = 14."""
    torch, bo, B = env
    rng = np.random.default_rng(4)
    n1 = (6, 5, 4)
    nvec, ld = 12, 14
    nrows = 2 * n1[0] * n1[1] * n1[2]
    X = (rng.standard_normal((nrows, ld)) + 1j * rng.standard_normal((nrows, ld))) * np.exp2(rng.uniform(-12, 2, (nrows, 1)))
    X = X.astype(cdtype)
    nodes = [(iz * n1[1] + iy) * n1[0] for iz in range(n1[2]) for iy in range(n1[1])]
    rows = np.array([2 * I + s for I in nodes for s in (0, 1)], dtype=np.int64)
    ref = bo.ghost_gather_encode(X[:, :nvec], rows, nbits)
    Xd, rd = torch.from_numpy(X).cuda(), torch.from_numpy(rows).cuda()
    out = torch.zeros(ref.size, dtype=torch.uint8, device="cuda")
    B.chfsi_bfp_gather_encode(nbits, Xd[:, :nvec], rd, out)
    assert np.array_equal(out.cpu().numpy(), ref)
    # receive side: rows listed once -> one add per element, bit-exact in Y's precision
    Y = (rng.standard_normal((nrows, ld)) + 1j * rng.standard_normal((nrows, ld))).astype(cdtype)
    Yd = torch.from_numpy(Y.copy()).cuda()
    B.chfsi_bfp_decode_scatter_add(nbits, out, rd, Yd[:, :nvec])
    Yref = Y.copy()
    bo.ghost_decode_scatter_add(ref, Yref[:, :nvec], rows, nbits)
    got = Yd.cpu().numpy()
    assert np.array_equal(got, Yref)
    # a row listed twice accumulates twice (atomic adds; order-independent here because both addends are equal)
    rows2 = np.concatenate([rows[:4], rows[:4]])
    s2 = bo.ghost_gather_encode(X[:, :nvec], rows2, nbits)
    Yd2 = torch.zeros((nrows, ld), dtype=getattr(torch, cdtype), device="cuda")
    B.chfsi_bfp_decode_scatter_add(nbits, torch.from_numpy(s2).cuda(), torch.from_numpy(rows2).cuda(), Yd2[:, :nvec])
    Yr2 = np.zeros((nrows, ld), dtype=cdtype)
    bo.ghost_decode_scatter_add(s2, Yr2[:, :nvec], rows2, nbits)
    assert np.array_equal(Yd2.cpu().numpy(), Yr2)


@pytest.mark.parametrize("nbits", RATES)
def test_full_size_slab_properties_and_samples(env, nbits):
    """A face slab of configs[3] (96^2 nodes x 2 spins x 256 vectors x (re, im) = 9.4M values) in the launch configuration
    bench.py times: sampled blocks against the oracle one by one, and properties that hold at any size (exponent byte,
    half-quantum error bound, zero blocks)."""
    torch, bo, B = env
    n = 96 * 96 * 2 * 256 * 2
    x = inp.make_ghost_values(n, seed=3)
    xd = torch.from_numpy(x).cuda()
    nb = nbits // 2
    sd = torch.empty(B.chfsi_bfp_stream_bytes(nbits, n), dtype=torch.uint8, device="cuda")
    B.chfsi_bfp_encode(nbits, xd, sd)
    yd = torch.empty_like(xd)
    B.chfsi_bfp_decode(nbits, sd, yd)
    s = sd.cpu().numpy().reshape(-1, nb)
    y = yd.cpu().numpy()
    rng = np.random.default_rng(9)
    for b in np.concatenate([[0, n // 4 - 1], rng.integers(0, n // 4, 400)]):
        xb = x[4 * b:4 * b + 4]
        assert np.array_equal(s[b], bo.bfp_encode(xb, nbits)), b
        assert np.array_equal(y[4 * b:4 * b + 4].view(np.uint32), bo.bfp_decode(s[b], 4, nbits).view(np.uint32))
    xb = x.reshape(-1, 4).astype(np.float64)
    amax = np.abs(xb).max(axis=1)
    e = s[:, 0].astype(np.int64)
    assert ((e == 0) == (amax == 0)).all()
    nz = amax > 0
    emax = e[nz] - 127
    assert (np.exp2(emax - 1.0) <= amax[nz]).all() and (amax[nz] < np.exp2(emax.astype(np.float64))).all()
    err = np.abs(xb[nz] - y.reshape(-1, 4)[nz])
    quantum = np.exp2(emax - (nbits - 2) + 1.0)[:, None]
    clamped = xb[nz] * np.exp2((nbits - 2) - 1.0 - emax)[:, None] > 2 ** (nbits - 3) - 1
    assert (err[~clamped] <= 0.5 * quantum.repeat(4, 1)[~clamped]).all()
    assert (err[clamped] <= quantum.repeat(4, 1)[clamped]).all()
    assert not y.reshape(-1, 4)[~nz].any()
