"""Pins of the BFP codec oracle (oracle/bfp_oracle.py) against what the paper and the mathematics fix
(PAPER.md:216-226).  CPU only."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import bfp_oracle as bo

GOLD = os.path.join(os.path.dirname(__file__), "golden", "bfp_worked_blocks.txt")


def _f(s):
    return float.fromhex(s) if "0x" in s else float(s)


def _worked():
    out = []
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        nb, xs, hx, dec = [t.strip() for t in line.split("|")]
        out.append((int(nb), [_f(t) for t in xs.split()], bytes.fromhex(hx), [_f(t) for t in dec.split()]))
    return out


@pytest.mark.parametrize("case", _worked(), ids=lambda c: f"n{c[0]}-{c[2].hex()}")
def test_worked_blocks(case):
    """Hand-worked blocks (tests/golden/bfp_worked_blocks.txt): quantiser, clamp, ties, bit order, zero flag, extremes."""
    nbits, x, stream, dec = case
    got = bo.bfp_encode(np.array(x, dtype=np.float32), nbits)
    assert got.tobytes() == stream
    back = bo.bfp_decode(np.frombuffer(stream, dtype=np.uint8), 4, nbits)
    assert back.tolist() == [np.float32(d) for d in dec]


def _random_blocks(seed, nblocks, spread=6.0):
    rng = np.random.default_rng(seed)
    mag = np.exp2(rng.uniform(-spread, spread, size=(nblocks, 1)) + rng.uniform(-3, 0, size=(nblocks, 4)))
    x = (mag * rng.choice([-1.0, 1.0], size=(nblocks, 4)) * rng.uniform(0.5, 1.0, size=(nblocks, 4))).astype(np.float32)
    x[rng.random((nblocks, 4)) < 0.05] = 0.0
    return x.ravel()


@pytest.mark.parametrize("nbits", bo.RATES)
def test_stream_size_and_error_bound(nbits):
    """Message size n n_bits / 8 bytes and |x - x~| <= half a quantum 2^(e_max - v) for values that are
    not clamped; clamped values (q would be 2^(v-1)) are off by at most one quantum."""
    x = _random_blocks(11, 500)
    s = bo.bfp_encode(x, nbits)
    assert s.size == x.size * nbits // 8
    y = bo.bfp_decode(s, x.size, nbits)
    v = nbits - 2
    for b in range(x.size // 4):
        xb = x[4 * b:4 * b + 4].astype(np.float64)
        amax = np.abs(xb).max()
        if amax == 0:
            assert not y[4 * b:4 * b + 4].any()
            continue
        emax = int(np.floor(np.log2(amax))) + 1
        assert 2.0 ** (emax - 1) <= amax < 2.0 ** emax
        assert s[b * (nbits // 2)] == emax + 127                 # the low byte is the biased exponent
        err = np.abs(xb - y[4 * b:4 * b + 4])
        quantum = 2.0 ** (emax - v + 1)
        clamped = xb * 2.0 ** (v - 1 - emax) > 2 ** (v - 1) - 1
        assert (err[~clamped] <= 0.5 * quantum).all()
        assert (err[clamped] <= quantum).all()


@pytest.mark.parametrize("nbits", bo.RATES)
def test_exact_on_multiples_of_the_quantum_and_idempotent(nbits):
    """Values q 2^(e_max - v + 1) with |q| < 2^(v-1) are reproduced exactly ("decoding exactly reconstructs the quantized
    representation") and re-encode to the same bytes; decoded values are a fixed point of the codec."""
    v = nbits - 2
    rng = np.random.default_rng(5)
    blocks = []
    for _ in range(300):
        emax = int(rng.integers(-20, 20))
        q = rng.integers(-(2 ** (v - 1)) + 1, 2 ** (v - 1), size=4)
        q[0] = (2 ** (v - 2)) * (1 if rng.random() < 0.5 else -1) + int(rng.integers(0, 2 ** (v - 2)))  # fixes e_max
        if q[0] < 0:
            q[0] = -abs(q[0])
        blocks.append(q * 2.0 ** (emax - v + 1))
    x = np.array(blocks, dtype=np.float32).ravel()
    s = bo.bfp_encode(x, nbits)
    y = bo.bfp_decode(s, x.size, nbits)
    assert np.array_equal(x, y)
    assert np.array_equal(bo.bfp_encode(y, nbits), s)
    # arbitrary data: re-encoding the decoded block gives the same bytes, except where a negative maximum rounded to
    # -2^e_max (q = -2^(v-1), legal: "bounds q_i from below by construction"), whose own block exponent is one higher
    x2 = _random_blocks(7, 300)
    s2 = bo.bfp_encode(x2, nbits)
    y2 = bo.bfp_decode(s2, x2.size, nbits)
    s3 = bo.bfp_encode(y2, nbits)
    nb = nbits // 2
    for b in range(x2.size // 4):
        yb = np.abs(y2[4 * b:4 * b + 4].astype(np.float64))
        e = int(s2[b * nb])
        if e and yb.max() < 2.0 ** (e - 127):
            assert np.array_equal(s2[b * nb:(b + 1) * nb], s3[b * nb:(b + 1) * nb])


@pytest.mark.parametrize("nbits", bo.RATES)
def test_against_exact_rational_quantiser(nbits):
    """An independent quantiser in exact rational arithmetic (fractions.Fraction; e_max by doubling, rounding by integer
    division) on random blocks: guards the float path of the oracle (frexp, ldexp, floor) against off-by-one mistakes."""
    v = nbits - 2
    x = _random_blocks(3, 400, spread=30.0)
    s = bo.bfp_encode(x, nbits)
    nb = nbits // 2
    for b in range(x.size // 4):
        xs = [Fraction(float(t)) for t in x[4 * b:4 * b + 4]]
        amax = max(abs(t) for t in xs)
        word = int.from_bytes(s[b * nb:(b + 1) * nb].tobytes(), "little")
        if amax == 0:
            assert word == 0
            continue
        emax = 0
        while Fraction(2) ** emax <= amax:
            emax += 1
        while Fraction(2) ** (emax - 1) > amax:
            emax -= 1
        assert word & 0xFF == emax + 127
        for i, t in enumerate(xs):
            y = t * Fraction(2) ** (v - 1 - emax)
            fl = y.numerator // y.denominator
            rem = y - fl
            q = fl + (1 if (rem > Fraction(1, 2) or (rem == Fraction(1, 2) and fl % 2 == 1)) else 0)
            q = min(q, 2 ** (v - 1) - 1)
            assert -(2 ** (v - 1)) <= q
            field = (word >> (8 + i * v)) & (2 ** v - 1)
            assert field == q % (2 ** v)


def test_rejects_partial_block_and_bad_rate():
    with pytest.raises(ValueError):
        bo.bfp_encode(np.zeros(6, dtype=np.float32), 16)
    with pytest.raises(ValueError):
        bo.bfp_encode(np.zeros(8, dtype=np.float32), 14)
    with pytest.raises(ValueError):
        bo.bfp_encode(np.array([np.inf, 0, 0, 0], dtype=np.float32), 16)


@pytest.mark.parametrize("nbits", bo.RATES)
def test_fused_ghost_forms_equal_the_unfused_ones(nbits):
    """gather + encode in one pass == encode of the gathered FP32 message; decode + scatter-add == adding
    the decoded message to the listed rows (rows repeated in the list accumulate)."""
    rng = np.random.default_rng(2)
    nrows, nvec = 40, 6
    X = rng.standard_normal((nrows, nvec)) + 1j * rng.standard_normal((nrows, nvec))
    rows = [3, 17, 4, 39, 0, 17]
    msg = np.stack([X[rows].real, X[rows].imag], axis=-1).astype(np.float32).ravel()
    s = bo.ghost_gather_encode(X, rows, nbits)
    assert np.array_equal(s, bo.bfp_encode(msg, nbits))
    Y = np.zeros((nrows, nvec), dtype=np.complex128)
    bo.ghost_decode_scatter_add(s, Y, rows, nbits)
    d = bo.bfp_decode(s, msg.size, nbits).reshape(len(rows), nvec, 2).astype(np.float64)
    ref = np.zeros_like(Y)
    for r, row in enumerate(rows):
        ref[row] += d[r, :, 0] + 1j * d[r, :, 1]
    assert np.array_equal(Y, ref)
    # decoded values are within the quantisation error of the originals on rows listed once
    assert np.abs(Y[3] - X[3]).max() < 2.0 ** (2 - (nbits - 2)) * np.abs(msg).max()
