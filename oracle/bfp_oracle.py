"""CPU oracle for the block floating-point (BFP) codec of the paper's compressed ghost exchange
(arxiv/paper_2605_30128, Sec. III-B 3, Fig. 3).

TEST INFRASTRUCTURE ONLY (same rules as fe_oracle.py): only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
cpu_baseline / `--impl reference` legs may import it; it shares no code with the CUDA path and imports nothing from it.

The codec is an *encoding*: the oracle follows the paper's algorithm step by step, in the paper's notation, one
four-value block at a time (a plain Python loop over blocks; integers are Python ints, so nothing can overflow).

  PAPER.md:218  "maps four FP32 values to N_bits = 4 x n_bits bits ... whose lower 8 bits store a shared biased
                exponent ... the remaining N_bits - 8 bits are divided equally among four signed coefficients, each of
                width v_bits = (N_bits - 8)/4 = n_bits - 2"; n_bits in {16, 12, 10} -> v_bits in {14, 10, 8}.
  PAPER.md:218  "The shared exponent e_max satisfies 2^(e_max-1) <= max_i |x_i| < 2^e_max.  A block whose four values
                are all zero is flagged by a zero exponent field.  Otherwise, the biased exponent e = e_max + 127 is
                stored, and each value is quantized as q_i = round(x_i 2^(v_bits-1-e_max)),
                q_i in [-2^(v_bits-1), 2^(v_bits-1)-1].  Round-to-nearest ...  Only the upper bound requires clamping
                ...  Each q_i is stored using its low v_bits bits in two's complement ...  Decoding recovers
                e_max = e - 127 and reconstructs x~_i = q_i 2^(e_max - v_bits + 1)."
  PAPER.md:222  "each thread writes its encoded block to a private region of the compressed byte stream ... At
                n_bits = 16, a block is stored as a single uint64_t ... At n_bits = 12 and 10, a block is stored using
                three uint16_t or five uint8_t stores".

Readings where the paper is silent (B1-B5):
  B1  ties of "round" go to even (IEEE round-to-nearest-even, the default rounding of every FP unit the paper runs on).
  B2  bit order inside the N_bits-bit word: exponent in bits 0..7, then q_0 in bits 8..8+v-1, q_1 above it, q_2, q_3;
      the word is stored little-endian (uint64 / three uint16 / five uint8 in increasing significance), block b at byte
      offset b * N_bits / 8 ("stored contiguously without padding").
  B3  FP32 subnormal maxima: e_max is clamped below at -126 (stored e = 1), so that the zero flag e = 0 stays
      unambiguous; such blocks are quantized against 2^-126 (values below 2^(-126-v) become 0).
  B4  inputs are finite FP32 numbers (the exchanged residuals); +-Inf / NaN are outside the codec's domain.
  B5  a trailing partial block (n not a multiple of 4) does not exist: "Choosing N_b as a multiple of four ensures that
      no four-value block straddles a message boundary"; n % 4 != 0 is an error.

Functions: bfp_encode(x, nbits) -> uint8 stream; bfp_decode(stream, n, nbits) -> float32;
ghost_gather_encode / ghost_decode_scatter_add: the fused forms of PAPER.md:226 (gather the rows of a ghost list from a
multivector and encode in the same pass; decode and scatter-add into the owned rows).

Pins (tests/test_bfp_pins.py, `-m "not gpu"`): hand-worked blocks (tests/golden/bfp_worked_blocks.txt), the error bound
|x - x~| <= 2^(e_max - v_bits) for unclamped values, exactness on values that are multiples of the quantum, stream size
n n_bits / 8, re-encoding a decoded stream reproduces it bit for bit, and an independent exact-rational (fractions)
implementation of the quantiser on random blocks.  No function here is unpinned.
"""
from __future__ import annotations

import math

import numpy as np

RATES = (16, 12, 10)


def vbits(nbits: int) -> int:
    if nbits not in RATES:
        raise ValueError("n_bits must be 16, 12 or 10 (PAPER.md:218)")
    return nbits - 2


def block_bytes(nbits: int) -> int:
    return 4 * nbits // 8


def shared_exponent(x4) -> int:
    """e_max with 2^(e_max-1) <= max|x_i| < 2^e_max; None for an all-zero block; clamped at -126 (B3)."""
    amax = max(abs(float(v)) for v in x4)
    if amax == 0.0:
        return None
    if not math.isfinite(amax):
        raise ValueError("BFP codec: non-finite input (reading B4)")
    mant, ex = math.frexp(amax)          # amax = mant * 2^ex, 0.5 <= mant < 1  =>  2^(ex-1) <= amax < 2^ex
    return max(ex, -126)


def round_half_even(t: float) -> int:
    """round-to-nearest, ties to even (reading B1).  t is an exactly representable double here: an FP32 value times a
    power of two."""
    f = math.floor(t)
    d = t - f
    if d > 0.5 or (d == 0.5 and (f % 2 == 1)):
        return int(f) + 1
    return int(f)


def encode_block(x4, nbits: int) -> int:
    """The N_bits-bit word of one block (bit order B2)."""
    v = vbits(nbits)
    emax = shared_exponent(x4)
    if emax is None:
        return 0                                            # zero exponent field flags the all-zero block
    word = emax + 127                                       # biased exponent, 1..255
    hi = (1 << (v - 1)) - 1
    for i, xi in enumerate(x4):
        q = round_half_even(math.ldexp(float(xi), v - 1 - emax))
        if q > hi:                                          # "only the upper bound requires clamping"
            q = hi
        assert q >= -(1 << (v - 1))
        word |= (q & ((1 << v) - 1)) << (8 + i * v)          # low v bits, two's complement
    return word


def decode_block(word: int, nbits: int):
    v = vbits(nbits)
    e = word & 0xFF
    if e == 0:
        return [0.0, 0.0, 0.0, 0.0]
    emax = e - 127
    out = []
    for i in range(4):
        q = (word >> (8 + i * v)) & ((1 << v) - 1)
        if q >= (1 << (v - 1)):                             # restore the dropped copies of the sign bit
            q -= 1 << v
        out.append(math.ldexp(float(q), emax - v + 1))
    return out


def bfp_encode(x, nbits: int) -> np.ndarray:
    """float32[n] (n % 4 == 0, B5) -> uint8[n * nbits / 8], block b at byte offset b * N_bits/8, little-endian (B2)."""
    x = np.asarray(x, dtype=np.float32).ravel()
    if x.size % 4 != 0:
        raise ValueError("BFP codec: the number of values must be a multiple of 4 (PAPER.md:224)")
    nb = block_bytes(nbits)
    out = np.zeros(x.size // 4 * nb, dtype=np.uint8)
    for b in range(x.size // 4):
        w = encode_block(x[4 * b:4 * b + 4], nbits)
        out[b * nb:(b + 1) * nb] = np.frombuffer(w.to_bytes(nb, "little"), dtype=np.uint8)
    return out


def bfp_decode(stream, n: int, nbits: int) -> np.ndarray:
    stream = np.asarray(stream, dtype=np.uint8).ravel()
    nb = block_bytes(nbits)
    if n % 4 != 0 or stream.size != n // 4 * nb:
        raise ValueError("BFP codec: stream size does not match n * n_bits / 8")
    out = np.zeros(n, dtype=np.float32)
    for b in range(n // 4):
        w = int.from_bytes(stream[b * nb:(b + 1) * nb].tobytes(), "little")
        out[4 * b:4 * b + 4] = decode_block(w, nbits)       # exact: |q| < 2^13, a power-of-two scale
    return out


# ------------------------------------------------------------------ fused forms
def ghost_gather_encode(X, rows, nbits: int) -> np.ndarray:
    """Ghost update, send side: "gathers the entries for each neighbour and encodes them in the same pass".
    X: complex multivector [nrows, nvec] (row = 2 I + alpha), rows: the (node, spin) rows of the message in order.
    The message is the FP32 values (re, im interleaved, vectors fastest) of those rows: 2 nvec values per row
    ("f x n_Gamma x N_b values ... f = 2 for complex"); nvec even so that blocks are complete."""
    X = np.asarray(X)
    msg = np.empty((len(rows), X.shape[1], 2), dtype=np.float32)
    for r, row in enumerate(rows):
        msg[r, :, 0] = X[row].real.astype(np.float32)       # FP64 -> FP32 round-to-nearest-even (S6 conversion)
        msg[r, :, 1] = X[row].imag.astype(np.float32)
    return bfp_encode(msg.ravel(), nbits)


def ghost_decode_scatter_add(stream, Y, rows, nbits: int) -> None:
    """Ghost accumulation, receive side: "decodes the data and atomically scatter-adds it to the corresponding owned
    entries".  Y (complex64 or complex128 [nrows, nvec]) is updated in place; a row may appear several times in `rows`."""
    nvec = Y.shape[1]
    vals = bfp_decode(stream, len(rows) * nvec * 2, nbits).reshape(len(rows), nvec, 2)
    for r, row in enumerate(rows):
        Y[row] += (vals[r, :, 0].astype(np.float64) + 1j * vals[r, :, 1].astype(np.float64)).astype(Y.dtype)
