"""Pins of the oracle's sample unpacking (Table 3 recording modes; reading R23).

The paper gives no packing, so there is no printed value; the pins are hand-decoded bytes and numpy's own
integer views / ``unpackbits`` (library routines that share nothing with the oracle's C loop).
"""
import numpy as np
import pytest

import oracle
from paper_1906_10598_b200 import workloads as W


def test_hand_decoded_bytes():
    xq = np.array([[0b11100100, 0x80]], dtype=np.uint8)
    # 2-bit fields of 0b11100100 from the least significant bit: 0, 1, 2, 3
    assert np.array_equal(oracle.unpack_samples(xq, 4, 2, False, 1.0, -1.5), [[-1.5, -0.5, 0.5, 1.5]])
    # the same fields as two's complement: 0, 1, -2, -1
    assert np.array_equal(oracle.unpack_samples(xq, 4, 2, True, 1.0, 0.0), [[0.0, 1.0, -2.0, -1.0]])
    # 1-bit: bits of 0xE4 from the LSB: 0 0 1 0 0 1 1 1
    assert np.array_equal(oracle.unpack_samples(xq, 8, 1, False, 2.0, -0.5), [[-1, -1, 1, -1, -1, 1, 1, 1]])
    # 4-bit: low nibble first: 4, 14
    assert np.array_equal(oracle.unpack_samples(xq, 2, 4, False, 1.0, 0.0), [[4.0, 14.0]])
    assert np.array_equal(oracle.unpack_samples(xq, 2, 4, True, 1.0, 0.0), [[4.0, -2.0]])
    # 8-bit: 0xE4 = 228 = -28, 0x80 = 128 = -128
    assert np.array_equal(oracle.unpack_samples(xq, 2, 8, False, 1.0, 0.0), [[228.0, 128.0]])
    assert np.array_equal(oracle.unpack_samples(xq, 2, 8, True, 0.5, 0.0), [[-14.0, -64.0]])
    # 16-bit little-endian: 0x80E4 = 32996 = -32540
    assert np.array_equal(oracle.unpack_samples(xq, 1, 16, False, 1.0, 0.0), [[32996.0]])
    assert np.array_equal(oracle.unpack_samples(xq, 1, 16, True, 1.0, 1.0), [[-32539.0]])


@pytest.mark.parametrize("bits", [1, 2, 4, 8, 16])
def test_against_numpy_views(bits):
    rng = np.random.default_rng(bits)
    B, N = 3, 4096
    row_bytes = N * bits // 8 + 3                   # rows may be longer than the samples need
    xq = rng.integers(0, 256, size=(B, row_bytes), dtype=np.uint8)
    scale, offset = 0.37, -1.25
    for signed in (False, True):
        got = oracle.unpack_samples(xq, N, bits, signed, scale, offset)
        if bits == 16:
            code = xq[:, :2 * N].copy().view("<i2" if signed else "<u2").astype(np.int64)
        elif bits == 8:
            code = xq[:, :N].view(np.int8 if signed else np.uint8).astype(np.int64)
        else:
            b = np.unpackbits(xq, axis=1, bitorder="little")[:, :N * bits].reshape(B, N, bits).astype(np.int64)
            code = (b << np.arange(bits)).sum(axis=-1)
            if signed:
                code = np.where(code >= (1 << (bits - 1)), code - (1 << bits), code)
        assert np.array_equal(got, (scale * (code + offset)).astype(np.float32))


@pytest.mark.parametrize("bits", [1, 2, 4, 8, 16])
def test_round_trip_of_the_workload_quantiser(bits):
    wl = W.config0(cases=range(2))
    xq, q = W.quantise(wl.x, bits)
    assert xq.shape == (2, wl.N * bits // 8)
    x = oracle.unpack_samples(xq, wl.N, q["bits"], q["is_signed"], q["scale"], q["offset"])
    err = x.astype(np.float64) - wl.x
    if bits >= 8:
        # rounding to the nearest level, plus the fp32 rounding of the unpacked value
        assert np.max(np.abs(err)) <= 0.5 * q["scale"] + 2.0**-23 * np.max(np.abs(wl.x))
    else:
        L = 1 << bits
        inside = np.abs(wl.x) < (L / 2) * q["scale"]                         # not clipped
        assert np.max(np.abs(err[inside])) <= 0.5 * q["scale"] * (1 + 1e-6)
        assert set(np.unique(np.rint(x / q["scale"] - q["offset"]).astype(int))) <= set(range(L))
    # quantisation noise adds to the receiver noise: a fit on 8-bit samples lands within the noise of the fp32 fit
    if bits == 8:
        a = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=40, generations=250, seed=2)
        b = oracle.fit_blocks(x, wl.fs, wl.lo, wl.hi, NP=40, generations=250, seed=2)
        assert np.max(np.abs(a["best"][:, 3] - b["best"][:, 3])) < 2e-3
        assert np.max(np.abs(a["best"][:, 2] - b["best"][:, 2])) < 5e-3


def test_invalid_arguments():
    xq = np.zeros((1, 4), dtype=np.uint8)
    with pytest.raises(ValueError):
        oracle.unpack_samples(xq, 4, 3, False, 1.0, 0.0)           # 3 bits is no recording mode
    with pytest.raises(ValueError):
        oracle.unpack_samples(xq, 5, 8, False, 1.0, 0.0)           # row too short
