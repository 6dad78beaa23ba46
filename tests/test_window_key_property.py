"""The packed window test of K4 (DESIGN.md §5 "K4 in detail"; kernels.cuh pack_key) never misses a close pair.

Restated here from the DESIGN.md text in numpy (this is a property of the arithmetic, checked on the CPU; the kernel's own
results are compared with the oracle in tests/test_gpu_parity.py):
  key = three fields (x: 10 bits, y and z: 8 bits of the coordinate >> shift) with two guard bits above each, the
  lower guard set; for keys a, b:  e = b + (K1 - a), K1 = T + 2^w per field;  pass iff ((e & LOW) + U) & GUARD == 0 with
  U = 2^w - 1 - 2T per field; shift = the smallest with T = ceil(R / 2^shift) <= 15.
Claim: |dx|, |dy|, |dz| <= R  =>  pass, for ANY coordinates (the fields are modular, so positions on either side of a
multiple of the field period are handled too).  The converse is not claimed: the test is a filter.
"""
import numpy as np
import pytest

LOW = 0x3FF | (0xFF << 12) | (0xFF << 22)
GUARD = (1 << 10) | (1 << 20) | (1 << 30)


def params(R):
    sh = 0
    while ((R + (1 << sh) - 1) >> sh) > 15:
        sh += 1
    T = (R + (1 << sh) - 1) >> sh
    k1 = (T + (1 << 10)) | ((T + (1 << 8)) << 12) | ((T + (1 << 8)) << 22)
    u = ((1 << 10) - 1 - 2 * T) | (((1 << 8) - 1 - 2 * T) << 12) | (((1 << 8) - 1 - 2 * T) << 22)
    return sh, T, k1, u


def pack(x, y, z, sh):
    return ((x >> sh) & 0x3FF) | (((y >> sh) & 0xFF) << 12) | (((z >> sh) & 0xFF) << 22) | GUARD


def passes(a, b, k1, u):
    e = (b + ((k1 - a) & 0xFFFFFFFF)) & 0xFFFFFFFF
    return ((((e & LOW) + u) & 0xFFFFFFFF) & GUARD) == 0


@pytest.mark.parametrize("R", [1, 7, 15, 16, 50, 51, 100, 500, 1000, 4096, 16384])
def test_every_pair_within_R_on_all_axes_passes(R):
    sh, T, k1, u = params(R)
    assert T <= 15 and 2 * T < 256
    rng = np.random.default_rng(R)
    n = 400_000
    # positions anywhere in the int32 range the library admits, including just below / above multiples of the field period
    base = rng.integers(0, 2**31 - 2 * R - 2, size=(n, 3), dtype=np.int64)
    period = np.array([1024 << sh, 256 << sh, 256 << sh])
    snap = rng.random((n, 3)) < 0.5
    base = np.where(snap, np.minimum((base // period) * period + rng.integers(-R, R + 1, size=(n, 3)), 2**31 - 2 * R - 2), base)
    base = np.maximum(base, R)
    d = rng.integers(-R, R + 1, size=(n, 3))
    d[: n // 8] = np.where(rng.random((n // 8, 3)) < 0.5, R, -R)          # the corners of the window
    other = base + d
    a = pack(base[:, 0], base[:, 1], base[:, 2], sh)
    b = pack(other[:, 0], other[:, 1], other[:, 2], sh)
    assert passes(a, b, k1, u).all() and passes(b, a, k1, u).all()


def test_the_filter_rejects_most_far_pairs_of_a_tile():
    # W4-like: R = 50, neighbours up to three cells (1,344 units) apart in x, inside one 448-unit row in y and z
    sh, T, k1, u = params(50)
    assert (sh, T) == (2, 13)
    rng = np.random.default_rng(1)
    n = 200_000
    p = rng.integers(100_000, 120_000, size=(n, 3), dtype=np.int64)
    q = p + np.stack([rng.integers(-1344, 1345, size=n), rng.integers(-448, 449, size=n), rng.integers(-448, 449, size=n)], axis=1)
    ok = passes(pack(p[:, 0], p[:, 1], p[:, 2], sh), pack(q[:, 0], q[:, 1], q[:, 2], sh), k1, u)
    near = (np.abs(q - p) <= 50).all(axis=1)
    assert ok[near].all()
    coarse = (np.abs(q - p) <= 55).all(axis=1)                              # T * 4 + 3: the widest box the filter lets through
    assert not ok[~coarse].any()
    assert ok.mean() < 2.5 * max(near.mean(), 1e-4)
