"""The kernels divide coordinates by the cell size with a multiply-high (device_types.cuh cell_coord; constants computed in
sim_create): with l = ceil(log2 d), m = floor(2^(31+l) / d) + 1 (< 2^32 for d >= 2),  v // d == ((v * m) >> 32) >> (l - 1)
for every 0 <= v < 2^31 (Granlund-Montgomery, N = 31).  Restated in numpy and checked for EVERY admissible cell size
(2..16384) at the values where a wrong constant shows first: around every multiple of d near 0, near 2^31, and at random.
A wrong quotient would put an agent in the wrong cell, i.e. outside its neighbours' 27-cell search.  CPU only."""
import numpy as np


def test_multiply_high_division_is_exact_for_every_cell_size():
    rng = np.random.default_rng(0)
    top = 2**31 - 1
    for d in range(2, 16385):
        l = (d - 1).bit_length()
        m = (1 << (31 + l)) // d + 1
        assert m < 2**32 and l >= 1
        k = np.concatenate([np.arange(0, 6), top // d - np.arange(0, 6), rng.integers(0, top // d + 1, size=24)])
        v = np.concatenate([k * d - 1, k * d, k * d + 1, k * d + d - 1, [top, top - 1]])
        v = v[(v >= 0) & (v <= top)].astype(np.uint64)
        q = ((v * np.uint64(m)) >> np.uint64(32)) >> np.uint64(l - 1)
        assert (q == v // np.uint64(d)).all(), d
