"""Host-side check of the arithmetic behind core.cuh's division-free site index: n / d == (n * ceil(2^32 / d)) >> 32 for
every n with n * d < 2^32 -- the condition lqcd_create enforces on V/2 and the extents (no GPU needed)."""
import numpy as np


def _exact(nmax, d):
    m = np.uint64((2 ** 32 + d - 1) // d)
    n = np.arange(max(0, nmax - 3_000_000), nmax, dtype=np.uint64)      # the top of the range is where it would fail first
    lo = np.arange(0, min(nmax, 1_000_000), dtype=np.uint64)
    for v in (n, lo):
        if not np.array_equal((v * m) >> np.uint64(32), v // np.uint64(d)):
            return False
    return True


def test_multiply_high_division_is_exact_under_the_documented_condition():
    for d in (2, 3, 6, 7, 12, 14, 16, 24, 26, 32, 48, 64, 96):
        nmax = (2 ** 32 - 1) // d                 # largest dividend range the condition admits: n * d < 2^32
        assert _exact(nmax, d), d
    # the lattices of BASELINE.json and the largest that fits one B200: V/2 as the dividend, X/2 as the divisor
    for dims in ((4, 4, 4, 4), (16, 16, 16, 32), (32, 32, 32, 64), (48, 48, 48, 96), (64, 64, 64, 128), (96, 96, 96, 192)):
        vh = dims[0] * dims[1] * dims[2] * dims[3] // 2
        assert vh * (dims[0] // 2) < 2 ** 32
        assert _exact(vh, dims[0] // 2) and _exact(vh // (dims[0] // 2), dims[1])


def test_condition_is_needed():
    # beyond the condition the product formula does fail somewhere (so the check in lqcd_create is not decoration)
    d = 96
    m = np.uint64((2 ** 32 + d - 1) // d)
    n = np.arange(2 ** 32 - 5_000_000, 2 ** 32, dtype=np.uint64)
    assert not np.array_equal((n * m) >> np.uint64(32), n // np.uint64(d))
