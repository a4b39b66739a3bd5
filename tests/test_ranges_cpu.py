"""The range list of the range-granular host access (include/skel.h skel_ranges_add; partial copies)
as a pure function, against a brute-force bitmap model. No GPU."""
import numpy as np

import skel_inputs as I
from paper_1405_2915_b200 import skel as S


def from_bitmap(bits):
    out, start = [], None
    for i, b in enumerate(list(bits) + [False]):
        if b and start is None:
            start = i
        if not b and start is not None:
            out.append((start, i))
            start = None
    return out


def test_ranges_add_matches_a_bitmap_model():
    u = I.raw_u64(1234, 4000)
    k = 0
    for trial in range(200):
        bits = np.zeros(64, bool)
        ranges = []
        for _ in range(10):
            a = int(u[k] % 64); b = int(u[k + 1] % 65); k += 2
            lo, hi = min(a, b), max(a, b)
            ranges = S.ranges_add(ranges, lo, hi)
            bits[lo:hi] = True
            # sorted, disjoint, non-adjacent, and exactly the union
            assert ranges == from_bitmap(bits), (trial, lo, hi, ranges)


def test_ranges_add_special_cases():
    assert S.ranges_add([], 5, 5) == []                      # empty range: no change
    assert S.ranges_add([], 3, 7) == [(3, 7)]
    assert S.ranges_add([(3, 7)], 7, 9) == [(3, 9)]          # adjacent ranges merge
    assert S.ranges_add([(3, 7)], 8, 9) == [(3, 7), (8, 9)]
    assert S.ranges_add([(3, 7), (10, 12)], 0, 2) == [(0, 2), (3, 7), (10, 12)]
    assert S.ranges_add([(3, 7), (10, 12), (20, 30)], 6, 21) == [(3, 30)]
    assert S.ranges_add([(3, 7), (10, 12)], 0, 100) == [(0, 100)]
    assert S.ranges_add([(0, 2 ** 40)], 2 ** 40, 2 ** 41) == [(0, 2 ** 41)]   # 64-bit bounds
