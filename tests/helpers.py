"""Shared checks of the parity tests (tolerances of BASELINE.json L5 / DESIGN.md "Tolerances")."""
import numpy as np

SIZES = [1, 2, 3, 4, 5, 7, 8, 31, 32, 33, 127, 128, 129, 1023, 1024, 1025, 4095, 4096, 4097, 8191, 8193,
         16385, 100003, (1 << 20) - 1, (1 << 20) + 1]
SIZES_SHORT = [1, 5, 33, 1025, 4097, 8193, 100003, (1 << 20) + 1]


def ulp_distance(got_f32: np.ndarray, ref_f64: np.ndarray) -> np.ndarray:
    """Distance in ordered fp32 bit patterns between got and RN_f32(ref) (reading (c).1 iv)."""
    ref = ref_f64.astype(np.float32)

    def ordered(a):
        i = a.view(np.int32).astype(np.int64)
        return np.where(i < 0, -(i & 0x7FFFFFFF), i)

    return np.abs(ordered(np.ascontiguousarray(got_f32)) - ordered(ref))


def assert_map_f32(got, ref64):
    d = ulp_distance(got, ref64)
    assert d.size == 0 or d.max() <= 1, f"map: max {d.max()} ulp at {int(d.argmax())}"


def assert_reduce_f32(got, ref64, abs_sum, rel=1e-5):
    assert abs(float(got) - ref64) <= rel * abs_sum, f"reduce: |{got} - {ref64}| > {rel} * {abs_sum}"


def assert_overlap(got, ref64, absref, rel=2e-6):
    err = np.abs(got.astype(np.float64) - ref64)
    bad = err > rel * absref
    assert not bad.any(), (f"overlap: {int(bad.sum())} elements out of tolerance; worst ratio "
                           f"{float((err / np.maximum(absref, 1e-300)).max()):.3e} at {np.argwhere(bad)[0]}")
    return float((err / np.maximum(absref, 1e-300)).max()) if err.size else 0.0
