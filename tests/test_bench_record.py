"""bench.py's record layout: the driver keeps the first 24 scalar keys of roofline / e2e, so the stated bars go first, flat."""
import bench


def test_priority_keys_first_then_scalars_then_text():
    assert len(bench.ROOFLINE_FIRST) == 24 and len(set(bench.ROOFLINE_FIRST)) == 24
    assert len(bench.E2E_FIRST) == 24 and len(set(bench.E2E_FIRST)) == 24
    assert bench.ROOFLINE_FIRST[:6] == ["bound", "achieved", "peak", "unit", "frac", "traffic"]
    assert bench.E2E_FIRST[:4] == ["value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"]
    d = {"kernel": "pack", "nested": {"a": 1}, "zzz": 3, "frac": 1.0, "bound": "hbm", "at4L_stream_GB": 42.5, "achieved": 5.0,
         "traffic": None, "list": [1, 2]}
    o = bench.ordered_for_record(d, bench.ROOFLINE_FIRST)
    assert list(o) == ["bound", "achieved", "frac", "traffic", "at4L_stream_GB", "zzz", "kernel", "nested", "list"]
    assert o == d and bench.ordered_for_record(None, bench.E2E_FIRST) is None
