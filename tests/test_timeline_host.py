"""Host logic of the timeline report (paper_2501_09308_b200/timeline.py) on synthetic stamp rows; no GPU."""
import numpy as np

from paper_2501_09308_b200.timeline import summarize


def _rows(t0, d1, d2, sm, rec):
    t0 = np.asarray(t0, dtype=np.uint64)
    t1 = t0 + np.asarray(d1, dtype=np.uint64)
    t2 = t1 + np.asarray(d2, dtype=np.uint64)
    tag = np.asarray(sm, dtype=np.uint64) | (np.asarray(rec, dtype=np.uint64) << np.uint64(32))
    return np.stack([t0, t1, t2, tag], axis=1)


def test_summary_of_two_back_to_back_waves():
    # 4 SMs x 2 slots: a first wave of 8 warps at t = 1 us, a second wave of 8 when the first ends at 31 us
    n = 16
    t0 = [1000] * 8 + [31000] * 8
    rows = _rows(t0, [10000] * n, [20000] * n, [i % 4 for i in range(n)], [10] * n)
    text = summarize(rows)
    assert "warps 16  SMs 4  span 60.0 us" in text
    assert "integrated warp-time 0.5 ms" in text               # 16 x 30 us
    assert "phase 1 per warp: mean 10.0 max 10.0 us   phase 2: mean 20.0 max 20.0 us" in text
    assert "(peak 8 = 2.0 per SM)" in text
    assert "last warp starts at 30.0 us" in text
    assert "phase 1 1000, phase 2 2000" in text                # ns per record: 10 us / 10 records, 20 us / 10


def test_unwritten_rows_and_empty_shares_are_ignored():
    rows = _rows([0, 5000, 6000], [0, 1000, 1000], [0, 1000, 1000], [0, 1, 2], [0, 0, 4])
    text = summarize(rows)
    assert text.startswith("warps 2  SMs 2")                   # the all-zero row was never written
