"""Per-warp timeline of one launch of the tile kernel (xrdvi_debug_timeline), as text.

``python -m paper_2501_09308_b200.timeline --config 1`` prints, for the synthetic workload of that config:
the launch span, the number of resident warps in 5 us bins, when the SMs run out of work, and the time a warp
needs per (peak, tile) record and phase as a function of when it started.  The measurement behind the
"drain of the last wave" statements in DESIGN.md and profiles/.
"""
from __future__ import annotations

import argparse

import numpy as np

from . import synth
from .binding import Xrdvi


def summarize(rows: np.ndarray, bin_us: float | None = None) -> str:
    rows = rows[rows[:, 0] > 0]
    t0 = rows[:, 0].astype(np.int64)
    t1 = rows[:, 1].astype(np.int64)
    t2 = rows[:, 2].astype(np.int64)
    sm = (rows[:, 3] & np.uint64(0xFFFFFFFF)).astype(np.int64)
    rec = (rows[:, 3] >> np.uint64(32)).astype(np.int64)
    base = t0.min()
    t0, t1, t2 = t0 - base, t1 - base, t2 - base
    n_sm = len(np.unique(sm))
    span_us = t2.max() / 1e3
    if bin_us is None:                                       # about 35 bins, at least 5 us wide
        bin_us = max(5.0, float(np.ceil(span_us / 35.0)))
    start_bin = max(10, int(np.ceil(span_us / 16.0)))
    out = [f"warps {len(rows)}  SMs {n_sm}  span {t2.max() / 1e3:.1f} us  "
           f"integrated warp-time {float((t2 - t0).sum()) / 1e6:.1f} ms"]
    out.append("phase 1 per warp: mean %.1f max %.1f us   phase 2: mean %.1f max %.1f us" % (
        (t1 - t0).mean() / 1e3, (t1 - t0).max() / 1e3, (t2 - t1).mean() / 1e3, (t2 - t1).max() / 1e3))
    w = int(bin_us * 1e3)
    peak = 0.0
    lines = []
    for lo in range(0, int(t2.max()) + w, w):
        res = np.clip(np.minimum(t2, lo + w) - np.maximum(t0, lo), 0, None).sum() / w
        in1 = np.clip(np.minimum(t1, lo + w) - np.maximum(t0, lo), 0, None).sum() / w
        peak = max(peak, res)
        lines.append((lo / 1e3, res, in1))
    out.append(f"resident warps per {bin_us:g} us bin (peak {peak:.0f} = {peak / n_sm:.1f} per SM):")
    for lo, res, in1 in lines:
        out.append("  %6.0f us  %6.0f  (%.2f of peak)  in phase 1: %6.0f" % (lo, res, res / peak, in1))
    ends = np.array([t2[sm == s].max() for s in np.unique(sm)]) / 1e3
    out.append("last warp of an SM ends: min %.1f  median %.1f  max %.1f us;  last warp starts at %.1f us" % (
        ends.min(), np.median(ends), ends.max(), t0.max() / 1e3))
    out.append("time per record and phase by start time (ns; warps with records only):")
    ok = rec > 0
    for lo in range(0, int(t0.max() / 1e3) + start_bin, start_bin):
        sel = ok & (t0 / 1e3 >= lo) & (t0 / 1e3 < lo + start_bin)
        if sel.sum() < 8:
            continue
        p1 = ((t1 - t0)[sel] / rec[sel]).mean()
        p2 = ((t2 - t1)[sel] / rec[sel]).mean()
        out.append("  start %5d-%5d us: %5d warps, %.1f records, phase 1 %.0f, phase 2 %.0f" % (
            lo, lo + start_bin, sel.sum(), rec[sel].mean(), p1, p2))
    return "\n".join(out)


def main() -> None:
    ap = argparse.ArgumentParser(description=__doc__)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--S", type=int, default=0, help="draws per instance (default: the config's)")
    ap.add_argument("--seed", type=int, default=1)
    args = ap.parse_args()
    wl = synth.make_workload(args.config, S=args.S) if args.S > 0 else synth.make_workload(args.config)
    g = Xrdvi.from_workload(wl)
    rows = g.debug_timeline(seed=args.seed)
    print(f"config {args.config}: S {g.S_max}, {g.pair_count} pairs per draw")
    print(summarize(rows))
    g.close()


if __name__ == "__main__":
    main()
