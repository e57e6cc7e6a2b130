"""Writes tests/golden/cfg0_oracle_values.txt: ELBO, log-likelihoods and gradient of config 0 at two fixed
states, computed by the fp64 oracle ONLY (oracle/ + the seeded input generator; no CUDA code is imported).
The file guards the oracle against silent drift: a later change of its arithmetic must regenerate it and say
why in the commit message.  Run:  python tests/golden/make_golden.py
"""
import pathlib
import sys

import numpy as np

ROOT = pathlib.Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

from oracle import xrdvi_oracle as orc            # noqa: E402
from paper_2501_09308_b200 import synth           # noqa: E402  (inputs only)


PHASE_WINDOWS = (22, 9, 15, 4, 22, 11)     # per-phase half-widths of the "gauss_windows" case (R27)


def cases():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    st0 = o.init_state()
    st1 = synth.random_state(wl.K, 1, 1, seed=21).astype(np.float64)
    st1[:, :, 0, :, 0] += np.log(1.0 / o.lambda_h()) - 2.0
    wlp = synth.make_workload(0, peak_counts=2.0e4)
    op = orc.from_workload(wlp)
    f32 = lambda a: a.astype(np.float32).astype(np.float64)     # states a float32 API can hold exactly
    yield "gauss_init", o, f32(st0), wl.S, 3, 1
    yield "gauss_rand", o, f32(st1), wl.S, 3, 7
    yield "poisson_init", op, f32(op.init_state()), wlp.S, 5, 2
    ow = orc.from_workload(wl)
    ow.set_phase_windows(PHASE_WINDOWS)
    yield "gauss_windows", ow, f32(st1), wl.S, 9, 4


def main():
    out = ["# case  quantity  index  value   (oracle/xrdvi_oracle.c, fp64; see make_golden.py)"]
    for name, o, st, S, seed, it in cases():
        elbo, grad, ll = o.elbo_grad(st, S, seed, it, want_ll=True)
        out.append(f"{name} elbo 0 {float(elbo[0, 0])!r}")
        for s in range(S):
            out.append(f"{name} ll {s} {float(ll[0, 0, s])!r}")
        g = grad.reshape(-1)
        for j in range(g.shape[0]):
            out.append(f"{name} grad {j} {float(g[j])!r}")
    path = pathlib.Path(__file__).resolve().parent / "cfg0_oracle_values.txt"
    path.write_text("\n".join(out) + "\n")
    print(f"wrote {path} ({len(out) - 1} values)")


if __name__ == "__main__":
    main()
