"""Long parity run, GPU vs oracle, printed as JSON lines (not collected by pytest: no test_ prefix).

    python tests/parity_report.py [--config 3] [--checkpoints 1 10 30 60 120]

Advances the CUDA path and the CPU oracle side by side on a BASELINE config and prints, at every checkpoint, the R13
error per conserved field, the cap-event counts of both sides and the differences of alpha and of the deposited totals.
The full 120-step config 3 run takes ~8 minutes of oracle time on the B200 box's 16 cores, which is why the default
GPU suite only compares the first steps (tests/test_gpu_parity.py::test_config3_full_size_first_steps); the record of the
full run is profiles/r1_i_parity_config3_120steps.txt."""
import argparse
import json
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_1511_02137_b200 import hydro as H, synthetic as S  # noqa: E402
from oracle import oracle as O  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--checkpoints", type=int, nargs="+", default=[1, 10, 30, 60, 120])
    args = ap.parse_args()
    c = S.CONFIGS[args.config]
    U0 = S.make_state(args.config)
    g = H.Hydro(*c["n"], c["dx"], c["dt"], nfields=c["nf"])
    o = O.Oracle(*c["n"], c["dx"], c["dt"], nfields=c["nf"])
    g.set_state(U0), o.set_state(U0)
    for pos, d in c["jets"]:
        g.add_jet(pos, d), o.add_jet(pos, d)
    done = 0
    for cp in args.checkpoints:
        t = time.time()
        g.step(cp - done), o.step(cp - done)
        done = cp
        Ug, Uo = g.get_fields(), o.get_fields()
        errs = [float(np.max(np.abs(Ug[f] - Uo[f])) / np.max(np.abs(Uo[f]))) for f in range(c["nf"])]
        dg, do = g.diag(), o.diag()
        print(json.dumps(dict(config=args.config, steps=done, r13_err_per_field=errs, ncap_gpu=dg["ncap"], ncap_oracle=do["ncap"],
                              dalpha=float(np.max(np.abs(dg["alpha"] - do["alpha"]))),
                              ddeposited=float(np.max(np.abs(dg["deposited"] - do["deposited"]))),
                              seconds=round(time.time() - t, 1))), flush=True)


if __name__ == "__main__":
    main()
