"""Writes tests/golden/oracle_fit_config1_8tracks.txt: the fp64 oracle's fit of the first 8 tracks of
config 1, event 0 (state, chi2, nhits at the outermost layer, and the smoothed state at the innermost).
Calls only oracle/ and the input generator.  The file is a regression anchor for the oracle itself: a change
of its arithmetic must be deliberate (commit message names the passage / reading) and re-run this script.

    python tests/golden/make_oracle_fit_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import kf_oracle as O          # noqa: E402
from workloads import barrel_events as W   # noqa: E402


def compute():
    b = W.simulate_event(W.get_config(1), 0, n_tracks=8)
    r = O.fit_refit_tracks(b.radius, b.x_over_X0, b.Bz, b.mass, b.par, b.cov, b.q, b.hpos, b.hcov, b.mask)
    rows = np.concatenate([r["par"].T, r["chi2"][:, None], r["nhits"][:, None].astype(float),
                           r["rpar"].T, r["rchi2"][:, None]], axis=1)
    return rows


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_fit_config1_8tracks.txt")
    np.savetxt(out, compute(), fmt="%.17g",
               header="oracle fit, config 1 event 0 tracks 0..7 (written by make_oracle_fit_golden.py)\n"
                      "x y z px py pz chi2 nhits | smoothed x y z px py pz chi2_backward")
    print(out)
