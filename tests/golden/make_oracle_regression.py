"""Writes tests/golden/oracle_regression.txt: digests of the ORACLE's own results on small seeded workloads, so that an
unintended change of the oracle's arithmetic (a refactoring that was meant to leave a code path alone) shows up as a
failed test.  Calls only oracle/ and the seeded input generator; no value here comes from the CUDA path or the paper.

    python tests/golden/make_oracle_regression.py          # rewrite the file (say why in the commit message)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2105_01796_b200 import workloads as W  # noqa: E402

CASES = [("cfg0", 0, {}), ("cfg1", 1, {}), ("cfg2", 2, {}), ("cfg3", 3, {}), ("cfg4", 4, {}), ("cfg4_gradient", 4, dict(field_gradient=1)),
         ("barrel", 5, {}), ("endcap", 6, {}), ("cfg2_inflated", 2, dict(cov_inflation=1e4)), ("cfg1_steps", 1, dict(max_step_mm=7.0))]
N = 200


def digest(name, cfg, over):
    wl = W.make_workload(cfg, n_tracks=N)
    r = oracle.fit_workload(wl, states=True, perigee=((0.0, 0.0, 0.0), (0.0, 0.0, 1.0)), **over)
    ok = (r.status & 7) == 0
    vals = [float(np.sum(r.chi2[ok])), float(np.sum(r.n_used)), float(np.sum(r.status))]
    vals += [float(v) for v in np.sum(np.abs(r.first_params[ok]), axis=0)]
    vals += [float(v) for v in np.sum(np.abs(r.last_params[ok]), axis=0)]
    vals += [float(v) for v in np.sum(np.einsum("nii->ni", r.first_cov[ok]), axis=0)]
    vals += [float(v) for v in np.sum(np.einsum("nii->ni", r.last_cov[ok]), axis=0)]
    vals += [float(np.nansum(np.abs(r.smooth_params))), float(np.nansum(np.abs(r.pred_cov)))]
    pk = ok & ((r.status & 128) == 0)
    vals += [float(np.sum(np.abs(r.perigee_params[pk]))), float(np.sum(np.einsum("nii->ni", r.perigee_cov[pk])))]
    return name, vals


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_oracle_regression.py (oracle/ only): name, then sums over %d tracks\n" % N)
        for c in CASES:
            name, vals = digest(*c)
            f.write(name + " " + " ".join("%.15e" % v for v in vals) + "\n")
    print(path)


if __name__ == "__main__":
    main()
