"""Writes tests/golden/c0_oracle.json from the CPU oracle alone (never from the CUDA path).

The paper prints no numeric worked example (PAPER.md has only three wall-clock pairs),
so this fixture is a regression guard for the oracle's own arithmetic on config C0
(BASELINE.json configs[0]); the facts that pin the oracle are in tests/test_oracle_pins.py.
Usage: python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "oracle"))

import pd_oracle  # noqa: E402
from paper_2006_09808_b200 import synth  # noqa: E402


def main():
    d = synth.generate(0)
    cfg = d["cfg"]
    out = pd_oracle.solve(d["field"], d["mask"], lambda_=cfg.lam, sigma=cfg.sigma, tau=cfg.tau, theta=cfg.theta,
                          max_iters=cfg.iters)
    chi = out["chi"][0]
    its = [1, 2, 3, 5, 10, 20, 30, 50, 70, 100]
    doc = {
        "source": "oracle/pd_oracle.cpp pdo_solve_f64 on synth.generate(0); written by tests/golden/make_golden.py",
        "config": "BASELINE.json configs[0]: 64x64, 100 iterations, lambda=0.01, sigma=tau=0.25, theta=1, B0 along y",
        "iters": its,
        "relgap": [float(out["relgap"][0, n - 1]) for n in its],
        "relres": [float(out["relres"][0, n - 1]) for n in its],
        "chi_max": float(chi.max()), "chi_min": float(chi.min()),
        "chi_l2": float(np.linalg.norm(chi)),
        "chi_argmax": [int(v) for v in np.unravel_index(chi.argmax(), chi.shape)],
        "chi_samples": {"%d,%d" % (y, x): float(chi[y, x]) for y, x in [(0, 0), (7, 13), (31, 32), (40, 9), (63, 63)]},
        "field_l2": float(np.linalg.norm(d["field"].astype(np.float64))),
    }
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "c0_oracle.json"), "w") as f:
        json.dump(doc, f, indent=1)
    print(json.dumps(doc, indent=1))


if __name__ == "__main__":
    main()
