"""Writes tests/golden/oracle_regression.json.  Calls only oracle/ and the seeded input generators."""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle as O  # noqa: E402
from paper_2007_14931_b200 import workloads as W  # noqa: E402


def build():
    out = {"note": "written by tests/golden/make_golden.py from oracle/ only; floats as hex", "configs": {}}
    for cfg in (0, 1, 2):
        Mo = O.Model(W.DECAY, W.resonances(cfg))
        c = W.couplings(cfg)
        xn, wn = W.norm_events(cfg, 400)
        x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=60)
        v = Mo.eval_events(c, x, eff)
        nll, integral = Mo.nll(c, x, eff, xn, wn)
        B = Mo.basis_terms(x[:, 0])
        out["configs"][str(cfg)] = {
            "n_data": 60, "n_norm": 400,
            "x0": [float(t).hex() for t in x[:, 0]],
            "eps_S": [float(t).hex() for t in v[:12]],
            "basis_terms_event0": [[float(z.real).hex(), float(z.imag).hex()] for z in B.ravel()],
            "nll": float(nll[0]).hex(), "integral": float(integral[0]).hex(),
        }
    return out


if __name__ == "__main__":
    with open(os.path.join(HERE, "oracle_regression.json"), "w") as f:
        json.dump(build(), f, indent=1)
    print("wrote oracle_regression.json")
