#!/usr/bin/env python
"""Writes tests/golden/oracle_tiny.json: the oracle's results on a tiny seeded case, so that a later change to
the oracle's arithmetic shows up as a diff of a committed file (such a change must cite the passage or DESIGN.md
reading that justifies it).  Calls only `oracle/` and the seeded generators; nothing here touches the CUDA path.

    python tests/golden/make_golden.py

The paper prints no usable worked example: Table 1 gives convolution / gradient values and
ratios without their inputs ("parity unpinned" for those values), Table 3 only timings.
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import fk_oracle as O  # noqa: E402
from paper_1909_10547_b200 import synth  # noqa: E402


def build():
    case = synth.hadronic_case(14, 3, 4, 5, 2, nfl=3, sub=1)
    sigma, scale = O.hadronic(case.fk, case.pairs, case.f)
    df, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    dis = synth.config1(R=1, N=4)
    sd, sds = O.dis(dis.fk, dis.flav, dis.f)
    dd, ddD = O.dis_vjp(dis.fk, dis.flav, dis.f, dis.g)
    return {
        "about": "oracle outputs (hex floats) on seeded inputs: hadronic_case(14, N=3, nx=4, C=5, R=2, nfl=3, sub=1); config1(R=1, N=4)",
        "hadronic_sigma": [float(x).hex() for x in sigma.ravel()],
        "hadronic_scale": [float(x).hex() for x in scale.ravel()],
        "hadronic_df": [float(x).hex() for x in df.ravel()],
        "hadronic_D": [float(x).hex() for x in D.ravel()],
        "dis_sigma": [float(x).hex() for x in sd.ravel()],
        "dis_scale": [float(x).hex() for x in sds.ravel()],
        "dis_df": [float(x).hex() for x in dd[:, dis.flav, :6].ravel()],      # active flavours, first 6 x-points
        "dis_D": [float(x).hex() for x in ddD[:, dis.flav, :6].ravel()],
    }


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny.json")
    with open(out, "w") as fh:
        json.dump(build(), fh, indent=1)
    print(out)
