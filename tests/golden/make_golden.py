"""Writes tests/golden/cfg0_oracle.txt: regression values of the CPU oracle on BASELINE.json:configs[0] (seed 0).

The paper (arXiv 2310.20103) prints no worked numerical example, so there is no paper value to store; this file freezes
what the ORACLE gives today so that a later change to its arithmetic shows up as a diff (such a change must name the
passage or DESIGN.md reading that justifies it).  It calls oracle/ and the seeded input generators only -- never
the CUDA path.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import gw_oracle as orc  # noqa: E402
from paper_2310_20103_b200 import synth  # noqa: E402


def compute():
    p = synth.make_problem(0)
    r = orc.run_chains(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, p.n_idx, p.m_idx, 12, p.omega, p.cfg.eta, reorth=True)
    sx = orc.exchange_eq6(p.phi_v, p.phi_c, p.V, p.cfg.n_v - 1)
    rows = []
    for j in range(p.cfg.n_chains):
        rows.append(("norm2", j, 0, r["norm2"][j]))
        for k in range(12):
            rows.append(("alpha", j, k, r["alpha"][j, k]))
            rows.append(("beta", j, k, r["beta"][j, k]))
        for iw in (0, 100, 200):
            rows.append(("sigma_re", j, iw, r["sigma"][j, iw].real))
            rows.append(("sigma_im", j, iw, r["sigma"][j, iw].imag))
    rows.append(("sigma_x_homo", 0, 0, sx))
    return rows


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle.txt")
    with open(out, "w") as f:
        f.write("# oracle/gw_oracle.py on BASELINE.json:configs[0], seed 0, 12 Lanczos steps, reorthogonalised; eV units\n")
        f.write("# PAPER.md:87-90 (Eq. 13: alpha = a_k, beta = b_{k+1}), :77 (Eq. 11: sigma), :57 (Eq. 6: sigma_x)\n")
        f.write("# written by tests/golden/make_golden.py (oracle only); quantity chain index value\n")
        for name, j, k, v in compute():
            f.write(f"{name} {j} {k} {float(v)!r}\n")
    print(out)
