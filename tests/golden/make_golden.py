"""Writes tests/golden/cfg0_oracle.txt: the ORACLE's outputs on configs[0] (BASELINE.json:7), a regression fixture.

    python tests/golden/make_golden.py

Calls only oracle/ and the seeded input generator (never the CUDA path).  The paper prints no worked example
and no numeric value, so there is nothing of the paper's to store; these values pin the oracle against silent change
(any later edit of its arithmetic must regenerate this file and say why in the commit message) and give the GPU tests a
second, stored, expectation.  Format: `name value` per line, floats as C99 hex (exact).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle  # noqa: E402
from sagecal_inputs import make_config  # noqa: E402


def compute():
    p = make_config(0)
    coh = oracle.predict(p)
    vis = oracle.simulate(p, coh)
    out = oracle.sage(p.N, p.T, p.F, vis, coh, p.jones_init(), p.n_em, p.n_lm, p.tau)
    phi, G, M = oracle.cost_grad_jtj(p.N, p.T, p.F, vis, coh[0], p.jones_init()[0])
    vals = {
        "coh_sum_re": float(coh.real.sum()), "coh_sum_im": float(coh.imag.sum()),
        "coh_norm2": float(np.vdot(coh, coh).real),
        "vis_norm2": float(np.vdot(vis, vis).real),
        "phi_identity": float(phi),
        "G_norm2_identity": float(np.vdot(G, G).real), "M_trace_identity": float(np.trace(M.sum(0)).real),
        "cost_cluster0": float(out["cost_per_cluster"][0]),
        "residual_norm2": float(np.vdot(out["residual"], out["residual"]).real),
        "n_accept": float(out["n_accept"]),
    }
    for i, c in enumerate(out["cost_trace"]):
        vals[f"cost_trace_{i}"] = float(c)
    return vals


def main():
    vals = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle.txt")
    with open(path, "w") as f:
        f.write("# oracle outputs on configs[0] (BASELINE.json:7), written by tests/golden/make_golden.py; C99 hex floats\n")
        for k, v in vals.items():
            f.write(f"{k} {float(v).hex()}\n")
    print(path)


if __name__ == "__main__":
    main()
