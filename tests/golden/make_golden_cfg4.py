"""Writes tests/golden/cfg4_oracle.txt: the ORACLE's outputs on the FULL configs[4] interval (BASELINE.json:11: N=512,
T=20, F=8, K=50 x 40 sources, 3 EM x 10 LM) -- the workload bench.py times -- so that the CUDA path can be compared with
the oracle at the bench's own size, not only on sampled outputs.

    python tests/golden/make_golden_cfg4.py [out_path]        # ~15 min on 16 cores, ~80 GB of host memory

Calls only oracle/ and the seeded input generator (never the CUDA path); SURVEY.md §8(d) "A full config-4 oracle run ...
is therefore feasible and should be run".  Stored: the 50 final per-cluster costs, the 151 entries of the cost trace,
||J||^2 per cluster, sampled Jones and residual entries, the oracle's min |rho| (parity seeds need > 1e-6, DESIGN.md §3
Q18).  Format: `name value` per line, floats as C99 hex (exact).
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle  # noqa: E402
from sagecal_inputs import make_config  # noqa: E402

SAMPLE_ROWS = 64          # residual rows stored (seeded choice)
SAMPLE_SEED = 4


def sample_rows(p):
    return np.sort(np.random.default_rng(SAMPLE_SEED).choice(p.rows, SAMPLE_ROWS, replace=False))


def compute(log=print):
    p = make_config(4)
    t0 = time.time()
    coh = np.empty((p.K, p.rows, p.F, 4), np.complex128)          # 67 GB: filled cluster by cluster, never copied
    for k in range(p.K):
        coh[k] = oracle.predict(p, clusters=[k])[0]
        if k % 10 == 9:
            log(f"predict {k + 1}/{p.K}  {time.time() - t0:.0f} s")
    vis = oracle.simulate(p, coh)
    log(f"simulate done {time.time() - t0:.0f} s")
    out = oracle.sage(p.N, p.T, p.F, vis, coh, p.jones_init(), p.n_em, p.n_lm, p.tau)
    log(f"sage done {time.time() - t0:.0f} s, min|rho| {out['min_abs_rho']:.3e}, accepted {out['n_accept']}")
    vals = {"vis_norm2": float(np.vdot(vis, vis).real), "min_abs_rho": float(out["min_abs_rho"]),
            "n_accept": float(out["n_accept"]),
            "residual_norm2": float(np.vdot(out["residual"], out["residual"]).real)}
    for k in range(p.K):
        vals[f"cost_cluster_{k}"] = float(out["cost_per_cluster"][k])
        vals[f"jones_norm2_{k}"] = float(np.vdot(out["jones"][k], out["jones"][k]).real)
    for i, c in enumerate(out["cost_trace"]):
        vals[f"cost_trace_{i}"] = float(c)
    for k in (0, 17, 49):
        for s in (0, 255, 511):
            for e, z in enumerate(out["jones"][k, s].reshape(4)):
                vals[f"jones_{k}_{s}_{e}_re"] = float(z.real)
                vals[f"jones_{k}_{s}_{e}_im"] = float(z.imag)
    rows = sample_rows(p)
    res = out["residual"][rows]                                    # [64, F, 4]
    vals["residual_sample_norm2"] = float(np.vdot(res, res).real)
    for i, r in enumerate(rows):
        for c in (0, p.F - 1):
            for e in (0, 1):
                vals[f"residual_{r}_{c}_{e}_re"] = float(res[i, c, e].real)
                vals[f"residual_{r}_{c}_{e}_im"] = float(res[i, c, e].imag)
    return vals


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    path = sys.argv[1] if len(sys.argv) > 1 else os.path.join(here, "cfg4_oracle.txt")
    oracle.build()
    vals = compute()
    with open(path, "w") as f:
        f.write("# oracle outputs on the full configs[4] interval (BASELINE.json:11), written by "
                "tests/golden/make_golden_cfg4.py; C99 hex floats\n")
        for k, v in vals.items():
            f.write(f"{k} {float(v).hex()}\n")
    print(path)


if __name__ == "__main__":
    main()
