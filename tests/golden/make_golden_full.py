"""Writes full-budget ORACLE fixtures at the sizes the bench and the paper's grid use, so that the CUDA path is compared
with the oracle on whole intervals (3 EM x 10 LM, every cluster), not only on sampled outputs:

    python tests/golden/make_golden_full.py cfg3    [outdir]   # configs[3]: N=256, T=20, F=4, K=50 x 20 sources
    python tests/golden/make_golden_full.py cfg4pol [outdir]   # configs[4]'s shape (N=512, T=20, F=8, 40 sources per
                                                               # cluster) with POLARISED sources, K cut to 4
    python tests/golden/make_golden_full.py cfg4    [outdir]   # configs[4] in full (about 80 GB of host memory)

Calls only oracle/ and the seeded input generator (never the CUDA path): SURVEY.md §8(d) "a full config-3 oracle run
takes 1-1.5 min", VERDICT r01 "next round" item 7.  cfg4pol exists because configs[4] is unpolarised (XY = YX = 0
exactly): with it the tensor-core statistics kernel sees non-zero off-diagonal coherencies at the bench's N, T, F.

Per fixture: <name>_oracle.txt (`name value` per line, floats as C99 hex: the final per-cluster costs, the cost trace,
||J_k||^2, ||V||^2, ||R||^2, sampled residual entries, the oracle's min |rho| -- parity seeds need > 1e-6, DESIGN.md
§3 Q18 -- and its host time) and <name>_oracle_jones.npy (the WHOLE Jones array [K, N, 2, 2] complex128).
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
VARIANTS = {
    "cfg3": dict(index=3, overrides={}, sample_seed=3),
    "cfg4pol": dict(index=4, overrides=dict(K=4, polarised=True), sample_seed=5),
    "cfg4": dict(index=4, overrides={}, sample_seed=4),
}


def problem(name):
    v = VARIANTS[name]
    return make_config(v["index"], **v["overrides"])


def sample_rows(name, p):
    return np.sort(np.random.default_rng(VARIANTS[name]["sample_seed"]).choice(p.rows, SAMPLE_ROWS, replace=False))


def compute(name, log=print):
    p = problem(name)
    t0 = time.time()
    coh = np.empty((p.K, p.rows, p.F, 4), np.complex128)          # filled cluster by cluster, never copied
    for k in range(p.K):
        coh[k] = oracle.predict(p, clusters=[k])[0]
        if k % 10 == 9 or k == p.K - 1:
            log(f"predict {k + 1}/{p.K}  {time.time() - t0:.0f} s")
    t_pred = time.time() - t0
    vis = oracle.simulate(p, coh)
    t1 = time.time()
    out = oracle.sage(p.N, p.T, p.F, vis, coh, p.jones_init(), p.n_em, p.n_lm, p.tau)
    t_sage = time.time() - t1
    log(f"sage done {time.time() - t0:.0f} s, min|rho| {out['min_abs_rho']:.3e}, accepted {out['n_accept']}")
    vals = {"vis_norm2": float(np.vdot(vis, vis).real), "min_abs_rho": float(out["min_abs_rho"]),
            "n_accept": float(out["n_accept"]),
            "residual_norm2": float(np.vdot(out["residual"], out["residual"]).real),
            "offdiag_coh_norm2": float(np.vdot(coh[..., 1:3], coh[..., 1:3]).real),
            "host_seconds_predict": t_pred, "host_seconds_sage": t_sage, "host_threads": float(oracle.num_threads())}
    for k in range(p.K):
        vals[f"cost_cluster_{k}"] = float(out["cost_per_cluster"][k])
        vals[f"jones_norm2_{k}"] = float(np.vdot(out["jones"][k], out["jones"][k]).real)
    for i, c in enumerate(out["cost_trace"]):
        vals[f"cost_trace_{i}"] = float(c)
    rows = sample_rows(name, p)
    res = out["residual"][rows]                                    # [64, F, 4]
    vals["residual_sample_norm2"] = float(np.vdot(res, res).real)
    for i, r in enumerate(rows):
        for c in (0, p.F - 1):
            for e in range(4):
                vals[f"residual_{r}_{c}_{e}_re"] = float(res[i, c, e].real)
                vals[f"residual_{r}_{c}_{e}_im"] = float(res[i, c, e].imag)
    return vals, np.ascontiguousarray(out["jones"])


def main():
    if len(sys.argv) < 2 or sys.argv[1] not in VARIANTS:
        raise SystemExit(__doc__)
    name = sys.argv[1]
    outdir = sys.argv[2] if len(sys.argv) > 2 else os.path.dirname(os.path.abspath(__file__))
    oracle.build()
    vals, jones = compute(name)
    path = os.path.join(outdir, f"{name}_oracle.txt")
    with open(path, "w") as f:
        f.write(f"# oracle outputs on the full-budget {name} interval, written by tests/golden/make_golden_full.py {name}; "
                "C99 hex floats\n")
        for k, v in vals.items():
            f.write(f"{k} {float(v).hex()}\n")
    np.save(os.path.join(outdir, f"{name}_oracle_jones.npy"), jones)
    print(path)


if __name__ == "__main__":
    main()
