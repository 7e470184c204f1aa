"""Writes the stored expected values tests/golden/cfg<N>.json.  Calls ONLY oracle/ (and the seeded input
generator); never the CUDA path.  Usage (from the repo root):

    python tests/golden/make_golden.py <cfg> <nsteps> [probe_step ...]

e.g.  python tests/golden/make_golden.py 2 200 1 2 10 200     (BASELINE.json config 2, full run)
      python tests/golden/make_golden.py 3 100 1 2 5 100      (config 3 = the metric shape)
      python tests/golden/make_golden.py shape 8 256 10 [base_cfg=2] [nsteps=1]
          -> tests/golden/shape_8_256_10.json: config `base_cfg` with the grids and rank overridden, for the parity of
             the n = 256 / r = 20 kernel paths, whose oracle steps take many minutes of host time
      python tests/golden/make_golden.py 5 1                  (config 5 at full size: ~35 GB, about an hour)
Stored: per-step electric energy / mass / kinetic energy / ||S||_F (step 0 = initial state) and
f at the 64 seeded probe pairs after each requested step.  No value here comes from the paper (it prints
none for these quantities, PAPER.md:472 gives only orders of magnitude); the citation for each quantity's
definition is in oracle/dlr_oracle.py (moments, f_at)."""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import dlr_oracle as O                      # noqa: E402
from paper_2110_13481_b200 import inputs                # noqa: E402


def main():
    if sys.argv[1] == "shape":
        n_x, n_v, r = int(sys.argv[2]), int(sys.argv[3]), int(sys.argv[4])
        idx = int(sys.argv[5]) if len(sys.argv) > 5 else 2
        nsteps = int(sys.argv[6]) if len(sys.argv) > 6 else 1
        probe_steps = list(range(1, nsteps + 1))
        cfg = inputs.make_config(idx, n_x=n_x, n_v=n_v, r=r)
        name, gen = f"shape_{n_x}_{n_v}_{r}.json", f"make_config({idx}, n_x={n_x}, n_v={n_v}, r={r})"
    else:
        idx, nsteps = int(sys.argv[1]), int(sys.argv[2])
        probe_steps = sorted({int(a) for a in sys.argv[3:]} | {nsteps})
        cfg = inputs.make_config(idx)
        name, gen = f"cfg{idx}.json", f"make_config({idx})"
    gx = O.Grid3((cfg["n_x"],) * 3, (cfg["x_lo"],) * 3, (cfg["x_hi"],) * 3)
    gv = O.Grid3((cfg["n_v"],) * 3, (cfg["v_lo"],) * 3, (cfg["v_hi"],) * 3)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    stats = {}
    hist = [O.moments(X, S, V, gx, gv)]
    probes = {"0": O.f_at(X, S, V, ix, iv).tolist()}
    t0 = time.time()
    for step in range(1, nsteps + 1):
        X, S, V = O.step_alg2(X, S, V, cfg["tau"], gx, gv, 1.0, stats)
        hist.append(O.moments(X, S, V, gx, gv))
        if step in probe_steps:
            probes[str(step)] = O.f_at(X, S, V, ix, iv).tolist()
        print(f"cfg {idx} step {step}/{nsteps}  ee={hist[-1]['electric_energy']:.12e}  {time.time() - t0:.0f}s", flush=True)
    out = {
        "config": idx, "n": cfg["n"], "n_x": cfg["n_x"], "n_v": cfg["n_v"], "r": cfg["r"], "tau": cfg["tau"], "steps": nsteps,
        "generator": "paper_2110_13481_b200.inputs.initial_factors(%s), probe_indices seed 7" % gen,
        "written_by": "tests/golden/make_golden.py (oracle/dlr_oracle.py step_alg2)",
        "qr_fallbacks": stats.get("qr_fallbacks", 0),
        "electric_energy": [h["electric_energy"] for h in hist],
        "mass": [h["mass"] for h in hist],
        "kinetic_energy": [h["kinetic_energy"] for h in hist],
        "s_fro": [h["s_fro"] for h in hist],
        "f_probe": probes,
    }
    with open(os.path.join(ROOT, "tests", "golden", name), "w") as f:
        json.dump(out, f, indent=0)


if __name__ == "__main__":
    main()
