"""Writes tests/golden/oracle_plan_<config>.json: the fp64 CPU oracle's free-running column-generation
plan (O9) on a BASELINE.json phantom -- per-iteration beam, reduced
cost and master optimum, the leaves of every aperture, and the final objective.  Calls ONLY the seeded input generator and
oracle/ (never the CUDA path).  The GPU parity test compares its own free-running plan against the
stored final objective within the north star's 1e-3.

    python tests/golden/make_oracle_plan.py cfg1 50      # ~2.5 min on one core
"""
import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import dao_oracle as orc                              # noqa: E402
from paper_1003_5402_b200.inputs import phantom                   # noqa: E402


def main():
    config = sys.argv[1] if len(sys.argv) > 1 else "cfg1"
    n_ap = int(sys.argv[2]) if len(sys.argv) > 2 else 50
    ph = phantom.make(config, 0)
    t0 = time.perf_counter()
    plan = orc.run(ph, n_ap)
    seconds = time.perf_counter() - t0
    out = {
        "written_by": "tests/golden/make_oracle_plan.py (oracle/ only)",
        "config": config, "seed": 0, "phantom": ph.name, "n_vox": int(ph.n_vox), "n_bl": int(ph.n_bl),
        "nnz": int(ph.nnz), "n_apertures": len(plan.beams), "converged": bool(plan.converged),
        "master": {"method": "projected Newton", "tol": 1e-10}, "price_tol": 1e-9,
        "oracle_seconds_one_core": round(seconds, 1),
        "objective": plan.objective,
        "beams": [int(b) for b in plan.beams],
        "price": [float(h.price) for h in plan.history],
        "master_objective": [float(h.objective) for h in plan.history],
        "master_iterations": [int(h.n_master_iter) for h in plan.history],
        "kkt": [float(h.kkt) for h in plan.history],
        "n_duplicates": int(plan.n_duplicates), "stalled": bool(plan.stalled),
        "n_open_beamlets": [int(sum(int(r) - int(l) for l, r in zip(h.left, h.right))) for h in plan.history],
        # the apertures themselves (half-open leaves of the rows of aperture k's beam, in row order), so that a test can
        # load the ORACLE's pool at any size K with dao_set_pool and solve the master on it (lock-step at large K)
        "left": [[int(v) for v in plan.lefts[k]] for k in range(len(plan.beams))],
        "right": [[int(v) for v in plan.rights[k]] for k in range(len(plan.beams))],
    }
    path = os.path.join(HERE, f"oracle_plan_{config}.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print(path, seconds, plan.objective)


if __name__ == "__main__":
    main()
