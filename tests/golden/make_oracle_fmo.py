"""Writes tests/golden/oracle_fmo_<config>.json: the oracle's FMO optimum
min_{x >= 0} F(D x) by the dense projected-Newton master on D^T (orc.fmo(method="newton"), tol 1e-10).
Calls ONLY the seeded input generator and oracle/.

    python tests/golden/make_oracle_fmo.py mini      # ~2 min on one core
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
    config = sys.argv[1] if len(sys.argv) > 1 else "mini"
    ph = phantom.make(config, 0)
    t0 = time.perf_counter()
    res = orc.fmo(ph, method="newton", tol=1e-10)
    out = {"written_by": "tests/golden/make_oracle_fmo.py (oracle/ only)", "config": config, "seed": 0,
           "n_vox": int(ph.n_vox), "n_bl": int(ph.n_bl), "nnz": int(ph.nnz), "method": "projected Newton on dense D^T",
           "tol": 1e-10, "objective": res.objective, "kkt_residual": res.kkt, "n_iter": res.n_iter,
           "n_positive": int((res.y > 0).sum()), "oracle_seconds_one_core": round(time.perf_counter() - t0, 1)}
    path = os.path.join(HERE, f"oracle_fmo_{config}.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print(path, out["objective"], out["oracle_seconds_one_core"])


if __name__ == "__main__":
    main()
