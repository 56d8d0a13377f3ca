"""Writes tests/golden/oracle_regression.json from the ORACLE ONLY (never the CUDA path).

The paper prints no worked numerical example (no E, F, rho or c for any geometry), so there is
no external value to store here; this file is a regression guard that freezes the oracle's
output on configs 0 and 1 once its pins (tests/test_oracle_*.py) are green. A later change of
these numbers must name, in its commit message, the PAPER.md passage or DESIGN.md reading
that justifies it. Run:  python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import gen      # noqa: E402
import oracle   # noqa: E402

out = {}
for k in (0, 1):
    cfg = gen.make_config(k)
    r = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    nb = oracle.neighbors(cfg["pos"], cfg["box"], cfg["rc"] + cfg["skin"])
    out[str(k)] = dict(E=r["E"], F_first3=r["F"][:3].tolist(), F_rms=float(np.sqrt((r["F"] ** 2).sum(1).mean())),
                       virial_trace=float(np.trace(r["virial"])), n_list_edges=int(len(nb)),
                       source="oracle/reann_oracle.c; no value in PAPER.md to cite")
with open(os.path.join(ROOT, "tests", "golden", "oracle_regression.json"), "w") as f:
    json.dump(out, f, indent=1)
print(json.dumps(out, indent=1))
