"""Writes tests/golden/pattern_counts.json from the CPU oracle only (never the CUDA path)."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import workloads  # noqa: E402

out = {"source": "oracle.knn(grid) + oracle.pattern; survey probe (SURVEY.md 8(c) Pins) gives the same counts"}
for name in ("patch", "cantilever"):
    w = workloads.config(name)
    s = oracle.knn(w.nodes, w.qpts, w.k, "grid")
    rp, ci = oracle.pattern(s, w.N)
    out[name] = {"blocks": int(rp[-1] // 9), "nnz": int(rp[-1])}
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "pattern_counts.json"), "w") as fh:
    json.dump(out, fh, indent=1)
print(out)
