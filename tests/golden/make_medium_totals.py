"""Writes tests/golden/medium_totals.json: the totals of the COMPLETE `medium` composition (BASELINE.json configs[1])
as the CPU oracle computes them.  Calls only oracle/ and the seeded input generators; nothing from the CUDA path.

    python tests/golden/make_medium_totals.py        (about 5 minutes on one core, ~10 GB of host memory)

tests/test_gpu_fullsize.py::test_medium_complete_properties_and_samples reads the file.
"""
from __future__ import annotations

import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle                                            # noqa: E402
from paper_1805_06383_b200 import workloads              # noqa: E402  (generators only: no method arithmetic)


def main() -> None:
    m1, m2 = workloads.make_config("medium")
    r = oracle.compose(m1, m2, keep_arcs=False)
    out = {
        "config": "medium", "seeds": list(workloads.CONFIGS["medium"]["seeds"]),
        "written_by": "tests/golden/make_medium_totals.py (oracle.compose, serial C++, fp64, Algorithm 1 PAPER.md:106-131)",
        "n_states": r.n_states, "n_arcs": r.n_arcs, "n_raw_arcs": r.n_raw_arcs, "n_levels": r.n_levels,
        "truncated": r.truncated, "n_expanded": r.n_expanded,
        "level_raw": [int(x) for x in r.level_raw], "level_size": [int(x) for x in r.level_size],
        "oracle_seconds": round(r.seconds, 1),
    }
    with open(os.path.join(HERE, "medium_totals.json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print(json.dumps(out))


if __name__ == "__main__":
    main()
