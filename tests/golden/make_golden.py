"""Writes the stored expected values under tests/golden/ by calling ONLY the CPU oracle.

    python tests/golden/make_golden.py

config1_oracle_fp64.json: BASELINE.json config 1 (tiny slab, 1e4 photons of 1 MeV, fp64, Philox seed 1):
run statistics, per-volume edep [MeV] and the first 16 history hashes.  These are a
regression pin of the oracle against itself across edits; the independent pins are the closed-form and
brute-force tests in tests/test_oracle_*.py."""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_1209_5235_b200 import workloads as W  # noqa: E402


def main():
    wl = W.config(1)
    og = oracle.OracleGeometry(wl.geometry)
    r = og.transport(wl.source, wl.seed, wl.n, 64, per_photon=True)
    out = {"citation": "BASELINE.json configs[0]; SURVEY.md 8(d) config 1", "n_photons": wl.n, "seed": wl.seed,
           "stats": {k: (int(v) if k.startswith("n_") else float(v)) for k, v in r["stats"].items()},
           "edep": [float(v) for v in r["edep"]], "hash_first16": [int(h) for h in r["hash"][:16]]}
    with open(os.path.join(HERE, "config1_oracle_fp64.json"), "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
