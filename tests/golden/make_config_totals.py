#!/usr/bin/env python
"""Writes tests/golden/config_totals.json: for every BASELINE.json configuration the number of
(query, primitive) pairs the ORACLE finds -- `sure` (outside the 1e-6 tolerance band) and `band`
(inside it).  Calls only oracle/ and the seeded generators; nothing here touches the CUDA path.
A correct result has sure <= total <= sure + band.

    python tests/golden/make_config_totals.py            # ~10 minutes on 8 cores
"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_2507_23700_b200 import datagen as dg  # noqa: E402


def main():
    oracle.build()
    out = {}
    for name in ("C1", "C2", "C3", "C4", "C5"):
        cfg = dg.config(name, 1.0)
        prims, pk = cfg["prims"], cfg["pkind"]
        grid = oracle.Grid(prims, pk, oracle.default_cell(prims, pk, "spatial", cfg["r"] if cfg["r"] else None))
        sure = band = 0
        for a in range(0, cfg["nq"], 1_000_000):
            off, _, bnd = oracle.spatial(prims, pk, cfg["queries"][a:a + 1_000_000], cfg["qkind"], grid)
            b = int(np.asarray(bnd, dtype=np.int64).sum())
            band += b
            sure += int(off[-1]) - b
        out[name] = dict(sure=sure, band=band, n=cfg["n"], nq=cfg["nq"])
        print(name, out[name], flush=True)
        del grid
    with open(os.path.join(HERE, "config_totals.json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
