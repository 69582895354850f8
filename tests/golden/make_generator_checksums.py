"""Writes tests/golden/generator_checksums.json.  Calls ONLY the generator (paper_2606_24647_b200.datagen)."""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from paper_2606_24647_b200 import datagen  # noqa: E402

SCALES = {1: 0.05, 2: 0.001, 3: 0.002, 4: 0.002, 5: 0.0002}


def snapshot():
    out = {}
    for cfg, sc in SCALES.items():
        t = datagen.make_config(cfg, scale=sc)
        out[f"C{cfg}@{sc}"] = {
            f"{tb}.{c}": dict(n=int(a.size), sum_xor_min_max=datagen.checksum(a), head=[int(x) for x in a[:4]],
                              tail=[int(x) for x in a[-4:]])
            for tb, cols in t.items() for c, a in cols.items()}
    return out


if __name__ == "__main__":
    with open(os.path.join(HERE, "generator_checksums.json"), "w") as f:
        json.dump(snapshot(), f, indent=1, sort_keys=True)
