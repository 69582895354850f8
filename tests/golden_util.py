"""Load tests/golden/worked_examples.json into numpy tables (column order as listed in the fixture)."""
import json
import os

import numpy as np

_DT = {"i8": np.int8, "i32": np.int32, "i64": np.int64}
_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "worked_examples.json")


def load():
    with open(_PATH) as f:
        return json.load(f)


def table(colspec, rows):
    """-> dict name -> array, in fixture order."""
    out = {}
    for i, spec in enumerate(colspec):
        name, dt = spec.split(":")
        out[name] = np.array([r[i] for r in rows], dtype=_DT[dt])
    return out
