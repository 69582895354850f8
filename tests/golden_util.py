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


def digest_columns(cols):
    """Digest of result columns (int64 numpy arrays already in key-tuple order): per column the wrapping u64 sum, the
    xor and the SHA-256 of the little-endian bytes. Pure bookkeeping — no arithmetic of the method."""
    import hashlib
    out = []
    for c in cols:
        a = np.ascontiguousarray(c, dtype=np.int64)
        u = a.view(np.uint64)
        out.append(dict(sum=int(np.sum(u, dtype=np.uint64)) if len(u) else 0,
                        xor=int(np.bitwise_xor.reduce(u)) if len(u) else 0,
                        sha256=hashlib.sha256(a.astype("<i8").tobytes()).hexdigest()))
    return out
