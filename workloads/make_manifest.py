"""Write workloads/MANIFEST.json: SHA-256 of every generated array of the five configs (numpy's Generator streams
are not guaranteed bit-stable across versions; tests/test_workloads.py fails loudly on a mismatch)."""
import json
import os

import numpy as np

from workloads import generators as gen

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    out = {"numpy": np.__version__, "configs": {}}
    for k in range(5):
        w = gen.make_config(k)
        out["configs"][str(k)] = dict(name=w.name, **w.digest())
    with open(os.path.join(HERE, "MANIFEST.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out, indent=1))


if __name__ == "__main__":
    main()
