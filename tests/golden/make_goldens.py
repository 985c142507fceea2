#!/usr/bin/env python
"""Writes the stored expected values under tests/golden/ for the full-size BASELINE.json configs.

Calls ONLY oracle/ (and the seeded input generators, which hold none of the method's arithmetic): no value
in these files comes from the CUDA path.  The oracle runs in sparse-DFT mode (accumulators only on the
receiver stencils and the check set: pointwise identical values, see test_convergence_rule).

    python tests/golden/make_goldens.py cfg2            # ~15 min on 8 cores
    python tests/golden/make_goldens.py cfg3 0 100        # configs[2] with aux_dx = 100 m, to convergence: ~50 min
    python tests/golden/make_goldens.py cfg4 300 100      # configs[3] with aux_dx = 100 m, 300 fixed steps: ~50 min

Output: tests/golden/<name>_converged[_aux<dx>].json or <name>_<n>steps[_aux<dx>].json with the inputs' SHA-256, nsteps, delta and the complex receivers.
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import emm_oracle as O  # noqa: E402
from paper_2304_00233_b200 import workloads as W  # noqa: E402


def input_hash(w):
    h = hashlib.sha256()
    for k in ("x", "y", "z", "sigma_h", "sigma_v", "freqs", "receivers"):
        v = w.get(k)
        if v is not None:
            h.update(np.ascontiguousarray(v).tobytes())
    h.update(repr(w["sources"]).encode())
    h.update(repr(sorted(w["grid"].items())).encode())
    return h.hexdigest()


def main():
    name = sys.argv[1]
    kw = {}
    fixed = int(sys.argv[2]) if len(sys.argv) > 2 else 0
    aux_dx = float(sys.argv[3]) if len(sys.argv) > 3 else 0.0
    if aux_dx:
        kw["aux_dx"] = aux_dx          # coarser auxiliary plane: the oracle's plain FFT makes the 25 m default take ~10 h on cfg3
    w = W.build(name, O.nugrid, **kw)
    g = O.Grid(w["x"], w["y"], w["z"], **w["grid"])
    g.model_set(w["sigma_h"], w.get("sigma_v"))
    opts = dict(w["run"])
    opts.pop("batched", None)
    opts["sparse_dft"] = 1
    if fixed:
        opts = dict(fixed_steps=fixed, sparse_dft=1)
    t = time.time()
    g.run_begin(w["sources"][:1], w["freqs"], w["receivers"], opts)
    done, ns = False, [0]
    while not done:
        ns, done = g.run_steps(100)
        print("steps", int(ns[0]), "delta", g.get("DELTA"), "elapsed %.0f s" % (time.time() - t), flush=True)
    out, ns = g.run_end()
    res = {"name": name, "sha256": input_hash(w), "info": g.info(), "opts": opts, "nsteps": int(ns[0]),
           "delta": [float(v) for v in g.get("DELTA")], "seconds": time.time() - t,
           "receivers_re": out[0].real.tolist(), "receivers_im": out[0].imag.tolist(),
           "written_by": "tests/golden/make_goldens.py %s (oracle only)" % " ".join(sys.argv[1:])}
    suffix = ("_converged" if not fixed else "_%dsteps" % fixed) + ("_aux%g" % aux_dx if aux_dx else "")
    with open(os.path.join(HERE, name + suffix + ".json"), "w") as f:
        json.dump(res, f)
    print("wrote", name + suffix + ".json", "nsteps", res["nsteps"])


if __name__ == "__main__":
    main()
