#!/usr/bin/env python
"""Writes the stored expected values under tests/golden/ for the full-size BASELINE.json configs.

Calls ONLY oracle/ (and the seeded input generators, which hold none of the method's arithmetic): no value
in these files comes from the CUDA path.  The oracle runs in sparse-DFT mode (accumulators only on the
receiver stencils and the check set: pointwise identical values, see test_convergence_rule).

    python tests/golden/make_goldens.py cfg2            # ~15 min on 8 cores
    python tests/golden/make_goldens.py cfg3 0 100        # configs[2] with aux_dx = 100 m, to convergence: ~50 min
    python tests/golden/make_goldens.py cfg3 0 0          # configs[2] as it ships (auxiliary plane at 25 m), to convergence: 2.4 h
    python tests/golden/make_goldens.py cfg4 300 100      # configs[3] with aux_dx = 100 m, 300 fixed steps: ~50 min
    python tests/golden/make_goldens.py cfg4s 1000 0 fields 500   # configs[3] on its default auxiliary plane (3125 x 3125,
                                                          # what bench.py times) with source and receivers 150 m below the
                                                          # surface and a 20 Hz wavelet (workloads.cfg4s), 1000 fixed
                                                          # steps, field planes: 92 min on 8 cores

Output: tests/golden/<name>_converged[_aux<dx>].json or <name>_<n>steps[_aux<dx>].json with the inputs' SHA-256, nsteps, delta and the complex receivers.
With `fields` also <name>_<n>steps[_aux<dx>]_fields.npz at every listed checkpoint and at the last step: the six time-domain
fields (float32 roundings of the oracle's fp64 values) on whole z planes -- the ghost plane above the surface that the
air-water boundary writes, the surface plane, the plane below it, the plane nearest the seabed -- and on the x-z slice
through the source, the L2 norm of every z plane of every field (fp64), and the partial Green's functions at the receivers.
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


def save_fields(g, w, name, nsteps, aux_dx, t0):
    """field planes + per-plane norms + receivers of the run in progress (oracle values only)"""
    info = g.info()
    out, ns = g.run_end()
    assert int(ns[0]) == nsteps
    k0 = info["k0"]
    z = g.coords(2)
    ksea = int(np.argmin(np.abs(z[:info["N3"]] - 1000.0)))
    y = g.coords(1)
    jsrc = int(np.argmin(np.abs(y[:info["N2"]] - w["sources"][0][0][1])))
    planes = [k0 - 1, k0, k0 + 1, ksea]
    res = {"planes_k": np.array(planes), "slice_j": np.array(jsrc), "nsteps": np.array(nsteps), "dt": np.array(info["dt"]),
           "dims": np.array([info["N3"], info["N2"], info["N1"]]), "aux": np.array([info["aux_M1"], info["aux_M2"]]),
           "receivers": out[0], "sha256": np.array(input_hash(w)), "seconds": np.array(time.time() - t0),
           "written_by": np.array("tests/golden/make_goldens.py %s (oracle only)" % " ".join(sys.argv[1:]))}
    for c in ("E1", "E2", "E3", "H1", "H2", "H3"):
        f = g.get(c)
        res["norm_" + c] = np.sqrt((f * f).sum(axis=(1, 2)))
        res["planes_" + c] = f[planes].astype(np.float32)
        res["slice_" + c] = f[:, jsrc, :].astype(np.float32)
    suffix = "_%dsteps" % nsteps + ("_aux%g" % aux_dx if aux_dx else "") + "_fields.npz"
    np.savez_compressed(os.path.join(HERE, name + suffix), **res)
    print("wrote", name + suffix, flush=True)


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
        if "fmax" in w["run"]:
            opts["fmax"] = w["run"]["fmax"]
    fields = len(sys.argv) > 4 and sys.argv[4] == "fields"
    marks = sorted(int(v) for v in sys.argv[5].split(",")) if len(sys.argv) > 5 else []
    t = time.time()
    g.run_begin(w["sources"][:1], w["freqs"], w["receivers"], opts)
    done, ns = False, [0]
    while not done:
        ns, done = g.run_steps(100)
        print("steps", int(ns[0]), "delta", g.get("DELTA"), "elapsed %.0f s" % (time.time() - t), flush=True)
        if fields and (int(ns[0]) in marks or done):
            save_fields(g, w, name, int(ns[0]), aux_dx, t)
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
