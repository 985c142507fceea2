"""CPU checks of the product's C-ABI library: it loads, exports every symbol include/emm.h declares, and
its host-side pre-computation (grid generator, FD weights, padded grid, coefficient tables) agrees with
the independently written oracle.  No compute call is made (no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2304_00233_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def emm():
    from paper_2304_00233_b200 import emm as m
    m.build()
    return m


def test_library_exports_every_declared_symbol(emm):
    hdr = open(os.path.join(ROOT, "include", "emm.h")).read()
    declared = set(re.findall(r"\b(emm_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(emm.SYMBOLS), declared ^ set(emm.SYMBOLS)
    L = emm.lib()
    for s in declared:
        assert hasattr(L, s), s


def test_oracle_and_product_share_no_symbols_or_sources(emm, oracle):
    """independence: different symbol prefixes, and neither source tree includes the other's files"""
    for root, pat in ((os.path.join(ROOT, "oracle"), r"paper_2304_00233_b200|emm\.h|emm_internal|emm_kernels|libemm_b200"),
                      (os.path.join(ROOT, "paper_2304_00233_b200"), r"oracle|emmo_")):
        for dp, _, files in os.walk(root):
            for f in files:
                if f.endswith((".c", ".h", ".cu", ".cuh", ".py")) and f != "workloads.py":
                    for line in open(os.path.join(dp, f)):
                        if re.match(r"\s*(#\s*include|import|from)\b", line) or "CDLL" in line or "dlopen" in line:
                            assert not re.search(pat, line), (f, line)


def test_nugrid_and_weights_agree_with_oracle(emm, oracle):
    for n, L, dx in ((28, 1000.0, 20.0), (50, 5000.0, 25.0), (40, 1000.0, 25.0)):
        xa, qa = emm.emm_nugrid(n, L, dx)
        xb, qb = oracle.nugrid(n, L, dx)
        assert abs(qa - qb) < 1e-12 and np.allclose(xa, xb, rtol=1e-12, atol=1e-9)
    rng = np.random.default_rng(3)
    for npts in (2, 4, 6):
        nodes = np.sort(rng.uniform(-50, 50, size=npts))
        a = emm.emm_fd_weights(nodes, 1.7)
        b = oracle.fd_weights(nodes, 1.7)
        assert np.allclose(a[0], b[0], rtol=1e-12, atol=1e-14) and np.allclose(a[1], b[1], rtol=1e-12, atol=1e-14)
    with pytest.raises(emm.EmmError):
        emm.emm_nugrid(10, 100.0, 20.0)


def test_acquisition_geometry_helpers(emm):
    """azimuth/dip columns of the paper's source/receiver files (L632-640), reading [R13]: unit vector, x at (0,0),
    y at azimuth pi/2, z (downward) at dip pi/2; a receiver channel is the projection of the six returned components."""
    assert np.allclose(emm.emm_dipole_direction(0.0, 0.0), [1, 0, 0], atol=1e-15)
    assert np.allclose(emm.emm_dipole_direction(np.pi / 2, 0.0), [0, 1, 0], atol=1e-15)
    assert np.allclose(emm.emm_dipole_direction(0.3, np.pi / 2), [0, 0, 1], atol=1e-15)
    rng = np.random.default_rng(11)
    az, dip = rng.uniform(-np.pi, np.pi, 9), rng.uniform(-np.pi / 2, np.pi / 2, 9)
    d = np.array([emm.emm_dipole_direction(a, b) for a, b in zip(az, dip)])
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-15)
    assert np.allclose(np.arctan2(d[:, 1], d[:, 0]), az, atol=1e-12) and np.allclose(np.arcsin(d[:, 2]), dip, atol=1e-12)
    g6 = rng.normal(size=(9, 6)) + 1j * rng.normal(size=(9, 6))
    ch = emm.emm_receiver_channels(g6, az, dip)
    assert np.allclose(ch[:, 0], np.einsum("qc,qc->q", d, g6[:, :3]), atol=1e-14)
    assert np.allclose(ch[:, 1], np.einsum("qc,qc->q", d, g6[:, 3:]), atol=1e-14)
    # an x-oriented receiver reads Ex and Hx
    assert np.allclose(emm.emm_receiver_channels(g6, 0.0, 0.0), g6[:, [0, 3]], atol=1e-15)
    with pytest.raises(emm.EmmError):
        emm.emm_dipole_direction(float("nan"), 0.0)


def _workloads():
    nug = None
    from oracle import emm_oracle
    nug = emm_oracle.nugrid
    yield W.cfg1(n=16, rd=1, nb=4)
    yield W.cfg1(n=16, rd=3, nb=5)
    yield W.cfg2(nx=20, nz=12, dx=100.0, rd=2, nb=6)
    yield W.cfg3(nug, nx=24, nz=20, rd=2, nb=6, n_water=6, n_rec_side=3)
    yield W.cfg4(nug, nx=24, nz=20, rd=3, nb=6, n_water=6, n_rec_side=3)


def test_padded_grid_and_tables_agree_with_oracle(emm, oracle):
    for w in _workloads():
        ga = emm.Grid(w["x"], w["y"], w["z"], **w["grid"])
        gb = oracle.Grid(w["x"], w["y"], w["z"], **w["grid"])
        ia, ib = ga.info(), gb.info()
        for k in ib:
            if k != "dt":
                assert ia[k] == ib[k], (w["name"], k, ia[k], ib[k])
        assert ia["pitch"] % 32 == 0 and ia["pitch"] >= ia["N1"]
        for axis in range(3):
            assert np.array_equal(ga.coords(axis), gb.coords(axis))
            for plus in (0, 1):
                a, b = ga.fdcoef(axis, plus), gb.fdcoef(axis, plus)
                assert np.allclose(a, b, rtol=1e-11, atol=1e-16), (w["name"], axis, plus)


def test_error_codes_without_device(emm):
    nodes = np.arange(9) * 10.0
    bad = nodes.copy()
    bad[4] = bad[3]
    with pytest.raises(emm.EmmError) as e:
        emm.Grid(bad, nodes, nodes, rd=1, nb=2)
    assert e.value.code == emm.EINVAL
    with pytest.raises(emm.EmmError):
        emm.Grid(nodes, nodes, nodes, rd=0, nb=2)
    g = emm.Grid(nodes, nodes, nodes, rd=1, nb=2)
    sig = np.ones((8, 8, 8), np.float32)
    # no workspace bound: the product path fails loudly instead of falling back to the CPU
    rc = emm.lib().emm_model_set(g._h, sig.ctypes.data_as(C.POINTER(C.c_float)), None)
    assert rc == emm.ECUDA and b"workspace" in emm.lib().emm_last_error()
    rc = emm.lib().emm_run_steps(g._h, 1, None, None)
    assert rc == emm.EINVAL
    # the sensitivity kernel needs a run in progress; the one-launch boundary is planned on the device, not before
    out = np.zeros((8, 8, 8), np.complex128)
    dp = out.ctypes.data_as(C.POINTER(C.c_double))
    assert emm.lib().emm_sensitivity(g._h, 0, 1, 0, dp, dp) == emm.EINVAL and b"no run" in emm.lib().emm_last_error()
    assert g.info()["air_cluster"] == 0
