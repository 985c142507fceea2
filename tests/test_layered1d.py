"""Self-checks of the semi-analytic layered-earth solution (tests/layered1d.py) that the oracle's layered-model pin is
held against: it must stand on something other than the oracle."""
import numpy as np

from helpers import wholespace_dipole
from layered1d import layered_hed, layered_hed_exy

REC = np.array([[500.0, 0, 300.0], [0, 500.0, 300.0], [400.0, 300.0, 320.0], [-300.0, 700.0, 200.0], [900.0, -200.0, 260.0]])


def test_hankel_form_of_the_primary_field_is_the_closed_form():
    """The two transmission-line amplitudes (i w mu / 2g for TE, -g / 2 sigma for TM), the split of the dipole into the
    two modes and the J0 / J2 angular integrals, all at once: integrated numerically, the primary field must be the
    closed-form whole-space dipole (Eq. 1) at in-line, broadside and oblique receivers above and below the source."""
    ref = wholespace_dipole((0, 0, 250.0), REC, 0.5, 1.0)
    got = layered_hed(250.0, REC, 0.5, [1.0], [None], primary="hankel")
    assert np.abs(got[:, :3] - ref[:, :3]).max() < 1e-5 * np.abs(ref[:, :3]).max()          # Ex, Ey, Ez
    assert np.abs(got[:, 3:] - ref[:, 3:]).max() < 1e-5 * np.abs(ref[:, 3:]).max()          # Hx (= 0), Hy, Hz: the z derivatives too
    assert np.abs(ref[[0, 2, 3, 4], 2]).min() > 0 and np.abs(ref[1:, 5]).min() > 0            # Ez (x != 0) and Hz (y != 0) take part


def test_reflection_machinery():
    """Interfaces without contrast reflect nothing; splitting a layer changes nothing; exchanging source and receiver depth
    (reciprocity of a horizontal dipole pair in one layer) changes nothing; the air matters; on a near-perfect conductor the
    tangential field vanishes."""
    ref = wholespace_dipole((0, 0, 250.0), REC, 0.5, 1.0)[:, :2]
    assert np.abs(layered_hed_exy(250.0, REC, 0.5, [1.0, 1.0, 1.0], [None, 0.0, 350.0]) - ref).max() < 1e-12 * np.abs(ref).max()
    a = layered_hed_exy(250.0, REC, 0.5, [0.0, 3.2, 1.0, 0.05, 1.0], [None, 0.0, 350.0, 900.0, 1000.0])
    b = layered_hed_exy(250.0, REC, 0.5, [0.0, 3.2, 1.0, 1.0, 0.05, 1.0], [None, 0.0, 350.0, 600.0, 900.0, 1000.0])
    assert np.abs(a - b).max() < 1e-10 * np.abs(a).max()
    r1 = layered_hed_exy(250.0, np.array([[600.0, 200.0, 320.0]]), 0.5, [0.0, 3.2, 1.0], [None, 0.0, 350.0])
    r2 = layered_hed_exy(320.0, np.array([[-600.0, -200.0, 250.0]]), 0.5, [0.0, 3.2, 1.0], [None, 0.0, 350.0])
    assert np.abs(r1 - r2).max() < 1e-10 * np.abs(r1).max()
    c = layered_hed_exy(250.0, REC, 0.5, [3.2, 3.2, 1.0, 0.05, 1.0], [None, 0.0, 350.0, 900.0, 1000.0])
    assert np.abs(a - c).max() > 0.1 * np.abs(a).max()
    s = layered_hed_exy(250.0, np.array([[400.0, 100.0, 350.0]]), 0.5, [1.0, 1e9], [None, 350.0])
    assert np.abs(s).max() < 1e-3 * np.abs(wholespace_dipole((0, 0, 250.0), [[400.0, 100.0, 350.0]], 0.5, 1.0)[0, :2]).max()


def test_vti_reduces_to_the_isotropic_solution_and_stretches_the_tm_mode():
    """sigma_v = sigma_h is the isotropic solution; and the textbook property of a uniaxial medium: its TM part is the
    isotropic TM part of a medium of conductivity sigma_v with the vertical axis stretched by lambda = sqrt(sigma_h / sigma_v)
    (here through Ez, which only the TM mode feeds: Ez_vti(sigma_h, sigma_v; x, z) = Ez_iso(sigma_v; x, lambda z))."""
    lay = ([0.0, 3.2, 1.0, 0.2, 1.0], [None, 0.0, 400.0, 800.0, 900.0])
    rec = REC.copy()
    rec[:, 2] = [300.0, 300.0, 320.0, 200.0, 260.0]
    a = layered_hed(350.0, rec, 0.75, *lay)
    b = layered_hed(350.0, rec, 0.75, *lay, sigma_v=lay[0])
    assert np.abs(a - b).max() < 1e-9 * np.abs(a).max()
    lam = np.sqrt(1.0 / 0.4)
    r1 = np.array([[400.0, 0.0, 100.0], [700.0, 0.0, 160.0], [1000.0, 0.0, 60.0]])
    r2 = r1 * np.array([1.0, 1.0, lam])
    vti = layered_hed(0.0, r1, 1.0, [1.0], [None], sigma_v=[0.4])[:, 2]
    iso = layered_hed(0.0, r2, 1.0, [0.4], [None], primary="hankel")[:, 2]
    assert np.abs(vti / iso - 1).max() < 1e-4

