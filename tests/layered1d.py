"""Semi-analytic field of a horizontal electric dipole in a horizontally layered earth (no code shared with oracle/ or
the CUDA path): the reference the layered-model pins of the oracle are held against.

Quasi-static Maxwell equations in the paper's convention (Eq. 1: e^{-i w t}, curl E = i w mu H,
curl H = sigma E + J), unit x-directed point dipole at (0, 0, zs), z positive downward.  In the horizontal wavenumber
domain the field splits into two scalar transmission lines along z (s = unit vector along the wavenumber, t = z x s):

  TE  (E along t):  e'' - g^2 e = -i w mu j_t delta(z - zs),                    g^2 = kappa^2 - i w mu sigma
                    whole space  e = i w mu / (2 g) * j_t * exp(-g |z - zs|);   e, e' continuous: r = (g1 - g2) / (g1 + g2)
  TM  (E along s):  e' = -(g^2 / sigma) h,  h' = -sigma e - j_s delta(z - zs)   (h = H along t, e_z = i kappa h / sigma)
                    whole space  e = -g / (2 sigma) * j_s * exp(-g |z - zs|);   e, h continuous: r = (Y1 - Y2) / (Y1 + Y2),
                    Y = sigma / g (air: Y = 0, r = +1)

With j_s = kx / kappa, j_t = -ky / kappa and Ex = e_s kx / kappa - e_t ky / kappa the angular integral leaves two Hankel
transforms (r, phi = horizontal offset and azimuth of the receiver):

  Ex = 1/(4 pi) int_0^inf [ (G_TM + G_TE) J0(kappa r) - cos(2 phi) (G_TM - G_TE) J2(kappa r) ] kappa d kappa
  Ey = -1/(4 pi) sin(2 phi) int_0^inf (G_TM - G_TE) J2(kappa r) kappa d kappa

The other four components follow from the same two lines (' = d/dz, sigma = conductivity of the layer of the receiver):
H_s = (i / w mu) e_t', H_z = (kappa / w mu) e_t (TE);  h = H_t = -(sigma / g^2) e_s', E_z = (i kappa / sigma) h (TM).  With
Q_TE = (i / w mu) G_TE', Q_TM = -(sigma / g^2) G_TM':

  Hx = 1/(4 pi) sin(2 phi) int (Q_TE + Q_TM) J2 kappa d kappa
  Hy = 1/(4 pi) int [ (Q_TM - Q_TE) J0 - cos(2 phi) (Q_TM + Q_TE) J2 ] kappa d kappa
  Hz = -i sin(phi) / (2 pi w mu) int G_TE J1 kappa^2 d kappa
  Ez = -cos(phi) / (2 pi sigma) int Q_TM J1 kappa^2 d kappa

Vertical transverse isotropy (sigma_v for E_z, sigma = sigma_h for the horizontal E) only enters the TM line:
i kappa h = sigma_v e_z turns its series impedance into kappa^2 / sigma_v - i w mu, so g_TM^2 = (sigma_h / sigma_v) kappa^2 -
i w mu sigma_h, Y = sigma_h / g_TM, whole-space amplitude -g_TM / (2 sigma_h), h = -(sigma_h / g_TM^2) e_s', E_z = i kappa h /
sigma_v; the TE line sees sigma_h only.

G = whole-space amplitude x [primary + reflections from the stacks above and below the source layer].  Source and receiver
sit in the same layer.  The primary part is the closed-form whole-space field (tests/helpers.py); only the reflected part
-- smooth, decaying like exp(-kappa x distance to the nearest image) -- is integrated numerically (composite Simpson on
a grid fine against both the decay and the Bessel oscillation)."""
import numpy as np
from scipy.special import jv

from helpers import MU0, wholespace_dipole


def _gamma(kappa, w, sh, sv, mode):
    lam2 = 1.0 if (mode == "TE" or sh == 0.0) else sh / sv
    return np.sqrt(lam2 * kappa ** 2 - 1j * w * MU0 * sh + 0j)


def _stack_reflection(kappa, w, sig, sigv, thick, mode):
    """Generalised reflection coefficient seen from a layer looking into the stack sig[0], sig[1], ... (sig[0] = the
    layer itself, thick[i] = thickness of sig[i], the last one a half-space), for the transmission-line voltage
    (tangential E) of the mode."""
    g = [_gamma(kappa, w, s, v, mode) for s, v in zip(sig, sigv)]
    Y = [gi if mode == "TE" else (s / gi) for s, gi in zip(sig, g)]
    R = np.zeros_like(kappa, dtype=complex)
    for i in range(len(sig) - 2, -1, -1):
        r = (Y[i] - Y[i + 1]) / (Y[i] + Y[i + 1])
        if i + 1 < len(sig) - 1:
            p = R * np.exp(-2 * g[i + 1] * thick[i + 1])
            R = (r + p) / (1 + r * p)
        else:
            R = r
    return R


def layered_hed(zs, rec, f, sigma, z_top, primary="closed form", sigma_v=None):
    """Ex, Ey, Ez, Hx, Hy, Hz of a unit x-directed electric dipole at (0, 0, zs) at the receivers rec[n] = (x, y, z).
    sigma[l] = conductivity of layer l (0 = air), z_top[l] = its upper boundary (z_top[0] = -inf for the top half-space,
    given as None); the last layer is a half-space.  Source and receivers must lie in the same (conductive) layer.
    sigma_v[l]: vertical conductivity of layer l (None: isotropic); with anisotropy in the source layer the primary field has
    no closed form here and is integrated numerically (primary = "hankel", needs z != zs).
    primary = "hankel" integrates the primary field numerically as well (needs z != zs): the self-check of the
    amplitudes and of the angular integrals against the closed form."""
    sigma = [float(s) for s in sigma]
    sigv = [float(s) for s in (sigma if sigma_v is None else sigma_v)]
    rec = np.asarray(rec, dtype=float)
    w = 2 * np.pi * f
    tops = [(-np.inf if t is None else float(t)) for t in z_top]
    bots = tops[1:] + [np.inf]
    fits = [l for l in range(len(sigma)) if tops[l] <= zs <= bots[l] and np.all((rec[:, 2] >= tops[l]) & (rec[:, 2] <= bots[l]))]
    assert fits, "source and receivers must lie in one layer"
    L = fits[0]
    zt, zb = tops[L], bots[L]
    sL, vL = sigma[L], sigv[L]
    if vL != sL:
        primary = "hankel"
    up_sigv = [sigv[l] for l in range(L, -1, -1)]
    dn_sigv = [sigv[l] for l in range(L, len(sigma))]
    up_sig = [sigma[l] for l in range(L, -1, -1)]
    up_thk = [bots[l] - tops[l] for l in range(L, -1, -1)]
    dn_sig = [sigma[l] for l in range(L, len(sigma))]
    dn_thk = [bots[l] - tops[l] for l in range(L, len(sigma))]
    out = np.zeros((len(rec), 6), dtype=complex)
    prim = wholespace_dipole((0.0, 0.0, zs), rec, f, sL)
    for n, (x, y, z) in enumerate(rec):
        r, phi = np.hypot(x, y), np.arctan2(y, x)
        # distance to the nearest image sets the decay of the reflected part, the offset its oscillation
        dimg = min((zs - zt) + (z - zt) if np.isfinite(zt) else np.inf, (zb - zs) + (zb - z) if np.isfinite(zb) else np.inf)
        if primary == "hankel":
            dimg = min(dimg, abs(z - zs))
        kmax = 50.0 / max(dimg, 1.0)
        dk = min(2 * np.pi / max(r, 1.0) / 40.0, kmax / 4000.0, 1.0 / max(dimg, 1.0) / 20.0)
        nk = int(np.ceil(kmax / dk)) // 2 * 2 + 2
        kap = np.linspace(0.0, kmax, nk + 1)
        kap[0] = 1e-12
        G, dG, gm = {}, {}, {}
        for mode in ("TE", "TM"):
            g = gm[mode] = _gamma(kap, w, sL, vL, mode)
            Ru = _stack_reflection(kap, w, up_sig, up_sigv, up_thk, mode) if len(up_sig) > 1 else 0.0 * kap
            Rd = _stack_reflection(kap, w, dn_sig, dn_sigv, dn_thk, mode) if len(dn_sig) > 1 else 0.0 * kap
            eu = np.exp(-g * (zs - zt)) if np.isfinite(zt) else 0.0 * kap      # source -> top
            ed = np.exp(-g * (zb - zs)) if np.isfinite(zb) else 0.0 * kap      # source -> bottom
            d = zb - zt
            ee = np.exp(-g * d) if np.isfinite(d) else 0.0 * kap
            den = 1 - Ru * Rd * ee * ee
            A = Ru * (eu + Rd * ee * ed) / den                                   # down-going wave leaving the top
            B = Rd * (ed + Ru * ee * eu) / den                                   # up-going wave leaving the bottom
            dn = A * np.exp(-g * (z - zt)) if np.isfinite(zt) else 0.0 * kap
            up = B * np.exp(-g * (zb - z)) if np.isfinite(zb) else 0.0 * kap
            F, dF = dn + up, g * (up - dn)
            if primary == "hankel":
                P = np.exp(-g * abs(z - zs))
                F, dF = F + P, dF - g * np.sign(z - zs) * P
            amp = 1j * w * MU0 / (2 * g) if mode == "TE" else -g / (2 * sL)
            G[mode], dG[mode] = amp * F, amp * dF
        QTE, QTM = 1j / (w * MU0) * dG["TE"], -(sL / gm["TM"] ** 2) * dG["TM"]
        wts = np.ones(nk + 1)
        wts[1:-1:2] = 4.0
        wts[2:-1:2] = 2.0
        wts *= (kap[-1] - 0.0) / nk / 3.0
        J0, J1, J2 = jv(0, kap * r), jv(1, kap * r), jv(2, kap * r)

        def hank(fk, J, power=1):
            return np.sum(wts * fk * J * kap ** power)

        p0 = prim[n] if primary != "hankel" else np.zeros(6)
        c2, s2 = np.cos(2 * phi), np.sin(2 * phi)
        out[n, 0] = p0[0] + (hank(G["TM"] + G["TE"], J0) - c2 * hank(G["TM"] - G["TE"], J2)) / (4 * np.pi)
        out[n, 1] = p0[1] - s2 * hank(G["TM"] - G["TE"], J2) / (4 * np.pi)
        out[n, 2] = p0[2] - np.cos(phi) / (2 * np.pi * vL) * hank(QTM, J1, 2)
        out[n, 3] = p0[3] + s2 * hank(QTE + QTM, J2) / (4 * np.pi)
        out[n, 4] = p0[4] + (hank(QTM - QTE, J0) - c2 * hank(QTM + QTE, J2)) / (4 * np.pi)
        out[n, 5] = p0[5] - 1j * np.sin(phi) / (2 * np.pi * w * MU0) * hank(G["TE"], J1, 2)
    return out


def layered_hed_exy(zs, rec, f, sigma, z_top, primary="closed form", sigma_v=None):
    """Ex, Ey only (see layered_hed)."""
    return layered_hed(zs, rec, f, sigma, z_top, primary, sigma_v)[:, :2]
