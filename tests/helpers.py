"""Closed forms and small utilities used by the pins (no code shared with oracle/ or the CUDA path)."""
import numpy as np

MU0 = 4e-7 * np.pi


def skin_depth(f, sigma):
    return np.sqrt(2.0 / (2 * np.pi * f * MU0 * sigma))


def wholespace_dipole(src, rec, f, sigma, p=(1.0, 0.0, 0.0)):
    """Frequency-domain E,H of a unit electric dipole p in a homogeneous whole space, e^{-i w t}
    convention (Eq. 1): E = (1/sigma)(k^2 + grad grad) g p, H = grad g x p,
    g = e^{ikr}/(4 pi r), k^2 = i w mu sigma.  Returns [nrec][6] (Ex,Ey,Ez,Hx,Hy,Hz)."""
    p = np.asarray(p, dtype=float)
    w = 2 * np.pi * f
    k = np.sqrt(1j * w * MU0 * sigma)
    d = np.asarray(rec, dtype=float) - np.asarray(src, dtype=float)
    r = np.linalg.norm(d, axis=1)
    rh = d / r[:, None]
    g = np.exp(1j * k * r) / (4 * np.pi * r)
    kr = k * r
    pr = rh @ p
    # (k^2 + grad grad) g p = g/r^2 [ (k^2 r^2 + i k r - 1) p + (-k^2 r^2 - 3 i k r + 3) rh (rh.p) ]
    E = (g / r ** 2)[:, None] * ((kr ** 2 + 1j * kr - 1)[:, None] * p[None, :]
                                 + ((-kr ** 2 - 3j * kr + 3) * pr)[:, None] * rh) / sigma
    H = ((1j * k - 1 / r) * g)[:, None] * np.cross(rh, p[None, :])
    return np.concatenate([E, H], axis=1)


def make_grid(mod, w, **over):
    """Build a Grid of binding module `mod` (oracle or product) from a workload dict."""
    opts = dict(w["grid"])
    opts.update(over)
    g = mod.Grid(w["x"], w["y"], w["z"], **opts)
    g.model_set(w["sigma_h"], w.get("sigma_v"))
    return g
