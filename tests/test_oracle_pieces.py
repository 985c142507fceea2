"""Pins of the oracle's building blocks against what the paper and the mathematics fix.
All CPU (`-m "not gpu"`).  None of these retypes an oracle formula: each compares with a closed
form, a textbook value, an independent library routine or an invariant."""
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy.optimize import brentq

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden_fornberg():
    tab = {}
    for line in open(os.path.join(HERE, "golden", "fornberg_staggered.txt")):
        if line.startswith("#") or not line.strip():
            continue
        parts = line.split()
        tab[int(parts[0])] = [float(Fraction(p)) for p in parts[1:]]
    return tab


# ---- FD / interpolation weights (Eq. 9-14) -------------------------------------
@pytest.mark.parametrize("r", [1, 2, 3])
def test_fd_weights_polynomial_exactness(oracle, r):
    """north_star pin (b): 2r non-equidistant nodes are exact for x^p, p <= 2r-1 (L200), not for p = 2r."""
    rng = np.random.default_rng(10 + r)
    for _ in range(20):
        nodes = np.cumsum(rng.uniform(0.5, 2.0, size=2 * r)) + rng.uniform(-5, 5)
        x0 = rng.uniform(nodes[r - 1], nodes[r])
        wi, wd = oracle.fd_weights(nodes, x0)
        scale = np.abs(nodes - x0).max()
        for p in range(2 * r):
            f = ((nodes - x0) / scale) ** p            # monomials about x0: f(x0)=[p==0], f'(x0)=[p==1]/scale
            assert abs(wi @ f - (1.0 if p == 0 else 0.0)) < 1e-11
            assert abs(wd @ f - ((1.0 / scale) if p == 1 else 0.0)) < 1e-11 / scale * 10
        f = ((nodes - x0) / scale) ** (2 * r)
        assert abs(wd @ f) * scale > 1e-6 or abs(wi @ f) > 1e-6


@pytest.mark.parametrize("r", [1, 2, 3])
def test_fd_weights_uniform_limit_is_fornberg(oracle, r):
    """Eq. 33 (L853-858): on a uniform grid c_i^+ = -c_{-i+1}^+ = c_i/dx, c_i = textbook staggered weights."""
    c = _golden_fornberg()[r]
    dx = 37.5
    nodes = (np.arange(2 * r) - r + 0.5) * dx           # half-offsets -(r-1/2) .. +(r-1/2)
    _, wd = oracle.fd_weights(nodes, 0.0)
    for i in range(1, r + 1):
        assert abs(wd[r - 1 + i] - c[i - 1] / dx) < 1e-14 / dx * 10
        assert abs(wd[r - i] + c[i - 1] / dx) < 1e-14 / dx * 10


def test_fd_weights_match_lagrange_closed_form(oracle):
    """Independent construction: derivative of the Lagrange basis (Bjorck-Pereyra equivalence)."""
    rng = np.random.default_rng(5)
    for n in (2, 4, 6):
        nodes = np.sort(rng.uniform(-3, 3, size=n))
        x0 = rng.uniform(-1, 1)
        wi, wd = oracle.fd_weights(nodes, x0)
        for j in range(n):
            others = np.delete(nodes, j)
            den = np.prod(nodes[j] - others)
            li = np.prod(x0 - others) / den
            dli = sum(np.prod(np.delete(x0 - others, m)) for m in range(n - 1)) / den
            assert abs(wi[j] - li) < 1e-11 * max(1, abs(li))
            assert abs(wd[j] - dli) < 1e-10 * max(1, abs(dli))


@pytest.mark.parametrize("r", [1, 2, 3])
def test_grid_tables_index_convention(oracle, r):
    """D- at x_i acts on half nodes i-r .. i+r-1 (listing L212-236), D+ at xh_i on nodes i-r+1 .. i+r
    (Eq. 13): applied to a cubic/quintic sampled on the padded coordinates they return its derivative."""
    rng = np.random.default_rng(r)
    x = np.concatenate(([0.0], np.cumsum(rng.uniform(20, 40, size=12))))
    y = np.arange(9) * 30.0
    z = np.concatenate(([0.0], np.cumsum(rng.uniform(10, 30, size=10))))
    g = oracle.Grid(x, y, z, rd=r, nb=3, ne=r + 1)
    deg = 2 * r - 1
    for axis in range(3):
        xn = g.coords(axis)
        N = len(xn) - 1
        xh = 0.5 * (xn[:-1] + xn[1:])
        L = xn[-1] - xn[0]
        poly = lambda t: ((t - xn[0]) / L) ** deg + 0.3 * ((t - xn[0]) / L)
        dpoly = lambda t: deg * ((t - xn[0]) / L) ** (deg - 1) / L + 0.3 / L
        cm, cp = g.fdcoef(axis, 0), g.fdcoef(axis, 1)
        for i in range(r, N - r):
            dm = sum(cm[i, m] * poly(xh[i - r + m]) for m in range(2 * r))
            dp = sum(cp[i, m] * poly(xn[i - r + 1 + m]) for m in range(2 * r))
            assert abs(dm - dpoly(xn[i])) < 1e-10 / L
            assert abs(dp - dpoly(xh[i])) < 1e-10 / L
        assert np.all(cm[:r] == 0) and np.all(cm[N - r:] == 0)     # outer r layers never updated (L563)


# ---- grid generator (Eq. 27-29) -------------------------------------------------------
@pytest.mark.parametrize("n,L,dx", [(28, 1000.0, 20.0), (50, 5000.0, 25.0), (10, 400.0, 39.0)])
def test_nugrid_solves_eq27(oracle, n, L, dx):
    x, q = oracle.nugrid(n, L, dx)
    assert q > 1
    assert abs(dx * (q ** n - 1) / (q - 1) - L) < 1e-10 * L                  # Eq. 27
    qb = brentq(lambda t: dx * (t ** n - 1) / (t - 1) - L, 1 + 1e-9, 3.0, xtol=1e-15)
    assert abs(q - qb) < 1e-10
    assert x[0] == 0 and abs(x[-1] - L) < 1e-9 * L
    w = np.diff(x)
    assert abs(w[0] - dx) < 1e-9 * dx and np.allclose(w[1:] / w[:-1], q, rtol=1e-9)


def test_nugrid_uniform_case_returns_q1(oracle):
    x, q = oracle.nugrid(40, 1000.0, 25.0)                                     # listing L430
    assert q == 1.0 and np.allclose(x, np.arange(41) * 25.0, rtol=0, atol=1e-12)


def test_nugrid_rejects_impossible(oracle):
    with pytest.raises(oracle.OracleError):
        oracle.nugrid(10, 100.0, 20.0)


# ---- FFT used by the air-wave boundary (L282-288; library-primitive step) -------------------------
@pytest.mark.parametrize("n1,n2", [(8, 6), (21, 10), (13, 7), (36, 30), (1, 5), (50, 49)])
def test_fft2_matches_numpy(oracle, n1, n2):
    rng = np.random.default_rng(n1 * 100 + n2)
    a = rng.standard_normal((n2, n1)) + 1j * rng.standard_normal((n2, n1))
    F = oracle.fft2(a, -1)
    assert np.allclose(F, np.fft.fft2(a) / (n1 * n2), rtol=0, atol=1e-13 * np.abs(a).max() * 10)
    back = oracle.fft2(F, +1)
    assert np.allclose(back, a, rtol=0, atol=1e-12)


def test_fft2_convention_plane_wave(oracle):
    """f(x) = sum F(k) e^{+ikx} (Eq. 32): a single e^{+i(2 pi 3 x/n1 + 2 pi 2 y/n2)} lands in bin (2,3)."""
    n1, n2 = 12, 10
    i, j = np.meshgrid(np.arange(n1), np.arange(n2), indexing="xy")
    a = np.exp(2j * np.pi * (3 * i / n1 + 2 * j / n2))
    F = oracle.fft2(a, -1)
    ref = np.zeros_like(F)
    ref[2, 3] = 1.0
    assert np.allclose(F, ref, atol=1e-13)


# ---- padding and time step (L305-312, Eq. 15-16) --------------------------------------------
def test_padding_and_box(oracle):
    nodes = np.arange(21) * 50.0
    g = oracle.Grid(nodes, nodes, nodes, rd=2, nb=5, ne=-1)
    i = g.info()
    assert (i["N1"], i["N2"], i["N3"]) == (20 + 2 * 12,) * 3               # n + 2*(nb+ne), ne = rd+5 (L308-311, L686)
    assert (i["box_lo1"], i["box_hi1"]) == (5, 44 - 1 - 5)                 # DFT excludes CPML (L365-370)
    xn = g.coords(0)
    assert np.allclose(np.diff(xn), 50.0) and abs(xn[12] - 0.0) < 1e-9
    ga = oracle.Grid(nodes, nodes, nodes, rd=2, nb=5, ne=-1, top=oracle.TOP_AIR)
    ia = ga.info()
    assert ia["k0"] == 2 and ia["N3"] == 20 + 2 + 12 and ia["box_lo3"] == 2
    assert ia["N1"] == 45 and ia["aux_M1"] == 45                             # 44 -> next 7-smooth size


@pytest.mark.parametrize("r,sumc", [(1, 2.0), (2, 2.0 * (9 / 8 + 1 / 24)), (3, 2.0 * (75 / 64 + 25 / 384 + 3 / 640))])
def test_dt_uniform_limit(oracle, r, sumc):
    """Eq. 15-16 with uniform spacing d: eta = v sqrt(3) sum|c| / (2 d); r=1 gives the textbook d/(v sqrt 3)."""
    d, sigma, cfl = 80.0, 0.7, 0.9
    nodes = np.arange(13) * d
    g = oracle.Grid(nodes, nodes, nodes, rd=r, nb=4, ne=-1, cfl=cfl)
    g.model_set(np.full((12, 12, 12), sigma, np.float32))
    sigma32 = float(np.float32(sigma))
    v = 1.0 / np.sqrt(4e-7 * np.pi * sigma32 / (2 * 2 * np.pi * 1.0))
    dt_ref = cfl / (0.5 * v * np.sqrt(3.0) * sumc / d)
    assert abs(g.info()["dt"] / dt_ref - 1) < 1e-12
    if r == 1:
        assert abs(g.info()["dt"] / (cfl * d / (v * np.sqrt(3))) - 1) < 1e-12


def test_effective_medium_at_interface(oracle):
    """[R3]/Eq. 26: tangential components on a horizontal interface see the arithmetic mean of the
    two layers; Ez (normal, inside a cell) sees its own cell; with top=AIR the surface plane sees sigma/2."""
    nodes = np.arange(11) * 100.0
    sig = np.ones((10, 10, 10), np.float32)
    sig[:4] = 3.0                                       # interface on the node plane z = 400
    g = oracle.Grid(nodes, nodes, nodes, rd=1, nb=2, ne=3, top=oracle.TOP_AIR)
    g.model_set(sig)
    i = g.info()
    dt, w0 = i["dt"], 2 * np.pi
    lo = (i["lo3"], i["lo2"], i["lo1"])
    s11 = 2 * w0 * dt / g.get("CE1")[lo[0] + 4, lo[1] + 5, lo[2] + 5]
    s33a = 2 * w0 * dt / g.get("CE3")[lo[0] + 3, lo[1] + 5, lo[2] + 5]
    s33b = 2 * w0 * dt / g.get("CE3")[lo[0] + 4, lo[1] + 5, lo[2] + 5]
    s_surf = 2 * w0 * dt / g.get("CE1")[i["k0"], lo[1] + 5, lo[2] + 5]
    assert abs(s11 - 2.0) < 1e-12 and abs(s33a - 3.0) < 1e-12 and abs(s33b - 1.0) < 1e-12
    assert abs(s_surf - 1.5) < 1e-12
    assert np.all(g.get("CE1")[: i["k0"]] == 0)         # ghost planes are never updated


def test_effective_medium_unequal_widths_is_the_dual_face_average(oracle):
    """[R3]/Eq. 26 on a grid whose neighbouring cells have UNEQUAL widths on all three axes (the rule every non-uniform
    config runs through).  The effective conductivity of an E component is the average of sigma over the face of the dual
    cell that its edge pierces (resistors in parallel, L400).  Checked two ways that share nothing with the oracle's
    loop: (i) a hand-computed number on a two-material model -- widths 100 | 300 m across the interface, sigma 1 | 4
    S/m: (1*100 + 4*300)/400 = 3.25, not the 2.5 an unweighted mean gives; (ii) brute force: the mean of the piecewise
    constant sigma sampled on a fine lattice over that dual face, for random cell values, for all three components
    (sigma_v for E3)."""
    x = np.cumsum(np.concatenate(([0.0], [100.0, 300.0, 120.0, 80.0, 260.0, 140.0, 90.0, 200.0])))
    y = np.cumsum(np.concatenate(([0.0], [100.0, 300.0, 70.0, 210.0, 130.0, 90.0, 170.0, 110.0])))
    z = np.cumsum(np.concatenate(([0.0], [50.0, 150.0, 40.0, 120.0, 60.0, 200.0, 80.0, 100.0])))
    n = 8
    w0 = 2 * np.pi

    def effective(sh, sv):
        g = oracle.Grid(x, y, z, rd=1, nb=2, ne=2)
        g.model_set(sh.astype(np.float32), sv.astype(np.float32))
        i = g.info()
        lo = (i["lo3"], i["lo2"], i["lo1"])
        sl = tuple(slice(lo[a], lo[a] + n) for a in range(3))
        return [2 * w0 * i["dt"] / g.get("CE%d" % (c + 1))[sl] for c in range(3)]           # sigma_bar at the model's own nodes

    # (i) vertical interface on the node plane y = y[1]: sigma = 1 for y < 100, 4 beyond; uniform otherwise
    sh = np.ones((n, n, n))
    sh[:, 1:, :] = 4.0
    s11, s22, s33 = effective(sh, sh)
    assert abs(s11[4, 1, 4] - 3.25) < 1e-12              # Ex on the interface: tangential, widths 100 | 300
    assert abs(s33[4, 1, 4] - 3.25) < 1e-12              # Ez on the interface: tangential too
    assert abs(s22[4, 1, 4] - 4.0) < 1e-12               # Ey at yh[1]: inside the second cell
    # the same across z (widths 50 | 150) for the horizontal components, with a different sigma_v that E3 alone must see
    sh = np.ones((n, n, n))
    sh[1:] = 4.0
    sv = np.full((n, n, n), 7.0)
    s11, s22, s33 = effective(sh, sv)
    assert abs(s11[1, 4, 4] - (1 * 50 + 4 * 150) / 200.0) < 1e-12 and abs(s22[1, 4, 4] - 3.25) < 1e-12
    assert abs(s33[1, 4, 4] - 7.0) < 1e-12

    # (ii) brute force over the dual face, random cells
    rng = np.random.default_rng(26)
    sh = rng.uniform(0.2, 5.0, size=(n, n, n))
    sv = rng.uniform(0.2, 5.0, size=(n, n, n))
    eff = effective(sh, sv)
    nodes = (x, y, z)

    def face_mean(c, idx, model, m=1500):
        """mean of model over the dual face of component c at node idx = (k, j, i), by midpoint sampling on an m x m
        lattice: the component sits at the half node of its own axis (inside cell i) and at nodes of the two others;
        the face spans from the previous to the next half node along those two"""
        pos = {a: idx[2 - a] for a in range(3)}           # node index along each coordinate axis (x = 0, y = 1, z = 2)
        others = [a for a in range(3) if a != c]
        t = (np.arange(m) + 0.5) / m
        cells = {c: np.array([pos[c]])}
        for a in others:
            u, i = nodes[a], pos[a]
            lo_, hi_ = 0.5 * (u[i - 1] + u[i]), 0.5 * (u[i] + u[i + 1])
            cells[a] = np.clip(np.searchsorted(u, lo_ + (hi_ - lo_) * t, side="right") - 1, 0, n - 1)
        return model[np.ix_(cells[2], cells[1], cells[0])].mean()

    for c, model in ((0, sh), (1, sh), (2, sv)):
        for idx in ((3, 4, 2), (1, 1, 1), (5, 2, 6), (2, 6, 3)):
            ref = face_mean(c, idx, model)
            got = eff[c][idx]
            assert abs(got / ref - 1) < 2e-3, (c, idx, got, ref)       # sampling error <= contrast / (2 m) per axis


# ---- CPML coefficients (Eq. 22-24; profile of DESIGN.md [R5]) ------------------------------
def test_cpml_coefficients_obey_eq24_and_the_profile_reflects_1e_minus_3(oracle):
    """The oracle's a, b tables read back and taken apart with Eq. 24 itself (kappa = 1): b = exp(-(d + alpha) dt) and
    a = d (b - 1) / (d + alpha) give rate = -ln b / dt, d = a rate / (b - 1), alpha = rate - d.  What must then hold:
    (i) 0 < b <= 1 and -1 < a <= 0 everywhere (a stable, decaying recursion); (ii) the limits of Eq. 24: where the
    frequency shift vanishes (depth = layer thickness and beyond) a = b - 1 exactly, and towards the inner edge a -> 0
    like depth^2 while b -> exp(-alpha dt) (no damping, d -> 0); (iii) the damping profile is the quadratic one, the same
    curve at node (D-) and half-node (D+) positions, and its theoretical normal-incidence reflection coefficient
    exp(-(2/v) integral_0^L d) is the 1e-3 that [R5] states; (iv) alpha falls linearly from pi fmax / 2 at the inner edge to 0
    at the outer one; (v) with top = AIR the surface side of z has no layer (a = 0, b = 1, L292).  A dropped factor, a
    sign, node and half-node tables swapped, the mirrored index of L324-326 reversed or a wrong reference speed fail one
    of these."""
    d_ax = (100.0, 80.0, 50.0)
    n, nb, fmax, sigma = 14, 6, 5.0, 0.8
    nodes = [np.arange(n + 1) * d for d in d_ax]
    for top in (oracle.TOP_CPML, oracle.TOP_AIR):
        g = oracle.Grid(nodes[0], nodes[1], nodes[2], rd=2, nb=nb, ne=-1, top=top)
        g.model_set(np.full((n, n, n), sigma, np.float32))
        dt = g.info()["dt"]
        g.run_begin([((650.0, 560.0, 350.0), (1, 0, 0))], [1.0], [[700.0, 560.0, 350.0]], dict(fixed_steps=2, fmax=fmax))
        v = np.sqrt(2 * 2 * np.pi * 1.0 / (4e-7 * np.pi * float(np.float32(sigma))))       # 1/sqrt(mu eps), eps = sigma / (2 omega0) (L47)
        for axis in range(3):
            am, bm, ap, bp = g.get("CPML", ifreq=axis)
            delta, L = d_ax[axis], nb * d_ax[axis]
            for side in (0, 1):
                sl = slice(0, nb) if side == 0 else slice(nb, 2 * nb)
                if axis == 2 and side == 0 and top == oracle.TOP_AIR:
                    assert np.all(am[sl] == 0) and np.all(ap[sl] == 0) and np.all(bm[sl] == 1) and np.all(bp[sl] == 1)      # (v)
                    continue
                q = np.arange(nb)
                # depth of slab entry q into the layer: low face entry q is index q, high face entry q is index N-1-q
                depth_node = (nb - q) * delta
                depth_half = (nb - q) * delta + (-0.5 if side == 0 else 0.5) * delta
                depth = np.concatenate([depth_node, depth_half])
                a, b = np.concatenate([am[sl], ap[sl]]), np.concatenate([bm[sl], bp[sl]])
                assert np.all((b > 0) & (b <= 1)) and np.all((a > -1) & (a <= 0))                                           # (i)
                rate = -np.log(b) / dt
                d = a * rate / np.expm1(-rate * dt)
                alpha = rate - d
                outer = depth >= L * (1 - 1e-12)
                assert outer.sum() >= 1 and np.allclose(a[outer], b[outer] - 1, rtol=1e-13, atol=0)                           # (ii) alpha = 0
                c = d / depth ** 2
                assert np.allclose(c, c[0], rtol=1e-9)                                                                      # (iii) quadratic, one curve
                refl = np.exp(-(2.0 / v) * c[0] * L ** 3 / 3.0)                                                             # integral of c xi^2 over [0, L]
                assert abs(refl / 1e-3 - 1) < 1e-9, (axis, side, refl)
                order = np.argsort(depth)
                assert np.all(np.diff(np.abs(a[order])) > 0)                                                                # (ii) |a| grows with depth ...
                inner = order[0]
                assert abs(a[inner] / (d[inner] * dt) + 1) < rate[inner] * dt                                               # ... a -> -d dt -> 0 as d -> 0
                assert abs(b[inner] - np.exp(-alpha[inner] * dt)) <= d[inner] * dt                                          # ... and b -> exp(-alpha dt)
                assert np.allclose(alpha, np.maximum(np.pi * fmax / 2 * (1 - depth / L), 0), rtol=1e-9, atol=1e-9)          # (iv)
        g.close()


# ---- argument checking (SURVEY 8b error codes) ----------------------------------------------------
def test_invalid_arguments(oracle):
    nodes = np.arange(9) * 10.0
    bad = nodes.copy()
    bad[3] = bad[2]
    with pytest.raises(oracle.OracleError):
        oracle.Grid(bad, nodes, nodes, rd=1, nb=2)
    with pytest.raises(oracle.OracleError):
        oracle.Grid(nodes, nodes, nodes, rd=4, nb=2)
    g = oracle.Grid(nodes, nodes, nodes, rd=1, nb=2)
    s = np.ones((8, 8, 8), np.float32)
    s[1, 2, 3] = -1
    with pytest.raises(oracle.OracleError):
        g.model_set(s)
    g.model_set(np.ones((8, 8, 8), np.float32))
    with pytest.raises(oracle.OracleError):          # source outside the interior
        g.run([((500.0, 40.0, 40.0), (1, 0, 0))], [1.0], [[40.0, 40.0, 40.0]], dict(fixed_steps=2))
    with pytest.raises(oracle.OracleError):          # non-positive frequency
        g.run([((40.0, 40.0, 40.0), (1, 0, 0))], [0.0], [[40.0, 40.0, 40.0]], dict(fixed_steps=2))
