"""GPU parity (`-m gpu`): the CUDA path, driven through the C ABI, against the fp64 oracle on the same
seeded inputs, element by element.  Tolerances are north_star's: fp32 fields after 200 steps within 1e-5
relative L2; converged receivers within 1e-3 at every receiver above 1e-3 of the peak; step counts exact.
Sizes span several thread tiles (64 x-nodes, 8 rows, 16-plane chunks) and ragged tails."""
import numpy as np
import pytest

from helpers import make_grid
from paper_2304_00233_b200 import workloads as W

pytestmark = pytest.mark.gpu
FIELDS = ("E1", "E2", "E3", "H1", "H2", "H3")


@pytest.fixture(scope="module")
def emm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2304_00233_b200 import emm as m
    m.build()
    return m


def _rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) else np.float64)
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a)


def _group_errors(ga, gb, s):
    """per field: ||a-b||_2, ||b||_2; plus the E and H group norms (a component that vanishes by symmetry,
    e.g. Hx of an x-dipole, is measured against its group)"""
    d, n = {}, {}
    for c in FIELDS:
        fa, fb = ga.get(c, isrc=s), gb.get(c, isrc=s)
        assert np.all(np.isfinite(fa)), c
        d[c] = np.linalg.norm(fa.astype(np.float64) - fb)
        n[c] = np.linalg.norm(fb)
    grp = {"E": max(n[c] for c in FIELDS[:3]), "H": max(n[c] for c in FIELDS[3:])}
    return d, n, grp


def _field_parity(emm, oracle, w, nsteps, tol=1e-5, ftol=2e-5, sources=None, batched=0, dtft_every=0, dtft_pair=0):
    """Field parity at four checkpoints up to `nsteps` (200 in north_star).

    Tolerance: relative L2 <= 1e-5 per field wherever the field still
    carries >= 10 % of its peak norm; everywhere ||a-b|| <= 1e-5 * peak norm.  The second form is needed
    because the fictitious wave domain is lossless: fp32 rounding at the source node leaves a static,
    curl-free residual of ~1e-8 of the peak that never radiates away, while on these small test grids the
    wave itself has left through the CPML long before step 200."""
    sources = sources or w["sources"]
    opts = dict(fixed_steps=nsteps, batched=batched, dtft_every=dtft_every)
    ga, gb = make_grid(emm, w), make_grid(oracle, w)
    assert abs(ga.info()["dt"] / gb.info()["dt"] - 1) < 1e-12
    for c in ("CE1", "CE2", "CE3"):
        assert _rel_l2(ga.get(c), gb.get(c)) < 1e-7, c
    ga.run_begin(sources, w["freqs"], w["receivers"], dict(opts, dtft_pair=dtft_pair))   # scheduling of the same sums: not an oracle option
    gb.run_begin(sources, w["freqs"], w["receivers"], opts)
    peak = [{"E": 0.0, "H": 0.0} for _ in sources]
    done_steps, strict_checks = 0, 0
    for q in range(4):
        n = nsteps * (q + 1) // 4 - done_steps
        nsa, da = ga.run_steps(n)
        nsb, db = gb.run_steps(n)
        done_steps += n
        assert list(nsa) == list(nsb) == [done_steps] * len(sources)
        for s in range(len(sources)):
            d, nrm, grp = _group_errors(ga, gb, s)
            for k in ("E", "H"):
                peak[s][k] = max(peak[s][k], grp[k])
            for c in FIELDS:
                k = c[0]
                assert d[c] <= tol * peak[s][k], (w["name"], done_steps, s, c, d[c] / peak[s][k])
                if grp[k] >= 0.1 * peak[s][k] and nrm[c] > 1e-3 * grp[k]:
                    strict_checks += 1
                    assert d[c] <= tol * nrm[c], (w["name"], done_steps, s, c, d[c] / nrm[c])
    assert da and db and strict_checks >= 5
    for s in range(len(sources)):
        for f in range(len(w["freqs"])):
            Fn = {c: gb.get("F_" + c, isrc=s, ifreq=f) for c in FIELDS}
            for c in FIELDS:
                grp = max(np.linalg.norm(Fn[x]) for x in FIELDS if x[0] == c[0])
                e = np.linalg.norm(ga.get("F_" + c, isrc=s, ifreq=f).astype(np.complex128) - Fn[c]) / grp
                assert e < ftol, (w["name"], s, f, "F_" + c, e)
    oa, _ = ga.run_end()
    ob, _ = gb.run_end()
    for s in range(len(sources)):
        for k in (slice(0, 3), slice(3, 6)):
            A, B = oa[s][..., k], ob[s][..., k]
            big = np.abs(B) > 1e-3 * np.abs(B).max()
            assert np.all(np.abs(A - B)[big] <= 1e-3 * np.abs(B)[big])
    ga.close()


@pytest.mark.parametrize("rd,pair", [(1, 0), (2, 0), (3, 0), (2, -1)])
def test_fields_wholespace_cpml(emm, oracle, rd, pair):
    """configs[0] scaled: homogeneous, CPML on six faces; 70 x-nodes (2 tiles + ragged tail), 200 steps.
    pair = 0: paired DTFT (default); -1: one term per step in every step."""
    w = W.cfg1(n=40 - 2 * rd, dx=100.0, rd=rd, nb=7)
    src = np.array(w["sources"][0][0])
    offs = np.array([300.0, 600.0, 900.0, 1200.0])        # off-axis, off-grid: all six components are non-zero
    w["receivers"] = np.stack([src[0] + 0.8 * offs, src[1] + 0.36 * offs, src[2] - 0.48 * offs], axis=1)
    _field_parity(emm, oracle, w, 200, dtft_pair=pair)


def test_wide_cpml_layer_in_an_exactly_sized_workspace(emm, oracle):
    """nb = 34: the twelve CPML coefficient tables are longer than one 256-byte allocation unit each; the workspace is the
    one emm_workspace_bytes asks for (the binding allocates exactly that), so the tables must be part of its count."""
    w = W.cfg1(n=14, dx=100.0, rd=2, nb=34)
    src = np.array(w["sources"][0][0])
    offs = np.array([150.0, 300.0, 420.0])                 # off-axis, off-grid: all six components are non-zero
    w["receivers"] = np.stack([src[0] + 0.8 * offs, src[1] + 0.36 * offs, src[2] - 0.48 * offs], axis=1)
    _field_parity(emm, oracle, w, 120)


@pytest.mark.parametrize("rd", [1, 2, 3])
def test_fields_layered_air_uniform(emm, oracle, rd):
    """configs[1] scaled: layered marine model, FFT air-water boundary on the padded plane itself."""
    w = W.cfg2(nx=36, nz=24, dx=100.0, rd=rd, nb=8)
    _field_parity(emm, oracle, w, 200)


def _small_receivers():
    g = np.array([-310.0, -95.0, 140.0, 330.0])
    X, Y = np.meshgrid(g, g * 0.9, indexing="xy")
    return np.stack([X.ravel(), Y.ravel(), np.full(X.size, 1000.0)], axis=1)


@pytest.mark.parametrize("rd,builder,pair", [(2, "cfg3", 0), (3, "cfg4", 0), (3, "cfg4", -1)])
def test_fields_nonuniform_aux_plane_vti(emm, oracle, rd, builder, pair):
    """configs[2]/[3] scaled: non-uniform x-y-z, VTI cells from sub-sampling, auxiliary-plane air boundary."""
    kw = dict(nx=40, nz=36, rd=rd, nb=8, n_water=8, n_rec_side=3, aux_dx=50.0)
    w = W.build(builder, oracle.nugrid, **kw)
    w["receivers"] = _small_receivers()
    w["sigma_v"] = (w["sigma_v"] * 0.6).astype(np.float32)                # make the anisotropy bite everywhere
    _field_parity(emm, oracle, w, 200, dtft_pair=pair)


def test_fields_batched_sources(emm, oracle):
    """configs[4] scaled: several sources advanced by one launch per kernel, each against its own oracle run."""
    w = W.cfg5(oracle.nugrid, nx=32, nz=30, rd=2, nb=6, n_water=6, nsrc=3, n_rec_side=3, aux_dx=100.0)
    srcs = [((-180.0 + 170.0 * i, 40.0 * i, 950.0), (1.0, 0.3 * i, 0.1)) for i in range(3)]
    w["receivers"] = _small_receivers()
    _field_parity(emm, oracle, w, 120, sources=srcs, batched=1)


@pytest.mark.parametrize("m", [3, -1])
def test_dtft_decimation_matches_oracle(emm, oracle, m):
    """only every m-th term of Eq. 25 is accumulated (m = -1: the automatic safe value);
    fields, accumulators, J', receivers and the converged step count follow the oracle's identical rule."""
    w = W.cfg2(nx=36, nz=24, dx=100.0, rd=2, nb=8)
    _field_parity(emm, oracle, w, 200, dtft_every=m)
    opts = dict(tol=1e-6, check_every=100, dtft_every=m)
    ga, gb = make_grid(emm, w), make_grid(oracle, w)
    oa, nsa = ga.run(w["sources"], w["freqs"], w["receivers"], opts)
    ob, nsb = gb.run(w["sources"], w["freqs"], w["receivers"], dict(opts, sparse_dft=1))
    assert list(nsa) == list(nsb) and nsa[0] > 0
    big = np.abs(ob) > 1e-3 * np.abs(ob).max()
    assert (np.abs(oa - ob)[big] / np.abs(ob)[big]).max() < 1e-3


@pytest.mark.parametrize("m", [0, -1])
def test_receivers_only_dtft_matches_full_grid_and_oracle(emm, oracle, m):
    """SURVEY 8f rank 1, second half: sparse_dft keeps the sums of Eq. 25 only at the receivers' stencil nodes (fp64)
    and on the check set.  Same receivers as the full-grid run and as the oracle, same converged step count, with
    and without decimation, on the non-uniform grid with the auxiliary-plane air boundary and two batched sources."""
    w = W.cfg3(oracle.nugrid, nx=36, nz=32, rd=2, nb=8, n_water=8, n_rec_side=3, aux_dx=50.0)
    w["receivers"] = _small_receivers()
    srcs = [((-150.0, 30.0, 950.0), (1.0, 0.2, 0.1)), ((120.0, -60.0, 930.0), (0.1, 1.0, 0.3), "M")]
    opts = dict(tol=1e-6, check_every=100, dtft_every=m, batched=1)
    ga, gb = make_grid(emm, w), make_grid(oracle, w)
    o_full, n_full = ga.run(srcs, w["freqs"], w["receivers"], opts)
    o_sp, n_sp = ga.run(srcs, w["freqs"], w["receivers"], dict(opts, sparse_dft=1))
    o_or, n_or = gb.run(srcs, w["freqs"], w["receivers"], dict(opts, sparse_dft=1))
    assert list(n_sp) == list(n_full) == list(n_or) and min(n_sp) > 0          # integer outputs: exact
    for s in range(2):
        for sl in (slice(0, 3), slice(3, 6)):
            ref = o_or[s][..., sl]
            big = np.abs(ref) > 1e-3 * np.abs(ref).max()
            assert big.sum() > 10
            assert (np.abs(o_sp[s][..., sl] - ref)[big] / np.abs(ref)[big]).max() < 1e-3
            assert (np.abs(o_full[s][..., sl] - ref)[big] / np.abs(ref)[big]).max() < 1e-3
    # no full-grid accumulator exists in this mode
    ga.run_begin(srcs[:1], w["freqs"], w["receivers"], dict(fixed_steps=5, sparse_dft=1))
    ga.run_steps(5)
    with pytest.raises(emm.EmmError) as e:
        ga.get("F_E1")
    assert e.value.code == emm.EINVAL
    ga.run_end()


@pytest.mark.parametrize("group", [0, 2, 8])
def test_paired_dtft_is_the_one_term_sum_bit_for_bit(emm, oracle, group):
    """Grouped DTFT (emm_run_opts.dtft_pair; 0 = default group, 2 = pairs, 8 = the largest group): m consecutive terms of
    Eq. 25 per pass over the accumulators, the earlier levels of a group copied by the passes before the closing one.
    Same fused multiply-adds in the same order as one term per step, so fields and accumulators are bit-identical to
    the dtft_pair = -1 run everywhere except at the injected nodes (where the missing product is added by the
    injection kernel, rounding order differs), whatever the batch sizes (odd batches leave single steps), for an
    electric and a magnetic dipole batched on the non-uniform grid with the air-water boundary.  Then run to
    convergence with an odd check interval: step counts identical, receivers the same to rounding, and both match
    the oracle."""
    w = W.cfg3(oracle.nugrid, nx=36, nz=32, rd=2, nb=8, n_water=8, n_rec_side=3, aux_dx=50.0)
    w["receivers"] = _small_receivers()
    srcs = [((-150.0, 30.0, 950.0), (1.0, 0.2, 0.1)), ((120.0, -60.0, 930.0), (0.1, 1.0, 0.3), "M")]
    ga, gs = make_grid(emm, w), make_grid(emm, w)
    ga.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=131, batched=1, dtft_pair=group))
    assert int(ga.get("DTFT_GROUP")[0]) == (group or 6)                # three frequencies: default group 6
    gs.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=131, batched=1, dtft_pair=-1))
    assert int(gs.get("DTFT_GROUP")[0]) == 1
    total = 0
    for n in (7, 50, 1, 33, 40):                     # 131 steps: odd and even batches, a pair split by a batch end
        na, _ = ga.run_steps(n)
        ns, _ = gs.run_steps(n)
        total += n
        assert list(na) == list(ns) == [total, total]
        for s in range(2):
            for c in FIELDS:
                assert np.array_equal(ga.get(c, isrc=s), gs.get(c, isrc=s)), (total, s, c)
            for f in (0, len(w["freqs"]) - 1):
                for c in FIELDS:
                    Fa, Fs = ga.get("F_" + c, isrc=s, ifreq=f), gs.get("F_" + c, isrc=s, ifreq=f)
                    differ = Fa != Fs
                    assert differ.sum() <= 6 ** 3, (total, s, f, c, int(differ.sum()))     # at most one source stencil
                    assert np.abs(Fa - Fs).max() <= 1e-5 * np.abs(Fs).max(), (total, s, f, c)
    assert np.abs(gs.get("F_E1", isrc=0, ifreq=0)).max() > 0 and np.abs(gs.get("F_H2", isrc=1, ifreq=0)).max() > 0
    oa, _ = ga.run_end()
    os_, _ = gs.run_end()
    assert np.abs(oa - os_).max() <= 1e-5 * np.abs(os_).max()
    opts = dict(tol=1e-6, check_every=75, batched=1)
    o_p, n_p = ga.run(srcs, w["freqs"], w["receivers"], dict(opts, dtft_pair=group))
    o_s, n_s = gs.run(srcs, w["freqs"], w["receivers"], dict(opts, dtft_pair=-1))
    o_or, n_or = make_grid(oracle, w).run(srcs, w["freqs"], w["receivers"], dict(opts, sparse_dft=1))
    assert list(n_p) == list(n_s) == list(n_or) and min(n_p) > 0 and n_p[0] % 75 == 0
    for s in range(2):
        for sl in (slice(0, 3), slice(3, 6)):
            ref = o_or[s][..., sl]
            big = np.abs(ref) > 1e-3 * np.abs(ref).max()
            assert (np.abs(o_p[s][..., sl] - ref)[big] / np.abs(ref)[big]).max() < 1e-3
            assert (np.abs(o_p[s][..., sl] - o_s[s][..., sl])[big] / np.abs(ref)[big]).max() < 1e-5


@pytest.mark.parametrize("rd", [1, 2, 3])
def test_paired_dtft_every_instance(emm, rd):
    """Every closing-pass instance k_update<rd, nf, ., PAIR>, nf = 1..5, with group sizes 6 (default), 2, 3, 5, 8, against
    the one-term schedule on a small whole-space grid (CPML on six faces), 41 steps in batches of 20 + 21 (whole groups,
    shorter groups and single steps): fields bit-identical, accumulators bit-identical away from the injected nodes and
    within rounding there.  nf = 6 has no such instance: the option is ignored."""
    w = W.cfg1(n=26, dx=100.0, rd=rd, nb=5)
    freqs_all = np.array([0.25, 0.5, 0.75, 1.0, 1.25, 1.5])
    for nf in range(1, 7):
        ga, gs = make_grid(emm, w), make_grid(emm, w)
        ga.run_begin(w["sources"], freqs_all[:nf], w["receivers"][:2], dict(fixed_steps=41, dtft_pair=(0, 2, 3, 5, 8, 0)[nf - 1]))
        assert int(ga.get("DTFT_GROUP")[0]) == (6, 2, 3, 5, 8, 1)[nf - 1]
        gs.run_begin(w["sources"], freqs_all[:nf], w["receivers"][:2], dict(fixed_steps=41, dtft_pair=-1))
        for n in (20, 21):
            ga.run_steps(n)
            gs.run_steps(n)
        for c in FIELDS:
            assert np.array_equal(ga.get(c), gs.get(c)), (rd, nf, c)
            for f in (0, nf - 1):
                Fa, Fs = ga.get("F_" + c, ifreq=f), gs.get("F_" + c, ifreq=f)
                assert (Fa != Fs).sum() <= (0 if nf == 6 else max(2 * rd, 4) ** 3), (rd, nf, c, f)
                assert np.abs(Fa - Fs).max() <= 1e-5 * max(np.abs(Fs).max(), 1e-30), (rd, nf, c, f)
        assert np.abs(gs.get("F_E1", ifreq=nf - 1)).max() > 0
        oa, _ = ga.run_end()
        ob, _ = gs.run_end()
        assert np.abs(oa - ob).max() <= 1e-5 * np.abs(ob).max()
        ga.close()
        gs.close()


def test_grouped_dtft_takes_the_largest_group_the_workspace_allows(emm):
    """A workspace short of three history slots: the run falls back from groups of 8 to groups of 5 (same sums, bit for
    bit); without room for any copy it runs pairs; without room for the run at all it fails with EMM_ENOMEM."""
    w = W.cfg1(n=26, dx=100.0, rd=2, nb=5)
    freqs = np.array([0.25, 0.5, 0.75, 1.0])            # four frequencies: default group 8
    ref = make_grid(emm, w)
    ref.run_begin(w["sources"], freqs, w["receivers"][:2], dict(fixed_steps=40, dtft_pair=-1))
    ref.run_steps(40)
    Fref = ref.get("F_E1", ifreq=3)
    info = ref.info()
    vol = info["pitch"] * info["N2"] * info["N3"] * 4                      # bytes of one field-sized array
    full = ref.workspace_bytes(1, len(freqs), 50, 2)
    for short, group in ((0, 8), (3 * 6 * vol, 5), (6 * 6 * vol, 2)):
        g = emm.Grid(w["x"], w["y"], w["z"], **w["grid"])
        g.bind(nsrc=1, nfreq=len(freqs), max_steps=50, nrec=2, ws_bytes=full - short)
        g.model_set(w["sigma_h"])
        g.run_begin(w["sources"], freqs, w["receivers"][:2], dict(fixed_steps=40))
        assert int(g.get("DTFT_GROUP")[0]) == group, (short, int(g.get("DTFT_GROUP")[0]))
        g.run_steps(40)
        F = g.get("F_E1", ifreq=3)
        assert (F != Fref).sum() <= 4 ** 3 and np.abs(F - Fref).max() <= 1e-5 * np.abs(Fref).max()
        g.close()
    g = emm.Grid(w["x"], w["y"], w["z"], **w["grid"])
    g.bind(nsrc=1, nfreq=len(freqs), max_steps=50, nrec=2, ws_bytes=full - 6 * 6 * vol - 30 * vol)
    g.model_set(w["sigma_h"])
    with pytest.raises(emm.EmmError) as e:
        g.run_begin(w["sources"], freqs, w["receivers"][:2], dict(fixed_steps=40))
    assert e.value.code == emm.ENOMEM


def test_plane_and_separable_air_routes_agree(emm, oracle):
    """Non-uniform x-y: the separable route (batched 1-D transforms, default) and the plane-sized 2-D route
    (emm_grid_opts.air_route = 1) are the same linear map up to rounding order; both are within the field tolerance of the oracle."""
    w = W.cfg4(oracle.nugrid, nx=40, nz=36, rd=3, nb=8, n_water=8, n_rec_side=3, aux_dx=50.0)
    w["receivers"] = _small_receivers()
    fields = {}
    for route in ("0", "1"):
        g = make_grid(emm, w, air_route=int(route))
        g.run_begin(w["sources"], w["freqs"], w["receivers"], dict(fixed_steps=150))
        g.run_steps(150)
        fields[route] = [g.get(c) for c in ("E1", "E2", "E3", "H1", "H2", "H3")]
        g.run_end()
        g.close()
    for a, b in zip(fields["0"], fields["1"]):
        assert np.abs(a).max() > 0
    ne = np.sqrt(sum(np.sum(np.asarray(a, np.float64) ** 2) for a in fields["0"][:3]))
    nh = np.sqrt(sum(np.sum(np.asarray(a, np.float64) ** 2) for a in fields["0"][3:]))
    de = np.sqrt(sum(np.sum((np.asarray(a, np.float64) - b) ** 2) for a, b in zip(fields["0"][:3], fields["1"][:3])))
    dh = np.sqrt(sum(np.sum((np.asarray(a, np.float64) - b) ** 2) for a, b in zip(fields["0"][3:], fields["1"][3:])))
    assert de / ne < 1e-5 and dh / nh < 1e-5


@pytest.mark.parametrize("rd,nx,ny_extra", [(1, 36, 0), (2, 52, 9), (3, 44, 5), (2, 200, 0)])
def test_cluster_and_library_air_routes_agree(emm, oracle, rd, nx, ny_extra):
    """Uniform x-y: the one-launch cluster route (hand-written shared-memory transforms, emm_air_cluster.cu, default) and the
    library route (emm_grid_opts.air_route = 1: pack, 2-D cuFFT, filter, 2-D cuFFT, unpack) are the same linear map up to
    rounding order.  Planes of several 7-smooth sizes (radix 2, 3, 4, 5 and 7 passes, rectangular, rows and columns that do
    not divide by the cluster size; a 240 x 240 plane whose two H ghost levels do not fit shared memory together and go
    through the kernel one after the other), two sources in one launch.  The ghost planes the boundary writes are compared directly,
    then every field; the oracle comparison of this route is test_fields_layered_air_uniform."""
    w = W.cfg2(nx=nx, nz=24, dx=100.0, rd=rd, nb=8)
    if ny_extra:                                                     # rectangular plane
        w["y"] = np.concatenate([w["y"], w["y"][-1] + 100.0 * np.arange(1, ny_extra + 1)])
        w["sigma_h"] = np.concatenate([w["sigma_h"], w["sigma_h"][:, -ny_extra:, :]], axis=1)
    srcs = [((-150.0, 30.0, 950.0), (1.0, 0.2, 0.1)), ((120.0, -60.0, 930.0), (0.1, 1.0, 0.3), "M")]
    fields, k0 = {}, None
    for route in (0, 1):
        g = make_grid(emm, w, air_route=route)
        info = g.info()
        assert (info["air_cluster"] > 0) == (route == 0), info
        k0 = info["k0"]
        g.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=150, batched=1))
        g.run_steps(150)
        fields[route] = [[np.asarray(g.get(c, isrc=q), np.float64) for c in FIELDS] for q in range(2)]
        g.run_end()
        g.close()
    for q in range(2):
        for lo, hi in ((0, 3), (3, 6)):
            n = np.sqrt(sum(np.sum(a ** 2) for a in fields[0][q][lo:hi]))
            d = np.sqrt(sum(np.sum((a - b) ** 2) for a, b in zip(fields[0][q][lo:hi], fields[1][q][lo:hi])))
            assert n > 0 and d / n < 1e-5, (q, lo, d / n)
            # the ghost planes above the surface are written by the boundary alone (Ex, Ey on rd - 1 levels; Hx, Hy on rd)
            for c in (lo, lo + 1):
                for m in range(1, rd + (1 if lo == 3 else 0)):
                    a, b = fields[0][q][c][k0 - m], fields[1][q][c][k0 - m]
                    assert np.linalg.norm(b) > 0
                    assert np.linalg.norm(a - b) < 2e-5 * np.linalg.norm(b), (q, c, m, np.linalg.norm(a - b) / np.linalg.norm(b))


def test_magnetic_and_mixed_sources_match_oracle(emm, oracle):
    """a magnetic dipole (injected into H at the half step), alone and batched together with
    an electric dipole; fields, accumulators and receivers against the oracle."""
    w = W.cfg2(nx=36, nz=24, dx=100.0, rd=2, nb=8)
    srcs = [((-130.0, 60.0, 870.0), (0.2, 1.0, 0.4), "M"), ((210.0, -40.0, 930.0), (1.0, 0.0, 0.3))]
    _field_parity(emm, oracle, w, 160, sources=srcs[:1])
    _field_parity(emm, oracle, w, 120, sources=srcs, batched=1)


@pytest.mark.parametrize("case", ["air_nonuniform_vti", "wholespace_cpml"])
def test_sensitivity_kernel_matches_oracle(emm, oracle, case):
    """SURVEY 8f rank 4 (gradient accumulation, DESIGN.md [R14]): emm_sensitivity against emmo_sensitivity, cell by cell,
    for d/d sigma_h and d/d sigma_v.  The oracle chains every E node through its Eq. 26 weights and node volume; the CUDA
    path gathers cell volume / 4 times the edge products per cell -- two derivations of the same sum.  Oblique off-grid
    dipoles so that all three components carry weight; the non-uniform case has the air layer (not a parameter) and VTI
    cells, the whole-space case a CPML on all six faces (padding cells fold into the edge cells on every side).
    Tolerance: the accumulators of either source are within 2e-5 relative L2 of the oracle's (the accumulator tolerance
    above), their product within 4e-5; 1e-4 on each kernel as a whole, and 1e-3 on the outermost shell of model cells taken
    alone (values 1e-3 .. 1e-6 of the peak: what the fold of the padding cells produces)."""
    if case == "air_nonuniform_vti":
        w = W.build("cfg3", oracle.nugrid, nx=40, nz=36, rd=2, nb=8, n_water=8, n_rec_side=3, aux_dx=50.0)
        w["sigma_v"] = (w["sigma_v"] * 0.6).astype(np.float32)
        srcs = [((-150.0, 30.0, 950.0), (1.0, 0.2, 0.1)), ((260.0, -110.0, 1000.0), (0.3, 0.8, 0.5))]
        nsteps = 300
    else:
        w = W.cfg1(n=30, dx=100.0, rd=3, nb=7)
        c = np.array(w["sources"][0][0])
        srcs = [(tuple(c + [-340.0, 30.0, 20.0]), (1.0, 0.4, -0.3)), (tuple(c + [330.0, -60.0, 110.0]), (0.2, 0.5, 0.8))]
        nsteps = 200
    ga, gb = make_grid(emm, w), make_grid(oracle, w)
    opts = dict(fixed_steps=nsteps, batched=1)
    for g in (ga, gb):
        g.run_begin(srcs, w["freqs"][:2] if len(w["freqs"]) > 1 else w["freqs"], w["receivers"], opts)
        g.run_steps(nsteps)
    f = 1 if len(w["freqs"]) > 1 else 0
    ka, kb = ga.sensitivity(0, 1, f), gb.sensitivity(0, 1, f)
    kswap = ga.sensitivity(1, 0, f)
    shell = np.ones(kb[0].shape, bool)
    shell[1:-1, 1:-1, 1:-1] = False
    for q, name in enumerate(("sigma_h", "sigma_v")):
        A, B = ka[q], kb[q]
        assert np.all(np.isfinite(A.view(np.float64)))
        assert np.array_equal(A, kswap[q])                                   # symmetric in the two sources, to the last bit
        assert np.linalg.norm(B) > 0 and np.abs(B[~shell]).max() > 0
        assert _rel_l2(A, B) < 1e-4, (case, name, _rel_l2(A, B))
        assert np.linalg.norm(B[shell]) > 0
        assert _rel_l2(A[shell], B[shell]) < 1e-3, (case, name, "shell", _rel_l2(A[shell], B[shell]))
        assert np.all(A[B == 0] == 0), (case, name)                          # cells out of reach of the DTFT box are exactly zero
    # the calls it must refuse
    with pytest.raises(emm.EmmError):
        ga.sensitivity(0, 2, f)
    with pytest.raises(emm.EmmError):
        ga.sensitivity(0, 1, 7)
    ga.run_end()
    ga.run_begin(srcs[:1], w["freqs"][:1], w["receivers"], dict(fixed_steps=8))
    ga.run_steps(8)
    with pytest.raises(emm.EmmError):
        ga.sensitivity(0, 0, 0)                                              # a run with a single resident source
    ga.run_end()
    ga.run_begin([srcs[0], srcs[1] + ("M",)], w["freqs"][:1], w["receivers"], dict(fixed_steps=8, batched=1))
    ga.run_steps(8)
    with pytest.raises(emm.EmmError):
        ga.sensitivity(0, 1, 0)                                              # magnetic receiver dipole
    ga.run_end()
    ga.close()
    gb.close()


@pytest.mark.parametrize("rd", [2, 3])
def test_layered_marine_model_matches_semi_analytic_solution_on_the_gpu(emm, rd):
    """The CUDA path against physics directly, no oracle in between: the layered marine model of the oracle's pin
    (tests/test_oracle_physics.py: air / 400 m of sea water / sediment with a resistive layer, dipole 50 m above the seabed,
    in-line, broadside and oblique receivers on the seabed and inside the water layer) run through the C ABI in fp32 with the
    one-launch air-water boundary, compared with the semi-analytic layered-earth solution (tests/layered1d.py).  Same bounds
    as for the oracle: Ex, Ey within 2 % and Hz within 1 % on the seabed, all six components within 1.5 % (E) / 3 % (H) inside
    the water layer (discretisation error of 50 m cells; fp32 adds nothing visible at this level)."""
    from test_oracle_physics import _layered_marine_case, _layered_marine_check
    x, z, sig, zs, f, rel, layers = _layered_marine_case()
    rec = rel + np.array([-25.0, 0.0, 0.0])
    g = emm.Grid(x, x, z, rd=rd, nb=8, ne=-1, top=emm.TOP_AIR)
    g.model_set(sig)
    assert g.info()["air_cluster"] > 0
    out, _ = g.run([((-25.0, 0.0, zs), (1, 0, 0))], [f], rec, dict(fixed_steps=int(4.0 / g.info()["dt"])))
    _layered_marine_check(out[0, 0], rel, zs, f, layers)
    g.close()


def test_stretched_grid_marine_model_matches_semi_analytic_solution_on_the_gpu(emm):
    """The separable auxiliary-plane route of the air-water boundary (non-uniform x-y, emm_air_sep.cu) against physics
    directly: the layered marine model on a grid stretched in x, y and z, same case and bounds as the oracle's pin
    (tests/test_oracle_physics.py::test_stretched_grid_marine_model_matches_semi_analytic_solution)."""
    from test_oracle_physics import _stretched_marine_case, _stretched_marine_check
    x, zb, sig, zs, f, rel, layers, shift = _stretched_marine_case()
    g = emm.Grid(x, x, zb, rd=2, nb=8, ne=-1, top=emm.TOP_AIR)
    g.model_set(sig)
    assert g.info()["uniform_xy"] == 0 and g.info()["air_cluster"] == 0
    out, _ = g.run([((shift[0], shift[1], zs), (1, 0, 0))], [f], rel + shift, dict(fixed_steps=int(4.0 / g.info()["dt"])))
    _stretched_marine_check(out[0, 0], rel, zs, f, layers)
    g.close()


def test_vti_whole_space_matches_semi_analytic_solution_on_the_gpu(emm):
    """sigma_v in the CUDA path against physics directly: an anisotropic whole space (sigma_h = 1, sigma_v = 0.4 S/m, CPML
    on six faces), all six components at in-line, broadside and oblique receivers 300 m below the dipole, against the
    semi-analytic solution whose TM line carries sigma_v (tests/layered1d.py).  Bound 1.5 % of the largest component of the
    field at the receiver (the oracle's pin measures < 0.7 %); the isotropic solution is more than 50 % away."""
    from layered1d import layered_hed
    n = 40
    xw = (np.arange(n + 1) - n // 2) * 100.0
    src = (-50.0, 0.0, 30.0)
    offs = np.array([600.0, 900.0, 1200.0])
    rel = np.concatenate([np.stack([offs, 0 * offs, 0 * offs + 330.0], axis=1), np.stack([0 * offs, offs, 0 * offs + 330.0], axis=1),
                          np.stack([0.6 * offs, 0.8 * offs, 0 * offs + 330.0], axis=1)])
    g = emm.Grid(xw, xw, xw, rd=2, nb=8, ne=-1, top=emm.TOP_CPML)
    g.model_set(np.full((n, n, n), 1.0, np.float32), np.full((n, n, n), 0.4, np.float32))
    out, _ = g.run([(src, (1, 0, 0))], [1.0], rel + np.array([src[0], src[1], 0.0]), dict(fixed_steps=int(5.0 / g.info()["dt"])))
    ref = layered_hed(src[2], rel, 1.0, [1.0], [None], sigma_v=[0.4])
    iso = layered_hed(src[2], rel, 1.0, [1.0], [None], primary="hankel")
    sE, sH = np.abs(ref[:, :3]).max(axis=1, keepdims=True), np.abs(ref[:, 3:]).max(axis=1, keepdims=True)
    sc = np.concatenate([sE, sE, sE, sH, sH, sH], axis=1)
    assert (np.abs(out[0, 0] - ref) / sc).max() < 1.5e-2
    assert (np.abs(iso - ref) / sc).max() > 0.5
    g.close()


def test_converged_run_matches_oracle_steps_and_receivers(emm, oracle):
    """configs[1] scaled, run to convergence: integer step count exact, receivers within 1e-3."""
    w = W.cfg2(nx=40, nz=28, dx=100.0, rd=2, nb=8)
    opts = dict(tol=1e-6, check_every=100)
    ga, gb = make_grid(emm, w), make_grid(oracle, w)
    oa, nsa = ga.run(w["sources"], w["freqs"], w["receivers"], opts)
    ob, nsb = gb.run(w["sources"], w["freqs"], w["receivers"], dict(opts, sparse_dft=1))
    assert list(nsa) == list(nsb) and nsa[0] % 100 == 0 and nsa[0] > 0
    big = np.abs(ob) > 1e-3 * np.abs(ob).max()
    rel = np.abs(oa - ob)[big] / np.abs(ob)[big]
    assert rel.max() < 1e-3, rel.max()
    da = ga.get("DELTA")
    assert np.all(da < 1e-6)


def test_converged_cfg1_fixed_500_steps(emm, oracle):
    """configs[0] itself (48^3, rd=1, 500 fixed steps, 20 in-line receivers)."""
    w = W.cfg1()
    ga, gb = make_grid(emm, w), make_grid(oracle, w)
    oa, nsa = ga.run(w["sources"], w["freqs"], w["receivers"], w["run"])
    ob, nsb = gb.run(w["sources"], w["freqs"], w["receivers"], w["run"])
    assert list(nsa) == list(nsb) == [500]
    ex_a, ex_b = oa[0, 0, :, 0], ob[0, 0, :, 0]
    assert np.abs(ex_a / ex_b - 1).max() < 1e-3


def test_batched_equals_sequential_and_nsteps_per_source(emm, oracle):
    w = W.cfg2(nx=32, nz=24, dx=100.0, rd=2, nb=8)
    srcs = [((-300.0, 0.0, 950.0), (1, 0, 0)), ((250.0, 100.0, 900.0), (0, 1, 0))]
    ga = make_grid(emm, w)
    opts = dict(tol=1e-6, check_every=100)
    o_seq, n_seq = ga.run(srcs, w["freqs"], w["receivers"], dict(opts, batched=0))
    o_bat, n_bat = ga.run(srcs, w["freqs"], w["receivers"], dict(opts, batched=1))
    assert list(n_seq) == list(n_bat)
    assert np.array_equal(o_seq, o_bat)               # same kernels, same arithmetic, source by source
    gb = make_grid(oracle, w)
    o_or, n_or = gb.run(srcs, w["freqs"], w["receivers"], dict(opts, sparse_dft=1))
    assert list(n_or) == list(n_bat)


def test_edge_cases(emm, oracle):
    w = W.cfg1(n=12, dx=100.0, rd=1, nb=3)
    ga = make_grid(emm, w)
    # no receivers: nothing to write, step count still returned
    out, ns = ga.run(w["sources"], w["freqs"], np.zeros((0, 3)), dict(fixed_steps=7))
    assert out.shape == (1, 1, 0, 6) and ns[0] == 7
    # max_steps reached -> EMM_ENOCONV, outputs still finite
    out, ns = ga.run(w["sources"], w["freqs"], w["receivers"][:2], dict(tol=1e-30, check_every=20, max_steps=60), allow_noconv=True)
    assert ga.last_rc == emm.ENOCONV and ns[0] == 60 and np.all(np.isfinite(out))
    # source / receiver outside the interior
    with pytest.raises(emm.EmmError) as e:
        ga.run([((5000.0, 600.0, 600.0), (1, 0, 0))], w["freqs"], w["receivers"][:1], dict(fixed_steps=3))
    assert e.value.code == emm.EINVAL
    with pytest.raises(emm.EmmError):
        ga.run(w["sources"], w["freqs"], [[-400.0, 600.0, 600.0]], dict(fixed_steps=3))
    with pytest.raises(emm.EmmError):
        ga.model_set(-np.ones((12, 12, 12), np.float32))
    # maximum number of frequencies on the unrolled path + the runtime fallback give the same accumulators as the oracle
    ga = make_grid(emm, w)
    gb = make_grid(oracle, w)
    freqs = np.array([0.25, 0.5, 0.75, 1.0, 1.25, 1.5, 2.0])
    ga.run_begin(w["sources"], freqs, w["receivers"][:2], dict(fixed_steps=40))
    gb.run_begin(w["sources"], freqs, w["receivers"][:2], dict(fixed_steps=40))
    ga.run_steps(40)
    gb.run_steps(40)
    for f in (0, 6):
        assert _rel_l2(ga.get("F_E1", ifreq=f), gb.get("F_E1", ifreq=f)) < 2e-5
        assert _rel_l2(ga.get("F_H2", ifreq=f), gb.get("F_H2", ifreq=f)) < 2e-5
