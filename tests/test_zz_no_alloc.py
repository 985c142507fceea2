"""GPU test (`-m gpu`) of emm_check_delta_static, the entry point that allocates nothing (include/emm.h): its output against
the existing path's -- the convergence measure the run driver computes with k_check_reduce / k_check_final on scratch carved
from the workspace, read back with emm_get(EMM_GET_DELTA) -- on calls made one after the other through the same static
scratch array.  Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the
other tests (it builds its own grid and shares no state with them)."""
import numpy as np
import pytest

from helpers import make_grid
from paper_2304_00233_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def emm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2304_00233_b200 import emm as m
    m.build()
    return m


def test_static_scratch_check_matches_the_run_drivers_check(emm):
    import torch
    # two sources advanced together (electric + magnetic) on a small marine grid, checks every 50 steps, no stop
    w = W.cfg2(nx=36, nz=24, dx=100.0, rd=2, nb=8)
    srcs = [((-130.0, 60.0, 870.0), (0.2, 1.0, 0.4), "M"), ((210.0, -40.0, 930.0), (1.0, 0.0, 0.3))]
    g = make_grid(emm, w)
    g.run_begin(srcs, w["freqs"], w["receivers"][:4], dict(fixed_steps=150, check_every=50, batched=1, fmax=12.0))
    nchk = int(g.get("CHECK_N")[0])
    assert nchk > 1000
    acc, ref = [], []
    for _ in range(3):                         # the checks at steps 50, 100, 150
        ns, _ = g.run_steps(50)
        acc.append(np.stack([g.get("CHECK_ACC", isrc=s) for s in range(2)]))          # [2][6][nchk], complete up to this step
        ref.append(np.stack([g.get("DELTA", isrc=s) for s in range(2)]))              # what the run driver's check found
    assert np.all(np.isfinite(ref[1])) and np.all(ref[1] > 0) and not np.array_equal(ref[1], ref[2])
    dev = "cuda:0"
    t = [torch.from_numpy(a).to(dev) for a in acc]
    zero = torch.zeros_like(t[0])
    # calls in a row through the same scratch, different inputs each time (stale partial sums would show): the first check
    # of a run compares with the all-zero accumulators, the later ones with the previous check
    out = torch.full((2, 2), -1.0, dtype=torch.float64, device=dev)
    got = []
    for now, prev in ((t[0], zero), (t[1], t[0]), (t[2], t[1]), (t[1], t[0])):
        emm.check_delta_static(now, prev, out=out)
        torch.cuda.synchronize()
        got.append(out.cpu().numpy().copy())
    # same fp64 sums, same block partition, same fixed order of the partial sums: equal to rounding (step-count parity in the
    # other tests rests on these numbers, so the tolerance is a few ulp, not a percentage)
    for q in range(3):
        assert np.allclose(got[q], ref[q], rtol=1e-13, atol=0.0), (q, got[q], ref[q])
    assert np.array_equal(got[3], got[1])                                               # and reproducible call after call
    assert np.allclose(got[0], 1.0, rtol=1e-13)                                         # ||C - 0|| / ||C||
    # sizes beyond the static scratch are refused with a clear error, before anything is launched
    too_many = torch.zeros((emm.CHECK_STATIC_MAX_NSRC + 1, 6, 8), dtype=torch.complex128, device=dev)
    with pytest.raises(emm.EmmError) as e:
        emm.check_delta_static(too_many, too_many)
    assert e.value.code == emm.EINVAL and "exceed the static scratch" in str(e.value)
    g.close()
