"""mg_compute_noalloc (include/mg5b200.h): the no-allocation variant of mg_compute must give mg_compute's results.

Collected last on purpose (the suite runs with pytest -x).  Two calls in a row share the library's static scratch
array, the second with another batch size and other momenta, so stale contents of the first call would show.
Tolerance: the 1e-12 of the FP64 parity tests (the kernels are the same, so the values are in fact identical).
"""
import ctypes as C

import numpy as np
import pytest

from paper_2507_21039_b200.workloads import WORKLOADS, SM_PARAMS, PRECISION_CODE

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2507_21039_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("cfg,sizes", [(1, (1000, 517)), (2, (4096 + 37, 1001)), (4, (512 + 37, 160)), (5, (96, 37))])
def test_noalloc_matches_compute_on_two_calls_in_a_row(B, cfg, sizes):
    wl = WORKLOADS[cfg]
    ctx = B.Context(wl.process, SM_PARAMS, PRECISION_CODE["d"], 0)
    ref = B.Context(wl.process, SM_PARAMS, PRECISION_CODE["d"], 0)
    first = 0
    for call, nevt in enumerate(sizes):
        mom, _ = ctx.sample_rambo(wl.seed, first, nevt, wl.sqrt_s)
        rh, rc = ctx.sample_uniforms(wl.seed, first, nevt)
        if call == 0:
            _, good = ref.filter_helicities(mom, nevt)
            ctx.set_good_helicities(good)
        me0, sh0, sc0 = ref.compute(mom, nevt, rnd_hel=rh, rnd_col=rc)
        me = torch.full((nevt,), -1.0, dtype=torch.float64, device="cuda")
        sh = torch.full((nevt,), -1, dtype=torch.int32, device="cuda")
        sc = torch.full((nevt,), -1, dtype=torch.int32, device="cuda")
        ctx.compute_noalloc(mom, nevt, me, rnd_hel=rh, rnd_col=rc, sel_hel=sh, sel_col=sc)
        torch.cuda.synchronize()
        a, b = me.cpu().numpy(), me0.cpu().numpy()
        assert np.all(np.isfinite(a)) and np.all(a > 0)
        assert np.abs(a / b - 1).max() <= 1e-12, (cfg, call, np.abs(a / b - 1).max())
        assert torch.equal(sh, sh0) and torch.equal(sc, sc0)
        first += nevt
    ctx.close()
    ref.close()


def test_noalloc_rejects_batches_beyond_the_static_scratch(B):
    wl = WORKLOADS[5]
    ctx = B.Context(wl.process, SM_PARAMS, PRECISION_CODE["d"], 0)
    nmax = ctx.noalloc_max_events()
    assert nmax == 8456
    n = nmax + 1
    mom, _ = ctx.sample_rambo(wl.seed, 0, n, wl.sqrt_s)
    ctx.filter_helicities(mom, 64)
    me = torch.zeros(n, dtype=torch.float64, device="cuda")
    lib = B.lib()
    rc = lib.mg_compute_noalloc(ctx._h, C.c_void_p(mom.data_ptr()), None, None, None, n, 0, C.c_void_p(me.data_ptr()), None, None, None)
    assert rc == B.MG_EINVAL
    msg = lib.mg_strerror(rc).decode()
    assert "at most 8456 events" in msg and "mg_compute_noalloc" in msg
    # the largest batch that fits runs and agrees with mg_compute
    ctx.compute_noalloc(mom, nmax, me)
    me0, _, _ = ctx.compute(mom, nmax)
    torch.cuda.synchronize()
    assert np.abs(me[:nmax].cpu().numpy() / me0.cpu().numpy() - 1).max() <= 1e-12
    ctx.close()
