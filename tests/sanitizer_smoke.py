"""Small invocation of every process through the C ABI, meant to be run under compute-sanitizer:
    compute-sanitizer --tool memcheck  python tests/sanitizer_smoke.py
    compute-sanitizer --tool racecheck python tests/sanitizer_smoke.py
(not collected by pytest; exits non-zero on a CUDA error)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import torch  # noqa: E402
from paper_2507_21039_b200 import binding as B  # noqa: E402
from paper_2507_21039_b200.workloads import WORKLOADS, SM_PARAMS, PRECISION_CODE  # noqa: E402

for cfg, nevt in ((1, 40), (2, 40), (3, 24), (4, 12), (5, 3)):
    wl = WORKLOADS[cfg]
    for prec in wl.precisions:
        ctx = B.Context(wl.process, SM_PARAMS, PRECISION_CODE[prec], 0)
        mom, w = ctx.sample_rambo(wl.seed, 0, nevt, wl.sqrt_s)
        rh, rc = ctx.sample_uniforms(wl.seed, 0, nevt)
        ctx.filter_helicities(mom, nevt)
        me, sh, sc = ctx.compute(mom, nevt, rnd_hel=rh, rnd_col=rc)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(me).all()) and bool((me > 0).all())
        print("cfg%d %s ok: %d events" % (cfg, prec, nevt), flush=True)
        ctx.close()
print("sanitizer smoke done")
