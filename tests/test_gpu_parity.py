"""Parity of the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs (-m gpu).

Tolerances (BASELINE.json north_star): FP64 per-event relative difference <= 1e-12 (1e-11 for gg -> ttbar ggg),
selected helicity / colour identical except within 1e-12 of a bin edge; FP32 and mixed: relative difference
<= 1e-3 for >= 99.9% of events with a median <= 1e-5.  ME parity always runs on bit-identical momenta
(SURVEY.md 8(c) C-R "parity protocol"); sampler parity is a separate test.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2507_21039_b200.workloads import WORKLOADS, SM_PARAMS, PRECISION_CODE

import os
import sys
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import parity_stats as PS  # noqa: E402  (tests/parity_stats.py: comparison records, appended to gpurun_out/parity_stats.jsonl)

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL64 = PS.TOL64


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2507_21039_b200 import binding
    binding.lib()
    return binding


def _ctx(B, cfg, prec="d"):
    return B.Context(WORKLOADS[cfg].process, SM_PARAMS, PRECISION_CODE[prec], 0)


def _check_fp64(orc, proc, p, me_gpu, me_orc, tol, what="parity test"):
    """FP64 comparator of SURVEY.md 8(c) C-T: events beyond `tol` are re-evaluated in extended precision; an event counts
    as ill-conditioned (recorded, not failed) only if the oracle's own FP64 value is as far from the extended value
    as the GPU's.  Configs 1-3 must not need the referee at all.  The record goes to gpurun_out/parity_stats.jsonl."""
    cfg = proc                                     # process ids equal config numbers (workloads.py)
    assert tol == PS.TOL64[cfg]
    rec = PS.record(PS.make_record(cfg, "d", p, me_gpu, me_orc, what))
    assert rec["referee_failed"] == 0, "gpu further from the extended-precision value than the oracle: %s" % rec.get("referee_failures")
    assert PS.passes(rec), rec
    return np.abs(me_gpu / me_orc - 1), rec["referee_exempted"]


def _check_selection(sel_gpu, r, w, mask, label):
    """Indices identical except for events within 1e-12 of a bin edge."""
    from oracle import binding as O
    ref = O.select(r, w, mask)
    diff = np.nonzero(sel_gpu != ref)[0]
    for i in diff:
        ww = w[i] * (mask if mask is not None else 1)
        T = ww.sum()
        edges = np.cumsum(ww)
        assert np.abs(r[i] * T - edges).min() <= 1e-12 * T, "%s index differs away from a bin edge (event %d)" % (label, i)
    return len(diff)


@pytest.mark.parametrize("cfg,nevt", [(1, 1000 + 37), (2, 2048 + 37), (3, 1024 + 37), (4, 512 + 37), (5, 96 + 5)])
@pytest.mark.parametrize("layout", ["aos", "aosoa"])
def test_fp64_parity_small_batches(B, orc, cfg, nevt, layout):
    """Element by element on a batch spanning several CTAs and a ragged tail."""
    wl = WORKLOADS[cfg]
    if layout == "aosoa":
        nevt = (nevt // 32) * 32
    p, _ = orc.rambo(wl.seed, 0, nevt, wl.final_masses, wl.sqrt_s)
    u = orc.uniforms(wl.seed, 0, nevt, 0, 1)
    ctx = _ctx(B, cfg)
    npar = p.shape[1]
    if layout == "aos":
        mom, lay = torch.tensor(p, device="cuda"), B.MG_LAYOUT_AOS
    else:
        mom = torch.tensor(p.reshape(nevt // 32, 32, npar, 4).transpose(0, 2, 3, 1).copy(), device="cuda")
        lay = B.MG_LAYOUT_AOSOA
    rh, rc = torch.tensor(u[:, 0].copy(), device="cuda"), torch.tensor(u[:, 1].copy(), device="cuda")
    ngood, good = ctx.filter_helicities(mom, nevt, layout=lay)
    me, sh, sc = ctx.compute(mom, nevt, layout=lay, rnd_hel=rh, rnd_col=rc)
    mh2g, wcg = ctx.last_details(nevt)
    torch.cuda.synchronize()
    ref, mh2, wcol = orc.matrix_elements(wl.process, p, sm=SM_PARAMS)
    gmask = np.frombuffer(good, np.uint8)
    assert np.array_equal(gmask, orc.filter_helicities(mh2))            # good-helicity mask: exact
    assert ngood == int(gmask.sum()) == {1: 4, 2: 16, 3: 32, 4: 64, 5: 128}[cfg]
    rel, ill = _check_fp64(orc, wl.process, p, me.cpu().numpy(), ref, TOL64[cfg], "small batch, layout %s" % layout)
    assert np.median(rel) < 1e-14
    # per-helicity values and colour-flow weights (what the selection is drawn from)
    assert np.abs(mh2g.cpu().numpy() - mh2).max(axis=1).max() <= 10 * TOL64[cfg] * mh2.sum(axis=1).max()
    assert (np.abs(mh2g.cpu().numpy() - mh2).max(axis=1) / mh2.sum(axis=1)).max() < 100 * TOL64[cfg]
    assert np.abs(wcg.cpu().numpy() / wcol - 1).max() < 1000 * TOL64[cfg]
    _check_selection(sh.cpu().numpy(), u[:, 0], mh2, gmask, "helicity")
    _check_selection(sc.cpu().numpy(), u[:, 1], wcol, None, "colour")
    ctx.close()


@pytest.mark.parametrize("cfg,prec", [(2, "f"), (3, "f"), (3, "m"), (4, "f"), (5, "f"), (2, "a"), (3, "a"), (4, "a"), (5, "a")])
def test_reduced_precision_parity(B, orc, cfg, prec):
    """FP32 (f), mixed (m) and all-FP32 (a: external wavefunctions and propagator denominators in FP32 too, reported beside f,
    SURVEY.md 8(c) C-M) against the FP64 oracle: <= 1e-3 for >= 99.9% of events, median <= 1e-5."""
    wl = WORKLOADS[cfg]
    # sizes at which ">= 99.9% of events" is resolved: the 2048-event oracle subset of config 5, 16384 events of config 4
    nevt = {2: 65536, 3: 32768, 4: 16384, 5: 2048}[cfg]
    rec = PS.record(PS.compare(cfg, prec, nevt, "first %d events, reduced precision" % nevt))
    assert rec["fraction_within_tol"] >= 0.999, "fraction within 1e-3: %.5f" % rec["fraction_within_tol"]
    assert rec["median_rel"] <= 1e-5, "median %.2e" % rec["median_rel"]


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_full_size_sampled_parity(B, orc, cfg):
    """BASELINE.json's full batch in the launch configuration bench.py times (device sampler -> compute), checked on
    sampled events the oracle evaluates one by one, plus properties that hold at any size."""
    wl = WORKLOADS[cfg]
    n = wl.nevt
    ctx = _ctx(B, cfg)
    mom, w = ctx.sample_rambo(wl.seed, 0, n, wl.sqrt_s)
    rh, rc = ctx.sample_uniforms(wl.seed, 0, n)
    nf = min(n, 16384)
    ngood, good = ctx.filter_helicities(mom, nf)
    me, sh, sc = ctx.compute(mom, n, rnd_hel=rh, rnd_col=rc)
    torch.cuda.synchronize()
    me = me.cpu().numpy()
    assert np.all(np.isfinite(me)) and np.all(me > 0)
    nsamp = {1: 256, 2: 256, 3: 128, 4: 64, 5: 24}[cfg]
    rng = np.random.default_rng(1234 + cfg)
    idx = np.unique(np.concatenate([[0, 1, n // 2, n - 2, n - 1], rng.integers(0, n, nsamp)]))
    p = mom[torch.tensor(idx, device="cuda")].cpu().numpy()             # bit-identical momenta
    ref, mh2, wcol = orc.matrix_elements(wl.process, p, sm=SM_PARAMS)
    _check_fp64(orc, wl.process, p, me[idx], ref, TOL64[cfg], "events sampled from the full batch (device sampler)")
    gmask = np.frombuffer(good, np.uint8)
    u = np.stack([rh.cpu().numpy()[idx], rc.cpu().numpy()[idx]], axis=1)
    _check_selection(sh.cpu().numpy()[idx], u[:, 0], mh2, gmask, "helicity")
    _check_selection(sc.cpu().numpy()[idx], u[:, 1], wcol, None, "colour")
    sh_all, sc_all = sh.cpu().numpy(), sc.cpu().numpy()
    assert sh_all.min() >= 0 and sh_all.max() < ctx.info.ncomb and np.all(gmask[sh_all] == 1)
    assert sc_all.min() >= 0 and sc_all.max() < ctx.info.ncolor
    ctx.close()


def test_ttggg_oracle_subset(B, orc):
    """Config 5: the 2048-event oracle subset of BASELINE.json (first 2048 global event indices), tolerance 1e-11."""
    wl = WORKLOADS[5]
    n = wl.oracle_events
    p, ref, _, _ = PS.oracle_batch(5, n)                   # shared with the FP32 test of the same subset
    ctx = _ctx(B, 5)
    mom = torch.tensor(p, device="cuda")
    ctx.filter_helicities(mom, n)
    me, _, _ = ctx.compute(mom, n)
    torch.cuda.synchronize()
    _check_fp64(orc, 5, p, me.cpu().numpy(), ref, TOL64[5], "the 2048-event oracle subset of BASELINE.json")
    ctx.close()


@pytest.mark.slow
@pytest.mark.parametrize("cfg,nevt", [(1, 16384), (2, 524288), (3, 524288), (4, 65536)])
def test_full_batch_parity(B, orc, cfg, nevt):
    """Every event of BASELINE.json's batch for configs 1-3 (65536 events of config 4) against the oracle: FP64 tolerance on
    each event, no extended-precision referee for configs 1-3 (minutes of oracle time on the host cores)."""
    rec = PS.record(PS.compare(cfg, "d", nevt, "full batch" if nevt == WORKLOADS[cfg].nevt else "first %d events" % nevt))
    assert rec["referee_failed"] == 0 and PS.passes(rec), rec


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_sampler_parity(B, orc, cfg):
    """Same Philox counters -> same uniforms (bit exact) and momenta equal to <= 1e-13 E per component, weights 1e-12."""
    wl = WORKLOADS[cfg]
    n, first = 4096 + 32, 1000
    ctx = _ctx(B, cfg)
    mom, w = ctx.sample_rambo(wl.seed, first, n, wl.sqrt_s)
    rh, rc = ctx.sample_uniforms(wl.seed, first, n)
    moma, _ = ctx.sample_rambo(wl.seed, first, n, wl.sqrt_s, layout=B.MG_LAYOUT_AOSOA)
    torch.cuda.synchronize()
    p, wr = orc.rambo(wl.seed, first, n, wl.final_masses, wl.sqrt_s)
    u = orc.uniforms(wl.seed, first, n, 0, 1)
    assert np.array_equal(rh.cpu().numpy(), u[:, 0]) and np.array_equal(rc.cpu().numpy(), u[:, 1])
    d = np.abs(mom.cpu().numpy() - p)
    # the rare n = 2 cancellation in Q^2 (SURVEY C-R) amplifies last-bit differences of log/sin/cos: bound the tail separately
    assert np.quantile(d, 0.999) <= 1e-13 * wl.sqrt_s and d.max() <= 1e-9 * wl.sqrt_s
    assert np.abs(w.cpu().numpy() / wr - 1).max() <= 1e-12
    npar = p.shape[1]
    assert torch.equal(moma, mom.reshape(n // 32, 32, npar, 4).permute(0, 2, 3, 1).contiguous())
    ctx.close()


def test_per_event_couplings_and_sharding(B, orc):
    """Couplings travel as per-event arrays; two shards by global event index reproduce one batch."""
    wl = WORKLOADS[3]
    n = 512
    ctx = _ctx(B, 3)
    mom, _ = ctx.sample_rambo(wl.seed, 0, n, wl.sqrt_s)
    gs0 = orc.sm_derive(SM_PARAMS)["gs"]
    gs = torch.tensor(gs0 * (1 + 0.1 * np.sin(np.arange(n))), device="cuda")
    ctx.filter_helicities(mom, n, gs=gs)
    me, _, _ = ctx.compute(mom, n, gs=gs)
    me0, _, _ = ctx.compute(mom, n)
    torch.cuda.synchronize()
    ref, _, _ = orc.matrix_elements(3, mom.cpu().numpy(), sm=SM_PARAMS, gs=gs.cpu().numpy())
    assert np.abs(me.cpu().numpy() / ref - 1).max() < 1e-12
    assert np.abs((me / me0).cpu().numpy() / (gs.cpu().numpy() / gs0) ** 6 - 1).max() < 1e-13     # |M|^2 ~ g_s^(2 n_g)
    from paper_2507_21039_b200 import sharding
    parts = []
    for r in range(2):
        first, cnt = sharding.shard_range(n, r, 2)
        m2, _ = ctx.sample_rambo(wl.seed, first, cnt, wl.sqrt_s)
        a, _, _ = ctx.compute(m2, cnt)
        parts.append(a)
    torch.cuda.synchronize()
    assert torch.equal(torch.cat(parts), me0)
    ctx.close()


def test_merged_mask_streams_and_details(B, orc):
    """(1) a good-helicity mask agreed between ranks can be installed (mg_set_good_helicities) and the helicity
    sum then runs over exactly that mask; (2) calls on one context from different streams are ordered by the library;
    (3) mg_get_last_details returns flow weights that carry the per-event couplings."""
    wl = WORKLOADS[1]
    n = 4096
    ctx = _ctx(B, 1)
    mom, _ = ctx.sample_rambo(wl.seed, 0, n, wl.sqrt_s)
    ngood, good = ctx.filter_helicities(mom, n)
    assert ngood == 4
    me, _, _ = ctx.compute(mom, n)
    mh2, _ = ctx.last_details(n)
    # two "ranks" that saw different halves of the good helicities: the union gives the full result, a half gives its partial sum
    half = bytearray(16)
    half[5] = half[6] = 1
    assert ctx.set_good_helicities(bytes(half)) == 2
    me_half, _, _ = ctx.compute(mom, n)
    torch.cuda.synchronize()
    assert np.allclose(me_half.cpu().numpy(), mh2.cpu().numpy()[:, [5, 6]].sum(axis=1) / 4, rtol=1e-15)
    other = bytearray(16)
    other[9] = other[10] = 1
    union = bytes(a | b for a, b in zip(half, other))
    assert union == good and ctx.set_good_helicities(union) == 4
    me_union, _, _ = ctx.compute(mom, n)
    assert torch.equal(me_union, me)
    lib = B.lib()
    assert lib.mg_set_good_helicities(ctx._h, bytes(16), None) == B.MG_EINVAL          # empty mask
    assert lib.mg_set_good_helicities(ctx._h, bytes([2] * 16), None) == B.MG_EINVAL     # not 0 / 1
    ctx.close()
    # (2) back-to-back calls on two streams without any synchronisation in between
    wl = WORKLOADS[4]
    ctx = _ctx(B, 4)
    n = 2048
    moms = [ctx.sample_rambo(wl.seed, k * n, n, wl.sqrt_s)[0] for k in range(2)]
    ctx.filter_helicities(moms[0], n)
    ref = [ctx.compute(m, n)[0].clone() for m in moms]
    torch.cuda.synchronize()
    outs = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(2)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for rep in range(3):
        for k in range(2):
            with torch.cuda.stream(streams[k]):
                ctx.compute(moms[k], n, me=outs[k])
    torch.cuda.synchronize()
    assert torch.equal(outs[0], ref[0]) and torch.equal(outs[1], ref[1])
    # (3) flow weights with per-event couplings
    gs0 = orc.sm_derive(SM_PARAMS)["gs"]
    gs = torch.tensor(gs0 * (1 + 0.1 * np.cos(np.arange(n))), device="cuda")
    ctx.compute(moms[0], n, gs=gs)
    _, wc = ctx.last_details(n)
    ctx.compute(moms[0], n)
    _, wc0 = ctx.last_details(n)
    torch.cuda.synchronize()
    ratio = (wc / wc0).cpu().numpy() / ((gs.cpu().numpy() / gs0) ** 8)[:, None]
    assert np.abs(ratio - 1).max() < 1e-13
    ctx.close()


def test_edge_cases_and_errors(B):
    lib = B.lib()
    ctx = _ctx(B, 2)
    mom, _ = ctx.sample_rambo(2, 0, 64, 1500.0)
    me = torch.empty(64, dtype=torch.float64, device="cuda")
    args = (ctx._h, C.c_void_p(mom.data_ptr()), None, None, None)
    # compute before the helicity filter
    assert lib.mg_compute(*args, 64, 0, C.c_void_p(me.data_ptr()), None, None, None) == B.MG_ENOTFILTERED
    assert lib.mg_filter_helicities(ctx._h, C.c_void_p(mom.data_ptr()), None, 0, 0, 0.0, None, None, None) == B.MG_EINVAL   # empty first batch
    ctx.filter_helicities(mom, 64)
    # empty batch is a no-op; AOSOA needs whole pages; NULL pointers and negative sizes are rejected
    assert lib.mg_compute(*args, 0, 0, C.c_void_p(me.data_ptr()), None, None, None) == 0
    assert lib.mg_compute(*args, 33, B.MG_LAYOUT_AOSOA, C.c_void_p(me.data_ptr()), None, None, None) == B.MG_EINVAL
    assert lib.mg_compute(*args, -1, 0, C.c_void_p(me.data_ptr()), None, None, None) == B.MG_EINVAL
    assert lib.mg_compute(*args, 64, 0, None, None, None, None) == B.MG_EINVAL
    assert lib.mg_compute(ctx._h, None, None, None, None, 64, 0, C.c_void_p(me.data_ptr()), None, None, None) == B.MG_EINVAL
    assert lib.mg_sample_rambo(ctx._h, 1, 0, 33, 1500.0, B.MG_LAYOUT_AOSOA, C.c_void_p(mom.data_ptr()), None, None) == B.MG_EINVAL
    # single event, no selection
    a, sh, sc = ctx.compute(mom, 1)
    b, _, _ = ctx.compute(mom, 64)
    torch.cuda.synchronize()
    assert sh is None and sc is None and a[0].item() == b[0].item()
    # host-buffer entry point gives the same numbers
    hm = mom.cpu().pin_memory()
    hme, _, _ = ctx.compute_host(hm, 64)
    assert torch.equal(hme, b.cpu())
    # selection with r -> 0 and r -> 1 stays inside the table
    r0 = torch.full((64,), 1e-300, dtype=torch.float64, device="cuda")
    r1 = torch.full((64,), 1 - 2.0 ** -53, dtype=torch.float64, device="cuda")
    _, s0, c0 = ctx.compute(mom, 64, rnd_hel=r0, rnd_col=r0)
    _, s1, c1 = ctx.compute(mom, 64, rnd_hel=r1, rnd_col=r1)
    torch.cuda.synchronize()
    assert int(s0.min()) >= 0 and int(s1.max()) < 16 and int(c0.min()) >= 0 and int(c1.max()) < 2
    ctx.close()


@pytest.mark.parametrize("cfg,nevt", [(2, 3 * 8192 + 1000), (4, 2 * 8192 + 96), (1, 5000)])
def test_host_bridge_layouts_and_chunks(B, cfg, nevt):
    """mg_compute_host: chunked two-lane pipeline, AOS / AOSOA / column-major (SOA) host layouts, pinned and
    pageable buffers -- bit-identical to mg_compute on device buffers, several chunks and a ragged last one."""
    wl = WORKLOADS[cfg]
    ctx = _ctx(B, cfg)
    nevt = (nevt // 32) * 32
    mom, _ = ctx.sample_rambo(wl.seed, 0, nevt, wl.sqrt_s)
    rh, rc = ctx.sample_uniforms(wl.seed, 0, nevt)
    gs = torch.full((nevt,), 1.2177157847767197, dtype=torch.float64, device="cuda") * (1 + 0.1 * torch.rand(nevt, dtype=torch.float64, device="cuda"))
    ctx.filter_helicities(mom, 4096)
    me, sh, sc = ctx.compute(mom, nevt, gs=gs if cfg > 1 else None, rnd_hel=rh, rnd_col=rc)
    torch.cuda.synchronize()
    npar = mom.shape[1]
    hosts = {
        B.MG_LAYOUT_AOS: mom.cpu(),
        B.MG_LAYOUT_AOSOA: mom.cpu().reshape(nevt // 32, 32, npar, 4).permute(0, 2, 3, 1).contiguous(),
        B.MG_LAYOUT_SOA: mom.cpu().permute(2, 1, 0).contiguous(),            # [4][npar][nevt]
    }
    for lay, hm in hosts.items():
        for pin in (True, False):
            f = (lambda t: t.pin_memory()) if pin else (lambda t: t)
            hme, hsh, hsc = ctx.compute_host(f(hm), nevt, layout=lay, gs=f(gs.cpu()) if cfg > 1 else None, rnd_hel=f(rh.cpu()), rnd_col=f(rc.cpu()),
                                             me=f(torch.zeros(nevt, dtype=torch.float64)), sel_hel=f(torch.zeros(nevt, dtype=torch.int32)),
                                             sel_col=f(torch.zeros(nevt, dtype=torch.int32)))
            assert torch.equal(hme, me.cpu()), (cfg, lay, pin)
            assert torch.equal(hsh, sh.cpu()) and torch.equal(hsc, sc.cpu()), (cfg, lay, pin)
    ctx.close()


@pytest.mark.parametrize("cfg,nevt", [(2, 2048 + 37), (3, 1024 + 37), (4, 512 + 37), (5, 64 + 5)])
def test_multichannel_parity(B, orc, cfg, nevt):
    """mg_compute_multichannel: numerator |A_k|^2 and denominator sum_k |A_k|^2 per event against the oracle's
    per-diagram evaluation, a channel per 32-event block; ME unchanged; colour selected among the channel's flows."""
    wl = WORKLOADS[cfg]
    tol = TOL64[cfg]
    p, _ = orc.rambo(wl.seed, 0, nevt, wl.final_masses, wl.sqrt_s)
    u = orc.uniforms(wl.seed, 0, nevt, 0, 1)
    names = orc.channels(wl.process)
    ctx = _ctx(B, cfg)
    assert ctx.info.nchannel == len(names)
    nblock = (nevt + 31) // 32
    rng = np.random.default_rng(cfg)
    chan = rng.integers(1, len(names) + 1, size=nblock).astype(np.int32)
    chan[0], chan[-1] = 1, len(names)
    if nblock > 3:
        chan[2] = 0                                        # a block without a channel
    mom = torch.tensor(p, device="cuda")
    rh, rc = torch.tensor(u[:, 0].copy(), device="cuda"), torch.tensor(u[:, 1].copy(), device="cuda")
    ngood, good = ctx.filter_helicities(mom, nevt)
    me0, sh0, sc0 = ctx.compute(mom, nevt, rnd_hel=rh, rnd_col=rc)
    me, sh, sc, num, den = ctx.compute_multichannel(mom, nevt, torch.tensor(chan, device="cuda"), rnd_hel=rh, rnd_col=rc)
    torch.cuda.synchronize()
    assert torch.equal(me, me0) and torch.equal(sh, sh0)
    c2 = orc.channel_sums(wl.process, p, sm=SM_PARAMS, good=np.frombuffer(good, np.uint8))
    evchan = np.repeat(chan, 32)[:nevt]
    ref_den = c2.sum(axis=1)
    ref_num = np.where(evchan > 0, c2[np.arange(nevt), np.maximum(evchan, 1) - 1], 0.0)
    num, den = num.cpu().numpy(), den.cpu().numpy()
    assert np.abs(den / ref_den - 1).max() <= tol, np.abs(den / ref_den - 1).max()
    assert np.all(num[evchan == 0] == 0)
    k = evchan > 0
    assert np.abs(num[k] / ref_num[k] - 1).max() <= 10 * tol, np.abs(num[k] / ref_num[k] - 1).max()    # a single diagram can be small against the sum
    assert np.all(num <= den * (1 + 1e-14))
    # colour: among the flows of the channel, first-above rule (bin-edge exemption as everywhere)
    _, _, wcol = orc.matrix_elements(wl.process, p, sm=SM_PARAMS)
    allowed = orc.channel_flows(wl.process)
    sc = sc.cpu().numpy()
    for b in range(nblock):
        sl = slice(32 * b, min(32 * b + 32, nevt))
        mask = allowed[chan[b] - 1] if chan[b] > 0 else None
        _check_selection(sc[sl], u[sl, 1], wcol[sl], mask, "colour (channel %d)" % chan[b])
        if mask is not None:
            assert np.all(mask[sc[sl]] == 1)
    ctx.close()


def test_input_validation(B):
    """mg_sample_rambo rejects sqrt_s at or below the sum of the final-state masses; mg_create rejects non-physical SM inputs."""
    ctx = _ctx(B, 2)
    lib = B.lib()
    mom = torch.zeros((64, 4, 4), dtype=torch.float64, device="cuda")
    for bad in (346.0, 100.0, float("nan")):
        rc = lib.mg_sample_rambo(ctx._h, 1, 0, 64, bad, 0, C.c_void_p(mom.data_ptr()), None, None)
        assert rc == B.MG_EINVAL and b"final-state masses" in lib.mg_strerror(rc)
    assert lib.mg_sample_rambo(ctx._h, 1, 0, 64, 346.5, 0, C.c_void_p(mom.data_ptr()), None, None) == 0
    torch.cuda.synchronize()
    assert torch.isfinite(mom).all()
    ctx.close()
    h = C.c_void_p()
    for k, v in ((2, -1.0), (4, 0.0), (5, 0.0), (6, -0.1), (0, float("nan")), (5, 1e-9)):     # MT < 0, 1/alpha = 0, G_F = 0, alpha_s < 0, MZ nan, MW^2 complex
        vals = list(SM_PARAMS)
        vals[k] = v
        assert lib.mg_create(C.byref(h), 2, C.byref(B.mg_sm_params(*vals)), 0, 0) == B.MG_EINVAL, (k, v)


@pytest.mark.parametrize("cfg,nevt", [(6, 2048 + 37), (7, 2048 + 37), (8, 1024 + 37), (9, 512 + 37)])
def test_drell_yan_parity(B, orc, cfg, nevt):
    """u u~ -> e+ e- + n g: ME, per-helicity values, good-helicity mask (exact zeros for the
    chirality-violating combinations), colour-flow weights and the selected indices against the oracle."""
    wl = WORKLOADS[cfg]
    p, _ = orc.rambo(wl.seed, 0, nevt, wl.final_masses, wl.sqrt_s)
    u = orc.uniforms(wl.seed, 0, nevt, 0, 1)
    ctx = _ctx(B, cfg)
    info = ctx.info
    n = cfg - 6
    assert (info.npar, info.ndiag, info.ncolor, info.ncomb, info.denom) == (4 + n, (1, 2, 8, 50)[n], (1, 1, 2, 6)[n], 16 << n, 36 * (1, 1, 2, 6)[n])
    mom = torch.tensor(p, device="cuda")
    rh, rc = torch.tensor(u[:, 0].copy(), device="cuda"), torch.tensor(u[:, 1].copy(), device="cuda")
    ngood, good = ctx.filter_helicities(mom, nevt)
    me, sh, sc = ctx.compute(mom, nevt, rnd_hel=rh, rnd_col=rc)
    mh2g, wcg = ctx.last_details(nevt)
    torch.cuda.synchronize()
    ref, mh2, wcol = orc.matrix_elements(wl.process, p, sm=SM_PARAMS)
    gmask = np.frombuffer(good, np.uint8)
    assert np.array_equal(gmask, orc.filter_helicities(mh2)) and ngood == 4 << n     # opposite helicities on both fermion lines
    assert np.all(mh2g.cpu().numpy()[:, gmask == 0] == 0)
    _check_fp64(orc, wl.process, p, me.cpu().numpy(), ref, TOL64[cfg], "Drell-Yan small batch")
    assert (np.abs(mh2g.cpu().numpy() - mh2).max(axis=1) / mh2.sum(axis=1)).max() < 100 * TOL64[cfg]
    if info.ncolor > 1:
        assert np.abs(wcg.cpu().numpy() / wcol - 1).max() < 1000 * TOL64[cfg]
    _check_selection(sh.cpu().numpy(), u[:, 0], mh2, gmask, "helicity")
    _check_selection(sc.cpu().numpy(), u[:, 1], wcol, None, "colour")
    # the device sampler and FP32 on the same process
    m2, _ = ctx.sample_rambo(wl.seed, 0, nevt, wl.sqrt_s)
    torch.cuda.synchronize()
    assert np.abs(m2.cpu().numpy() - p).max() <= 1e-12 * wl.sqrt_s
    ctx.close()
    rec = PS.record(PS.compare(cfg, "f", nevt, "Drell-Yan, FP32"))
    assert rec["fraction_within_tol"] >= 0.999 and rec["median_rel"] <= 1e-5, rec


@pytest.mark.parametrize("cfg,nevt,prec", [(2, 8388608 + 37, "d"), (3, 4194304 + 37, "d"), (4, 2097152 + 5, "d"), (5, 262144 + 3, "d"),
                                             (9, 1048576 + 5, "d"), (4, 1048576 + 5, "f")])
def test_large_batches(B, orc, cfg, nevt, prec):
    """Maximum sizes: batches 4 to 16 times the BASELINE.json size with a ragged tail (index arithmetic in 64 bits, workspace growth):
    the first, middle and last events against the oracle (momenta from the device sampler, oracle momenta for the same indices)."""
    wl = WORKLOADS[cfg]
    ctx = _ctx(B, cfg, prec)
    mom, _ = ctx.sample_rambo(wl.seed, 0, nevt, wl.sqrt_s)
    ctx.filter_helicities(mom, 8192)
    me, _, _ = ctx.compute(mom, nevt)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(me).all()) and bool((me > 0).all())
    n = 128
    for first in (0, nevt // 2 - 50, nevt - n):
        p, _ = orc.rambo(wl.seed, first, n, wl.final_masses, wl.sqrt_s)
        ref, _, _ = orc.matrix_elements(wl.process, p, sm=SM_PARAMS)
        rel = np.abs(me[first:first + n].cpu().numpy() / ref - 1)
        # the device sampler's momenta differ from the oracle's by <= 1e-13 E (test_sampler_parity), which the matrix element amplifies
        assert rel.max() <= (1e-10 if prec == "d" else 1e-3), (cfg, first, rel.max())
    ctx.close()
    del mom, me
    torch.cuda.empty_cache()


def test_native_library_is_loaded(B):
    maps = open("/proc/self/maps").read()
    assert "libmg5b200.so" in maps
