"""Host logic of the CUDA path: the emitter's diagram/colour tables and the scheduled task program."""
import numpy as np
import pytest

from paper_2507_21039_b200.emitter import diagrams as D
from paper_2507_21039_b200.emitter import emit
from paper_2507_21039_b200.emitter import program as PR
from paper_2507_21039_b200.workloads import WORKLOADS, SM_PARAMS

import vm_sim


@pytest.fixture(scope="module")
def programs():
    return {ng: emit.build_program(ng) for ng in (2, 3, 4, 5)}


def test_diagram_counts():
    # BASELINE.json: 3 / 16 / 123 / 1240 diagrams; SURVEY C-D: 3 / 18 / 159 / 1890 amplitudes; subtrees 1, 1, 4, 25, 220
    expect = {2: (3, 3), 3: (16, 18), 4: (123, 159), 5: (1240, 1890)}
    for ng, e in expect.items():
        ts = D.TreeSet(ng)
        assert D.count_diagrams(ts) == e
    ts = D.TreeSet(5)
    unexp = [sum(1 for i in range(ts.ntrees(m)) if ts.first_structure_only(m, i)) for m in (1, 3, 7, 15, 31)]
    assert unexp == [1, 1, 4, 25, 220]
    assert [ts.ntrees(m) for m in (1, 3, 7, 15, 31)] == [1, 1, 6, 45, 510]


@pytest.mark.parametrize("ng,den", [(2, 3), (3, 9), (4, 54), (5, 324)])
def test_colour_matrix_fierz_vs_gell_mann(orc, ng, den):
    # emitter: exact Fierz reduction; oracle: explicit Gell-Mann matrices -- two independent computations
    num, d = D.colour_matrix_integer(ng)
    assert d == den
    C = orc.colour_matrix(ng, full=(ng <= 4))
    assert np.abs(np.array(num) / den - C).max() < 1e-9
    assert np.abs(np.array(num)).max() <= 4096


def test_kappa_values_and_flow_counts():
    for ng in (2, 3, 4, 5):
        ts = D.TreeSet(ng)
        for m in range(1, 1 << ng):
            for i in range(ts.ntrees(m)):
                poly = ts.colour(m, i)
                assert set(poly.values()) <= {1, -1, 1j, -1j}
                assert len(poly) == 2 ** (bin(m).count("1") - 1)      # a block of k gluons touches 2^(k-1) orderings


def test_ordered_basis_regroups_the_colour_dressed_current():
    """sum_tree C_tree x_tree == sum_ordering C_ordering (sum_tree sign x_tree) for arbitrary tree values x: the ordered
    currents are an exact regrouping; k!/2 orderings with two T-strings each, related by reversal with (-1)^(k-1)."""
    rng = np.random.default_rng(5)
    ts = D.TreeSet(5, merged=True)
    for mask, nord in ((0b111, 3), (0b10110, 3), (0b1111, 12), (0b11101, 12)):
        perms, comb = ts.ordered_basis(mask)
        k = bin(mask).count("1")
        assert len(perms) == nord and all(p[0] < p[-1] for p in perms)
        x = rng.normal(size=ts.ntrees(mask)) + 1j * rng.normal(size=ts.ntrees(mask))
        dressed = {}
        for i in range(ts.ntrees(mask)):
            for p, c in ts.colour(mask, i).items():
                dressed[p] = dressed.get(p, 0) + c * x[i]
        regrouped = {}
        for o, terms in enumerate(comb):
            val = sum(sg * x[i] for i, sg in terms)
            poly = ts.colour_ordered(mask, o)
            assert len(poly) == 2 and poly[perms[o][::-1]] == poly[perms[o]] * (-1) ** (k - 1)
            for p, c in poly.items():
                regrouped[p] = regrouped.get(p, 0) + c * val
        assert set(dressed) == set(regrouped)
        assert max(abs(dressed[p] - regrouped[p]) for p in dressed) < 1e-12


def _jamp_owners_ok(P):
    """Emitted unit lists: within a phase two units that add into the same jamp storage slot run in the SAME warp (a warp's units
    run in order, csrc/mg_vm.cuh __syncwarp): an accumulation unit and the closing sums of its flows."""
    stats = []
    emit.emit_program(P, "chk", stats=stats)
    nshared = 0
    for st in stats:
        owner = {}
        for w, units in enumerate(st.get("jamp_units", [])):
            for pos, (ty, slots) in enumerate(units):
                for sl in slots:
                    if sl in owner:
                        w0, ty0 = owner[sl]
                        assert w0 == w and {ty0, ty} == {PR.T_ACC, PR.T_QSUM}, (sl, w0, w, ty0, ty)
                        nshared += 1
                    else:
                        owner[sl] = (w, ty)
    return nshared


def _hazard_free(P):
    """Inside one phase no task reads a slot or amplitude column written in that phase and no two tasks write the same one."""
    for phase in P.phases:
        w_slots, w_cols = set(), set()
        reads_s, reads_c = set(), set()
        j_flows, acc_slots = set(), set()
        for t in phase:
            if t["type"] == PR.T_ACC:
                for lst in t["lists"]:
                    reads_c |= {c for c, _ in lst}
                continue
            n = t["nitems"]
            if t["type"] == PR.T_COMB:
                for q in range(PR.COMB_MAX):
                    sel = (t["idx"][:, PR.COMB_MAX] & 7) > q
                    reads_s |= set((t["in_base"][0] + t["idx"][sel, q]).tolist())
                out = set(range(t["out_base"], t["out_base"] + n))
                assert not (out & w_slots)
                w_slots |= out
                continue
            if t["type"] == PR.T_QSUM:
                # colour-ordered quark line: (row spinor, current) pairs of both row sums, R1 for both t~ helicities, v
                ix = t["idx"]
                for c, base in zip(t["in_cols"], t["in_base"]):
                    if c < 2 * PR.QSUM_MAX:
                        sel = (ix[:, PR.QS_FLAGS_A] & 15) > c // 2
                    elif c < PR.QS_R1:
                        sel = (ix[:, PR.QS_FLAGS_B] & 15) > (c - 2 * PR.QSUM_MAX) // 2
                    else:
                        sel = np.ones(n, dtype=bool)
                    reads_s |= set((base + ix[sel, c]).tolist())
                    if c == PR.QS_R1:
                        reads_s |= set((base + ix[:, c] + (1 << ix[:, PR.QS_SH_TB])).tolist())
                    if c == PR.QS_V:
                        reads_s.add(base + 1)
                if t["aux"] & 1:
                    # closing sums add into jamp: one task per flow; beside an accumulation task only in a program that was built
                    # for it (then the emitted unit lists are checked by _jamp_owners_ok: same warp, after the accumulation unit)
                    assert t["flow"] not in j_flows and (P.fuse_closing or not any(u["type"] == PR.T_ACC for u in phase))
                    j_flows.add(t["flow"])
                else:
                    out = set(range(t["out_base"], t["out_base"] + n))
                    assert not (out & w_slots)
                    w_slots |= out
                continue
            if t["type"] == PR.T_VVVF:
                # fused tree current: the two children's currents and the children of its composite children
                reads_s |= set((t["in_base"][0] + t["idx"][:, 0]).tolist()) | set((t["in_base"][1] + t["idx"][:, 1]).tolist())
                for q in range(2):
                    sel = ((t["xflags"] >> (2 * q)) & 1) == 1
                    reads_s |= set(t["xslots"][sel, 2 * q].tolist()) | set(t["xslots"][sel, 2 * q + 1].tolist())
                out = set(range(t["out_base"], t["out_base"] + n))
                assert not (out & w_slots)
                w_slots |= out
                continue
            nin = {PR.T_EXT: 0, PR.T_VVV: 2, PR.T_VVVV: 3, PR.T_FFV: 2, PR.T_FFVR: 2, PR.T_WCUR: 2, PR.T_AMP_DOT: 2, PR.T_AMP_FFV: 3,
                   PR.T_AMP_VVV: 2, PR.T_AMP_VVVV: 3}[t["type"]]
            for k in range(nin):
                reads_s |= set((t["in_base"][k] + t["idx"][:, k]).tolist())
            if t["type"] == PR.T_AMP_VVVV and (t["aux"] & 4):
                cols = set(t["col_of_item"].tolist())          # folded top level: adds into columns stored in an earlier phase
                assert not (cols & w_cols)
                w_cols |= cols
            elif t["type"] in (PR.T_AMP_DOT, PR.T_AMP_FFV, PR.T_AMP_VVV, PR.T_AMP_VVVV):
                cols = set(range(t["out_base"], t["out_base"] + n // t["rpc"]))
                assert not (cols & w_cols)
                w_cols |= cols
            elif t["type"] == PR.T_VVVV and (t["aux"] & 4):
                out = set((t["out_base"] + (t["idx"][:, 3] & 0x7fff)).tolist())
                assert len(out) == n
                # read-modify-write: the targets were stored in an earlier phase and no other task of this phase touches them
                assert not (out & w_slots) and not (out & acc_slots)
                acc_slots |= out
                w_slots |= out
            else:
                out = set(range(t["out_base"], t["out_base"] + n))
                assert not (out & w_slots)
                w_slots |= out
        assert not (reads_s & w_slots) and not (reads_c & w_cols)
        assert max(w_slots | {0}) < P.nslot and max(w_cols | {0}) < P.ncol


def _task_reads(t):
    """wavefunction slots a slot-producing task reads (the same rules as _hazard_free)."""
    ix, n = t["idx"], t["nitems"]
    if t["type"] == PR.T_COMB:
        return set().union(*[set((t["in_base"][0] + ix[(ix[:, PR.COMB_MAX] & 7) > q, q]).tolist()) for q in range(PR.COMB_MAX)])
    if t["type"] == PR.T_QSUM:
        r = set()
        for c, base in zip(t["in_cols"], t["in_base"]):
            r |= set((base + ix[(ix[:, PR.QS_FLAGS_A] & 15) > c // 2, c]).tolist())
        return r
    r = set((t["in_base"][0] + ix[:, 0]).tolist()) | set((t["in_base"][1] + ix[:, 1]).tolist())
    if t["type"] == PR.T_VVVF:
        for q in range(2):
            sel = ((t["xflags"] >> (2 * q)) & 1) == 1
            r |= set(t["xslots"][sel, 2 * q].tolist()) | set(t["xslots"][sel, 2 * q + 1].tolist())
    return r


def test_pass_invariant_tasks(programs):
    """Tasks marked first_only (run in the first outer-helicity pass only when the kernel keeps the wavefunction file) read only
    external wavefunctions of inner legs and results of other such tasks, and nothing else ever writes their slots."""
    for ng in (4, 5):
        P = programs[ng]
        inv, other_writes, nfirst = set(), set(), 0
        for phase in P.phases:
            for t in phase:
                if t["type"] == PR.T_EXT:
                    legs = t["idx"][:, 0]
                    out = set(range(t["out_base"], t["out_base"] + t["nitems"]))
                    if all(int(l) in P.inner for l in legs):
                        inv |= out
                    else:
                        other_writes |= out
                elif t.get("first_only"):
                    assert t["type"] in (PR.T_VVVF, PR.T_QSUM, PR.T_FFVR, PR.T_WCUR, PR.T_COMB) and not t["aux"] & 1
                    assert _task_reads(t) <= inv
                    inv |= set(range(t["out_base"], t["out_base"] + t["nitems"]))
                    nfirst += t["nitems"]
                elif "out_base" in t and t["type"] in (PR.T_VVV, PR.T_VVVF, PR.T_FFV, PR.T_FFVR, PR.T_WCUR, PR.T_COMB) or (t["type"] == PR.T_QSUM and not t["aux"] & 1):
                    other_writes |= set(range(t["out_base"], t["out_base"] + t["nitems"]))
        assert nfirst == {4: 136, 5: 232}[ng] and not (inv & other_writes)
        # skipping them in the later passes would remove 3.3% (gg->ttgg) / 1.4% (gg->ttggg) of an event's flops: why it buys nothing
        assert 0 < P.first_only_flops * (P.nouter - 1) < 0.04 * P.flops_executed_per_event()
        assert P.flops_executed_per_event(True) == P.flops_executed_per_event() - P.first_only_flops * (P.nouter - 1)


def test_program_structure(programs):
    # (flow, column) pairs: gg->ttgg and gg->ttggg keep amplitude columns only for the single-block diagrams (the quark line with
    # two or more blocks is the colour-ordered recursion, emitter/program.py _chains_bg)
    pairs = {2: 4, 3: 42, 4: 216, 5: 1920}
    for ng, P in programs.items():
        _hazard_free(P)
        # gg->ttggg: the closing sums share a phase with an accumulation task; every flow's closing sum follows its accumulation unit
        # in the same warp
        assert _jamp_owners_ok(P) == (P.ncolor if P.fuse_closing else 0) and P.fuse_closing == (ng == 5)
        assert P.acc_pairs == pairs[ng]
        ncols = sum(t["nitems"] // t["rpc"] for ph in P.phases for t in ph
                    if t["type"] in (PR.T_AMP_DOT, PR.T_AMP_FFV, PR.T_AMP_VVV, PR.T_AMP_VVVV) and not (t["type"] == PR.T_AMP_VVVV and t["aux"] & 4))
        assert ncols == {2: 3, 3: 18, 4: 33, 5: 225}[ng]     # amplitude columns (ng >= 4: the full-set vertices on ordered currents)
        if P.bg:
            finals = [t for ph in P.phases for t in ph if t["type"] == PR.T_QSUM and t["aux"] & 1]
            assert sorted(t["flow"] for t in finals) == list(range(P.ncolor))       # one closing sum per colour flow
        assert P.NL >= 32 and P.NL & (P.NL - 1) == 0
        # the kernel generates the code of at most 2 (n_g <= 4) / 5 (n_g = 5) operands of an ordered-current sum and of n_g - 1 terms of a
        # quark-line sum (csrc/mg_vm.cuh T_COMB, T_QSUM)
        for ph in P.phases:
            for t in ph:
                if t["type"] == PR.T_COMB:
                    assert int((t["idx"][:, PR.COMB_MAX] & 7).max()) <= (2 if ng <= 4 else 5)
                if t["type"] == PR.T_QSUM and t["aux"] & 1:
                    assert np.all((t["idx"][:, PR.QS_FLAGS_A] & 7) == ng - 1) and np.all((t["idx"][:, PR.QS_FLAGS_B] & 7) == ng - 2)
                elif t["type"] == PR.T_QSUM:
                    assert int((t["idx"][:, PR.QS_FLAGS_A] & 7).max()) <= ng - 2
        assert P.flops_executed_per_event() <= P.flops_canonical_per_event()[0]


def test_shared_memory_budget(programs):
    # bytes the kernel carves (csrc/mg_vm.cuh): doubles [8*4*E + E + NT], T [8*nslot*E + 2^ng*12*E + (ncolor + ncol + 1)*2*NL]
    for ng, P in programs.items():
        E, NL = P.E, P.NL
        b = (8 * 4 * E + ((E + 1) & ~1) + P.nthreads) * 8 + (8 * P.nslot * E + (1 << ng) * 12 * E + (P.ncolor + P.ncol + 1) * 2 * NL) * 8
        assert b <= 227 * 1024, (ng, b)


def test_accumulation_units_partition_the_flows(programs):
    """acc_groups: every touched flow of an accumulation task lands in exactly one unit of at most ACC_R flows."""
    for ng, P in programs.items():
        for phase in P.phases:
            for t in phase:
                if t["type"] != PR.T_ACC:
                    continue
                groups = emit.acc_groups(t["lists"], P.nthreads // 32)
                flat = sorted(k for g in groups for k in g)
                assert flat == list(range(len(t["lists"])))
                assert max(len(g) for g in groups) <= emit.ACC_R


@pytest.mark.parametrize("ng,opts", [(4, dict(mitm=False)), (4, dict(ordered=True)), (4, dict(mitm=False, ordered=True)),
                                     (3, dict(mitm=False)), (4, dict(outer_legs=(0, 1))), (4, dict(outer_legs=())),
                                     (4, dict(block_r=2)), (4, dict(block_r=1)), (3, dict(block_r=0))])
def test_program_options_reproduce_oracle(orc, ng, opts):
    """The optional forms of the program (left-only chains, ordered basis on/off, other outer legs) stay exact regroupings."""
    cfg = dict(emit.CONFIGS[ng])
    cfg.pop("chunk_warps", None)
    cfg.update(slot_budget=600)
    cfg.update(opts)
    P = PR.QCDProgram(ng, **cfg)
    _hazard_free(P)
    _check_against_oracle(orc, P, ng)


@pytest.mark.parametrize("ng", [4, 5])
def test_fp32_program_reproduces_oracle(orc, ng):
    """The FP32 programs of gg->ttgg / gg->ttggg (more events per CTA, emit.F32_CONFIGS) are the same exact regrouping."""
    P = emit.build_program(ng, f32=True)
    _hazard_free(P)
    assert P.pid == ng + 10 and P.E > emit.CONFIGS[ng]["E"]
    E, NL = P.E, P.NL
    assert (8 * 4 * E + ((E + 1) & ~1) + P.nthreads) * 8 + (8 * P.nslot * E + (1 << ng) * 12 * E + (P.ncolor + P.ncol + 1) * 2 * NL) * 4 <= 227 * 1024
    _check_against_oracle(orc, P, ng)


@pytest.mark.parametrize("ng", [2, 3, 4, 5])
def test_program_reproduces_oracle(orc, programs, ng):
    """The scheduled program, interpreted in numpy, gives the oracle's per-helicity |M_h|^2 and flow weights."""
    _check_against_oracle(orc, programs[ng], ng)


def _check_against_oracle(orc, P, ng):
    wl = WORKLOADS[ng]
    pm, _ = orc.rambo(wl.seed, 7, 1, wl.final_masses, wl.sqrt_s)
    p = pm[0]
    mt, wt = SM_PARAMS[2], SM_PARAMS[3]
    gs = orc.sm_derive(SM_PARAMS)["gs"]
    num, den = D.colour_matrix_integer(ng)
    Cm = np.array(num) / den

    def ext(kind, leg, lam):
        if kind < 2:
            e = orc.wavefunction("eps", p[leg], 0.0, lam)
            return e.conj() if kind == 1 else e
        return orc.wavefunction("ubar" if kind == 2 else "v", p[leg], mt, lam)

    _, mh2, wcol = orc.matrix_elements(ng, pm, sm=SM_PARAMS)
    npar = ng + 2
    mine, wc = np.zeros(1 << npar), np.zeros(P.ncolor)
    for o in range(P.nouter):
        J = vm_sim.simulate(P, p, mt, wt, o, ext)
        assert np.all(np.isfinite(J))
        ho = sum(((o >> (len(P.outer) - 1 - k)) & 1) << (npar - 1 - leg) for k, leg in enumerate(P.outer))
        for c in range(P.NC):
            hi = sum(((c >> (len(P.inner) - 1 - k)) & 1) << (npar - 1 - leg) for k, leg in enumerate(P.inner))
            mine[ho + hi] = (J[:, c].conj() @ Cm @ J[:, c]).real * gs ** (2 * ng)
        wc += (np.abs(J) ** 2).sum(axis=1) * gs ** (2 * ng)
    assert np.abs(mine - mh2[0]).max() < 1e-11 * mh2[0].sum()
    assert np.abs(wc / wcol[0] - 1).max() < 1e-11


def test_flop_counts_are_counted_and_cross_checked(orc, programs):
    """the per-routine flops come from a counting scalar (emitter/flops.py); executed <= canonical; the oracle
    built on ITS counting scalar (orc_count_flops) gives the order-of-magnitude cross-check: it performs a constant multiple of
    the canonical count (explicit 4x4 gamma matrices against two-component chiral forms), the same multiple for every process."""
    from paper_2507_21039_b200.emitter import flops as F
    assert F.FFV == 146 and F.ROW_SLASH == 64 and F.CLOSE4 == 4 * 30          # hand counts of three routines (csrc/mg_vm.cuh)
    assert F.ee_flops(4) < F.ee_flops(16)
    ratios = {}
    for ng, P in programs.items():
        canon, ex = P.flops_canonical_per_event()[0], P.flops_executed_per_event()
        assert 0 < ex <= canon
        wl = WORKLOADS[ng]
        p, _ = orc.rambo(wl.seed, 0, 1, wl.final_masses, wl.sqrt_s)
        ops, me = orc.count_flops(ng, p[0], sm=SM_PARAMS)
        ref, _, _ = orc.matrix_elements(ng, p, sm=SM_PARAMS)
        assert abs(me / ref[0] - 1) < 1e-14                                   # the counting build computes the same thing
        ratios[ng] = ops / canon
        assert 1.0 <= ratios[ng] <= 10.0, ratios                              # same order of magnitude, never below the canonical count
    assert max(ratios.values()) / min(ratios.values()) < 1.25, ratios         # both scale with the same wavefunction / amplitude counts
    ops1, _ = orc.count_flops(1, orc.rambo(1, 0, 1, (0.0, 0.0), 500.0)[0][0], sm=SM_PARAMS)
    assert F.ee_flops(16) <= ops1 <= 40 * F.ee_flops(16)


# ---- Drell-Yan u u~ -> e+ e- + n g: the programs of the same emitter against the oracle (process ids 6..9) -------
def _dy_ext(orc, p):
    """external wavefunctions of the Drell-Yan programs for the numpy interpreter, from the oracle's spinors and couplings."""
    d = orc.sm_derive(SM_PARAMS)
    MZ, WZ = SM_PARAMS[0], SM_PARAMS[1]
    sw, cw = np.sqrt(d["sw2"]), np.sqrt(1 - d["sw2"])
    Qu, T3 = 2.0 / 3.0, 0.5
    gq = [[d["ee"] * Qu, d["ee"] * Qu], [d["ee"] / (sw * cw) * (T3 - Qu * d["sw2"]), d["ee"] / (sw * cw) * (-Qu * d["sw2"])]]
    gl = [[d["gLA"], d["gRA"]], [d["gLZ"], d["gRZ"]]]
    g0 = np.array([[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]], complex)
    sig = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]], complex), np.array([[1, 0], [0, -1]], complex)]
    gam = [g0] + [np.block([[np.zeros((2, 2)), s], [-s, np.zeros((2, 2))]]) for s in sig]
    PL, PR = np.diag([1, 1, 0, 0]).astype(complex), np.diag([0, 0, 1, 1]).astype(complex)
    sll = 2 * (p[2][0] * p[3][0] - p[2][1:] @ p[3][1:])
    den = [sll, sll - MZ * MZ + 1j * MZ * WZ]

    def ext(kind, leg, lam, lam2=None):
        if kind == 1:
            return orc.wavefunction("eps", p[leg], 0.0, lam).conj()
        if kind == 4:
            return orc.wavefunction("vbar", p[leg], 0.0, lam)
        if kind == 5:
            return orc.wavefunction("u", p[leg], 0.0, lam)
        assert kind in (6, 7)
        ub, v = orc.wavefunction("ubar", p[3], 0.0, lam2), orc.wavefunction("v", p[2], 0.0, lam)
        jL = np.array([ub @ gam[mu] @ PL @ v for mu in range(4)])
        jR = np.array([ub @ gam[mu] @ PR @ v for mu in range(4)])
        chi = kind - 6
        return sum(gq[V][chi] / den[V] * (gl[V][0] * jL + gl[V][1] * jR) for V in range(2))
    return ext


@pytest.mark.parametrize("n", [0, 1, 2, 3])
def test_drell_yan_program_reproduces_oracle(orc, n):
    P = emit.build_program(n + 6)
    assert P.dy and (P.ndiag, P.ncolor) == {0: (1, 1), 1: (2, 1), 2: (8, 2), 3: (50, 6)}[n]
    _hazard_free(P)
    pm, _ = orc.rambo(40 + n, 3, 1, (0.0,) * (n + 2), 700.0)
    p = pm[0]
    gs = orc.sm_derive(SM_PARAMS)["gs"]
    num, den = D.colour_matrix_integer(n)
    Cm = np.array(num) / den
    _, mh2, wcol = orc.matrix_elements(n + 6, pm, sm=SM_PARAMS)
    J = vm_sim.simulate(P, p, 0.0, 0.0, 0, _dy_ext(orc, p))
    assert np.all(np.isfinite(J))
    npar = n + 4
    mine = np.zeros(1 << npar)
    for c in range(P.NC):
        hi = sum(((c >> (len(P.inner) - 1 - k)) & 1) << (npar - 1 - leg) for k, leg in enumerate(P.inner))
        mine[hi] = (J[:, c].conj() @ Cm @ J[:, c]).real * gs ** (2 * n)
    assert np.abs(mine - mh2[0]).max() < 1e-11 * mh2[0].sum()
    assert np.array_equal(mine == 0, mh2[0] == 0)                      # the vanishing helicity combinations vanish exactly on both sides
    wc = (np.abs(J) ** 2).sum(axis=1) * gs ** (2 * n)
    assert np.abs(wc / wcol[0] - 1).max() < 1e-11
