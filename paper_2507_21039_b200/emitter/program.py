"""Scheduler: turns the diagram/colour tables of g g -> t t~ + (ng-2) g into a task program for the CUDA
wavefunction VM (csrc/mg_vm.cuh).

Design: one CTA evaluates E events for one assignment of the OUTER helicities
(legs whose helicity is fixed per CTA) and all 2^|inner| assignments of the INNER helicities.  Every stored
wavefunction family (external legs, gluon subtree currents per label set, quark-line chains per ordered block
prefix, W currents) keeps one entry per (tree choice, helicity assignment of the inner legs it depends on), so a
sub-wavefunction is evaluated once per ITS OWN helicity sub-combination (helicity recycling)
and shared by every helicity combination that contains it.  A task is warp-uniform: one routine (PAPER.md:130-136
FFV / VVV / VVVV families) applied to `nitems` gathered operand tuples; consecutive lanes take consecutive items.
Tasks are grouped in phases separated by CTA barriers; the scheduler keeps everything in shared memory.
"""
import numpy as np

from . import diagrams as D
from . import flops as F

# task types (keep in sync with csrc/mg_vm.cuh)
T_EXT, T_VVV, T_VVVV, T_FFV, T_WCUR, T_AMP_DOT, T_AMP_FFV, T_AMP_VVV, T_AMP_VVVV, T_ACC, T_COMB, T_FFVR, T_QSUM, T_CHAN, T_VVVF = range(15)
TYPE_NAMES = ["EXT", "VVV", "VVVV", "FFV", "WCUR", "AMP_DOT", "AMP_FFV", "AMP_VVV", "AMP_VVVV", "ACC", "COMB", "FFVR", "QSUM", "CHAN", "VVVF"]
QSUM_MAX = 4                # terms per row sum of a QSUM item
# QSUM index columns (program level): row sum A = (row spinor, current) x QSUM_MAX in columns 0..7, row sum B x (QSUM_MAX - 1) in
# columns 8..13, then the right current R1, v(t~), helicity combination, flags (terms | orientation signs << 4), flow, bit of t~ in R1
QS_R1, QS_V, QS_H, QS_FLAGS_A, QS_FLAGS_B, QS_FLOW, QS_SH_TB, QSUM_COLS = 14, 15, 16, 17, 18, 19, 20, 24
COMB_MAX = 6                # operands per COMB item (index-table fields u0..u3, u5, u6)

# flops per item: counted by running each routine's operation sequence on a counting scalar (emitter/flops.py), not tallied by hand.
# Amplitude routines are multi-output: AMP_DOT 4 amplitudes per item (4 dots), AMP_FFV 4 per helicity assignment of the blocked legs
# (two row*slash per item + four dots each), AMP_VVV / AMP_VVVV 4 (one vertex current + 4 dots)
FLOPS = {T_EXT: F.EXT_SPINOR, T_VVV: F.VVV, T_VVVV: F.VVVV, T_FFV: F.FFV, T_WCUR: F.WCUR, T_AMP_DOT: F.AMP_DOT,
         T_AMP_FFV: F.AMP_FFV_ROWS + F.AMP_FFV_DOTS, T_AMP_VVV: F.AMP_VVV, T_AMP_VVVV: F.AMP_VVVV, T_COMB: 0, T_FFVR: F.FFV}
# the same routines as the paper's method calls them, one amplitude per call (canonical count)
FLOPS_CANON = {T_AMP_FFV: F.CANON_AMP_FFV, T_AMP_VVV: F.CANON_AMP_VVV, T_AMP_VVVV: F.CANON_AMP_VVVV}
FLOPS_AMP_FFV_ROWS, FLOPS_AMP_FFV_DOTS = F.AMP_FFV_ROWS, F.AMP_FFV_DOTS
FLOPS_ACC_PAIR = F.ACC_PAIR     # one complex add per (flow, diagram) pair
FLOPS_QSUM_TERM, FLOPS_QSUM_PROP, FLOPS_QSUM_CLOSE = F.QSUM_TERM, F.QSUM_PROP, F.QSUM_CLOSE
FLOPS_COMB_TERM = F.COMB_TERM   # one signed 4-vector add per (ordered current, tree) term
EXT_G, EXT_UBAR, EXT_V = 0, 2, 3   # EXT kinds: 0 gluon incoming, 1 gluon outgoing, 2 ubar(t), 3 v(tbar)
# Drell-Yan: 4 vbar of the incoming antiquark (row end), 5 u of the incoming quark (column end), 6 / 7 the gamma*/Z "current" seen by a
# left- / right-chiral quark line: sum_V g^q_chi g^l / (s_ll - M_V^2 + i M_V W_V) ubar(e-) gamma^mu (P_L, P_R) v(e+)
EXT_VBAR_IN, EXT_U_IN, EXT_EW_L, EXT_EW_R = 4, 5, 6, 7


def task_access(t):
    """(slots read, slots written, amplitude columns read, columns written) of one scheduled task (a dict of QCDProgram.phases).
    Accumulate-mode tasks read what they add into.  Used by the emitter to decide which tasks of a phase may start before
    the previous phase has finished on every warp (split arrive / wait barriers, emitter/emit.py)."""
    ty, n = t["type"], t["nitems"]
    rs, ws, rc, wc = set(), set(), set(), set()
    if ty == T_ACC:
        for lst in t["lists"]:
            rc |= {c for c, _ in lst}
        return rs, ws, rc, wc
    if ty == T_CHAN:
        return rs, ws, set(range(len(t["names"]))), wc
    ix = t["idx"]
    if ty == T_COMB:
        for q in range(COMB_MAX):
            sel = (ix[:, COMB_MAX] & 7) > q
            rs |= set((t["in_base"][0] + ix[sel, q]).tolist())
        ws |= set(range(t["out_base"], t["out_base"] + n))
        return rs, ws, rc, wc
    if ty == T_QSUM:
        for c, b in zip(t["in_cols"], t["in_base"]):
            if c < 2 * QSUM_MAX:
                sel = (ix[:, QS_FLAGS_A] & 15) > c // 2
            elif c < QS_R1:
                sel = (ix[:, QS_FLAGS_B] & 15) > (c - 2 * QSUM_MAX) // 2
            else:
                sel = np.ones(n, dtype=bool)
            rs |= set((b + ix[sel, c]).tolist())
            if c == QS_R1:
                rs |= set((b + ix[:, c] + (1 << ix[:, QS_SH_TB])).tolist())
            if c == QS_V:
                rs |= {b + 1}
        if not (t["aux"] & 1):
            ws |= set(range(t["out_base"], t["out_base"] + n))
        return rs, ws, rc, wc
    if ty == T_VVVF:
        rs |= set((t["in_base"][0] + ix[:, 0]).tolist()) | set((t["in_base"][1] + ix[:, 1]).tolist())
        xs, fl = t["xslots"], t["xflags"]
        for q in range(2):
            sel = ((fl >> (2 * q)) & 1) == 1
            rs |= set(xs[sel, 2 * q].tolist()) | set(xs[sel, 2 * q + 1].tolist())
        ws |= set(range(t["out_base"], t["out_base"] + n))
        return rs, ws, rc, wc
    nin = {T_EXT: 0, T_VVV: 2, T_VVVV: 3, T_FFV: 2, T_FFVR: 2, T_WCUR: 2, T_AMP_DOT: 2, T_AMP_FFV: 3, T_AMP_VVV: 2, T_AMP_VVVV: 3}[ty]
    for k in range(nin):
        rs |= set((t["in_base"][k] + ix[:, k]).tolist())
    if ty == T_AMP_VVV or (ty == T_AMP_VVVV):
        rs |= set(range(t["in_base"][nin], t["in_base"][nin] + 4))            # the four (t, t~) variants of W0
    if ty == T_AMP_DOT:
        # the W family entry of every (t, t~) variant: bit positions mA (t), mB (t~) of the variant index
        base = t["in_base"][0] + ix[:, 0]
        for tt in range(4):
            rs |= set((base + ((tt >> 1) << t["mA"]) + ((tt & 1) << t["mB"])).tolist())
    if ty == T_AMP_FFV:
        sh_tb, sh_g, sh_t = t["mA"] & 15, (t["mA"] >> 4) & 15, t["mB"] & 15
        sh_g1 = (ix[:, 4] & 15) if ix.shape[1] > 4 else 0 * ix[:, 0]
        rs |= set((t["in_base"][0] + ix[:, 0] + (1 << sh_t)).tolist())
        for hg in range(1 << (t["aux"] & 3)):
            rb = t["in_base"][2] + ix[:, 2] + ((hg & 1) << sh_g) + ((hg >> 1) << sh_g1)
            for tb in range(2):
                rs |= set((rb + (tb << sh_tb)).tolist())
    if ty == T_AMP_VVVV and (t["aux"] & 4):
        cols = set(t["col_of_item"].tolist())
        rc |= cols
        wc |= cols
    elif ty in (T_AMP_DOT, T_AMP_FFV, T_AMP_VVV, T_AMP_VVVV):
        wc |= set(range(t["out_base"], t["out_base"] + n // t["rpc"]))
    elif ty == T_VVVV and (t["aux"] & 4):
        out = set((t["out_base"] + (ix[:, 3] & 0x7fff)).tolist())
        rs |= out
        ws |= out
    else:
        ws |= set(range(t["out_base"], t["out_base"] + n))
    return rs, ws, rc, wc


def mark_free_tasks(phases):
    """Sets t["free"] on every task: True when the task touches nothing that the PREVIOUS phase reads or writes in a conflicting
    way (no input written there, no output read or written there), so it may run while other warps are still in that phase.
    Accumulation tasks (they update jamp and read the columns just written) and the first phase are never free."""
    prev = None
    for phase in phases:
        acc = [task_access(t) for t in phase]
        for t, (rs, ws, rc, wc) in zip(phase, acc):
            free = prev is not None and t["type"] != T_ACC
            if free:
                prs, pws, prc, pwc = prev
                free = not (rs & pws) and not (ws & (prs | pws)) and not (rc & pwc) and not (wc & (prc | pwc))
            t["free"] = bool(free)
        prev = tuple(set().union(*[a[k] for a in acc]) for k in range(4))


class Fam:
    def __init__(self, name, ntree, deps, arena):
        self.name, self.ntree, self.deps, self.arena = name, ntree, tuple(deps), arena
        self.nv = 1 << len(self.deps)
        self.nitems = ntree * self.nv
        self.base = None
        self.producers_left = 0
        self.consumers_left = 0
        self.complete = False


class Task:
    def __init__(self, ttype, nitems, ins, idx, out=None, out_off=0, aux=0, mA=0, mB=0, depth=0):
        self.type, self.nitems, self.ins, self.idx = ttype, nitems, ins, idx
        self.out, self.out_off, self.aux, self.mA, self.mB, self.depth = out, out_off, aux, mA, mB, depth
        self.cols = None          # amp tasks: list of {flow: kappa code} per diagram column
        self.rpc = 0              # amp tasks: index-table rows (operand tuples) per column
        self.done = False
        self.accumulate = False   # VVVV tasks of the merged scheme: += into slots written by earlier tasks
        self.after = []           # tasks that must have run in an earlier phase
        self.out_slots = None     # accumulate tasks: relative output slots (or amplitude columns) they touch
        self.flops_item = None    # flops per item when they differ from FLOPS[type]
        self.flops = None         # flops of the whole task when they are not FLOPS[type] * nitems (COMB)
        self.top = None           # folded top level: 'store' (cubic-top columns at fixed positions) / 'acc' (quartic, += into them)
        self.done_cols = 0


class Arena:
    def __init__(self, start, size):
        self.start, self.size = start, size
        self.free = [(start, size)]

    def alloc(self, n):
        for k, (s, z) in enumerate(self.free):
            if z >= n:
                if z == n:
                    self.free.pop(k)
                else:
                    self.free[k] = (s + n, z - n)
                return s
        return None

    def release(self, s, n):
        self.free.append((s, n))
        self.free.sort()
        merged = []
        for a, z in self.free:
            if merged and merged[-1][0] + merged[-1][1] == a:
                merged[-1] = (merged[-1][0], merged[-1][1] + z)
            else:
                merged.append((a, z))
        self.free = merged


def _restrict(hv, sup, sub):
    """helicity-variant index over leg tuple `sup` (first leg = MSB) -> index over the sub-tuple `sub`."""
    out = np.zeros_like(hv)
    for leg in sub:
        pos = len(sup) - 1 - sup.index(leg)
        out = (out << 1) | ((hv >> pos) & 1)
    return out


class QCDProgram:
    def __init__(self, ng, outer_legs=(), E=1, ncol=32, slot_budget=1024, nthreads=256, chunk_items=None, stream_top=False, top_factor=2.0, double_buffer=False, merge_quartic=True, fold_top=False, arena_weights=None, ordered=True, mitm=True, block_r=1, bg=False, chan=False, dy=False, fuse_quartic=True, fuse_closing=False):
        # stream_top: the currents on the (ng-1)-gluon label sets are not kept resident; they live in an arena and are
        # freed once their consumers (single-block vertices, chains, closing amplitudes) have run
        # dy: Drell-Yan u(0) u~(1) -> e+(2) e-(3) + gluons (legs 4..).  `ng` then counts the labels on the quark
        # line: the gluons and, as the LAST label, the gamma*/Z, a colourless block with a left- and a right-chiral current.  The
        # row end of the line is the incoming u~ (vbar), the column end the incoming u; all gluons are outgoing; massless, no width.
        # fuse_quartic: the four-gluon structures merged into a cubic tree ((X, Y), Z) are evaluated INSIDE the item that builds the
        # tree (task VVVF) instead of being added by a separate accumulate task one phase later: the merged structure only needs X, Y
        # (the children of the composite child) and Z, and always has the form (x.z) y - (y.z) x.  Two phases fewer on the critical
        # path of g g -> t t~ g g g (tree -> ordered current instead of tree -> quartic add -> ordered current, at two levels).
        self.fuse_quartic = fuse_quartic and merge_quartic and not chan
        # fuse_closing: the closing sums of the colour-ordered quark line may share a phase with an accumulation task.  Both add into
        # jamp, so the emitter gives the closing sums of a flow to the WARP that runs the accumulation unit of that flow, after it
        # (emit.py, "owner"): the shared-memory-bound accumulation of some warps then overlaps the FP64-bound closing sums of others.
        self.fuse_closing = fuse_closing and bg and not chan
        self.dy = dy
        self.ngl = ng - 1 if dy else ng                   # gluons
        self.vmask = 1 << (ng - 1) if dy else 0
        self.leg_row, self.leg_col = (1, 0) if dy else (2, 3)
        self.ng, self.E, self.ncol, self.nthreads, self.stream_top = ng, E, ncol, nthreads, stream_top
        self.top_factor = top_factor
        self.double_buffer = double_buffer
        self.arena_weights = arena_weights or {}      # arena name -> weight of its share of the spare slots
        self.npar = ng + 3 if dy else ng + 2
        # merge_quartic: four-gluon structures below the full label set are added into the nested three-gluon tree with
        # the same colour factor (emitter/diagrams.py); ts_full keeps the paper's one-amplitude-per-structure enumeration
        self.fold_top = fold_top and merge_quartic and not double_buffer
        # ordered: chains, closing amplitudes and the full-set vertices take the currents of the 3..(ng-1)-gluon label sets in
        # the colour-ordered basis (diagrams.TreeSet.ordered_basis): k!/2 ordered currents with two colour flows each
        # instead of (2k-3)!! trees with 2^(k-1) flows each -- fewer amplitude columns, far fewer (flow, column) pairs
        self.ordered = ordered and merge_quartic and not self.fold_top
        # mitm: quark chains are grown from both ends (row spinors from ubar(t), column spinors from v(t~)) and a diagram is
        # closed on a middle block: chain depth (ng - 1) -> (ng - 1) / 2 and far fewer chain wavefunctions
        self.mitm = mitm
        self.block_r = block_r
        # bg: the quark line as a colour-ordered recursion (Berends-Giele form): one quark current per ORDERED gluon prefix, the
        # sum over its last block taken in registers, and one closing sum per colour flow written straight into jamp -- no
        # amplitude columns and no kappa accumulation for the diagrams with two or more blocks (see _chains_bg)
        if dy:
            ordered, bg, fold_top = False, False, False
        self.bg = bg and self.ordered and not chan
        # chan: the multichannel program.  Gluon trees without four-gluon vertices, one amplitude column per
        # diagram = per channel; instead of the kappa accumulation a CHAN task adds |A_k|^2 of every pending column into the
        # channel sums.  No jamp, no colour sum.
        self.chan = chan
        if chan:
            self.ordered, self.fold_top, merge_quartic = False, False, False
        self.ts = D.TreeSet(ng, merged=merge_quartic, fold_top=self.fold_top, cubic_only=chan, vlabel=ng - 1 if dy else None)
        self.ts_full = D.TreeSet(ng, vlabel=ng - 1 if dy else None)
        self.full = self.ts.full
        self.outer = tuple(sorted(outer_legs))
        self.inner = tuple(l for l in range(self.npar) if l not in self.outer)
        self.NC = 1 << len(self.inner)
        self.NL = self.NC * E
        self.nouter = 1 << len(self.outer)
        self.flows = D.flows(self.ngl)
        self.flow_index = {f: i for i, f in enumerate(self.flows)}
        self.ncolor = len(self.flows)
        self.slot_budget = slot_budget
        self.chunk_items = chunk_items
        self.ndiag, self.namp = D.count_diagrams(self.ts_full)
        self._build_tasks()
        self._schedule()

    # ------------------------------------------------------------------------------------------------ helpers
    def leg_of_gluon(self, g):
        return 4 + g if self.dy else D.gluon_leg(g)

    def gdeps(self, mask):
        """inner legs whose helicities a current on this label set depends on (the boson: both lepton legs)."""
        legs = set()
        for g in D.bits(mask):
            legs |= {2, 3} if (self.dy and g == self.ng - 1) else {self.leg_of_gluon(g)}
        return tuple(sorted(l for l in legs if l in self.inner))

    def nchoice(self, mask):
        """number of currents of a label set as the chains / amplitudes see it (trees, or ordered currents)."""
        if self.dy and mask & self.vmask:
            return 1 if mask == self.vmask else 0            # the boson never shares a block with gluons
        return self.use[mask].ntree

    def choice_colour(self, mask, i):
        if self.use[mask] is self.cur[mask]:
            return self.ts.colour(mask, i)
        return self.ts.colour_ordered(mask, i)

    def _deposit(self, H, src, dst):
        """variant index over leg tuple `src` -> index over `dst` (legs of dst missing in src get bit 0)."""
        out = np.zeros_like(H)
        for leg in dst:
            out = out << 1
            if leg in src:
                out = out | ((H >> (len(src) - 1 - src.index(leg))) & 1)
        return out

    def _bitpos(self, deps, leg):
        """bit position of `leg` inside a variant index over `deps`."""
        return len(deps) - 1 - deps.index(leg)

    def _deps_union(self, *deps):
        return tuple(sorted(set().union(*[set(d) for d in deps])))

    # ------------------------------------------------------------------------------------------------ task graph
    def _build_tasks(self):
        ts, ng = self.ts, self.ng
        self.fams, self.tasks = [], []
        self.store_tasks = {}
        self.top_store_tasks = []
        inner = self.inner
        t_in = (self.leg_row,) if self.leg_row in inner else ()
        tb_in = (self.leg_col,) if self.leg_col in inner else ()

        def fam(name, ntree, deps, arena):
            f = Fam(name, ntree, deps, arena)
            self.fams.append(f)
            return f

        def add(task):
            self.tasks.append(task)
            if task.out is not None:
                task.out.producers_left += 1
            for f in task.ins:
                f.consumers_left += 1
            return task

        def ext_task(f, leg, kind):
            # idx columns: leg, helicity code (0: -1, 1: +1, 2+k: k-th outer leg's bit of the CTA), kind
            nv = f.nv
            code = np.arange(nv) if nv == 2 else np.array([2 + self.outer.index(leg)])
            idx = np.stack([np.full(nv, leg), code, np.full(nv, kind), np.zeros(nv, int)], axis=1)
            t = add(Task(T_EXT, nv, [], idx, out=f))
            t.flops_item = F.EXT_EPS if kind < 2 else F.EXT_SPINOR

        # external legs
        self.cur = {}
        for g in range(self.ngl):
            leg = self.leg_of_gluon(g)
            f = fam("g%d" % leg, 1, self.gdeps(1 << g), "perm")
            self.cur[1 << g] = f
            ext_task(f, leg, 1 if (self.dy or g >= 2) else 0)
        if self.dy:
            # the gamma*/Z: two currents (left- and right-chiral quark line) per helicity assignment of the two leptons
            assert self.outer == () and 2 in inner and 3 in inner
            f = fam("JV", 2, (2, 3), "perm")
            self.cur[self.vmask] = f
            hv = np.arange(4)
            for chi, kind in ((0, EXT_EW_L), (1, EXT_EW_R)):
                idx = np.stack([np.full(4, 2), hv >> 1, np.full(4, kind), hv & 1], axis=1)      # codes: helicity of e+ (leg 2), of e- (leg 3)
                t = add(Task(T_EXT, 4, [], idx, out=f, out_off=chi * 4))
                t.flops_item = 2 * F.EXT_SPINOR + F.WCUR + 60
            self.ubar = fam("vbar", 1, t_in, "perm")
            ext_task(self.ubar, self.leg_row, EXT_VBAR_IN)
            self.vsp = fam("u", 1, tb_in, "perm")
            ext_task(self.vsp, self.leg_col, EXT_U_IN)
            self.W0 = None
        else:
            self.ubar = fam("ubar", 1, t_in, "perm")
            ext_task(self.ubar, 2, EXT_UBAR)
            self.vsp = fam("v", 1, tb_in, "perm")
            ext_task(self.vsp, 3, EXT_V)
            # W0 = i ubar gamma^mu v
            self.W0 = fam("W0", 1, t_in + tb_in, "perm")
            hv = np.arange(self.W0.nv)
            idx = np.stack([_restrict(hv, self.W0.deps, t_in), _restrict(hv, self.W0.deps, tb_in), 0 * hv, 0 * hv], axis=1)
            add(Task(T_WCUR, self.W0.nv, [self.ubar, self.vsp], idx, out=self.W0))

        # gluon subtree currents on proper subsets
        for mask in sorted(range(1, self.full), key=lambda m: (bin(m).count("1"), m)):
            if bin(mask).count("1") < 2 or (mask & self.vmask):
                continue
            top = self.stream_top and bin(mask).count("1") == ng - 1
            f = fam("J%x" % mask, ts.ntrees(mask), self.gdeps(mask), "top" if top else "perm")
            self.cur[mask] = f
            for sp in ts.splits[mask]:
                self._vertex_task(sp, f, None, add)
        # colour-ordered currents: signed sums of the tree currents of the same label set and helicities
        self.use = dict(self.cur)
        for mask in sorted(self.cur, key=lambda m: (bin(m).count("1"), m)):
            k = bin(mask).count("1")
            if not self.ordered or k < 3:
                continue
            src = self.cur[mask]
            perms, comb = ts.ordered_basis(mask)
            assert max(len(c) for c in comb) <= COMB_MAX
            f = fam("O%x" % mask, len(perms), src.deps, "perm" if self.bg else src.arena)   # bg: every closing sum reads them
            O, H = np.meshgrid(np.arange(len(perms)), np.arange(f.nv), indexing="ij")
            O, H = O.ravel(), H.ravel()
            idx = np.zeros((len(O), COMB_MAX + 1), dtype=np.int64)       # operand slots (relative to the tree family), flags
            for j, o in enumerate(O):
                terms = comb[o]
                for q, (tree, sg) in enumerate(terms):
                    idx[j, q] = tree * src.nv + H[j]
                    idx[j, COMB_MAX] |= (1 if sg < 0 else 0) << (3 + q)
                idx[j, COMB_MAX] |= len(terms)
            t = add(Task(T_COMB, len(O), [src], idx, out=f))
            t.flops = FLOPS_COMB_TERM * sum(len(comb[o]) for o in O)
            self.use[mask] = f
        # single-block diagrams: the full-set vertex closed with W0 (none with an electroweak boson on the line)
        for sp in ts.splits[self.full]:
            self._vertex_task(sp, None, self.W0, add)

        # quark-line chains, depth-first over ordered block prefixes
        self.chain_depth_max = 0
        if self.bg:
            self._chains_bg(add, fam)
        elif self.mitm:
            self._chains_mitm(add, fam)
        else:
            self._chains(prefix=(), parent=self.ubar, parent_trees=[()], used=0, add=add, fam=fam)

    def _ordered_block(self, block):
        """(family, entry index, sign) of the current on the ordered gluon tuple `block` as the quark line sees it: the stored
        current of the label set in canonical orientation (first label < last label) times the sign that is left of its colour
        coefficient for this orientation once the phase (-i)^(k-1) carried by every k-gluon current is split off."""
        mask = 0
        for g in block:
            mask |= 1 << g
        k = len(block)
        fam = self.use[mask]
        canon = tuple(block) if block[0] <= block[-1] else tuple(block[::-1])
        if fam is self.cur[mask]:
            assert k <= 2 and fam.ntree == 1
            o = 0
        else:
            o = self.ts.ordered_basis(mask)[0].index(canon)
        coeff = self.choice_colour(mask, o)[tuple(block)] / ((-1j) ** (k - 1))
        assert coeff in (1, -1)
        return fam, o, int(coeff.real)

    def _chains_bg(self, add, fam):
        """Colour-ordered quark line.  For an ordered tuple pi = (g_1 .. g_k) of distinct gluons, k <= ng - 2,
            Q[pi] = S(p_t - K(pi)) sum_{j=0}^{k-1} r_j  Q[g_1 .. g_j] slash(J[g_{j+1} .. g_k]),   Q[()] = ubar(t),
        where J[..] is the colour-ordered current of the block and r_j its orientation sign (_ordered_block), and for a colour
        flow sigma (a permutation of all ng gluons), with n = ng and R1[g] = S(p_t - K(all but g)) slash(eps_g) v(t~),
            jamp[sigma] += i ( sum_{j=0}^{n-2} r_j Q[sigma_1..sigma_j] slash(J[sigma_{j+1}..sigma_{n-1}]) ) R1[sigma_n]
                         + i ( sum_{j=1}^{n-2} r_j Q[sigma_1..sigma_j] slash(J[sigma_{j+1}..sigma_n]) ) v(t~).
        The first bracket is the quark current on sigma_1..sigma_{n-1} without its propagator (which sits in R1: the line is cut
        at its last propagator, so the (n-1)-gluon quark currents are never stored).  Expanding the recursion gives every
        ordered partition of sigma into two or more consecutive blocks exactly once: the same diagram sum as the block-sequence
        enumeration, with the sums over blocks taken in registers (task QSUM) instead of one amplitude
        column per block sequence followed by the kappa accumulation.  The single-block diagrams stay amplitude columns closed
        with W0 (their vertex values are shared between flows).  PAPER.md:110, 130-136."""
        from itertools import permutations
        ng, full = self.ng, self.full
        t_in = (2,) if 2 in self.inner else ()
        tb_in = (3,) if 3 in self.inner else ()
        assert t_in and tb_in, "the quark helicities are inner legs in every configuration"
        gl = tuple(l for l in self.inner if l not in (2, 3))
        assert ng - 1 <= QSUM_MAX
        Q = {(): self.ubar}

        def terms_of(pi, j_lo, j_hi):
            out = []
            for j in range(j_lo, j_hi):
                Jf, o, r = self._ordered_block(pi[j:])
                out.append((Q[pi[:j]], Jf, o, r))
            return out

        def fill(idx, col0, flag_col, H, deps, terms):
            flags = np.zeros(len(H), dtype=np.int64) + len(terms)
            for q, (Af, Jf, o, r) in enumerate(terms):
                idx[:, col0 + 2 * q] = _restrict(H, deps, Af.deps)
                idx[:, col0 + 2 * q + 1] = o * Jf.nv + _restrict(H, deps, Jf.deps)
                if r < 0:
                    flags |= 1 << (4 + q)
            idx[:, flag_col] = flags

        self.chain_depth_max = ng - 2
        for k in range(1, ng - 1):
            for pi in permutations(range(ng), k):
                mask = 0
                for g in pi:
                    mask |= 1 << g
                deps = self._deps_union(t_in, self.gdeps(mask))
                f = fam("Q" + "".join(str(g) for g in pi), 1, deps, "perm")
                terms = terms_of(pi, 0, k)
                idx = np.zeros((f.nv, QSUM_COLS), dtype=np.int64)
                fill(idx, 0, QS_FLAGS_A, np.arange(f.nv), deps, terms)
                ins = [x for (Af, Jf, _, _) in terms for x in (Af, Jf)]
                t = add(Task(T_QSUM, f.nv, ins, idx, out=f, mA=mask, depth=k))
                t.in_cols = list(range(2 * len(terms)))
                t.flops_item = FLOPS_QSUM_TERM * len(terms) + FLOPS_QSUM_PROP
                Q[pi] = f
        # right currents of one gluon: R1[g] = S(p_t - K(full ^ g)) slash(eps_g) v
        R1 = {}
        for g in range(ng):
            J = self.cur[1 << g]
            deps = self._deps_union(tb_in, J.deps)
            f = fam("R%d" % g, 1, deps, "perm")
            H = np.arange(f.nv)
            idx = np.zeros((f.nv, 4), dtype=np.int64)
            idx[:, 0] = _restrict(H, deps, self.vsp.deps)
            idx[:, 1] = _restrict(H, deps, J.deps)
            add(Task(T_FFVR, f.nv, [self.vsp, J], idx, out=f, mA=full ^ (1 << g), depth=1))
            R1[g] = f
        self.final_tasks = []
        deps = self._deps_union(t_in, gl)
        nv = 1 << len(deps)
        H = np.arange(nv)
        for sigma in self.flows:
            last = sigma[-1]
            termsA = terms_of(sigma[:-1], 0, ng - 1)          # the quark current on sigma_1..sigma_{n-1}, propagator cut off
            termsB = terms_of(sigma, 1, ng - 1)
            idx = np.zeros((nv, QSUM_COLS), dtype=np.int64)
            fill(idx, 0, QS_FLAGS_A, H, deps, termsA)
            fill(idx, 2 * QSUM_MAX, QS_FLAGS_B, H, deps, termsB)
            Rf = R1[last]
            idx[:, QS_R1] = self._deposit(H, deps, Rf.deps)              # variant with t~ = -1
            idx[:, QS_SH_TB] = self._bitpos(Rf.deps, 3)
            idx[:, QS_H] = self._deposit(H, deps, self.inner)            # helicity combination with t~ = -1
            idx[:, QS_FLOW] = self.flow_index[sigma]
            ins = ([x for (Af, Jf, _, _) in termsA for x in (Af, Jf)] + [x for (Af, Jf, _, _) in termsB for x in (Af, Jf)] + [Rf, self.vsp])
            t = add(Task(T_QSUM, nv, ins, idx, aux=1, depth=ng))
            t.in_cols = (list(range(2 * len(termsA))) + [2 * QSUM_MAX + c for c in range(2 * len(termsB))] + [QS_R1, QS_V])
            t.flops_item = FLOPS_QSUM_TERM * (len(termsA) + len(termsB)) + FLOPS_QSUM_CLOSE
            t.flow = self.flow_index[sigma]
            self.final_tasks.append(t)

    def _chains_mitm(self, add, fam):
        """Meet in the middle.  A diagram with blocks (B1..Bm), m >= 2, along the quark line is
        ubar S.. slash(J_B1) S slash(J_B2) .. slash(J_Bm) v.  If the last block has many currents (> 2) the diagram is closed as
        before: W^mu = i (left chain of B1..B(m-1)) gamma^mu v once, then one dot product per current of Bm.  Otherwise the
        diagram is cut at the middle block Bc, c = (m - 1) // 2 + 1: left chain L(B1..B(c-1)) (row spinor grown from ubar),
        right chain R(B(c+1)..Bm) (column spinor grown from v) and the amplitude i L slash(J_Bc) R.  The propagator after block k
        carries p_t - K(B1..Bk) in both directions, so the right chain reads the momentum table at the complement of its label
        set: the same numbers as the left-only evaluation (and the oracle), only the association of the matrix product changes."""
        ts, full = self.ts, self.full
        lr, lc = self.leg_row, self.leg_col
        t_in = (lr,) if lr in self.inner else ()
        tb_in = (lc,) if lc in self.inner else ()
        assert t_in and tb_in, "the quark helicities are inner legs in every configuration"
        gl = tuple(l for l in self.inner if l not in (lr, lc))     # helicity legs of the currents (gluons; Drell-Yan: and the leptons)
        left = {(): (self.ubar, [()])}
        right = {(): (self.vsp, [()])}

        def union(blocks):
            m = 0
            for b in blocks:
                m |= b
            return m

        def chain(blocks, is_left):
            table = left if is_left else right
            if blocks in table:
                return table[blocks]
            S = blocks[-1] if is_left else blocks[0]
            parent, ptrees = chain(blocks[:-1] if is_left else blocks[1:], is_left)
            J = self.use[S]
            ntS, ntP = self.nchoice(S), len(ptrees)
            deps = self._deps_union(parent.deps, self.gdeps(S))
            nv = 1 << len(deps)
            depth = len(blocks)
            self.chain_depth_max = max(self.chain_depth_max, depth)
            f = fam(("C" if is_left else "R") + "_".join("%x" % m for m in blocks), ntP * ntS, deps,
                    "dt" if (J.arena == "top" or parent.arena == "dt") else "d%d" % depth)
            T, H = np.meshgrid(np.arange(ntP * ntS), np.arange(nv), indexing="ij")
            T, H = T.ravel(), H.ravel()
            tp, tS = T // ntS, T % ntS
            idx = np.zeros((len(T), 4), dtype=np.int64)
            idx[:, 0] = tp * parent.nv + _restrict(H, deps, parent.deps)
            idx[:, 1] = tS * J.nv + _restrict(H, deps, J.deps)
            U = union(blocks)
            if S == self.vmask and self.dy:
                idx[:, 2] = J.nv               # chiral current: its right-handed partner sits J.nv entries further (index field u7)
            add(Task(T_FFV if is_left else T_FFVR, len(T), [parent, J], idx, out=f, mA=U if is_left else full ^ U, depth=depth))
            if is_left:
                trees = [tuple(ptrees[a]) + ((S, b),) for a in range(ntP) for b in range(ntS)]
            else:
                trees = [((S, b),) + tuple(ptrees[a]) for a in range(ntP) for b in range(ntS)]
            table[blocks] = (f, trees)
            return table[blocks]

        for part in D.ordered_partitions(full):
            m = len(part)
            if m < 2 and not self.dy:
                continue                       # (single-block diagrams of g g -> t t~ + gluons: full-set vertices closed with W0)
            if self.dy and any(self.nchoice(b) == 0 for b in part):
                continue                       # the electroweak boson is a block of its own
            last = part[-1]
            if self.nchoice(last) > 2:
                # W trick; one item per gluon-helicity assignment closes with the four (t, t~) variants of W
                parent, ptrees = chain(part[:-1], True)
                R, ntR, ntP = self.use[last], self.nchoice(last), len(ptrees)
                Wd = self._deps_union(parent.deps, tb_in)
                W = fam("W" + "_".join("%x" % b for b in part[:-1]), ntP, Wd, "W")
                T, H = np.meshgrid(np.arange(ntP), np.arange(W.nv), indexing="ij")
                T, H = T.ravel(), H.ravel()
                widx = np.zeros((len(T), 4), dtype=np.int64)
                widx[:, 0] = T * parent.nv + _restrict(H, Wd, parent.deps)
                widx[:, 1] = _restrict(H, Wd, tb_in)
                add(Task(T_WCUR, len(T), [parent, self.vsp], widx, out=W, depth=m - 1))
                DV, Hh = np.meshgrid(np.arange(ntP * ntR), np.arange(1 << len(gl)), indexing="ij")
                DV, Hh = DV.ravel(), Hh.ravel()
                tp, tr = DV // ntR, DV % ntR
                idx = np.zeros((len(DV), 4), dtype=np.int64)
                idx[:, 0] = tp * W.nv + self._deposit(Hh, gl, W.deps)          # W variant with t = t~ = -1
                idx[:, 1] = tr * R.nv + _restrict(Hh, gl, R.deps)
                idx[:, 2] = self._deposit(Hh, gl, self.inner)
                t = add(Task(T_AMP_DOT, len(DV), [W, R], idx, depth=m - 1,
                             mA=self._bitpos(W.deps, lr), mB=self._bitpos(W.deps, lc)))
                t.rpc = 1 << len(gl)
                t.cols = [self._kappa(list(ptrees[a]) + [(last, b)]) for a in range(ntP) for b in range(ntR)]
                t.col_names = [self._name(list(ptrees[a]) + [(last, b)]) for a in range(ntP) for b in range(ntR)]
            else:
                nl = (m - 1) // 2
                Lf, ltrees = chain(part[:nl], True)
                Rf, rtrees = chain(part[nl + 1:], False)
                S = part[nl]
                J, ntS, ntL, ntQ = self.use[S], self.nchoice(S), len(ltrees), len(rtrees)
                # one item per gluon-helicity assignment closes the four (t, t~) variants: L(t) slash(J) R(t~).  If a gluon leg
                # enters only through the right chain, the item also runs over its two helicities (aux = number of such legs,
                # at most block_r): both rows L(t) slash(J) stay in registers for 8 or 16 amplitudes (28 operand loads
                # instead of 40, 44 instead of 80)
                only_r = [l for l in gl if l in Rf.deps and l not in Lf.deps and l not in J.deps][:self.block_r]
                glh = tuple(l for l in gl if l not in only_r)
                DV, Hh = np.meshgrid(np.arange(ntL * ntS * ntQ), np.arange(1 << len(glh)), indexing="ij")
                DV, Hh = DV.ravel(), Hh.ravel()
                tl, tS, tq = DV // (ntS * ntQ), (DV // ntQ) % ntS, DV % ntQ
                idx = np.zeros((len(DV), 5), dtype=np.int64)
                idx[:, 0] = tl * Lf.nv + self._deposit(Hh, glh, Lf.deps)       # left-chain variant with t = -1
                idx[:, 1] = tS * J.nv + _restrict(Hh, glh, J.deps)
                idx[:, 2] = tq * Rf.nv + self._deposit(Hh, glh, Rf.deps)       # right-chain variant with t~ = -1 (blocked legs = -1)
                idx[:, 3] = self._deposit(Hh, glh, self.inner)                 # helicity combination with t = t~ = -1
                sh = [self._bitpos(Rf.deps, l) for l in only_r] + [0, 0]       # bit positions of the blocked legs in the right chain's
                lsh = [self._bitpos(self.inner, l) for l in only_r] + [0, 0]   # variant index and in the helicity combination
                assert max(sh + lsh + [self._bitpos(Rf.deps, lc), self._bitpos(Lf.deps, lr)]) < 16
                idx[:, 4] = sh[1] | lsh[1] << 4                                 # second blocked leg (index-table field u7)
                if S == self.vmask and self.dy:
                    idx[:, 4] |= J.nv << 8                                      # chiral current: offset of its right-handed partner
                t = add(Task(T_AMP_FFV, len(DV), [Lf, J, Rf], idx, depth=m - 1, aux=len(only_r),
                             mA=self._bitpos(Rf.deps, lc) | sh[0] << 4, mB=self._bitpos(Lf.deps, lr) | lsh[0] << 4))
                t.rpc = 1 << len(glh)
                t.flops_item = FLOPS_AMP_FFV_ROWS + FLOPS_AMP_FFV_DOTS * (1 << len(only_r))
                t.cols = [self._kappa(list(ltrees[a]) + [(S, b)] + list(rtrees[c]))
                          for a in range(ntL) for b in range(ntS) for c in range(ntQ)]
                t.col_names = [self._name(list(ltrees[a]) + [(S, b)] + list(rtrees[c]))
                               for a in range(ntL) for b in range(ntS) for c in range(ntQ)]

    def _vertex_task(self, sp, outfam, W, add):
        """One vertex group: current (outfam) or closing amplitude with W (single-block diagrams)."""
        ts = self.ts
        kids = sp[1:3] if sp[0] == "v3" else sp[2:5]
        merged_v4 = sp[0] == "v4" and len(sp) == 7          # ('v4', s, A, B, C, targets, signs)
        first_tree = None if merged_v4 else sp[-1]
        s = 0 if sp[0] == "v3" else sp[1]
        mask = 0
        for m in kids:
            mask |= m
        kf = [(self.cur if outfam is not None else self.use)[m] for m in kids]     # currents are built from trees
        nts = [f.ntree for f in kf]
        ntree = int(np.prod(nts))
        gl = tuple(l for l in self.inner if l not in (self.leg_row, self.leg_col))     # inner gluon legs
        if outfam is not None:
            deps, nv = outfam.deps, outfam.nv
        else:
            deps, nv = gl, 1 << len(gl)      # one item per gluon-helicity assignment: it closes with all (t, t~) variants of W
        tt = np.arange(ntree)
        hv = np.arange(nv)
        T, H = np.meshgrid(tt, hv, indexing="ij")
        T, H = T.ravel(), H.ravel()
        rem = T.copy()
        tidx = []
        for n in reversed(nts):
            tidx.append(rem % n)
            rem = rem // n
        tidx = tidx[::-1]
        idx = np.zeros((len(T), 4), dtype=np.int64)
        for k, f in enumerate(kf):
            idx[:, k] = tidx[k] * f.nv + _restrict(H, deps, f.deps)
        if outfam is not None and merged_v4 and self.fuse_quartic:
            return                               # evaluated inside the VVVF items of the trees it is merged into
        if outfam is not None and sp[0] == "v3" and self.fuse_quartic:
            # fused tree current: V3(A, B) plus, for every composite child c = (x, y) of the tree, the merged quartic structure
            # sign * ((x.z) y - (y.z) x) with z the other child
            qsign = self._quartic_signs(mask)
            xfam = np.full((len(T), 4), None, dtype=object)
            xrel = np.zeros((len(T), 4), dtype=np.int64)
            xflags = np.zeros(len(T), dtype=np.int64)
            extra = []
            nterm = 0
            for j in range(len(T)):
                tree = first_tree + int(T[j])
                node = ts.trees[mask][tree]
                assert node[0] == "v3" and node[1][0] == kids[0] and node[2][0] == kids[1]
                for q, c in enumerate((node[1], node[2])):
                    cn = ts.trees[c[0]][c[1]]
                    if cn[0] != "v3":
                        continue
                    sg = qsign[(tree, c)]
                    xflags[j] |= (1 | (2 if sg < 0 else 0)) << (2 * q)
                    nterm += 1
                    for r, (cm, ci) in enumerate((cn[1], cn[2])):
                        f = self.cur[cm]
                        xfam[j, 2 * q + r] = f
                        xrel[j, 2 * q + r] = ci * f.nv + _restrict(H[j:j + 1], deps, f.deps)[0]
                        if f not in extra:
                            extra.append(f)
            t = add(Task(T_VVVF, len(T), kf + [f for f in extra if f not in kf], idx, out=outfam, out_off=first_tree * nv, aux=0,
                         mA=kids[0], mB=kids[1], depth=0))
            t.xfam, t.xrel, t.xflags = xfam, xrel, xflags
            t.flops = FLOPS[T_VVV] * len(T) + F.VVVV_ACC * nterm
            self.store_tasks.setdefault(id(outfam), []).append(t)
            return
        if outfam is not None and merged_v4:
            # accumulate into the matching cubic trees: output slot and sign per item in index column 3
            tgt = np.array(sp[5])[T] * nv + H
            neg = (np.array(sp[6])[T] < 0).astype(np.int64)
            assert tgt.max() < 32768
            idx[:, 3] = tgt | (neg << 15)
            t = add(Task(T_VVVV, len(T), kf, idx, out=outfam, out_off=0, aux=s | 4, mA=mask, mB=0, depth=0))
            t.accumulate = True
            t.flops_item = F.VVVV_ACC
            t.out_slots = set(tgt.tolist())
            t.after = list(self.store_tasks.get(id(outfam), []))
        elif outfam is not None:
            ttype = T_VVV if sp[0] == "v3" else T_VVVV
            t = add(Task(ttype, len(T), kf, idx, out=outfam, out_off=first_tree * nv, aux=s,
                         mA=kids[0] if sp[0] == "v3" else mask, mB=kids[1] if sp[0] == "v3" else 0, depth=0))
            self.store_tasks.setdefault(id(outfam), []).append(t)
        else:
            assert W.deps == (2, 3)
            idx[:, len(kf)] = self._deposit(H, gl, self.inner)          # helicity combination with t = t~ = -1
            ttype = T_AMP_VVV if sp[0] == "v3" else T_AMP_VVVV
            t = add(Task(ttype, len(T), kf + [W], idx, aux=s | (4 if merged_v4 else 0), mA=kids[0] if sp[0] == "v3" else mask,
                         mB=kids[1] if sp[0] == "v3" else 0, depth=0))
            t.rpc = nv
            if merged_v4:
                # folded top level: += into the amplitude column of the cubic tree with the same colour factor
                t.accumulate = True
                t.col_of_item = np.array(sp[5])[T]
                t.neg_of_item = (np.array(sp[6])[T] < 0).astype(np.int64)
                t.out_slots = set(t.col_of_item.tolist())
                t.top = "acc"
                t.after = list(self.top_store_tasks)
            else:
                t.cols = []
                t.col_names = []
                for dv in range(ntree):
                    if self.chan:
                        assert sp[0] == "v3"
                        t.col_names.append("(" + "".join(self.ts.name(m, int(tidx[k][dv * nv])) for k, m in enumerate(kids)) + ")")
                    pol = [self.choice_colour(m, int(tidx[k][dv * nv])) for k, m in enumerate(kids)]
                    if sp[0] == "v3":
                        poly = D._scale(-1j, D._comm(pol[0], pol[1]))
                    else:
                        a, b, c = [(0, 1, 2), (0, 2, 1), (1, 2, 0)][s]
                        poly = D._scale(-1, D._comm(D._comm(pol[a], pol[b]), pol[c]))
                    t.cols.append(self._kappa_poly(poly, 1))
                if self.fold_top:
                    t.top = "store"
                    t.first_tree = first_tree
                    self.top_store_tasks.append(t)

    def _quartic_signs(self, mask):
        """{(tree index, composite child (mask, index)): sign} of the four-gluon structures merged into the cubic trees of `mask`."""
        if not hasattr(self, "_qsigns"):
            self._qsigns = {}
        if mask not in self._qsigns:
            ts, out = self.ts, {}
            for sp in ts.splits[mask]:
                if sp[0] != "v4" or len(sp) != 7:
                    continue
                s, (A, B, Cm) = sp[1], sp[2:5]
                k = 0
                for iA in range(ts.ntrees(A)):
                    for iB in range(ts.ntrees(B)):
                        for iC in range(ts.ntrees(Cm)):
                            X, Y, Z = (A, iA), (B, iB), (Cm, iC)
                            pair = [(X, Y), (X, Z), (Y, Z)][s]
                            pm = pair[0][0] | pair[1][0]
                            inner = (pm, ts.cubic_index[pm][frozenset(pair)])
                            assert (sp[5][k], inner) not in out
                            out[(sp[5][k], inner)] = sp[6][k]
                            k += 1
            self._qsigns[mask] = out
        return self._qsigns[mask]

    def _name(self, blocks):
        """channel name of the diagram with these blocks along the quark line (multichannel program only)."""
        return "|".join(self.ts.name(m, i) for m, i in blocks) if self.chan else None

    def _kappa(self, blocks):
        """{flow index: kappa code} of a diagram given as [(mask, tree index)] along the quark line."""
        poly = {(): 1 + 0j}
        for m, i in blocks:
            poly = D._mul(poly, self.choice_colour(m, i))
        return self._kappa_poly(poly, len(blocks))

    def _kappa_poly(self, poly, nblocks):
        # every k-gluon current carries the phase (-i)^(k-1) of its colour factor (the three-gluon vertex stores
        # -V/K^2 instead of -i V/K^2, the four-gluon structures +L/K^2): what is left of kappa is a sign, code 0 or 2
        phase = (-1j) ** (self.ng - nblocks)
        out = {self.flow_index[p]: D.kappa_code(c / phase) for p, c in poly.items() if c != 0}
        assert all(code in (0, 2) for code in out.values())
        return out

    def _chains(self, prefix, parent, parent_trees, used, add, fam):
        """parent: chain family of `prefix` (ubar for the empty prefix); parent_trees: list of block-tree tuples, one per
        tree entry of the parent family, each a tuple of (mask, tree index)."""
        ts = self.ts
        rest = self.full ^ used
        depth = len(prefix)
        t_in = (2,) if 2 in self.inner else ()
        tb_in = (3,) if 3 in self.inner else ()
        # closing amplitudes (final block = rest), not for the empty prefix (handled by the full-set vertices)
        if depth > 0:
            R = self.use[rest]
            ntR = self.nchoice(rest)
            ntP = len(parent_trees)
            ndv = ntP * ntR
            cols = [self._kappa(list(parent_trees[a]) + [(rest, b)]) for a in range(ntP) for b in range(ntR)]
            gl = tuple(l for l in self.inner if l not in (2, 3))
            assert t_in and tb_in, "the quark helicities are inner legs in every configuration"
            if ntR > 2:
                # W trick; one item per gluon-helicity assignment closes with the four (t, t~) variants of W
                Wd = self._deps_union(parent.deps, tb_in)
                W = fam("W" + "_".join("%x" % m for m in prefix), ntP, Wd, "W")
                T, H = np.meshgrid(np.arange(ntP), np.arange(W.nv), indexing="ij")
                T, H = T.ravel(), H.ravel()
                widx = np.zeros((len(T), 4), dtype=np.int64)
                widx[:, 0] = T * parent.nv + _restrict(H, Wd, parent.deps)
                widx[:, 1] = _restrict(H, Wd, tb_in)
                add(Task(T_WCUR, len(T), [parent, self.vsp], widx, out=W, depth=depth))
                legsH = gl
                DV, Hh = np.meshgrid(np.arange(ndv), np.arange(1 << len(legsH)), indexing="ij")
                DV, Hh = DV.ravel(), Hh.ravel()
                tp, tr = DV // ntR, DV % ntR
                idx = np.zeros((len(DV), 4), dtype=np.int64)
                idx[:, 0] = tp * W.nv + self._deposit(Hh, legsH, W.deps)         # W variant with t = t~ = -1
                idx[:, 1] = tr * R.nv + _restrict(Hh, legsH, R.deps)
                idx[:, 2] = self._deposit(Hh, legsH, self.inner)
                t = add(Task(T_AMP_DOT, len(DV), [W, R], idx, depth=depth,
                             mA=self._bitpos(W.deps, 2), mB=self._bitpos(W.deps, 3)))
                t.rpc = 1 << len(legsH)
            else:
                # one item per gluon-helicity assignment closes the four (t, t~) variants
                DV, Hh = np.meshgrid(np.arange(ndv), np.arange(1 << len(gl)), indexing="ij")
                DV, Hh = DV.ravel(), Hh.ravel()
                tp, tr = DV // ntR, DV % ntR
                idx = np.zeros((len(DV), 4), dtype=np.int64)
                idx[:, 0] = tp * parent.nv + self._deposit(Hh, gl, parent.deps)
                idx[:, 1] = tr * R.nv + _restrict(Hh, gl, R.deps)
                idx[:, 3] = self._deposit(Hh, gl, self.inner)
                t = add(Task(T_AMP_FFV, len(DV), [parent, R, self.vsp], idx, depth=depth, mA=0, mB=self._bitpos(parent.deps, 2)))
                t.rpc = 1 << len(gl)
            t.cols = cols
        # extend the chain by one more block S (proper subset of rest)
        for S in sorted(D.submasks(rest)):
            if S == rest:
                continue
            J = self.use[S]
            ntS = self.nchoice(S)
            deps = self._deps_union(parent.deps if depth else t_in, self.gdeps(S))
            nv = 1 << len(deps)
            ntP = len(parent_trees)
            # chunk the tree range of the new block so that no family exceeds chunk_items
            per_tree = ntP * nv
            step = ntS
            if self.chunk_items and per_tree * ntS > self.chunk_items:
                step = max(1, self.chunk_items // per_tree)
            for lo in range(0, ntS, step):
                hi = min(ntS, lo + step)
                ntree = ntP * (hi - lo)
                f = fam("C" + "_".join("%x" % m for m in prefix + (S,)) + ("[%d:%d]" % (lo, hi) if step < ntS else ""),
                        ntree, deps, "dt" if J.arena == "top" else "d%d" % (depth + 1))
                self.chain_depth_max = max(self.chain_depth_max, depth + 1)
                T, H = np.meshgrid(np.arange(ntree), np.arange(nv), indexing="ij")
                T, H = T.ravel(), H.ravel()
                tp, tS = T // (hi - lo), T % (hi - lo) + lo
                idx = np.zeros((len(T), 4), dtype=np.int64)
                idx[:, 0] = tp * parent.nv + _restrict(H, deps, parent.deps)
                idx[:, 1] = tS * J.nv + _restrict(H, deps, J.deps)
                add(Task(T_FFV, len(T), [parent, J], idx, out=f, mA=used | S, depth=depth + 1))
                trees = [tuple(parent_trees[a]) + ((S, b),) for a in range(ntP) for b in range(lo, hi)]
                self._chains(prefix + (S,), f, trees, used | S, add, fam)

    # ------------------------------------------------------------------------------------------------ scheduling
    def _schedule(self):
        perm = [f for f in self.fams if f.arena == "perm"]
        base = 0
        for f in perm:
            f.base = base
            base += f.nitems
        self.perm_slots = base
        # arenas for chain depths and W, sized by demand with the largest family as floor
        if self.bg:
            names = ["top"] if self.stream_top else []
        else:
            names = ["d%d" % d for d in range(1, self.chain_depth_max + 1)] + ["W"] + (["top", "dt"] if self.stream_top else [])
        demand = {n: sum(f.nitems for f in self.fams if f.arena == n) for n in names}
        floor = {n: max([f.nitems for f in self.fams if f.arena == n] + [0]) for n in names}
        if self.stream_top:
            # room for two of the largest streamed families (one being consumed while the next is produced)
            floor["top"] = min(demand["top"], int(self.top_factor * floor["top"]))
            demand["top"] = floor["top"]
        avail = self.slot_budget - base
        if sum(floor.values()) > avail:
            raise ValueError("slot budget %d too small: permanent %d + largest families %s" % (self.slot_budget, base, floor))
        extra = avail - sum(floor.values())
        want = {n: (demand[n] - floor[n]) * self.arena_weights.get(n, 1.0) for n in names}
        tot = max(1, sum(want.values()))
        self.arenas = {}
        for n in names:
            size = floor[n] + int(min(demand[n] - floor[n], extra * want[n] // tot))
            self.arenas[n] = Arena(base, size)
            base += size
        self.nslot = base

        # Pass-invariant items: a wavefunction that depends on no OUTER leg is the same in every outer-helicity pass of an event.  Where
        # the kernel runs the passes of an event back to back and keeps the wavefunction file (csrc/mg_vm.cuh KEEP_EXT) the units of
        # such tasks run in the first pass only ("first_only"); they must live in permanent slots.
        dep = {}
        for t in self.tasks:
            if t.type == T_EXT:
                d = any(int(l) in self.outer for l in t.idx[:, 0])
            else:
                d = any(dep[id(f)] for f in t.ins)
            t.first_only = (not d) and t.out is not None and t.out.arena == "perm" and t.type != T_EXT and not t.accumulate
            if t.out is not None:
                dep[id(t.out)] = dep.get(id(t.out), False) or d
        pending = list(self.tasks)
        self.phases = []            # list of lists of emitted task dicts
        col_used = 0                # amp columns waiting for accumulation
        col_kappa = []              # kappa dict per pending column
        self._col_names = []        # multichannel program: channel name per pending column
        prio = {T_EXT: 0, T_WCUR: 1, T_VVV: 1, T_VVVV: 1, T_VVVF: 1, T_COMB: 1, T_FFV: 2, T_FFVR: 2, T_QSUM: 2}
        self.exec_flops = 0
        self.first_only_flops = 0     # part of exec_flops in pass-invariant tasks
        self.acc_pairs = 0
        guard = 0
        if self.double_buffer:
            return self._schedule_double(pending, prio)
        while pending or col_used:
            guard += 1
            if guard > 100000:
                raise RuntimeError("scheduler made no progress")
            ready = [t for t in pending if all(f.complete for f in t.ins) and all(x.done for x in t.after)]
            top_acc = [t for t in ready if t.top == "acc"]
            top_store = [t for t in ready if t.top == "store"]
            amps = [t for t in ready if t.cols is not None and t.top is None]
            others = [t for t in ready if t.cols is None and t.top is None]
            others.sort(key=lambda t: (0 if any(f.arena == "top" for f in t.ins) else 1, prio[t.type], -t.depth))
            phase = []
            finished = []
            # folded top level: the cubic-top columns sit at fixed positions [0, ntop) of an empty buffer; the quartic
            # structures are then added into them in the following phases, and only after that the buffer is accumulated
            top_pending_acc = any(t.top == "acc" and not t.done for t in self.tasks)
            top_stored = all(t.done for t in self.top_store_tasks)
            want_top_store = bool(self.top_store_tasks) and not top_stored and len(top_store) == len(self.top_store_tasks)
            # accumulate when the buffer cannot take the next amp task's columns, or nothing else is ready
            want_acc = col_used > 0 and (not amps or col_used == self.ncol or
                                         all(len(t.cols) - t.done_cols > self.ncol - col_used for t in amps) and col_used * 2 >= self.ncol)
            if not amps and not others and col_used:
                want_acc = True
            if want_top_store and col_used > 0:
                want_acc = True                                   # empty the buffer first
            if top_stored and top_pending_acc:
                want_acc = False                                  # columns [0, ntop) still receive the quartic structures
            if want_acc:
                phase.extend(self._acc_tasks(col_kappa))
                col_used, col_kappa, self._col_names = 0, [], []
            else:
                if want_top_store:
                    ntop = self.ts.ntrees(self.full)
                    assert ntop <= self.ncol and col_used == 0
                    col_kappa = [None] * ntop
                    for t in top_store:
                        ncols_t = len(t.cols)
                        phase.append(dict(type=t.type, aux=t.aux, mA=t.mA, mB=t.mB, nitems=ncols_t * t.rpc, rpc=t.rpc,
                                          idx=t.idx, in_base=[f.base for f in t.ins], out_base=t.first_tree))
                        self.exec_flops += FLOPS[t.type] * ncols_t * t.rpc
                        col_kappa[t.first_tree:t.first_tree + ncols_t] = t.cols
                        t.done_cols = ncols_t
                        finished.append(t)
                    assert all(k is not None for k in col_kappa)
                    col_used = ntop
                busy_cols = set()
                for t in top_acc:
                    if busy_cols & t.out_slots:
                        continue                                  # two structures adding into the same column: next phase
                    busy_cols |= t.out_slots
                    phase.append(dict(type=t.type, aux=t.aux, mA=t.mA, mB=t.mB, nitems=t.nitems, rpc=t.rpc, idx=t.idx,
                                      in_base=[f.base for f in t.ins], out_base=0,
                                      col_of_item=t.col_of_item, neg_of_item=t.neg_of_item))
                    self.exec_flops += FLOPS[t.type] * t.nitems
                    finished.append(t)
                amps.sort(key=lambda t: (0 if any(f.arena == "top" for f in t.ins) else 1, -t.depth))
                for t in amps:
                    if col_used == self.ncol:
                        break
                    ncols = len(t.cols) - t.done_cols
                    take = min(ncols, self.ncol - col_used)
                    lo = t.done_cols
                    phase.append(dict(type=t.type, aux=t.aux, mA=t.mA, mB=t.mB, nitems=take * t.rpc, rpc=t.rpc,
                                      idx=t.idx[lo * t.rpc:(lo + take) * t.rpc], in_base=[f.base for f in t.ins],
                                      out_base=col_used))
                    self.exec_flops += (FLOPS[t.type] if t.flops_item is None else t.flops_item) * take * t.rpc
                    col_kappa.extend(t.cols[lo:lo + take])
                    if self.chan:
                        self._col_names.extend(t.col_names[lo:lo + take])
                    col_used += take
                    t.done_cols += take
                    if t.done_cols == len(t.cols):
                        finished.append(t)
            acc_busy = {}
            for t in others:
                f = t.out
                if f is None:
                    # closing sum of a colour flow (QSUM, aux = 1): adds into jamp, so never beside an accumulation task
                    assert t.type == T_QSUM
                    if want_acc and not self.fuse_closing:
                        continue
                    phase.append(dict(type=t.type, aux=t.aux, mA=t.mA, mB=t.mB, nitems=t.nitems, idx=t.idx,
                                      in_base=[g.base for g in t.ins], in_cols=t.in_cols, out_base=0, flow=t.flow))
                    self.exec_flops += t.flops_item * t.nitems
                    finished.append(t)
                    continue
                if t.accumulate:
                    busy = acc_busy.setdefault(id(f), set())
                    if busy & t.out_slots:
                        continue                  # another task adds into the same slots in this phase
                    busy |= t.out_slots
                if f.base is None:
                    b = self.arenas[f.arena].alloc(f.nitems)
                    if b is None:
                        continue
                    f.base = b
                phase.append(dict(type=t.type, aux=t.aux, mA=t.mA, mB=t.mB, nitems=t.nitems, idx=t.idx,
                                  in_base=[g.base for g in t.ins], out_base=f.base + t.out_off, first_only=t.first_only))
                if t.type == T_QSUM:
                    phase[-1]["in_cols"] = t.in_cols
                if t.type == T_VVVF:
                    xs = np.zeros(t.xrel.shape, dtype=np.int64)
                    for (j, q), fm in np.ndenumerate(t.xfam):
                        if fm is not None:
                            assert fm.base is not None and fm.complete
                            xs[j, q] = fm.base + t.xrel[j, q]
                    phase[-1]["xslots"], phase[-1]["xflags"] = xs, t.xflags
                before = self.exec_flops
                if t.flops is not None:
                    self.exec_flops += t.flops
                else:
                    self.exec_flops += (FLOPS[t.type] if t.flops_item is None else t.flops_item) * t.nitems
                if t.first_only:
                    self.first_only_flops += self.exec_flops - before
                finished.append(t)
            if not phase:
                raise RuntimeError("deadlock: %d tasks pending, arenas %s" % (len(pending), {n: a.free for n, a in self.arenas.items()}))
            self.phases.append(phase)
            for t in finished:
                t.done = True
                pending.remove(t)
                if t.out is not None:
                    t.out.producers_left -= 1
                    if t.out.producers_left == 0:
                        t.out.complete = True
                for f in t.ins:
                    f.consumers_left -= 1
            for f in self.fams:
                if f.arena != "perm" and f.complete and f.consumers_left == 0 and f.base is not None:
                    self.arenas[f.arena].release(f.base, f.nitems)
                    f.base = None
                    f.consumers_left = -1
        self.exec_flops += FLOPS_ACC_PAIR * self.acc_pairs * self.NC

    def _schedule_double(self, pending, prio):
        """Amplitude buffer used as two halves: while one half is filled by the amplitude tasks of a phase, the other half
        (filled in the previous phase) is accumulated into jamp, so that the shared-memory-bound accumulation overlaps
        with the FP64-bound arithmetic."""
        half = self.ncol // 2
        cur = 0
        pend = {0: [], 1: []}
        guard = 0
        while pending or pend[0] or pend[1]:
            guard += 1
            if guard > 100000:
                raise RuntimeError("scheduler made no progress")
            ready = [t for t in pending if all(f.complete for f in t.ins) and all(x.done for x in t.after)]
            amps = [t for t in ready if t.cols is not None]
            others = [t for t in ready if t.cols is None]
            others.sort(key=lambda t: (0 if any(f.arena == "top" for f in t.ins) else 1, prio[t.type], -t.depth))
            phase, finished = [], []
            other = 1 - cur
            if pend[other]:
                phase.extend(self._acc_tasks(pend[other], other * half))
                pend[other] = []
            if pend[cur] and not amps:
                cur = other
            else:
                amps.sort(key=lambda t: (0 if any(f.arena == "top" for f in t.ins) else 1, -t.depth))
                for t in amps:
                    used = len(pend[cur])
                    if used == half:
                        break
                    take = min(len(t.cols) - t.done_cols, half - used)
                    lo = t.done_cols
                    phase.append(dict(type=t.type, aux=t.aux, mA=t.mA, mB=t.mB, nitems=take * t.rpc, rpc=t.rpc,
                                      idx=t.idx[lo * t.rpc:(lo + take) * t.rpc], in_base=[f.base for f in t.ins],
                                      out_base=cur * half + used))
                    self.exec_flops += (FLOPS[t.type] if t.flops_item is None else t.flops_item) * take * t.rpc
                    pend[cur].extend(t.cols[lo:lo + take])
                    t.done_cols += take
                    if t.done_cols == len(t.cols):
                        finished.append(t)
                if pend[cur]:
                    cur = other
            acc_busy = {}
            for t in others:
                f = t.out
                if t.accumulate:
                    busy = acc_busy.setdefault(id(f), set())
                    if busy & t.out_slots:
                        continue                  # another task adds into the same slots in this phase
                    busy |= t.out_slots
                if f.base is None:
                    b = self.arenas[f.arena].alloc(f.nitems)
                    if b is None:
                        continue
                    f.base = b
                phase.append(dict(type=t.type, aux=t.aux, mA=t.mA, mB=t.mB, nitems=t.nitems, idx=t.idx,
                                  in_base=[g.base for g in t.ins], out_base=f.base + t.out_off))
                self.exec_flops += FLOPS[t.type] * t.nitems if t.flops is None else t.flops
                finished.append(t)
            if not phase:
                raise RuntimeError("deadlock: %d tasks pending" % len(pending))
            self.phases.append(phase)
            for t in finished:
                t.done = True
                pending.remove(t)
                if t.out is not None:
                    t.out.producers_left -= 1
                    if t.out.producers_left == 0:
                        t.out.complete = True
                for f in t.ins:
                    f.consumers_left -= 1
            for f in self.fams:
                if f.arena != "perm" and f.complete and f.consumers_left == 0 and f.base is not None:
                    self.arenas[f.arena].release(f.base, f.nitems)
                    f.base = None
                    f.consumers_left = -1
        self.exec_flops += FLOPS_ACC_PAIR * self.acc_pairs * self.NC

    def _acc_tasks(self, col_kappa, col_base=0):
        """One ACC task: for every flow touched by the pending columns, the list of (column, kappa code).
        Multichannel program: one CHAN task instead, which adds |A|^2 of every pending column into the channel sums."""
        if self.chan:
            assert len(self._col_names) == len(col_kappa) and col_base == 0
            self.exec_flops += 4 * len(col_kappa) * self.NC
            self.exec_flops += (F.CHAN_COL - 4) * len(col_kappa) * self.NC
            return [dict(type=T_CHAN, aux=0, mA=0, mB=0, nitems=len(col_kappa), names=list(self._col_names), kappas=list(col_kappa),
                         in_base=[], out_base=0)]
        per_flow = {}
        for col, kd in enumerate(col_kappa):
            for fl, code in kd.items():
                per_flow.setdefault(fl, []).append((col_base + col, code))
        flows = sorted(per_flow)
        lists = [per_flow[f] for f in flows]
        self.acc_pairs += sum(len(l) for l in lists)
        return [dict(type=T_ACC, aux=0, mA=0, mB=0, nitems=len(flows), flows=flows, lists=lists, in_base=[], out_base=0)]

    # ------------------------------------------------------------------------------------------------ accounting
    def flops_executed_per_event(self, keep_first=False):
        """Flops this program executes per event (all outer assignments): the scheduled items (counted per routine,
        emitter/flops.py), the colour stage as csrc/mg_vm.cuh runs it, the colour-flow weights and the per-event setup.
        keep_first: the pass-invariant tasks run in the first outer pass only (emit.py keep_first)."""
        NL = self.NL
        if self.chan:
            colour = weights = 0
        elif self.E == 1 and NL == 32 and self.ncolor % 8 == 0 and self.ncolor >= 24:
            # FP64 tensor cores: 64 rows x block pairs kb <= nb of 8 x 8 blocks, m8n8k4 = 512 flops; then Y o X (one FMA per element)
            # (J+- form: two half-size diagonal blocks; block pairs kb <= nb with kb >= (ncolor / 2) // 8 once the column block lies
            # in the second half), plus the butterfly J+- = J_sigma +- J_reversed
            nb, hb = self.ncolor // 8, (self.ncolor // 2) // 8
            pairs = sum(n - (hb if n * 8 >= self.ncolor // 2 else 0) + 1 for n in range(nb))
            colour = pairs * 2 * 8 * 512 + 2 * 64 * self.ncolor + 2 * 64 * self.ncolor // 2
        else:
            # symmetric blocked form: RPT rows per thread against the columns t >= g * RPT, two FMAs per (row, column, lane)
            G = max(1, self.nthreads // NL)
            RPT = (self.ncolor + G - 1) // G
            GU = (self.ncolor + RPT - 1) // RPT
            nit = GU * self.ncolor - RPT * (GU * (GU - 1) // 2)
            colour = (4 * nit * RPT + 4 * self.ncolor) * self.NC * self.E // self.E
        if not self.chan:
            weights = 4 * self.ncolor * self.NC                        # |J|^2: two FMAs per (flow, helicity lane)
        # subset momenta and propagator denominators: once per event when the outer passes share a CTA (four or more), else per pass
        setup = F.setup_flops(self.ng)          # once per event: the outer passes of an event share a CTA (csrc/mg_vm.cuh MG_PER_TILE_MIN)
        skipped = self.first_only_flops * (self.nouter - 1) if keep_first else 0
        return (self.exec_flops + colour + weights) * self.nouter - skipped + setup + (1 << self.npar)     # + helicity sum

    def flops_canonical_per_event(self):
        if self.dy:
            return self._flops_canonical_dy()
        return self._flops_canonical_tt()

    def _flops_canonical_dy(self):
        """Drell-Yan: per helicity combination (all 2^npar, no recycling) the external wavefunctions, the boson current, every distinct
        gluon subtree current once, and per diagram structure its chain of quark propagators plus one closing."""
        ts = self.ts_full
        per_hel = F.EXT_EPS * self.ngl + 2 * F.EXT_SPINOR + (2 * F.EXT_SPINOR + F.WCUR + 60) + F.setup_flops(self.ng)
        for mask in range(1, self.full + 1):
            for sp in ts.splits[mask]:
                kids = sp[1:3] if sp[0] == "v3" else sp[2:5]
                per_hel += int(np.prod([ts.ntrees(m) for m in kids])) * (FLOPS[T_VVV] if sp[0] == "v3" else FLOPS[T_VVVV])
        nchain = namp = pairs = 0
        for part in D.ordered_partitions(self.full):
            n = int(np.prod([ts.ntrees(S) for S in part]))
            namp += n
            nchain += n * (len(part) - 1)
            pairs += n * int(np.prod([1 << max(0, bin(S & ~self.vmask).count("1") - 1) for S in part]))
        per_hel += nchain * FLOPS[T_FFV] + namp * FLOPS_CANON[T_AMP_FFV]
        per_hel += FLOPS_ACC_PAIR * pairs + 4 * self.ncolor * self.ncolor + 2 * self.ncolor
        return per_hel * (1 << self.npar), dict(nchain=nchain, namp_multi=namp, pairs=pairs)

    def _flops_canonical_tt(self):
        """the method as the paper runs it -- per helicity combination every distinct off-shell
        wavefunction once, one amplitude per diagram structure, kappa accumulation, dense colour form; no recycling."""
        ts = self.ts_full
        per_hel = F.EXT_EPS * self.ng + F.EXT_SPINOR * 2 + F.setup_flops(self.ng)
        for mask in range(1, self.full + 1):
            for sp in ts.splits[mask]:
                kids = sp[1:3] if sp[0] == "v3" else sp[2:5]
                n = int(np.prod([ts.ntrees(m) for m in kids]))
                if mask == self.full:
                    per_hel += n * (FLOPS_CANON[T_AMP_VVV] if sp[0] == "v3" else FLOPS_CANON[T_AMP_VVVV])
                else:
                    per_hel += n * (FLOPS[T_VVV] if sp[0] == "v3" else FLOPS[T_VVVV])
        per_hel += FLOPS[T_WCUR]
        nchain = namp2 = 0
        for part in D.ordered_partitions(self.full):
            if len(part) < 2:
                continue
            n = 1
            for S in part:
                n *= ts.ntrees(S)
            namp2 += n
        # distinct chains: every proper ordered prefix with its tree choices
        def chains(used):
            tot = 0
            rest = self.full ^ used
            for S in D.submasks(rest):
                if S == rest:
                    continue
                sub = chains(used | S)
                tot += ts.ntrees(S) * (1 + sub)
            return tot
        nchain = chains(0)
        per_hel += nchain * FLOPS[T_FFV] + namp2 * FLOPS_CANON[T_AMP_FFV]
        pairs = 0
        for part in D.ordered_partitions(self.full):
            n = 1
            for S in part:
                n *= ts.ntrees(S) * (1 << (bin(S).count("1") - 1))
            pairs += n
        per_hel += FLOPS_ACC_PAIR * pairs + 4 * self.ncolor * self.ncolor + 2 * self.ncolor
        return per_hel * (1 << self.npar), dict(nchain=nchain, namp_multi=namp2, pairs=pairs)

    def summary(self):
        nt = sum(len(p) for p in self.phases)
        items = sum(t["nitems"] for p in self.phases for t in p if t["type"] != T_ACC)
        return dict(ng=self.ng, ndiag=self.ndiag, namp=self.namp, ncolor=self.ncolor, NC=self.NC, nouter=self.nouter, E=self.E,
                    nslot=self.nslot, perm_slots=self.perm_slots, phases=len(self.phases), tasks=nt, items=items,
                    acc_pairs=self.acc_pairs, flops_exec=self.flops_executed_per_event(),
                    flops_canonical=self.flops_canonical_per_event()[0])
