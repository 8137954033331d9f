"""Diagram and colour tables for g g -> t t~ + (ng-2) g, written for the CUDA path's emitter.

This is the emitter's OWN enumeration (it shares no code with oracle/): gluon subtrees on label sets, diagrams as
ordered block sequences along the quark line, colour coefficients kappa(d, sigma) from
commutator expansion and the colour matrix from the SU(3) Fierz identity in exact rational arithmetic (C-C;
PAPER.md:200 "colour matrix of integer coefficients").
Gluon index g = 0..ng-1 stands for leg g (g < 2, initial state) or leg g + 2 (final state).
"""
from fractions import Fraction
from functools import lru_cache
from itertools import permutations


def gluon_leg(g):
    return g if g < 2 else g + 2


def bits(mask):
    return [i for i in range(mask.bit_length()) if mask >> i & 1]


def submasks(mask):
    s = mask
    while s:
        yield s
        s = (s - 1) & mask


class TreeSet:
    """All gluon subtrees (quartic vertices expanded into their 3 colour/Lorentz structures) on every label set.

    trees[mask] is a list of nodes; a node is ('leaf', g) | ('v3', (maskA, iA), (maskB, iB)) |
    ('v4', s, (maskA, iA), (maskB, iB), (maskC, iC)); children are (mask, index into trees[mask]).
    splits[mask] lists the vertex groups in the same order: ('v3', A, B, first_tree) / ('v4', s, A, B, C, first_tree):
    within a group the trees run over (iA, iB[, iC]) in row-major order starting at first_tree.
    """

    def __init__(self, ng, merged=False, fold_top=False, cubic_only=False, vlabel=None):
        """merged=True: below the full label set, a four-gluon structure is not a tree of its own.  Its colour factor
        -[[X,Y],Z] equals that of the nested three-gluon tree ((X,Y),Z) ((-i)^2 [[X,Y],Z]), so its kinematic value is
        ADDED (with the relative sign of the two colour polynomials) to that tree's current: an exact regrouping that
        leaves (2k-3)!! = 1, 1, 3, 15 trees per k-gluon label set.  splits[mask] then lists for every quartic group
        ('v4', s, A, B, C, targets, signs): the tree index and sign per (iA, iB, iC) in row-major order.
        On the full label set quartic structures stay separate amplitude columns."""
        self.ng = ng
        self.merged = merged
        self.fold_top = fold_top      # merged only: fold the quartic structures of the FULL label set too
        self.cubic_only = cubic_only  # no four-gluon vertices at all: the trees of the multichannel channels
        # vlabel: label of a colourless electroweak boson on the quark line (Drell-Yan): a block of its own (node
        # ('ew',), colour factor 1), never part of a gluon subtree.  ng then counts the gluons AND this label.
        self.vlabel = vlabel
        self.full = (1 << ng) - 1
        self.trees = {}
        self.splits = {}
        self.cubic_index = {}
        for mask in sorted(range(1, 1 << ng), key=lambda m: (bin(m).count("1"), m)):
            self._build(mask)

    def _build(self, mask):
        b = bits(mask)
        trees, splits = [], []
        if self.vlabel is not None and mask >> self.vlabel & 1:
            self.trees[mask] = [("ew",)] if len(b) == 1 else []
            self.splits[mask] = []
            self.cubic_index[mask] = {}
            return
        if len(b) == 1:
            trees.append(("leaf", b[0]))
        else:
            low = mask & -mask
            for A in sorted(submasks(mask)):
                if A == mask or not (A & low):
                    continue
                B = mask ^ A
                splits.append(("v3", A, B, len(trees)))
                for iA in range(len(self.trees[A])):
                    for iB in range(len(self.trees[B])):
                        trees.append(("v3", (A, iA), (B, iB)))
            self.cubic_index[mask] = {frozenset(n[1:]): i for i, n in enumerate(trees)}
            self.trees[mask] = trees           # colour() of the cubic trees of this mask is needed below
            for A in ([] if self.cubic_only else sorted(submasks(mask))):
                if A == mask or not (A & low):
                    continue
                rest = mask ^ A
                low2 = rest & -rest
                for B in sorted(submasks(rest)):
                    if B == rest or not (B & low2):
                        continue
                    Cm = rest ^ B
                    for s in range(3):
                        if self.merged and (mask != self.full or self.fold_top):
                            targets, signs = [], []
                            for iA in range(len(self.trees[A])):
                                for iB in range(len(self.trees[B])):
                                    for iC in range(len(self.trees[Cm])):
                                        X, Y, Z = (A, iA), (B, iB), (Cm, iC)
                                        pair, third = [((X, Y), Z), ((X, Z), Y), ((Y, Z), X)][s]
                                        inner = (pair[0][0] | pair[1][0], self.cubic_index[pair[0][0] | pair[1][0]][frozenset(pair)])
                                        tgt = self.cubic_index[mask][frozenset((inner, third))]
                                        cq, ct = self.colour_v4(s, X, Y, Z), self.colour(mask, tgt)
                                        if cq == ct:
                                            sg = 1
                                        else:
                                            assert cq == _scale(-1, ct), "quartic structure does not match its cubic tree"
                                            sg = -1
                                        targets.append(tgt)
                                        signs.append(sg)
                            splits.append(("v4", s, A, B, Cm, targets, signs))
                        else:
                            splits.append(("v4", s, A, B, Cm, len(trees)))
                            for iA in range(len(self.trees[A])):
                                for iB in range(len(self.trees[B])):
                                    for iC in range(len(self.trees[Cm])):
                                        trees.append(("v4", s, (A, iA), (B, iB), (Cm, iC)))
        self.trees[mask] = trees
        self.splits[mask] = splits

    def ntrees(self, mask):
        return len(self.trees[mask])

    def name(self, mask, idx):
        """Canonical name of a cubic tree: a leaf is its gluon index as one digit, a vertex over the split {A, B} (A holds the
        lowest label) is "(" name(A) name(B) ")".  Channel names join the blocks along the quark line by "|" (DESIGN.md reading
        "channels"); the channels are numbered in ascending byte order of their names."""
        node = self.trees[mask][idx]
        if node[0] == "leaf":
            return str(node[1])
        assert node[0] == "v3"
        return "(" + self.name(*node[1]) + self.name(*node[2]) + ")"

    # ---- colour: polynomial in T-strings, dict {tuple(gluon order): Gaussian integer as complex} -------------
    @lru_cache(maxsize=None)
    def colour(self, mask, idx):
        node = self.trees[mask][idx]
        if node[0] == "leaf":
            return {(node[1],): 1 + 0j}
        if node[0] == "ew":
            return {(): 1 + 0j}
        if node[0] == "v3":
            X, Y = self.colour(*node[1]), self.colour(*node[2])
            return _scale(-1j, _comm(X, Y))                 # f^{abc} x^a y^b T^c = -i [X, Y]
        s = node[1]
        X, Y, Z = self.colour(*node[2]), self.colour(*node[3]), self.colour(*node[4])
        if s == 0:
            return _scale(-1, _comm(_comm(X, Y), Z))        # f^{abe} f^{cde}
        if s == 1:
            return _scale(-1, _comm(_comm(X, Z), Y))        # f^{ace} f^{bde}
        return _scale(-1, _comm(_comm(Y, Z), X))            # f^{ade} f^{bce}

    # ---- colour-ordered basis of the currents on a label set ------------------------------------------------------
    @lru_cache(maxsize=None)
    def ordered_basis(self, mask):
        """The colour-dressed current on a k-gluon label set is sum_tree C_tree J_tree = sum_pi pi Jord[pi] with
        Jord[pi] = sum_tree c_tree(pi) J_tree (c = coefficient of the T-string pi in C_tree, a sign once the phase
        (-i)^(k-1) of the current is split off).  Every commutator changes sign under reversal of the string, so
        Jord[reversed pi] = (-1)^(k-1) Jord[pi]: k!/2 independent ordered currents instead of (2k-3)!! trees, each
        with a two-term colour polynomial instead of 2^(k-1) terms.  An exact regrouping of the same diagram sum.
        Returns (orderings with pi[0] < pi[-1] in lexicographic order, per ordering [(tree index, sign)])."""
        b = bits(mask)
        k = len(b)
        phase = (-1j) ** (k - 1)
        perms = [p for p in permutations(b) if p[0] < p[-1]]
        comb = {p: [] for p in perms}
        for i in range(self.ntrees(mask)):
            poly = self.colour(mask, i)
            for p, c in poly.items():
                sg = c / phase
                assert sg in (1, -1)
                r = p[::-1]
                assert poly[r] == c * (-1) ** (k - 1)
                if p in comb:
                    comb[p].append((i, int(sg.real)))
        return perms, [comb[p] for p in perms]

    def colour_ordered(self, mask, o):
        """colour polynomial of ordered current o of `mask` (same convention as colour(): includes the phase)."""
        p = self.ordered_basis(mask)[0][o]
        k = len(p)
        phase = (-1j) ** (k - 1)
        return {p: phase, p[::-1]: phase * (-1) ** (k - 1)}

    def colour_v4(self, s, X, Y, Z):
        """colour polynomial of quartic structure s on subtrees X, Y, Z (each (mask, index))."""
        cx, cy, cz = self.colour(*X), self.colour(*Y), self.colour(*Z)
        if s == 0:
            return _scale(-1, _comm(_comm(cx, cy), cz))
        if s == 1:
            return _scale(-1, _comm(_comm(cx, cz), cy))
        return _scale(-1, _comm(_comm(cy, cz), cx))

    def n_quartic(self, mask, idx):
        node = self.trees[mask][idx]
        if node[0] in ("leaf", "ew"):
            return 0
        if node[0] == "v3":
            return self.n_quartic(*node[1]) + self.n_quartic(*node[2])
        return 1 + sum(self.n_quartic(*c) for c in node[2:])

    def first_structure_only(self, mask, idx):
        node = self.trees[mask][idx]
        if node[0] in ("leaf", "ew"):
            return True
        if node[0] == "v3":
            return self.first_structure_only(*node[1]) and self.first_structure_only(*node[2])
        return node[1] == 0 and all(self.first_structure_only(*c) for c in node[2:])


def _mul(a, b):
    r = {}
    for pa, ca in a.items():
        for pb, cb in b.items():
            r[pa + pb] = r.get(pa + pb, 0) + ca * cb
    return r


def _comm(a, b):
    r = _mul(a, b)
    for p, c in _mul(b, a).items():
        r[p] = r.get(p, 0) - c
    return {p: c for p, c in r.items() if c != 0}


def _scale(c, a):
    return {p: c * v for p, v in a.items()}


def flows(ng):
    """Colour flows = permutations of the gluon legs in lexicographic order of leg numbers (C-C)."""
    return list(permutations(range(ng)))


def kappa_code(c):
    """kappa in {1, i, -1, -i} -> 0..3 (power of i)."""
    table = {1 + 0j: 0, 1j: 1, -1 + 0j: 2, -1j: 3}
    return table[complex(c)]


def ordered_partitions(mask):
    """All ordered sequences of disjoint non-empty blocks with union `mask`."""
    if mask == 0:
        yield ()
        return
    for S in sorted(submasks(mask)):
        for rest in ordered_partitions(mask ^ S):
            yield (S,) + rest


def count_diagrams(ts):
    """(number of Feynman diagrams, number of amplitudes with 3 structures per quartic vertex)."""
    ndiag = namp = 0
    for part in ordered_partitions(ts.full):
        n_all = n_first = 1
        for S in part:
            n_all *= ts.ntrees(S)
            n_first *= sum(1 for i in range(ts.ntrees(S)) if ts.first_structure_only(S, i))
        namp += n_all
        ndiag += n_first
    return ndiag, namp


# ---- colour matrix from the Fierz identity, exact ---------------------------------------------------------------
def _trace_product(cycles_of_indices):
    """Evaluate a product of traces of generators with every adjoint index appearing exactly twice (summed).

    Representation: list of cyclic words (lists of index labels).  SU(N) Fierz:
      T^a_ij T^a_kl = 1/2 (delta_il delta_jk - 1/N delta_ij delta_kl), N = 3, tr(1) = N.
    Returns a Fraction.
    """
    N = 3
    words = [list(w) for w in cycles_of_indices]
    # find an index to contract
    for wi, w in enumerate(words):
        if w:
            a = w[0]
            break
    else:
        r = Fraction(1)
        for w in words:
            r *= N                                         # empty trace = tr(1)
        return r
    # locate the second occurrence of a
    pos = [(i, j) for i, w in enumerate(words) for j, x in enumerate(w) if x == a]
    (i1, j1), (i2, j2) = pos
    if i1 == i2:
        w = words[i1]
        # tr(T^a X T^a Y) with X = w[j1+1:j2], Y = w[j2+1:] + w[:j1]
        X = w[j1 + 1:j2]
        Y = w[j2 + 1:] + w[:j1]
        rest = words[:i1] + words[i1 + 1:]
        # = 1/2 ( tr(X) tr(Y) - 1/N tr(X Y) )
        return Fraction(1, 2) * (_trace_product(rest + [X, Y]) - Fraction(1, N) * _trace_product(rest + [X + Y]))
    w1, w2 = words[i1], words[i2]
    X = w1[j1 + 1:] + w1[:j1]                               # tr(T^a X)
    Y = w2[j2 + 1:] + w2[:j2]                               # tr(T^a Y)
    rest = [w for k, w in enumerate(words) if k not in (i1, i2)]
    # tr(T^a X) tr(T^a Y) = 1/2 ( tr(X Y) - 1/N tr(X) tr(Y) )
    return Fraction(1, 2) * (_trace_product(rest + [X + Y]) - Fraction(1, N) * _trace_product(rest + [X, Y]))


def colour_matrix(ng):
    """C[s][s'] = sum_a tr(T^{a_s(1)}..T^{a_s(n)} T^{a_s'(n)}..T^{a_s'(1)}) as exact Fractions (list of lists)."""
    fl = flows(ng)
    index = {f: i for i, f in enumerate(fl)}
    ident = fl[0]
    row = {}
    for f in fl:
        row[f] = _trace_product([list(ident) + list(reversed(f))])
    nc = len(fl)
    C = [[None] * nc for _ in range(nc)]
    for s, fs in enumerate(fl):
        relab = {fs[k]: ident[k] for k in range(ng)}        # relabel summed indices so that flow s becomes the identity
        for t, ft in enumerate(fl):
            C[s][t] = row[tuple(relab[x] for x in ft)]
    return C


def colour_matrix_integer(ng):
    """(numerators[nc][nc] as ints, common denominator)."""
    C = colour_matrix(ng)
    den = 1
    for r in C:
        for x in r:
            den = den * x.denominator // _gcd(den, x.denominator)
    return [[int(x * den) for x in r] for r in C], den


def _gcd(a, b):
    while b:
        a, b = b, a % b
    return a
