"""Flop counts of the device routines, counted instead of tallied by hand (real add / sub / mul = 1, FMA = 2,
div / sqrt = 1; a complex multiply is 6, a complex add 2).

Every routine of csrc/mg_vm.cuh is restated here on a counting scalar, operation by operation and in the same order, and run
once; the number of arithmetic operations it performed is the routine's flop count.  Multiplications by a literal +-1 and
sign flips are not counted (the compiler folds them into negated FMA operands), a multiply-add counts 2 whether or not it is
contracted.  emitter/program.py takes its per-item costs from here, so the flop total of a program is the sum over the items it
actually schedules.
"""


class _Counter:
    n = 0


class S:
    """counting real scalar (no value: only the operation count matters)"""
    __slots__ = ()

    def _op(self, other=None):
        if isinstance(other, (int, float)) and abs(other) == 1:
            return self                      # literal +-1: a sign, not a flop
        _Counter.n += 1
        return self
    __add__ = __radd__ = __sub__ = __rsub__ = __mul__ = __rmul__ = __truediv__ = __rtruediv__ = _op

    def __neg__(self):
        return self


def sqrt(x):
    _Counter.n += 1
    return x


class Cx:
    __slots__ = ("re", "im")

    def __init__(self, re=None, im=None):
        self.re, self.im = re if re is not None else S(), im if im is not None else S()


def cmul(a, b):
    return Cx(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re)


def cadd(a, b):
    return Cx(a.re + b.re, a.im + b.im)


csub = cadd


def cscale(s, a):
    return Cx(s * a.re, s * a.im)


def cneg(a):
    return a


def cfma(a, b, c):                  # a += b * c: four FMAs
    a.re = a.re + b.re * c.re - b.im * c.im
    a.im = a.im + b.re * c.im + b.im * c.re
    return a


def vec():
    return [Cx() for _ in range(4)]


def mdot(a, b):
    r = cmul(a[0], b[0])
    q = cmul(cneg(a[2]), b[2])
    cfma(r, cneg(a[1]), b[1])
    cfma(q, cneg(a[3]), b[3])
    return cadd(r, q)


def rdot(k, a):
    re = k[0] * a[0].re
    im = k[0] * a[0].im
    for c in (1, 2, 3):
        re = re - k[c] * a[c].re
        im = im - k[c] * a[c].im
    return Cx(re, im)


def row_slash(a, J):                # also slash_col: the same operations on a column
    Jp, Jm = cadd(J[0], J[3]), csub(J[0], J[3])
    Jr = Cx(J[1].re - J[2].im, J[1].im + J[2].re)
    Jl = Cx(J[1].re + J[2].im, J[1].im - J[2].re)
    r = [cmul(a[2], Jp), cmul(a[2], Jl), cmul(a[0], Jm), cmul(a[1], Jp)]
    cfma(r[0], a[3], Jr)
    cfma(r[1], a[3], Jm)
    cfma(r[2], cneg(a[1]), Jr)
    cfma(r[3], cneg(a[0]), Jl)
    return r


def row_slash_real_m(r, q, m):      # also slash_real_m_col
    qp, qm = q[0] + q[3], q[0] - q[3]
    qr, ql = Cx(q[1], q[2]), Cx(q[1], -q[2])
    s = []
    for c, (qq, rr, cc, qc) in enumerate(((qp, r[2], r[3], qr), (qm, r[3], r[2], ql), (qm, r[0], r[1], qr), (qp, r[1], r[0], ql))):
        x = cscale(m, r[c])
        x.re = x.re + qq * rr.re
        x.im = x.im + qq * rr.im
        cfma(x, cc, qc)
        s.append(x)
    return s


def count(fn, *args):
    _Counter.n = 0
    fn(*args)
    return _Counter.n


# ---- the routines of the task types ------------------------------------------------------------------------------------
def _vvv_current():
    X, Y = vec(), vec()
    kA, kB = [S() for _ in range(4)], [S() for _ in range(4)]
    d = [kA[c] - kB[c] for c in range(4)]
    ka2 = [kA[c] + 2 * kB[c] for c in range(4)]
    kb2 = [2 * kA[c] + kB[c] for c in range(4)]
    f = S()
    xy, ax, by = mdot(X, Y), rdot(ka2, X), rdot(kb2, Y)
    J = []
    for c in range(4):
        v = cscale(d[c], xy)
        cfma(v, ax, Y[c])
        cfma(v, cneg(by), X[c])
        J.append(Cx(-f * v.re, -f * v.im))
    return J


def _vvvv_current():
    X, Y, Z = vec(), vec(), vec()
    f = S()
    c1, c2 = mdot(X, Z), mdot(Y, Z)
    J = []
    for c in range(4):
        v = cmul(c1, Y[c])
        cfma(v, cneg(c2), X[c])
        J.append(cscale(f, v))
    return J


def _signed_add(O, J):              # O += sign * J: the sign is not a flop
    for c in range(4):
        O[c].re = O[c].re + J[c].re
        O[c].im = O[c].im + J[c].im


def _close4(J):                     # one current against the four (t, t~) variants of W
    for _ in range(4):
        mdot(J, vec())


def _ffv():
    A, J = vec(), vec()
    q, mt, nd = [S() for _ in range(4)], S(), Cx()
    s = row_slash_real_m(row_slash(A, J), q, mt)
    return [cmul(nd, x) for x in s]


def _wcur():
    a, v = vec(), vec()
    t = [cmul(a[0], v[2]), cmul(a[1], v[3]), cmul(a[2], v[0]), cmul(a[3], v[1])]
    u = [cmul(a[0], v[3]), cmul(a[1], v[2]), cmul(a[2], v[1]), cmul(a[3], v[0])]
    cadd(cadd(t[0], t[1]), cadd(t[2], t[3]))
    csub(cadd(u[0], u[1]), cadd(u[2], u[3]))
    cadd(csub(u[1], u[0]), csub(u[2], u[3]))
    csub(csub(t[0], t[1]), csub(t[2], t[3]))


def _spin_dot(r, V):                # row . column: cmul + three cfma
    v = cmul(r[0], V[0])
    for c in (1, 2, 3):
        cfma(v, r[c], V[c])
    return v


def _amp_ffv_dots():                # per helicity assignment of the blocked legs: two rows against two columns
    r0, r1 = vec(), vec()
    for _ in range(2):
        V = vec()
        _spin_dot(r0, V)
        _spin_dot(r1, V)


def _qsum_term():
    rA = vec()
    _signed_add(rA, row_slash(vec(), vec()))


def _qsum_prop():
    s = row_slash_real_m(vec(), [S() for _ in range(4)], S())
    nd = Cx()
    return [cmul(nd, x) for x in s]


def _qsum_close():
    rA, rB = vec(), vec()
    for _ in range(2):
        R, V = vec(), vec()
        v = _spin_dot(rA, R)
        for c in range(4):
            cfma(v, rB[c], V[c])
        j = Cx()
        j.re, j.im = j.re - v.im, j.im + v.re


def _ext_eps():
    p = [S() for _ in range(4)]
    pt2 = p[1] * p[1] + p[2] * p[2]
    pp = sqrt(pt2 + p[3] * p[3])
    pt = sqrt(pt2)
    inv = 1.0 / (pp * pt)
    e1 = [p[1] * p[3] * inv, p[2] * p[3] * inv, -pt2 * inv]
    e2 = [-p[2] / pt, p[1] / pt]
    s = S()
    for x in e1:
        x * s                           # (-lam) e1 s: lam is a sign
    for x in e2:
        x * s


def _ext_spinor():
    p, m = [S() for _ in range(4)], S()
    pp = sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3])
    wp = sqrt(p[0] + pp)
    wm = m / wp
    s = (p[1] * p[1] + p[2] * p[2]) / (pp - p[3])           # the longer branch of |p| + p_z
    N = 1.0 / sqrt(2 * pp * s)
    x = [N * s, N * p[1], N * p[2]]
    for w in (wp, wm):
        for k in range(2):
            w * x[0]
            w * x[1]


def setup_flops(ng):
    """per event and tile: subset momenta, K^2 from pairwise products, top propagator denominators for all 2^ng subsets."""
    def run():
        for sub in range(1 << ng):
            gl = [g for g in range(ng) if sub >> g & 1]
            K = [S() for _ in range(4)]
            K2, D = S(), S()
            for i, g in enumerate(gl):
                for c in range(4):
                    K[c] = K[c] + S()
                for h in gl[i + 1:]:
                    kg, kh = [S() for _ in range(4)], [S() for _ in range(4)]
                    ee = kg[0] * kh[0]
                    d3 = kg[1] * kh[1] + kg[2] * kh[2] + kg[3] * kh[3]
                    cx, cy, cz = kg[2] * kh[3] - kg[3] * kh[2], kg[3] * kh[1] - kg[1] * kh[3], kg[1] * kh[2] - kg[2] * kh[1]
                    gh = (cx * cx + cy * cy + cz * cz) / (ee + d3)
                    K2 = K2 + 2 * gh
            for g in gl:
                p2, kg = [S() for _ in range(4)], [S() for _ in range(4)]
                D = D - 2 * (p2[0] * kg[0] - p2[1] * kg[1] - p2[2] * kg[2] - p2[3] * kg[3])
            for c in range(4):
                S() - K[c]
            1.0 / K2
            gw = S() * S()
            nrm = D * D + gw * gw
            D / nrm
            -gw / nrm
    return count(run)


VVV = count(_vvv_current)
VVVV = count(_vvvv_current)
VVVV_ACC = VVVV + count(_signed_add, vec(), vec())
CLOSE4 = count(_close4, vec())
FFV = count(_ffv)                               # FFVR performs the same operations on a column
WCUR = count(_wcur)
ROW_SLASH = count(row_slash, vec(), vec())
AMP_FFV_ROWS = 2 * ROW_SLASH
AMP_FFV_DOTS = count(_amp_ffv_dots)
AMP_DOT = CLOSE4
AMP_VVV = VVV + CLOSE4
AMP_VVVV = VVVV + CLOSE4
COMB_TERM = count(_signed_add, vec(), vec())
QSUM_TERM = count(_qsum_term)
QSUM_PROP = count(_qsum_prop)
QSUM_CLOSE = count(_qsum_close)
EXT_EPS = count(_ext_eps)
EXT_SPINOR = count(_ext_spinor)
ACC_PAIR = 2                                    # one complex add per (flow, column) pair
CHAN_COL = 5                                    # |A|^2 (mul + FMA) and two adds per column and lane
# the same routines as the paper's method calls them, one amplitude per call (canonical count)
CANON_AMP_FFV = ROW_SLASH + count(_spin_dot, vec(), vec())
CANON_AMP_VVV = VVV + count(mdot, vec(), vec())
CANON_AMP_VVVV = VVVV + count(mdot, vec(), vec())


def ee_flops(nhel):
    """e+ e- -> mu+ mu- kernel (csrc/mg_lib.cu mg_ee_kernel) per event with `nhel` evaluated helicity combinations."""
    def run():
        for _ in range(4):                                      # massless spinors of the four legs
            p = [S() for _ in range(4)]
            pp = sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3])
            w = sqrt(2 * pp)
            for _ in range(2):                                  # chi_+ and chi_-
                s = (p[1] * p[1] + p[2] * p[2]) / (pp - p[3])
                N = 1.0 / sqrt(2 * pp * s)
                x = [N * s, N * p[1], N * p[2]]
            for _ in range(2):
                w * x[0]; w * x[1]; w * x[1]; w * x[2]        # cscale of the two components
        k = [S() + S() for _ in range(4)]
        s = k[0] * k[0] - k[1] * k[1] - k[2] * k[2] - k[3] * k[3]
        1.0 / s
        dz, gz = s - S() * S(), S() * S()
        nz = dz * dz + gz * gz
        gz / nz; dz / nz
        for _ in range(nhel):
            for _ in range(2):                                  # chiral currents of the electron and the muon line
                a, b = vec(), vec()
                t = [cmul(a[2], b[0]), cmul(a[3], b[1]), cmul(a[2], b[1]), cmul(a[3], b[0])]
                cadd(t[0], t[1]); cadd(t[2], t[3]); csub(t[2], t[3]); csub(t[0], t[1])
                u = [cmul(a[0], b[2]), cmul(a[1], b[3]), cmul(a[0], b[3]), cmul(a[1], b[2])]
                cadd(u[0], u[1]); cadd(u[2], u[3]); csub(u[3], u[2]); csub(u[0], u[1])
            M = Cx()
            for _ in range(2):                                  # photon and Z
                gL, gR = S(), S()
                Je = [cadd(cscale(gL, Cx()), cscale(gR, Cx())) for _ in range(4)]
                Jm = [cadd(cscale(gL, Cx()), cscale(gR, Cx())) for _ in range(4)]
                M = cadd(M, cmul(Cx(), mdot(Je, Jm)))
            M.re * M.re + M.im * M.im
    return count(run)
