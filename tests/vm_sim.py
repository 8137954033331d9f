"""numpy interpreter of the emitter's task program -- TEST INFRASTRUCTURE for the host logic (emitter/scheduler).

It executes a QCDProgram phase by phase exactly as csrc/mg_vm.cuh does (same task types, operand gathering, slot
reuse, amplitude buffer and kappa accumulation) with the vertex formulas of DESIGN.md written in numpy, so that the
scheduler, index tables, colour coefficients and helicity maps can be checked against the oracle without a GPU.
It is not part of the product path and is not the oracle.
"""
import numpy as np

from paper_2507_21039_b200.emitter import diagrams as D
from paper_2507_21039_b200.emitter import program as PR


def mdot(a, b):
    return a[..., 0] * b[..., 0] - a[..., 1] * b[..., 1] - a[..., 2] * b[..., 2] - a[..., 3] * b[..., 3]


def row_slash(a, J):
    Jp, Jm = J[..., 0] + J[..., 3], J[..., 0] - J[..., 3]
    Jr, Jl = J[..., 1] + 1j * J[..., 2], J[..., 1] - 1j * J[..., 2]
    return np.stack([a[..., 2] * Jp + a[..., 3] * Jr, a[..., 2] * Jl + a[..., 3] * Jm,
                     a[..., 0] * Jm - a[..., 1] * Jr, a[..., 1] * Jp - a[..., 0] * Jl], axis=-1)


def col_slash(J, c):
    """slash(J) . column spinor (chiral representation)."""
    Jp, Jm = J[..., 0] + J[..., 3], J[..., 0] - J[..., 3]
    Jr, Jl = J[..., 1] + 1j * J[..., 2], J[..., 1] - 1j * J[..., 2]
    return np.stack([Jm * c[..., 2] - Jl * c[..., 3], -Jr * c[..., 2] + Jp * c[..., 3],
                     Jp * c[..., 0] + Jl * c[..., 1], Jr * c[..., 0] + Jm * c[..., 1]], axis=-1)


def row_slash2(a, JL, JR):
    """row . (slash(JL) P_L + slash(JR) P_R): upper result components from JL, lower ones from JR (chiral representation)."""
    rl, rr = row_slash(a, JL), row_slash(a, JR)
    return np.concatenate([rl[..., :2], rr[..., 2:]], axis=-1)


def col_slash2(JL, JR, c):
    """(slash(JL) P_L + slash(JR) P_R) . column: P_L keeps the upper column components, which feed the LOWER result components."""
    rl, rr = col_slash(JL, c), col_slash(JR, c)
    return np.concatenate([rr[..., :2], rl[..., 2:]], axis=-1)


def wcur(a, v):
    t0, t1, t2, t3 = a[..., 0] * v[..., 2], a[..., 1] * v[..., 3], a[..., 2] * v[..., 0], a[..., 3] * v[..., 1]
    u0, u1, u2, u3 = a[..., 0] * v[..., 3], a[..., 1] * v[..., 2], a[..., 2] * v[..., 1], a[..., 3] * v[..., 0]
    return 1j * np.stack([t0 + t1 + t2 + t3, u0 + u1 - u2 - u3, 1j * (u1 - u0 + u2 - u3), t0 - t1 - t2 + t3], axis=-1)


def simulate(P, p, mt, wt, outer_idx, ext):
    """p[npar][4] -> jamp[ncolor][NC] for one outer helicity assignment; ext(kind, leg, lam) gives external wavefunctions."""
    ng = P.ng
    if P.dy:
        # labels: gluons (legs 4.., outgoing) and, last, the gamma*/Z with incoming momentum -(p_e+ + p_e-); line momentum -p_u~
        k = np.array([-p[4 + g] for g in range(ng - 1)] + [-(p[2] + p[3])])
        p2 = -p[1]
    else:
        k = np.array([p[D.gluon_leg(g)] * (1 if g < 2 else -1) for g in range(ng)])
        p2 = p[2]
    nsub = 1 << ng
    K, K2, Dt = np.zeros((nsub, 4)), np.zeros(nsub), np.zeros(nsub)
    for S in range(nsub):
        gl = D.bits(S)
        for g in gl:
            K[S] += k[g]
        K2[S] = sum(2 * mdot(k[g], k[h]) for i, g in enumerate(gl) for h in gl[i + 1:]) + sum(mdot(k[g], k[g]) for g in gl if P.dy and g == ng - 1)
        Dt[S] = K2[S] - sum(2 * mdot(p2, k[g]) for g in gl)
    pos_t = len(P.inner) - 1 - P.inner.index(P.leg_row)
    pos_tb = len(P.inner) - 1 - P.inner.index(P.leg_col)

    def put_amp(staged, ob, rpc, cbase, tt_bits, vals):
        """vals[item] -> amplitude column ob + item // rpc, helicity combination cbase | t, t~ bits."""
        staged.append(("ampl", ob + np.arange(len(vals)) // rpc, cbase | tt_bits, vals))

    wf = np.full((P.nslot, 4), np.nan, complex)
    amp = np.full((P.ncol, P.NC), np.nan, complex)
    jamp = np.zeros((P.ncolor, P.NC), complex)
    chan = {}                # multichannel program: channel name -> |A|^2 per helicity lane
    for phase in P.phases:
        staged = []          # writes become visible at the end of the phase (tasks of a phase are unordered)
        for t in phase:
            ty = t["type"]
            if ty == PR.T_ACC:
                for fl, lst in zip(t["flows"], t["lists"]):
                    for col, code in lst:
                        jamp[fl] += (1j ** code) * amp[col]
                continue
            if ty == PR.T_CHAN:
                for col, name in enumerate(t["names"]):
                    chan[name] = chan.get(name, 0) + np.abs(amp[col]) ** 2        # per helicity lane
                continue
            idx, n, ib, ob = t["idx"], t["nitems"], t["in_base"], t["out_base"]
            if ty == PR.T_EXT:
                def lam_of(code):
                    return 1 if (code if code < 2 else (outer_idx >> (len(P.outer) - 1 - (code - 2))) & 1) else -1
                out = np.array([ext(int(idx[j, 2]), int(idx[j, 0]), lam_of(idx[j, 1])) if idx[j, 2] < 6 else
                                ext(int(idx[j, 2]), int(idx[j, 0]), lam_of(idx[j, 1]), lam_of(idx[j, 3])) for j in range(n)])
                staged.append(("wf", ob, out))
                continue
            if ty == PR.T_COMB:
                out = np.zeros((n, 4), complex)
                for j in range(n):
                    flags = int(idx[j, PR.COMB_MAX])
                    for q in range(flags & 7):
                        out[j] += (-1.0 if (flags >> (3 + q)) & 1 else 1.0) * wf[ib[0] + idx[j, q]]
                staged.append(("wf", ob, out))
                continue
            if ty == PR.T_QSUM:
                base = dict(zip(t["in_cols"], ib))

                def rowsum(col0, flag_col):
                    r = np.zeros((n, 4), complex)
                    fl = idx[:, flag_col]
                    for q in range(int(fl[0] & 15)):
                        A = wf[base[col0 + 2 * q] + idx[:, col0 + 2 * q]]
                        J = wf[base[col0 + 2 * q + 1] + idx[:, col0 + 2 * q + 1]]
                        sg = np.where((fl >> (4 + q)) & 1, -1.0, 1.0)
                        r += sg[:, None] * row_slash(A, J)
                    return r
                rA = rowsum(0, PR.QS_FLAGS_A)
                if not (t["aux"] & 1):
                    U = t["mA"]
                    q = p2 - K[U]
                    s = row_slash(rA, np.broadcast_to(q.astype(complex), rA.shape)) + mt * rA
                    staged.append(("wf", ob, -s / (Dt[U] + 1j * mt * wt)))
                else:
                    rB = rowsum(2 * PR.QSUM_MAX, PR.QS_FLAGS_B)
                    for tb in range(2):
                        R = wf[base[PR.QS_R1] + idx[:, PR.QS_R1] + (tb << idx[:, PR.QS_SH_TB])]
                        V = np.broadcast_to(wf[base[PR.QS_V] + tb], R.shape)
                        staged.append(("jampadd", idx[:, PR.QS_FLOW], idx[:, PR.QS_H] | (tb << pos_tb),
                                       1j * ((rA * R).sum(axis=-1) + (rB * V).sum(axis=-1))))
                continue
            X = wf[ib[0] + idx[:, 0]]
            Y = wf[ib[1] + idx[:, 1]]
            if ty == PR.T_VVVF:
                kA, kB = K[t["mA"]], K[t["mB"]]
                f = 1 / K2[t["mA"] | t["mB"]]
                xy = mdot(X, Y)
                ax = mdot(np.broadcast_to(kA + 2 * kB, X.shape), X)
                by = mdot(np.broadcast_to(2 * kA + kB, Y.shape), Y)
                Jv = -f * (xy[:, None] * (kA - kB)[None, :] + ax[:, None] * Y - by[:, None] * X)
                xs, fl = t["xslots"], t["xflags"]
                for q, Z in ((0, Y), (1, X)):                     # merged quartic structure of the first / second composite child
                    sel = ((fl >> (2 * q)) & 1) == 1
                    if sel.any():
                        Pq, Qq = wf[xs[:, 2 * q]], wf[xs[:, 2 * q + 1]]
                        sg = np.where((fl >> (2 * q + 1)) & 1, -1.0, 1.0) * sel
                        Jv = Jv + (sg * f)[:, None] * (mdot(Pq, Z)[:, None] * Qq - mdot(Qq, Z)[:, None] * Pq)
                staged.append(("wf", ob, Jv))
            elif ty in (PR.T_VVV, PR.T_AMP_VVV):
                kA, kB = K[t["mA"]], K[t["mB"]]
                f = 1 / K2[t["mA"] | t["mB"]]
                xy = mdot(X, Y)
                ax = mdot(np.broadcast_to(kA + 2 * kB, X.shape), X)
                by = mdot(np.broadcast_to(2 * kA + kB, Y.shape), Y)
                if ty == PR.T_VVV:
                    staged.append(("wf", ob, -f * (xy[:, None] * (kA - kB)[None, :] + ax[:, None] * Y - by[:, None] * X)))
                else:
                    Jv = -f * (xy[:, None] * (kA - kB)[None, :] + ax[:, None] * Y - by[:, None] * X)
                    for tt in range(4):
                        W = np.broadcast_to(wf[ib[2] + tt], Jv.shape)
                        put_amp(staged, ob, t["rpc"], idx[:, 2], ((tt >> 1) << pos_t) | ((tt & 1) << pos_tb), mdot(Jv, W))
            elif ty in (PR.T_VVVV, PR.T_AMP_VVVV):
                Z = wf[ib[2] + idx[:, 2]]
                f, s = 1 / K2[t["mA"]], t["aux"] & 3
                if s == 0:
                    c1, c2, V1, V2 = mdot(X, Z), mdot(Y, Z), Y, X
                elif s == 1:
                    c1, c2, V1, V2 = mdot(X, Y), mdot(Y, Z), Z, X
                else:
                    c1, c2, V1, V2 = mdot(X, Y), mdot(X, Z), Z, Y
                if ty == PR.T_VVVV and (t["aux"] & 4):
                    sg = np.where(idx[:, 3] & 0x8000, -1.0, 1.0)
                    staged.append(("wfadd", ob + (idx[:, 3] & 0x7fff), sg[:, None] * f * (c1[:, None] * V1 - c2[:, None] * V2)))
                elif ty == PR.T_VVVV:
                    staged.append(("wf", ob, f * (c1[:, None] * V1 - c2[:, None] * V2)))
                else:
                    Jv = f * (c1[:, None] * V1 - c2[:, None] * V2)
                    for tt in range(4):
                        W = np.broadcast_to(wf[ib[3] + tt], Jv.shape)
                        if t["aux"] & 4:      # folded top level: += into the cubic tree's column
                            sg = np.where(t["neg_of_item"] > 0, -1.0, 1.0)
                            staged.append(("ampadd", t["col_of_item"], idx[:, 3] | ((tt >> 1) << pos_t) | ((tt & 1) << pos_tb), sg * mdot(Jv, W)))
                        else:
                            put_amp(staged, ob, t["rpc"], idx[:, 3], ((tt >> 1) << pos_t) | ((tt & 1) << pos_tb), mdot(Jv, W))
            elif ty == PR.T_FFV:
                U = t["mA"]
                q = p2 - K[U]
                r = row_slash2(X, Y, wf[ib[1] + idx[:, 1] + idx[:, 2]]) if idx[0, 2] else row_slash(X, Y)
                s = row_slash(r, np.broadcast_to(q.astype(complex), r.shape)) + mt * r
                staged.append(("wf", ob, -s / (Dt[U] + 1j * mt * wt)))
            elif ty == PR.T_FFVR:
                U = t["mA"]                     # complement of the right chain's label set: q = p_t - K[U]
                q = p2 - K[U]
                r = col_slash2(Y, wf[ib[1] + idx[:, 1] + idx[:, 2]], X) if idx[0, 2] else col_slash(Y, X)
                s = col_slash(np.broadcast_to(q.astype(complex), r.shape), r) + mt * r
                staged.append(("wf", ob, -s / (Dt[U] + 1j * mt * wt)))
            elif ty == PR.T_WCUR:
                staged.append(("wf", ob, wcur(X, Y)))
            elif ty == PR.T_AMP_DOT:
                for tt in range(4):
                    W = wf[ib[0] + idx[:, 0] + ((tt >> 1) << t["mA"]) + ((tt & 1) << t["mB"])]
                    put_amp(staged, ob, t["rpc"], idx[:, 2], ((tt >> 1) << pos_t) | ((tt & 1) << pos_tb), mdot(W, Y))
            elif ty == PR.T_AMP_FFV:
                sh_tb, sh_g, sh_t, lsh_g = t["mA"] & 15, t["mA"] >> 4, t["mB"] & 15, t["mB"] >> 4
                u7 = idx[:, 4] if idx.shape[1] > 4 else np.zeros(n, dtype=np.int64)
                sh_g1, lsh_g1 = u7 & 15, (u7 >> 4) & 15
                chir = (u7 >> 8)[0]
                for tq in range(2):
                    A = wf[ib[0] + idx[:, 0] + (tq << sh_t)]
                    r = row_slash2(A, Y, wf[ib[1] + idx[:, 1] + chir]) if chir else row_slash(A, Y)
                    for hg in range(1 << (t["aux"] & 3)):
                        for tb in range(2):
                            V = wf[ib[2] + idx[:, 2] + (tb << sh_tb) + ((hg & 1) << sh_g) + ((hg >> 1) << sh_g1)]
                            comb = idx[:, 3] | ((hg & 1) << lsh_g) | ((hg >> 1) << lsh_g1)
                            put_amp(staged, ob, t["rpc"], comb, (tq << pos_t) | (tb << pos_tb), 1j * (r * V).sum(axis=-1))
        for item in staged:
            if item[0] == "ampl":
                amp[item[1], item[2]] = item[3]
            elif item[0] == "ampadd":
                assert len(set(zip(item[1].tolist(), item[2].tolist()))) == len(item[1])
                amp[item[1], item[2]] += item[3]
            elif item[0] == "jampadd":
                assert len(set(zip(item[1].tolist(), item[2].tolist()))) == len(item[1])
                jamp[item[1], item[2]] += item[3]
            elif item[0] == "wfadd":
                assert len(set(item[1].tolist())) == len(item[1])
                wf[item[1]] += item[2]
            else:
                wf[item[1]:item[1] + len(item[2])] = item[2]
    return chan if P.chan else jamp
