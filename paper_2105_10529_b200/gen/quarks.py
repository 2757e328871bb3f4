"""Build-time generator of the |M|^2 code of the LO channels with a second (light, massless) quark line and one gluon
(SURVEY 8(f)2 "q q~ -> t t~ (g), q g -> t t~ q"; "any process generated (at LO)"):

    q q~ -> t t~ g   light line  u(pa) ... vbar(pb),   gluon outgoing
    q g  -> t t~ q   light line  u(pa) ... ubar(k3),   gluon incoming

Both are one amplitude with different external lines.  With all couplings and the common phase -i g_s^3
factored out, the five diagrams (Feynman gauge, rules of reading O6.3) are

    A1 = ubar eslash (q1slash + m) jslash v / (PL^2 (q1^2 - m^2)),   q1 = PL - k2        gluon off the heavy line, top side
    A2 = ubar jslash (q2slash + m) eslash v / (PL^2 (q2^2 - m^2)),   q2 = K - k2         ... antitop side
    A3 = h . [lrow gamma^mu q3slash eslash lcol] / (P^2 q3^2),       q3 = pc + K         gluon off the light line, next to lcol
    A4 = h . [lrow eslash q4slash gamma^mu lcol] / (P^2 q4^2),       q4 = -(pr + K)      ... next to lrow
    A5 = h . V3(-P, PL, K; j, e) / (P^2 PL^2)                                            three-gluon vertex
    j^mu = lrow gamma^mu lcol,  h^mu = ubar gamma^mu v,  PL = pc + pr,  P = PL + K = k1 + k2

(pc, pr, K: all-incoming momenta of the light line's ends and of the gluon; e: real polarisation vector, linear basis).
Colour: t1 = (T^a T^b)_{34} T^b_{ji}, t2 = (T^b T^a)_{34} T^b_{ji}, t3 = T^b_{34} (T^b T^a)_{ji}, t4 = T^b_{34} (T^a T^b)_{ji};
the three-gluon vertex carries i f^{cba} T^c_{34} T^b_{ji} = t2 - t1 (checked numerically below), so
    M ~ (A1 - A5) t1 + (A2 + A5) t2 + A3 t3 + A4 t4,     |M|^2 = g_s^6 / avg  sum_hel sum_{kl} B_k C_kl conj(B_l),
C_kl = sum_colours t_k conj(t_l) by brute force from the Gell-Mann matrices (real, symmetric; numerators over 9).
"""
import itertools
import numpy as np
from .dag import Dag, Cx, csum_prod
from .amplitudes import gell_mann_T, SlashC, slash_terms, mdot, mdot_r, mdot_rr, Gen, GenEE


def colour_matrix_2q():
    """C_kl (4 x 4) of the structures t1..t4 and the check i f^{cba} T^c T^b = t2 - t1; integers over 9"""
    T = gell_mann_T()
    f = np.zeros((8, 8, 8))
    for a, b, c in itertools.product(range(8), repeat=3):
        f[a, b, c] = (-2j * np.trace((T[a] @ T[b] - T[b] @ T[a]) @ T[c])).real
    # t[k][c3, c4, j, i, a]
    ab = np.einsum("aij,bjk->abik", T, T)                      # (T^a T^b)_{ik}
    t1 = np.einsum("abmn,bji->mnjia", ab, T)
    t2 = np.einsum("bamn,bji->mnjia", ab, T)
    t3 = np.einsum("bmn,baji->mnjia", T, ab)
    t4 = np.einsum("bmn,abji->mnjia", T, ab)
    t5 = 1j * np.einsum("cba,cmn,bji->mnjia", f, T, T)
    assert np.abs(t5 - (t2 - t1)).max() < 1e-14
    ts = [t.reshape(-1) for t in (t1, t2, t3, t4)]
    C = np.array([[np.vdot(b, a) for b in ts] for a in ts])
    assert np.abs(C.imag).max() < 1e-14
    num = np.rint(C.real * 9)
    assert np.abs(num - C.real * 9).max() < 1e-9 and (num == num.T).all()
    return num.astype(int), 9


def row_slash_terms(w, s):
    """(w aslash) components as complex product lists, for a row spinor w: the transpose of slash_terms"""
    return [[(w[2], s.p), (w[3], s.t)], [(w[2], s.tb), (w[3], s.m)], [(w[0], s.m), (-w[1], s.t)], [(-w[0], s.tb), (w[1], s.p)]]


class Gen2Q:
    """kind "qq": q q~ -> t t~ g;  kind "qg": q g -> t t~ q.  Inputs are generic (no axis is special), so that the
    beam-exchanged and charge-conjugated channels are the same code on relabelled momenta."""

    def __init__(self, kind, loop_pol=False):
        """loop_pol: the gluon's polarisation (eps1 / eps2) is a run-time loop of two trips (symbol lam5 = +-1 blends the two
        vectors) instead of being unrolled: half the straight-line code, no spills"""
        assert kind in ("qq", "qg")
        self.kind, self.g = kind, Dag()
        self.loop_pol = loop_pol
        self.input_names = []
        inp = self._inp
        self.mt = inp("mt")
        self.k2 = [inp("k2" + c) for c in "exyz"]                       # antitop momentum
        self.t_ing = [inp("t_" + n) for n in ("wp", "wm", "c0", "cx", "cy")]
        self.b_ing = [inp("b_" + n) for n in ("wp", "wm", "c0", "cx", "cy")]
        self.pc = [inp("pc" + c) for c in "exyz"]                       # light line: all-incoming momenta of its two ends
        self.pr = [inp("pr" + c) for c in "exyz"]
        zero = self.g.const(0.0)                                        # massless: w- = 0 (chirality zeros become structural)
        self.c_ing = [inp("c_wp"), zero] + [inp("c_" + n) for n in ("c0", "cx", "cy")]
        self.r_ing = [inp("r_wp"), zero] + [inp("r_" + n) for n in ("c0", "cx", "cy")]
        self.K = [inp("K" + c) for c in "exyz"]                         # gluon: all-incoming momentum, two real unit polarisations
        self.e = [[inp("e%d%s" % (i, c)) for c in "xyz"] for i in (1, 2)]
        self.loop_legs = (5,) if loop_pol else ()
        self.lam5 = self.g.sym("lam5") if loop_pol else None

    def _inp(self, name):
        self.input_names.append(name)
        return self.g.inp(name)

    def _prop(self, q, m, x):
        """(qslash + m) x for a real momentum q (list of R) and a column spinor x; m an R or None"""
        g = self.g
        zero = g.const(0.0)
        qp, qm = q[0] + q[3], q[0] - q[3]
        qt, qtb = Cx(q[1], q[2]), Cx(q[1], -q[2])
        cqp, cqm = Cx(qp, zero), Cx(qm, zero)
        rows = [[(cqm, x[2]), (-qtb, x[3])], [(-qt, x[2]), (cqp, x[3])], [(cqp, x[0]), (qtb, x[1])], [(qt, x[0]), (cqm, x[1])]]
        if m is not None:
            cm = Cx(m, zero)
            for r in range(4):
                rows[r].append((cm, x[r]))
        return [csum_prod(g, rows[r]) for r in range(4)]

    def _slash(self, a, x):
        return [csum_prod(self.g, t) for t in slash_terms(SlashC(a), x)]

    def build(self):
        g = self.g
        zero = g.const(0.0)
        cvec = lambda v: [Cx(c, zero) for c in v]
        PL = [a + b for a, b in zip(self.pc, self.pr)]
        P = [a + b for a, b in zip(PL, self.K)]
        q1 = [a - b for a, b in zip(PL, self.k2)]
        q2 = [a - b for a, b in zip(self.K, self.k2)]
        q3 = [a + b for a, b in zip(self.pc, self.K)]
        q4 = [-(a + b) for a, b in zip(self.pr, self.K)]
        iPL2, iP2 = g.rcp(mdot_rr(g, PL, PL)), g.rcp(mdot_rr(g, P, P))
        d1 = g.rcp(mdot_rr(g, q1, q1) - self.mt * self.mt) * iPL2
        d2 = g.rcp(mdot_rr(g, q2, q2) - self.mt * self.mt) * iPL2
        d3 = g.rcp(mdot_rr(g, q3, q3)) * iP2
        d4 = g.rcp(mdot_rr(g, q4, q4)) * iP2
        d5 = iP2 * iPL2
        num, den = colour_matrix_2q()
        total = g.const(0.0)
        for lc, lr in itertools.product((1, -1), repeat=2):
            lcol = GenEE._u(self, self.c_ing, lc)
            lrow = GenEE._bar(GenEE._v(self, self.r_ing, lr) if self.kind == "qq" else GenEE._u(self, self.r_ing, lr))
            j = GenEE._current(self, lrow, lcol)                        # lrow gamma^mu lcol, upper index
            if all(c.re.is_zero() and c.im.is_zero() for c in j):
                continue                                                # chirality: the massless line flips no helicity
            for pol in ((None,) if self.loop_pol else (0, 1)):
                if pol is None:                                         # e = (1 + lam5)/2 e1 + (1 - lam5)/2 e2
                    s1, s2 = 0.5 * self.lam5 + 0.5, 0.5 - 0.5 * self.lam5
                    evec = [g.sop([(s1, a), (s2, b)]) for a, b in zip(self.e[0], self.e[1])]
                else:
                    evec = self.e[pol]
                e = [Cx(zero, zero)] + cvec(evec)
                es = SlashC(e)
                # light line with the gluon attached
                b3 = GenEE._current(self, lrow, self._prop(q3, None, self._slash(e, lcol)))
                w4 = [csum_prod(g, t) for t in row_slash_terms(lrow, es)]               # lrow eslash
                w4 = [csum_prod(g, t) for t in row_slash_terms(w4, SlashC(cvec(q4)))]   # ... q4slash
                b4 = GenEE._current(self, w4, lcol)
                # three-gluon vertex: V3(-P, PL, K; j, e) = j ((-P - PL).e) + (PL - K) (j.e) + e ((K + P).j)
                c1 = mdot_rr(g, [-(a + b) for a, b in zip(P, PL)], [zero] + list(evec))
                c2 = mdot(g, j, e)
                c3 = mdot_r(g, [a + b for a, b in zip(self.K, P)], j)
                dPK = [a - b for a, b in zip(PL, self.K)]
                v3 = [j[m] * c1 + Cx(dPK[m] * c2.re, dPK[m] * c2.im) + e[m] * c3 for m in range(4)]
                for l4 in (1, -1):
                    v = GenEE._v(self, self.b_ing, l4)
                    x1 = self._prop(q1, self.mt, self._slash(j, v))                     # (q1slash + m) jslash v
                    x1 = self._slash(e, x1)
                    x2 = self._slash(j, self._prop(q2, self.mt, self._slash(e, v)))     # jslash (q2slash + m) eslash v
                    for l3 in (1, -1):
                        ub = GenEE._bar(GenEE._u(self, self.t_ing, l3))
                        h = GenEE._current(self, ub, v)
                        A1 = csum_prod(g, [(ub[r], x1[r]) for r in range(4)]) * d1
                        A2 = csum_prod(g, [(ub[r], x2[r]) for r in range(4)]) * d2
                        A3 = mdot(g, h, b3) * d3
                        A4 = mdot(g, h, b4) * d4
                        A5 = mdot(g, h, v3) * d5
                        B = [A1 - A5, A2 + A5, A3, A4]
                        for part in ("re", "im"):
                            x = [getattr(b, part) for b in B]
                            pairs = []
                            for s in range(4):
                                y = g.sop([(g.const(2.0 * num[s][t]), x[t]) for t in range(s + 1, 4)], g.const(float(num[s][s])) * x[s])
                                pairs.append((x[s], y))
                            total = g.sop(pairs, total)
        self.out = total
        # |M|^2 = g_s^6 * scale * out: colour denominator, average over the incoming pair's helicities and colours
        self.scale = 1.0 / den / (36.0 if self.kind == "qq" else 96.0)
        self.loop_assign = [(-1.0,), (1.0,)] if self.loop_pol else [()]
        return total


# the gluon polarisation as a run-time loop: stack 1424 -> 944 B per thread, q q~ -> t t~ g 0.99 -> 0.94 ms per 1e6 events on the B200
# (q g -> t t~ q unchanged: 1.60 ms; profiles/r2_tuning.md)
PROCESSES_2Q = {"mf_me2_qq_ttg": lambda: Gen2Q("qq", loop_pol=True), "mf_me2_qg_ttq": lambda: Gen2Q("qg", loop_pol=True)}
