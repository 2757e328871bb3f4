"""Build-time generator of the per-process |M|^2 device code (PAPER.md:47 wavefunctions, vertices,
propagators; "loops over initial and final state particle helicities and aggregates"
the squared amplitude; PAPER.md:69 the algebraic routines are "elementary algebraic operations").

Organisation: colour-ordered Berends-Giele recursion, i.e. the sum of all
tree diagrams of DESIGN.md reading O6.5 regrouped by colour word T^{a_s(1)}...T^{a_s(n)}:

  gluon currents   j(pi) = (1/P^2) { - sum_{pi=L|R} v3(L,R) - sum_{pi=X|Y|Z} q4(X,Y,Z) },  j(g) = e_g
      v3(L,R)^mu  = V3^{mu nu rho}(-P,P_L,P_R) j_L,nu j_R,rho
                  = -j_L^mu ((2P_L+P_R).j_R) + (P_L-P_R)^mu (j_L.j_R) + j_R^mu ((2P_R+P_L).j_L)
      q4(X,Y,Z)   = X (Y.Z) + Z (X.Y) - 2 Y (X.Z)
  quark line       chi(()) = v(p4,l4);  chi(tau) = -S(q_tau) sum_{tau=b|tau'} jslash(b) chi(tau'),
                   S(q) = (qslash+m)/(q^2-m^2),  q_tau = P_tau - p4
  partial amps     a_s = -ubar(p3,l3) sum_{s=b|tau'} jslash(b) chi(tau')
  |M|^2            = g_s^{2n}/256 sum_hel sum_{s,s'} a_s C_{ss'} a*_{s'}   (overall phase -i dropped)

with all g_s factored out (real coefficients everywhere).  Obtained from the Feynman rules of O6.3
by expanding every tree's colour word (-i[T_A,T_B], -[T_A,[T_B,T_C]], ...) into ordered words; the
derivation is written out in DESIGN.md.  The parity relation |M(-lambda)|^2 = |M(lambda)|^2
(colour-summed) halves the helicity sum (reading O6.7 allows it on the GPU side only).
"""
import itertools
import math
import numpy as np
from .dag import Dag, R, Cx, csum_prod

SQ2I = 1.0 / math.sqrt(2.0)
METRIC = (1.0, -1.0, -1.0, -1.0)


# ---- SU(3) colour matrix (own brute force; integers over a common denominator) -----------------
def gell_mann_T():
    T = np.zeros((8, 3, 3), complex)
    T[0][0, 1] = T[0][1, 0] = 0.5
    T[1][0, 1], T[1][1, 0] = -0.5j, 0.5j
    T[2][0, 0], T[2][1, 1] = 0.5, -0.5
    T[3][0, 2] = T[3][2, 0] = 0.5
    T[4][0, 2], T[4][2, 0] = -0.5j, 0.5j
    T[5][1, 2] = T[5][2, 1] = 0.5
    T[6][1, 2], T[6][2, 1] = -0.5j, 0.5j
    T[7] = np.diag([1.0, 1.0, -2.0]) / (2.0 * math.sqrt(3.0))
    return T


def colour_matrix(ng):
    """C_{ss'} = sum_{a} Tr(T^{a_s(1)}..T^{a_s(n)} (T^{a_s'(1)}..T^{a_s'(n)})^dagger); perms in
    lexicographic order.  Returns (integer numerators, denominator)."""
    T = gell_mann_T()
    perms = list(itertools.permutations(range(ng)))
    letters = "abcd"[:ng]
    words = []
    for p in perms:
        # W[a_0..a_{n-1}, i, j] = (T^{a_p0} T^{a_p1} ...)_{ij}
        W = T[:, :, :]
        sub = letters[p[0]] + "ij"
        for k in range(1, ng):
            W = np.einsum(sub + "," + letters[p[k]] + "jk->" + "".join(sorted(sub[:-2] + letters[p[k]])) + "ik", W, T)
            sub = "".join(sorted(sub[:-2] + letters[p[k]])) + "ij"
        words.append(W.reshape(-1))
    Wm = np.array(words)
    Cm = (Wm @ Wm.conj().T).real
    den = {2: 3, 3: 9, 4: 54}[ng]
    num = np.rint(Cm * den)
    assert np.abs(num - Cm * den).max() < 1e-9
    return num.astype(int), den, perms


# ---- vectors and spinors over the DAG ------------------------------------------------------------
def mdot(g, a, b):
    """Minkowski product of two complex 4-vectors."""
    return csum_prod(g, [(a[m] if METRIC[m] > 0 else -a[m], b[m]) for m in range(4)])


def mdot_r(g, p, b):
    """Minkowski product of a real 4-vector p (list of R) with a complex one."""
    return Cx(g.sop([(p[m] if METRIC[m] > 0 else -p[m], b[m].re) for m in range(4)]),
              g.sop([(p[m] if METRIC[m] > 0 else -p[m], b[m].im) for m in range(4)]))


def mdot_rr(g, p, q):
    return g.sop([(p[m] if METRIC[m] > 0 else -p[m], q[m]) for m in range(4)])


class SlashC:
    """light-cone pieces of a complex 4-vector a for aslash psi (chiral representation, O6.1)"""

    def __init__(self, a):
        self.p = a[0] + a[3]
        self.m = a[0] - a[3]
        self.t = Cx(a[1].re - a[2].im, a[1].im + a[2].re)     # a1 + i a2
        self.tb = Cx(a[1].re + a[2].im, a[1].im - a[2].re)    # a1 - i a2


def slash_terms(s, psi):
    """rows of (aslash psi) as lists of complex products (so that several can share one FMA chain):
    r0 = am psi2 - atb psi3; r1 = -at psi2 + ap psi3; r2 = ap psi0 + atb psi1; r3 = at psi0 + am psi1"""
    return [[(s.m, psi[2]), (-s.tb, psi[3])], [(-s.t, psi[2]), (s.p, psi[3])],
            [(s.p, psi[0]), (s.tb, psi[1])], [(s.t, psi[0]), (s.m, psi[1])]]


class Gen:
    """gg -> t tbar + (ng-2) g.  Gluon legs 0,1 incoming along +z/-z, legs 2.. outgoing."""

    def __init__(self, ng, loop_legs=(), parity=True, loop_lam4=False, basis="circular"):
        """loop_legs: gluon legs whose helicity is a run-time loop symbol; loop_lam4: the antitop
        helicity is a loop symbol too (leg id 4 in the loop list; v(lam4) is blended arithmetically).
        basis: "circular" = helicity states eps(k, +-1) of O6.2; "linear" = the two REAL polarisation
        vectors eps1, eps2 of O6.2 (label +1 -> eps1, -1 -> eps2).  The spin sum over a gluon is the
        same in any orthonormal basis of its two physical polarisations (sum_lam eps_lam^mu
        eps_lam^nu* = eps1^mu eps1^nu + eps2^mu eps2^nu), and with real vectors every gluon current
        is real: the DAG drops the imaginary parts as structural zeros."""
        self.basis = basis
        self.loop_lam4 = loop_lam4
        self.ng, self.g = ng, Dag()
        g = self.g
        self.loop_legs = tuple(loop_legs)
        self.parity = parity
        self.input_names = []
        inp = self._inp
        E = inp("E")
        zero = g.const(0.0)
        self.mt = inp("mt")
        self.p3 = [inp("p3e"), inp("p3x"), inp("p3y"), inp("p3z")]
        self.p4 = [inp("p4e"), inp("p4x"), inp("p4y"), inp("p4z")]
        self.t_ing = [inp("t_" + n) for n in ("wp", "wm", "c0", "cx", "cy")]
        self.b_ing = [inp("b_" + n) for n in ("wp", "wm", "c0", "cx", "cy")]
        # all-incoming gluon momenta K_g
        self.K = [[E, zero, zero, E], [E, zero, zero, -E]]
        self.g_ing = [None, None]
        for l in range(2, ng):
            k = [inp("k%d%s" % (l, c)) for c in "exyz"]
            self.K.append([-c for c in k])
            self.g_ing.append([inp("g%d_%s" % (l, n)) for n in ("e1x", "e1y", "e1z", "e2x", "e2y")])
        self.lam_sym = {l: g.sym("lam%d" % l) for l in self.loop_legs}
        self.lam4_sym = g.sym("lam9") if loop_lam4 else None
        self._P, self._j, self._sl, self._chi = {}, {}, {}, {}

    def _inp(self, name):
        self.input_names.append(name)
        return self.g.inp(name)

    # ---- external wavefunctions (O6.2) ----------------------------------------------------------
    def pol(self, leg, lam):
        """e_g: eps(k,lam) for incoming legs, eps^*(k,lam) for outgoing; lam is +-1 or a symbol R"""
        g = self.g
        z = Cx(g.const(0.0), g.const(0.0))
        if self.basis == "linear":
            return self.pol_linear(leg, lam)
        lamR = lam if isinstance(lam, R) else g.const(float(lam))
        if leg == 0:      # k along +z: eps = (0, -lam/sqrt2, -i/sqrt2, 0)
            return [z, Cx(-lamR * SQ2I, g.const(0.0)), Cx(g.const(0.0), g.const(-SQ2I)), z]
        if leg == 1:      # k along -z: eps = (0, -lam/sqrt2, +i/sqrt2, 0)
            return [z, Cx(-lamR * SQ2I, g.const(0.0)), Cx(g.const(0.0), g.const(SQ2I)), z]
        e1x, e1y, e1z, e2x, e2y = self.g_ing[leg]      # already divided by sqrt 2
        return [z, Cx(-lamR * e1x, e2x), Cx(-lamR * e1y, e2y), Cx(-lamR * e1z, g.const(0.0))]

    def pol_linear(self, leg, lam):
        """real polarisation vectors: label +1 -> eps1, -1 -> eps2 (O6.2: eps1 = (0, kx kz, ky kz, -kT^2)/(|k| kT),
        eps2 = (0, -ky, kx, 0)/kT; kT = 0: eps1 = x, eps2 = sgn(kz) y).  Incoming legs: unit vectors;
        outgoing legs: the ingredients are eps_i/sqrt2 (the factor 2 per outgoing gluon goes into
        `scale`).  A loop symbol lam = +-1 selects by blending: s1 = (1+lam)/2, s2 = (1-lam)/2."""
        g = self.g
        zero = g.const(0.0)
        z = Cx(zero, zero)
        re = lambda x: Cx(x, zero)
        if isinstance(lam, R):
            s1, s2 = 0.5 * lam + 0.5, 0.5 - 0.5 * lam
        else:
            s1, s2 = g.const(1.0 if lam > 0 else 0.0), g.const(0.0 if lam > 0 else 1.0)
        if leg in (0, 1):
            sg = 1.0 if leg == 0 else -1.0
            return [z, re(s1), re(s2 * sg), z]
        e1x, e1y, e1z, e2x, e2y = self.g_ing[leg]
        return [z, re(g.sop([(s1, e1x), (s2, e2x)])), re(g.sop([(s1, e1y), (s2, e2y)])), re(s1 * e1z)]

    @staticmethod
    def _chi_pm(ing):
        wp, wm, c0, cx, cy = ing
        g = wp.g
        zero = g.const(0.0)
        chi_p = [Cx(c0, zero), Cx(cx, cy)]
        chi_m = [Cx(-cx, cy), Cx(c0, zero)]
        return wp, wm, chi_p, chi_m

    def ubar3(self, lam):
        wp, wm, cp, cm = self._chi_pm(self.t_ing)
        if lam > 0:      # u = (w- chi+ ; w+ chi+)
            u = [cp[0] * wm, cp[1] * wm, cp[0] * wp, cp[1] * wp]
        else:            # u = (w+ chi- ; w- chi-)
            u = [cm[0] * wp, cm[1] * wp, cm[0] * wm, cm[1] * wm]
        return [u[2].conj(), u[3].conj(), u[0].conj(), u[1].conj()]      # u^dagger gamma^0

    def v4(self, lam):
        if isinstance(lam, R):       # symbolic: v = (1+lam)/2 v(+) + (1-lam)/2 v(-)
            vp, vm = self.v4(1), self.v4(-1)
            sp, sm = 0.5 * lam + 0.5, 0.5 - 0.5 * lam
            return [Cx(self.g.sop([(sp, a.re), (sm, b.re)]), self.g.sop([(sp, a.im), (sm, b.im)])) for a, b in zip(vp, vm)]
        wp, wm, cp, cm = self._chi_pm(self.b_ing)
        if lam > 0:      # v(+) = (-w+ chi- ; w- chi-)
            return [-(cm[0] * wp), -(cm[1] * wp), cm[0] * wm, cm[1] * wm]
        return [cp[0] * wm, cp[1] * wm, -(cp[0] * wp), -(cp[1] * wp)]   # v(-) = (w- chi+ ; -w+ chi+)

    # ---- gluon currents ---------------------------------------------------------------------------
    def P(self, legs):
        key = tuple(sorted(legs))
        if key not in self._P:
            v = [self.g.const(0.0)] * 4
            for l in key:
                v = [a + b for a, b in zip(v, self.K[l])]
            self._P[key] = v
        return self._P[key]

    def _hk(self, legs, hel):
        """memo key of the helicity labels of `legs` (symbols by identity)"""
        return tuple(id(hel[l]) if isinstance(hel[l], R) else hel[l] for l in legs)

    def j(self, pi, hel):
        """ordered current j(pi) for helicities hel (dict leg -> +-1 or symbol); memoised with the
        reflection identity j(reversed pi) = (-1)^(k-1) j(pi)"""
        pi = tuple(pi)
        rev = tuple(reversed(pi))
        if rev < pi:
            cur = self.j(rev, hel)
            return cur if len(pi) % 2 == 1 else [-c for c in cur]
        key = (pi, self._hk(pi, hel))
        if key not in self._j:
            self._j[key] = self.pol(pi[0], hel[pi[0]]) if len(pi) == 1 else self._bg(pi, hel)
        return self._j[key]

    def _bg(self, pi, hel):
        """one step of the Berends-Giele recursion: j(pi), len(pi) >= 2, from the currents of its splits"""
        g = self.g
        k = len(pi)
        terms = [[] for _ in range(4)]        # complex product lists per component
        rterms = [[] for _ in range(4)]       # (real, complex) products per component
        for s in range(1, k):                 # cubic: split L | R
            L, Rr = pi[:s], pi[s:]
            PL, PR = self.P(L), self.P(Rr)
            jL, jR = self.j(L, hel), self.j(Rr, hel)
            c1 = mdot_r(g, [2.0 * a + b for a, b in zip(PL, PR)], jR)
            c2 = mdot(g, jL, jR)
            c3 = mdot_r(g, [2.0 * b + a for a, b in zip(PL, PR)], jL)
            d = [a - b for a, b in zip(PL, PR)]
            for m in range(4):                # accumulate  -v3 = +jL c1 - d c2 - jR c3
                terms[m] += [(jL[m], c1), (-jR[m], c3)]
                rterms[m] += [(-d[m], c2)]
        for s1 in range(1, k - 1):            # quartic: X | Y | Z
            for s2 in range(s1 + 1, k):
                X, Y, Z = self.j(pi[:s1], hel), self.j(pi[s1:s2], hel), self.j(pi[s2:], hel)
                yz, xy, xz = mdot(g, Y, Z), mdot(g, X, Y), mdot(g, X, Z)
                for m in range(4):            # accumulate -q4 = -X yz - Z xy + 2 Y xz
                    terms[m] += [(-X[m], yz), (-Z[m], xy), (2.0 * Y[m], xz)]
        Pv = self.P(pi)
        inv = g.rcp(mdot_rr(g, Pv, Pv))
        cur = []
        for m in range(4):
            acc = csum_prod(g, terms[m])
            re = g.sop([(a, c.re) for a, c in rterms[m]], acc.re)
            im = g.sop([(a, c.im) for a, c in rterms[m]], acc.im)
            cur.append(Cx(re * inv, im * inv))
        return cur

    def jsl(self, pi, hel):
        pi = tuple(pi)
        key = (pi, self._hk(pi, hel))
        if key not in self._sl:
            self._sl[key] = SlashC(self.j(pi, hel))
        return self._sl[key]

    # ---- quark line ---------------------------------------------------------------------------------
    def attach(self, seq, hel, lam4):
        """sum over splits seq = b | tail of jslash(b) chi(tail): 4 complex rows"""
        g = self.g
        rows = [[] for _ in range(4)]
        for s in range(1, len(seq) + 1):
            b, tail = seq[:s], seq[s:]
            t = slash_terms(self.jsl(b, hel), self.chi(tail, hel, lam4))
            for r in range(4):
                rows[r] += t[r]
        return [csum_prod(g, rows[r]) for r in range(4)]

    def chi(self, tau, hel, lam4):
        tau = tuple(tau)
        key = (tau, self._hk(tau, hel), id(lam4) if isinstance(lam4, R) else lam4)
        if key in self._chi:
            return self._chi[key]
        g = self.g
        if len(tau) == 0:
            out = self.v4(lam4)
        else:
            xi = self.attach(tau, hel, lam4)
            q = [a - b for a, b in zip(self.P(tau), self.p4)]
            den = mdot_rr(g, q, q) - self.mt * self.mt
            ninv = -g.rcp(den)
            qp, qm = q[0] + q[3], q[0] - q[3]
            zero = g.const(0.0)
            qt, qtb = Cx(q[1], q[2]), Cx(q[1], -q[2])
            cqp, cqm, cm = Cx(qp, zero), Cx(qm, zero), Cx(self.mt, zero)
            rows = [[(cqm, xi[2]), (-qtb, xi[3]), (cm, xi[0])], [(-qt, xi[2]), (cqp, xi[3]), (cm, xi[1])],
                    [(cqp, xi[0]), (qtb, xi[1]), (cm, xi[2])], [(qt, xi[0]), (cqm, xi[1]), (cm, xi[3])]]
            out = [csum_prod(g, rows[r]) * ninv for r in range(4)]
        self._chi[key] = out
        return out

    def partial_amps(self, sigma, hel, lam4):
        """a_sigma for lam3 = +1 and -1 (shared closing spinor)"""
        xi = self.attach(tuple(sigma), hel, lam4)
        out = {}
        for lam3 in (1, -1):
            ub = self.ubar3(lam3)
            out[lam3] = -csum_prod(self.g, [(ub[r], xi[r]) for r in range(4)])
        return out

    # ---- helicity and colour sums ----------------------------------------------------------------
    def colour_form(self, amps, num):
        """sum_{s,s'} C_{ss'} (Re a_s Re a_s' + Im a_s Im a_s') with integer numerators (symmetric)"""
        g = self.g
        total = g.const(0.0)
        n = len(amps)
        for part in ("re", "im"):
            x = [getattr(a, part) for a in amps]
            pairs = []
            for s in range(n):
                y = g.sop([(g.const(2.0 * num[s][t]), x[t]) for t in range(s + 1, n)],
                          g.const(float(num[s][s])) * x[s])
                pairs.append((x[s], y))
            total = g.sop(pairs, total)
        return total

    def build(self):
        """returns (body output R, list of loop symbol assignments, scale) where
        |M|^2_avg = g_s^{2 ng}/256 * scale * sum_{loop assignments} body"""
        ng = self.ng
        num, den, perms = colour_matrix(ng)
        # parity: circular basis |M(-lam)|^2 = |M(lam)|^2 (colour-summed) fixes the helicity of gluon 0;
        # linear basis: real polarisation vectors are their own conjugates, so flipping the two quark
        # helicities conjugates every partial amplitude: the antitop helicity is fixed instead
        linear = self.basis == "linear"
        fix0 = self.parity and not linear
        free = [l for l in range(ng) if l not in self.loop_legs and not (fix0 and l == 0)]
        lam4s = (self.lam4_sym,) if self.loop_lam4 else ((1,) if (self.parity and linear) else (1, -1))
        total = self.g.const(0.0)
        for combo in itertools.product((1, -1), repeat=len(free)):
            hel = dict(self.lam_sym)
            if fix0:
                hel[0] = 1
            hel.update(dict(zip(free, combo)))
            for lam4 in lam4s:
                amps = {1: [], -1: []}
                for sg in perms:
                    a = self.partial_amps(sg, hel, lam4)
                    amps[1].append(a[1])
                    amps[-1].append(a[-1])
                for lam3 in (1, -1):
                    total = total + self.colour_form(amps[lam3], num)
        self.out = total
        self.scale = (2.0 if self.parity else 1.0) / den * (2.0 ** (ng - 2) if linear else 1.0)
        if self.loop_lam4:
            self.loop_legs = self.loop_legs + (9,)          # symbol lam9 = antitop helicity
        self.loop_assign = list(itertools.product((-1.0, 1.0), repeat=len(self.loop_legs)))
        return total


class GenEE:
    """e+ e- -> gamma* -> mu+ mu- (O6.4): M = e^2 [vbar(pb) gamma^mu u(pa)][ubar(p1) gamma_mu v(p2)]/s"""

    def __init__(self):
        self.g = Dag()
        self.input_names = []
        names = ("wp", "wm", "c0", "cx", "cy")
        self.ing = {p: [self._inp("%s_%s" % (p, n)) for n in names] for p in ("a", "b", "m", "n")}
        self.loop_legs = ()

    def _inp(self, name):
        self.input_names.append(name)
        return self.g.inp(name)

    def _u(self, ing, lam):
        wp, wm, cp, cm = Gen._chi_pm(ing)
        if lam > 0:
            return [cp[0] * wm, cp[1] * wm, cp[0] * wp, cp[1] * wp]
        return [cm[0] * wp, cm[1] * wp, cm[0] * wm, cm[1] * wm]

    def _v(self, ing, lam):
        wp, wm, cp, cm = Gen._chi_pm(ing)
        if lam > 0:
            return [-(cm[0] * wp), -(cm[1] * wp), cm[0] * wm, cm[1] * wm]
        return [cp[0] * wm, cp[1] * wm, -(cp[0] * wp), -(cp[1] * wp)]

    @staticmethod
    def _bar(u):
        return [u[2].conj(), u[3].conj(), u[0].conj(), u[1].conj()]

    def _current(self, row, col):
        """w gamma^mu psi, mu = 0..3 (upper index): gamma^mu = g_mumu * slash(unit vector mu)"""
        g = self.g
        zero, one = g.const(0.0), g.const(1.0)
        out = []
        for mu in range(4):
            a = [Cx(one if m == mu else zero, zero) for m in range(4)]
            t = slash_terms(SlashC(a), col)
            v = csum_prod(g, [(row[r], csum_prod(g, t[r])) for r in range(4)])
            out.append(v * METRIC[mu])
        return out

    def build(self):
        """body = sum_hel |L.R|^2 ; |M|^2_avg = e^4/s^2 * scale * body, scale = 1/4"""
        g = self.g
        total = g.const(0.0)
        for la, lb, l1, l2 in itertools.product((1, -1), repeat=4):
            L = self._current(self._bar(self._v(self.ing["b"], lb)), self._u(self.ing["a"], la))
            Rc = self._current(self._bar(self._u(self.ing["m"], l1)), self._v(self.ing["n"], l2))
            M = mdot(g, L, Rc)
            total = g.sop([(M.re, M.re), (M.im, M.im)], total)
        self.out, self.scale, self.loop_assign = total, 0.25, [()]
        return total


# ---- emission ---------------------------------------------------------------------------------------
def emit_function(gen, fname):
    """CUDA/C++ text of `template <typename T> T fname(const T* in)` (T = double, or float for the fp32
    variant of the |M|^2 stage) plus the flop-count macros."""
    g, out = gen.g, gen.out
    sync = SYNC_MACRO.get(fname, "MF_SYNC_POINT")
    nh = len(gen.loop_assign)
    looped = bool(gen.loop_legs)
    pro_ids, body_ids, hoisted = g.plan([out], getattr(gen, "max_hoist_cost", None) if looped else None)
    pro, body = g.count_list(pro_ids), g.count_list(body_ids)
    if not looped:
        tot = {k: pro[k] + body[k] for k in pro}
    else:
        tot = {k: pro[k] + nh * (body[k] + (1 if k == "add" else 0)) for k in pro}
    emitted = dict(tot)
    if looped:      # ALGORITHMIC count = every loop invariant computed once (recomputation is not counted)
        p0, b0, _h = g.plan([out], None)
        c0, c1 = g.count_list(p0), g.count_list(b0)
        tot = {k: c0[k] + nh * (c1[k] + (1 if k == "add" else 0)) for k in c0}
    U = fname.upper()
    L = ["// GENERATED by paper_2105_10529_b200/gen/amplitudes.py -- do not edit.",
         "// per event (algorithmic): %d add, %d mul, %d fma, %d rcp  (flops = add + mul + 2 fma = %d)"
         % (tot["add"], tot["mul"], tot["fma"], tot["rcp"], tot["add"] + tot["mul"] + 2 * tot["fma"]),
         "// emitted (cheap loop invariants recomputed per helicity-loop trip): %d add, %d mul, %d fma"
         % (emitted["add"], emitted["mul"], emitted["fma"]),
         "#define %s_NADD %dull" % (U, tot["add"]), "#define %s_NMUL %dull" % (U, tot["mul"]),
         "#define %s_NFMA %dull" % (U, tot["fma"]), "#define %s_NIN %d" % (U, len(gen.input_names)),
         "#define %s_SCALE %r" % (U, gen.scale)]
    L.append("enum { " + ", ".join("%s_IN_%s = %d" % (U, n.upper(), i) for i, n in enumerate(gen.input_names)) + " };")
    L.append("template <typename T>")
    L.append("MF_DEVFN T %s(const T* __restrict__ in) {" % fname)
    for i, n in enumerate(gen.input_names):
        L.append("  const T %s = in[%d];" % (n, i))
    leaf = lambda j: g.nodes[j][0] in ("in", "sym")
    pname = lambda j: g.names[j] if leaf(j) else "p%d" % j
    if not looped:
        ids = sorted(set(pro_ids) | set(body_ids))
        for i, line in enumerate(g.emit_list(ids, pname, "p")):
            if i % 64 == 0 and len(ids) > 1024:
                L.append("  %s(%d);" % (sync, i // 64))
            L.append(line)
        L.append("  return %s;" % _ref(g, out, pname))
    else:
        L += g.emit_list(pro_ids, pname, "p")
        L.append("  T acc = T(0.0);")
        L.append("#pragma unroll 1")
        L.append("  for (int ih = 0; ih < %d; ++ih) {" % nh)
        for b, l in enumerate(reversed(gen.loop_legs)):
            L.append("    const T lam%d = (ih & %d) ? T(1.0) : T(-1.0);" % (l, 1 << b))
        launder = getattr(gen, "max_hoist_cost", None) is not None
        used_inputs = sorted({o for i in body_ids for o in g._operands(i) if g.nodes[o][0] == "in"})
        if launder:       # opaque copies: keeps NVVM from hoisting the cheap invariants out again
            for j in used_inputs:
                L.append("    T %s_l = %s; MF_LAUNDER(%s_l);" % (g.names[j], g.names[j], g.names[j]))

        def bname(j):
            if g.nodes[j][0] == "in":
                return g.names[j] + ("_l" if launder else "")
            if g.nodes[j][0] == "sym":
                return g.names[j]
            return "p%d" % j if (j in hoisted and not g.dep[j] and j not in body_set) else "v%d" % j

        body_set = set(body_ids)
        body_ids = g.schedule(body_ids, SCHED_WINDOW, SCHED_DISTANCE)
        body_lines = g.emit_list(body_ids, bname, "v", indent="    ")
        for i, line in enumerate(body_lines):      # barrier points: keep the block's warps on the same I-cache lines
            if i % 64 == 0:
                L.append("    %s(%d);" % (sync, i // 64))
            L.append(line)
        L.append("    acc += %s;" % _ref(g, out, bname))
        L.append("  }")
        L.append("  return acc;")
    L.append("}")
    return "\n".join(L) + "\n", tot


def emit_function_smem(gen, fname, clobber_every=256, max_hoist_cost=2, rcp_leaf=False):
    """The same helicity-loop function with its loop-entering values in SHARED MEMORY instead of registers:
        template <typename T, int S> T fname_s(T* W)
    W: the thread's column of a [slot][S] tile (S = threads of the CTA: conflict-free): slots 0..NIN-1 hold the inputs, the
    following NV slots receive the hoisted loop invariants.  The body re-reads them where they are used; a compiler barrier
    every `clobber_every` statements keeps the loads from being hoisted to the loop head (where they would be spilled again)
    while letting the compiler share a loaded value inside a stretch.  With ~50 doubles out of the register file the body
    has the register file to itself: no spills at 255 registers (672 B before), |M|^2 stage of gg -> tt~g 5.64 -> 5.40 ms per
    1e7 events (profiles/r2_tuning.md; 384 threads at 168 registers still spill 1.2 KB and take 8.0 ms)."""
    g, out = gen.g, gen.out
    nh = len(gen.loop_assign)
    pro_ids, body_ids, hoisted = g.plan([out], max_hoist_cost, rcp_leaf)     # parking costs shared memory, not registers: hoist more
    body_set = set(body_ids)
    leaf = lambda j: g.nodes[j][0] in ("in", "sym")
    parked = sorted({o for i in body_ids for o in g._operands(i) if o not in body_set and not leaf(o)})
    nin = len(gen.input_names)
    slot = {j: nin + n for n, j in enumerate(parked)}
    idx = {n: i for i, n in enumerate(gen.input_names)}
    U = fname.upper()
    p0, b0, _h = g.plan([out], None)              # ALGORITHMIC count of this organisation: every loop invariant computed once
    c0, c1 = g.count_list(p0), g.count_list(b0)
    alg = {k: c0[k] + nh * (c1[k] + (1 if k == "add" else 0)) for k in c0}
    cp, cb = g.count_list(pro_ids), g.count_list(body_ids)
    emitted = {k: cp[k] + nh * (cb[k] + (1 if k == "add" else 0)) for k in cp}
    L = ["// %s_s: helicity loop over gluon legs %s (%d trips); algorithmic %d add, %d mul, %d fma (flops = %d); emitted with recomputed invariants: flops = %d"
         % (fname, gen.loop_legs, nh, alg["add"], alg["mul"], alg["fma"], alg["add"] + alg["mul"] + 2 * alg["fma"],
            emitted["add"] + emitted["mul"] + 2 * emitted["fma"]),
         "#define %s_S_NADD %dull" % (U, alg["add"]), "#define %s_S_NMUL %dull" % (U, alg["mul"]), "#define %s_S_NFMA %dull" % (U, alg["fma"]),
         "#define %s_S_NFLOPS_EMITTED %dull" % (U, emitted["add"] + emitted["mul"] + 2 * emitted["fma"]),
         "#define %s_S_SCALE %r" % (U, gen.scale),
         "#define %s_NW %d      // slots of the shared-memory tile of %s_s: inputs, then parked invariants" % (U, nin + len(parked), fname),
         "#if defined(__CUDACC__)",
         "template <typename T, int S>",
         "__device__ __forceinline__ T %s_s(T* W) {" % fname,
         "  {"]
    used_pro = sorted({o for i in pro_ids for o in g._operands(i) if g.nodes[o][0] == "in"})
    for j in used_pro:
        L.append("    const T %s = W[%d * S];" % (g.names[j], idx[g.names[j]]))
    pname = lambda j: g.names[j] if leaf(j) else "p%d" % j
    L += g.emit_list(pro_ids, pname, "p", indent="    ")
    for j in parked:
        L.append("    W[%d * S] = p%d;" % (slot[j], j))
    L += ["  }", "  T acc = T(0.0);", "#pragma unroll 1", "  for (int ih = 0; ih < %d; ++ih) {" % nh]
    for b, l in enumerate(reversed(gen.loop_legs)):
        L.append("    const T lam%d = (ih & %d) ? T(1.0) : T(-1.0);" % (l, 1 << b))

    def bname(j):
        if g.nodes[j][0] == "in":
            return "W[%d * S]" % idx[g.names[j]]
        if g.nodes[j][0] == "sym":
            return g.names[j]
        return "v%d" % j if j in body_set else "W[%d * S]" % slot[j]

    body_ids = g.schedule(body_ids, SCHED_WINDOW, SCHED_DISTANCE)
    for i, line in enumerate(g.emit_list(body_ids, bname, "v", indent="    ")):
        if i % 64 == 0:
            L.append("    MF_SYNC_POINT(%d);" % (i // 64))
        if i % clobber_every == 0:
            L.append("    asm volatile(\"\" ::: \"memory\");")
        L.append(line)
    L += ["    acc += %s;" % _ref(g, out, bname), "  }", "  return acc;", "}", "#endif"]
    return "\n".join(L) + "\n"


def _ref(g, r, name):
    if r.n is None:
        return g._k(r.c)
    return name(r.n) if r.s > 0 else "-" + name(r.n)


def evaluate(gen, inputs):
    """numeric evaluation of the generated function (host self-test of the generator)"""
    total = 0.0
    for assign in gen.loop_assign:
        vals = dict(inputs)
        vals.update({"lam%d" % l: v for l, v in zip(gen.loop_legs, assign)})
        total = total + gen.g.evaluate([gen.out], vals)[0]
    return total


# Organisation of the emitted code per process (tuned on the B200, profiles/r1_tuning.md): polarisation basis, the gluon
# legs whose polarisation is a run-time loop, parity; gg -> tt~gg is emitted by gen/lanes.py (one event over four lanes)
PROCESSES = {
    "mf_me2_ee_mumu": lambda: GenEE(),
    "mf_me2_gg_tt": lambda: Gen(2, loop_legs=(), parity=True, basis="circular"),      # 514 flops (linear: 715)
    "mf_me2_gg_ttg": lambda: Gen(3, loop_legs=(0, 2), parity=True, basis="linear"),
}

# loop-invariant values with a cone of at most this many operations are recomputed in the loop body
# (Dag.plan); tuned on B200, see DESIGN.md "Kernels / S7"
DEMOTE = {"mf_me2_gg_ttg": 6}

# barrier-point macro of the generated code (csrc/mf_device.cuh): 128-thread groups (default), or the whole CTA
SYNC_MACRO = {}

# emission order of the helicity-loop body (Dag.schedule): window 0 = creation order
SCHED_WINDOW = 48
SCHED_DISTANCE = 5
# shared-memory-operand variant of gg -> tt~g (emit_function_smem; the |M|^2 stage of the staged path): with the loop invariants parked
# in shared memory a SHORTER loop pays -- gluon leg 2 only (2 trips, 6 806 operations per event instead of 8 712 with legs (0, 2)):
# 102 slots per thread (reciprocals always parked, values built on them recomputed when their cone has <= 16 operations), 5.40 -> 5.05 ms
# per 1e7 events (profiles/r2_tuning.md).  Statements between compiler barriers: 64 .. 1024 make no difference on the B200.
SMEM_LOOP_LEGS = (2,)
SMEM_CLOBBER_EVERY = 256
SMEM_HOIST_COST = 16
SMEM_RCP_LEAF = True


def generate_smem(fname):
    """the organisation of fname's shared-memory-operand variant (a second Gen: the register version keeps PROCESSES[fname])"""
    assert fname == "mf_me2_gg_ttg"
    gen = Gen(3, loop_legs=SMEM_LOOP_LEGS, parity=True, basis="linear")
    gen.build()
    return gen


def generate(fname):
    gen = PROCESSES[fname]()
    gen.build()
    if DEMOTE.get(fname, 0) > 0:
        gen.max_hoist_cost = DEMOTE[fname]
    return gen
