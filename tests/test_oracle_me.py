"""Pins of the oracle's squared matrix elements (O6) and of the full weight chain (O8-O10):
wavefunction identities, closed forms (e+e- -> mu+mu-, gg -> tt~, sigma_hat_gg), brute-force colour
algebra written here from scratch, the literal colour-dressed recursion, Ward / Lorentz / Bose /
parity, golden points, sigma(config 0) and sigma(config 1).  CPU only."""
import itertools
import math
import numpy as np
import pytest
from scipy import integrate
from conftest import read_golden
from paper_2105_10529_b200 import workloads as W

MT, AS = 173.0, 0.118
GS2 = 4 * math.pi * AS


def golden():
    return {k: np.array([float(t) for t in v]) for k, v in read_golden("points.txt").items()}


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def tt_momenta(rts, ct, phi):
    E = rts / 2; p = math.sqrt(E * E - MT * MT); st = math.sqrt(1 - ct * ct)
    v = np.array([p * st * math.cos(phi), p * st * math.sin(phi), p * ct])
    return np.array([[E, 0, 0, E], [E, 0, 0, -E], [E, *v], [E, *(-v)]])


def momenta(mfo, n, rts, rs):
    r = mfo.phase_space(n, rts ** 2, [MT, MT] + [0.0] * (n - 2), rs)
    return np.vstack([[rts / 2, 0, 0, rts / 2], [rts / 2, 0, 0, -rts / 2], r["k"]])


def gg_tt_closed_form(mom):
    """|M|^2 avg = g^4 (1/(6 t1 t2) - 3/8)(t1^2 + t2^2 + rho - rho^2/(4 t1 t2)) (textbook)"""
    shat = mdot(mom[0] + mom[1], mom[0] + mom[1])
    t1 = 2 * mdot(mom[0], mom[2]) / shat; t2 = 2 * mdot(mom[1], mom[2]) / shat; rho = 4 * MT * MT / shat
    return GS2 ** 2 * (1 / (6 * t1 * t2) - 3 / 8) * (t1 * t1 + t2 * t2 + rho - rho * rho / (4 * t1 * t2))


def lorentz(mom, rap, ang):
    """boost along z with rapidity rap, then rotate by ang about x"""
    ch, sh = math.cosh(rap), math.sinh(rap); c, s = math.cos(ang), math.sin(ang)
    out = mom.copy()
    out[:, 0] = ch * mom[:, 0] + sh * mom[:, 3]; z = sh * mom[:, 0] + ch * mom[:, 3]
    out[:, 2] = c * mom[:, 2] - s * z; out[:, 3] = s * mom[:, 2] + c * z
    return out


# ---------------------------------------------------------------- P12 wavefunctions
def test_wavefunction_identities(mfo):
    G = mfo.gamma(); g0 = G[0]
    assert all(np.allclose(G[m] @ G[n] + G[n] @ G[m], 2 * np.diag([1, -1, -1, -1])[m, n] * np.eye(4)) for m in range(4) for n in range(4))
    slash = lambda p: G[0] * p[0] - G[1] * p[1] - G[2] * p[2] - G[3] * p[3]
    rng = np.random.default_rng(0)
    cases = [rng.normal(size=3) * 300 for _ in range(20)] + [np.array([0, 0, 250.0]), np.array([0, 0, -250.0]),
                                                               np.array([1e-7, -2e-7, -300.0]), np.array([30.0, -40.0, -1e4])]
    for pv in cases:
        for m in (0.0, MT):
            p = np.array([math.sqrt(m * m + pv @ pv), *pv])
            su = np.zeros((4, 4), complex); sv = np.zeros((4, 4), complex)
            for lam in (1, -1):
                u = mfo.wf_fermion(0, p, m, lam); v = mfo.wf_fermion(1, p, m, lam)
                ub = u.conj() @ g0; vb = v.conj() @ g0
                scale = p[0] ** 1.5
                assert np.abs((slash(p) - m * np.eye(4)) @ u).max() < 1e-12 * scale       # Dirac equation
                assert np.abs((slash(p) + m * np.eye(4)) @ v).max() < 1e-12 * scale
                assert np.isclose(ub @ u, 2 * m, atol=1e-10 * p[0]) and np.isclose(vb @ v, -2 * m, atol=1e-10 * p[0])
                assert np.isclose(u.conj() @ u, 2 * p[0], rtol=1e-13)
                # helicity: (Sigma.p) u = lam |p| u, (Sigma.p) v = -lam |p| v
                sig = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
                S = sum(np.kron(np.eye(2), sig[i]) * pv[i] for i in range(3)); pa = math.sqrt(pv @ pv)
                assert np.abs(S @ u - lam * pa * u).max() < 1e-11 * scale and np.abs(S @ v + lam * pa * v).max() < 1e-11 * scale
                su += np.outer(u, ub); sv += np.outer(v, vb)
            assert np.allclose(su, slash(p) + m * np.eye(4), atol=1e-11 * p[0])          # completeness
            assert np.allclose(sv, slash(p) - m * np.eye(4), atol=1e-11 * p[0])
        k = np.array([math.sqrt(pv @ pv), *pv])
        e = {lam: mfo.wf_vector(k, lam) for lam in (1, -1)}
        for lam in (1, -1):
            assert abs(mdot(e[lam], k)) < 1e-12 * k[0] and e[lam][0] == 0                # transverse
            assert np.isclose(mdot(e[lam], e[lam].conj()), -1) and abs(mdot(e[lam], e[-lam].conj())) < 1e-14
        # helicity +1: i k_hat x eps = eps ;  sum over polarisations = delta_ij - k_i k_j / k^2
        kh = pv / k[0]
        assert np.allclose(1j * np.cross(kh, e[1][1:]), e[1][1:], atol=1e-13)
        P = sum(np.outer(e[l][1:], e[l][1:].conj()) for l in (1, -1))
        assert np.allclose(P, np.eye(3) - np.outer(kh, kh), atol=1e-13)


# ---------------------------------------------------------------- P11 e+e- -> mu+mu-
def test_ee_mumu_closed_form_and_sigma(mfo):
    alpha = 1 / 132.5; e4 = (4 * math.pi * alpha) ** 2
    for ct in (0.3, -0.77, 0.0, 0.999):
        st = math.sqrt(1 - ct * ct); phi = 0.7
        mom = np.array([[50, 0, 0, 50], [50, 0, 0, -50], [50, 50 * st * math.cos(phi), 50 * st * math.sin(phi), 50 * ct],
                        [50, -50 * st * math.cos(phi), -50 * st * math.sin(phi), -50 * ct]])
        got = mfo.me2(W.EE_MUMU, mom)
        t = -2 * mdot(mom[0], mom[2]); u = -2 * mdot(mom[0], mom[3]); s = 1e4
        assert np.isclose(got, e4 * (1 + ct * ct), rtol=1e-13) and np.isclose(got, 2 * e4 * (t * t + u * u) / s ** 2, rtol=1e-13)
    st = math.sqrt(1 - 0.09)
    m03 = np.array([[50, 0, 0, 50], [50, 0, 0, -50], [50, 50 * st, 0, 15], [50, -50 * st, 0, -15]])
    assert np.isclose(mfo.me2(W.EE_MUMU, m03), 0.009804252089996, rtol=1e-12)    # SURVEY O6.4 value at cos(theta) = 0.3
    sigma_exact = float(read_golden("points.txt")["sigma_cfg0_pb"][0])
    assert np.isclose(sigma_exact, 4 * math.pi * alpha ** 2 / (3 * 1e4) * 0.3894e9, rtol=1e-15)
    v = mfo.Vegas(W.config(W.EE_MUMU, seed=0))
    for _ in range(3):
        it = v.iterate(100_000, n_threads=4)
    r = v.result()
    assert abs(r["integral"] - sigma_exact) < 4 * r["sigma"] and r["sigma"] < 1e-3 and it["n_nonfinite"] == 0


# ---------------------------------------------------------------- P13, P14 gg -> tt~
def test_gg_tt_closed_form_per_event(mfo):
    g = golden()
    m1 = tt_momenta(700.0, 0.37, 1.1)
    assert np.isclose(gg_tt_closed_form(m1), g["G1_me2"][0], rtol=1e-14)
    assert np.isclose(mfo.me2(W.GG_TT, m1), g["G1_me2"][0], rtol=1e-13)
    rng = np.random.default_rng(1)
    for _ in range(60):
        rts = math.exp(rng.uniform(math.log(347.0), math.log(13000.0)))
        m = tt_momenta(rts, rng.uniform(-0.9999, 0.9999), rng.uniform(0, 2 * math.pi))
        assert np.isclose(mfo.me2(W.GG_TT, m), gg_tt_closed_form(m), rtol=2e-12)


def test_sigma_hat_gg(mfo):
    xs, ws = np.polynomial.legendre.leggauss(48)
    for rts in (400.0, 700.0, 3000.0):
        shat = rts * rts; rho = 4 * MT * MT / shat; beta = math.sqrt(1 - rho)
        ang = sum(w * mfo.me2(W.GG_TT, tt_momenta(rts, x, 0.3)) for x, w in zip(xs, ws))
        sig = ang * beta / (16 * math.pi) / (2 * shat)
        exact = math.pi * AS ** 2 / (3 * shat) * ((1 + rho + rho * rho / 16) * math.log((1 + beta) / (1 - beta)) - beta * (7 / 4 + 31 * rho / 16))
        assert np.isclose(sig, exact, rtol=1e-9)


# ---------------------------------------------------------------- P15 sigma(config 1)
def test_config1_cross_section_against_quadrature(mfo):
    """sigma = int dx1 dx2 g(x1) g(x2) sigma_hat(x1 x2 s) = int dln(tau) sigma_hat(tau s) int dln(x1) x1 g(x1) x2 g(x2):
    nested quadrature with the interpolated PDF and the closed-form sigma_hat, against the oracle's VEGAS chain."""
    xf = W.synthetic_gluon_grid(); a = (W.PDF_XMIN, W.PDF_XMAX, W.PDF_QMIN, W.PDF_QMAX)
    s = 13000.0 ** 2; tau0 = 4 * MT * MT / s
    f = lambda x: mfo.pdf_interp(xf, *a, x, MT * MT) / x

    def sighat(shat):
        rho = 4 * MT * MT / shat; beta = math.sqrt(max(1 - rho, 0.0))
        return math.pi * AS ** 2 / (3 * shat) * ((1 + rho + rho * rho / 16) * math.log((1 + beta) / (1 - beta)) - beta * (7 / 4 + 31 * rho / 16))
    knots = np.linspace(math.log(1e-6), 0, 100)

    def lum(lt):        # int d ln x1 of x1 f(x1) x2 f(x2), x2 = tau/x1, piecewise between the PDF knots
        tau = math.exp(lt)
        pts = sorted(set([lt, 0.0] + [k for k in knots if lt < k < 0] + [lt - k for k in knots if lt < lt - k < 0]))
        return sum(integrate.fixed_quad(np.vectorize(lambda l1: math.exp(l1) * f(math.exp(l1)) * (tau / math.exp(l1)) * f(tau / math.exp(l1))), p, q, n=8)[0]
                   for p, q in zip(pts[:-1], pts[1:]))
    edges = np.concatenate([[math.log(tau0)], [k for k in np.linspace(math.log(tau0), 0, 41)[1:]]])
    tot = sum(integrate.fixed_quad(np.vectorize(lambda lt: lum(lt) * sighat(math.exp(lt) * s)), p, q, n=10)[0]
              for p, q in zip(edges[:-1], edges[1:]))
    sigma_q = tot * 0.3894e9
    assert np.isclose(sigma_q, float(read_golden("points.txt")["sigma_cfg1_pb"][0]), rtol=3e-5)
    v = mfo.Vegas(W.config(W.GG_TT, seed=0))
    for _ in range(5):
        v.iterate(100_000, n_threads=mfo.max_threads())
    r = v.result()
    assert abs(r["integral"] - sigma_q) < 4 * r["sigma"] and r["sigma"] / sigma_q < 2e-3


# ---------------------------------------------------------------- P16, P17 colour algebra from scratch
def gell_mann_T():
    l = np.zeros((8, 3, 3), complex)
    l[0][0, 1] = l[0][1, 0] = 1; l[1][0, 1] = -1j; l[1][1, 0] = 1j; l[2][0, 0] = 1; l[2][1, 1] = -1
    l[3][0, 2] = l[3][2, 0] = 1; l[4][0, 2] = -1j; l[4][2, 0] = 1j; l[5][1, 2] = l[5][2, 1] = 1
    l[6][1, 2] = -1j; l[6][2, 1] = 1j; l[7] = np.diag([1, 1, -2]) / math.sqrt(3)
    return l / 2


def test_su3_and_colour_matrices(mfo):
    T, f = mfo.su3(); Tm = gell_mann_T()
    assert np.allclose(T, Tm)
    for a in range(8):
        for b in range(8):
            assert np.isclose(np.trace(Tm[a] @ Tm[b]), 0.5 * (a == b))
            assert np.allclose(Tm[a] @ Tm[b] - Tm[b] @ Tm[a], 1j * np.einsum("c,cij->ij", f[a, b], Tm))
    assert np.isclose(f[0, 1, 2], 1) and np.isclose(f[3, 4, 7], math.sqrt(3) / 2) and np.isclose(f[0, 3, 6], 0.5)
    g = golden()
    for ng in (2, 3, 4):
        num, den = mfo.colour_matrix(ng)
        assert den == g["C%d_den" % ng][0]
        assert np.allclose(num[0], g["C%d_row0" % ng], atol=1e-9)
        assert np.allclose(num, num.T, atol=1e-9) and np.linalg.eigvalsh(num).min() > 0
        assert mfo.diagram_counts(ng) == tuple(int(x) for x in g["counts_ng%d" % ng])
        if ng < 4:                                              # full brute force here (8^ng traces)
            perms = list(itertools.permutations(range(ng)))
            C = np.zeros((len(perms), len(perms)), complex)
            for cols in itertools.product(range(8), repeat=ng):
                Wm = [np.linalg.multi_dot([Tm[cols[i]] for i in p]) if ng > 1 else Tm[cols[0]] for p in perms]
                for i, wi in enumerate(Wm):
                    for j, wj in enumerate(Wm):
                        C[i, j] += np.trace(wi @ wj.conj().T)
            assert np.allclose(C.imag, 0, atol=1e-12) and np.allclose(C.real * den, num, atol=1e-9)
        nf = num.shape[0]
        assert np.isclose(num[0, 0] / den, 3 * (4 / 3) ** ng)     # diagonal = N C_F^ng


# ---------------------------------------------------------------- P18-P23 tt~g, tt~gg
def test_golden_matrix_elements(mfo):
    g = golden()
    m2 = momenta(mfo, 3, 1000.0, g["G2_rs"]); m3 = momenta(mfo, 4, 1500.0, g["G3_rs"])
    assert np.isclose(mfo.me2(W.GG_TTG, m2), g["G2_me2"][0], rtol=1e-12)
    assert np.isclose(mfo.me2(W.GG_TTGG, m3), g["G3_me2"][0], rtol=1e-12)


def test_diagram_list_equals_literal_recursion(mfo):
    """Algorithm A (diagram list + colour flows) against algorithm B (colour-dressed recursion with
    explicit SU(3) indices), amplitude by amplitude and colour-summed."""
    g = golden(); T = gell_mann_T(); rng = np.random.default_rng(2)
    pts = {W.GG_TT: tt_momenta(700.0, 0.37, 1.1), W.GG_TTG: momenta(mfo, 3, 1000.0, g["G2_rs"]), W.GG_TTGG: momenta(mfo, 4, 1500.0, g["G3_rs"])}
    for proc, mom in pts.items():
        ng = proc + 1; perms = list(itertools.permutations(range(ng)))
        for _ in range(12 if proc < W.GG_TTGG else 6):
            hel = rng.choice([-1, 1], size=ng + 2); col = rng.integers(0, 8, size=ng); c3, c4 = rng.integers(0, 3, size=2)
            jamp, _ = mfo.jamps(proc, mom, hel)
            viaA = sum(np.linalg.multi_dot([T[col[i]] for i in p])[c3, c4] * jamp[s] for s, p in enumerate(perms))
            viaB = mfo.amp_literal(proc, mom, hel, col, c3, c4)
            assert abs(viaA - viaB) < 1e-11 * np.abs(jamp).max(), (proc, hel, col)
    # colour-summed: one helicity of tt~gg (36864 colour terms) and a few of tt~g (4608 each)
    hel = [1, -1, 1, 1, -1, 1]; hidx = sum(1 << l for l, h in enumerate(hel) if h > 0)
    assert np.isclose(mfo.me2_literal(W.GG_TTGG, pts[W.GG_TTGG], hel_only=hidx), mfo.jamps(W.GG_TTGG, pts[W.GG_TTGG], hel)[1], rtol=1e-12)
    for hidx in (0, 5, 22, 31):
        hel = [1 if hidx >> l & 1 else -1 for l in range(5)]
        assert np.isclose(mfo.me2_literal(W.GG_TTG, pts[W.GG_TTG], hel_only=hidx), mfo.jamps(W.GG_TTG, pts[W.GG_TTG], hel)[1], rtol=1e-12)
    assert np.isclose(mfo.me2_literal(W.GG_TT, pts[W.GG_TT]), mfo.me2(W.GG_TT, pts[W.GG_TT]), rtol=1e-13)


def test_ward_identity_per_flow(mfo):
    g = golden(); rng = np.random.default_rng(3)
    for proc, n in ((W.GG_TT, 2), (W.GG_TTG, 3), (W.GG_TTGG, 4)):
        for _ in range(3):
            mom = momenta(mfo, n, math.exp(rng.uniform(math.log(500), math.log(6000))), rng.uniform(0.05, 0.95, size=3 * n - 4))
            hel = rng.choice([-1, 1], size=n + 2)
            # scale: the largest flow amplitude over all helicities (a single helicity can vanish)
            scale = max(np.abs(mfo.jamps(proc, mom, [1 if h >> l & 1 else -1 for l in range(n + 2)])[0]).max() for h in range(1 << (n + 2)))
            for leg in range(n):
                jw, mw = mfo.jamps(proc, mom, hel, ward_leg=leg)
                # eps -> k scales the amplitude by ~E; compare with |jamp| * E
                assert np.abs(jw).max() < 1e-9 * scale * mom[0, 0], (proc, leg)


def test_lorentz_bose_parity(mfo):
    rng = np.random.default_rng(4)
    for proc, n in ((W.GG_TT, 2), (W.GG_TTG, 3), (W.GG_TTGG, 4)):
        for _ in range(2):
            mom = momenta(mfo, n, 1200.0, rng.uniform(0.05, 0.95, size=3 * n - 4))
            ref = mfo.me2(proc, mom)
            assert np.isclose(mfo.me2(proc, lorentz(mom, 0.4, 0.7)), ref, rtol=1e-11)           # P20
            swapped = mom.copy(); swapped[[0, 1]] = mom[[1, 0]]                                   # P21 incoming gluons
            assert np.isclose(mfo.me2(proc, lorentz(swapped, 0.0, math.pi)), ref, rtol=1e-11)
            if n == 4:
                sw = mom.copy(); sw[[4, 5]] = mom[[5, 4]]                                         # P21 final gluons
                assert np.isclose(mfo.me2(proc, sw), ref, rtol=1e-12)
            hel = rng.choice([-1, 1], size=n + 2)                                                 # P22 parity
            assert np.isclose(mfo.jamps(proc, mom, hel)[1], mfo.jamps(proc, mom, -hel)[1], rtol=1e-11)


# ---------------------------------------------------------------- P24 collinear factorisation: absolute normalisation
# Ward, Lorentz, Bose and the A = B comparison are blind to a common normalisation or convention slip (coupling powers,
# 1/256, colour matrix).  The collinear limits are not: they tie |M(gg -> tt~g)|^2 to the closed form of gg -> tt~ and
# |M(gg -> tt~gg)|^2 to |M(gg -> tt~g)|^2 through the unregularised Altarelli-Parisi function (textbook; azimuth averaged)
#   P_gg(z) = 2 C_A [ z/(1-z) + (1-z)/z + z(1-z) ],  C_A = 3:
#   final state   k3 || k4:  |M_{n+1}|^2 -> (2 g_s^2 / s_34) P_gg(z) |M_n|^2,          z = E_3 / (E_3 + E_4)
#   initial state k || p_a:  |M_{n+1}|^2 -> (2 g_s^2 / (2 p_a.k)) P_gg(x)/x |M_n(x p_a, p_b)|^2,   x = (p_a + p_b - k)^2 / shat
# (both sides averaged over the incoming gluons' spins and colours, summed over the final ones, no symmetry factor).
def p_gg(z):
    return 2 * 3.0 * (z / (1 - z) + (1 - z) / z + z * (1 - z))


def boost_from_rest(p, K):
    """p given in the rest frame of K -> the frame in which K is given"""
    M = math.sqrt(mdot(K, K)); E = (K[0] * p[0] + K[1:] @ p[1:]) / M
    return np.array([E, *(p[1:] + K[1:] * (p[0] + E) / (K[0] + M))])


@pytest.mark.parametrize("rts,x,cts,phis", [(900.0, 0.7, 0.3, 1.1), (2500.0, 0.45, -0.6, 4.0)])
def test_initial_state_collinear_limit_ties_ttg_to_closed_form_tt(mfo, rts, x, cts, phis):
    E = rts / 2
    pa, pb = np.array([E, 0, 0, E]), np.array([E, 0, 0, -E])
    dev = {}
    for theta in (1e-2, 1e-3):
        acc = 0.0
        for j in range(8):                                        # azimuth average: kills the cos(2 phi) spin correlation
            phi = 0.37 + 2 * math.pi * j / 8
            k = (1 - x) * E * np.array([1, math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
            K = pa + pb - k
            M = math.sqrt(mdot(K, K))
            b = tt_momenta(M, cts, phis)                           # t t~ in the rest frame of K, same angles as the Born point
            mom = np.array([pa, pb, boost_from_rest(b[2], K), boost_from_rest(b[3], K), k])
            xx = M * M / rts ** 2
            born = gg_tt_closed_form(b)                            # the CLOSED FORM, not the oracle
            acc += mfo.me2(W.GG_TTG, mom) / (2 * GS2 / (2 * mdot(pa, k)) * p_gg(xx) / xx * born)
        dev[theta] = acc / 8 - 1
    assert abs(dev[1e-3]) < 2e-6 and abs(dev[1e-2]) < 1e-4, dev   # approached like theta^2


@pytest.mark.parametrize("rts,rs,ctd", [(900.0, [0.31, 0.62, 0.44, 0.83, 0.27], 0.2), (3000.0, [0.7, 0.2, 0.9, 0.55, 0.4], -0.5)])
def test_final_state_collinear_limit_ties_ttgg_to_ttg(mfo, rts, rs, ctd):
    E = rts / 2
    beams = [[E, 0, 0, E], [E, 0, 0, -E]]
    born = mfo.me2(W.GG_TTG, np.vstack([beams, mfo.phase_space(3, rts * rts, [MT, MT, 0.0], rs)["k"]]))
    dev = {}
    for m34 in (5.0, 0.5):                                         # the gluon pair as a particle of small mass m34
        ks = mfo.phase_space(3, rts * rts, [MT, MT, m34], rs)["k"]
        K = ks[2]
        n = K[1:] / np.linalg.norm(K[1:]); a = np.cross(n, [0.3, -0.5, 0.8]); a /= np.linalg.norm(a); b = np.cross(n, a)
        acc = 0.0
        for j in range(8):
            phid = 0.11 + 2 * math.pi * j / 8
            d = math.sqrt(1 - ctd * ctd) * (math.cos(phid) * a + math.sin(phid) * b) + ctd * n
            k3 = boost_from_rest(np.array([m34 / 2, *(m34 / 2 * d)]), K)
            k4 = boost_from_rest(np.array([m34 / 2, *(-m34 / 2 * d)]), K)
            mom = np.vstack([beams, ks[:2], k3, k4])
            acc += mfo.me2(W.GG_TTGG, mom) / (2 * GS2 / m34 ** 2 * p_gg(k3[0] / K[0]) * born)
        dev[m34] = acc / 8 - 1
    assert abs(dev[0.5]) < 1e-4 and abs(dev[5.0]) < 1e-2, dev      # approached like m34^2 / shat


# ---------------------------------------------------------------- P26-P28 weight chain and reductions
@pytest.mark.parametrize("proc", [W.EE_MUMU, W.GG_TT, W.GG_TTG])
def test_weight_chain_and_reductions(mfo, proc):
    cfg = W.config(proc, seed=3); v = mfo.Vegas(cfg); N = 3000
    rng = np.random.default_rng(9)
    e = np.zeros((v.d, 51)); e[:, 1:] = np.cumsum(rng.uniform(0.5, 2, size=(v.d, 50)), axis=1); e /= e[:, -1:]
    v.set_grid(e)
    out = v.eval(0, 0, N, n_threads=4)
    # chunking: evaluating a sub-range gives identical events (counter RNG keyed on the global index)
    sub = v.eval(0, 1000, 500)
    for k in out:
        assert np.array_equal(out[k][1000:1500], sub[k])
    # per-event chain recomputed here from the recorded stage outputs
    s = cfg["sqrt_s"] ** 2
    for i in range(0, N, 37):
        x = out["x"][i]; J = np.prod([50 * (e[j, out["bins"][i, j] + 1] - e[j, out["bins"][i, j]]) for j in range(v.d)])
        mom = out["momenta"][i]
        if proc == W.EE_MUMU:
            F = J * out["me2"][i] / (8 * math.pi) * 0.3894e9 / (2 * s)
        else:
            smin = (2 * MT + (proc - 1) * cfg["ptmin_g"]) ** 2; tau0 = smin / s
            tau = tau0 ** (1 - x[0]); x1 = tau ** x[1]; x2 = tau / x1; shat = tau * s
            assert np.isclose(mom[0, 0], math.sqrt(shat) / 2, rtol=1e-13)
            Jx = tau * math.log(tau0) * math.log(tau)
            ps = mfo.phase_space(v.n_final, shat, [MT, MT] + [0.0] * (v.n_final - 2), x[2:])
            assert np.allclose(ps["k"], mom[2:], rtol=1e-12, atol=1e-9)
            assert np.isclose(out["me2"][i], mfo.me2(proc, mom), rtol=1e-12) or not out["pass_"][i]
            F = J * Jx * out["pdf"][i, 0] / x1 * out["pdf"][i, 1] / x2 * out["me2"][i] * ps["W0"] * ps["Wm"] * 0.3894e9 / (2 * shat) * out["pass_"][i]
        assert np.isclose(out["weight"][i], F, rtol=1e-12)
    # reductions against exact sums (math.fsum) and the two-pass variance
    acc, cnt = v.accumulate(0, 0, N, N, n_threads=3)
    t = out["weight"] / N
    assert np.isclose(acc[0], math.fsum(t), rtol=1e-14) and np.isclose(acc[1], math.fsum(t * t), rtol=1e-14)
    H = acc[2:].reshape(v.d, 50)
    for j in range(v.d):
        for k in range(50):
            assert np.isclose(H[j, k], math.fsum((t * t)[out["bins"][:, j] == k]), rtol=1e-13, atol=0)
    assert cnt[0] == out["pass_"].sum() and cnt[1] == 0
    # sharding: two halves accumulate to the same sums
    a2, c2 = v.accumulate(0, 0, 1234, N, n_threads=2); a2, c3 = v.accumulate(0, 1234, N - 1234, N, n_threads=2, acc=a2)
    assert np.allclose(a2, acc, rtol=1e-13, atol=0) and c2[0] + c3[0] == cnt[0]
    it = v.finalize(acc, N, cnt[0], cnt[1])
    var_two_pass = np.var(out["weight"], ddof=1) / N
    assert np.isclose(it["sigma"] ** 2, var_two_pass, rtol=1e-9) and np.isclose(it["integral"], out["weight"].mean(), rtol=1e-13)
    assert np.allclose(v.get_grid(), mfo.refine(e, H, 1.5), rtol=0, atol=0)
