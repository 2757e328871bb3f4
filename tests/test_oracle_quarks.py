"""Pins of the oracle's quark channel (q q~ -> t t~ with flavour-summed PDFs on an
11-flavour synthetic grid; readings O5q, O6q of DESIGN.md).  Checked against what the mathematics fixes: the
textbook closed form of the spin/colour-averaged |M|^2, the textbook partonic cross section (by angular
quadrature of the oracle's |M|^2), Lorentz invariance and beam-exchange symmetry, the flavour sum rebuilt from
single-table interpolations, and the hadronic cross section by nested quadrature through the whole chain."""
import math

import numpy as np
from scipy import integrate

from paper_2105_10529_b200 import workloads as W

MT, AS = 173.0, 0.118


def tt_momenta(rts, ct, phi, m=MT):
    E = rts / 2; p = math.sqrt(E * E - m * m); st = math.sqrt(1 - ct * ct)
    k = np.array([E, p * st * math.cos(phi), p * st * math.sin(phi), p * ct])
    return np.array([[E, 0, 0, E], [E, 0, 0, -E], k, [E, -k[1], -k[2], -k[3]]])


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def qq_tt_closed_form(mom, m=MT, alpha_s=AS):
    """sum-bar |M|^2 = (4 g^4 / 9) [(m^2 - t)^2 + (m^2 - u)^2 + 2 m^2 s] / s^2  (Combridge 1979; Ellis-Stirling-Webber
    table 10.2 in the massive case)"""
    g4 = (4 * math.pi * alpha_s) ** 2
    s = mdot(mom[0] + mom[1], mom[0] + mom[1])
    t = mdot(mom[0] - mom[2], mom[0] - mom[2]); u = mdot(mom[0] - mom[3], mom[0] - mom[3])
    return 4 * g4 / 9 * ((m * m - t) ** 2 + (m * m - u) ** 2 + 2 * m * m * s) / s ** 2


def sighat_qq(shat, m=MT, alpha_s=AS):
    """sigma_hat(q q~ -> Q Q~) = 8 pi alpha_s^2 / (27 shat) * beta * (1 + rho/2), rho = 4 m^2 / shat
    (Nason, Dawson, Ellis 1988: f_qq~ = pi beta rho (2 + rho) / 27 in units alpha_s^2 / m^2)"""
    rho = 4 * m * m / shat; beta = math.sqrt(max(1 - rho, 0.0))
    return 8 * math.pi * alpha_s ** 2 / (27 * shat) * beta * (1 + rho / 2)


def test_qq_tt_closed_form_per_event(mfo):
    rng = np.random.default_rng(5)
    for _ in range(80):
        rts = math.exp(rng.uniform(math.log(347.0), math.log(13000.0)))
        m = tt_momenta(rts, rng.uniform(-0.9999, 0.9999), rng.uniform(0, 2 * math.pi))
        assert np.isclose(mfo.me2(W.QQ_TT, m), qq_tt_closed_form(m), rtol=2e-12)
    # massless limit = the QED-like 1 + cos^2 shape: (4 g^4/9) (t^2 + u^2)/s^2 = (2 g^4/9)(1 + cos^2 theta)
    m = tt_momenta(1000.0, 0.3, 0.7, m=1e-9)
    g4 = (4 * math.pi * AS) ** 2
    assert np.isclose(mfo.me2(W.QQ_TT, m, m_top=1e-9), 2 * g4 / 9 * (1 + 0.09), rtol=1e-10)
    # threshold: t = u = -m^2, s = 4 m^2: (4 g^4/9) (4 m^4 + 4 m^4 + 8 m^4) / (16 m^4) = 4 g^4 / 9
    m = tt_momenta(2 * MT * (1 + 1e-9), 0.5, 0.1)
    assert np.isclose(mfo.me2(W.QQ_TT, m), 4 * g4 / 9, rtol=1e-7)


def test_qq_tt_symmetries(mfo):
    """beam exchange (t <-> u), azimuthal rotation, and a boost along the beam leave |M|^2 unchanged"""
    m = tt_momenta(800.0, 0.41, 0.9)
    ref = mfo.me2(W.QQ_TT, m)
    sw = m.copy(); sw[[0, 1]] = sw[[1, 0]]
    assert np.isclose(mfo.me2(W.QQ_TT, sw), ref, rtol=1e-12)
    assert np.isclose(mfo.me2(W.QQ_TT, tt_momenta(800.0, 0.41, 2.3)), ref, rtol=1e-12)
    assert np.isclose(mfo.me2(W.QQ_TT, tt_momenta(800.0, -0.41, 0.9)), ref, rtol=1e-12)
    y = 0.7; ch, sh = math.cosh(y), math.sinh(y)
    b = m.copy(); b[:, 0] = ch * m[:, 0] + sh * m[:, 3]; b[:, 3] = sh * m[:, 0] + ch * m[:, 3]
    assert np.isclose(mfo.me2(W.QQ_TT, b), ref, rtol=1e-11)


def test_sigma_hat_qq(mfo):
    xs, ws = np.polynomial.legendre.leggauss(16)
    for rts in (350.0, 400.0, 700.0, 3000.0):
        shat = rts * rts; beta = math.sqrt(1 - 4 * MT * MT / shat)
        ang = sum(w * mfo.me2(W.QQ_TT, tt_momenta(rts, x, 0.3)) for x, w in zip(xs, ws))
        sig = ang * beta / (16 * math.pi) / (2 * shat)
        assert np.isclose(sig, sighat_qq(shat), rtol=1e-11)


def test_flavour_grid_and_luminosity_record(mfo):
    """the 11-flavour input grid (index = PDG id + 5), and the per-event flavour sums against single-table lookups"""
    g = W.synthetic_flavour_grid()
    assert g.shape == (11, W.PDF_NX, W.PDF_NQ)
    assert np.array_equal(g[5], W.synthetic_gluon_grid())
    assert (g[:, -1, :] == 0).all() and (g[:, :-1, :] > 0).all()
    assert np.array_equal(g[2], g[8]) and np.array_equal(g[1], g[9]) and np.array_equal(g[0], g[10])   # s, c, b: sea only
    assert (g[7, :-1] > g[3, :-1]).all() and (g[6, :-1] > g[4, :-1]).all()                               # u > u~, d > d~
    # valence number sum rules of the synthetic shapes: int (u - u~) dx = 2.2 B(0.5, 4), int (d - d~) dx = 1.1 B(0.5, 5)
    lx = np.linspace(math.log(W.PDF_XMIN), 0.0, W.PDF_NX)
    for fl, exact in ((2, 2.2 * math.gamma(0.5) * math.gamma(4) / math.gamma(4.5)), (1, 1.1 * math.gamma(0.5) * math.gamma(5) / math.gamma(5.5))):
        num = integrate.trapezoid(g[5 + fl, :, 0] - g[5 - fl, :, 0], lx)       # int x f dln x
        assert abs(num / exact - 1) < 2e-2
    cfg = W.config(W.QQ_TT, seed=3)
    v = mfo.Vegas(cfg)
    assert v.d == 4 and v.n_final == 2
    out = v.eval(0, 0, 50)
    a = (W.PDF_XMIN, W.PDF_XMAX, W.PDF_QMIN, W.PDF_QMAX)
    s = cfg["sqrt_s"] ** 2
    for i in range(50):
        mom = out["momenta"][i]; shat = 4 * mom[0, 0] ** 2
        x1, x2, _, jx = mfo.x_map(out["x"][i, 0], out["x"][i, 1], s, 4 * MT * MT)
        assert np.isclose(x1 * x2 * s, shat, rtol=1e-13)
        f = lambda fl, x: mfo.pdf_interp(g[5 + fl], *a, x, MT * MT)
        l12 = sum(f(q, x1) * f(-q, x2) for q in range(1, 6)); l21 = sum(f(-q, x1) * f(q, x2) for q in range(1, 6))
        assert np.allclose(out["pdf"][i], [l12, l21], rtol=1e-13)
        assert np.isclose(out["me2"][i], qq_tt_closed_form(mom), rtol=2e-12)
        # weight chain on the uniform grid (J_V = 1): F = J_x (L12 + L21)/(x1 x2) |M|^2 /(8 pi) beta K / (2 shat)
        beta = math.sqrt(1 - 4 * MT * MT / shat)
        F = jx * (l12 + l21) / (x1 * x2) * out["me2"][i] / (8 * math.pi) * beta * 0.3894e9 / (2 * shat)
        assert np.isclose(out["weight"][i], F, rtol=1e-11)


def test_qq_tt_cross_section_against_quadrature(mfo):
    """sigma = sum_q int dx1 dx2 [f_q(x1) f_q~(x2) + f_q~(x1) f_q(x2)] sigma_hat(x1 x2 s): nested quadrature with the
    interpolated flavour tables and the closed-form sigma_hat, against the oracle's VEGAS chain (both tau maps)."""
    g = W.synthetic_flavour_grid(); a = (W.PDF_XMIN, W.PDF_XMAX, W.PDF_QMIN, W.PDF_QMAX)
    s = 13000.0 ** 2; tau0 = 4 * MT * MT / s
    xf = lambda fl, x: mfo.pdf_interp(g[5 + fl], *a, x, MT * MT)
    knots = np.linspace(math.log(1e-6), 0, 100)

    def lum(lt):        # int d ln x1 of sum_q [x1 f_q(x1) x2 f_q~(x2) + (q <-> q~)], x2 = tau/x1
        tau = math.exp(lt)
        pts = sorted(set([lt, 0.0] + [k for k in knots if lt < k < 0] + [lt - k for k in knots if lt < lt - k < 0]))

        def integrand(l1):
            x1 = math.exp(l1); x2 = tau / x1
            return sum(xf(q, x1) * xf(-q, x2) + xf(-q, x1) * xf(q, x2) for q in range(1, 6))
        return sum(integrate.fixed_quad(np.vectorize(integrand), p, q, n=6)[0] for p, q in zip(pts[:-1], pts[1:]))
    edges = np.linspace(math.log(tau0), 0, 31)
    tot = sum(integrate.fixed_quad(np.vectorize(lambda lt: lum(lt) * sighat_qq(math.exp(lt) * s)), p, q, n=8)[0]
              for p, q in zip(edges[:-1], edges[1:]))
    sigma_q = tot * 0.3894e9
    for gen in (0, W.GEN_LINEAR_TAU):
        v = mfo.Vegas(W.config(W.QQ_TT, seed=0, generator=gen))
        for _ in range(5):
            v.iterate(100_000, n_threads=mfo.max_threads())
        r = v.result()
        assert abs(r["integral"] - sigma_q) < 4 * r["sigma"] and r["sigma"] / sigma_q < 3e-3, (gen, r, sigma_q)


def test_pp_tt_is_the_sum_of_its_subprocesses(mfo):
    """process 5 (p p -> t t~: g g and q q~ in one integrand): event by event the weight is the sum of the weights of the
    two pinned subprocesses on the same points (same seed, same grid: d = 4 for all three), the record holds the two
    luminosities, and the cross section is the sum of the two quadrature values (1074.39 + 79.96 pb)"""
    g11 = W.synthetic_flavour_grid()
    cfg5 = W.config(W.PP_TT, seed=21)
    v5, v1, v4 = mfo.Vegas(cfg5), mfo.Vegas(W.config(W.GG_TT, seed=21)), mfo.Vegas(W.config(W.QQ_TT, seed=21))
    assert v5.d == 4 and v5.n_final == 2
    rng = np.random.default_rng(2)
    w = rng.uniform(0.4, 1.6, size=(4, 50))
    e = np.concatenate([np.zeros((4, 1)), np.cumsum(w, axis=1) / w.sum(axis=1, keepdims=True)], axis=1); e[:, -1] = 1.0
    for v in (v5, v1, v4):
        v.set_grid(e)
    n = 400
    o5, o1, o4 = v5.eval(2, 10, n), v1.eval(2, 10, n), v4.eval(2, 10, n)
    assert np.array_equal(o5["x"], o1["x"]) and np.array_equal(o5["momenta"], o4["momenta"])
    np.testing.assert_allclose(o5["weight"], o1["weight"] + o4["weight"], rtol=1e-13)
    np.testing.assert_allclose(o5["pdf"][:, 0], o1["pdf"][:, 0] * o1["pdf"][:, 1], rtol=1e-14)
    np.testing.assert_allclose(o5["pdf"][:, 1], o4["pdf"].sum(axis=1), rtol=1e-14)
    lum = o5["pdf"]
    np.testing.assert_allclose(o5["me2"] * lum.sum(axis=1), lum[:, 0] * o1["me2"] + lum[:, 1] * o4["me2"], rtol=1e-13)
    v = mfo.Vegas(W.config(W.PP_TT, seed=0))
    for _ in range(5):
        v.iterate(100_000, n_threads=mfo.max_threads())
    r = v.result()
    assert abs(r["integral"] - (1074.393 + 79.96)) < 4 * r["sigma"] + 0.03 and r["sigma"] < 1.5, r


# ---- the channels with a second quark line and one gluon: q q~ -> t t~ g (process 6), q g -> t t~ q (process 7) ------------
# oracle/mfo_amp2q.cpp writes the five diagrams out with explicit gamma matrices and the literal colour sum.  Pins: the Ward
# identity of the external gluon; the four initial-state collinear limits, which tie both processes to the CLOSED FORMS of
# q q~ -> t t~ and g g -> t t~ through the textbook (unregularised, azimuth-averaged) Altarelli-Parisi functions
#   |M_{n+1}|^2 -> (2 g_s^2 / (2 p.k)) P(x)/x |M_n(x p, p')|^2,  x = (p + p' - k)^2 / shat:
#   q -> q(x) g:  P_qq = C_F (1 + x^2)/(1 - x)      q -> g(x) q:  P_gq = C_F (1 + (1 - x)^2)/x      g -> q(x) q~:  P_qg = T_R (x^2 + (1 - x)^2)
# (coupling power, colour factors C_F = 4/3 and T_R = 1/2, the 1/36 and 1/96 averages and the relative signs of the diagrams
# all enter); Lorentz invariance; positivity; and the cross sections through both oracle generators.
def gg_tt_closed_form(mom, m=MT, alpha_s=AS):
    g4 = (4 * math.pi * alpha_s) ** 2
    s = mdot(mom[0] + mom[1], mom[0] + mom[1])
    t1 = 2 * mdot(mom[0], mom[2]) / s; t2 = 2 * mdot(mom[1], mom[2]) / s; rho = 4 * m * m / s
    return g4 * (1 / (6 * t1 * t2) - 3 / 8) * (t1 * t1 + t2 * t2 + rho - rho * rho / (4 * t1 * t2))


def boost_from_rest(p, K):
    M = math.sqrt(mdot(K, K)); E = (K[0] * p[0] + K[1:] @ p[1:]) / M
    return np.array([E, *(p[1:] + K[1:] * (p[0] + E) / (K[0] + M))])


def three_body(mfo, rts, rs):
    ks = mfo.phase_space(3, rts * rts, [MT, MT, 0.0], rs)["k"]
    return np.vstack([[rts / 2, 0, 0, rts / 2], [rts / 2, 0, 0, -rts / 2], ks])


def test_two_quark_lines_ward_identity_lorentz_and_positivity(mfo):
    rng = np.random.default_rng(31)
    for proc in (W.QQ_TTG, W.QG_TTQ):
        for _ in range(6):
            mom = three_body(mfo, math.exp(rng.uniform(math.log(450.0), math.log(6000.0))), rng.uniform(0.03, 0.97, 5))
            ref = mfo.me2_2q(proc, mom)
            assert ref > 0 and mfo.me2(proc, mom) == ref
            assert abs(mfo.me2_2q(proc, mom, ward=1)) < 1e-9 * ref          # eps -> k: the five diagrams cancel
            ch, sh, c, s = math.cosh(0.6), math.sinh(0.6), math.cos(0.8), math.sin(0.8)
            lor = mom.copy()
            lor[:, 0] = ch * mom[:, 0] + sh * mom[:, 3]; z = sh * mom[:, 0] + ch * mom[:, 3]
            lor[:, 2] = c * mom[:, 2] - s * z; lor[:, 3] = s * mom[:, 2] + c * z
            assert np.isclose(mfo.me2_2q(proc, lor), ref, rtol=1e-10)        # boost along z, rotation about x


def collinear_ratio(mfo, proc, side, born, split, rts, x, theta):
    """azimuth average of |M_{n+1}|^2 / [ (2 g^2 / (2 p.k)) P(x')/x' |M_n|^2 ] for the emitted parton k at angle theta to beam `side`"""
    E = rts / 2
    pa, pb = np.array([E, 0, 0, E]), np.array([E, 0, 0, -E])
    gs2 = 4 * math.pi * AS
    acc = 0.0
    for j in range(8):
        phi = 0.37 + 2 * math.pi * j / 8
        k = (1 - x) * E * np.array([1, math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), (1 if side == 0 else -1) * math.cos(theta)])
        K = pa + pb - k
        M = math.sqrt(mdot(K, K))
        b = tt_momenta(M, 0.3, 1.1)
        mom = np.array([pa, pb, boost_from_rest(b[2], K), boost_from_rest(b[3], K), k])
        xx = M * M / rts ** 2
        acc += mfo.me2_2q(proc, mom) / (2 * gs2 / (2 * mdot(pa if side == 0 else pb, k)) * split(xx) / xx * born(b))
    return acc / 8


def test_two_quark_lines_collinear_limits_tie_to_closed_forms(mfo):
    CF, TR = 4.0 / 3.0, 0.5
    p_qq = lambda x: CF * (1 + x * x) / (1 - x)
    p_gq = lambda x: CF * (1 + (1 - x) ** 2) / x
    p_qg = lambda x: TR * (x * x + (1 - x) ** 2)
    cases = [(W.QQ_TTG, 0, qq_tt_closed_form, p_qq),      # g || q:   q -> q g,   hard q q~ -> t t~
             (W.QQ_TTG, 1, qq_tt_closed_form, p_qq),      # g || q~
             (W.QG_TTQ, 0, gg_tt_closed_form, p_gq),      # outgoing q || incoming q: q -> g q, hard g g -> t t~
             (W.QG_TTQ, 1, qq_tt_closed_form, p_qg)]      # outgoing q || incoming g: g -> q~ q, hard q q~ -> t t~
    for proc, side, born, split in cases:
        for rts, x in ((1100.0, 0.65), (3000.0, 0.3)):
            d2, d3 = (collinear_ratio(mfo, proc, side, born, split, rts, x, th) - 1 for th in (1e-2, 1e-3))
            assert abs(d3) < 5e-6 and abs(d2) < 5e-4, (proc, side, rts, x, d2, d3)     # approached like theta^2


def test_two_quark_lines_integrand_chain(mfo):
    """the event weight of processes 6 and 7 rebuilt here from the oracle's per-event records and single calls: luminosities from
    single-table interpolations, the channels' |M|^2 from mfo_me2_2q on relabelled momenta (beam exchange, t <-> t~)"""
    for proc in (W.QQ_TTG, W.QG_TTQ):
        cfg = W.config(proc, seed=2)
        orc = mfo.Vegas(cfg)
        assert orc.d == 7 and orc.n_final == 3
        ev = orc.eval(1, 100, 40)
        xf = cfg["pdf_xf"]
        pdf = lambda f, x: mfo.pdf_interp(xf[5 + f], W.PDF_XMIN, W.PDF_XMAX, W.PDF_QMIN, W.PDF_QMAX, x, cfg["mu_f"] ** 2)
        ref2 = mfo.Vegas(W.config(W.GG_TTG, seed=2, pdf_xf=xf[5])).eval(1, 100, 40)      # same kinematics, cuts and Jacobians
        np.testing.assert_array_equal(ev["pass_"], ref2["pass_"])
        np.testing.assert_array_equal(ev["momenta"], ref2["momenta"])
        for i in range(40):
            mom = ev["momenta"][i]
            shat = 4 * mom[0][0] ** 2
            # x1, x2 from the records of the gluon run: weight_gg = J ... xg(x1) xg(x2)/(x1 x2) |M_gg|^2 ...
            y0, y1 = ev["x"][i][0], ev["x"][i][1]
            tau0 = (2 * MT + 30.0) ** 2 / 13000.0 ** 2
            tau = tau0 ** (1 - y0); x1 = tau ** y1; x2 = tau / x1
            assert np.isclose(tau * 13000.0 ** 2, shat, rtol=1e-12)
            beams = mom.copy(); beams[[0, 1]] = mom[[1, 0]]
            cc = mom.copy(); cc[[2, 3]] = mom[[3, 2]]
            both = beams.copy(); both[[2, 3]] = beams[[3, 2]]
            if proc == W.QQ_TTG:
                lum = [sum(pdf(f, x1) * pdf(-f, x2) for f in range(1, 6)), sum(pdf(-f, x1) * pdf(f, x2) for f in range(1, 6))]
                me = [mfo.me2_2q(proc, mom), mfo.me2_2q(proc, beams)]
                np.testing.assert_allclose(ev["pdf"][i], lum, rtol=1e-13)
            else:
                q1 = sum(pdf(f, x1) for f in range(1, 6)); a1 = sum(pdf(-f, x1) for f in range(1, 6))
                q2 = sum(pdf(f, x2) for f in range(1, 6)); a2 = sum(pdf(-f, x2) for f in range(1, 6))
                lum = [q1 * pdf(0, x2), pdf(0, x1) * q2, a1 * pdf(0, x2), pdf(0, x1) * a2]
                me = [mfo.me2_2q(proc, mom), mfo.me2_2q(proc, beams), mfo.me2_2q(proc, cc), mfo.me2_2q(proc, both)]
                np.testing.assert_allclose(ev["pdf"][i], [lum[0] + lum[2], lum[1] + lum[3]], rtol=1e-13)
            if not ev["pass_"][i]:
                assert ev["weight"][i] == 0.0
                continue
            tot = sum(l * m for l, m in zip(lum, me))
            assert np.isclose(ev["me2"][i], tot / sum(lum), rtol=1e-12)
            # everything but luminosity x |M|^2 is the gluon run's factor: F / (L |M|^2) agrees between the two processes
            gg = ref2["weight"][i] / (ref2["pdf"][i][0] * ref2["pdf"][i][1] * ref2["me2"][i])
            assert np.isclose(ev["weight"][i] / tot, gg, rtol=1e-12)
