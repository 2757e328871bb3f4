"""Pins of the oracle's non-matrix-element steps (O1-O5, O7, O9-O11) against what the paper's
configs and the mathematics fix: known-answer vectors, closed forms, invariants, library routines.
CPU only.  Pin numbers P1..P29 refer to DESIGN.md ("Pins")."""
import math
import numpy as np
import pytest
from scipy import integrate, interpolate
from conftest import read_golden
from paper_2105_10529_b200 import workloads as W

MT = 173.0


# ---------------------------------------------------------------- P1, P2  RNG
def test_philox_known_answers(mfo):
    for name, v in read_golden("philox_kat.txt").items():
        w = [int(t, 16) for t in v]
        out = mfo.philox4x32_10(w[0:4], w[4:6])
        assert [int(o) for o in out] == w[6:10], name


def test_uniforms_exact_open_interval(mfo):
    us = np.array([mfo.uniforms(7, 3, ev, 7) for ev in range(4000)])
    assert us.min() > 0.0 and us.max() < 1.0
    k = us * 2.0 ** 52 - 0.5                       # u = (X>>12 + 1/2) 2^-52 is exact in fp64
    assert np.all(k == np.floor(k))
    assert np.all(np.floor(us * 50) <= 49)
    assert abs(us.mean() - 0.5) < 4 / math.sqrt(12 * us.size)
    assert abs((us ** 2).mean() - 1 / 3) < 0.01
    # counter layout (A1): dims (2j, 2j+1) come from block j of (event lo, event hi, j, iteration), key = seed
    seed, it, ev = 0x123456789ABCDEF, 5, (3 << 32) | 17
    u = mfo.uniforms(seed, it, ev, 5)
    for j in range(3):
        o = [int(t) for t in mfo.philox4x32_10([17, 3, j, it], [seed & 0xFFFFFFFF, seed >> 32])]
        X0, X1 = (o[1] << 32) | o[0], (o[3] << 32) | o[2]
        assert u[2 * j] == ((X0 >> 12) + 0.5) * 2.0 ** -52
        if 2 * j + 1 < 5:
            assert u[2 * j + 1] == ((X1 >> 12) + 0.5) * 2.0 ** -52
    # chunk independence: the same (seed, iteration, event) always gives the same numbers
    assert np.array_equal(mfo.uniforms(seed, it, ev, 5)[:4], mfo.uniforms(seed, it, ev, 4))


# ---------------------------------------------------------------- P3  VEGAS map
def test_vegas_map_uniform_grid_is_identity(mfo):
    edges = np.tile(np.arange(51) / 50.0, (4, 1))
    rng = np.random.default_rng(0)
    for _ in range(200):
        u = rng.uniform(size=4)
        x, b, J = mfo.vegas_map(edges, u)
        assert np.allclose(x, u, rtol=0, atol=2e-16) and abs(J - 1) < 1e-13
        assert np.array_equal(b, np.floor(u * 50).astype(np.uint8))


def test_vegas_map_random_grid_integrates_one(mfo):
    rng = np.random.default_rng(1)
    edges = np.zeros((3, 51)); edges[:, 1:] = np.cumsum(rng.uniform(0.2, 3.0, size=(3, 50)), axis=1)
    edges /= edges[:, -1:]
    assert np.allclose(np.diff(edges, axis=1).sum(axis=1), 1.0)
    N = 20000; Js = np.zeros(N); g = np.zeros(N)
    for i in range(N):
        u = rng.uniform(size=3)
        x, b, J = mfo.vegas_map(edges, u)
        for j in range(3):
            assert edges[j, b[j]] <= x[j] <= edges[j, b[j] + 1]
        # J is the inverse of the sampling density: prod 1/(Nb * width of the bin holding x)
        k = [np.searchsorted(edges[j], x[j], side="right") - 1 for j in range(3)]
        assert np.isclose(J, np.prod([50 * (edges[j, k[j] + 1] - edges[j, k[j]]) for j in range(3)]), rtol=1e-13)
        Js[i] = J; g[i] = J * 8 * x[0] * x[1] * x[2]          # integral of 8xyz over the cube = 1
    assert abs(Js.mean() - 1) < 5 * Js.std() / math.sqrt(N)
    assert abs(g.mean() - 1) < 5 * g.std() / math.sqrt(N)


# ---------------------------------------------------------------- P4  refinement
def _bin_mass(edges_old, r, edges_new):
    """integral over each new bin of the piecewise-constant density r_k/width_k (independent check)"""
    cum = np.concatenate([[0], np.cumsum(r)]) / r.sum()
    return np.diff(np.interp(edges_new, edges_old, cum))


def test_refine_flat_histogram_is_fixed_point(mfo):
    rng = np.random.default_rng(2)
    e = np.zeros((2, 51)); e[:, 1:] = np.cumsum(rng.uniform(0.5, 2, size=(2, 50)), axis=1); e /= e[:, -1:]
    out = mfo.refine(e, np.ones((2, 50)), 1.5)
    assert np.allclose(out, e, rtol=0, atol=1e-15)
    out0 = mfo.refine(e, rng.uniform(0.1, 5, size=(2, 50)), 0.0)      # alpha = 0 => r = 1 => unchanged
    assert np.allclose(out0, e, rtol=0, atol=1e-15)
    outz = mfo.refine(e, np.zeros((2, 50)), 1.5)                      # empty histogram => unchanged
    assert np.array_equal(outz, e)


def test_refine_equalises_compressed_mass(mfo):
    rng = np.random.default_rng(3)
    e = np.tile(np.arange(51) / 50.0, (3, 1))
    H = rng.uniform(0, 1, size=(3, 50)) ** 4
    H[1] = 0; H[1, 17] = 2.5                                           # all weight in one bin
    out = mfo.refine(e, H, 1.5)
    assert np.all(out[:, 0] == 0) and np.all(out[:, -1] == 1) and np.all(np.diff(out, axis=1) > 0)
    for j in range(3):
        h = H[j]
        s = np.concatenate([[(h[0] + h[1]) / 2], (h[:-2] + h[1:-1] + h[2:]) / 3, [(h[-2] + h[-1]) / 2]])
        s = np.maximum(s / s.sum(), 1e-30)
        r = ((s - 1) / np.log(s)) ** 1.5
        assert np.allclose(_bin_mass(e[j], r, out[j]), 1 / 50, rtol=1e-10)
    # closed form for the one-bin case: three bins share s = 1/3, the rest sit at the floor
    r_hi = ((1 / 3 - 1) / math.log(1 / 3)) ** 1.5; r_lo = ((1e-30 - 1) / math.log(1e-30)) ** 1.5
    tot = 3 * r_hi + 47 * r_lo
    # new edge m = 25 lies inside old bin 17 (the middle one): cumulative mass before it = 16 r_lo + r_hi
    frac = (tot * 25 / 50 - (16 * r_lo + r_hi)) / r_hi
    assert np.isclose(out[1, 25], (17 + frac) / 50, rtol=1e-13)


# ---------------------------------------------------------------- P29 combination
def test_combine_inverse_variance(mfo):
    I = np.array([10.0, 11.0, 9.5, 10.2]); s = np.array([1.0, 0.5, 2.0, 0.25])
    w = 1 / s ** 2; mean = (w * I).sum() / w.sum()
    got = mfo.combine(I, s)
    assert np.isclose(got[0], mean, rtol=1e-14) and np.isclose(got[1], w.sum() ** -0.5, rtol=1e-14)
    assert np.isclose(got[2], (w * (I - mean) ** 2).sum() / 3, rtol=1e-13)
    assert mfo.combine([3.0], [0.1])[2] == 0.0
    assert np.isclose(mfo.combine([1.0, 3.0], [0.0, 1.0])[0], 2.0)       # a zero error => plain mean


# ---------------------------------------------------------------- O3 x map
def test_x_map_jacobian_and_range(mfo):
    s, smin = 13000.0 ** 2, 376.0 ** 2
    rng = np.random.default_rng(4)
    for _ in range(100):
        y0, y1 = rng.uniform(0.01, 0.99, size=2)
        x1, x2, shat, jx = mfo.x_map(y0, y1, s, smin)
        assert smin <= shat <= s and 0 < x1 <= 1 and 0 < x2 <= 1 and np.isclose(x1 * x2 * s, shat, rtol=1e-14)
        h = 1e-6                                                   # numerical Jacobian d(x1,x2)/d(y0,y1)
        a = np.array(mfo.x_map(y0 + h, y1, s, smin)[:2]) - np.array(mfo.x_map(y0 - h, y1, s, smin)[:2])
        b = np.array(mfo.x_map(y0, y1 + h, s, smin)[:2]) - np.array(mfo.x_map(y0, y1 - h, s, smin)[:2])
        det = abs(a[0] * b[1] - a[1] * b[0]) / (4 * h * h)
        assert np.isclose(det, jx, rtol=1e-6)
    # the map covers {x1 x2 >= tau0}: integral of 1 over that region = 1 - tau0 + tau0 ln tau0
    tau0 = smin / s; n = 200
    y = (np.arange(n) + 0.5) / n
    tot = np.mean([mfo.x_map(a, b, s, smin)[3] for a in y for b in y])
    assert np.isclose(tot, 1 - tau0 + tau0 * math.log(tau0), rtol=2e-3)


# ---------------------------------------------------------------- P5-P9 phase space
def test_two_body_closed_forms(mfo):
    r = mfo.phase_space(2, 700.0 ** 2, [0, 0], [0.685, 0.3])
    assert np.isclose(r["W0"] * r["Wm"], 1 / (8 * math.pi), rtol=1e-15) and r["xi"] == 1.0
    r = mfo.phase_space(2, 700.0 ** 2, [MT, MT], [0.685, 0.3])
    beta = math.sqrt(1 - 4 * MT * MT / 700.0 ** 2)
    assert np.isclose(r["xi"], beta, rtol=1e-14) and np.isclose(r["W0"] * r["Wm"], beta / (8 * math.pi), rtol=1e-13)
    ct, phi = 2 * 0.685 - 1, 2 * math.pi * 0.3; p = 350 * beta; st = math.sqrt(1 - ct * ct)
    assert np.allclose(r["k"][0], [350, p * st * math.cos(phi), p * st * math.sin(phi), p * ct], rtol=1e-13)
    assert np.allclose(r["k"][1][1:], -r["k"][0][1:], rtol=1e-13)


def test_w0_formula(mfo):
    assert np.isclose(mfo.w0(2, 123.0), 1 / (8 * math.pi), rtol=1e-15)
    assert np.isclose(mfo.w0(3, 1e6), 1e6 / (256 * math.pi ** 3), rtol=1e-14)
    assert np.isclose(mfo.w0(4, 1e6), 1e12 / (24576 * math.pi ** 5), rtol=1e-14)   # shat^2/(2^13 3 pi^5)


def test_golden_phase_space_points(mfo):
    g = {k: np.array([float(t) for t in v]) for k, v in read_golden("points.txt").items()}
    r = mfo.phase_space(3, 1000.0 ** 2, [MT, MT, 0], g["G2_rs"])
    assert np.isclose(r["Mint"][1], g["G2_M2"][0], rtol=1e-13)
    for i in range(3):
        assert np.allclose(r["p0"][i], g["G2_p%d" % (i + 1)], rtol=1e-12, atol=1e-11)
        assert np.allclose(r["k"][i], g["G2_k%d" % (i + 1)], rtol=1e-12, atol=1e-11)
    assert np.isclose(r["xi"], g["G2_xi"][0], rtol=1e-14) and np.isclose(r["Wm"], g["G2_Wm"][0], rtol=1e-13)
    r = mfo.phase_space(4, 1500.0 ** 2, [MT, MT, 0, 0], g["G3_rs"])
    assert np.isclose(r["Mint"][1], g["G3_M2"][0], rtol=1e-13) and np.isclose(r["Mint"][2], g["G3_M3"][0], rtol=1e-13)
    for i in range(4):
        assert np.allclose(r["k"][i], g["G3_k%d" % (i + 1)], rtol=1e-12, atol=1e-11)
    assert np.isclose(r["xi"], g["G3_xi"][0], rtol=1e-14) and np.isclose(r["Wm"], g["G3_Wm"][0], rtol=1e-13)


@pytest.mark.parametrize("n", [3, 4])
def test_kinematics_conservation_and_flat_moments(mfo, n):
    rng = np.random.default_rng(10 + n); N = 20000; rts = 2000.0
    masses = [MT, MT] + [0.0] * (n - 2)
    s12 = np.zeros(N); cz = np.zeros((N, n)); e2 = np.zeros(N)
    for i in range(N):
        r = mfo.phase_space(n, rts ** 2, masses, rng.uniform(size=3 * n - 4))
        for mom, ms in ((r["p0"], [0.0] * n), (r["k"], masses)):            # P8
            tot = mom.sum(axis=0)
            assert abs(tot[0] - rts) < 1e-9 and np.abs(tot[1:]).max() < 1e-9
            m2 = mom[:, 0] ** 2 - (mom[:, 1:] ** 2).sum(axis=1)
            assert np.allclose(m2, np.array(ms) ** 2, rtol=0, atol=1e-7)
        p = r["p0"]; q = p[0] + p[1]
        s12[i] = (q[0] ** 2 - (q[1:] ** 2).sum()) / rts ** 2
        cz[i] = p[:, 3] / p[:, 0]; e2[i] = (p[0, 0] / rts) ** 2
    err = lambda a: 5 * a.std() / math.sqrt(N)
    exp1 = {3: 1 / 3, 4: 1 / 6}[n]                                            # P6: <s12/shat>
    assert abs(s12.mean() - exp1) < err(s12)
    if n == 3:
        assert abs((s12 ** 2).mean() - 1 / 6) < err(s12 ** 2)
        assert abs(e2.mean() - 1 / 8) < err(e2)       # x = 2E/rts has density 2x on (0,1): <E^2/shat> = <x^2>/4 = 1/8
    for j in range(n):                                                        # isotropy of every particle
        assert abs(cz[:, j].mean()) < err(cz[:, j]) and abs((cz[:, j] ** 2).mean() - 1 / 3) < err(cz[:, j] ** 2)


def test_massive_three_body_volume(mfo):
    g = read_golden("points.txt")
    rng = np.random.default_rng(5); N = 40000

    def phi2(s, a, b):
        lam = (s - (a + b) ** 2) * (s - (a - b) ** 2)
        return math.sqrt(max(lam, 0.0)) / (8 * math.pi * s)
    for rts in (400.0, 1000.0, 5000.0):
        s = rts * rts
        exact = integrate.quad(lambda M2: phi2(s, math.sqrt(M2), 0.0) * phi2(M2, MT, MT) / (2 * math.pi),
                               4 * MT * MT, s, epsabs=0, epsrel=1e-10)[0]
        assert np.isclose(exact, float(g["vol3_%d" % int(rts)][0]), rtol=2e-5)       # the survey's number
        w = np.zeros(N)
        for i in range(N):
            r = mfo.phase_space(3, s, [MT, MT, 0.0], rng.uniform(size=5)); w[i] = r["W0"] * r["Wm"]
        assert abs(w.mean() - exact) < 4.5 * w.std() / math.sqrt(N), (rts, w.mean(), exact)


# ---------------------------------------------------------------- P10 PDF
def test_pdf_interpolation_properties(mfo):
    xf = W.synthetic_gluon_grid(); a = (W.PDF_XMIN, W.PDF_XMAX, W.PDF_QMIN, W.PDF_QMAX)
    lx = np.linspace(math.log(1e-6), 0.0, 100); lq = np.linspace(0.0, math.log(1e8), 50)
    for ix in (0, 1, 37, 98, 99):                      # knots reproduced
        for iq in (0, 1, 20, 49):
            v = mfo.pdf_interp(xf, *a, math.exp(lx[ix]), math.exp(lq[iq]))
            assert np.isclose(v, xf[ix, iq], rtol=1e-12, atol=1e-15)
    rng = np.random.default_rng(6)
    for _ in range(200):                               # Q-independent table => Q-independent value (to rounding)
        x = math.exp(rng.uniform(math.log(7e-4), 0)); q2a, q2b = np.exp(rng.uniform(0, math.log(1e8), size=2))
        assert np.isclose(mfo.pdf_interp(xf, *a, x, q2a), mfo.pdf_interp(xf, *a, x, q2b), rtol=1e-15, atol=0)
        if x < 0.5:                                    # close to the tabulated formula away from x -> 1
            assert abs(mfo.pdf_interp(xf, *a, x, q2a) / (3 * (1 - x) ** 5 * x ** -0.1) - 1) < 6.5e-4
    # exact for a product of quadratics in (ln x, ln Q^2) away from the edges
    X, Q = np.meshgrid(lx, lq, indexing="ij")
    quad = (1 + 0.3 * X + 0.02 * X * X) * (2 - 0.1 * Q + 0.005 * Q * Q)
    for _ in range(200):
        zx = rng.uniform(lx[1], lx[-2]); zq = rng.uniform(lq[1], lq[-2])
        want = (1 + 0.3 * zx + 0.02 * zx * zx) * (2 - 0.1 * zq + 0.005 * zq * zq)
        assert np.isclose(mfo.pdf_interp(quad, *a, math.exp(zx), math.exp(zq)), want, rtol=5e-14)


def test_pdf_matches_library_hermite_spline(mfo):
    """Same rule through scipy's CubicHermiteSpline (library routine as a step), Q-dependent table."""
    t = W.q_dependent_test_grid(); nx, nq = t.shape
    a = (1e-4, 1.0, 2.0, 500.0)
    lx = np.linspace(math.log(a[0]), math.log(a[1]), nx); lq = np.linspace(math.log(a[2] ** 2), math.log(a[3] ** 2), nq)

    def slopes(z, f):
        sec = np.diff(f) / np.diff(z)
        return np.concatenate([[sec[0]], 0.5 * (sec[1:] + sec[:-1]), [sec[-1]]])
    rng = np.random.default_rng(7)
    for _ in range(300):
        zx = rng.uniform(lx[0], lx[-1]); zq = rng.uniform(lq[0], lq[-1])
        rows = np.array([interpolate.CubicHermiteSpline(lx, t[:, q], slopes(lx, t[:, q]))(zx) for q in range(nq)])
        want = interpolate.CubicHermiteSpline(lq, rows, slopes(lq, rows))(zq)
        got = mfo.pdf_interp(t, *a, math.exp(zx), math.exp(zq))
        assert np.isclose(got, want, rtol=1e-11), (zx, zq)


# ---------------------------------------------------------------- P25 cuts
def test_cuts_against_explicit_lab_boost(mfo):
    rng = np.random.default_rng(8)
    for _ in range(500):
        x1, x2 = np.exp(rng.uniform(math.log(1e-3), 0, size=2))
        kg = np.zeros((2, 4))
        for i in range(2):
            p = rng.uniform(10, 400); ct = rng.uniform(-0.999, 0.999); ph = rng.uniform(-math.pi, math.pi); st = math.sqrt(1 - ct * ct)
            kg[i] = [p, p * st * math.cos(ph), p * st * math.sin(ph), p * ct]
        ok, obs = mfo.cuts(kg, x1, x2, 30.0, 2.5, 0.4)
        # boost to the lab frame with beta = (x1-x2)/(x1+x2), then textbook definitions
        b = (x1 - x2) / (x1 + x2); ga = 1 / math.sqrt(1 - b * b)
        lab = kg.copy(); lab[:, 0] = ga * (kg[:, 0] + b * kg[:, 3]); lab[:, 3] = ga * (kg[:, 3] + b * kg[:, 0])
        pt = np.hypot(lab[:, 1], lab[:, 2]); pabs = np.sqrt((lab[:, 1:] ** 2).sum(axis=1))
        eta = 0.5 * np.log((pabs + lab[:, 3]) / (pabs - lab[:, 3])); phi = np.arctan2(lab[:, 2], lab[:, 1])
        dphi = abs(phi[0] - phi[1]); dphi = min(dphi, 2 * math.pi - dphi)
        dr = math.hypot(eta[0] - eta[1], dphi)
        assert np.allclose(obs[[0, 2]], pt, rtol=1e-12) and np.allclose(obs[[1, 3]], eta, rtol=1e-9, atol=1e-11)
        assert np.isclose(obs[4], dr, rtol=1e-9)
        assert ok == bool(np.all(pt > 30) and np.all(np.abs(eta) < 2.5) and dr > 0.4)
    ok, _ = mfo.cuts(kg[:1], 0.1, 0.1, 0.0, 0.0, 0.0)       # disabled cuts always pass
    assert ok


# ---- observable histograms ("histogram accumulation") ----------------------
def test_observable_hist_config0_matches_closed_form_dsigma_dpt(mfo):
    """e+e- -> mu+mu-: pT = (sqrt(s)/2) sin(theta) and dsigma/dcos = (3 sigma/8)(1 + cos^2), so the cross
    section with pT in [a, b) is 2 (3 sigma/8) [c + c^3/3] between c(b) and c(a), c(pT) = sqrt(1 - (2 pT/sqrt s)^2)"""
    cfg = W.config(0, seed=0)
    orc = mfo.Vegas(cfg)
    n, nb, lo, hi = 200_000, 10, 0.0, 50.0
    (s1, s2), = orc.observable_hist(0, 0, n, n, [(0, nb, lo, hi)], n_threads=mfo.max_threads())
    sigma = 4 * math.pi * cfg["alpha_em"] ** 2 / (3 * cfg["sqrt_s"] ** 2) * cfg["gev2_to_pb"]
    c = lambda pt: math.sqrt(max(0.0, 1 - (2 * pt / cfg["sqrt_s"]) ** 2))
    prim = lambda x: x + x ** 3 / 3
    edges = np.linspace(lo, hi, nb + 1)
    exact = np.array([2 * (3 * sigma / 8) * (prim(c(a)) - prim(c(b))) for a, b in zip(edges[:-1], edges[1:])])
    err = np.sqrt(np.maximum(s2[:nb] * n - s1[:nb] ** 2, 0) / (n - 1))      # per-bin MC error of sum t
    assert s1[nb] == 0 and s1[nb + 1] == 0                                   # pT never leaves [0, sqrt(s)/2)
    assert (np.abs(s1[:nb] - exact) < 5 * err + 1e-12).all(), (s1[:nb], exact, err)
    acc, _ = orc.accumulate(0, 0, n, n, n_threads=mfo.max_threads())
    assert abs(s1.sum() / acc[0] - 1) < 1e-12 and abs(s2.sum() / acc[1] - 1) < 1e-12   # every event lands in one slot


def test_observable_hist_definitions_against_numpy(mfo):
    """all four kinds, under/overflow slots, on gg -> tt~g: rebuilt in NumPy from the per-event records"""
    cfg = W.config(W.GG_TTG, seed=4)
    orc = mfo.Vegas(cfg)
    n = 4000
    obs = [(0, 7, 20.0, 300.0), (1, 5, 0.0, 150.0), (2, 9, 400.0, 2000.0), (3, 6, 30.0, 200.0)]
    got = orc.observable_hist(1, 100, n, n, obs, n_threads=mfo.max_threads())
    ev = orc.eval(1, 100, n, n_threads=mfo.max_threads())
    k = ev["momenta"][:, 2:]
    tot = k[:, 0] + k[:, 1]
    vals = [np.hypot(k[:, 0, 1], k[:, 0, 2]), np.hypot(k[:, 1, 1], k[:, 1, 2]),
            np.sqrt(tot[:, 0] ** 2 - (tot[:, 1:] ** 2).sum(1)), np.hypot(k[:, 2, 1], k[:, 2, 2])]
    t = ev["weight"] / n
    for (kind, nb, lo, hi), v, (s1, s2) in zip(obs, vals, got):
        b = np.floor((v - lo) / (hi - lo) * nb).astype(int)
        b = np.where(v < lo, nb, np.where(v >= hi, nb + 1, np.minimum(b, nb - 1)))
        ref1 = np.bincount(b, weights=t, minlength=nb + 2); ref2 = np.bincount(b, weights=t * t, minlength=nb + 2)
        np.testing.assert_allclose(s1, ref1, rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(s2, ref2, rtol=1e-12, atol=1e-300)
        assert s1[nb] > 0 or s1[nb + 1] > 0 or kind == 3                     # the ranges above cut into the spectra
