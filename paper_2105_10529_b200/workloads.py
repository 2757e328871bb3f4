"""Seeded, synthetic workload definitions (BASELINE.json configs 0-4) shared by the product's
tests/bench and by the oracle's tests.  Holds NONE of the method's arithmetic: only the run
parameters the configs state and the tabulated input PDF grid (input data).
"""
import numpy as np

EE_MUMU, GG_TT, GG_TTG, GG_TTGG = 0, 1, 2, 3
QQ_TT = 4                                      # q q~ -> t t~ summed over five light flavours
PP_TT = 5                                      # p p -> t t~ at LO: g g -> t t~ and q q~ -> t t~ in one integrand
QQ_TTG = 6                                     # p p -> t t~ g through q q~ -> t t~ g (both beam orientations, five flavours)
QG_TTQ = 7                                     # p p -> t t~ + quark jet through q g, g q, q~ g, g q~ -> t t~ q
PROCESS_NAMES = {EE_MUMU: "ee_mumu", GG_TT: "gg_tt", GG_TTG: "gg_ttg", GG_TTGG: "gg_ttgg", QQ_TT: "qq_tt", PP_TT: "pp_tt",
                 QQ_TTG: "qq_ttg", QG_TTQ: "qg_ttq"}
PDF_NF = 11                                    # flavour tables of the 11-flavour grid, index = PDG id + 5 (b~ .. g .. b)

GEN_CLASSIC_RAMBO, GEN_LINEAR_TAU = 1, 2      # `generator` flags; 0 = the generators of the configs

PDF_NX, PDF_NQ = 100, 50
PDF_XMIN, PDF_XMAX, PDF_QMIN, PDF_QMAX = 1e-6, 1.0, 1.0, 1e4


def synthetic_gluon_grid(nx=PDF_NX, nq=PDF_NQ, xmin=PDF_XMIN, xmax=PDF_XMAX):
    """Input table x*g(x) = 3 (1-x)^5 x^-0.1 on nx knots uniform in ln x, repeated at every Q^2 knot
    (config 1 text; reading A9).  The last row (x = 1) is exactly 0.  Row-major [ix][iq]."""
    lx = np.linspace(np.log(xmin), np.log(xmax), nx)
    x = np.exp(lx)
    x[-1] = xmax
    xf = 3.0 * (1.0 - x) ** 5 * x ** (-0.1)
    xf[-1] = 0.0 if xmax == 1.0 else xf[-1]
    return np.ascontiguousarray(np.repeat(xf[:, None], nq, axis=1))


def synthetic_flavour_grid(nx=PDF_NX, nq=PDF_NQ, xmin=PDF_XMIN, xmax=PDF_XMAX, qmin=PDF_QMIN, qmax=PDF_QMAX):
    """Input tables x*f_i(x, Q^2) of an 11-flavour synthetic proton, [11][ix][iq], flavour index =
    PDG id + 5 (0..4 = b~ c~ s~ u~ d~, 5 = g, 6..10 = d u s c b), same knots as the gluon grid.  Shapes: gluon as in
    synthetic_gluon_grid; sea x*S_i = k_i 0.2 (1-x)^7 x^-0.1 (1 + 0.04 ln(Q^2/Q0^2)), k = 1, 1, 0.5, 0.15, 0.05 for
    d, u, s, c, b; valence x*u_v = 2.2 x^0.5 (1-x)^3, x*d_v = 1.1 x^0.5 (1-x)^4 (Q-independent); q = valence + sea,
    q~ = sea.  The sea evolves with Q so that the Q direction of the interpolation is exercised.  x = 1 row: exactly 0."""
    lx = np.linspace(np.log(xmin), np.log(xmax), nx)
    x = np.exp(lx); x[-1] = xmax
    lq2 = np.linspace(np.log(qmin * qmin), np.log(qmax * qmax), nq)
    evo = 1.0 + 0.04 * (lq2 - lq2[0])
    sea = 0.2 * (1.0 - x) ** 7 * x ** (-0.1)
    g = np.zeros((PDF_NF, nx, nq))
    g[5] = synthetic_gluon_grid(nx, nq, xmin, xmax)
    kappa = {1: 1.0, 2: 1.0, 3: 0.5, 4: 0.15, 5: 0.05}
    val = {1: 1.1 * x ** 0.5 * (1.0 - x) ** 4, 2: 2.2 * x ** 0.5 * (1.0 - x) ** 3}
    for fl, k in kappa.items():
        s_ = k * sea[:, None] * evo[None, :]
        g[5 - fl] = s_
        g[5 + fl] = s_ + (val[fl][:, None] if fl in val else 0.0)
    if xmax == 1.0:
        g[:, -1, :] = 0.0
    return np.ascontiguousarray(g)


def q_dependent_test_grid(nx=24, nq=12):
    """A Q-dependent table used only by the interpolation tests (exercises the Q direction)."""
    rng = np.random.default_rng(1234)
    return np.ascontiguousarray(rng.uniform(0.1, 2.0, size=(nx, nq)))


def config(process, seed=0, **over):
    """Run parameters of BASELINE.json's configs (process 0..3), and of the quark channel (process 4)."""
    c = dict(process=process, precision=64, device=0, seed=seed, n_bins=50, alpha_damp=1.5,
             sqrt_s=13000.0, m_top=173.0, alpha_s=0.118, alpha_em=1.0 / 132.5, mu_f=173.0,
             ptmin_g=0.0, etamax_g=0.0, drmin_gg=0.0, gev2_to_pb=0.3894e9,
             pdf_xf=synthetic_gluon_grid(), pdf_xmin=PDF_XMIN, pdf_xmax=PDF_XMAX,
             pdf_qmin=PDF_QMIN, pdf_qmax=PDF_QMAX, generator=0)
    if process == EE_MUMU:
        c.update(sqrt_s=100.0, pdf_xf=None)
    if process in (QQ_TT, PP_TT, QQ_TTG, QG_TTQ):
        c.update(pdf_xf=synthetic_flavour_grid())
    if process in (GG_TTG, GG_TTGG, QQ_TTG, QG_TTQ):      # cuts of config 2 on the third final particle (gluon / light-quark jet)
        c.update(ptmin_g=30.0, etamax_g=2.5)
    if process == GG_TTGG:
        c.update(drmin_gg=0.4)
    c.update(over)
    return c


# (process, iterations, events per iteration, seed) of configs 0..3; config 4 is a sweep of config 2
CONFIGS = [
    dict(process=EE_MUMU, n_iter=3, n_events=100_000, seed=0),
    dict(process=GG_TT, n_iter=5, n_events=1_000_000, seed=0),
    dict(process=GG_TTG, n_iter=5, n_events=10_000_000, seed=0),
    dict(process=GG_TTGG, n_iter=5, n_events=1_000_000, seed=0),
]
SWEEP = dict(process=GG_TTG, seed=1, n_iter=1, sizes=[10_000, 100_000, 1_000_000, 10_000_000, 100_000_000])
