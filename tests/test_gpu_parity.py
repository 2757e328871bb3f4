"""GPU parity tests proper: the CUDA path, called through the C-ABI (ctypes binding), against the
oracle element by element on the same seeded inputs.  Tolerances (BASELINE.json north_star):
1e-10 relative per event and on the integrals in fp64; integer work (bins, pass flags) bit-exact."""
import numpy as np
import pytest

from paper_2105_10529_b200 import workloads as W

pytestmark = pytest.mark.gpu
RTOL_EVENT = 1e-10
RTOL_INT = 1e-10


@pytest.fixture(scope="module")
def mf():
    import torch
    assert torch.cuda.is_available()
    from paper_2105_10529_b200 import binding
    binding.lib()
    return binding


def random_grid(d, nb, seed):
    rng = np.random.default_rng(seed)
    w = rng.uniform(0.3, 1.7, size=(d, nb))
    e = np.concatenate([np.zeros((d, 1)), np.cumsum(w, axis=1) / w.sum(axis=1, keepdims=True)], axis=1)
    e[:, -1] = 1.0
    return e


def compare_events(out, ref, proc, mom_tol=(1e-11, 1e-9), lumi_abs=0.0):
    g = {k: v.cpu().numpy() for k, v in out.items()}
    assert (g["bins"] == ref["bins"]).all()
    assert (g["pass_"] == ref["pass_"]).all()
    np.testing.assert_allclose(g["x"], ref["x"], rtol=1e-14, atol=0)
    np.testing.assert_allclose(g["momenta"], ref["momenta"], rtol=mom_tol[0], atol=mom_tol[1])
    if proc:
        np.testing.assert_allclose(g["pdf"], ref["pdf"], rtol=1e-12, atol=1e-15)
    nz = ref["weight"] != 0
    assert (g["weight"][~nz] == 0).all()
    rel_w = np.abs(g["weight"][nz] / ref["weight"][nz] - 1)
    rel_m = np.abs(g["me2"][nz] / ref["me2"][nz] - 1)
    # (process 5 records the luminosity-weighted mean of two |M|^2: it inherits the absolute error of the luminosities)
    tol_m = RTOL_EVENT + (lumi_abs / np.abs(ref["pdf"][nz].sum(axis=1)) if lumi_abs else 0.0)
    assert (rel_m < tol_m).all(), (rel_m / tol_m).max()
    # the weight carries xf(x1) xf(x2); where the interpolant crosses zero (x -> 1)
    # its absolute rounding error (1e-15, the bound used on the PDF values above) sets the relative one
    tol_w = np.full(int(nz.sum()), RTOL_EVENT)
    if proc:
        tol_w = tol_w + (1e-15 / np.abs(ref["pdf"][nz])).sum(axis=1)
    if lumi_abs:            # quark channel: the weight carries the SUM of the two flavour sums, each good to lumi_abs absolutely
        tol_w = tol_w + lumi_abs / np.abs(ref["pdf"][nz].sum(axis=1))
    assert (rel_w < tol_w).all(), (rel_w / tol_w).max()


# sizes span several 128-thread tiles and a ragged tail; iteration/first_event exercise the counter
@pytest.mark.parametrize("proc,n", [(0, 5003), (1, 5003), (2, 3001), (3, 333)])
def test_per_event_parity_uniform_and_adapted_grid(mf, mfo, proc, n):
    cfg = W.config(proc, seed=W.CONFIGS[proc]["seed"])
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    ref = orc.eval(0, 0, n, n_threads=mfo.max_threads())
    compare_events(gpu.integrand_eval(0, 0, n, debug=True), ref, proc)
    e = random_grid(orc.d, 50, 100 + proc)
    gpu.set_grid(e); orc.set_grid(e)
    np.testing.assert_array_equal(gpu.get_grid(), e)
    ref = orc.eval(3, 2**33 + 17, n, n_threads=mfo.max_threads())
    compare_events(gpu.integrand_eval(3, 2**33 + 17, n, debug=True), ref, proc)


def test_chunking_invariance(mf):
    """event indices are global: one call == concatenated chunks, bit for bit"""
    cfg = W.config(W.GG_TTG, seed=1)
    gpu = mf.Vegas(cfg)
    a = gpu.integrand_eval(0, 0, 10000)["weight"].cpu().numpy()
    b = np.concatenate([gpu.integrand_eval(0, s, m)["weight"].cpu().numpy() for s, m in ((0, 1), (1, 4095), (4096, 5904))])
    assert (a == b).all()


@pytest.mark.parametrize("proc,n_iter,n", [(0, 3, 100_000), (1, 3, 40_000), (2, 2, 20_000), (3, 2, 1_500)])
def test_iteration_parity(mf, mfo, proc, n_iter, n):
    """fused kernel + finalize vs the oracle: I, sigma, raw sums, histogram, refined grid, counters"""
    cfg = W.config(proc, seed=W.CONFIGS[proc]["seed"])
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    for it in range(n_iter):
        g = gpu.vegas_iterate(n)
        o = orc.iterate(n, n_threads=mfo.max_threads())
        assert g["n_events"] == n and g["n_pass"] == o["n_pass"] and g["n_nonfinite"] == 0 == o["n_nonfinite"]
        assert abs(g["integral"] / o["integral"] - 1) < RTOL_INT
        assert abs(g["sigma"] / o["sigma"] - 1) < 1e-8          # sigma^2 = N S2 - I^2 cancels ~2 digits
        acc, cnt = gpu.get_accum()
        np.testing.assert_allclose(acc, orc.get_accum(), rtol=RTOL_INT, atol=1e-300)
        np.testing.assert_allclose(gpu.get_grid(), orc.get_grid(), rtol=0, atol=1e-11)
        gpu.set_grid(orc.get_grid())          # keep the two in lock-step for the next iteration
    rg, ro = gpu.result(), orc.result()
    assert rg["n_iter"] == n_iter
    for k in ("integral", "sigma"):
        assert abs(rg[k] / ro[k] - 1) < 1e-8
    assert abs(rg["chi2_dof"] - ro["chi2_dof"]) < 1e-6 * max(1.0, ro["chi2_dof"])


def test_config0_cross_section(mf):
    """config 0 end to end on the GPU: sigma = 4 pi alpha^2/(3s) K = 9.290793339943443 pb"""
    c = W.CONFIGS[0]
    gpu = mf.Vegas(W.config(0, seed=c["seed"]))
    for _ in range(c["n_iter"]):
        gpu.vegas_iterate(c["n_events"])
    r = gpu.result()
    assert abs(r["integral"] - 9.290793339943443) < 5 * r["sigma"] and r["sigma"] < 2e-3


def test_config1_cross_section_and_closed_form(mf):
    """config 1 at full size: per-event |M|^2 vs the closed form of gg -> tt~ (sampled), sigma vs quadrature"""
    c = W.CONFIGS[1]
    cfg = W.config(1, seed=c["seed"])
    gpu = mf.Vegas(cfg)
    out = gpu.integrand_eval(0, 0, 20000, debug=True)
    mom = out["momenta"].cpu().numpy(); me2 = out["me2"].cpu().numpy()
    shat = 4 * mom[:, 0, 0] ** 2
    dot = lambda a, b: a[:, 0] * b[:, 0] - (a[:, 1:] * b[:, 1:]).sum(1)
    t1 = 2 * dot(mom[:, 0], mom[:, 2]) / shat; t2 = 2 * dot(mom[:, 1], mom[:, 2]) / shat
    rho = 4 * cfg["m_top"] ** 2 / shat
    gs4 = (4 * np.pi * cfg["alpha_s"]) ** 2
    closed = gs4 * (1 / (6 * t1 * t2) - 3.0 / 8) * (t1 ** 2 + t2 ** 2 + rho - rho ** 2 / (4 * t1 * t2))
    assert np.abs(me2 / closed - 1).max() < 1e-10
    for _ in range(c["n_iter"]):
        gpu.vegas_iterate(c["n_events"])
    r = gpu.result()
    assert abs(r["integral"] - 1074.393) < 5 * r["sigma"] + 0.02 and r["sigma"] < 0.5


def test_full_size_launch_sampled_parity(mf, mfo):
    """gg->tt~g at BASELINE's 1e7 events in the launch configuration bench.py times: integrals of
    the fused kernel == sums of the eval kernel's weights; sampled events == oracle"""
    import torch
    cfg = W.config(W.GG_TTG, seed=0)
    n = 10_000_000
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    g = gpu.vegas_iterate(n)
    acc, cnt = gpu.get_accum()
    gpu2 = mf.Vegas(cfg)
    w = gpu2.integrand_eval(0, 0, n)["weight"]
    t = w / n
    assert abs(float(t.sum()) / acc[0] - 1) < 1e-10 and abs(float((t * t).sum()) / acc[1] - 1) < 1e-10
    assert int((w != 0).sum()) <= cnt[0] <= n and g["n_nonfinite"] == 0
    idx = [0, 1, 127, 128, 4097, 999_999, 5_000_001, n - 1]
    for i in idx:
        ref = orc.eval(0, i, 1)["weight"][0]
        got = float(w[i])
        assert (ref == 0 and got == 0) or abs(got / ref - 1) < RTOL_EVENT


@pytest.mark.parametrize("proc,n", [(2, 70_001)])
def test_staged_path_equals_fused_path(mf, proc, n):
    """the staged iteration (front end -> |M|^2 -> reductions through HBM records) and the fused kernel
    evaluate the same events: equal counters, sums equal to summation order, same refined grid"""
    cfg = W.config(proc, seed=2)
    a, b = mf.Vegas(cfg), mf.Vegas(cfg)
    b.set_path(False)
    for _ in range(2):
        ia, ib = a.vegas_iterate(n), b.vegas_iterate(n)
        assert ia["n_pass"] == ib["n_pass"] and ia["n_nonfinite"] == 0 == ib["n_nonfinite"]
        np.testing.assert_allclose(a.get_accum()[0], b.get_accum()[0], rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(a.get_grid(), b.get_grid(), rtol=0, atol=1e-13)
    st = a.last_stage_ms()
    assert st["front"] > 0 and st["me"] > 0 and st["reduce"] > 0
    with pytest.raises(mf.MfError) as e:
        mf.Vegas(W.config(W.GG_TT)).set_path(True)
    assert e.value.code == mf.MF_EUNSUPPORTED
    with pytest.raises(mf.MfError) as e:                      # gg -> tt~gg: staged path only (four lanes per event)
        mf.Vegas(W.config(W.GG_TTGG)).set_path(False)
    assert e.value.code == mf.MF_EUNSUPPORTED


def test_staged_path_slices_large_iterations(mf):
    """more than 2^24 events per iteration: the staged path runs in slices that reuse the workspace;
    raw sums == sums of the eval kernel's per-event weights"""
    cfg = W.config(W.GG_TTG, seed=1)
    n = (1 << 24) + 12_345
    gpu = mf.Vegas(cfg)
    g = gpu.vegas_iterate(n)
    acc, cnt = gpu.get_accum()
    w = mf.Vegas(cfg).integrand_eval(0, 0, n)["weight"]
    t = w / n
    assert abs(float(t.sum()) / acc[0] - 1) < 1e-10 and abs(float((t * t).sum()) / acc[1] - 1) < 1e-10
    assert int((w != 0).sum()) <= cnt[0] <= n and g["n_events"] == n


@pytest.mark.parametrize("proc,n", [(0, 60_000), (1, 30_000), (2, 20_000), (3, 1_500)])
def test_observable_histograms_match_oracle(mf, mfo, proc, n):
    """observable histograms filled in the same pass ("histogram accumulation"): two iterations
    against the oracle's plain definition on the same grids; slots incl. under/overflow to 1e-10"""
    cfg = W.config(proc, seed=W.CONFIGS[proc]["seed"])
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    obs = [(0, 12, 0.0, 45.0), (2, 5, 99.0, 101.0)] if proc == 0 else \
          [(0, 20, 0.0, 400.0), (1, 7, 10.0, 250.0), (2, 16, 350.0, 1500.0)] + ([(3, 10, 30.0, 230.0)] if proc >= 2 else [])
    gpu.set_observables(obs)
    assert gpu.accum_len() == 2 + gpu.d * gpu.n_bins + 2 * 4 * 64
    ref = [(np.zeros(o[1] + 2), np.zeros(o[1] + 2)) for o in obs]
    for it in range(2):
        for (a, b), (r1, r2) in zip(orc.observable_hist(it, 0, n, n, obs, n_threads=mfo.max_threads()), ref):
            r1 += a; r2 += b
        g = gpu.vegas_iterate(n)
        o = orc.iterate(n, n_threads=mfo.max_threads())
        assert abs(g["integral"] / o["integral"] - 1) < RTOL_INT
        gpu.set_grid(orc.get_grid())
    got, n_it = gpu.get_observables()
    assert n_it == 2
    for (g1, g2), (r1, r2), ob in zip(got, ref, obs):
        scale1, scale2 = np.abs(r1).max(), np.abs(r2).max()
        np.testing.assert_allclose(g1, r1, rtol=1e-10, atol=1e-13 * scale1)
        np.testing.assert_allclose(g2, r2, rtol=1e-10, atol=1e-13 * scale2)
    tot = sum(it["integral"] for it in gpu.get_iterations())
    assert abs(got[0][0].sum() / tot - 1) < 1e-12            # every weighted event lands in exactly one slot
    gpu.set_observables([])                                   # off again: plain record length
    assert gpu.accum_len() == 2 + gpu.d * gpu.n_bins
    if proc >= 2:                                             # heavy processes: observables on the staged path only
        gpu.set_observables(obs)
        with pytest.raises(mf.MfError) as e:
            gpu.set_path(False)                               # (gg -> tt~gg has no fused path at all)
            gpu.vegas_iterate(1000)
        assert e.value.code == mf.MF_EUNSUPPORTED


def test_fp32_matrix_element_variant(mf, mfo):
    """precision = 32 (gg -> tt~g only): |M|^2 in fp32, everything else fp64, so the events, bins and cut
    decisions are those of the fp64 path.  north_star: 1e-4 relative per event for the optional fp32 path;
    gauge cancellations push a small fraction of the events beyond it -- the fraction is bounded here"""
    cfg32 = W.config(W.GG_TTG, seed=1, precision=32)
    gpu, orc = mf.Vegas(cfg32), mfo.Vegas(W.config(W.GG_TTG, seed=1))
    n = 20_000
    out = gpu.integrand_eval(0, 0, n, debug=True)
    ref = orc.eval(0, 0, n, n_threads=mfo.max_threads())
    assert (out["bins"].cpu().numpy() == ref["bins"]).all() and (out["pass_"].cpu().numpy() == ref["pass_"]).all()
    np.testing.assert_allclose(out["momenta"].cpu().numpy(), ref["momenta"], rtol=1e-11, atol=1e-9)   # front end is fp64
    w = out["weight"].cpu().numpy()
    nz = ref["weight"] != 0
    rel = np.abs(w[nz] / ref["weight"][nz] - 1)
    assert (w[~nz] == 0).all()
    assert np.median(rel) < 2e-6 and np.quantile(rel, 0.99) < 1e-4 and (rel > 1e-4).mean() < 2e-3 and rel.max() < 1e-2, \
        (np.median(rel), np.quantile(rel, 0.99), (rel > 1e-4).mean(), rel.max())
    g64 = mf.Vegas(W.config(W.GG_TTG, seed=1))
    a, b = g64.vegas_iterate(200_000), gpu.vegas_iterate(200_000)
    assert a["n_pass"] == b["n_pass"] and abs(b["integral"] / a["integral"] - 1) < 1e-6
    np.testing.assert_allclose(gpu.get_grid(), g64.get_grid(), rtol=0, atol=5e-6)          # fp32 weights move the edges ~2e-7
    with pytest.raises(mf.MfError) as e:
        gpu.set_path(False)                                   # the fp32 variant exists on the staged path only
    assert e.value.code == mf.MF_EUNSUPPORTED
    for proc in (0, 1, 3):
        with pytest.raises(mf.MfError) as e:
            mf.Vegas(W.config(proc, precision=32))
        assert e.value.code == mf.MF_EUNSUPPORTED


def test_config3_full_size_launch_and_config2_cross_section(mf, mfo):
    """config 3 at its full size (1e6 events per iteration, staged path): raw sums == sums of the eval kernel's
    weights, sampled events == oracle.  Config 2 at its full size (5 x 1e7): the cross section agrees with the
    oracle-side determinations (VEGAS 1054.3 +- 6.6 pb, classic RAMBO 1047 +- 28 pb: tests/test_oracle_crosscheck.py)"""
    cfg = W.config(W.GG_TTGG, seed=0)
    n = W.CONFIGS[3]["n_events"]
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    g = gpu.vegas_iterate(n)
    acc, cnt = gpu.get_accum()
    w = mf.Vegas(cfg).integrand_eval(0, 0, n)["weight"]
    t = w / n
    assert abs(float(t.sum()) / acc[0] - 1) < 1e-10 and abs(float((t * t).sum()) / acc[1] - 1) < 1e-10
    assert int((w != 0).sum()) <= cnt[0] <= n and g["n_nonfinite"] == 0
    for i in (0, 255, 256, 77_777, n - 1):
        ref = orc.eval(0, i, 1)["weight"][0]
        got = float(w[i])
        assert (ref == 0 and got == 0) or abs(got / ref - 1) < RTOL_EVENT
    c = W.CONFIGS[2]
    gpu = mf.Vegas(W.config(W.GG_TTG, seed=c["seed"]))
    for _ in range(c["n_iter"]):
        gpu.vegas_iterate(c["n_events"])
    r = gpu.result()
    assert r["n_iter"] == c["n_iter"] and r["sigma"] < 0.5 and abs(r["integral"] - 1054.3) < 4 * 6.6 and r["chi2_dof"] < 5


def test_sharded_accumulate_equals_iterate(mf):
    """mf_vegas_accumulate over two event ranges + finalize == mf_vegas_iterate (to summation order)"""
    cfg = W.config(W.GG_TT, seed=5)
    n = 50_000
    a, b = mf.Vegas(cfg), mf.Vegas(cfg)
    ia = a.vegas_iterate(n)
    acc0 = np.zeros(2 + b.d * b.n_bins); b.set_accum(acc0, np.zeros(2, np.uint64))
    b.vegas_accumulate(0, 20_000, n); b.vegas_accumulate(20_000, 30_000, n)
    ib = b.vegas_finalize(n)
    assert abs(ia["integral"] / ib["integral"] - 1) < 1e-13 and ia["n_pass"] == ib["n_pass"]
    np.testing.assert_allclose(a.get_grid(), b.get_grid(), rtol=0, atol=1e-13)


def test_staged_path_edge_cases(mf, mfo):
    """staged path: minimum iteration, fewer events than one CTA, no event passing the cuts (empty record
    set: zero integral, grid kept), one passing event per region at most"""
    cfg = W.config(W.GG_TTG, seed=9)
    for n in (2, 3, 255, 257):
        gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
        g, o = gpu.vegas_iterate(n), orc.iterate(n)
        assert g["n_pass"] == o["n_pass"] and g["n_events"] == n
        assert (o["integral"] == 0 and g["integral"] == 0) or abs(g["integral"] / o["integral"] - 1) < RTOL_INT
        np.testing.assert_allclose(gpu.get_grid(), orc.get_grid(), rtol=0, atol=1e-11)
    none = dict(cfg); none["etamax_g"] = 1e-9            # |eta| < 1e-9: nothing passes
    gpu = mf.Vegas(none)
    before = gpu.get_grid()
    g = gpu.vegas_iterate(5000)
    assert g["n_pass"] == 0 and g["integral"] == 0.0 and g["sigma"] == 0.0 and g["n_nonfinite"] == 0
    np.testing.assert_array_equal(gpu.get_grid(), before)
    g = gpu.vegas_iterate(5000)                           # and again (workspace reuse with empty records)
    assert g["n_pass"] == 0 and gpu.result()["n_iter"] == 2


def test_errors_and_edge_cases(mf):
    cfg = W.config(W.GG_TT)
    gpu = mf.Vegas(cfg)
    with pytest.raises(mf.MfError) as e:
        gpu.result()
    assert e.value.code == mf.MF_ESTATE
    with pytest.raises(mf.MfError):
        gpu.vegas_iterate(1)
    out = gpu.integrand_eval(0, 0, 0)            # empty input
    assert out["weight"].numel() == 0
    one = gpu.integrand_eval(0, 5, 1)["weight"]  # single event (ragged warp)
    assert one.shape == (1,)
    bad = dict(cfg); bad["precision"] = 32
    with pytest.raises(mf.MfError) as e:
        mf.Vegas(bad)
    assert e.value.code == mf.MF_EUNSUPPORTED
    bad = dict(cfg); bad["sqrt_s"] = 300.0       # below threshold: kinematics outside the grid
    with pytest.raises(mf.MfError) as e:
        mf.Vegas(bad)
    assert e.value.code == mf.MF_EINVAL
    g = gpu.get_grid(); g[0, 3] = g[0, 2]
    with pytest.raises(mf.MfError):
        gpu.set_grid(g)
    gpu.vegas_iterate(2)                          # minimum iteration
    assert gpu.result()["n_iter"] == 1


# ---- selectable generators: classic 4n-random RAMBO (flag 1, d = 2 + 4 n_final) and linear tau (flag 2)
@pytest.mark.parametrize("proc,gen,n", [(1, 1, 5003), (1, 2, 5003), (1, 3, 5003), (2, 1, 3001), (2, 2, 3001), (2, 3, 3001),
                                        (3, 1, 333), (3, 2, 333), (3, 3, 333)])
def test_generator_variants_per_event_parity(mf, mfo, proc, gen, n):
    cfg = W.config(proc, seed=4, generator=gen)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    assert gpu.d == orc.d == (2 + 4 * orc.n_final if gen & W.GEN_CLASSIC_RAMBO else 3 * orc.n_final - 2)
    # the boost of the classic RAMBO (gamma = Q0/M of the generated system) amplifies the rounding of its inputs
    mom_tol = (1e-10, 1e-8) if gen & W.GEN_CLASSIC_RAMBO else (1e-11, 1e-9)
    ref = orc.eval(0, 0, n, n_threads=mfo.max_threads())
    compare_events(gpu.integrand_eval(0, 0, n, debug=True), ref, proc, mom_tol)
    e = random_grid(orc.d, 50, 200 + proc)
    gpu.set_grid(e); orc.set_grid(e)
    ref = orc.eval(2, 2**32 + 5, n, n_threads=mfo.max_threads())
    compare_events(gpu.integrand_eval(2, 2**32 + 5, n, debug=True), ref, proc, mom_tol)
    w = gpu.integrand_eval(2, 2**32 + 5, n)["weight"].cpu().numpy()      # weights-only call: same values
    nz = ref["weight"] != 0
    assert (w[~nz] == 0).all() and np.abs(w[nz] / ref["weight"][nz] - 1).max() < 2 * RTOL_EVENT


@pytest.mark.parametrize("proc,gen,n_iter,n", [(1, 1, 3, 40_000), (1, 2, 2, 40_000), (2, 1, 2, 20_000), (2, 3, 2, 20_000),
                                               (3, 1, 2, 1_500), (3, 2, 2, 1_500)])
def test_generator_variants_iteration_parity(mf, mfo, proc, gen, n_iter, n):
    """whole iterations with the variant generators (process 1: fused kernel with d = 10; processes 2, 3: staged
    path with d = 14 / 18, bins of dimensions 10.. in the second packed word) vs the oracle"""
    cfg = W.config(proc, seed=6, generator=gen)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    for it in range(n_iter):
        g = gpu.vegas_iterate(n)
        o = orc.iterate(n, n_threads=mfo.max_threads())
        assert g["n_events"] == n and g["n_pass"] == o["n_pass"] and g["n_nonfinite"] == 0 == o["n_nonfinite"]
        assert abs(g["integral"] / o["integral"] - 1) < RTOL_INT
        assert abs(g["sigma"] / o["sigma"] - 1) < 1e-8
        acc, cnt = gpu.get_accum()
        assert acc.shape == (2 + orc.d * 50,)
        np.testing.assert_allclose(acc, orc.get_accum(), rtol=RTOL_INT, atol=1e-300)
        np.testing.assert_allclose(gpu.get_grid(), orc.get_grid(), rtol=0, atol=1e-11)
        gpu.set_grid(orc.get_grid())
    rg, ro = gpu.result(), orc.result()
    assert rg["n_iter"] == n_iter and abs(rg["integral"] / ro["integral"] - 1) < 1e-8


def test_generator_variants_observables_errors_and_cross_section(mf, mfo):
    """observables through the d = 14 staged path; argument errors; and the physics check: config 1's cross section
    through every generator variant on the GPU (quadrature value 1074.39 pb, tests/test_oracle_generators.py)"""
    cfg = W.config(W.GG_TTG, seed=3, generator=W.GEN_CLASSIC_RAMBO)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    obs = [(0, 20, 0.0, 400.0), (3, 10, 30.0, 230.0)]
    gpu.set_observables(obs)
    n = 20_000
    ref = orc.observable_hist(0, 0, n, n, obs, n_threads=mfo.max_threads())
    gpu.vegas_iterate(n)
    got, n_it = gpu.get_observables()
    for (g1, g2), (r1, r2) in zip(got, ref):
        np.testing.assert_allclose(g1, r1, rtol=1e-10, atol=1e-13 * np.abs(r1).max())
        np.testing.assert_allclose(g2, r2, rtol=1e-10, atol=1e-13 * np.abs(r2).max())
    with pytest.raises(mf.MfError) as e:
        gpu.set_path(False)                                   # heavy processes: classic RAMBO on the staged path only
    assert e.value.code == mf.MF_EUNSUPPORTED
    for bad in (dict(process=W.EE_MUMU, generator=1), dict(process=W.GG_TT, generator=4)):
        with pytest.raises(mf.MfError) as e:
            mf.Vegas(W.config(bad["process"], generator=bad["generator"]))
        assert e.value.code == mf.MF_EINVAL
    c = W.CONFIGS[1]
    for gen in (1, 2, 3):
        gpu = mf.Vegas(W.config(W.GG_TT, seed=c["seed"], generator=gen))
        for _ in range(c["n_iter"]):
            gpu.vegas_iterate(c["n_events"])
        r = gpu.result()
        assert abs(r["integral"] - 1074.393) < 5 * r["sigma"] + 0.02 and r["sigma"] < 1.5, (gen, r)


# ---- quark channel: q q~ -> t t~, luminosity summed over five flavours on the 11-flavour grid (process 4),
# and p p -> t t~ = g g -> t t~ + q q~ -> t t~ in one integrand (process 5)
@pytest.mark.parametrize("proc,gen,n", [(4, 0, 5003), (4, 1, 5003), (4, 2, 5003), (5, 0, 5003), (5, 3, 5003)])
def test_quark_channel_per_event_parity(mf, mfo, proc, gen, n):
    cfg = W.config(proc, seed=8, generator=gen)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    assert gpu.d == orc.d == (10 if gen & 1 else 4) and gpu.n_final == 2
    mom_tol = (1e-10, 1e-8) if gen & 1 else (1e-11, 1e-9)
    ref = orc.eval(0, 0, n, n_threads=mfo.max_threads())
    # proc = 0: the pdf record (the two flavour sums of ten products of O(1) interpolants, each good to 1e-15) is compared
    # below; towards x -> 1 (sampled often by the linear-tau map) the sums go to zero and their absolute error shows
    compare_events(gpu.integrand_eval(0, 0, n, debug=True), ref, 0, mom_tol, lumi_abs=2e-14)
    e = random_grid(orc.d, 50, 300)
    gpu.set_grid(e); orc.set_grid(e)
    ref = orc.eval(4, 2**34 + 3, n, n_threads=mfo.max_threads())
    out = gpu.integrand_eval(4, 2**34 + 3, n, debug=True)
    compare_events(out, ref, 0, mom_tol, lumi_abs=2e-14)
    np.testing.assert_allclose(out["pdf"].cpu().numpy(), ref["pdf"], rtol=1e-12, atol=1e-14)   # the two flavour sums
    assert (ref["pdf"][:, 0] != ref["pdf"][:, 1]).all()      # distinct sums (process 4: the beam orientations; 5: the two luminosities)


@pytest.mark.parametrize("proc,sigma_pb", [(W.QQ_TT, 79.96), (W.PP_TT, 1074.393 + 79.96)])
def test_quark_channel_iterations_cross_section_and_errors(mf, mfo, proc, sigma_pb):
    """fused iterations against the oracle (raw sums, histogram, grid), observables, the cross section against the
    quadrature values pinned on the oracle side (tests/test_oracle_quarks.py, test_oracle_me.py), argument errors"""
    cfg = W.config(proc, seed=0)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    obs = [(0, 20, 0.0, 400.0), (2, 16, 350.0, 1500.0)]
    gpu.set_observables(obs)
    n = 40_000
    ref = [(np.zeros(o[1] + 2), np.zeros(o[1] + 2)) for o in obs]
    for it in range(3):
        for (a, b), (r1, r2) in zip(orc.observable_hist(it, 0, n, n, obs, n_threads=mfo.max_threads()), ref):
            r1 += a; r2 += b
        g = gpu.vegas_iterate(n)
        o = orc.iterate(n, n_threads=mfo.max_threads())
        assert g["n_pass"] == o["n_pass"] == n and g["n_nonfinite"] == 0
        assert abs(g["integral"] / o["integral"] - 1) < RTOL_INT and abs(g["sigma"] / o["sigma"] - 1) < 1e-8
        np.testing.assert_allclose(gpu.get_accum()[0][:2 + 4 * 50], orc.get_accum(), rtol=RTOL_INT, atol=1e-300)
        np.testing.assert_allclose(gpu.get_grid(), orc.get_grid(), rtol=0, atol=1e-11)
        gpu.set_grid(orc.get_grid())
    got, n_it = gpu.get_observables()
    for (g1, g2), (r1, r2) in zip(got, ref):
        np.testing.assert_allclose(g1, r1, rtol=1e-10, atol=1e-13 * np.abs(r1).max())
        np.testing.assert_allclose(g2, r2, rtol=1e-10, atol=1e-13 * np.abs(r2).max())
    gpu = mf.Vegas(cfg)
    for _ in range(5):
        gpu.vegas_iterate(1_000_000)
    r = gpu.result()
    assert abs(r["integral"] - sigma_pb) < 5 * r["sigma"] + 3e-4 * sigma_pb and r["sigma"] < 6e-4 * sigma_pb, r
    with pytest.raises(mf.MfError) as e:
        gpu.set_path(True)                                    # light process: fused path only
    assert e.value.code == mf.MF_EUNSUPPORTED
    for bad in (W.config(proc, pdf_xf=W.synthetic_gluon_grid()), W.config(W.GG_TT, pdf_xf=W.synthetic_flavour_grid()),
                W.config(proc, precision=32)):
        with pytest.raises(mf.MfError):
            mf.Vegas(bad)
    two_current = mf.Vegas(W.config(W.EE_MUMU)).me_flops()["flops"]
    extra = mf.Vegas(W.config(W.GG_TT)).me_flops()["flops"] + 3 if proc == W.PP_TT else 0   # + the luminosity-weighted sum
    assert gpu.me_flops()["flops"] == two_current + extra


def test_config2_full_iteration_against_oracle(mf, mfo):
    """configs[2] at its full size, every event through the oracle: the raw sums (I, S2), the 7 x 50 histogram, the pass
    counter and the refined grid of a whole 1e7-event iteration on the GPU (staged path, the launch configuration
    bench.py times) against the oracle's (about two minutes on 16 host cores; 2e6 events on a box with fewer than 8)"""
    n = 10_000_000 if mfo.max_threads() >= 8 else 2_000_000
    cfg = W.config(W.GG_TTG, seed=0)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    g = gpu.vegas_iterate(n)
    o = orc.iterate(n, n_threads=mfo.max_threads())
    assert g["n_pass"] == o["n_pass"] and g["n_nonfinite"] == 0 == o["n_nonfinite"]
    assert abs(g["integral"] / o["integral"] - 1) < RTOL_INT and abs(g["sigma"] / o["sigma"] - 1) < 1e-8
    np.testing.assert_allclose(gpu.get_accum()[0], orc.get_accum(), rtol=RTOL_INT, atol=1e-300)
    np.testing.assert_allclose(gpu.get_grid(), orc.get_grid(), rtol=0, atol=1e-11)


def test_device_side_sharded_iteration(mf):
    """multi-GPU exchange without host round trips (mf_zero_accum / mf_get_accum_device / mf_set_accum_device around an
    NCCL all-reduce on the device buffer), on the one GPU of this box with a world-size-1 NCCL group: identical to
    mf_vegas_iterate bit for bit (same launches); and two event ranges accumulated one after the other, as two ranks
    would, agree to summation order"""
    import os
    import torch
    import torch.distributed as dist
    from paper_2105_10529_b200 import sharding
    dev = torch.device("cuda", 0)
    cfg = W.config(W.GG_TTG, seed=11)
    n = 300_001
    a, b, c = mf.Vegas(cfg), mf.Vegas(cfg), mf.Vegas(cfg)
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", str(29700 + os.getpid() % 200))
    group = False
    if not dist.is_initialized():
        try:
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
            group = True
        except Exception as exc:                                   # no NCCL rendezvous on this box: the exchange kernels are
            print("NCCL group not available (%s): running without the collective" % exc)   # still checked, without all_reduce
            dist = None
    try:
        for _ in range(2):
            ia = a.vegas_iterate(n)
            ib = sharding.sharded_iterate_device(b, n, 0, 1, dist, dev)
            assert ia["integral"] == ib["integral"] and ia["sigma"] == ib["sigma"] and ia["n_pass"] == ib["n_pass"]
            np.testing.assert_array_equal(a.get_grid(), b.get_grid())
            # two "ranks" on one handle: ranges [0, n/2) and [n/2, n), packed sums added on the device
            c.zero_accum()
            bufs = []
            for r in range(2):
                first, m = sharding.shard_range(n, r, 2)
                c.zero_accum(); c.vegas_accumulate(first, m, n)
                t = torch.empty(c.accum_len() + 2, dtype=torch.float64, device=dev)
                c.get_accum_device(t.data_ptr()); bufs.append(t)
            tot = bufs[0] + bufs[1]
            if dist is not None:
                dist.all_reduce(tot)                               # world size 1: identity, through NCCL
            c.set_accum_device(tot.data_ptr())
            ic = c.vegas_finalize(n)
            assert ic["n_pass"] == ia["n_pass"] and abs(ic["integral"] / ia["integral"] - 1) < 1e-13
            np.testing.assert_allclose(c.get_grid(), a.get_grid(), rtol=0, atol=1e-13)
    finally:
        if group:
            dist.destroy_process_group()


@pytest.mark.parametrize("proc,gen,n", [(W.QQ_TT, 0, 1_000_000), (W.GG_TTG, W.GEN_CLASSIC_RAMBO, 10_000_000),
                                        (W.GG_TTGG, W.GEN_CLASSIC_RAMBO | W.GEN_LINEAR_TAU, 1_000_000)])
def test_widened_rows_full_size_launch_sampled_parity(mf, mfo, proc, gen, n):
    """the quark channel and the selectable generators at the full size of the config they vary, in the launch
    configuration `bench.py --processes` times: raw sums of the iteration == sums of the eval kernel's weights, counters
    consistent, sampled events == oracle"""
    cfg = W.config(proc, seed=0, generator=gen)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    g = gpu.vegas_iterate(n)
    acc, cnt = gpu.get_accum()
    w = mf.Vegas(cfg).integrand_eval(0, 0, n)["weight"]
    t = w / n
    assert abs(float(t.sum()) / acc[0] - 1) < 1e-10 and abs(float((t * t).sum()) / acc[1] - 1) < 1e-10
    assert int((w != 0).sum()) <= cnt[0] <= n and g["n_nonfinite"] == 0 and g["n_events"] == n
    for i in (0, 1, 255, 256, 65_537, n // 2 + 1, n - 1):
        ref = orc.eval(0, i, 1)["weight"][0]
        got = float(w[i])
        assert (ref == 0 and got == 0) or abs(got / ref - 1) < RTOL_EVENT, (i, got, ref)


def test_fp32_matrix_element_with_generator_variants(mf):
    """the fp32 |M|^2 stage never sees the VEGAS dimensions, so it runs unchanged behind the variant generators: same
    events and counters as the fp64 run of the same variant, integral within fp32 rounding"""
    for gen in (W.GEN_CLASSIC_RAMBO, W.GEN_LINEAR_TAU):
        a = mf.Vegas(W.config(W.GG_TTG, seed=5, generator=gen))
        b = mf.Vegas(W.config(W.GG_TTG, seed=5, generator=gen, precision=32))
        ia, ib = a.vegas_iterate(200_000), b.vegas_iterate(200_000)
        assert ia["n_pass"] == ib["n_pass"] and ib["n_nonfinite"] == 0 and abs(ib["integral"] / ia["integral"] - 1) < 1e-5
        wa = a.integrand_eval(1, 0, 4000, debug=True); wb = b.integrand_eval(1, 0, 4000, debug=True)
        assert (wa["bins"] == wb["bins"]).all() and (wa["pass_"] == wb["pass_"]).all()
        nz = wa["weight"] != 0
        rel = (wb["weight"][nz] / wa["weight"][nz] - 1).abs()
        assert float(rel.median()) < 1e-5 and float((rel > 1e-4).double().mean()) < 5e-3      # north_star: 1e-4 for the fp32 path


# ---- config 3 (gg -> tt~gg, one event over four lanes in the |M|^2 stage) at sizes that reach the full-size code path ------
def test_config3_large_iteration_against_oracle(mf, mfo):
    """a 1e5-event iteration of gg -> tt~gg on the staged path (several hundred record regions, prefix + binary search over the
    region counts, 4-lane |M|^2 stage) on a random adapted grid, every event through the oracle: raw sums, all 10 x 50 histogram
    bins, pass counter, refined grid (about a minute of oracle time on 16 host cores)"""
    n = 100_000 if mfo.max_threads() >= 8 else 20_000
    cfg = W.config(W.GG_TTGG, seed=0)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    e = random_grid(orc.d, 50, 77)
    gpu.set_grid(e); orc.set_grid(e)
    g = gpu.vegas_iterate(n)
    o = orc.iterate(n, n_threads=mfo.max_threads())
    assert g["n_pass"] == o["n_pass"] and g["n_nonfinite"] == 0 == o["n_nonfinite"] and g["n_events"] == n
    assert abs(g["integral"] / o["integral"] - 1) < RTOL_INT and abs(g["sigma"] / o["sigma"] - 1) < 1e-8
    acc = gpu.get_accum()[0]
    assert acc.shape == (2 + 10 * 50,)
    np.testing.assert_allclose(acc, orc.get_accum(), rtol=RTOL_INT, atol=1e-300)
    np.testing.assert_allclose(gpu.get_grid(), orc.get_grid(), rtol=0, atol=1e-11)


def test_config3_full_index_range_per_event(mf, mfo):
    """1e4 events of the 1e6-event config-3 iteration, in 20 chunks of 500 spread over the whole index range (and a second
    iteration counter), event by event against the oracle: bins, cut flags, points, momenta, PDFs, |M|^2, weights"""
    cfg = W.config(W.GG_TTGG, seed=0)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    n = W.CONFIGS[3]["n_events"]
    for j in range(20):
        first = j * (n // 20) + 37 * j
        it = 0 if j % 2 == 0 else 4
        ref = orc.eval(it, first, 500, n_threads=mfo.max_threads())
        compare_events(gpu.integrand_eval(it, first, 500, debug=True), ref, 3)


def test_streams_and_stage_time_sums(mf):
    """calls under a non-default torch stream (the binding passes the current stream of the handle's device); two streams
    without host synchronisation in between (the library orders a call behind the last writer of the integrator state);
    stage times summed over every slice of a sliced iteration; flop bounds"""
    import torch
    from paper_2105_10529_b200 import sharding
    cfg = W.config(W.GG_TTG, seed=12)
    n = 200_003
    a, b, c = mf.Vegas(cfg), mf.Vegas(cfg), mf.Vegas(cfg)
    ia = [a.vegas_iterate(n) for _ in range(2)]
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(s1):
        ib = [b.vegas_iterate(n) for _ in range(2)]
        ic = [sharding.sharded_iterate_device(c, n, 0, 1, None, torch.device("cuda", 0)) for _ in range(2)]
    for x, y, z in zip(ia, ib, ic):
        assert x == y or {k: x[k] for k in x if k != "kernel_ms"} == {k: y[k] for k in y if k != "kernel_ms"}
        assert x["integral"] == z["integral"] and x["n_pass"] == z["n_pass"]
    np.testing.assert_array_equal(a.get_grid(), b.get_grid())
    np.testing.assert_array_equal(a.get_grid(), c.get_grid())
    # iterate on s1 (enqueue only), evaluate on s2 at once: the evaluation must see the refined grid
    ref = a.vegas_iterate(n) and a.integrand_eval(0, 0, 4096)["weight"].clone()
    with torch.cuda.stream(s1):
        b.vegas_iterate(n, sync=False)
    with torch.cuda.stream(s2):
        w = b.integrand_eval(0, 0, 4096)["weight"]
    s2.synchronize()
    assert torch.equal(w, ref)
    assert b.result()["n_iter"] == 3 and b.result()["integral"] == a.result()["integral"]
    # stage times: one entry per staged launch; an iteration of more than 2^24 events runs as two slices
    a.stage_ms_sum()
    a.vegas_iterate((1 << 24) + 1000)
    sums, launches = a.stage_ms_sum()
    assert launches == 2 and sums["front"] > 0 and sums["me"] > sums["front"] and sums["reduce"] > 0
    assert a.stage_ms_sum()[1] == 0
    fb = a.me_flops_bounds()
    assert fb["min"] == 11302 and a.me_flops()["flops"] == 11591 and fb["executed"] == 11975      # staged path: loop over gluon leg 2 only
    a.set_path(False)
    fb = a.me_flops_bounds()
    assert a.me_flops()["flops"] == 15023 == fb["executed"] and fb["min"] == 11302                 # fused path: the register-resident organisation
    a.set_path(True)
    fb = mf.Vegas(W.config(W.GG_TTGG)).me_flops_bounds()
    assert fb["min"] == 170880 < 256020 < fb["executed"]


# ---- channels with a second quark line and one gluon: q q~ -> t t~ g (6), q g -> t t~ q (7) -----------------
@pytest.mark.parametrize("proc,gen,n", [(6, 0, 3001), (6, 3, 2001), (7, 0, 3001), (7, 1, 2001)])
def test_two_quark_line_channels_per_event_parity(mf, mfo, proc, gen, n):
    cfg = W.config(proc, seed=8, generator=gen)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    assert gpu.d == orc.d == (14 if gen & 1 else 7) and gpu.n_final == 3
    mom_tol = (1e-10, 1e-8) if gen & 1 else (1e-11, 1e-9)
    ref = orc.eval(0, 0, n, n_threads=mfo.max_threads())
    # the luminosity record: the absolute-error term of the quark channel (DESIGN.md 5.9 / section 6)
    compare_events(gpu.integrand_eval(0, 0, n, debug=True), ref, 0, mom_tol, lumi_abs=2e-14)
    e = random_grid(orc.d, 50, 400 + proc)
    gpu.set_grid(e); orc.set_grid(e)
    ref = orc.eval(3, 2**33 + 5, n, n_threads=mfo.max_threads())
    out = gpu.integrand_eval(3, 2**33 + 5, n, debug=True)
    compare_events(out, ref, 0, mom_tol, lumi_abs=2e-14)
    np.testing.assert_allclose(out["pdf"].cpu().numpy(), ref["pdf"], rtol=1e-12, atol=1e-14)
    assert 0.5 < ref["pass_"].mean() < 0.999                  # the cuts act on the third final particle


@pytest.mark.parametrize("proc", [W.QQ_TTG, W.QG_TTQ])
def test_two_quark_line_channels_iterations_and_errors(mf, mfo, proc):
    """fused iterations against the oracle (raw sums, histogram, pass counter, grid), observables incl. the jet pT, full-size
    launch with sampled events, argument errors"""
    cfg = W.config(proc, seed=0)
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    obs = [(0, 20, 0.0, 400.0), (3, 10, 30.0, 230.0)]
    gpu.set_observables(obs)
    n = 30_000
    ref = [(np.zeros(o[1] + 2), np.zeros(o[1] + 2)) for o in obs]
    for it in range(3):
        for (a, b), (r1, r2) in zip(orc.observable_hist(it, 0, n, n, obs, n_threads=mfo.max_threads()), ref):
            r1 += a; r2 += b
        g = gpu.vegas_iterate(n)
        o = orc.iterate(n, n_threads=mfo.max_threads())
        assert g["n_pass"] == o["n_pass"] and g["n_nonfinite"] == 0 == o["n_nonfinite"]
        assert abs(g["integral"] / o["integral"] - 1) < RTOL_INT and abs(g["sigma"] / o["sigma"] - 1) < 1e-8
        np.testing.assert_allclose(gpu.get_accum()[0][:2 + 7 * 50], orc.get_accum(), rtol=RTOL_INT, atol=1e-300)
        np.testing.assert_allclose(gpu.get_grid(), orc.get_grid(), rtol=0, atol=1e-11)
        gpu.set_grid(orc.get_grid())
    got, n_it = gpu.get_observables()
    for (g1, g2), (r1, r2) in zip(got, ref):
        np.testing.assert_allclose(g1, r1, rtol=1e-10, atol=1e-13 * np.abs(r1).max())
        np.testing.assert_allclose(g2, r2, rtol=1e-10, atol=1e-13 * np.abs(r2).max())
    # full-size launch (1e6 events per iteration): raw sums == sums of the eval kernel's weights; sampled events == oracle
    n = 1_000_000
    gpu, orc = mf.Vegas(cfg), mfo.Vegas(cfg)
    g = gpu.vegas_iterate(n)
    acc, cnt = gpu.get_accum()
    w = mf.Vegas(cfg).integrand_eval(0, 0, n)["weight"]
    t = w / n
    assert abs(float(t.sum()) / acc[0] - 1) < 1e-10 and abs(float((t * t).sum()) / acc[1] - 1) < 1e-10
    assert int((w != 0).sum()) == cnt[0] and g["n_nonfinite"] == 0
    for i in (0, 1, 255, 256, 65_537, n // 2 + 1, n - 1):
        r = orc.eval(0, i, 1)["weight"][0]
        assert (r == 0 and float(w[i]) == 0) or abs(float(w[i]) / r - 1) < RTOL_EVENT
    with pytest.raises(mf.MfError) as e:
        gpu.set_path(True)                                    # fused path only
    assert e.value.code == mf.MF_EUNSUPPORTED
    for bad in (W.config(proc, pdf_xf=W.synthetic_gluon_grid()), W.config(proc, precision=32)):
        with pytest.raises(mf.MfError):
            mf.Vegas(bad)
    assert gpu.me_flops()["flops"] == (2 if proc == W.QQ_TTG else 4) * (5661 + 2)


def test_checkpoint_and_resume(mf):
    """mf_get_state / mf_set_state: a run saved after two iterations and restored into a fresh handle continues bit for bit (grid,
    iteration records, Philox iteration word, observable sums); states of another configuration or damaged blobs are rejected"""
    for proc, n in ((W.GG_TTG, 100_003), (W.PP_TT, 50_001)):
        cfg = W.config(proc, seed=21)
        obs = [(0, 20, 0.0, 400.0), (2, 16, 350.0, 1500.0)]
        a = mf.Vegas(cfg)
        a.set_observables(obs)
        for _ in range(2):
            a.vegas_iterate(n)
        blob = a.get_state()
        assert len(blob) == len(a.get_state()) and blob == a.get_state()
        b = mf.Vegas(cfg)
        b.set_observables(obs)
        b.set_state(blob)
        np.testing.assert_array_equal(a.get_grid(), b.get_grid())
        assert b.get_iterations() == a.get_iterations() and b.result() == a.result()
        ia, ib = a.vegas_iterate(n), b.vegas_iterate(n)
        assert {k: ia[k] for k in ia if k != "kernel_ms"} == {k: ib[k] for k in ib if k != "kernel_ms"}
        np.testing.assert_array_equal(a.get_grid(), b.get_grid())
        assert a.result() == b.result() and b.result()["n_iter"] == 3
        (ga, na), (gb, nb_) = a.get_observables(), b.get_observables()
        assert na == nb_ == 3
        for (x1, x2), (y1, y2) in zip(ga, gb):
            np.testing.assert_array_equal(x1, y1); np.testing.assert_array_equal(x2, y2)
        assert len(b.get_state()) == len(blob) + 40                    # one more iteration record
        # the restored run saw the same random numbers as the uninterrupted one: per-event weights of the next iteration agree too
        assert bool((a.integrand_eval(3, 0, 2048)["weight"] == b.integrand_eval(3, 0, 2048)["weight"]).all())
        for bad_cfg in (W.config(proc, seed=22), W.config(W.GG_TT if proc != W.GG_TT else W.GG_TTG, seed=21)):
            c = mf.Vegas(bad_cfg)
            if bad_cfg["process"] == proc:
                c.set_observables(obs)
            with pytest.raises(mf.MfError) as e:
                c.set_state(blob)
            assert e.value.code == mf.MF_EINVAL
        c = mf.Vegas(cfg)                                               # observables not set as when the state was saved
        with pytest.raises(mf.MfError):
            c.set_state(blob)
        c.set_observables(obs)
        for damaged in (blob[:-8], b"XXXX" + blob[4:], blob[:64]):
            with pytest.raises(mf.MfError):
                c.set_state(damaged)
        c.set_state(blob)                                               # and the intact blob still goes in
        assert c.result()["n_iter"] == 2
