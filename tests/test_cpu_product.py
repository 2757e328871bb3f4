"""CPU-side tests of the product's host logic: the C-ABI library loads and exports every symbol the
header declares (no compute calls without a GPU), argument validation, the build-time amplitude
generator evaluated numerically against the oracle, and the sharded-iteration plumbing under gloo."""
import ctypes as C
import math
import os
import re
import numpy as np
import pytest

from paper_2105_10529_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2105_10529_b200 import build, binding as b
    build.build()
    b.lib()
    return b


def test_library_exports_every_declared_symbol(binding):
    hdr = open(os.path.join(ROOT, "include", "madflow_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mf_[a-z0-9_]+)\s*\(", hdr))
    assert {"mf_vegas_create", "mf_integrand_eval", "mf_vegas_iterate", "mf_result"} <= declared
    lib = binding.lib()
    for name in sorted(declared):
        assert getattr(lib, name) is not None, name
    assert declared == set(binding.EXPORTS)


def test_argument_validation_and_no_cpu_path(binding):
    import torch
    lib = binding.lib()
    h = C.c_void_p()
    cfg, pdf = binding.make_config(W.config(W.GG_TTG))
    cfg.n_bins = 100                                   # invalid: validated before any device work
    assert lib.mf_vegas_create(C.byref(cfg), C.byref(h)) == binding.MF_EINVAL
    assert b"n_bins" in lib.mf_last_error()
    cfg, pdf = binding.make_config(W.config(W.GG_TTG))
    cfg.struct_size = 8
    assert lib.mf_vegas_create(C.byref(cfg), C.byref(h)) == binding.MF_EINVAL
    cfg, pdf = binding.make_config(W.config(W.GG_TT))  # the fp32 |M|^2 variant exists for gg -> tt~g only
    cfg.precision = 32
    assert lib.mf_vegas_create(C.byref(cfg), C.byref(h)) == binding.MF_EUNSUPPORTED
    cfg, pdf = binding.make_config(W.config(W.GG_TTG))
    cfg.precision = 16
    assert lib.mf_vegas_create(C.byref(cfg), C.byref(h)) == binding.MF_EUNSUPPORTED
    if not torch.cuda.is_available():                  # no CPU fallback: a valid config fails loudly
        cfg, pdf = binding.make_config(W.config(W.GG_TTG))
        assert lib.mf_vegas_create(C.byref(cfg), C.byref(h)) == binding.MF_ECUDA
        assert b"no CUDA device" in lib.mf_last_error()
        with pytest.raises(binding.MfError):
            binding.Vegas(W.config(W.GG_TT))
    assert lib.mf_result(None, None) == binding.MF_EINVAL


# ---- the amplitude generator, evaluated with NumPy, against the oracle -----------------------------
def _ferm(p, m):
    E, px, py, pz = p
    pabs = math.sqrt(px * px + py * py + pz * pz); pt2 = px * px + py * py
    wp = math.sqrt(E + pabs); wm = 0.0 if m == 0 else m / wp
    if pabs < 1e-12 * abs(E) or (pt2 == 0 and pz < 0):
        return wp, wm, 0.0, 1.0, 0.0
    ppz = pabs + pz if pz >= 0 else pt2 / (pabs - pz)
    N = 1 / math.sqrt(2 * pabs * ppz)
    return wp, wm, N * ppz, N * px, N * py


def _glu(k):
    E, px, py, pz = k
    pt = math.hypot(px, py); pabs = math.sqrt(px * px + py * py + pz * pz); s = 1 / math.sqrt(2)
    return px * pz / (pabs * pt) * s, py * pz / (pabs * pt) * s, -pt / pabs * s, -py / pt * s, px / pt * s


def _inputs(gen, mom, mt=173.0):
    v = dict(E=mom[0][0], mt=mt)
    for n, c in zip(("p3e", "p3x", "p3y", "p3z"), mom[2]): v[n] = c
    for n, c in zip(("p4e", "p4x", "p4y", "p4z"), mom[3]): v[n] = c
    for n, c in zip(("wp", "wm", "c0", "cx", "cy"), _ferm(mom[2], mt)): v["t_" + n] = c
    for n, c in zip(("wp", "wm", "c0", "cx", "cy"), _ferm(mom[3], mt)): v["b_" + n] = c
    for l in range(2, gen.ng):
        for n, c in zip("exyz", mom[2 + l]): v["k%d%s" % (l, n)] = c
        for n, c in zip(("e1x", "e1y", "e1z", "e2x", "e2y"), _glu(mom[2 + l])): v["g%d_%s" % (l, n)] = c
    return v


@pytest.mark.parametrize("proc,fname,n", [(1, "mf_me2_gg_tt", 2), (2, "mf_me2_gg_ttg", 3)])
def test_generated_amplitude_dag_matches_oracle(mfo, proc, fname, n):
    from paper_2105_10529_b200.gen import amplitudes as A
    gen = A.generate(fname)
    text, tot = A.emit_function(gen, fname)
    assert "%s_NFMA %dull" % (fname.upper(), tot["fma"]) in text
    gs2 = 4 * math.pi * 0.118
    rng = np.random.default_rng(17 + proc)
    for trial in range(4 if proc < 3 else 2):
        rts = rng.uniform(450, 4000)
        ps = mfo.phase_space(n, rts * rts, [173.0, 173.0] + [0.0] * (n - 2), rng.uniform(0.03, 0.97, 3 * n - 4))
        mom = np.zeros((2 + n, 4)); mom[0] = [rts / 2, 0, 0, rts / 2]; mom[1] = [rts / 2, 0, 0, -rts / 2]; mom[2:] = ps["k"]
        ref = mfo.me2(proc, mom)
        val = float(A.evaluate(gen, _inputs(gen, mom))) * gen.scale * gs2 ** n / 256
        assert abs(val / ref - 1) < 1e-11
        if fname == "mf_me2_gg_ttg":      # the organisation of the shared-memory-operand variant (loop over gluon leg 2 only)
            gs_ = A.generate_smem(fname)
            assert gs_.input_names == gen.input_names and gs_.scale == gen.scale and len(gs_.loop_assign) == 2
            assert abs(float(A.evaluate(gs_, _inputs(gs_, mom))) * gs_.scale * gs2 ** n / 256 / ref - 1) < 1e-11


def test_four_lane_decomposition_matches_oracle(mfo):
    """gg -> tt~gg with one event over four lanes (gen/lanes.py): the per-lane DAG evaluated for the four lanes with the
    exchanges of currents and amplitudes played out, against the oracle; the orbit structure of the shared currents; and
    the one-thread organisation of the same amplitude (the algorithmic flop count) against both"""
    from paper_2105_10529_b200.gen import amplitudes as A, lanes as L
    gen = L.GenLanes()
    gen.build()
    assert [len(gen.reps[s]) for s in (2, 3, 4)] == [2, 3, 4]          # orbits of the cyclic relabelling
    assert len(gen.local) == 6 and all(sg[-1] == 0 for sg in gen.local) and gen.n_slots == 36
    text, tot, parts = L.emit_lanes(gen, "mf_me2_gg_ttgg_lanes")
    assert text.count("__syncwarp();") == 6 and "MF_ME2_GG_TTGG_LANES_NFMA %dull" % tot["fma"] in text
    one = A.Gen(4, loop_legs=(0, 1, 2, 3), parity=True, basis="linear")
    one.build()

    def glu_units(k):
        e = np.array(_glu(k)) * math.sqrt(2)
        return e[:3], np.array([e[3], e[4], 0.0])

    gs2 = 4 * math.pi * 0.118
    rng = np.random.default_rng(23)
    for trial in range(3):
        rts = rng.uniform(450, 4000)
        ps = mfo.phase_space(4, rts * rts, [173.0, 173.0, 0.0, 0.0], rng.uniform(0.03, 0.97, 8))
        mom = np.zeros((6, 4)); mom[0] = [rts / 2, 0, 0, rts / 2]; mom[1] = [rts / 2, 0, 0, -rts / 2]; mom[2:] = ps["k"]
        ref = mfo.me2(3, mom)
        val = L.evaluate_event(gen, mom, 173.0, _ferm, glu_units) * gen.scale * gs2 ** 4 / 256
        assert abs(val / ref - 1) < 1e-11
        if trial == 0:
            v1 = float(A.evaluate(one, _inputs(one, mom))) * one.scale * gs2 ** 4 / 256
            assert abs(v1 / ref - 1) < 1e-11


def test_two_quark_line_generator_matches_oracle(mfo):
    """gen/quarks.py (q q~ -> t t~ g, q g -> t t~ q: four colour structures, linear polarisations, generic external lines)
    evaluated with NumPy against the oracle's five explicit diagrams with the literal colour sum, on the basic channel and on the
    beam-exchanged + charge-conjugated one"""
    from paper_2105_10529_b200.gen import amplitudes as A, quarks as Q
    num, den = Q.colour_matrix_2q()
    assert den == 9 and (num == num.T).all() and num[0][0] == num[1][1] and num[2][2] == num[3][3]
    gs2 = 4 * math.pi * 0.118
    rng = np.random.default_rng(29)
    for kind, proc in (("qq", W.QQ_TTG), ("qg", W.QG_TTQ)):
        gen = Q.Gen2Q(kind)
        gen.build()
        assert len(gen.input_names) == 41
        looped = Q.PROCESSES_2Q["mf_me2_%s" % ("qq_ttg" if kind == "qq" else "qg_ttq")]()      # the emitted form: polarisation loop
        looped.build()
        assert looped.loop_pol and looped.input_names == gen.input_names and looped.scale == gen.scale and len(looped.loop_assign) == 2
        for trial in range(3):
            rts = rng.uniform(450, 4000)
            ps = mfo.phase_space(3, rts * rts, [173.0, 173.0, 0.0], rng.uniform(0.03, 0.97, 5))
            mom = np.vstack([[rts / 2, 0, 0, rts / 2], [rts / 2, 0, 0, -rts / 2], ps["k"]])
            for swap in (False, True):
                m = mom.copy()
                if swap:
                    m[[0, 1]] = m[[1, 0]]; m[[2, 3]] = m[[3, 2]]
                pa, pb, k1, k2, k3 = m
                v = dict(mt=173.0)
                for n, c in zip("exyz", k2): v["k2" + n] = c
                for n, c in zip(("wp", "wm", "c0", "cx", "cy"), _ferm(k1, 173.0)): v["t_" + n] = c
                for n, c in zip(("wp", "wm", "c0", "cx", "cy"), _ferm(k2, 173.0)): v["b_" + n] = c
                pr, K, kg = (pb, -k3, k3) if kind == "qq" else (-k3, pb, pb)
                for n, c in zip("exyz", pa): v["pc" + n] = c
                for n, c in zip("exyz", pr): v["pr" + n] = c
                for n, c in zip("exyz", K): v["K" + n] = c
                for n, c in zip(("wp", "wm", "c0", "cx", "cy"), _ferm(pa, 0.0)): v["c_" + n] = c
                for n, c in zip(("wp", "wm", "c0", "cx", "cy"), _ferm(pb if kind == "qq" else k3, 0.0)): v["r_" + n] = c
                if math.hypot(kg[1], kg[2]) == 0:
                    e1, e2 = [1.0, 0.0, 0.0], [0.0, 1.0 if kg[3] >= 0 else -1.0, 0.0]
                else:
                    e = np.array(_glu(kg)) * math.sqrt(2); e1, e2 = e[:3], [e[3], e[4], 0.0]
                for n, c in zip("xyz", e1): v["e1" + n] = c
                for n, c in zip("xyz", e2): v["e2" + n] = c
                for form in (gen, looped):
                    val = float(A.evaluate(form, {k: x for k, x in v.items() if k in form.input_names})) * form.scale * gs2 ** 3
                    assert abs(val / mfo.me2_2q(proc, m) - 1) < 1e-12


def test_generator_colour_matrices_match_golden():
    from paper_2105_10529_b200.gen import amplitudes as A
    from conftest import read_golden
    g = read_golden("points.txt")
    for ng in (2, 3, 4):
        num, den, perms = A.colour_matrix(ng)
        assert den == int(g["C%d_den" % ng][0])
        assert list(num[0]) == [int(v) for v in g["C%d_row0" % ng]]
        assert (num == num.T).all()
