"""CPU check of the product's per-event arithmetic (csrc/mf_event.cuh + generated |M|^2 code),
compiled for the host by tests/host_harness (test harness only), against the oracle, event by
event on the same seeded inputs.  The GPU parity tests proper are in test_gpu_parity.py."""
import ctypes as C
import os
import subprocess
import numpy as np
import pytest

from paper_2105_10529_b200 import workloads as W
from paper_2105_10529_b200.binding import Config, make_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "host_harness", "mf_host_harness.cpp")
LIB = os.path.join(ROOT, "tests", "host_harness", "libmfh.so")


@pytest.fixture(scope="module")
def harness():
    from paper_2105_10529_b200.gen.__main__ import main as gen_main
    gen_main()
    csrc = os.path.join(ROOT, "paper_2105_10529_b200", "csrc")
    deps = [SRC] + [os.path.join(csrc, f) for f in ("mf_event.cuh", "mf_device.cuh", "mf_params.h")]
    deps += [os.path.join(csrc, "generated", f) for f in os.listdir(os.path.join(csrc, "generated"))]
    if not os.path.exists(LIB) or any(os.path.getmtime(LIB) < os.path.getmtime(p) for p in deps):
        subprocess.check_call(["g++", "-O1", "-std=c++20", "-pthread", "-fPIC", "-shared", "-o", LIB, SRC])
    lib = C.CDLL(LIB)
    lib.mfh_event.restype = C.c_double
    lib.mfh_event.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.mfh_fill_params.argtypes = [C.POINTER(Config), C.c_void_p]
    lib.mfh_event_ttg_f32.restype = C.c_double
    lib.mfh_event_ttg_f32.argtypes = lib.mfh_event.argtypes
    return lib


def random_grid(d, nb, seed):
    rng = np.random.default_rng(seed)
    w = rng.uniform(0.3, 1.7, size=(d, nb))
    e = np.concatenate([np.zeros((d, 1)), np.cumsum(w, axis=1) / w.sum(axis=1, keepdims=True)], axis=1)
    e[:, -1] = 1.0
    return e


@pytest.mark.parametrize("proc,n,tol", [(0, 300, 1e-12), (1, 300, 1e-11), (2, 300, 1e-10), (3, 40, 1e-10)])
def test_host_compiled_event_matches_oracle(mfo, harness, proc, n, tol):
    cfg = W.config(proc, seed=7)
    c, pdf = make_config(cfg)
    P = C.create_string_buffer(harness.mfh_params_size())
    assert harness.mfh_fill_params(C.byref(c), P) == 0
    orc = mfo.Vegas(cfg)
    edges = random_grid(orc.d, 50, 11 + proc)
    orc.set_grid(edges)
    ref = orc.eval(2, 1000, n)
    d, nl = orc.d, 2 + orc.n_final
    bins = np.zeros(16, np.int32); ok = np.zeros(1, np.int32); rec = np.zeros(37)
    worst = 0.0
    for i in range(n):
        F = harness.mfh_event(P, edges.ctypes.data, pdf.ctypes.data if pdf is not None else None, 2, 1000 + i,
                              bins.ctypes.data, ok.ctypes.data, rec.ctypes.data)
        assert list(bins[:d]) == list(ref["bins"][i])
        assert ok[0] == ref["pass_"][i]
        np.testing.assert_allclose(rec[:d], ref["x"][i], rtol=1e-14, atol=0)
        np.testing.assert_allclose(rec[10:10 + 4 * nl].reshape(nl, 4), ref["momenta"][i], rtol=1e-11, atol=1e-9)
        if proc:
            np.testing.assert_allclose(rec[35:37], ref["pdf"][i], rtol=1e-12, atol=1e-15)   # interpolant ~0 near x -> 1: absolute
        if ref["weight"][i] != 0:
            worst = max(worst, abs(F / ref["weight"][i] - 1), abs(rec[34] / ref["me2"][i] - 1))
        else:
            assert F == 0.0
    assert worst < tol, worst


def test_host_compiled_fp32_matrix_element_variant(mfo, harness):
    """the precision = 32 variant (|M|^2 in float, the rest in double) compiled for the host: same events,
    bins and cut flags as the oracle; |M|^2 within float rounding times the gauge cancellations"""
    cfg = W.config(W.GG_TTG, seed=7)
    c, pdf = make_config(cfg)
    P = C.create_string_buffer(harness.mfh_params_size())
    assert harness.mfh_fill_params(C.byref(c), P) == 0
    orc = mfo.Vegas(cfg)
    edges = orc.get_grid()
    n = 400
    ref = orc.eval(0, 0, n)
    bins = np.zeros(16, np.int32); ok = np.zeros(1, np.int32); rec = np.zeros(37)
    rel = []
    for i in range(n):
        F = harness.mfh_event_ttg_f32(P, edges.ctypes.data, pdf.ctypes.data, 0, i, bins.ctypes.data, ok.ctypes.data, rec.ctypes.data)
        assert list(bins[:orc.d]) == list(ref["bins"][i]) and ok[0] == ref["pass_"][i]
        if ref["weight"][i] != 0:
            rel.append(abs(F / ref["weight"][i] - 1))
        else:
            assert F == 0.0
    rel = np.array(rel)
    assert np.median(rel) < 2e-6 and (rel > 1e-4).mean() < 0.02 and rel.max() < 1e-2, (np.median(rel), rel.max())


@pytest.mark.parametrize("proc,gen,n", [(1, 1, 200), (1, 2, 200), (1, 3, 200), (2, 1, 200), (2, 2, 100), (2, 3, 200), (3, 1, 30), (3, 3, 30)])
def test_host_compiled_generator_variants_match_oracle(mfo, harness, proc, gen, n):
    """selectable generators (classic 4n-random RAMBO = 1, linear tau = 2) of the product's per-event
    code, compiled for the host, against the oracle's mfo_rambo_classic / mfo_x_map_linear path"""
    harness.mfh_event_gen.restype = C.c_double
    harness.mfh_event_gen.argtypes = harness.mfh_event.argtypes
    cfg = W.config(proc, seed=9, generator=gen)
    c, pdf = make_config(cfg)
    P = C.create_string_buffer(harness.mfh_params_size())
    assert harness.mfh_fill_params(C.byref(c), P) == 0
    orc = mfo.Vegas(cfg)
    d, nl = orc.d, 2 + orc.n_final
    assert d == (2 + 4 * orc.n_final if gen & 1 else 3 * orc.n_final - 2)
    edges = random_grid(d, 50, 21 + proc)
    orc.set_grid(edges)
    ref = orc.eval(1, 500, n)
    bins = np.zeros(24, np.int32); ok = np.zeros(1, np.int32); rec = np.zeros(45)
    worst = 0.0
    for i in range(n):
        F = harness.mfh_event_gen(P, edges.ctypes.data, pdf.ctypes.data, 1, 500 + i, bins.ctypes.data, ok.ctypes.data, rec.ctypes.data)
        assert list(bins[:d]) == list(ref["bins"][i])
        assert ok[0] == ref["pass_"][i]
        np.testing.assert_allclose(rec[:d], ref["x"][i], rtol=1e-14, atol=0)
        np.testing.assert_allclose(rec[18:18 + 4 * nl].reshape(nl, 4), ref["momenta"][i], rtol=1e-10, atol=1e-8)
        np.testing.assert_allclose(rec[43:45], ref["pdf"][i], rtol=1e-11, atol=1e-15)
        if ref["weight"][i] != 0:
            worst = max(worst, abs(F / ref["weight"][i] - 1), abs(rec[42] / ref["me2"][i] - 1))
        else:
            assert F == 0.0
    assert worst < 1e-10, worst


def test_generator_flag_validation(harness):
    """mf_config_t.generator (host logic of mf_vegas_create): unknown flags and process 0 are rejected; d follows the flag"""
    P = C.create_string_buffer(harness.mfh_params_size())
    for proc, gen, rc in [(1, 0, 0), (1, 1, 0), (2, 2, 0), (3, 3, 0), (1, 4, -1), (2, 8, -1), (0, 1, -1), (0, 2, -1)]:
        c, pdf = make_config(W.config(proc, generator=gen))
        assert harness.mfh_fill_params(C.byref(c), P) == rc, (proc, gen)
        if rc == 0:
            d = np.frombuffer(P, dtype=np.int32, count=5)          # MfParams: process, d, n_final, nb, gen
            nf = {1: 2, 2: 3, 3: 4}[proc]
            assert d[0] == proc and d[2] == nf and d[4] == gen and d[1] == (2 + 4 * nf if gen & 1 else 3 * nf - 2)


def flavour_slice(harness, P, pdf11):
    """the library's device copy of the 11-flavour grid (mf_params.h mf_flavour_slice): the tables flavour-innermost
    (slot = PDG id + 5), the Q^2 rows around mu_F only; checked here against a NumPy re-layout"""
    n = harness.mfh_flavour_slice(P, pdf11.ctypes.data, None)
    out = np.zeros(n)
    harness.mfh_flavour_slice(P, pdf11.ctypes.data, out.ctypes.data)
    nx, nq = pdf11.shape[1:]
    iq = int(np.floor((np.log(173.0 ** 2) - np.log(W.PDF_QMIN ** 2)) / (np.log(W.PDF_QMAX ** 2) - np.log(W.PDF_QMIN ** 2)) * (nq - 1)))
    ref = np.transpose(pdf11[:, :, iq - 1:iq + 3], (1, 2, 0))
    assert n == nx * (ref.shape[1] * 11 + 1) and np.array_equal(out.reshape(nx, -1)[:, :-1].reshape(ref.shape), ref)   # one pad double per ln-x row
    return out


@pytest.mark.parametrize("proc,gen,n", [(6, 0, 200), (6, 3, 100), (7, 0, 200), (7, 1, 100)])
def test_host_compiled_two_quark_line_channels_match_oracle(mfo, harness, proc, gen, n):
    """q q~ -> t t~ g (6) and q g -> t t~ q (7): the product's per-event code compiled for the host against the
    oracle: bins, cut flags, momenta, the luminosity record, the luminosity-weighted |M|^2 and the weight"""
    harness.mfh_event_gen.restype = C.c_double
    harness.mfh_event_gen.argtypes = harness.mfh_event.argtypes
    cfg = W.config(proc, seed=17, generator=gen)
    c, pdf = make_config(cfg)
    P = C.create_string_buffer(harness.mfh_params_size())
    assert harness.mfh_fill_params(C.byref(c), P) == 0
    tab = flavour_slice(harness, P, pdf)
    orc = mfo.Vegas(cfg)
    d = orc.d
    assert d == (14 if gen & 1 else 7)
    edges = random_grid(d, 50, 41)
    orc.set_grid(edges)
    ref = orc.eval(2, 900, n)
    bins = np.zeros(24, np.int32); ok = np.zeros(1, np.int32); rec = np.zeros(45)
    worst, n_pass = 0.0, 0
    for i in range(n):
        F = harness.mfh_event_gen(P, edges.ctypes.data, tab.ctypes.data, 2, 900 + i, bins.ctypes.data, ok.ctypes.data, rec.ctypes.data)
        assert list(bins[:d]) == list(ref["bins"][i]) and ok[0] == ref["pass_"][i]
        np.testing.assert_allclose(rec[:d], ref["x"][i], rtol=1e-14, atol=0)
        np.testing.assert_allclose(rec[18:38].reshape(5, 4), ref["momenta"][i], rtol=1e-10, atol=1e-8)
        np.testing.assert_allclose(rec[43:45], ref["pdf"][i], rtol=1e-12, atol=1e-16)
        if ref["weight"][i] != 0:
            n_pass += 1
            worst = max(worst, abs(F / ref["weight"][i] - 1), abs(rec[42] / ref["me2"][i] - 1))
        else:
            assert F == 0.0
    assert worst < 1e-10 and n_pass > n // 2, (worst, n_pass)
    if gen == 0:                                              # and through the plain entry point
        rec37 = np.zeros(37)
        F = harness.mfh_event(P, edges.ctypes.data, tab.ctypes.data, 2, 900, bins.ctypes.data, ok.ctypes.data, rec37.ctypes.data)
        assert F == 0.0 and ref["weight"][0] == 0 or abs(F / ref["weight"][0] - 1) < 1e-10


@pytest.mark.parametrize("proc,gen,n", [(4, 0, 300), (4, 1, 150), (4, 2, 150), (5, 0, 300), (5, 3, 150)])
def test_host_compiled_quark_channel_matches_oracle(mfo, harness, proc, gen, n):
    """q q~ -> t t~ with the flavour-summed luminosity of the product's per-event code, compiled for
    the host, against the oracle: bins, momenta, the two flavour sums, |M|^2 and the weight"""
    harness.mfh_event_gen.restype = C.c_double
    harness.mfh_event_gen.argtypes = harness.mfh_event.argtypes
    cfg = W.config(proc, seed=13, generator=gen)                  # 4 = q q~ -> t t~, 5 = p p -> t t~ (g g + q q~)
    c, pdf = make_config(cfg)
    assert c.pdf_nf == 11
    P = C.create_string_buffer(harness.mfh_params_size())
    assert harness.mfh_fill_params(C.byref(c), P) == 0
    tab = flavour_slice(harness, P, pdf)
    orc = mfo.Vegas(cfg)
    d = orc.d
    edges = random_grid(d, 50, 31)
    orc.set_grid(edges)
    ref = orc.eval(1, 77, n)
    bins = np.zeros(24, np.int32); ok = np.zeros(1, np.int32); rec = np.zeros(45)
    worst = 0.0
    for i in range(n):
        F = harness.mfh_event_gen(P, edges.ctypes.data, tab.ctypes.data, 1, 77 + i, bins.ctypes.data, ok.ctypes.data, rec.ctypes.data)
        assert list(bins[:d]) == list(ref["bins"][i]) and ok[0] == 1
        np.testing.assert_allclose(rec[:d], ref["x"][i], rtol=1e-14, atol=0)
        np.testing.assert_allclose(rec[18:34].reshape(4, 4), ref["momenta"][i], rtol=1e-10, atol=1e-8)
        np.testing.assert_allclose(rec[43:45], ref["pdf"][i], rtol=1e-12, atol=1e-16)
        worst = max(worst, abs(F / ref["weight"][i] - 1), abs(rec[42] / ref["me2"][i] - 1))
    assert worst < 1e-10, worst
    if gen == 0:                                              # and through the plain entry point
        rec37 = np.zeros(37)
        F = harness.mfh_event(P, edges.ctypes.data, tab.ctypes.data, 1, 77, bins.ctypes.data, ok.ctypes.data, rec37.ctypes.data)
        assert abs(F / ref["weight"][0] - 1) < 1e-10
    bad, _ = make_config(W.config(W.QQ_TT, pdf_xf=W.synthetic_gluon_grid()))     # needs the flavour grid
    assert harness.mfh_fill_params(C.byref(bad), P) == -1
    bad, _ = make_config(W.config(W.GG_TT, pdf_xf=W.synthetic_flavour_grid()))   # and the gluon processes the gluon table
    assert harness.mfh_fill_params(C.byref(bad), P) == -1
