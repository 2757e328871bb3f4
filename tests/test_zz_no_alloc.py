"""mf_reduce_weights_noalloc (include/madflow_b200.h; csrc/mf_noalloc.cu): S9 through the ONE entry point that allocates nothing
(static __device__ scratch of 296 x (2 + 18 x 64) doubles) against the existing path (mf_vegas_accumulate: the library-owned,
cudaMalloc'ed per-CTA partial records and, for gg -> tt~g, the on-demand record workspace), on two calls in a row of different
shape, within the tolerance the parity tests use for raw sums (1e-10 relative).  Collected last on purpose (the suite runs with
pytest -x); passes alone in a fresh process and after the other tests."""
import os
import re

import numpy as np
import pytest

from paper_2105_10529_b200 import workloads as W

RTOL_INT = 1e-10
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_noalloc_source_calls_no_allocator():
    """static check (no GPU): the translation unit of the entry point names no allocating CUDA routine, resolves the address of its
    static array with cudaGetSymbolAddress, and the array is the stated size"""
    src = open(os.path.join(ROOT, "paper_2105_10529_b200", "csrc", "mf_noalloc.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)                               # comments may name what the code must not call
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "cudaMemPool", "new ", "malloc("):
        assert banned not in code, banned
    assert "cudaGetSymbolAddress(&p, mf_na_scratch)" in code
    assert re.search(r"static __device__ __align__\(256\) double mf_na_scratch\[MF_NA_MAX_BLOCKS \* MF_NA_ROW\];", code)
    assert "#define MF_NA_MAX_BLOCKS 296" in code and "#define MF_NA_MAX_D 18" in code and "#define MF_NA_MAX_NB 64" in code


def random_grid(d, nb, seed):
    rng = np.random.default_rng(seed)
    w = rng.uniform(0.3, 1.7, size=(d, nb))
    e = np.concatenate([np.zeros((d, 1)), np.cumsum(w, axis=1) / w.sum(axis=1, keepdims=True)], axis=1)
    e[:, -1] = 1.0
    return e


@pytest.mark.gpu
def test_noalloc_reduction_matches_existing_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available()
    from paper_2105_10529_b200 import binding as mf
    mf.lib()
    dev = torch.device("cuda", 0)
    # two calls in a row that share the static scratch: a large gg -> tt~g launch (d = 7, the full grid of 296 CTAs, cut-failed events
    # with weight 0), then a SMALLER gg -> tt~ launch (d = 4, fewer CTAs, shorter records): stale partial records of the first call
    # lie behind and between the second call's and must not be read
    cases = [(W.GG_TTG, 3, 300_001, 1_000, 301_001), (W.GG_TT, 5, 40_003, 0, 40_003), (W.GG_TTG, 3, 300_001, 1_000, 301_001)]
    for proc, seed, n, first, n_total in cases:
        cfg = W.config(proc, seed=seed)
        a, b = mf.Vegas(cfg), mf.Vegas(cfg)
        e = random_grid(a.d, 50, 900 + proc)
        a.set_grid(e); b.set_grid(e)
        # existing path: raw sums of the event range through mf_vegas_accumulate
        b.zero_accum()
        b.vegas_accumulate(first, n, n_total)
        ref, cnt = b.get_accum()
        # new entry point: per-event weights and bins from mf_integrand_eval, reduced without any allocation by the library
        out = a.integrand_eval(0, first, n, debug=True)
        acc = torch.full((2 + a.d * 50,), float("nan"), dtype=torch.float64, device=dev)      # overwritten, not accumulated
        mf.reduce_weights_noalloc(out["weight"].data_ptr(), out["bins"].data_ptr(), n, a.d, 50, n_total, acc.data_ptr())
        got = acc.cpu().numpy()
        assert ref[0] > 0 and np.isfinite(got).all()
        np.testing.assert_allclose(got, ref, rtol=RTOL_INT, atol=1e-300)
        assert int((out["weight"] != 0).sum()) <= cnt[0] <= n
        # accumulate != 0 adds: two halves of the range on top of each other's sums == the whole
        h = n // 2
        acc2 = torch.zeros_like(acc)
        mf.reduce_weights_noalloc(out["weight"].data_ptr(), out["bins"].data_ptr(), h, a.d, 50, n_total, acc2.data_ptr(), accumulate=True)
        mf.reduce_weights_noalloc(out["weight"][h:].data_ptr(), out["bins"][h:].data_ptr(), n - h, a.d, 50, n_total, acc2.data_ptr(), accumulate=True)
        np.testing.assert_allclose(acc2.cpu().numpy(), ref, rtol=RTOL_INT, atol=1e-300)
        # the sums feed the rest of the iteration without an allocation either: set_accum_device + finalize == the existing path's finalize
        buf = torch.cat([acc, torch.tensor([float(cnt[0]), float(cnt[1])], dtype=torch.float64, device=dev)])
        a.set_accum_device(buf.data_ptr())
        ia, ib = a.vegas_finalize(n_total), b.vegas_finalize(n_total)
        assert abs(ia["integral"] / ib["integral"] - 1) < RTOL_INT and abs(ia["sigma"] / ib["sigma"] - 1) < 1e-8
        np.testing.assert_allclose(a.get_grid(), b.get_grid(), rtol=0, atol=1e-11)
    # empty input: zeros (or, accumulating, nothing); sizes beyond the static scratch are rejected with a clear error
    acc = torch.full((2 + 4 * 50,), 7.0, dtype=torch.float64, device=dev)
    mf.reduce_weights_noalloc(0, 0, 0, 4, 50, 10.0, acc.data_ptr(), accumulate=True)
    assert bool((acc == 7.0).all())
    mf.reduce_weights_noalloc(0, 0, 0, 4, 50, 10.0, acc.data_ptr())
    assert bool((acc == 0.0).all())
    w = torch.ones(10, dtype=torch.float64, device=dev); bn = torch.zeros((10, 19), dtype=torch.uint8, device=dev)
    for d, nb in ((19, 50), (7, 65), (0, 50)):
        with pytest.raises(mf.MfError) as err:
            mf.reduce_weights_noalloc(w.data_ptr(), bn.data_ptr(), 10, d, nb, 10.0, acc.data_ptr())
        assert err.value.code == mf.MF_EINVAL and "18" in str(err.value) and "64" in str(err.value)
    with pytest.raises(mf.MfError):
        mf.reduce_weights_noalloc(w.data_ptr(), bn.data_ptr(), 10, 4, 50, 10.0, 0)            # null output
