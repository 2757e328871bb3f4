"""Thin ctypes binding of the C-ABI library (include/madflow_b200.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of libmadflow_b200.so; PyTorch is used by callers
for device memory and streams (tensors' data_ptr(), torch.cuda.current_stream()).  There is no CPU
path: if the library is missing or no CUDA device is present the calls raise.
"""
import ctypes as C
import os
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmadflow_b200.so")

MF_OK, MF_EINVAL, MF_ENOMEM, MF_ECUDA, MF_ESTATE, MF_EUNSUPPORTED = 0, -1, -2, -3, -4, -5
EXPORTS = ["mf_vegas_create", "mf_vegas_destroy", "mf_ndim", "mf_integrand_eval", "mf_vegas_iterate",
           "mf_vegas_accumulate", "mf_get_accum", "mf_set_accum", "mf_vegas_finalize", "mf_result",
           "mf_get_iterations", "mf_get_grid", "mf_set_grid", "mf_set_launch", "mf_me_flops",
           "mf_fp64_peak", "mf_last_kernel_ms", "mf_last_error", "mf_set_path", "mf_last_stage_ms",
           "mf_set_observables", "mf_get_observables", "mf_accum_len", "mf_zero_accum", "mf_get_accum_device",
           "mf_set_accum_device", "mf_stage_ms_sum", "mf_me_flops_bounds", "mf_reduce_weights_noalloc",
           "mf_state_size", "mf_get_state", "mf_set_state"]


class MfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("madflow_b200 error %d: %s" % (code, msg))
        self.code = code


class Config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("process", C.c_int32), ("precision", C.c_int32),
                ("device", C.c_int32), ("seed", C.c_uint64), ("n_bins", C.c_uint32), ("generator", C.c_uint32),
                ("alpha_damp", C.c_double), ("sqrt_s", C.c_double), ("m_top", C.c_double),
                ("alpha_s", C.c_double), ("alpha_em", C.c_double), ("mu_f", C.c_double),
                ("ptmin_g", C.c_double), ("etamax_g", C.c_double), ("drmin_gg", C.c_double),
                ("gev2_to_pb", C.c_double), ("pdf_xf", C.POINTER(C.c_double)),
                ("pdf_nx", C.c_uint32), ("pdf_nq", C.c_uint32), ("pdf_xmin", C.c_double),
                ("pdf_xmax", C.c_double), ("pdf_qmin", C.c_double), ("pdf_qmax", C.c_double),
                ("pdf_nf", C.c_uint32), ("reserved1", C.c_uint32)]


class EvalOut(C.Structure):
    _fields_ = [("weight", C.c_void_p), ("x", C.c_void_p), ("bins", C.c_void_p), ("momenta", C.c_void_p),
                ("me2", C.c_void_p), ("pdf", C.c_void_p), ("pass_", C.c_void_p)]


class Iter(C.Structure):
    _fields_ = [("integral", C.c_double), ("sigma", C.c_double), ("n_events", C.c_uint64),
                ("n_pass", C.c_uint64), ("n_nonfinite", C.c_uint64), ("kernel_ms", C.c_float)]


class Result(C.Structure):
    _fields_ = [("integral", C.c_double), ("sigma", C.c_double), ("chi2_dof", C.c_double), ("n_iter", C.c_uint32)]


def make_config(cfg: dict):
    """dict (paper_2105_10529_b200.workloads.config) -> (Config, keep-alive host PDF array)"""
    c = Config()
    c.struct_size = C.sizeof(Config)
    for k in ("process", "precision", "device", "seed", "n_bins", "alpha_damp", "sqrt_s", "m_top", "alpha_s",
              "alpha_em", "mu_f", "ptmin_g", "etamax_g", "drmin_gg", "gev2_to_pb", "pdf_xmin", "pdf_xmax",
              "pdf_qmin", "pdf_qmax"):
        setattr(c, k, cfg[k])
    c.generator = int(cfg.get("generator", 0))
    pdf = None
    if cfg.get("pdf_xf") is not None:
        pdf = np.ascontiguousarray(cfg["pdf_xf"], dtype=np.float64)
        c.pdf_xf = pdf.ctypes.data_as(C.POINTER(C.c_double))
        c.pdf_nx, c.pdf_nq = pdf.shape[-2:]
        c.pdf_nf = pdf.shape[0] if pdf.ndim == 3 else 1
    return c, pdf


_lib = None


def lib():
    """Load libmadflow_b200.so (built in-tree by __graft_entry__.build()); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("CUDA library %s is missing: run `python -c 'import __graft_entry__ as g; g.build()'`"
                               " (there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        L.mf_last_error.restype = C.c_char_p
        vp, u32, u64 = C.c_void_p, C.c_uint32, C.c_uint64
        L.mf_vegas_create.argtypes = [C.POINTER(Config), C.POINTER(vp)]
        L.mf_vegas_destroy.argtypes = [vp]
        L.mf_ndim.argtypes = [vp, C.POINTER(u32), C.POINTER(u32)]
        L.mf_integrand_eval.argtypes = [vp, u32, u64, u64, C.POINTER(EvalOut), vp]
        L.mf_vegas_iterate.argtypes = [vp, u64, vp, C.POINTER(Iter)]
        L.mf_vegas_accumulate.argtypes = [vp, u64, u64, u64, vp]
        L.mf_get_accum.argtypes = [vp, vp, vp]
        L.mf_set_accum.argtypes = [vp, vp, vp]
        L.mf_vegas_finalize.argtypes = [vp, u64, vp, C.POINTER(Iter)]
        L.mf_result.argtypes = [vp, C.POINTER(Result)]
        L.mf_get_iterations.argtypes = [vp, vp, u32, C.POINTER(u32)]
        L.mf_get_grid.argtypes = [vp, vp]
        L.mf_set_grid.argtypes = [vp, vp]
        L.mf_set_launch.argtypes = [vp, u32, u32]
        L.mf_set_path.argtypes = [vp, C.c_int32]
        L.mf_set_observables.argtypes = [vp, vp, u32]
        L.mf_get_observables.argtypes = [vp, vp, vp, C.POINTER(u32)]
        L.mf_accum_len.argtypes = [vp, C.POINTER(u32)]
        L.mf_zero_accum.argtypes = [vp, vp]
        L.mf_get_accum_device.argtypes = [vp, vp, vp]
        L.mf_set_accum_device.argtypes = [vp, vp, vp]
        L.mf_last_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.mf_stage_ms_sum.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(u32)]
        L.mf_me_flops_bounds.argtypes = [vp, C.POINTER(u64), C.POINTER(u64)]
        L.mf_state_size.argtypes = [vp, C.POINTER(u64)]
        L.mf_get_state.argtypes = [vp, vp, u64]
        L.mf_set_state.argtypes = [vp, vp, u64]
        L.mf_reduce_weights_noalloc.argtypes = [C.c_int32, vp, vp, u64, u32, u32, C.c_double, C.c_int32, vp, vp]
        L.mf_me_flops.argtypes = [vp, C.POINTER(u64), C.POINTER(u64), C.POINTER(u64)]
        L.mf_last_kernel_ms.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.mf_fp64_peak.argtypes = [C.c_int32, C.c_double, C.POINTER(C.c_double)]
        _lib = L
    return _lib


class Observable(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_bins", C.c_uint32), ("lo", C.c_double), ("hi", C.c_double)]


OBS_PT_1, OBS_PT_2, OBS_M_12, OBS_PT_3 = 0, 1, 2, 3


def _check(rc):
    if rc != 0:
        raise MfError(rc, lib().mf_last_error().decode())


def _stream_ptr(stream, device=None):
    """cudaStream_t of `stream` (an int / torch stream pointer), default: torch's current stream ON THE HANDLE'S DEVICE"""
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)
    return C.c_void_p(int(getattr(stream, "cuda_stream", stream)))


class Vegas:
    """mf_vegas_t handle.  Methods carry the names of the C calls."""

    def __init__(self, cfg: dict):
        self._cfg, self._pdf = make_config(cfg)
        self._h = C.c_void_p()
        _check(lib().mf_vegas_create(C.byref(self._cfg), C.byref(self._h)))
        d, nf = C.c_uint32(), C.c_uint32()
        _check(lib().mf_ndim(self._h, C.byref(d), C.byref(nf)))
        self.d, self.n_final, self.n_bins = d.value, nf.value, cfg["n_bins"]
        self.device = cfg.get("device", 0)

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:    # at interpreter shutdown the module globals may be gone already
            _lib.mf_vegas_destroy(self._h)
            self._h = None

    __del__ = close

    def integrand_eval(self, iteration, first_event, n_events, debug=False, stream=None):
        """mf_integrand_eval: returns a dict of torch tensors on the handle's device"""
        import torch
        dev = torch.device("cuda", self.device)
        n, d, nl = int(n_events), self.d, 2 + self.n_final
        out = dict(weight=torch.empty(n, dtype=torch.float64, device=dev))
        if debug:
            out.update(x=torch.empty((n, d), dtype=torch.float64, device=dev),
                       bins=torch.empty((n, d), dtype=torch.uint8, device=dev),
                       momenta=torch.empty((n, nl, 4), dtype=torch.float64, device=dev),
                       me2=torch.empty(n, dtype=torch.float64, device=dev),
                       pdf=torch.empty((n, 2), dtype=torch.float64, device=dev),
                       pass_=torch.empty(n, dtype=torch.uint8, device=dev))
        eo = EvalOut(**{k: (v.data_ptr() if n else None) for k, v in out.items()})
        with torch.cuda.device(dev):
            _check(lib().mf_integrand_eval(self._h, iteration, int(first_event), n, C.byref(eo), _stream_ptr(stream, self.device)))
        return out

    def integrand_eval_into(self, iteration, first_event, n_events, weight_ptr, stream=None):
        """mf_integrand_eval writing only the weights to a caller-owned device pointer"""
        eo = EvalOut(weight=weight_ptr)
        _check(lib().mf_integrand_eval(self._h, iteration, int(first_event), int(n_events), C.byref(eo), _stream_ptr(stream, self.device)))

    def vegas_iterate(self, n_events, stream=None, sync=True):
        it = Iter()
        _check(lib().mf_vegas_iterate(self._h, int(n_events), _stream_ptr(stream, self.device), C.byref(it) if sync else None))
        return _iter_dict(it) if sync else None

    def vegas_accumulate(self, first_event, n_events, n_total, stream=None):
        _check(lib().mf_vegas_accumulate(self._h, int(first_event), int(n_events), int(n_total), _stream_ptr(stream, self.device)))

    def accum_len(self):
        n = C.c_uint32()
        _check(lib().mf_accum_len(self._h, C.byref(n)))
        return n.value

    def set_observables(self, obs):
        """obs: list of (kind, n_bins, lo, hi), kinds OBS_PT_1 / OBS_PT_2 / OBS_M_12 / OBS_PT_3; [] turns them off"""
        arr = (Observable * max(1, len(obs)))(*[Observable(int(k), int(nb), float(lo), float(hi)) for k, nb, lo, hi in obs])
        _check(lib().mf_set_observables(self._h, C.cast(arr, C.c_void_p), len(obs)))
        self._obs = list(obs)

    def get_observables(self):
        """[(sum, sum2)] per observable, each n_bins + 2 slots (last two: underflow, overflow), summed over the
        iterations since set_observables; and the number of those iterations"""
        n = len(self._obs)
        s1 = np.zeros((n, 64)); s2 = np.zeros((n, 64)); it = C.c_uint32()
        _check(lib().mf_get_observables(self._h, s1.ctypes.data, s2.ctypes.data, C.byref(it)))
        out = []
        for o, (k, nb, lo, hi) in enumerate(self._obs):
            pick = list(range(int(nb))) + [62, 63]
            out.append((s1[o, pick].copy(), s2[o, pick].copy()))
        return out, it.value

    def get_accum(self):
        acc = np.zeros(self.accum_len()); cnt = np.zeros(2, np.uint64)
        _check(lib().mf_get_accum(self._h, acc.ctypes.data, cnt.ctypes.data))
        return acc, cnt

    def set_accum(self, acc, counts):
        acc = np.ascontiguousarray(acc, dtype=np.float64); cnt = np.ascontiguousarray(counts, dtype=np.uint64)
        _check(lib().mf_set_accum(self._h, acc.ctypes.data, cnt.ctypes.data))

    def zero_accum(self, stream=None):
        _check(lib().mf_zero_accum(self._h, _stream_ptr(stream, self.device)))

    def get_accum_device(self, dev_ptr, stream=None):
        """raw sums + the two counters (as doubles) into a device buffer of accum_len() + 2 doubles; enqueue only"""
        _check(lib().mf_get_accum_device(self._h, C.c_void_p(int(dev_ptr)), _stream_ptr(stream, self.device)))

    def set_accum_device(self, dev_ptr, stream=None):
        _check(lib().mf_set_accum_device(self._h, C.c_void_p(int(dev_ptr)), _stream_ptr(stream, self.device)))

    def vegas_finalize(self, n_total, stream=None, sync=True):
        it = Iter()
        _check(lib().mf_vegas_finalize(self._h, int(n_total), _stream_ptr(stream, self.device), C.byref(it) if sync else None))
        return _iter_dict(it) if sync else None

    def result(self):
        r = Result()
        _check(lib().mf_result(self._h, C.byref(r)))
        return dict(integral=r.integral, sigma=r.sigma, chi2_dof=r.chi2_dof, n_iter=r.n_iter)

    def get_iterations(self, max_iter=1024):
        arr = (Iter * max_iter)(); n = C.c_uint32()
        _check(lib().mf_get_iterations(self._h, C.cast(arr, C.c_void_p), max_iter, C.byref(n)))
        return [_iter_dict(arr[i]) for i in range(n.value)]

    def get_grid(self):
        e = np.zeros((self.d, self.n_bins + 1))
        _check(lib().mf_get_grid(self._h, e.ctypes.data))
        return e

    def set_grid(self, edges):
        e = np.ascontiguousarray(edges, dtype=np.float64)
        assert e.shape == (self.d, self.n_bins + 1)
        _check(lib().mf_set_grid(self._h, e.ctypes.data))

    def set_launch(self, blocks_per_sm=0, threads_per_block=0):
        _check(lib().mf_set_launch(self._h, blocks_per_sm, threads_per_block))

    def set_path(self, staged):
        _check(lib().mf_set_path(self._h, 1 if staged else 0))

    def last_stage_ms(self):
        ms = (C.c_float * 3)()
        _check(lib().mf_last_stage_ms(self._h, ms))
        return dict(front=ms[0], me=ms[1], reduce=ms[2])

    def last_kernel_ms(self):
        a, b = C.c_float(), C.c_float()
        _check(lib().mf_last_kernel_ms(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def get_state(self):
        """checkpoint of the integrator state (grid, iteration records, counter, observable sums) as bytes"""
        n = C.c_uint64()
        _check(lib().mf_state_size(self._h, C.byref(n)))
        buf = (C.c_char * n.value)()
        _check(lib().mf_get_state(self._h, buf, n.value))
        return bytes(buf)

    def set_state(self, blob):
        """resume from a checkpoint taken on a handle of the same configuration"""
        _check(lib().mf_set_state(self._h, C.c_char_p(blob), len(blob)))

    def stage_ms_sum(self):
        """sums of the stage times over all staged launches since the previous call, and their number"""
        ms = (C.c_float * 3)(); n = C.c_uint32()
        _check(lib().mf_stage_ms_sum(self._h, ms, C.byref(n)))
        return dict(front=ms[0], me=ms[1], reduce=ms[2]), n.value

    def me_flops_bounds(self):
        lo, ex = C.c_uint64(), C.c_uint64()
        _check(lib().mf_me_flops_bounds(self._h, C.byref(lo), C.byref(ex)))
        return dict(min=lo.value, executed=ex.value)

    def me_flops(self):
        a, m, f = C.c_uint64(), C.c_uint64(), C.c_uint64()
        _check(lib().mf_me_flops(self._h, C.byref(a), C.byref(m), C.byref(f)))
        return dict(add=a.value, mul=m.value, fma=f.value, flops=a.value + m.value + 2 * f.value)


def _iter_dict(it):
    return dict(integral=it.integral, sigma=it.sigma, n_events=it.n_events, n_pass=it.n_pass,
                n_nonfinite=it.n_nonfinite, kernel_ms=it.kernel_ms)


def reduce_weights_noalloc(weight_ptr, bins_ptr, n_events, d, n_bins, n_total, acc_ptr, accumulate=False, device=0, stream=None):
    """mf_reduce_weights_noalloc: raw sums (sum t, sum t^2, d x n_bins histogram) of per-event weights and bins into a caller-owned
    device buffer of 2 + d*n_bins doubles; allocates nothing (static device scratch); enqueue only"""
    _check(lib().mf_reduce_weights_noalloc(int(device), C.c_void_p(int(weight_ptr)), C.c_void_p(int(bins_ptr)), int(n_events), int(d),
                                           int(n_bins), float(n_total), 1 if accumulate else 0, C.c_void_p(int(acc_ptr)),
                                           _stream_ptr(stream, device)))


def fp64_peak(device=0, seconds=0.5):
    v = C.c_double()
    _check(lib().mf_fp64_peak(device, seconds, C.byref(v)))
    return v.value
