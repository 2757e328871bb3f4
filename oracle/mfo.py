"""ctypes binding of the ORACLE (oracle/libmfo.so).  Test infrastructure, NOT the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the product package (paper_2105_10529_b200).
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "libmfo.so")


def build(force=False):
    """Compile oracle/libmfo.so with g++ (building the checker is not using it)."""
    srcs = [os.path.join(_HERE, f) for f in ("mfo_core.cpp", "mfo_amp.cpp", "mfo_amp2q.cpp", "mfo_integrand.cpp", "mfo.h")]
    if (not force and os.path.exists(_LIB)
            and all(os.path.getmtime(_LIB) >= os.path.getmtime(s) for s in srcs)):
        return _LIB
    subprocess.check_call(["make", "-C", _HERE, "-B", "libmfo.so"], stdout=subprocess.DEVNULL)
    return _LIB


class Config(C.Structure):
    _fields_ = [("process", C.c_int32), ("seed", C.c_uint64), ("n_bins", C.c_uint32),
                ("alpha_damp", C.c_double), ("sqrt_s", C.c_double), ("m_top", C.c_double),
                ("alpha_s", C.c_double), ("alpha_em", C.c_double), ("mu_f", C.c_double),
                ("ptmin_g", C.c_double), ("etamax_g", C.c_double), ("drmin_gg", C.c_double),
                ("gev2_to_pb", C.c_double), ("pdf_xf", C.POINTER(C.c_double)),
                ("pdf_nx", C.c_uint32), ("pdf_nq", C.c_uint32), ("pdf_xmin", C.c_double),
                ("pdf_xmax", C.c_double), ("pdf_qmin", C.c_double), ("pdf_qmax", C.c_double),
                ("generator", C.c_uint32), ("pdf_nf", C.c_uint32)]


class EvalOut(C.Structure):
    _fields_ = [("weight", C.c_void_p), ("x", C.c_void_p), ("bins", C.c_void_p), ("momenta", C.c_void_p),
                ("me2", C.c_void_p), ("pdf", C.c_void_p), ("pass_", C.c_void_p)]


class Iter(C.Structure):
    _fields_ = [("integral", C.c_double), ("sigma", C.c_double), ("n_events", C.c_uint64),
                ("n_pass", C.c_uint64), ("n_nonfinite", C.c_uint64)]


class Observable(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_bins", C.c_uint32), ("lo", C.c_double), ("hi", C.c_double)]


class Result(C.Structure):
    _fields_ = [("integral", C.c_double), ("sigma", C.c_double), ("chi2_dof", C.c_double), ("n_iter", C.c_uint32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.mfo_last_error.restype = C.c_char_p
        _lib.mfo_pdf_interp.restype = C.c_double
        _lib.mfo_pdf_interp.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32] + [C.c_double] * 6
        _lib.mfo_w0.restype = C.c_double
        _lib.mfo_w0.argtypes = [C.c_uint32, C.c_double]
        _lib.mfo_x_map.argtypes = [C.c_double] * 4 + [C.c_void_p] * 4
        _lib.mfo_x_map_linear.argtypes = [C.c_double] * 4 + [C.c_void_p] * 4
        _lib.mfo_rambo_classic.argtypes = [C.c_uint32, C.c_double, C.c_void_p, C.c_void_p]
        _lib.mfo_massive_rescale.argtypes = [C.c_uint32, C.c_double] + [C.c_void_p] * 4
        _lib.mfo_phase_space.argtypes = [C.c_uint32, C.c_double] + [C.c_void_p] * 6
        _lib.mfo_me2.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_void_p]
        _lib.mfo_me2_2q.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_void_p]
        _lib.mfo_me2_literal.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_void_p]
        _lib.mfo_jamps.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        _lib.mfo_amp_literal.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p,
                                         C.c_int, C.c_int, C.c_int, C.c_void_p]
        _lib.mfo_cuts.argtypes = [C.c_uint32, C.c_void_p] + [C.c_double] * 5 + [C.c_void_p]
        _lib.mfo_wf_fermion.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_int, C.c_void_p]
        _lib.mfo_wf_vector.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        _lib.mfo_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint32, C.c_void_p]
        _lib.mfo_vegas_map.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.mfo_refine.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_double, C.c_void_p]
        _lib.mfo_combine.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
        _lib.mfo_integrand_eval.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_uint64, C.c_void_p, C.c_int]
        _lib.mfo_vegas_iterate.argtypes = [C.c_void_p, C.c_uint64, C.c_int, C.c_void_p]
        _lib.mfo_vegas_accumulate.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_uint64, C.c_uint64, C.c_int,
                                              C.c_void_p, C.c_void_p]
        _lib.mfo_observable_hist.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_uint64, C.c_uint64, C.c_int,
                                             C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]
        _lib.mfo_vegas_finalize.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p]
        for f in ("mfo_vegas_destroy", "mfo_result", "mfo_get_grid", "mfo_set_grid", "mfo_get_accum", "mfo_ndim"):
            getattr(_lib, f).argtypes = [C.c_void_p] + [C.c_void_p] * (2 if f == "mfo_ndim" else 0 if f == "mfo_vegas_destroy" else 1)
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _check(rc):
    if rc != 0:
        raise RuntimeError("oracle error %d: %s" % (rc, lib().mfo_last_error().decode()))


# ---- single steps ---------------------------------------------------------------------------
def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32); o = np.zeros(4, np.uint32)
    lib().mfo_philox4x32_10(_p(c), _p(k), _p(o)); return o


def uniforms(seed, iteration, event, d):
    u = np.zeros(d); lib().mfo_uniforms(seed, iteration, event, d, _p(u)); return u


def vegas_map(edges, u):
    edges = _f64(edges); d, nb1 = edges.shape; u = _f64(u)
    x = np.zeros(d); b = np.zeros(d, np.uint8); j = np.zeros(1)
    lib().mfo_vegas_map(_p(edges), d, nb1 - 1, _p(u), _p(x), _p(b), _p(j)); return x, b, j[0]


def refine(edges, H, alpha):
    edges = _f64(edges); H = _f64(H); d, nb1 = edges.shape; out = np.zeros_like(edges)
    lib().mfo_refine(_p(edges), _p(H), d, nb1 - 1, alpha, _p(out)); return out


def combine(I, sig):
    I = _f64(I); sig = _f64(sig); r = Result()
    lib().mfo_combine(_p(I), _p(sig), len(I), C.byref(r)); return r.integral, r.sigma, r.chi2_dof


def x_map(y0, y1, s, shat_min):
    o = [C.c_double() for _ in range(4)]
    lib().mfo_x_map(y0, y1, s, shat_min, *[C.byref(v) for v in o]); return tuple(v.value for v in o)


def x_map_linear(y0, y1, s, shat_min):
    o = [C.c_double() for _ in range(4)]
    lib().mfo_x_map_linear(y0, y1, s, shat_min, *[C.byref(v) for v in o]); return tuple(v.value for v in o)


def rambo_classic(n, shat, rs):
    rs = _f64(rs); p0 = np.zeros((n, 4)); lib().mfo_rambo_classic(n, shat, _p(rs), _p(p0)); return p0


def massive_rescale(n, shat, masses, p0):
    masses = _f64(masses); p0 = _f64(p0); k = np.zeros((n, 4)); o2 = np.zeros(2)
    steps = lib().mfo_massive_rescale(n, shat, _p(masses), _p(p0), _p(k), _p(o2))
    return dict(k=k, Wm=o2[0], xi=o2[1], steps=steps)


def phase_space(n, shat, masses, rs):
    masses = _f64(masses); rs = _f64(rs); p0 = np.zeros((n, 4)); k = np.zeros((n, 4)); Mi = np.zeros(n); o3 = np.zeros(3)
    steps = lib().mfo_phase_space(n, shat, _p(masses), _p(rs), _p(p0), _p(k), _p(Mi), _p(o3))
    return dict(p0=p0, k=k, Mint=Mi, W0=o3[0], Wm=o3[1], xi=o3[2], steps=steps)


def w0(n, shat):
    return lib().mfo_w0(n, shat)


def pdf_interp(xf, xmin, xmax, qmin, qmax, x, q2):
    xf = _f64(xf); return lib().mfo_pdf_interp(_p(xf), xf.shape[0], xf.shape[1], xmin, xmax, qmin, qmax, x, q2)


def wf_fermion(kind, p, m, lam):
    p = _f64(p); o = np.zeros(8); lib().mfo_wf_fermion(kind, _p(p), m, lam, _p(o)); return o[0::2] + 1j * o[1::2]


def wf_vector(p, lam):
    p = _f64(p); o = np.zeros(8); lib().mfo_wf_vector(_p(p), lam, _p(o)); return o[0::2] + 1j * o[1::2]


def gamma():
    o = np.zeros(128); lib().mfo_gamma(_p(o)); o = o.reshape(4, 4, 4, 2); return o[..., 0] + 1j * o[..., 1]


def su3():
    T = np.zeros(8 * 9 * 2); f = np.zeros(512); lib().mfo_su3(_p(T), _p(f))
    T = T.reshape(8, 3, 3, 2); return T[..., 0] + 1j * T[..., 1], f.reshape(8, 8, 8)


def colour_matrix(ng):
    nf = {2: 2, 3: 6, 4: 24}[ng]; num = np.zeros((nf, nf)); den = np.zeros(1)
    _check(lib().mfo_colour_matrix(ng, _p(num), _p(den))); return num, den[0]


def diagram_counts(ng):
    a, b, c = C.c_uint32(), C.c_uint32(), C.c_uint32()
    _check(lib().mfo_diagram_counts(ng, C.byref(a), C.byref(b), C.byref(c))); return a.value, b.value, c.value


def me2(process, mom, m_top=173.0, alpha_s=0.118, alpha_em=1 / 132.5):
    mom = _f64(mom); o = np.zeros(1); _check(lib().mfo_me2(process, _p(mom), m_top, alpha_s, alpha_em, _p(o))); return o[0]


def me2_2q(process, mom, m_top=173.0, alpha_s=0.118, ward=0):
    """|M|^2 of q q~ -> t t~ g (process 6) / q g -> t t~ q (process 7) for mom = [pa, pb, k1, k2, k3]; ward: e -> K"""
    mom = _f64(mom); o = np.zeros(1); _check(lib().mfo_me2_2q(process, _p(mom), m_top, alpha_s, ward, _p(o))); return o[0]


def me2_literal(process, mom, m_top=173.0, alpha_s=0.118, hel_only=-1):
    mom = _f64(mom); o = np.zeros(1); _check(lib().mfo_me2_literal(process, _p(mom), m_top, alpha_s, hel_only, _p(o))); return o[0]


def jamps(process, mom, hel, m_top=173.0, alpha_s=0.118, ward_leg=-1):
    mom = _f64(mom); hel = np.asarray(hel, dtype=np.int32); nf = {1: 2, 2: 6, 3: 24}[process]
    j = np.zeros(2 * nf); m = np.zeros(1)
    _check(lib().mfo_jamps(process, _p(mom), m_top, alpha_s, _p(hel), ward_leg, _p(j), _p(m)))
    return j[0::2] + 1j * j[1::2], m[0]


def amp_literal(process, mom, hel, col_g, c3, c4, m_top=173.0, alpha_s=0.118, ward_leg=-1):
    mom = _f64(mom); hel = np.asarray(hel, dtype=np.int32); col = np.asarray(col_g, dtype=np.int32); o = np.zeros(2)
    _check(lib().mfo_amp_literal(process, _p(mom), m_top, alpha_s, _p(hel), _p(col), c3, c4, ward_leg, _p(o)))
    return o[0] + 1j * o[1]


def cuts(kg, x1, x2, ptmin, etamax, drmin):
    kg = _f64(kg); ng = kg.shape[0]; obs = np.zeros(2 * ng + 1)
    ok = lib().mfo_cuts(ng, _p(kg), x1, x2, ptmin, etamax, drmin, _p(obs)); return bool(ok), obs


def max_threads():
    return lib().mfo_max_threads()


# ---- the path -------------------------------------------------------------------------------
class Vegas:
    """Host-memory twin of the product's handle (mfo_vegas_*)."""

    def __init__(self, cfg: dict):
        self._pdf = _f64(cfg["pdf_xf"]) if cfg.get("pdf_xf") is not None else None
        c = Config()
        for k in ("process", "seed", "n_bins", "alpha_damp", "sqrt_s", "m_top", "alpha_s", "alpha_em", "mu_f",
                  "ptmin_g", "etamax_g", "drmin_gg", "gev2_to_pb", "pdf_xmin", "pdf_xmax", "pdf_qmin", "pdf_qmax"):
            setattr(c, k, cfg[k])
        c.generator = int(cfg.get("generator", 0))
        if self._pdf is not None:
            c.pdf_xf = self._pdf.ctypes.data_as(C.POINTER(C.c_double)); c.pdf_nx, c.pdf_nq = self._pdf.shape[-2:]
            c.pdf_nf = self._pdf.shape[0] if self._pdf.ndim == 3 else 1
        self._h = C.c_void_p()
        _check(lib().mfo_vegas_create(C.byref(c), C.byref(self._h)))
        d, nf = C.c_uint32(), C.c_uint32(); lib().mfo_ndim(self._h, C.byref(d), C.byref(nf))
        self.d, self.n_final, self.n_bins = d.value, nf.value, cfg["n_bins"]

    def __del__(self):
        if getattr(self, "_h", None):
            lib().mfo_vegas_destroy(self._h); self._h = None

    def eval(self, iteration, first, n, n_threads=1, debug=True):
        d, nl = self.d, 2 + self.n_final
        out = dict(weight=np.zeros(n))
        if debug:
            out.update(x=np.zeros((n, d)), bins=np.zeros((n, d), np.uint8), momenta=np.zeros((n, nl, 4)),
                       me2=np.zeros(n), pdf=np.zeros((n, 2)), pass_=np.zeros(n, np.uint8))
        eo = EvalOut(**{k: v.ctypes.data for k, v in out.items()})
        _check(lib().mfo_integrand_eval(self._h, iteration, first, n, C.byref(eo), n_threads)); return out

    def iterate(self, n, n_threads=1):
        it = Iter(); _check(lib().mfo_vegas_iterate(self._h, n, n_threads, C.byref(it)))
        return dict(integral=it.integral, sigma=it.sigma, n_events=it.n_events, n_pass=it.n_pass, n_nonfinite=it.n_nonfinite)

    def accumulate(self, iteration, first, n, n_total, n_threads=1, acc=None):
        acc = np.zeros(2 + self.d * self.n_bins) if acc is None else acc; cnt = np.zeros(2, np.uint64)
        _check(lib().mfo_vegas_accumulate(self._h, iteration, first, n, n_total, n_threads, _p(acc), _p(cnt))); return acc, cnt

    def finalize(self, acc, n_total, n_pass=0, n_nonfinite=0):
        acc = _f64(acc); it = Iter(); _check(lib().mfo_vegas_finalize(self._h, _p(acc), n_total, int(n_pass), int(n_nonfinite), C.byref(it)))
        return dict(integral=it.integral, sigma=it.sigma, n_events=it.n_events, n_pass=it.n_pass, n_nonfinite=it.n_nonfinite)

    def result(self):
        r = Result(); _check(lib().mfo_result(self._h, C.byref(r)))
        return dict(integral=r.integral, sigma=r.sigma, chi2_dof=r.chi2_dof, n_iter=r.n_iter)

    def get_grid(self):
        e = np.zeros((self.d, self.n_bins + 1)); _check(lib().mfo_get_grid(self._h, _p(e))); return e

    def set_grid(self, e):
        e = _f64(e); _check(lib().mfo_set_grid(self._h, _p(e)))

    def observable_hist(self, iteration, first, n, n_total, obs, n_threads=1):
        """obs: list of (kind, n_bins, lo, hi); returns a list of (sum, sum2) arrays of n_bins + 2 slots
        (the last two: underflow, overflow) for the events [first, first+n) of `iteration` on the current grid"""
        arr = (Observable * len(obs))(*[Observable(int(k), int(nb), float(lo), float(hi)) for k, nb, lo, hi in obs])
        tot = sum(int(o[1]) + 2 for o in obs)
        s1, s2 = np.zeros(tot), np.zeros(tot)
        _check(lib().mfo_observable_hist(self._h, iteration, first, n, n_total, n_threads, arr, len(obs), _p(s1), _p(s2)))
        out, off = [], 0
        for o in obs:
            m = int(o[1]) + 2
            out.append((s1[off:off + m].copy(), s2[off:off + m].copy())); off += m
        return out

    def get_accum(self):
        a = np.zeros(2 + self.d * self.n_bins); _check(lib().mfo_get_accum(self._h, _p(a))); return a
