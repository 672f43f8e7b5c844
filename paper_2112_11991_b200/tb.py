"""ctypes binding of libtb (include/tb.h).  Argument marshalling only: every step of the hot path
runs inside the shared library's CUDA kernels.  There is no CPU fallback -- importing this module
raises if libtb.so has not been built (``python -m paper_2112_11991_b200.build``), and every call
raises ``TbError`` when the library reports a failure (e.g. no CUDA device).

The module-level functions carry the C names (tb_plan_create, tb_search_templates, ...) and take /
return plain Python and numpy objects; ``Plan`` is a small RAII convenience over them.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "lib", "libtb.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2112_11991_b200.build` "
                      "(there is no CPU fallback)")
lib = C.CDLL(_LIB_PATH)

TB_OK, TB_ERR_INVALID_ARG, TB_ERR_CUDA, TB_ERR_CUFFT, TB_ERR_NOMEM, TB_ERR_OVERFLOW, TB_ERR_CAPACITY = 0, -1, -2, -3, -4, -5, -6

TB_NOALLOC_MAX_SAMPLES, TB_NOALLOC_SCRATCH_BYTES = 1 << 28, 33024

TEMPLATE_DTYPE = np.dtype([("p_orb_s", "<f8"), ("tau_lts", "<f8"), ("phi0_rad", "<f8"), ("ecc", "<f8"),
                           ("omega_rad", "<f8")])
CANDIDATE_DTYPE = np.dtype([("template_id", "<u4"), ("fold", "<u4"), ("bin", "<u4"), ("power", "<f4"),
                            ("sigma", "<f4"), ("pad", "<u4")])
GROUP_DTYPE = np.dtype([("template_id", "<u4"), ("fold", "<u4"), ("bin", "<u4"), ("power", "<f4"), ("sigma", "<f4"),
                        ("n_peaks", "<u4"), ("n_detections", "<u4"), ("n_templates", "<u4")])
assert TEMPLATE_DTYPE.itemsize == 40 and CANDIDATE_DTYPE.itemsize == 24 and GROUP_DTYPE.itemsize == 32


class PlanOpts(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("device", C.c_int32), ("stream", C.c_void_p),
                ("median_window", C.c_uint32), ("f_min_hz", C.c_double), ("max_candidates", C.c_uint64),
                ("chunk_templates", C.c_uint32), ("series_is_device_ptr", C.c_int32), ("has_fill", C.c_int32),
                ("fill_value", C.c_float), ("enable_timings", C.c_int32), ("fft_path", C.c_int32),
                ("whiten", C.c_int32), ("n_zap_ranges", C.c_uint32), ("zap_ranges", C.c_void_p),
                ("delay_model", C.c_int32), ("interbin_oversample", C.c_int32)]


class BankSpace(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("device", C.c_int32), ("t_obs_s", C.c_double), ("f_max_hz", C.c_double),
                ("p_orb_min_s", C.c_double), ("p_orb_max_s", C.c_double), ("m_pulsar_min", C.c_double),
                ("m_comp_max", C.c_double), ("theta", C.c_double), ("e_max", C.c_double), ("elliptical", C.c_int32),
                ("pad", C.c_int32)]


class Timings(C.Structure):
    _fields_ = [("ms_resample", C.c_double), ("ms_fft", C.c_double), ("ms_spectrum", C.c_double),
                ("ms_normalise", C.c_double), ("ms_hsum", C.c_double), ("ms_total", C.c_double),
                ("n_templates", C.c_uint64), ("n_samples", C.c_uint64), ("n_chunks", C.c_uint64),
                ("chunk_templates", C.c_uint64), ("model_bytes_per_template", C.c_uint64),
                ("n_kernel_launches", C.c_uint64), ("n_median_fallbacks", C.c_uint64),
                ("ms_delay", C.c_double), ("fft_path_used", C.c_uint64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


EXPORTS = ["tb_plan_create", "tb_plan_set_series", "tb_search_templates", "tb_get_candidates", "tb_clear_candidates", "tb_plan_destroy",
           "tb_reduce_candidates", "tb_debug_set_candidates",
           "tb_strerror", "tb_last_error", "tb_get_timings", "tb_debug_resample_indices", "tb_debug_spectrum",
           "tb_debug_resampled", "tb_debug_hsums", "tb_debug_series", "tb_sigma_to_power", "tb_plan_info", "tb_template_knot_log2",
           "tb_bank_density", "tb_bank_generate", "tb_bank_n_templates", "tb_series_mean_noalloc"]

_vp, _u64, _u32 = C.c_void_p, C.c_uint64, C.c_uint32
lib.tb_plan_create.argtypes = [C.POINTER(_vp), _vp, _u64, C.c_double, C.POINTER(PlanOpts)]
lib.tb_plan_set_series.argtypes = [_vp, _vp]
lib.tb_search_templates.argtypes = [_vp, _vp, _u64, _u32, _vp, _u32, C.c_double]
lib.tb_get_candidates.argtypes = [_vp, _vp, _u64, C.POINTER(_u64)]
lib.tb_clear_candidates.argtypes = [_vp]
lib.tb_debug_set_candidates.argtypes = [_vp, _vp, _u64]
lib.tb_reduce_candidates.argtypes = [_vp, C.c_double, _vp, _u64, C.POINTER(_u64), _vp, _u64]
lib.tb_plan_destroy.argtypes = [_vp]
lib.tb_strerror.argtypes = [C.c_int]
lib.tb_strerror.restype = C.c_char_p
lib.tb_last_error.argtypes = [_vp]
lib.tb_last_error.restype = C.c_char_p
lib.tb_get_timings.argtypes = [_vp, C.POINTER(Timings)]
lib.tb_debug_resample_indices.argtypes = [_vp, _vp, _vp]
lib.tb_debug_spectrum.argtypes = [_vp, _vp, _vp, _vp, _vp]
lib.tb_debug_resampled.argtypes = [_vp, _vp, _vp]
lib.tb_debug_hsums.argtypes = [_vp, _vp, _vp]
lib.tb_debug_series.argtypes = [_vp, _vp, C.POINTER(C.c_double)]
lib.tb_sigma_to_power.argtypes = [_u32, C.c_double, C.POINTER(C.c_double)]
lib.tb_plan_info.argtypes = [_vp, C.POINTER(C.c_float), C.POINTER(_u32), C.POINTER(_u32)]
lib.tb_template_knot_log2.argtypes = [_vp, _vp, C.POINTER(C.c_int32)]
lib.tb_bank_density.argtypes = [C.POINTER(BankSpace), _vp, _u64, _vp]
lib.tb_bank_generate.argtypes = [C.POINTER(BankSpace), _vp, _u64, C.c_double, _vp, _u64, C.POINTER(_u64), _vp, C.POINTER(C.c_double)]
lib.tb_bank_n_templates.argtypes = [C.c_double, C.c_double, _u32, C.c_double, C.c_int32, C.POINTER(C.c_double)]
lib.tb_series_mean_noalloc.argtypes = [_vp, _u64, _vp, _vp, C.c_char_p, _u64]
for _name in EXPORTS:
    if _name not in ("tb_strerror", "tb_last_error"):
        getattr(lib, _name).restype = C.c_int


class TbError(RuntimeError):
    def __init__(self, code, detail=""):
        self.code = code
        super().__init__(f"libtb: {lib.tb_strerror(code).decode()} ({code}) {detail}")


def _check(code, plan=None):
    if code != TB_OK:
        detail = lib.tb_last_error(plan).decode() if plan else ""
        raise TbError(code, detail)


def as_templates(templates) -> np.ndarray:
    """float64[K,5] (P_orb, tau, phi0, e, omega) or a structured array -> contiguous tb_template[K]."""
    t = np.asarray(templates)
    if t.dtype == TEMPLATE_DTYPE:
        return np.ascontiguousarray(t).reshape(-1)
    t = np.ascontiguousarray(np.asarray(t, dtype=np.float64).reshape(-1, 5))
    return t.view(TEMPLATE_DTYPE).reshape(-1)


def tb_plan_create(series, n_samples, tsamp_s, *, device=0, stream=None, median_window=0, f_min_hz=0.0,
                   max_candidates=0, chunk_templates=0, series_is_device_ptr=False, fill_value=None,
                   enable_timings=False, fft_path=0, whiten=False, zap_ranges=(), delay_model=0, interbin_oversample=False):
    """series: numpy float32[N] (host) or an integer device address when series_is_device_ptr."""
    o = PlanOpts()
    o.struct_size = C.sizeof(PlanOpts)
    o.device, o.stream = int(device), stream
    o.median_window, o.f_min_hz, o.max_candidates = int(median_window), float(f_min_hz), int(max_candidates)
    o.chunk_templates, o.series_is_device_ptr = int(chunk_templates), int(bool(series_is_device_ptr))
    o.has_fill, o.fill_value = (0, 0.0) if fill_value is None else (1, float(fill_value))
    o.enable_timings = int(bool(enable_timings))
    o.fft_path = int(fft_path)
    o.whiten = int(bool(whiten))
    o.delay_model = int(delay_model)
    o.interbin_oversample = int(bool(interbin_oversample))
    zap = np.ascontiguousarray(np.asarray(zap_ranges, dtype=np.uint32).reshape(-1, 2))
    o.n_zap_ranges, o.zap_ranges = len(zap), (zap.ctypes.data if len(zap) else None)
    if series_is_device_ptr:
        ptr = int(series)
    else:
        series = np.ascontiguousarray(series, dtype=np.float32)
        ptr = series.ctypes.data
    plan = _vp()
    _check(lib.tb_plan_create(C.byref(plan), ptr, int(n_samples), float(tsamp_s), C.byref(o)))
    return plan


def tb_plan_set_series(plan, series, series_is_device_ptr=False):
    """series: numpy float32[N] (host; pinned memory makes the copy asynchronous) or a device address."""
    if series_is_device_ptr:
        ptr = int(series)
    else:
        assert series.dtype == np.float32 and series.flags.c_contiguous
        ptr = series.ctypes.data
    _check(lib.tb_plan_set_series(plan, ptr), plan)


def tb_search_templates(plan, templates, first_template_id=0, folds=(0, 1, 2, 3, 4), sigma_threshold=6.0):
    t = as_templates(templates)
    f = np.ascontiguousarray(folds, dtype=np.uint32)
    _check(lib.tb_search_templates(plan, t.ctypes.data, t.size, int(first_template_id), f.ctypes.data, f.size,
                                   float(sigma_threshold)), plan)


def tb_get_candidates(plan, capacity=None):
    """Returns (candidates structured array sorted by (template, fold, bin), n_total).  Raises
    TbError(TB_ERR_OVERFLOW) if the device buffer overflowed (``.n_total`` on the exception)."""
    n = _u64(0)
    if capacity is None:
        code = lib.tb_get_candidates(plan, None, 0, C.byref(n))
        if code == TB_OK:
            return np.zeros(0, dtype=CANDIDATE_DTYPE), 0
        if code not in (TB_ERR_CAPACITY,):
            _check(code, plan)
        capacity = n.value
    out = np.zeros(int(capacity), dtype=CANDIDATE_DTYPE)
    code = lib.tb_get_candidates(plan, out.ctypes.data, out.size, C.byref(n))
    if code == TB_ERR_OVERFLOW:
        err = TbError(code, lib.tb_last_error(plan).decode())
        err.n_total = n.value
        err.partial = out
        raise err
    _check(code, plan)
    return out[: n.value], n.value


def tb_reduce_candidates(plan, freq_tol_bins=0.0, with_members=False, n_detections=0):
    """Returns (groups structured array in head order, member_of or None).  member_of (uint32 per
    detection, in tb_get_candidates order) needs n_detections = the current candidate count.
    One reduction per call: there are never more groups than detections, so groups_out is sized by the
    detection count (n_detections, or the count tb_get_candidates reports) instead of by a first pass."""
    n = _u64(0)
    n_det = int(n_detections)
    if n_det == 0:
        code = lib.tb_get_candidates(plan, None, 0, C.byref(n))            # count only
        if code not in (TB_OK, TB_ERR_CAPACITY):
            _check(code, plan)
        n_det = int(n.value)
    out = np.zeros(max(n_det, 1), dtype=GROUP_DTYPE)
    members = np.zeros(int(n_detections), dtype=np.uint32) if with_members else None
    _check(lib.tb_reduce_candidates(plan, float(freq_tol_bins), out.ctypes.data, out.size, C.byref(n),
                                    members.ctypes.data if with_members else None, int(n_detections)), plan)
    return out[: n.value].copy(), members


def tb_debug_set_candidates(plan, cands):
    c = np.ascontiguousarray(cands, dtype=CANDIDATE_DTYPE)
    _check(lib.tb_debug_set_candidates(plan, c.ctypes.data, c.size), plan)


def tb_clear_candidates(plan):
    _check(lib.tb_clear_candidates(plan), plan)


def tb_plan_destroy(plan):
    _check(lib.tb_plan_destroy(plan))


def tb_get_timings(plan) -> dict:
    t = Timings()
    _check(lib.tb_get_timings(plan, C.byref(t)), plan)
    return t.as_dict()


def tb_plan_info(plan):
    f, b, k = C.c_float(), _u32(), _u32()
    _check(lib.tb_plan_info(plan, C.byref(f), C.byref(b), C.byref(k)), plan)
    return {"fill_value": np.float32(f.value), "chunk_templates": b.value, "k_lo": k.value}


def tb_template_knot_log2(plan, template) -> int:
    t = as_templates(template)
    v = C.c_int32()
    _check(lib.tb_template_knot_log2(plan, t.ctypes.data, C.byref(v)), plan)
    return v.value


def tb_debug_resample_indices(plan, template, n_samples) -> np.ndarray:
    t = as_templates(template)
    out = np.empty(int(n_samples), dtype=np.int64)
    _check(lib.tb_debug_resample_indices(plan, t.ctypes.data, out.ctypes.data), plan)
    return out


def tb_debug_resampled(plan, template, n_samples) -> np.ndarray:
    t = as_templates(template)
    out = np.empty(int(n_samples), dtype=np.float32)
    _check(lib.tb_debug_resampled(plan, t.ctypes.data, out.ctypes.data), plan)
    return out


def tb_debug_series(plan, n_samples):
    """(the plan's working series float32[N] -- whitened if the plan whitens --, kappa)."""
    x = np.empty(int(n_samples), dtype=np.float32)
    k = C.c_double()
    _check(lib.tb_debug_series(plan, x.ctypes.data, C.byref(k)), plan)
    return x, k.value


def tb_debug_hsums(plan, template, n_samples, oversample=False) -> np.ndarray:
    """float32[5, N/2] (N half bins with interbin_oversample): S_L[k] of every fold and bin through the production harmonic summer."""
    t = as_templates(template)
    out = np.empty((5, int(n_samples) // (1 if oversample else 2)), dtype=np.float32)
    _check(lib.tb_debug_hsums(plan, t.ctypes.data, out.ctypes.data), plan)
    return out


def tb_debug_spectrum(plan, template, n_samples, median_window=1024, oversample=False):
    t = as_templates(template)
    nb = int(n_samples) // (1 if oversample else 2)
    p = np.empty(nb, dtype=np.float32)
    ph = np.empty(nb, dtype=np.float32)
    m = np.empty(nb // int(median_window), dtype=np.float32)
    _check(lib.tb_debug_spectrum(plan, t.ctypes.data, p.ctypes.data, ph.ctypes.data, m.ctypes.data), plan)
    return p, ph, m


def tb_sigma_to_power(fold, sigma) -> float:
    v = C.c_double()
    _check(lib.tb_sigma_to_power(int(fold), float(sigma), C.byref(v)))
    return v.value


class Plan:
    """RAII wrapper: ``with Plan(series, tsamp) as p: p.search(templates); cands, n = p.candidates()``."""

    def __init__(self, series, tsamp_s, n_samples=None, **opts):
        self.n_samples = int(n_samples if n_samples is not None else len(series))
        self.tsamp = float(tsamp_s)
        self.median_window = int(opts.get("median_window", 0) or 1024)
        self.oversample = bool(opts.get("interbin_oversample", False))
        self._series = series                        # keep host/device memory alive
        self.handle = tb_plan_create(series, self.n_samples, tsamp_s, **opts)

    def set_series(self, series, series_is_device_ptr=False):
        self._series = series
        tb_plan_set_series(self.handle, series, series_is_device_ptr)

    def search(self, templates, first_template_id=0, folds=(0, 1, 2, 3, 4), sigma_threshold=6.0):
        tb_search_templates(self.handle, templates, first_template_id, folds, sigma_threshold)

    def candidates(self, capacity=None):
        return tb_get_candidates(self.handle, capacity)

    def reduce(self, freq_tol_bins=0.0, with_members=False, n_detections=0):
        return tb_reduce_candidates(self.handle, freq_tol_bins, with_members, n_detections)

    def debug_set_candidates(self, cands):
        tb_debug_set_candidates(self.handle, cands)

    def clear(self):
        tb_clear_candidates(self.handle)

    def timings(self):
        return tb_get_timings(self.handle)

    def info(self):
        return tb_plan_info(self.handle)

    def knot_log2(self, template):
        return tb_template_knot_log2(self.handle, template)

    def debug_indices(self, template):
        return tb_debug_resample_indices(self.handle, template, self.n_samples)

    def debug_resampled(self, template):
        return tb_debug_resampled(self.handle, template, self.n_samples)

    def debug_series(self):
        return tb_debug_series(self.handle, self.n_samples)

    def debug_hsums(self, template):
        return tb_debug_hsums(self.handle, template, self.n_samples, self.oversample)

    def debug_spectrum(self, template):
        return tb_debug_spectrum(self.handle, template, self.n_samples, self.median_window, self.oversample)

    def close(self):
        if self.handle is not None:
            tb_plan_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---------------------------------------------------------------------------------- template bank (f3)
def bank_space(t_obs_s, f_max_hz, p_orb_min_s, p_orb_max_s, m_pulsar_min=1.4, m_comp_max=8.0, theta=1.0, e_max=0.1,
               elliptical=False, device=0) -> BankSpace:
    s = BankSpace()
    s.struct_size = C.sizeof(BankSpace)
    s.device = int(device)
    s.t_obs_s, s.f_max_hz, s.p_orb_min_s, s.p_orb_max_s = float(t_obs_s), float(f_max_hz), float(p_orb_min_s), float(p_orb_max_s)
    s.m_pulsar_min, s.m_comp_max, s.theta, s.e_max = float(m_pulsar_min), float(m_comp_max), float(theta), float(e_max)
    s.elliptical = int(bool(elliptical))
    return s


def tb_bank_density(space: BankSpace, lam) -> np.ndarray:
    """lam: float64[n, 5] = (tau, Omega, alpha, psi, e) -> rho float64[n]."""
    lam = np.ascontiguousarray(np.asarray(lam, dtype=np.float64).reshape(-1, 5))
    rho = np.zeros(len(lam), dtype=np.float64)
    _check(lib.tb_bank_density(C.byref(space), lam.ctypes.data, len(lam), rho.ctypes.data))
    return rho


def tb_bank_generate(space: BankSpace, uniforms, rho_max, capacity=None):
    """uniforms: float64[n, 6] in [0, 1).  Returns (templates float64[k, 5], rho float64[n], volume estimate)."""
    u = np.ascontiguousarray(np.asarray(uniforms, dtype=np.float64).reshape(-1, 6))
    cap = len(u) if capacity is None else int(capacity)
    out = np.zeros(max(cap, 1), dtype=TEMPLATE_DTYPE)
    rho = np.zeros(len(u), dtype=np.float64)
    n_acc, vol = _u64(0), C.c_double(0.0)
    rc = lib.tb_bank_generate(C.byref(space), u.ctypes.data, len(u), float(rho_max), out.ctypes.data, cap, C.byref(n_acc),
                              rho.ctypes.data, C.byref(vol))
    if rc != TB_OK:
        err = TbError(rc)
        err.n_total = int(n_acc.value)
        raise err
    k = int(n_acc.value)
    return out[:k].view(np.float64).reshape(k, 5).copy(), rho, float(vol.value)


def tb_bank_n_templates(eta, m_star, n_dim, volume, exact=True) -> float:
    out = C.c_double(0.0)
    _check(lib.tb_bank_n_templates(float(eta), float(m_star), int(n_dim), float(volume), int(bool(exact)), C.byref(out)))
    return float(out.value)


def tb_series_mean_noalloc(d_series, n_samples, d_mean_out, stream=None) -> None:
    """Queue the fp64 mean of a device-resident float32 series (the default fill value of a plan) on
    `stream`, for callers that must not allocate device memory: a real-time loop that cannot take the
    device-wide stall of cudaMalloc / cudaFree, or a process whose own pool already holds all GPU memory.

    d_series, d_mean_out: integer device addresses (float32[n_samples] and float64[1]) on the current CUDA
    device; stream: an integer cudaStream_t or None.  Nothing is allocated and nothing is synchronised:
    read d_mean_out after the stream has got there.  n_samples <= TB_NOALLOC_MAX_SAMPLES, else TbError
    (TB_ERR_CAPACITY).  All calls share one static scratch array per GPU: do not let two of them overlap
    on the device.  See include/tb.h."""
    err = C.create_string_buffer(384)
    code = lib.tb_series_mean_noalloc(int(d_series) if d_series else None, int(n_samples),
                                      int(d_mean_out) if d_mean_out else None, stream, err, len(err))
    if code != TB_OK:
        raise TbError(code, err.value.decode())
