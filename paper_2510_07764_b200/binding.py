"""ctypes binding of libppm_b200.so (include/ppm.h).  Same names as the C entry points, argument
marshalling only.  torch tensors are passed as raw device pointers; the stream is torch's current
stream at construction."""
import ctypes as C
import os

import numpy as np

from . import _build

EMISSION_BLACKBODY, EMISSION_TABLE_CUBIC, EMISSION_TABLE_MIXED, EMISSION_TABLE_CUBIC_LINEDGE = 0, 1, 2, 3
EMISSION_TABLE_CUBIC_CLIP = 4

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_u8p = C.POINTER(C.c_uint8)
_vp = C.c_void_p


class PPMError(RuntimeError):
    pass


class _Config(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_spots", "n_theta", "n_phi", "n_phase", "n_fp", "n_energy", "emission",
                                         "precision", "oblate", "max_batch", "device", "mesh", "beaming",
                                         "scratch_mb", "phase_interp", "interp_domain")]


# every symbol include/ppm.h declares: name -> (restype, argtypes)
EXPORTS = {
    "ppm_create": (C.c_int, [C.POINTER(_Config), _dp, _vp, C.POINTER(_vp)]),
    "ppm_destroy": (C.c_int, [_vp]),
    "ppm_load_atmosphere": (C.c_int, [_vp, _dp, C.c_int, _dp, C.c_int, _dp, C.c_int, _dp, C.c_int, _vp, C.c_int]),
    "ppm_set_response": (C.c_int, [_vp, C.c_int, C.c_int, _ip, _vp, C.c_int, _dp]),
    "ppm_evaluate": (C.c_int, [_vp, _vp, C.c_int, _vp, _vp]),
    "ppm_evaluate_map": (C.c_int, [_vp, _vp, _vp, C.c_int, _vp, _vp]),
    "ppm_fold_response": (C.c_int, [_vp, _vp, _vp, C.c_int, _vp]),
    "ppm_loglike": (C.c_int, [_vp, _vp, C.c_int, _vp, _vp, C.c_double, _vp]),
    "ppm_evaluate_host": (C.c_int, [_vp, _dp, C.c_int, _dp, _ip]),
    "ppm_loglike_host": (C.c_int, [_vp, _dp, C.c_int, _vp, _vp, C.c_double, _dp, _ip]),
    "ppm_chain_create": (C.c_int, [_vp, C.c_int, _dp, _dp, _dp, _dp, _dp, C.c_uint64, _vp, _vp, C.c_double]),
    "ppm_chain_run": (C.c_int, [_vp, C.c_int]),
    "ppm_chain_read": (C.c_int, [_vp, _dp, _dp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]),
    "ppm_debug_rows": (C.c_int, [_vp, C.c_int, _dp]),
    "ppm_debug_mask": (C.c_int, [_vp, C.c_int, _u8p]),
    "ppm_debug_template": (C.c_int, [_vp, C.c_int, _dp]),
    "ppm_debug_lookup": (C.c_int, [_vp, C.c_int, C.c_int, _dp, C.c_int, _dp, _dp, _dp]),
    "ppm_launch_count": (C.c_int64, [_vp]),
    "ppm_n_fp": (C.c_int, [_vp]),
    "ppm_sub_batch": (C.c_int, [_vp]),
    "ppm_uniform_energy": (C.c_int, [_vp]),
    "ppm_profile_enable": (C.c_int, [_vp, C.c_int]),
    "ppm_profile_read": (C.c_int, [_vp, _dp, C.POINTER(C.c_int64), _dp]),
    "ppm_measure_fp64_peak": (C.c_int, [C.c_int, _dp]),
    "ppm_last_error": (C.c_char_p, []),
    "ppm_loglike_noalloc": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int, _vp, _vp, C.c_double, _vp, _vp]),
    "ppm_loglike_noalloc_error": (C.c_char_p, []),
}

_lib = None


def lib_path():
    return _build.LIB


def load_library():
    """Build (if stale) and load the C-ABI library; raises PPMError when that is impossible."""
    global _lib
    if _lib is None:
        try:
            path = _build.build()
        except Exception as exc:  # no nvcc and no prebuilt library
            if os.path.exists(_build.LIB):
                path = _build.LIB
            else:
                raise PPMError(f"libppm_b200.so is missing and cannot be built: {exc}") from exc
        lib = C.CDLL(path)
        for name, (res, args) in EXPORTS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(rc):
    if rc != 0:
        raise PPMError(f"ppm error {rc}: {load_library().ppm_last_error().decode()}")


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _np(a):
    return a.ctypes.data_as(_dp)


def _dev(t, dtype=None, what="tensor", shape=None):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise PPMError(f"{what} must be a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise PPMError(f"{what} must have dtype {dtype}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise PPMError(f"{what} must have shape {tuple(shape)}, got {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


NOALLOC_MAX_BATCH = 1024      # PPM_NOALLOC_MAX_BATCH of include/ppm.h


def loglike_noalloc(counts, data, bkg, exposure_s, out):
    """ppm_loglike_noalloc: Poisson ln L without a context and without any allocation (static device scratch; see
    include/ppm.h).  counts [B][n_phase][n_channel], data [n_phase][n_channel], bkg [n_channel] or None, out [B]: contiguous
    float64 CUDA tensors on the current device; runs on torch's current stream.  `out` is the caller's (nothing is
    allocated here either).  Calls that overlap on the GPU race on the shared scratch."""
    import torch
    lib = load_library()
    if not isinstance(counts, torch.Tensor) or counts.dim() != 3:
        raise PPMError("counts must be a [B][n_phase][n_channel] CUDA tensor")
    B, n_phase, n_channel = counts.shape
    bp = _dev(bkg, torch.float64, "bkg", (n_channel,)) if bkg is not None else C.c_void_p(0)
    rc = lib.ppm_loglike_noalloc(_dev(counts, torch.float64, "counts"), int(B), int(n_phase), int(n_channel),
                                 _dev(data, torch.float64, "data", (n_phase, n_channel)), bp, float(exposure_s),
                                 _dev(out, torch.float64, "loglike", (B,)),
                                 C.c_void_p(torch.cuda.current_stream(counts.device).cuda_stream))
    if rc != 0:
        raise PPMError(f"ppm error {rc}: {lib.ppm_loglike_noalloc_error().decode()}")
    return out


def _host(a, dtype, shape, what):
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous or a.shape != tuple(shape):
        raise PPMError(f"{what} must be a C-contiguous numpy array of dtype {np.dtype(dtype)} and shape {tuple(shape)}")
    return a


def measure_fp64_peak(device=0):
    out = C.c_double()
    _check(load_library().ppm_measure_fp64_peak(int(device), C.byref(out)))
    return out.value


class PPM:
    """One context (ppm_create).  cfg: dict(n_spots, n_theta, n_phi, n_phase, n_fp, emission, oblate)."""

    def __init__(self, cfg, energies, max_batch=1, device=0, precision=0, scratch_mb=0):
        import torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise PPMError("no CUDA device: the PPM hot path has no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        energies = _f64(energies)
        self.n_energy = len(energies)
        self.cfg = dict(cfg)
        self.n_spots, self.n_theta, self.n_phi, self.n_phase = (int(cfg[k]) for k in
                                                                ("n_spots", "n_theta", "n_phi", "n_phase"))
        c = _Config(self.n_spots, self.n_theta, self.n_phi, self.n_phase, int(cfg.get("n_fp", 0)), self.n_energy,
                    int(cfg["emission"]), int(precision), int(cfg.get("oblate", 1)), int(max_batch), int(device),
                    int(cfg.get("mesh", 0)), int(cfg.get("beaming", 0)), int(scratch_mb),
                    int(cfg.get("phase_interp", 0)), int(cfg.get("interp_domain", 0)))
        self.P = 8 + 8 * self.n_spots
        self.max_batch = int(max_batch)
        with torch.cuda.device(self.device):
            stream = torch.cuda.current_stream().cuda_stream
        self._stream = stream
        self._h = C.c_void_p()
        _check(self.lib.ppm_create(C.byref(c), _np(energies), C.c_void_p(stream), C.byref(self._h)))
        self.n_fp = self.lib.ppm_n_fp(self._h)
        self.n_rows = self.n_spots * self.n_theta
        self.n_channel = 0

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self.lib.ppm_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _on_stream(self):
        """Single-stream contract (include/ppm.h): all work is enqueued on the stream that was current at construction;
        a call made under another torch stream would not be ordered with the caller's tensors."""
        if self.torch.cuda.current_stream(self.device).cuda_stream != self._stream:
            raise PPMError("this context was created on another CUDA stream: call it under the same torch stream")

    def _params(self, params):
        if params.dim() != 2 or params.shape[1] != self.P:
            raise PPMError(f"params must have shape [B][{self.P}]")
        if params.shape[0] > self.max_batch:
            raise PPMError(f"ppm error -5: B = {params.shape[0]} exceeds max_batch = {self.max_batch}")
        return params.shape[0]

    # ---- tables ----
    def load_atmosphere(self, logT, logg, mu, logx, values):
        logT, logg, mu, logx = map(_f64, (logT, logg, mu, logx))
        on_dev = hasattr(values, "is_cuda") and values.is_cuda
        if on_dev:
            vp = _dev(values, self.torch.float64, "values")
            n = values.numel()
        else:
            values = _f64(values)
            vp = C.c_void_p(values.ctypes.data)
            n = values.size
        if n != len(logT) * len(logg) * len(mu) * len(logx):
            raise PPMError("values has the wrong number of elements")
        _check(self.lib.ppm_load_atmosphere(self._h, _np(logT), len(logT), _np(logg), len(logg), _np(mu), len(mu),
                                            _np(logx), len(logx), vp, int(on_dev)))

    def set_response(self, n_channel, first_chan, rsp_band, tau_ref):
        first = np.ascontiguousarray(first_chan, dtype=np.int32)
        band = _f64(rsp_band)
        tau = _f64(tau_ref)
        if band.shape[0] != self.n_energy or len(first) != self.n_energy or len(tau) != self.n_energy:
            raise PPMError("response arrays must have n_energy rows")
        _check(self.lib.ppm_set_response(self._h, int(n_channel), band.shape[1], first.ctypes.data_as(_ip),
                                         C.c_void_p(band.ctypes.data), 0, _np(tau)))
        self.n_channel = int(n_channel)

    # ---- device-pointer calls (asynchronous on the context's stream) ----
    def evaluate(self, params, flux=None, status=None):
        t = self.torch
        self._on_stream()
        B = self._params(params)
        if flux is None:
            flux = t.empty((B, self.n_phase, self.n_energy), dtype=t.float64, device=self.device)
        if status is None:
            status = t.empty((B,), dtype=t.int32, device=self.device)
        _check(self.lib.ppm_evaluate(self._h, _dev(params, t.float64, "params"), B,
                                     _dev(flux, t.float64, "flux", (B, self.n_phase, self.n_energy)),
                                     _dev(status, t.int32, "status", (B,))))
        return flux, status

    def evaluate_map(self, params, logT_map, flux=None, status=None):
        """ppm_evaluate_map: logT_map [B][n_spots][n_theta][n_phi] float64 CUDA tensor, NaN = cell does not emit."""
        t = self.torch
        self._on_stream()
        B = self._params(params)
        if flux is None:
            flux = t.empty((B, self.n_phase, self.n_energy), dtype=t.float64, device=self.device)
        if status is None:
            status = t.empty((B,), dtype=t.int32, device=self.device)
        _check(self.lib.ppm_evaluate_map(self._h, _dev(params, t.float64, "params"),
                                         _dev(logT_map, t.float64, "logT_map", (B, self.n_spots, self.n_theta, self.n_phi)),
                                         B, _dev(flux, t.float64, "flux", (B, self.n_phase, self.n_energy)),
                                         _dev(status, t.int32, "status", (B,))))
        return flux, status

    def fold_response(self, flux, params, counts=None):
        t = self.torch
        self._on_stream()
        B = self._params(params)
        if counts is None:
            counts = t.empty((B, self.n_phase, self.n_channel), dtype=t.float64, device=self.device)
        _check(self.lib.ppm_fold_response(self._h, _dev(flux, t.float64, "flux", (B, self.n_phase, self.n_energy)),
                                          _dev(params, t.float64, "params"), B,
                                          _dev(counts, t.float64, "counts", (B, self.n_phase, self.n_channel))))
        return counts

    def loglike(self, counts, data, bkg, exposure_s, out=None):
        t = self.torch
        self._on_stream()
        B = counts.shape[0]
        if out is None:
            out = t.empty((B,), dtype=t.float64, device=self.device)
        bp = _dev(bkg, t.float64, "bkg", (self.n_channel,)) if bkg is not None else C.c_void_p(0)
        _check(self.lib.ppm_loglike(self._h, _dev(counts, t.float64, "counts", (B, self.n_phase, self.n_channel)), B,
                                    _dev(data, t.float64, "data", (self.n_phase, self.n_channel)), bp,
                                    float(exposure_s), _dev(out, t.float64, "loglike", (B,))))
        return out

    # ---- host-buffer calls (copies inside, synchronous) ----
    def evaluate_host(self, params, flux=None, status=None):
        params = _f64(params).reshape(-1, self.P)
        B = params.shape[0]
        if flux is None:
            flux = np.empty((B, self.n_phase, self.n_energy))
        if status is None:
            status = np.empty((B,), dtype=np.int32)
        _host(flux, np.float64, (B, self.n_phase, self.n_energy), "flux")
        _host(status, np.int32, (B,), "status")
        _check(self.lib.ppm_evaluate_host(self._h, _np(params), B, _np(flux), status.ctypes.data_as(_ip)))
        return flux, status

    def loglike_host(self, params, data, bkg, exposure_s, out=None, status=None):
        t = self.torch
        params = _f64(params).reshape(-1, self.P)
        B = params.shape[0]
        if out is None:
            out = np.empty((B,))
        if status is None:
            status = np.empty((B,), dtype=np.int32)
        _host(out, np.float64, (B,), "loglike")
        _host(status, np.int32, (B,), "status")
        bp = _dev(bkg, t.float64, "bkg", (self.n_channel,)) if bkg is not None else C.c_void_p(0)
        _check(self.lib.ppm_loglike_host(self._h, _np(params), B, _dev(data, t.float64, "data", (self.n_phase, self.n_channel)), bp, float(exposure_s),
                                         _np(out), status.ctypes.data_as(_ip)))
        return out, status

    # ---- device-resident sampler loop ----
    def chain_create(self, params0, lo, hi, sigma, data, bkg, exposure_s, beta=None, seed=0):
        t = self.torch
        self._on_stream()
        params0 = _f64(params0).reshape(-1, self.P)
        W = params0.shape[0]
        lo, hi, sigma = (_host(_f64(a), np.float64, (self.P,), n) for a, n in ((lo, "lo"), (hi, "hi"), (sigma, "sigma")))
        bp = None
        if beta is not None:
            beta = _host(_f64(beta), np.float64, (W,), "beta")
            bp = _np(beta)
        bk = _dev(bkg, t.float64, "bkg", (self.n_channel,)) if bkg is not None else C.c_void_p(0)
        self._chain_keep = (data, bkg)                       # the chain reads these device buffers at every step
        _check(self.lib.ppm_chain_create(self._h, W, _np(params0), _np(lo), _np(hi), _np(sigma), bp, int(seed),
                                         _dev(data, t.float64, "data", (self.n_phase, self.n_channel)), bk, float(exposure_s)))
        self._chain_w = W

    def chain_run(self, n_steps):
        self._on_stream()
        _check(self.lib.ppm_chain_run(self._h, int(n_steps)))

    def chain_read(self):
        """-> (params [W][P], loglike [W], accepted [W], swapped [W], steps)"""
        W = self._chain_w
        p, ll = np.empty((W, self.P)), np.empty(W)
        acc, swp = np.zeros(W, dtype=np.int64), np.zeros(W, dtype=np.int64)
        st = C.c_int64()
        i64 = C.POINTER(C.c_int64)
        _check(self.lib.ppm_chain_read(self._h, _np(p), _np(ll), acc.ctypes.data_as(i64), swp.ctypes.data_as(i64), C.byref(st)))
        return p, ll, acc, swp, st.value

    # ---- introspection of the last evaluate (tests) ----
    def debug_rows(self, b=0):
        out = np.zeros((self.n_rows, 16))
        _check(self.lib.ppm_debug_rows(self._h, b, _np(out)))
        return out

    def debug_mask(self, b=0):
        out = np.zeros((self.n_rows, self.n_phi), dtype=np.uint8)
        _check(self.lib.ppm_debug_mask(self._h, b, out.ctypes.data_as(_u8p)))
        return out

    def debug_template(self, b=0):
        out = np.zeros((self.n_rows, 4, self.n_fp + 1))
        _check(self.lib.ppm_debug_template(self._h, b, _np(out)))
        return out

    def debug_lookup(self, row, alpha, b=0):
        alpha = _f64(alpha)
        psi, dpsi, lag = (np.zeros(len(alpha)) for _ in range(3))
        _check(self.lib.ppm_debug_lookup(self._h, b, int(row), _np(alpha), len(alpha), _np(psi), _np(dpsi), _np(lag)))
        return psi, dpsi, lag

    KERNELS = ("star", "rows", "lookup", "template", "slice", "cells", "reduce", "fold", "loglike")

    def profile_enable(self, on=True):
        _check(self.lib.ppm_profile_enable(self._h, int(bool(on))))

    def profile_read(self):
        """-> (dict kernel -> (ms, launches), triples) since the last profile_enable."""
        ms = np.zeros(len(self.KERNELS))
        n = np.zeros(len(self.KERNELS), dtype=np.int64)
        tr = C.c_double()
        _check(self.lib.ppm_profile_read(self._h, _np(ms), n.ctypes.data_as(C.POINTER(C.c_int64)), C.byref(tr)))
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(self.KERNELS)}, tr.value

    def launch_count(self):
        return int(self.lib.ppm_launch_count(self._h))

    def sub_batch(self):
        return int(self.lib.ppm_sub_batch(self._h))

    def uniform_energy(self):
        return bool(self.lib.ppm_uniform_energy(self._h))
