"""Thin ctypes binding of libgpumonty_b200.so (include/gpumonty_b200.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C-ABI.  PyTorch is used for device
memory (the fluid grid may be a CUDA tensor) and for the stream the work is enqueued on.  There is no
CPU fallback: without the built library, or without a CUDA device, these calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# GPUMONTY_B200_LIB selects another build of the same library (tuning experiments: launch bounds etc.)
LIB_PATH = os.environ.get("GPUMONTY_B200_LIB") or os.path.join(_HERE, "libgpumonty_b200.so")

GM_ABI_VERSION = 3
TABLE_LNK2, TABLE_LNF, TABLE_LNSIGH, TABLE_LNW, TABLE_NEXP, TABLE_QMAX = range(6)
EVAL_ACCEL, EVAL_GEOM, EVAL_PLASMA, EVAL_OPAC, EVAL_PUSH, EVAL_RAD, EVAL_NB, EVAL_BOUND = range(8)
_EVAL_SHAPES = {EVAL_ACCEL: (8, 4), EVAL_GEOM: (4, 33), EVAL_PLASMA: (4, 12), EVAL_OPAC: (8, 3),
                EVAL_PUSH: (13, 13), EVAL_RAD: (5, 3), EVAL_NB: (1, 3), EVAL_BOUND: (8, 6)}
FATE_ALIVE, FATE_RECORDED, FATE_HORIZON, FATE_ROULETTE, FATE_MAXSTEP, FATE_OUTOFRANGE, FATE_ANALOG = range(7)

EXPORTS = ["gm_create", "gm_destroy", "gm_last_error", "gm_set_grid", "gm_prepare", "gm_get_zone_counts",
           "gm_get_table", "gm_run", "gm_set_batch", "gm_set_phase_passes", "gm_get_spectrum", "gm_get_tally", "gm_get_stats",
           "gm_reset_tally", "gm_emit", "gm_trace", "gm_eval", "gm_fp64_peak", "gm_build_tables", "gm_timing", "gm_spectrum_device",
           "gm_get_bias_table", "gm_set_bias_table", "gm_get_zone_offsets", "gm_scan_counts_static"]
SCAN_STATIC_MAX_ZONES = 4194304  # GM_SCAN_STATIC_MAX_ZONES


class GmParams(C.Structure):
    _fields_ = [
        ("abi_version", C.c_uint32), ("metric_kind", C.c_int32), ("seed", C.c_uint64),
        ("Ns_target", C.c_double), ("a_spin", C.c_double), ("hslope", C.c_double),
        ("startx", C.c_double * 4), ("dx", C.c_double * 4),
        ("n1", C.c_int32), ("n2", C.c_int32), ("n3", C.c_int32), ("thetae_mode", C.c_int32),
        ("L_unit", C.c_double), ("M_unit", C.c_double),
        ("thetae_fixed", C.c_double), ("trat", C.c_double), ("R_low", C.c_double), ("R_high", C.c_double),
        ("gam_ad", C.c_double), ("thetae_min", C.c_double), ("thetae_max", C.c_double),
        ("nu_min", C.c_double), ("nu_max", C.c_double), ("w_min", C.c_double),
        ("step_eps", C.c_double), ("verlet_tol", C.c_double), ("r_max", C.c_double),
        ("r_horizon_stop", C.c_double), ("bias0", C.c_double), ("roulette", C.c_double),
        ("nu_lo", C.c_double), ("nu_hi", C.c_double), ("max_steps", C.c_int64),
        ("verlet_maxit", C.c_int32), ("scattering_on", C.c_int32), ("nsc_max", C.c_int32),
        ("bias_p_theta", C.c_int32), ("bias_q_nsc", C.c_int32),
        ("n_th", C.c_int32), ("n_nu", C.c_int32), ("fold_theta", C.c_int32),
        ("emit_mode", C.c_int32), ("bias_target", C.c_double), ("bias_tune", C.c_int32), ("pad_", C.c_int32),
    ]


class GmStats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in (
        "n_primary", "n_spawned", "n_recorded", "n_horizon", "n_roulette_killed", "n_roulette_survived",
        "n_maxstep", "n_outofrange", "n_steps_total", "n_verlet_iters", "n_verlet_capped", "n_bad_scatter",
        "n_analog_killed", "n_steps_free", "n_reentered", "n_bound_violations")] + [(n, C.c_double) for n in (
        "sum_w_emit", "sum_w_rec", "sum_w_horizon", "sum_w_roulette_killed", "sum_w_roulette_gain",
        "sum_w_outofrange", "sum_w_maxstep", "sum_w_absorbed", "sum_wE_emit", "sum_wE_rec", "sum_w_bad",
        "sum_w_spawned")]


TRACE_DTYPE = np.dtype([("x", "f8", 4), ("k", "f8", 4), ("w", "f8"), ("E_inf", "f8"), ("nstep", "i8"),
                        ("fate", "i4"), ("nsc", "i4"), ("ith", "i4"), ("inu", "i4"), ("jscat", "u4"),
                        ("pad_", "u4"), ("fam_wE", "f8"), ("fam_nspawn", "i8")])
EMIT_DTYPE = np.dtype([("x", "f8", 4), ("k", "f8", 4), ("a", "f8", 4), ("w", "f8"), ("nua_a", "f8"),
                       ("nua_s", "f8"), ("bias", "f8"), ("E0", "f8")])


class GmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gpumonty_b200 error {code}: {msg}")
        self.code = code


_lib = None


def load_library(build_if_missing: bool = True) -> C.CDLL:
    """Load the C-ABI library (building it in-tree with nvcc if it is absent)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise GmError(-3, f"{LIB_PATH} not built; run `python -m paper_2602_13198_b200.build`")
        from . import build as _build
        _build.build()
    L = C.CDLL(LIB_PATH)
    vp, i64p = C.c_void_p, C.POINTER(C.c_int64)
    L.gm_create.argtypes = [C.POINTER(vp), C.POINTER(GmParams)]
    L.gm_destroy.argtypes = [vp]
    L.gm_destroy.restype = None
    L.gm_last_error.argtypes = [vp]
    L.gm_last_error.restype = C.c_char_p
    L.gm_set_grid.argtypes = [vp, vp, C.c_int, C.c_size_t, vp]
    L.gm_prepare.argtypes = [vp, vp, i64p]
    L.gm_get_zone_counts.argtypes = [vp, vp]
    L.gm_get_table.argtypes = [vp, C.c_int, vp, C.c_size_t]
    L.gm_run.argtypes = [vp, C.c_int64, C.c_int64, vp]
    L.gm_set_batch.argtypes = [vp, C.c_int64, C.c_int64]
    L.gm_set_phase_passes.argtypes = [vp, C.c_int, C.c_int]
    L.gm_get_spectrum.argtypes = [vp, vp, vp, vp]
    L.gm_get_tally.argtypes = [vp, vp, vp, vp, vp]
    L.gm_get_stats.argtypes = [vp, C.POINTER(GmStats)]
    L.gm_reset_tally.argtypes = [vp]
    L.gm_emit.argtypes = [vp, vp, C.c_int, vp]
    L.gm_trace.argtypes = [vp, vp, C.c_int, vp]
    L.gm_eval.argtypes = [vp, C.c_int, vp, C.c_int, vp]
    L.gm_fp64_peak.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.gm_abi_sizes.argtypes = [C.POINTER(C.c_int)]
    L.gm_build_tables.argtypes = [vp, vp]
    L.gm_spectrum_device.argtypes = [vp, vp, vp, vp]
    L.gm_timing.argtypes = [vp, C.c_int, vp, vp]
    L.gm_get_bias_table.argtypes = [vp, vp, vp, C.POINTER(C.c_int)]
    L.gm_set_bias_table.argtypes = [vp, vp]
    L.gm_get_zone_offsets.argtypes = [vp, vp]
    L.gm_scan_counts_static.argtypes = [vp, C.c_int64, vp, vp]
    L.gm_abi_sizes.restype = None
    _lib = L
    return L


def make_params(d: dict) -> GmParams:
    p = GmParams()
    for name, _ in GmParams._fields_:
        if name == "pad_":
            continue
        v = d[name] if name != "abi_version" else d.get("abi_version", GM_ABI_VERSION)
        if name in ("startx", "dx"):
            for i in range(4):
                getattr(p, name)[i] = float(v[i])
        else:
            setattr(p, name, v)
    return p


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _stream_ptr(stream):
    if stream is None:
        try:
            import torch
            if torch.cuda.is_available():
                return C.c_void_p(torch.cuda.current_stream().cuda_stream)
        except ImportError:
            pass
        return C.c_void_p(0)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


def fp64_peak():
    """(FLOP/s of the FP64 pipe measured by a DFMA chain, SM clock from the device properties in MHz)."""
    L = load_library()
    f, c = C.c_double(0), C.c_double(0)
    rc = L.gm_fp64_peak(C.byref(f), C.byref(c))
    if rc:
        raise GmError(rc, L.gm_last_error(None).decode())
    return f.value, c.value


def scan_counts_static(counts, offsets, n_zones=None, stream=None):
    """gm_scan_counts_static: exclusive prefix sum of `counts` (CUDA int32 tensor) into `offsets` (CUDA int64 tensor,
    one element longer), for callers that may not allocate device memory: no context, no cudaMalloc; the scan's
    partial sums go to a fixed array inside the library, hence n_zones <= SCAN_STATIC_MAX_ZONES and no two calls in
    flight at once on a device.  Both tensors are the caller's; nothing is returned and nothing is synchronised.
    `n_zones` defaults to counts.numel() (passing it explicitly exists for the size-limit test)."""
    import torch
    L = load_library()
    assert counts.is_cuda and offsets.is_cuda and counts.dtype == torch.int32 and offsets.dtype == torch.int64
    assert counts.is_contiguous() and offsets.is_contiguous()
    n = counts.numel() if n_zones is None else int(n_zones)
    if n_zones is None:
        assert offsets.numel() == n + 1
    rc = L.gm_scan_counts_static(C.c_void_p(counts.data_ptr()), n, C.c_void_p(offsets.data_ptr()), _stream_ptr(stream))
    if rc:
        raise GmError(rc, L.gm_last_error(None).decode())


class GPUMonty:
    """One library context: same verbs as the C-ABI (gm_create .. gm_destroy)."""

    def __init__(self, params: dict):
        self.L = load_library()
        self.params = dict(params)
        self._P = make_params(params)
        self.nz = params["n1"] * params["n2"] * params["n3"]
        self.shape = (params["n_th"], params["n_nu"])
        self.h = C.c_void_p(0)
        rc = self.L.gm_create(C.byref(self.h), C.byref(self._P))
        if rc:
            raise GmError(rc, self.L.gm_last_error(None).decode())
        self.n_primaries = None

    def _ck(self, rc):
        if rc:
            raise GmError(rc, self.L.gm_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.L.gm_destroy(self.h)
            self.h = None

    __del__ = close

    # ---- inputs -------------------------------------------------------------------------------
    def set_grid(self, prim, stream=None):
        """prim: numpy array (host) or torch CUDA tensor (device), [n1][n2][n3][8] fp64."""
        if isinstance(prim, np.ndarray):
            a = np.ascontiguousarray(prim, dtype=np.float64)
            self._ck(self.L.gm_set_grid(self.h, _np_ptr(a), 0, a.nbytes, _stream_ptr(stream)))
            self._keep = a
        else:  # torch tensor
            import torch
            assert prim.dtype == torch.float64 and prim.is_contiguous()
            on_dev = 1 if prim.is_cuda else 0
            self._ck(self.L.gm_set_grid(self.h, C.c_void_p(prim.data_ptr()), on_dev,
                                        prim.numel() * 8, _stream_ptr(stream)))
            self._keep = prim

    def prepare(self, stream=None) -> int:
        n = C.c_int64(0)
        self._ck(self.L.gm_prepare(self.h, _stream_ptr(stream), C.byref(n)))
        self.n_primaries = n.value
        return n.value

    def set_batch(self, batch_primaries=0, queue_records=0):
        self._ck(self.L.gm_set_batch(self.h, int(batch_primaries), int(queue_records)))

    def set_phase_passes(self, pairs=-1, k_cold=4):
        self._ck(self.L.gm_set_phase_passes(self.h, int(pairs), int(k_cold)))

    def run(self, first=0, n=None, stream=None):
        if n is None:
            n = self.n_primaries - first
        self._ck(self.L.gm_run(self.h, int(first), int(n), _stream_ptr(stream)))

    def build_tables(self, stream=None):
        self._ck(self.L.gm_build_tables(self.h, _stream_ptr(stream)))

    def timing(self, enable=True):
        """{category: (ms, launches)} since the previous call; switches per-kernel event timing on/off."""
        ms, nl = np.zeros(7), np.zeros(7, dtype=np.int64)
        self._ck(self.L.gm_timing(self.h, int(enable), _np_ptr(ms), _np_ptr(nl)))
        names = ("tables", "prepare", "emit", "track", "compton", "spectrum", "escape")
        return {n: (float(ms[i]), int(nl[i])) for i, n in enumerate(names)}

    def bias_table(self):
        """(per-generation bias factors [64], scattered superphotons spawned by each generation [64], pilot passes)"""
        f, g, it = np.zeros(64), np.zeros(64, dtype=np.int64), C.c_int(0)
        self._ck(self.L.gm_get_bias_table(self.h, _np_ptr(f), _np_ptr(g), C.byref(it)))
        return f, g, it.value

    def set_bias_table(self, fac):
        f = np.ascontiguousarray(fac, dtype=np.float64)
        assert f.size == 64
        self._ck(self.L.gm_set_bias_table(self.h, _np_ptr(f)))

    def reset_tally(self):
        self._ck(self.L.gm_reset_tally(self.h))

    # ---- outputs ------------------------------------------------------------------------------
    def zone_counts(self):
        o = np.zeros(self.nz, dtype=np.int32)
        self._ck(self.L.gm_get_zone_counts(self.h, _np_ptr(o)))
        return o

    def zone_offsets(self):
        o = np.zeros(self.nz + 1, dtype=np.int64)
        self._ck(self.L.gm_get_zone_offsets(self.h, _np_ptr(o)))
        return o

    def table(self, which):
        n = {TABLE_LNK2: 201, TABLE_LNF: 261, TABLE_LNSIGH: 221 * 81, TABLE_LNW: 201,
             TABLE_NEXP: self.nz, TABLE_QMAX: self.nz}[which]
        o = np.zeros(n)
        self._ck(self.L.gm_get_table(self.h, which, _np_ptr(o), n))
        return o

    def spectrum(self):
        nb = self.shape[0] * self.shape[1]
        a, s, n = np.zeros(nb), np.zeros(nb), np.zeros(nb, dtype=np.int64)
        self._ck(self.L.gm_get_spectrum(self.h, _np_ptr(a), _np_ptr(s), _np_ptr(n)))
        return a.reshape(self.shape), s.reshape(self.shape), n.reshape(self.shape)

    def spectrum_device(self, nuLnu, sigma, stream=None):
        """nu L_nu and sigma into caller-owned CUDA tensors (fp64, n_th*n_nu elements), asynchronously."""
        self._ck(self.L.gm_spectrum_device(self.h, C.c_void_p(nuLnu.data_ptr()), C.c_void_p(sigma.data_ptr()),
                                           _stream_ptr(stream)))

    def tally(self):
        nb = self.shape[0] * self.shape[1]
        A, Q, W, n = np.zeros(nb), np.zeros(nb), np.zeros(nb), np.zeros(nb, dtype=np.int64)
        self._ck(self.L.gm_get_tally(self.h, _np_ptr(A), _np_ptr(Q), _np_ptr(W), _np_ptr(n)))
        return tuple(v.reshape(self.shape) for v in (A, Q, W, n))

    def stats(self) -> dict:
        s = GmStats()
        self._ck(self.L.gm_get_stats(self.h, C.byref(s)))
        return {n: getattr(s, n) for n, _ in GmStats._fields_}

    def emit(self, ids):
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        out = np.zeros(len(ids), dtype=EMIT_DTYPE)
        self._ck(self.L.gm_emit(self.h, _np_ptr(ids), len(ids), _np_ptr(out)))
        return out

    def trace(self, ids):
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        out = np.zeros(len(ids), dtype=TRACE_DTYPE)
        self._ck(self.L.gm_trace(self.h, _np_ptr(ids), len(ids), _np_ptr(out)))
        return out

    def eval(self, what, rows):
        nin, nout = _EVAL_SHAPES[what]
        a = np.ascontiguousarray(rows, dtype=np.float64).reshape(-1, nin)
        o = np.zeros((a.shape[0], nout))
        self._ck(self.L.gm_eval(self.h, what, _np_ptr(a), a.shape[0], _np_ptr(o)))
        return o
