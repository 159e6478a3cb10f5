"""ctypes binding of the CPU oracle (oracle/liboracle.so) -- test infrastructure only.

Imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
It marshals the parameter dict of paper_2602_13198_b200.workloads into the oracle's own struct.
"""
from __future__ import annotations

import ctypes as C
import importlib.util
import os

import numpy as np

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _load():
    spec = importlib.util.spec_from_file_location("oracle_build", os.path.join(_ROOT, "oracle", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return C.CDLL(mod.build())


class Params(C.Structure):
    _fields_ = [
        ("Ns_target", C.c_double), ("a_spin", C.c_double), ("hslope", C.c_double),
        ("startx", C.c_double * 4), ("dx", C.c_double * 4),
        ("L_unit", C.c_double), ("M_unit", C.c_double),
        ("thetae_fixed", C.c_double), ("trat", C.c_double), ("R_low", C.c_double), ("R_high", C.c_double),
        ("gam_ad", C.c_double), ("thetae_min", C.c_double), ("thetae_max", C.c_double),
        ("nu_min", C.c_double), ("nu_max", C.c_double), ("w_min", C.c_double),
        ("step_eps", C.c_double), ("verlet_tol", C.c_double),
        ("r_max", C.c_double), ("r_horizon_stop", C.c_double),
        ("bias0", C.c_double), ("roulette", C.c_double),
        ("nu_lo", C.c_double), ("nu_hi", C.c_double),
        ("seed", C.c_uint64), ("max_steps", C.c_int64),
        ("metric_kind", C.c_int32), ("n1", C.c_int32), ("n2", C.c_int32), ("n3", C.c_int32),
        ("thetae_mode", C.c_int32), ("verlet_maxit", C.c_int32),
        ("scattering_on", C.c_int32), ("nsc_max", C.c_int32), ("bias_p_theta", C.c_int32),
        ("bias_q_nsc", C.c_int32), ("n_th", C.c_int32), ("n_nu", C.c_int32), ("fold_theta", C.c_int32),
        ("emit_mode", C.c_int32), ("bias_target", C.c_double), ("bias_tune", C.c_int32), ("pad_", C.c_int32),
    ]


class Stats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in (
        "n_primary", "n_spawned", "n_recorded", "n_horizon", "n_roulette_killed", "n_roulette_survived",
        "n_maxstep", "n_outofrange", "n_steps_total", "n_verlet_iters", "n_verlet_capped", "n_bad_scatter",
        "n_analog_killed")] + [(n, C.c_double) for n in (
        "sum_w_emit", "sum_w_rec", "sum_w_horizon", "sum_w_roulette_killed", "sum_w_roulette_gain",
        "sum_w_outofrange", "sum_w_maxstep", "sum_w_absorbed", "sum_wE_emit", "sum_wE_rec", "sum_w_bad",
        "sum_w_spawned")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class TraceRec(C.Structure):
    _fields_ = [("x", C.c_double * 4), ("k", C.c_double * 4), ("w", C.c_double), ("E_inf", C.c_double),
                ("nstep", C.c_int64), ("fate", C.c_int32), ("nsc", C.c_int32), ("ith", C.c_int32),
                ("inu", C.c_int32), ("jscat", C.c_uint32), ("pad_", C.c_uint32)]


def make_params(d: dict) -> Params:
    p = Params()
    for name, _ in Params._fields_:
        if name == "pad_":
            continue
        v = d.get(name, 0) if name in ("emit_mode", "bias_target", "bias_tune") else d[name]
        if name in ("startx", "dx"):
            for i in range(4):
                getattr(p, name)[i] = float(v[i])
        else:
            setattr(p, name, v)
    return p


_dp = C.POINTER(C.c_double)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class OracleLib:
    def __init__(self):
        L = self.L = _load()
        assert L.orc_sizeof_params() == C.sizeof(Params), (L.orc_sizeof_params(), C.sizeof(Params))
        assert L.orc_sizeof_stats() == C.sizeof(Stats)
        assert L.orc_sizeof_trace() == C.sizeof(TraceRec)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(Params), C.c_void_p, C.c_size_t]
        L.orc_destroy.argtypes = [C.c_void_p]
        for f in ("orc_prepare", "orc_get_zone_counts", "orc_reset_tally", "orc_get_stats"):
            getattr(L, f).argtypes = [C.c_void_p, C.c_void_p] if f != "orc_reset_tally" else [C.c_void_p]
        L.orc_get_zone_info.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_weight_table.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_run.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int]
        L.orc_get_tally.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.orc_get_spectrum.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        L.orc_emit.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
        L.orc_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_plasma_at.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_fluid_frame.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        for f, n in (("orc_K2_direct", 1), ("orc_F_direct", 1), ("orc_sigma_kn", 1), ("orc_sigma_hot_direct", 2),
                     ("orc_K2_eval", 1), ("orc_F_eval", 1), ("orc_sigma_hot_eval", 2), ("orc_jnu", 5),
                     ("orc_jnu_integrated", 4), ("orc_nu_alpha_abs", 5)):
            getattr(L, f).restype = C.c_double
            getattr(L, f).argtypes = [C.c_double] * n
        L.orc_get_table.argtypes = [C.c_int, C.c_void_p, C.c_int]
        L.orc_philox.argtypes = [C.c_void_p] * 3
        L.orc_uniform_pair.argtypes = [C.c_uint64] + [C.c_uint32] * 5 + [C.c_void_p]
        L.orc_stream.argtypes = [C.c_uint64] + [C.c_uint32] * 4 + [C.c_int, C.c_void_p]
        L.orc_child_ids.argtypes = [C.c_uint64, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        for f in ("orc_gcov", "orc_gcon", "orc_dgcov", "orc_conn"):
            getattr(L, f).argtypes = [C.POINTER(Params), C.c_void_p, C.c_void_p]
        L.orc_gdet.restype = C.c_double
        L.orc_gdet.argtypes = [C.POINTER(Params), C.c_void_p]
        L.orc_step_size.restype = C.c_double
        L.orc_step_size.argtypes = [C.POINTER(Params), C.c_void_p, C.c_void_p]
        L.orc_push.argtypes = [C.POINTER(Params)] + [C.c_void_p] * 3 + [C.c_double] + [C.c_void_p] * 3
        L.orc_geodesic.argtypes = [C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.orc_tetrad.argtypes = [C.POINTER(Params)] + [C.c_void_p] * 4
        L.orc_get_bias_table.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_set_bias_table.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_zone_volume.restype = C.c_double
        L.orc_zone_volume.argtypes = [C.POINTER(Params), C.c_int, C.c_int, C.c_int]
        L.orc_sample_positions.argtypes = [C.POINTER(Params), C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.orc_sample_mj.argtypes = [C.c_double, C.c_uint64, C.c_int, C.c_void_p]
        L.orc_compton_sample.argtypes = [C.c_double, C.c_double, C.c_uint64, C.c_int] + [C.c_void_p] * 3

    # ---- bare functions ------------------------------------------------------------
    def philox(self, ctr, key):
        c = np.asarray(ctr, dtype=np.uint32)
        k = np.asarray(key, dtype=np.uint32)
        o = np.zeros(4, dtype=np.uint32)
        self.L.orc_philox(_p(c), _p(k), _p(o))
        return o

    def stream(self, seed, tag, c0, c1, c2, n):
        o = np.zeros(n)
        self.L.orc_stream(seed, tag, c0, c1, c2, n, _p(o))
        return o

    def child_ids(self, seed, parents, j):
        """ids [n][3] of the scattered superphotons spawned by event j[n] of parents[n][3] (G11)"""
        par = np.ascontiguousarray(parents, dtype=np.uint32).reshape(-1, 3)
        jj = np.ascontiguousarray(j, dtype=np.uint32)
        assert len(jj) == len(par)
        o = np.zeros_like(par)
        self.L.orc_child_ids(seed, _p(par), _p(jj), len(jj), _p(o))
        return o

    def table(self, which):
        n = -self.L.orc_get_table(which, None, -1)
        o = np.zeros(n)
        assert self.L.orc_get_table(which, _p(o), n) == 0
        return o

    def gcov(self, P, x):
        g = np.zeros((4, 4)); x = np.ascontiguousarray(x, dtype=float)
        self.L.orc_gcov(C.byref(P), _p(x), _p(g)); return g

    def gcon(self, P, x):
        g = np.zeros((4, 4)); x = np.ascontiguousarray(x, dtype=float)
        self.L.orc_gcon(C.byref(P), _p(x), _p(g)); return g

    def gdet(self, P, x):
        x = np.ascontiguousarray(x, dtype=float)
        return self.L.orc_gdet(C.byref(P), _p(x))

    def dgcov(self, P, x):
        g = np.zeros((4, 4, 4)); x = np.ascontiguousarray(x, dtype=float)
        self.L.orc_dgcov(C.byref(P), _p(x), _p(g)); return g

    def conn(self, P, x):
        g = np.zeros((4, 4, 4)); x = np.ascontiguousarray(x, dtype=float)
        self.L.orc_conn(C.byref(P), _p(x), _p(g)); return g

    def push(self, P, x0, k0, a0, dl):
        x0, k0, a0 = (np.ascontiguousarray(v, dtype=float) for v in (x0, k0, a0))
        x1, k1, a1 = np.zeros(4), np.zeros(4), np.zeros(4)
        it = self.L.orc_push(C.byref(P), _p(x0), _p(k0), _p(a0), dl, _p(x1), _p(k1), _p(a1))
        return x1, k1, a1, it

    def geodesic(self, P, x0, k0, nmax=100000):
        x0, k0 = (np.ascontiguousarray(v, dtype=float) for v in (x0, k0))
        traj = np.zeros((nmax, 8))
        n = self.L.orc_geodesic(C.byref(P), _p(x0), _p(k0), nmax, _p(traj))
        return traj[:n]

    def tetrad(self, P, x, ucon, trial):
        x, ucon, trial = (np.ascontiguousarray(v, dtype=float) for v in (x, ucon, trial))
        e = np.zeros((4, 4))
        self.L.orc_tetrad(C.byref(P), _p(x), _p(ucon), _p(trial), _p(e))
        return e

    def sample_mj(self, thetae, seed, n):
        o = np.zeros(n)
        self.L.orc_sample_mj(thetae, seed, n, _p(o))
        return o

    def compton_sample(self, thetae, eps, seed, n):
        e, c, kk = np.zeros(n), np.zeros(n), np.zeros(n)
        self.L.orc_compton_sample(thetae, eps, seed, n, _p(e), _p(c), _p(kk))
        return e, c, kk


_LIB = None


def lib() -> OracleLib:
    global _LIB
    if _LIB is None:
        _LIB = OracleLib()
    return _LIB


class Oracle:
    """One oracle context: params dict + prim grid."""

    def __init__(self, params: dict, prim: np.ndarray):
        self.lib = lib()
        self.L = self.lib.L
        self.params = dict(params)
        self.P = make_params(params)
        prim = np.ascontiguousarray(prim, dtype=np.float64)
        self.nz = params["n1"] * params["n2"] * params["n3"]
        self.nb = params["n_th"] * params["n_nu"]
        self.h = self.L.orc_create(C.byref(self.P), _p(prim), prim.size)
        assert self.h, "orc_create failed"
        self.n_primaries = None

    def __del__(self):
        if getattr(self, "h", None):
            self.L.orc_destroy(self.h)
            self.h = None

    def prepare(self) -> int:
        n = C.c_int64(0)
        assert self.L.orc_prepare(self.h, C.byref(n)) == 0
        self.n_primaries = n.value
        return n.value

    def zone_counts(self):
        o = np.zeros(self.nz, dtype=np.int32)
        self.L.orc_get_zone_counts(self.h, _p(o))
        return o

    def zone_info(self):
        a, b = np.zeros(self.nz), np.zeros(self.nz)
        self.L.orc_get_zone_info(self.h, _p(a), _p(b))
        return a, b

    def weight_table(self):
        nu, w = np.zeros(201), np.zeros(201)
        self.L.orc_get_weight_table(self.h, _p(nu), _p(w))
        return nu, w

    def run(self, first=0, n=None, nthreads=0) -> int:
        if n is None:
            n = self.n_primaries - first
        r = self.L.orc_run(self.h, first, n, nthreads)
        assert r > 0
        return r

    def reset_tally(self):
        self.L.orc_reset_tally(self.h)

    def tally(self):
        A, Q, W = np.zeros(self.nb), np.zeros(self.nb), np.zeros(self.nb)
        n = np.zeros(self.nb, dtype=np.int64)
        self.L.orc_get_tally(self.h, _p(A), _p(Q), _p(W), _p(n))
        sh = (self.params["n_th"], self.params["n_nu"])
        return A.reshape(sh), Q.reshape(sh), W.reshape(sh), n.reshape(sh)

    def spectrum(self):
        a, s = np.zeros(self.nb), np.zeros(self.nb)
        n = np.zeros(self.nb, dtype=np.int64)
        self.L.orc_get_spectrum(self.h, _p(a), _p(s), _p(n))
        sh = (self.params["n_th"], self.params["n_nu"])
        return a.reshape(sh), s.reshape(sh), n.reshape(sh)

    def stats(self) -> dict:
        s = Stats()
        self.L.orc_get_stats(self.h, C.byref(s))
        return s.as_dict()

    def emit(self, pid):
        o = np.zeros(20)
        self.L.orc_emit(self.h, pid, _p(o))
        return dict(x=o[0:4].copy(), k=o[4:8].copy(), a=o[8:12].copy(), w=o[12], nua_a=o[13], nua_s=o[14],
                    bias=o[15], E0=o[16])

    def trace(self, pids):
        pids = np.ascontiguousarray(pids, dtype=np.int64)
        n = len(pids)
        recs = (TraceRec * n)()
        fam_wE = np.zeros(n)
        fam_n = np.zeros(n, dtype=np.int64)
        self.L.orc_trace(self.h, _p(pids), n, C.byref(recs), _p(fam_wE), _p(fam_n))
        out = np.zeros(n, dtype=[("x", "f8", 4), ("k", "f8", 4), ("w", "f8"), ("E_inf", "f8"), ("nstep", "i8"),
                                 ("fate", "i4"), ("nsc", "i4"), ("ith", "i4"), ("inu", "i4"), ("jscat", "u4"),
                                 ("pad_", "u4")])
        C.memmove(out.ctypes.data, C.byref(recs), C.sizeof(recs))
        return out, fam_wE, fam_n

    def plasma_at(self, x):
        x = np.ascontiguousarray(x, dtype=float)
        o = np.zeros(12)
        self.L.orc_plasma_at(self.h, _p(x), _p(o))
        return dict(ne=o[0], thetae=o[1], B=o[2], ucon=o[3:7].copy(), bcon=o[7:11].copy(), vacuum=bool(o[11]))

    def fluid_frame(self, x, k, nsc=0):
        x = np.ascontiguousarray(x, dtype=float); k = np.ascontiguousarray(k, dtype=float)
        o = np.zeros(6)
        self.L.orc_fluid_frame(self.h, _p(x), _p(k), nsc, _p(o))
        return dict(eps=o[0], cos_b=o[1], nua_a=o[2], nua_s=o[3], bias=o[4], vacuum=bool(o[5]))

    def bias_table(self):
        """(per-generation bias factors [64], scattered superphotons spawned by each generation [64], pilot iterations)"""
        f = np.zeros(64); g = np.zeros(64, dtype=np.int64)
        it = self.L.orc_get_bias_table(self.h, _p(f), _p(g))
        return f, g, it

    def set_bias_table(self, fac):
        f = np.ascontiguousarray(fac, dtype=np.float64)
        assert f.size == 64
        self.L.orc_set_bias_table(self.h, _p(f))
