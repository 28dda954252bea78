"""ctypes wrapper around oracle/pm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It imports nothing from the CUDA package (paper_2509_18261_b200) except nothing at all: the parameter
dicts and numpy arrays it takes are produced by paper_2509_18261_b200/inputs.py, which the callers pass in.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_pm.so")
_LIB_OMP = os.path.join(_HERE, "liboracle_pm_omp.so")     # the same source with -fopenmp: bench.py's all-cores timing leg only
_lock = threading.Lock()
_lib = None
_lib_omp = None

c_dp = C.POINTER(C.c_double)
c_ip = C.POINTER(C.c_int32)
c_lp = C.POINTER(C.c_int64)


class OrcParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("sn_nsub", C.c_int32), ("sn_regime", C.c_int32), ("pad_", C.c_int32),
        ("dx", C.c_double), ("x0", C.c_double * 3),
        ("G", C.c_double), ("gamma", C.c_double), ("cs_iso", C.c_double),
        ("rk_sink", C.c_double), ("rk_sn", C.c_double),
        ("bondi_lambda", C.c_double), ("f_max_remove", C.c_double), ("rho_floor", C.c_double),
        ("sn_eps_k", C.c_double), ("sn_rm_ej", C.c_double), ("sn_rm_mc", C.c_double),
        ("sn_msf_coeff", C.c_double), ("sn_msf_exp", C.c_double),
        ("sn_psnr_coeff", C.c_double), ("sn_psnr_exp", C.c_double),
        ("sn_mu_h", C.c_double), ("sn_nh_unit", C.c_double),
        ("sn_eint_theta", C.c_double), ("truelove_J", C.c_double),
    ]


class OrcState(C.Structure):
    _fields_ = [(f, c_dp) for f in ("rho", "mx", "my", "mz", "etot", "eint")]


class OrcSinks(C.Structure):
    _fields_ = ([("n", C.c_int64)] +
                [(f, c_dp) for f in ("x", "y", "z", "vx", "vy", "vz", "m",
                                     "rho_inf", "v_inf", "c_inf", "r_bh", "mdot", "r_acc", "wsum",
                                     "dm", "dpx", "dpy", "dpz")] +
                [("n_member", c_ip), ("dpabs", c_dp)])


class OrcSNe(C.Structure):
    _fields_ = ([("n", C.c_int64)] +
                [(f, c_dp) for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej",
                                     "m_snr", "v_snr", "vcx", "vcy", "vcz", "n_h", "r_m", "p_rad")] +
                [("regime", c_ip)])


class OrcMeshOut(C.Structure):
    _fields_ = [("A", c_dp * 6), ("S", c_dp * 5), ("Aabs", c_dp * 6), ("Sabs", c_dp * 5),
                ("eta", c_dp), ("lam", c_dp), ("sn_count", c_ip), ("sink_count", c_ip), ("Tp", c_dp), ("Te", c_dp),
                ("Scond", c_dp * 5)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-ffp-contract=off so no FMA contraction changes a membership test)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
            subprocess.check_call(cmd)
    return _LIB


def build_omp(force: bool = False) -> str:
    """The same file compiled with -fopenmp: timed by bench.py on all host cores, never compared
    against -- its sums depend on the order of the atomic additions."""
    with _lock:
        stale = (not os.path.exists(_LIB_OMP)) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC)
        if force or stale:
            subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", _LIB_OMP, _SRC, "-lm"])
    return _LIB_OMP


def lib_omp():
    """The OpenMP build; only orc_step and orc_threads are called on it."""
    global _lib_omp
    if _lib_omp is None:
        build_omp()
        L = C.CDLL(_LIB_OMP)
        L.orc_sizeof_params.restype = C.c_int32
        assert L.orc_sizeof_params() == C.sizeof(OrcParams), "orc_params layout mismatch"
        L.orc_threads.restype = C.c_int32
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), C.POINTER(OrcSinks), C.POINTER(OrcSNe),
                               C.c_double, C.POINTER(OrcMeshOut), c_dp]
        _lib_omp = L
    return _lib_omp


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_sizeof_params.restype = C.c_int32
        assert L.orc_sizeof_params() == C.sizeof(OrcParams), "orc_params layout mismatch"
        L.orc_sink_stencil.restype = C.c_int32
        L.orc_sink_stencil.argtypes = [C.POINTER(OrcParams), C.c_double, C.c_double, C.c_double, c_ip, C.c_int32]
        L.orc_sn_omega_box.restype = C.c_int32
        L.orc_sn_omega_box.argtypes = [C.POINTER(OrcParams), C.c_double, C.c_double, C.c_double, c_ip, c_ip]
        L.orc_deposit.restype = C.c_int
        L.orc_deposit.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), C.POINTER(OrcSinks), C.POINTER(OrcSNe),
                                  C.c_double, C.POINTER(OrcMeshOut)]
        L.orc_apply.restype = C.c_int
        L.orc_apply.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), C.POINTER(OrcMeshOut), c_ip]
        L.orc_return.restype = C.c_int
        L.orc_return.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), c_dp, C.POINTER(OrcSinks), C.c_double]
        L.orc_return_from_list.restype = C.c_double
        L.orc_return_from_list.argtypes = [c_dp, c_lp, c_dp, C.c_int64, C.c_double]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), C.POINTER(OrcSinks), C.POINTER(OrcSNe),
                               C.c_double, C.POINTER(OrcMeshOut), c_dp]
        L.orc_step_repro.restype = C.c_int
        L.orc_step_repro.argtypes = L.orc_step.argtypes + [C.c_int32]
        L.orc_repro_bits.restype = C.c_int32
        L.orc_repro_bits.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_int32]
        L.orc_repro_round.restype = C.c_double
        L.orc_repro_round.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_int32]
        L.orc_repro_buffers.restype = C.c_int
        L.orc_repro_buffers.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), C.POINTER(OrcMeshOut), C.c_int32]
        L.orc_create_sinks.restype = C.c_int64
        L.orc_create_sinks.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), c_dp, C.c_int64] + [c_dp] * 7 + [c_lp]
        L.orc_sample_cells.restype = C.c_int
        L.orc_sample_cells.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), C.POINTER(OrcSinks), C.POINTER(OrcSNe),
                                       C.c_double, c_lp, C.c_int64, c_dp, c_dp, c_dp, c_dp, c_dp, c_dp, c_dp, c_ip]
        L.orc_particle_scalars.restype = C.c_int
        L.orc_particle_scalars.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState), C.POINTER(OrcSinks), C.POINTER(OrcSNe)]
        L.orc_sink_amounts.restype = C.c_int32
        L.orc_sink_amounts.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcState)] + [C.c_double] * 8 + [c_lp, c_dp, C.c_int32]
        _lib = L
    return _lib


def _dp(a):
    if a is None:
        return C.cast(None, c_dp)
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(c_dp)


def _ip(a):
    if a is None:
        return C.cast(None, c_ip)
    assert a.dtype == np.int32 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(c_ip)


def _lp(a):
    assert a.dtype == np.int64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(c_lp)


def make_params(p: dict) -> OrcParams:
    o = OrcParams()
    for k, _ in OrcParams._fields_:
        if k == "pad_":
            continue
        if k == "x0":
            o.x0[0], o.x0[1], o.x0[2] = (float(v) for v in p["x0"])
        elif k == "truelove_J":
            o.truelove_J = float(p.get("truelove_J", 0.0))      # 0 = Truelove terms off (R10)
        else:
            setattr(o, k, p[k])
    return o


SINK_DIAG = ("rho_inf", "v_inf", "c_inf", "r_bh", "mdot", "r_acc", "wsum", "dm", "dpx", "dpy", "dpz")
SN_DIAG = ("m_snr", "v_snr", "vcx", "vcy", "vcz", "n_h", "r_m", "p_rad")


class Oracle:
    """Holds one problem (params, state, particles; all numpy, modified in place by step())."""

    def __init__(self, params: dict, state, sinks, sne, keep_abs: bool = True, mesh: bool = True, abs_channels=None,
                 omp: bool = False):
        """abs_channels = (accretion channels, SN channels) whose error-scale meshes (Aabs, Sabs) are kept; None: all of them
        (with keep_abs) -- a 512^3 run keeps only the ones its comparisons read.  omp=True: the OpenMP build (step() only;
        for timing, not for comparisons)."""
        self.L = lib_omp() if omp else lib()
        self.pd = dict(params)
        self.p = make_params(params)
        self.state, self.sinks, self.sne = state, sinks, sne
        self.N = int(params["nx"]) * int(params["ny"]) * int(params["nz"])
        self.shape = (int(params["nz"]), int(params["ny"]), int(params["nx"]))
        N = self.N if mesh else 0          # mesh=False: only sample_cells / particle_scalars / sink_amounts are used
        self.A = [np.zeros(N) for _ in range(6)]
        self.S = [np.zeros(N) for _ in range(5)]
        ka, ks = (range(6), range(5)) if abs_channels is None else abs_channels
        self.Aabs = [np.zeros(N) if (keep_abs and f in ka) else None for f in range(6)]
        self.Sabs = [np.zeros(N) if (keep_abs and f in ks) else None for f in range(5)]
        # how strongly a cell's SN terms depend on the rounding of v_COM, a cancelling stencil sum (error scale only, see the C file)
        self.Scond = [np.zeros(N) if (keep_abs and f in ks and f > 0) else None for f in range(5)]
        self.eta = np.ones(N)
        self.lam = np.ones(N)
        self.sn_count = np.zeros(N, dtype=np.int32)
        self.sink_count = np.zeros(N, dtype=np.int32)
        self.Tp = np.zeros(N) if (keep_abs and abs_channels is None) else None      # Appendix A error scales (sum of |values added| per cell)
        self.Te = np.zeros(N) if (keep_abs and abs_channels is None) else None
        self.sink_diag = {k: np.zeros(sinks.n) for k in SINK_DIAG}
        self.sink_diag["n_member"] = np.zeros(sinks.n, dtype=np.int32)
        self.sink_diag["dpabs"] = np.zeros(sinks.n)          # error scale of the momentum gains (see the C file)
        self.sn_diag = {k: np.zeros(sne.n) for k in SN_DIAG}
        self.sn_diag["regime"] = np.zeros(sne.n, dtype=np.int32)
        self._old = None

    # -- ctypes views ------------------------------------------------------------------------
    def _cstate(self, st=None):
        st = st or self.state
        o = OrcState()
        for f in ("rho", "mx", "my", "mz", "etot", "eint"):
            setattr(o, f, _dp(getattr(st, f).reshape(-1)))
        return o

    def _csinks(self):
        o = OrcSinks()
        o.n = self.sinks.n
        for f in ("x", "y", "z", "vx", "vy", "vz", "m"):
            setattr(o, f, _dp(getattr(self.sinks, f)))
        for f in SINK_DIAG:
            setattr(o, f, _dp(self.sink_diag[f]))
        o.n_member = _ip(self.sink_diag["n_member"])
        o.dpabs = _dp(self.sink_diag["dpabs"])
        return o

    def _csne(self):
        o = OrcSNe()
        o.n = self.sne.n
        for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej"):
            setattr(o, f, _dp(getattr(self.sne, f)))
        for f in SN_DIAG:
            setattr(o, f, _dp(self.sn_diag[f]))
        o.regime = _ip(self.sn_diag["regime"])
        return o

    def _cmesh(self):
        o = OrcMeshOut()
        for f in range(6):
            o.A[f] = _dp(self.A[f])
            o.Aabs[f] = _dp(self.Aabs[f])
        for f in range(5):
            o.S[f] = _dp(self.S[f])
            o.Sabs[f] = _dp(self.Sabs[f])
            o.Scond[f] = _dp(self.Scond[f])
        o.eta, o.lam = _dp(self.eta), _dp(self.lam)
        o.sn_count, o.sink_count = _ip(self.sn_count), _ip(self.sink_count)
        o.Tp, o.Te = _dp(self.Tp), _dp(self.Te)
        return o

    # -- stages ------------------------------------------------------------------------------
    def deposit(self, dt: float):
        cs, ck, cn, cm = self._cstate(), self._csinks(), self._csne(), self._cmesh()
        rc = self.L.orc_deposit(C.byref(self.p), C.byref(cs), C.byref(ck), C.byref(cn), dt, C.byref(cm))
        assert rc == 0, f"orc_deposit rc={rc}"

    def apply(self, sn_touched=None):
        cs, cm = self._cstate(), self._cmesh()
        t = self.sn_count if sn_touched is None else sn_touched
        rc = self.L.orc_apply(C.byref(self.p), C.byref(cs), C.byref(cm), _ip(t))
        assert rc == 0

    def return_to_particles(self, state_old, dt: float):
        cs, ck = self._cstate(state_old), self._csinks()
        rc = self.L.orc_return(C.byref(self.p), C.byref(cs), _dp(self.eta), C.byref(ck), dt)
        assert rc == 0

    def step(self, dt: float, repro_M=None):
        """One whole step; repro_M = margin bits M of Appendix A (None: no rounding of the buffers)."""
        if self._old is None:
            self._old = np.empty(6 * self.N)
        cs, ck, cn, cm = self._cstate(), self._csinks(), self._csne(), self._cmesh()
        if repro_M is None:
            rc = self.L.orc_step(C.byref(self.p), C.byref(cs), C.byref(ck), C.byref(cn), dt, C.byref(cm), _dp(self._old))
        else:
            rc = self.L.orc_step_repro(C.byref(self.p), C.byref(cs), C.byref(ck), C.byref(cn), dt, C.byref(cm), _dp(self._old), int(repro_M))
        assert rc == 0, f"orc_step rc={rc}"

    def create_sinks(self, max_new: int, use_buffer: bool = True):
        """Sec. 3.1.2 on the current state (and the retained accretion buffer A[0]).  Returns (n_found, dict of arrays)."""
        out = {k: np.zeros(max_new) for k in ("x", "y", "z", "vx", "vy", "vz", "m")}
        cells = np.zeros(max_new, dtype=np.int64)
        cs = self._cstate()
        n = self.L.orc_create_sinks(C.byref(self.p), C.byref(cs), _dp(self.A[0]) if use_buffer else C.cast(None, c_dp), max_new,
                                    *(_dp(out[k]) for k in ("x", "y", "z", "vx", "vy", "vz", "m")), _lp(cells))
        assert n >= 0
        k = min(int(n), max_new)
        res = {key: v[:k] for key, v in out.items()}
        res["cells"] = cells[:k]
        return int(n), res

    def repro_buffers(self, M: int):
        """Appendix A rounding of the deposited buffers (call between deposit() and apply())."""
        cs, cm = self._cstate(), self._cmesh()
        rc = self.L.orc_repro_buffers(C.byref(self.p), C.byref(cs), C.byref(cm), int(M))
        assert rc == 0

    def state_old(self):
        """Views of the pre-step state kept by the last step()."""
        N = self.N
        return [self._old[f * N:(f + 1) * N].reshape(self.shape) for f in range(6)]

    def particle_scalars(self):
        cs, ck, cn = self._cstate(), self._csinks(), self._csne()
        rc = self.L.orc_particle_scalars(C.byref(self.p), C.byref(cs), C.byref(ck), C.byref(cn))
        assert rc == 0

    def sample_cells(self, cells: np.ndarray, dt: float):
        cells = np.ascontiguousarray(cells, dtype=np.int64)
        n = cells.shape[0]
        out = dict(A=np.zeros((n, 6)), S=np.zeros((n, 5)), Aabs=np.zeros((n, 6)), Sabs=np.zeros((n, 5)),
                   eta=np.zeros(n), lam=np.zeros(n), unew=np.zeros((n, 6)), sn_count=np.zeros(n, dtype=np.int32))
        cs, ck, cn = self._cstate(), self._csinks(), self._csne()
        rc = self.L.orc_sample_cells(C.byref(self.p), C.byref(cs), C.byref(ck), C.byref(cn), dt, _lp(cells), n,
                                     _dp(out["A"]), _dp(out["S"]), _dp(out["Aabs"]), _dp(out["Sabs"]),
                                     _dp(out["eta"]), _dp(out["lam"]), _dp(out["unew"]), _ip(out["sn_count"]))
        assert rc == 0
        return out

    def sink_amounts(self, s: int, dt: float):
        k = self.sinks
        cells = np.zeros(4096, dtype=np.int64)
        a = np.zeros(4096)
        cs = self._cstate()
        n = self.L.orc_sink_amounts(C.byref(self.p), C.byref(cs), k.x[s], k.y[s], k.z[s], k.vx[s], k.vy[s], k.vz[s],
                                    k.m[s], dt, _lp(cells), _dp(a), 4096)
        assert 0 <= n <= 4096
        return cells[:n].copy(), a[:n].copy()


def sink_stencil(params: dict, x: float, y: float, z: float) -> np.ndarray:
    """Unwrapped member cells (n, 3) as (i, j, k) of a sink kernel."""
    L = lib()
    p = make_params(params)
    buf = np.zeros(3 * 8192, dtype=np.int32)
    n = L.orc_sink_stencil(C.byref(p), x, y, z, _ip(buf), 8192)
    assert n <= 8192
    return buf[:3 * n].reshape(n, 3).copy()


def sn_omega_box(params: dict, x: float, y: float, z: float):
    """(counts[(2g+1)^3] in (k,j,i) order reshaped (2g+1,)*3, host cell (i,j,k))."""
    L = lib()
    p = make_params(params)
    import math
    side = 2 * int(math.ceil(params["rk_sn"] / params["dx"])) + 1
    counts = np.zeros(side ** 3, dtype=np.int32)
    host = np.zeros(3, dtype=np.int32)
    s = L.orc_sn_omega_box(C.byref(p), x, y, z, _ip(counts), _ip(host))
    assert s == side
    return counts.reshape(side, side, side), host


def return_from_list(eta: np.ndarray, cells: np.ndarray, a: np.ndarray, V: float) -> float:
    L = lib()
    cells = np.ascontiguousarray(cells, dtype=np.int64)
    a = np.ascontiguousarray(a, dtype=np.float64)
    eta = np.ascontiguousarray(eta.reshape(-1), dtype=np.float64)
    return float(L.orc_return_from_list(_dp(eta), _lp(cells), _dp(a), cells.shape[0], V))


def repro_bits(x: float, T: float, k: int, M: int) -> int:
    return int(lib().orc_repro_bits(float(x), float(T), int(k), int(M)))


def repro_round(x: float, T: float, k: int, M: int) -> float:
    return float(lib().orc_repro_round(float(x), float(T), int(k), int(M)))
