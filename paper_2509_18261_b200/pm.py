"""Thin Python binding over the C ABI of libpm_b200.so (include/pm.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of csrc/pm_b200.cu.  torch is
used for device memory and the stream handle.  There is no CPU fallback: if the library is missing or was
not built, importing/using this module raises.
"""
from __future__ import annotations

import ctypes as C
import glob
import math
import os
import subprocess

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpm_b200.so")
SRC = [os.path.join(_HERE, "csrc", "pm_b200.cu")]
HDRS = sorted(glob.glob(os.path.join(_HERE, "csrc", "*.cuh"))) + [os.path.join(os.path.dirname(_HERE), "include", "pm.h")]

PM_OK, PM_EINVAL, PM_ENOMEM, PM_ECUDA, PM_EORDER, PM_EDOMAIN = 0, -1, -2, -3, -4, -5
PM_FLAG_DEBUG_SCALARS, PM_FLAG_DEBUG_LAMBDA, PM_FLAG_GENERIC_KERNELS, PM_FLAG_TIMING, PM_FLAG_REPRODUCIBLE, PM_FLAG_SMEM_TILES = 1, 2, 4, 8, 16, 32
KERNEL_GROUPS = ("bin", "zero", "sinks", "sne", "fold", "apply", "return")
STATUS_NAMES = {0: "PM_OK", -1: "PM_EINVAL", -2: "PM_ENOMEM", -3: "PM_ECUDA", -4: "PM_EORDER", -5: "PM_EDOMAIN"}

EXPORTS = ["pm_create", "pm_deposit", "pm_fold_ghosts", "pm_apply_limited", "pm_return_to_particles", "pm_check",
           "pm_step_host", "pm_step_host_begin", "pm_step_host_end", "pm_step_graph", "pm_destroy", "pm_last_error", "pm_launch_count", "pm_kernel_times", "pm_probe_red_f64", "pm_set_repro_margin", "pm_create_sinks", "pm_gravity_deposit", "pm_gravity_kick", "pm_drift", "pm_slab_describe", "pm_slab_pack", "pm_debug_round_buffers", "pm_debug_buffer", "pm_debug_tile_counts", "pm_debug_graph_state",
           "pm_debug_return_mesh", "pm_debug_lambda", "pm_debug_sink_scalars", "pm_debug_sn_scalars",
           "pm_debug_stencil", "pm_slab_ipc_export", "pm_slab_connect_ipc", "pm_slab_connect_local", "pm_slab_put", "pm_noalloc_setup", "pm_gravity_deposit_noalloc", "pm_noalloc_last_error"]

c_dp = C.POINTER(C.c_double)
PM_NOALLOC_MAX_GHOSTED_CELLS = 327680      # include/pm.h


class PmParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("sn_nsub", C.c_int32), ("sn_regime", C.c_int32), ("flags", C.c_int32),
        ("dx", C.c_double), ("x0", C.c_double * 3),
        ("G", C.c_double), ("gamma", C.c_double), ("cs_iso", C.c_double),
        ("rk_sink", C.c_double), ("rk_sn", C.c_double),
        ("bondi_lambda", C.c_double), ("f_max_remove", C.c_double), ("rho_floor", C.c_double),
        ("sn_eps_k", C.c_double), ("sn_rm_ej", C.c_double), ("sn_rm_mc", C.c_double),
        ("sn_msf_coeff", C.c_double), ("sn_msf_exp", C.c_double),
        ("sn_psnr_coeff", C.c_double), ("sn_psnr_exp", C.c_double),
        ("sn_mu_h", C.c_double), ("sn_nh_unit", C.c_double),
        ("sn_eint_theta", C.c_double), ("truelove_J", C.c_double),
        ("z_slab", C.c_int32), ("pad_", C.c_int32),
    ]


class PmSlabDesc(C.Structure):
    _fields_ = ([(f, C.c_void_p) for f in ("buf_send_lo", "buf_send_hi", "buf_recv_lo", "buf_recv_hi")] + [("buf_bytes", C.c_int64)] +
                [(f, C.c_void_p) for f in ("ret_send_lo", "ret_send_hi", "ret_recv_lo", "ret_recv_hi")] + [("ret_bytes", C.c_int64)] +
                [(f, C.c_void_p) for f in ("rtr_send_lo", "rtr_send_hi", "rtr_recv_lo", "rtr_recv_hi")] + [("rtr_bytes", C.c_int64)] +
                [("state_ghost_planes", C.c_int32), ("pad_", C.c_int32)])


class PmState(C.Structure):
    _fields_ = [(f, C.c_void_p) for f in ("rho", "mx", "my", "mz", "etot", "eint")]


class PmSinks(C.Structure):
    _fields_ = [("n", C.c_int64)] + [(f, C.c_void_p) for f in
                                     ("x", "y", "z", "vx", "vy", "vz", "m", "dm", "dpx", "dpy", "dpz")]


class PmSNe(C.Structure):
    _fields_ = [("n", C.c_int64)] + [(f, C.c_void_p) for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")]


class PmError(RuntimeError):
    def __init__(self, status: int, where: str, msg: str = ""):
        self.status = status
        super().__init__(f"{where}: {STATUS_NAMES.get(status, status)} {msg}".strip())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libpm_b200.so in-tree for sm_100a (nvcc cross-compiles without a GPU)."""
    newest = max(os.path.getmtime(p) for p in SRC + HDRS)
    if not force and os.path.exists(LIB_PATH) and os.path.getmtime(LIB_PATH) >= newest:
        return LIB_PATH
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo", "-fmad=false",
           "-Xcompiler", "-fPIC", "-shared", "-o", LIB_PATH] + SRC
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return LIB_PATH


_lib = None


def lib():
    """Load the CUDA library; fail loudly when it is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -c 'import __graft_entry__ as g; g.build()'`")
        L = C.CDLL(LIB_PATH)
        vp, i32p, i64p = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        L.pm_create.argtypes = [C.POINTER(PmParams), C.c_int, vp, C.POINTER(vp)]
        L.pm_deposit.argtypes = [vp, C.POINTER(PmState), C.POINTER(PmSinks), C.POINTER(PmSNe), C.c_double]
        L.pm_fold_ghosts.argtypes = [vp]
        L.pm_apply_limited.argtypes = [vp, C.POINTER(PmState)]
        L.pm_return_to_particles.argtypes = [vp, C.POINTER(PmSinks)]
        L.pm_check.argtypes = [vp]
        L.pm_step_host.argtypes = [vp, C.POINTER(PmState), C.POINTER(PmSinks), C.POINTER(PmSNe), C.c_double]
        L.pm_step_host_begin.argtypes = [vp, C.c_int, C.POINTER(PmState), C.POINTER(PmSinks), C.POINTER(PmSNe), C.c_double]
        L.pm_step_host_end.argtypes = [vp, C.c_int]
        L.pm_step_graph.argtypes = [vp, C.POINTER(PmState), C.POINTER(PmSinks), C.POINTER(PmSNe), C.c_double]
        L.pm_destroy.argtypes = [vp]
        L.pm_last_error.argtypes = [vp]
        L.pm_last_error.restype = C.c_char_p
        L.pm_launch_count.argtypes = [vp]
        L.pm_launch_count.restype = C.c_int64
        L.pm_set_repro_margin.argtypes = [vp, C.c_int32]
        L.pm_create_sinks.argtypes = [vp, C.POINTER(PmState), C.c_int64] + [vp] * 7 + [i64p]
        L.pm_gravity_deposit.argtypes = [vp, vp, C.c_int64, vp, vp, vp, vp, vp]
        L.pm_gravity_kick.argtypes = [vp] + [vp] * 3 + [C.c_int64] + [vp] * 6 + [C.c_double] + [vp] * 3
        L.pm_drift.argtypes = [vp, C.c_int64] + [vp] * 6 + [C.c_double]
        L.pm_kernel_times.argtypes = [vp, C.POINTER(C.c_float), C.c_int32]
        L.pm_probe_red_f64.argtypes = [vp, C.c_int64, C.c_int32, C.POINTER(C.c_double)]
        L.pm_debug_round_buffers.argtypes = [vp]
        L.pm_debug_buffer.argtypes = [vp, C.c_int, C.POINTER(vp), i64p, i64p, i32p]
        L.pm_debug_tile_counts.argtypes = [vp, i64p, i64p, i64p]
        L.pm_debug_graph_state.argtypes = [vp, i32p]
        L.pm_slab_describe.argtypes = [vp, C.POINTER(PmSlabDesc)]
        L.pm_slab_pack.argtypes = [vp]
        L.pm_slab_put.argtypes = [vp]
        L.pm_slab_ipc_export.argtypes = [vp, C.c_char_p, i64p]
        L.pm_slab_connect_ipc.argtypes = [vp, C.c_char_p, C.c_char_p]
        L.pm_slab_connect_local.argtypes = [vp, vp, vp]
        L.pm_debug_return_mesh.argtypes = [vp, C.c_int, C.POINTER(vp)]
        L.pm_debug_lambda.argtypes = [vp, C.POINTER(vp)]
        L.pm_debug_sink_scalars.argtypes = [vp, C.POINTER(vp), i64p]
        L.pm_debug_sn_scalars.argtypes = [vp, C.POINTER(vp), i64p]
        L.pm_debug_stencil.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_double, vp, i32p, i32p]
        L.pm_noalloc_setup.argtypes = [C.c_int]
        L.pm_gravity_deposit_noalloc.argtypes = [C.c_int, vp, C.c_int32, C.c_int32, C.c_int32, c_dp, C.c_double, vp, C.c_int64] + [vp] * 6
        L.pm_noalloc_last_error.argtypes = []
        L.pm_noalloc_last_error.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("pm_last_error", "pm_launch_count", "pm_noalloc_last_error"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def make_params(p: dict, flags: int = 0) -> PmParams:
    o = PmParams()
    for k, _ in PmParams._fields_:
        if k == "flags":
            o.flags = flags
        elif k == "x0":
            o.x0[0], o.x0[1], o.x0[2] = (float(v) for v in p["x0"])
        elif k == "truelove_J":
            o.truelove_J = float(p.get("truelove_J", 0.0))
        elif k == "z_slab":
            o.z_slab = int(p.get("z_slab", 0))
        elif k == "pad_":
            o.pad_ = 0
        else:
            setattr(o, k, p[k])
    return o


def _ptr(t, n=None):
    """Device pointer of a contiguous fp64 CUDA tensor of n elements (None -> NULL): the kernels get a raw pointer, so a CPU
    tensor or a short array must be refused here."""
    if t is None:
        return None
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), "fp64 contiguous CUDA tensors only"
    assert n is None or t.numel() == n, f"array of {t.numel()} elements where {n} are expected"
    return t.data_ptr()


def _dptr(t):
    """Device pointer of a contiguous fp64 CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _from_ptr(ptr: int, n: int, device, dtype=torch.float64):
    """Wrap library-owned device memory in a tensor (debug views only) via __cuda_array_interface__."""
    typestr = {torch.float64: "<f8", torch.int32: "<i4"}[dtype]

    class _Holder:
        __cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 2}
    return torch.as_tensor(_Holder(), device=device)


class DeviceState:
    FIELDS = ("rho", "mx", "my", "mz", "etot", "eint")

    def __init__(self, *fields):
        assert len(fields) == 6
        self.rho, self.mx, self.my, self.mz, self.etot, self.eint = fields

    @classmethod
    def from_host(cls, st, device):
        return cls(*(torch.from_numpy(getattr(st, f)).to(device) for f in cls.FIELDS))

    def fields(self):
        return [getattr(self, f) for f in self.FIELDS]

    def c(self, n_cells=None) -> PmState:
        s = PmState()
        dev = {getattr(self, f).device for f in self.FIELDS}
        assert len(dev) == 1, "state fields live on different devices"
        for f in self.FIELDS:
            setattr(s, f, _ptr(getattr(self, f), n_cells))
        return s


class DeviceSinks:
    IN = ("x", "y", "z", "vx", "vy", "vz", "m")
    OUT = ("dm", "dpx", "dpy", "dpz")

    def __init__(self, n, **t):
        self.n = n
        for f in self.IN + self.OUT:
            setattr(self, f, t.get(f))

    @classmethod
    def from_host(cls, sk, device, with_outputs=True):
        t = {f: torch.from_numpy(getattr(sk, f)).to(device) for f in cls.IN}
        if with_outputs:
            for f in cls.OUT:
                t[f] = torch.zeros(sk.n, dtype=torch.float64, device=device)
        return cls(sk.n, **t)

    def c(self) -> PmSinks:
        s = PmSinks()
        s.n = self.n
        for f in self.IN + self.OUT:
            setattr(s, f, _ptr(getattr(self, f), self.n))
        return s


class DeviceSNe:
    IN = ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")

    def __init__(self, n, **t):
        self.n = n
        for f in self.IN:
            setattr(self, f, t.get(f))

    @classmethod
    def from_host(cls, sn, device):
        return cls(sn.n, **{f: torch.from_numpy(getattr(sn, f)).to(device) for f in cls.IN})

    def c(self) -> PmSNe:
        s = PmSNe()
        s.n = self.n
        for f in self.IN:
            setattr(s, f, _ptr(getattr(self, f), self.n))
        return s


class Context:
    """One pm_ctx.  Methods have the names of the C entry points and only marshal arguments."""

    def __init__(self, params: dict, device="cuda:0", stream=None, flags: int = 0):
        self.L = lib()
        self.device = torch.device(device)
        self.params = dict(params)
        idx = self.device.index if self.device.index is not None else 0
        self.device = torch.device(self.device.type, idx)          # with an explicit index, so that tensor.device compares equal
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        self._p = make_params(params, flags)
        h = C.c_void_p()
        rc = self.L.pm_create(C.byref(self._p), idx, C.c_void_p(stream.cuda_stream), C.byref(h))
        if rc != PM_OK:
            raise PmError(rc, "pm_create")
        self.h = h

    def _chk(self, rc, where):
        if rc != PM_OK:
            raise PmError(rc, where, self.L.pm_last_error(self.h).decode())

    def _cells(self):
        """Length of a state array: owned cells, plus g ghost planes below and above on a z slab."""
        p = self.params
        nz = p["nz"] + (2 * self.ghost_width() if p.get("z_slab", 0) else 0)
        return p["nx"] * p["ny"] * nz

    def ghost_width(self) -> int:
        p = self.params
        return max(math.ceil(p["rk_sink"] / p["dx"]) if p["rk_sink"] > 0 else 0, math.ceil(p["rk_sn"] / p["dx"]) if p["rk_sn"] > 0 else 0)

    # ---- z-slab decomposition -------------------------------------------------------
    def pm_slab_pack(self):
        self._chk(self.L.pm_slab_pack(self.h), "pm_slab_pack")

    def pm_slab_put(self):
        """Pack + put: this rank's z ghost planes go straight into the neighbours' receive slabs (peer memory)."""
        self._chk(self.L.pm_slab_put(self.h), "pm_slab_put")

    def pm_slab_ipc_export(self) -> bytes:
        """The 64-byte CUDA IPC handle of this ctx's slab memory, to be handed to the two neighbours."""
        buf = C.create_string_buffer(64)
        self._chk(self.L.pm_slab_ipc_export(self.h, buf, None), "pm_slab_ipc_export")
        return buf.raw

    def pm_slab_connect_ipc(self, handle_lower, handle_upper):
        """Neighbours in other processes (handles from their pm_slab_ipc_export); None = this ctx is its own neighbour there."""
        self._chk(self.L.pm_slab_connect_ipc(self.h, handle_lower, handle_upper), "pm_slab_connect_ipc")

    def pm_slab_connect_local(self, lower=None, upper=None):
        """Neighbours in this process (other Context objects); None = this ctx itself."""
        self._chk(self.L.pm_slab_connect_local(self.h, lower.h if lower is not None else None, upper.h if upper is not None else None),
                  "pm_slab_connect_local")

    def pm_slab_describe(self) -> dict:
        """Device tensors (views of ctx-owned memory) of the slab messages: buf / ret / rtr x send_lo, send_hi, recv_lo, recv_hi."""
        d = PmSlabDesc()
        self._chk(self.L.pm_slab_describe(self.h, C.byref(d)), "pm_slab_describe")
        out = {"state_ghost_planes": int(d.state_ghost_planes)}
        for grp in ("buf", "ret", "rtr"):
            nbytes = getattr(d, grp + "_bytes")
            for side in ("send_lo", "send_hi", "recv_lo", "recv_hi"):
                ptr = getattr(d, f"{grp}_{side}")
                out[f"{grp}_{side}"] = _from_ptr(ptr, nbytes // 8, self.device) if (ptr and nbytes) else None
        return out

    def _on_device(self, *objs):
        for o in objs:
            if o is None:
                continue
            for f in getattr(o, "FIELDS", None) or (o.IN + getattr(o, "OUT", ())):
                t = getattr(o, f, None)
                assert t is None or t.device == self.device, f"{f} lives on {t.device}, the ctx on {self.device}"

    def pm_deposit(self, state: DeviceState, sinks, sne, dt: float):
        self._on_device(state, sinks, sne)
        cs = state.c(self._cells())
        ck = sinks.c() if sinks is not None else None
        cn = sne.c() if sne is not None else None
        self._chk(self.L.pm_deposit(self.h, C.byref(cs), C.byref(ck) if ck else None, C.byref(cn) if cn else None, dt),
                  "pm_deposit")

    def pm_step_graph(self, state: DeviceState, sinks, sne, dt: float, reuse_args: bool = False):
        """The four calls of a step as one call, replayed from a CUDA graph while the arguments stay the same.
        reuse_args=True keeps the marshalled structs of the previous call (the caller promises that state, sinks and sne still
        hold the same tensors): a replay then costs one ctypes call."""
        hit = getattr(self, "_graph_args", None) if reuse_args else None
        if hit is None:
            self._on_device(state, sinks, sne)
            cs = state.c(self._cells())
            ck = sinks.c() if sinks is not None else None
            cn = sne.c() if sne is not None else None
            hit = self._graph_args = (cs, ck, cn, (state, sinks, sne))       # the owners are kept alive with the pointers
        cs, ck, cn, _ = hit
        self._chk(self.L.pm_step_graph(self.h, C.byref(cs), C.byref(ck) if ck else None, C.byref(cn) if cn else None, dt),
                  "pm_step_graph")

    def pm_fold_ghosts(self):
        self._chk(self.L.pm_fold_ghosts(self.h), "pm_fold_ghosts")

    def pm_apply_limited(self, state: DeviceState):
        self._on_device(state)
        cs = state.c(self._cells())
        self._chk(self.L.pm_apply_limited(self.h, C.byref(cs)), "pm_apply_limited")

    def pm_return_to_particles(self, sinks):
        self._on_device(sinks)
        ck = sinks.c() if sinks is not None else None
        self._chk(self.L.pm_return_to_particles(self.h, C.byref(ck) if ck else None), "pm_return_to_particles")

    def pm_check(self):
        self._chk(self.L.pm_check(self.h), "pm_check")

    def step(self, state, sinks, sne, dt):
        """deposit -> fold -> apply -> return (four C calls, all asynchronous on the ctx stream)."""
        self.pm_deposit(state, sinks, sne, dt)
        self.pm_fold_ghosts()
        self.pm_apply_limited(state)
        self.pm_return_to_particles(sinks)

    def pm_step_host(self, st, sk, sn, dt: float):
        """Host-buffer step: st / sk / sn hold numpy arrays or CPU (pinned) tensors; updated in place."""
        self.pm_step_host_begin(0, st, sk, sn, dt)
        self.pm_step_host_end(0)

    def pm_step_host_end(self, slot: int):
        self._chk(self.L.pm_step_host_end(self.h, int(slot)), "pm_step_host_end")

    def pm_step_host_begin(self, slot: int, st, sk, sn, dt: float):
        """Enqueue one host-buffer step in slot 0 / 1 (upload, four calls, download) without waiting; see include/pm.h."""
        def hp(a):
            if a is None:
                return None
            if isinstance(a, torch.Tensor):
                assert a.device.type == "cpu" and a.dtype == torch.float64 and a.is_contiguous()
                return a.data_ptr()
            assert a.dtype.name == "float64" and a.flags["C_CONTIGUOUS"]
            return a.ctypes.data
        cs = PmState()
        for f in DeviceState.FIELDS:
            setattr(cs, f, hp(getattr(st, f)))
        ck = PmSinks()
        ck.n = sk.n if sk is not None else 0
        if sk is not None:
            for f in DeviceSinks.IN + DeviceSinks.OUT:
                setattr(ck, f, hp(getattr(sk, f, None)))
        cn = PmSNe()
        cn.n = sn.n if sn is not None else 0
        if sn is not None:
            for f in DeviceSNe.IN:
                setattr(cn, f, hp(getattr(sn, f)))
        self._chk(self.L.pm_step_host_begin(self.h, int(slot), C.byref(cs), C.byref(ck), C.byref(cn), dt), "pm_step_host_begin")

    def pm_create_sinks(self, state: DeviceState, max_new: int):
        """Sec. 3.1.2.  Returns (n_found, dict of device tensors x, y, z, vx, vy, vz, m of length min(n_found, max_new))."""
        out = {k: torch.zeros(max(max_new, 1), dtype=torch.float64, device=self.device) for k in ("x", "y", "z", "vx", "vy", "vz", "m")}
        n = C.c_int64(0)
        self._on_device(state)
        cs = state.c(self._cells())
        self._chk(self.L.pm_create_sinks(self.h, C.byref(cs), int(max_new), *(out[k].data_ptr() for k in ("x", "y", "z", "vx", "vy", "vz", "m")),
                                         C.byref(n)), "pm_create_sinks")
        k = n.value if n.value <= max_new else 0
        return int(n.value), {key: v[:k] for key, v in out.items()}

    # ---- PM gravity (Steps 1, 2, 5; L95, L107) ---------------------------------------------------
    def pm_gravity_deposit(self, rho_gas, x, y, z, m, rho_tot):
        """rho_tot := rho_gas + CIC deposit of the particle masses (device tensors; rho_gas may be None)."""
        n = int(x.numel())
        self._chk(self.L.pm_gravity_deposit(self.h, _dptr(rho_gas), n, _dptr(x), _dptr(y), _dptr(z), _dptr(m), _dptr(rho_tot)),
                  "pm_gravity_deposit")

    def pm_gravity_kick(self, gx, gy, gz, x, y, z, v=None, dt: float = 0.0, a=None):
        """a_s = CIC interpolation of (gx, gy, gz); v += a dt when v = (vx, vy, vz) is given; a = (ax, ay, az) optional outputs."""
        n = int(x.numel())
        vv = v if v is not None else (None, None, None)
        aa = a if a is not None else (None, None, None)
        self._chk(self.L.pm_gravity_kick(self.h, _dptr(gx), _dptr(gy), _dptr(gz), n, _dptr(x), _dptr(y), _dptr(z),
                                         _dptr(vv[0]), _dptr(vv[1]), _dptr(vv[2]), float(dt), _dptr(aa[0]), _dptr(aa[1]), _dptr(aa[2])),
                  "pm_gravity_kick")

    def pm_drift(self, x, y, z, vx, vy, vz, dt: float):
        n = int(x.numel())
        self._chk(self.L.pm_drift(self.h, n, _dptr(x), _dptr(y), _dptr(z), _dptr(vx), _dptr(vy), _dptr(vz), float(dt)), "pm_drift")

    def pm_set_repro_margin(self, M: int):
        self._chk(self.L.pm_set_repro_margin(self.h, int(M)), "pm_set_repro_margin")

    def pm_kernel_times(self) -> dict:
        """ms of each kernel group in the last step (needs PM_FLAG_TIMING)."""
        ms = (C.c_float * len(KERNEL_GROUPS))()
        self._chk(self.L.pm_kernel_times(self.h, ms, len(KERNEL_GROUPS)), "pm_kernel_times")
        return {k: float(v) for k, v in zip(KERNEL_GROUPS, ms)}

    def pm_probe_red_f64(self, footprint_bytes: int, channels: int) -> float:
        g = C.c_double(0.0)
        self._chk(self.L.pm_probe_red_f64(self.h, int(footprint_bytes), int(channels), C.byref(g)), "pm_probe_red_f64")
        return g.value

    def debug_graph_state(self) -> int:
        v = C.c_int32()
        self._chk(self.L.pm_debug_graph_state(self.h, C.byref(v)), "pm_debug_graph_state")
        return int(v.value)

    def pm_launch_count(self) -> int:
        return int(self.L.pm_launch_count(self.h))

    # ---- test-only views ------------------------------------------------------------------------
    def pm_debug_round_buffers(self):
        self._chk(self.L.pm_debug_round_buffers(self.h), "pm_debug_round_buffers")

    def debug_buffer(self, channel: int):
        """Returns (ghosted tensor (nz+2g, ny+2g, pitch), owned view (nz, ny, nx), g)."""
        ptr = C.c_void_p()
        dims = (C.c_int64 * 3)()
        origin = C.c_int64()
        g = C.c_int32()
        self._chk(self.L.pm_debug_buffer(self.h, channel, C.byref(ptr), dims, C.byref(origin), C.byref(g)), "pm_debug_buffer")
        d = [int(v) for v in dims]
        t = _from_ptr(ptr.value, d[0] * d[1] * d[2], self.device).view(d[0], d[1], d[2])
        nx, ny, nz = self.params["nx"], self.params["ny"], self.params["nz"]
        gz = g.value
        ox = origin.value - (gz * d[1] + gz) * d[2]
        owned = t[gz:gz + nz, gz:gz + ny, ox:ox + nx]
        return t, owned, gz, ox

    def debug_tile_counts(self):
        """(tiles of the buffer mesh, tiles live in group K, tiles live in group N) after the last pm_deposit."""
        n, k, m = C.c_int64(), C.c_int64(), C.c_int64()
        self._chk(self.L.pm_debug_tile_counts(self.h, C.byref(n), C.byref(k), C.byref(m)), "pm_debug_tile_counts")
        return int(n.value), int(k.value), int(m.value)

    def debug_return_mesh(self, word: int):
        ptr = C.c_void_p()
        self._chk(self.L.pm_debug_return_mesh(self.h, word, C.byref(ptr)), "pm_debug_return_mesh")
        nx, ny, nz = self.params["nx"], self.params["ny"], self.params["nz"]
        n = nx * ny * nz
        return _from_ptr(ptr.value, 4 * n - word, self.device)[::4][:n].view(nz, ny, nx)

    def debug_lambda(self):
        ptr = C.c_void_p()
        self._chk(self.L.pm_debug_lambda(self.h, C.byref(ptr)), "pm_debug_lambda")
        nx, ny, nz = self.params["nx"], self.params["ny"], self.params["nz"]
        return _from_ptr(ptr.value, nx * ny * nz, self.device).view(nz, ny, nx)

    def debug_sink_scalars(self):
        ptr, n = C.c_void_p(), C.c_int64()
        self._chk(self.L.pm_debug_sink_scalars(self.h, C.byref(ptr), C.byref(n)), "pm_debug_sink_scalars")
        return _from_ptr(ptr.value, 8 * n.value, self.device).view(8, n.value)

    def debug_sn_scalars(self):
        ptr, n = C.c_void_p(), C.c_int64()
        self._chk(self.L.pm_debug_sn_scalars(self.h, C.byref(ptr), C.byref(n)), "pm_debug_sn_scalars")
        return _from_ptr(ptr.value, 9 * n.value, self.device).view(9, n.value)

    def debug_stencil(self, kind: int, x: float, y: float, z: float):
        """(counts reshaped (side, side, side) in (k, j, i) order as a CPU int32 tensor, host cell (i, j, k))."""
        counts = torch.zeros(17 ** 3, dtype=torch.int32, device=self.device)
        host = (C.c_int32 * 3)()
        side = C.c_int32()
        self._chk(self.L.pm_debug_stencil(self.h, kind, x, y, z, C.c_void_p(counts.data_ptr()), host, C.byref(side)),
                  "pm_debug_stencil")
        s = side.value
        return counts[:s ** 3].view(s, s, s).cpu(), tuple(int(v) for v in host)

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            self.L.pm_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- the entry point that allocates nothing (include/pm.h) ------------------------------------------------------
def pm_gravity_deposit_noalloc(params: dict, rho_gas, x, y, z, m, rho_tot, outside=None, stream=None):
    """rho_tot := rho_gas + CIC deposit of the particle masses, through the static scratch array of the library: no ctx, no
    allocation.  params: nx, ny, nz, x0, dx.  outside: optional int32 CUDA tensor of one element (1 = a particle lay outside)."""
    L = lib()
    dev = rho_tot.device
    assert dev.type == "cuda", "device tensors only"
    idx = dev.index if dev.index is not None else 0
    if stream is None:
        stream = torch.cuda.current_stream(dev)
    n = int(x.numel()) if x is not None else 0
    ncell = params["nx"] * params["ny"] * params["nz"]
    _ptr(rho_tot, ncell), _ptr(rho_gas, ncell)
    for t in (x, y, z, m):
        _ptr(t, n)
    if outside is not None:
        assert outside.is_cuda and outside.dtype == torch.int32 and outside.numel() == 1
    x0 = (C.c_double * 3)(*(float(v) for v in params["x0"]))
    rc = L.pm_gravity_deposit_noalloc(idx, C.c_void_p(stream.cuda_stream), params["nx"], params["ny"], params["nz"], x0,
                                      float(params["dx"]), _dptr(rho_gas), n, _dptr(x), _dptr(y), _dptr(z), _dptr(m),
                                      _dptr(rho_tot), C.c_void_p(outside.data_ptr()) if outside is not None else None)
    if rc != PM_OK:
        raise PmError(rc, "pm_gravity_deposit_noalloc", L.pm_noalloc_last_error().decode())


def pm_noalloc_setup(device=0):
    L = lib()
    rc = L.pm_noalloc_setup(int(device))
    if rc != PM_OK:
        raise PmError(rc, "pm_noalloc_setup", L.pm_noalloc_last_error().decode())
