"""Shared helpers of the GPU parity tests: run the CUDA path and the oracle on the same seeded inputs and
compare element by element.  Tolerances (BASELINE.json north_star):

  * integer work (host cell, stencil membership, omega counts, regime): bit-exact;
  * per-cell values: |gpu - oracle| <= 1e-12 |oracle| + 1e-300, strictly, for everything whose terms share a
    sign (accretion d rho, SN d rho, SN d E, eta, rho, E);
  * channels that are cancelling sums (SN momentum, and through it p and e_int after the apply) add the
    paper's own bound on a floating-point sum (Appendix A: every addition errs by at most eps times the
    partial sum):  + eps * (C_TERM + k - 1) * sum_s |dU^s_ijk|  (R36), k = the number of particles that
    contributed to the cell (k - 1 additions, each partial sum <= sum |terms|), C_TERM = 32 ulp for the
    per-term arithmetic that differs between the two sides by design (explicit fma forms, x * (1/rho) for
    x / rho, d * rsqrt(r^2), exp(e ln x) for pow, tree instead of sequential stencil sums);
    the number of cells that needed the second term is reported;
  * the apply pass is ill-conditioned where Eq. 21 binds; there the bound is the oracle's own response to each
    buffer channel perturbed by exactly the bound it was verified to, summed over the channels with the worst
    sign each (first order), times 2;
  * global conserved totals: 1e-13 relative.
"""
from __future__ import annotations

import json
import math
import os

import numpy as np
import torch

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs, pm

REL = 1e-12
ABS_FLOOR = 1e-300
EPS = float(np.finfo(np.float64).eps)
C_TERM = 32.0            # ulp budget of one particle's term (see the module docstring)
K_STENCIL = 16.0         # v_COM = (sum omega rho V v + M_ej v_s) / M_snr (Eq. 18) is a sum over the 7^3 box that CANCELS once the gas
                         # streams away from the particle (every step after the first here); the GPU adds it as a tree, the oracle
                         # sequentially.  The two differ by at most (n - 1) eps sum|terms| and by ~ sqrt(n) eps sum|terms| for
                         # roundings of random sign (n = 343: 18); the bound takes 16 eps sum|terms| / M_snr for v_COM and lets it
                         # enter every cell's d p and d E with the factors of Eq. 17 (the oracle accumulates them as Scond).
                         # Found on config 4, step 4: a cell with ONE contribution off by 93 ulp of its sum|terms| -- which is
                         # 1.4 eps Scond.
REORDER = 1e-14          # unit in which close_reorder takes its `scale` (kept from round 1: 1e-14 = 45 eps)
TOTALS_REL = 1e-13
PROPAGATION_SAFETY = 2.0


def sum_bound(abs_terms: np.ndarray, k: np.ndarray, cond=None) -> np.ndarray:
    """eps [(C_TERM + k - 1) sum|terms| + K_STENCIL cond] in units of REORDER (the `scale` argument of close_reorder)."""
    b = (C_TERM + np.maximum(k, 1) - 1.0) * abs_terms
    if cond is not None:
        b = b + K_STENCIL * cond
    return (EPS / REORDER) * b


# Every comparison records how much of its bound it used (max over elements of err / tol), and every failure is also appended
# to a file: the log tail of a GPU run may lose the assertion message, the file does not.  MARGINS feeds the table in DESIGN.md
# section 5; the files land in gpurun_out/ (the one folder that comes back from the GPU box).
LOG_DIR = os.environ.get("PM_PARITY_LOG_DIR", os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out"))
MARGINS: dict = {}
CONTEXT = {"test": ""}


def _record(what: str, err: np.ndarray, tol: np.ndarray):
    ratio = float(np.max(err / np.maximum(tol, 1e-320))) if err.size else 0.0
    key = (CONTEXT["test"], what.split(" (")[0])
    MARGINS[key] = max(MARGINS.get(key, 0.0), ratio)
    return ratio


def dump_margins():
    """Append this process's margins (used fraction of each bound) to gpurun_out/parity_margins.jsonl."""
    try:
        os.makedirs(LOG_DIR, exist_ok=True)
        with open(os.path.join(LOG_DIR, "parity_margins.jsonl"), "a") as f:
            for (test, what), r in sorted(MARGINS.items()):
                f.write(json.dumps({"test": test, "quantity": what, "used_fraction_of_bound": r}) + "\n")
    except OSError:
        pass


def _fail(msg: str):
    try:
        os.makedirs(LOG_DIR, exist_ok=True)
        with open(os.path.join(LOG_DIR, "parity_failures.log"), "a") as f:
            f.write(f"[{CONTEXT['test']}] {msg}\n")
    except OSError:
        pass
    raise AssertionError(msg)


def close_strict(gpu: np.ndarray, ref: np.ndarray, what: str, rel: float = REL):
    err = np.abs(gpu - ref)
    tol = rel * np.abs(ref) + ABS_FLOOR
    _record(what, err, tol)
    bad = err > tol
    if bad.any():
        w = int(np.argmax(err / np.maximum(tol, 1e-320)))
        _fail(f"{what}: {bad.sum()} of {bad.size} outside {rel:g} rel; worst at flat index {w}: "
              f"gpu={gpu.reshape(-1)[w]!r} ref={ref.reshape(-1)[w]!r} err={err.reshape(-1)[w]:.3e} bound={tol.reshape(-1)[w]:.3e}")


def close_reorder(gpu: np.ndarray, ref: np.ndarray, scale: np.ndarray, what: str, rel: float = REL):
    """rel*|ref| + REORDER*scale; returns how many entries needed the second term."""
    err = np.abs(gpu - ref)
    tol1 = rel * np.abs(ref) + ABS_FLOOR
    tol = tol1 + REORDER * scale
    _record(what, err, tol)
    bad = err > tol
    if bad.any():
        w = int(np.argmax(err / np.maximum(tol, 1e-320)))
        _fail(f"{what}: {bad.sum()} of {bad.size} outside tolerance; worst at flat index {w}: "
              f"gpu={gpu.reshape(-1)[w]!r} ref={ref.reshape(-1)[w]!r} err={err.reshape(-1)[w]:.3e} "
              f"bound={tol.reshape(-1)[w]:.3e} (rel part {tol1.reshape(-1)[w]:.3e}, scale={np.broadcast_to(scale, err.shape).reshape(-1)[w]!r})")
    return int((err > tol1).sum())


class GpuRun:
    """The CUDA path on one workload, stage by stage, keeping what the tests inspect."""

    def __init__(self, w: inputs.Workload, device="cuda:0", flags=pm.PM_FLAG_DEBUG_SCALARS | pm.PM_FLAG_DEBUG_LAMBDA):
        self.w = w
        self.dev = torch.device(device)
        self.ctx = pm.Context(w.params, device=device, flags=flags)
        self.state = pm.DeviceState.from_host(w.state, self.dev)
        self.sinks = pm.DeviceSinks.from_host(w.sinks, self.dev) if w.sinks.n else None
        self.sne = pm.DeviceSNe.from_host(w.sne, self.dev) if w.sne.n else None

    def step(self, dt=None):
        self.ctx.step(self.state, self.sinks, self.sne, self.w.dt if dt is None else dt)

    def owned_buffer(self, ch):
        return self.ctx.debug_buffer(ch)[1].cpu().numpy()

    def state_np(self):
        return [f.cpu().numpy() for f in self.state.fields()]

    def totals(self):
        """(mass, momentum[3]) of gas + sinks, summed on the device in fp64."""
        V = float(self.w.params["dx"]) ** 3
        mass = V * float(self.state.rho.sum())
        mom = [V * float(f.sum()) for f in (self.state.mx, self.state.my, self.state.mz)]
        if self.sinks is not None:
            mass += float(self.sinks.m.sum())
            mom = [p + float((self.sinks.m * v).sum()) for p, v in
                   zip(mom, (self.sinks.vx, self.sinks.vy, self.sinks.vz))]
        return mass, mom


def make_oracle(w: inputs.Workload, lean: bool = False):
    """lean: keep only the error-scale meshes the comparisons read (accretion d rho, SN d p and d E) -- 512^3 needs it."""
    return po.Oracle(w.params, w.state.copy(), w.sinks.copy(), w.sne.copy(), abs_channels=((0,), (1, 2, 3, 4)) if lean else None)


def compare_buffers(g: GpuRun, o: po.Oracle):
    """After deposit + fold: the six GPU channels against the oracle's wrapped sums."""
    shp = o.shape
    ksk, ksn = o.sink_count.reshape(shp), o.sn_count.reshape(shp)
    # a ~ exp(-r^2/r_acc^2): Aabs carries the condition number 1 + r^2/r_acc^2 of each term (<= 257), which multiplies the
    # rounding of the exponent on both sides (the oracle's single exp and the kernel's three per-axis factors alike)
    n0 = close_reorder(g.owned_buffer(0), o.A[0].reshape(shp), sum_bound(o.Aabs[0].reshape(shp), ksk), "accretion d rho")
    close_strict(g.owned_buffer(1), o.S[0].reshape(shp), "SN d rho")
    n2 = n0
    for f in (1, 2, 3):
        n2 += close_reorder(g.owned_buffer(1 + f), o.S[f].reshape(shp), sum_bound(o.Sabs[f].reshape(shp), ksn, o.Scond[f].reshape(shp)), f"SN d p[{f - 1}]")
    # d E = thermal part (same sign) + v_COM . p_rad (either sign, small): bounded the same way
    n2 += close_reorder(g.owned_buffer(5), o.S[4].reshape(shp), sum_bound(o.Sabs[4].reshape(shp), ksn, o.Scond[4].reshape(shp)), "SN d E")
    # R29: the GPU keeps one accretion channel; the oracle's literal six are rank one in the cell state
    return n2


def compare_particle_scalars(g: GpuRun, o: po.Oracle):
    if g.sinks is not None:
        d = g.ctx.debug_sink_scalars().cpu().numpy()
        for row, key in enumerate(("rho_inf", "v_inf", "c_inf", "r_bh", "mdot", "r_acc", "wsum")):
            close_strict(d[row], o.sink_diag[key], f"sink {key}")
        assert np.array_equal(d[7].astype(np.int64), o.sink_diag["n_member"].astype(np.int64)), "sink member counts"
    if g.sne is not None:
        d = g.ctx.debug_sn_scalars().cpu().numpy()
        for row, key in enumerate(("m_snr", "v_snr")):
            close_strict(d[row], o.sn_diag[key], f"SN {key}")
        for row, key in zip((5, 6, 7), ("n_h", "r_m", "p_rad")):
            close_strict(d[row], o.sn_diag[key], f"SN {key}")
        # v_COM is a mass-weighted mean of signed velocities: bound by the momentum scale / M_snr
        vscale = np.abs(o.sn_diag["vcx"]) + np.abs(o.sn_diag["vcy"]) + np.abs(o.sn_diag["vcz"]) + 0.05
        for row, key in zip((2, 3, 4), ("vcx", "vcy", "vcz")):
            close_reorder(d[row], o.sn_diag[key], vscale, f"SN {key}", rel=REL)
        assert np.array_equal(d[8].astype(np.int32), o.sn_diag["regime"]), "SN regimes"


def propagated_apply_tolerance(o: po.Oracle, st_old):
    """First-order propagation of the buffer tolerance through the limiters, worst sign per channel.

    The apply step is ill-conditioned where Eq. 21 binds (lambda is the root of a quadratic whose coefficients
    are cancelling sums, and e_int = E - KE subtracts nearly equal numbers), so "1e-12 of the result" is not a
    meaningful bound there.  We re-run the ORACLE's apply with ONE buffer channel at a time moved by exactly the bound
    that channel was just verified to (+ and -), take the larger response per channel, and add the channels up:
    the first-order bound for any combination of signs.  The accretion group moves as one channel (it is rank one in
    the cell state, R29: all six components scale with d rho).  The apply pass is cell-local, so only the cells some
    particle touched are run (as a one-dimensional mesh).  Returns per-field response arrays (6 fields, lam*|S_p|)."""
    shp = o.shape
    resp = [np.zeros(shp) for _ in range(7)]
    idx = np.flatnonzero((o.sn_count > 0) | (o.A[0] != 0.0))
    if idx.size == 0:
        return resp
    m = idx.size
    A = [a[idx] for a in o.A]
    S = [s_[idx] for s_ in o.S]
    old = [f.reshape(-1)[idx] for f in st_old]
    ref_state = [f.reshape(-1)[idx] for f in o.state.fields()]
    ksk, ksn = o.sink_count[idx], o.sn_count[idx].copy()
    lam_ref = o.lam[idx]
    sp_ref = np.sqrt(sum(S[f] ** 2 for f in (1, 2, 3)))
    tolA = REL * np.abs(A[0]) + EPS * (C_TERM + np.maximum(ksk, 1) - 1.0) * o.Aabs[0][idx]
    relA = np.divide(tolA, np.abs(A[0]), out=np.zeros_like(tolA), where=A[0] != 0)
    tolS = [REL * np.abs(S[0])] + [REL * np.abs(S[f]) + EPS * ((C_TERM + np.maximum(ksn, 1) - 1.0) * o.Sabs[f][idx] + K_STENCIL * o.Scond[f][idx])
                                   for f in range(1, 5)]          # SN d rho has same-sign terms: verified strictly, no sum term
    pd = dict(o.pd, nx=m, ny=1, nz=1)
    t = po.Oracle(pd, inputs.State(*(f.copy() for f in old)), inputs.empty_sinks(), inputs.empty_sne(), keep_abs=False)
    chans = ([0] if o.sinks.n else []) + (list(range(1, 6)) if o.sne.n else [])
    tot = [np.zeros(m) for _ in range(7)]
    for ch in chans:                                      # 0: accretion group, 1..5: SN d rho, d p (3), d E
        worst = [np.zeros(m) for _ in range(7)]
        for sign in (1.0, -1.0):
            for f, fld in enumerate(t.state.fields()):
                fld[...] = old[f]
            for f in range(6):
                t.A[f][:] = A[f] * (1.0 + sign * relA) if ch == 0 else A[f]
            for f in range(5):
                t.S[f][:] = S[f] + sign * tolS[f] if ch == f + 1 else S[f]
            t.apply(sn_touched=ksn)
            for f in range(6):
                np.maximum(worst[f], np.abs(t.state.fields()[f] - ref_state[f]), out=worst[f])
            sp = np.sqrt(sum(t.S[f] ** 2 for f in (1, 2, 3)))
            np.maximum(worst[6], np.abs(t.lam * sp - lam_ref * sp_ref), out=worst[6])
        for f in range(7):
            tot[f] += worst[f]
    for f in range(7):
        resp[f].reshape(-1)[idx] = PROPAGATION_SAFETY * tot[f]
    return resp


def compare_state(g: GpuRun, o: po.Oracle, st_old, check_eta=True):
    """After apply: the six fields, eta, lambda.  st_old = pre-step oracle state (list of 6 arrays)."""
    shp = o.shape
    gs = g.state_np()
    os_ = o.state.fields()
    touched = o.sn_count.reshape(shp) > 0
    close_strict(gs[0], os_[0], "rho")
    resp = propagated_apply_tolerance(o, st_old)
    # E_2 = E_1 - eta A_E + S_E: strict wherever no SN touched the cell; S_E carries v_COM . p_rad, a signed part that is only
    # known to its own (verified) bound -- propagated like everything else
    close_reorder(gs[4], os_[4], resp[4] / REORDER, "E")
    eps = np.finfo(np.float64).eps
    n2 = 0
    for f in (1, 2, 3):
        n2 += close_reorder(gs[f], os_[f], resp[f] / REORDER, f"p[{f - 1}]")
    # e_int = E - KE in SN cells: add the rounding of the subtraction itself (E and KE, 4 ulp each)
    ke = 0.5 * (os_[1] ** 2 + os_[2] ** 2 + os_[3] ** 2) / os_[0]
    n2 += close_reorder(gs[5], os_[5], (resp[5] + 4 * eps * (np.abs(os_[4]) + ke) * touched) / REORDER, "e_int")
    if check_eta and g.sinks is not None:
        eta = g.ctx.debug_return_mesh(0).cpu().numpy()
        has = o.A[0].reshape(shp) != 0
        # eta = min(a, f rho, rho - floor)/a: a relative error of rho (1e-12) enters as 1e-12 rho/a through the floor
        a_req = -o.A[0].reshape(shp)[has]
        close_reorder(eta[has], o.eta.reshape(shp)[has], 4.0 * st_old[0][has] / a_req, "eta")
        for word, f in ((1, 1), (2, 2), (3, 3)):
            v = g.ctx.debug_return_mesh(word).cpu().numpy()
            close_strict(v[has], (st_old[f] / st_old[0])[has], f"v_old[{f - 1}]")
    lam = g.ctx.debug_lambda().cpu().numpy()
    lo = o.lam.reshape(shp)
    assert np.all(lam[~touched] == 1.0)
    assert lam.min() >= 0.0 and lam.max() <= 1.0
    sp = np.sqrt(sum(o.S[f].reshape(shp) ** 2 for f in (1, 2, 3)))
    close_reorder(lam * sp, lo * sp, resp[6] / REORDER, "lambda |S_p|")
    return n2


def compare_sinks(g: GpuRun, o: po.Oracle):
    """m, dm strict; the momentum gains are signed sums of gain * v_old over the ~264 member cells (a tree on the GPU, sequential
    in the oracle): bounded by eps (C_TERM + 264) sum |gain v|, the oracle's dpabs."""
    if g.sinks is None:
        return
    k = g.sinks
    close_strict(k.m.cpu().numpy(), o.sinks.m, "sink m")
    close_strict(k.dm.cpu().numpy(), o.sink_diag["dm"], "sink dm")
    bound = (EPS / REORDER) * (C_TERM + 264.0) * o.sink_diag["dpabs"]
    for f in ("dpx", "dpy", "dpz"):
        close_reorder(getattr(k, f).cpu().numpy(), o.sink_diag[f], bound, f"sink {f}")
    m_new = np.maximum(np.abs(o.sinks.m), 1e-300)
    for f in ("vx", "vy", "vz"):
        ref = getattr(o.sinks, f)
        close_reorder(getattr(k, f).cpu().numpy(), ref, bound / m_new + (EPS / REORDER) * 4.0 * np.abs(ref), f"sink {f}")


def run_and_compare(w: inputs.Workload, steps: int, stagewise_first: bool = True, lean: bool = False, trajectory: bool = True):
    """Full element-by-element parity over `steps` steps.  Returns (GpuRun, Oracle, cells needing the R36 term).

    Every step is compared from IDENTICAL inputs: from the second step on the oracle starts from the GPU's own state and sink
    masses / velocities (downloaded; they were verified against the oracle's at the end of the step before).  Otherwise the
    difference the bounds already allowed in step s (1e-12 relative, more where Eq. 21 binds) re-enters step s + 1's deposits as
    a difference of INPUTS that no bound of step s + 1 knows about -- measured: after ten free-running steps of config 4 a
    momentum deposit differs by 110 ulp of sum |terms|, against 5-10 ulp in any first step.  With trajectory=True a second,
    free-running oracle is stepped alongside and the final states are required to agree to 1e-9 (no drift, no blow-up)."""
    g = GpuRun(w)
    o = make_oracle(w, lean)
    free = make_oracle(w, lean=True) if (trajectory and steps > 1) else None
    n2 = 0
    for it in range(steps):
        if it > 0:                                # identical inputs: the oracle takes the GPU's state and sinks
            for dst, src in zip(o.state.fields(), g.state_np()):
                dst[...] = src
            if g.sinks is not None:
                for f in ("vx", "vy", "vz", "m"):
                    getattr(o.sinks, f)[:] = getattr(g.sinks, f).cpu().numpy()
        st_old = [f.copy() for f in o.state.fields()]
        m0, p0 = g.totals()
        o.step(w.dt)
        if free is not None:
            free.step(w.dt)
        if it == 0 and stagewise_first:
            g.ctx.pm_deposit(g.state, g.sinks, g.sne, w.dt)
            ghosted = [g.ctx.debug_buffer(ch)[0].clone() for ch in range(6)]
            g.ctx.pm_fold_ghosts()
            # fold invariant (O6): sum over ALL buffer cells before == sum over owned cells after
            for ch in range(6):
                before = float(ghosted[ch].sum())
                after = float(g.ctx.debug_buffer(ch)[1].sum())
                scale = float(ghosted[ch].abs().sum())
                assert abs(before - after) <= TOTALS_REL * max(scale, 1e-300), f"fold total, channel {ch}"
            del ghosted
            n2 += compare_buffers(g, o)
            compare_particle_scalars(g, o)
            g.ctx.pm_apply_limited(g.state)
            n2 += compare_state(g, o, st_old)
            g.ctx.pm_return_to_particles(g.sinks)
        else:
            g.step()
            n2 += compare_buffers(g, o)
            n2 += compare_state(g, o, st_old)
        compare_sinks(g, o)
        g.ctx.pm_check()
        # Eq. 1 on the GPU result alone: mass changes by exactly sum M_ej; sink exchange conserves momentum
        m1, _ = g.totals()
        dm_expect = float(w.sne.m_ej.sum())
        assert abs((m1 - m0) - dm_expect) <= TOTALS_REL * abs(m1), f"mass budget step {it}: {m1 - m0} vs {dm_expect}"
    if free is not None:                          # the free-running oracle trajectory: no drift beyond rounding-level growth
        for a, b, nm in zip(g.state_np(), free.state.fields(), inputs.State.FIELDS):
            err = np.abs(a - b)
            tol = 1e-9 * (np.abs(b) + np.abs(b).mean())
            _record(f"trajectory {nm}", err, tol)
            if (err > tol).any():
                wq = int(np.argmax(err / tol))
                _fail(f"trajectory {nm} after {steps} free-running steps: worst at flat index {wq}: gpu={a.reshape(-1)[wq]!r} "
                      f"oracle={b.reshape(-1)[wq]!r}")
        if g.sinks is not None:
            close_strict(g.sinks.m.cpu().numpy(), free.sinks.m, "trajectory sink m", rel=1e-9)
    return g, o, n2
