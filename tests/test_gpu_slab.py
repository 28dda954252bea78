"""z-slab decomposition on ONE GPU: the kernels and the C calls of the sharded path, with the exchanges
between the slabs done by device copies that follow sharded.py's neighbour rule.  (Real multi-GPU runs need more than the one
GPU this box has; the exchange plumbing itself is covered by the world-size-2 gloo test in test_sharded_host.py.)

  * one rank that is its own neighbour reproduces the periodic fold bit for bit on arbitrary buffer contents;
  * two half-domains, each with its own ctx, particles and ghost-zoned state, give the single-domain ORACLE's step: buffers,
    state, eta, lambda and sinks within the usual bounds -- including sinks and supernovae whose kernels cross the cut;
  * call-order errors.
"""
import numpy as np
import pytest
import torch

from paper_2509_18261_b200 import inputs, pm, sharded
from tests import parity

pytestmark = pytest.mark.gpu
DEV = torch.device("cuda:0")


def slab_state(st: inputs.State, z0: int, nz: int, g: int, fill_ghosts: bool):
    """Planes [z0 - g, z0 + nz + g) of a global state (periodic), as a DeviceState of (nz + 2g) planes; ghost planes are
    poisoned unless fill_ghosts (then the halo exchange has to fill them)."""
    n = st.rho.shape[0]
    idx = np.arange(z0 - g, z0 + nz + g) % n
    fields = []
    for f in st.fields():
        a = np.ascontiguousarray(f[idx])
        if not fill_ghosts:
            a[:g] = np.nan
            a[-g:] = np.nan
        fields.append(torch.from_numpy(a).to(DEV))
    return pm.DeviceState(*fields)


def pick(prt, sel, cls, names, shift_z=0.0):
    arrs = [np.ascontiguousarray(getattr(prt, f)[sel]) for f in names]
    out = cls(*arrs)
    out.z[:] = out.z - shift_z
    return out


class Pair:
    """Two slab contexts on one GPU and the copies between them (rank 0: planes [0, h), rank 1: planes [h, n))."""

    def __init__(self, w, flags=pm.PM_FLAG_DEBUG_SCALARS | pm.PM_FLAG_DEBUG_LAMBDA, put=False):
        self.w = w
        self.put = put
        n = w.params["nz"]
        self.h = h = n // 2
        self.n = n
        p = dict(w.params, nz=h, z_slab=1)
        self.ctx, self.steps, self.state, self.sinks, self.sne, self.sel_k, self.sel_n = [], [], [], [], [], [], []
        for r in range(2):
            z0 = r * h
            c = pm.Context(dict(p, x0=(p["x0"][0], p["x0"][1], p["x0"][2] + z0 * p["dx"])), device="cuda:0", flags=flags)
            self.ctx.append(c)
            g = c.ghost_width()
            self.g = g
            self.state.append(slab_state(w.state, z0, h, g, fill_ghosts=False))
            sk_sel = (w.sinks.z >= z0) & (w.sinks.z < z0 + h)
            sn_sel = (w.sne.z >= z0) & (w.sne.z < z0 + h)
            self.sel_k.append(np.nonzero(sk_sel)[0]); self.sel_n.append(np.nonzero(sn_sel)[0])
            sk = pick(w.sinks, sk_sel, inputs.Sinks, ("x", "y", "z", "vx", "vy", "vz", "m"))
            sn = pick(w.sne, sn_sel, inputs.SNe, ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej"))
            self.sinks.append(pm.DeviceSinks.from_host(sk, DEV) if sk.n else None)
            self.sne.append(pm.DeviceSNe.from_host(sn, DEV) if sn.n else None)
        self.desc = [c.pm_slab_describe() for c in self.ctx]
        if put:                                     # peer-memory exchange: each ctx stores into the other's receive slabs
            self.ctx[0].pm_slab_connect_local(self.ctx[1], self.ctx[1])
            self.ctx[1].pm_slab_connect_local(self.ctx[0], self.ctx[0])

    def xchg(self, grp):
        d0, d1 = self.desc
        if d0[grp + "_send_lo"] is None:
            return
        for a, b in ((d0, d1), (d1, d0)):          # with two ranks the lower and the upper neighbour are the same peer
            b[grp + "_recv_hi"].copy_(a[grp + "_send_lo"])
            b[grp + "_recv_lo"].copy_(a[grp + "_send_hi"])

    def halo(self):
        g, plane, h = self.g, self.w.params["nx"] * self.w.params["ny"], self.h
        gp = g * plane
        for f in range(6):
            v = [s.fields()[f].view(-1) for s in self.state]
            for a, b in ((0, 1), (1, 0)):
                v[b][(h + g) * plane:(h + 2 * g) * plane].copy_(v[a][gp:2 * gp])      # a's bottom owned planes -> b's high ghosts
                v[b][0:gp].copy_(v[a][h * plane:h * plane + gp])                        # a's top owned planes -> b's low ghosts

    def step(self, stop_after=None):
        dt = self.w.dt
        self.halo()
        for r in range(2):
            self.ctx[r].pm_deposit(self.state[r], self.sinks[r], self.sne[r], dt)
            self.ctx[r].pm_slab_put() if self.put else self.ctx[r].pm_slab_pack()
        if not self.put:
            self.xchg("buf")
        for r in range(2):
            self.ctx[r].pm_fold_ghosts()
        if stop_after == "fold":
            return
        for r in range(2):
            self.ctx[r].pm_apply_limited(self.state[r])
        self.xchg("ret")
        self.xchg("rtr")
        for r in range(2):
            self.ctx[r].pm_return_to_particles(self.sinks[r])
            self.ctx[r].pm_check()

    # ---- what the parity helpers read, glued back to the global domain --------------------------------------
    def owned_buffer(self, ch):
        return np.concatenate([c.debug_buffer(ch)[1].cpu().numpy() for c in self.ctx], axis=0)

    def state_np(self):
        g = self.g
        return [np.concatenate([s.fields()[f][g:-g].cpu().numpy() for s in self.state], axis=0) for f in range(6)]

    def sink_field(self, name):
        out = np.zeros(self.w.sinks.n)
        for r in range(2):
            if self.sinks[r] is not None:
                out[self.sel_k[r]] = getattr(self.sinks[r], name).cpu().numpy()
        return out


def test_one_rank_as_its_own_neighbour_is_the_periodic_fold_bit_for_bit():
    """Arbitrary (random, sign-mixed) contents in every cell of the ghosted buffer, ghost planes included: periodic fold
    against pack -> self-exchange -> slab fold.  Same image order, same additions (Appendix A)."""
    for n, repro in ((24, 0), (21, 0), (24, pm.PM_FLAG_REPRODUCIBLE)):
        p = inputs.default_params(n)
        outs = []
        rng = np.random.default_rng(5)
        filled = None
        for slab in (0, 1):
            c = pm.Context(dict(p, z_slab=slab), device="cuda:0", flags=repro)
            g = c.ghost_width()
            nzs = n + (2 * g if slab else 0)
            st = pm.DeviceState(*(torch.ones(nzs * n * n, dtype=torch.float64, device=DEV) for _ in range(6)))
            c.pm_deposit(st, None, None, 0.1)                       # no particles: every tile stale
            views = [c.debug_buffer(ch)[0] for ch in range(6)]       # the debug view stores the zeros and marks every tile live
            if filled is None:
                filled = [torch.from_numpy(rng.standard_normal(tuple(v.shape))).to(DEV) for v in views]
            for v, f in zip(views, filled):
                v.copy_(f)
            if slab:
                c.pm_slab_pack()
                d = c.pm_slab_describe()
                sharded.exchange_slabs(d["buf_send_lo"], d["buf_send_hi"], d["buf_recv_lo"], d["buf_recv_hi"])
            c.pm_fold_ghosts()
            outs.append([c.debug_buffer(ch)[1].clone() for ch in range(6)])
            c.pm_check()
            c.close()
        for a, b in zip(*outs):
            assert torch.equal(a, b)


def test_fold_before_the_exchange_is_refused():
    p = dict(inputs.default_params(24), z_slab=1)
    c = pm.Context(p, device="cuda:0")
    st = pm.DeviceState(*(torch.ones(32 * 24 * 24, dtype=torch.float64, device=DEV) for _ in range(6)))
    c.pm_deposit(st, None, None, 0.1)
    with pytest.raises(pm.PmError) as e:
        c.pm_fold_ghosts()
    assert e.value.status == pm.PM_EORDER
    c.pm_slab_pack()
    c.pm_fold_ghosts()
    with pytest.raises(pm.PmError):
        c.pm_slab_pack()                                             # only directly after pm_deposit
    plain = pm.Context(inputs.default_params(24), device="cuda:0")
    with pytest.raises(pm.PmError):
        plain.pm_slab_pack()
    with pytest.raises(pm.PmError):
        plain.pm_slab_describe()
    with pytest.raises(AssertionError):                              # a state without ghost planes is refused by the binding
        c.pm_deposit(pm.DeviceState(*(torch.ones(24 ** 3, dtype=torch.float64, device=DEV) for _ in range(6))), None, None, 0.1)


@pytest.mark.parametrize("n,npart,seed", [(48, 1500, 5), (40, 900, 7)])
def test_two_half_domains_give_the_single_domain_oracle_step(n, npart, seed):
    """Every quantity the single-domain parity tests check, on a domain cut in two along z: particles are handed to the slab
    that holds their host cell; several sinks and supernovae are put right at the cut and at the periodic seam, so that their
    kernels reach into the other slab (ghost planes of the buffer out, ghost planes of state and return mesh in)."""
    w = inputs.scaled_mixed(n, npart, seed_index=seed)
    h = n // 2
    rng = np.random.default_rng(seed)
    for prt in (w.sinks, w.sne):                                     # a fifth of the particles within 3 cells of a cut
        k = max(prt.n // 5, 2)
        prt.z[:k] = np.mod(rng.choice([0.0, float(h)], size=k) + rng.uniform(-3.0, 3.0, size=k), float(n))
    o = parity.make_oracle(w)
    st_old = [f.copy() for f in o.state.fields()]
    g = Pair(w)
    o.step(w.dt)
    g.step(stop_after="fold")
    parity.CONTEXT["test"] = "two_slabs"
    n2 = parity.compare_buffers(g, o)
    # per-particle scalars, glued back into the global particle order
    for r in range(2):
        if g.sinks[r] is not None:
            d = g.ctx[r].debug_sink_scalars().cpu().numpy()
            for row, key in enumerate(("rho_inf", "v_inf", "c_inf", "r_bh", "mdot", "r_acc", "wsum")):
                parity.close_strict(d[row], o.sink_diag[key][g.sel_k[r]], f"sink {key}")
            assert np.array_equal(d[7].astype(np.int64), o.sink_diag["n_member"][g.sel_k[r]].astype(np.int64))
        if g.sne[r] is not None:
            d = g.ctx[r].debug_sn_scalars().cpu().numpy()
            for row, key in ((0, "m_snr"), (1, "v_snr"), (5, "n_h"), (6, "r_m"), (7, "p_rad")):
                parity.close_strict(d[row], o.sn_diag[key][g.sel_n[r]], f"SN {key}")
            assert np.array_equal(d[8].astype(np.int32), o.sn_diag["regime"][g.sel_n[r]])
    for r in range(2):
        g.ctx[r].pm_apply_limited(g.state[r])
    # state, eta, lambda
    gs, os_ = g.state_np(), o.state.fields()
    parity.close_strict(gs[0], os_[0], "rho")
    resp = parity.propagated_apply_tolerance(o, st_old)
    parity.close_reorder(gs[4], os_[4], resp[4] / parity.REORDER, "E")
    touched = o.sn_count.reshape(o.shape) > 0
    for f in (1, 2, 3):
        parity.close_reorder(gs[f], os_[f], resp[f] / parity.REORDER, f"p[{f - 1}]")
    ke = 0.5 * (os_[1] ** 2 + os_[2] ** 2 + os_[3] ** 2) / os_[0]
    parity.close_reorder(gs[5], os_[5], (resp[5] + 4 * parity.EPS * (np.abs(os_[4]) + ke) * touched) / parity.REORDER, "e_int")
    eta = np.concatenate([c.debug_return_mesh(0).cpu().numpy() for c in g.ctx], axis=0)
    has = o.A[0].reshape(o.shape) != 0
    parity.close_reorder(eta[has], o.eta.reshape(o.shape)[has], 4.0 * st_old[0][has] / (-o.A[0].reshape(o.shape)[has]), "eta")
    lam = np.concatenate([c.debug_lambda().cpu().numpy() for c in g.ctx], axis=0)
    sp = np.sqrt(sum(o.S[f].reshape(o.shape) ** 2 for f in (1, 2, 3)))
    parity.close_reorder(lam * sp, o.lam.reshape(o.shape) * sp, resp[6] / parity.REORDER, "lambda |S_p|")
    assert (o.eta < 1).sum() > 0 and (o.lam < 1).sum() > 0
    # Step 4 with the fill-back of (eta, v_old)
    g.xchg("ret")
    for r in range(2):
        g.ctx[r].pm_return_to_particles(g.sinks[r])
        g.ctx[r].pm_check()
    parity.close_strict(g.sink_field("m"), o.sinks.m, "sink m")
    parity.close_strict(g.sink_field("dm"), o.sink_diag["dm"], "sink dm")
    for f in ("dpx", "dpy", "dpz"):
        parity.close_reorder(g.sink_field(f), o.sink_diag[f], (parity.EPS / parity.REORDER) * (parity.C_TERM + 264.0) * o.sink_diag["dpabs"], f"sink {f}")
    # sinks at the cut really used the neighbour's cells
    near = np.minimum(np.abs(w.sinks.z - h), np.minimum(w.sinks.z, n - w.sinks.z)) < 3.0
    assert near.sum() >= 2 and np.all(o.sink_diag["dm"][near] > 0)
    # Eq. 1 over both slabs: mass changed by the ejecta only
    V = float(w.params["dx"]) ** 3
    mass = V * gs[0].sum() + g.sink_field("m").sum()
    mass0 = V * w.state.rho.sum() + w.sinks.m.sum()
    assert abs((mass - mass0) - w.sne.m_ej.sum()) <= 1e-12 * mass
    parity.dump_margins()
    for c in g.ctx:
        c.close()


def test_second_step_and_truelove_fill_back():
    """Two steps with the Truelove terms on (the Step 4 re-evaluation then also needs rho - rho_Tr of the neighbour's cells:
    the rtr_* slabs), against the oracle; the second step starts from the oracle's state on both sides."""
    n = 40
    w = inputs.scaled_mixed(n, 600, seed_index=9)
    w.params["truelove_J"] = 0.6
    h = n // 2
    w.sinks.z[:6] = np.array([0.3, h - 0.4, h + 1.2, n - 0.7, h + 2.6, 1.9])
    o = parity.make_oracle(w)
    for step in range(2):
        g = Pair(inputs.Workload(w.name, w.params, o.state.copy(), o.sinks.copy(), w.sne.copy(), w.dt, 1))
        o.step(w.dt)
        g.step()
        parity.close_strict(g.state_np()[0], o.state.rho, "rho")
        parity.close_strict(g.sink_field("m"), o.sinks.m, "sink m")
        parity.close_strict(g.sink_field("dm"), o.sink_diag["dm"], "sink dm")
        for c in g.ctx:
            c.close()


def test_put_to_itself_is_the_periodic_fold_bit_for_bit():
    """pm_slab_put with the ctx as its own neighbour (the pack kernel stores into the ctx's own receive slabs) over three
    consecutive steps -- both receive sets -- against the periodic fold of the same arbitrary buffer contents."""
    n = 24
    p = inputs.default_params(n)
    rng = np.random.default_rng(11)
    plain = pm.Context(dict(p, z_slab=0), device="cuda:0")
    slab = pm.Context(dict(p, z_slab=1), device="cuda:0")
    slab.pm_slab_connect_ipc(None, None)
    g = slab.ghost_width()
    st_plain = pm.DeviceState(*(torch.ones(n ** 3, dtype=torch.float64, device=DEV) for _ in range(6)))
    st_slab = pm.DeviceState(*(torch.ones((n + 2 * g) * n * n, dtype=torch.float64, device=DEV) for _ in range(6)))
    for step in range(3):
        outs = []
        filled = None
        for c, st in ((plain, st_plain), (slab, st_slab)):
            c.pm_deposit(st, None, None, 0.1)
            views = [c.debug_buffer(ch)[0] for ch in range(6)]
            if filled is None:
                filled = [torch.from_numpy(rng.standard_normal(tuple(v.shape))).to(DEV) for v in views]
            for v, f in zip(views, filled):
                v.copy_(f)
            if c is slab:
                c.pm_slab_put()
            c.pm_fold_ghosts()
            outs.append([c.debug_buffer(ch)[1].clone() for ch in range(6)])
            c.pm_check()                                             # (the next pm_deposit abandons the step)
        for a, b in zip(*outs):
            assert torch.equal(a, b), f"step {step}"
    slab.pm_deposit(st_slab, None, None, 0.1)
    slab.pm_slab_put()
    with pytest.raises(pm.PmError) as e:                             # a second put in one step
        slab.pm_slab_put()
    assert e.value.status == pm.PM_EORDER
    fresh = pm.Context(dict(p, z_slab=1), device="cuda:0")
    fresh.pm_deposit(st_slab, None, None, 0.1)
    with pytest.raises(pm.PmError) as e:                             # a put without neighbours
        fresh.pm_slab_put()
    assert e.value.status == pm.PM_EORDER
    for c in (plain, slab, fresh):
        c.close()


def test_two_half_domains_with_peer_puts_follow_the_oracle_for_three_steps():
    """The two slab contexts store their ghost planes straight into each other's receive slabs (pm_slab_connect_local +
    pm_slab_put), three steps in a row on the same contexts, so that both receive sets and their alternation are used; the
    oracle runs alongside.  Step 1 to the strict tolerances, the free-running trajectory to 1e-9 (as in tests/parity.py)."""
    n = 40
    w = inputs.scaled_mixed(n, 900, seed_index=8)
    h = n // 2
    rng = np.random.default_rng(8)
    for prt in (w.sinks, w.sne):
        k = max(prt.n // 5, 2)
        prt.z[:k] = np.mod(rng.choice([0.0, float(h)], size=k) + rng.uniform(-3.0, 3.0, size=k), float(n))
    o = parity.make_oracle(w)
    g = Pair(w, put=True)
    for step in range(3):
        o.step(w.dt)
        g.step()
        rho, m = g.state_np()[0], g.sink_field("m")
        if step == 0:
            parity.close_strict(rho, o.state.rho, "rho")
            parity.close_strict(m, o.sinks.m, "sink m")
            parity.close_strict(g.sink_field("dm"), o.sink_diag["dm"], "sink dm")
        assert np.all(np.abs(rho - o.state.rho) <= 1e-9 * np.abs(o.state.rho)), f"rho, step {step}"
        assert np.all(np.abs(m - o.sinks.m) <= 1e-9 * np.abs(o.sinks.m)), f"sink m, step {step}"
        E = g.state_np()[4]
        assert np.all(np.abs(E - o.state.etot) <= 1e-9 * np.abs(o.state.etot)), f"E, step {step}"
    V = float(w.params["dx"]) ** 3
    mass = V * rho.sum() + m.sum()
    mass0 = V * w.state.rho.sum() + w.sinks.m.sum()
    assert abs((mass - mass0) - 3 * w.sne.m_ej.sum()) <= 1e-12 * mass
    for c in g.ctx:
        c.close()
