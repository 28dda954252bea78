"""Truelove terms (Eqs. 12-14, 16) on the GPU against the oracle, through the C ABI."""
import numpy as np
import pytest
import torch

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs, pm
from tests import parity

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("flags", [0, pm.PM_FLAG_GENERIC_KERNELS])
@pytest.mark.parametrize("J", [0.8, 0.45])
def test_truelove_mixed_workload_matches_oracle(flags, J):
    """Lognormal gas (sigma_ln = 1.5) with c_s = 1: rho_Tr = J^2 pi (2.0 / 0.64), so a good part of the sink-touched cells
    sit above it and take the Eq. 14 branch, the others the Bondi-Hoyle branch; three steps so that the return pass reads
    entries invalidated and rewritten across steps."""
    n = 40 if flags == 0 else 37                     # 37: odd row length, scalar apply / fold variants
    w = inputs.scaled_mixed(n, 600, seed_index=5, n_clusters=3)
    w.params["truelove_J"] = J
    g = parity.GpuRun(w, flags=pm.PM_FLAG_DEBUG_SCALARS | pm.PM_FLAG_DEBUG_LAMBDA | flags)
    o = parity.make_oracle(w)
    rho_tr = J * J * np.pi
    for it in range(3):
        st_old = [f.copy() for f in o.state.fields()]
        if it > 0:
            # rho - rho_Tr amplifies the (verified, 1e-12) differences the previous step left in rho and e_int by rho / (rho -
            # rho_Tr): start every step from the oracle's state, so that each step is compared on identical inputs
            g.state = pm.DeviceState.from_host(o.state, g.dev)
            g.sinks = pm.DeviceSinks.from_host(o.sinks, g.dev)
        o.step(w.dt)
        g.step()
        touched = o.sink_count.reshape(o.shape) > 0
        if it == 0:
            above = touched & (st_old[0] > rho_tr)
            assert above.sum() > 100 and (touched & ~above).sum() > 100       # both branches are exercised
        parity.compare_buffers(g, o)
        parity.compare_state(g, o, st_old)
        parity.compare_sinks(g, o)
        g.ctx.pm_check()


def test_truelove_density_falls_to_rho_tr_on_gpu():
    """The paper's statement (L146) checked on the GPU result alone: uniform gas above rho_Tr, negligible Bondi-Hoyle rate."""
    n = 24
    w = inputs.config1_tiny_sink()
    p = dict(w.params)
    p.update(nx=n, ny=n, nz=n, truelove_J=0.4, f_max_remove=0.25)
    st = inputs._uniform_state(n, 1.0, 0.6, p["gamma"])            # c_s^2 = 1
    sinks = inputs._pack_sinks(np.array([[12.3, 12.1, 12.7]]), np.zeros((1, 3)), np.array([1e-3]))
    ww = inputs.Workload("tl", p, st, sinks, inputs.empty_sne(), 0.01, 1)
    g = parity.GpuRun(ww)
    g.step()
    rho = g.state_np()[0]
    rho_tr = 0.16 * np.pi
    changed = rho != 1.0
    assert changed.sum() == 264
    assert np.allclose(rho[changed], rho_tr, rtol=1e-14, atol=0)
    assert abs(float(g.sinks.m[0]) - 1e-3 - 264 * (1.0 - rho_tr)) < 1e-10


def test_truelove_params_validation():
    w = inputs.config1_tiny_sink()
    p = dict(w.params)
    p["truelove_J"] = -0.1
    with pytest.raises(pm.PmError):
        pm.Context(p)
