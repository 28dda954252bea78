"""Appendix A on the GPU (PM_FLAG_REPRODUCIBLE): the rounded buffers do not depend on the order of the atomic additions.
Through the C ABI, against the oracle's orc_repro_* (tests/test_oracle_repro.py pins that)."""
import numpy as np
import pytest
import torch

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs, pm
from tests import parity

pytestmark = pytest.mark.gpu

FLAGS = pm.PM_FLAG_DEBUG_SCALARS | pm.PM_FLAG_DEBUG_LAMBDA


def _permuted(w, seed):
    rng = np.random.default_rng(seed)
    pk, pn = rng.permutation(w.sinks.n), rng.permutation(w.sne.n)
    w2 = inputs.Workload("perm", w.params, w.state.copy(),
                         inputs.Sinks(*(getattr(w.sinks, f)[pk].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "m"))),
                         inputs.SNe(*(getattr(w.sne, f)[pn].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej"))),
                         w.dt, w.steps)
    return w2, pk, pn


def _run(w, flags, steps=1, view_buffers=True):
    """view_buffers: round the folded buffers in place (pm_debug_round_buffers) at step 0 and copy them out.  In the product
    path the apply pass rounds the sums as it reads them and the buffers stay unrounded; the rounding is idempotent, so
    both ways must leave the same state (checked below), and every later step runs the product path only."""
    g = parity.GpuRun(w, flags=FLAGS | flags)
    bufs = None
    for it in range(steps):
        g.ctx.pm_deposit(g.state, g.sinks, g.sne, w.dt)
        g.ctx.pm_fold_ghosts()
        if it == 0 and view_buffers:
            if flags & pm.PM_FLAG_REPRODUCIBLE:
                g.ctx.pm_debug_round_buffers()
            bufs = [g.owned_buffer(ch).copy() for ch in range(6)]
        g.ctx.pm_apply_limited(g.state)
        g.ctx.pm_return_to_particles(g.sinks)
    g.ctx.pm_check()
    return g, bufs


@pytest.mark.parametrize("n", [40, 37])
@pytest.mark.parametrize("flags", [0, pm.PM_FLAG_GENERIC_KERNELS])
def test_particle_order_does_not_change_a_bit(flags, n):
    """Heavily overlapping stencils (3 clusters): same particles, different order, two steps -> identical buffers, state, sinks.
    n = 37 (odd) takes the scalar fold / rounding / apply variants."""
    w = inputs.scaled_mixed(n, 800, seed_index=5, n_clusters=3)
    w2, pk, pn = _permuted(w, 7)
    ga, ba = _run(w, pm.PM_FLAG_REPRODUCIBLE | flags, steps=2)
    gb, bb = _run(w2, pm.PM_FLAG_REPRODUCIBLE | flags, steps=2)
    for ch in range(6):
        assert np.array_equal(ba[ch], bb[ch]), f"buffer channel {ch} depends on the particle order"
    for fa, fb in zip(ga.state_np(), gb.state_np()):
        assert np.array_equal(fa, fb)
    assert np.array_equal(ga.sinks.m.cpu().numpy()[pk], gb.sinks.m.cpu().numpy())
    assert np.array_equal(ga.sinks.vx.cpu().numpy()[pk], gb.sinks.vx.cpu().numpy())
    # the product path alone (rounding inside the apply pass, buffers never rounded in place) gives the same bits
    gc, _ = _run(w2, pm.PM_FLAG_REPRODUCIBLE | flags, steps=2, view_buffers=False)
    for fa, fc in zip(ga.state_np(), gc.state_np()):
        assert np.array_equal(fa, fc)
    assert np.array_equal(gb.sinks.m.cpu().numpy(), gc.sinks.m.cpu().numpy())


def test_without_the_flag_the_order_shows():
    w = inputs.scaled_mixed(40, 800, seed_index=5, n_clusters=3)
    w2, _, _ = _permuted(w, 7)
    _, ba = _run(w, 0)
    _, bb = _run(w2, 0)
    assert any(not np.array_equal(ba[ch], bb[ch]) for ch in range(2, 5))      # SN momentum: cancelling sums, order dependent


@pytest.mark.parametrize("flags", [0, pm.PM_FLAG_GENERIC_KERNELS])
def test_rounded_buffers_match_the_oracle(flags):
    """GPU and oracle round to the same value wherever neither sits within a reorder error of a rounding boundary (all but a
    ~2^-20 fraction of cells); everywhere they agree to the rounding interval; the state then follows as in the plain step."""
    w = inputs.scaled_mixed(40, 800, seed_index=5, n_clusters=3)
    g, bufs = _run(w, pm.PM_FLAG_REPRODUCIBLE | flags)
    o = parity.make_oracle(w)
    st_old = [f.copy() for f in o.state.fields()]
    o.step(w.dt, repro_M=28)
    shp = o.shape
    ref = [o.A[0].reshape(shp)] + [o.S[f].reshape(shp) for f in range(5)]
    multi = [(o.sink_count.reshape(shp) > 1)] + [(o.sn_count.reshape(shp) > 1)] * 5
    for ch in range(6):
        differ = (bufs[ch] != ref[ch]) & multi[ch]          # rounded cells: same bits; single contributions are not rounded
        assert differ.sum() <= max(2, int(1e-3 * multi[ch].sum())), f"channel {ch}: {differ.sum()} rounded cells differ bitwise"
        err = np.abs(bufs[ch] - ref[ch])
        assert np.all(err <= 2.0 ** -22 * np.abs(ref[ch]) + 1e-300)
        single = ~multi[ch] & (ref[ch] != 0)
        if ch in (0, 1, 5):           # single contributions are not rounded: plain parity there
            parity.close_strict(bufs[ch][single], ref[ch][single], f"channel {ch}, single contribution")
    parity.compare_sinks(g, o)
    parity.close_strict(g.state_np()[0], o.state.rho, "rho", rel=2.0 ** -22)


def test_margin_setter_and_errors():
    w = inputs.scaled_mixed(16, 40, seed_index=5, n_clusters=1)
    plain = pm.Context(w.params)
    with pytest.raises(pm.PmError):
        plain.pm_set_repro_margin(20)
    ctx = pm.Context(w.params, flags=pm.PM_FLAG_REPRODUCIBLE)
    with pytest.raises(pm.PmError):
        ctx.pm_set_repro_margin(53)
    ctx.pm_set_repro_margin(8)
    dev = torch.device("cuda:0")
    st = pm.DeviceState.from_host(w.state, dev)
    sk = pm.DeviceSinks.from_host(w.sinks, dev)
    sn = pm.DeviceSNe.from_host(w.sne, dev)
    ctx.step(st, sk, sn, w.dt)
    ctx.pm_check()
    o = po.Oracle(w.params, w.state.copy(), w.sinks.copy(), w.sne.copy())
    o.step(w.dt, repro_M=8)
    assert np.allclose(st.rho.cpu().numpy(), o.state.rho, rtol=1e-12)      # M = 8 keeps 40+ bits


def test_full_size_reproducible_step_twice_identical():
    """Config 5 (512^3, 10^6 particles) in the launch configuration bench.py --reproducible times: independent runs of the
    same step (different atomic order, as always) give bit-identical rounded buffers and a bit-identical state (momentum,
    internal energy, sink masses).  Runs 0 and 1 round the buffers in place to look at them; run 2 is the product path
    alone (rounding inside the apply pass)."""
    w = inputs.make(5)
    dev = torch.device("cuda:0")
    outs = []
    for rep in range(3):
        ctx = pm.Context(w.params, device="cuda:0", flags=pm.PM_FLAG_REPRODUCIBLE)
        st = pm.DeviceState.from_host(w.state, dev)
        sk = pm.DeviceSinks.from_host(w.sinks, dev)
        sn = pm.DeviceSNe.from_host(w.sne, dev)
        ctx.pm_deposit(st, sk, sn, w.dt)
        ctx.pm_fold_ghosts()
        sums = None
        if rep < 2:
            ctx.pm_debug_round_buffers()
            sums = [ctx.debug_buffer(ch)[1].clone() for ch in (0, 2, 5)]
        ctx.pm_apply_limited(st)
        ctx.pm_return_to_particles(sk)
        ctx.pm_check()
        outs.append((sums, st.mx.clone(), st.eint.clone(), sk.m.clone()))
        ctx.close()
        del st, sk, sn
    for a, b in zip(outs[0][0], outs[1][0]):
        assert torch.equal(a, b)
    for rep in (1, 2):
        assert torch.equal(outs[0][1], outs[rep][1]) and torch.equal(outs[0][2], outs[rep][2]) and torch.equal(outs[0][3], outs[rep][3])
