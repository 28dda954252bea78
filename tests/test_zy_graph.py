"""pm_step_graph: the four calls of a step replayed from a CUDA graph.  Same kernels in the same order, so in Appendix A mode
(PM_FLAG_REPRODUCIBLE: results independent of the order of the atomic additions) the graph path must equal the plain calls BIT
FOR BIT, step after step, while particles and gas evolve; without the flag the two agree to the reorder tolerance and the
graph path agrees with the oracle like any other step.

Appendix A makes two orders of the additions land on the same bits "except with probability ~2^-M per cell" (L612): the
comparisons here run with M = 40 instead of the default 28, which leaves that chance below 1e-6 per run.  The file is named to
be collected after the core parity tests (pytest -x)."""
import numpy as np
import pytest
import torch

from paper_2509_18261_b200 import inputs, pm
from tests import parity

pytestmark = pytest.mark.gpu
DEV = torch.device("cuda:0")


def device_copy(w):
    st = pm.DeviceState.from_host(w.state.copy(), DEV)
    sk = pm.DeviceSinks.from_host(w.sinks.copy(), DEV) if w.sinks.n else None
    sn = pm.DeviceSNe.from_host(w.sne.copy(), DEV) if w.sne.n else None
    return st, sk, sn


def plain_step(ctx, st, sk, sn, dt):
    ctx.pm_deposit(st, sk, sn, dt)
    ctx.pm_fold_ghosts()
    ctx.pm_apply_limited(st)
    if sk is not None:
        ctx.pm_return_to_particles(sk)


@pytest.mark.parametrize("n,npart", [(32, 300), (37, 500)])
def test_graph_replay_is_bit_identical_to_the_plain_calls_in_appendix_a_mode(n, npart):
    w = inputs.scaled_mixed(n, npart, seed_index=5)
    stream = torch.cuda.Stream(DEV)                      # a stream of its own: default streams cannot be captured
    with torch.cuda.stream(stream):
        a = pm.Context(w.params, device="cuda:0", stream=stream, flags=pm.PM_FLAG_REPRODUCIBLE)
        b = pm.Context(w.params, device="cuda:0", stream=stream, flags=pm.PM_FLAG_REPRODUCIBLE)
        a.pm_set_repro_margin(40)
        b.pm_set_repro_margin(40)
        sa, ka, na = device_copy(w)
        sb, kb, nb = device_copy(w)
        launches = []

        def same(x, y, what):
            bad = int((x != y).sum())
            assert bad == 0, f"{what}: {bad} of {x.numel()} values differ, largest difference {float((x - y).abs().max()):.3e}"

        for step in range(5):                            # 1: plain calls, 2: capture + launch, 3-5: replays
            l0 = a.pm_launch_count()
            a.pm_step_graph(sa, ka, na, w.dt)
            launches.append(a.pm_launch_count() - l0)
            assert a.debug_graph_state() == min(step + 1, 2)       # plain calls, then captured, then replayed
            plain_step(b, sb, kb, nb, w.dt)
            a.pm_check(); b.pm_check()
            for name, fa, fb in zip(pm.DeviceState.FIELDS, sa.fields(), sb.fields()):
                same(fa, fb, f"{name}, step {step}")
            for f in ("m", "vx", "vy", "vz", "dm"):
                same(getattr(ka, f), getattr(kb, f), f"sink {f}, step {step}")
        assert len(set(launches)) == 1 and launches[0] > 0, launches       # the count advances as if the calls had been made
        # another dt: back to plain calls, capture again, replay -- still the same bits
        for step in range(3):
            a.pm_step_graph(sa, ka, na, 0.5 * w.dt)
            plain_step(b, sb, kb, nb, 0.5 * w.dt)
            for name, fa, fb in zip(pm.DeviceState.FIELDS, sa.fields(), sb.fields()):
                same(fa, fb, f"{name} after the change of dt, step {step}")
        # the retained buffer is the step's (sink creation and the debug views read it)
        # (the buffers keep the UNROUNDED sums -- the apply pass rounds as it reads -- so here the order of the additions shows)
        ra, rb = a.debug_buffer(0)[1], b.debug_buffer(0)[1]
        assert torch.equal(ra != 0, rb != 0) and bool(((ra - rb).abs() <= 1e-12 * rb.abs()).all())
        a.close(); b.close()


def test_graph_step_follows_the_oracle():
    w = inputs.scaled_mixed(40, 600, seed_index=6)
    o = parity.make_oracle(w)
    stream = torch.cuda.Stream(DEV)
    with torch.cuda.stream(stream):
        c = pm.Context(w.params, device="cuda:0", stream=stream)
        st, sk, sn = device_copy(w)
        for step in range(4):
            o.step(w.dt)
            c.pm_step_graph(st, sk, sn, w.dt, reuse_args=step > 0)
            c.pm_check()
            rho, m = st.rho.cpu().numpy(), sk.m.cpu().numpy()
            if step == 0:
                parity.close_strict(rho, o.state.rho, "rho")
                parity.close_strict(m, o.sinks.m, "sink m")
            assert np.all(np.abs(rho - o.state.rho) <= 1e-9 * np.abs(o.state.rho)), f"rho, step {step}"
            assert np.all(np.abs(st.etot.cpu().numpy() - o.state.etot) <= 1e-9 * np.abs(o.state.etot)), f"E, step {step}"
            assert np.all(np.abs(m - o.sinks.m) <= 1e-9 * np.abs(o.sinks.m)), f"sink m, step {step}"
        c.close()


def test_fallbacks_and_refusals():
    w = inputs.scaled_mixed(32, 200, seed_index=5)
    # the default stream of torch is the legacy default stream, which cannot be captured: the graph lives on a stream of the
    # ctx's own, ordered against the default stream by events -- interleaved with torch work on the default stream
    c = pm.Context(w.params, device="cuda:0", flags=pm.PM_FLAG_REPRODUCIBLE)
    d = pm.Context(w.params, device="cuda:0", flags=pm.PM_FLAG_REPRODUCIBLE)
    c.pm_set_repro_margin(40)
    d.pm_set_repro_margin(40)
    sc, kc, nc = device_copy(w)
    sd, kd, nd = device_copy(w)
    for step in range(5):
        sc.rho.mul_(1.0 + 1e-3 * step)                    # torch kernels on the default stream between the steps
        sd.rho.mul_(1.0 + 1e-3 * step)
        c.pm_step_graph(sc, kc, nc, w.dt)
        assert c.debug_graph_state() == min(step + 1, 2)
        plain_step(d, sd, kd, nd, w.dt)
        for fa, fb in zip(sc.fields(), sd.fields()):
            assert torch.equal(fa, fb), step
    # PM_FLAG_TIMING: plain calls every time
    t = pm.Context(w.params, device="cuda:0", flags=pm.PM_FLAG_TIMING)
    for _ in range(3):
        t.pm_step_graph(sc, kc, nc, w.dt)
        assert t.debug_graph_state() == 0
    assert t.pm_kernel_times()["sne"] > 0.0
    t.close()
    # only SNe: no return pass, the ctx is left where pm_apply_limited leaves it
    e = pm.Context(w.params, device="cuda:0")
    e.pm_step_graph(sc, None, nc, w.dt)
    e.pm_check()
    # a z slab has an exchange between the calls
    z = pm.Context(dict(w.params, z_slab=1), device="cuda:0")
    g = z.ghost_width()
    zs = pm.DeviceState(*(torch.ones((32 + 2 * g) * 32 * 32, dtype=torch.float64, device=DEV) for _ in range(6)))
    with pytest.raises(pm.PmError) as err:
        z.pm_step_graph(zs, None, None, w.dt)
    assert err.value.status == pm.PM_EINVAL
    for x in (c, d, e, z):
        x.close()
