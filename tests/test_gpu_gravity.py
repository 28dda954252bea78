"""GPU parity of the PM-gravity calls (pm_gravity_deposit / pm_gravity_kick / pm_drift) against oracle/pm_gravity_oracle.py,
through the C ABI.  Cell membership and wrapped indices bit-exact (which cells are non-zero); deposited densities within
1e-12 relative + the reorder term (atomic order varies); interpolated accelerations, kicks and drifts are fixed-order
sums and must agree to the last bit; totals within 1e-13."""
import numpy as np
import pytest
import torch

from oracle import pm_gravity_oracle as go
from paper_2509_18261_b200 import inputs, pm

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def fold_x_only(buf, g):
    """The oracle's ghost-zoned buffer (nz + 2g, ny + 2g, nx + 2g) with its x ghost columns added to the owned columns they
    image and then emptied: the kernels wrap x where they add (csrc/pm_device.cuh: deposit_index), so on the GPU only the y
    and z ghost zones ever hold anything before the fold."""
    out = buf.copy()
    out[:, :, g:2 * g] += buf[:, :, -g:]
    out[:, :, -2 * g:-g] += buf[:, :, :g]
    out[:, :, :g] = 0.0
    out[:, :, -g:] = 0.0
    return out


def run_deposit(w, with_gas=True):
    ctx = pm.Context(w.params, device=DEV)
    out = torch.empty(w.rho_gas.shape, dtype=torch.float64, device=DEV)
    ctx.pm_gravity_deposit(dev(w.rho_gas) if with_gas else None, dev(w.x), dev(w.y), dev(w.z), dev(w.m), out)
    ctx.pm_check()
    return ctx, out


def check_deposit(w, with_gas=True):
    ctx, out = run_deposit(w, with_gas)
    p = w.params
    ghosted, owned, g, ox = ctx.debug_buffer(1)
    # Step 1 alone: the ghost cells keep what was deposited into them (the fold leaves them in place)
    ref_buf = fold_x_only(go.gravity_deposit_buffer(p, w.x, w.y, w.z, w.m, g=g), g)
    gb = ghosted[:, :, ox - g:ox - g + p["nx"] + 2 * g].cpu().numpy()
    ghost_mask = np.ones(ref_buf.shape, dtype=bool)
    ghost_mask[g:-g, g:-g, g:-g] = False
    assert np.array_equal(gb[ghost_mask] != 0, ref_buf[ghost_mask] != 0), "ghost cell membership"
    # sum of positive terms: every partial sum is within n eps of the exact one
    tol = 1e-12 * np.abs(ref_buf) + 1e-300
    assert np.all(np.abs(gb - ref_buf)[ghost_mask] <= tol[ghost_mask]), "ghost cell values"
    # Steps 1 + 2: the folded buffer
    ref_owned = go.fold_ghosts(ref_buf, g)
    go_ = owned.cpu().numpy()
    assert np.array_equal(go_ != 0, ref_owned != 0), "owned cell membership"
    assert np.all(np.abs(go_ - ref_owned) <= 1e-12 * np.abs(ref_owned) + 1e-300), "folded buffer"
    # Steps 1, 2, 5: the density handed to the Poisson solver, against the oracle's own (ghost width 1) path
    ref = go.gravity_deposit(p, w.rho_gas if with_gas else None, w.x, w.y, w.z, w.m)
    got = out.cpu().numpy()
    assert np.all(np.abs(got - ref) <= 1e-12 * np.abs(ref) + 1e-300), "rho_tot"
    if not with_gas:
        assert np.array_equal(got != 0, ref != 0)
    # total mass
    V = float(p["dx"]) ** 3
    gas = float(w.rho_gas.sum()) if with_gas else 0.0
    total = float(out.sum().item()) * V
    assert abs(total - (gas * V + w.m.sum())) <= 1e-13 * (gas * V + w.m.sum())
    ctx.close()


def test_deposit_parity_cubic_even():
    check_deposit(inputs.gravity_workload(48, 20000))
    check_deposit(inputs.gravity_workload(48, 20000, seed_index=7), with_gas=False)


def test_deposit_parity_odd_noncubic_offset_origin():
    # nx odd: scalar fold / apply variants; non-cubic; dx != 1 and a shifted origin
    w = inputs.gravity_workload(33, 5000, seed_index=8, shape=(35, 33, 40), dx=0.37, x0=(-3.0, 11.5, 0.125))
    check_deposit(w)
    w = inputs.gravity_workload(40, 5000, seed_index=9, shape=(40, 37, 33), dx=2.5, x0=(1.0, 2.0, 3.0))
    check_deposit(w, with_gas=False)


def test_deposit_hand_placed_particles():
    """Cell centre, cell corner, box corner (all eight ghost octants), last half cell: exact binary fractions, so the GPU
    result is bit-equal to the hand-worked values whatever the order of the additions."""
    p = inputs.default_params(16)
    ctx = pm.Context(p, device=DEV)
    x = np.array([5.5, 3.0, 0.0, 15.75])
    y = np.array([2.5, 5.0, 0.0, 8.5])
    z = np.array([7.5, 2.0, 0.0, 0.25])
    m = np.array([3.0, 8.0, 16.0, 4.0])
    out = torch.empty((16, 16, 16), dtype=torch.float64, device=DEV)
    ctx.pm_gravity_deposit(None, dev(x), dev(y), dev(z), dev(m), out)
    ctx.pm_check()
    e = np.zeros((16, 16, 16))
    e[7, 2, 5] += 3.0
    e[1:3, 4:6, 2:4] += 1.0
    for k in (0, 15):
        for j in (0, 15):
            for i in (0, 15):
                e[k, j, i] += 2.0
    # (15.75, 8.5, 0.25): x cells 15 (0.75) and 16 -> 0 (0.25); y cell 8; z cells -1 -> 15 (0.25) and 0 (0.75)
    for k, wz in ((15, 0.25), (0, 0.75)):
        for i, wx in ((15, 0.75), (0, 0.25)):
            e[k, 8, i] += 4.0 * wx * wz
    assert np.array_equal(out.cpu().numpy(), e)
    assert np.array_equal(go.gravity_deposit(p, None, x, y, z, m), e)
    ctx.close()


def test_deposit_empty_and_order_errors():
    w = inputs.gravity_workload(24, 10)
    ctx = pm.Context(w.params, device=DEV)
    out = torch.empty((24, 24, 24), dtype=torch.float64, device=DEV)
    e = torch.empty(0, dtype=torch.float64, device=DEV)
    gas = dev(w.rho_gas)
    ctx.pm_gravity_deposit(gas, e, e, e, e, out)           # no particles: rho_tot = rho_gas
    ctx.pm_check()
    assert torch.equal(out, gas)
    ctx.pm_gravity_deposit(gas, dev(w.x), dev(w.y), dev(w.z), dev(w.m), gas)   # in place on the gas field
    ctx.pm_check()
    assert abs(float(gas.sum()) - (w.rho_gas.sum() + w.m.sum())) <= 1e-13 * (w.rho_gas.sum() + w.m.sum())
    # outside the box -> PM_EDOMAIN at the next pm_check
    bad = dev(np.array([24.0]))
    ok = dev(np.array([1.0]))
    ctx.pm_gravity_deposit(None, bad, ok, ok, ok, out)
    with pytest.raises(pm.PmError):
        ctx.pm_check()
    # mid-step: the buffer mesh is in use
    wk = inputs.scaled_mixed(24, 20)
    c2 = pm.Context(wk.params, device=DEV)
    st = pm.DeviceState.from_host(wk.state, torch.device(DEV))
    sk = pm.DeviceSinks.from_host(wk.sinks, torch.device(DEV))
    sn = pm.DeviceSNe.from_host(wk.sne, torch.device(DEV))
    c2.pm_deposit(st, sk, sn, wk.dt)
    with pytest.raises(pm.PmError):
        c2.pm_gravity_deposit(None, ok, ok, ok, ok, out)
    c2.pm_fold_ghosts()
    c2.pm_apply_limited(st)
    with pytest.raises(pm.PmError):
        c2.pm_drift(sk.x, sk.y, sk.z, sk.vx, sk.vy, sk.vz, 0.1)    # Step 4 still needs the positions
    c2.pm_return_to_particles(sk)
    c2.pm_gravity_deposit(None, ok, ok, ok, ok, out)
    c2.pm_check()
    ctx.close()
    c2.close()


def check_kick_and_drift(w):
    p = w.params
    ctx = pm.Context(p, device=DEV)
    gx, gy, gz = (dev(a) for a in w.g)
    x, y, z = dev(w.x), dev(w.y), dev(w.z)
    v = [dev(w.vx), dev(w.vy), dev(w.vz)]
    a = [torch.empty_like(x) for _ in range(3)]
    ctx.pm_gravity_kick(gx, gy, gz, x, y, z, v=None, a=a)          # interpolate only
    ctx.pm_check()
    ref_a = [go.gravity_interpolate(p, w.g[c], w.x, w.y, w.z) for c in range(3)]
    for c in range(3):
        assert np.array_equal(a[c].cpu().numpy(), ref_a[c]), f"a[{c}] not bit-equal"
    half = 0.5 * w.dt
    ctx.pm_gravity_kick(gx, gy, gz, x, y, z, v=v, dt=half, a=None)  # kick only
    ref_v = [go.kick(vv, aa, half) for vv, aa in zip((w.vx, w.vy, w.vz), ref_a)]
    for c in range(3):
        assert np.array_equal(v[c].cpu().numpy(), ref_v[c]), f"v[{c}] after the kick"
    # a long drift: many particles cross the seam, some by more than one box
    dt = 400.0
    ctx.pm_drift(x, y, z, v[0], v[1], v[2], dt)
    ctx.pm_check()
    n = (p["nx"], p["ny"], p["nz"])
    for c, (q, q0) in enumerate(zip((x, y, z), (w.x, w.y, w.z))):
        ref = go.drift(q0, ref_v[c], dt, p["x0"][c], n[c], p["dx"])
        got = q.cpu().numpy()
        assert np.array_equal(got, ref), f"drift axis {c}"
        assert got.min() >= p["x0"][c] and got.max() < p["x0"][c] + n[c] * p["dx"]
    assert (np.abs(ref_v[0] * dt) > n[0] * p["dx"]).any()            # the multi-box case did occur
    ctx.close()


def test_kick_and_drift_bit_equal():
    check_kick_and_drift(inputs.gravity_workload(48, 20000))
    check_kick_and_drift(inputs.gravity_workload(33, 5000, seed_index=8, shape=(35, 33, 40), dx=0.37, x0=(-3.0, 11.5, 0.125)))


def test_kdk_steps_match_the_oracle_with_a_deposit_in_the_loop():
    """Three kick-drift-kick steps where the acceleration mesh depends on the deposited density (a local stand-in for the
    Poisson solve, evaluated with torch on the GPU side and numpy on the oracle side from the SAME formula on the
    respective rho_tot): exercises deposit -> kick -> drift -> deposit -> kick chaining.  rho_tot differs by rounding
    order (atomics), so positions and velocities are compared to 1e-11 rather than bit for bit."""
    w = inputs.gravity_workload(32, 3000, seed_index=10)
    p = w.params
    n = 32

    def mesh_np(rho):
        return tuple(-1e-3 * (np.roll(rho, -1, ax) - np.roll(rho, 1, ax)) for ax in (2, 1, 0))

    def mesh_t(rho):
        return tuple((-1e-3 * (torch.roll(rho, -1, ax) - torch.roll(rho, 1, ax))).contiguous() for ax in (2, 1, 0))

    pos = (w.x.copy(), w.y.copy(), w.z.copy())
    vel = (w.vx.copy(), w.vy.copy(), w.vz.copy())
    ctx = pm.Context(p, device=DEV)
    x, y, z, m = dev(w.x), dev(w.y), dev(w.z), dev(w.m)
    v = [dev(w.vx), dev(w.vy), dev(w.vz)]
    gas = dev(w.rho_gas)
    rho = torch.empty_like(gas)
    dt = 0.5
    for _ in range(3):
        pos, vel = go.kdk_step(p, pos, vel, lambda q: mesh_np(go.gravity_deposit(p, w.rho_gas, q[0], q[1], q[2], w.m)), dt)
        ctx.pm_gravity_deposit(gas, x, y, z, m, rho)
        ctx.pm_gravity_kick(*mesh_t(rho), x, y, z, v=v, dt=0.5 * dt)
        ctx.pm_drift(x, y, z, v[0], v[1], v[2], dt)
        ctx.pm_gravity_deposit(gas, x, y, z, m, rho)
        ctx.pm_gravity_kick(*mesh_t(rho), x, y, z, v=v, dt=0.5 * dt)
    ctx.pm_check()
    for c, q in enumerate((x, y, z)):
        d = np.abs(q.cpu().numpy() - pos[c])
        d = np.minimum(d, n - d)                                   # a particle within rounding of the seam may wrap differently
        assert d.max() <= 1e-11 * n
        assert np.abs(v[c].cpu().numpy() - vel[c]).max() <= 1e-11
    ctx.close()


def test_full_size_sampled_and_invariants():
    """512^3 with 10^6 particles (the configuration bench.py times): total mass, non-negativity, and the densities of
    sampled cells against a one-by-one evaluation of the oracle's weights over the particles near them."""
    w = inputs.gravity_workload(512, 1_000_000)
    p = w.params
    ctx = pm.Context(p, device=DEV)
    out = torch.empty((512, 512, 512), dtype=torch.float64, device=DEV)
    x, y, z, m = dev(w.x), dev(w.y), dev(w.z), dev(w.m)
    ctx.pm_gravity_deposit(None, x, y, z, m, out)
    ctx.pm_check()
    total = float(out.sum().item())
    assert abs(total - w.m.sum()) <= 1e-13 * w.m.sum()
    assert float(out.min().item()) >= 0.0
    # sampled cells: host cells of random particles, their +1 neighbours, and the box corners
    rng = np.random.default_rng(77)
    pick = rng.choice(w.x.size, 200, replace=False)
    cells = set()
    for s in pick:
        i, j, k = int(w.x[s]), int(w.y[s]), int(w.z[s])
        cells.add((k, j, i))
        cells.add(((k + 1) % 512, (j + 1) % 512, (i + 1) % 512))
    cells |= {(a, b, c) for a in (0, 511) for b in (0, 511) for c in (0, 511)}
    i0, wx0, wx1 = go.cic_axis(w.x, 0.0, 1.0)
    j0, wy0, wy1 = go.cic_axis(w.y, 0.0, 1.0)
    k0, wz0, wz1 = go.cic_axis(w.z, 0.0, 1.0)
    got = out.cpu().numpy()
    for (k, j, i) in cells:
        ref = 0.0
        for dk, wz in ((0, wz0), (1, wz1)):
            for dj, wy in ((0, wy0), (1, wy1)):
                for di, wx in ((0, wx0), (1, wx1)):
                    sel = ((k0 + dk) % 512 == k) & ((j0 + dj) % 512 == j) & ((i0 + di) % 512 == i)
                    if sel.any():
                        ref += float((w.m[sel] * ((wz[sel] * wy[sel]) * wx[sel]) / 1.0).sum())
        assert abs(got[k, j, i] - ref) <= 1e-12 * abs(ref) + 1e-300, (k, j, i)
    # interpolation at full size: sampled particles, bit-equal
    gx, gy, gz = (dev(a) for a in w.g)
    a = [torch.empty_like(x) for _ in range(3)]
    ctx.pm_gravity_kick(gx, gy, gz, x, y, z, a=a)
    ctx.pm_check()
    for c in range(3):
        ref = go.gravity_interpolate(p, w.g[c], w.x[pick], w.y[pick], w.z[pick])
        assert np.array_equal(a[c].cpu().numpy()[pick], ref)
    ctx.close()


def test_bin_ordered_path_above_the_sort_threshold():
    """n >= 65536 particles: the library takes the particles in a1 bin order (a cached permutation shared by the deposit and
    the kick, invalidated by pm_drift).  Same checks as the small cases, then a drift and a second deposit + kick, which must
    follow the NEW positions (a stale order would still be a valid permutation; a stale index would not be)."""
    w = inputs.gravity_workload(64, 100_000, seed_index=11)
    check_deposit(w)
    check_kick_and_drift(w)
    p = w.params
    ctx = pm.Context(p, device=DEV)
    x, y, z, m = dev(w.x), dev(w.y), dev(w.z), dev(w.m)
    v = [dev(w.vx), dev(w.vy), dev(w.vz)]
    gx, gy, gz = (dev(a) for a in w.g)
    rho = torch.empty((64, 64, 64), dtype=torch.float64, device=DEV)
    ctx.pm_gravity_deposit(None, x, y, z, m, rho)                  # builds and caches the order
    ctx.pm_drift(x, y, z, v[0], v[1], v[2], 37.0)                  # invalidates it
    ctx.pm_gravity_deposit(None, x, y, z, m, rho)
    a = [torch.empty_like(x) for _ in range(3)]
    ctx.pm_gravity_kick(gx, gy, gz, x, y, z, a=a)                  # reuses the order of the second deposit
    ctx.pm_check()
    pos = [go.drift(q, vv, 37.0, 0.0, 64, 1.0) for q, vv in zip((w.x, w.y, w.z), (w.vx, w.vy, w.vz))]
    for c, q in enumerate((x, y, z)):
        assert np.array_equal(q.cpu().numpy(), pos[c])
    ref = go.gravity_deposit(p, None, pos[0], pos[1], pos[2], w.m)
    got = rho.cpu().numpy()
    assert np.array_equal(got != 0, ref != 0)
    assert np.all(np.abs(got - ref) <= 1e-12 * np.abs(ref) + 1e-300)
    for c in range(3):
        assert np.array_equal(a[c].cpu().numpy(), go.gravity_interpolate(p, w.g[c], *pos))
    # an exchange step in between reuses the bin memory: the gravity order must be rebuilt, not reused
    wk = inputs.scaled_mixed(64, 2000)
    st = pm.DeviceState.from_host(wk.state, torch.device(DEV))
    sk = pm.DeviceSinks.from_host(wk.sinks, torch.device(DEV))
    sn = pm.DeviceSNe.from_host(wk.sne, torch.device(DEV))
    ctx.step(st, sk, sn, wk.dt)
    ctx.pm_gravity_kick(gx, gy, gz, x, y, z, a=a)
    ctx.pm_check()
    for c in range(3):
        assert np.array_equal(a[c].cpu().numpy(), go.gravity_interpolate(p, w.g[c], *pos))
    ctx.close()


def test_kick_between_deposit_and_return_keeps_the_sink_order():
    """ADVICE r1 / VERDICT r1: a pm_gravity_kick with n >= 65536 particles between pm_deposit and pm_return_to_particles used
    to rebuild its particle order in the memory Step 4 reads the sink order from.  Gravity has its own scratch now: deposit ->
    kick -> fold -> kick -> apply -> kick -> return must give the oracle's sinks (m, dm strictly; v within the reorder bound),
    conserve mass, and interpolate exactly as a kick outside a step does."""
    from tests import parity
    w = inputs.scaled_mixed(64, 3000, seed_index=5)
    gw = inputs.gravity_workload(64, 70_000, seed_index=12)
    g = parity.GpuRun(w)
    o = parity.make_oracle(w)
    x, y, z = dev(gw.x), dev(gw.y), dev(gw.z)
    gx, gy, gz = (dev(a) for a in gw.g)
    acc = [[torch.empty_like(x) for _ in range(3)] for _ in range(3)]
    m0, _ = g.totals()
    g.ctx.pm_deposit(g.state, g.sinks, g.sne, w.dt)
    g.ctx.pm_gravity_kick(gx, gy, gz, x, y, z, a=acc[0])
    g.ctx.pm_fold_ghosts()
    g.ctx.pm_gravity_kick(gx, gy, gz, x, y, z, a=acc[1])
    g.ctx.pm_apply_limited(g.state)
    g.ctx.pm_gravity_kick(gx, gy, gz, x, y, z, a=acc[2])
    g.ctx.pm_return_to_particles(g.sinks)
    g.ctx.pm_check()
    o.step(w.dt)
    parity.compare_sinks(g, o)
    m1, _ = g.totals()
    assert abs((m1 - m0) - float(w.sne.m_ej.sum())) <= 1e-13 * abs(m1)
    for c in range(3):
        ref = go.gravity_interpolate(gw.params, gw.g[c], gw.x, gw.y, gw.z)
        for k in range(3):
            assert np.array_equal(acc[k][c].cpu().numpy(), ref)
    # a gravity deposit between apply and return (it works in buffer channel 1) does not disturb Step 4 either
    g2 = parity.GpuRun(w)
    rho = torch.empty((64, 64, 64), dtype=torch.float64, device=DEV)
    g2.ctx.pm_deposit(g2.state, g2.sinks, g2.sne, w.dt)
    g2.ctx.pm_fold_ghosts()
    g2.ctx.pm_apply_limited(g2.state)
    g2.ctx.pm_gravity_deposit(None, x, y, z, dev(gw.m), rho)
    g2.ctx.pm_return_to_particles(g2.sinks)
    g2.ctx.pm_check()
    parity.compare_sinks(g2, o)
    ref = go.gravity_deposit(gw.params, None, gw.x, gw.y, gw.z, gw.m)
    assert np.all(np.abs(rho.cpu().numpy() - ref) <= 1e-12 * np.abs(ref) + 1e-300)
    g.ctx.close(); g2.ctx.close()
