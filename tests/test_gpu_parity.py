"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs."""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs, pm
from tests import parity

pytestmark = pytest.mark.gpu


def test_native_library_loaded():
    L = pm.lib()
    assert L.pm_create is not None
    assert torch.cuda.is_available()
    assert torch.cuda.get_device_capability(0)[0] == 10, "sm_100a library needs a Blackwell GPU"


# ---------------------------------------------------------------------------------------------
# bit-exact integer work
# ---------------------------------------------------------------------------------------------
def _positions(n, rng, count):
    pos = rng.uniform(0.0, n, size=(count, 3))
    special = np.array([[0.0, 0.0, 0.0], [n - 1e-9, 0.5, n / 2], [0.5, 0.5, 0.5], [n / 2, n / 2, n / 2],
                        [1e-12, n - 1e-12, 3.25], [n - 0.5, n - 0.5, n - 0.5], [2.0, 3.0, 4.0], [2.5, 3.5, 4.5],
                        [7.125, 7.375, 7.625], [0.3, 0.1, 0.7]])
    return np.concatenate([special, pos])


@pytest.mark.parametrize("n,dx,x0,rk", [(16, 1.0, (0.0, 0.0, 0.0), 4.0), (20, 0.37, (-1.3, 2.2, 0.11), 4 * 0.37),
                                        (12, 1.0, (0.0, 0.0, 0.0), 2.6), (24, 2.0, (5.0, 5.0, 5.0), 7.0)])
def test_sink_membership_bit_exact(n, dx, x0, rk):
    p = inputs.default_params(n)
    p.update(dx=dx, x0=x0, rk_sink=rk, rk_sn=min(rk, 3 * dx))
    ctx = pm.Context(p)
    rng = np.random.default_rng(11)
    for q in _positions(n, rng, 60):
        x, y, z = (x0[a] + q[a] * dx for a in range(3))
        cnt, host = ctx.debug_stencil(0, x, y, z)
        cells = po.sink_stencil(p, x, y, z)
        g = cnt.shape[0] // 2
        want = np.zeros(cnt.shape, dtype=np.int32)
        for i, j, k in cells:
            want[k - host[2] + g, j - host[1] + g, i - host[0] + g] = 1
        assert np.array_equal(cnt.numpy(), want), f"membership differs at {(x, y, z)}"
    ctx.close()


@pytest.mark.parametrize("nsub", [1, 2, 3, 4, 8])
@pytest.mark.parametrize("n,dx,x0,rk", [(16, 1.0, (0.0, 0.0, 0.0), 3.0), (20, 0.37, (-1.3, 2.2, 0.11), 3 * 0.37),
                                        (12, 1.0, (0.0, 0.0, 0.0), 2.2)])
def test_sn_omega_counts_bit_exact(nsub, n, dx, x0, rk):
    p = inputs.default_params(n)
    p.update(dx=dx, x0=x0, rk_sn=rk, rk_sink=rk, sn_nsub=nsub)
    ctx = pm.Context(p)
    rng = np.random.default_rng(13)
    for q in _positions(n, rng, 40):
        x, y, z = (x0[a] + q[a] * dx for a in range(3))
        cnt, host = ctx.debug_stencil(1, x, y, z)
        want, host_o = po.sn_omega_box(p, x, y, z)
        assert tuple(host_o) == host
        assert np.array_equal(cnt.numpy(), want), f"omega counts differ at {(x, y, z)} nsub={nsub}"
    ctx.close()


# ---------------------------------------------------------------------------------------------
# element-by-element parity, stage by stage
# ---------------------------------------------------------------------------------------------
def test_config1_tiny_sink():
    w = inputs.make(1)
    g, o, _ = parity.run_and_compare(w, steps=1)
    # the closed form the oracle is pinned to (Bondi, L326) holds for the GPU result too
    assert float(g.sinks.dm[0]) == pytest.approx(6.543626026975605, rel=1e-12)


def test_config3_single_sn():
    w = inputs.make(3)
    g, o, _ = parity.run_and_compare(w, steps=1)
    assert float(g.ctx.debug_buffer(1)[1].sum()) == pytest.approx(1.0, rel=1e-13)        # sum d rho V = M_ej
    assert float(g.ctx.debug_buffer(5)[1].sum()) == pytest.approx(1e4, rel=1e-13)        # sum d E V = E_sn (v = 0)


@pytest.mark.parametrize("n,npart", [(40, 500), (37, 400), (48, 1200)])
def test_mixed_small_grids(n, npart):
    """Config-5-shaped mixes on grids that span several tiles with ragged tails; odd n takes the scalar apply path."""
    w = inputs.scaled_mixed(n, npart, seed_index=5)
    g, o, n2 = parity.run_and_compare(w, steps=3)
    assert (o.eta < 1).sum() > 0 and (o.lam < 1).sum() > 0           # both limiters exercised
    print(f"cells needing the R36 reorder term: {n2}")


def test_generic_kernels_same_contract(monkeypatch):
    """PM_FLAG_GENERIC_KERNELS: the any-radius / any-n_sub kernels on the shapes the specialised ones normally take."""
    w = inputs.scaled_mixed(40, 500, seed_index=5)
    flags = pm.PM_FLAG_DEBUG_SCALARS | pm.PM_FLAG_DEBUG_LAMBDA | pm.PM_FLAG_GENERIC_KERNELS
    orig = parity.GpuRun.__init__
    monkeypatch.setattr(parity.GpuRun, "__init__", lambda self, w_, device="cuda:0", flags=flags: orig(self, w_, device, flags))
    parity.run_and_compare(w, steps=2)


def test_seam_particles():
    """Particles whose stencils straddle the periodic seam in every direction exercise ghosts + fold (L284 analogue)."""
    w = inputs.scaled_mixed(32, 64, seed_index=5)
    n = 32.0
    edge = np.array([0.0, 0.2, n - 0.2, n - 1e-9, 1.5, n - 1.5, 3.9, n - 3.9])
    rng = np.random.default_rng(5)
    for prt in (w.sinks, w.sne):
        for f in ("x", "y", "z"):
            getattr(prt, f)[:] = rng.choice(edge, size=prt.n)
    g, o, _ = parity.run_and_compare(w, steps=2)
    ghosted, owned, gz, ox = g.ctx.debug_buffer(1)
    ghost_sum = float(ghosted.abs().sum() - owned.abs().sum())
    assert ghost_sum > 0.0, "seam particles must have deposited into ghost zones"
    # x is wrapped where the particles add (deposit_index): the x ghost columns stay empty, y and z ghost zones are used
    xg = torch.cat([ghosted[:, :, :ox], ghosted[:, :, ox + 32:]], dim=2)
    assert float(xg.abs().sum()) == 0.0


def test_stacked_particles_contention():
    """100 SNe and 20 sinks on (nearly) the same spot: maximum atomic contention on a few hundred cells."""
    w = inputs.scaled_mixed(32, 120, seed_index=5)
    rng = np.random.default_rng(9)
    for prt in (w.sinks, w.sne):
        prt.x[:] = 15.7 + 1e-3 * rng.standard_normal(prt.n)
        prt.y[:] = 16.2 + 1e-3 * rng.standard_normal(prt.n)
        prt.z[:] = 0.4 + 1e-3 * rng.standard_normal(prt.n)
    w.sinks.z[:] = np.mod(w.sinks.z, 32.0)
    w.sne.z[:] = np.mod(w.sne.z, 32.0)
    parity.run_and_compare(w, steps=1)


def test_shared_memory_tile_accumulator_path(monkeypatch):
    """PM_FLAG_SMEM_TILES: supernova bins with >= 48 particles go through the shared-memory-privatised tile accumulator (one
    CTA per tile, flushed once), the rest through the direct path; both in one step.  Clustered workloads, a stack of 100
    supernovae on one spot, a cluster on the periodic corner (the flush reaches ghost zones in all three directions)."""
    flags = pm.PM_FLAG_DEBUG_SCALARS | pm.PM_FLAG_DEBUG_LAMBDA | pm.PM_FLAG_SMEM_TILES
    orig = parity.GpuRun.__init__
    monkeypatch.setattr(parity.GpuRun, "__init__", lambda self, w_, device="cuda:0", flags=flags: orig(self, w_, device, flags))
    w = inputs.scaled_mixed(48, 4000, seed_index=5, n_clusters=2)       # two clusters of ~900 supernovae: bins of 50-300
    g, o, _ = parity.run_and_compare(w, steps=2)
    sn_bins = np.bincount((np.floor(w.sne.z / 8) * 36 + np.floor(w.sne.y / 8) * 6 + np.floor(w.sne.x / 8)).astype(int), minlength=216)
    assert (sn_bins >= 48).sum() >= 3 and ((sn_bins > 0) & (sn_bins < 48)).sum() >= 20      # both paths are taken
    w = inputs.scaled_mixed(32, 120, seed_index=5)
    rng = np.random.default_rng(9)
    for prt, c in ((w.sinks, (15.7, 16.2, 0.4)), (w.sne, (31.6, 0.3, 31.9))):          # the SN stack sits on the periodic corner
        prt.x[:] = np.mod(c[0] + 1e-3 * rng.standard_normal(prt.n), 32.0)
        prt.y[:] = np.mod(c[1] + 1e-3 * rng.standard_normal(prt.n), 32.0)
        prt.z[:] = np.mod(c[2] + 1e-3 * rng.standard_normal(prt.n), 32.0)
    parity.run_and_compare(w, steps=1)
    w = inputs.scaled_mixed(37, 3000, seed_index=5, n_clusters=1)       # odd grid: scalar paths, ragged last tile
    parity.run_and_compare(w, steps=1)


def test_only_sinks_and_only_sne_and_empty():
    w = inputs.scaled_mixed(32, 200, seed_index=5)
    w1 = inputs.Workload("sinks", w.params, w.state.copy(), w.sinks.copy(), inputs.empty_sne(), w.dt, 1)
    parity.run_and_compare(w1, steps=2)
    w2 = inputs.Workload("sne", w.params, w.state.copy(), inputs.empty_sinks(), w.sne.copy(), w.dt, 1)
    parity.run_and_compare(w2, steps=2)
    w3 = inputs.Workload("empty", w.params, w.state.copy(), inputs.empty_sinks(), inputs.empty_sne(), w.dt, 1)
    g = parity.GpuRun(w3)
    g.step()
    g.ctx.pm_check()
    for a, b in zip(g.state_np(), w.state.fields()):
        assert np.array_equal(a, b)                                  # nothing deposited: state bit-identical
    for ch in range(6):
        assert float(g.ctx.debug_buffer(ch)[0].abs().sum()) == 0.0


def test_sn_only_params_ghost3():
    """rk_sink = 0: ghost width 3 (odd), exercising the padded x-origin; minimum grid 2g+1 = 7."""
    w = inputs.scaled_mixed(7, 12, seed_index=5, n_clusters=1)
    w.params["rk_sink"] = 0.0
    w = inputs.Workload("sn7", w.params, w.state, inputs.empty_sinks(), w.sne, w.dt, 1)
    parity.run_and_compare(w, steps=1)


def test_regimes_and_nsub1():
    """EJ / ST / MC each hit (R27's unit cases) and the binary-omega variant."""
    for rho0, regime in ((0.01, 1), (0.3, 2), (3.0, 3)):
        w = inputs.scaled_mixed(24, 30, seed_index=5)
        w.state = inputs.State(*(f * rho0 for f in w.state.fields()))
        w.params["sn_nsub"] = 1 if regime == 2 else 4
        g, o, _ = parity.run_and_compare(w, steps=1)
        assert (o.sn_diag["regime"] == regime).sum() > 0


def test_cs_iso_and_theta0_and_f_quarter():
    w = inputs.scaled_mixed(32, 300, seed_index=5)
    w.params.update(cs_iso=1.3, sn_eint_theta=0.0, f_max_remove=0.25, rho_floor=0.05)
    parity.run_and_compare(w, steps=2)


def test_permutation_invariance_gpu():
    """L243: particle order changes the result only at rounding level (and only through atomic order)."""
    w = inputs.scaled_mixed(32, 300, seed_index=5)
    outs = []
    for seed in (None, 3):
        ww = inputs.Workload(w.name, w.params, w.state.copy(), w.sinks.copy(), w.sne.copy(), w.dt, 1)
        if seed is not None:
            rng = np.random.default_rng(seed)
            pk, pn = rng.permutation(ww.sinks.n), rng.permutation(ww.sne.n)
            ww.sinks = inputs.Sinks(*(getattr(ww.sinks, f)[pk].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "m")))
            ww.sne = inputs.SNe(*(getattr(ww.sne, f)[pn].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")))
        g = parity.GpuRun(ww)
        g.step()
        outs.append(g.state_np())
    for a, b in zip(outs[0], outs[1]):
        assert np.allclose(a, b, rtol=1e-9, atol=1e-9 * np.abs(a).max())
    assert np.allclose(outs[0][0], outs[1][0], rtol=1e-12, atol=0)


def test_eq21_fallback_branch_on_the_gpu():
    """R25 fall-back (a reading, "parity unpinned"): exercised on BOTH sides.  (a) Gas far hotter than the ejecta
    (e_int / rho = 1e6 against (E_sn + E_kin) / M_ej ~ 1): adding the SN mass at the cell's own specific internal energy needs
    more energy than the SN brings, K < 0, no lambda satisfies Eq. 21 (discriminant < 0 by Cauchy-Schwarz): lambda = 0 in
    every touched cell.  (b) A state with E < KE (inconsistent input): e_int = E_2 - KE comes out negative and is clipped to 0."""
    w = inputs.scaled_mixed(32, 200, seed_index=5)
    st = w.state
    for f in ("mx", "my", "mz"):
        getattr(st, f)[...] *= 20.0                                  # |v| ~ 1
    ke = 0.5 * (st.mx ** 2 + st.my ** 2 + st.mz ** 2) / st.rho
    st.eint[...] = 1e6 * st.rho
    st.etot[...] = st.eint + ke
    w.sne.e_sn[:] = 1.0
    g, o, _ = parity.run_and_compare(w, steps=1)
    touched = o.sn_count > 0
    assert touched.sum() > 1000 and np.all(o.lam[touched] == 0.0)
    lam = g.ctx.debug_lambda().cpu().numpy().reshape(-1)
    assert np.all(lam[touched] == 0.0) and np.all(lam[~touched] == 1.0)
    # (b)
    w = inputs.scaled_mixed(32, 200, seed_index=5)
    st = w.state
    for f in ("mx", "my", "mz"):
        getattr(st, f)[...] *= 40.0
    ke = 0.5 * (st.mx ** 2 + st.my ** 2 + st.mz ** 2) / st.rho
    st.eint[...] = 1e-8 * st.rho
    st.etot[...] = 0.5 * ke
    w.sne.e_sn[:] = 1e-3
    w = inputs.Workload("clip", w.params, st, inputs.empty_sinks(), w.sne, w.dt, 1)
    g, o, _ = parity.run_and_compare(w, steps=1)
    touched = (o.sn_count > 0).reshape(o.shape)
    assert (o.state.eint[touched] == 0.0).sum() > 100
    assert np.array_equal(g.state.eint.cpu().numpy() == 0.0, o.state.eint == 0.0)


# ---------------------------------------------------------------------------------------------
# the BASELINE configs at full size
# ---------------------------------------------------------------------------------------------
def test_config2_bondi_100_steps():
    w = inputs.make(2)
    g, o, n2 = parity.run_and_compare(w, steps=w.steps)
    assert float(g.sinks.m[0]) > 100.0
    assert (o.eta < 1).sum() > 0                                     # limiter-dominated (requested mdot dt >> gas)


def test_config4_clustered_10_steps():
    """BASELINE config 4 at its stated size, ALL ten steps element by element against the oracle (about 5 s of oracle time
    per step).  No retry: a failure names quantity, cell, both values and the bound (also in gpurun_out/parity_failures.log)."""
    w = inputs.make(4)
    g, o, n2 = parity.run_and_compare(w, steps=w.steps)
    print(f"config 4: cells needing the R36 reorder term over {w.steps} steps: {n2}")
    g.ctx.pm_check()
    assert float(g.state.rho.min()) > 0 and float(g.state.eint.min()) >= 0
    assert (o.lam < 1).sum() > 100 and (o.eta < 1).sum() > 0          # both limiters are at work in the last step too


def test_config5_full_mesh_one_step():
    """BASELINE config 5 (512^3, 10^6 particles) in the launch configuration bench.py times: ONE whole step compared on
    every one of the 1.3e8 cells and on every particle (the oracle needs about 90 s for it); the sampled test below covers
    the following steps."""
    w = inputs.make(5)
    g, o, n2 = parity.run_and_compare(w, steps=1, lean=True)
    print(f"config 5: cells needing the R36 reorder term: {n2}")
    assert (o.lam < 1).sum() > 1000 and (o.eta < 1).sum() > 1000


def test_config5_large_sampled():
    """512^3 with 10^6 particles in the launch configuration bench.py times: sampled cells and particles against
    the oracle evaluated one by one (orc_sample_cells / orc_particle_scalars), plus invariants at full size."""
    w = inputs.make(5)
    g = parity.GpuRun(w)
    o = po.Oracle(w.params, w.state, w.sinks, w.sne, mesh=False)     # sampled evaluation only: no 512^3 meshes
    N = o.N
    rng = np.random.default_rng(55)
    # cells: random + neighbourhoods of random particles (dense) + domain corners
    hosts = []
    for prt, k in ((w.sne, 150), (w.sinks, 60)):
        idx = rng.choice(prt.n, k, replace=False)
        off = rng.integers(-3, 4, size=(k, 3))
        i = (np.floor(prt.x[idx]).astype(np.int64) + off[:, 0]) % 512
        j = (np.floor(prt.y[idx]).astype(np.int64) + off[:, 1]) % 512
        kk = (np.floor(prt.z[idx]).astype(np.int64) + off[:, 2]) % 512
        hosts.append((kk * 512 + j) * 512 + i)
    cells = np.unique(np.concatenate(hosts + [rng.integers(0, N, 150), np.array([0, 511, N - 1, N - 512])])).astype(np.int64)
    ref = o.sample_cells(cells, w.dt)
    m0, _ = g.totals()
    g.ctx.pm_deposit(g.state, g.sinks, g.sne, w.dt)
    g.ctx.pm_fold_ghosts()
    kz, jy, ix = cells // (512 * 512), (cells // 512) % 512, cells % 512
    kz_t, jy_t, ix_t = (torch.from_numpy(a).to(g.dev) for a in (kz, jy, ix))

    def owned_at(ch):
        return g.ctx.debug_buffer(ch)[1][kz_t, jy_t, ix_t].cpu().numpy()
    parity.close_reorder(owned_at(0), ref["A"][:, 0], ref["Aabs"][:, 0], "accretion d rho (sampled)")
    parity.close_strict(owned_at(1), ref["S"][:, 0], "SN d rho (sampled)")
    for f in (1, 2, 3, 4):
        parity.close_reorder(owned_at(1 + f), ref["S"][:, f], ref["Sabs"][:, f], f"SN channel {f} (sampled)")
    assert (ref["sn_count"] > 3).sum() > 20                          # overlapping stencils are in the sample
    g.ctx.pm_apply_limited(g.state)
    new = [f.reshape(-1)[torch.from_numpy(cells).to(g.dev)].cpu().numpy() for f in g.state.fields()]
    parity.close_strict(new[0], ref["unew"][:, 0], "rho (sampled)")
    parity.close_strict(new[4], ref["unew"][:, 4], "E (sampled)")
    eps = np.finfo(np.float64).eps
    for f in (1, 2, 3):
        scale = 100.0 * ref["Sabs"][:, f] + 100.0 * np.abs(ref["unew"][:, f])
        parity.close_reorder(new[f], ref["unew"][:, f], scale, f"p[{f - 1}] (sampled)")
    parity.close_reorder(new[5], ref["unew"][:, 5], 1e3 * np.abs(ref["unew"][:, 4]), "e_int (sampled)")
    lam = g.ctx.debug_lambda().reshape(-1)[torch.from_numpy(cells).to(g.dev)].cpu().numpy()
    assert np.all(lam[ref["sn_count"] == 0] == 1.0)
    assert np.abs(lam - ref["lam"]).max() < 1e-6
    # sampled sinks: Eq. 5 from the oracle's (cell, a) lists and the oracle's eta at those cells
    g.ctx.pm_return_to_particles(g.sinks)
    g.ctx.pm_check()
    for s in rng.choice(w.sinks.n, 3, replace=False):
        cl, a = o.sink_amounts(int(s), w.dt)
        eta = o.sample_cells(cl, w.dt)["eta"]
        dm = float(np.sum(eta * a * 1.0))
        assert float(g.sinks.dm[s]) == pytest.approx(dm, rel=1e-12)
    # sampled per-particle scalars (the oracle evaluates only the sampled particles)
    ks, ns = np.sort(rng.choice(w.sinks.n, 300, replace=False)), np.sort(rng.choice(w.sne.n, 300, replace=False))
    sk = inputs.Sinks(*(getattr(w.sinks, f)[ks].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "m")))
    sn = inputs.SNe(*(getattr(w.sne, f)[ns].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")))
    op = po.Oracle(w.params, w.state, sk, sn, mesh=False)
    op.particle_scalars()
    dk = g.ctx.debug_sink_scalars().cpu().numpy()[:, ks]
    for row, key in enumerate(("rho_inf", "v_inf", "c_inf", "r_bh", "mdot", "r_acc", "wsum")):
        parity.close_strict(dk[row], op.sink_diag[key], f"sink {key} (sampled)")
    assert np.array_equal(dk[7].astype(np.int64), op.sink_diag["n_member"].astype(np.int64))
    dn = g.ctx.debug_sn_scalars().cpu().numpy()[:, ns]
    for row, key in ((0, "m_snr"), (1, "v_snr"), (5, "n_h"), (6, "r_m"), (7, "p_rad")):
        parity.close_strict(dn[row], op.sn_diag[key], f"SN {key} (sampled)")
    assert np.array_equal(dn[8].astype(np.int32), op.sn_diag["regime"])
    # full-size invariants on the GPU result: Eq. 1 and limiter bounds
    m1, _ = g.totals()
    assert abs((m1 - m0) - float(w.sne.m_ej.sum())) <= 1e-13 * abs(m1)
    rho_old = torch.from_numpy(w.state.rho).to(g.dev)
    f, fl = w.params["f_max_remove"], w.params["rho_floor"]
    assert bool((g.state.rho >= torch.minimum(rho_old, torch.tensor(fl, device=g.dev, dtype=torch.float64)) * (1 - 1e-15)).all())
    assert float(g.state.eint.min()) >= 0.0
    del rho_old
    # the remaining steps of the config: invariants
    for _ in range(2):
        ma, _ = g.totals()
        g.step()
        mb, _ = g.totals()
        assert abs((mb - ma) - float(w.sne.m_ej.sum())) <= 1e-13 * abs(mb)
    g.ctx.pm_check()


# ---------------------------------------------------------------------------------------------
# error behaviour of the C ABI
# ---------------------------------------------------------------------------------------------
def test_errors():
    p = inputs.default_params(8)                                    # 8 < 2*4+1
    with pytest.raises(pm.PmError) as e:
        pm.Context(p)
    assert e.value.status == pm.PM_EINVAL
    w = inputs.scaled_mixed(16, 20, seed_index=5, n_clusters=1)
    g = parity.GpuRun(w)
    with pytest.raises(pm.PmError) as e:
        g.ctx.pm_apply_limited(g.state)
    assert e.value.status == pm.PM_EORDER
    with pytest.raises(pm.PmError) as e:
        g.ctx.pm_fold_ghosts()
    assert e.value.status == pm.PM_EORDER
    # a particle outside the domain is skipped and reported by pm_check
    g.sne.x[0] = 16.5
    g.step()
    with pytest.raises(pm.PmError) as e:
        g.ctx.pm_check()
    assert e.value.status == pm.PM_EDOMAIN
    g.sne.x[0] = 3.5
    g.step()
    g.ctx.pm_check()


def test_step_host_matches_device_path():
    w = inputs.scaled_mixed(32, 300, seed_index=5)
    g = parity.GpuRun(w)
    g.step()
    g.ctx.pm_check()
    hs, hk, hn = w.state.copy(), w.sinks.copy(), w.sne.copy()
    hk.dm = np.zeros(hk.n); hk.dpx = np.zeros(hk.n); hk.dpy = np.zeros(hk.n); hk.dpz = np.zeros(hk.n)
    ctx = pm.Context(w.params)
    ctx.pm_step_host(hs, hk, hn, w.dt)
    for a, b in zip(g.state_np(), hs.fields()):
        assert np.allclose(a, b, rtol=1e-10, atol=1e-10 * np.abs(a).max())
    assert np.allclose(g.sinks.m.cpu().numpy(), hk.m, rtol=1e-12)
    assert np.allclose(g.sinks.dm.cpu().numpy(), hk.dm, rtol=1e-12)
    assert ctx.pm_launch_count() == 12      # 4 binning, 3 reset (stamp, tile-wise zero, sweep), 2 deposits, fold, apply, return
    # two slots in flight: same results as one step at a time, each slot in its own host buffers
    a, b = (w.state.copy(), w.sinks.copy()), (w.state.copy(), w.sinks.copy())
    for _, k in (a, b):
        k.dm = np.zeros(k.n); k.dpx = np.zeros(k.n); k.dpy = np.zeros(k.n); k.dpz = np.zeros(k.n)
    ctx.pm_step_host_begin(0, a[0], a[1], hn, w.dt)
    ctx.pm_step_host_begin(1, b[0], b[1], hn, w.dt)
    with pytest.raises(pm.PmError) as e:
        ctx.pm_step_host_begin(1, b[0], b[1], hn, w.dt)          # slot 1 is in flight
    assert e.value.status == pm.PM_EORDER
    ctx.pm_step_host_end(0)
    ctx.pm_step_host_begin(0, a[0], a[1], hn, w.dt)              # second step of a, while b may still be downloading
    ctx.pm_step_host_end(1)
    ctx.pm_step_host_end(0)
    for x, y in zip(hs.fields(), b[0].fields()):
        assert np.allclose(x, y, rtol=1e-10, atol=1e-10 * np.abs(x).max())
    assert np.allclose(hk.m, b[1].m, rtol=1e-12) and np.all(a[1].m > b[1].m)     # a has taken two steps


def test_kernel_times_and_red_probe():
    """pm_kernel_times (PM_FLAG_TIMING) reports every group that ran; pm_probe_red_f64 returns a positive rate."""
    w = inputs.scaled_mixed(48, 1200, seed_index=5)
    dev = torch.device("cuda:0")
    ctx = pm.Context(w.params, device="cuda:0", flags=pm.PM_FLAG_TIMING)
    st = pm.DeviceState.from_host(w.state, dev)
    sk = pm.DeviceSinks.from_host(w.sinks, dev)
    sn = pm.DeviceSNe.from_host(w.sne, dev)
    ctx.step(st, sk, sn, w.dt)
    ms = ctx.pm_kernel_times()
    assert set(ms) == set(pm.KERNEL_GROUPS)
    assert all(v > 0.0 for v in ms.values()), ms
    ctx.pm_deposit(st, None, sn, w.dt)            # no sinks: that group reports 0
    ctx.pm_fold_ghosts(); ctx.pm_apply_limited(st); ctx.pm_return_to_particles(None)
    ms = ctx.pm_kernel_times()
    assert ms["sinks"] == 0.0 and ms["return"] == 0.0 and ms["sne"] > 0.0
    assert ctx.pm_probe_red_f64(8 << 20, 5) > 1.0
    plain = pm.Context(w.params, device="cuda:0")
    with pytest.raises(pm.PmError):
        plain.pm_kernel_times()


@pytest.mark.parametrize("n,npart", [(72, 3000), (130, 6000)])
def test_mixed_ragged_grids_clustered(n, npart):
    """Grid sizes that are no multiple of the 8-cell tile or the 64-cell super-block, few dense clusters (heavy stencil overlap)."""
    w = inputs.scaled_mixed(n, npart, seed_index=5, n_clusters=3)
    g, o, _ = parity.run_and_compare(w, steps=1)
    g.ctx.close()


@pytest.mark.parametrize("rk_sink,rk_sn,dx", [(3.3, 2.6, 1.0), (4.0 * 0.37, 3.0 * 0.37, 0.37), (3.01, 2.01, 1.0)])
def test_fast_kernels_other_radii_and_spacing(rk_sink, rk_sn, dx):
    """The specialised kernels serve every radius with ceil(r_K / dx) = 4 (sinks) / 3 (SNe), any dx and origin: member masks,
    omega counts and the separable Gaussian must follow r_K and dx, not the BASELINE values 4 dx / 3 dx."""
    w = inputs.scaled_mixed(40, 500, seed_index=5)
    n = 40
    w.params.update(dx=dx, x0=(-1.3, 2.2, 0.11), rk_sink=rk_sink, rk_sn=rk_sn)
    for p in (w.sinks, w.sne):                      # positions were drawn in [0, n): map them into the shifted, scaled box
        p.x[:] = p.x * dx + w.params["x0"][0]; p.y[:] = p.y * dx + w.params["x0"][1]; p.z[:] = p.z * dx + w.params["x0"][2]
    for p in (w.sinks, w.sne):
        for arr, o in ((p.x, 0), (p.y, 1), (p.z, 2)):
            np.clip(arr, w.params["x0"][o], np.nextafter(w.params["x0"][o] + n * dx, -np.inf), out=arr)
    parity.run_and_compare(w, steps=2)


def test_generic_and_fast_kernels_agree_bitwise_on_integers():
    """Member counts (sinks) and regimes (SNe) from the generic and the specialised kernels are identical."""
    w = inputs.scaled_mixed(40, 500, seed_index=5)
    outs = []
    for flags in (0, pm.PM_FLAG_GENERIC_KERNELS):
        g = parity.GpuRun(w, flags=pm.PM_FLAG_DEBUG_SCALARS | pm.PM_FLAG_DEBUG_LAMBDA | flags)
        g.ctx.pm_deposit(g.state, g.sinks, g.sne, w.dt)
        outs.append((g.ctx.debug_sink_scalars().cpu().numpy()[7].copy(), g.ctx.debug_sn_scalars().cpu().numpy()[8].copy(),
                     g.ctx.debug_sn_scalars().cpu().numpy()[1].copy()))
        g.ctx.pm_fold_ghosts(); g.ctx.pm_apply_limited(g.state); g.ctx.pm_return_to_particles(g.sinks); g.ctx.pm_check()
    assert np.array_equal(outs[0][0], outs[1][0])
    assert np.array_equal(outs[0][1], outs[1][1])
    assert np.allclose(outs[0][2], outs[1][2], rtol=1e-13, atol=0)     # V_snr = (sum of omega counts) V / 64


def test_sn_subsamples_exactly_on_the_kernel_radius():
    """Supernovae an odd multiple of dx/8 off a cell corner: every sub-sample offset is a multiple of dx/4, 30 of them lie
    exactly ON r_K = 3 dx and many more within a few ulp of the rounding boundary of the test (L203).  The specialised
    kernel's threshold form of the test must give the oracle's counts: V_snr bit for bit, buffers within tolerance."""
    w = inputs.scaled_mixed(24, 64, seed_index=5)
    assert w.params["dx"] == 1.0 and w.params["rk_sn"] == 3.0 and w.params["sn_nsub"] == 4
    rng = np.random.default_rng(11)
    eighths = np.array([0.125, 0.375, 0.625, 0.875])
    for f in ("x", "y", "z"):
        getattr(w.sne, f)[:] = rng.integers(0, 24, size=w.sne.n) + rng.choice(eighths, size=w.sne.n)
    # a few more a hair off the exact positions: sums that straddle the rounding boundary of r_K^2
    k = w.sne.n // 2
    w.sne.x[:k] = np.nextafter(w.sne.x[:k], np.where(rng.random(k) < 0.5, -np.inf, np.inf))
    g, o, _ = parity.run_and_compare(w, steps=1)
    v_gpu = g.ctx.debug_sn_scalars().cpu().numpy()[1]
    assert np.array_equal(v_gpu, o.sn_diag["v_snr"]), "V_snr = (sum of omega counts) V / 64 must match bit for bit"
    exact = w.sne.x == np.round(w.sne.x * 8) / 8
    assert np.all(v_gpu[exact] == 7153.0 / 64.0)
