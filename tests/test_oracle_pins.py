"""Pins of the CPU oracle (oracle/pm_oracle.c) against what the paper and the mathematics fix.

None of these tests re-types an oracle formula: each compares the oracle with a printed value
(tests/golden/*.txt), a closed form, an invariant, a special case or a brute-force evaluation over
ALL cells with minimum-image distances (independent of the oracle's stencil walk + index wrapping).
Citations are PAPER.md line numbers; R-numbers are DESIGN.md readings.
"""
import math
import os

import numpy as np
import pytest

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs


# ---------------------------------------------------------------------------------------------
def read_golden(path):
    out = {}
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()[:2]
                out[k] = float(v)
    return out


def uniform_workload(n, rho0=1.0, pressure=1.0, v=(0.0, 0.0, 0.0)):
    p = inputs.default_params(n)
    shp = (n, n, n)
    rho = np.full(shp, rho0)
    eint = np.full(shp, pressure / (p["gamma"] - 1.0))
    st = inputs.State(rho, rho * v[0], rho * v[1], rho * v[2], eint + 0.5 * rho * sum(c * c for c in v), eint)
    return p, st


def one_sink(pos, m, v=(0.0, 0.0, 0.0)):
    a = lambda x: np.array([float(x)])
    return inputs.Sinks(a(pos[0]), a(pos[1]), a(pos[2]), a(v[0]), a(v[1]), a(v[2]), a(m))


def one_sn(pos, e_sn=1e4, m_ej=1.0, v=(0.0, 0.0, 0.0)):
    a = lambda x: np.array([float(x)])
    return inputs.SNe(a(pos[0]), a(pos[1]), a(pos[2]), a(v[0]), a(v[1]), a(v[2]), a(e_sn), a(m_ej))


def min_image_r2(n, dx, pos, sub=None):
    """r^2 from `pos` to every cell centre (or sub-sample centres) with minimum-image wrapping; shape (n,n,n[,..])."""
    idx = np.arange(n)
    L = n * dx

    def axis(c, off):
        d = (idx + off) * dx - c
        return d - L * np.round(d / L)
    if sub is None:
        dxs, dys, dzs = axis(pos[0], 0.5), axis(pos[1], 0.5), axis(pos[2], 0.5)
        return dzs[:, None, None] ** 2 + dys[None, :, None] ** 2 + dxs[None, None, :] ** 2
    q = (np.arange(sub) + 0.5) / sub
    r2 = np.zeros((n, n, n, sub, sub, sub))
    for a, qz in enumerate(q):
        for b, qy in enumerate(q):
            for c, qx in enumerate(q):
                dxs, dys, dzs = axis(pos[0], qx), axis(pos[1], qy), axis(pos[2], qz)
                r2[..., a, b, c] = dzs[:, None, None] ** 2 + dys[None, :, None] ** 2 + dxs[None, None, :] ** 2
    return r2


# ---------------------------------------------------------------------------------------------
# O1 / membership
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,pos", [(12, (6.3, 6.1, 6.7)), (16, (0.2, 15.9, 7.5)), (13, (12.99, 0.01, 3.3)),
                                   (9, (4.5, 4.5, 4.5))])
def test_sink_membership_bruteforce(n, pos):
    """Stencil walk + wrapping == all-cells minimum-image test |x_ijk - x_s| <= r_K (L51-53, R2)."""
    p = inputs.default_params(n)
    cells = po.sink_stencil(p, *pos)
    got = np.zeros((n, n, n), dtype=int)
    for i, j, k in cells:
        got[k % n, j % n, i % n] += 1
    want = (min_image_r2(n, 1.0, pos) <= p["rk_sink"] ** 2).astype(int)
    assert got.max() == 1
    assert np.array_equal(got, want)


def test_sink_member_count_config1():
    """264 cells for config 1's offset (SURVEY probe; cross-checked here by brute force above as well)."""
    w = inputs.make(1)
    assert len(po.sink_stencil(w.params, 16.3, 16.1, 16.7)) == 264


def test_sink_membership_cube_symmetry():
    """A particle at a cell centre has a member set with the 48-fold symmetry of the cube."""
    p = inputs.default_params(16)
    p["rk_sink"] = 3.7
    cells = po.sink_stencil(p, 8.5, 8.5, 8.5) - np.array([8, 8, 8])
    s = {tuple(c) for c in cells}
    for perm in [(0, 1, 2), (1, 0, 2), (2, 1, 0), (0, 2, 1), (1, 2, 0), (2, 0, 1)]:
        for sx in (1, -1):
            for sy in (1, -1):
                for sz in (1, -1):
                    t = {(sx * c[perm[0]], sy * c[perm[1]], sz * c[perm[2]]) for c in s}
                    assert t == s


def test_membership_seam_shift():
    """Shifting the particle by whole cells across the periodic seam shifts the member set (L284 analogue)."""
    p = inputs.default_params(16)
    base = po.sink_stencil(p, 8.3, 8.1, 8.7)
    for shift in [(-8, 0, 0), (7, -8, 5), (0, 7, -8)]:
        moved = po.sink_stencil(p, 8.3 + shift[0], 8.1 + shift[1], 8.7 + shift[2])
        assert np.array_equal(moved, base + np.array(shift))


@pytest.mark.parametrize("nsub", [1, 2, 4])
@pytest.mark.parametrize("pos", [(6.3, 6.1, 6.7), (0.2, 11.9, 5.5)])
def test_sn_omega_bruteforce(nsub, pos):
    """omega counts == number of sub-cell centres within r_K over ALL cells, minimum image (L203, R17)."""
    n = 12
    p = inputs.default_params(n)
    p["sn_nsub"] = nsub
    counts, host = po.sn_omega_box(p, *pos)
    g = counts.shape[0] // 2
    got = np.zeros((n, n, n), dtype=int)
    for a in range(2 * g + 1):
        for b in range(2 * g + 1):
            for c in range(2 * g + 1):
                got[(host[2] - g + a) % n, (host[1] - g + b) % n, (host[0] - g + c) % n] += counts[a, b, c]
    want = (min_image_r2(n, 1.0, pos, sub=nsub) <= p["rk_sn"] ** 2).sum(axis=(3, 4, 5))
    assert np.array_equal(got, want)
    assert counts.min() >= 0 and counts.max() <= nsub ** 3


def test_sn_volume_converges_to_sphere():
    """V_snr = sum omega V -> 4 pi r_K^3 / 3 as n_sub grows (R17-R18); n_sub = 1 gives the member count."""
    want = 4.0 * math.pi * 27.0 / 3.0
    errs = []
    for nsub in (1, 4, 8, 16):
        p = inputs.default_params(12)
        p["sn_nsub"] = nsub
        counts, _ = po.sn_omega_box(p, 6.3, 6.1, 6.7)
        vol = counts.sum() / nsub ** 3
        if nsub == 1:
            assert vol == (min_image_r2(12, 1.0, (6.3, 6.1, 6.7)) <= 9.0).sum()
        errs.append(abs(vol - want) / want)
    assert errs[1] < 0.01 and errs[2] < 0.003 and errs[3] < 0.001
    assert errs[3] < errs[1] < errs[0] + 1e-12


# ---------------------------------------------------------------------------------------------
# O2 / O3 sink accretion
# ---------------------------------------------------------------------------------------------
def test_bondi_closed_form_config1():
    """Uniform gas at rest: mdot = 4 pi lambda rho (G m)^2 / c^3 (Eq. 8 with v_inf = 0, Eq. 32; L326).
    Config 1: c^2 = gamma P / rho = 5/3, so mdot dt = 6.5436..., r_BH = G m / c^2 = 6 (Eq. 7)."""
    w = inputs.make(1)
    rho0, m_s = 1.0, 10.0
    m0 = w.state.rho.sum() + w.sinks.m.sum()
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o.step(w.dt)
    c2 = 5.0 / 3.0
    closed = 4.0 * math.pi * (math.exp(1.5) / 4.0) * rho0 * (1.0 * m_s) ** 2 / c2 ** 1.5
    assert o.sink_diag["r_bh"][0] == pytest.approx(6.0, rel=1e-13)
    assert o.sink_diag["mdot"][0] == pytest.approx(closed, rel=1e-13)
    assert closed * w.dt == pytest.approx(6.543626026975605, rel=1e-13)
    # Sigma phi = 1 (Eq. 11): requested removal == mdot dt independent of the sub-cell offset
    assert -(o.A[0].sum()) == pytest.approx(closed * w.dt, rel=1e-13)
    # limiter inactive (max removal 0.145 < f rho = 0.5) => sink gains exactly the closed form
    assert o.eta.min() == 1.0
    assert w.sinks.m[0] - m_s == pytest.approx(closed * w.dt, rel=1e-13)
    # Eq. 1: total mass conserved
    assert w.state.rho.sum() + w.sinks.m.sum() == pytest.approx(m0, rel=1e-14)
    # gas at rest: the sink gains no momentum
    assert abs(w.sinks.vx[0]) + abs(w.sinks.vy[0]) + abs(w.sinks.vz[0]) == 0.0


def test_bondi_golden_lambda():
    g = read_golden(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt"))
    assert inputs.default_params(8)["bondi_lambda"] == pytest.approx(g["bondi_lambda"], abs=5e-4)


@pytest.mark.parametrize("offset", [(0.0, 0.0, 0.0), (0.5, 0.5, 0.5), (0.3, 0.1, 0.7), (0.999, 0.001, 0.5)])
def test_sink_total_request_independent_of_offset(offset):
    """Sigma phi = 1 (Eq. 11): sum a V = mdot dt for any sub-cell position."""
    p, st = uniform_workload(16)
    sk = one_sink((8 + offset[0], 8 + offset[1], 8 + offset[2]), 0.5)
    o = po.Oracle(p, st, sk, inputs.empty_sne())
    o.deposit(0.01)
    assert -(o.A[0].sum()) == pytest.approx(o.sink_diag["mdot"][0] * 0.01, rel=1e-13)


@pytest.mark.parametrize("rbh_over_dx,want", [(0.1, 0.25), (1.0, 1.0), (10.0, 2.0)])
def test_r_acc_three_branches(rbh_over_dx, want):
    """Eq. 10 (L136): r_acc = dx/4, r_BH, r_K/2 in the three ranges (r_K = 4 dx)."""
    p, st = uniform_workload(16)
    c2 = 5.0 / 3.0
    sk = one_sink((8.3, 8.1, 8.7), rbh_over_dx * c2 / p["G"])
    o = po.Oracle(p, st, sk, inputs.empty_sne())
    o.deposit(0.01)
    assert o.sink_diag["r_bh"][0] == pytest.approx(rbh_over_dx, rel=1e-14)
    assert o.sink_diag["r_acc"][0] == pytest.approx(want, rel=1e-14)


def test_gaussian_kernel_ratio():
    """Eq. 9 (L132): the ratio of two cells' removal equals exp(-(r1^2 - r2^2)/r_acc^2)."""
    p, st = uniform_workload(16)
    pos = (8.3, 8.1, 8.7)
    sk = one_sink(pos, 1.0 * (5.0 / 3.0))          # r_BH = 1 => r_acc = 1
    o = po.Oracle(p, st, sk, inputs.empty_sne())
    o.deposit(0.01)
    A = o.A[0].reshape(16, 16, 16)
    r2 = min_image_r2(16, 1.0, pos)
    c1, c2 = (8, 8, 8), (10, 7, 9)
    assert A[c1] / A[c2] == pytest.approx(math.exp(-(r2[c1] - r2[c2]) / 1.0), rel=1e-12)
    # truncated at r_K (R8): nothing outside
    assert np.all(A[r2 > 16.0] == 0.0) and np.all(A[r2 <= 16.0] < 0.0)


def test_bondi_hoyle_two_forms_and_moving_gas():
    """Eq. 8's two printed forms agree (L125-127); v_inf is the speed relative to the sink (R5)."""
    p, st = uniform_workload(16, v=(0.3, -0.2, 0.1))
    vs = (0.1, 0.1, -0.4)
    m_s = 2.0
    sk = one_sink((8.3, 8.1, 8.7), m_s, v=vs)
    o = po.Oracle(p, st, sk, inputs.empty_sne())
    o.deposit(0.01)
    vinf2 = (0.3 - 0.1) ** 2 + (-0.2 - 0.1) ** 2 + (0.1 + 0.4) ** 2
    c2 = 5.0 / 3.0
    lam = p["bondi_lambda"]
    first_form = 4 * math.pi * 1.0 * p["G"] ** 2 * m_s ** 2 * math.sqrt((lam ** 2 * c2 + vinf2) / (c2 + vinf2) ** 4)
    assert o.sink_diag["v_inf"][0] == pytest.approx(math.sqrt(vinf2), rel=1e-13)
    assert o.sink_diag["c_inf"][0] == pytest.approx(math.sqrt(c2), rel=1e-13)
    assert o.sink_diag["mdot"][0] == pytest.approx(first_form, rel=1e-13)
    # removed gas carries its own velocity (Eq. 13): momentum removed / mass removed = v_gas
    for f, v in zip((1, 2, 3), (0.3, -0.2, 0.1)):
        assert o.A[f].sum() / o.A[0].sum() == pytest.approx(v, rel=1e-13)


def test_cs_iso_overrides_eos():
    p, st = uniform_workload(16)
    p["cs_iso"] = 2.0
    o = po.Oracle(p, st, one_sink((8.3, 8.1, 8.7), 1.0), inputs.empty_sne())
    o.deposit(0.01)
    assert o.sink_diag["c_inf"][0] == pytest.approx(2.0, rel=1e-14)
    assert o.sink_diag["r_bh"][0] == pytest.approx(0.25, rel=1e-14)


# ---------------------------------------------------------------------------------------------
# O6-O8: fold (sum), limiter, return -- Fig. 1 worked example
# ---------------------------------------------------------------------------------------------
def test_fig1_worked_example(golden_dir):
    """Fig. 1 (L83): rho = 1, two sinks each request -0.5, overlap sums to -1, limiter gives -0.8."""
    g = read_golden(os.path.join(golden_dir, "fig1_worked_example.txt"))
    n = 8
    p = inputs.default_params(n)
    p["f_max_remove"] = -g["drho_lim_overlap"] / g["rho0"]          # the 80 % the figure implies (R11)
    p, st = p, uniform_workload(n, rho0=g["rho0"])[1]
    o = po.Oracle(p, st, inputs.empty_sinks(), inputs.empty_sne())
    N = n ** 3
    # two 2-cell-wide kernels overlapping in x = 3,4 on row (j,k) = (4,4): cells 1..4 and 3..6
    row = lambda i: (4 * n + 4) * n + i
    k1, k2 = [row(i) for i in (1, 2, 3, 4)], [row(i) for i in (3, 4, 5, 6)]
    for f in range(6):
        o.A[f][:] = 0.0
    for cells in (k1, k2):                                           # Steps 1-2: buffer sum (Eqs. 2-3)
        for c in cells:
            frac = g["drho_each"] / g["rho0"]
            for f, fld in enumerate(st.fields()):
                o.A[f][c] += frac * fld.reshape(-1)[c]
    assert o.A[0][row(3)] == g["drho_sum_overlap"] and o.A[0][row(1)] == g["drho_each"]
    o.apply(sn_touched=np.zeros(N, dtype=np.int32))                  # Steps 3 + 5
    rho = st.rho.reshape(-1)
    for c in (row(3), row(4)):
        assert o.eta[c] == pytest.approx(g["eta_overlap"], rel=1e-15)
        assert rho[c] == pytest.approx(g["rho_after_overlap"], rel=1e-14)
    for c in (row(1), row(2), row(5), row(6)):
        assert o.eta[c] == 1.0
        assert rho[c] == pytest.approx(g["rho_after_single"], rel=1e-15)
    assert o.eta[row(0)] == 1.0 and rho[row(0)] == g["rho0"]
    # Step 4 (Eq. 5): each sink gains eta * 0.5 * V per cell
    a = np.full(4, -g["drho_each"])
    gain1 = po.return_from_list(o.eta, np.array(k1), a, 1.0)
    gain2 = po.return_from_list(o.eta, np.array(k2), a, 1.0)
    want = 2 * g["sink_gain_per_single_cell_over_V"] + 2 * g["sink_gain_per_shared_cell_over_V"]
    assert gain1 == pytest.approx(want, rel=1e-15) and gain2 == pytest.approx(want, rel=1e-15)
    # Eq. 1: gas lost == sinks gained
    assert (n ** 3 * g["rho0"] - rho.sum()) == pytest.approx(gain1 + gain2, rel=1e-13)


def test_limiter_eq16_quarter_and_floor():
    """Eq. 16 with rho_Tr = inf (L168): d rho_lim = min(d rho, rho/4); plus BASELINE's density floor."""
    n = 8
    p, st = uniform_workload(n)
    p["f_max_remove"] = 0.25
    p["rho_floor"] = 0.9
    o = po.Oracle(p, st, inputs.empty_sinks(), inputs.empty_sne())
    for f in range(6):
        o.A[f][:] = 0.0
    req = {0: 0.1, 1: 0.25, 2: 0.6, 3: 0.05, 4: 3.0}
    st.rho.reshape(-1)[3] = 0.92          # floor binds: room = 0.02 < 0.05
    st.rho.reshape(-1)[4] = 0.5           # already below the floor: nothing may be removed
    for c, a in req.items():
        for f, fld in enumerate(st.fields()):
            o.A[f][c] = -a * fld.reshape(-1)[c] / st.rho.reshape(-1)[c]
    rho_old = st.rho.reshape(-1).copy()
    eint_old = st.eint.reshape(-1).copy()
    o.apply(sn_touched=np.zeros(n ** 3, dtype=np.int32))
    rho = st.rho.reshape(-1)
    assert rho[0] == pytest.approx(0.9, rel=1e-15) and o.eta[0] == pytest.approx(1.0, rel=1e-15)   # floor just reached
    assert rho[1] == pytest.approx(0.9, rel=1e-15)                       # 0.25 requested, room 0.1 binds
    assert rho[2] == pytest.approx(0.9, rel=1e-15)
    assert rho[3] == pytest.approx(0.9, rel=1e-15)
    assert rho[4] == 0.5 and o.eta[4] == 0.0
    # same factor for every field (L161): specific internal energy unchanged
    for c in range(4):
        assert st.eint.reshape(-1)[c] / rho[c] == pytest.approx(eint_old[c] / rho_old[c], rel=1e-14)
    # now without a binding floor: the 25 % cap
    p2, st2 = uniform_workload(n)
    p2["f_max_remove"] = 0.25
    o2 = po.Oracle(p2, st2, inputs.empty_sinks(), inputs.empty_sne())
    for f in range(6):
        o2.A[f][:] = 0.0
    for c, a in {0: 0.1, 1: 0.25, 2: 0.6}.items():
        for f, fld in enumerate(st2.fields()):
            o2.A[f][c] = -a * fld.reshape(-1)[c]
    o2.apply(sn_touched=np.zeros(n ** 3, dtype=np.int32))
    assert st2.rho.reshape(-1)[:3] == pytest.approx([0.9, 0.75, 0.75], rel=1e-15)
    assert o2.eta[:3] == pytest.approx([1.0, 1.0, 0.25 / 0.6], rel=1e-15)


def test_limiter_invariants_random():
    """rho' >= (1-f) rho, rho' >= min(rho, floor), 0 <= eta <= 1 on a limiter-dominated case (config 2 start)."""
    w = inputs.config2_bondi(n=32)
    rho_old = w.state.rho.copy()
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o.step(w.dt)
    f, fl = w.params["f_max_remove"], w.params["rho_floor"]
    assert (o.eta < 1).sum() > 50                    # requested mdot dt >> gas in kernel
    assert o.eta.min() >= 0.0 and o.eta.max() <= 1.0
    assert np.all(w.state.rho >= (1 - f) * rho_old * (1 - 1e-15))
    assert np.all(w.state.rho >= np.minimum(rho_old, fl))


# ---------------------------------------------------------------------------------------------
# whole-step conservation (Eq. 1)
# ---------------------------------------------------------------------------------------------
def totals(st, sk):
    mass = math.fsum(st.rho.reshape(-1)) + math.fsum(sk.m)
    mom = [math.fsum(f.reshape(-1)) + math.fsum(sk.m * v) for f, v in
           ((st.mx, sk.vx), (st.my, sk.vy), (st.mz, sk.vz))]
    return mass, mom


def test_conservation_sinks_only_limited():
    w = inputs.scaled_mixed(32, 400, seed_index=5)
    w.sne = inputs.empty_sne()
    sk = w.sinks
    sk.vx[:] = 0.1
    sk.vy[:] = -0.2
    m0, p0 = totals(w.state, sk)
    o = po.Oracle(w.params, w.state, sk, w.sne)
    for _ in range(3):
        o.step(0.05)
    assert (o.eta < 1).sum() > 0
    m1, p1 = totals(w.state, sk)
    assert m1 == pytest.approx(m0, rel=1e-13)
    scale = math.fsum(np.abs(w.state.mx).reshape(-1)) + math.fsum(np.abs(sk.m * sk.vx))
    for a, b in zip(p0, p1):
        assert abs(a - b) <= 1e-13 * scale


def test_mass_budget_with_sne():
    """Sum d rho V = M_ej per SN (Eq. 17 first row, R18): total mass rises by exactly sum M_ej."""
    w = inputs.scaled_mixed(32, 400, seed_index=5)
    m0, _ = totals(w.state, w.sinks)
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o.step(w.dt)
    m1, _ = totals(w.state, w.sinks)
    assert m1 - m0 == pytest.approx(w.sne.m_ej.sum(), rel=1e-10)
    assert math.fsum(o.S[0]) == pytest.approx(w.sne.m_ej.sum(), rel=1e-13)


# ---------------------------------------------------------------------------------------------
# O4 / O5 supernovae
# ---------------------------------------------------------------------------------------------
def test_sn_budgets_uniform_centered():
    """Cell-centred SN in gas at rest: sum d rho V = M_ej; sum dE V = E_sn; sum dp V = 0 (isotropy, L217)."""
    p, st = uniform_workload(16, pressure=1e-3)
    p["sn_regime"] = inputs.SN_FORCE_ST
    o = po.Oracle(p, st, inputs.empty_sinks(), one_sn((8.5, 8.5, 8.5)))
    o.deposit(0.01)
    assert math.fsum(o.S[0]) == pytest.approx(1.0, rel=1e-14)
    assert math.fsum(o.S[4]) == pytest.approx(1e4, rel=1e-14)
    for f in (1, 2, 3):
        assert abs(math.fsum(o.S[f])) < 1e-11 * math.fsum(np.abs(o.S[f]))
    # sum |p_rad| V = |P| (R21): in gas at rest dp = p_rad + d rho * v_COM and v_COM = 0
    pmag = np.sqrt(o.S[1] ** 2 + o.S[2] ** 2 + o.S[3] ** 2)
    # the host cell (r = 0) gets no radial momentum, so the sum misses its omega share
    V_snr = o.sn_diag["v_snr"][0]
    assert math.fsum(pmag) == pytest.approx(o.sn_diag["p_rad"][0] * (V_snr - 1.0) / V_snr, rel=1e-13)


def test_sn_st_kinetic_fraction():
    """ST regime deposits the Sedov-Taylor kinetic fraction: |P|^2 / (2 M_snr) = eps_K E_sn = 0.28 E_sn (L225, R23)."""
    p, st = uniform_workload(16, pressure=1e-3)
    p["sn_regime"] = inputs.SN_FORCE_ST
    p["sn_nsub"] = 1
    o = po.Oracle(p, st, inputs.empty_sinks(), one_sn((8.3, 8.1, 8.7)))
    o.deposit(0.01)
    d = o.sn_diag
    assert d["v_snr"][0] == (min_image_r2(16, 1.0, (8.3, 8.1, 8.7)) <= 9.0).sum()     # n_sub = 1: member count
    assert d["m_snr"][0] == pytest.approx(d["v_snr"][0] * 1.0 + 1.0, rel=1e-14)
    assert d["p_rad"][0] ** 2 / (2 * d["m_snr"][0]) == pytest.approx(0.28 * 1e4, rel=1e-14)


def test_sn_physical_units_continuity_R23(golden_dir):
    """Paper's physical constants: ST momentum with the REMNANT mass is continuous-ish with P_snr at R_M = 1
    (2.17e5 vs 2.8e5 M_sun km/s), and P_snr^2 / (2 * 1679 M_sun) = 4.6e50 erg = 0.46 E_sn (L225) -- R23."""
    g = read_golden(os.path.join(golden_dir, "paper_constants.txt"))
    msun_g, kms = 1.98841e33, 1e5
    e_sn_code = g["e_sn_erg"] / (msun_g * kms * kms)              # E_sn in M_sun (km/s)^2
    # pure constants check of the paper's sentence
    ke = g["psnr_coeff_msun_kms"] ** 2 / (2 * g["msf_coeff_msun"]) * msun_g * kms * kms
    assert ke == pytest.approx(g["mc_kinetic_erg"], rel=0.02)
    assert ke / g["e_sn_erg"] == pytest.approx(g["mc_kinetic_fraction"], abs=0.01)
    # oracle in the paper's units: choose rho so that M_snr = M_sf(n_H) i.e. R_M ~ 1
    n = 16
    p, st = uniform_workload(n, pressure=1e-3)
    p.update(sn_msf_coeff=g["msf_coeff_msun"], sn_msf_exp=g["msf_exp"], sn_psnr_coeff=g["psnr_coeff_msun_kms"],
             sn_psnr_exp=g["psnr_exp"], sn_eps_k=g["eps_K"], sn_rm_ej=g["rm_ej"], sn_rm_mc=g["rm_mc"],
             sn_mu_h=1.0, sn_nh_unit=1.0)
    out = {}
    for rho0, tag in ((8.0, "ST"), (9.0, "MC")):
        st_ = inputs.State(*(f * rho0 for f in uniform_workload(n, pressure=1e-3)[1].fields()))
        o = po.Oracle(p, st_, inputs.empty_sinks(), one_sn((8.3, 8.1, 8.7), e_sn=e_sn_code, m_ej=10.0))
        o.deposit(0.01)
        out[tag] = (o.sn_diag["regime"][0], o.sn_diag["r_m"][0], o.sn_diag["p_rad"][0], o.sn_diag["n_h"][0])
    assert out["ST"][0] == 2 and out["MC"][0] == 3
    assert 0.8 < out["ST"][1] <= 1.0 < out["MC"][1] < 1.3
    # with M_ej in Eq. 19 instead of M_snr the ST value would be ~17x smaller (1.7e4): a discontinuity the
    # paper's own sentence "changes in kinetic and internal energy match ... Sedov-Taylor" (L225) excludes
    assert out["ST"][2] == pytest.approx(2.17e5 * math.sqrt(out["ST"][1] * (out["ST"][3]) ** -0.26), rel=0.01)
    assert 0.6 < out["ST"][2] / out["MC"][2] < 1.0
    assert out["MC"][2] == pytest.approx(g["psnr_coeff_msun_kms"] * out["MC"][3] ** g["psnr_exp"], rel=1e-13)


@pytest.mark.parametrize("rho0,regime", [(0.01, 1), (0.3, 2), (3.0, 3)])
def test_sn_regimes_auto(rho0, regime):
    """Eq. 19 thresholds with R27's stand-in constants: rho = 0.01, 0.3, 3 land in EJ, ST, MC."""
    p, st = uniform_workload(16, rho0=rho0, pressure=1e-3)
    o = po.Oracle(p, st, inputs.empty_sinks(), one_sn((8.3, 8.1, 8.7)))
    o.deposit(0.01)
    assert o.sn_diag["regime"][0] == regime
    if regime == 1:
        assert o.sn_diag["p_rad"][0] == 0.0
        assert o.sn_diag["r_m"][0] <= 0.027


def test_sn_momentum_energy_identities_offcentre_moving():
    """R21 identities: sum dp V = M_ej v_s + (|P|/V_snr) sum omega rhat V and
    sum dE V = E_sn + E_kin + v_COM . (that residual), for an off-centre moving SN in moving lognormal gas."""
    w = inputs.scaled_mixed(24, 20, seed_index=5)
    w.sne = one_sn((11.3, 12.1, 10.7), v=(0.3, -0.1, 0.2))
    w.sinks = inputs.empty_sinks()
    n, pos = 24, (11.3, 12.1, 10.7)
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o.deposit(0.01)
    d = {k: v[0] for k, v in o.sn_diag.items()}
    counts, host = po.sn_omega_box(w.params, *pos)
    g = counts.shape[0] // 2
    resid = np.zeros(3)
    for a in range(2 * g + 1):
        for b in range(2 * g + 1):
            for c in range(2 * g + 1):
                if counts[a, b, c] == 0:
                    continue
                dvec = np.array([host[0] - g + c + 0.5 - pos[0], host[1] - g + b + 0.5 - pos[1],
                                 host[2] - g + a + 0.5 - pos[2]])
                resid += counts[a, b, c] / 64.0 * dvec / np.linalg.norm(dvec)
    resid *= d["p_rad"] / d["v_snr"]
    vs = np.array([0.3, -0.1, 0.2])
    vcom = np.array([d["vcx"], d["vcy"], d["vcz"]])
    for f in range(3):
        assert math.fsum(o.S[1 + f]) == pytest.approx(1.0 * vs[f] + resid[f], rel=1e-9, abs=1e-9)
    e_kin = 0.5 * 1.0 * vs.dot(vs)
    assert math.fsum(o.S[4]) == pytest.approx(1e4 + e_kin + vcom.dot(resid), rel=1e-12)
    # Eq. 18: v_COM is the mass-weighted mean of gas-in-stencil and ejecta, so smoothing conserves momentum:
    # sum omega rho (v_COM - v) V + M_ej v_COM = M_ej v_s  (checked through the identity above)


def test_sn_galilean_invariance():
    """L217: boosting gas and particle by a constant velocity changes dp, dE only by the boost terms."""
    base = inputs.scaled_mixed(24, 20, seed_index=5)
    pos = (11.3, 12.1, 10.7)
    u = np.array([0.7, -0.4, 0.25])
    res = []
    for boost in (np.zeros(3), u):
        st = base.state.copy()
        vx, vy, vz = st.mx / st.rho + boost[0], st.my / st.rho + boost[1], st.mz / st.rho + boost[2]
        st = inputs.State(st.rho, st.rho * vx, st.rho * vy, st.rho * vz,
                          st.eint + 0.5 * st.rho * (vx * vx + vy * vy + vz * vz), st.eint)
        o = po.Oracle(base.params, st, inputs.empty_sinks(), one_sn(pos, v=tuple(np.array([0.3, -0.1, 0.2]) + boost)))
        o.deposit(0.01)
        res.append([s.copy() for s in o.S] + [o.sn_diag["p_rad"][0]])
    S0, S1 = res
    assert S1[5] == pytest.approx(S0[5], rel=1e-13)
    assert np.allclose(S1[0], S0[0], rtol=1e-13, atol=0)
    scale = np.abs(S0[1]).max()
    for f in range(3):                               # dp' = dp + d rho * u
        assert np.allclose(S1[1 + f], S0[1 + f] + S0[0] * u[f], rtol=0, atol=1e-12 * scale)
    # energy: Eq. 17's last row is frame-covariant in the stencil SUM ("ensuring global energy conservation", L217):
    # sum dE' V = sum dE V + u . sum dp V + 1/2 M_ej u^2
    dsum = math.fsum(S1[4]) - math.fsum(S0[4])
    want = sum(u[f] * math.fsum(S0[1 + f]) for f in range(3)) + 0.5 * 1.0 * u.dot(u)
    assert dsum == pytest.approx(want, rel=1e-9)


def test_sn_limiter_single_cell_closed_form():
    """Eq. 21 (L238): rho = 1, p = 0, S_rho = 0, S_p = (4,0,0), S_E = 2 => lambda = 0.5, e_int unchanged, KE = 2."""
    n = 8
    p, st = uniform_workload(n, pressure=2.0 / 3.0)        # e_int = 1
    o = po.Oracle(p, st, inputs.empty_sinks(), inputs.empty_sne())
    for f in range(6):
        o.A[f][:] = 0.0
    for f in range(5):
        o.S[f][:] = 0.0
    o.S[1][5], o.S[4][5] = 4.0, 2.0
    # opposite-momentum midpoint: S_p = 0 => lambda = 1, all energy thermal (L241)
    o.S[4][9] = 2.0
    touched = np.zeros(n ** 3, dtype=np.int32)
    touched[[5, 9]] = 1
    o.apply(sn_touched=touched)
    assert o.lam[5] == pytest.approx(0.5, rel=1e-15)
    assert st.mx.reshape(-1)[5] == pytest.approx(2.0, rel=1e-15)
    assert st.etot.reshape(-1)[5] == pytest.approx(3.0, rel=1e-15)
    assert st.eint.reshape(-1)[5] == pytest.approx(1.0, rel=1e-14)
    assert o.lam[9] == 1.0 and st.eint.reshape(-1)[9] == pytest.approx(3.0, rel=1e-15)
    assert o.lam[0] == 1.0 and st.eint.reshape(-1)[0] == pytest.approx(1.0, rel=1e-15)


def test_sn_limiter_invariant_config4_shape():
    """Where Eq. 21 has a root, e_int,2 >= e_min = rho_2 e_int,1/rho_1 (theta = 1); lambda in [0,1]; e_int >= 0."""
    w = inputs.config4_clustered(n=48, n_sn=300, n_sink=10)
    st0 = w.state.copy()
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o.step(w.dt)
    t = o.sn_count.reshape(w.state.rho.shape) > 0
    lam = o.lam.reshape(w.state.rho.shape)
    assert (lam[t] < 1).sum() > 10 and lam.min() >= 0 and lam.max() <= 1
    assert np.all(lam[~t] == 1.0)
    eta = o.eta.reshape(w.state.rho.shape)
    rho1 = st0.rho + eta * o.A[0].reshape(t.shape)
    eint1 = st0.eint + eta * o.A[5].reshape(t.shape)
    emin = w.state.rho * eint1 / rho1
    ok = lam > 0
    assert np.all(w.state.eint[t & ok] >= emin[t & ok] * (1 - 1e-9))
    assert np.all(w.state.eint >= 0)


# ---------------------------------------------------------------------------------------------
# whole step: order independence, translation, sampled evaluation
# ---------------------------------------------------------------------------------------------
def test_order_independence():
    """L243: the result does not depend on the order in which particles are processed (to rounding, R36)."""
    w = inputs.scaled_mixed(32, 300, seed_index=5)
    res = []
    for perm_seed in (None, 7):
        st, sk, sn = w.state.copy(), w.sinks.copy(), w.sne.copy()
        if perm_seed is not None:
            rng = np.random.default_rng(perm_seed)
            pk, pn = rng.permutation(sk.n), rng.permutation(sn.n)
            sk = inputs.Sinks(*(getattr(sk, f)[pk].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "m")))
            sn = inputs.SNe(*(getattr(sn, f)[pn].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")))
        o = po.Oracle(w.params, st, sk, sn)
        o.step(w.dt)
        inv = np.argsort(pk) if perm_seed is not None else np.arange(sk.n)
        res.append((st, sk.m[inv].copy(), [a.copy() for a in o.Sabs], [s.copy() for s in o.S]))
    (st0, m0, Sabs, S0), (st1, m1, _, S1) = res
    for f in range(5):
        assert np.all(np.abs(S0[f] - S1[f]) <= 1e-12 * np.abs(S0[f]) + 1e-14 * Sabs[f])
    assert np.allclose(st0.rho, st1.rho, rtol=1e-12, atol=0)
    assert np.allclose(m0, m1, rtol=1e-13, atol=0)


def test_translation_equivariance_across_seam():
    """Shifting everything by whole cells (periodic roll) commutes with the step (seam / wrap test)."""
    w = inputs.scaled_mixed(24, 120, seed_index=5)
    shift = (5, -7, 11)
    st, sk, sn = w.state.copy(), w.sinks.copy(), w.sne.copy()
    o = po.Oracle(w.params, st, sk, sn)
    o.step(w.dt)
    st2 = inputs.State(*(np.ascontiguousarray(np.roll(f, (shift[2], shift[1], shift[0]), axis=(0, 1, 2)))
                         for f in w.state.fields()))
    sk2, sn2 = w.sinks.copy(), w.sne.copy()
    for prt in (sk2, sn2):
        prt.x[:] = np.mod(prt.x + shift[0], 24.0)
        prt.y[:] = np.mod(prt.y + shift[1], 24.0)
        prt.z[:] = np.mod(prt.z + shift[2], 24.0)
    o2 = po.Oracle(w.params, st2, sk2, sn2)
    o2.step(w.dt)
    # positions x + shift are not exactly representable shifts, so compare to tolerance only
    for a, b in zip(st.fields(), st2.fields()):
        b_back = np.roll(b, (-shift[2], -shift[1], -shift[0]), axis=(0, 1, 2))
        assert np.allclose(a, b_back, rtol=1e-9, atol=1e-9 * np.abs(a).max())
    assert np.allclose(sk.m, sk2.m, rtol=1e-10)


def test_sample_cells_matches_full_step():
    w = inputs.scaled_mixed(32, 300, seed_index=5)
    st0 = w.state.copy()
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o_s = po.Oracle(w.params, st0, w.sinks.copy(), w.sne.copy())
    rng = np.random.default_rng(3)
    cells = np.concatenate([rng.integers(0, 32 ** 3, 200), np.array([0, 31, 32 ** 3 - 1])]).astype(np.int64)
    smp = o_s.sample_cells(cells, w.dt)
    o.step(w.dt)
    for f in range(6):
        assert np.array_equal(smp["A"][:, f], o.A[f][cells])
        assert np.array_equal(smp["unew"][:, f], w.state.fields()[f].reshape(-1)[cells])
    for f in range(5):
        assert np.array_equal(smp["S"][:, f], o.S[f][cells])
    assert np.array_equal(smp["eta"], o.eta[cells]) and np.array_equal(smp["lam"], o.lam[cells])
    assert np.array_equal(smp["sn_count"], o.sn_count[cells])
    assert (smp["sn_count"] > 0).sum() > 20


def test_return_matches_list_form():
    """orc_return == Eq. 5 evaluated from explicit (cell, a) lists (ties the step to the Fig. 1 pin's routine)."""
    w = inputs.scaled_mixed(32, 300, seed_index=5)
    st0 = w.state.copy()
    sk0 = w.sinks.copy()
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o.step(w.dt)
    o0 = po.Oracle(w.params, st0, sk0, w.sne.copy())
    for s in (0, 5, sk0.n - 1):
        cells, a = o0.sink_amounts(s, w.dt)
        dm = po.return_from_list(o.eta, cells, a, 1.0)
        assert dm == pytest.approx(o.sink_diag["dm"][s], rel=1e-14)
        assert w.sinks.m[s] == pytest.approx(sk0.m[s] + dm, rel=1e-15)


@pytest.mark.parametrize("off", [(0.125, 0.125, 0.125), (0.625, 0.375, 0.875)])
def test_sn_omega_subsamples_exactly_on_the_radius(off):
    """A supernova an odd multiple of dx/8 off a cell corner sees every sub-cell centre (n_sub = 4) at a multiple of
    dx/4: with r_K = 3 dx the test of L203 is m1^2 + m2^2 + m3^2 <= 144 on the integer lattice, every operand exact
    in binary, and the sub-samples ON the radius (30 of them) count as inside.  The sum of the omega counts is the
    number of lattice points in the closed ball of radius 12, counted here by plain integer enumeration."""
    n = 12
    p = inputs.default_params(n)
    assert p["dx"] == 1.0 and p["rk_sn"] == 3.0 and p["sn_nsub"] == 4
    pos = (5.0 + off[0], 6.0 + off[1], 4.0 + off[2])
    counts, _ = po.sn_omega_box(p, *pos)
    r = range(-12, 13)
    inside = sum(1 for a in r for b in r for c in r if a * a + b * b + c * c <= 144)
    on_radius = sum(1 for a in r for b in r for c in r if a * a + b * b + c * c == 144)
    assert on_radius == 30
    assert int(counts.sum()) == inside
