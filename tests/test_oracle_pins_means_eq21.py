"""More pins of the CPU oracle: what PAPER.md fixes about the kernel MEANS of the accretion recipe (L121) and about the
Eq. 21 limiter (L236-241) beyond the cases of test_oracle_pins.py.

* L121: "mass-weighted mean relative velocity and mass-weighted mean sound speed" -- pinned in a two-phase gas, where
  volume weights, or the root of the mean c_s^2, give different numbers.  The expected values are closed forms in the
  member counts of the two phases (counted by brute force over all cells with minimum-image distances).
* Eq. 21 with p_1 != 0: the cross term 2 (p_1 . S_p) lambda of the quadratic, the LARGER root, and equality
  e_int,2 = e_min wherever 0 < lambda < 1.
* R25 fall-back (no admissible root => lambda = 0, e_int clipped at 0): defined by DESIGN.md's reading only, so it stays
  "parity unpinned"; the cases below fix what the reading says and make sure the branch is exercised.
"""
import math

import numpy as np
import pytest

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs
from tests.test_oracle_pins import min_image_r2, one_sink


# ---------------------------------------------------------------------------------------------
# L121: mass-weighted means over the cells within the kernel
# ---------------------------------------------------------------------------------------------
def two_phase(n, rho, vel, cs, gamma):
    """Half-spaces k < n/2 (phase 0) and k >= n/2 (phase 1), each uniform."""
    shp = (n, n, n)
    ph = (np.arange(n) >= n // 2).astype(int)[:, None, None] * np.ones(shp, dtype=int)
    pick = lambda a, b: np.where(ph == 0, a, b).astype(np.float64)
    r = pick(rho[0], rho[1])
    vx, vy, vz = (pick(vel[0][c], vel[1][c]) for c in range(3))
    c = pick(cs[0], cs[1])
    eint = r * c * c / (gamma * (gamma - 1.0))
    st = inputs.State(r, r * vx, r * vy, r * vz, eint + 0.5 * r * (vx * vx + vy * vy + vz * vz), eint)
    return st, ph


@pytest.mark.parametrize("pos", [(8.3, 8.1, 8.7), (7.9, 8.5, 6.2), (8.5, 8.5, 10.4)])
def test_kernel_means_are_mass_weighted_two_phase_gas(pos):
    n = 16
    p = inputs.default_params(n)
    rho, cs = (1.0, 4.0), (1.0, 2.0)
    vel = ((0.3, 0.0, -0.1), (-0.1, 0.2, 0.05))
    vs = (0.05, -0.02, 0.1)
    m_s = 3.0
    st, ph = two_phase(n, rho, vel, cs, p["gamma"])
    o = po.Oracle(p, st, one_sink(pos, m_s, v=vs), inputs.empty_sne())
    o.deposit(0.01)
    member = min_image_r2(n, 1.0, pos) <= p["rk_sink"] ** 2
    n0, n1 = int((member & (ph == 0)).sum()), int((member & (ph == 1)).sum())
    assert n0 > 20 and n1 > 20 and n0 != n1                     # both phases inside the kernel, unequal shares
    M = n0 * rho[0] + n1 * rho[1]
    # L121: mass-weighted mean of the RELATIVE velocity (vector), then its magnitude (R5)
    vrel = [(n0 * rho[0] * (vel[0][c] - vs[c]) + n1 * rho[1] * (vel[1][c] - vs[c])) / M for c in range(3)]
    v_inf = math.sqrt(sum(x * x for x in vrel))
    c_inf = (n0 * rho[0] * cs[0] + n1 * rho[1] * cs[1]) / M          # mass-weighted mean of c_s (R6)
    rho_inf = (n0 * rho[0] + n1 * rho[1]) / (n0 + n1)                # R4 (a reading): plain mean over the member cells
    assert o.sink_diag["n_member"][0] == n0 + n1
    assert o.sink_diag["v_inf"][0] == pytest.approx(v_inf, rel=1e-13)
    assert o.sink_diag["c_inf"][0] == pytest.approx(c_inf, rel=1e-13)
    assert o.sink_diag["rho_inf"][0] == pytest.approx(rho_inf, rel=1e-13)
    # the wrong weights give clearly different numbers here (what this test is for)
    v_vol = math.sqrt(sum(((n0 * (vel[0][c] - vs[c]) + n1 * (vel[1][c] - vs[c])) / (n0 + n1)) ** 2 for c in range(3)))
    c_vol = (n0 * cs[0] + n1 * cs[1]) / (n0 + n1)
    c_rms = math.sqrt((n0 * rho[0] * cs[0] ** 2 + n1 * rho[1] * cs[1] ** 2) / M)
    assert abs(v_vol - v_inf) > 1e-3 * v_inf and abs(c_vol - c_inf) > 1e-2 * c_inf and abs(c_rms - c_inf) > 1e-3 * c_inf
    # Eq. 7 and Eq. 8 from those means (L119, L127)
    r_bh = p["G"] * m_s / (v_inf ** 2 + c_inf ** 2)
    mdot = 4.0 * math.pi * rho_inf * r_bh ** 2 * math.sqrt(p["bondi_lambda"] ** 2 * c_inf ** 2 + v_inf ** 2)
    assert o.sink_diag["r_bh"][0] == pytest.approx(r_bh, rel=1e-13)
    assert o.sink_diag["mdot"][0] == pytest.approx(mdot, rel=1e-13)
    # Eq. 13: every cell loses gas with ITS OWN velocity and specific energies (R9)
    A = [a.reshape(n, n, n) for a in o.A]
    for phase in (0, 1):
        sel = member & (ph == phase)
        for f in range(3):
            assert A[1 + f][sel].sum() == pytest.approx(vel[phase][f] * A[0][sel].sum(), rel=1e-12, abs=1e-18)
        assert A[5][sel].sum() / A[0][sel].sum() == pytest.approx(cs[phase] ** 2 / (p["gamma"] * (p["gamma"] - 1.0)), rel=1e-12)


# ---------------------------------------------------------------------------------------------
# Eq. 21: the quadratic with p_1 != 0
# ---------------------------------------------------------------------------------------------
def apply_cells(cells):
    """Run the oracle's apply pass on hand-made cells.  cells: list of dicts with rho, p (3), E, eint, S = (S_rho, S_p (3), S_E).
    Returns (lambda, new state rows) per cell."""
    n = 8
    p = inputs.default_params(n)
    shp = (n, n, n)
    st = inputs.State(*(np.ones(shp) for _ in range(6)))
    o = po.Oracle(p, st, inputs.empty_sinks(), inputs.empty_sne())
    for f in range(6):
        o.A[f][:] = 0.0
    for f in range(5):
        o.S[f][:] = 0.0
    touched = np.zeros(n ** 3, dtype=np.int32)
    flat = [f.reshape(-1) for f in st.fields()]
    for q, c in enumerate(cells):
        flat[0][q] = c["rho"]
        flat[1][q], flat[2][q], flat[3][q] = c["p"]
        flat[4][q], flat[5][q] = c["E"], c["eint"]
        o.S[0][q] = c["S"][0]
        o.S[1][q], o.S[2][q], o.S[3][q] = c["S"][1]
        o.S[4][q] = c["S"][2]
        touched[q] = 1
    o.apply(sn_touched=touched)
    return [(o.lam[q], [fl[q] for fl in flat]) for q in range(len(cells))]


def consistent(rho, p, eint):
    return dict(rho=rho, p=p, E=eint + 0.5 * sum(x * x for x in p) / rho, eint=eint)


def test_eq21_cross_term_and_larger_root():
    """(L238) |p_1 + lambda S_p|^2 / (2 rho_2) <= E_2 - e_min, largest root in [0, 1].
    a: p_1 = (1,0,0), S_p = (3,0,0), e_int = 1, S_E = 2.625: (1 + 3 lambda)^2 = 6.25 -> lambda = 1/2 (other root -7/6).
    b: p_1 = (-1,0,0), S_p = (3,0,0), S_E = 0: (3 lambda - 1)^2 = 1 -> roots 0 and 2/3: BOTH in [0,1], the larger one counts.
    c: p_1 = (0,2,0), S_p = (0,0,4), S_E = 2.5: 4 + 16 lambda^2 = 2 (2 + 2.5) = 9 -> lambda = sqrt(5)/4 (no cross term).
    d: mass loading, rho_2 = 2: p_1 = (1,0,0), S_p = (3,0,0), S_rho = 1, e_int = 1 -> e_min = 2; S_E = 3.0625:
       K = 4 (1.5 + 3.0625 - 2) = 10.25 = (1 + 3 lambda)^2 -> lambda = (sqrt(10.25) - 1) / 3."""
    cells = [
        dict(consistent(1.0, (1.0, 0.0, 0.0), 1.0), S=(0.0, (3.0, 0.0, 0.0), 2.625)),
        dict(consistent(1.0, (-1.0, 0.0, 0.0), 1.0), S=(0.0, (3.0, 0.0, 0.0), 0.0)),
        dict(consistent(1.0, (0.0, 2.0, 0.0), 1.0), S=(0.0, (0.0, 0.0, 4.0), 2.5)),
        dict(consistent(1.0, (1.0, 0.0, 0.0), 1.0), S=(1.0, (3.0, 0.0, 0.0), 3.0625)),
    ]
    want = [0.5, 2.0 / 3.0, math.sqrt(5.0) / 4.0, (math.sqrt(10.25) - 1.0) / 3.0]
    res = apply_cells(cells)
    for (lam, u), c, lw in zip(res, cells, want):
        assert lam == pytest.approx(lw, rel=1e-14)
        rho2 = c["rho"] + c["S"][0]
        for f in range(3):
            assert u[1 + f] == pytest.approx(c["p"][f] + lw * c["S"][1][f], rel=1e-14, abs=1e-15)
        assert u[0] == rho2 and u[4] == pytest.approx(c["E"] + c["S"][2], rel=1e-15)
        # the limited momentum leaves exactly e_min of internal energy (the inequality of Eq. 21 holds with equality)
        assert u[5] == pytest.approx(rho2 * c["eint"] / c["rho"], rel=1e-13)


def test_eq21_not_binding_keeps_all_momentum():
    """lambda = 1 when the inequality holds at lambda = 1; e_int = E - KE then exceeds e_min (L241)."""
    c = dict(consistent(1.0, (1.0, 0.0, 0.0), 1.0), S=(0.0, (3.0, 0.0, 0.0), 8.0))      # 16 <= 2 (1.5 + 8 - 1) = 17
    (lam, u), = apply_cells([c])
    assert lam == 1.0 and u[1] == 4.0
    assert u[5] == pytest.approx(9.5 - 8.0, rel=1e-15) and u[5] > 1.0


def test_eq21_equality_where_limited_config4_shape():
    """On a clustered workload every cell with 0 < lambda < 1 ends with e_int,2 = e_min = rho_2 e_int,1 / rho_1 (theta = 1),
    to the rounding of E - KE; a lambda that is too small would leave e_int,2 > e_min."""
    w = inputs.config4_clustered(n=48, n_sn=300, n_sink=10)
    st0 = w.state.copy()
    o = po.Oracle(w.params, w.state, w.sinks, w.sne)
    o.step(w.dt)
    shp = w.state.rho.shape
    lam, eta = o.lam.reshape(shp), o.eta.reshape(shp)
    lim = (lam > 0.0) & (lam < 1.0)
    assert lim.sum() > 50
    rho1 = st0.rho + eta * o.A[0].reshape(shp)
    eint1 = st0.eint + eta * o.A[5].reshape(shp)
    emin = w.state.rho * eint1 / rho1
    ke = 0.5 * (w.state.mx ** 2 + w.state.my ** 2 + w.state.mz ** 2) / w.state.rho
    err = np.abs(w.state.eint - emin)[lim]
    assert np.all(err <= 1e-9 * emin[lim] + 64 * np.finfo(float).eps * (w.state.etot + ke)[lim])


# ---------------------------------------------------------------------------------------------
# R25: the fall-back branch (a reading; exercised, not pinned)
# ---------------------------------------------------------------------------------------------
def test_eq21_fallback_branch_R25():
    """No root in [0, 1] even at lambda = 0 (the cell's own momentum already violates the inequality once the SN mass is
    added): R25 sets lambda = 0, keeps p_1, adds S_rho and S_E, and clips e_int = E_2 - KE at 0.
    a: negative larger root (p_1 . S_p > 0, |p_1|^2 > K);  b: complex roots (S_p perpendicular to p_1);
    c: E_2 < KE (inconsistent input) -> e_int clipped to 0."""
    hot = consistent(1.0, (2.0, 0.0, 0.0), 1.0)                    # E_1 = 3
    a = dict(hot, S=(2.0, (1.0, 0.0, 0.0), 0.2))                   # rho_2 = 3, e_min = 3, K = 6 * 0.2 = 1.2 < |p_1|^2 = 4
    b = dict(hot, S=(2.0, (0.0, 1.0, 0.0), 0.2))
    c = dict(rho=1.0, p=(4.0, 0.0, 0.0), E=7.9, eint=0.1, S=(0.0, (1.0, 0.0, 0.0), 0.0))
    res = apply_cells([a, b, c])
    for (lam, u), cell in zip(res, (a, b, c)):
        assert lam == 0.0
        assert [u[1], u[2], u[3]] == list(cell["p"])               # no SN momentum at all
        assert u[0] == cell["rho"] + cell["S"][0] and u[4] == pytest.approx(cell["E"] + cell["S"][2], rel=1e-15)
    assert res[0][1][5] == pytest.approx(3.2 - 4.0 / 6.0, rel=1e-14) and res[0][1][5] < 3.0       # below e_min: the inequality cannot be met
    assert res[1][1][5] == pytest.approx(3.2 - 4.0 / 6.0, rel=1e-14)
    assert res[2][1][5] == 0.0


def test_eq21_lambda_against_a_root_finder_that_shares_nothing_with_the_oracle():
    """Eq. 21 (L238-241) on 500 random cells: lambda must be the LARGEST value in [0, 1] at which the inequality
    |p_1 + lambda S_p|^2 / (2 rho_2) <= E_2 - e_min holds, found here by scanning the inequality itself on a fine grid from 1
    downwards and bisecting the crossing -- no quadratic formula, no discriminant, no branch logic in common with the oracle.
    The cells cover every case: not binding (lambda = 1), the inequality holding on [0, lambda], holding only on an interval
    inside (0, 1) (momentum that first has to cancel p_1: two roots in [0, 1], the larger one counts), and holding nowhere (the
    R25 fall-back, lambda = 0)."""
    rng = np.random.default_rng(21)
    cells = []
    for q in range(500):
        rho = float(rng.uniform(0.5, 2.0))
        eint = float(rng.uniform(0.2, 2.0))
        s_rho = float(rng.uniform(0.0, 1.0))
        s_p = rng.normal(0.0, 3.0, size=3)
        if q % 4 == 0:                                         # p_1 against S_p and a small energy budget: interval cases
            p1 = -rng.uniform(0.2, 0.8) * s_p + rng.normal(0.0, 0.1, size=3)
            s_e = float(rng.uniform(-0.9, 0.3) * eint)
        else:
            p1 = rng.normal(0.0, 1.5, size=3)
            s_e = float(rng.uniform(-0.5, 6.0))
        cells.append(dict(consistent(rho, tuple(float(x) for x in p1), eint), S=(s_rho, tuple(float(x) for x in s_p), s_e)))
    res = apply_cells(cells)
    kinds = {"from_zero": 0, "not_binding": 0, "fallback": 0, "interval": 0}
    grid = np.linspace(1.0, 0.0, 20001)
    for (lam, u), c in zip(res, cells):
        rho2 = c["rho"] + c["S"][0]
        e2 = c["E"] + c["S"][2]
        emin = rho2 * c["eint"] / c["rho"]                     # theta = 1 (R25)
        p1, sp = np.array(c["p"]), np.array(c["S"][1])

        def slack(x):                                          # >= 0: the inequality holds at lambda = x (x: scalar or array)
            v = p1[None, :] + np.atleast_1d(x)[:, None] * sp[None, :]
            return (e2 - emin) - np.einsum("ij,ij->i", v, v) / (2.0 * rho2)

        if slack(1.0)[0] >= 0.0:
            want = 1.0
            kinds["not_binding"] += 1
        else:
            ok = slack(grid) >= 0.0
            if not ok.any():
                want = 0.0
                kinds["fallback"] += 1
            else:
                i = int(np.argmax(ok))                          # first grid point from the top where it holds
                lo, hi = grid[i], grid[i - 1]                   # holds at lo, fails at hi
                for _ in range(80):
                    mid = 0.5 * (lo + hi)
                    if slack(mid)[0] >= 0.0:
                        lo = mid
                    else:
                        hi = mid
                want = lo
                kinds["from_zero" if slack(0.0)[0] >= 0.0 else "interval"] += 1
        # the crossing is a root of a quadratic: its position moves by ~eps |terms| / |slope|; 2e-9 covers every case drawn
        assert lam == pytest.approx(want, abs=2e-9), (lam, want, c)
        if want == 0.0 and slack(0.0)[0] < 0.0:                 # fall-back: no momentum added, e_int clipped at >= 0 (R25)
            assert u[5] >= 0.0
    assert min(kinds.values()) >= 10, kinds
