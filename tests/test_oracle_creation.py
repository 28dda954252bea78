"""Pins of the oracle's sink creation (Sec. 3.1.2) on hand-built fields where the paper's words fix the
answer: which cells create (above rho_Tr, local maximum within r_K, not inside another sink's kernel), the new particle
(m = (rho - rho_Tr) V, momentum m v, L183) and what is left in the cell (rho_Tr, same v and specific energies)."""
import math

import numpy as np

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs

J = 0.4                      # with c_s = 1, G = dx = 1: rho_Tr = 0.16 pi
RHO_TR = J * J * math.pi


def _setup(n=20, bumps=(), v=(0.1, -0.2, 0.05)):
    w = inputs.config1_tiny_sink()
    p = dict(w.params)
    p.update(nx=n, ny=n, nz=n, truelove_J=J, cs_iso=1.0)
    rho = np.full((n, n, n), 0.3)                      # background below rho_Tr
    for (k, j, i, val) in bumps:
        rho[k, j, i] = val
    vx, vy, vz = (np.full((n, n, n), c) for c in v)
    st = inputs._state_from_primitives(rho, vx, vy, vz, 0.9 * rho)
    return p, st


def _oracle(p, st, sinks=None):
    return po.Oracle(p, st, sinks if sinks is not None else inputs.empty_sinks(), inputs.empty_sne())


def test_single_peak_closed_form():
    p, st = _setup(bumps=[(7, 8, 9, 2.0), (7, 8, 10, 1.0)])          # the neighbour is above rho_Tr too, but not a maximum
    old = st.copy()
    o = _oracle(p, st)
    n, s = o.create_sinks(16, use_buffer=False)
    assert n == 1 and s["cells"][0] == (7 * 20 + 8) * 20 + 9
    assert (s["x"][0], s["y"][0], s["z"][0]) == (9.5, 8.5, 7.5)       # cell centre
    assert abs(s["m"][0] - (2.0 - RHO_TR)) < 1e-15                   # V = 1
    assert abs(s["vx"][0] - 0.1) < 1e-16 and abs(s["vy"][0] + 0.2) < 1e-16 and abs(s["vz"][0] - 0.05) < 1e-16
    assert abs(st.rho[7, 8, 9] - RHO_TR) < 1e-15
    assert abs(st.mx[7, 8, 9] / st.rho[7, 8, 9] - 0.1) < 1e-15       # velocity kept (L183)
    assert abs(st.eint[7, 8, 9] / st.rho[7, 8, 9] - 0.9) < 1e-15     # specific internal energy kept
    assert abs(st.etot[7, 8, 9] / st.rho[7, 8, 9] - old.etot[7, 8, 9] / 2.0) < 1e-15
    # conservation: gas + new particle
    assert abs(st.rho.sum() + s["m"][0] - old.rho.sum()) < 1e-12
    assert abs(st.mx.sum() + s["m"][0] * s["vx"][0] - old.mx.sum()) < 1e-12
    st.rho[7, 8, 9] = old.rho[7, 8, 9]
    assert np.array_equal(st.rho, old.rho)                           # nothing else touched (the 1.0 neighbour stays)


def test_two_peaks_nearer_and_farther_than_r_k():
    # r_K = 4: offset (3, 2, 0) has r = 3.6 < 4 -> only the higher one creates; offset (4, 1, 0), r = 4.12 > 4 -> both
    p, st = _setup(bumps=[(5, 5, 5, 2.0), (5, 7, 8, 1.5)])
    n, s = _oracle(p, st).create_sinks(16, use_buffer=False)
    assert n == 1 and abs(s["m"][0] - (2.0 - RHO_TR)) < 1e-15
    p, st = _setup(bumps=[(5, 5, 5, 2.0), (5, 6, 9, 1.5)])
    n, s = _oracle(p, st).create_sinks(16, use_buffer=False)
    assert n == 2
    assert list(s["cells"]) == sorted(s["cells"])                    # ordered by cell index
    assert abs(s["m"].sum() - (3.5 - 2 * RHO_TR)) < 1e-14


def test_plateau_creates_nothing_and_seam_neighbour_counts():
    p, st = _setup(bumps=[(5, 5, 5, 2.0), (5, 5, 6, 2.0)])            # a tie is not a strict maximum (R39)
    n, _ = _oracle(p, st).create_sinks(16, use_buffer=False)
    assert n == 0
    p, st = _setup(bumps=[(0, 0, 0, 1.5), (19, 19, 18, 2.0)])         # across the periodic corner: offset (-2, -1, -1), r = 2.4
    n, s = _oracle(p, st).create_sinks(16, use_buffer=False)
    assert n == 1 and s["cells"][0] == (19 * 20 + 19) * 20 + 18


def test_no_creation_inside_an_existing_sinks_kernel():
    """L177: cells where the retained accretion buffer is non-zero are excluded; outside the kernel creation goes on."""
    p, st = _setup(bumps=[(10, 10, 12, 2.0), (3, 3, 3, 1.8)])
    p0 = dict(p, truelove_J=0.0)                                     # plain accretion step, so that the bump stays above rho_Tr
    sinks = inputs._pack_sinks(np.array([[10.5, 10.5, 10.5]]), np.zeros((1, 3)), np.array([1e-6]))
    o0 = _oracle(p0, st, sinks)
    o0.step(0.01)                                                    # deposits: A[0] != 0 within 4 dx of the sink
    assert o0.A[0].reshape(o0.shape)[10, 10, 12] != 0.0 and o0.A[0].reshape(o0.shape)[3, 3, 3] == 0.0
    assert st.rho[10, 10, 12] > 1.9                                  # still far above rho_Tr: only criterion (iii) can exclude it
    o = _oracle(p, st, sinks)
    o.A[0][:] = o0.A[0]
    n, s = o.create_sinks(16)
    assert n == 1 and s["cells"][0] == (3 * 20 + 3) * 20 + 3
    n2, _ = _oracle(p, st.copy(), sinks).create_sinks(16, use_buffer=False)
    assert n2 == 1                                                   # (3,3,3) was consumed above; without the buffer the in-kernel bump creates


def test_capacity_is_respected_and_count_reported():
    p, st = _setup(bumps=[(2, 2, 2, 2.0), (2, 2, 12, 2.1), (12, 12, 12, 2.2)])
    n, s = _oracle(p, st).create_sinks(2, use_buffer=False)
    assert n == 3 and len(s["m"]) == 2
