"""Pins of the oracle's Appendix A rounding (reading R34) against what the paper and the
mathematics fix, none of which re-types the oracle's formula:
  * the paper's own example: a few same-sign terms with M = 28 costs about half the mantissa (L612: "roughly
    equivalent to rounding the results from double precision to single precision");
  * the PURPOSE of the rounding, by brute force: sums of the same terms in many random orders round to the same bits;
  * the error it introduces is below 2^(N_bit - 52) |x| and towards zero; single contributions are left alone;
  * on a whole step: particle order no longer changes a single bit of the buffers or of the final state.
"""
import struct

import numpy as np
import pytest

from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs


def bits(x: float) -> int:
    return struct.unpack("<Q", struct.pack("<d", x))[0]


def test_two_equal_terms_margin_28_is_29_bits():
    """k = 2 equal same-sign terms: T = |x|, log2 r + 52 = log2((k-1) eps T / |x|) + 52 = 0, so N_bit = M (+1 from rounding the
    logarithm up): 28-29 of the 52 mantissa bits, i.e. about single precision is left (L612)."""
    nb = po.repro_bits(2.0, 2.0, 2, 28)
    assert nb in (28, 29)
    assert 52 - nb in (23, 24)            # fp32 has a 23-bit mantissa
    x = 1.0 + 2.0 ** -30                  # a bit far below the kept mantissa is cleared
    assert po.repro_round(x, x, 2, 28) == 1.0
    y = 1.0 + 2.0 ** -20                  # a bit inside the kept mantissa survives
    assert po.repro_round(y, y, 2, 28) == y


def test_single_contribution_and_zero_are_untouched():
    assert po.repro_round(0.1234567890123, 0.1234567890123, 1, 28) == 0.1234567890123
    assert po.repro_round(0.0, 5.0, 7, 28) == 0.0
    assert po.repro_bits(3.0, 3.0, 0, 28) == 0


@pytest.mark.parametrize("M", [8, 28])
def test_rounding_is_truncation_within_its_interval(M):
    rng = np.random.default_rng(1)
    for _ in range(2000):
        k = int(rng.integers(2, 40))
        t = rng.standard_normal(k) * 10.0 ** rng.uniform(-3, 3)
        x, T = float(t.sum()), float(np.abs(t).sum())
        nb = po.repro_bits(x, T, k, M)
        r = po.repro_round(x, T, k, M)
        assert 0 <= nb <= 52
        assert abs(r) <= abs(x) and (r == 0.0 or np.sign(r) == np.sign(x))
        assert abs(x - r) < 2.0 ** (nb - 52) * abs(x) * (1 + 1e-15) + 0.0
        assert bits(r) & ((1 << nb) - 1) == 0
        assert po.repro_round(r, T, k, M) == r                      # idempotent


def test_reordered_sums_round_to_the_same_bits():
    """The point of Appendix A: the rounding interval is 2^M times wider than anything a re-ordering of the additions can do
    to the sum, so every order lands on the same value except with probability ~2^-M per case (here M = 28, 300 cases x 20
    orders: the chance of a single failure is ~1e-5).  Without the rounding most cases differ in the last bits."""
    rng = np.random.default_rng(2)
    differ_raw = 0
    for case in range(300):
        k = int(rng.integers(2, 60))
        t = rng.standard_normal(k) * 10.0 ** rng.uniform(-2, 2, size=k)
        T = float(np.abs(t).sum())
        raw, rounded = set(), set()
        for _ in range(20):
            s = 0.0
            for v in rng.permutation(t):
                s += float(v)
            raw.add(bits(s))
            rounded.add(bits(po.repro_round(s, T, k, 28)))
        differ_raw += len(raw) > 1
        assert len(rounded) == 1, f"case {case}: {len(rounded)} different rounded values"
    assert differ_raw > 100           # the unrounded sums really are order dependent


def test_whole_step_is_order_independent_bit_for_bit():
    """Same particles in a different order: with the rounding, buffers and the final state agree in every bit; the sink channel
    of the oracle's literal six accretion buffers is rebuilt from the rounded mass channel (R29), so it agrees too."""
    w = inputs.scaled_mixed(24, 260, seed_index=5, n_clusters=2)
    rng = np.random.default_rng(3)
    pk, pn = rng.permutation(w.sinks.n), rng.permutation(w.sne.n)
    w2 = inputs.Workload("perm", w.params, w.state.copy(),
                         inputs.Sinks(*(getattr(w.sinks, f)[pk].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "m"))),
                         inputs.SNe(*(getattr(w.sne, f)[pn].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej"))),
                         w.dt, 1)
    a = po.Oracle(w.params, w.state.copy(), w.sinks.copy(), w.sne.copy())
    b = po.Oracle(w2.params, w2.state.copy(), w2.sinks.copy(), w2.sne.copy())
    a.step(w.dt, repro_M=28)
    b.step(w.dt, repro_M=28)
    assert (a.sn_count.max() > 3) and (a.sink_count.max() >= 1)          # the case has real overlaps
    for f in range(5):
        assert np.array_equal(a.S[f], b.S[f]), f"SN buffer channel {f}"
    for f in range(6):
        assert np.array_equal(a.A[f], b.A[f]), f"accretion buffer channel {f}"
    for fa, fb in zip(a.state.fields(), b.state.fields()):
        assert np.array_equal(fa, fb)
    # and without the rounding the same comparison fails somewhere (so the test above is not vacuous)
    c = po.Oracle(w.params, w.state.copy(), w.sinks.copy(), w.sne.copy())
    d = po.Oracle(w2.params, w2.state.copy(), w2.sinks.copy(), w2.sne.copy())
    c.step(w.dt)
    d.step(w.dt)
    assert any(not np.array_equal(c.S[f], d.S[f]) for f in range(5))


def test_rounded_step_stays_within_the_rounding_error_of_the_plain_step():
    w = inputs.scaled_mixed(24, 260, seed_index=5, n_clusters=2)
    a = po.Oracle(w.params, w.state.copy(), w.sinks.copy(), w.sne.copy())
    b = po.Oracle(w.params, w.state.copy(), w.sinks.copy(), w.sne.copy())
    a.step(w.dt)
    b.step(w.dt, repro_M=28)
    assert np.allclose(a.state.rho, b.state.rho, rtol=2.0 ** -20, atol=0)
    assert np.allclose(a.state.etot, b.state.etot, rtol=2.0 ** -20, atol=0)
    assert np.allclose(a.sinks.m, b.sinks.m, rtol=2.0 ** -20, atol=0)
