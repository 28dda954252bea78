"""Pins of oracle/pm_gravity_oracle.py (PM-gravity deposit / interpolate / KDK leapfrog).

None of these retypes the oracle's formula: they are hand-worked values, conservation laws, exactness on linear
fields, the transpose relation between deposit and interpolation, zero self-force through an independent FFT Poisson
solve, and closed forms of the leapfrog.
"""
import numpy as np
import pytest

from oracle import pm_gravity_oracle as go


def params(n, dx=1.0, x0=(0.0, 0.0, 0.0), ny=None, nz=None):
    return dict(nx=n, ny=ny or n, nz=nz or n, dx=dx, x0=x0)


def test_particle_on_cell_centre_fills_one_cell():
    p = params(8, dx=0.5, x0=(-1.0, 2.0, 0.25))
    # centre of cell (i, j, k) = (5, 2, 7)
    x, y, z = -1.0 + 5.5 * 0.5, 2.0 + 2.5 * 0.5, 0.25 + 7.5 * 0.5
    rho = go.gravity_deposit(p, None, [x], [y], [z], [3.0])
    expect = np.zeros((8, 8, 8))
    expect[7, 2, 5] = 3.0 / 0.125            # m / V, array order (k, j, i)
    assert np.array_equal(rho, expect)


def test_particle_on_cell_corner_splits_in_eight():
    p = params(8)
    rho = go.gravity_deposit(p, None, [3.0], [5.0], [2.0], [8.0])     # the corner shared by cells 2|3, 4|5, 1|2
    expect = np.zeros((8, 8, 8))
    expect[1:3, 4:6, 2:4] = 1.0
    assert np.array_equal(rho, expect)


def test_particle_on_box_corner_wraps_through_the_ghosts():
    p = params(6, x0=(1.0, 1.0, 1.0))
    buf = go.gravity_deposit_buffer(p, [1.0], [1.0], [1.0], [8.0], g=2)
    # Step 1 puts 1/8 into the 2x2x2 block around the corner, half of it in ghost cells (index -1 -> array index g-1 = 1)
    assert buf.sum() == 8.0 and np.all(buf[1:3, 1:3, 1:3] == 1.0)
    rho = go.fold_ghosts(buf, 2)
    expect = np.zeros((6, 6, 6))
    for k in (0, 5):
        for j in (0, 5):
            for i in (0, 5):
                expect[k, j, i] = 1.0
    assert np.array_equal(rho, expect)


def test_hand_worked_off_centre_particle():
    """Offsets from the centre of cell (4, 2, 6): (+0.25, -0.5, +0.125) dx.  Per axis the weights are
    x: cell 4 -> 0.75, cell 5 -> 0.25;  y: cell 1 -> 0.5, cell 2 -> 0.5;  z: cell 6 -> 0.875, cell 7 -> 0.125.
    All are binary fractions, so the expected densities are exact, and they differ per axis (a transposed axis fails)."""
    p = params(8, dx=2.0)
    x, y, z = (4.5 + 0.25) * 2.0, (2.5 - 0.5) * 2.0, (6.5 + 0.125) * 2.0
    m, V = 16.0, 8.0
    rho = go.gravity_deposit(p, None, [x], [y], [z], [m])
    expect = np.zeros((8, 8, 8))
    for k, wz in ((6, 0.875), (7, 0.125)):
        for j, wy in ((1, 0.5), (2, 0.5)):
            for i, wx in ((4, 0.75), (5, 0.25)):
                expect[k, j, i] = m * wx * wy * wz / V
    assert np.array_equal(rho, expect)
    assert rho[6, 1, 4] == 16.0 * 0.75 * 0.5 * 0.875 / 8.0


def test_gas_density_is_added_not_replaced():
    p = params(4)
    gas = np.arange(64, dtype=np.float64).reshape(4, 4, 4)
    rho = go.gravity_deposit(p, gas, [0.5], [0.5], [0.5], [2.0])
    expect = gas.copy()
    expect[0, 0, 0] += 2.0
    assert np.array_equal(rho, expect)


def test_total_mass_and_centre_of_mass():
    rng = np.random.default_rng(11)
    n, dx, x0 = 12, 0.7, (0.3, -2.0, 5.0)
    p = params(n, dx=dx, x0=x0)
    N = 500
    pos = [x0[c] + rng.uniform(0, n * dx, N) for c in range(3)]
    m = rng.uniform(0.5, 3.0, N)
    V = dx ** 3
    rho = go.gravity_deposit(p, None, *pos, m)
    assert abs(rho.sum() * V - m.sum()) <= 1e-13 * m.sum()
    assert rho.min() >= 0.0
    # first moment on the UNFOLDED buffer (unwrapped cell centres): CIC reproduces each particle's position exactly
    g = 1
    buf = go.gravity_deposit_buffer(p, *pos, m, g=g)
    idx = np.arange(-g, n + g)
    centres = [x0[c] + (idx + 0.5) * dx for c in range(3)]
    mx = (buf * centres[0][None, None, :]).sum() * V
    my = (buf * centres[1][None, :, None]).sum() * V
    mz = (buf * centres[2][:, None, None]).sum() * V
    for got, c in ((mx, 0), (my, 1), (mz, 2)):
        want = (m * pos[c]).sum()
        assert abs(got - want) <= 1e-12 * abs(want)


def test_interpolation_is_exact_on_linear_fields_and_at_cell_centres():
    rng = np.random.default_rng(12)
    n, dx, x0 = 10, 0.5, (1.0, 2.0, 3.0)
    p = params(n, dx=dx, x0=x0)
    idx = np.arange(n)
    X = x0[0] + (idx + 0.5) * dx
    Y = x0[1] + (idx + 0.5) * dx
    Z = x0[2] + (idx + 0.5) * dx
    fld = 2.0 + 0.3 * X[None, None, :] - 1.1 * Y[None, :, None] + 0.7 * Z[:, None, None]
    # particles between the first and last cell centres (a linear field is not periodic: stay off the seam)
    N = 200
    pos = [x0[c] + rng.uniform(0.5 * dx, (n - 0.5) * dx, N) for c in range(3)]
    a = go.gravity_interpolate(p, fld, *pos)
    want = 2.0 + 0.3 * pos[0] - 1.1 * pos[1] + 0.7 * pos[2]
    assert np.max(np.abs(a - want)) <= 1e-13 * np.max(np.abs(want))
    # a particle on a cell centre reads that cell
    rnd = rng.standard_normal((n, n, n))
    a = go.gravity_interpolate(p, rnd, [X[3]], [Y[9]], [Z[0]])
    assert a[0] == rnd[0, 9, 3]
    # across the seam: a particle on the lower box face reads the mean of the first and last cell along that axis
    a = go.gravity_interpolate(p, rnd, [x0[0]], [Y[4]], [Z[7]])
    assert abs(a[0] - 0.5 * (rnd[7, 4, 0] + rnd[7, 4, n - 1])) <= 1e-15


def test_deposit_and_interpolation_are_transposes():
    """sum_s m_s (interp phi)(x_s) = sum_ijk phi_ijk (deposit m)_ijk V for any mesh phi (same kernel both ways: the
    property that removes the self-force in PM codes).  Non-cubic grid, particles everywhere including the seam."""
    rng = np.random.default_rng(13)
    p = dict(nx=9, ny=7, nz=5, dx=1.3, x0=(0.0, -1.0, 2.0))
    N = 300
    x = rng.uniform(0, 9 * 1.3, N)
    y = -1.0 + rng.uniform(0, 7 * 1.3, N)
    z = 2.0 + rng.uniform(0, 5 * 1.3, N)
    m = rng.uniform(0.1, 2.0, N)
    phi = rng.standard_normal((5, 7, 9))
    lhs = (m * go.gravity_interpolate(p, phi, x, y, z)).sum()
    rhs = (phi * go.gravity_deposit(p, None, x, y, z, m)).sum() * 1.3 ** 3
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs), 1.0)


def fft_accel(rho, dx, G=1.0):
    """Independent periodic Poisson solve (test tool, not part of the path): del^2 phi = 4 pi G rho with the spectral
    Green's function, g = -grad phi by spectral differentiation.  Any translation-invariant, odd force law will do."""
    nz, ny, nx = rho.shape
    kx = 2 * np.pi * np.fft.fftfreq(nx, dx)
    ky = 2 * np.pi * np.fft.fftfreq(ny, dx)
    kz = 2 * np.pi * np.fft.fftfreq(nz, dx)
    KX, KY, KZ = kx[None, None, :], ky[None, :, None], kz[:, None, None]
    k2 = KX ** 2 + KY ** 2 + KZ ** 2
    k2[0, 0, 0] = 1.0
    rk = np.fft.fftn(rho)
    phik = -4 * np.pi * G * rk / k2
    phik[0, 0, 0] = 0.0
    # zero the Nyquist planes of the derivative (odd symmetry of the force)
    def d(K, axis_len, axis):
        Kc = K.copy()
        if axis_len % 2 == 0:
            sl = [slice(None)] * 3
            sl[axis] = axis_len // 2
            Kc = np.broadcast_to(Kc, phik.shape).copy()
            Kc[tuple(sl)] = 0.0
        return np.real(np.fft.ifftn(-1j * Kc * phik))
    return d(KX, nx, 2), d(KY, ny, 1), d(KZ, nz, 0)


def test_no_self_force_and_pairwise_momentum_conservation():
    n = 16
    p = params(n)
    # one particle at a generic position: the force it feels from its own deposited mass vanishes
    x, y, z, m = [5.37], [9.81], [2.26], [4.0]
    g = fft_accel(go.gravity_deposit(p, None, x, y, z, m), 1.0)
    gmax = max(np.abs(c).max() for c in g)
    for c in range(3):
        a = go.gravity_interpolate(p, g[c], x, y, z)
        assert abs(a[0]) <= 1e-12 * gmax
    # two particles: m1 a1 + m2 a2 = 0
    x, y, z, m = [5.37, 8.9], [9.81, 7.2], [2.26, 15.8], [4.0, 1.5]
    g = fft_accel(go.gravity_deposit(p, None, x, y, z, m), 1.0)
    for c in range(3):
        a = go.gravity_interpolate(p, g[c], x, y, z)
        assert abs(m[0] * a[0] + m[1] * a[1]) <= 1e-12 * gmax * 4.0
        assert abs(a[0]) > 1e-4                    # they do attract one another
    # and the attraction points from 1 to 2 along x
    ax = go.gravity_interpolate(p, g[0], x, y, z)
    assert ax[0] > 0 > ax[1]


def test_kdk_constant_acceleration_closed_form_and_reversibility():
    n = 32
    p = params(n)
    acc = (0.3, -0.2, 0.05)
    mesh = tuple(np.full((n, n, n), a) for a in acc)
    pos = (np.array([10.0]), np.array([20.0]), np.array([5.0]))
    vel = (np.array([0.5]), np.array([0.1]), np.array([-0.3]))
    dt, steps = 0.25, 8
    q, v = pos, vel
    for _ in range(steps):
        q, v = go.kdk_step(p, q, v, lambda _pos: mesh, dt)
    t = dt * steps
    for c in range(3):
        assert abs(q[c][0] - (pos[c][0] + vel[c][0] * t + 0.5 * acc[c] * t * t)) <= 1e-13 * 32
        assert abs(v[c][0] - (vel[c][0] + acc[c] * t)) <= 1e-14
    # time reversal: the same steps with -dt return to the start
    for _ in range(steps):
        q, v = go.kdk_step(p, q, v, lambda _pos: mesh, -dt)
    for c in range(3):
        assert abs(q[c][0] - pos[c][0]) <= 1e-13 * 32 and abs(v[c][0] - vel[c][0]) <= 1e-14


def test_kdk_second_order_on_a_harmonic_oscillator():
    """g = -w^2 (x - c) is linear, so CIC interpolation is exact and the only error is the leapfrog's: halving dt
    divides the position error after a fixed time by 4."""
    n = 64
    p = params(n)
    idx = np.arange(n) + 0.5
    w2, c = 0.04, 32.0
    gx = np.broadcast_to(-w2 * (idx[None, None, :] - c), (n, n, n)).copy()
    zero = np.zeros((n, n, n))
    amp, T = 10.0, 20.0

    def run(dt):
        q = (np.array([c + amp]), np.array([32.0]), np.array([32.0]))
        v = (np.array([0.0]), np.array([0.0]), np.array([0.0]))
        for _ in range(int(round(T / dt))):
            q, v = go.kdk_step(p, q, v, lambda _pos: (gx, zero, zero), dt)
        return q[0][0]

    exact = c + amp * np.cos(np.sqrt(w2) * T)
    e1, e2 = abs(run(0.5) - exact), abs(run(0.25) - exact)
    assert 3.6 < e1 / e2 < 4.4
    assert e2 < 0.02


def test_drift_wraps_into_the_box():
    lo, n, dx = -3.0, 10, 0.5          # box [-3, 2)
    x = np.array([1.9, -2.9, 0.0, 1.0])
    v = np.array([1.0, -1.0, 0.0, 11.0])
    xn = go.drift(x, v, 0.5, lo, n, dx)
    assert np.allclose(xn, [-2.6, 1.6, 0.0, 1.5], rtol=0, atol=1e-15)
    assert np.all((xn >= lo) & (xn < lo + n * dx))
    # a result that rounds onto the upper face goes to the lower face (R41)
    xn = go.drift(np.array([-3.0]), np.array([-1e-30]), 1.0, lo, n, dx)
    assert xn[0] == lo


def test_gravity_workload_is_seeded_and_inside_the_box():
    """The shared input generator (no method arithmetic): same seed -> same arrays; every particle inside [x0, x0 + n dx)."""
    from paper_2509_18261_b200 import inputs
    a = inputs.gravity_workload(24, 500, seed_index=8, shape=(24, 20, 28), dx=0.37, x0=(-3.0, 11.5, 0.125))
    b = inputs.gravity_workload(24, 500, seed_index=8, shape=(24, 20, 28), dx=0.37, x0=(-3.0, 11.5, 0.125))
    for f in ("x", "y", "z", "vx", "vy", "vz", "m", "rho_gas"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    p = a.params
    for q, lo, n in ((a.x, -3.0, 24), (a.y, 11.5, 20), (a.z, 0.125, 28)):
        assert q.min() >= lo and q.max() < lo + n * 0.37
        i0, w0, w1 = go.cic_axis(q, lo, 0.37)
        assert i0.min() >= -1 and i0.max() <= n - 1 and w0.min() >= 0 and w1.min() >= 0
    assert a.rho_gas.shape == (28, 20, 24) and a.g[0].shape == (28, 20, 24)
    assert p["rk_sink"] / p["dx"] <= 4 and p["rk_sn"] / p["dx"] <= 3
    c = inputs.gravity_workload(24, 500, seed_index=9)
    assert not np.array_equal(c.x[:10], inputs.gravity_workload(24, 500, seed_index=8).x[:10])
