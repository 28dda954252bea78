"""PM-gravity deposit / interpolate / kick-drift-kick oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy, fp64, one statement per step of the paper's algorithm; shares no code with the CUDA path and imports
nothing from it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.

What it computes ("L" = /root/reference/PAPER.md line, "R" = DESIGN.md reading):

  The paper moves its particles with "a standard PM gravity method, which we implement using steps 1, 2, and 5 of
  the algorithm described in Sec. 2" (L107), "because there is no limiting and because interactions do not modify
  particle properties, only mesh properties" (L95); the deposition is "depositing particle mass into the gas density
  field for the purposes of computing the gravitational potential" (L51), "simply additive" (L27).  The Poisson solve
  between the deposit and the interpolation is the multigrid gravity solver of the host code (L427) and is NOT part
  of this path: the acceleration mesh is an input.

  gravity_deposit     Step 1 (Eq. 2): every particle adds m_s W(x_ijk - x_s) / V_ijk into a zeroed ghost-zoned
                      buffer; Step 2 (Eq. 3): ghost contents are added to the periodically wrapped owned cell;
                      Step 5 (Eq. 6 with eta = 1, L89-95): rho_tot = rho_gas + buffer.
  gravity_interpolate "conversely interpolation of mesh data back to particles" (L27): a_s = sum_ijk W(x_ijk - x_s) g_ijk
                      with the SAME weights W as the deposit.
  kick, drift, kdk_step  "kick-drift-kick" leapfrog (L107, L189; Springel 2005): v += a dt/2; x += v dt; v += a' dt/2.

  W is the cloud-in-cell (trilinear) kernel, the "standard" PM choice (reading R40: the paper names no kernel; its
  kernel radius is r_K = dx in the sense of L51-53, so one ghost layer contains it).  Per axis, for a cell-centred mesh:
      s = (x - x0) / dx - 1/2,  i0 = floor(s),  f = s - i0,  W(i0) = 1 - f,  W(i0 + 1) = f,  0 elsewhere,
  and W_ijk = (W_z(k) W_y(j)) W_x(i).  i0 ranges over [-1, n-1]: a particle in the first or last half cell reaches the
  ghost layer.

Pins (tests/test_oracle_gravity.py): particle on a cell centre / cell corner / the box corner, a hand-worked off-centre
particle with binary-fraction offsets that differ per axis, total mass and centre of mass of the deposit, exactness of
the interpolation on linear fields, deposit and interpolation as transposes of one another, zero self-force and
pairwise momentum conservation through an FFT Poisson solve, the constant-acceleration closed form and time
reversibility of the leapfrog, second-order convergence on a harmonic oscillator, drift wrap into the box.
"""
from __future__ import annotations

import numpy as np


def cic_axis(x, x0: float, dx: float):
    """Lower cell index i0 (may be -1) and the weights of cells i0 and i0 + 1 along one axis."""
    inv_dx = 1.0 / dx
    s = (np.asarray(x, dtype=np.float64) - x0) * inv_dx - 0.5
    i0f = np.floor(s)
    f = s - i0f
    return i0f.astype(np.int64), 1.0 - f, f


def gravity_deposit_buffer(p: dict, x, y, z, m, g: int = 1) -> np.ndarray:
    """Step 1.  Ghost-zoned buffer of shape (nz + 2g, ny + 2g, nx + 2g): sum_s m_s W / V, particle by particle in
    index order, the eight cells of a particle in the order k (low, high), j (low, high), i (low, high)."""
    nx, ny, nz = int(p["nx"]), int(p["ny"]), int(p["nz"])
    dx = float(p["dx"])
    x0 = p["x0"]
    V = dx * dx * dx
    assert g >= 1
    buf = np.zeros((nz + 2 * g, ny + 2 * g, nx + 2 * g), dtype=np.float64)
    i0, wx0, wx1 = cic_axis(x, x0[0], dx)
    j0, wy0, wy1 = cic_axis(y, x0[1], dx)
    k0, wz0, wz1 = cic_axis(z, x0[2], dx)
    m = np.asarray(m, dtype=np.float64)
    for dk, wz in ((0, wz0), (1, wz1)):
        for dj, wy in ((0, wy0), (1, wy1)):
            for di, wx in ((0, wx0), (1, wx1)):
                w = (wz * wy) * wx
                np.add.at(buf, (k0 + dk + g, j0 + dj + g, i0 + di + g), m * w / V)
    return buf


def fold_ghosts(buf: np.ndarray, g: int) -> np.ndarray:
    """Step 2 on one rank with periodic boundaries: every ghost cell's contents are added to the owned cell at the
    periodically wrapped index.  Returns the owned (nz, ny, nx) array."""
    nzb, nyb, nxb = buf.shape
    nz, ny, nx = nzb - 2 * g, nyb - 2 * g, nxb - 2 * g
    out = np.zeros((nz, ny, nx), dtype=np.float64)
    kk = (np.arange(nzb) - g) % nz
    jj = (np.arange(nyb) - g) % ny
    ii = (np.arange(nxb) - g) % nx
    np.add.at(out, (kk[:, None, None], jj[None, :, None], ii[None, None, :]), buf)
    return out


def gravity_deposit(p: dict, rho_gas, x, y, z, m) -> np.ndarray:
    """Steps 1, 2, 5 (L95, L107): the density the Poisson solver sees, rho_gas + sum_s m_s W / V.  rho_gas may be None
    (particles only)."""
    owned = fold_ghosts(gravity_deposit_buffer(p, x, y, z, m, 1), 1)
    if rho_gas is None:
        return owned
    return np.asarray(rho_gas, dtype=np.float64).reshape(owned.shape) + owned


def gravity_interpolate(p: dict, field, x, y, z) -> np.ndarray:
    """a_s = sum W_ijk field_ijk over the particle's eight cells (periodic), summed in the order k, j, i (low first)."""
    nx, ny, nz = int(p["nx"]), int(p["ny"]), int(p["nz"])
    dx = float(p["dx"])
    x0 = p["x0"]
    fld = np.asarray(field, dtype=np.float64).reshape(nz, ny, nx)
    i0, wx0, wx1 = cic_axis(x, x0[0], dx)
    j0, wy0, wy1 = cic_axis(y, x0[1], dx)
    k0, wz0, wz1 = cic_axis(z, x0[2], dx)
    a = np.zeros(i0.shape, dtype=np.float64)
    for dk, wz in ((0, wz0), (1, wz1)):
        for dj, wy in ((0, wy0), (1, wy1)):
            for di, wx in ((0, wx0), (1, wx1)):
                w = (wz * wy) * wx
                a = a + w * fld[(k0 + dk) % nz, (j0 + dj) % ny, (i0 + di) % nx]
    return a


def kick(v, a, dt: float) -> np.ndarray:
    """v + a dt (one half of the "kick" pair when dt is half the step)."""
    return np.asarray(v, dtype=np.float64) + np.asarray(a, dtype=np.float64) * dt


def drift(x, v, dt: float, lo: float, n: int, dx: float) -> np.ndarray:
    """x + v dt, brought back into the periodic box [lo, lo + n dx) by whole box lengths (reading R41: a result that
    rounds onto the upper face is put on the lower face, so that the host cell of L43 always exists)."""
    L = n * dx
    hi = lo + L
    xn = np.asarray(x, dtype=np.float64) + np.asarray(v, dtype=np.float64) * dt
    xn = xn.copy()
    while np.any(xn >= hi):
        xn = np.where(xn >= hi, xn - L, xn)
    while np.any(xn < lo):
        xn = np.where(xn < lo, xn + L, xn)
    return np.where(xn >= hi, lo, xn)


def kdk_step(p: dict, pos, vel, accel_mesh_of, dt: float):
    """One kick-drift-kick step (L107).  pos, vel: tuples (x, y, z), (vx, vy, vz).  accel_mesh_of(pos) returns the three
    acceleration meshes (gx, gy, gz) for the given particle positions -- the caller's Poisson solve (out of scope here).
    Returns (pos', vel')."""
    g = accel_mesh_of(pos)
    a = [gravity_interpolate(p, g[c], *pos) for c in range(3)]
    vh = [kick(vel[c], a[c], 0.5 * dt) for c in range(3)]
    n = (int(p["nx"]), int(p["ny"]), int(p["nz"]))
    pn = tuple(drift(pos[c], vh[c], dt, p["x0"][c], n[c], float(p["dx"])) for c in range(3))
    g = accel_mesh_of(pn)
    a = [gravity_interpolate(p, g[c], *pn) for c in range(3)]
    vn = tuple(kick(vh[c], a[c], 0.5 * dt) for c in range(3))
    return pn, vn
