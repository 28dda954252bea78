"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of
the method's arithmetic: it only draws initial gas fields and particle sets with numpy
(PCG64) and packs the run-time parameters of the particle-mesh-particle step
(mesh U_ijk, particles (x_s, u_s), kernel radius r_K, deposition
function and limiter constants) into plain dicts / arrays.

Recipe: SeedSequence(250918261 + config
index).spawn(5) -> streams [density, velocity, cluster centres, particle positions,
particle masses/velocities], always consumed in that order.  The paper's own workloads
(AGORA disk, MIST / Sukhbold tables, QUOKKA checkpoints) are not
available, so these synthetic fields stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 250918261

# regime selector values (shared vocabulary, "EJ / ST / MC")
SN_AUTO, SN_FORCE_EJ, SN_FORCE_ST, SN_FORCE_MC = 0, 1, 2, 3


def default_params(n: int) -> dict:
    """Run-time parameters; every key is a plain number (copied into C structs by the users)."""
    return dict(
        nx=n, ny=n, nz=n, dx=1.0, x0=(0.0, 0.0, 0.0),
        G=1.0, gamma=5.0 / 3.0, cs_iso=0.0,
        rk_sink=4.0, rk_sn=3.0,
        bondi_lambda=math.exp(1.5) / 4.0,
        f_max_remove=0.5, rho_floor=1e-6,          # BASELINE.json configs
        sn_nsub=4, sn_regime=SN_AUTO,
        sn_eps_k=0.28, sn_rm_ej=0.027, sn_rm_mc=1.0,
        # dimensionless stand-ins for Eqs. 19-20: R_M ~ 1 at rho ~ 1
        sn_msf_coeff=114.0, sn_msf_exp=-0.26,
        sn_psnr_coeff=1030.0, sn_psnr_exp=-0.17,
        sn_mu_h=1.0, sn_nh_unit=1.0,
        sn_eint_theta=1.0,
        truelove_J=0.0,                            # Eq. 12 Jeans number; 0 = off in all BASELINE configs (paper: 0.25, L148)
    )


@dataclass
class Sinks:
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray
    m: np.ndarray

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    def copy(self) -> "Sinks":
        return Sinks(*(np.array(getattr(self, f), dtype=np.float64, copy=True)
                       for f in ("x", "y", "z", "vx", "vy", "vz", "m")))


@dataclass
class SNe:
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray
    e_sn: np.ndarray
    m_ej: np.ndarray

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    def copy(self) -> "SNe":
        return SNe(*(np.array(getattr(self, f), dtype=np.float64, copy=True)
                     for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")))


@dataclass
class State:
    """Conserved gas state, each field a C-contiguous fp64 array of shape (nz, ny, nx), x fastest."""
    rho: np.ndarray
    mx: np.ndarray
    my: np.ndarray
    mz: np.ndarray
    etot: np.ndarray
    eint: np.ndarray

    FIELDS = ("rho", "mx", "my", "mz", "etot", "eint")

    def copy(self) -> "State":
        return State(*(np.array(getattr(self, f), dtype=np.float64, copy=True) for f in self.FIELDS))

    def fields(self):
        return [getattr(self, f) for f in self.FIELDS]


@dataclass
class Workload:
    name: str
    params: dict
    state: State
    sinks: Sinks
    sne: SNe
    dt: float
    steps: int
    notes: dict = field(default_factory=dict)


def empty_sinks() -> Sinks:
    z = np.zeros(0, dtype=np.float64)
    return Sinks(z, z.copy(), z.copy(), z.copy(), z.copy(), z.copy(), z.copy())


def empty_sne() -> SNe:
    z = np.zeros(0, dtype=np.float64)
    return SNe(z, z.copy(), z.copy(), z.copy(), z.copy(), z.copy(), z.copy(), z.copy())


def _streams(config_index: int):
    ss = np.random.SeedSequence(SEED_BASE + config_index).spawn(5)
    return [np.random.Generator(np.random.PCG64(s)) for s in ss]


def _state_from_primitives(rho, vx, vy, vz, eint_density) -> State:
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    mx = rho * vx
    my = rho * vy
    mz = rho * vz
    eint = np.ascontiguousarray(eint_density, dtype=np.float64)
    etot = eint + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return State(rho, np.ascontiguousarray(mx), np.ascontiguousarray(my), np.ascontiguousarray(mz),
                 np.ascontiguousarray(etot), eint)


def _uniform_state(n: int, rho0: float, pressure: float, gamma: float) -> State:
    shp = (n, n, n)
    rho = np.full(shp, rho0, dtype=np.float64)
    zero = np.zeros(shp, dtype=np.float64)
    eint = np.full(shp, pressure / (gamma - 1.0), dtype=np.float64)
    return _state_from_primitives(rho, zero, zero, zero, eint)


def _turbulent_state(n: int, rho: np.ndarray, g_vel, sigma_v: float, gamma: float, cs: float) -> State:
    """Random velocities N(0, sigma_v) per component; sound speed cs through e_int = rho cs^2/(gamma(gamma-1))."""
    shp = (n, n, n)
    vx = g_vel.standard_normal(shp) * sigma_v
    vy = g_vel.standard_normal(shp) * sigma_v
    vz = g_vel.standard_normal(shp) * sigma_v
    eint = rho * (cs * cs / (gamma * (gamma - 1.0)))
    return _state_from_primitives(rho, vx, vy, vz, eint)


def _clustered_positions(g_centres, g_pos, count: int, n: int, n_clusters: int, sigma: float,
                         frac_clustered: float) -> np.ndarray:
    """(count, 3) positions in [0, n): a uniform part and a part in Gaussian clusters, wrapped periodically."""
    n_cl = int(round(count * frac_clustered))
    n_un = count - n_cl
    centres = g_centres.uniform(0.0, n, size=(n_clusters, 3))
    pos_un = g_pos.uniform(0.0, n, size=(n_un, 3))
    if n_cl > 0:
        # equal cluster sizes (remainder to the first clusters)
        owner = np.arange(n_cl) % n_clusters
        pos_cl = centres[owner] + g_pos.standard_normal((n_cl, 3)) * sigma
    else:
        pos_cl = np.zeros((0, 3))
    pos = np.concatenate([pos_un, pos_cl], axis=0)
    pos = np.mod(pos, float(n))
    pos[pos >= float(n)] = 0.0           # np.mod can round up to n for tiny negatives
    return pos


def _pack_sinks(pos, vel, m) -> Sinks:
    c = np.ascontiguousarray
    return Sinks(c(pos[:, 0]), c(pos[:, 1]), c(pos[:, 2]), c(vel[:, 0]), c(vel[:, 1]), c(vel[:, 2]), c(m))


def _pack_sne(pos, vel, e_sn, m_ej) -> SNe:
    c = np.ascontiguousarray
    return SNe(c(pos[:, 0]), c(pos[:, 1]), c(pos[:, 2]), c(vel[:, 0]), c(vel[:, 1]), c(vel[:, 2]),
               c(e_sn), c(m_ej))


# ---------------------------------------------------------------------------------------------
def config1_tiny_sink() -> Workload:
    """32^3, rho=1, v=0, P=1; one sink at centre + (0.3, 0.1, 0.7) dx, m=10, r_K = 4 dx, dt = 0.01."""
    n = 32
    p = default_params(n)
    st = _uniform_state(n, 1.0, 1.0, p["gamma"])
    pos = np.array([[16.3, 16.1, 16.7]])
    sinks = _pack_sinks(pos, np.zeros((1, 3)), np.array([10.0]))
    return Workload("config1_tiny_sink_32", p, st, sinks, empty_sne(), dt=0.01, steps=1)


def config2_bondi(n: int = 128) -> Workload:
    """128^3, rho = 1 + 0.01 N(0,1), v ~ N(0, 0.05), c_s = 1; one sink at the centre, m = 100; 100 steps."""
    g_rho, g_vel, _, _, _ = _streams(2)
    p = default_params(n)
    rho = 1.0 + 0.01 * g_rho.standard_normal((n, n, n))
    st = _turbulent_state(n, rho, g_vel, 0.05, p["gamma"], 1.0)
    pos = np.array([[n / 2.0, n / 2.0, n / 2.0]])
    sinks = _pack_sinks(pos, np.zeros((1, 3)), np.array([100.0]))
    return Workload(f"config2_bondi_{n}", p, st, sinks, empty_sne(), dt=0.005, steps=100)


def config3_single_sn(n: int = 64) -> Workload:
    """64^3, rho = 1, P = 1e-3, one SN (E = 1e4, M_ej = 1, r_K = 3 dx, ST regime forced); 1 step."""
    _, _, _, g_pos, _ = _streams(3)
    p = default_params(n)
    p["sn_regime"] = SN_FORCE_ST
    st = _uniform_state(n, 1.0, 1e-3, p["gamma"])
    pos = g_pos.uniform(0.0, n, size=(1, 3))
    sne = _pack_sne(pos, np.zeros((1, 3)), np.array([1e4]), np.array([1.0]))
    return Workload(f"config3_single_sn_{n}", p, st, empty_sinks(), sne, dt=0.005, steps=1)


def _mixed(config_index: int, n: int, sigma_ln: float, n_sn: int, n_sink: int, n_clusters: int,
           sigma_cl: float, sn_frac_clustered: float, sink_frac_clustered: float, m_hi: float,
           steps: int, name: str) -> Workload:
    g_rho, g_vel, g_cen, g_pos, g_pm = _streams(config_index)
    p = default_params(n)
    gauss = g_rho.standard_normal((n, n, n))
    rho = np.exp(sigma_ln * gauss - 0.5 * sigma_ln * sigma_ln)     # lognormal, mean 1
    del gauss
    st = _turbulent_state(n, rho, g_vel, 0.05, p["gamma"], 1.0)
    sn_pos = _clustered_positions(g_cen, g_pos, n_sn, n, n_clusters, sigma_cl, sn_frac_clustered)
    sink_pos = _clustered_positions(g_cen, g_pos, n_sink, n, n_clusters, sigma_cl, sink_frac_clustered)
    sink_m = g_pm.uniform(1.0, m_hi, size=n_sink)
    sink_v = np.zeros((n_sink, 3))
    sn_v = g_pm.standard_normal((n_sn, 3)) * 0.05
    sne = _pack_sne(sn_pos, sn_v, np.full(n_sn, 1e4), np.full(n_sn, 1.0))
    sinks = _pack_sinks(sink_pos, sink_v, sink_m)
    return Workload(name, p, st, sinks, sne, dt=0.005, steps=steps)


def config4_clustered(n: int = 256, n_sn: int = 10_000, n_sink: int = 500) -> Workload:
    """256^3 lognormal (sigma_ln = 1); 1e4 SNe in 20 Gaussian clusters (sigma = 8 dx); 500 uniform sinks."""
    return _mixed(4, n, 1.0, n_sn, n_sink, 20, 8.0, 1.0, 0.0, 50.0, 10, f"config4_clustered_{n}")


def config5_large(n: int = 512, n_particles: int = 1_000_000) -> Workload:
    """512^3 lognormal (sigma_ln = 1.5); 1e6 particles, 90 % SN / 10 % sinks, half uniform, half in 200 clusters."""
    n_sink = n_particles // 10
    n_sn = n_particles - n_sink
    return _mixed(5, n, 1.5, n_sn, n_sink, 200, 6.0, 0.5, 0.5, 100.0, 10, f"config5_large_{n}")


def scaled_mixed(n: int, n_particles: int, seed_index: int = 5, n_clusters: int | None = None) -> Workload:
    """Config-5-shaped workload at a reduced size (same particle density per cell by default callers);
    used by parity tests that the oracle must finish in seconds."""
    n_sink = max(n_particles // 10, 1)
    n_sn = n_particles - n_sink
    if n_clusters is None:
        n_clusters = max(1, int(round(200 * (n / 512.0) ** 3)))
    return _mixed(seed_index, n, 1.5, n_sn, n_sink, n_clusters, 6.0, 0.5, 0.5, 100.0, 10,
                  f"config5_shape_{n}_{n_particles}")


@dataclass
class GravityWorkload:
    """Inputs of the PM-gravity calls: collisionless particles, the gas density they are deposited
    onto, and an acceleration mesh standing in for the host code's Poisson solve (out of scope, L427)."""
    name: str
    params: dict
    rho_gas: np.ndarray          # (nz, ny, nx)
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray
    m: np.ndarray
    g: tuple                     # (gx, gy, gz), each (nz, ny, nx)
    dt: float


def gravity_workload(n: int, n_particles: int, seed_index: int = 6, n_clusters: int | None = None,
                     shape: tuple | None = None, dx: float = 1.0, x0=(0.0, 0.0, 0.0)) -> GravityWorkload:
    """Config-5-shaped particle set for the gravity path: positions half uniform, half in Gaussian clusters (sigma = 6 dx),
    masses U(1, 100), velocities N(0, 0.05), lognormal gas (sigma_ln = 1.5), acceleration mesh N(0, 0.01) per component.
    shape = (nx, ny, nz) for a non-cubic box (positions are drawn in the cube of side min(shape))."""
    g_rho, g_vel, g_cen, g_pos, g_pm = _streams(seed_index)
    nx, ny, nz = shape if shape is not None else (n, n, n)
    p = default_params(n)
    p.update(nx=nx, ny=ny, nz=nz, dx=dx, x0=tuple(x0))
    if dx != 1.0:                      # kernel radii of the exchange step in cells, not length units (ghost width 4)
        p.update(rk_sink=3.5 * dx, rk_sn=2.5 * dx)
    if n_clusters is None:
        n_clusters = max(1, int(round(200 * (n / 512.0) ** 3)))
    rho = np.exp(1.5 * g_rho.standard_normal((nz, ny, nx)) - 0.5 * 1.5 * 1.5)
    acc = tuple(0.01 * g_vel.standard_normal((nz, ny, nx)) for _ in range(3))
    pos = _clustered_positions(g_cen, g_pos, n_particles, min(nx, ny, nz), n_clusters, 6.0, 0.5)
    m = g_pm.uniform(1.0, 100.0, size=n_particles)
    vel = 0.05 * g_pm.standard_normal((n_particles, 3))
    xs = [np.ascontiguousarray(x0[c] + pos[:, c] * dx) for c in range(3)]
    # x0 + pos dx can round onto the upper face; such a particle is put on the lower face
    for c, nn in enumerate((nx, ny, nz)):
        xs[c][xs[c] >= x0[c] + nn * dx] = x0[c]
    return GravityWorkload(f"gravity_{nx}x{ny}x{nz}_{n_particles}", p, rho, xs[0], xs[1], xs[2],
                           np.ascontiguousarray(vel[:, 0]), np.ascontiguousarray(vel[:, 1]), np.ascontiguousarray(vel[:, 2]),
                           m, acc, dt=0.5)


CONFIGS = {
    1: config1_tiny_sink,
    2: config2_bondi,
    3: config3_single_sn,
    4: config4_clustered,
    5: config5_large,
}


def make(config_index: int, **kw) -> Workload:
    return CONFIGS[config_index](**kw)
