"""Seeded synthetic inputs for the DD-4DVar workloads (BASELINE.json `configs`).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no model step, no functional, no decomposition.  It produces only what
the paper calls the inputs of Algorithm 1 (u0^b, R_k, B, H, v): a truth initial
state, a background, a station set and observation noise.  The truth *trajectory* (needed to
sample observations, "simulated observations are created by sampling the model
states and adding random errors") is produced by whoever calls `make_observations`, through a
`forecast(x0, levels)` callable that the caller supplies (the oracle in tests, the CUDA library
in bench.py's GPU arm).

Field order everywhere: (h, u, v); arrays are [3][nlat][nlon], longitude fastest.
Recipe:
  truth(t0): u = u0 cos(theta), v = 0, h = h0 - (a*Omega*u0 + u0^2/2) sin^2(theta)/g,
             plus `nbumps` Gaussian height bumps A*exp(-d^2/(2 w^2)), d = great-circle angle,
             A = 50 m, w = 15 deg, centres lambda~U[0,2pi), theta~U[-60,60] deg;
             config 2/4 add a zonal-wavenumber-4 perturbation 2*sin(4 lambda)*cos(theta) m/s to v.
  sigma:     "field RMS" read as: h -> RMS of the departure from the grid mean,
             u and v -> the wind RMS sqrt(mean(u^2+v^2)); sigma_b = 5 %, sigma_o = 1 % of it.
             (`literal_rms=True` gives the literal raw-field RMS reading.)
  background = truth(t0) + N(0, sigma_b^2), independent per value.
  stations:  one seeded subset of round(frac*nlon*nlat) grid points, the same at every
             observation level, all three fields observed.
  levels:    k = 0, every, 2*every, ... <= nsteps.
  seeds:     numpy SeedSequence(1000 + cfg).spawn(4) -> bumps, background noise, stations,
             observation noise (PCG64 default_rng).
"""
from __future__ import annotations

import dataclasses
import numpy as np

RADIUS = 6.371e6
OMEGA = 7.292e-5
GRAVITY = 9.806
H0 = 1.0e4
U0 = 20.0
COS_CLAMP = float(np.cos(np.deg2rad(50.0)))
DIFFUSION = 0.02


@dataclasses.dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: grid, window, decomposition and data density."""
    cfg: int
    nlon: int
    nlat: int
    dt: float
    nsteps: int
    nbumps: int
    obs_frac: float
    obs_every: int
    p_lon: int
    p_lat: int
    q_time: int
    overlap: int
    outer_iters: int
    wave4: float = 0.0
    seed_cfg: int | None = None   # config whose seeds are used (config 4 reuses config 2's)
    mu: float = 1.0
    lam: float = 1.0
    bg_later: float = 0.0         # weight of the background term (25a) in windows j > 0 (R7)
    lbfgs_m: int = 5
    n_inner: int = 5
    max_backtrack: int = 20
    armijo_c1: float = 1e-4
    name: str = ""

    def with_layout(self, p_lon, p_lat, q_time, overlap):
        return dataclasses.replace(self, p_lon=p_lon, p_lat=p_lat, q_time=q_time,
                                   overlap=overlap)


CONFIGS = {
    0: Workload(0, 36, 18, 600.0, 16, 3, 0.50, 2, 2, 2, 2, 1, 10, name="10deg 36x18 N=16 2x2x2 o1"),
    1: Workload(1, 360, 180, 300.0, 64, 10, 0.10, 4, 4, 4, 4, 2, 20, name="1deg 360x180 N=64 4x4x4 o2"),
    2: Workload(2, 720, 360, 150.0, 128, 20, 0.05, 4, 8, 8, 8, 2, 20, wave4=2.0,
                name="0.5deg 720x360 N=128 8x8x8 o2"),
    3: Workload(3, 1440, 720, 75.0, 256, 40, 0.02, 8, 16, 16, 8, 2, 30,
                name="0.25deg 1440x720 N=256 16x16x8 o2"),
}
# config 4: the decomposition sweep on config 2's problem
SWEEP_LAYOUTS = [(1, 1, 1), (2, 2, 2), (4, 4, 4), (8, 8, 8), (16, 16, 8)]
SWEEP_OVERLAPS = [1, 2]


def sweep_workloads():
    """Config 4: config 2's problem under 5 layouts x 2 overlaps (same seeds as config 2)."""
    out = []
    for (a, b, q) in SWEEP_LAYOUTS:
        for o in SWEEP_OVERLAPS:
            w = dataclasses.replace(CONFIGS[2], cfg=4, seed_cfg=2, p_lon=a, p_lat=b, q_time=q,
                                    overlap=o, name=f"0.5deg sweep {a}x{b}x{q} o{o}")
            out.append(w)
    return out


def _streams(w: Workload):
    base = w.seed_cfg if w.seed_cfg is not None else w.cfg
    return [np.random.default_rng(s) for s in np.random.SeedSequence(1000 + base).spawn(4)]


def grid_angles(nlon, nlat):
    """Longitudes lambda_i = i*dlambda and cell-centred latitudes theta_j = -pi/2+(j+1/2)*dtheta."""
    lam = np.arange(nlon) * (2.0 * np.pi / nlon)
    theta = -0.5 * np.pi + (np.arange(nlat) + 0.5) * (np.pi / nlat)
    return lam, theta


def truth_initial(w: Workload) -> np.ndarray:
    lam, theta = grid_angles(w.nlon, w.nlat)
    L, T = np.meshgrid(lam, theta)              # [nlat][nlon]
    h = H0 - (RADIUS * OMEGA * U0 + 0.5 * U0 * U0) * np.sin(T) ** 2 / GRAVITY
    u = U0 * np.cos(T)
    v = np.zeros_like(u)
    rng = _streams(w)[0]
    lam_c = rng.uniform(0.0, 2.0 * np.pi, size=w.nbumps)
    th_c = np.deg2rad(rng.uniform(-60.0, 60.0, size=w.nbumps))
    width = np.deg2rad(15.0)
    for lc, tc in zip(lam_c, th_c):
        cosd = np.sin(T) * np.sin(tc) + np.cos(T) * np.cos(tc) * np.cos(L - lc)
        d = np.arccos(np.clip(cosd, -1.0, 1.0))
        h = h + 50.0 * np.exp(-d * d / (2.0 * width * width))
    if w.wave4:
        v = v + w.wave4 * np.sin(4.0 * L) * np.cos(T)
    return np.ascontiguousarray(np.stack([h, u, v]), dtype=np.float64)


def field_rms(x0: np.ndarray, literal_rms: bool = False) -> np.ndarray:
    h, u, v = x0
    if literal_rms:
        r = np.array([np.sqrt(np.mean(h * h)), np.sqrt(np.mean(u * u)), np.sqrt(np.mean(v * v))])
        return r
    wind = np.sqrt(np.mean(u * u + v * v))
    return np.array([np.sqrt(np.mean((h - h.mean()) ** 2)), wind, wind])


def sigmas(x0: np.ndarray, literal_rms: bool = False):
    r = field_rms(x0, literal_rms)
    return 0.05 * r, 0.01 * r


def background(w: Workload, truth0: np.ndarray, sigma_b: np.ndarray) -> np.ndarray:
    rng = _streams(w)[1]
    noise = rng.standard_normal(truth0.shape)
    return np.ascontiguousarray(truth0 + sigma_b[:, None, None] * noise)


def stations(w: Workload) -> np.ndarray:
    """Sorted flat cell indices (into [nlat][nlon]) of the observed grid points."""
    rng = _streams(w)[2]
    ncell = w.nlon * w.nlat
    n = int(round(w.obs_frac * ncell))
    return np.sort(rng.choice(ncell, size=n, replace=False)).astype(np.int64)


def obs_levels(w: Workload) -> np.ndarray:
    return np.arange(0, w.nsteps + 1, w.obs_every, dtype=np.int32)


@dataclasses.dataclass
class Observations:
    levels: np.ndarray     # int32 [n_times], ascending
    offsets: np.ndarray    # int64 [n_times+1]
    index: np.ndarray      # int32 flat into [3][nlat][nlon], ascending per level
    value: np.ndarray      # float64
    sigma_o: np.ndarray    # float64 [3]


def make_observations(w: Workload, truth_at_levels: np.ndarray, sigma_o: np.ndarray) -> Observations:
    """truth_at_levels: [n_times][3][nlat][nlon] = the truth trajectory at obs_levels(w)."""
    lev = obs_levels(w)
    st = stations(w)
    ncell = w.nlon * w.nlat
    idx1 = np.concatenate([st + f * ncell for f in range(3)]).astype(np.int32)   # ascending
    fld = np.repeat(np.arange(3), st.size)
    rng = _streams(w)[3]
    vals = []
    for k in range(lev.size):
        flat = truth_at_levels[k].reshape(-1)
        noise = rng.standard_normal(idx1.size)
        vals.append(flat[idx1] + sigma_o[fld] * noise)
    offsets = np.arange(lev.size + 1, dtype=np.int64) * idx1.size
    return Observations(lev, offsets, np.tile(idx1, lev.size), np.concatenate(vals),
                        np.asarray(sigma_o, dtype=np.float64))


@dataclasses.dataclass
class Problem:
    w: Workload
    truth0: np.ndarray
    xb: np.ndarray
    sigma_b: np.ndarray
    sigma_o: np.ndarray
    obs: Observations | None = None


def make_problem(w: Workload, forecast=None, literal_rms: bool = False) -> Problem:
    """Build all inputs.  `forecast(x0, levels) -> [len(levels)][3][nlat][nlon]` runs the
    caller's model (oracle or CUDA library); without it the problem has no observations."""
    t0 = truth_initial(w)
    sb, so = sigmas(t0, literal_rms)
    xb = background(w, t0, sb)
    prob = Problem(w, t0, xb, sb, so)
    if forecast is not None:
        tl = np.asarray(forecast(t0, obs_levels(w)))
        prob.obs = make_observations(w, tl, so)
    return prob


def random_fields(shape, seed, scale=1.0) -> np.ndarray:
    """Seeded N(0, scale^2) array for tests (directions for dot-product / finite-difference pins)."""
    return scale * np.random.default_rng(seed).standard_normal(shape)
