"""The five BASELINE.json workloads as seeded synthetic inputs.

They stand in for the paper's Hurricane Harvey / TX2008 workload (6,675,517
elements, p=1, tidal boundary on one side, moving hurricane wind,
PAPER.md:529), whose mesh and HURDAT2 track are not available here.  Every
generator takes size arguments so the same recipe can be built small (tests the
oracle finishes in seconds) or at BASELINE.json's full size (bench, full-size
parity).  numpy default_rng(seed), seed = 2508212080 + config number.

This module serves both the oracle and the CUDA path and contains no method
arithmetic: it returns node coordinates, connectivity, edge tables, nodal
bathymetry, parameters, the time step and the initial modal state (the
element-wise linear interpolant of a nodal field, see mesh.vertex_to_modal_p1).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

from .mesh import Mesh, rect_mesh, vertex_to_modal_p1

SEED0 = 2508212080
G = 9.81
M2_OMEGA = 1.405189e-4   # rad/s


@dataclass
class Workload:
    name: str
    mesh: Mesh
    bathy: np.ndarray            # [n_nodes], positive down
    params: dict                 # p, rk_order, g, cf, coriolis_f, h0_dry, limiter, wetdry
    ze: np.ndarray               # [ndof, n_elem]
    qx: np.ndarray
    qy: np.ndarray
    dt: float
    nsteps: int
    tide: tuple | None = None    # (amp, omega, phase)
    holland: dict | None = None  # x0,y0,vx,vy,rmax,dp,B,rho_air,rho_water,f
    notes: dict = field(default_factory=dict)

    @property
    def ndof(self) -> int:
        p = self.params["p"]
        return (p + 1) * (p + 2) // 2

    @property
    def n_stage(self) -> int:
        return self.params.get("rk_stages", 0) or self.params["rk_order"]

    @property
    def dofs(self) -> int:
        return 3 * self.ndof * self.mesh.n_elem


def ndof_of(p: int) -> int:
    return (p + 1) * (p + 2) // 2


def default_params(**kw) -> dict:
    d = dict(p=1, rk_order=2, g=G, cf=0.0, coriolis_f=0.0, h0_dry=1e-3, limiter=0, wetdry=0, flux=0)
    d.update(kw)
    return d


def round_down_2sig(x: float) -> float:
    e = math.floor(math.log10(x))
    m = math.floor(x / 10.0 ** (e - 1) + 1e-9)
    return m * 10.0 ** (e - 1)


def cfl_dt(mesh: Mesh, bathy: np.ndarray, p: int, g: float = G, safety: float = 0.25) -> float:
    """dt = safety * min_e(2 r_in) / ((2p+1) sqrt(g max(h_b, 1 m))), rounded down to 2
    significant digits."""
    xy, tri = mesh.xy, mesh.tri
    p0, p1, p2 = xy[tri[:, 0]], xy[tri[:, 1]], xy[tri[:, 2]]
    area = 0.5 * ((p1[:, 0] - p0[:, 0]) * (p2[:, 1] - p0[:, 1]) - (p2[:, 0] - p0[:, 0]) * (p1[:, 1] - p0[:, 1]))
    per = (np.linalg.norm(p1 - p0, axis=1) + np.linalg.norm(p2 - p1, axis=1) + np.linalg.norm(p0 - p2, axis=1))
    two_r = 4.0 * area / per
    hmax = np.maximum(bathy[tri].max(axis=1), 1.0)
    dt = safety * float(np.min(two_r / ((2 * p + 1) * np.sqrt(g * hmax))))
    return round_down_2sig(dt)


def _modal(fn_nodes: np.ndarray, mesh: Mesh, p: int) -> np.ndarray:
    return vertex_to_modal_p1(fn_nodes, mesh.tri, ndof_of(p))


def _zeros(mesh: Mesh, p: int) -> np.ndarray:
    return np.zeros((ndof_of(p), mesh.n_elem), dtype=np.float64)


def hump(xy: np.ndarray, cx: float, cy: float, amp: float, sigma: float) -> np.ndarray:
    r2 = (xy[:, 0] - cx) ** 2 + (xy[:, 1] - cy) ** 2
    return amp * np.exp(-r2 / (2.0 * sigma * sigma))


def perturbed(w: Workload, amp_z: float = 0.3, amp_q: float = 1.0, seed: int = 0, min_depth: float = 2.0) -> Workload:
    """The same workload started from a non-trivial state: a smooth wave pattern (amplitude amp_z in zeta,
    amp_q in Qx, Qy; wavelength ~ 40 cells) plus seeded white noise (10 % of the amplitude) in ALL modes of all
    three variables, added in every element whose shallowest vertex is deeper than min_depth (dry land and the
    swash zone keep the recipe's state).  Used by the parity tests so that every gather, permutation and mode is
    compared on data that is not zero; the bench keeps BASELINE.json's initial states."""
    rng = np.random.default_rng(SEED0 + 100 + seed)
    m = w.mesh
    p = w.params["p"]
    nd = ndof_of(p)
    xy = m.xy
    span = float(max(np.ptp(xy[:, 0]), np.ptp(xy[:, 1])))
    cell = span / math.sqrt(max(m.n_elem / 2.0, 1.0))
    k = 2.0 * math.pi / (40.0 * cell)
    ph = rng.uniform(0.0, 2.0 * math.pi, 6)
    nodal = [amp_z * np.sin(k * xy[:, 0] + ph[0]) * np.cos(0.7 * k * xy[:, 1] + ph[1]),
             amp_q * np.cos(0.8 * k * xy[:, 0] + ph[2]) * np.cos(k * xy[:, 1] + ph[3]),
             amp_q * np.sin(k * xy[:, 0] + ph[4]) * np.sin(0.6 * k * xy[:, 1] + ph[5])]
    deep = (w.bathy[m.tri].min(axis=1) > min_depth)[None, :]
    decay = (1.0 / (1.0 + np.arange(nd)))[:, None]            # higher modes carry less
    out = []
    for c, base in enumerate((w.ze, w.qx, w.qy)):
        amp = amp_z if c == 0 else amp_q
        d = _modal(nodal[c], m, p) + 0.1 * amp * decay * rng.uniform(-1.0, 1.0, (nd, m.n_elem))
        out.append(base + np.where(deep, d, 0.0))
    return Workload(w.name + "+perturbed", m, w.bathy, w.params, out[0], out[1], out[2], w.dt, w.nsteps,
                    tide=w.tide, holland=w.holland, notes=dict(w.notes, perturbed=(amp_z, amp_q, seed)))


def with_forcing(w: Workload, pressure: bool = False, rain: float = 0.0) -> Workload:
    """The same workload with the surface-pressure gradient of its Holland vortex switched on and / or a uniform rain
    rate (m/s) -- SURVEY.md 8(f) NEXT-4; both sides' from_workload read these notes."""
    notes = dict(w.notes)
    if pressure:
        notes["pressure"] = True
    if rain:
        notes["rain"] = float(rain)
    return Workload(w.name + ("+pressure" if pressure else "") + ("+rain" if rain else ""), w.mesh, w.bathy, w.params,
                    w.ze, w.qx, w.qy, w.dt, w.nsteps, tide=w.tide, holland=w.holland, notes=notes)


# --------------------------------------------------------------------------- C1
def c1(nq: int = 32, nsteps: int = 100, p: int = 1, rk_order: int = 2) -> Workload:
    """Square basin 10 km x 10 km, nq x nq quads (same diagonal), flat 10 m, closed walls,
    Gaussian hump 0.5 m / sigma 1 km, Q=0, no friction/wind, SSP-RK2, dt=1 s (scaled with
    the cell size when nq != 32)."""
    L = 10_000.0
    mesh = rect_mesh(nq, nq, L, L, diag="same", meta=dict(config="C1", nq=nq))
    bathy = np.full(mesh.n_nodes, 10.0)
    ze = _modal(hump(mesh.xy, L / 2, L / 2, 0.5, 1000.0), mesh, p)
    dt = 1.0 * (32.0 / nq) * (3.0 / (2 * p + 1))
    return Workload(f"C1[{nq}x{nq},p{p}]", mesh, bathy,
                    default_params(p=p, rk_order=rk_order), ze, _zeros(mesh, p), _zeros(mesh, p),
                    dt, nsteps)


# --------------------------------------------------------------------------- C2
def c2_bathy(xy: np.ndarray, L: float, rng: np.random.Generator) -> np.ndarray:
    r2 = (xy[:, 0] - L / 2) ** 2 + (xy[:, 1] - L / 2) ** 2
    h = 10.0 + 40.0 * np.exp(-r2 / 3000.0 ** 2)
    for _ in range(5):
        nx_, ny_ = rng.integers(1, 5, size=2)
        ph = rng.uniform(0.0, 2.0 * np.pi)
        h = h + 0.2 * np.sin(2.0 * np.pi * (nx_ * xy[:, 0] + ny_ * xy[:, 1]) / L + ph)
    return h


def c2(nq: int = 512, p: int = 1, state: str = "hump", nsteps: int = 200) -> Workload:
    """Same basin, nq x nq quads with a random diagonal per quad, bathymetry
    10+40 exp(-r^2/(3 km)^2) + 5 seeded sinusoid modes (sum amplitude 1 m), Cf=0.0025,
    f=1e-4, lake-at-rest (zeta=0.3) or hump initial state, SSP-RK2."""
    L = 10_000.0
    rng = np.random.default_rng(SEED0 + 2)
    mesh = rect_mesh(nq, nq, L, L, diag="random", rng=rng, meta=dict(config="C2", nq=nq))
    bathy = c2_bathy(mesh.xy, L, rng)
    if state == "rest":
        zn = np.full(mesh.n_nodes, 0.3)
    elif state == "hump":
        zn = hump(mesh.xy, L / 2, L / 2, 0.5, 1000.0)
    else:
        raise ValueError(state)
    params = default_params(p=p, rk_order=2, cf=0.0025, coriolis_f=1e-4)
    dt = cfl_dt(mesh, bathy, p)
    return Workload(f"C2[{nq}x{nq},p{p},{state}]", mesh, bathy, params,
                    _modal(zn, mesh, p), _zeros(mesh, p), _zeros(mesh, p), dt, nsteps)


# --------------------------------------------------------------------------- C3
def c3(nn: int = 1500, nsteps: int = 100, spacing: float = 200.0, wetdry: int = 1) -> Workload:
    """Unstructured-like mesh: nn x nn node grid, interior nodes jittered by U(-0.3,0.3)
    cell, random diagonal, elements and edges randomly permuted; shelf bathymetry linear
    in x from 5 m to 3000 m; M2 tidal elevation (1 m) on the east side, land elsewhere;
    rest start; p=1, SSP-RK2.  The wet/dry pass runs (every element stays wet)."""
    rng = np.random.default_rng(SEED0 + 3)
    L = spacing * (nn - 1)
    mesh = rect_mesh(nn - 1, nn - 1, L, L, diag="random", jitter=0.3, permute=True, rng=rng,
                     ocean_pred=lambda xm, ym: xm > L - 1e-6 * L, meta=dict(config="C3", nn=nn))
    bathy = 5.0 + (3000.0 - 5.0) * mesh.xy[:, 0] / L
    params = default_params(p=1, rk_order=2, wetdry=wetdry)
    dt = cfl_dt(mesh, bathy, 1)
    z = _zeros(mesh, 1)
    return Workload(f"C3[{nn}x{nn} nodes]", mesh, bathy, params, z, z.copy(), z.copy(), dt, nsteps,
                    tide=(1.0, M2_OMEGA, 0.0))


# --------------------------------------------------------------------------- C4
def holland_default(x0, y0, vx, vy, rmax=40_000.0, dp=6000.0, f=7.0e-5) -> dict:
    return dict(x0=x0, y0=y0, vx=vx, vy=vy, rmax=rmax, dp=dp, B=1.5, rho_air=1.15, rho_water=1025.0, f=f)


def c4(nqx: int = 1024, nqy: int = 512, nsteps: int = 500, spacing: float = 200.0) -> Workload:
    """Wetting/drying channel: nqx x nqy quads (same diagonal), bed elevation linear in x
    from -20 m to +5 m (h_b from 20 to -5) so about 20 % of the elements start dry,
    zeta_v = max(0, H0/2 - h_v), Q=0, all land boundaries, translating Holland vortex wind,
    slope limiter on, H0 = 1e-3 m, Cf = 0.0025 (added, the config is
    silent), p=1, SSP-RK2."""
    Lx, Ly = spacing * nqx, spacing * nqy
    mesh = rect_mesh(nqx, nqy, Lx, Ly, diag="same", meta=dict(config="C4", nqx=nqx, nqy=nqy))
    bathy = 20.0 - 25.0 * mesh.xy[:, 0] / Lx
    h0 = 1e-3
    zn = np.maximum(0.0, 0.5 * h0 - bathy)   # dry land carries a film of H0/2 (clearly below the tolerance)
    params = default_params(p=1, rk_order=2, cf=0.0025, h0_dry=h0, limiter=1, wetdry=1)
    dt = cfl_dt(mesh, bathy, 1)
    hol = holland_default(40_000.0 * Lx / 204_800.0, 0.5 * Ly, 5.0, 0.0,
                          rmax=40_000.0 * Lx / 204_800.0)
    return Workload(f"C4[{nqx}x{nqy}]", mesh, bathy, params,
                    _modal(zn, mesh, 1), _zeros(mesh, 1), _zeros(mesh, 1), dt, nsteps, holland=hol)


# --------------------------------------------------------------------------- C5
def graded_coords(n_cells: int, L: float, centre: float = 0.7, half_band: float = 0.2,
                  ramp: float = 0.1, ratio: float = 10.0) -> np.ndarray:
    """Node x-coordinates with cells `ratio` times smaller in an index band around
    `centre` (fractions of the cell index range), geometric ramps on both sides."""
    s = (np.arange(n_cells) + 0.5) / n_cells
    d = np.abs(s - centre)
    t = np.clip((d - half_band) / ramp, 0.0, 1.0)
    size = ratio ** (t - 1.0)          # 1/ratio inside the band ... 1 outside
    x = np.concatenate([[0.0], np.cumsum(size)])
    return x * (L / x[-1])


def c5(nn: int = 1323, nsteps: int = 200, p: int = 2, rk_order: int = 3, spacing: float = 500.0) -> Workload:
    """Storm-surge scale: nn x nn nodes, x-spacing graded 10x finer around a synthetic
    coastline, jitter 0.3 local cell, random diagonal, random permutation; shelf
    bathymetry crossing zero at the coastline (wet/dry active); tidal ocean side (west);
    friction, Coriolis, moving Holland wind, limiter; p=2, SSP-RK3."""
    rng = np.random.default_rng(SEED0 + 5)
    L = spacing * (nn - 1)
    xs = graded_coords(nn - 1, L)
    x_coast = float(xs[int(round(0.7 * (nn - 1)))])
    mesh = rect_mesh(nn - 1, nn - 1, L, L, diag="random", jitter=0.3, permute=True, rng=rng,
                     ocean_pred=lambda xm, ym: xm < 1e-6 * L, x_coords=xs,
                     meta=dict(config="C5", nn=nn, x_coast=x_coast))
    x = mesh.xy[:, 0]
    bathy = np.where(x < x_coast, 200.0 * (x_coast - x) / x_coast,
                     -5.0 * (x - x_coast) / (L - x_coast))
    h0 = 1e-3
    zn = np.maximum(0.0, 0.5 * h0 - bathy)   # dry land carries a film of H0/2 (clearly below the tolerance)
    params = default_params(p=p, rk_order=rk_order, cf=0.0025, coriolis_f=7.0e-5, h0_dry=h0,
                            limiter=1, wetdry=1)
    dt = cfl_dt(mesh, bathy, p)
    hol = holland_default(0.35 * L, 0.5 * L, 5.0, 0.0, rmax=min(40_000.0, 0.15 * L))
    return Workload(f"C5[{nn}x{nn} nodes,p{p}]", mesh, bathy, params,
                    _modal(zn, mesh, p), _zeros(mesh, p), _zeros(mesh, p), dt, nsteps,
                    tide=(1.0, M2_OMEGA, 0.0), holland=hol)


FULL = {
    "C1": lambda: c1(),
    "C2p1": lambda: c2(p=1),
    "C2p2": lambda: c2(p=2),
    "C3": lambda: c3(),
    "C4": lambda: c4(),
    "C5": lambda: c5(),
}
