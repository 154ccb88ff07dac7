"""Seeded synthetic two-strip J-PET event lists (inputs only; none of the reconstruction arithmetic).

This module stands in for the paper's "simulated data using realistic parameters" (PAPER.md:204,
sigma_z ~ 10 mm and sigma_dl ~ 40 mm from PAPER.md:124), which is not available here.  It is the one
module that both the CPU oracle's tests and the CUDA path's tests / bench read; it holds the detector
*forward* model only (Eq. 1: where a photon pair from (y, z, theta) hits the strips
and the path difference it produces) and no part of Eq. 2-12 / Listing 1.

Recipe (restated in DESIGN.md "Input recipe"):
  1. draw (y, z) uniformly in the phantom's bounding rectangle, accept with probability
     intensity(y, z) / max_intensity; where primitives overlap the FIRST one in the list wins
     (the paper's phantom rule);
  2. draw the in-plane LOR angle theta uniformly on (-pi/2, pi/2); hits z_u = z + (R - y) tan(theta),
     z_d = z - (R + y) tan(theta); keep the emission only if |z_u| <= L/2 and |z_d| <= L/2;
     dl = -2 y / cos(theta)  (Eq. 1 evaluated on the LOR);
  3. smear: z_u, z_d with N(0, sigma_z), dl with N(0, sigma_dl); no cut afterwards;
  4. repeat until exactly n detected events.
Output: float32 array [n, 3] = (z_u~, z_d~, dl~), C-contiguous - the layout of `events` in include/jpet.h.
RNG: numpy Generator(PCG64(seed)); draws are made in fixed-size chunks so a given (config, seed, n)
always yields the same array.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

_CHUNK = 1 << 21  # emissions drawn per RNG round; part of the recipe (changing it changes the stream)


@dataclasses.dataclass(frozen=True)
class Primitive:
    """One phantom primitive. kind 'E' = ellipse, 'B' = box; centre (cy, cz), half sizes (hy, hz) in mm,
    rotation phi in degrees counter-clockwise in the (z horizontal, y vertical) plane, relative intensity."""

    kind: str
    cy: float
    cz: float
    hy: float
    hz: float
    phi_deg: float
    intensity: float


@dataclasses.dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json `configs`, made concrete as in SURVEY.md section 8(d)."""

    name: str
    R: float  # strips at y = +-R  [mm]
    L: float  # strip length, |z| <= L/2  [mm]
    n_y: int
    n_z: int
    pixel: float  # mm
    n_events: int
    n_iter: int
    sigma_z: float
    sigma_dl: float
    phantom: tuple
    seed: int = 0
    batch: int = 0  # >0: events are streamed in batches of this many (config 5)


def _E(cy, cz, hy, hz, phi, rho):
    return Primitive("E", cy, cz, hy, hz, phi, rho)


def _B(cy, cz, hy, hz, phi, rho):
    return Primitive("B", cy, cz, hy, hz, phi, rho)


# BASELINE.json configs[0..4]; phantoms are SURVEY.md section 8(d)'s concrete choices (our own tables).
CONFIGS = {
    "cfg1": Config("cfg1", 450.0, 500.0, 64, 64, 5.0, 20_000, 1, 10.0, 40.0,
                   (_E(0, 0, 30, 30, 0, 4.0), _E(0, 0, 100, 150, 0, 1.0))),
    "cfg2": Config("cfg2", 450.0, 500.0, 200, 200, 2.5, 1_000_000, 10, 10.0, 40.0,
                   (_E(-40, 60, 20, 20, 0, 0.0), _E(40, -50, 15, 15, 0, 4.0),
                    _E(0, 40, 40, 60, 30, 2.0), _E(0, 0, 120, 160, 0, 1.0))),
    "cfg3": Config("cfg3", 450.0, 500.0, 400, 400, 1.25, 10_000_000, 10, 5.0, 20.0,
                   tuple(_B(cy, 0, 1, 100, 0, 1.0) for cy in (-40, -20, 0, 20, 40))),
    "cfg4": Config("cfg4", 450.0, 500.0, 200, 200, 2.5, 10_000_000, 5, 20.0, 80.0,
                   (_E(0, 0, 180, 180, 0, 1.0),)),
    "cfg5": Config("cfg5", 450.0, 500.0, 512, 512, 1.0, 100_000_000, 20, 10.0, 40.0,
                   (_E(0, -90, 12, 12, 0, 4.0), _E(-50, 70, 18, 18, 0, 3.0), _E(60, 20, 45, 25, -20, 0.0),
                    _E(-60, -20, 55, 30, 20, 2.0), _E(0, 0, 150, 200, 0, 1.0), _E(0, 0, 165, 215, 0, 2.0)),
                   batch=10_000_000),
    # The paper's own set-up: Fig. 4 geometry R = 130 mm, L = 300 mm, 4 x 4 mm pixels
    # and the phantom of Table 2 (rows (x, y, a, b, phi, rho), centre (x, y),
    # half-axes a, b, rotated by phi counter-clockwise, topmost row wins; x is the coordinate along the strips = z,
    # reading R21), sigma_z = 10 mm, sigma_dl = 40 mm.  The paper does not print the number of events
    # or the grid of Fig. 4; 64 x 80 pixels cover |y| < R and |z| <= L/2 + 8 mm, 2 x 10^6 events, 10 iterations.
    "fig4": Config("fig4", 130.0, 300.0, 64, 80, 4.0, 2_000_000, 10, 10.0, 40.0,
                   (_E(0, 0, 60, 30, 0, 0.3), _E(-62, 50, 33, 10, -40, 0.3), _E(-63, -50, 33, 20, 45, 0.5),
                    _E(65, 60, 14, 13, 0, 0.5), _E(55, 35, 12, 12, 0, 0.7), _E(0, 0, 110, 120, 0, 0.1))),
}


def _inside(p: Primitive, y: np.ndarray, z: np.ndarray) -> np.ndarray:
    """Membership of points in a primitive rotated by phi CCW in the (z, y) plane."""
    c, s = math.cos(math.radians(p.phi_deg)), math.sin(math.radians(p.phi_deg))
    dz, dy = z - p.cz, y - p.cy
    a = c * dz + s * dy   # coordinate along the primitive's own z axis
    b = -s * dz + c * dy  # ... and its own y axis
    if p.kind == "E":
        return (a / p.hz) ** 2 + (b / p.hy) ** 2 <= 1.0
    if p.kind == "B":
        return (np.abs(a) <= p.hz) & (np.abs(b) <= p.hy)
    raise ValueError(f"unknown primitive kind {p.kind!r}")


def phantom_intensity(phantom, y: np.ndarray, z: np.ndarray) -> np.ndarray:
    """Relative tracer density at points (y, z); first primitive in the list wins."""
    out = np.zeros(np.shape(y), dtype=np.float64)
    undecided = np.ones(np.shape(y), dtype=bool)
    for p in phantom:
        hit = undecided & _inside(p, y, z)
        out[hit] = p.intensity
        undecided &= ~hit
    return out


def _bounding_rectangle(phantom):
    ys, zs = [], []
    for p in phantom:
        c, s = abs(math.cos(math.radians(p.phi_deg))), abs(math.sin(math.radians(p.phi_deg)))
        if p.kind == "E":
            ez = math.hypot(p.hz * c, p.hy * s)
            ey = math.hypot(p.hz * s, p.hy * c)
        else:
            ez = p.hz * c + p.hy * s
            ey = p.hz * s + p.hy * c
        ys += [p.cy - ey, p.cy + ey]
        zs += [p.cz - ez, p.cz + ez]
    return min(ys), max(ys), min(zs), max(zs)


def generate_events(phantom, n: int, R: float, L: float, sigma_z: float, sigma_dl: float,
                    seed: int = 0, return_truth: bool = False):
    """n detected, smeared events as float32 [n, 3] = (z_u~, z_d~, dl~).

    With return_truth=True also returns the float64 emission points/angles [n, 3] = (y, z, theta)."""
    if n < 0:
        raise ValueError("n must be >= 0")
    rng = np.random.Generator(np.random.PCG64(seed))
    y0, y1, z0, z1 = _bounding_rectangle(phantom)
    rho_max = max(p.intensity for p in phantom)
    out = np.empty((n, 3), dtype=np.float32)
    truth = np.empty((n, 3), dtype=np.float64) if return_truth else None
    filled = 0
    half = 0.5 * L
    while filled < n:
        y = rng.uniform(y0, y1, _CHUNK)
        z = rng.uniform(z0, z1, _CHUNK)
        keep = rng.uniform(0.0, rho_max, _CHUNK) < phantom_intensity(phantom, y, z)
        theta = rng.uniform(-0.5 * math.pi, 0.5 * math.pi, _CHUNK)
        noise = rng.standard_normal((_CHUNK, 3))
        tan_t = np.tan(theta)
        z_u = z + (R - y) * tan_t
        z_d = z - (R + y) * tan_t
        keep &= (np.abs(z_u) <= half) & (np.abs(z_d) <= half)
        idx = np.flatnonzero(keep)[: n - filled]
        m = idx.size
        dl = -2.0 * y[idx] / np.cos(theta[idx])
        out[filled:filled + m, 0] = z_u[idx] + sigma_z * noise[idx, 0]
        out[filled:filled + m, 1] = z_d[idx] + sigma_z * noise[idx, 1]
        out[filled:filled + m, 2] = dl + sigma_dl * noise[idx, 2]
        if return_truth:
            truth[filled:filled + m, 0] = y[idx]
            truth[filled:filled + m, 1] = z[idx]
            truth[filled:filled + m, 2] = theta[idx]
        filled += m
    return (out, truth) if return_truth else out


def config_events(cfg: Config | str, n: int | None = None, seed: int | None = None) -> np.ndarray:
    """Events of a named config; `n` takes the first n events of that config's stream (a prefix of the
    full array, because events are produced in order)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    return generate_events(cfg.phantom, cfg.n_events if n is None else n, cfg.R, cfg.L,
                           cfg.sigma_z, cfg.sigma_dl, cfg.seed if seed is None else seed)


def noise_free_events(n: int, R: float, L: float, seed: int = 0, y_max: float | None = None):
    """Exact (unsmeared) events for emissions uniform in |y| <= y_max, |z| <= L/2 that hit both strips.

    Returns (events float64 [n,3], truth float64 [n,3] = (y, z, tan theta)); used to check that Eq. 2
    inverts Eq. 1."""
    rng = np.random.Generator(np.random.PCG64(seed))
    y_max = 0.8 * R if y_max is None else y_max
    ev = np.empty((n, 3))
    tr = np.empty((n, 3))
    filled = 0
    while filled < n:
        y = rng.uniform(-y_max, y_max, 4 * n + 16)
        z = rng.uniform(-0.5 * L, 0.5 * L, 4 * n + 16)
        theta = rng.uniform(-0.5 * math.pi, 0.5 * math.pi, 4 * n + 16)
        t = np.tan(theta)
        z_u = z + (R - y) * t
        z_d = z - (R + y) * t
        idx = np.flatnonzero((np.abs(z_u) <= 0.5 * L) & (np.abs(z_d) <= 0.5 * L))[: n - filled]
        m = idx.size
        # Eq. 1 written with the two hit points: distance to upper hit minus distance to lower hit
        dl = np.hypot(R - y[idx], z_u[idx] - z[idx]) - np.hypot(R + y[idx], z_d[idx] - z[idx])
        ev[filled:filled + m] = np.stack([z_u[idx], z_d[idx], dl], axis=1)
        tr[filled:filled + m] = np.stack([y[idx], z[idx], t[idx]], axis=1)
        filled += m
    return ev, tr
