"""Counter-based seeded generators for the five synthetic grids of BASELINE.json.

Recipe: SURVEY.md §8(d) / DESIGN.md "Input recipe".  The paper's own matrices
(Table I, exported from 3D-ICE) and floorplan power maps
 are not available; these grids take their structure
(7-point FV, layered stack, convective top, adiabatic sides, hotspot power maps
on active layers, same range of N) and stand in for them.

Random numbers: splitmix64 finaliser applied to a 64-bit key built from
(seed, stream id, element index); top 53 bits -> uniform in [0,1); Box-Muller
for normals.  No library random stream is used, so values never change with
the numpy version.

Nothing here computes conductances, matrices or solves anything.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

_U64 = np.uint64
_MASK = (1 << 64) - 1

CONFIG_NAMES = {
    1: "cfg1_steady_32x32x8",
    2: "cfg2_steady_256x256x16",
    3: "cfg3_steady_1024x1024x16_lognormal",
    4: "cfg4_steady_4096x4096x8",
    5: "cfg5_transient_512x512x16",
    6: "cfg6_paperlike_anisotropic_256x256x10",
}
SEEDS = {1: 178501, 2: 178502, 3: 178503, 4: 178504, 5: 178505, 6: 178506}

# stream ids (the second key component)
_ST_KAPPA_U1, _ST_KAPPA_U2 = 1, 2
_ST_HOT_X, _ST_HOT_Y, _ST_HOT_AMP = 3, 4, 5
_ST_CELL_POWER = 6
_ST_ACTIVITY = 7

# layer stacks, bottom -> top (W/m.K); BASELINE.json configs 1, 2, 4
S8 = [130.0, 2.0, 5.0, 130.0, 400.0, 130.0, 2.0, 130.0]
S8P = [130.0, 2.0, 2.0, 130.0, 5.0, 400.0, 400.0, 400.0]
# volumetric heat capacity by material (J/m^3.K); silicon from BASELINE.json cfg 5,
# the others are this build's choice (cfg 5)
_CV = {130.0: 1.63e6, 2.0: 2.2e6, 5.0: 2.0e6, 400.0: 3.45e6}

W_PER_MM2 = 1.0e6  # 1 W/mm^2 in W/m^2

# cfg 6: the layer THICKNESSES of the paper's 10-layer Memory-on-Logic stack,
# bottom to top (logic bulk 10, logic FEOL 2, logic BEOL 10, hybrid bonding 2, memory BEOL 10,
# memory FEOL 2, memory bulk 200, TIM 100, heat spreader 400, heat sink 1000 um).  Conductivities and the
# lateral cell size are not given in the paper: this build's choice (Si 130, BEOL / bonding 2, TIM 5,
# spreader and sink 400 W/m.K; 50 um cells).  Power on the two FEOL layers.  The floorplan power maps
# (SPARC / EV6 / 9-core) are not available: the synthetic hotspot maps are used instead.
PAPER_DZ_UM = [10.0, 2.0, 10.0, 2.0, 10.0, 2.0, 200.0, 100.0, 400.0, 1000.0]
PAPER_KAPPA = [130.0, 130.0, 2.0, 2.0, 2.0, 130.0, 130.0, 5.0, 400.0, 400.0]


def splitmix64(key: np.ndarray) -> np.ndarray:
    """splitmix64 output function on an array of uint64 keys (wrapping arithmetic)."""
    z = np.asarray(key, dtype=_U64).copy()
    with np.errstate(over="ignore"):
        z += _U64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)
        z = z ^ (z >> _U64(31))
    return z


def _key(seed: int, stream: int, idx: np.ndarray) -> np.ndarray:
    base = ((seed & 0xFFFFFFFF) << 32 | (stream & 0xFF) << 24) & _MASK
    hi = splitmix64(np.array([base], dtype=_U64))[0]
    with np.errstate(over="ignore"):
        return hi + np.asarray(idx, dtype=_U64) * _U64(0xD1342543DE82EF95)


def uniform01(seed: int, stream: int, idx) -> np.ndarray:
    """Uniform doubles in [0,1): top 53 bits of splitmix64(key(seed, stream, idx))."""
    bits = splitmix64(_key(seed, stream, np.asarray(idx)))
    return (bits >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(seed: int, stream_a: int, stream_b: int, idx) -> np.ndarray:
    """Standard normals by Box-Muller from two uniform streams."""
    u1 = uniform01(seed, stream_a, idx)
    u2 = uniform01(seed, stream_b, idx)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


@dataclass
class Workload:
    """Plain arrays describing one thermal problem (inputs only, no matrix)."""
    cfg: int
    name: str
    seed: int
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: np.ndarray                      # [nz] m
    kappa_layer: np.ndarray             # [nz] W/m.K (layer means)
    kappa_cell: Optional[np.ndarray]    # [N] W/m.K or None (layered)
    h_top: float                        # W/m^2.K on z = nz-1
    cvol: Optional[np.ndarray]          # [nz] J/m^3.K or None (steady)
    dt: float                           # s, 0 => steady
    active: list                        # active layer indices
    power: np.ndarray                   # [N] W per cell (b for steady; P_1 for transient)
    mixed: bool                         # BASELINE's mode for this config
    rtol: float = 1e-8
    true_resid_period: int = 20
    n_steps: int = 0
    n_sites: int = 0
    extra: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def transient(self) -> bool:
        return self.dt > 0.0


def _stack(nz: int, base):
    reps = (nz + len(base) - 1) // len(base)
    return np.array((base * reps)[:nz], dtype=np.float64)


def _active_layers(nz: int, base_len: int = 8):
    out = []
    for z0 in range(0, nz, base_len):
        for a in (0, 3):
            if z0 + a < nz:
                out.append(z0 + a)
    return out


def _add_gaussian_hotspots(q, nx, ny, active, n_hot, seed, peak, sigma=3.0):
    """q: [nz, ny, nx] areal density (W/m^2); adds truncated (6 sigma) Gaussians in place."""
    j = np.arange(n_hot)
    cx = np.minimum((uniform01(seed, _ST_HOT_X, j) * nx).astype(np.int64), nx - 1)
    cy = np.minimum((uniform01(seed, _ST_HOT_Y, j) * ny).astype(np.int64), ny - 1)
    rad = int(np.ceil(6.0 * sigma))
    for k in range(n_hot):
        z = active[k % len(active)]
        x0, x1 = max(0, cx[k] - rad), min(nx, cx[k] + rad + 1)
        y0, y1 = max(0, cy[k] - rad), min(ny, cy[k] + rad + 1)
        xs = np.arange(x0, x1, dtype=np.float64) - cx[k]
        ys = np.arange(y0, y1, dtype=np.float64) - cy[k]
        r2 = ys[:, None] ** 2 + xs[None, :] ** 2
        g = peak * np.exp(-r2 / (2.0 * sigma * sigma))
        g[r2 > (6.0 * sigma) ** 2] = 0.0
        q[z, y0:y1, x0:x1] += g
    return cx, cy


def _sites(seed, nx, ny, n_sites):
    j = np.arange(n_sites)
    cx = np.minimum((uniform01(seed, _ST_HOT_X, j) * nx).astype(np.int64), nx - 1)
    cy = np.minimum((uniform01(seed, _ST_HOT_Y, j) * ny).astype(np.int64), ny - 1)
    return cx, cy


def make_workload(cfg: int, nx: int = 0, ny: int = 0, nz: int = 0, n_hot: int = -1,
                  seed: int = 0) -> Workload:
    """Build config `cfg` (1..5 = BASELINE.json; 6 = paper-like anisotropic stack).  nx/ny/nz/n_hot override the full size to get a
    small grid with the same recipe (used by the parity tests)."""
    full = {1: (32, 32, 8, 4), 2: (256, 256, 16, 64), 3: (1024, 1024, 16, 1024),
            4: (4096, 4096, 8, 4096), 5: (512, 512, 16, 256), 6: (256, 256, 10, 64)}[cfg]
    nx = nx or full[0]
    ny = ny or full[1]
    nz = nz or full[2]
    n_hot = full[3] if n_hot < 0 else n_hot
    seed = seed or SEEDS[cfg]
    n = nx * ny * nz
    dx = dy = 1.0e-6
    dz = np.full(nz, 1.0e-6)
    h = 1.0e4
    base = S8P if cfg == 4 else S8
    kl = _stack(nz, base)
    active = [0, 3] if cfg == 4 else _active_layers(nz)
    active = [a for a in active if a < nz]
    bg = 0.5 * W_PER_MM2
    q = np.zeros((nz, ny, nx), dtype=np.float64)
    kappa_cell = None
    cvol = None
    dt = 0.0
    mixed = cfg in (2, 3, 4, 5, 6)
    period = 20
    n_steps = 0
    n_sites = 0
    extra = {}

    if cfg == 6:
        assert nz == 10, "cfg 6 is the paper's 10-layer stack"
        dx = dy = 50.0e-6
        dz = np.array(PAPER_DZ_UM) * 1e-6
        kl = np.array(PAPER_KAPPA)
        active = [1, 5]
        bg = 0.05 * W_PER_MM2
        for z in active:
            q[z] += bg
        _add_gaussian_hotspots(q, nx, ny, active, n_hot, seed, 1.0 * W_PER_MM2)
    elif cfg in (1, 2):
        for z in active:
            q[z] += bg
        _add_gaussian_hotspots(q, nx, ny, active, n_hot, seed, 20.0 * W_PER_MM2)
    elif cfg == 3:
        idx = np.arange(n, dtype=np.uint64)
        nrm = normal01(seed, _ST_KAPPA_U1, _ST_KAPPA_U2, idx)
        kappa_cell = (np.repeat(kl, nx * ny) * np.exp(0.2 * nrm - 0.02)).astype(np.float64)
        for z in active:
            q[z] += bg
        cx, cy = _sites(seed, nx, ny, n_hot)
        u = uniform01(seed, _ST_HOT_AMP, np.arange(n_hot))
        for k in range(n_hot):
            q[active[k % len(active)], cy[k], cx[k]] = bg * (1.0 + 5.0 * u[k])
    elif cfg == 4:
        for a_i, z in enumerate(active):
            idx = np.arange(nx * ny, dtype=np.uint64) + np.uint64(a_i * nx * ny)
            q[z] = (2.0 * W_PER_MM2) * uniform01(seed, _ST_CELL_POWER, idx).reshape(ny, nx)
        _add_gaussian_hotspots(q, nx, ny, active, n_hot, seed, 20.0 * W_PER_MM2)
    elif cfg == 5:
        cvol = np.array([_CV[k] for k in kl], dtype=np.float64)
        dt = 1.0e-5
        period = 5
        n_steps = 200
        n_sites = n_hot
        for z in active:
            q[z] += bg
        extra["background_q"] = q.copy()
        cx, cy = _sites(seed, nx, ny, n_hot)
        extra["site_x"], extra["site_y"] = cx, cy
    else:
        raise ValueError("cfg must be 1..5")

    power = (q * (dx * dy)).reshape(n)
    w = Workload(cfg=cfg, name=CONFIG_NAMES[cfg] if (nx, ny, nz) == full[:3] else
                 f"cfg{cfg}_small_{nx}x{ny}x{nz}", seed=seed, nx=nx, ny=ny, nz=nz, dx=dx, dy=dy,
                 dz=dz, kappa_layer=kl, kappa_cell=kappa_cell, h_top=h, cvol=cvol, dt=dt,
                 active=active, power=power, mixed=mixed, true_resid_period=period,
                 n_steps=n_steps, n_sites=n_sites, extra=extra)
    if cfg == 5:
        w.power = power_for_step(w, 1)
    return w


def power_for_step(w: Workload, step: int) -> np.ndarray:
    """Power map P_step (W per cell) of the transient config: background plus the
    hotspot sites that are ON at this step (each site on with probability 1/2,
    independently per (step, site))."""
    assert w.cfg == 5
    q = w.extra["background_q"].copy()
    sites = np.arange(w.n_sites, dtype=np.uint64)
    on = uniform01(w.seed, _ST_ACTIVITY, np.uint64(step) * np.uint64(1 << 20) + sites) < 0.5
    sigma, peak = 3.0, 20.0 * W_PER_MM2
    rad = int(np.ceil(6.0 * sigma))
    cx, cy = w.extra["site_x"], w.extra["site_y"]
    for k in range(w.n_sites):
        if not on[k]:
            continue
        z = w.active[k % len(w.active)]
        x0, x1 = max(0, cx[k] - rad), min(w.nx, cx[k] + rad + 1)
        y0, y1 = max(0, cy[k] - rad), min(w.ny, cy[k] + rad + 1)
        xs = np.arange(x0, x1, dtype=np.float64) - cx[k]
        ys = np.arange(y0, y1, dtype=np.float64) - cy[k]
        r2 = ys[:, None] ** 2 + xs[None, :] ** 2
        g = peak * np.exp(-r2 / (2.0 * sigma * sigma))
        g[r2 > (6.0 * sigma) ** 2] = 0.0
        q[z, y0:y1, x0:x1] += g
    return (q * (w.dx * w.dy)).reshape(w.n)
