"""Seeded synthetic inputs for the coupled flood-pedestrian step.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only draws terrain, walls, water, crowds and the navigation field
(an *input* the paper says the user specifies) and hands them over
as plain numpy arrays.  It imports neither the CUDA binding nor the oracle.

The paper's case study (a 332 m shopping centre; Fig. 4 unreadable) is not available,
so these generators stand in for it with the same shapes: a walled hall, an inflow breach on the
south side, an exit on the opposite side, ~1 pedestrian per 100 m2, n_M = 0.01
(P:L138).  The five recipes are BASELINE.json `configs[0..4]` as completed by SURVEY 8(d); every
value the configs leave open is listed in DESIGN.md.

Arrays are row-major [j][i]; cell (i, j) has centre ((i+.5)dx, (j+.5)dy).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# direction codes of the navigation field: E, NE, N, NW, W, SW, S, SE ; 255 = none
DIR_DI = np.array([1, 1, 0, -1, -1, -1, 0, 1])
DIR_DJ = np.array([0, 1, 1, 1, 0, -1, -1, -1])
DIR_NONE = 255
SIDE_W, SIDE_E, SIDE_S, SIDE_N = 0, 1, 2, 3


@dataclass
class Scenario:
    name: str
    nx: int
    ny: int
    dx: float
    dy: float
    real_bits: int
    z: np.ndarray
    manning: np.ndarray
    mask: np.ndarray
    h0: np.ndarray
    u0: np.ndarray | None
    v0: np.ndarray | None
    px: np.ndarray
    py: np.ndarray
    pvx: np.ndarray
    pvy: np.ndarray
    pvpref: np.ndarray
    prole: np.ndarray
    nav_dir: np.ndarray                      # [n_targets, ny*nx] uint8
    exit_cells: np.ndarray
    # hydrodynamics
    g: float = 9.81
    cfl: float = 0.5
    dt_max: float = 0.0                      # <= 0: default of SURVEY C10
    h_dry: float = 1e-3
    couple_roughness: int = 1
    n_cap: int = 20
    inflow_cell: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))
    inflow_side: np.ndarray = field(default_factory=lambda: np.zeros(0, np.uint8))
    hydro_t: np.ndarray = field(default_factory=lambda: np.zeros(0))
    hydro_q: np.ndarray = field(default_factory=lambda: np.zeros(0))
    # Table 1
    hr_edges: tuple = (0.75, 1.5, 2.5, 20.0)
    speed_wet: tuple = (1.8, 0.9, 0.45, 0.0)
    # social force defaults
    tau: float = 0.5
    A_s: float = 25.0
    B_s: float = 0.08
    radius: float = 0.3
    R_int: float = 1.0
    vmax_factor: float = 1.3
    # navigation targets
    exit_target: int = 0
    storage_target: int = 0
    drop_target: int = 0
    storage_cell: int = 0
    drop_cell: int = 0
    arrive_cells: int = 1
    # barrier
    line_cells: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))
    bags_per_cell_layer: int = 1
    n_layers: int = 0
    layer_thickness: float = 0.25
    t_pick: float = 30.0
    t_drop: float = 30.0
    t_end: float = float("inf")
    steps: int = 0                           # the run length the config names (0: until t_end)
    # widened scope
    flood_order: int = 1                     # 1: the paper's first-order scheme; 2: MUSCL-Hancock (8f-2)
    # 8f-3 (D1-D9): open edges, entrance doors, pre-flood phase, trigger
    open_sides: int = 0                      # bit 0 W, 1 E, 2 S, 3 N: that domain edge is open (transmissive)
    door_cells: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))
    door_target: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))   # nav field index per door
    spawn_rate: float = 0.0                  # pedestrians per second per door
    target_population: int = 0
    spawn_seed: int = 0
    spawn_vpref_lo: float = 1.0
    spawn_vpref_hi: float = 1.4
    pactive0: np.ndarray | None = None       # initial active flag per slot (None: all active)

    @property
    def real(self):
        return np.float64 if self.real_bits == 64 else np.float32

    @property
    def n_peds(self) -> int:
        return int(self.px.shape[0])


def _as_real(a, real_bits):
    """Round to the storage precision (float32 arrays for fp32 configs) so that both sides
    receive identical values: float32 -> float64 is exact."""
    return np.ascontiguousarray(a, dtype=np.float32 if real_bits == 32 else np.float64)


# --------------------------------------------------------------------------- navigation field

def _grid_distance(mask: np.ndarray, targets: np.ndarray) -> np.ndarray:
    """8-connected shortest-path length (in cells; diagonal sqrt(2), no corner cutting) from
    every walkable cell to the nearest target cell; inf where unreachable."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import dijkstra

    ny, nx = mask.shape
    walk = mask == 0
    idx = np.arange(ny * nx).reshape(ny, nx)
    rows, cols, w = [], [], []
    for code in range(8):
        di, dj = int(DIR_DI[code]), int(DIR_DJ[code])
        src = walk.copy()
        dst_ok = np.zeros_like(walk)
        js, je = max(0, -dj), ny - max(0, dj)
        is_, ie = max(0, -di), nx - max(0, di)
        dst_ok[js:je, is_:ie] = walk[js + dj:je + dj, is_ + di:ie + di]
        ok = src & dst_ok
        if di != 0 and dj != 0:               # no corner cutting: both side cells walkable
            a = np.zeros_like(walk); b = np.zeros_like(walk)
            a[:, is_:ie] = walk[:, is_ + di:ie + di]
            b[js:je, :] = walk[js + dj:je + dj, :]
            ok &= a & b
        s = idx[ok]
        rows.append(s); cols.append(s + dj * nx + di)
        w.append(np.full(s.shape, np.sqrt(2.0) if (di and dj) else 1.0))
    g = csr_matrix((np.concatenate(w), (np.concatenate(rows), np.concatenate(cols))),
                   shape=(ny * nx, ny * nx))
    d = dijkstra(g, directed=False, indices=np.asarray(targets, dtype=np.int64), min_only=True)
    return d.reshape(ny, nx)


def nav_field(mask: np.ndarray, targets) -> tuple[np.ndarray, np.ndarray]:
    """Direction code of the first step of a shortest 8-connected path to the nearest target
    (ties -> lowest code); 255 on targets, solids and unreachable cells.  Returns (dir, dist)."""
    ny, nx = mask.shape
    targets = np.atleast_1d(np.asarray(targets, dtype=np.int64))
    dist = _grid_distance(mask, targets)
    walk = mask == 0
    best = np.full((ny, nx), np.inf)
    code_out = np.full((ny, nx), DIR_NONE, dtype=np.uint8)
    big = np.where(np.isfinite(dist), dist, np.inf)
    for code in range(8):
        di, dj = int(DIR_DI[code]), int(DIR_DJ[code])
        cand = np.full((ny, nx), np.inf)
        js, je = max(0, -dj), ny - max(0, dj)
        is_, ie = max(0, -di), nx - max(0, di)
        cand[js:je, is_:ie] = big[js + dj:je + dj, is_ + di:ie + di]
        if di != 0 and dj != 0:
            a = np.zeros_like(walk); b = np.zeros_like(walk)
            a[:, is_:ie] = walk[:, is_ + di:ie + di]
            b[js:je, :] = walk[js + dj:je + dj, :]
            cand[~(a & b)] = np.inf
        cand = np.round(cand + (np.sqrt(2.0) if (di and dj) else 1.0), 9)
        better = cand < best
        best[better] = cand[better]
        code_out[better] = code
    code_out[~walk] = DIR_NONE
    code_out[~np.isfinite(dist)] = DIR_NONE
    code_out.reshape(-1)[targets] = DIR_NONE
    return code_out.reshape(-1), dist


def nav_field_open(nx: int, ny: int, targets) -> np.ndarray:
    """Navigation field of an obstacle-free hall: step towards the nearest target in the
    8-connected (octile) metric, diagonal first.  Used where a graph search over the full grid
    would be wasteful (Config 5: 6.7e7 cells, no walls)."""
    targets = np.atleast_1d(np.asarray(targets, dtype=np.int64))
    i = np.arange(nx, dtype=np.int32)[None, :]
    j = np.arange(ny, dtype=np.int32)[:, None]
    best = np.full((ny, nx), np.inf, dtype=np.float32)
    code = np.full((ny, nx), DIR_NONE, dtype=np.uint8)
    lut = np.full((3, 3), DIR_NONE, dtype=np.uint8)          # [sign(dj)+1][sign(di)+1]
    for c in range(8):
        lut[DIR_DJ[c] + 1, DIR_DI[c] + 1] = c
    for t in targets:
        ti, tj = int(t % nx), int(t // nx)
        di, dj = ti - i, tj - j
        a, b = np.abs(di), np.abs(dj)
        d = (np.maximum(a, b) + (np.sqrt(2.0) - 1.0) * np.minimum(a, b)).astype(np.float32)
        c = lut[np.sign(dj) + 1, np.sign(di) + 1]
        better = d < best
        best[better] = d[better]
        code[better] = c[better]
    return code.reshape(-1)


# --------------------------------------------------------------------------- terrain helpers

def _value_noise(rng, ny, nx, spacings, weights):
    """Multi-octave bilinear value noise normalised to [0, 1]."""
    z = np.zeros((ny, nx))
    jj = np.arange(ny)[:, None]
    ii = np.arange(nx)[None, :]
    for sp, w in zip(spacings, weights):
        gy, gx = ny // sp + 2, nx // sp + 2
        lat = rng.random((gy, gx))
        fj, fi = jj / sp, ii / sp
        j0, i0 = np.floor(fj).astype(int), np.floor(fi).astype(int)
        tj, ti = fj - j0, fi - i0
        z += w * ((1 - tj) * (1 - ti) * lat[j0, i0] + (1 - tj) * ti * lat[j0, i0 + 1]
                  + tj * (1 - ti) * lat[j0 + 1, i0] + tj * ti * lat[j0 + 1, i0 + 1])
    z -= z.min()
    z /= z.max()
    return z


def _place_in_cells(rng, cells, nx, dx, dy, n):
    """n positions: a uniformly drawn cell of `cells` each, uniform inside the cell."""
    pick = cells[rng.integers(0, cells.shape[0], size=n)]
    x = (pick % nx + rng.random(n)) * dx
    y = (pick // nx + rng.random(n)) * dy
    return x, y


def _keep_inside(x, n, d, real_bits):
    """Round to storage precision and keep strictly inside [0, n*d)."""
    x = _as_real(x, real_bits)
    hi = np.nextafter(np.float32(n * d), np.float32(0)) if real_bits == 32 else np.nextafter(n * d, 0.0)
    return np.clip(x, x.dtype.type(0), hi).astype(x.dtype)


def _triangle(t0, t_peak, t1, q_peak):
    return np.array([t0, t_peak, t1], dtype=np.float64), np.array([0.0, q_peak, 0.0])


def _vpref(rng, n):
    return np.clip(rng.normal(1.2, 0.2, size=n), 0.6, 1.8)


# --------------------------------------------------------------------------- Config 1

def tiny_dam_break(n: int = 64, n_peds: int = 256, bump: bool = True, friction: float = 0.02,
                   steps: int = 100) -> Scenario:
    """BASELINE.json configs[0]: 64x64, dx = 1 m, fp64, Gaussian bump 0.3 m / sigma 5 cells
    centred at (44, 32) [centre: SURVEY C40], n = 0.02, depth 1.0 m for i < n/2 else 0.1 m,
    closed walls; 256 pedestrians (seed 0) in the shallow half heading for exit (n-1, n/2)."""
    nx = ny = n
    ii, jj = np.meshgrid(np.arange(nx), np.arange(ny))
    z = 0.3 * np.exp(-((ii - 44 * n / 64) ** 2 + (jj - 32 * n / 64) ** 2) / (2.0 * (5.0 * n / 64) ** 2)) \
        if bump else np.zeros((ny, nx))
    h0 = np.where(ii < nx // 2, 1.0, 0.1)
    mask = np.zeros((ny, nx), np.uint8)
    rng = np.random.Generator(np.random.PCG64(0))
    x = nx / 2 + nx / 2 * rng.random(n_peds)
    y = ny * rng.random(n_peds)
    exit_cell = (ny // 2) * nx + (nx - 1)
    nav, _ = nav_field(mask, [exit_cell])
    return Scenario(
        name="config1_tiny_dam_break", nx=nx, ny=ny, dx=1.0, dy=1.0, real_bits=64,
        z=z.reshape(-1), manning=np.full(nx * ny, friction), mask=mask.reshape(-1),
        h0=h0.reshape(-1).astype(np.float64), u0=None, v0=None,
        px=_keep_inside(x, nx, 1.0, 64), py=_keep_inside(y, ny, 1.0, 64),
        pvx=np.zeros(n_peds), pvy=np.zeros(n_peds), pvpref=np.full(n_peds, 1.2),
        prole=np.zeros(n_peds, np.uint8), nav_dir=nav[None, :].copy(),
        exit_cells=np.array([exit_cell], np.int32), steps=steps)


# --------------------------------------------------------------------------- Configs 2 and 3

def _hall(n: int, seed: int):
    """Walls (20 random rectangles, 15 % of cells) and bed (smooth 0..0.2 m) of the synthetic
    shopping centre, scaled from the 256-cell recipe."""
    from scipy.ndimage import gaussian_filter

    s = n / 256.0
    rng = np.random.Generator(np.random.PCG64(seed))
    lo, hi = max(2, int(round(12 * s))), max(3, int(round(32 * s)))
    w = rng.integers(lo, hi + 1, size=20).astype(float)
    hgt = rng.integers(lo, hi + 1, size=20).astype(float)
    cx = rng.random(20)
    cy = rng.random(20)
    edge = max(1, int(round(4 * s)))
    # keep-out: barrier line of Config 3 (j = 40, i in [104, 152)) so that both configs share walls
    ko_j0, ko_j1 = int(36 * s), int(45 * s) + 1
    ko_i0, ko_i1 = int(104 * s), int(152 * s)

    def raster(scale):
        m = np.zeros((n, n), np.uint8)
        for k in range(20):
            ww = max(1, int(round(w[k] * scale)))
            hh = max(1, int(round(hgt[k] * scale)))
            i0 = edge + int(cx[k] * max(1, n - 2 * edge - ww))
            j0 = edge + int(cy[k] * max(1, n - 2 * edge - hh))
            m[j0:min(j0 + hh, n - edge), i0:min(i0 + ww, n - edge)] = 1
        m[ko_j0:ko_j1, ko_i0:ko_i1] = 0
        return m

    scale, mask = 1.0, None
    for _ in range(60):                      # resize until the union covers 15 % +- 0.5 %
        mask = raster(scale)
        frac = mask.mean()
        if abs(frac - 0.15) <= 0.005:
            break
        scale *= np.sqrt(0.15 / max(frac, 1e-6)) ** 0.7
    zn = gaussian_filter(rng.normal(size=(n, n)), sigma=8 * s, mode="reflect")
    zn -= zn.min()
    z = 0.2 * zn / zn.max()
    return mask, z, rng


def shopping_centre(n: int = 256, n_evac: int = 2000, n_resp: int = 0, q_peak: float = 2.0,
                    t_release: float = 0.0, t_end: float = 3600.0, seed: int = 1,
                    name: str = "config2_shopping_centre") -> Scenario:
    """BASELINE.json configs[1] (and [2] through `pre_flood_intervention`): n x n cells at
    0.5 m * 256/n, fp32, dry start, triangular hydrograph through a south-edge breach
    i in [90, 166) * n/256, one exit at (n/2, n-1)."""
    nx = ny = n
    s = n / 256.0
    dx = 0.5 / s
    mask, z, _ = _hall(n, seed)
    exit_cell = (ny - 1) * nx + nx // 2
    i0, i1 = int(round(90 * s)), int(round(166 * s))
    inflow_cell = np.arange(i0, i1, dtype=np.int32)            # j = 0
    mask.reshape(-1)[inflow_cell] = 0
    mask.reshape(-1)[exit_cell] = 0
    nav_exit, dist = nav_field(mask, [exit_cell])
    reachable = np.flatnonzero(np.isfinite(dist.reshape(-1)) & (mask.reshape(-1) == 0))
    rng = np.random.Generator(np.random.PCG64(100 + (3 if n_resp else 2)))
    n_p = n_resp + n_evac
    x, y = _place_in_cells(rng, reachable, nx, dx, dx, n_p)     # responders are the first n_resp
    vpref = _vpref(rng, n_p)
    role = np.zeros(n_p, np.uint8)
    role[:n_resp] = 1
    ht, hq = _triangle(t_release, t_release + 300.0, t_release + 600.0, q_peak)
    sc = Scenario(
        name=name, nx=nx, ny=ny, dx=dx, dy=dx, real_bits=32,
        z=_as_real(z.reshape(-1), 32), manning=_as_real(np.full(nx * ny, 0.01), 32),
        mask=mask.reshape(-1).copy(), h0=np.zeros(nx * ny, np.float32), u0=None, v0=None,
        px=_keep_inside(x, nx, dx, 32), py=_keep_inside(y, ny, dx, 32),
        pvx=np.zeros(n_p, np.float32), pvy=np.zeros(n_p, np.float32), pvpref=_as_real(vpref, 32), prole=role,
        nav_dir=nav_exit[None, :].copy(), exit_cells=np.array([exit_cell], np.int32),
        inflow_cell=inflow_cell, inflow_side=np.full(inflow_cell.shape, SIDE_S, np.uint8),
        hydro_t=ht, hydro_q=hq, t_end=t_end)
    if n_resp:
        line_j = int(round(40 * s))
        line = np.array([line_j * nx + i for i in range(int(round(108 * s)), int(round(148 * s)))], np.int32)
        line = line[mask.reshape(-1)[line] == 0]
        drop_cell = int(line[0])
        want = int(round(200 * s)) * nx + int(round(30 * s))
        jj, ii = np.divmod(reachable, nx)
        storage_cell = int(reachable[np.argmin((ii - want % nx) ** 2 + (jj - want // nx) ** 2)])
        nav_sto, _ = nav_field(mask, [storage_cell])
        nav_drop, _ = nav_field(mask, [drop_cell])
        sc.nav_dir = np.stack([nav_exit, nav_sto, nav_drop])
        sc.exit_target, sc.storage_target, sc.drop_target = 0, 1, 2
        sc.storage_cell, sc.drop_cell = storage_cell, drop_cell
        sc.line_cells = line
        sc.bags_per_cell_layer, sc.n_layers, sc.layer_thickness = 1, 12, 0.05
        sc.t_pick = sc.t_drop = 30.0
    return sc


def door_hall(n: int = 64, slots: int = 400, n_init: int = 0, target_population: int = 200,
              spawn_rate: float = 10.0 / 60.0, t_pre: float = 300.0, q_peak: float = 1.0,
              t_end: float = 1800.0, seed: int = 7, open_north: bool = False, real_bits: int = 32) -> Scenario:
    """Scenario 1 of the paper in miniature (Fig. 4 unreadable, so the
    geometry is synthetic): an n x n hall at 0.5 m * 256/n with the walls and bed of the shopping
    centre, SEVEN entrance doors (three on the west wall, three on the east, one on the south), a
    pre-flood phase of `t_pre` seconds during which pedestrians enter at `spawn_rate` per second and
    door, each bound for one of the seven doors with probability 1/7, then the triangular flood
    through the southern breach; the emergency exit is at the middle of the north wall.  `slots`
    agent slots, the first `n_init` of them already walking at t = 0."""
    nx = ny = n
    s = n / 256.0
    dx = 0.5 / s
    mask, z, _ = _hall(n, seed)
    m = mask.reshape(-1)
    exit_cell = (ny - 1) * nx + nx // 2
    i0, i1 = int(round(90 * s)), int(round(166 * s))
    inflow_cell = np.arange(i0, i1, dtype=np.int32)
    doors = [(0, ny // 4), (0, ny // 2), (0, 3 * ny // 4), (nx - 1, ny // 4), (nx - 1, ny // 2), (nx - 1, 3 * ny // 4),
             (max(i0 - 4, 1), 0)]
    door_cells = np.array([j * nx + i for i, j in doors], np.int32)
    m[inflow_cell] = 0; m[exit_cell] = 0; m[door_cells] = 0
    nav_exit, dist = nav_field(mask, [exit_cell])
    assert np.all(np.isfinite(dist.reshape(-1)[door_cells])), "a door cannot reach the exit"
    navs = [nav_exit] + [nav_field(mask, [int(c)])[0] for c in door_cells]
    reachable = np.flatnonzero(np.isfinite(dist.reshape(-1)) & (m == 0))
    rng = np.random.Generator(np.random.PCG64(100 + seed))
    x, y = _place_in_cells(rng, reachable, nx, dx, dx, slots)
    vpref = _vpref(rng, slots)
    act = np.zeros(slots, np.uint8); act[:n_init] = 1
    ht, hq = _triangle(t_pre, t_pre + 300.0, t_pre + 600.0, q_peak)
    return Scenario(
        name="door_hall", nx=nx, ny=ny, dx=dx, dy=dx, real_bits=real_bits,
        z=_as_real(z.reshape(-1), real_bits), manning=_as_real(np.full(nx * ny, 0.01), real_bits),
        mask=m.copy(), h0=np.zeros(nx * ny, np.float32 if real_bits == 32 else np.float64), u0=None, v0=None,
        px=_keep_inside(x, nx, dx, real_bits), py=_keep_inside(y, ny, dx, real_bits),
        pvx=np.zeros(slots), pvy=np.zeros(slots), pvpref=_as_real(vpref, real_bits), prole=np.zeros(slots, np.uint8),
        nav_dir=np.stack(navs), exit_cells=np.array([exit_cell], np.int32), exit_target=0,
        inflow_cell=inflow_cell, inflow_side=np.full(inflow_cell.shape, SIDE_S, np.uint8),
        hydro_t=ht, hydro_q=hq, t_end=t_end,
        open_sides=(1 << SIDE_N) if open_north else 0,
        door_cells=door_cells, door_target=np.arange(1, 8, dtype=np.int32),
        spawn_rate=spawn_rate, target_population=target_population, spawn_seed=0x5eed0000 + seed,
        spawn_vpref_lo=1.0, spawn_vpref_hi=1.4, pactive0=act)


def pre_flood_intervention(n: int = 256, n_evac: int = 1000, n_resp: int = 100,
                           t_end: float = 3900.0) -> Scenario:
    """BASELINE.json configs[2]: Config 2's hall; 100 responders build a 40-cell barrier line at
    j = 40, each deposit raising the bed 0.05 m up to 0.6 m; flood released after 300 s."""
    return shopping_centre(n=n, n_evac=n_evac, n_resp=n_resp, t_release=300.0, t_end=t_end,
                           name="config3_pre_flood_intervention")


# --------------------------------------------------------------------------- Config 4

def scaled_flood(n: int = 2048, n_peds: int = 100_000, steps: int = 1000, seed: int = 3) -> Scenario:
    """BASELINE.json configs[3]: n x n at 0.25 m, fp32, 5-octave bed (1 m), Manning U[0.012, 0.05],
    16x16-cell building blocks solid with p = 0.25, reservoir eta = 2 m for i < n/4 [SURVEY C40],
    pedestrians on reachable cells with i >= n/4, exits at the 4 edge midpoints."""
    nx = ny = n
    dx = 0.25
    rng = np.random.Generator(np.random.PCG64(seed))
    sp = [max(2, n // 8 >> o) for o in range(5)]               # 256,128,...,16 at n = 2048
    z = _value_noise(rng, ny, nx, sp, [2.0 ** -o for o in range(5)])
    manning = rng.uniform(0.012, 0.05, size=(ny, nx))
    blk = 16
    nb = (n + blk - 1) // blk
    solid_blk = rng.random((nb, nb)) < 0.25
    exits = np.array([(ny // 2) * nx + 0, (ny // 2) * nx + nx - 1, 0 * nx + nx // 2, (ny - 1) * nx + nx // 2], np.int32)
    for e in exits:
        solid_blk[(e // nx) // blk, (e % nx) // blk] = False
    mask = np.kron(solid_blk.astype(np.uint8), np.ones((blk, blk), np.uint8))[:ny, :nx].copy()
    ii = np.arange(nx)[None, :]
    h0 = np.where((ii < nx // 4) & (mask == 0), np.maximum(0.0, 2.0 - z), 0.0)
    nav, dist = nav_field(mask, exits)
    ok = np.isfinite(dist) & (mask == 0) & (ii >= nx // 4)
    cells = np.flatnonzero(ok.reshape(-1))
    prng = np.random.Generator(np.random.PCG64(104))
    x, y = _place_in_cells(prng, cells, nx, dx, dx, n_peds)
    vpref = _vpref(prng, n_peds)
    return Scenario(
        name="config4_scaled_flood", nx=nx, ny=ny, dx=dx, dy=dx, real_bits=32,
        z=_as_real(z.reshape(-1), 32), manning=_as_real(manning.reshape(-1), 32),
        mask=mask.reshape(-1), h0=_as_real(h0.reshape(-1), 32),
        u0=None, v0=None,
        px=_keep_inside(x, nx, dx, 32), py=_keep_inside(y, ny, dx, 32),
        pvx=np.zeros(n_peds, np.float32), pvy=np.zeros(n_peds, np.float32), pvpref=_as_real(vpref, 32),
        prole=np.zeros(n_peds, np.uint8), nav_dir=nav[None, :].copy(), exit_cells=exits, steps=steps)


# --------------------------------------------------------------------------- Config 5

def throughput_stress(n: int = 8192, n_peds: int = 1_000_000, steps: int = 500, seed: int = 4) -> Scenario:
    """BASELINE.json configs[4]: n x n fp32 at 0.25 m [dx: SURVEY C40], multi-octave bed, n = 0.02,
    no walls, still water at the 60th percentile of z (exactly 60 % of cells wet) plus a 0.5 m
    Gaussian mound (sigma 100 m) at the centre, inflow over the whole south edge ramping to
    2000 m3/s * (n/8192) in 60 s; 8 Gaussian crowds (sigma 20 m) in the central half."""
    nx = ny = n
    dx = 0.25
    rng = np.random.Generator(np.random.PCG64(seed))
    sp = [max(2, n // 8 >> o) for o in range(5)]               # 1024,...,64 at n = 8192
    z = _value_noise(rng, ny, nx, sp, [2.0 ** -o for o in range(5)]).astype(np.float32)
    eta0 = np.float32(np.quantile(z, 0.6))
    jj = (np.arange(ny, dtype=np.float32)[:, None] + 0.5) * dx - ny * dx / 2
    ii = (np.arange(nx, dtype=np.float32)[None, :] + 0.5) * dx - nx * dx / 2
    sig = np.float32(100.0 * n / 8192)
    eta = eta0 + np.float32(0.5) * np.exp(-(ii * ii + jj * jj) / (2 * sig * sig))
    h0 = np.where(z < eta0, eta - z, 0.0).astype(np.float32)   # only already-wet cells carry the mound
    exits = np.array([(ny // 2) * nx + 0, (ny // 2) * nx + nx - 1, 0 * nx + nx // 2, (ny - 1) * nx + nx // 2], np.int32)
    nav = nav_field_open(nx, ny, exits)
    prng = np.random.Generator(np.random.PCG64(105))
    L = nx * dx
    centres = L * (0.25 + 0.5 * prng.random((8, 2)))
    per = n_peds // 8
    xs, ys = [], []
    sigma_c = 20.0 * n / 8192
    for k in range(8):
        m = per if k < 7 else n_peds - 7 * per
        x = np.empty(0); y = np.empty(0)
        while x.size < m:
            cand = centres[k] + prng.normal(0.0, sigma_c, size=(m, 2))
            good = (cand[:, 0] > 0) & (cand[:, 0] < L) & (cand[:, 1] > 0) & (cand[:, 1] < L)
            x = np.concatenate([x, cand[good, 0]]); y = np.concatenate([y, cand[good, 1]])
        xs.append(x[:m]); ys.append(y[:m])
    x = np.concatenate(xs); y = np.concatenate(ys)
    vpref = _vpref(prng, n_peds)
    inflow_cell = np.arange(nx, dtype=np.int32)
    return Scenario(
        name="config5_throughput_stress", nx=nx, ny=ny, dx=dx, dy=dx, real_bits=32,
        z=z.reshape(-1), manning=np.full(nx * ny, 0.02, np.float32),
        mask=np.zeros(nx * ny, np.uint8), h0=h0.reshape(-1),
        u0=None, v0=None,
        px=_keep_inside(x, nx, dx, 32), py=_keep_inside(y, ny, dx, 32),
        pvx=np.zeros(n_peds, np.float32), pvy=np.zeros(n_peds, np.float32), pvpref=_as_real(vpref, 32),
        prole=np.zeros(n_peds, np.uint8), nav_dir=nav[None, :].copy(), exit_cells=exits,
        inflow_cell=inflow_cell, inflow_side=np.full(nx, SIDE_S, np.uint8),
        hydro_t=np.array([0.0, 60.0, 1e9]), hydro_q=np.array([0.0, 2000.0 * n / 8192, 2000.0 * n / 8192]),
        steps=steps)


# --------------------------------------------------------------------------- mid-run states

def synthetic_flow(sc: Scenario, seed: int, speed: float = 1.5, ped_speed: float = 1.0) -> dict:
    """A seeded state that looks like the middle of a run, for single-step parity at sizes the
    oracle cannot evolve itself: the scenario's initial depth modulated by +-20 % smooth noise,
    smooth velocities in [-speed, speed] m/s (conserved variables q = h * u rounded to storage
    precision), pedestrians with uniform random velocities of up to ped_speed.  Input generation
    only; nothing here is the method's arithmetic."""
    rng = np.random.Generator(np.random.PCG64(seed))
    ny, nx = sc.ny, sc.nx
    sp = [max(2, nx // 32), max(2, nx // 128)]

    def smooth():
        return (_value_noise(rng, ny, nx, sp, [1.0, 0.5]).astype(np.float32) - np.float32(0.5)) * np.float32(2.0)

    h = sc.h0.reshape(ny, nx).astype(np.float32) * (np.float32(1.0) + np.float32(0.2) * smooth())
    h = np.where(sc.mask.reshape(ny, nx) != 0, np.float32(0.0), h).astype(np.float32)
    qx = (h * (np.float32(speed) * smooth())).astype(np.float32)
    qy = (h * (np.float32(speed) * smooth())).astype(np.float32)
    n = sc.n_peds
    ang = rng.random(n) * 2.0 * np.pi
    mag = rng.random(n) * ped_speed
    real = sc.real
    return dict(h=h.reshape(-1).astype(real), qx=qx.reshape(-1).astype(real), qy=qy.reshape(-1).astype(real),
                pvx=(mag * np.cos(ang)).astype(real), pvy=(mag * np.sin(ang)).astype(real))


def window(sc: Scenario, state: dict, i0: int, j0: int, w: int, hgt: int):
    """The sub-box [i0, i0+w) x [j0, j0+hgt) of a scenario and of a state of it as a Scenario of
    its own (closed walls; inflow faces kept where the window touches the inflow edge, the
    hydrograph scaled so that the discharge per unit width is unchanged; pedestrians inside the
    window, coordinates shifted by a whole number of cells).  Returns (scenario, state, ids):
    ids = indices of the window's pedestrians in the parent.  One first-order step of the parent
    restricted to the window's interior depends on nothing outside the window."""
    nx, ny = sc.nx, sc.ny
    sl = np.s_[j0:j0 + hgt, i0:i0 + w]

    def cut(a, dtype=None):
        a = np.asarray(a).reshape(ny, nx)[sl].reshape(-1)
        return np.ascontiguousarray(a if dtype is None else a.astype(dtype))

    ci, cj = (sc.px / sc.dx).astype(np.int64), (sc.py / sc.dy).astype(np.int64)
    ids = np.flatnonzero((ci >= i0) & (ci < i0 + w) & (cj >= j0) & (cj < j0 + hgt))
    real = sc.real
    ox, oy = real(i0) * real(sc.dx), real(j0) * real(sc.dy)
    keep = [k for k, c in enumerate(sc.exit_cells)
            if i0 <= c % nx < i0 + w and j0 <= c // nx < j0 + hgt]
    exits = np.array([(sc.exit_cells[k] // nx - j0) * w + (sc.exit_cells[k] % nx - i0) for k in keep], np.int32)
    fi, fj = sc.inflow_cell % nx, sc.inflow_cell // nx
    fk = np.flatnonzero((fi >= i0) & (fi < i0 + w) & (fj >= j0) & (fj < j0 + hgt))
    nav = np.stack([cut(sc.nav_dir[t]) for t in range(sc.nav_dir.shape[0])])
    scale = fk.size / max(sc.inflow_cell.size, 1)
    sub = Scenario(
        name=f"{sc.name}[{i0}:{i0 + w},{j0}:{j0 + hgt}]", nx=w, ny=hgt, dx=sc.dx, dy=sc.dy, real_bits=sc.real_bits,
        z=cut(sc.z), manning=cut(sc.manning), mask=cut(sc.mask), h0=cut(state["h"]), u0=None, v0=None,
        px=(sc.px[ids] - ox).astype(real), py=(sc.py[ids] - oy).astype(real),
        pvx=np.ascontiguousarray(state["pvx"][ids]), pvy=np.ascontiguousarray(state["pvy"][ids]),
        pvpref=np.ascontiguousarray(sc.pvpref[ids]), prole=np.ascontiguousarray(sc.prole[ids]),
        nav_dir=nav, exit_cells=exits,
        g=sc.g, cfl=sc.cfl, dt_max=sc.dt_max, h_dry=sc.h_dry, couple_roughness=sc.couple_roughness, n_cap=sc.n_cap,
        inflow_cell=((fj[fk] - j0) * w + (fi[fk] - i0)).astype(np.int32), inflow_side=np.ascontiguousarray(sc.inflow_side[fk]),
        hydro_t=sc.hydro_t.copy(), hydro_q=sc.hydro_q * scale,
        hr_edges=sc.hr_edges, speed_wet=sc.speed_wet, tau=sc.tau, A_s=sc.A_s, B_s=sc.B_s, radius=sc.radius,
        R_int=sc.R_int, vmax_factor=sc.vmax_factor, arrive_cells=sc.arrive_cells)
    sub_state = dict(h=cut(state["h"]), qx=cut(state["qx"]), qy=cut(state["qy"]))
    return sub, sub_state, ids


CONFIGS = {
    1: tiny_dam_break,
    2: shopping_centre,
    3: pre_flood_intervention,
    4: scaled_flood,
    5: throughput_stress,
}


def make(config: int, **kw) -> Scenario:
    """Scenario for BASELINE.json configs[config-1]; keyword arguments shrink it for tests."""
    return CONFIGS[config](**kw)
