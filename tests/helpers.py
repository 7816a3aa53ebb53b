"""Small scenario builders and comparison utilities shared by the tests (no method arithmetic)."""
from __future__ import annotations

import os

import numpy as np

from paper_1908_05232_b200.scenarios import Scenario, nav_field, DIR_NONE

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden_rows(fname, kind):
    rows = []
    with open(os.path.join(GOLDEN, fname)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line and line.split()[0] == kind:
                rows.append([float(v) for v in line.split()[1:]])
    return rows


def box(nx, ny, dx=1.0, real_bits=64, z=None, h0=None, u0=None, v0=None, manning=0.0, mask=None,
        peds=None, exit_cell=None, **kw) -> Scenario:
    """Closed nx x ny box; peds = dict(x, y[, vx, vy, vpref, role])."""
    nc = nx * ny
    real = np.float64 if real_bits == 64 else np.float32
    def arr(a, fill):
        if a is None:
            return np.full(nc, fill, real)
        a = np.asarray(a, real)
        return np.full(nc, a, real) if a.ndim == 0 else np.ascontiguousarray(a.reshape(-1))

    mask = np.zeros(nc, np.uint8) if mask is None else np.ascontiguousarray(mask, np.uint8).reshape(-1)
    peds = peds or {}
    n_p = len(peds.get("x", []))
    pa = lambda k, fill: np.ascontiguousarray(peds.get(k, np.full(n_p, fill)), real)
    if exit_cell is None:
        nav = np.full((1, nc), DIR_NONE, np.uint8)
        exits = np.zeros(0, np.int32)
    else:
        nav1, _ = nav_field(mask.reshape(ny, nx), [exit_cell])
        nav = nav1[None, :]
        exits = np.array([exit_cell], np.int32)
    base = dict(
        name="box", nx=nx, ny=ny, dx=dx, dy=dx, real_bits=real_bits,
        z=arr(z, 0.0), manning=arr(manning, 0.0), mask=mask, h0=arr(h0, 0.0),
        u0=None if u0 is None else arr(u0, 0.0), v0=None if v0 is None else arr(v0, 0.0),
        px=pa("x", 0.0), py=pa("y", 0.0), pvx=pa("vx", 0.0), pvy=pa("vy", 0.0),
        pvpref=pa("vpref", 1.4), prole=np.ascontiguousarray(peds.get("role", np.zeros(n_p)), np.uint8),
        nav_dir=nav, exit_cells=exits, dt_max=1.0)
    base.update(kw)
    return Scenario(**base)


def mixed_err(a, b):
    """max |a-b| / max(|b|_inf, tiny): the mixed norm of SURVEY C39 (a scalar)."""
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    scale = max(float(np.max(np.abs(b))) if b.size else 0.0, 1e-300)
    return float(np.max(np.abs(a - b))) / scale if b.size else 0.0


def doors_box(n=24, slots=64, rate=0.5, target=1000, n_doors=3, **kw):
    """dry closed box, dt = dt_max = 0.25 s exactly, doors on the west wall, exit at the east wall"""
    mask = np.zeros((n, n), np.uint8)
    doors = np.array([(3 + 6 * d) * n + 0 for d in range(n_doors)], np.int32)
    exit_cell = (n // 2) * n + n - 1
    navs = [nav_field(mask, [exit_cell])[0]] + [nav_field(mask, [int(c)])[0] for c in doors]
    sc = box(n, n, dx=1.0, h0=0.0, manning=0.0, dt_max=0.25,
             peds=dict(x=np.full(slots, 12.5), y=np.full(slots, 12.5)), **kw)
    sc.nav_dir = np.stack(navs); sc.exit_cells = np.array([exit_cell], np.int32); sc.exit_target = 0
    sc.door_cells = doors; sc.door_target = np.arange(1, n_doors + 1, dtype=np.int32)
    sc.spawn_rate = rate; sc.target_population = target; sc.spawn_seed = 1234
    sc.spawn_vpref_lo, sc.spawn_vpref_hi = 1.0, 1.4
    sc.pactive0 = np.zeros(slots, np.uint8)
    return sc


def compass_scene(code, real_bits=64):
    """one agent in the middle of a dry 64 x 64 hall whose navigation field holds `code` in every cell"""
    n = 64
    sc = box(n, n, dx=1.0, real_bits=real_bits, peds=dict(x=[32.5], y=[32.5], vpref=[1.3]), exit_cell=0, dt_max=0.2)
    sc.nav_dir = np.full_like(sc.nav_dir, code)
    return sc
