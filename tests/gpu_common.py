"""Helpers for the GPU parity tests: put the oracle and the CUDA path into the same state."""
from __future__ import annotations

import numpy as np

import oracle
from paper_1908_05232_b200 import binding


def rounded(a, real):
    return np.asarray(a, np.float64).astype(real).astype(np.float64)


def make_pair(sc, evolve=0, variant=None):
    """Oracle evolved `evolve` steps, then that state (rounded to the storage precision) injected
    into both sides so that they start one step from IDENTICAL inputs."""
    o = oracle.Oracle(sc)
    g = binding.Sim(sc)
    if variant is not None:
        g.set_flood_variant(variant)
    if evolve:
        o.step(evolve)
        sync(o, g, sc)
    return o, g


def sync(o, g, sc):
    real = np.float64 if sc.real_bits == 64 else np.float32
    c = o.read_conserved(); z = o.read_flood()["z"]; p = o.read_peds(); st = o.stats()
    h, qx, qy, zz = (rounded(a, real) for a in (c["h"], c["qx"], c["qy"], z))
    o.write_flood(h, qx, qy, zz)
    g.write_flood(h, qx, qy, zz)
    if sc.n_peds:
        x, y, vx, vy, tm = (rounded(p[k], real) for k in ("x", "y", "vx", "vy", "timer"))
        o.write_peds(x, y, vx, vy, p["fsm"], p["active"], tm)
        g.write_peds(x, y, vx, vy, p["fsm"], p["active"], tm)
    dt = float(rounded(st["dt"], real))
    o.set_time(st["t"], dt); g.set_time(st["t"], dt)
    g.set_barrier(st["cursor"], st["layer"], st["bags"], st["barrier_complete"])
    return st


def mixed(a, b):
    """max |a-b| / max(|b|_inf, tiny) -- the mixed norm of DESIGN.md C39."""
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    if b.size == 0:
        return 0.0
    return float(np.max(np.abs(a - b))) / max(float(np.max(np.abs(b))), 1e-300)
