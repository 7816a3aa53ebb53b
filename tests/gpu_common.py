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


def force_magnitude_sum(x, y, sc):
    """S_i = sum over partners within R_int of |f_ij| = A_s exp((2r - d)/B_s) (C24): the
    scale that the rounding of the social-force sum is relative to.  Agents in a dense crowd sit
    between forces of thousands of m/s2 that nearly cancel, so their new velocity carries an
    absolute error of about eps * dt * S_i whatever the order of summation."""
    from scipy.spatial import cKDTree
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64)
    S_i = np.zeros(x.shape[0])
    if x.shape[0] > 1:
        pr = cKDTree(np.c_[x, y]).query_pairs(sc.R_int, output_type="ndarray")
        d = np.hypot(x[pr[:, 0]] - x[pr[:, 1]], y[pr[:, 0]] - y[pr[:, 1]])
        f = sc.A_s * np.exp((2.0 * sc.radius - d) / sc.B_s)
        np.add.at(S_i, pr[:, 0], f); np.add.at(S_i, pr[:, 1], f)
    return S_i


def force_sum_tolerance(x, y, sc, dt):
    """absolute tolerance on a new velocity component from the conditioning of the force sum: each
    term carries <= 16 ulp (ex2/rsqrt.approx and the rounding of the exponent argument d/B_s <= 12.5
    in fp32; a few ulp in fp64), the sum is multiplied by dt."""
    eps = 2.0 ** -23 if sc.real_bits == 32 else 2.0 ** -52
    return 16.0 * eps * dt * force_magnitude_sum(x, y, sc)
