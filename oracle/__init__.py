"""CPU oracle of the coupled flood-pedestrian step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper around `floodped_oracle.c` (plain C99, fp64, single thread).  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import
this package.  It imports nothing from `paper_1908_05232_b200`; scenarios are duck-typed.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "floodped_oracle.c")
_HDR = os.path.join(_HERE, "floodped_oracle.h")
_LIB = os.path.join(_HERE, "liboracle.so")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_bp = C.POINTER(C.c_ubyte)


class OrcConfig(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("dx", C.c_double), ("dy", C.c_double),
        ("real_bits", C.c_int),
        ("z", _dp), ("manning", _dp), ("mask", _bp), ("h0", _dp), ("u0", _dp), ("v0", _dp),
        ("n_peds", C.c_int),
        ("px", _dp), ("py", _dp), ("pvx", _dp), ("pvy", _dp), ("pvpref", _dp), ("prole", _bp),
        ("g", C.c_double), ("cfl", C.c_double), ("dt_max", C.c_double), ("h_dry", C.c_double),
        ("couple_roughness", C.c_int), ("n_cap", C.c_int),
        ("n_inflow", C.c_int), ("inflow_cell", _ip), ("inflow_side", _bp),
        ("n_hydro", C.c_int), ("hydro_t", _dp), ("hydro_q", _dp),
        ("hr_edges", C.c_double * 4), ("speed_wet", C.c_double * 4),
        ("tau", C.c_double), ("A_s", C.c_double), ("B_s", C.c_double), ("radius", C.c_double),
        ("R_int", C.c_double), ("vmax_factor", C.c_double),
        ("n_targets", C.c_int), ("nav_dir", _bp),
        ("exit_target", C.c_int), ("storage_target", C.c_int), ("drop_target", C.c_int),
        ("n_exit_cells", C.c_int), ("exit_cells", _ip),
        ("storage_cell", C.c_int), ("drop_cell", C.c_int), ("arrive_cells", C.c_int),
        ("n_line", C.c_int), ("line_cells", _ip),
        ("bags_per_cell_layer", C.c_int), ("n_layers", C.c_int),
        ("layer_thickness", C.c_double), ("t_pick", C.c_double), ("t_drop", C.c_double),
        ("t_end", C.c_double),
        ("flood_order", C.c_int),
        ("open_sides", C.c_int), ("n_doors", C.c_int), ("door_cells", _ip), ("door_target", _ip),
        ("spawn_rate", C.c_double), ("target_population", C.c_int), ("spawn_seed", C.c_ulonglong),
        ("spawn_vpref_lo", C.c_double), ("spawn_vpref_hi", C.c_double), ("pactive0", _bp),
    ]


class OrcStats(C.Structure):
    _fields_ = [
        ("t", C.c_double), ("dt", C.c_double), ("step", C.c_longlong),
        ("volume", C.c_double), ("max_h", C.c_double), ("max_hr", C.c_double),
        ("hist", C.c_longlong * 6), ("neg_depth_clamps", C.c_longlong),
        ("clamped_volume", C.c_double),
        ("cursor", C.c_int), ("layer", C.c_int), ("bags", C.c_int), ("barrier_complete", C.c_int),
        ("deposits", C.c_longlong),
        ("outflow_volume", C.c_double), ("spawned", C.c_longlong), ("triggered", C.c_int),
    ]


def build(force: bool = False) -> str:
    """Compile liboracle.so with gcc (-O2, no fast-math, no FMA contraction)."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", "-std=c99", "-O2", "-fno-fast-math", "-ffp-contract=off", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        d = C.c_double
        L.orc_riemann_flux.argtypes = [d] * 7 + [_dp]
        L.orc_riemann_flux.restype = None
        L.orc_face.argtypes = [d] * 9 + [_dp, _dp, _dp]
        L.orc_face.restype = None
        L.orc_minmod.argtypes = [d, d]
        L.orc_minmod.restype = d
        L.orc_friction.argtypes = [d, d, d, d, d, _dp, _dp]
        L.orc_friction.restype = None
        L.orc_cell_dt.argtypes = [d] * 7
        L.orc_cell_dt.restype = d
        L.orc_hazard_rate.argtypes = [C.c_int, d, d, d]
        L.orc_hazard_rate.restype = d
        L.orc_risk_state.argtypes = [C.c_int, d, d, d, _dp]
        L.orc_risk_state.restype = C.c_int
        L.orc_roughness.argtypes = [d, C.c_int, C.c_int]
        L.orc_roughness.restype = d
        L.orc_hydrograph.argtypes = [C.c_int, _dp, _dp, d]
        L.orc_hydrograph.restype = d
        L.orc_social_bruteforce.argtypes = [C.c_int, _dp, _dp, _bp, d, d, d, d, C.c_int, _dp, _dp]
        L.orc_social_bruteforce.restype = None
        L.orc_philox4x32.argtypes = [C.POINTER(C.c_uint), C.POINTER(C.c_uint), C.POINTER(C.c_uint)]
        L.orc_philox4x32.restype = None
        L.orc_create.argtypes = [C.POINTER(OrcConfig)]
        L.orc_create.restype = C.c_void_p
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_step.argtypes = [C.c_void_p, C.c_longlong]
        L.orc_step.restype = C.c_int
        L.orc_get_stats.argtypes = [C.c_void_p, C.POINTER(OrcStats)]
        L.orc_get_stats.restype = None
        L.orc_read_flood.argtypes = [C.c_void_p] + [_dp] * 5
        L.orc_read_flood.restype = None
        L.orc_read_conserved.argtypes = [C.c_void_p] + [_dp] * 3
        L.orc_read_conserved.restype = None
        L.orc_read_occupancy.argtypes = [C.c_void_p, _ip]
        L.orc_read_occupancy.restype = None
        L.orc_read_peds.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _bp, _bp, _bp, _ip, _dp]
        L.orc_read_peds.restype = None
        L.orc_social_celllist.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_social_celllist.restype = None
        L.orc_binning.argtypes = [C.c_void_p, _ip, _ip, _ip, _ip, _ip, _ip]
        L.orc_binning.restype = C.c_int
        L.orc_write_flood.argtypes = [C.c_void_p] + [_dp] * 4
        L.orc_write_flood.restype = None
        L.orc_write_peds.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _bp, _bp, _dp]
        L.orc_write_peds.restype = None
        L.orc_set_time.argtypes = [C.c_void_p, d, d]
        L.orc_set_time.restype = None
        L.orc_set_barrier.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
        L.orc_set_barrier.restype = None
        _lib = L
    return _lib


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a, typ):
    return None if a is None else a.ctypes.data_as(typ)


# ---- building blocks (thin wrappers) ----------------------------------------------------------

def riemann_flux(g, hL, unL, utL, hR, unR, utR):
    out = (C.c_double * 3)()
    lib().orc_riemann_flux(g, hL, unL, utL, hR, unR, utR, out)
    return np.array(out[:])


def face(g, hi, uni, uti, zi, hk, unk, utk, zk):
    out = (C.c_double * 3)()
    fi, fk = C.c_double(), C.c_double()
    lib().orc_face(g, hi, uni, uti, zi, hk, unk, utk, zk, out, C.byref(fi), C.byref(fk))
    return np.array(out[:]), fi.value, fk.value


def minmod(a, b):
    return lib().orc_minmod(a, b)


def philox4x32(counter, key):
    """Philox4x32-10 of the oracle (spawning, D5): 4 + 2 uint32 in, 4 uint32 out."""
    c = (C.c_uint * 4)(*[int(v) & 0xffffffff for v in counter])
    k = (C.c_uint * 2)(*[int(v) & 0xffffffff for v in key])
    out = (C.c_uint * 4)()
    lib().orc_philox4x32(c, k, out)
    return [int(v) for v in out]


def friction(g, n, dt, h_dry, h, qx, qy):
    a, b = C.c_double(qx), C.c_double(qy)
    lib().orc_friction(g, n, dt, h_dry, h, C.byref(a), C.byref(b))
    return a.value, b.value


def cell_dt(g, cfl, dx, dy, h, u, v):
    return lib().orc_cell_dt(g, cfl, dx, dy, h, u, v)


def hazard_rate(h, u, v, real_bits=64):
    return lib().orc_hazard_rate(real_bits, h, u, v)


def risk_state(h, hr, h_dry=1e-3, edges=(0.75, 1.5, 2.5, 20.0), real_bits=64):
    e = (C.c_double * 4)(*edges)
    return lib().orc_risk_state(real_bits, h, hr, h_dry, e)


def roughness(n0, Np, cap=20):
    return lib().orc_roughness(n0, Np, cap)


def hydrograph(t, q, time):
    t = _f64(t); q = _f64(q)
    return lib().orc_hydrograph(len(t), _ptr(t, _dp), _ptr(q, _dp), time)


def social_bruteforce(x, y, active, A_s, B_s, radius, R_int):
    x = _f64(x); y = _f64(y)
    act = np.ascontiguousarray(active, dtype=np.uint8)
    n = len(x)
    ax = np.zeros(n); ay = np.zeros(n)
    a, b = C.c_double(), C.c_double()
    for i in range(n):
        if not act[i]:
            continue
        lib().orc_social_bruteforce(n, _ptr(x, _dp), _ptr(y, _dp), _ptr(act, _bp),
                                    A_s, B_s, radius, R_int, i, C.byref(a), C.byref(b))
        ax[i], ay[i] = a.value, b.value
    return ax, ay


# ---- the simulator ----------------------------------------------------------------------------

class Oracle:
    """fp64 single-threaded CPU simulator built from a Scenario-like object."""

    def __init__(self, sc):
        L = lib()
        self._keep = []
        self.nx, self.ny, self.n_peds = int(sc.nx), int(sc.ny), int(sc.px.shape[0])
        self.ncell = self.nx * self.ny
        cfg = OrcConfig()

        def keep(a, dtype):
            if a is None:
                return None
            a = np.ascontiguousarray(a, dtype=dtype)
            self._keep.append(a)
            return a

        def setp(name, a, dtype, typ):
            a = keep(a, dtype)
            setattr(cfg, name, _ptr(a, typ) if a is not None and a.size else C.cast(None, typ))
            return a

        cfg.nx, cfg.ny, cfg.dx, cfg.dy, cfg.real_bits = sc.nx, sc.ny, sc.dx, sc.dy, sc.real_bits
        setp("z", sc.z, np.float64, _dp); setp("manning", sc.manning, np.float64, _dp)
        setp("mask", sc.mask, np.uint8, _bp); setp("h0", sc.h0, np.float64, _dp)
        setp("u0", sc.u0, np.float64, _dp); setp("v0", sc.v0, np.float64, _dp)
        cfg.n_peds = self.n_peds
        setp("px", sc.px, np.float64, _dp); setp("py", sc.py, np.float64, _dp)
        setp("pvx", sc.pvx, np.float64, _dp); setp("pvy", sc.pvy, np.float64, _dp)
        setp("pvpref", sc.pvpref, np.float64, _dp); setp("prole", sc.prole, np.uint8, _bp)
        cfg.g, cfg.cfl, cfg.dt_max, cfg.h_dry = sc.g, sc.cfl, sc.dt_max, sc.h_dry
        cfg.couple_roughness, cfg.n_cap = sc.couple_roughness, sc.n_cap
        cfg.n_inflow = int(len(sc.inflow_cell))
        setp("inflow_cell", sc.inflow_cell, np.int32, _ip); setp("inflow_side", sc.inflow_side, np.uint8, _bp)
        cfg.n_hydro = int(len(sc.hydro_t))
        setp("hydro_t", sc.hydro_t, np.float64, _dp); setp("hydro_q", sc.hydro_q, np.float64, _dp)
        cfg.hr_edges = (C.c_double * 4)(*sc.hr_edges)
        cfg.speed_wet = (C.c_double * 4)(*sc.speed_wet)
        cfg.tau, cfg.A_s, cfg.B_s, cfg.radius = sc.tau, sc.A_s, sc.B_s, sc.radius
        cfg.R_int, cfg.vmax_factor = sc.R_int, sc.vmax_factor
        nav = np.ascontiguousarray(sc.nav_dir, dtype=np.uint8).reshape(-1, self.ncell)
        cfg.n_targets = nav.shape[0]
        setp("nav_dir", nav, np.uint8, _bp)
        cfg.exit_target, cfg.storage_target, cfg.drop_target = sc.exit_target, sc.storage_target, sc.drop_target
        cfg.n_exit_cells = int(len(sc.exit_cells))
        setp("exit_cells", sc.exit_cells, np.int32, _ip)
        cfg.storage_cell, cfg.drop_cell, cfg.arrive_cells = sc.storage_cell, sc.drop_cell, sc.arrive_cells
        cfg.n_line = int(len(sc.line_cells))
        setp("line_cells", sc.line_cells, np.int32, _ip)
        cfg.bags_per_cell_layer, cfg.n_layers = sc.bags_per_cell_layer, sc.n_layers
        cfg.layer_thickness, cfg.t_pick, cfg.t_drop = sc.layer_thickness, sc.t_pick, sc.t_drop
        cfg.t_end = sc.t_end
        cfg.flood_order = int(getattr(sc, "flood_order", 1))
        cfg.open_sides = int(getattr(sc, "open_sides", 0))
        doors = np.asarray(getattr(sc, "door_cells", np.zeros(0, np.int32)), np.int32)
        cfg.n_doors = int(len(doors))
        setp("door_cells", doors, np.int32, _ip)
        setp("door_target", getattr(sc, "door_target", np.zeros(0, np.int32)), np.int32, _ip)
        cfg.spawn_rate = float(getattr(sc, "spawn_rate", 0.0))
        cfg.target_population = int(getattr(sc, "target_population", 0))
        cfg.spawn_seed = int(getattr(sc, "spawn_seed", 0))
        cfg.spawn_vpref_lo = float(getattr(sc, "spawn_vpref_lo", 1.0)); cfg.spawn_vpref_hi = float(getattr(sc, "spawn_vpref_hi", 1.4))
        setp("pactive0", getattr(sc, "pactive0", None), np.uint8, _bp)
        self._h = L.orc_create(C.byref(cfg))
        if not self._h:
            raise ValueError("orc_create failed")
        self._keep = []                      # the C side copied everything

    def close(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    __del__ = close

    def step(self, n=1):
        lib().orc_step(self._h, int(n))

    def stats(self) -> dict:
        st = OrcStats()
        lib().orc_get_stats(self._h, C.byref(st))
        d = {k: getattr(st, k) for k, _ in OrcStats._fields_ if k != "hist"}
        d["hist"] = list(st.hist)
        return d

    def read_flood(self):
        out = {k: np.empty(self.ncell) for k in ("h", "u", "v", "z", "hr")}
        lib().orc_read_flood(self._h, *[_ptr(out[k], _dp) for k in ("h", "u", "v", "z", "hr")])
        return out

    def read_conserved(self):
        out = {k: np.empty(self.ncell) for k in ("h", "qx", "qy")}
        lib().orc_read_conserved(self._h, *[_ptr(out[k], _dp) for k in ("h", "qx", "qy")])
        return out

    def read_occupancy(self):
        a = np.empty(self.ncell, np.int32)
        lib().orc_read_occupancy(self._h, _ptr(a, _ip))
        return a

    def read_peds(self):
        n = self.n_peds
        out = {k: np.empty(n) for k in ("x", "y", "vx", "vy", "timer")}
        out.update({k: np.empty(n, np.uint8) for k in ("state", "fsm", "active")})
        out["cell"] = np.empty(n, np.int32)
        lib().orc_read_peds(self._h, _ptr(out["x"], _dp), _ptr(out["y"], _dp), _ptr(out["vx"], _dp),
                            _ptr(out["vy"], _dp), _ptr(out["state"], _bp), _ptr(out["fsm"], _bp),
                            _ptr(out["active"], _bp), _ptr(out["cell"], _ip), _ptr(out["timer"], _dp))
        return out

    def social_celllist(self):
        ax = np.empty(self.n_peds); ay = np.empty(self.n_peds)
        lib().orc_social_celllist(self._h, _ptr(ax, _dp), _ptr(ay, _dp))
        return ax, ay

    def binning(self):
        nbx, nby, k = C.c_int(), C.c_int(), C.c_int()
        nb = lib().orc_binning(self._h, None, None, None, C.byref(nbx), C.byref(nby), C.byref(k))
        key = np.empty(self.n_peds, np.int32)
        count = np.empty(nb, np.int32)
        start = np.empty(nb + 1, np.int32)
        lib().orc_binning(self._h, _ptr(key, _ip), _ptr(count, _ip), _ptr(start, _ip), None, None, None)
        return {"key": key, "count": count, "start": start, "nbx": nbx.value, "nby": nby.value, "k": k.value}

    def write_flood(self, h=None, qx=None, qy=None, z=None):
        a = [_f64(v) for v in (h, qx, qy, z)]
        lib().orc_write_flood(self._h, *[_ptr(v, _dp) for v in a])

    def write_peds(self, x=None, y=None, vx=None, vy=None, fsm=None, active=None, timer=None):
        f = [_f64(v) for v in (x, y, vx, vy)]
        b = [None if v is None else np.ascontiguousarray(v, dtype=np.uint8) for v in (fsm, active)]
        t = _f64(timer)
        lib().orc_write_peds(self._h, *[_ptr(v, _dp) for v in f], *[_ptr(v, _bp) for v in b], _ptr(t, _dp))

    def set_time(self, t, dt):
        lib().orc_set_time(self._h, float(t), float(dt))

    def set_barrier(self, cursor, layer, bags, complete):
        lib().orc_set_barrier(self._h, int(cursor), int(layer), int(bags), int(complete))
