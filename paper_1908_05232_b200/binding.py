"""Thin ctypes binding over the C ABI of libfloodped.so (include/floodped.h).

Argument marshalling only: every step of the path runs in the CUDA kernels.  PyTorch supplies
the device workspace (`torch.empty`) and the stream; there is no CPU fallback -- if the library
or a CUDA device is missing, construction raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfloodped.so")

SIM_OK, SIM_EINVAL, SIM_ENOMEM, SIM_ECUDA, SIM_ENOTFINITE = 0, -1, -2, -3, -4

EXPORTS = [
    "sim_workspace_bytes", "sim_create", "sim_step", "sim_step_profiled", "sim_read_flood", "sim_read_conserved",
    "sim_read_occupancy", "sim_read_peds", "sim_get_stats", "sim_bin_peds", "sim_write_flood",
    "sim_write_peds", "sim_set_time", "sim_set_barrier", "sim_test_philox", "sim_set_flood_variant", "sim_get_flood_variant", "sim_set_march_rows", "sim_set_overlap", "sim_set_dry_skip", "sim_set_deterministic",
    "sim_kernels_per_step", "sim_slab_link", "sim_slab_step", "sim_slab_describe", "sim_slab_attach", "sim_slab_enqueue", "sim_cfl_dt_static", "sim_last_error", "sim_destroy",
]

SIM_CFL_STATIC_MAX_CELLS = 1 << 28

_vp = C.c_void_p
_u8p = C.POINTER(C.c_uint8)
_i32p = C.POINTER(C.c_int32)
_f64p = C.POINTER(C.c_double)


class SimGrid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("dx", C.c_double), ("dy", C.c_double),
                ("real_bits", C.c_int32), ("slab_j0", C.c_int32), ("slab_ny_global", C.c_int32)]


class SimTopo(C.Structure):
    _fields_ = [("z", _vp), ("mask", _u8p), ("h0", _vp), ("u0", _vp), ("v0", _vp)]


class SimPeds(C.Structure):
    _fields_ = [("n", C.c_int32), ("x", _vp), ("y", _vp), ("vx", _vp), ("vy", _vp), ("v_pref", _vp),
                ("role", _u8p), ("active", _u8p)]


class SimParams(C.Structure):
    _fields_ = [
        ("g", C.c_double), ("cfl", C.c_double), ("dt_max", C.c_double), ("h_dry", C.c_double),
        ("couple_roughness", C.c_int32), ("n_cap", C.c_int32),
        ("n_inflow_faces", C.c_int32), ("inflow_cell", _i32p), ("inflow_side", _u8p),
        ("n_hydro", C.c_int32), ("hydro_t", _f64p), ("hydro_q", _f64p),
        ("hr_edges", C.c_double * 4), ("speed_wet", C.c_double * 4),
        ("tau", C.c_double), ("A_s", C.c_double), ("B_s", C.c_double), ("radius", C.c_double),
        ("R_int", C.c_double), ("vmax_factor", C.c_double),
        ("n_targets", C.c_int32), ("nav_dir", _u8p),
        ("exit_target", C.c_int32), ("storage_target", C.c_int32), ("drop_target", C.c_int32),
        ("n_exit_cells", C.c_int32), ("exit_cells", _i32p),
        ("storage_cell", C.c_int32), ("drop_cell", C.c_int32), ("arrive_cells", C.c_int32),
        ("n_line", C.c_int32), ("line_cells", _i32p),
        ("bags_per_cell_layer", C.c_int32), ("n_layers", C.c_int32),
        ("layer_thickness", C.c_double), ("t_pick", C.c_double), ("t_drop", C.c_double),
        ("t_end", C.c_double),
        ("flood_order", C.c_int32),
        ("open_sides", C.c_int32), ("n_doors", C.c_int32), ("door_cells", _i32p), ("door_target", _i32p),
        ("spawn_rate", C.c_double), ("target_population", C.c_int32), ("spawn_seed", C.c_uint64),
        ("spawn_vpref_lo", C.c_double), ("spawn_vpref_hi", C.c_double),
    ]


class SlabDesc(C.Structure):
    _fields_ = [("j0", C.c_int32), ("ny", C.c_int32),
                ("h", C.c_uint64 * 2), ("qx", C.c_uint64 * 2), ("qy", C.c_uint64 * 2),
                ("zs", C.c_uint64), ("occ", C.c_uint64), ("ctl", C.c_uint64), ("lam_bits", C.c_uint64),
                ("workspace", C.c_uint64), ("workspace_bytes", C.c_uint64)]

    ADDRS = ("zs", "occ", "ctl", "lam_bits")

    def to_dict(self):
        d = {k: int(getattr(self, k)) for k in ("j0", "ny", "workspace", "workspace_bytes") + self.ADDRS}
        d.update({k: [int(v) for v in getattr(self, k)] for k in ("h", "qx", "qy")})
        return d

    @classmethod
    def rebased(cls, d, new_base):
        """the description `d` (a dict made by to_dict in the owner's process) with every address moved
        from the owner's workspace base to `new_base`, where this process has that workspace mapped"""
        o, delta = cls(), int(new_base) - int(d["workspace"])
        o.j0, o.ny, o.workspace, o.workspace_bytes = d["j0"], d["ny"], int(new_base), d["workspace_bytes"]
        for k in cls.ADDRS:
            setattr(o, k, d[k] + delta)
        for k in ("h", "qx", "qy"):
            setattr(o, k, (C.c_uint64 * 2)(*[v + delta for v in d[k]]))
        return o


class SimStats(C.Structure):
    _fields_ = [
        ("t", C.c_double), ("dt", C.c_double), ("step", C.c_int64),
        ("volume", C.c_double), ("max_h", C.c_double), ("max_hr", C.c_double),
        ("hist", C.c_int64 * 6), ("neg_depth_clamps", C.c_int64), ("clamped_volume", C.c_double),
        ("cursor", C.c_int32), ("layer", C.c_int32), ("bags", C.c_int32), ("barrier_complete", C.c_int32),
        ("deposits", C.c_int64),
        ("outflow_volume", C.c_double), ("spawned", C.c_int64), ("triggered", C.c_int32),
    ]


class FloodpedError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libfloodped error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen libfloodped.so and declare the prototypes.  Raises if the library is missing:
    there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(
            f"{path} is missing: build it with `python -m paper_1908_05232_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(path)
    L.sim_workspace_bytes.argtypes = [C.POINTER(SimGrid), C.c_int32, C.POINTER(SimParams), C.POINTER(C.c_size_t)]
    L.sim_create.argtypes = [C.POINTER(SimGrid), C.POINTER(SimTopo), _vp, C.POINTER(SimPeds),
                             C.POINTER(SimParams), _vp, _vp, C.POINTER(_vp)]
    L.sim_step.argtypes = [_vp, C.c_int64]
    L.sim_step_profiled.argtypes = [_vp, C.c_int64, _f64p]
    L.sim_read_flood.argtypes = [_vp] * 6
    L.sim_read_conserved.argtypes = [_vp] * 4
    L.sim_read_occupancy.argtypes = [_vp, _vp]
    L.sim_read_peds.argtypes = [_vp] * 10
    L.sim_get_stats.argtypes = [_vp, C.POINTER(SimStats)]
    L.sim_bin_peds.argtypes = [_vp, _vp, _vp, _vp, _i32p, _i32p, _i32p]
    L.sim_write_flood.argtypes = [_vp] * 5
    L.sim_write_peds.argtypes = [_vp] * 8
    L.sim_set_time.argtypes = [_vp, C.c_double, C.c_double]
    L.sim_set_barrier.argtypes = [_vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32]
    L.sim_test_philox.argtypes = [_vp, _vp, _vp, C.c_int32]
    L.sim_set_flood_variant.argtypes = [_vp, C.c_int32]
    L.sim_get_flood_variant.argtypes = [_vp]
    L.sim_set_march_rows.argtypes = [_vp, C.c_int32]
    L.sim_set_overlap.argtypes = [_vp, C.c_int32]
    L.sim_set_dry_skip.argtypes = [_vp, C.c_int32]
    L.sim_set_deterministic.argtypes = [_vp, C.c_int32]
    L.sim_kernels_per_step.argtypes = [_vp]
    L.sim_slab_link.argtypes = [C.POINTER(_vp), C.c_int32]
    L.sim_slab_step.argtypes = [C.POINTER(_vp), C.c_int32, C.c_int64]
    L.sim_slab_describe.argtypes = [_vp, C.POINTER(SlabDesc)]
    L.sim_slab_attach.argtypes = [_vp, C.c_int32, C.c_int32, C.POINTER(SlabDesc)]
    L.sim_slab_enqueue.argtypes = [_vp, C.c_int32]
    L.sim_cfl_dt_static.argtypes = [_vp, _vp, _vp, _vp, C.c_int64, C.c_int32] + [C.c_double] * 6 + [_vp, _vp]
    L.sim_last_error.argtypes = [_vp]
    L.sim_last_error.restype = C.c_char_p
    L.sim_destroy.argtypes = [_vp]
    L.sim_destroy.restype = None
    for name in EXPORTS:
        if name not in ("sim_last_error", "sim_destroy"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _np_ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


class _Marshalled:
    """Host-side C structs for a Scenario; keeps the numpy arrays alive."""

    def __init__(self, sc, slab=None, with_peds=True):
        real = np.float64 if sc.real_bits == 64 else np.float32
        self.real = real
        self.keep = []

        def arr(a, dtype):
            if a is None:
                return None
            a = np.ascontiguousarray(a, dtype=dtype)
            self.keep.append(a)
            return a

        def typed(a, dtype, ptype):
            a = arr(a, dtype)
            return C.cast(None, ptype) if a is None or a.size == 0 else a.ctypes.data_as(ptype)

        if slab is None:
            self.grid = SimGrid(sc.nx, sc.ny, sc.dx, sc.dy, sc.real_bits, 0, 0)
        else:                                       # rows [j0, j0 + ny_local) of the grid; arrays stay those of the whole grid
            self.grid = SimGrid(sc.nx, slab[1], sc.dx, sc.dy, sc.real_bits, slab[0], sc.ny)
        self.topo = SimTopo(_np_ptr(arr(sc.z, real)), typed(sc.mask, np.uint8, _u8p),
                            _np_ptr(arr(sc.h0, real)), _np_ptr(arr(sc.u0, real)), _np_ptr(arr(sc.v0, real)))
        self.manning = arr(sc.manning, real)
        n = int(sc.px.shape[0]) if with_peds else 0
        self.peds = SimPeds(n, _np_ptr(arr(sc.px, real)), _np_ptr(arr(sc.py, real)),
                            _np_ptr(arr(sc.pvx, real)), _np_ptr(arr(sc.pvy, real)),
                            _np_ptr(arr(sc.pvpref, real)), typed(sc.prole, np.uint8, _u8p),
                            typed(getattr(sc, "pactive0", None), np.uint8, _u8p))
        p = SimParams()
        p.g, p.cfl, p.dt_max, p.h_dry = sc.g, sc.cfl, sc.dt_max, sc.h_dry
        p.couple_roughness, p.n_cap = sc.couple_roughness, sc.n_cap
        p.n_inflow_faces = len(sc.inflow_cell)
        p.inflow_cell = typed(sc.inflow_cell, np.int32, _i32p)
        p.inflow_side = typed(sc.inflow_side, np.uint8, _u8p)
        p.n_hydro = len(sc.hydro_t)
        p.hydro_t = typed(sc.hydro_t, np.float64, _f64p)
        p.hydro_q = typed(sc.hydro_q, np.float64, _f64p)
        p.hr_edges = (C.c_double * 4)(*sc.hr_edges)
        p.speed_wet = (C.c_double * 4)(*sc.speed_wet)
        p.tau, p.A_s, p.B_s, p.radius, p.R_int, p.vmax_factor = sc.tau, sc.A_s, sc.B_s, sc.radius, sc.R_int, sc.vmax_factor
        nav = np.ascontiguousarray(sc.nav_dir, dtype=np.uint8).reshape(-1, sc.nx * sc.ny)
        p.n_targets = nav.shape[0]
        p.nav_dir = typed(nav, np.uint8, _u8p)
        p.exit_target, p.storage_target, p.drop_target = sc.exit_target, sc.storage_target, sc.drop_target
        p.n_exit_cells = len(sc.exit_cells)
        p.exit_cells = typed(sc.exit_cells, np.int32, _i32p)
        p.storage_cell, p.drop_cell, p.arrive_cells = sc.storage_cell, sc.drop_cell, sc.arrive_cells
        p.n_line = len(sc.line_cells)
        p.line_cells = typed(sc.line_cells, np.int32, _i32p)
        p.bags_per_cell_layer, p.n_layers = sc.bags_per_cell_layer, sc.n_layers
        p.layer_thickness, p.t_pick, p.t_drop, p.t_end = sc.layer_thickness, sc.t_pick, sc.t_drop, sc.t_end
        p.flood_order = int(getattr(sc, "flood_order", 1))
        p.open_sides = int(getattr(sc, "open_sides", 0))
        doors = getattr(sc, "door_cells", np.zeros(0, np.int32))
        p.n_doors = len(doors)
        p.door_cells = typed(doors, np.int32, _i32p)
        p.door_target = typed(getattr(sc, "door_target", np.zeros(0, np.int32)), np.int32, _i32p)
        p.spawn_rate = float(getattr(sc, "spawn_rate", 0.0))
        p.target_population = int(getattr(sc, "target_population", 0))
        p.spawn_seed = int(getattr(sc, "spawn_seed", 0))
        p.spawn_vpref_lo = float(getattr(sc, "spawn_vpref_lo", 1.0)); p.spawn_vpref_hi = float(getattr(sc, "spawn_vpref_hi", 1.4))
        self.params = p


def workspace_bytes(sc) -> int:
    L = load_library()
    m = _Marshalled(sc)
    out = C.c_size_t()
    rc = L.sim_workspace_bytes(C.byref(m.grid), m.peds.n, C.byref(m.params), C.byref(out))
    if rc != SIM_OK:
        raise FloodpedError(rc, L.sim_last_error(None).decode())
    return out.value


def cfl_dt_static(h_ptr, qx_ptr, qy_ptr, mask_ptr, n_cells, real_bits, dx, dy, g, h_dry, cfl, dt_max, stream_ptr, out_ptr):
    """sim_cfl_dt_static (include/floodped.h): largest wave speed and CFL time step of a flood state
    that already sits in device memory, for callers that must not allocate on the device (a host
    framework's pool owns the GPU's memory, a loop that cannot afford cudaMalloc's device-wide
    synchronisation, a plug-in that is only handed pointers).  All `*_ptr` are raw DEVICE addresses
    (ints; `mask_ptr` and `stream_ptr` may be None / 0); `out_ptr` receives two doubles (lam, dt)
    once the stream has run.  Enqueues only; no handle, no workspace, no allocation: the scratch is
    a fixed array inside the library, so n_cells <= SIM_CFL_STATIC_MAX_CELLS and calls that could
    overlap on the GPU must be serialised by the caller.  Marshalling only."""
    L = load_library()
    rc = L.sim_cfl_dt_static(_vp(h_ptr), _vp(qx_ptr), _vp(qy_ptr), _vp(mask_ptr or None), int(n_cells), int(real_bits),
                             float(dx), float(dy), float(g), float(h_dry), float(cfl), float(dt_max),
                             _vp(stream_ptr or None), _vp(out_ptr))
    if rc != SIM_OK:
        raise FloodpedError(rc, L.sim_last_error(None).decode())


class Sim:
    """One simulation handle on the current CUDA device / current torch stream."""

    def __init__(self, sc, device="cuda:0", use_torch_workspace=True, stream=None, slab=None, with_peds=True):
        import torch

        L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libfloodped has no CPU fallback")
        self._L = L
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.real = np.float64 if sc.real_bits == 64 else np.float32
        self.nx, self.ny = sc.nx, (sc.ny if slab is None else slab[1])
        self.ncell, self.n_peds = self.nx * self.ny, (int(sc.px.shape[0]) if with_peds else 0)
        self.dx, self.dy = float(sc.dx), float(sc.dy)
        m = _Marshalled(sc, slab, with_peds)
        self._ws = None
        ws_ptr = None
        if use_torch_workspace:
            nbytes = C.c_size_t()
            rc = L.sim_workspace_bytes(C.byref(m.grid), m.peds.n, C.byref(m.params), C.byref(nbytes))
            if rc != SIM_OK:
                raise FloodpedError(rc, L.sim_last_error(None).decode())
            self._ws = torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
            ws_ptr = C.c_void_p(self._ws.data_ptr())
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = L.sim_create(C.byref(m.grid), C.byref(m.topo), _np_ptr(m.manning), C.byref(m.peds),
                          C.byref(m.params), ws_ptr, C.c_void_p(self._stream.cuda_stream), C.byref(h))
        if rc != SIM_OK:
            raise FloodpedError(rc, L.sim_last_error(None).decode())
        self._h = h

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            self._L.sim_destroy(self._h)
            self._h = None
            self._ws = None

    __del__ = close

    def _chk(self, rc):
        if rc != SIM_OK:
            raise FloodpedError(rc, self._L.sim_last_error(self._h).decode())

    # -- the path
    def step(self, n=1):
        self._chk(self._L.sim_step(self._h, int(n)))

    KERNELS = ("bin_count", "bin_scan", "scatter", "ped_step", "flood_step", "tail", "occupancy")

    def step_profiled(self, n=1) -> dict:
        """n steps with per-kernel CUDA-event timing; returns summed ms per kernel."""
        ms = (C.c_double * 8)()
        self._chk(self._L.sim_step_profiled(self._h, int(n), ms))
        return {k: ms[i] for i, k in enumerate(self.KERNELS)}

    def kernels_per_step(self) -> int:
        return self._L.sim_kernels_per_step(self._h)

    def set_flood_variant(self, v):
        self._chk(self._L.sim_set_flood_variant(self._h, int(v)))

    def set_march_rows(self, rows):
        self._chk(self._L.sim_set_march_rows(self._h, int(rows)))

    def set_overlap(self, on):
        self._chk(self._L.sim_set_overlap(self._h, int(bool(on))))

    def set_dry_skip(self, on):
        self._chk(self._L.sim_set_dry_skip(self._h, int(bool(on))))

    def set_deterministic(self, on):
        """Bins ordered by original agent id: same bits on every run (include/floodped.h)."""
        self._chk(self._L.sim_set_deterministic(self._h, int(bool(on))))

    def flood_variant(self) -> int:
        return self._L.sim_get_flood_variant(self._h)

    # -- read-back (host numpy)
    def read_flood(self, fields=("h", "u", "v", "z", "hr")):
        out = {k: np.empty(self.ncell, self.real) for k in fields}
        self._chk(self._L.sim_read_flood(self._h, *[_np_ptr(out.get(k)) for k in ("h", "u", "v", "z", "hr")]))
        return out

    def read_conserved(self):
        out = {k: np.empty(self.ncell, self.real) for k in ("h", "qx", "qy")}
        self._chk(self._L.sim_read_conserved(self._h, *[_np_ptr(out[k]) for k in ("h", "qx", "qy")]))
        return out

    def read_conserved_into(self, h_ptr, qx_ptr, qy_ptr):
        """Raw pointers (host or device), e.g. pinned torch tensors' data_ptr()."""
        self._chk(self._L.sim_read_conserved(self._h, C.c_void_p(h_ptr), C.c_void_p(qx_ptr), C.c_void_p(qy_ptr)))

    def read_occupancy(self):
        a = np.empty(self.ncell, np.uint8)
        self._chk(self._L.sim_read_occupancy(self._h, _np_ptr(a)))
        return a

    def read_peds(self):
        n = self.n_peds
        out = {k: np.empty(n, self.real) for k in ("x", "y", "vx", "vy", "timer")}
        out.update({k: np.empty(n, np.uint8) for k in ("state", "fsm", "active")})
        out["cell"] = np.empty(n, np.int32)
        self._chk(self._L.sim_read_peds(self._h, *[_np_ptr(out[k]) for k in
                                                    ("x", "y", "vx", "vy", "state", "fsm", "active", "cell", "timer")]))
        return out

    def stats(self) -> dict:
        st = SimStats()
        self._chk(self._L.sim_get_stats(self._h, C.byref(st)))
        d = {k: getattr(st, k) for k, _ in SimStats._fields_ if k != "hist"}
        d["hist"] = list(st.hist)
        return d

    # -- test hooks
    def bin_peds(self):
        nbx, nby, k = C.c_int32(), C.c_int32(), C.c_int32()
        self._chk(self._L.sim_bin_peds(self._h, None, None, None, C.byref(nbx), C.byref(nby), C.byref(k)))
        nb = nbx.value * nby.value
        key = np.empty(self.n_peds, np.int32); order = np.empty(self.n_peds, np.int32)
        start = np.empty(nb + 2, np.int32)
        self._chk(self._L.sim_bin_peds(self._h, _np_ptr(key), _np_ptr(order), _np_ptr(start), None, None, None))
        return {"key": key, "order": order, "start": start, "nbx": nbx.value, "nby": nby.value, "k": k.value}

    def write_flood(self, h=None, qx=None, qy=None, z=None):
        a = [None if v is None else np.ascontiguousarray(v, self.real) for v in (h, qx, qy, z)]
        self._chk(self._L.sim_write_flood(self._h, *[_np_ptr(v) for v in a]))

    def write_peds(self, x=None, y=None, vx=None, vy=None, fsm=None, active=None, timer=None):
        f = [None if v is None else np.ascontiguousarray(v, self.real) for v in (x, y, vx, vy)]
        b = [None if v is None else np.ascontiguousarray(v, np.uint8) for v in (fsm, active)]
        t = None if timer is None else np.ascontiguousarray(timer, self.real)
        self._chk(self._L.sim_write_peds(self._h, *[_np_ptr(v) for v in f], *[_np_ptr(v) for v in b], _np_ptr(t)))

    def set_time(self, t, dt):
        self._chk(self._L.sim_set_time(self._h, float(t), float(dt)))

    def philox(self, counters_keys):
        """the device's Philox4x32-10 on rows of (c0, c1, c2, c3, k0, k1)"""
        a = np.ascontiguousarray(counters_keys, np.uint32).reshape(-1, 6)
        out = np.empty((a.shape[0], 4), np.uint32)
        self._chk(self._L.sim_test_philox(self._h, _np_ptr(a), _np_ptr(out), a.shape[0]))
        return out

    def set_barrier(self, cursor, layer, bags, complete):
        self._chk(self._L.sim_set_barrier(self._h, int(cursor), int(layer), int(bags), int(complete)))


class SlabSim:
    """The grid cut into `n_slabs` row slabs, one handle each (include/floodped.h
    sim_slab_link): `devices` names one CUDA device per slab (all in this process, with peer access),
    default all on `cuda:0`, which is how the path is tested on one GPU.  All pedestrians live on
    the first slab's handle.  Marshalling only."""

    def __init__(self, sc, n_slabs, devices=None):
        from .replicas import slab_cuts
        self.cuts = slab_cuts(sc.ny, n_slabs)
        devices = devices or ["cuda:0"] * len(self.cuts)
        self.sims = [Sim(sc, device=devices[r], slab=cut, with_peds=(r == 0)) for r, cut in enumerate(self.cuts)]
        self._L = self.sims[0]._L
        self._arr = (_vp * len(self.sims))(*[g._h for g in self.sims])
        self._chk(self._L.sim_slab_link(self._arr, len(self.sims)))

    def _chk(self, rc):
        if rc != SIM_OK:
            raise FloodpedError(rc, self._L.sim_last_error(self.sims[0]._h).decode())

    def step(self, n=1):
        self._chk(self._L.sim_slab_step(self._arr, len(self.sims), int(n)))

    def read_conserved(self):
        parts = [g.read_conserved() for g in self.sims]
        return {k: np.concatenate([p[k] for p in parts]) for k in ("h", "qx", "qy")}

    def read_flood(self, fields=("h", "u", "v", "z", "hr")):
        parts = [g.read_flood(fields) for g in self.sims]
        return {k: np.concatenate([p[k] for p in parts]) for k in fields}

    def read_occupancy(self):
        return np.concatenate([g.read_occupancy() for g in self.sims])

    def read_peds(self):
        return self.sims[0].read_peds()

    def stats(self) -> dict:
        """the first slab's record (time, pedestrians, barrier) with the flood sums taken over all slabs"""
        st = [g.stats() for g in self.sims]
        d = dict(st[0])
        d["volume"] = float(sum(s["volume"] for s in st))
        d["clamped_volume"] = float(sum(s["clamped_volume"] for s in st))
        d["neg_depth_clamps"] = int(sum(s["neg_depth_clamps"] for s in st))
        d["max_h"] = max(s["max_h"] for s in st); d["max_hr"] = max(s["max_hr"] for s in st)
        d["per_slab"] = st
        return d

    def close(self):
        for g in self.sims:
            g.close()


class SlabRank:
    """One row slab per PROCESS and GPU (include/floodped.h sim_slab_attach), under an
    initialised torch.distributed group: rank r holds slab r (rank 0 also all pedestrians).  The
    workspaces are shared between the processes as CUDA-IPC tensors (torch.multiprocessing's
    reductions), so that a slab's flood kernel reads its halo rows, and the pedestrian kernels read
    and write the cells of other slabs, in place; the one collective per step is the MAX all-reduce of
    the 8-byte wave speed (NCCL on the device; any other backend through a host copy, for tests).
    Marshalling and sequencing only."""

    def __init__(self, sc, device=None):
        import torch
        import torch.distributed as dist
        from torch.multiprocessing.reductions import reduce_tensor
        from .replicas import slab_cuts
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        cuts = slab_cuts(sc.ny, self.world)
        if len(cuts) != self.world:
            raise ValueError("fewer rows than ranks")
        self.cut = cuts[self.rank]
        self.sim = Sim(sc, device=device or f"cuda:{torch.cuda.current_device()}", slab=self.cut, with_peds=(self.rank == 0))
        self._L = self.sim._L
        mine = SlabDesc()
        self.sim._chk(self._L.sim_slab_describe(self.sim._h, C.byref(mine)))
        ws = self.sim._ws
        assert ws.data_ptr() == mine.workspace
        torch.cuda.synchronize()
        offer = (mine.to_dict(), reduce_tensor(ws))
        offers = [None] * self.world
        dist.all_gather_object(offers, offer)
        self._peers = []                                   # mapped workspaces of the other ranks: keep them alive
        descs = (SlabDesc * self.world)()
        for r, (d, (rebuild, args)) in enumerate(offers):
            if r == self.rank:
                descs[r] = mine
            else:
                t = rebuild(*args)                         # the peer's workspace, mapped into this process
                self._peers.append(t)
                descs[r] = SlabDesc.rebased(d, t.data_ptr())
        self.sim._chk(self._L.sim_slab_attach(self.sim._h, self.rank, self.world, descs))
        off = mine.lam_bits - mine.workspace
        self._lam = ws[off:off + 8].view(torch.int64)      # bit pattern of a non-negative double: ordered like an integer
        self._nccl = dist.get_backend() == "nccl"
        dist.barrier()
        self.resync()

    def resync(self):
        """(re)make the bins and N_p of the state in place and the time step from the global wave speed;
        collective: every rank calls it, after attaching and after any change of pedestrians or modes"""
        self._phase(2); self._reduce(); self._phase(3)

    def set_deterministic(self, on):
        """collective: sim_set_deterministic on this rank's handle, then resync()"""
        self.sim.set_deterministic(on)
        self.resync()

    def _phase(self, k):
        self.sim._chk(self._L.sim_slab_enqueue(self.sim._h, int(k)))

    def _reduce(self):
        import torch
        import torch.distributed as dist
        if self._nccl:
            dist.all_reduce(self._lam, op=dist.ReduceOp.MAX)
        else:                                              # CPU backends (tests): through the host
            torch.cuda.synchronize()
            v = self._lam.cpu()
            dist.all_reduce(v, op=dist.ReduceOp.MAX)
            self._lam.copy_(v)
            torch.cuda.synchronize()

    def step(self, n=1):
        for _ in range(int(n)):
            self._phase(0); self._reduce(); self._phase(1)

    def close(self):
        import torch
        import torch.distributed as dist
        torch.cuda.synchronize()
        dist.barrier()                                     # nobody unmaps a workspace another rank may still read
        self.sim.close()
        self._peers = []
