"""ctypes binding of oracle/liborc.so (double-precision CPU oracle; test infrastructure).

Argument marshalling only; all arithmetic is in sph_oracle.cpp.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MAX_PHASES = 4
TAG_WALL = -1
FLAG_REINIT = 1
FLAG_WALL_VEL_MIRROR = 2
FLAG_WALL_ADAMI_ONLY = 8
VAR_REINIT_LITERAL = 1   # study-only variants (NEXT-2): see sph_oracle.cpp
VAR_SUM_RAW = 2
VAR_SIGMA_ALL = 4


class OrcParams(C.Structure):
    _fields_ = [
        ("dim", C.c_int32), ("n_phases", C.c_int32),
        ("dp", C.c_double), ("h", C.c_double),
        ("rho0", C.c_double * MAX_PHASES), ("c0", C.c_double * MAX_PHASES),
        ("g", C.c_double * 3), ("g_osc_amp", C.c_double * 3), ("g_osc_period", C.c_double),
        ("cfl", C.c_double), ("penalty_strength", C.c_double),
        ("penalty_phase_mask", C.c_uint32), ("free_surface_mask", C.c_uint32),
        ("flags", C.c_uint32), ("variant", C.c_uint32),
        ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("wall_osc_amp", C.c_double * 3), ("wall_osc_freq", C.c_double), ("t_start", C.c_double),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        d, i32, i64, vp = C.c_double, C.c_int32, C.c_int64, C.c_void_p
        L.orc_kernel_w.restype = d; L.orc_kernel_w.argtypes = [C.c_int, d, d]
        L.orc_kernel_dw.restype = d; L.orc_kernel_dw.argtypes = [C.c_int, d, d]
        L.orc_sigma0.restype = d; L.orc_sigma0.argtypes = [C.c_int, d, d]
        L.orc_reinit_density.restype = d; L.orc_reinit_density.argtypes = [d, d, d, d, C.c_int]
        L.orc_riemann.restype = None; L.orc_riemann.argtypes = [C.c_int] + [d] * 8 + [vp]
        L.orc_create.restype = vp; L.orc_create.argtypes = [C.POINTER(OrcParams)]
        L.orc_destroy.restype = None; L.orc_destroy.argtypes = [vp]
        L.orc_set_particles.restype = C.c_int; L.orc_set_particles.argtypes = [vp, i64, vp, vp, vp, vp]
        L.orc_step.restype = C.c_int; L.orc_step.argtypes = [vp, i32, vp, vp]
        L.orc_get_fields.restype = None; L.orc_get_fields.argtypes = [vp] * 8
        L.orc_get_normals.restype = None; L.orc_get_normals.argtypes = [vp, vp]
        L.orc_get_stats.restype = None; L.orc_get_stats.argtypes = [vp, vp]
        L.orc_neighbour_count.restype = i64; L.orc_neighbour_count.argtypes = [vp]
        L.orc_get_neighbours.restype = None; L.orc_get_neighbours.argtypes = [vp, vp, vp]
        L.orc_neighbours_bruteforce.restype = i64; L.orc_neighbours_bruteforce.argtypes = [vp, vp, vp]
        L.orc_f32_ncell.restype = i64; L.orc_f32_ncell.argtypes = [C.POINTER(OrcParams)]
        L.orc_f32_cells.restype = None
        L.orc_f32_cells.argtypes = [C.POINTER(OrcParams), i64, vp, vp, vp, vp, vp, vp]
        L.orc_f32_neighbours.restype = i64
        L.orc_f32_neighbours.argtypes = [C.POINTER(OrcParams), i64, vp, vp, vp, vp, i64]
        L.orc_f32_neighbours_grid.restype = i64
        L.orc_f32_neighbours_grid.argtypes = [C.POINTER(OrcParams), i64, vp, vp, vp, vp, i64]
        _lib = L
    return _lib


def make_params(cfg: dict) -> OrcParams:
    """cfg: the plain dict produced by paper_2110_02621_b200.inputs (no arithmetic here)."""
    P = OrcParams()
    P.dim = cfg["dim"]; P.n_phases = cfg["n_phases"]
    P.dp = cfg["dp"]; P.h = cfg["h"]
    for k in range(MAX_PHASES):
        P.rho0[k] = cfg["rho0"][k] if k < len(cfg["rho0"]) else 0.0
        P.c0[k] = cfg["c0"][k] if k < len(cfg["c0"]) else 0.0
    for k in range(3):
        P.g[k] = cfg["g"][k]
        P.g_osc_amp[k] = cfg.get("g_osc_amp", (0, 0, 0))[k]
        P.domain_min[k] = cfg["domain_min"][k]
        P.domain_max[k] = cfg["domain_max"][k]
        P.wall_osc_amp[k] = cfg.get("wall_osc_amp", (0, 0, 0))[k]
    P.wall_osc_freq = cfg.get("wall_osc_freq", 0.0)
    P.t_start = cfg.get("t_start", 0.0)
    P.g_osc_period = cfg.get("g_osc_period", 0.0)
    P.cfl = cfg.get("cfl", 0.25)
    P.penalty_strength = cfg.get("penalty_strength", 1.0)
    P.penalty_phase_mask = cfg.get("penalty_phase_mask", 0)
    P.free_surface_mask = cfg.get("free_surface_mask", 1)
    P.flags = cfg.get("flags", FLAG_REINIT | FLAG_WALL_VEL_MIRROR)
    P.variant = cfg.get("oracle_variant", 0)
    return P


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def kernel_w(dim, h, r):
    return lib().orc_kernel_w(dim, h, r)


def kernel_dw(dim, h, r):
    return lib().orc_kernel_dw(dim, h, r)


def sigma0(dim, h, dp):
    return lib().orc_sigma0(dim, h, dp)


def reinit_density(rho_star, rho0, sigma, sig0, free_surface):
    return lib().orc_reinit_density(rho_star, rho0, sigma, sig0, int(free_surface))


def riemann(rL, UL, pL, cL, rR, UR, pR, cR, mode=0):
    out = np.zeros(5)
    lib().orc_riemann(mode, rL, UL, pL, cL, rR, UR, pR, cR, _p(out))
    return dict(Ustar=out[0], pstar=out[1], Ubar=out[2], wL=out[3], wR=out[4])


class Oracle:
    def __init__(self, cfg: dict):
        self.P = make_params(cfg)
        self.h = lib().orc_create(C.byref(self.P))
        self.n = 0

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_destroy(self.h)
            self.h = None

    def set_particles(self, pos, vel, rho, tag):
        pos = np.ascontiguousarray(pos, np.float32); vel = np.ascontiguousarray(vel, np.float32)
        rho = np.ascontiguousarray(rho, np.float32); tag = np.ascontiguousarray(tag, np.int32)
        self.n = len(tag)
        assert pos.shape == (self.n, 3) and vel.shape == (self.n, 3)
        rc = lib().orc_set_particles(self.h, self.n, _p(pos), _p(vel), _p(rho), _p(tag))
        if rc != 0:
            raise ValueError("orc_set_particles failed")

    def step(self, nsteps=1, dts=None):
        out = np.zeros(nsteps)
        din = None if dts is None else np.ascontiguousarray(dts, np.float64)
        lib().orc_step(self.h, nsteps, _p(din), _p(out))
        return out

    def fields(self):
        n = self.n
        f = dict(pos=np.zeros((n, 3)), vel=np.zeros((n, 3)), rho=np.zeros(n), p=np.zeros(n),
                 acc=np.zeros((n, 3)), sigma=np.zeros(n), drho=np.zeros(n))
        lib().orc_get_fields(self.h, _p(f["pos"]), _p(f["vel"]), _p(f["rho"]), _p(f["p"]),
                             _p(f["acc"]), _p(f["sigma"]), _p(f["drho"]))
        return f

    def normals(self):
        nw = np.zeros((self.n, 3))
        lib().orc_get_normals(self.h, _p(nw))
        return nw

    def stats(self):
        o = np.zeros(8)
        lib().orc_get_stats(self.h, _p(o))
        return dict(t=o[0], dt=o[1], steps=int(o[2]), npairs=int(o[3]), ek=o[4], mass=o[5],
                    x_front=o[6], escaped=int(o[7]))

    def neighbours(self):
        tot = lib().orc_neighbour_count(self.h)
        off = np.zeros(self.n + 1, np.int64); ids = np.zeros(max(tot, 1), np.int32)
        lib().orc_get_neighbours(self.h, _p(off), _p(ids))
        return off, ids[:tot]

    def neighbours_bruteforce(self):
        off = np.zeros(self.n + 1, np.int64)
        tot = lib().orc_neighbours_bruteforce(self.h, _p(off), None)
        ids = np.zeros(max(tot, 1), np.int32)
        lib().orc_neighbours_bruteforce(self.h, _p(off), _p(ids))
        return off, ids[:tot]


def f32_cells(cfg, pos, tag):
    P = make_params(cfg)
    pos = np.ascontiguousarray(pos, np.float32); tag = np.ascontiguousarray(tag, np.int32)
    n = len(tag)
    ncell = lib().orc_f32_ncell(C.byref(P))
    cell_id = np.zeros(n, np.int32); perm = np.zeros(n, np.int32)
    cs = np.zeros(2 * ncell, np.int32); ce = np.zeros(2 * ncell, np.int32)
    lib().orc_f32_cells(C.byref(P), n, _p(pos), _p(tag), _p(cell_id), _p(perm), _p(cs), _p(ce))
    return cell_id, perm, cs, ce


def f32_neighbours(cfg, pos, tag, grid=False):
    P = make_params(cfg)
    pos = np.ascontiguousarray(pos, np.float32); tag = np.ascontiguousarray(tag, np.int32)
    n = len(tag)
    fn = lib().orc_f32_neighbours_grid if grid else lib().orc_f32_neighbours
    off = np.zeros(n + 1, np.int64)
    tot = fn(C.byref(P), n, _p(pos), _p(tag), _p(off), None, 0)
    ids = np.zeros(max(tot, 1), np.int32)
    fn(C.byref(P), n, _p(pos), _p(tag), _p(off), _p(ids), tot)
    return off, ids[:tot]
