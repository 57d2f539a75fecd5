"""ctypes binding of libsph (include/sph.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/sph.cu.  torch is used for device
memory and streams.  There is no CPU fallback: loading fails loudly if libsph.so is missing,
and every call raises SphError if the library reports an error (e.g. no CUDA device).
"""
import ctypes as C
import os

import numpy as np

MAX_PHASES = 4
TAG_WALL = -1
FLAG_REINIT = 1
FLAG_WALL_VEL_MIRROR = 2
FLAG_NO_GRAPH = 4
FLAG_WALL_ADAMI_ONLY = 8
DEFAULT_LIST_SKIN = 0.1   # what sph_create takes for list_skin < 0 (include/sph.h)
STAGES = ("predict", "sort", "reorder", "wall", "pass_a", "pass_b", "build")

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsph.so")


class SphError(RuntimeError):
    pass


class SphParams(C.Structure):
    _fields_ = [
        ("dim", C.c_int32), ("n_phases", C.c_int32),
        ("dp", C.c_double), ("h", C.c_double),
        ("rho0", C.c_double * MAX_PHASES), ("c0", C.c_double * MAX_PHASES),
        ("g", C.c_double * 3), ("g_osc_amp", C.c_double * 3), ("g_osc_period", C.c_double),
        ("cfl", C.c_double), ("penalty_strength", C.c_double),
        ("penalty_phase_mask", C.c_uint32), ("free_surface_mask", C.c_uint32),
        ("flags", C.c_uint32), ("max_neighbours", C.c_uint32),
        ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("wall_osc_amp", C.c_double * 3), ("wall_osc_freq", C.c_double), ("list_skin", C.c_double),
    ]


class SphStats(C.Structure):
    _fields_ = [
        ("t", C.c_double), ("dt", C.c_double), ("steps", C.c_int64), ("n_fluid", C.c_int64),
        ("n_wall", C.c_int64), ("n_pairs", C.c_int64), ("e_kin", C.c_double), ("mass", C.c_double),
        ("x_front", C.c_double), ("escaped", C.c_int64), ("nonfinite", C.c_int64), ("rebuilds", C.c_int64), ("list_skin", C.c_double),
    ]


EXPORTS = (
    "sph_create", "sph_destroy", "sph_set_particles", "sph_set_particles_host", "sph_step",
    "sph_step_dt", "sph_get_fields", "sph_get_fields_host", "sph_get_stats", "sph_get_stats_ex", "sph_set_profiling",
    "sph_get_timings", "sph_num_cells", "sph_debug_cells", "sph_debug_neighbours", "sph_debug_list_check", "sph_probe_pressure", "sph_probe_gauge",
    "sph_debug_normals", "sph_debug_sigma", "sph_launch_count", "sph_last_error", "sph_debug_step_lists", "sph_debug_fma_peak", "sph_debug_time_pointwise", "sph_debug_gather_floor", "sph_debug_gather_patterns",
    "sph_cell_sort_static", "sph_cell_sort_static_error",
)

_lib = None


def load():
    """dlopen libsph.so; raises if it has not been built (python -m paper_2110_02621_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise SphError("libsph.so is missing: build it with `python paper_2110_02621_b200/build.py` "
                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.sph_create.restype = C.c_int; L.sph_create.argtypes = [C.POINTER(SphParams), C.POINTER(vp)]
    L.sph_destroy.restype = None; L.sph_destroy.argtypes = [vp]
    for name in ("sph_set_particles", "sph_set_particles_host"):
        f = getattr(L, name); f.restype = C.c_int; f.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    L.sph_step.restype = C.c_int; L.sph_step.argtypes = [vp, i32, vp]
    L.sph_step_dt.restype = C.c_int; L.sph_step_dt.argtypes = [vp, i32, vp, vp]
    for name in ("sph_get_fields", "sph_get_fields_host"):
        f = getattr(L, name); f.restype = C.c_int; f.argtypes = [vp] * 7
    L.sph_get_stats.restype = C.c_int; L.sph_get_stats.argtypes = [vp, C.POINTER(SphStats), vp]
    L.sph_get_stats_ex.restype = C.c_int; L.sph_get_stats_ex.argtypes = [vp, C.POINTER(SphStats), i32, vp]
    L.sph_set_profiling.restype = C.c_int; L.sph_set_profiling.argtypes = [vp, i32]
    L.sph_get_timings.restype = C.c_int; L.sph_get_timings.argtypes = [vp, vp, vp, vp]
    L.sph_num_cells.restype = i64; L.sph_num_cells.argtypes = [vp]
    L.sph_debug_cells.restype = C.c_int; L.sph_debug_cells.argtypes = [vp] * 6
    L.sph_debug_neighbours.restype = C.c_int; L.sph_debug_neighbours.argtypes = [vp, vp, vp, i64, vp, vp]
    L.sph_debug_step_lists.restype = C.c_int; L.sph_debug_step_lists.argtypes = [vp, vp, vp, i64, vp, vp]
    L.sph_debug_time_pointwise.restype = C.c_int; L.sph_debug_time_pointwise.argtypes = [vp, vp, vp]
    L.sph_debug_fma_peak.restype = C.c_int; L.sph_debug_fma_peak.argtypes = [vp, vp]
    L.sph_debug_gather_floor.restype = C.c_int; L.sph_debug_gather_floor.argtypes = [vp, i32, vp, vp, vp]
    L.sph_debug_gather_patterns.restype = C.c_int; L.sph_debug_gather_patterns.argtypes = [vp, vp]
    L.sph_debug_normals.restype = C.c_int; L.sph_debug_normals.argtypes = [vp, vp, vp]
    L.sph_debug_list_check.restype = C.c_int; L.sph_debug_list_check.argtypes = [vp, vp, vp]
    L.sph_probe_pressure.restype = C.c_int; L.sph_probe_pressure.argtypes = [vp, C.c_int32, vp, vp, vp, vp]
    L.sph_probe_gauge.restype = C.c_int; L.sph_probe_gauge.argtypes = [vp, C.c_int32, vp, vp, vp]
    L.sph_debug_sigma.restype = C.c_int; L.sph_debug_sigma.argtypes = [vp, vp, vp]
    L.sph_launch_count.restype = i64; L.sph_launch_count.argtypes = [vp]
    L.sph_last_error.restype = C.c_char_p; L.sph_last_error.argtypes = [vp]
    L.sph_cell_sort_static.restype = C.c_int; L.sph_cell_sort_static.argtypes = [i32, vp, vp, i32, vp, vp, vp]
    L.sph_cell_sort_static_error.restype = C.c_char_p; L.sph_cell_sort_static_error.argtypes = []
    _lib = L
    return L


def make_params(cfg: dict) -> SphParams:
    P = SphParams()
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
    P.g_osc_period = cfg.get("g_osc_period", 0.0)
    P.cfl = cfg.get("cfl", 0.25)
    P.penalty_strength = cfg.get("penalty_strength", 1.0)
    P.penalty_phase_mask = cfg.get("penalty_phase_mask", 0)
    P.free_surface_mask = cfg.get("free_surface_mask", 1)
    P.flags = cfg.get("flags", FLAG_REINIT | FLAG_WALL_VEL_MIRROR)
    P.max_neighbours = cfg.get("max_neighbours", 0)
    P.list_skin = cfg.get("list_skin", -1.0)   # < 0: library default
    return P


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Sph:
    """One simulation context (sph_ctx).  Methods mirror the C entry points."""

    def __init__(self, cfg: dict, stream=None):
        self.L = load()
        self.P = make_params(cfg)
        self.ctx = C.c_void_p()
        self.n = 0
        self._stream = stream
        rc = self.L.sph_create(C.byref(self.P), C.byref(self.ctx))
        if rc != 0:
            self.ctx = C.c_void_p()
            raise SphError("sph_create failed with code %d (no CUDA device or bad parameters)" % rc)

    def _st(self):
        import torch
        s = self._stream if self._stream is not None else torch.cuda.current_stream()
        return C.c_void_p(s.cuda_stream)

    def _ck(self, rc):
        if rc != 0:
            raise SphError("libsph error %d: %s" % (rc, self.L.sph_last_error(self.ctx).decode()))

    def close(self):
        if getattr(self, "ctx", None) and self.ctx.value:
            self.L.sph_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- sph_set_particles / _host ------------------------------------------------------------
    def set_particles(self, pos, vel, rho, tag):
        """torch CUDA tensors (float32 [n,3], [n,3], [n]; int32 [n]) -> device-pointer entry;
        numpy arrays -> host-pointer entry."""
        import torch
        if isinstance(pos, np.ndarray):
            pos = np.ascontiguousarray(pos, np.float32); vel = np.ascontiguousarray(vel, np.float32)
            rho = np.ascontiguousarray(rho, np.float32); tag = np.ascontiguousarray(tag, np.int32)
            self.n = len(tag)
            self._ck(self.L.sph_set_particles_host(self.ctx, self.n, _hp(pos), _hp(vel), _hp(rho), _hp(tag), self._st()))
            return
        assert pos.is_cuda and pos.dtype == torch.float32 and tag.dtype == torch.int32
        pos, vel, rho, tag = pos.contiguous(), vel.contiguous(), rho.contiguous(), tag.contiguous()
        self.n = tag.numel()
        self._ck(self.L.sph_set_particles(self.ctx, self.n, pos.data_ptr(), vel.data_ptr(), rho.data_ptr(),
                                          tag.data_ptr(), self._st()))

    # -- sph_step / sph_step_dt ------------------------------------------------------------------
    def step(self, n_steps=1, dts=None):
        if dts is None:
            self._ck(self.L.sph_step(self.ctx, int(n_steps), self._st()))
        else:
            d = np.ascontiguousarray(dts, np.float64)
            assert len(d) >= n_steps
            self._ck(self.L.sph_step_dt(self.ctx, int(n_steps), _hp(d), self._st()))

    # -- sph_get_fields / _host ----------------------------------------------------------------------
    def get_fields(self, device=True, which=("pos", "vel", "rho", "p", "acc")):
        import torch
        n = self.n
        shapes = dict(pos=(n, 3), vel=(n, 3), rho=(n,), p=(n,), acc=(n, 3))
        if device:
            out = {k: torch.empty(shapes[k], dtype=torch.float32, device="cuda") for k in which}
            ptr = lambda k: out[k].data_ptr() if k in out else None
            self._ck(self.L.sph_get_fields(self.ctx, ptr("pos"), ptr("vel"), ptr("rho"), ptr("p"), ptr("acc"), self._st()))
            return out
        out = {k: np.empty(shapes[k], np.float32) for k in which}
        ptr = lambda k: _hp(out[k]) if k in out else None
        self._ck(self.L.sph_get_fields_host(self.ctx, ptr("pos"), ptr("vel"), ptr("rho"), ptr("p"), ptr("acc"), self._st()))
        return out

    def get_fields_into_host(self, pos=None, vel=None, rho=None, p=None, acc=None):
        """Host-pointer entry writing into caller-provided (e.g. pinned) numpy arrays."""
        self._ck(self.L.sph_get_fields_host(self.ctx, _hp(pos), _hp(vel), _hp(rho), _hp(p), _hp(acc), self._st()))

    # -- sph_get_stats ---------------------------------------------------------------------------
    def get_stats(self, check=True, with_pairs=True):
        s = SphStats()
        rc = self.L.sph_get_stats_ex(self.ctx, C.byref(s), 1 if with_pairs else 0, self._st())
        if check:
            self._ck(rc)
        return dict(t=s.t, dt=s.dt, steps=s.steps, n_fluid=s.n_fluid, n_wall=s.n_wall, npairs=s.n_pairs,
                    ek=s.e_kin, mass=s.mass, x_front=s.x_front, escaped=s.escaped, nonfinite=s.nonfinite,
                    rebuilds=s.rebuilds, list_skin=s.list_skin, rc=rc)

    # -- profiling ---------------------------------------------------------------------------------
    def set_profiling(self, on=True):
        self._ck(self.L.sph_set_profiling(self.ctx, 1 if on else 0))

    def get_timings(self):
        ms = np.zeros(len(STAGES), np.float32)
        ns, nr = C.c_int32(0), C.c_int32(0)
        self._ck(self.L.sph_get_timings(self.ctx, _hp(ms), C.byref(ns), C.byref(nr)))
        self.last_timing_rebuilds = nr.value
        return dict(zip(STAGES, ms.tolist())), ns.value

    def time_pointwise(self):
        """sph_debug_time_pointwise: stand-alone density-reinitialisation kernel, integrator kernel (kick + drift +
        cell hash) and the fused predictor the step runs, ms per launch (state untouched)."""
        ms = np.zeros(3, np.float32)
        self._ck(self.L.sph_debug_time_pointwise(self.ctx, _hp(ms), self._st()))
        return dict(reinit=float(ms[0]), integrator=float(ms[1]), fused_predict=float(ms[2]))

    def gather_floor(self, body_fma=0):
        """sph_debug_gather_floor: the passes' list walk with an empty pair body on the current lists (ms per launch)
        and the number of warp-wide gather requests of one walk; body_fma > 0: with a synthetic pair body of that many
        FFMAs per pair."""
        ms = np.zeros(5, np.float32)
        req = C.c_int64(0)
        self._ck(self.L.sph_debug_gather_floor(self.ctx, int(body_fma), _hp(ms), C.byref(req), self._st()))
        return dict(own_entries=float(ms[0]), lane_pair_shared=float(ms[1]), quad_shared=float(ms[2]),
                    coalesced=float(ms[3]), own_entries_sm_affine=float(ms[4]), requests=req.value)

    def launch_count(self):
        return self.L.sph_launch_count(self.ctx)

    def num_cells(self):
        return self.L.sph_num_cells(self.ctx)

    # -- debug (integer contract) --------------------------------------------------------------------
    def debug_cells(self):
        nc = self.num_cells()
        cell_id = np.zeros(self.n, np.int32); perm = np.zeros(self.n, np.int32)
        cs = np.zeros(2 * nc, np.int32); ce = np.zeros(2 * nc, np.int32)
        self._ck(self.L.sph_debug_cells(self.ctx, _hp(cell_id), _hp(perm), _hp(cs), _hp(ce), self._st()))
        return cell_id, perm, cs, ce

    def debug_neighbours(self):
        off = np.zeros(self.n + 1, np.int64)
        tot = C.c_int64(0)
        self._ck(self.L.sph_debug_neighbours(self.ctx, _hp(off), None, 0, C.byref(tot), self._st()))
        ids = np.zeros(max(tot.value, 1), np.int32)
        self._ck(self.L.sph_debug_neighbours(self.ctx, _hp(off), _hp(ids), tot.value, C.byref(tot), self._st()))
        return off, ids[:tot.value]

    def debug_step_lists(self):
        """The lists the passes read (caller ids, list order, self and filter extras included)."""
        off = np.zeros(self.n + 1, np.int64)
        tot = C.c_int64(0)
        self._ck(self.L.sph_debug_step_lists(self.ctx, _hp(off), None, 0, C.byref(tot), self._st()))
        ids = np.zeros(max(tot.value, 1), np.int32)
        self._ck(self.L.sph_debug_step_lists(self.ctx, _hp(off), _hp(ids), tot.value, C.byref(tot), self._st()))
        return off, ids[:tot.value]

    def probe_pressure(self, points):
        """Shepard-averaged fluid pressure at points (m,3) -> (p (m,), wsum (m,)); reading A29."""
        pts = np.ascontiguousarray(points, np.float32).reshape(-1, 3)
        p = np.zeros(len(pts), np.float32); w = np.zeros(len(pts), np.float32)
        self._ck(self.L.sph_probe_pressure(self.ctx, len(pts), _hp(pts), _hp(p), _hp(w), self._st()))
        return p, w

    def probe_gauge(self, points):
        """Free-surface height of phase 0 at the horizontal positions of points (m,3); reading A30."""
        pts = np.ascontiguousarray(points, np.float32).reshape(-1, 3)
        eta = np.zeros(len(pts), np.float32)
        self._ck(self.L.sph_probe_gauge(self.ctx, len(pts), _hp(pts), _hp(eta), self._st()))
        return eta

    def debug_list_check(self):
        """(missing, extra, total) of the step's neighbour lists against the float32 contract."""
        out = np.zeros(3, np.int64)
        self._ck(self.L.sph_debug_list_check(self.ctx, _hp(out), self._st()))
        return int(out[0]), int(out[1]), int(out[2])

    def debug_normals(self):
        nw = np.zeros((self.n, 3), np.float32)
        self._ck(self.L.sph_debug_normals(self.ctx, _hp(nw), self._st()))
        return nw

    def debug_sigma(self):
        buf = np.zeros(2 * max(self.n, 1), np.float32)
        self._ck(self.L.sph_debug_sigma(self.ctx, _hp(buf), self._st()))
        return buf[:self.n].copy(), buf[self.n:2 * self.n].copy()


def fma_peak_tflops(stream=None):
    """sph_debug_fma_peak: measured non-tensor FP32 peak of the current device in TFLOP/s."""
    import torch
    L = load()
    out = C.c_double(0.0)
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = L.sph_debug_fma_peak(C.byref(out), C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise SphError("sph_debug_fma_peak failed with code %d" % rc)
    return out.value


GATHER_PATTERNS = ("random_32_records", "consecutive_32_records", "16_lines_lane_pairs", "8_lines_quads_4_records",
                   "8_records_quads", "one_record", "32_lines", "random_32_of_64_records")


def gather_pattern_cycles(stream=None):
    """sph_debug_gather_patterns: SM cycles per warp-wide 32-byte-record gather for eight address patterns (L1-resident)."""
    import torch
    L = load()
    out = (C.c_double * 8)()
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = L.sph_debug_gather_patterns(out, C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise SphError("sph_debug_gather_patterns failed with code %d" % rc)
    return dict(zip(GATHER_PATTERNS, [float(x) for x in out]))


STATIC_SORT_MAX_KEYS = 1 << 20


def cell_sort_static(keys, vals, key_bits, keys_out, vals_out, stream=None):
    """sph_cell_sort_static: stable radix sort of (keys, vals) by the low `key_bits` bits of the keys with the
    library's static device scratch (no allocation; at most STATIC_SORT_MAX_KEYS keys).  All tensors are the
    caller's: contiguous 4-byte integer CUDA tensors of n elements; `vals` None = the indices 0..n-1.
    Asynchronous on `stream` (default: torch's current stream)."""
    import torch
    L = load()
    n = keys.numel()
    for t in (keys, vals, keys_out, vals_out):
        if t is not None and not (t.is_cuda and t.is_contiguous() and t.element_size() == 4 and t.numel() == n):
            raise SphError("cell_sort_static: contiguous 4-byte CUDA tensors of one length are needed")
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = L.sph_cell_sort_static(n, C.c_void_p(keys.data_ptr()), C.c_void_p(vals.data_ptr()) if vals is not None else None,
                                int(key_bits), C.c_void_p(keys_out.data_ptr()), C.c_void_p(vals_out.data_ptr()),
                                C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise SphError("sph_cell_sort_static failed with code %d: %s" % (rc, L.sph_cell_sort_static_error().decode()))
