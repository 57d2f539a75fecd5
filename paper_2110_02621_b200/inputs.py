"""Seeded synthetic particle configurations (BASELINE.json configs 0-4).

This module serves both the CUDA library and the CPU oracle and holds none of the
method's arithmetic: it only places particles on lattices, tags them and sets the
initial (hydrostatic) density.  numpy only.  The inputs stand in for the paper's
cases — dam break with obstacle, two-phase tank/sloshing
(PAPER.md:220-252), arbitrary geometry; the benchmark records
themselves are not reproduced here.

Conventions: lattice sites at (k+1/2) dp from the inner wall face; wall dummy layers
at -(k+1/2) dp, k = 0,1,2; fluid at rest; rho = rho0 + p_hydrostatic / c0^2.
Every generator returns a dict with the parameters (plain numbers) and the float32
arrays pos[n,3], vel[n,3], rho[n], tag[n] (phase id >= 0, -1 = wall), fluid first.
"""
import math

import numpy as np

TAG_WALL = -1
FLAG_REINIT = 1
FLAG_WALL_VEL_MIRROR = 2
G0 = 9.81
NWALL = 3  # dummy layers


def _finish(cfg, pos_f, tag_f, rho_f, pos_w):
    pos = np.concatenate([pos_f, pos_w]).astype(np.float64)
    if pos.shape[1] == 2:
        pos = np.concatenate([pos, np.zeros((len(pos), 1))], axis=1)
    tag = np.concatenate([tag_f, np.full(len(pos_w), TAG_WALL)]).astype(np.int32)
    rho = np.concatenate([rho_f, np.full(len(pos_w), cfg["rho0"][0])])
    cfg["pos"] = np.ascontiguousarray(pos, np.float32)
    cfg["vel"] = np.zeros_like(cfg["pos"])
    cfg["rho"] = np.ascontiguousarray(rho, np.float32)
    cfg["tag"] = tag
    cfg["n_fluid"] = int(len(pos_f))
    cfg["n_wall"] = int(len(pos_w))
    return cfg


def _base(dim, dp, rho0, c0, g, lo, hi, **kw):
    cfg = dict(dim=dim, n_phases=len(rho0), dp=float(dp), h=1.3 * float(dp),
               rho0=[float(x) for x in rho0], c0=[float(x) for x in c0],
               g=[float(x) for x in g], g_osc_amp=[0.0, 0.0, 0.0], g_osc_period=0.0,
               cfl=0.25, penalty_strength=1.0, penalty_phase_mask=0, free_surface_mask=1,
               flags=FLAG_REINIT | FLAG_WALL_VEL_MIRROR,
               domain_min=[float(x) for x in lo] + [0.0] * (3 - dim),
               domain_max=[float(x) for x in hi] + [0.0] * (3 - dim))
    cfg.update(kw)
    return cfg


def _lattice(shape, dp, start=0):
    """Sites (k + 1/2) dp, k = start .. start+shape-1 per axis; returns [prod(shape), dim]."""
    axes = [(np.arange(start, start + s) + 0.5) * dp for s in shape]
    grid = np.meshgrid(*axes, indexing="ij")
    return np.stack([g.ravel() for g in grid], axis=1)


def _shell(shape, dp):
    """3-layer closed shell around an interior of `shape` sites: index arrays (integer sites)."""
    ext = [s + 2 * NWALL for s in shape]
    idx = np.stack([g.ravel() for g in np.meshgrid(*[np.arange(-NWALL, s + NWALL) for s in shape],
                                                   indexing="ij")], axis=1)
    inside = np.ones(len(idx), bool)
    for k, s in enumerate(shape):
        inside &= (idx[:, k] >= 0) & (idx[:, k] < s)
    del ext
    return idx[~inside]


def dam_break_2d(dp=0.05, tank=(4.0, 3.0), column=(1.0, 2.0)):
    """Config 0: 2-D single-phase dam break, about 800 fluid particles."""
    H = column[1]
    c0 = 10.0 * math.sqrt(2.0 * G0 * H)
    nx, ny = int(round(tank[0] / dp)), int(round(tank[1] / dp))
    cfg = _base(2, dp, [1000.0], [c0], [0.0, -G0, 0.0], [-NWALL * dp] * 2,
                [tank[0] + NWALL * dp, tank[1] + NWALL * dp], name="cfg0_dam_break_2d", H=H)
    cx, cy = int(math.floor(column[0] / dp + 1e-9)), int(math.floor(column[1] / dp + 1e-9))
    pos_f = _lattice((cx, cy), dp)
    rho_f = 1000.0 * (1.0 + G0 * (H - pos_f[:, 1]) / c0 ** 2)
    pos_w = (_shell((nx, ny), dp) + 0.5) * dp
    return _finish(cfg, pos_f, np.zeros(len(pos_f)), rho_f, pos_w)


def dam_break_3d_box(dp=0.01, tank=(3.22, 1.0, 1.0), column=(1.228, 1.0, 0.55),
                     box_lo=(2.40, 0.30, 0.0), box_hi=(2.56, 0.70, 0.16)):
    """Config 1: 3-D dam break with a box obstacle (geometry from BASELINE.json; reading A27)."""
    H = column[2]
    c0 = 10.0 * math.sqrt(2.0 * G0 * H)
    n = [int(round(t / dp)) for t in tank]
    cfg = _base(3, dp, [1000.0], [c0], [0.0, 0.0, -G0], [-NWALL * dp] * 3,
                [t + NWALL * dp for t in tank], name="cfg1_dam_break_3d_box", H=H)
    cn = [int(math.floor(c / dp + 1e-9)) for c in column]
    pos_f = _lattice(cn, dp)
    rho_f = 1000.0 * (1.0 + G0 * (H - pos_f[:, 2]) / c0 ** 2)
    pos_w = (_shell(n, dp) + 0.5) * dp
    # obstacle: lattice sites inside the box within 3 layers of its five exposed faces
    b0 = [int(round(a / dp)) for a in box_lo]
    b1 = [int(round(a / dp)) for a in box_hi]
    bs = [b1[k] - b0[k] for k in range(3)]
    bi = np.stack([g.ravel() for g in np.meshgrid(*[np.arange(s) for s in bs], indexing="ij")], 1)
    depth = np.minimum.reduce([bi[:, 0], bs[0] - 1 - bi[:, 0], bi[:, 1], bs[1] - 1 - bi[:, 1],
                               bs[2] - 1 - bi[:, 2]])
    band = bi[depth < NWALL]
    pos_b = (band + np.array(b0) + 0.5) * dp
    return _finish(cfg, pos_f, np.zeros(len(pos_f)), rho_f, np.concatenate([pos_w, pos_b]))


def two_phase_2d(dp=0.0125, tank=(5.366, 3.0), column=(2.0, 1.0), equal_c=False):
    """Config 2: 2-D water/air dam break, density ratio 1000, tank fully filled.
    equal_c=True is variant 2a (same c both phases); False is 2b
    (BASELINE.json: air c0 chosen so the air pressure scale matches the water's)."""
    H = column[1]
    cw = 10.0 * math.sqrt(2.0 * G0 * H)
    ca = cw if equal_c else cw * math.sqrt(1000.0)
    nx, ny = int(math.floor(tank[0] / dp + 1e-9)), int(math.floor(tank[1] / dp + 1e-9))
    top = ny * dp
    cfg = _base(2, dp, [1000.0, 1.0], [cw, ca], [0.0, -G0, 0.0], [-NWALL * dp] * 2,
                [nx * dp + NWALL * dp, top + NWALL * dp],
                name="cfg2a_two_phase_2d" if equal_c else "cfg2b_two_phase_2d", H=H,
                penalty_phase_mask=2, free_surface_mask=1)
    pos = _lattice((nx, ny), dp)
    water = (pos[:, 0] < column[0]) & (pos[:, 1] < column[1])
    p_air = 1.0 * G0 * (top - pos[:, 1])
    p_wat = 1.0 * G0 * (top - H) + 1000.0 * G0 * (H - pos[:, 1])
    rho = np.where(water, 1000.0 + p_wat / cw ** 2, 1.0 + p_air / ca ** 2)
    order = np.argsort(~water, kind="stable")  # water first
    pos, rho, tag = pos[order], rho[order], (~water[order]).astype(np.int64)
    pos_w = (_shell((nx, ny), dp) + 0.5) * dp
    return _finish(cfg, pos, tag, rho, pos_w)


def hydrostatic_tank_x1(dp=0.01, L=1.0, H=0.5, c_rule="baseline"):
    """The paper's two-phase hydrostatic tank, case X1 (section 4.1): 2-D tank of
    length L = 2H = 1 m and height L, lower half water, upper half air (density ratio 1000), both at
    rest on a Cartesian lattice, same speed of sound in both phases.  The paper's
    spacings are dx = 0.01, 0.005, 0.0025, 0.00125 m.  c_rule: "baseline" = 10 sqrt(2 g H) (BASELINE.json,
    reading A2), "paper" = 10 * 2 sqrt(g H).  Initial density hydrostatic in both phases."""
    cfg = two_phase_2d(dp=dp, tank=(L, L), column=(L, H), equal_c=True)
    cfg["name"] = "x1_hydrostatic_tank_dp%g" % dp
    if c_rule == "paper":
        c = 20.0 * math.sqrt(G0 * H)
        pos, tag = cfg["pos"].astype(np.float64), cfg["tag"]
        top = cfg["domain_max"][1] - NWALL * dp
        p = np.where(tag == 0, G0 * (top - H) + 1000.0 * G0 * (H - pos[:, 1]), G0 * (top - pos[:, 1]))
        rho = np.where(tag == 0, 1000.0, 1.0) + p / c ** 2
        cfg["rho"] = np.where(tag < 0, 1000.0, rho).astype(np.float32)
        cfg["c0"] = [c, c]
    cfg["top"] = cfg["domain_max"][1] - NWALL * dp
    return cfg


def x1_analytic_pressure(cfg, y):
    """Hydrostatic pressure of case X1 at height y (Fig. 4): p = rho_a g (top - y) above the
    interface, + (rho_w - rho_a) g (H - y) below it (p = 0 at the lid, as the linear EOS has it)."""
    y = np.asarray(y, np.float64)
    ra, rw = cfg["rho0"][1], cfg["rho0"][0]
    return ra * G0 * (cfg["top"] - y) + (rw - ra) * G0 * np.maximum(cfg["H"] - y, 0.0)


def sloshing_spheres_3d(dp=0.004, tank=(2.0, 1.0, 1.0), fill=0.4, n_spheres=8, seed=211002621):
    """Config 3: 3-D sloshing box with spherical obstacles; walls = 3-layer band of the
    signed distance to union(tank walls, spheres); gravity tilted sinusoidally."""
    H = fill * tank[2]
    c0 = 10.0 * math.sqrt(2.0 * G0 * H)
    rng = np.random.Generator(np.random.PCG64(seed))
    rad = rng.uniform(0.05, 0.15, n_spheres)
    cen = np.stack([rng.uniform(0.2, 1.8, n_spheres) * tank[0] / 2.0,
                    rng.uniform(0.15, 0.85, n_spheres) * tank[1],
                    rng.uniform(0.0, 0.5, n_spheres) * tank[2]], axis=1)
    n = [int(round(t / dp)) for t in tank]
    cfg = _base(3, dp, [1000.0], [c0], [0.0, 0.0, -G0], [-NWALL * dp] * 3,
                [t + NWALL * dp for t in tank], name="cfg3_sloshing_spheres_3d", H=H,
                g_osc_amp=[0.3 * G0, 0.0, 0.0], g_osc_period=1.5)
    cfg["spheres"] = dict(centre=cen, radius=rad)
    pos_f, pos_w = [], []
    # slab-wise over x to bound memory
    ys = (np.arange(-NWALL, n[1] + NWALL) + 0.5) * dp
    zs = (np.arange(-NWALL, n[2] + NWALL) + 0.5) * dp
    Y, Z = np.meshgrid(ys, zs, indexing="ij")
    for ix in range(-NWALL, n[0] + NWALL):
        x = (ix + 0.5) * dp
        sd = np.minimum.reduce([np.full_like(Y, min(x, tank[0] - x)), Y, tank[1] - Y, Z,
                                tank[2] - Z])
        for c, r in zip(cen, rad):
            sd = np.minimum(sd, np.sqrt((x - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2) - r)
        fl = (sd >= 0) & (Z < H)
        wl = (sd < 0) & (sd >= -NWALL * dp)
        pos_f.append(np.stack([np.full(fl.sum(), x), Y[fl], Z[fl]], 1))
        pos_w.append(np.stack([np.full(wl.sum(), x), Y[wl], Z[wl]], 1))
    pos_f, pos_w = np.concatenate(pos_f), np.concatenate(pos_w)
    rho_f = 1000.0 * (1.0 + G0 * (H - pos_f[:, 2]) / c0 ** 2)
    return _finish(cfg, pos_f, np.zeros(len(pos_f)), rho_f, pos_w)


def box_sweep_3d(n=100, dp=0.01, jitter=0.1, seed=None):
    """Config 4: closed cube, n^3 fluid particles on a lattice jittered by +-jitter*dp,
    hydrostatic density, 3-layer walls on all faces.  seed defaults to 4000 + n."""
    seed = 4000 + n if seed is None else seed
    H = n * dp
    c0 = 10.0 * math.sqrt(2.0 * G0 * H)
    cfg = _base(3, dp, [1000.0], [c0], [0.0, 0.0, -G0], [-NWALL * dp] * 3,
                [H + NWALL * dp] * 3, name="cfg4_box_%d" % n, H=H)
    rng = np.random.Generator(np.random.PCG64(seed))
    ax = (np.arange(n, dtype=np.float32) + np.float32(0.5)) * np.float32(dp)
    pos_f = np.empty((n, n, n, 3), np.float32)
    pos_f[..., 0] = ax[:, None, None]
    pos_f[..., 1] = ax[None, :, None]
    pos_f[..., 2] = ax[None, None, :]
    pos_f = pos_f.reshape(-1, 3)
    pos_f += rng.uniform(-jitter * dp, jitter * dp, pos_f.shape).astype(np.float32)
    rho_f = 1000.0 * (1.0 + G0 * (H - pos_f[:, 2].astype(np.float64)) / c0 ** 2)
    pos_w = (_shell((n, n, n), dp) + 0.5) * dp
    return _finish(cfg, pos_f, np.zeros(len(pos_f)), rho_f, pos_w)


def box_2d(n=24, dp=0.01, jitter=0.0, seed=7, two_phase=False):
    """Small closed 2-D box used by tests (same recipe as config 4, two dimensions)."""
    H = n * dp
    c0 = 10.0 * math.sqrt(2.0 * G0 * H)
    rho0 = [1000.0, 1.0] if two_phase else [1000.0]
    cfg = _base(2, dp, rho0, [c0] * len(rho0), [0.0, -G0, 0.0], [-NWALL * dp] * 2,
                [H + NWALL * dp] * 2, name="box2d_%d" % n, H=H,
                penalty_phase_mask=2 if two_phase else 0)
    rng = np.random.Generator(np.random.PCG64(seed))
    pos_f = _lattice((n, n), dp)
    pos_f = pos_f + rng.uniform(-jitter * dp, jitter * dp, pos_f.shape)
    if two_phase:
        air = pos_f[:, 1] >= 0.5 * H
        p = np.where(air, 1.0 * G0 * (H - pos_f[:, 1]),
                     1.0 * G0 * 0.5 * H + 1000.0 * G0 * (0.5 * H - pos_f[:, 1]))
        rho_f = np.where(air, 1.0, 1000.0) + p / c0 ** 2
        tag_f = air.astype(np.int64)
    else:
        rho_f = 1000.0 * (1.0 + G0 * (H - pos_f[:, 1]) / c0 ** 2)
        tag_f = np.zeros(len(pos_f))
    pos_w = (_shell((n, n), dp) + 0.5) * dp
    return _finish(cfg, pos_f, tag_f, rho_f, pos_w)


def shuffled(cfg, seed=1):
    """Same configuration with the particle order permuted (fluid and wall interleaved)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    perm = rng.permutation(len(cfg["tag"]))
    out = dict(cfg)
    for k in ("pos", "vel", "rho", "tag"):
        out[k] = np.ascontiguousarray(cfg[k][perm])
    out["perm"] = perm
    return out
