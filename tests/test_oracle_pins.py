"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Pin ids follow SURVEY.md §8(c) / DESIGN.md.  None of these compares the oracle with
itself: expected values are the paper's (tests/golden), closed forms, invariants,
lattice constants computed outside oracle/, or brute force.
"""
import math
import os

import numpy as np
import pytest

from oracle import orc
from paper_2110_02621_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def custom(dim, pos, tag, rho, vel=None, dp=1.0 / 64, rho0=(1000.0,), c0=(10.0,), g=(0, 0, 0),
           **kw):
    """Hand-built configuration (arrays given directly; no generator)."""
    pos = np.asarray(pos, np.float64)
    if pos.shape[1] == 2:
        pos = np.concatenate([pos, np.zeros((len(pos), 1))], 1)
    lo = pos.min(0) - 4 * dp
    hi = pos.max(0) + 4 * dp
    cfg = dict(dim=dim, n_phases=len(rho0), dp=dp, h=1.3 * dp, rho0=list(rho0), c0=list(c0),
               g=list(g), cfl=0.25, penalty_strength=1.0, penalty_phase_mask=0,
               free_surface_mask=1, flags=orc.FLAG_REINIT | orc.FLAG_WALL_VEL_MIRROR,
               domain_min=list(lo), domain_max=list(hi))
    cfg.update(kw)
    cfg["pos"] = pos.astype(np.float32)
    cfg["vel"] = np.zeros_like(cfg["pos"]) if vel is None else np.asarray(vel, np.float32)
    cfg["rho"] = np.asarray(rho, np.float32)
    cfg["tag"] = np.asarray(tag, np.int32)
    return cfg


def run(cfg):
    o = orc.Oracle(cfg)
    o.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    return o


def lattice(dim, n, dp):
    ax = (np.arange(n) + 0.5) * dp
    return np.stack([g.ravel() for g in np.meshgrid(*([ax] * dim), indexing="ij")], 1)


# ------------------------------------------------------------------ P1 kernel
@pytest.mark.parametrize("dim", [2, 3])
def test_P1_kernel_unit_integral_and_derivative(dim):
    h = 0.37
    r = np.linspace(0, 2 * h, 200001)
    w = np.array([orc.kernel_w(dim, h, x) for x in r[::100]])
    rr = r[::100]
    jac = 2 * math.pi * rr if dim == 2 else 4 * math.pi * rr ** 2
    integral = np.trapezoid(w * jac, rr)
    assert abs(integral - 1.0) < 1e-6
    assert orc.kernel_w(dim, h, 2 * h) == 0.0 and orc.kernel_w(dim, h, 2.5 * h) == 0.0
    assert orc.kernel_dw(dim, h, 0.0) == 0.0
    for x in (0.1 * h, 0.7 * h, 1.3 * h, 1.9 * h):
        e = 1e-6 * h
        fd = (orc.kernel_w(dim, h, x + e) - orc.kernel_w(dim, h, x - e)) / (2 * e)
        assert abs(fd - orc.kernel_dw(dim, h, x)) < 1e-6 * abs(orc.kernel_dw(dim, h, 0.7 * h))
        assert orc.kernel_dw(dim, h, x) < 0


# ------------------------------------------------------------------ P2 lattice constants
def test_P2_lattice_constants_golden():
    g = _gold("lattice_constants.txt")
    assert abs(orc.sigma0(2, 1.3, 1.0) - g["sigma0_2d"]) < 2e-9
    assert abs(orc.sigma0(3, 1.3, 1.0) - g["sigma0_3d"]) < 2e-9
    assert abs(orc.kernel_w(2, 1.3, 0.0) - g["w0_2d"]) < 2e-9
    assert abs(orc.kernel_w(3, 1.3, 0.0) - g["w0_3d"]) < 2e-9


@pytest.mark.parametrize("dim,n", [(2, 9), (3, 9)])
def test_P2_partition_of_unity_and_neighbour_count(dim, n):
    g = _gold("lattice_constants.txt")
    dp = 1.0 / 64
    pos = lattice(dim, n, dp)
    cfg = custom(dim, pos, np.zeros(len(pos)), np.full(len(pos), 1000.0), dp=dp)
    o = run(cfg)
    f = o.fields()
    centre = np.argmin(np.linalg.norm(pos - pos.mean(0), axis=1))
    key = "%dd" % dim
    assert abs(f["sigma"][centre] * dp ** dim - g["sigma0_" + key]) < 2e-9
    off, ids = o.neighbours()
    assert off[centre + 1] - off[centre] == int(g["neigh_" + key])
    # half-space sum: particle on the top face of the block sees own layer and below only
    top = np.argmin(np.linalg.norm(pos - (pos.mean(0) + np.eye(dim)[dim - 1] * (n // 2) * dp), axis=1))
    assert abs(f["sigma"][top] * dp ** dim - g["halfspace_" + key]) < 2e-9


# ------------------------------------------------------------------ P3 momentum sum
@pytest.mark.parametrize("dim", [2, 3])
def test_P3_linear_pressure_gives_M1_gradient(dim):
    """Eq. 2.10 on a full lattice with an (almost) uniform density and a linear p:
    a = -M1 grad p / rho, M1 the first-moment lattice constant."""
    g = _gold("lattice_constants.txt")
    dp, n, c = 1.0 / 64, 9, 10.0
    pos = lattice(dim, n, dp)
    k = np.round(pos[:, 0] / dp - 0.5)
    rho = 1000.0 + k * 2.0 ** -10            # exactly representable in float32
    o = run(custom(dim, pos, np.zeros(len(pos)), rho, dp=dp, c0=(c,)))
    f = o.fields()
    centre = np.argmin(np.linalg.norm(pos - pos.mean(0), axis=1))
    gradp = c * c * 2.0 ** -10 / dp
    expect = -g["M1_%dd" % dim] * gradp / rho[centre]
    assert abs(f["acc"][centre, 0] - expect) < 2e-5 * abs(expect)
    assert np.all(np.abs(f["acc"][centre, 1:]) < 1e-9 * abs(expect))


@pytest.mark.parametrize("dim", [2, 3])
def test_P7_linear_velocity_gives_M1_divergence(dim):
    """Eq. 2.9 with uniform p, rho reduces to Eq. 2.5: d rho/dt = -rho M1 div v."""
    g = _gold("lattice_constants.txt")
    dp, n, A = 1.0 / 64, 9, 0.5
    pos = lattice(dim, n, dp)
    vel = np.zeros((len(pos), 3))
    vel[:, 0] = A * pos[:, 0]
    vel[:, 1] = -0.25 * A * pos[:, 1]
    o = run(custom(dim, pos, np.zeros(len(pos)), np.full(len(pos), 1000.0), vel=vel, dp=dp,
                   flags=0))
    o.step(1, dts=[1e-13])
    f = o.fields()
    centre = np.argmin(np.linalg.norm(pos - pos.mean(0), axis=1))
    expect = -1000.0 * g["M1_%dd" % dim] * (A - 0.25 * A)
    assert abs(f["drho"][centre] - expect) < 1e-6 * abs(expect)


# ------------------------------------------------------------------ P4 wall extrapolation
@pytest.mark.parametrize("multi", [False, True])
def test_P4_wall_pressure_exact_for_linear_hydrostatic_field(multi):
    dp, nx, K, c = 1.0 / 64, 12, 10, 10.0
    fl = lattice(2, nx, dp)
    fl = fl[fl[:, 1] < K * dp]
    k = np.round(fl[:, 1] / dp - 0.5)
    rho_f = 1000.0 + (K - k) * 2.0 ** -10
    gmag = c * c * 2.0 ** -10 / (dp * 1000.0)
    H = (K + 0.5) * dp
    wl = np.array([[(i + 0.5) * dp, -(j + 0.5) * dp] for i in range(nx) for j in range(3)])
    pos = np.concatenate([fl, wl])
    tag = np.concatenate([np.zeros(len(fl)), -np.ones(len(wl))])
    rho = np.concatenate([rho_f, np.full(len(wl), 1000.0)])
    kw = dict(rho0=(1000.0, 1.0), c0=(c, c)) if multi else dict(c0=(c,))
    o = run(custom(2, pos, tag, rho, dp=dp, g=(0, -gmag, 0), **kw))
    f = o.fields()
    pw = f["p"][len(fl):]
    expect = 1000.0 * gmag * (H - wl[:, 1])
    # rho_f is uniform to 1e-5, so Eq. 2.12 reproduces the linear field to that level
    near = wl[:, 1] > -2.4 * dp                  # the third layer has no fluid neighbour
    assert np.max(np.abs(pw - expect)[near]) < 3e-5 * expect.max()
    assert np.all(pw[~near] == 0.0)              # reading A7
    # dropping the lever term would miss by more than one lattice unit of pressure
    assert 1000.0 * gmag * dp > 1e3 * 3e-5 * expect.max() / 40


# ------------------------------------------------------------------ P5 / P17 whole step
def test_P5_resting_column_relaxes_to_hydrostatic_and_P17_mass():
    """BASELINE.json north_star: closed-form p = rho0 g (H - z) in a resting column
    (PAPER.md:224).  The scheme is low-dissipation, so the column rings acoustically about
    the hydrostatic state; the time average over the ringing is compared."""
    cfg = inputs.dam_break_2d(dp=0.02, tank=(0.6, 0.9), column=(0.6, 0.6))
    o = run(cfg)
    nf, H = cfg["n_fluid"], cfg["H"]
    m0 = o.stats()["mass"]
    o.step(1000)
    psum, cnt = np.zeros(nf), 0
    for _ in range(40):
        o.step(50)
        psum += o.fields()["p"][:nf]
        cnt += 1
    f = o.fields()
    y = f["pos"][:nf, 1]
    pa = 1000.0 * 9.81 * (H - y)
    pavg = psum / cnt
    rel = math.sqrt(np.mean((pavg - pa) ** 2)) / (1000.0 * 9.81 * H)
    assert rel < 0.03
    slope = np.polyfit(y, pavg, 1)[0]
    assert abs(slope / (-1000.0 * 9.81) - 1.0) < 0.03
    s = o.stats()
    assert s["mass"] == m0 and abs(m0 - 1000.0 * cfg["dp"] ** 2 * nf) < 1e-9 * m0
    assert s["escaped"] == 0
    assert np.abs(f["vel"][:nf]).max() < 0.1 * math.sqrt(9.81 * H)


def test_P14_potential_energy_of_paper_column():
    """T_tot = 1226.25 J for L = 1 m, H = 0.5 m of water; the lattice
    midpoint rule is exact for a linear integrand, for every dp of PAPER.md:222."""
    T = _gold("paper_values.txt")["T_tot_J"]
    for dp in (0.01, 0.005):
        cfg = inputs.dam_break_2d(dp=dp, tank=(1.0, 1.0), column=(1.0, 0.5))
        nf = cfg["n_fluid"]
        m = 1000.0 * dp ** 2
        ep = np.sum(m * 9.81 * cfg["pos"][:nf, 1].astype(np.float64))
        assert abs(ep - T) < 1e-4 * T
    o = run(inputs.dam_break_2d(dp=0.02, tank=(1.0, 1.0), column=(1.0, 0.5)))
    assert abs(o.stats()["mass"] - 1000.0 * 1.0 * 0.5) < 1e-9


# ------------------------------------------------------------------ P6 neighbour search
def test_P6_cell_list_equals_brute_force():
    cfg = inputs.dam_break_2d()
    o = run(cfg)
    o.step(150)
    a, b = o.neighbours(), o.neighbours_bruteforce()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    cfg = inputs.box_sweep_3d(n=8)
    o = run(cfg)
    a, b = o.neighbours(), o.neighbours_bruteforce()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    assert o.stats()["npairs"] == int((a[0][1:] - a[0][:-1])[:cfg["n_fluid"]].sum())


def test_f32_contract_grid_walk_equals_brute_force():
    for cfg in (inputs.dam_break_2d(), inputs.box_sweep_3d(n=10), inputs.shuffled(inputs.box_2d(n=20, jitter=0.3))):
        a = orc.f32_neighbours(cfg, cfg["pos"], cfg["tag"], grid=False)
        b = orc.f32_neighbours(cfg, cfg["pos"], cfg["tag"], grid=True)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
        cell_id, perm, cs, ce = orc.f32_cells(cfg, cfg["pos"], cfg["tag"])
        n = len(cfg["tag"])
        assert sorted(perm.tolist()) == list(range(n))
        nf = int((cfg["tag"] >= 0).sum())
        for blk in (perm[:nf], perm[nf:]):
            key = cell_id[blk].astype(np.int64) * n + blk
            assert np.all(np.diff(key) > 0)          # sorted by cell, ids ascending within


# ------------------------------------------------------------------ P7 / P18 Riemann terms
def test_P7_riemann_reduces_to_plain_averages():
    s = orc.riemann(1000.0, -0.3, 5000.0, 40.0, 1000.0, 0.2, 5000.0, 40.0)
    assert s["pstar"] == 5000.0                     # U_L <= U_R: beta = 0
    assert abs(s["Ustar"] - (-0.05)) < 1e-15
    s = orc.riemann(1000.0, 0.3, 5000.0, 40.0, 1000.0, -0.2, 7000.0, 40.0)
    # Eq. 2.8 by hand: beta = min(1.5, 40) = 1.5
    assert abs(s["pstar"] - (6000.0 + 500.0 * 1.5 * 0.5)) < 1e-9
    assert abs(s["Ustar"] - (0.05 + 0.5 * (-2000.0) / (40.0 * 1000.0))) < 1e-15
    # limiter saturates at c
    s = orc.riemann(1000.0, 30.0, 0.0, 40.0, 1000.0, -30.0, 0.0, 40.0)
    assert abs(s["pstar"] - 500.0 * 40.0 * 60.0) < 1e-6


def test_P18_acoustic_extension_equals_paper_at_equal_c():
    rng = np.random.default_rng(3)
    for _ in range(50):
        rL, rR = rng.uniform(0.5, 1200.0, 2)
        UL, UR = rng.uniform(-3, 3, 2)
        pL, pR = rng.uniform(-1e3, 1e4, 2)
        c = rng.uniform(10, 100)
        a = orc.riemann(rL, UL, pL, c, rR, UR, pR, c, mode=1)
        b = orc.riemann(rL, UL, pL, c, rR, UR, pR, c, mode=2)
        for k in a:
            assert abs(a[k] - b[k]) <= 1e-12 * max(1.0, abs(a[k]))
    # symmetric under exchange of the two particles: p*(L,R) = p*(R,L) with
    # U -> -U (e_ji = -e_ij)
    a = orc.riemann(1000.0, 0.4, 3e3, 44.0, 1.2, -0.7, 1e3, 1400.0)
    b = orc.riemann(1.2, 0.7, 1e3, 1400.0, 1000.0, -0.4, 3e3, 44.0)
    assert abs(a["pstar"] - b["pstar"]) < 1e-9 * abs(a["pstar"])
    assert abs(a["Ustar"] + b["Ustar"]) < 1e-12


# ------------------------------------------------------------------ P8 antisymmetry
@pytest.mark.parametrize("dim,two_phase", [(2, False), (3, False), (2, True)])
def test_P8_total_momentum_of_internal_forces_vanishes(dim, two_phase):
    rng = np.random.default_rng(11)
    dp = 1.0 / 64
    pos = lattice(dim, 6, dp) + rng.uniform(-0.2 * dp, 0.2 * dp, (6 ** dim, dim))
    n = len(pos)
    vel = np.zeros((n, 3))
    vel[:, :dim] = rng.uniform(-1, 1, (n, dim))
    if two_phase:
        tag = (pos[:, 1] > 3 * dp).astype(int)
        rho0, c0 = (1000.0, 1.0), (20.0, 20.0 * math.sqrt(1000.0))
        rho = np.where(tag == 0, 1000.0, 1.0) * (1 + rng.uniform(0, 0.01, n))
    else:
        tag, rho0, c0 = np.zeros(n, int), (1000.0,), (20.0,)
        rho = 1000.0 * (1 + rng.uniform(0, 0.01, n))
    o = run(custom(dim, pos, tag, rho, vel=vel, dp=dp, rho0=rho0, c0=c0))
    f = o.fields()
    m = np.array(rho0)[tag] * dp ** dim
    tot = (m[:, None] * f["acc"]).sum(0)
    scale = np.abs(m[:, None] * f["acc"]).sum()
    assert np.all(np.abs(tot) < 1e-12 * scale)
    # two isolated particles: m_i a_i = -m_j a_j exactly as vectors
    p2 = np.array([[0.0] * dim, [1.1 * dp] + [0.3 * dp] * (dim - 1)])
    v2 = np.zeros((2, 3)); v2[0, 0], v2[1, 0] = 0.7, -0.4
    o = run(custom(dim, p2, tag[:2] * 0, [1004.0, 1001.0], vel=v2, dp=dp, c0=(20.0,)))
    a = o.fields()["acc"]
    assert np.allclose(a[0], -a[1], rtol=1e-13, atol=0) and abs(a[0, 0]) > 0


# ------------------------------------------------------------------ P9 / P10
def test_P9_continuity_scalar_identity_two_particles():
    """(v_i - v*).grad_i W_ij = (U* - U_L) W'(r) because v*.e = U* (SURVEY P9); with
    U* - U_L = [(p_i - p_j)/c - rho_j v_ij.e] / (rho_i + rho_j) for equal c."""
    dp, c = 1.0 / 64, 20.0
    f32 = lambda a: np.asarray(a, np.float32).astype(np.float64)   # the oracle sees float32 inputs
    pos = f32([[0.0, 0.0, 0.0], [0.9 * dp, 0.5 * dp, -0.4 * dp]])
    vel = f32([[0.3, -0.2, 0.5], [-0.1, 0.4, 0.2]])
    rho = np.array([1003.0, 1001.0])
    o = run(custom(3, pos, [0, 0], rho, vel=vel, dp=dp, c0=(c,), flags=0))
    o.step(1, dts=[1e-14])
    d = pos[0] - pos[1]
    r = np.linalg.norm(d)
    e = -d / r
    p = c * c * (rho - 1000.0)
    vij_e = (vel[0] - vel[1]) @ e
    dU = ((p[0] - p[1]) / c - rho[1] * vij_e) / (rho[0] + rho[1])
    V1 = 1000.0 * dp ** 3 / rho[1]
    expect = 2 * rho[0] * V1 * dU * orc.kernel_dw(3, 1.3 * dp, r)
    got = o.fields()["drho"][0]
    assert abs(got - expect) < 1e-9 * abs(expect)


def test_P10_galilean_invariance():
    rng = np.random.default_rng(5)
    dp = 1.0 / 64
    pos = lattice(3, 5, dp) + rng.uniform(-0.2 * dp, 0.2 * dp, (125, 3))
    vel = rng.uniform(-1, 1, (125, 3))
    rho = 1000.0 * (1 + rng.uniform(0, 0.01, 125))
    out = []
    for boost in (np.zeros(3), np.array([3.0, -2.0, 1.0])):
        o = run(custom(3, pos, np.zeros(125), rho, vel=vel + boost, dp=dp, c0=(20.0,), flags=0))
        a0 = o.fields()["acc"].copy()
        o.step(1, dts=[1e-14])
        out.append((a0, o.fields()["drho"].copy()))
    assert np.allclose(out[0][0], out[1][0], rtol=0, atol=1e-5 * np.abs(out[0][0]).max())
    assert np.allclose(out[0][1], out[1][1], rtol=0, atol=1e-5 * np.abs(out[0][1]).max())
    # uniform v, p, rho on a lattice: d rho/dt = 0
    pos = lattice(3, 7, dp)
    o = run(custom(3, pos, np.zeros(343), np.full(343, 1002.0), vel=np.tile([1.0, 2.0, 3.0], (343, 1)),
                   dp=dp, c0=(20.0,), flags=0))
    o.step(1, dts=[1e-14])
    assert np.abs(o.fields()["drho"]).max() < 1e-6      # pair terms are O(1e3) each


def test_P11_tangential_flow_along_mirror_wall_keeps_density():
    dp, nx = 1.0 / 64, 15
    fl = lattice(2, nx, dp)
    fl = fl[fl[:, 1] < 6 * dp]
    wl = np.array([[(i + 0.5) * dp, -(j + 0.5) * dp] for i in range(nx) for j in range(3)])
    pos = np.concatenate([fl, wl])
    tag = np.concatenate([np.zeros(len(fl)), -np.ones(len(wl))])
    vel = np.zeros((len(pos), 3)); vel[:len(fl), 0] = 0.8
    o = run(custom(2, pos, tag, np.full(len(pos), 1002.0), vel=vel, dp=dp, c0=(20.0,), flags=orc.FLAG_WALL_VEL_MIRROR))
    o.step(1, dts=[1e-14])
    f = o.fields()
    centre = np.argmin(np.linalg.norm(fl - np.array([nx / 2 * dp, 0.5 * dp]), axis=1))
    assert abs(f["drho"][centre]) < 1e-8
    # the mirrored wall velocity is minus the fluid's tangential velocity
    wc = len(fl) + np.argmin(np.linalg.norm(wl - np.array([nx / 2 * dp, -0.5 * dp]), axis=1))
    assert abs(f["vel"][wc, 0] + float(np.float32(0.8))) < 1e-12


# ------------------------------------------------------------------ P12 integrator
def test_P12_free_fall_is_exact_and_dt_body_force():
    dp, g = 0.05, 9.81
    v0 = np.array([[0.25, 0.125, 0.0]])     # exactly representable in float32
    cfg = custom(3, np.array([[0.0, 0.0, 10.0]]), [0], [1000.0], vel=v0, dp=dp, c0=(0.05,), g=(0, 0, -g),
                 domain_min=[-5, -5, -5], domain_max=[5, 5, 15])
    o = run(cfg)
    dts = o.step(7)
    assert abs(dts[0] - 0.25 * math.sqrt(1.3 * dp / g)) < 1e-15
    t = dts.sum()
    f = o.fields()
    expect = np.array([0.25 * t, 0.125 * t, 10.0 - 0.5 * g * t * t])
    assert np.allclose(f["pos"][0], expect, rtol=0, atol=1e-12)
    assert np.allclose(f["vel"][0], [0.25, 0.125, -g * t], rtol=0, atol=1e-12)
    # CFL branch, Eq. 2.23 with U_max = current max |v| (reading A17)
    cfg = custom(3, np.array([[0.0, 0.0, 0.0]]), [0], [1000.0], vel=[[3.0, 4.0, 0.0]], dp=dp, c0=(50.0,))
    assert abs(run(cfg).step(1)[0] - 0.25 * 1.3 * dp / 55.0) < 1e-15


# ------------------------------------------------------------------ P13 reinitialisation
def test_P13_reinitialisation_cases():
    s0 = 1.0095
    assert orc.reinit_density(1001.0, 1000.0, 1.002 * s0, s0, 1) == pytest.approx(1002.0, abs=1e-10)
    got = orc.reinit_density(1004.0, 1000.0, 0.6 * s0, s0, 1)   # free surface: rho_s < rho*
    assert got == pytest.approx(600.0 + 404.0 * 1000.0 / 1004.0, abs=1e-10)
    lo = orc.reinit_density(1003.0, 1000.0, 1.003 * s0 * (1 - 1e-12), s0, 1)
    hi = orc.reinit_density(1003.0, 1000.0, 1.003 * s0 * (1 + 1e-12), s0, 1)
    assert abs(lo - hi) < 1e-6                                   # continuous at rho_s = rho*
    assert orc.reinit_density(1004.0, 1.0, 0.9 * s0, s0, 0) == pytest.approx(0.9, abs=1e-12)  # Eq. 2.18


# ------------------------------------------------------------------ P15 penalty
def _wall_patch(nx, dp):
    return np.array([[(i + 0.5) * dp, -(j + 0.5) * dp] for i in range(nx) for j in range(3)])


def test_P15_penalty_zero_on_lattice_and_pushes_along_normal():
    dp, nx, c = 1.0 / 64, 13, 20.0
    wl = _wall_patch(nx, dp)
    x0 = (nx // 2 + 0.5) * dp

    def acc(y, mask, rho=1003.0):
        pos = np.concatenate([[[x0, y]], wl])
        tag = np.concatenate([[0], -np.ones(len(wl))])
        rho_a = np.concatenate([[rho], np.full(len(wl), 1000.0)])
        return run(custom(2, pos, tag, rho_a, dp=dp, c0=(c,), penalty_phase_mask=mask)).fields()["acc"][0]

    # undisturbed lattice position: normal distance dp >= dp/2 -> no penalty
    assert np.array_equal(acc(0.5 * dp, 1), acc(0.5 * dp, 0))
    assert np.array_equal(acc(0.0 * dp + 1e-9, 1), acc(0.0 * dp + 1e-9, 0))   # exactly dp/2 away
    # closer than dp/2 to the first layer: extra push along +n_w = +y, none along x
    d = acc(-0.2 * dp, 1) - acc(-0.2 * dp, 0)
    assert d[1] > 0 and abs(d[0]) < 1e-9 * d[1]
    # closed form of reading A8/A9b for this geometry (flat wall, n = (0,1)):
    # sum over first-layer particles of 2 V0/rho_i * gamma*(1-delta)^2*|p_i s| * |W'(r)|
    rho_i, y = 1003.0, -0.2 * dp
    p_i = c * c * (rho_i - 1000.0)
    tot = 0.0
    for w in wl[np.isclose(wl[:, 1], -0.5 * dp)]:
        dvec = np.array([x0, y]) - w
        r = np.linalg.norm(dvec)
        if r >= 2.6 * dp:
            continue
        delta = 2 * dvec[1] / dp
        if -1 < delta < 1:
            tot += 2 * dp ** 2 / rho_i * (1 - delta) ** 2 * abs(p_i * dvec[1] / r) * -orc.kernel_dw(2, 1.3 * dp, r)
    assert tot > 0 and abs(d[1] - tot) < 1e-6 * tot      # float32-rounded input positions
    # scales linearly with gamma_p and vanishes with p_i
    assert np.allclose(acc(-0.2 * dp, 1, rho=1000.0), acc(-0.2 * dp, 0, rho=1000.0))


# ------------------------------------------------------------------ P16 normals
def test_P16_wall_normals():
    cfg = inputs.dam_break_2d()
    o = run(cfg)
    n, pos, dp = o.normals(), cfg["pos"].astype(np.float64), cfg["dp"]

    def at(x, y):
        i = np.argmin(np.abs(pos[:, 0] - x * dp) + np.abs(pos[:, 1] - y * dp))
        assert cfg["tag"][i] == -1
        return n[i]

    assert np.allclose(at(40.5, -0.5), [0, 1, 0], atol=2e-5)        # floor, first layer: into fluid
    assert np.allclose(at(40.5, -1.5), [0, 0, 0], atol=0)            # middle layer: degenerate -> 0
    assert np.allclose(at(40.5, -2.5), [0, -1, 0], atol=2e-5)       # outer layer: away from the wall bulk
    assert np.allclose(at(-0.5, 30.5), [1, 0, 0], atol=2e-5)        # left wall
    assert np.allclose(at(-0.5, -0.5), [math.sqrt(0.5)] * 2 + [0], atol=2e-5)   # corner -> diagonal
    assert np.all(n[cfg["tag"] >= 0] == 0)


def test_long_run_keeps_particles_inside_P17():
    cfg = inputs.dam_break_2d()
    o = run(cfg)
    o.step(1500)
    s = o.stats()
    assert s["escaped"] == 0 and s["mass"] == pytest.approx(2000.0, rel=1e-12)
    assert 1.2 < s["x_front"] < 4.0 and s["ek"] > 0


# ------------------------------------------------------------------------- probes (readings A29, A30)
def _lattice_block(dim, n, dp):
    ax = (np.arange(n) + 0.5) * dp
    g = np.meshgrid(*([ax] * dim), indexing="ij")
    pos = np.stack([a.ravel() for a in g], 1)
    if dim == 2:
        pos = np.concatenate([pos, np.zeros((len(pos), 1))], 1)
    return pos


@pytest.mark.parametrize("dim", [2, 3])
def test_P19_pressure_probe_constant_linear_and_kernel_values(dim):
    """oracle/probes.py, reading A29.  (i) Normalised average of a constant is the constant at any
    point; (ii) of a field linear in the coordinates, at a point about which the lattice is
    symmetric (a particle site or a cell centre), the field's value there — the first moments cancel
    by symmetry; (iii) the kernel it uses has the Wendland C2 values W(0) = alpha_d and
    W(h) = alpha_d (1/2)^4 * 3 and vanishes at 2h (closed forms, not the oracle's C routine);
    (iv) no fluid within 2h gives 0; walls do not count."""
    from oracle import probes
    dp, n = 0.02, 12
    h = 1.3 * dp
    pos = _lattice_block(dim, n, dp)
    tag = np.zeros(len(pos), np.int32)
    cfg = dict(dim=dim, h=h, dp=dp)
    up = dim - 1
    rng = np.random.default_rng(5)
    pts = np.zeros((4, 3))
    pts[:, :dim] = 0.5 * n * dp + (rng.random((4, dim)) - 0.5) * 2 * dp
    pc, ws = probes.pressure_probes(cfg, pos, np.full(len(pos), 123.5), tag, pts)
    assert np.allclose(pc, 123.5, rtol=1e-13) and np.all(ws > 0)
    # linear field a + b.x at a site and at a cell centre
    b = np.array([3.0, -7.0, 11.0])[:dim]
    field = 5.0 + pos[:, :dim] @ b
    site = np.zeros(3); site[:dim] = (n // 2 + 0.5) * dp          # an interior particle site
    centre = site.copy(); centre[:dim] += 0.5 * dp
    for x in (site, centre):
        got, _ = probes.pressure_probes(cfg, pos, field, tag, x[None, :])
        assert got[0] == pytest.approx(5.0 + x[:dim] @ b, rel=1e-12)
    alpha = 7.0 / (4 * math.pi * h * h) if dim == 2 else 21.0 / (16 * math.pi * h ** 3)
    assert probes.wendland_c2(0.0, h, dim) == pytest.approx(alpha, rel=1e-14)
    assert probes.wendland_c2(h, h, dim) == pytest.approx(alpha * 3.0 / 16.0, rel=1e-14)
    assert probes.wendland_c2(2.0 * h, h, dim) == 0.0 and probes.wendland_c2(1.999 * h, h, dim) > 0.0
    # one particle: the sum of weights at distance r is W(r), the average is its pressure
    one = np.zeros((1, 3)); x = np.zeros((1, 3)); x[0, 0] = 0.7 * h
    got, ws = probes.pressure_probes(cfg, one, np.array([42.0]), np.zeros(1, np.int32), x)
    assert got[0] == pytest.approx(42.0) and ws[0] == pytest.approx(alpha * (1 - 0.35) ** 4 * (1 + 1.4), rel=1e-13)
    far = np.full((1, 3), 10.0); far[0, 2] = 0.0 if dim == 2 else 10.0
    got, ws = probes.pressure_probes(cfg, pos, field, tag, far)
    assert got[0] == 0.0 and ws[0] == 0.0
    got, ws = probes.pressure_probes(cfg, pos, field, np.full(len(pos), -1, np.int32), site[None, :])
    assert got[0] == 0.0 and ws[0] == 0.0


@pytest.mark.parametrize("dim", [2, 3])
def test_P20_wave_gauge_of_a_resting_block(dim):
    """oracle/probes.py, reading A30: a block of n layers at spacing dp whose lowest layer sits at
    dp/2 gauges n dp = H; only phase 0 counts; a gauge with no particle within h horizontally is NaN."""
    from oracle import probes
    dp, n = 0.05, 8
    pos = _lattice_block(dim, n, dp)
    cfg = dict(dim=dim, h=1.3 * dp, dp=dp)
    up = dim - 1
    tag = np.zeros(len(pos), np.int32)
    pts = np.zeros((2, 3)); pts[0, :up] = 0.5 * n * dp; pts[1, :up] = -3.0
    eta = probes.wave_gauges(cfg, pos, tag, pts)
    assert eta[0] == pytest.approx(n * dp, rel=1e-14) and np.isnan(eta[1])
    tag2 = tag.copy(); tag2[pos[:, up] > 0.5 * n * dp] = 1            # upper half is the light phase
    eta = probes.wave_gauges(cfg, pos, tag2, pts)
    assert eta[0] == pytest.approx(0.5 * n * dp, rel=1e-14)


# ------------------------------------------------------------------------- NEXT-1: moving walls (oracle side)
def test_P21_wall_kinematics_and_accelerating_frame_wall_pressure():
    """PAPER.md:116 (a_w in Eq. 2.12), :252 (x = A0 sin(2 pi f0 t)).
    (i) Kinematics: after steps of given dt the wall particles sit at x(t_start) + A [sin(w t) - sin(w t_start)],
    fluid-independent (closed form).
    (ii) Eq. 2.12 with a_w: a tank accelerating upwards with a_w = gmag in zero gravity holds the same
    hydrostatic field as the tank at rest under gravity -gmag, so the wall pressures must equal pin P4's
    closed form rho0 gmag (H - y_w): t_start = 3T/4 gives a_w = +A w^2, v_wall = 0."""
    dp, nx, K, c = 1.0 / 64, 12, 10, 10.0
    fl = lattice(2, nx, dp)
    fl = fl[fl[:, 1] < K * dp]
    k = np.round(fl[:, 1] / dp - 0.5)
    rho_f = 1000.0 + (K - k) * 2.0 ** -10
    gmag = c * c * 2.0 ** -10 / (dp * 1000.0)
    H = (K + 0.5) * dp
    wl = np.array([[(i + 0.5) * dp, -(j + 0.5) * dp] for i in range(nx) for j in range(3)])
    pos = np.concatenate([fl, wl])
    tag = np.concatenate([np.zeros(len(fl)), -np.ones(len(wl))])
    rho = np.concatenate([rho_f, np.full(len(wl), 1000.0)])
    f0 = 2.0
    w = 2.0 * math.pi * f0
    A = gmag / (w * w)
    cfg = custom(2, pos, tag, rho, dp=dp, g=(0, 0, 0), c0=(c,), wall_osc_amp=(0.0, A, 0.0), wall_osc_freq=f0,
                 t_start=0.75 / f0)
    o = run(cfg)
    pw = o.fields()["p"][len(fl):]
    expect = 1000.0 * gmag * (H - wl[:, 1])
    near = wl[:, 1] > -2.4 * dp
    assert np.max(np.abs(pw - expect)[near]) < 3e-5 * expect.max()
    # without the a_w term the lever vanishes (g = 0) and the miss is of the size of the term itself
    o_static = run(custom(2, pos, tag, rho, dp=dp, g=(0, 0, 0), c0=(c,)))
    pw0 = o_static.fields()["p"][len(fl):]
    assert np.max(np.abs(pw0 - expect)[near]) > 100 * 3e-5 * expect.max()
    # (i) kinematics over three steps of unequal dt
    dts = np.array([1.0e-4, 2.5e-4, 0.7e-4])
    x0 = o.fields()["pos"][len(fl):].copy()
    o.step(3, dts=dts)
    t0, t1 = 0.75 / f0, 0.75 / f0 + dts.sum()
    x1 = o.fields()["pos"][len(fl):]
    assert np.allclose(x1[:, 1] - x0[:, 1], A * (math.sin(w * t1) - math.sin(w * t0)), rtol=0, atol=1e-15)
    assert np.array_equal(x1[:, 0], x0[:, 0])


def test_P22_fluid_moving_with_the_walls_feels_no_wall_motion():
    """Mirror velocity with a moving wall (reading A6, v_w = 2 v_wall - <v_f>) and Galilean invariance:
    at t = 0 the wall velocity is A w e_x and a_w = 0; a fluid moving uniformly with that velocity must
    get the density rates (Eq. 2.9, the only place the wall velocity enters: Eq. 2.11 has no velocity
    term, reading A20) and the accelerations of the same fluid at rest between walls at rest."""
    cfg0 = inputs.dam_break_2d(dp=0.05, tank=(1.0, 0.8), column=(1.0, 0.4))
    dt = np.array([1.0e-9])

    def rates(cfg):
        o = run(cfg)
        o.step(1, dts=dt)
        f = o.fields()
        return f["drho"], f["acc"]

    d0, a0 = rates(cfg0)
    f0, A = 1.5, 0.02
    u = A * 2.0 * math.pi * f0
    vel = cfg0["vel"].copy()
    vel[cfg0["tag"] >= 0, 0] = np.float32(u)
    cfg1 = dict(cfg0, wall_osc_amp=(A, 0.0, 0.0), wall_osc_freq=f0, vel=vel)
    d1, a1 = rates(cfg1)
    fl = cfg0["tag"] >= 0
    sa = np.abs(a0[fl]).max()
    sd = 1000.0 * u / cfg0["h"]          # size of a density rate that a relative velocity u would cause
    # u is rounded to float32 on input, the wall moves with the float64 value: residual relative motion 1e-8 u
    assert np.max(np.abs(a1[fl] - a0[fl])) < 1e-6 * sa
    assert np.max(np.abs(d1[fl] - d0[fl])) < 1e-6 * sd
    # with the walls at rest the same moving fluid is compressed against them (the pin is not vacuous)
    d2, _ = rates(dict(cfg0, vel=vel))
    assert np.max(np.abs(d2[fl] - d0[fl])) > 1e-2 * sd


# ------------------------------------------------------------------ P23-P25: what round 1 left unpinned
def _two_phase_lattice(n=24, dp=1.0 / 64, rho_w=1005.0, rho_a=1.3, **kw):
    """Unperturbed two-phase box (water below y = H/2, air above), every particle given one
    off-reference density per phase so that each formula leaves a distinct value."""
    cfg = dict(inputs.box_2d(n=n, dp=dp, jitter=0.0, two_phase=True))
    rho = np.where(cfg["tag"] == 0, rho_w, np.where(cfg["tag"] == 1, rho_a, 1000.0)).astype(np.float32)
    cfg["rho"] = rho
    cfg["g"] = [0.0, 0.0, 0.0]
    cfg.update(kw)
    return cfg


def test_P23_two_phase_step_dispatch_reinit_and_density_update():
    """Readings A13 / A13b / A15 inside orc.step (the dispatch, not the kernel): one step with dt = 0 on
    the unperturbed two-phase lattice leaves the positions alone, so every density follows by hand from
    the lattice constants of pin P2 (tests/golden/lattice_constants.txt, computed outside oracle/):
      water, bulk          sigma (own phase + walls) = sigma0          -> Eq. 2.17 with rho_s = rho0 < rho*:
                           rho = rho0 + (rho* - rho0) rho0 / rho*      (continuity adds dt * drho = 0)
      water, interface row sigma = half-space sum (own row and below)  -> rho_s = rho0 * halfspace / sigma0
      air (any)            sigma over every neighbour = sigma0         -> Eq. 2.4 / 2.18: rho = rho0_air,
                           whatever rho* was (summation overwrites)
    A wrong phase in either dispatch, the light phase counted in the water's sigma, or Eq. 2.18 on the water
    changes one of these values by >= 0.5 %."""
    gold = _gold("lattice_constants.txt")
    n, dp = 24, 1.0 / 64
    rw, ra = 1005.0, 1.3
    cfg = _two_phase_lattice(n, dp, rw, ra)
    o = run(cfg)
    o.step(1, dts=[0.0])
    f = o.fields()
    y = cfg["pos"][:, 1].astype(np.float64)
    tag = cfg["tag"]
    H = n * dp
    water, air = tag == 0, tag == 1
    x = cfg["pos"][:, 0].astype(np.float64)
    # interface row away from the side walls (the wall particles above the interface still count for a water particle)
    top_row = water & (np.abs(y - (0.5 * H - 0.5 * dp)) < 1e-6) & (x > 3 * dp) & (x < H - 3 * dp)
    bulk = water & (y < 0.5 * H - 3 * dp)
    assert top_row.sum() == n - 6 and bulk.sum() == n * (n // 2 - 3)
    want_bulk = 1000.0 + (rw - 1000.0) * 1000.0 / rw
    assert np.max(np.abs(f["rho"][bulk] - want_bulk)) < 1e-6
    rs = 1000.0 * gold["halfspace_2d"] / gold["sigma0_2d"]
    want_top = rs + (rw - rs) * 1000.0 / rw
    assert np.max(np.abs(f["rho"][top_row] - want_top)) < 1e-4     # golden constants carry 9 digits
    assert np.max(np.abs(f["rho"][air] - 1.0)) < 2e-9              # sigma0 is a 20-neighbour sum
    # Eq. 2.3 with each phase's own rho0 (c equal here)
    c2 = cfg["c0"][0] ** 2
    assert np.max(np.abs(f["p"][bulk] - c2 * (want_bulk - 1000.0))) < 1e-6 * c2
    assert np.max(np.abs(f["p"][air])) < 1e-8 * c2
    # the study-only variants really are the other readings (they must NOT reproduce the values above)
    o2 = run(dict(cfg, oracle_variant=orc.VAR_SIGMA_ALL))
    o2.step(1, dts=[0.0])
    assert np.max(np.abs(o2.fields()["rho"][top_row] - want_bulk)) < 1e-6      # air counted: no deficiency
    o3 = run(dict(cfg, oracle_variant=orc.VAR_SUM_RAW))
    o3.step(1, dts=[0.0])
    assert np.max(np.abs(o3.fields()["rho"][air] - gold["sigma0_2d"])) < 2e-9  # Eq. 2.4 raw: m sigma = rho0 V0 sigma0
    o4 = run(dict(cfg, oracle_variant=orc.VAR_REINIT_LITERAL))
    o4.step(1, dts=[0.0])
    assert np.max(np.abs(o4.fields()["rho"][bulk] - 1000.0)) < 1e-6            # Eq. 2.18 on the water


def test_P24_stats_kinetic_energy_and_front_closed_form():
    """orc.stats: E_k = 1/2 M |v|^2 for a uniformly moving block, mass = N rho0 dp^d, x_front = the
    largest x of the phase-0 particles within 3 dp of the floor: all closed forms of the generator's
    lattice (config 0: column 20 x 40 sites of dp = 0.05 from the corner, PAPER.md:244 for the energy
    definition)."""
    cfg = dict(inputs.dam_break_2d())
    v = np.array([0.3, -0.4, 0.0], np.float32)
    vel = np.zeros_like(cfg["pos"])
    vel[cfg["tag"] >= 0] = v
    cfg["vel"] = vel
    o = run(cfg)
    s = o.stats()
    nf, dp = cfg["n_fluid"], cfg["dp"]
    M = nf * 1000.0 * dp * dp
    assert nf == 800 and abs(s["mass"] - M) < 1e-9 * M
    v64 = v.astype(np.float64)
    assert abs(s["ek"] - 0.5 * M * float(v64 @ v64)) < 1e-12 * M
    assert abs(s["x_front"] - (1.0 - 0.5 * dp)) < 1e-6          # float32 input positions
    # a block that does not touch the floor band has no front
    cfg2 = dict(inputs.dam_break_2d())
    pos = cfg2["pos"].copy()
    pos[cfg2["tag"] >= 0, 1] += 0.5
    cfg2["pos"] = pos
    assert run(cfg2).stats()["x_front"] < -1e100
    # two phases: only phase 0 counts for the front, both for the energy
    cfg3 = _two_phase_lattice(24, 1.0 / 64, 1000.0, 1.0)
    vel3 = np.zeros_like(cfg3["pos"]); vel3[cfg3["tag"] >= 0] = (0.0, 2.0, 0.0)
    cfg3["vel"] = vel3
    s3 = run(cfg3).stats()
    n = 24
    M3 = (n * n // 2) * (1000.0 + 1.0) * (1.0 / 64) ** 2
    assert abs(s3["ek"] - 0.5 * M3 * 4.0) < 1e-12 * M3 and abs(s3["mass"] - M3) < 1e-12 * M3
    assert abs(s3["x_front"] - (n - 0.5) / 64.0) < 1e-6


@pytest.mark.parametrize("dim", [2, 3])
def test_P25_sigma_of_the_continuity_pass_on_the_lattice(dim):
    """pass_continuity's own sigma (the one the reinitialisation of the next step reads) equals the
    lattice constant of pin P2 for every particle of a closed, unperturbed single-phase box after a
    step (dt = 0 keeps the lattice): sigma dp^d = 1.010473152 / 1.009500784, walls included."""
    gold = _gold("lattice_constants.txt")
    dp = 1.0 / 64
    cfg = dict(inputs.box_2d(n=12, dp=dp)) if dim == 2 else dict(inputs.box_sweep_3d(n=9, dp=dp, jitter=0.0))
    cfg["g"] = [0.0, 0.0, 0.0]
    cfg["rho"] = np.full_like(cfg["rho"], 1000.0)
    o = run(cfg)
    o.step(1, dts=[0.0])
    f = o.fields()
    fl = cfg["tag"] >= 0
    assert np.max(np.abs(f["sigma"][fl] * dp ** dim - gold["sigma0_%dd" % dim])) < 2e-9
    assert np.max(np.abs(f["drho"][fl])) < 1e-6     # at rest with uniform rho and p: Eq. 2.9 gives 0


# ------------------------------------------------------------------ P26-P27: the paper's hydrostatic tank X1 (NEXT-2) and Fig. 7 (NEXT-4)
def _x1(dp, **kw):
    cfg = dict(inputs.hydrostatic_tank_x1(dp=dp))
    cfg.update(kw)
    return cfg, run(cfg)


def _ek_by_phase(cfg, o):
    f = o.fields()
    v2 = (f["vel"] ** 2).sum(1)
    m = np.where(cfg["tag"] == 0, cfg["rho0"][0], cfg["rho0"][1]) * cfg["dp"] ** 2
    return [0.5 * float((m * v2)[cfg["tag"] == ph].sum()) for ph in (0, 1)], f


def test_P26_x1_tank_stays_at_rest_and_reading_A13b_decides():
    """PAPER.md:220-244 (section 4.1): the two-phase tank at rest stays at rest: "the energy variation vanishes",
    0.26 % of T_tot = 1226.25 J is all that is ever dissipated, the pressure follows the analytic hydrostatic
    profile.  At dx = 0.01 (the paper's coarsest) over the first 0.3 s the kinetic energy stays at 1e-4 T_tot under
    reading A13b (sigma of the water over water + walls) while it GROWS past 1e-3 T_tot, with water particles at
    1.5 m/s at the interface, when the air is counted in the water's number density (the first build's reading,
    kept as ORC_VAR_SIGMA_ALL): the evidence DESIGN.md section 3 cites for A13b."""
    T_tot = _gold("paper_values.txt")["T_tot_J"]
    cfg, o = _x1(0.01)
    o.step(3000)
    (ekw, eka), f = _ek_by_phase(cfg, o)
    s = o.stats()
    assert s["escaped"] == 0 and abs(s["ek"] - (ekw + eka)) < 1e-9 * (ekw + eka)
    assert ekw + eka < 3e-4 * T_tot, (ekw, eka)
    fl = cfg["tag"] >= 0
    y = f["pos"][:, 1]
    pex = inputs.x1_analytic_pressure(cfg, y)
    l2 = math.sqrt(((f["p"][fl] - pex[fl]) ** 2).sum() / (pex[fl] ** 2).sum())
    assert l2 < 0.2, l2          # start-up acoustic wave still present at t = 0.3 s (0.14 measured; 0.012 at t = 10 s on the GPU)
    v_w = np.sqrt((f["vel"][cfg["tag"] == 0] ** 2).sum(1)).max()
    assert v_w < 0.3, v_w
    cfg2, o2 = _x1(0.01, oracle_variant=orc.VAR_SIGMA_ALL)
    o2.step(3000)
    (ekw2, eka2), f2 = _ek_by_phase(cfg2, o2)
    assert ekw2 + eka2 > 7e-4 * T_tot, (ekw2, eka2)
    assert np.sqrt((f2["vel"][cfg2["tag"] == 0] ** 2).sum(1)).max() > 0.8


def test_P27_without_the_papers_wall_extensions_air_leaves_the_tank():
    """PAPER.md:258-260 (Fig. 7): "without applying the F_p penalty force ... several particles of the light
    phase have penetrated into the wall boundaries ... and ultimately leave the computational domain"; the paper
    compares with the wall model of Adami et al. (2012).  The X1 tank at dx = 0.02: with the paper's wall treatment
    (Eq. 2.12 divided by rho_f, F_p on the air) no particle leaves in 2000 steps; with ORC_FLAG_WALL_ADAMI_ONLY
    (single-phase Eq. 2.12 for both phases, no F_p) air particles are through the walls within 0.12 s."""
    cfg, o = _x1(0.02)
    o.step(2000)
    assert o.stats()["escaped"] == 0
    (ekw, eka), _ = _ek_by_phase(cfg, o)
    fl = inputs.FLAG_REINIT | inputs.FLAG_WALL_VEL_MIRROR | orc.FLAG_WALL_ADAMI_ONLY
    cfg2, o2 = _x1(0.02, flags=fl)
    o2.step(2000)
    (ekw2, eka2), f2 = _ek_by_phase(cfg2, o2)
    assert o2.stats()["escaped"] >= 1
    assert eka2 > 100.0 * eka, (eka, eka2)


# ------------------------------------------------------------------ P28-P29: the unequal-c solver and the fluid-wall pair
def test_P28_acoustic_solver_satisfies_the_characteristic_relations():
    """Reading A3 away from c_L = c_R.  The linearised (acoustic) Riemann problem has a textbook solution (Toro 1989,
    cited at PAPER.md:77) fixed by the two characteristic relations
        p* - p_L = Z_L (U_L - U*),   p* - p_R = Z_R (U* - U_R),   Z = rho c.
    The oracle's U* must satisfy both with the fully dissipative p* (limiter saturated, beta = c~: U_L - U_R >= c~/3),
    its p* must equal that textbook p* there, and below saturation p* must lie between the non-dissipative average and
    the textbook value, reaching the average when the states separate (U_L <= U_R, the limiter of Eq. 2.8)."""
    rng = np.random.Generator(np.random.PCG64(28))
    for _ in range(200):
        rL, rR = rng.uniform(0.5, 2000.0, 2)
        cL, cR = rng.uniform(5.0, 2000.0, 2)
        pL, pR = rng.uniform(-1e4, 1e4, 2)
        ZL, ZR = rL * cL, rR * cR
        ctil = (ZL + ZR) / (rL + rR)
        UR = rng.uniform(-5.0, 5.0)
        # saturated limiter
        UL = UR + ctil * rng.uniform(0.34, 3.0)
        s = orc.riemann(rL, UL, pL, cL, rR, UR, pR, cR, mode=2)
        scale = abs(pL) + abs(pR) + ZL * abs(UL) + ZR * abs(UR) + 1.0
        assert abs((s["pstar"] - pL) - ZL * (UL - s["Ustar"])) < 1e-12 * scale
        assert abs((s["pstar"] - pR) - ZR * (s["Ustar"] - UR)) < 1e-12 * scale
        # separating states: no dissipation, p* = impedance-weighted average, U* unchanged in form
        UL2 = UR - rng.uniform(0.0, 5.0)
        s2 = orc.riemann(rL, UL2, pL, cL, rR, UR, pR, cR, mode=2)
        assert abs(s2["pstar"] - (ZL * pR + ZR * pL) / (ZL + ZR)) < 1e-12 * scale
        assert abs((ZL + ZR) * s2["Ustar"] - (ZL * UL2 + ZR * UR + pL - pR)) < 1e-12 * scale
        # in between: monotone in the limiter
        UL3 = UR + ctil * rng.uniform(0.0, 0.33)
        s3 = orc.riemann(rL, UL3, pL, cL, rR, UR, pR, cR, mode=2)
        p_avg = (ZL * pR + ZR * pL) / (ZL + ZR)
        p_full = p_avg + ZL * ZR / (ZL + ZR) * (UL3 - UR)
        assert p_avg - 1e-9 * scale <= s3["pstar"] <= p_full + 1e-9 * scale
    # the dispatcher takes the paper's formulas at equal c and the acoustic ones otherwise
    a = orc.riemann(1000.0, 1.0, 50.0, 30.0, 1.0, -2.0, 10.0, 30.0, mode=0)
    b = orc.riemann(1000.0, 1.0, 50.0, 30.0, 1.0, -2.0, 10.0, 30.0, mode=1)
    assert a == b
    c = orc.riemann(1000.0, 1.0, 50.0, 30.0, 1.0, -2.0, 10.0, 900.0, mode=0)
    d = orc.riemann(1000.0, 1.0, 50.0, 30.0, 1.0, -2.0, 10.0, 900.0, mode=2)
    assert c == d


def test_P29_one_fluid_particle_over_one_wall_particle_closed_form():
    """Eq. 2.12, the wall density of reading A5 and Eq. 2.11 on the smallest case that separates them: one fluid
    particle a distance d above one wall particle, a slow sound speed so that rho_w = rho0 + p_w / c^2 is far from
    rho_f.  By hand: p_w = p_f + rho_f g . r_wf (one neighbour: the Shepard average is the value, the lever is the
    printed one), p* = (rho_f p_w + rho_w p_f) / (rho_f + rho_w), a = g - 2 V0 (p* / rho_f) W'(d) e, e = r_fw / d.
    Swapping the weights of Eq. 2.11, taking rho_w = rho_f, or dropping / flipping the lever each changes a by > 5 %."""
    dp, c0, rho0 = 1.0 / 64, 1.0, 1000.0
    d = 1.1 * dp
    rho_f = 1100.0
    g = (0.0, -50.0, 0.0)
    pos = [[0.0, d], [0.0, 0.0]]
    cfg = custom(2, pos, [0, -1], [rho_f, rho0], dp=dp, c0=(c0,), g=g, penalty_phase_mask=0)
    cfg["pos"] = np.asarray([[0.0, d, 0.0], [0.0, 0.0, 0.0]], np.float32)
    f = run(cfg).fields()
    d32 = float(cfg["pos"][0, 1])
    h = 1.3 * dp
    p_f = c0 ** 2 * (rho_f - rho0)
    p_w = p_f + rho_f * (g[1] * (0.0 - d32))          # r_wf = r_w - r_f = (0, -d)
    rho_w = rho0 + p_w / c0 ** 2
    assert rho_w > 1.5 * rho_f                          # the case does separate the readings
    pstar = (rho_f * p_w + rho_w * p_f) / (rho_f + rho_w)
    dw = orc.kernel_dw(2, h, d32)
    ay = g[1] - 2.0 * dp * dp * (pstar / rho_f) * dw * 1.0    # grad_i W = W' (r_i - r_w) / d = W' (0, 1)
    assert abs(f["p"][1] - p_w) < 1e-9 * abs(p_w)
    assert abs(f["acc"][0, 1] - ay) < 1e-9 * abs(ay) and abs(f["acc"][0, 0]) < 1e-12
    wrong = [(rho_w * p_w + rho_f * p_f) / (rho_f + rho_w), 0.5 * (p_w + p_f)]
    for pw in wrong:
        assert abs((g[1] - 2.0 * dp * dp * (pw / rho_f) * dw) - ay) > 0.05 * abs(ay)
