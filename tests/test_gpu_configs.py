"""GPU parity at BASELINE.json's configurations (full sizes where the oracle finishes in seconds,
the stated reduced variant otherwise), in the launch configuration bench.py times: same kernels,
same block sizes, device-resident state, sph_step_dt driven by the oracle's dt sequence.

Run on a B200 with `pytest -m gpu`.
"""
import numpy as np
import pytest

from oracle import orc
from paper_2110_02621_b200 import inputs, sph

from parity_util import TOL, acc_tol, check_step_lists, compare_fields, extra_bound, make_pair

pytestmark = pytest.mark.gpu


def _steps_and_compare(cfg, nsteps, names=("rho", "p", "acc", "vel", "pos"), light_acc_tol=None):
    """light_acc_tol: DECLARED DEVIATION from the north_star's 1e-4 (A26b) for the
    acceleration of the light phase when it has its own, larger speed of sound (config 2b); every other
    field and phase is held to TOL with the acceleration scale |g|."""
    from parity_util import acc_err_by_phase
    o, g = make_pair(cfg)
    e0 = compare_fields(cfg, o, g, names=("rho", "p", "acc"))
    if light_acc_tol is not None:
        ph0 = acc_err_by_phase(cfg, o, g)
        print("set-up: acceleration error / |g| per phase:", ph0)
        assert ph0[0] < TOL and max(ph0.values()) < light_acc_tol, ("set-up", ph0)
        e0.pop("acc")
    assert max(e0.values()) < TOL, ("set-up", e0)
    dts = o.step(nsteps)
    g.step(nsteps, dts=dts)
    e = compare_fields(cfg, o, g, names=names)
    ph = acc_err_by_phase(cfg, o, g)
    print("after %d steps: acceleration error / |g| per phase:" % nsteps, ph)
    if light_acc_tol is not None:
        assert ph[0] < TOL and max(ph.values()) < light_acc_tol, ("after %d steps" % nsteps, ph)
        e.pop("acc")
    elif acc_tol(cfg) > TOL:       # declared deviation for H / h > 66 (parity_util.acc_tol)
        assert e.pop("acc") < acc_tol(cfg), ("after %d steps" % nsteps, ph, acc_tol(cfg))
    assert max(e.values()) < TOL, ("after %d steps" % nsteps, e, ph)
    so, sg = o.stats(), g.get_stats()
    # after steps the two position sets differ in the last bits: pairs at r = 2h to rounding may flip
    # (reading A25: the integer contract is per snapshot)
    assert abs(sg["npairs"] - so["npairs"]) <= max(2, 1e-7 * so["npairs"])
    assert sg["escaped"] == 0 and sg["nonfinite"] == 0
    assert abs(sg["mass"] - so["mass"]) <= 1e-9 * so["mass"]   # the oracle adds up to 16.8 M doubles one by one (1.9e-10 seen at 12 M)
    assert abs(sg["ek"] - so["ek"]) <= 1e-3 * so["ek"] + 1e-12
    # the lists the passes read hold every float32-contract neighbour (k_build's float16 filter)
    missing, extra, total = g.debug_list_check()
    assert missing == 0 and extra <= extra_bound(cfg) * total
    # probes (readings A29 / A30) on the oracle's own state, sampled points
    from oracle import probes
    fo = o.fields()
    fl = cfg["tag"] >= 0
    lo, hi = fo["pos"][fl].min(0), fo["pos"][fl].max(0)
    pts = (lo + np.random.default_rng(23).random((16, 3)) * (hi - lo)).astype(np.float32)
    if cfg["dim"] == 2:
        pts[:, 2] = 0.0
    p_ref, _ = probes.pressure_probes(cfg, fo["pos"], fo["p"], cfg["tag"], pts.astype(np.float64))
    p_gpu, _ = g.probe_pressure(pts)
    S = cfg["rho0"][0] * float(np.linalg.norm(cfg["g"]) or 1.0) * float(cfg.get("H", 1.0))
    assert np.max(np.abs(p_gpu - p_ref)) / S < TOL
    e_ref = probes.wave_gauges(cfg, fo["pos"], cfg["tag"], pts.astype(np.float64))
    e_gpu = g.probe_gauge(pts)
    ok = ~np.isnan(e_ref)
    assert np.array_equal(ok, ~np.isnan(e_gpu))
    assert ok.sum() == 0 or np.max(np.abs(e_gpu[ok] - e_ref[ok])) < 1e-5 * float(cfg.get("H", 1.0))
    return o, g


def test_cfg1_dam_break_3d_box_full_size():
    """Config 1 at full size (671 000 fluid + 471 228 wall): set-up, then 3 steps."""
    cfg = inputs.dam_break_3d_box()
    assert cfg["n_fluid"] == 671000
    _steps_and_compare(cfg, 3)


def test_cfg1_moving_walls_full_size():
    """Config 1 at full size with the wall motion `bench.py --wall-osc 0.01,0.5` times (NEXT-1,
    PAPER.md:252, :116): set-up, then 3 steps on the oracle's dt sequence; the walls sit on
    x_w(0) + A0 sin(2 pi f0 t)."""
    cfg = dict(inputs.dam_break_3d_box())
    cfg["wall_osc_amp"], cfg["wall_osc_freq"] = (0.01, 0.0, 0.0), 0.5
    o, g = make_pair(cfg)
    e0 = compare_fields(cfg, o, g, names=("rho", "p", "acc"))
    assert max(e0.values()) < TOL, ("set-up", e0)
    dts = o.step(3)
    g.step(3, dts=dts)
    e = compare_fields(cfg, o, g, names=("rho", "p", "acc", "vel", "pos"))
    assert max(e.values()) < TOL, e
    wall = cfg["tag"] < 0
    pg = g.get_fields(device=False, which=("pos",))["pos"]
    want = cfg["pos"][wall].astype(np.float64)
    want[:, 0] += 0.01 * np.sin(2.0 * np.pi * 0.5 * float(np.sum(dts)))
    assert np.max(np.abs(pg[wall] - want)) < 2e-7 * max(1.0, np.abs(want).max())
    sg = g.get_stats()
    assert sg["escaped"] == 0 and sg["nonfinite"] == 0
    missing, extra, total = g.debug_list_check()
    assert missing == 0 and extra <= extra_bound(cfg) * total
    # all three lists the passes read (fluid-fluid, fluid-wall, wall-fluid) against the oracle's contract lists, host side
    check_step_lists(cfg, g, grid=True)


def test_cfg1_cells_bit_exact_full_size():
    cfg = inputs.dam_break_3d_box()
    g = sph.Sph(cfg)
    g.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    cid, perm, cs, ce = g.debug_cells()
    rcid, rperm, rcs, rce = orc.f32_cells(cfg, cfg["pos"], cfg["tag"])
    assert np.array_equal(cid, rcid) and np.array_equal(perm, rperm)
    assert np.array_equal(cs, rcs) and np.array_equal(ce, rce)
    off, ids = g.debug_neighbours()
    roff, rids = orc.f32_neighbours(cfg, cfg["pos"], cfg["tag"], grid=True)
    assert np.array_equal(off, roff) and np.array_equal(ids, rids)


@pytest.mark.parametrize("equal_c", [True, False])
def test_cfg2_two_phase_2d_full_size(equal_c):
    """Config 2a (paper: one c) and 2b (BASELINE.json: per-phase c), 102 960 fluid, 10 steps."""
    cfg = inputs.two_phase_2d(equal_c=equal_c)
    assert cfg["n_fluid"] == 102960
    # 2a (the paper's equal c): every phase to 1e-4 |g|.  2b (c_air^2 = 1000 c_w^2): the air's
    # acceleration responds to a relative change ds of its number density by c_air^2 ds / h, 1.2e8 m/s^2 here,
    # so positions held to Q/1024 = 1.8e-12 m (oracle: float64) leave 1e-3 |g|: measured 2.8e-3, bound 5e-3.
    _steps_and_compare(cfg, 10, light_acc_tol=None if equal_c else 5e-3)


def test_cfg3_sloshing_spheres_reduced():
    """Config 3's geometry (signed-distance walls around 8 seeded spheres, tilted gravity) at
    dp = 0.0125 (≈ 0.4 M fluid) so that the oracle takes seconds; 5 steps."""
    cfg = inputs.sloshing_spheres_3d(dp=0.0125)
    assert 3.0e5 < cfg["n_fluid"] < 6.0e5
    _steps_and_compare(cfg, 5)


def test_cfg4_box_sweep_1m():
    """Config 4 at N_f = 1 M: 2 steps, all fields."""
    cfg = inputs.box_sweep_3d(n=100)
    _steps_and_compare(cfg, 2)


def test_cfg4_box_sweep_16m_properties():
    """Config 4 at N_f = 16.8 M (the size the roofline bar is quoted at): the oracle is too slow
    for a full comparison, so check what holds at any size: mass, no escapes, the pair count
    against the lattice count of pin P2, finite accelerations, and
    sigma / sigma0 = 1 in the bulk to the jitter-induced spread."""
    n = 256
    cfg = inputs.box_sweep_3d(n=n)
    g = sph.Sph(cfg)
    g.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    g.step(2)
    s = g.get_stats()
    assert s["n_fluid"] == n ** 3 and s["escaped"] == 0 and s["nonfinite"] == 0
    assert abs(s["mass"] - 1000.0 * (n * cfg["dp"]) ** 3) < 1e-6 * s["mass"]
    # 80 neighbours on the undisturbed lattice (pin P2); a jitter of 0.1 dp moves few pairs across 2h; walls complete the support
    assert 78.0 < s["npairs"] / n ** 3 < 81.0
    f = g.get_fields(device=False, which=("pos", "acc"))
    fl = cfg["tag"] >= 0
    H = n * cfg["dp"]
    assert np.isfinite(f["acc"]).all() and np.all(f["acc"][~fl] == 0)
    sig, _ = g.debug_sigma()
    s0 = orc.sigma0(3, cfg["h"], cfg["dp"])
    x = f["pos"][fl]
    inner = np.all((x > 0.05) & (x < H - 0.05), axis=1)
    # a jitter of +-0.1 dp raises the mean of sigma by the second-order term (3e-3 measured)
    assert abs(np.mean(sig[fl][inner], dtype=np.float64) / s0 - 1.0) < 6e-3


# ------------------------------------------------------------------------- round 2: the sizes the roofline bar is quoted at
def _cells_bit_exact(cfg):
    g = sph.Sph(cfg)
    g.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    cid, perm, cs, ce = g.debug_cells()
    rcid, rperm, rcs, rce = orc.f32_cells(cfg, cfg["pos"], cfg["tag"])
    assert np.array_equal(cid, rcid) and np.array_equal(perm, rperm)
    assert np.array_equal(cs, rcs) and np.array_equal(ce, rce)
    return g


def test_cfg4_160_cells_and_neighbour_lists_bit_exact():
    """4.1 M fluid keys: the radix sort's 16-keys-per-thread path (n >= 2 M, sph_sort.cuh) with 18-bit cell
    ids (2 passes of 9 bits); cell ids, permutation, ranges and the full CSR neighbour lists (368 M
    entries) bit-exact against the oracle's float32 contract (std::stable_sort, grid walk)."""
    cfg = inputs.box_sweep_3d(n=160)
    assert cfg["n_fluid"] >= (2 << 20)
    g = _cells_bit_exact(cfg)
    assert 17 <= int(np.ceil(np.log2(g.num_cells()))) <= 18
    off, ids = g.debug_neighbours()
    roff, rids = orc.f32_neighbours(cfg, cfg["pos"], cfg["tag"], grid=True)
    assert np.array_equal(off, roff) and np.array_equal(ids, rids)


def test_cfg4_256_cells_bit_exact():
    """16.8 M fluid keys, cell ids beyond 18 bits (3 radix passes): cell ids, permutation and ranges
    bit-exact against std::stable_sort on the oracle's float32 cell hash."""
    cfg = inputs.box_sweep_3d(n=256)
    g = _cells_bit_exact(cfg)
    assert g.num_cells() > (1 << 18)


def test_cfg4_256_fields_after_setup_and_2_steps():
    """Config 4 at N_f = 16.8 M, the size the >= 0.5 roofline bar is quoted at and the default bench.py
    workload: every field of every particle against the oracle after the set-up and after 2 steps."""
    cfg = inputs.box_sweep_3d(n=256)
    assert cfg["n_fluid"] == 256 ** 3
    _steps_and_compare(cfg, 2)


def test_cfg3_sloshing_spheres_full_size_dp_0_004():
    """Config 3 as BASELINE.json writes it (dp = 0.004: 12.05 M fluid + 1.9 M wall, reading A27): set-up
    and 2 steps against the oracle."""
    cfg = inputs.sloshing_spheres_3d()
    assert cfg["n_fluid"] > 1.1e7
    _steps_and_compare(cfg, 2)


# ------------------------------------------------------------------------- NEXT-2: the paper's two-phase hydrostatic tank study (X1)
def test_x1_hydrostatic_tank_study():
    """PAPER.md:220-244 (section 4.1) through the committed driver paper_2110_02621_b200/x1_study.py: dx = 0.02, 0.01
    (the paper's coarsest) and 0.005, from rest to t = 10 s (the paper's instant of Fig. 3 / 4).  What the paper states
    and what is checked: a stable interface with no particle leaving the tank; "after the initial effects of gravity, the
    energy variation vanishes and the system reaches a steady state" with the energy at the 1e-3 level of T_tot =
    1226.25 J (0.26 % dissipated); the pressure follows the analytic hydrostatic profile, with an L2 error
    that falls with the spacing.  Measured (profiles/r02_x1.md): L2 = 1.6-1.8 %, 1.2 %, 1.0-1.2 %, i.e. a floor near
    1 % that does not depend on the spacing: the pressure gradient of Eq. 2.10 on a particle arrangement with h / dx =
    1.3 is short by the first-moment constant of pin P3 (M1 = 0.974), so the settled column is 2-3 % over-compressed at
    the bottom: a property of the discretisation the paper prints (no kernel-gradient correction), not of a reading."""
    from paper_2110_02621_b200 import x1_study
    rows = [x1_study.run_case(dp, 10.0, samples=40) for dp in (0.02, 0.01, 0.005)]
    for r in rows:
        print({k: v for k, v in r.items() if k != "history"})
        assert r["escaped"] == 0 and r["nonfinite"] == 0 and r["t_end"] >= 10.0
        assert r["ek_max_over_T"] < 1e-3            # never more than 0.1 % of T_tot in motion (paper: 0.26 % dissipated in all)
        assert r["ek_end_over_T"] < 3e-5            # at rest at t = 10 s
        assert abs(r["ep_end_minus_ep0_over_T"]) < 1e-2
        assert r["l2_end"] < 0.03 and r["l2_avg"] < 0.03
        tail = [h["ek"] for h in r["history"] if h["t"] > 5.0]
        assert max(tail) < 1e-4 * 1226.25           # "the total energy stayed conserved afterwards"
    # the error falls from dx = 0.02 to 0.01 and then sits on the h / dx consistency floor near 1 %; the values scatter by
    # +-0.002 between realisations (chaotic air motion, residual acoustic wave), so the bounds are on the time averages
    assert rows[0]["l2_avg"] > 1.1 * rows[1]["l2_avg"]      # measured 0.0156 / 0.0125 and 0.0181 / 0.0117
    assert rows[1]["l2_avg"] < 0.015 and rows[2]["l2_avg"] < 0.015


# ------------------------------------------------------------------------- the launch configuration bench.py times, at full sizes
def _sampled_sigma_check(cfg, g, nsample=24, seed=5):
    """sigma_i of sampled fluid particles, one by one, from the oracle's kernel (orc.kernel_w, pin P1) over ALL particles
    at the library's current positions (brute force in float64), against the sigma_i the last pass A summed."""
    pos = g.get_fields(device=False, which=("pos",))["pos"]
    sig, _ = g.debug_sigma()
    fl = np.flatnonzero(cfg["tag"] >= 0)
    pick = np.random.default_rng(seed).choice(fl, nsample, replace=False)
    h, dim = cfg["h"], cfg["dim"]
    s0 = orc.sigma0(dim, h, cfg["dp"])
    p64 = pos.astype(np.float64)
    worst = 0.0
    for i in pick:
        d = p64 - p64[i]
        near = np.flatnonzero((np.abs(d) < 2.0 * h).all(axis=1))
        r = np.sqrt((d[near] ** 2).sum(axis=1))
        s = sum(orc.kernel_w(dim, h, float(x)) for x in r[r < 2.0 * h])     # includes the self term r = 0
        worst = max(worst, abs(float(sig[i]) - s) / s0)
    return worst


def test_cfg4_256_graph_replay_is_the_direct_path_bitwise_and_sampled_sigma():
    """The configuration `python bench.py` times (config 4 at 16.8 M, sph_step = CUDA-graph replay with the rebuild
    branch as an IF node, device-computed dt) against the plain-launch path the oracle comparisons above drive
    (`test_cfg4_256_fields_after_setup_and_2_steps`): 6 steps, every field bit for bit; then sigma_i of sampled particles
    against the oracle's kernel summed by brute force."""
    cfg = inputs.box_sweep_3d(n=256)
    out = []
    for flags in (cfg["flags"], cfg["flags"] | sph.FLAG_NO_GRAPH):
        g = sph.Sph(dict(cfg, flags=flags))
        g.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
        g.step(6)
        s = g.get_stats(with_pairs=False)
        assert s["steps"] == 6 and s["escaped"] == 0 and s["nonfinite"] == 0 and s["rebuilds"] >= 2
        out.append((g.get_fields(device=False), s["rebuilds"], s["dt"]))
        if flags == cfg["flags"]:
            # float32 positions at 2.6 m carry 2.4e-7 m: sigma from them is good to 1e-5 sigma0 (the library sums it from
            # its 32-bit fixed-point positions); a dropped neighbour would show as >= 1e-3 sigma0
            assert _sampled_sigma_check(cfg, g) < 5e-5
        g.close()
    assert out[0][1] == out[1][1] and out[0][2] == out[1][2]
    for k in out[0][0]:
        assert np.array_equal(out[0][0][k], out[1][0][k]), k


def test_cfg4_400_64m_properties_and_sampled_sigma():
    """Config 4 at its largest size (64 M fluid + 2.9 M wall particles, 84 GB on the device): what holds at any size
    (mass, no escapes, no list overflow, the pair count against the lattice count of pin P2, finite fields) after the
    set-up and 3 graph-replayed steps, and sigma_i of sampled particles against the oracle's kernel by brute force."""
    n = 400
    cfg = inputs.box_sweep_3d(n=n)
    g = sph.Sph(cfg)
    g.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    g.step(3)
    s = g.get_stats()
    assert s["n_fluid"] == n ** 3 and s["escaped"] == 0 and s["nonfinite"] == 0 and s["steps"] == 3
    assert abs(s["mass"] - 1000.0 * (n * cfg["dp"]) ** 3) < 1e-6 * s["mass"]
    assert 78.0 < s["npairs"] / n ** 3 < 81.0
    assert _sampled_sigma_check(cfg, g, nsample=12) < 1e-4        # float32 positions at 4 m: 4.8e-7 m
    f = g.get_fields(device=False, which=("acc", "rho"))
    fl = cfg["tag"] >= 0
    assert np.isfinite(f["acc"]).all() and np.all(f["acc"][~fl] == 0)
    dev = np.abs(f["rho"][fl] / 1000.0 - 1.0)     # hydrostatic 0.5 % + the jittered lattice's sigma spread through Eq. 2.17
    assert float(dev.mean()) < 0.03 and float(dev.max()) < 0.25, (float(dev.mean()), float(dev.max()))
    g.close()


# ------------------------------------------------------------------------- long runs: integral quantities (BASELINE.json north_star)
def _long_run(cfg, nsteps, chunk, ek_tol=0.01, front=True):
    """sph_step (graph replay, device-computed dt, kept lists) against the oracle's own run with its own dt, `nsteps`
    steps (BASELINE.json's step count of the configuration): total mass exact, kinetic energy and surge front within
    1 % at every `chunk` steps, no particle lost, the lists rebuilt now and then but not every step."""
    o, g = make_pair(cfg)
    m0 = g.get_stats(with_pairs=False)["mass"]
    done = 0
    while done < nsteps:
        o.step(chunk)
        g.step(chunk)
        done += chunk
        so, sg = o.stats(), g.get_stats(with_pairs=False)
        assert sg["escaped"] == 0 and sg["nonfinite"] == 0 and so["escaped"] == 0, (done, sg)
        assert sg["mass"] == m0 and abs(m0 - so["mass"]) <= 1e-9 * so["mass"]
        assert abs(sg["t"] - so["t"]) < 1e-4 * so["t"], (done, sg["t"], so["t"])
        assert abs(sg["ek"] - so["ek"]) <= ek_tol * so["ek"] + 1e-12, (done, sg["ek"], so["ek"])
        if front:
            assert abs(sg["x_front"] - so["x_front"]) < 0.01 * abs(so["x_front"]), (done, sg["x_front"], so["x_front"])
    assert 2 <= sg["rebuilds"] < nsteps, sg["rebuilds"]
    return so, sg


def test_cfg1_geometry_1000_steps_integral_quantities():
    """Config 1 (3-D dam break with the box obstacle) over its 1000 steps at dp = 0.02 (83 875 fluid particles: the
    oracle takes a minute)."""
    cfg = inputs.dam_break_3d_box(dp=0.02)
    _long_run(cfg, 1000, 250)


@pytest.mark.parametrize("equal_c", [True, False])
def test_cfg2_geometry_2000_steps_integral_quantities(equal_c):
    """Config 2 (2-D water / air dam break, density ratio 1000) over its 2000 steps at dp = 0.025 (25 680 fluid)."""
    cfg = inputs.two_phase_2d(dp=0.025, equal_c=equal_c)
    _long_run(cfg, 2000, 500)


def test_cfg3_geometry_500_steps_integral_quantities():
    """Config 3 (sloshing box with 8 seeded spheres, gravity tilting) over its 500 steps at dp = 0.02."""
    cfg = inputs.sloshing_spheres_3d(dp=0.02)
    _long_run(cfg, 500, 250, front=False)      # a filled box has no surge front; E_k and mass are the integral quantities
