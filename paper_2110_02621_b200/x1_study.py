"""The paper's two-phase hydrostatic tank study, case X1 (section 4.1), run through
the public binding: `python -m paper_2110_02621_b200.x1_study --dp 0.02 0.01 0.005 --t-end 10`.

For every spacing it advances the tank from rest to t_end with sph_step (device-computed dt, Eq.
2.23-2.24), samples the kinetic and potential energies (Fig. 5) at `--samples` instants
and, at the end, compares the pressure with the analytic hydrostatic profile (Fig. 4):
  L2      = sqrt( sum_i (p_i - p_exact(y_i))^2 / sum_i p_exact(y_i)^2 ) over the fluid particles
            (the L2 norm of error the paper cites, Fatehi & Manzari 2011), instantaneous at t_end and
            from the pressure averaged over the last fifth of the run (the residual acoustic standing
            wave of the start-up averages out; the low-dissipation limiter of Eq. 2.8 damps it slowly);
  E_k/T   = kinetic energy over T_tot = rho_w g L H^2 / 2 = 1226.25 J.
Evaluation only: no method arithmetic here; everything the method computes runs in libsph's kernels.
Prints one JSON object per spacing and a final table."""
import argparse
import json
import math
import time

import numpy as np

from . import inputs, sph


def run_case(dp, t_end, samples=50, c_rule="baseline", flags=None, penalty=True, chunk_max=5000, verbose=False):
    cfg = inputs.hydrostatic_tank_x1(dp=dp, c_rule=c_rule)
    if flags is not None:
        cfg["flags"] = flags
    if not penalty:
        cfg["penalty_phase_mask"] = 0
    g = sph.Sph(cfg)
    g.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    tag = cfg["tag"]
    fl = tag >= 0
    m = np.where(tag == 0, cfg["rho0"][0], cfg["rho0"][1] if cfg["n_phases"] > 1 else 0.0) * dp * dp
    T_tot = cfg["rho0"][0] * inputs.G0 * 1.0 * cfg["H"] ** 2 / 2.0
    dt0 = 0.25 * cfg["h"] / max(cfg["c0"])
    hist = []
    p_acc, n_acc = None, 0
    t, steps, t0 = 0.0, 0, time.time()
    next_sample = t_end / samples
    while t < t_end:
        k = int(min(chunk_max, max(1, (min(next_sample, t_end) - t) / dt0)))
        g.step(k)
        steps += k
        s = g.get_stats(with_pairs=False)
        t = s["t"]
        if t + 0.5 * dt0 < next_sample and t < t_end:
            continue
        next_sample += t_end / samples
        f = g.get_fields(device=False, which=("pos", "p"))
        y = f["pos"][:, 1].astype(np.float64)
        ep = float((m[fl] * inputs.G0 * y[fl]).sum())
        hist.append(dict(t=t, steps=steps, ek=s["ek"], ep=ep))
        if t >= 0.8 * t_end:
            p_acc = f["p"].astype(np.float64) if p_acc is None else p_acc + f["p"]
            n_acc += 1
        if verbose:
            print("  dp=%g t=%.3f steps=%d E_k/T=%.3e (%.0f s)" % (dp, t, steps, s["ek"] / T_tot, time.time() - t0), flush=True)
        if s["escaped"] or s["nonfinite"]:
            break
    f = g.get_fields(device=False, which=("pos", "p"))
    y = f["pos"][:, 1].astype(np.float64)
    pex = inputs.x1_analytic_pressure(cfg, y)
    l2 = lambda p: math.sqrt(float(((p[fl] - pex[fl]) ** 2).sum() / (pex[fl] ** 2).sum()))
    ep0 = float((m[fl] * inputs.G0 * cfg["pos"][fl, 1].astype(np.float64)).sum())
    # where the error sits: mean of (p - p_exact) / (rho_w g H) over the water in ten bands of height (time-averaged p)
    S = cfg["rho0"][0] * inputs.G0 * cfg["H"]
    pbar = p_acc / max(n_acc, 1) if p_acc is not None else f["p"].astype(np.float64)
    water = tag == 0
    profile = []
    for k in range(10):
        lo, hi = k * cfg["H"] / 10.0, (k + 1) * cfg["H"] / 10.0
        sel = water & (y >= lo) & (y < hi)
        if sel.any():
            profile.append([0.5 * (lo + hi), float(((pbar - pex)[sel]).mean() / S)])
    y_water_mean = float(y[water].mean())
    out = dict(dp=dp, n_fluid=cfg["n_fluid"], n_wall=cfg["n_wall"], t_end=t, steps=steps,
               l2_end=l2(f["p"].astype(np.float64)), l2_avg=l2(p_acc / max(n_acc, 1)) if p_acc is not None else None,
               ek_max_over_T=max(h["ek"] for h in hist) / T_tot, ek_end_over_T=hist[-1]["ek"] / T_tot,
               ep0=ep0, ep_end_minus_ep0_over_T=(hist[-1]["ep"] - ep0) / T_tot,
               escaped=int(s["escaped"]), nonfinite=int(s["nonfinite"]), seconds=time.time() - t0,
               c0=cfg["c0"][0], error_profile=profile, water_mean_height=y_water_mean, history=hist)
    g.close()
    return out


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--dp", type=float, nargs="+", default=[0.02, 0.01, 0.005])
    ap.add_argument("--t-end", type=float, default=10.0)
    ap.add_argument("--samples", type=int, default=50)
    ap.add_argument("--c-rule", default="baseline", choices=["baseline", "paper"])
    ap.add_argument("--no-penalty", action="store_true", help="Fig. 7 ablation: F_p off")
    ap.add_argument("--adami-only", action="store_true", help="NEXT-4 ablation: SPH_FLAG_WALL_ADAMI_ONLY")
    ap.add_argument("--out", default="")
    ap.add_argument("-v", "--verbose", action="store_true")
    a = ap.parse_args()
    flags = inputs.FLAG_REINIT | inputs.FLAG_WALL_VEL_MIRROR | (sph.FLAG_WALL_ADAMI_ONLY if a.adami_only else 0)
    rows = []
    for dp in a.dp:
        r = run_case(dp, a.t_end, a.samples, a.c_rule, flags, not a.no_penalty, verbose=a.verbose)
        rows.append(r)
        print(json.dumps({k: v for k, v in r.items() if k != "history"}), flush=True)
    print("%-9s %9s %9s %10s %10s %11s %11s %8s" % ("dp", "n_fluid", "steps", "L2(t_end)", "L2(avg)", "maxE_k/T", "E_k(end)/T", "escaped"))
    for r in rows:
        print("%-9g %9d %9d %10.5f %10.5f %11.3e %11.3e %8d" % (r["dp"], r["n_fluid"], r["steps"], r["l2_end"], r["l2_avg"] or float("nan"),
                                                               r["ek_max_over_T"], r["ek_end_over_T"], r["escaped"]))
    for r in rows:
        print("dp %g: mean (p - p_exact) / (rho_w g H) of the water by height: " % r["dp"] +
              " ".join("%.2f:%+.4f" % (yy, e) for yy, e in r["error_profile"]) + "; mean water height %.5f" % r["water_mean_height"])
    for a_, b_ in zip(rows[:-1], rows[1:]):
        if a_["l2_avg"] and b_["l2_avg"]:
            print("order dp %g -> %g: L2(avg) ratio %.3f (observed order %.2f)" % (
                a_["dp"], b_["dp"], b_["l2_avg"] / a_["l2_avg"], math.log(a_["l2_avg"] / b_["l2_avg"]) / math.log(a_["dp"] / b_["dp"])))
    if a.out:
        with open(a.out, "w") as fh:
            json.dump(rows, fh)


if __name__ == "__main__":
    main()
