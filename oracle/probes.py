"""CPU oracle of the on-device probes — TEST INFRASTRUCTURE ONLY.

Plain numpy, float64, brute force over all particles; shares no code with the CUDA path.
Only tests/ may import this module.

What the paper says: pressure signals at sensors P1-P4 "are obtained by the method explained by
Zhang et al. (2017)" and water levels are "recorded at three different probes" (PAPER.md:296,
:304); it prints neither formula.  Readings (A29 / A30):

  A29  pressure probe at a point x: the Shepard (kernel-normalised) average of the fluid pressure,
           p(x) = sum_f p_f W(|x - r_f|, h) / sum_f W(|x - r_f|, h)      over fluid particles with |x - r_f| < 2h,
       0 where no fluid particle is in reach; W is the Wendland C2 kernel of reading A1.  The same
       weights as the fluid part of Eq. 2.12 without the lever term.
  A30  wave gauge at a horizontal position (x[, y]): the free-surface height
           eta = max { z_f + dp/2 : phase_f = 0, horizontal distance to the gauge < h },
       -inf (reported as the domain floor by the library: here NaN) when no such particle exists.
       In 2-D "z" is the y coordinate and the horizontal distance is |x_f - x|.

Pins (tests/test_oracle_pins.py): a constant field returns the constant; a field linear in z on
an unperturbed lattice returns the field value at a lattice-symmetric point; a resting block of
height H gauges H.
"""
import numpy as np


def wendland_c2(r, h, dim):
    """W(r, h) = alpha_d (1 - q/2)^4 (1 + 2q), q = r/h < 2 (reading A1)."""
    q = np.asarray(r, np.float64) / h
    alpha = 7.0 / (4.0 * np.pi * h * h) if dim == 2 else 21.0 / (16.0 * np.pi * h ** 3)
    w = alpha * (1.0 - 0.5 * q) ** 4 * (1.0 + 2.0 * q)
    return np.where(q < 2.0, w, 0.0)


def pressure_probes(cfg, pos, p, tag, points):
    """Reading A29.  pos (n,3), p (n,), tag (n,), points (m,3) -> (p_probe (m,), wsum (m,))."""
    dim, h = int(cfg["dim"]), float(cfg["h"])
    pos = np.asarray(pos, np.float64)
    p = np.asarray(p, np.float64)
    fluid = np.asarray(tag) >= 0
    pf, xf = p[fluid], pos[fluid]
    out = np.zeros(len(points))
    ws = np.zeros(len(points))
    for k, x in enumerate(np.asarray(points, np.float64)):
        d = xf - x[None, :]
        if dim == 2:
            d = d[:, :2]
        r = np.sqrt((d * d).sum(axis=1))
        w = wendland_c2(r, h, dim)
        s = w.sum()
        ws[k] = s
        out[k] = (w * pf).sum() / s if s > 0.0 else 0.0
    return out, ws


def wave_gauges(cfg, pos, tag, points):
    """Reading A30.  points (m,3): the horizontal coordinates are used ((x, y) in 3-D, x in 2-D)."""
    dim, h, dp = int(cfg["dim"]), float(cfg["h"]), float(cfg["dp"])
    pos = np.asarray(pos, np.float64)
    heavy = np.asarray(tag) == 0
    xf = pos[heavy]
    up = dim - 1                      # vertical axis: z in 3-D, y in 2-D
    out = np.full(len(points), np.nan)
    for k, x in enumerate(np.asarray(points, np.float64)):
        d = xf[:, :up] - x[None, :up]
        m = (d * d).sum(axis=1) < h * h
        if m.any():
            out[k] = xf[m, up].max() + 0.5 * dp
    return out
