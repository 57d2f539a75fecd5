// sph_probe.cuh — on-device probes: pressure sensors and wave gauges
// as small reduction kernels over the current fluid state, so a long run needs no full download.
// The paper reports pressure signals "by the method explained by Zhang et al. (2017)" and water levels
// at probes without printing either formula: readings A29 / A30.
// Included by sph.cu only.  Not on the per-step path.
#pragma once
#include "sph_common.cuh"

// Reading A29: p(x) = sum_f p_f W(|x - r_f|) / sum_f W over the fluid particles within 2h of x (0 if
// none).  One warp per probe: the 27 (9) cells around the probe from the step's cell list, positions
// from the fixed-point records in float64 (a handful of probes: precision costs nothing here).
__global__ void __launch_bounds__(32)
k_probe_pressure(const DP p, const int nf, const int m, const float* __restrict__ xyz, const XB* __restrict__ R,
                 const int* __restrict__ lbF, float* __restrict__ out_p, float* __restrict__ out_w) {
  const int k = blockIdx.x, lane = threadIdx.x;
  if (k >= m) return;
  const float xf = xyz[3 * k], yf = xyz[3 * k + 1], zf = p.dim == 3 ? xyz[3 * k + 2] : 0.0f;
  const double x = xf, y = yf, z = zf;
  const int cx = cell_coord(xf, p.ox, p.inv_edge, p.nx), cy = cell_coord(yf, p.oy, p.inv_edge, p.ny);
  const int cz = p.dim == 3 ? cell_coord(zf, p.oz, p.inv_edge, p.nz) : 0;
  const double ih = 1.0 / p.hD;
  double sw = 0.0, sp = 0.0;
  const int RC = p.reach;
  for (int dz = (p.dim == 3 ? -RC : 0); dz <= (p.dim == 3 ? RC : 0); ++dz)
    for (int dy = -RC; dy <= RC; ++dy) {
      const int yy = cy + dy, zz = cz + dz;
      if (yy < 0 || yy >= p.ny || zz < 0 || zz >= p.nz) continue;
      const int rb = (zz * p.ny + yy) * p.nx;
      const int s = lbF[rb + max(cx - RC, 0)], e = lbF[rb + min(cx + RC, p.nx - 1) + 1];
      for (int j = s + lane; j < e; j += 32) {
        const XB r = R[j];
        const double ddx = fx_pos(p, r.x, 0) - x, ddy = fx_pos(p, r.x, 1) - y;
        const double ddz = p.dim == 3 ? fx_pos(p, r.x, 2) - z : 0.0;
        const double q = sqrt(ddx * ddx + ddy * ddy + ddz * ddz) * ih;
        if (q < 2.0) {
          const double t = 1.0 - 0.5 * q, t2 = t * t;
          const double w = t2 * t2 * (1.0 + 2.0 * q);  // W / alpha_d: alpha_d cancels in the ratio
          sw += w;
          sp += w * (double)p.c2[phase_of(r.x)] * (double)r.b.w;
        }
      }
    }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sw += __shfl_xor_sync(FULL, sw, o);
    sp += __shfl_xor_sync(FULL, sp, o);
  }
  if (lane == 0) {
    out_p[k] = sw > 0.0 ? (float)(sp / sw) : 0.0f;
    out_w[k] = (float)(sw * (double)p.alpha);
  }
}

// Reading A30: eta = max { z_f + dp/2 : phase_f = 0, horizontal distance to the gauge < h }, NaN if
// there is no such particle ("z" is y in 2-D).  One block per gauge over all fluid particles.
__global__ void __launch_bounds__(256)
k_probe_gauge(const DP p, const int nf, const int m, const float* __restrict__ xyz, const XB* __restrict__ R,
              float* __restrict__ out) {
  __shared__ double sm[8];
  const int k = blockIdx.x;
  if (k >= m) return;
  const double x = xyz[3 * k], y = xyz[3 * k + 1];
  const int up = p.dim - 1;
  const double h2 = p.hD * p.hD;
  double best = -1.0e300;
  for (int j = threadIdx.x; j < nf; j += 256) {
    const XB r = R[j];
    if (phase_of(r.x) != 0) continue;
    const double px = fx_pos(p, r.x, 0), py = fx_pos(p, r.x, 1);
    const double ddx = px - x, ddy = p.dim == 3 ? py - y : 0.0;
    if (ddx * ddx + ddy * ddy < h2) best = fmax(best, up == 2 ? fx_pos(p, r.x, 2) : py);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(FULL, best, o));
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) best = fmax(best, sm[w]);
    out[k] = best > -1.0e299 ? (float)(best + 0.5 * p.dpD) : __int_as_float(0x7fc00000);
  }
}
