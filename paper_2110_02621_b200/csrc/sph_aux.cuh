// sph_aux.cuh — loading, time step, predictor, reorder, wall normals and near-wall flags.
// Included by sph.cu only.  Citations: PAPER.md:<line>; readings Axx: DESIGN.md §3.
#pragma once
#include <cuda_fp16.h>

#include "sph_common.cuh"


// ------------------------------------------------------------------------------------------
// Loading (sph_set_particles): split caller arrays into the fluid / wall structures.
// ------------------------------------------------------------------------------------------
__global__ void k_load(DP p, int n, int is_wall, const int* __restrict__ idx, const float* __restrict__ pos,
                       const float* __restrict__ vel, const float* __restrict__ rho,
                       const int* __restrict__ tag, uint4* __restrict__ TX, float4* __restrict__ TB,
                       unsigned* __restrict__ ID, unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int o = idx[i];
  const int ph = is_wall ? 0 : tag[o];
  uint4 x;
  unsigned fx, fy, fz = 0u;
  fx_split(p, fx_tot_from_double((double)pos[3 * o], p.O[0], p.Q), x.x, fx);
  fx_split(p, fx_tot_from_double((double)pos[3 * o + 1], p.O[1], p.Q), x.y, fy);
  x.z = 0u;
  if (p.dim == 3) fx_split(p, fx_tot_from_double((double)pos[3 * o + 2], p.O[2], p.Q), x.z, fz);
  x.w = fx_pack(fx, fy, fz, (unsigned)ph);
  TX[i] = x;
  if (is_wall) {
    TB[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  } else {
    const float drho = (float)((double)rho[o] - (double)p.rho0[ph]);
    TB[i] = make_float4(vel[3 * o], vel[3 * o + 1], p.dim == 3 ? vel[3 * o + 2] : 0.0f, drho);
  }
  ID[i] = (unsigned)o;
  keys[i] = sort_key(p, fx_image(p, x, 0), fx_image(p, x, 1), p.dim == 3 ? fx_image(p, x, 2) : 0.0f);
  vals[i] = (unsigned)i;
}

// sph_set_particles: class of every caller entry as a sort key (0 fluid, 1 wall, 2 tag out of range) with its index;
// a stable sort by this key leaves the fluid entries first, then the wall entries, each in ascending caller order.
__global__ void __launch_bounds__(256)
k_classify(int n, int n_phases, const int* __restrict__ tag, unsigned* __restrict__ keys, unsigned* __restrict__ vals,
           unsigned long long* __restrict__ counts) {
  __shared__ unsigned sm[3];
  if (threadIdx.x < 3) sm[threadIdx.x] = 0u;
  __syncthreads();
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i < n) {
    const int t = tag[i];
    const unsigned k = t == SPH_TAG_WALL ? 1u : (t >= 0 && t < n_phases ? 0u : 2u);
    keys[i] = k;
    vals[i] = (unsigned)i;
    atomicAdd(&sm[k], 1u);
  }
  __syncthreads();
  if (threadIdx.x < 3 && sm[threadIdx.x]) atomicAdd(&counts[threadIdx.x], (unsigned long long)sm[threadIdx.x]);
}

// NEXT-1: the wall normals are invariant under the rigid translation: kept in set-up order (k_unsort4 at
// the set-up), gathered into the new cell order every step (k_gather4) instead of being recomputed.
__global__ void __launch_bounds__(256)
k_unsort4(int n, const unsigned* __restrict__ vals, const float4* __restrict__ in, float4* __restrict__ out) {
  const int s = blockIdx.x * 256 + threadIdx.x;
  if (s < n) out[vals[s]] = in[s];
}
__global__ void __launch_bounds__(256)
k_gather4(int n, const unsigned* __restrict__ vals, const float4* __restrict__ in, float4* __restrict__ out) {
  const int s = blockIdx.x * 256 + threadIdx.x;
  if (s < n) out[s] = in[vals[s]];
}

__global__ void __launch_bounds__(256)
k_gatherx(int n, const unsigned* __restrict__ vals, const uint4* __restrict__ in, uint4* __restrict__ out) {
  const int s = blockIdx.x * 256 + threadIdx.x;
  if (s < n) out[s] = in[vals[s]];
}

// a wall particle's set-up position displaced by the wall motion of t^{n+1} (S->sq: units of Q = 1024 units of the
// 42-bit coordinate); the sum stays inside the span because the domain box contains the whole excursion
__device__ __forceinline__ uint4 wall_shifted(const DP& p, const SS* __restrict__ S, uint4 x) {
  unsigned f[3] = {fx_field(x, 0), fx_field(x, 1), fx_field(x, 2)};
  unsigned w[3] = {x.x, x.y, x.z};
  for (int k = 0; k < p.dim; ++k) {
    const long long t = (long long)fx_tot(p, w[k], f[k]) + ((long long)S->sq[k] << 10);
    fx_split(p, (unsigned long long)min(max(t, 0ll), 4398046511103ll), w[k], f[k]);
  }
  return make_uint4(w[0], w[1], w[2], fx_pack(f[0], f[1], f[2], x.w & 3u));
}

// NEXT-1 (moving walls): wall particles in set-up order at their displaced positions X0 + sq, with the
// cell hash of the new position; input of the per-step wall re-sort.
__global__ void __launch_bounds__(256)
k_wall_shift(DP p, const SS* __restrict__ S, int nw, const uint4* __restrict__ X0, uint4* __restrict__ TX,
             float4* __restrict__ TB, unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= nw) return;
  const uint4 x = wall_shifted(p, S, X0[i]);
  TX[i] = x;
  TB[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  keys[i] = sort_key(p, fx_image(p, x, 0), fx_image(p, x, 1), p.dim == 3 ? fx_image(p, x, 2) : 0.0f);
  vals[i] = (unsigned)i;
}

// Gather into cell-sorted order and derive the centred float32 image used by the candidate filter;
// the same launch computes the cell lower bounds (one thread per cell, independent work: one graph
// node less per step).  lb[c] = number of sorted particles with key < c, c = 0..ncell: the three cells
// of an x-row of the stencil are one contiguous range [lb[c0], lb[c1+1]).  Binary search in the
// sorted keys (the tank may be mostly dry: no serial gap filling).
__global__ void __launch_bounds__(256)
k_reorder(DP p, int n, const unsigned* __restrict__ vals, const uint4* __restrict__ TX,
          const float4* __restrict__ TB, const unsigned* __restrict__ IDin, XB* __restrict__ R,
          float4* __restrict__ A, unsigned* __restrict__ IDout,
          const unsigned* __restrict__ keys, int ncell, int* __restrict__ lb) {
  const int s = blockIdx.x * 256 + threadIdx.x;
  if (s <= ncell) {
    int lo = 0, hi = n;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if ((keys[mid] >> p.sub_bits) < (unsigned)s) lo = mid + 1; else hi = mid;
    }
    lb[s] = lo;
  }
  if (s >= n) return;
  const unsigned v = vals[s];
  const uint4 x = TX[v];
  R[s] = XB{x, TB[v]};
  A[s] = centred_image(p, x);
  IDout[s] = IDin[v];
}

// ------------------------------------------------------------------------------------------
// Time step, Eq. 2.23-2.24 (reading A17): grid-stride max |v|^2 with warp
// shuffles, one atomicMax per block; the last block to finish computes dt and g(t^{n+1}).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_dt(DP p, SS* __restrict__ S, int nf, const float4* __restrict__ B, const double* __restrict__ dt_seq,
     int seq_idx) {
  __shared__ float sm[8];
  float m = 0.f;
  for (int i = blockIdx.x * 256 + threadIdx.x; i < nf; i += gridDim.x * 256) {
    const float4 v = B[i];
    m = fmaxf(m, fmaf(v.z, v.z, fmaf(v.y, v.y, v.x * v.x)));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(FULL, m, o));
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x != 0) return;
  for (int w = 1; w < 8; ++w) m = fmaxf(m, sm[w]);
  if (!(m == m) || isinf(m)) { atomicAdd(&S->nonfinite, 1ull); m = 0.f; }
  atomicMax(&S->vmax2_bits, __float_as_uint(m));
  __threadfence();
  const unsigned done = atomicAdd(&S->blocks_done, 1u);
  if (done != gridDim.x - 1) return;
  __threadfence();
  const double vmax = sqrt((double)__uint_as_float(atomicMax(&S->vmax2_bits, 0u)));
  double g[3];
  auto grav = [&](double t) {
    const double s = p.gperiod > 0.0 ? sin(6.283185307179586476925286766559 * t / p.gperiod) : 0.0;
    for (int k = 0; k < 3; ++k) g[k] = p.g[k] + p.gamp[k] * s;
  };
  double dt;
  if (dt_seq) {
    dt = dt_seq[seq_idx];
  } else {
    dt = p.cfl * p.hD / (p.cmax + vmax);  // Eq. 2.23
    grav(S->t);
    const double gn = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
    if (gn > 0.0) dt = fmin(dt, p.cfl * sqrt(p.hD / gn));  // Eq. 2.24
    if (!(dt > 1e-12)) S->dt_underflow = 1;
  }
  grav(S->t + dt);
  S->g[0] = (float)g[0]; S->g[1] = (float)g[1]; S->g[2] = (float)g[2];
  {  // NEXT-1: rigid wall motion at t^{n+1}: displacement, velocity, g - a_w
    double sn = 0.0, cs = 1.0;
    if (p.womega != 0.0) sincos(p.womega * (S->t + dt), &sn, &cs);  // static walls: gw = g, v_wall = 0, no displacement
    for (int k = 0; k < 3; ++k) {
      S->sq[k] = (int)rint(p.wamp[k] * sn / p.Q);
      S->vwall[k] = (float)(p.wamp[k] * p.womega * cs);
      S->gw[k] = (float)(g[k] + p.wamp[k] * p.womega * p.womega * sn);
    }
  }
  S->dt_d = dt;
  S->dt = (float)dt;
  S->t += dt;
  S->steps += 1;
  S->vmax2_bits = 0u;
  S->blocks_done = 0u;
  S->escaped = 0ull;
}

// One axis of the drift Eq. 2.20 on the fixed-point master position: the coordinate is a 42-bit integer in units
// of Q/1024; the displacement dt*v is rounded to that unit.
__device__ __forceinline__ void drift_axis(const DP& p, unsigned& mid, unsigned& field, double disp_sub) {
  long long tot = (long long)fx_tot(p, mid, field) + __double2ll_rn(disp_sub);
  tot = min(max(tot, 0ll), 4398046511103ll);
  fx_split(p, (unsigned long long)tot, mid, field);
}

// Predictor: density reinitialisation Eq. 2.17 / 2.18 from the sigma_i of the last pass A
// (same positions, reading A13), first half kick Eq. 2.19, drift Eq. 2.20,
// cell hash of the new position.  In place on (v, rho); the new record goes to Rout (the input of the
// pair passes when the lists are kept) and the new position to TX (the input of the reorder when
// they are rebuilt).
// Verlet skin: the block maxima of |dx_i|^2 are combined with atomicMax and the last block to finish
// adds this step's largest displacement to S->disp, decides whether the lists (built with radius
// 2h(1 + skin)) still hold every pair within 2h, and publishes the decision: S->rebuild and, when
// the step runs as a CUDA graph, the condition of the IF node that holds the rebuild branch.
// DO_REINIT / DO_MOVE = false give the stand-alone "density reinitialisation kernel" and "integrator"
// that BASELINE.json's config 4 asks to be timed separately (sph_debug_time_pointwise); the step
// itself runs the fused <true, true> form.
template <bool DO_REINIT, bool DO_MOVE>
__global__ void __launch_bounds__(256)
k_predict(DP p, SS* __restrict__ S, int nf, const XB* __restrict__ R, float4* __restrict__ B,
          const float4* __restrict__ ACC, const float* __restrict__ SIG, uint4* __restrict__ TX,
          XB* __restrict__ Rout, unsigned* __restrict__ keys, unsigned* __restrict__ vals,
          cudaGraphConditionalHandle cond, int use_cond, int decide) {
  __shared__ float smax[8];
  const int i = blockIdx.x * 256 + threadIdx.x;
  float d2 = 0.f;
  if (i < nf) {
    uint4 x = R[i].x;
    float4 b = B[i];
    const int ph = phase_of(x);
    if (DO_REINIT && (p.flags & SPH_FLAG_REINIT)) {
      const float rho0 = p.rho0[ph];
      const float ds = rho0 * SIG[i];  // rho0 sigma/sigma0 - rho0; SIG holds sigma/sigma0 - 1
      float d = ds;
      // Eq. 2.17 for rho* > rho_s: rho - rho0 = rho_s (rho* - rho0) / rho*  (same value as
      // rho_s + (rho* - rho_s) rho0 / rho*, without the cancellation of two O(rho0) terms)
      if (((p.fs_mask >> ph) & 1u) && b.w > ds) d = b.w * ((rho0 + ds) / (rho0 + b.w));
      b.w = d;
    }
    if (DO_MOVE) {
      const float4 a = ACC[i];
      const float hdt = 0.5f * S->dt;
      b.x = fmaf(hdt, a.x, b.x); b.y = fmaf(hdt, a.y, b.y); b.z = fmaf(hdt, a.z, b.z);  // Eq. 2.19
      const bool fin = isfinite(b.x) && isfinite(b.y) && isfinite(b.z);
      if (fin) {
        const double k = S->dt_d * p.sub_per_m;
        unsigned fx = fx_field(x, 0), fy = fx_field(x, 1), fz = fx_field(x, 2);
        drift_axis(p, x.x, fx, k * (double)b.x);
        drift_axis(p, x.y, fy, k * (double)b.y);
        if (p.dim == 3) drift_axis(p, x.z, fz, k * (double)b.z);
        x.w = fx_pack(fx, fy, fz, (unsigned)ph);
        // this step's displacement, rounded up: |dx| <= dt |v| (1 + 2^-20) + one sub-quantum per axis
        const float dtf = S->dt * 1.000001f;
        d2 = dtf * dtf * fmaf(b.z, b.z, fmaf(b.y, b.y, b.x * b.x));
      } else {
        atomicAdd(&S->nonfinite, 1ull);
      }
      TX[i] = x;
      const float gx = fx_image(p, x, 0), gy = fx_image(p, x, 1);
      const float gz = p.dim == 3 ? fx_image(p, x, 2) : 0.0f;
      bool out = gx < p.dmin[0] || gx >= p.dmax[0] || gy < p.dmin[1] || gy >= p.dmax[1];
      if (p.dim == 3) out = out || gz < p.dmin[2] || gz >= p.dmax[2];
      if (out || !fin) atomicAdd(&S->escaped, 1ull);
      keys[i] = sort_key(p, gx, gy, gz);
      vals[i] = (unsigned)i;
    }
    B[i] = b;
    Rout[i] = XB{x, b};
  }
  if (!decide) return;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) d2 = fmaxf(d2, __shfl_xor_sync(FULL, d2, o));
  if ((threadIdx.x & 31) == 0) smax[threadIdx.x >> 5] = d2;
  __syncthreads();
  if (threadIdx.x != 0) return;
  for (int w = 1; w < 8; ++w) d2 = fmaxf(d2, smax[w]);
  if (d2 > 0.f) atomicMax(&S->dmax2_bits, __float_as_uint(d2));
  __threadfence();
  if (atomicAdd(&S->blocks_done2, 1u) != gridDim.x - 1) return;
  __threadfence();
  const double dstep = sqrt((double)__uint_as_float(atomicMax(&S->dmax2_bits, 0u))) + 2.0 * p.Q;
  double disp = S->disp + dstep;
  double dw2 = 0.0, dws2 = 0.0;
  for (int k = 0; k < 3; ++k) {
    const double d = p.Q * (double)(S->sq[k] - S->sq_build[k]), e = p.Q * (double)(S->sq[k] - S->sq_prev[k]);
    dw2 += d * d;
    dws2 += e * e;
    S->sq_prev[k] = S->sq[k];
  }
  // the skin the next build should take: optimum for this step's displacement, 20 % head room
  const double delta = (dstep + sqrt(dws2)) / p.hD, beta = 0.65;
  double snext = 1.2 * (-2.0 * beta * delta + sqrt(4.0 * beta * beta * delta * delta + 12.0 * beta * delta)) / 6.0;
  snext = fmin(fmax(snext, p.skin_min), p.skin);
  const int since = S->since + 1;
  const bool stale = 2.0 * disp > S->budget || disp + sqrt(dw2) > S->budget;   // a pair beyond the list radius may be within 2h
  const bool loose = S->skin_cur > 1.5 * snext + 0.004 && since >= 4;          // the lists carry far more entries than they need to
  const int rb = (p.skin <= 0.0 || stale || loose) ? 1 : 0;
  if (rb) {
    disp = 0.0;
    for (int k = 0; k < 3; ++k) S->sq_build[k] = S->sq[k];
    S->rebuilds += 1;
    if (p.skin > 0.0) {
      const double rl = 2.0 * p.hD * (1.0 + snext);
      S->skin_cur = snext;
      S->budget = 2.0 * p.hD * snext * (1.0 - 1e-6);
      S->rl2m = __double2float_ru(rl * rl + p.marg32);
      const double thr = 4.08 * (1.0 + snext) * (1.0 + snext) + p.marg16;
      __half th = __double2half(thr);
      if ((double)__half2float(th) < thr) th = __ushort_as_half((unsigned short)(__half_as_ushort(th) + 1));
      S->thr_h2 = (unsigned)__half_as_ushort(th) * 0x10001u;
    }
  }
  S->since = rb ? 0 : since;
  S->disp = disp;
  S->rebuild = rb;
  S->dmax2_bits = 0u;
  S->blocks_done2 = 0u;
  if (use_cond) cudaGraphSetConditional(cond, (unsigned)rb);
}

// NEXT-1 with kept lists: the wall records in their cell order of the last list build, at the displacement of
// t^{n+1} (WXB: the positions of sph_set_particles in that order).
__global__ void __launch_bounds__(256)
k_wall_move(DP p, const SS* __restrict__ S, int nw, const uint4* __restrict__ WXB, XB* __restrict__ WR) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= nw) return;
  WR[i].x = wall_shifted(p, S, WXB[i]);
}

// Wall normals, Eq. 2.16, once, in float64 (reading A10).
template <int DIM>
__global__ void k_normals(DP p, int nw, const XB* __restrict__ WR, const unsigned* __restrict__ WK,
                          const int* __restrict__ lbW, float4* __restrict__ WN) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= nw) return;
  const uint4 xi = WR[w].x;
  const unsigned key = WK[w] >> p.sub_bits;
  const unsigned row = key / (unsigned)p.nx;
  const int cx = (int)(key - row * (unsigned)p.nx), cz = (int)(row / (unsigned)p.ny),
            cy = (int)(row - (unsigned)cz * (unsigned)p.ny);
  const double h = p.hD, rc2 = 4.0 * h * h;
  const double PI = 3.14159265358979323846264338327950288;
  const double alpha = DIM == 2 ? 7.0 / (4.0 * PI * h * h) : 21.0 / (16.0 * PI * h * h * h);
  const double dpd = p.dpD;
  const double V0 = DIM == 2 ? dpd * dpd : dpd * dpd * dpd;
  double px = 0, py = 0, pz = 0;
  const int RC = p.reach;
  for (int dz = (DIM == 3 ? -RC : 0); dz <= (DIM == 3 ? RC : 0); ++dz)
    for (int dy = -RC; dy <= RC; ++dy) {
      const int y = cy + dy, z = cz + dz;
      if (y < 0 || y >= p.ny || z < 0 || z >= p.nz) continue;
      const int rb = (z * p.ny + y) * p.nx;
      const int s = lbW[rb + max(cx - RC, 0)], e = lbW[rb + min(cx + RC, p.nx - 1) + 1];
      for (int j = s; j < e; ++j) {
        if (j == w) continue;
        const uint4 xj = WR[j].x;
        const double dx = p.Qp * (double)(int)(xi.x - xj.x), dyy = p.Qp * (double)(int)(xi.y - xj.y),
                     dzz = DIM == 3 ? p.Qp * (double)(int)(xi.z - xj.z) : 0.0;
        const double r2 = dx * dx + dyy * dyy + dzz * dzz;
        if (!(r2 < rc2) || r2 == 0.0) continue;
        const double r = sqrt(r2), q = r / h, t = 1.0 - 0.5 * q;
        const double dw = -5.0 * alpha / h * q * t * t * t;
        const double f = -V0 * dw / r;  // -(m_j/rho_j) grad_i W_ij = f * r_ij
        px += f * dx; py += f * dyy; pz += f * dzz;
      }
    }
  const double nrm = sqrt(px * px + py * py + pz * pz);
  float4 n = make_float4(0.f, 0.f, 0.f, 0.f);
  if (nrm * h >= 1e-3) n = make_float4((float)(px / nrm), (float)(py / nrm), (float)(pz / nrm), 0.f);
  WN[w] = n;
}

// wnear[c] = 1 if any wall particle lies in the 27 / 9-cell stencil of cell c (static, set-up):
// lets the fluid pair kernels skip the wall walk for warps in the bulk.
__global__ void k_wnear(DP p, int ncell, const int* __restrict__ lbW, unsigned char* __restrict__ wnear) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  const int row = c / p.nx, cx = c - row * p.nx, cz = row / p.ny, cy = row - cz * p.ny;
  int any = 0;
  const int RC = p.reach;
  for (int dz = (p.dim == 3 ? -RC : 0); dz <= (p.dim == 3 ? RC : 0); ++dz)
    for (int dy = -RC; dy <= RC; ++dy) {
      const int y = cy + dy, z = cz + dz;
      if (y < 0 || y >= p.ny || z < 0 || z >= p.nz) continue;
      const int rb = (z * p.ny + y) * p.nx;
      any |= lbW[rb + min(cx + RC, p.nx - 1) + 1] > lbW[rb + max(cx - RC, 0)];
    }
  wnear[c] = (unsigned char)any;
}
