// paper_2110_02621_b200/csrc/sph.cu — libsph: the per-time-step SPH pipeline of
// arXiv 2110.02621 as hand-written CUDA for B200 (sm_100a) behind the C ABI of include/sph.h.
//
// Citations: PAPER.md:<line> / equation; readings Axx are listed in DESIGN.md §3.
// Nothing here is shared with oracle/ (the CPU checker); there is no CPU fallback.
//
// Data layout: fluid and wall particles live in separate cell-sorted
// structure-of-arrays float4 buffers.  pos4 = (x, y, z, rho - rho0_phase), vel4 = (vx, vy, vz,
// phase id bits); wall pos4 = (x, y, z, p_w), wall vel4 = (v_w, 0), wall nrm4 = (n_w, 0).
// The wall structure is built once; the fluid one every step.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <string>
#include <vector>

#include "sph.h"

namespace {

// ------------------------------------------------------------------------------------------
// Device-side parameter block (passed by value to every kernel).
// ------------------------------------------------------------------------------------------
struct DP {
  int dim, n_phases;
  float h, hinv, dp, rc2;
  float alpha;   // kernel normalisation alpha_d (reading A1)
  float gradc;   // W'(r)/r = gradc * (1 - q/2)^3,  gradc = -5 alpha / h^2
  float w0;      // W(0)
  float V0;      // dp^dim
  float rho0[SPH_MAX_PHASES], c0[SPH_MAX_PHASES], c2[SPH_MAX_PHASES], inv_c2[SPH_MAX_PHASES],
      mass[SPH_MAX_PHASES];
  float sigma0, inv_sigma0;
  float gamma_p, two_over_dp;
  unsigned pen_mask, fs_mask, flags;
  float ox, oy, oz, inv_edge;
  int nx, ny, nz;
  float dmin[3], dmax[3];
  double cmax, cfl, hD;
  double massD[SPH_MAX_PHASES];
  double hinvD, a_over_s0, sigma0D;
  double g[3], gamp[3], gperiod;
};

// Device-resident per-step state: written by k_dt, read by every other kernel, so that
// sph_step(n) needs no host synchronisation between steps.
struct SS {
  double t;
  double dt_d;
  float dt;
  float g[3];            // gravity at t^{n+1} (reading A28)
  unsigned vmax2_bits;   // max |v|^2 over fluid, float bits (non-negative -> ordered as uint)
  unsigned blocks_done;
  long long steps;
  unsigned long long escaped, nonfinite;
  int dt_underflow;
};

#define FULL 0xffffffffu

__device__ __forceinline__ int cell_coord(float x, float o, float inv, int n) {
  // Integer contract (reading A24): one FP32 subtract, one FP32 multiply, no contraction.
  float u = __fmul_rn(__fsub_rn(x, o), inv);
  u = fminf(fmaxf(floorf(u), 0.0f), (float)(n - 1));  // NaN -> 0
  return (int)u;
}

__device__ __forceinline__ float dist2(float dx, float dy, float dz) {
  // reading A24: r2 = fmaf(dz,dz,fmaf(dy,dy,dx*dx)); in 2-D dz = 0 adds exactly 0.
  return fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx)));
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}

// ------------------------------------------------------------------------------------------
// Loading (sph_set_particles): split caller arrays into the fluid / wall structures.
// ------------------------------------------------------------------------------------------
__global__ void k_load_fluid(DP p, int nf, const int* __restrict__ fid, const float* __restrict__ pos,
                             const float* __restrict__ vel, const float* __restrict__ rho,
                             const int* __restrict__ tag, float4* __restrict__ TP,
                             float4* __restrict__ TV, double2* __restrict__ TDxy, double* __restrict__ TDz,
                             unsigned* __restrict__ ID,
                             unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nf) return;
  int o = fid[i];
  int ph = tag[o];
  float x = pos[3 * o], y = pos[3 * o + 1], z = p.dim == 3 ? pos[3 * o + 2] : 0.0f;
  float drho = (float)((double)rho[o] - (double)p.rho0[ph]);
  TP[i] = make_float4(x, y, z, drho);
  TDxy[i] = make_double2((double)x, (double)y);
  TDz[i] = (double)z;
  TV[i] = make_float4(vel[3 * o], vel[3 * o + 1], p.dim == 3 ? vel[3 * o + 2] : 0.0f,
                      __int_as_float(ph));
  ID[i] = (unsigned)o;
  int cx = cell_coord(x, p.ox, p.inv_edge, p.nx), cy = cell_coord(y, p.oy, p.inv_edge, p.ny);
  int cz = p.dim == 3 ? cell_coord(z, p.oz, p.inv_edge, p.nz) : 0;
  keys[i] = (unsigned)((cz * p.ny + cy) * p.nx + cx);
  vals[i] = (unsigned)i;
}

__global__ void k_load_wall(DP p, int nw, const int* __restrict__ wid, const float* __restrict__ pos,
                            float4* __restrict__ TP, unsigned* __restrict__ ID,
                            unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nw) return;
  int o = wid[i];
  float x = pos[3 * o], y = pos[3 * o + 1], z = p.dim == 3 ? pos[3 * o + 2] : 0.0f;
  TP[i] = make_float4(x, y, z, 0.0f);
  ID[i] = (unsigned)o;
  int cx = cell_coord(x, p.ox, p.inv_edge, p.nx), cy = cell_coord(y, p.oy, p.inv_edge, p.ny);
  int cz = p.dim == 3 ? cell_coord(z, p.oz, p.inv_edge, p.nz) : 0;
  keys[i] = (unsigned)((cz * p.ny + cy) * p.nx + cx);
  vals[i] = (unsigned)i;
}

// ------------------------------------------------------------------------------------------
// Device radix sort (stable LSD, 8-bit digits) of (cell id, index).  BASELINE.json north_star
// "cell hash, device radix sort"; the paper only names the step.
// Per pass: tile histograms -> row sums -> scan -> stable scatter with warp match ranking.
// ------------------------------------------------------------------------------------------
constexpr int RS_THREADS = 256, RS_ITEMS = 16, RS_TILE = RS_THREADS * RS_ITEMS, RS_WARPS = 8;

__global__ void __launch_bounds__(RS_THREADS)
k_radix_hist(const unsigned* __restrict__ keys, int n, int shift, unsigned* __restrict__ hist,
             int nblk) {
  __shared__ unsigned h[256];
  h[threadIdx.x] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int base = blockIdx.x * RS_TILE;
#pragma unroll 4
  for (int it = 0; it < RS_ITEMS; ++it) {
    int idx = base + it * RS_THREADS + threadIdx.x;
    bool ok = idx < n;
    unsigned d = ok ? ((keys[idx] >> shift) & 255u) : 256u;
    unsigned peers = __match_any_sync(FULL, d);
    if (ok && lane == __ffs(peers) - 1) atomicAdd(&h[d], (unsigned)__popc(peers));
  }
  __syncthreads();
  hist[threadIdx.x * nblk + blockIdx.x] = h[threadIdx.x];
}

__global__ void __launch_bounds__(256)
k_scan_rowsum(const unsigned* __restrict__ hist, int nblk, unsigned* __restrict__ rowsum) {
  __shared__ unsigned sm[8];
  unsigned s = 0;
  const unsigned* row = hist + (size_t)blockIdx.x * nblk;
  for (int i = threadIdx.x; i < nblk; i += 256) s += row[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned t = 0;
    for (int w = 0; w < 8; ++w) t += sm[w];
    rowsum[blockIdx.x] = t;
  }
}

// Exclusive scan of hist in (digit-major, block-minor) order, in place.
__global__ void __launch_bounds__(256)
k_scan_apply(unsigned* __restrict__ hist, int nblk, const unsigned* __restrict__ rowsum) {
  __shared__ unsigned sm[8];
  __shared__ unsigned carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // base = sum of rowsum[d'] for d' < digit
  unsigned b = (threadIdx.x < blockIdx.x) ? rowsum[threadIdx.x] : 0u;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) b += __shfl_xor_sync(FULL, b, o);
  if (lane == 0) sm[wid] = b;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned t = 0;
    for (int w = 0; w < 8; ++w) t += sm[w];
    carry_s = t;
  }
  __syncthreads();
  unsigned* row = hist + (size_t)blockIdx.x * nblk;
  for (int i0 = 0; i0 < nblk; i0 += 256) {
    int i = i0 + threadIdx.x;
    unsigned v = i < nblk ? row[i] : 0u;
    unsigned x = v;  // inclusive warp scan
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      unsigned y = __shfl_up_sync(FULL, x, o);
      if (lane >= o) x += y;
    }
    __syncthreads();  // previous iteration's readers of sm / carry_s are done
    if (lane == 31) sm[wid] = x;
    __syncthreads();
    unsigned woff = 0;
    for (int w = 0; w < wid; ++w) woff += sm[w];
    unsigned carry = carry_s;
    if (i < nblk) row[i] = carry + woff + x - v;
    __syncthreads();
    if (threadIdx.x == 255) carry_s = carry + woff + x;
  }
}

__global__ void __launch_bounds__(RS_THREADS)
k_radix_scatter(const unsigned* __restrict__ keys, const unsigned* __restrict__ vals, int n, int shift,
                const unsigned* __restrict__ hist, int nblk, unsigned* __restrict__ keys_out,
                unsigned* __restrict__ vals_out) {
  __shared__ unsigned wc[RS_WARPS][256];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < RS_WARPS * 256; i += RS_THREADS) (&wc[0][0])[i] = 0;
  __syncthreads();
  const int base = blockIdx.x * RS_TILE + wid * (RS_ITEMS * 32);
  unsigned k[RS_ITEMS], rank[RS_ITEMS];
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int it = 0; it < RS_ITEMS; ++it) {
    int idx = base + it * 32 + lane;  // warp-contiguous order keeps the sort stable
    bool ok = idx < n;
    k[it] = ok ? keys[idx] : 0xffffffffu;
    unsigned d = ok ? ((k[it] >> shift) & 255u) : 256u;
    unsigned peers = __match_any_sync(FULL, d);
    int leader = __ffs(peers) - 1;
    unsigned old = 0;
    if (ok && lane == leader) {
      old = wc[wid][d];
      wc[wid][d] = old + __popc(peers);
    }
    old = __shfl_sync(FULL, old, leader);
    rank[it] = old + __popc(peers & lt);
    __syncwarp();
  }
  __syncthreads();
  {  // exclusive prefix over warps per digit, plus the scanned global base of this tile
    unsigned d = threadIdx.x, run = hist[d * nblk + blockIdx.x];
#pragma unroll
    for (int w = 0; w < RS_WARPS; ++w) {
      unsigned t = wc[w][d];
      wc[w][d] = run;
      run += t;
    }
  }
  __syncthreads();
#pragma unroll
  for (int it = 0; it < RS_ITEMS; ++it) {
    int idx = base + it * 32 + lane;
    if (idx < n) {
      unsigned d = (k[it] >> shift) & 255u;
      unsigned dst = wc[wid][d] + rank[it];
      keys_out[dst] = k[it];
      vals_out[dst] = vals[idx];
    }
  }
}

// lb[c] = number of sorted particles with key < c, c = 0..ncell (dense lower bounds: the three
// cells of an x-row of the stencil are one contiguous range [lb[c0], lb[c1+1])).
__global__ void k_cell_bounds(const unsigned* __restrict__ keys, int n, int ncell, int* __restrict__ lb) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s > n) return;
  int kprev = s == 0 ? -1 : (int)keys[s - 1];
  int kcur = s == n ? ncell : (int)keys[s];
  for (int c = kprev + 1; c <= kcur; ++c) lb[c] = s;
}

__global__ void k_reorder(int n, const unsigned* __restrict__ vals, const float4* __restrict__ TP,
                          const float4* __restrict__ TV, const double2* __restrict__ TDxy,
                          const double* __restrict__ TDz, const unsigned* __restrict__ IDin,
                          float4* __restrict__ P, float4* __restrict__ V, double2* __restrict__ Dxy,
                          double* __restrict__ Dz, float4* __restrict__ L, unsigned* __restrict__ IDout) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  unsigned v = vals[s];
  const float4 r = TP[v];
  P[s] = r;
  if (TV) V[s] = TV[v];
  if (TDxy) {
    // float64 master position; (P.xyz, L.xyz) is its two-float image: hi = float32 rounding, lo = remainder
    const double2 xy = TDxy[v];
    const double z = TDz[v];
    Dxy[s] = xy;
    Dz[s] = z;
    L[s] = make_float4((float)(xy.x - (double)r.x), (float)(xy.y - (double)r.y), (float)(z - (double)r.z), 0.f);
  }
  IDout[s] = IDin[v];
}

// Static wall positions as float64 (exact images of the caller's float32), for the sigma sum.
__global__ void k_wall_double(int n, const float4* __restrict__ WP, double2* __restrict__ Dxy,
                              double* __restrict__ Dz) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const float4 r = WP[s];
  Dxy[s] = make_double2((double)r.x, (double)r.y);
  Dz[s] = (double)r.z;
}

// ------------------------------------------------------------------------------------------
// Stencil walk: one warp per particle, lanes over the candidates of each x-row of the
// 27 (3-D) / 9 (2-D) cell stencil (coalesced float4 loads), hits compacted through a
// per-warp shared-memory queue so that the expensive pair body runs with full warps.
// ------------------------------------------------------------------------------------------
template <typename Body>
__device__ __forceinline__ void walk(const DP& p, const float4* __restrict__ P, const int* __restrict__ lb,
                                     float xi, float yi, float zi, int self, unsigned* q, Body&& body) {
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  const int cx = cell_coord(xi, p.ox, p.inv_edge, p.nx), cy = cell_coord(yi, p.oy, p.inv_edge, p.ny);
  const int cz = p.dim == 3 ? cell_coord(zi, p.oz, p.inv_edge, p.nz) : 0;
  const int nrow = p.dim == 3 ? 9 : 3;
  int rs = 0, re = 0;
  if (lane < nrow) {
    int y = cy + (lane % 3) - 1, z = cz + (lane / 3) - 1;
    if (p.dim != 3) z = 0;
    if (y >= 0 && y < p.ny && z >= 0 && z < p.nz) {
      int rb = (z * p.ny + y) * p.nx;
      rs = lb[rb + max(cx - 1, 0)];
      re = lb[rb + min(cx + 1, p.nx - 1) + 1];
    }
  }
  int qn = 0, qh = 0;
  for (int r = 0; r < nrow; ++r) {
    const int s = __shfl_sync(FULL, rs, r), e = __shfl_sync(FULL, re, r);
    for (int j0 = s; j0 < e; j0 += 32) {
      const int j = j0 + lane;
      bool hit = false;
      if (j < e) {
        float4 pj = P[j];
        float r2 = dist2(xi - pj.x, yi - pj.y, zi - pj.z);
        hit = (r2 < p.rc2) && (j != self);
      }
      const unsigned m = __ballot_sync(FULL, hit);
      if (m) {
        if (hit) q[(qh + qn + __popc(m & lt)) & 63] = (unsigned)j;
        qn += __popc(m);
        __syncwarp();
        if (qn >= 32) {
          body((int)q[(qh + lane) & 63]);
          qh = (qh + 32) & 63;
          qn -= 32;
          __syncwarp();
        }
      }
    }
  }
  if (qn > 0) {
    __syncwarp();
    if (lane < qn) body((int)q[(qh + lane) & 63]);
  }
  __syncwarp();
}

constexpr int PW = 8;  // warps per block in the pair kernels

// W(r)/alpha_d = (1 - q/2)^4 (1 + 2q) in float64 from a float64 separation (reading A1).  Used only
// for the number density sigma_i, whose relative error is amplified by c0^2 ~ 200 g H into the
// pressure (DESIGN.md §4 "precision").  sqrt: one MUFU.RSQ64H seed + one Newton step (~1e-13).
__device__ __forceinline__ double wendland64(const DP& p, double dx, double dy, double dz) {
  const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(r2));
  const double e = fma(-r2 * y, y, 1.0);
  y = fma(0.5 * y, e, y);
  const double q = r2 > 0.0 ? r2 * y * p.hinvD : 0.0;
  const double t = fmax(fma(-0.5, q, 1.0), 0.0), t2 = t * t;
  return t2 * t2 * fma(2.0, q, 1.0);
}

// Wall extrapolation, Eq. 2.12 (readings A4-A7); a_w = 0, v_wall = 0.
template <bool MULTI, bool WITH_VEL>
__global__ void __launch_bounds__(PW * 32)
k_wall(DP p, const SS* __restrict__ S, int nw, float4* __restrict__ WP, float4* __restrict__ WV,
       const float4* __restrict__ P, const float4* __restrict__ V, const float4* __restrict__ LO,
       const int* __restrict__ lbF) {
  __shared__ unsigned qs[PW][64];
  const int w = blockIdx.x * PW + (threadIdx.x >> 5);
  if (w >= nw) return;
  const int lane = threadIdx.x & 31;
  const float4 pw = WP[w];
  float sW = 0, sp = 0, sWr = 0, srx = 0, sry = 0, srz = 0, svx = 0, svy = 0, svz = 0;
  walk(p, P, lbF, pw.x, pw.y, pw.z, -1, qs[threadIdx.x >> 5], [&](int j) {
    const float4 pj = P[j], lj = LO[j];
    // r_wf with the low-order part of the fluid position (two-float positions)
    const float dx = (pw.x - pj.x) - lj.x, dy = (pw.y - pj.y) - lj.y, dz = (pw.z - pj.z) - lj.z;
    const float r2 = dist2(dx, dy, dz);
    const float r = r2 > 0.f ? r2 * rsqrtf(r2) : 0.f;
    const float q = r * p.hinv, t = fmaf(-0.5f, q, 1.0f), t2 = t * t;
    const float W = p.alpha * t2 * t2 * fmaf(2.0f, q, 1.0f);
    int ph = 0;
    float4 vj;
    if (MULTI || WITH_VEL) vj = V[j];
    if (MULTI) ph = __float_as_int(vj.w);
    const float rhof = p.rho0[ph] + pj.w, pf = p.c2[ph] * pj.w;
    sW += W;
    if (MULTI) {
      const float ir = __fdividef(W, rhof);
      sp = fmaf(pf, ir, sp);
      sWr += ir;
      srx = fmaf(dx, W, srx); sry = fmaf(dy, W, sry); srz = fmaf(dz, W, srz);
    } else {
      sp = fmaf(pf, W, sp);
      const float rw = rhof * W;
      srx = fmaf(dx, rw, srx); sry = fmaf(dy, rw, sry); srz = fmaf(dz, rw, srz);
    }
    if (WITH_VEL) { svx = fmaf(vj.x, W, svx); svy = fmaf(vj.y, W, svy); svz = fmaf(vj.z, W, svz); }
  });
  sW = warp_sum(sW); sp = warp_sum(sp); srx = warp_sum(srx); sry = warp_sum(sry); srz = warp_sum(srz);
  if (MULTI) sWr = warp_sum(sWr);
  if (WITH_VEL) { svx = warp_sum(svx); svy = warp_sum(svy); svz = warp_sum(svz); }
  if (lane == 0) {
    float pwall = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
    if (sW > 0.f) {
      const float lever = S->g[0] * srx + S->g[1] * sry + S->g[2] * srz;
      pwall = (sp + lever) / (MULTI ? sWr : sW);
      if (WITH_VEL && (p.flags & SPH_FLAG_WALL_VEL_MIRROR)) {
        const float is = 1.0f / sW;
        vx = -svx * is; vy = -svy * is; vz = -svz * is;
      }
    }
    WP[w].w = pwall;
    if (WITH_VEL) WV[w] = make_float4(vx, vy, vz, 0.f);
  }
}

// Pair pass A: sigma_i + Riemann continuity Eq. 2.9 with Eq. 2.8
// in the scalar form (v_i - v*).grad W = (U* - U_L) W', then the density update
// Eq. 2.21 / summation Eq. 2.4 in the normalised form of Eq. 2.18 (readings A3, A5, A15).
template <bool MULTI>
__global__ void __launch_bounds__(PW * 32)
k_pass_a(DP p, const SS* __restrict__ S, int nf, int init, const float4* __restrict__ P,
         const float4* __restrict__ V, const double2* __restrict__ Dxy, const double* __restrict__ Dz,
         const int* __restrict__ lbF, const float4* __restrict__ WP, const float4* __restrict__ WV,
         const double2* __restrict__ WDxy, const double* __restrict__ WDz, const int* __restrict__ lbW,
         float4* __restrict__ Pout, float* __restrict__ SIG, float* __restrict__ DRHO, const unsigned* __restrict__ IDin,
         unsigned* __restrict__ IDout) {
  __shared__ unsigned qs[PW][64];
  const int i = blockIdx.x * PW + (threadIdx.x >> 5);
  if (i >= nf) return;
  const int lane = threadIdx.x & 31;
  unsigned* q = qs[threadIdx.x >> 5];
  const float4 pi = P[i], vi = V[i];
  const double2 xyi = Dxy[i];
  const double zi = p.dim == 3 ? Dz[i] : 0.0;
  const bool d3 = p.dim == 3;
  const int phi = MULTI ? __float_as_int(vi.w) : 0;
  const float rhoi = p.rho0[phi] + pi.w, prsi = p.c2[phi] * pi.w, ci = p.c0[phi], ZL = rhoi * ci;
  double sig = 0.0;
  float acc = 0.f;
  walk(p, P, lbF, pi.x, pi.y, pi.z, i, q, [&](int j) {
    const float4 pj = P[j], vj = V[j];
    const double2 xyj = Dxy[j];
    sig += wendland64(p, xyi.x - xyj.x, xyi.y - xyj.y, d3 ? zi - Dz[j] : 0.0);
    const float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;  // r_ij (float32 image)
    const float r2 = dist2(dx, dy, dz);
    const float r = r2 > 0.f ? r2 * rsqrtf(r2) : 0.f;
    const float qq = r * p.hinv, t = fmaf(-0.5f, qq, 1.0f), t2 = t * t;
    const float Fg = p.gradc * t2 * t;  // W'(r)/r
    const int phj = MULTI ? __float_as_int(vj.w) : 0;
    const float rhoj = p.rho0[phj] + pj.w;
    const float ZR = rhoj * p.c0[phj];
    const float dpr = (!MULTI || phj == phi) ? p.c2[phi] * (pi.w - pj.w) : prsi - p.c2[phj] * pj.w;
    const float vd = (vi.x - vj.x) * dx + (vi.y - vj.y) * dy + (vi.z - vj.z) * dz;
    const float num = fmaf(ZR, vd, dpr * r);  // (U* - U_L) W' (Z_L + Z_R) / Fg
    acc = fmaf(p.mass[phj] * Fg, __fdividef(num, rhoj * (ZL + ZR)), acc);
  });
  float accw = 0.f;
  walk(p, WP, lbW, pi.x, pi.y, pi.z, -1, q, [&](int j) {
    const float4 pj = WP[j], vj = WV[j];  // (x, y, z, p_w), v_w
    const double2 xyj = WDxy[j];
    sig += wendland64(p, xyi.x - xyj.x, xyi.y - xyj.y, d3 ? zi - WDz[j] : 0.0);
    const float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
    const float r2 = dist2(dx, dy, dz);
    const float r = r2 > 0.f ? r2 * rsqrtf(r2) : 0.f;
    const float qq = r * p.hinv, t = fmaf(-0.5f, qq, 1.0f), t2 = t * t;
    const float Fg = p.gradc * t2 * t;
    const float rhow = fmaf(pj.w, p.inv_c2[phi], p.rho0[phi]);  // reading A5
    const float ZR = rhow * ci;
    const float vd = (vi.x - vj.x) * dx + (vi.y - vj.y) * dy + (vi.z - vj.z) * dz;
    const float num = fmaf(ZR, vd, (prsi - pj.w) * r);
    accw = fmaf(Fg, __fdividef(num, ZL + ZR), accw);
  });
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sig += __shfl_xor_sync(FULL, sig, o);
  acc = warp_sum(acc);
  accw = warp_sum(accw);
  if (lane == 0) {
    // sigma_i / sigma0 - 1 in float64 (self term W(0) = alpha, reading A14), stored as float32:
    // the density of Eq. 2.17 / 2.18 is rho0 (1 + dev), so the deviation carries the precision.
    const float dev = (float)(p.a_over_s0 * (1.0 + sig) - 1.0);
    const float drho = 2.0f * rhoi * fmaf(p.V0, accw, acc);  // Eq. 2.9
    float d = pi.w;
    if (!init) {
      if ((p.fs_mask >> phi) & 1u) d = fmaf(S->dt, drho, d);          // Eq. 2.21
      else d = p.rho0[phi] * dev;                                      // Eq. 2.4 / 2.18
    }
    Pout[i] = make_float4(pi.x, pi.y, pi.z, d);
    SIG[i] = dev;
    DRHO[i] = drho;
    IDout[i] = IDin[i];
  }
}

// Pair pass B: momentum Eq. 2.10 with p* of Eq. 2.8 (fluid j) / Eq. 2.11 (wall j), penalty
// Eq. 2.13-2.15 (readings A8, A9b, A11), gravity, then the second half kick Eq. 2.22.
template <bool MULTI>
__global__ void __launch_bounds__(PW * 32)
k_pass_b(DP p, const SS* __restrict__ S, int nf, const float4* __restrict__ P,
         const float4* __restrict__ V, const float4* __restrict__ LO, const int* __restrict__ lbF,
         const float4* __restrict__ WP, const float4* __restrict__ WN, const int* __restrict__ lbW,
         float4* __restrict__ Vout,
         float4* __restrict__ ACC) {
  __shared__ unsigned qs[PW][64];
  const int i = blockIdx.x * PW + (threadIdx.x >> 5);
  if (i >= nf) return;
  const int lane = threadIdx.x & 31;
  unsigned* q = qs[threadIdx.x >> 5];
  const float4 pi = P[i], vi = V[i], li = LO[i];
  const int phi = MULTI ? __float_as_int(vi.w) : 0;
  const float rhoi = p.rho0[phi] + pi.w, prsi = p.c2[phi] * pi.w, ZL = rhoi * p.c0[phi];
  float ax = 0.f, ay = 0.f, az = 0.f;
  walk(p, P, lbF, pi.x, pi.y, pi.z, i, q, [&](int j) {
    const float4 pj = P[j], vj = V[j], lj = LO[j];
    const float dx = (pi.x - pj.x) + (li.x - lj.x), dy = (pi.y - pj.y) + (li.y - lj.y),
                dz = (pi.z - pj.z) + (li.z - lj.z);
    const float r2 = dist2(dx, dy, dz);
    const float rinv = r2 > 0.f ? rsqrtf(r2) : 0.f;
    const float qq = r2 * rinv * p.hinv, t = fmaf(-0.5f, qq, 1.0f);
    const float Fg = p.gradc * t * t * t;
    const int phj = MULTI ? __float_as_int(vj.w) : 0;
    const float rhoj = p.rho0[phj] + pj.w, prsj = p.c2[phj] * pj.w, ZR = rhoj * p.c0[phj];
    const float vd = (vi.x - vj.x) * dx + (vi.y - vj.y) * dy + (vi.z - vj.z) * dz;
    const float dU = -vd * rinv;  // U_L - U_R
    const float izs = __fdividef(1.0f, ZL + ZR);
    const float ctil = (ZL + ZR) * __fdividef(1.0f, rhoi + rhoj);
    const float beta = fminf(3.0f * fmaxf(dU, 0.f), ctil);
    const float pstar = fmaf(ZL, prsj, ZR * prsi) * izs + ZL * ZR * izs * __fdividef(beta, ctil) * dU;
    const float coef = -2.0f * __fdividef(p.mass[phj] * pstar, rhoj * rhoi) * Fg;  // Eq. 2.10
    ax = fmaf(coef, dx, ax); ay = fmaf(coef, dy, ay); az = fmaf(coef, dz, az);
  });
  const bool pen = (p.pen_mask >> phi) & 1u;
  walk(p, WP, lbW, pi.x, pi.y, pi.z, -1, q, [&](int j) {
    const float4 pj = WP[j];
    const float dx = (pi.x - pj.x) + li.x, dy = (pi.y - pj.y) + li.y, dz = (pi.z - pj.z) + li.z;
    const float r2 = dist2(dx, dy, dz);
    const float rinv = r2 > 0.f ? rsqrtf(r2) : 0.f;
    const float r = r2 * rinv;
    const float qq = r * p.hinv, t = fmaf(-0.5f, qq, 1.0f);
    const float Fg = p.gradc * t * t * t;
    const float rhow = fmaf(pj.w, p.inv_c2[phi], p.rho0[phi]);
    const float pstar = __fdividef(fmaf(rhoi, pj.w, rhow * prsi), rhoi + rhow);  // Eq. 2.11
    const float coef = -2.0f * p.V0 * __fdividef(pstar, rhoi) * Fg;
    ax = fmaf(coef, dx, ax); ay = fmaf(coef, dy, ay); az = fmaf(coef, dz, az);
    if (pen) {
      const float4 n = WN[j];
      if (n.x != 0.f || n.y != 0.f || n.z != 0.f) {
        const float nd = n.x * dx + n.y * dy + n.z * dz;   // n_w . (r_i - r_w)
        const float delta = nd * p.two_over_dp;            // Eq. 2.15 (reading A9b)
        if (delta < 1.0f && delta > -1.0f) {
          const float lam = (1.0f - delta) * (1.0f - delta);  // Eq. 2.14 (reading A8)
          const float Pn = p.gamma_p * lam * fabsf(prsi * nd * rinv);
          const float c = -2.0f * p.V0 * __fdividef(Pn, rhoi) * (Fg * r);  // Eq. 2.13, W' = Fg r
          ax = fmaf(c, n.x, ax); ay = fmaf(c, n.y, ay); az = fmaf(c, n.z, az);
        }
      }
    }
  });
  ax = warp_sum(ax); ay = warp_sum(ay); az = warp_sum(az);
  if (lane == 0) {
    ax += S->g[0]; ay += S->g[1]; az += S->g[2];
    if (p.dim != 3) az = 0.f;
    ACC[i] = make_float4(ax, ay, az, 0.f);
    const float hdt = 0.5f * S->dt;
    Vout[i] = make_float4(fmaf(hdt, ax, vi.x), fmaf(hdt, ay, vi.y), fmaf(hdt, az, vi.z), vi.w);  // Eq. 2.22
  }
}

// Time step, Eq. 2.23-2.24 (reading A17): grid-stride max |v|^2 with warp
// shuffles, one atomicMax per block; the last block to finish computes dt and g(t^{n+1}).
__global__ void __launch_bounds__(256)
k_dt(DP p, SS* __restrict__ S, int nf, const float4* __restrict__ V, const double* __restrict__ dt_seq,
     int seq_idx) {
  __shared__ float sm[8];
  float m = 0.f;
  for (int i = blockIdx.x * 256 + threadIdx.x; i < nf; i += gridDim.x * 256) {
    float4 v = V[i];
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
  unsigned done = atomicAdd(&S->blocks_done, 1u);
  if (done != gridDim.x - 1) return;
  __threadfence();
  const double vmax = sqrt((double)__uint_as_float(atomicMax(&S->vmax2_bits, 0u)));
  double g[3];
  auto grav = [&](double t) {
    double s = p.gperiod > 0.0 ? sin(6.283185307179586476925286766559 * t / p.gperiod) : 0.0;
    for (int k = 0; k < 3; ++k) g[k] = p.g[k] + p.gamp[k] * s;
  };
  double dt;
  if (dt_seq) {
    dt = dt_seq[seq_idx];
  } else {
    dt = p.cfl * p.hD / (p.cmax + vmax);  // Eq. 2.23
    grav(S->t);
    double gn = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
    if (gn > 0.0) dt = fmin(dt, p.cfl * sqrt(p.hD / gn));  // Eq. 2.24
    if (!(dt > 1e-12)) S->dt_underflow = 1;
  }
  grav(S->t + dt);
  S->g[0] = (float)g[0]; S->g[1] = (float)g[1]; S->g[2] = (float)g[2];
  S->dt_d = dt;
  S->dt = (float)dt;
  S->t += dt;
  S->steps += 1;
  S->vmax2_bits = 0u;
  S->blocks_done = 0u;
  S->escaped = 0ull;
}

// Predictor: density reinitialisation Eq. 2.17 / 2.18 from the sigma_i of the last pass A
// (same positions, reading A13), first half kick Eq. 2.19, drift Eq. 2.20,
// cell hash of the new position.
__global__ void __launch_bounds__(256)
k_predict(DP p, SS* __restrict__ S, int nf, const float4* __restrict__ P, const float4* __restrict__ V,
          const float4* __restrict__ ACC, const float* __restrict__ SIG, const double2* __restrict__ Dxy,
          const double* __restrict__ Dz, float4* __restrict__ TP, float4* __restrict__ TV,
          double2* __restrict__ TDxy, double* __restrict__ TDz,
          unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= nf) return;
  float4 r = P[i], v = V[i];
  const float4 a = ACC[i];
  const int ph = __float_as_int(v.w);
  if (p.flags & SPH_FLAG_REINIT) {
    const float rho0 = p.rho0[ph];
    const float ds = rho0 * SIG[i];  // rho0 sigma/sigma0 - rho0; SIG holds sigma/sigma0 - 1
    float d = ds;
    // Eq. 2.17 for rho* > rho_s: rho - rho0 = rho_s (rho* - rho0) / rho*  (same value as
    // rho_s + (rho* - rho_s) rho0 / rho*, without the cancellation of two O(rho0) terms)
    if (((p.fs_mask >> ph) & 1u) && r.w > ds) d = r.w * ((rho0 + ds) / (rho0 + r.w));
    r.w = d;
  }
  const float hdt = 0.5f * S->dt;
  v.x = fmaf(hdt, a.x, v.x); v.y = fmaf(hdt, a.y, v.y); v.z = fmaf(hdt, a.z, v.z);
  // Eq. 2.20 on the float64 master position: r.xyz is its float32 rounding, which is
  // what the cell hash and the neighbour test see (integer contract, reading A24).
  double2 xy = Dxy[i];
  double zd = Dz[i];
  const double dtd = S->dt_d;
  xy.x = fma(dtd, (double)v.x, xy.x); xy.y = fma(dtd, (double)v.y, xy.y); zd = fma(dtd, (double)v.z, zd);
  r.x = (float)xy.x; r.y = (float)xy.y; r.z = (float)zd;
  TP[i] = r;
  TV[i] = v;
  TDxy[i] = xy;
  TDz[i] = zd;
  const bool fin = isfinite(r.x) && isfinite(r.y) && isfinite(r.z);
  if (!fin) atomicAdd(&S->nonfinite, 1ull);
  bool out = r.x < p.dmin[0] || r.x >= p.dmax[0] || r.y < p.dmin[1] || r.y >= p.dmax[1];
  if (p.dim == 3) out = out || r.z < p.dmin[2] || r.z >= p.dmax[2];
  if (out || !fin) atomicAdd(&S->escaped, 1ull);
  const int cx = cell_coord(r.x, p.ox, p.inv_edge, p.nx), cy = cell_coord(r.y, p.oy, p.inv_edge, p.ny);
  const int cz = p.dim == 3 ? cell_coord(r.z, p.oz, p.inv_edge, p.nz) : 0;
  keys[i] = (unsigned)((cz * p.ny + cy) * p.nx + cx);
  vals[i] = (unsigned)i;
}

// Wall normals, Eq. 2.16, once, in float64 (reading A10).
__global__ void k_normals(DP p, int nw, const float4* __restrict__ WP, const int* __restrict__ lbW,
                          float4* __restrict__ WN) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= nw) return;
  const float4 pw = WP[w];
  const int cx = cell_coord(pw.x, p.ox, p.inv_edge, p.nx), cy = cell_coord(pw.y, p.oy, p.inv_edge, p.ny);
  const int cz = p.dim == 3 ? cell_coord(pw.z, p.oz, p.inv_edge, p.nz) : 0;
  const double h = p.hD, rc2 = 4.0 * h * h;
  const double PI = 3.14159265358979323846264338327950288;
  const double alpha = p.dim == 2 ? 7.0 / (4.0 * PI * h * h) : 21.0 / (16.0 * PI * h * h * h);
  const double V0 = p.dim == 2 ? (double)p.dp * (double)p.dp : (double)p.dp * (double)p.dp * (double)p.dp;
  double px = 0, py = 0, pz = 0;
  for (int dz = (p.dim == 3 ? -1 : 0); dz <= (p.dim == 3 ? 1 : 0); ++dz)
    for (int dy = -1; dy <= 1; ++dy) {
      int y = cy + dy, z = cz + dz;
      if (y < 0 || y >= p.ny || z < 0 || z >= p.nz) continue;
      int rb = (z * p.ny + y) * p.nx;
      int s = lbW[rb + max(cx - 1, 0)], e = lbW[rb + min(cx + 1, p.nx - 1) + 1];
      for (int j = s; j < e; ++j) {
        if (j == w) continue;
        const float4 pj = WP[j];
        double dx = (double)pw.x - (double)pj.x, dyy = (double)pw.y - (double)pj.y,
               dzz = (double)pw.z - (double)pj.z;
        double r2 = dx * dx + dyy * dyy + dzz * dzz;
        if (!(r2 < rc2) || r2 == 0.0) continue;
        double r = sqrt(r2), q = r / h, t = 1.0 - 0.5 * q;
        double dw = -5.0 * alpha / h * q * t * t * t;
        double f = -V0 * dw / r;  // -(m_j/rho_j) grad_i W_ij = f * r_ij
        px += f * dx; py += f * dyy; pz += f * dzz;
      }
    }
  double nrm = sqrt(px * px + py * py + pz * pz);
  float4 n = make_float4(0.f, 0.f, 0.f, 0.f);
  if (nrm * h >= 1e-3) n = make_float4((float)(px / nrm), (float)(py / nrm), (float)(pz / nrm), 0.f);
  WN[w] = n;
}

// ------------------------------------------------------------------------------------------
// Output / diagnostics
// ------------------------------------------------------------------------------------------
__global__ void k_get_fluid(DP p, int nf, const float4* __restrict__ P, const float4* __restrict__ V,
                            const float4* __restrict__ ACC, const unsigned* __restrict__ ID, float* pos,
                            float* vel, float* rho, float* prs, float* acc) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nf) return;
  const float4 r = P[i], v = V[i], a = ACC[i];
  const int ph = __float_as_int(v.w);
  const size_t o = ID[i];
  if (pos) { pos[3 * o] = r.x; pos[3 * o + 1] = r.y; pos[3 * o + 2] = r.z; }
  if (vel) { vel[3 * o] = v.x; vel[3 * o + 1] = v.y; vel[3 * o + 2] = v.z; }
  if (acc) { acc[3 * o] = a.x; acc[3 * o + 1] = a.y; acc[3 * o + 2] = a.z; }
  if (rho) rho[o] = p.rho0[ph] + r.w;
  if (prs) prs[o] = p.c2[ph] * r.w;
}

__global__ void k_get_wall(DP p, int nw, const float4* __restrict__ WP, const float4* __restrict__ WV,
                           const unsigned* __restrict__ ID, float* pos, float* vel, float* rho,
                           float* prs, float* acc) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nw) return;
  const float4 r = WP[i], v = WV[i];
  const size_t o = ID[i];
  if (pos) { pos[3 * o] = r.x; pos[3 * o + 1] = r.y; pos[3 * o + 2] = r.z; }
  if (vel) { vel[3 * o] = v.x; vel[3 * o + 1] = v.y; vel[3 * o + 2] = v.z; }
  if (acc) { acc[3 * o] = 0.f; acc[3 * o + 1] = 0.f; acc[3 * o + 2] = 0.f; }
  if (rho) rho[o] = fmaf(r.w, p.inv_c2[0], p.rho0[0]);
  if (prs) prs[o] = r.w;
}

__global__ void k_scatter_f(int n, const float* __restrict__ src, const unsigned* __restrict__ ID,
                            float* dst, float scale, float shift) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[ID[i]] = scale * (src[i] + shift);
}

__global__ void k_scatter_n(int n, const float4* __restrict__ src, const unsigned* __restrict__ ID,
                            float* dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float4 v = src[i];
  const size_t o = ID[i];
  dst[3 * o] = v.x; dst[3 * o + 1] = v.y; dst[3 * o + 2] = v.z;
}

struct StatAcc {
  double ek;
  unsigned long long count[SPH_MAX_PHASES];  // fluid particles per phase (mass = sum count * m_phase, exact)
  unsigned long long pairs;
  unsigned xfront_bits;  // ordered encoding of float
};

__device__ __forceinline__ unsigned f2ord(float f) {
  unsigned u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

__global__ void __launch_bounds__(256)
k_stats(DP p, int nf, const float4* __restrict__ P, const float4* __restrict__ V, StatAcc* out) {
  double ek = 0;
  unsigned cnt[SPH_MAX_PHASES] = {0, 0, 0, 0};
  float xf = -INFINITY;
  const int up = p.dim - 1;
  const float zlim = p.dmin[up] + 6.0f * p.dp;
  for (int i = blockIdx.x * 256 + threadIdx.x; i < nf; i += gridDim.x * 256) {
    const float4 r = P[i], v = V[i];
    const int ph = __float_as_int(v.w);
    ek += 0.5 * p.massD[ph] * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
#pragma unroll
    for (int k = 0; k < SPH_MAX_PHASES; ++k) cnt[k] += (ph == k);
    const float zz = up == 2 ? r.z : r.y;
    if (ph == 0 && zz < zlim) xf = fmaxf(xf, r.x);
  }
  for (int o = 16; o > 0; o >>= 1) {
    ek += __shfl_xor_sync(FULL, ek, o);
#pragma unroll
    for (int k = 0; k < SPH_MAX_PHASES; ++k) cnt[k] += __shfl_xor_sync(FULL, cnt[k], o);
    xf = fmaxf(xf, __shfl_xor_sync(FULL, xf, o));
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&out->ek, ek);
#pragma unroll
    for (int k = 0; k < SPH_MAX_PHASES; ++k)
      if (cnt[k]) atomicAdd(&out->count[k], (unsigned long long)cnt[k]);
    atomicMax(&out->xfront_bits, f2ord(xf));
  }
}

// Hit counting / listing for sph_get_stats (n_pairs) and sph_debug_neighbours.
// mode 0: count into cnt[caller id] (and total pairs); mode 1: fill ids at off[caller id].
__global__ void __launch_bounds__(PW * 32)
k_neigh(DP p, int n, int is_wall, int mode, const float4* __restrict__ Pself, const unsigned* __restrict__ IDself,
        const float4* __restrict__ P, const unsigned* __restrict__ ID, const int* __restrict__ lbF,
        const float4* __restrict__ WP, const unsigned* __restrict__ WID, const int* __restrict__ lbW,
        int* __restrict__ cnt, const long long* __restrict__ off, int* __restrict__ ids, long long cap,
        unsigned long long* total) {
  __shared__ unsigned qs[PW][64];
  const int i = blockIdx.x * PW + (threadIdx.x >> 5);
  if (i >= n) return;
  const int lane = threadIdx.x & 31;
  unsigned* q = qs[threadIdx.x >> 5];
  const float4 pi = Pself[i];
  const unsigned me = IDself[i];
  const long long base = mode ? off[me] : 0;
  // the body runs with full warps except in the tail; tot is re-broadcast from lane 0 after
  int tot = 0;
  walk(p, P, lbF, pi.x, pi.y, pi.z, is_wall ? -1 : i, q, [&](int j) {
    unsigned act = __activemask();
    int k = __popc(act & ((1u << lane) - 1u));
    if (mode && base + tot + k < cap) ids[base + tot + k] = (int)ID[j];
    tot += __popc(act);
  });
  tot = __shfl_sync(FULL, tot, 0);
  if (!is_wall) {
    walk(p, WP, lbW, pi.x, pi.y, pi.z, -1, q, [&](int j) {
      unsigned act = __activemask();
      int k = __popc(act & ((1u << lane) - 1u));
      if (mode && base + tot + k < cap) ids[base + tot + k] = (int)WID[j];
      tot += __popc(act);
    });
    tot = __shfl_sync(FULL, tot, 0);
  }
  __syncwarp();
  if (lane == 0) {
    if (!mode) {
      if (cnt) cnt[me] = tot;
      if (total) atomicAdd(total, (unsigned long long)tot);
    } else {
      // ascending caller ids within the row (insertion sort; debug path, rows of ~20-100)
      long long m = tot;
      if (base + m > cap) m = cap > base ? cap - base : 0;
      __threadfence_block();
      for (long long a = 1; a < m; ++a) {
        int x = ids[base + a];
        long long b = a - 1;
        while (b >= 0 && ids[base + b] > x) { ids[base + b + 1] = ids[base + b]; --b; }
        ids[base + b + 1] = x;
      }
    }
  }
}

__global__ void k_dbg_cells(DP p, int n, const float4* __restrict__ P, const unsigned* __restrict__ ID,
                            int* cell_id, int* perm, int perm_base) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float4 r = P[i];
  const int cx = cell_coord(r.x, p.ox, p.inv_edge, p.nx), cy = cell_coord(r.y, p.oy, p.inv_edge, p.ny);
  const int cz = p.dim == 3 ? cell_coord(r.z, p.oz, p.inv_edge, p.nz) : 0;
  if (cell_id) cell_id[ID[i]] = (cz * p.ny + cy) * p.nx + cx;
  if (perm) perm[perm_base + i] = (int)ID[i];
}

__global__ void k_dbg_ranges(int ncell, const int* __restrict__ lb, int* cs, int* ce) {
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  int s = lb[c], e = lb[c + 1];
  if (s == e) s = e = 0;
  cs[c] = s;
  ce[c] = e;
}

}  // namespace

// ============================================================================================
// Host side
// ============================================================================================
struct sph_ctx {
  sph_params prm;
  DP dp;
  int device = 0;
  int64_t n = 0, nf = 0, nw = 0, ncell = 0;
  bool multi = false, loaded = false;
  std::string err;
  int64_t launches = 0;
  // fluid
  float4 *P0 = nullptr, *V0 = nullptr, *P1 = nullptr, *V1 = nullptr, *TP = nullptr, *TV = nullptr,
         *ACC = nullptr, *LO = nullptr;
  double2 *Dxy = nullptr, *TDxy = nullptr, *WDxy = nullptr;
  double *Dz = nullptr, *TDz = nullptr, *WDz = nullptr;
  float *SIG = nullptr, *DRHO = nullptr;
  unsigned *ID0 = nullptr, *ID1 = nullptr;
  unsigned *keyA = nullptr, *valA = nullptr, *keyB = nullptr, *valB = nullptr, *hist = nullptr,
           *rowsum = nullptr;
  int *lbF = nullptr, *lbW = nullptr;
  // wall
  float4 *WP = nullptr, *WV = nullptr, *WN = nullptr;
  unsigned* WID = nullptr;
  SS* S = nullptr;
  double* dt_seq = nullptr;
  int64_t dt_seq_cap = 0;
  StatAcc* stat = nullptr;
  int sort_passes = 1;
  // profiling
  bool prof = false;
  std::vector<cudaEvent_t> ev;
  int ev_steps = 0;
  static constexpr int EV_MAX_STEPS = 64, EV_PER_STEP = 14;
};

namespace {

#define CK(call)                                                                         \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess) {                                                             \
      c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                       \
      return e_ == cudaErrorMemoryAllocation ? SPH_ENOMEM : SPH_ECUDA;                   \
    }                                                                                    \
  } while (0)

#define LAUNCH(kern, grid, block, st, ...)                 \
  do {                                                     \
    kern<<<(grid), (block), 0, (st)>>>(__VA_ARGS__);       \
    c->launches++;                                         \
  } while (0)

inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

template <typename T>
int dalloc(sph_ctx* c, T** p, size_t count) {
  if (*p) { cudaFree(*p); *p = nullptr; }
  if (count == 0) count = 1;
  CK(cudaMalloc((void**)p, count * sizeof(T)));
  return SPH_OK;
}

void free_all(sph_ctx* c) {
  void* ptrs[] = {c->P0, c->V0, c->P1, c->V1, c->TP, c->TV, c->ACC, c->SIG, c->DRHO, c->ID0, c->ID1,
                  c->keyA, c->valA, c->keyB, c->valB, c->hist, c->rowsum, c->lbF, c->lbW, c->WP, c->LO, c->Dxy, c->TDxy, c->WDxy, c->Dz, c->TDz, c->WDz,
                  c->WV, c->WN, c->WID, c->S, c->dt_seq, c->stat};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (auto e : c->ev) cudaEventDestroy(e);
}

// Stable radix sort of (keys, vals); result pointers returned in *ko, *vo.
int radix_sort(sph_ctx* c, cudaStream_t st, int n, unsigned* kA, unsigned* vA, unsigned* kB, unsigned* vB,
               unsigned** ko, unsigned** vo) {
  unsigned *ki = kA, *vi = vA, *kt = kB, *vt = vB;
  if (n > 0) {
    int nblk = cdiv(n, RS_TILE);
    for (int pass = 0; pass < c->sort_passes; ++pass) {
      int shift = 8 * pass;
      LAUNCH(k_radix_hist, nblk, RS_THREADS, st, ki, n, shift, c->hist, nblk);
      LAUNCH(k_scan_rowsum, 256, 256, st, c->hist, nblk, c->rowsum);
      LAUNCH(k_scan_apply, 256, 256, st, c->hist, nblk, c->rowsum);
      LAUNCH(k_radix_scatter, nblk, RS_THREADS, st, ki, vi, n, shift, c->hist, nblk, kt, vt);
      std::swap(ki, kt);
      std::swap(vi, vt);
    }
  }
  *ko = ki;
  *vo = vi;
  CK(cudaGetLastError());
  return SPH_OK;
}

struct Prof {
  sph_ctx* c;
  cudaStream_t st;
  int slot = 0;
  bool on;
  Prof(sph_ctx* c_, cudaStream_t s) : c(c_), st(s) {
    on = c->prof && c->ev_steps < sph_ctx::EV_MAX_STEPS;
  }
  void mark() {
    if (!on) return;
    cudaEventRecord(c->ev[c->ev_steps * sph_ctx::EV_PER_STEP + slot++], st);
  }
  void done() {
    if (on) c->ev_steps++;
  }
};

// wall extrapolation launcher
int launch_wall(sph_ctx* c, cudaStream_t st, bool with_vel, const float4* P, const float4* V) {
  if (c->nw == 0 || c->nf == 0) return SPH_OK;
  int grid = cdiv(c->nw, PW);
  if (c->multi) {
    if (with_vel) LAUNCH((k_wall<true, true>), grid, PW * 32, st, c->dp, c->S, (int)c->nw, c->WP, c->WV, P, V, c->LO, c->lbF);
    else LAUNCH((k_wall<true, false>), grid, PW * 32, st, c->dp, c->S, (int)c->nw, c->WP, c->WV, P, V, c->LO, c->lbF);
  } else {
    if (with_vel) LAUNCH((k_wall<false, true>), grid, PW * 32, st, c->dp, c->S, (int)c->nw, c->WP, c->WV, P, V, c->LO, c->lbF);
    else LAUNCH((k_wall<false, false>), grid, PW * 32, st, c->dp, c->S, (int)c->nw, c->WP, c->WV, P, V, c->LO, c->lbF);
  }
  return SPH_OK;
}

// Everything after the drift: sort, reorder, cell ranges, wall pass, pass A, wall pass, pass B.
int pipeline_after_hash(sph_ctx* c, cudaStream_t st, int init, Prof& pf) {
  const int nf = (int)c->nf;
  unsigned *ks, *vs;
  int rc = radix_sort(c, st, nf, c->keyA, c->valA, c->keyB, c->valB, &ks, &vs);
  if (rc) return rc;
  pf.mark();  // end sort
  if (nf > 0) LAUNCH(k_reorder, cdiv(nf, 256), 256, st, nf, vs, c->TP, c->TV, c->TDxy, c->TDz, c->ID0, c->P1, c->V1,
                     c->Dxy, c->Dz, c->LO, c->ID1);
  LAUNCH(k_cell_bounds, cdiv(nf + 1, 256), 256, st, ks, nf, (int)c->ncell, c->lbF);
  pf.mark();  // end reorder
  launch_wall(c, st, true, c->P1, c->V1);
  pf.mark();  // end wall 1
  if (nf > 0) {
    if (c->multi)
      LAUNCH((k_pass_a<true>), cdiv(nf, PW), PW * 32, st, c->dp, c->S, nf, init, c->P1, c->V1, c->Dxy, c->Dz, c->lbF, c->WP,
             c->WV, c->WDxy, c->WDz, c->lbW, c->P0, c->SIG, c->DRHO, c->ID1, c->ID0);
    else
      LAUNCH((k_pass_a<false>), cdiv(nf, PW), PW * 32, st, c->dp, c->S, nf, init, c->P1, c->V1, c->Dxy, c->Dz, c->lbF, c->WP,
             c->WV, c->WDxy, c->WDz, c->lbW, c->P0, c->SIG, c->DRHO, c->ID1, c->ID0);
  }
  pf.mark();  // end pass A
  launch_wall(c, st, false, c->P0, c->V1);
  pf.mark();  // end wall 2
  if (nf > 0) {
    if (c->multi)
      LAUNCH((k_pass_b<true>), cdiv(nf, PW), PW * 32, st, c->dp, c->S, nf, c->P0, c->V1, c->LO, c->lbF, c->WP, c->WN,
             c->lbW, c->V0, c->ACC);
    else
      LAUNCH((k_pass_b<false>), cdiv(nf, PW), PW * 32, st, c->dp, c->S, nf, c->P0, c->V1, c->LO, c->lbF, c->WP, c->WN,
             c->lbW, c->V0, c->ACC);
  }
  pf.mark();  // end pass B
  CK(cudaGetLastError());
  return SPH_OK;
}

int do_steps(sph_ctx* c, int32_t n_steps, const double* dt_host, cudaStream_t st) {
  if (!c->loaded) { c->err = "sph_step before sph_set_particles"; return SPH_EINVAL; }
  if (n_steps < 0) { c->err = "n_steps < 0"; return SPH_EINVAL; }
  if (dt_host && n_steps > 0) {
    if (c->dt_seq_cap < n_steps) {
      int rc = dalloc(c, &c->dt_seq, (size_t)n_steps);
      if (rc) return rc;
      c->dt_seq_cap = n_steps;
    }
    CK(cudaMemcpyAsync(c->dt_seq, dt_host, sizeof(double) * n_steps, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));  // dt_host may be pageable; keep ownership rules simple
  }
  const int nf = (int)c->nf;
  const int dt_grid = std::max(1, std::min(cdiv(nf, 256), 148 * 4));
  for (int s = 0; s < n_steps; ++s) {
    Prof pf(c, st);
    pf.mark();  // start
    LAUNCH(k_dt, dt_grid, 256, st, c->dp, c->S, nf, c->V0, dt_host ? c->dt_seq : nullptr, s);
    if (nf > 0)
      LAUNCH(k_predict, cdiv(nf, 256), 256, st, c->dp, c->S, nf, c->P0, c->V0, c->ACC, c->SIG, c->Dxy, c->Dz, c->TP, c->TV, c->TDxy, c->TDz,
             c->keyA, c->valA);
    pf.mark();  // end predict
    int rc = pipeline_after_hash(c, st, 0, pf);
    if (rc) return rc;
    pf.done();
  }
  return SPH_OK;
}

}  // namespace

extern "C" {

int sph_create(const sph_params* prm, sph_ctx** out) {
  if (!prm || !out) return SPH_EINVAL;
  *out = nullptr;
  if ((prm->dim != 2 && prm->dim != 3) || prm->n_phases < 1 || prm->n_phases > SPH_MAX_PHASES ||
      !(prm->dp > 0) || !(prm->h > 0) || !(prm->cfl > 0))
    return SPH_EINVAL;
  for (int k = 0; k < prm->n_phases; ++k)
    if (!(prm->rho0[k] > 0) || !(prm->c0[k] > 0)) return SPH_EINVAL;
  for (int k = 0; k < prm->dim; ++k)
    if (!(prm->domain_max[k] > prm->domain_min[k])) return SPH_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return SPH_ECUDA;
  sph_ctx* c = new sph_ctx();
  c->prm = *prm;
  cudaGetDevice(&c->device);
  DP& d = c->dp;
  memset(&d, 0, sizeof(d));
  const double PI = 3.14159265358979323846264338327950288;
  const double h = prm->h, dp = prm->dp;
  d.dim = prm->dim; d.n_phases = prm->n_phases;
  d.h = (float)h; d.hinv = (float)(1.0 / h); d.dp = (float)dp; d.rc2 = (float)(4.0 * h * h);
  const double alpha = prm->dim == 2 ? 7.0 / (4.0 * PI * h * h) : 21.0 / (16.0 * PI * h * h * h);
  d.alpha = (float)alpha; d.gradc = (float)(-5.0 * alpha / (h * h)); d.w0 = (float)alpha;
  const double V0 = prm->dim == 2 ? dp * dp : dp * dp * dp;
  d.V0 = (float)V0;
  double cmax = 0;
  for (int k = 0; k < SPH_MAX_PHASES; ++k) {
    bool live = k < prm->n_phases;
    double r0 = live ? prm->rho0[k] : 1.0, c0 = live ? prm->c0[k] : 1.0;
    d.rho0[k] = (float)r0; d.c0[k] = (float)c0; d.c2[k] = (float)(c0 * c0);
    d.inv_c2[k] = (float)(1.0 / (c0 * c0)); d.mass[k] = (float)(r0 * V0); d.massD[k] = live ? r0 * V0 : 0.0;
    if (live) cmax = std::max(cmax, c0);
  }
  // sigma0: full undisturbed lattice incl. self term (readings A12, A14)
  {
    int m = (int)ceil(2.0 * h / dp) + 1;
    double s = 0;
    for (int k = (prm->dim == 3 ? -m : 0); k <= (prm->dim == 3 ? m : 0); ++k)
      for (int j = -m; j <= m; ++j)
        for (int i = -m; i <= m; ++i) {
          double q = dp * sqrt((double)(i * i + j * j + k * k)) / h;
          if (q < 2.0) {
            double t = 1.0 - 0.5 * q;
            s += alpha * t * t * t * t * (1.0 + 2.0 * q);
          }
        }
    d.sigma0 = (float)s; d.inv_sigma0 = (float)(1.0 / s);
    d.sigma0D = s; d.a_over_s0 = alpha / s; d.hinvD = 1.0 / h;
  }
  d.gamma_p = (float)prm->penalty_strength; d.two_over_dp = (float)(2.0 / dp);
  d.pen_mask = prm->penalty_phase_mask; d.fs_mask = prm->free_surface_mask; d.flags = prm->flags;
  const double edge = 2.0 * h * (1.0 + 1.0 / 1024.0);  // reading A24
  d.inv_edge = (float)(1.0 / edge);
  d.ox = (float)prm->domain_min[0]; d.oy = (float)prm->domain_min[1]; d.oz = (float)prm->domain_min[2];
  int nc[3] = {1, 1, 1};
  for (int k = 0; k < prm->dim; ++k)
    nc[k] = std::max(1, (int)ceil((prm->domain_max[k] - prm->domain_min[k]) / edge));
  d.nx = nc[0]; d.ny = nc[1]; d.nz = nc[2];
  for (int k = 0; k < 3; ++k) {
    d.dmin[k] = (float)prm->domain_min[k]; d.dmax[k] = (float)prm->domain_max[k];
    d.g[k] = prm->g[k]; d.gamp[k] = prm->g_osc_amp[k];
  }
  d.gperiod = prm->g_osc_period; d.cmax = cmax; d.cfl = prm->cfl; d.hD = h;
  c->ncell = (int64_t)nc[0] * nc[1] * nc[2];
  if (c->ncell >= (1ll << 31) - 2) { delete c; return SPH_EINVAL; }
  int bits = 1;
  while ((1ll << bits) < c->ncell) ++bits;
  c->sort_passes = (bits + 7) / 8;
  c->multi = prm->n_phases > 1;
  *out = c;
  return SPH_OK;
}

void sph_destroy(sph_ctx* c) {
  if (!c) return;
  free_all(c);
  delete c;
}

const char* sph_last_error(const sph_ctx* c) { return c ? c->err.c_str() : "null context"; }
int64_t sph_launch_count(const sph_ctx* c) { return c ? c->launches : 0; }
int64_t sph_num_cells(const sph_ctx* c) { return c ? c->ncell : 0; }

int sph_set_particles(sph_ctx* c, int64_t n, const float* pos, const float* vel, const float* rho,
                      const int32_t* tag, void* stream) {
  if (!c) return SPH_EINVAL;
  if (n < 0 || n >= (1ll << 31) - 64 || (n > 0 && (!pos || !vel || !rho || !tag))) {
    c->err = "bad arguments to sph_set_particles";
    return SPH_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)stream;
  c->loaded = false;
  // classify on the host (one-off): caller indices of fluid and wall particles, order kept
  std::vector<int32_t> htag((size_t)n);
  if (n) CK(cudaMemcpyAsync(htag.data(), tag, sizeof(int32_t) * n, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  std::vector<int32_t> fid, wid;
  fid.reserve(n); wid.reserve(n / 4 + 1);
  for (int64_t i = 0; i < n; ++i) {
    if (htag[i] == SPH_TAG_WALL) wid.push_back((int32_t)i);
    else if (htag[i] >= 0 && htag[i] < c->prm.n_phases) fid.push_back((int32_t)i);
    else { c->err = "tag out of range"; return SPH_EINVAL; }
  }
  c->n = n; c->nf = (int64_t)fid.size(); c->nw = (int64_t)wid.size();
  const int nf = (int)c->nf, nw = (int)c->nw;
  const size_t cap = (size_t)std::max(nf, nw);
  int rc = 0;
  rc |= dalloc(c, &c->P0, nf); rc |= dalloc(c, &c->V0, nf); rc |= dalloc(c, &c->P1, nf);
  rc |= dalloc(c, &c->V1, nf); rc |= dalloc(c, &c->TP, cap); rc |= dalloc(c, &c->TV, nf);
  rc |= dalloc(c, &c->LO, nf); rc |= dalloc(c, &c->Dxy, nf); rc |= dalloc(c, &c->TDxy, nf);
  rc |= dalloc(c, &c->Dz, nf); rc |= dalloc(c, &c->TDz, nf); rc |= dalloc(c, &c->WDxy, nw); rc |= dalloc(c, &c->WDz, nw);
  rc |= dalloc(c, &c->ACC, nf); rc |= dalloc(c, &c->SIG, nf); rc |= dalloc(c, &c->DRHO, nf);
  rc |= dalloc(c, &c->ID0, cap); rc |= dalloc(c, &c->ID1, nf);
  rc |= dalloc(c, &c->keyA, cap); rc |= dalloc(c, &c->valA, cap); rc |= dalloc(c, &c->keyB, cap);
  rc |= dalloc(c, &c->valB, cap);
  rc |= dalloc(c, &c->hist, (size_t)256 * cdiv(std::max<size_t>(cap, 1), RS_TILE));
  rc |= dalloc(c, &c->rowsum, 256);
  rc |= dalloc(c, &c->lbF, c->ncell + 1); rc |= dalloc(c, &c->lbW, c->ncell + 1);
  rc |= dalloc(c, &c->WP, nw); rc |= dalloc(c, &c->WV, nw); rc |= dalloc(c, &c->WN, nw);
  rc |= dalloc(c, &c->WID, nw);
  rc |= dalloc(c, &c->S, 1); rc |= dalloc(c, &c->stat, 1);
  if (rc) return c->err.find("out of memory") != std::string::npos ? SPH_ENOMEM : SPH_ECUDA;
  CK(cudaMemsetAsync(c->S, 0, sizeof(SS), st));
  CK(cudaMemsetAsync(c->ACC, 0, sizeof(float4) * std::max(nf, 1), st));
  CK(cudaMemsetAsync(c->WV, 0, sizeof(float4) * std::max(nw, 1), st));
  {  // gravity at t = 0 (sin(0) = 0)
    float g0[3] = {(float)c->prm.g[0], (float)c->prm.g[1], (float)c->prm.g[2]};
    CK(cudaMemcpyAsync((char*)c->S + offsetof(SS, g), g0, sizeof(g0), cudaMemcpyHostToDevice, st));
  }
  int* idx = nullptr;
  CK(cudaMalloc((void**)&idx, sizeof(int) * std::max<size_t>(cap, 1)));
  // ---- wall structure, built once ----
  if (nw > 0) {
    CK(cudaMemcpyAsync(idx, wid.data(), sizeof(int) * nw, cudaMemcpyHostToDevice, st));
    LAUNCH(k_load_wall, cdiv(nw, 256), 256, st, c->dp, nw, idx, pos, c->TP, c->ID0, c->keyA, c->valA);
    unsigned *ks, *vs;
    rc = radix_sort(c, st, nw, c->keyA, c->valA, c->keyB, c->valB, &ks, &vs);
    if (rc) { cudaFree(idx); return rc; }
    LAUNCH(k_reorder, cdiv(nw, 256), 256, st, nw, vs, c->TP, (const float4*)nullptr, (const double2*)nullptr,
           (const double*)nullptr, c->ID0, c->WP, (float4*)nullptr, (double2*)nullptr, (double*)nullptr,
           (float4*)nullptr, c->WID);
    LAUNCH(k_wall_double, cdiv(nw, 256), 256, st, nw, c->WP, c->WDxy, c->WDz);
    LAUNCH(k_cell_bounds, cdiv(nw + 1, 256), 256, st, ks, nw, (int)c->ncell, c->lbW);
    LAUNCH(k_normals, cdiv(nw, 128), 128, st, c->dp, nw, c->WP, c->lbW, c->WN);
  } else {
    LAUNCH(k_cell_bounds, 1, 256, st, c->keyA, 0, (int)c->ncell, c->lbW);
  }
  CK(cudaStreamSynchronize(st));  // wid host buffer / idx reuse
  // ---- fluid: load, then the common pipeline in init mode (dt = 0: sigma_i, p_w, (dv/dt)^0) ----
  if (nf > 0) {
    CK(cudaMemcpyAsync(idx, fid.data(), sizeof(int) * nf, cudaMemcpyHostToDevice, st));
    LAUNCH(k_load_fluid, cdiv(nf, 256), 256, st, c->dp, nf, idx, pos, vel, rho, tag, c->TP, c->TV, c->TDxy, c->TDz, c->ID0,
           c->keyA, c->valA);
  }
  Prof pf(c, st);
  pf.on = false;
  rc = pipeline_after_hash(c, st, 1, pf);
  cudaError_t e = cudaStreamSynchronize(st);
  cudaFree(idx);
  if (rc) return rc;
  if (e != cudaSuccess) { c->err = cudaGetErrorString(e); return SPH_ECUDA; }
  c->loaded = true;
  c->ev_steps = 0;
  return SPH_OK;
}

int sph_set_particles_host(sph_ctx* c, int64_t n, const float* pos, const float* vel, const float* rho,
                           const int32_t* tag, void* stream) {
  if (!c) return SPH_EINVAL;
  if (n < 0 || (n > 0 && (!pos || !vel || !rho || !tag))) { c->err = "bad arguments"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  float *dpos = nullptr, *dvel = nullptr, *drho = nullptr;
  int32_t* dtag = nullptr;
  size_t m = (size_t)std::max<int64_t>(n, 1);
  CK(cudaMalloc((void**)&dpos, m * 12)); CK(cudaMalloc((void**)&dvel, m * 12));
  CK(cudaMalloc((void**)&drho, m * 4)); CK(cudaMalloc((void**)&dtag, m * 4));
  int rc = SPH_OK;
  cudaError_t e = cudaSuccess;
  if (n) {
    e = cudaMemcpyAsync(dpos, pos, n * 12, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dvel, vel, n * 12, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(drho, rho, n * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dtag, tag, n * 4, cudaMemcpyHostToDevice, st);
  }
  if (e != cudaSuccess) { c->err = cudaGetErrorString(e); rc = SPH_ECUDA; }
  if (rc == SPH_OK) rc = sph_set_particles(c, n, dpos, dvel, drho, dtag, stream);
  cudaStreamSynchronize(st);
  cudaFree(dpos); cudaFree(dvel); cudaFree(drho); cudaFree(dtag);
  return rc;
}

int sph_step(sph_ctx* c, int32_t n_steps, void* stream) {
  if (!c) return SPH_EINVAL;
  return do_steps(c, n_steps, nullptr, (cudaStream_t)stream);
}

int sph_step_dt(sph_ctx* c, int32_t n_steps, const double* dt_host, void* stream) {
  if (!c) return SPH_EINVAL;
  if (!dt_host && n_steps > 0) { c->err = "dt_host is NULL"; return SPH_EINVAL; }
  return do_steps(c, n_steps, dt_host, (cudaStream_t)stream);
}

int sph_get_fields(sph_ctx* c, float* pos, float* vel, float* rho, float* p, float* acc, void* stream) {
  if (!c) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  if (c->nf) LAUNCH(k_get_fluid, cdiv(c->nf, 256), 256, st, c->dp, (int)c->nf, c->P0, c->V0, c->ACC, c->ID0, pos, vel, rho, p, acc);
  if (c->nw) LAUNCH(k_get_wall, cdiv(c->nw, 256), 256, st, c->dp, (int)c->nw, c->WP, c->WV, c->WID, pos, vel, rho, p, acc);
  CK(cudaGetLastError());
  return SPH_OK;
}

int sph_get_fields_host(sph_ctx* c, float* pos, float* vel, float* rho, float* p, float* acc, void* stream) {
  if (!c) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)std::max<int64_t>(c->n, 1);
  float* buf = nullptr;
  CK(cudaMalloc((void**)&buf, n * 11 * sizeof(float)));
  float *dpos = buf, *dvel = buf + 3 * n, *dacc = buf + 6 * n, *drho = buf + 9 * n, *dp = buf + 10 * n;
  int rc = sph_get_fields(c, pos ? dpos : nullptr, vel ? dvel : nullptr, rho ? drho : nullptr,
                          p ? dp : nullptr, acc ? dacc : nullptr, stream);
  cudaError_t e = cudaSuccess;
  if (rc == SPH_OK && c->n) {
    if (pos) e = cudaMemcpyAsync(pos, dpos, c->n * 12, cudaMemcpyDeviceToHost, st);
    if (vel && e == cudaSuccess) e = cudaMemcpyAsync(vel, dvel, c->n * 12, cudaMemcpyDeviceToHost, st);
    if (acc && e == cudaSuccess) e = cudaMemcpyAsync(acc, dacc, c->n * 12, cudaMemcpyDeviceToHost, st);
    if (rho && e == cudaSuccess) e = cudaMemcpyAsync(rho, drho, c->n * 4, cudaMemcpyDeviceToHost, st);
    if (p && e == cudaSuccess) e = cudaMemcpyAsync(p, dp, c->n * 4, cudaMemcpyDeviceToHost, st);
  }
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(buf);
  if (rc) return rc;
  if (e != cudaSuccess || e2 != cudaSuccess) {
    c->err = cudaGetErrorString(e != cudaSuccess ? e : e2);
    return SPH_ECUDA;
  }
  return SPH_OK;
}

int sph_get_stats(sph_ctx* c, sph_stats* out, void* stream) {
  if (!c || !out) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  StatAcc z;
  memset(&z, 0, sizeof(z));
  CK(cudaMemcpyAsync(c->stat, &z, sizeof(z), cudaMemcpyHostToDevice, st));
  const int nf = (int)c->nf;
  if (nf) {
    LAUNCH(k_stats, std::min(cdiv(nf, 256), 1184), 256, st, c->dp, nf, c->P0, c->V0, c->stat);
    LAUNCH(k_neigh, cdiv(nf, PW), PW * 32, st, c->dp, nf, 0, 0, c->P0, c->ID0, c->P0, c->ID0, c->lbF, c->WP,
           c->WID, c->lbW, (int*)nullptr, (const long long*)nullptr, (int*)nullptr, 0ll, &c->stat->pairs);
  }
  SS hs;
  CK(cudaMemcpyAsync(&z, c->stat, sizeof(z), cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(&hs, c->S, sizeof(hs), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  out->t = hs.t; out->dt = hs.dt_d; out->steps = hs.steps; out->n_fluid = c->nf; out->n_wall = c->nw;
  out->n_pairs = (int64_t)z.pairs; out->e_kin = z.ek;
  out->mass = 0.0;
  for (int k = 0; k < SPH_MAX_PHASES; ++k) out->mass += (double)z.count[k] * c->dp.massD[k];
  {
    unsigned u = z.xfront_bits;
    float f;
    u = (u & 0x80000000u) ? (u & 0x7fffffffu) : ~u;
    memcpy(&f, &u, 4);
    out->x_front = z.xfront_bits == 0 ? -INFINITY : (double)f;
  }
  out->escaped = (int64_t)hs.escaped; out->nonfinite = (int64_t)hs.nonfinite;
  if (hs.nonfinite) { c->err = "non-finite particle state"; return SPH_ENONFINITE; }
  if (hs.dt_underflow) { c->err = "time step underflow"; return SPH_EDTUNDERFLOW; }
  return SPH_OK;
}

int sph_set_profiling(sph_ctx* c, int32_t on) {
  if (!c) return SPH_EINVAL;
  if (on && c->ev.empty()) {
    c->ev.resize((size_t)sph_ctx::EV_MAX_STEPS * sph_ctx::EV_PER_STEP);
    for (auto& e : c->ev) CK(cudaEventCreate(&e));
  }
  c->prof = on != 0;
  c->ev_steps = 0;
  return SPH_OK;
}

int sph_get_timings(sph_ctx* c, float* ms, int32_t* n_steps) {
  if (!c || !ms || !n_steps) return SPH_EINVAL;
  for (int k = 0; k < SPH_STAGE_COUNT; ++k) ms[k] = 0.f;
  *n_steps = c->ev_steps;
  if (c->ev_steps == 0) return SPH_OK;
  CK(cudaEventSynchronize(c->ev[(c->ev_steps - 1) * sph_ctx::EV_PER_STEP + 7]));
  // marks per step: 0 start, 1 predict, 2 sort, 3 reorder, 4 wall1, 5 passA, 6 wall2, 7 passB
  static const int stage_of[7] = {SPH_STAGE_PREDICT, SPH_STAGE_SORT, SPH_STAGE_REORDER, SPH_STAGE_WALL,
                                  SPH_STAGE_PASS_A, SPH_STAGE_WALL, SPH_STAGE_PASS_B};
  for (int s = 0; s < c->ev_steps; ++s)
    for (int k = 0; k < 7; ++k) {
      float t = 0.f;
      CK(cudaEventElapsedTime(&t, c->ev[s * sph_ctx::EV_PER_STEP + k], c->ev[s * sph_ctx::EV_PER_STEP + k + 1]));
      ms[stage_of[k]] += t;
    }
  c->ev_steps = 0;
  return SPH_OK;
}

int sph_debug_cells(sph_ctx* c, int32_t* cell_id, int32_t* perm, int32_t* cs, int32_t* ce, void* stream) {
  if (!c) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)std::max<int64_t>(c->n, 1), nc = (size_t)c->ncell;
  int *dcid = nullptr, *dperm = nullptr, *dcs = nullptr, *dce = nullptr;
  CK(cudaMalloc((void**)&dcid, n * 4)); CK(cudaMalloc((void**)&dperm, n * 4));
  CK(cudaMalloc((void**)&dcs, 2 * nc * 4)); CK(cudaMalloc((void**)&dce, 2 * nc * 4));
  if (c->nf) LAUNCH(k_dbg_cells, cdiv(c->nf, 256), 256, st, c->dp, (int)c->nf, c->P0, c->ID0, dcid, dperm, 0);
  if (c->nw) LAUNCH(k_dbg_cells, cdiv(c->nw, 256), 256, st, c->dp, (int)c->nw, c->WP, c->WID, dcid, dperm, (int)c->nf);
  LAUNCH(k_dbg_ranges, cdiv(nc, 256), 256, st, (int)nc, c->lbF, dcs, dce);
  LAUNCH(k_dbg_ranges, cdiv(nc, 256), 256, st, (int)nc, c->lbW, dcs + nc, dce + nc);
  cudaError_t e = cudaSuccess;
  if (cell_id && c->n) e = cudaMemcpyAsync(cell_id, dcid, c->n * 4, cudaMemcpyDeviceToHost, st);
  if (perm && c->n && e == cudaSuccess) e = cudaMemcpyAsync(perm, dperm, c->n * 4, cudaMemcpyDeviceToHost, st);
  if (cs && e == cudaSuccess) e = cudaMemcpyAsync(cs, dcs, 2 * nc * 4, cudaMemcpyDeviceToHost, st);
  if (ce && e == cudaSuccess) e = cudaMemcpyAsync(ce, dce, 2 * nc * 4, cudaMemcpyDeviceToHost, st);
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(dcid); cudaFree(dperm); cudaFree(dcs); cudaFree(dce);
  if (e != cudaSuccess || e2 != cudaSuccess) {
    c->err = cudaGetErrorString(e != cudaSuccess ? e : e2);
    return SPH_ECUDA;
  }
  return SPH_OK;
}

int sph_debug_neighbours(sph_ctx* c, int64_t* offsets, int32_t* ids, int64_t cap, int64_t* total, void* stream) {
  if (!c || !offsets || !total) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = c->n;
  int* dcnt = nullptr;
  CK(cudaMalloc((void**)&dcnt, std::max<int64_t>(n, 1) * 4));
  CK(cudaMemsetAsync(dcnt, 0, std::max<int64_t>(n, 1) * 4, st));
  auto run = [&](int mode, const long long* doff, int* dids, long long dcap) {
    if (c->nf)
      LAUNCH(k_neigh, cdiv(c->nf, PW), PW * 32, st, c->dp, (int)c->nf, 0, mode, c->P0, c->ID0, c->P0, c->ID0, c->lbF,
             c->WP, c->WID, c->lbW, dcnt, doff, dids, dcap, (unsigned long long*)nullptr);
    if (c->nw && c->nf)
      LAUNCH(k_neigh, cdiv(c->nw, PW), PW * 32, st, c->dp, (int)c->nw, 1, mode, c->WP, c->WID, c->P0, c->ID0, c->lbF,
             c->WP, c->WID, c->lbW, dcnt, doff, dids, dcap, (unsigned long long*)nullptr);
  };
  run(0, nullptr, nullptr, 0);
  std::vector<int> hc((size_t)n);
  if (n) CK(cudaMemcpyAsync(hc.data(), dcnt, n * 4, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  offsets[0] = 0;
  for (int64_t i = 0; i < n; ++i) offsets[i + 1] = offsets[i] + hc[i];
  *total = offsets[n];
  int rc = SPH_OK;
  if (ids && cap > 0 && n > 0) {
    long long* doff = nullptr;
    int* dids = nullptr;
    CK(cudaMalloc((void**)&doff, (n + 1) * 8));
    CK(cudaMalloc((void**)&dids, std::max<int64_t>(cap, 1) * 4));
    CK(cudaMemcpyAsync(doff, offsets, (n + 1) * 8, cudaMemcpyHostToDevice, st));
    run(1, doff, dids, cap);
    int64_t m = std::min<int64_t>(cap, *total);
    cudaError_t e = cudaMemcpyAsync(ids, dids, m * 4, cudaMemcpyDeviceToHost, st);
    cudaError_t e2 = cudaStreamSynchronize(st);
    cudaFree(doff); cudaFree(dids);
    if (e != cudaSuccess || e2 != cudaSuccess) {
      c->err = cudaGetErrorString(e != cudaSuccess ? e : e2);
      rc = SPH_ECUDA;
    }
  }
  cudaFree(dcnt);
  return rc;
}

int sph_debug_normals(sph_ctx* c, float* normals, void* stream) {
  if (!c || !normals) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  float* d = nullptr;
  const size_t n = (size_t)std::max<int64_t>(c->n, 1);
  CK(cudaMalloc((void**)&d, n * 12));
  CK(cudaMemsetAsync(d, 0, n * 12, st));
  if (c->nw) LAUNCH(k_scatter_n, cdiv(c->nw, 256), 256, st, (int)c->nw, c->WN, c->WID, d);
  cudaError_t e = cudaMemcpyAsync(normals, d, c->n * 12, cudaMemcpyDeviceToHost, st);
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(d);
  if (e != cudaSuccess || e2 != cudaSuccess) { c->err = cudaGetErrorString(e != cudaSuccess ? e : e2); return SPH_ECUDA; }
  return SPH_OK;
}

int sph_debug_sigma(sph_ctx* c, float* sigma, void* stream) {
  if (!c || !sigma) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  float* d = nullptr;
  const size_t n = (size_t)std::max<int64_t>(c->n, 1);
  CK(cudaMalloc((void**)&d, n * 8));
  CK(cudaMemsetAsync(d, 0, n * 8, st));
  if (c->nf) {
    LAUNCH(k_scatter_f, cdiv(c->nf, 256), 256, st, (int)c->nf, c->SIG, c->ID0, d, c->dp.sigma0, 1.0f);
    LAUNCH(k_scatter_f, cdiv(c->nf, 256), 256, st, (int)c->nf, c->DRHO, c->ID0, d + n, 1.0f, 0.0f);
  }
  cudaError_t e = cudaMemcpyAsync(sigma, d, c->n * 4, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(sigma + c->n, d + n, c->n * 4, cudaMemcpyDeviceToHost, st);
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(d);
  if (e != cudaSuccess || e2 != cudaSuccess) { c->err = cudaGetErrorString(e != cudaSuccess ? e : e2); return SPH_ECUDA; }
  return SPH_OK;
}

}  // extern "C"
