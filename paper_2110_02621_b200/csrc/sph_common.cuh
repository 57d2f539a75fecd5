// sph_common.cuh — parameter blocks and device helpers shared by the kernels of libsph.
// Included by sph.cu only.  Citations: PAPER.md:<line>; readings Axx: DESIGN.md §3.
//
// Data layout.  Fluid and wall particles live in separate cell-sorted arrays:
//   (X4 and B4 are interleaved in one 32-byte record XB per particle)
//   X4  uint4   fixed-point master position: the middle 32 bits of each 42-bit coordinate (units of Qp = Q / 2^mbits,
//               modulo 2^32; Q = 2^-k m), .w = the 10 bits above and below them per axis (3 x 10 bits) << 2 | phase
//   A4  float4  float32 image centred on the domain centre (xc, yc, zc, |xc|^2): candidate test only
//   B4  float4  (vx, vy, vz, rho - rho0_phase); walls: (v_w, p_w)
// Pair geometry is an exact wrapping integer subtraction of X4 followed by int->float, in units of Qp.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "sph.h"

struct DP {
  int dim, n_phases;
  float rc2;       // (2h)^2, contract neighbour test on float32 images (reading A24)
  float rc2m;      // candidate filter threshold on the centred images: rc2 + rounding margin
  int exact_filter;  // 1: margin too large for the expanded form, use the difference form
  int subq;          // 1: sigma from separations that include the 10-bit residuals (k_pass_a<.., SUBQ>)
  float inv_h;       // float16 filter of k_build: coordinates in units of h
  unsigned thr_h2;   // its threshold on r^2 / h^2 (half2, both halves): 4.08 + the float32 image margin
  int mbits, lobits;  // pair unit Qp = Q / 2^mbits; lobits = 10 - mbits bits of a coordinate lie below the record's word
  float sub_scale, sub_half_inv;  // 2^lobits and 0.5 / 2^lobits (float64 sigma term with the low bits, w64)
  float qh;        // Qp / h: q = r_Qp * qh
  float Qf;        // Qp
  float gradcQ;    // W'(r)/r * r_ij = gradcQ * (1 - q/2)^3 * d_Qp,   gradc = -5 alpha / h^2
  float alpha, V0;
  float rho0[SPH_MAX_PHASES], c0[SPH_MAX_PHASES], c2[SPH_MAX_PHASES], inv_c2[SPH_MAX_PHASES],
      mass[SPH_MAX_PHASES];
  float gamma_p, two_over_dp;  // two_over_dp holds 2 Qp / dp (delta of Eq. 2.15 from Qp units)
  unsigned pen_mask, fs_mask, flags;
  float ox, oy, oz, inv_edge;  // contract cell hash (reading A24)
  int nx, ny, nz;
  float dmin[3], dmax[3];
  double O[3], C[3], Q, sub_per_m;  // fixed point: origin, image centre, quantum, 1024 / Q
  double Qs, Qp;                    // Q / 1024 (unit of the 42-bit coordinate), Q / 2^mbits (unit of the pair geometry)
  double cmax, cfl, hD, dpD, qhD;  // qhD = Qp / h
  double mhqD[2], tqD[2];          // -q/2 and 2q per unit of r: [0] r in Qp, [1] r in Q/1024 (w64)
  double massD[SPH_MAX_PHASES];
  double a_over_s0;
  double g[3], gamp[3], gperiod;
  double wamp[3], womega;  // NEXT-1: wall motion x_w(t) = x_w(0) + wamp sin(womega t); womega = 0: static walls
  // Verlet skin: the lists are built with radius 2h(1 + skin) on a cell grid of that edge
  // and kept while 2 * (fluid displacement bound) and (fluid + wall displacement) stay below skin_budget
  int reach;           // cells per axis a neighbour walk reaches on each side: 1 (cell edge = list radius, 27 / 9 cells) or
                       // 2 (cell edge = half of it, 125 / 25 cells: NEXT-4 measurement)
  int sub_bits;        // sort key = (cell id << sub_bits) | Morton code of the position inside the cell (sub_bits / dim bits
                       // per axis; 0 when skin = 0, where the order inside a cell is the contract's id order, reading A25)
  double skin;         // largest skin s_max >= 0 (the cell edge is 2h(1 + s_max)); 0: the lists are rebuilt every step
  double skin_min;     // smallest skin the adaptive choice takes
  double marg32;       // rounding margin of the float32 filter forms on r^2 (m^2): threshold = rl^2 + marg32
  double marg16;       // float32-image part of the float16 filter's margin on r^2 / h^2: threshold = 4.08 (rl / 2h)^2 + marg16
};

// Per-particle record gathered by the pair bodies: one 32-byte sector, one 256-bit load.
struct __align__(32) XB {
  uint4 x;   // fixed-point master position (+ residual / phase, or the wall's own index)
  float4 b;  // (vx, vy, vz, rho - rho0_phase); walls: (v_w, p_w)
};
__device__ __forceinline__ XB ldg256(const XB* p) {  // LDG.E.256 (sm_100+): the whole record in one request
  XB r;
  asm("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
      : "=r"(r.x.x), "=r"(r.x.y), "=r"(r.x.z), "=r"(r.x.w), "=f"(r.b.x), "=f"(r.b.y), "=f"(r.b.z), "=f"(r.b.w)
      : "l"(p));
  return r;
}

// Device-resident per-step state: written by k_dt, read by every other kernel, so that
// sph_step(n) needs no host synchronisation between steps.
struct SS {
  double t;
  double dt_d;
  float dt;
  float g[3];            // gravity at t^{n+1} (reading A28)
  float gw[3];           // g - a_w at t^{n+1}: the lever term of Eq. 2.12; = g for static walls
  float vwall[3];        // wall velocity at t^{n+1} (mirror of reading A6)
  int sq[3];             // wall displacement since sph_set_particles, in units of Q
  unsigned vmax2_bits;   // max |v|^2 over fluid, float bits (non-negative -> ordered as uint)
  unsigned blocks_done;
  long long steps;
  unsigned long long escaped, nonfinite;
  int dt_underflow;
  int list_overflow;     // largest neighbour count seen above the list capacity (0 = none); sticky
  // Verlet skin: written by k_predict's last block (and by sph_set_particles for the first build).
  // The skin is ADAPTIVE: every build takes the skin that minimises (pass cost + build cost / steps between builds)
  // for the displacement per step seen at that time, s = (-2 b d + sqrt(4 b^2 d^2 + 12 b d)) / 6 with d = max_i |dx_i| / h
  // and b = build cost / pass cost (0.65 measured), within [skin_min, skin]; k_build / k_wall_build read the
  // thresholds of the current skin from here.
  double skin_cur;         // skin of the lists in use
  double budget;           // 2 h skin_cur (1 - 1e-6): the lists hold every pair within 2h while 2 disp (or disp + wall displacement) stays below it
  float rl2m;              // float32 filter threshold of the current skin: (2h(1 + skin_cur))^2 + marg32
  unsigned thr_h2;         // float16 filter threshold (half2, both halves)
  int since;               // steps since the last build
  int sq_prev[3];          // wall displacement of the previous step (units of Q)
  double disp;             // sum over the steps since the last list build of max_i |dx_i| (metres): a bound on
                           // every fluid particle's displacement since then
  int sq_build[3];         // wall displacement (units of Q) at the last list build
  int rebuild;             // 1: this step rebuilds the cell list and the neighbour lists
  unsigned dmax2_bits;     // max_i |dx_i|^2 of this step (float bits)
  unsigned blocks_done2;
  long long rebuilds;      // list builds since sph_set_particles (the set-up's included)
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

// ---- fixed-point master positions ---------------------------------------------------------
// A coordinate is a 42-bit unsigned integer T in units of Q/1024 from the origin O (span 2^32 Q >= 1.5 L + 16 h).
// The record does not hold its top 32 bits but its MIDDLE 32 bits, T >> lobits (lobits = 10 - mbits): positions
// modulo 2^32 quanta of Qp = Q / 2^mbits.  The separation of two particles that are within a stencil of each other
// is then still one exact wrapping 32-bit subtraction (mbits is chosen so that 2.5 list radii stay below 2^30 Qp),
// but in units 2^mbits times finer than Q: on metre-sized domains the pair geometry resolves 10^-11 m instead of
// 10^-9 m at no cost in the pair loops.  The mbits bits above and the lobits bits below the word sit in a 10-bit
// field per axis of the record's fourth word, (top << lobits) | low; only the drift, the cell hash, the output and
// (multi-phase runs) the residual-exact sigma term read them.  Saturates outside the span; NaN -> 0.
__device__ __forceinline__ unsigned long long fx_tot_from_double(double x, double O, double Q) {
  double u = rint((x - O) / Q * 1024.0);
  u = fmin(fmax(u, 0.0), 4398046511103.0);   // 2^42 - 1
  return (unsigned long long)u;
}
__device__ __forceinline__ unsigned long long fx_tot(const DP& p, unsigned mid, unsigned field) {
  const unsigned lomask = (1u << p.lobits) - 1u;
  return ((unsigned long long)(field >> p.lobits) << (32 + p.lobits)) | ((unsigned long long)mid << p.lobits) |
         (unsigned long long)(field & lomask);
}
__device__ __forceinline__ void fx_split(const DP& p, unsigned long long tot, unsigned& mid, unsigned& field) {
  const unsigned lomask = (1u << p.lobits) - 1u;
  mid = (unsigned)(tot >> p.lobits);
  field = ((unsigned)(tot >> (32 + p.lobits)) << p.lobits) | ((unsigned)tot & lomask);
}
__device__ __forceinline__ unsigned fx_field(const uint4& x, int k) { return (x.w >> (22 - 10 * k)) & 1023u; }
__device__ __forceinline__ unsigned fx_word(const uint4& x, int k) { return k == 0 ? x.x : (k == 1 ? x.y : x.z); }
__device__ __forceinline__ unsigned fx_pack(unsigned fx, unsigned fy, unsigned fz, unsigned phase) {
  return (fx << 22) | (fy << 12) | (fz << 2) | phase;
}
// the coordinate in metres: exact (Q a power of two, O a multiple of Q, 42 + few bits)
__device__ __forceinline__ double fx_pos(const DP& p, const uint4& x, int k) {
  return fma((double)fx_tot(p, fx_word(x, k), fx_field(x, k)), p.Qs, p.O[k]);
}
// float32 image of the master position (what sph_get_fields returns and the cell hash sees)
__device__ __forceinline__ float fx_image(const DP& p, const uint4& x, int k) { return (float)fx_pos(p, x, k); }

__device__ __forceinline__ int phase_of(const uint4& x) { return (int)(x.w & 3u); }

__device__ __forceinline__ float4 centred_image(const DP& p, const uint4& x) {
  const float a = (float)(fx_pos(p, x, 0) - p.C[0]);
  const float b = (float)(fx_pos(p, x, 1) - p.C[1]);
  const float c = p.dim == 3 ? (float)(fx_pos(p, x, 2) - p.C[2]) : 0.0f;
  return make_float4(a, b, c, fmaf(c, c, fmaf(b, b, a * a)));
}

// Sort key of the step's cell list: the cell id of reading A24's hash on the step's grid, and below it the Morton code
// of the position inside the cell, so that particles that are neighbours in memory are neighbours in space: the
// lanes of a warp then gather from few cache lines at a time (profiles/r02).
__device__ __forceinline__ unsigned spread_bits(unsigned v, const int dim) {  // v < 8: bit k -> bit k * dim
  return dim == 3 ? ((v & 1u) | ((v & 2u) << 2) | ((v & 4u) << 4)) : ((v & 1u) | ((v & 2u) << 1) | ((v & 4u) << 2));
}
__device__ __forceinline__ unsigned sort_key(const DP& p, float x, float y, float z) {
  const float ux = __fmul_rn(__fsub_rn(x, p.ox), p.inv_edge), uy = __fmul_rn(__fsub_rn(y, p.oy), p.inv_edge);
  const float uz = p.dim == 3 ? __fmul_rn(__fsub_rn(z, p.oz), p.inv_edge) : 0.0f;
  const float fx = fminf(fmaxf(floorf(ux), 0.0f), (float)(p.nx - 1)), fy = fminf(fmaxf(floorf(uy), 0.0f), (float)(p.ny - 1));
  const float fz = p.dim == 3 ? fminf(fmaxf(floorf(uz), 0.0f), (float)(p.nz - 1)) : 0.0f;
  unsigned key = (unsigned)(((int)fz * p.ny + (int)fy) * p.nx + (int)fx);
  if (p.sub_bits) {
    const int b = p.sub_bits / p.dim;
    const float sc = (float)(1 << b), top = sc - 1.0f;
    const unsigned sx = (unsigned)fminf(fmaxf((ux - fx) * sc, 0.0f), top), sy = (unsigned)fminf(fmaxf((uy - fy) * sc, 0.0f), top);
    const unsigned sz = p.dim == 3 ? (unsigned)fminf(fmaxf((uz - fz) * sc, 0.0f), top) : 0u;
    key = (key << p.sub_bits) | spread_bits(sx, p.dim) | (spread_bits(sy, p.dim) << 1) | (p.dim == 3 ? spread_bits(sz, 3) << 2 : 0u);
  }
  return key;
}

__device__ __forceinline__ unsigned cell_key(const DP& p, float x, float y, float z) {
  const int cx = cell_coord(x, p.ox, p.inv_edge, p.nx), cy = cell_coord(y, p.oy, p.inv_edge, p.ny);
  const int cz = p.dim == 3 ? cell_coord(z, p.oz, p.inv_edge, p.nz) : 0;
  return (unsigned)((cz * p.ny + cy) * p.nx + cx);
}
