// sph_pair.cuh — the neighbour-list builds and the pair kernels (wall extrapolation, pass A, pass B).
// Included by sph.cu only.  DESIGN.md §5 describes the scheme:
//   one thread per particle i (cell-sorted order, so a warp covers ~2 cells);
//   list builds (k_build, k_wall_build; only on the steps that rebuild the lists): each lane walks the 9 (3-D) /
//            3 (2-D) x-rows of its own 27 / 9-cell stencil, every row one contiguous index range; a conservative
//            filter (float16 staged tile in k_build, float32 otherwise) with radius 2h(1 + skin); survivors are
//            staged in the lane's shared-memory queue and written four at a time to the warp's slot-major list;
//   list walks (k_wall, k_pass_a, k_pass_b; every step): one coalesced 16-byte load gives 4 neighbour indices,
//            their 256-bit records are gathered together; exact geometry from the fixed-point positions (integer
//            subtract + I2F), then the pair physics.  Entries beyond 2h add exactly zero.
#pragma once
#include <cuda_fp16.h>

#include "sph_common.cuh"

#ifndef SPH_PB
#define SPH_PB 128
#endif
#ifndef SPH_MINB
#define SPH_MINB 8
#endif
#ifndef SPH_QCAP
#define SPH_QCAP 32
#endif
#ifndef SPH_CH
#define SPH_CH 4
#endif
constexpr int PB = SPH_PB;     // threads per block in the pair kernels
constexpr int QCAP = SPH_QCAP; // queue entries per lane (QCAP * PB * 4 bytes of shared memory per block)
constexpr int CH = SPH_CH;     // candidates per lane between two queue-occupancy votes (loads issued together)

// Body = struct with  Ld load(unsigned j) const  and  void apply(const Ld&)  so that the gathers of
// four list entries are issued before the arithmetic of the first one.
//
// ListSink: what happens to a candidate that passes the filter: the per-warp neighbour list in global memory,
// slot-major: NL[(warp * caps + slot) * 32 + lane] (the list walks then read it with coalesced loads).
struct ListSink {
  // Survivors are staged in the lane's shared-memory queue and written out four at a time as one
  // 16-byte store: NL is an array of uint4 groups, group g of lane l of warp w at
  // NL[(w * capg + g) * 32 + l], so the readers' loads are coalesced and the scattered 4-byte
  // stores of a compact per-lane list become 16-byte ones (0.8 -> 0.3 ms at 4.1 M).
  unsigned* q;
  unsigned qa0, qa;
  uint4* __restrict__ g;  // this lane's column of the warp's groups: g[group * 32]
  int ng, capg, n;
  __device__ __forceinline__ ListSink(unsigned* q_, uint4* g_, int capg_) : q(q_), g(g_), ng(0), capg(capg_), n(0) {
    qa0 = (unsigned)__cvta_generic_to_shared(q_);
    qa = qa0;
  }
  __device__ __forceinline__ void push(const unsigned j) {
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(qa), "r"(j) : "memory");
    qa += PB * 4;
  }
  // Two candidates at once: r2 and thr are half2; candidates C and C + 1 of the chunk (list indices
  // j0 and j0 + 1) are pushed iff r2 < thr, C (+1) < rem (the lane's remaining range) and, for the
  // first one, ok0 (false only for the padding candidate in front of an odd range start).
  template <int C>
  __device__ __forceinline__ void push2(const unsigned r2, const unsigned thr, const int rem, const int ok0, const unsigned j0) {
    asm volatile(
        "{\n"
        ".reg .pred p, q, v;\n"
        ".reg .u32 t;\n"
        "setp.lt.f16x2 p|q, %1, %2;\n"
        "setp.ne.s32 v, %4, 0;\n"
        "and.pred p, p, v;\n"
        "setp.gt.and.s32 p, %3, %7, p;\n"
        "setp.gt.and.s32 q, %3, %8, q;\n"
        "@p st.shared.u32 [%0], %5;\n"
        "@p add.u32 %0, %0, %6;\n"
        "add.u32 t, %5, 1;\n"
        "@q st.shared.u32 [%0], t;\n"
        "@q add.u32 %0, %0, %6;\n"
        "}"
        : "+r"(qa)
        : "r"(r2), "r"(thr), "r"(rem), "r"(ok0), "r"(j0), "n"(PB * 4), "n"(C), "n"(C + 1)
        : "memory");
  }
  __device__ __forceinline__ void flush(const bool last) {
    const int qn = (int)(qa - qa0) / (PB * 4);
    const int ngr = last ? (qn + 3) >> 2 : qn >> 2;
    if (last) n = 4 * ng + qn;  // counts past the capacity too: the overflow is reported, never silently dropped
    const int nm = __reduce_max_sync(FULL, ngr);
#pragma unroll 1
    for (int t = 0; t < nm; ++t)
      if (t < ngr && ng + t < capg)
        g[(size_t)(ng + t) * 32] = make_uint4(q[(4 * t) * PB], q[(4 * t + 1) * PB], q[(4 * t + 2) * PB], q[(4 * t + 3) * PB]);
    ng += ngr;
    const int rem = last ? 0 : qn & 3;  // entries of an incomplete group go back to the queue front
    for (int r = 0; r < rem; ++r) q[r * PB] = q[(4 * ngr + r) * PB];
    qa = qa0 + rem * PB * 4;
  }
  __device__ __forceinline__ void after_chunk(const int ch = CH) {
    if (__any_sync(FULL, qa > qa0 + (QCAP - ch) * PB * 4)) flush(false);
  }
  __device__ __forceinline__ void finish() { flush(true); }
};

// Staged filter of k_build.  The lanes of a warp sit in 2-3 neighbouring cells, so their 3-cell
// ranges of one stencil row overlap in one index interval [smin, emax) of ~4-5 cells.  The warp reads
// it once with coalesced 16-byte loads and stages it in shared memory as float16 coordinates
// relative to the warp's first particle, in units of h, two candidates per record (x0 x1 y0 y1 |
// z0 z1); every lane then tests its own sub-range two candidates at a time with packed half
// arithmetic (difference form).  What bounds the walk is the L1/shared data pipe, which moves 128
// bytes per cycle whatever the address pattern: 16-byte float4 candidates cost 4 wavefronts per
// warp-wide read (staged float32: 98 % of the pipe's peak, profiles/r01d_README.md), the 6-byte
// float16 candidate 1.5.
// Margin of the float16 test (units of h, r_c = 2): coordinates are below 16 in magnitude (checked
// per row, else the row falls back to the float32 path), so each is rounded by at most 2^-8; the
// difference by 2^-11 |d| <= 1.1e-3: 8.9e-3 per axis, 1.54e-2 in norm, 2 r |e| + |e|^2 <= 6.2e-2 on
// r^2 at r = 2; the three roundings of the sum of squares add 3 * 2^-11 * 4 = 5.9e-3.  A true
// neighbour therefore computes r^2 < 4.068; the threshold is 4.08 plus the float32 image margin.
// A false positive has q >= 2 in the passes and adds exactly 0 (reading B2).
constexpr int TW = 128;   // candidates per warp tile
constexpr int TP = TW / 2 + 4;  // pair records per tile, padded for the chunk over-read
constexpr int CHS = 8;    // candidates (4 pair records) per lane between two occupancy votes
struct HCtx {          // per-lane constants of the float16 test
  float ox, oy, oz;    // origin: centred image of the warp's first particle
  unsigned xi, yi, zi; // this lane's coordinates, each duplicated in both halves
  bool bad;            // a coordinate of this lane is outside the float16 working range
};
struct HTile {
  uint2 xy[TP];     // (x0 x1), (y0 y1) as half2
  unsigned z[TP];   // (z0 z1)
};
__device__ __forceinline__ unsigned h2(const float a, const float b) {
  const __half2 h = __floats2half2_rn(a, b);
  return *reinterpret_cast<const unsigned*>(&h);
}
__device__ __forceinline__ unsigned hsub2(const unsigned a, const unsigned b) {
  unsigned d;
  asm("sub.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}
__device__ __forceinline__ unsigned hmul2(const unsigned a, const unsigned b) {
  unsigned d;
  asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}
__device__ __forceinline__ unsigned hfma2(const unsigned a, const unsigned b, const unsigned c) {
  unsigned d;
  asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}
template <int DIM, bool EXACT>
__device__ __forceinline__ float filter_t(const float4& ai, const float m2x, const float m2y, const float m2z,
                                          const float4& pj) {
  if (EXACT) return dist2(ai.x - pj.x, ai.y - pj.y, DIM == 3 ? ai.z - pj.z : 0.0f);
  if (DIM == 3) return fmaf(m2x, pj.x, fmaf(m2y, pj.y, fmaf(m2z, pj.z, pj.w)));
  return fmaf(m2x, pj.x, fmaf(m2y, pj.y, pj.w));
}
template <int DIM, bool EXACT, bool STAGE, class Sink>
__device__ __forceinline__ void walk_f(const DP& p, const float4* __restrict__ A, const int* __restrict__ lb,
                                       const bool act, const float4 ai, const int cx, const int cy,
                                       const int cz, HTile* __restrict__ tile, const HCtx& hc, Sink& sink,
                                       const float rl2m, const unsigned thr_h2) {
  const float m2x = -2.0f * ai.x, m2y = -2.0f * ai.y, m2z = -2.0f * ai.z;
  const float thr = EXACT ? rl2m : rl2m - ai.w;
  const int lane = threadIdx.x & 31;
  const int RC = p.reach, NR = DIM == 3 ? (2 * RC + 1) * (2 * RC + 1) : 2 * RC + 1;
  int ry = -RC, rz = DIM == 3 ? -RC : 0;
#pragma unroll 1
  for (int r = 0; r < NR; ++r) {
    int s = 0x7fffffff, e = 0;
    const int y = cy + ry, z = cz + rz;
    if (act && y >= 0 && y < p.ny && z >= 0 && z < p.nz) {
      const int rb = (z * p.ny + y) * p.nx;
      const int s1 = __ldg(lb + rb + max(cx - RC, 0));
      e = __ldg(lb + rb + min(cx + RC, p.nx - 1) + 1);
      if (e > s1) s = s1; else e = 0;
    }
    if (++ry > RC) { ry = -RC; ++rz; }
    const int smin = STAGE ? __reduce_min_sync(FULL, s) : 0, emax = STAGE ? __reduce_max_sync(FULL, e) : 0;
    bool staged = false;
    if constexpr (STAGE) if (emax > smin && emax - smin <= TW) {  // warp-uniform; a row in which no lane has a candidate (emax <= smin) skips the tile
      const int t0 = smin, n = emax - smin;
      bool bad = hc.bad;
      __syncwarp();
#pragma unroll
      for (int k = 0; k < TW; k += 32) {
        const int c = k + lane;
        if (c < n) {
          const float4 a = __ldg(A + t0 + c);
          const float x = (a.x - hc.ox) * p.inv_h, y = (a.y - hc.oy) * p.inv_h, z = DIM == 3 ? (a.z - hc.oz) * p.inv_h : 0.0f;
          bad |= !(fmaxf(fabsf(x), fmaxf(fabsf(y), fabsf(z))) < 15.9f);
          __half* xy = reinterpret_cast<__half*>(tile->xy + (c >> 1)) + (c & 1);
          xy[0] = __float2half_rn(x);
          xy[2] = __float2half_rn(y);
          if (DIM == 3) reinterpret_cast<__half*>(tile->z + (c >> 1))[c & 1] = __float2half_rn(z);
        }
      }
      staged = !__any_sync(FULL, bad);
      __syncwarp();
      if (staged) {
        const int lo = min(s, emax) - t0;  // this lane's part of the tile: [lo, lo + len), len <= 0: none
        const int len = max(e - t0 - lo, 0), odd = lo & 1, np = (odd + len + 1) >> 1;
        const int npmax = __reduce_max_sync(FULL, np);
        const int pb = lo >> 1, plast = (n + 1) >> 1;
#pragma unroll 1
        for (int kp = 0; kp < npmax; kp += CHS / 2) {
          const int pi = min(pb + kp, plast);  // reads run up to 3 records past the last one: the tile is padded
          uint2 xy[CHS / 2];
          unsigned zz[CHS / 2];
#pragma unroll
          for (int u = 0; u < CHS / 2; ++u) {
            xy[u] = tile->xy[pi + u];
            if (DIM == 3) zz[u] = tile->z[pi + u];
          }
          const int rem = odd + len - 2 * kp;    // candidates C of this chunk with C < rem are in the lane's range,
          const int ok0 = (kp > 0) | (odd ^ 1);  // except the one in front of an odd range start
          const unsigned j0 = (unsigned)(t0 + 2 * (pb + kp));
          unsigned r2[CHS / 2];
#pragma unroll
          for (int u = 0; u < CHS / 2; ++u) {
            const unsigned dx = hsub2(hc.xi, xy[u].x), dy = hsub2(hc.yi, xy[u].y);
            r2[u] = hfma2(dy, dy, hmul2(dx, dx));
            if (DIM == 3) {
              const unsigned dz = hsub2(hc.zi, zz[u]);
              r2[u] = hfma2(dz, dz, r2[u]);
            }
          }
          static_assert(CHS == 8, "four pair records per chunk");
          sink.template push2<0>(r2[0], thr_h2, rem, ok0, j0);
          sink.template push2<2>(r2[1], thr_h2, rem, 1, j0 + 2);
          sink.template push2<4>(r2[2], thr_h2, rem, 1, j0 + 4);
          sink.template push2<6>(r2[3], thr_h2, rem, 1, j0 + 6);
          sink.after_chunk(CHS);
        }
      }
    }
    if (!staged) {
      // the lanes' ranges are far apart (a warp that straddles the end of a cell row, wall particles
      // of a thin layer): every lane reads its own range from global memory
      const int len = e > 0 ? e - s : 0, jb0 = e > 0 ? s : 0;
      const int nmax = __reduce_max_sync(FULL, len);
      const int last = len > 0 ? e - 1 : 0;
#pragma unroll 1
      for (int k0 = 0; k0 < nmax; k0 += CH) {
        const int jb = jb0 + k0, rem = len - k0;
        const float4* __restrict__ ap = A + min(jb, last);  // clamp of the chunk base (arrays are padded by CH)
        float4 pj[CH];
#pragma unroll
        for (int u = 0; u < CH; ++u) pj[u] = __ldg(ap + u);
#pragma unroll
        for (int u = 0; u < CH; ++u)
          if (u < rem && filter_t<DIM, EXACT>(ai, m2x, m2y, m2z, pj[u]) < thr) sink.push((unsigned)(jb + u));
        sink.after_chunk(STAGE ? CHS : CH);  // the head room the next chunk of either path needs
      }
    }
  }
  sink.finish();
}

// List walk: every lane runs over its own column of the warp's neighbour groups; the loop is
// warp-uniform (to the largest count in the warp), one coalesced 16-byte load gives 4 neighbours
// whose records are gathered together before the arithmetic.
// RO = false: the list was written by this thread earlier in the same kernel (no read-only path).
template <bool RO = true, class Body>
__device__ __forceinline__ void walk_l(const uint4* g, const int cnt, Body& body) {
  const int nm = __reduce_max_sync(FULL, cnt);
#pragma unroll 1
  for (int k = 0; k < nm; k += 4) {
    if (k < cnt) {
      // the list entries are read once per pass: LDG.E.NA (no L1 allocation) leaves the L1 to the records, which are
      // gathered ~85 times each (pass A / pass B -1.3 % / -2.3 % at 16.8 M, the bare walk -3 %; eviction hints on the
      // record loads themselves change nothing: profiles/r02_README.md)
      uint4 e;
      if (RO) asm("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(e.x), "=r"(e.y), "=r"(e.z), "=r"(e.w) : "l"(g + (size_t)(k >> 2) * 32));
      else e = g[(size_t)(k >> 2) * 32];
      decltype(body.load(0u)) ld[4];
      ld[0] = body.load(e.x);
      if (k + 1 < cnt) ld[1] = body.load(e.y);
      if (k + 2 < cnt) ld[2] = body.load(e.z);
      if (k + 3 < cnt) ld[3] = body.load(e.w);
      body.apply(ld[0]);
      if (k + 1 < cnt) body.apply(ld[1]);
      if (k + 2 < cnt) body.apply(ld[2]);
      if (k + 3 < cnt) body.apply(ld[3]);
    }
  }
}

// Exact pair geometry in units of Qp from the fixed-point positions: d = X_i - X_j (wrapping
// integer subtract, exact), r^2, 1/r (r = 0 -> r = 0 with a finite 1/r), q = r/h and the
// Wendland C2 factors (reading A1): w = (1 - q/2)^4 (1 + 2q) = W / alpha_d,  f = (1 - q/2)^3.
// MUFU.RSQ / MUFU.RCP are accurate to about 2^-22 and their error is a smooth function of the
// operand, i.e. of the neighbour's distance and density: in the momentum sum, whose terms cancel to
// 1e-3 of their size, that is a systematic bias of 1e-4 g at H / dp = 100 (measured against the oracle).
// One Newton step each makes the error rounding-sized and random.
__device__ __forceinline__ float rsqrt_fast(float x) {  // x >= 0.5 here: no denormal fix-up needed
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  const float e = fmaf(-x * y, y, 1.0f);
  return fmaf(0.5f * y, e, y);
}
__device__ __forceinline__ float div_fast(float a, float b) {  // b normal and finite here
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(b));
  y = fmaf(y, fmaf(-b, y, 1.0f), y);
  return a * y;
}
// Compensated (Kahan) float32 accumulator.  The momentum sum cancels to O(g) from terms whose
// partial sums reach O(g H / h): plain float32 accumulation loses 1e-4 g at H / dp = 100
// (measured against the oracle); sigma needs 5e-7 relative for the same reason.
struct KSum {
  float s = 0.f, c = 0.f;
  __device__ __forceinline__ void add(const float x) {
    const float y = x - c, t = s + y;
    c = (t - s) - y;
    s = t;
  }
  __device__ __forceinline__ float value() const { return s - c; }
};
struct Geo {
  float dx, dy, dz, r, rinv, w, f;
};
__device__ __forceinline__ float rsqrt_raw(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// REFINE = false: 1 / r straight from MUFU.RSQ (2^-22).  Measured in pass A (profiles/r02_README.md): -3 % on the
// pass, but the 10-step acceleration error of box2d_jitter goes from 0.99e-4 to 1.05e-4 of |g| (bar 1e-4): not used.
template <int DIM, bool REFINE = true>
__device__ __forceinline__ Geo geometry(const DP& p, const uint4& xi, const uint4& xj) {
  Geo g;
  g.dx = (float)(int)(xi.x - xj.x);
  g.dy = (float)(int)(xi.y - xj.y);
  g.dz = DIM == 3 ? (float)(int)(xi.z - xj.z) : 0.0f;
  const float r2 = DIM == 3 ? fmaf(g.dz, g.dz, fmaf(g.dy, g.dy, g.dx * g.dx)) : fmaf(g.dy, g.dy, g.dx * g.dx);
  g.rinv = REFINE ? rsqrt_fast(fmaxf(r2, 0.5f)) : rsqrt_raw(fmaxf(r2, 0.5f));
  g.r = r2 * g.rinv;
  const float qq = g.r * p.qh;
  const float t = fmaxf(fmaf(-0.5f, qq, 1.0f), 0.0f), t2 = t * t;
  g.w = t2 * t2 * fmaf(2.0f, qq, 1.0f);
  g.f = t2 * t;
  return g;
}

// W / alpha_d in float64 from the exact integer separation (reading A1), for the number density
// sigma_i only.  p = c0^2 rho0 (sigma/sigma0 - 1) with c0^2 = 200 g H amplifies a relative error of
// sigma by 200, and the momentum sum amplifies a pressure error by another H / h: float32 terms
// (2e-7 each) leave 3e-5 of rho0 g H in p and 2.5e-4 g in a at H / dp = 100 (measured against the
// oracle).  r^2 is an exact 64-bit integer; its root is one float64 Newton step from the float32 r.
template <int DIM, bool SUBQ>
__device__ __forceinline__ double w64(const DP& p, const uint4& xi, const uint4& xj, const Geo& g) {
  const long long dx = (int)(xi.x - xj.x), dy = (int)(xi.y - xj.y), dz = DIM == 3 ? (int)(xi.z - xj.z) : 0;
  double r2, r0, hy;
  if (SUBQ) {
    // include the lobits bits of each coordinate below the record's word (units of Q/1024): every multi-phase run
    // (for a light phase with its own large c0, config 2b: c_air^2 = 1000 c_w^2, sigma must be good to 1e-11, i.e.
    // positions to 1e-12 m) and single-phase runs whose pair unit Qp is coarse for their size (DP::subq)
    const unsigned lm = (1u << p.lobits) - 1u;
    const double ex = (double)((dx << p.lobits) + (int)((xi.w >> 22) & lm) - (int)((xj.w >> 22) & lm));
    const double ey = (double)((dy << p.lobits) + (int)((xi.w >> 12) & lm) - (int)((xj.w >> 12) & lm));
    const double ez = DIM == 3 ? (double)((dz << p.lobits) + (int)((xi.w >> 2) & lm) - (int)((xj.w >> 2) & lm)) : 0.0;
    r2 = fma(ez, ez, fma(ey, ey, ex * ex));
    r0 = (double)(g.r * p.sub_scale);
    hy = (double)(g.rinv * p.sub_half_inv);
  } else {
    r2 = (double)(dx * dx + dy * dy + dz * dz);
    r0 = (double)g.r;
    hy = (double)(0.5f * g.rinv);
  }
  // sqrt by one Newton step in float64 from the float32 r of the geometry (relative error e <= 2e-7,
  // with the residuals 1e-6): r = r0 + (r2 - r0^2) / (2 r0), error e^2 / 2.  r2 = 0 gives r0 = 0, r = 0.
  const double r = fma(fma(-r0, r0, r2), hy, r0);
  const double t = fma(r, p.mhqD[SUBQ], 1.0), u = fma(r, p.tqD[SUBQ], 1.0), t2 = t * t;
  // outside the support (decided on the float32 q of the geometry, as for every other term) the
  // term is exactly 0; within a rounding of q = 2 the value is below 1e-26
  return g.f > 0.0f ? t2 * t2 * u : 0.0;
}

// Pair body = the neighbour's record (one 256-bit gather) + the arithmetic on it.
struct LdXB {
  XB r;
  unsigned j;
};
template <class F>
struct BodyXB {
  const XB* __restrict__ R;
  F f;
  __device__ __forceinline__ LdXB load(const unsigned j) const { return LdXB{ldg256(R + j), j}; }
  __device__ __forceinline__ void apply(const LdXB& l) { f(l.r.x, l.r.b, l.j); }
};
template <class F>
__device__ __forceinline__ BodyXB<F> make_body(const XB* R, F f) { return BodyXB<F>{R, f}; }

__device__ __forceinline__ void cell_of_key(const DP& p, unsigned key, int& cx, int& cy, int& cz) {
  const unsigned row = key / (unsigned)p.nx;
  cx = (int)(key - row * (unsigned)p.nx);
  cz = (int)(row / (unsigned)p.ny);
  cy = (int)(row - (unsigned)cz * (unsigned)p.ny);
}

// ------------------------------------------------------------------------------------------
// Neighbour list build (once per step, after the reorder): the filter walk of every fluid particle
// over the fluid arrays, survivors written to the warp's slot-major list.  Both fluid pair passes
// of the step read it, so the 27-cell candidate walk is done once per step, not once per pass.
// ------------------------------------------------------------------------------------------
template <int DIM, bool EXACT>
__global__ void __launch_bounds__(PB)
k_build(const DP p, SS* __restrict__ S, const int nf, const float4* __restrict__ A,
        const unsigned* __restrict__ K, const int* __restrict__ lbF, uint4* __restrict__ NL,
        int* __restrict__ NC, const int caps,
        const float4* __restrict__ WA, const int* __restrict__ lbW, const unsigned char* __restrict__ wnear,
        uint4* __restrict__ NLW, int* __restrict__ NCW, const int capsw,
        unsigned* __restrict__ IDcur, const unsigned* __restrict__ IDnext) {
  __shared__ unsigned qs[QCAP * PB];
  __shared__ HTile tiles[PB / 32];
  const int i0 = blockIdx.x * PB + threadIdx.x;
  const bool act = i0 < nf;
  const int i = act ? i0 : nf - 1;
  const float4 ai = A[i];
  const unsigned key = K[i] >> p.sub_bits;   // the cell id sits above the sub-cell Morton bits of the sort key
  int cx, cy, cz;
  cell_of_key(p, key, cx, cy, cz);
  HCtx hc;
  hc.ox = __shfl_sync(FULL, ai.x, 0); hc.oy = __shfl_sync(FULL, ai.y, 0); hc.oz = DIM == 3 ? __shfl_sync(FULL, ai.z, 0) : 0.0f;
  {
    const float x = (ai.x - hc.ox) * p.inv_h, y = (ai.y - hc.oy) * p.inv_h, z = DIM == 3 ? (ai.z - hc.oz) * p.inv_h : 0.0f;
    hc.bad = act && !(fmaxf(fabsf(x), fmaxf(fabsf(y), fabsf(z))) < 15.9f);
    hc.xi = h2(x, x); hc.yi = h2(y, y); hc.zi = h2(z, z);
  }
  const float rl2m = S->rl2m;          // thresholds of the skin this build takes (adaptive: SS, k_predict)
  const unsigned thr_h2 = S->thr_h2;
  int n = 0, nw = 0;
  {
    ListSink sink(qs + threadIdx.x, NL + (size_t)(i0 >> 5) * (caps >> 2) * 32 + (threadIdx.x & 31), caps >> 2);
    walk_f<DIM, EXACT, true>(p, A, lbF, act, ai, cx, cy, cz, tiles + (threadIdx.x >> 5), hc, sink, rl2m, thr_h2);
    n = sink.n;
  }
  // fluid-wall lists (same filter over the static wall arrays) for the warps that have a wall
  // particle in a stencil: both pair passes read them, so the wall candidate walk is also paid once
  if (__any_sync(FULL, act && wnear[key])) {
    ListSink sink(qs + threadIdx.x, NLW + (size_t)(i0 >> 5) * (capsw >> 2) * 32 + (threadIdx.x & 31), capsw >> 2);
    walk_f<DIM, EXACT, true>(p, WA, lbW, act, ai, cx, cy, cz, tiles + (threadIdx.x >> 5), hc, sink, rl2m, thr_h2);
    nw = sink.n;
  }
  if (act) {
    IDcur[i] = IDnext[i];  // caller ids of the new order (k_reorder wrote IDnext from IDcur: no ping-pong of pointers)
    NC[i] = min(n, caps);
    NCW[i] = min(nw, capsw);
    if (n > caps) atomicMax(&S->list_overflow, n);
    if (nw > capsw) atomicMax(&S->list_overflow, nw);
  }
}

// ------------------------------------------------------------------------------------------
// Wall extrapolation, Eq. 2.12 (readings A4-A7); a_w = 0, v_wall = 0.
// One thread per wall dummy particle, summing over its fluid neighbours.  WB = (v_w, p_w).
// ------------------------------------------------------------------------------------------
// k_wall_build (list build only, in the rebuild branch of a step): the float32 filter walk of every wall
// particle over the fluid arrays, survivors written to its wall-fluid neighbour list NLF / NCF.
template <int DIM, bool EXACT>
__global__ void __launch_bounds__(PB)
k_wall_build(const DP p, SS* __restrict__ S, const int nw, const float4* __restrict__ WA,
             const unsigned* __restrict__ WK, const float4* __restrict__ A, const int* __restrict__ lbF,
             uint4* __restrict__ NLF, int* __restrict__ NCF, const int capsf) {
  __shared__ unsigned qs[QCAP * PB];
  const int w0 = blockIdx.x * PB + threadIdx.x;
  const bool act = w0 < nw;
  const int w = act ? w0 : nw - 1;
  uint4* col = NLF + (size_t)(w0 >> 5) * (capsf >> 2) * 32 + (threadIdx.x & 31);
  const float4 ai = WA[w];
  int cx, cy, cz;
  cell_of_key(p, WK[w] >> p.sub_bits, cx, cy, cz);
  ListSink sink(qs + threadIdx.x, col, capsf >> 2);
  walk_f<DIM, EXACT, false>(p, A, lbF, act, ai, cx, cy, cz, nullptr, HCtx{}, sink, S->rl2m, S->thr_h2);
  if (act) {
    NCF[w] = min(sink.n, capsf);
    if (sink.n > capsf) atomicMax(&S->list_overflow, sink.n);
  }
}

// k_wall: Eq. 2.12 for every wall particle from its wall-fluid neighbour list; WITH_VEL: pressure and the
// velocity of reading A6 (first wall pass of a step), else the pressure only (second pass, after pass A).
template <int DIM, bool MULTI, bool WITH_VEL>
__global__ void __launch_bounds__(PB)
k_wall(const DP p, const SS* __restrict__ S, const int nw, XB* __restrict__ WR, const XB* __restrict__ R,
       const uint4* __restrict__ NLF, const int* __restrict__ NCF, const int capsf) {
  const int w0 = blockIdx.x * PB + threadIdx.x;
  const bool act = w0 < nw;
  const int w = act ? w0 : nw - 1;
  const uint4 xi = WR[w].x;
  const uint4* col = NLF + (size_t)(w0 >> 5) * (capsf >> 2) * 32 + (threadIdx.x & 31);
  const int cnt = act ? NCF[w] : 0;
  float sW = 0, sp = 0, sWr = 0, srx = 0, sry = 0, srz = 0, svx = 0, svy = 0, svz = 0;
  // multi-phase form of Eq. 2.12 (every fluid term divided by rho_f) unless the run asks for the
  // wall model of Adami et al. (2012) without the paper's extensions (NEXT-4 ablation)
  const bool mw = MULTI && !(p.flags & SPH_FLAG_WALL_ADAMI_ONLY);
  {
    auto body = make_body(R, [&](const uint4& xj, const float4& bj, const unsigned j) {
    const Geo g = geometry<DIM>(p, xi, xj);  // r_wf = r_w - r_f
    const int ph = MULTI ? phase_of(xj) : 0;
    const float rhof = p.rho0[ph] + bj.w, pf = p.c2[ph] * bj.w;
    sW += g.w;
    if (MULTI && mw) {
      const float ir = div_fast(g.w, rhof);
      sp = fmaf(pf, ir, sp);
      sWr += ir;
      srx = fmaf(g.dx, g.w, srx); sry = fmaf(g.dy, g.w, sry); srz = fmaf(g.dz, g.w, srz);
    } else {
      sp = fmaf(pf, g.w, sp);
      const float rw = rhof * g.w;
      srx = fmaf(g.dx, rw, srx); sry = fmaf(g.dy, rw, sry); srz = fmaf(g.dz, rw, srz);
    }
    if (WITH_VEL) { svx = fmaf(bj.x, g.w, svx); svy = fmaf(bj.y, g.w, svy); svz = fmaf(bj.z, g.w, svz); }
    });
    walk_l(col, cnt, body);
  }
  if (!act) return;
  float pwall = 0.f, vx = S->vwall[0], vy = S->vwall[1], vz = S->vwall[2];  // reading A7: v_w = v_wall
  if (sW > 0.f) {
    const float lever = p.Qf * (S->gw[0] * srx + S->gw[1] * sry + S->gw[2] * srz);  // (g - a_w) . sum
    pwall = (sp + lever) / (mw ? sWr : sW);
    if (WITH_VEL && (p.flags & SPH_FLAG_WALL_VEL_MIRROR)) {
      const float is = 1.0f / sW;  // reading A6: v_w = 2 v_wall - <v_f>
      vx = fmaf(2.0f, vx, -svx * is); vy = fmaf(2.0f, vy, -svy * is); vz = fmaf(2.0f, vz, -svz * is);
    }
  }
  if (WITH_VEL) WR[w].b = make_float4(vx, vy, vz, pwall);
  else WR[w].b.w = pwall;
}

// ------------------------------------------------------------------------------------------
// Pair pass A: sigma_i + Riemann continuity Eq. 2.9 with Eq. 2.8
// in the scalar form (v_i - v*).grad W = (U* - U_L) W', then the density update
// Eq. 2.21 / summation Eq. 2.4 in the normalised form of Eq. 2.18 (readings A3, A5, A15).
// The self pair is a candidate like any other: it adds W(0) to sigma (reading A14) and, with
// r = 0 and v_ij = 0, nothing to the continuity sum.
// ------------------------------------------------------------------------------------------
// SUBQ: sigma_i from separations that include the 10-bit residuals of the master positions (units of
// Q/1024): every multi-phase run, and single-phase runs whose quantum is coarse for their size (sph.cu:
// DP::subq; the 1e-4 bar on a needs sigma to about 1e-6 h / H relative).
template <int DIM, bool MULTI, bool SUBQ>
__global__ void __launch_bounds__(PB, SPH_MINB)
k_pass_a(const DP p, const SS* __restrict__ S, const int nf, const int init,
         const XB* __restrict__ R, const XB* __restrict__ WR,
         XB* __restrict__ Rout, float* __restrict__ SIG, float* __restrict__ DRHO,
         const uint4* __restrict__ NL, const int* __restrict__ NC, const int caps,
         const uint4* __restrict__ NLW, const int* __restrict__ NCW, const int capsw) {
  const int i0 = blockIdx.x * PB + threadIdx.x;
  const bool act = i0 < nf;
  const int i = act ? i0 : nf - 1;
  const uint4 xi = R[i].x;
  const float4 bi = R[i].b;
  const int ncw = act ? NCW[i] : 0;
  const int phi = MULTI ? phase_of(xi) : 0;
  const float rho0i = p.rho0[phi], c2i = p.c2[phi], ci = p.c0[phi];
  const float rhoi = rho0i + bi.w, prsi = c2i * bi.w, ZL = rhoi * ci;
  double sig = 0.0;  // sum of W/alpha in float64 (DESIGN.md §4 "precision")
  float acc = 0.f;
  // reading A13b: the number density of a free-surface (heavy) phase particle of a multi-phase
  // run counts its own phase and the walls only; an internal-flow (light) phase particle counts every neighbour
  const bool sig_all = !MULTI || !((p.fs_mask >> phi) & 1u);
  {
    constexpr bool RF = true;
    auto body = make_body(R, [&](const uint4& xj, const float4& bj, const unsigned j) {
    const Geo g = geometry<DIM, RF>(p, xi, xj);
    if (!MULTI || sig_all || phase_of(xj) == phi) sig += w64<DIM, SUBQ>(p, xi, xj, g);
    const float vd = fmaf(bi.z - bj.z, g.dz, fmaf(bi.y - bj.y, g.dy, (bi.x - bj.x) * g.dx));
    if (!MULTI) {
      // equal c: (U* - U_L)(Z_L + Z_R) = c (rho_j v_ij.e + c (rho_i - rho_j)) with p = c^2 (rho - rho0)
      const float rhoj = rho0i + bj.w;
      const float num = fmaf(rhoj, vd, (ci * (bi.w - bj.w)) * g.r);
      acc = fmaf(g.f, div_fast(num, rhoj * (rhoi + rhoj)), acc);
    } else {
      const int phj = phase_of(xj);
      const float rhoj = p.rho0[phj] + bj.w, ZR = rhoj * p.c0[phj];
      const float dpr = phj == phi ? c2i * (bi.w - bj.w) : prsi - p.c2[phj] * bj.w;
      const float num = fmaf(ZR, vd, dpr * g.r);  // (U* - U_L) W' (Z_L + Z_R) / (W'/r), units of Q
      acc = fmaf(p.mass[phj] * g.f, div_fast(num, rhoj * (ZL + ZR)), acc);
    }
    });
    walk_l(NL + (size_t)(i0 >> 5) * (caps >> 2) * 32 + (threadIdx.x & 31), act ? NC[i] : 0, body);
  }
  float accw = 0.f;
  if (__any_sync(FULL, ncw > 0)) {
    {
      auto body = make_body(WR, [&](const uint4& xj, const float4& bj, const unsigned j) {  // (v_w, p_w)
      const Geo g = geometry<DIM>(p, xi, xj);
      sig += w64<DIM, SUBQ>(p, xi, xj, g);
      const float rhow = fmaf(bj.w, p.inv_c2[phi], rho0i);  // reading A5
      const float ZR = rhow * ci;
      const float vd = fmaf(bi.z - bj.z, g.dz, fmaf(bi.y - bj.y, g.dy, (bi.x - bj.x) * g.dx));
      const float num = fmaf(ZR, vd, (prsi - bj.w) * g.r);
      accw = fmaf(g.f, div_fast(num, ZL + ZR), accw);
      });
      walk_l(NLW + (size_t)(i0 >> 5) * (capsw >> 2) * 32 + (threadIdx.x & 31), ncw, body);
    }
  }
  if (!act) return;
  // sigma_i / sigma0 - 1 in float64, stored as float32: the density of
  // Eq. 2.17 / 2.18 is rho0 (1 + dev), so the deviation carries the precision.
  const float dev = (float)(p.a_over_s0 * sig - 1.0);
  const float accf = MULTI ? acc : p.mass[0] * acc;
  const float drho = 2.0f * rhoi * p.gradcQ * fmaf(p.V0, accw, accf);  // Eq. 2.9
  float d = bi.w;
  if (!init) {
    if ((p.fs_mask >> phi) & 1u) d = fmaf(S->dt, drho, d);  // Eq. 2.21
    else d = rho0i * dev;                                   // Eq. 2.4 / 2.18
  }
  Rout[i] = XB{xi, make_float4(bi.x, bi.y, bi.z, d)};
  SIG[i] = dev;
  DRHO[i] = drho;
}

// ------------------------------------------------------------------------------------------
// Pair pass B: momentum Eq. 2.10 with p* of Eq. 2.8 (fluid j) / Eq. 2.11 (wall j), penalty
// Eq. 2.13-2.15 (readings A8, A9, A11), gravity, then the second half kick Eq. 2.22.
// ------------------------------------------------------------------------------------------
template <int DIM, bool MULTI, bool EXACT>
__global__ void __launch_bounds__(PB, SPH_MINB)
k_pass_b(const DP p, const SS* __restrict__ S, const int nf,
         const XB* __restrict__ R, const XB* __restrict__ WR,
         const float4* __restrict__ WN, float4* __restrict__ Bout, float4* __restrict__ ACC,
         const uint4* __restrict__ NL, const int* __restrict__ NC, const int caps,
         const uint4* __restrict__ NLW, const int* __restrict__ NCW, const int capsw) {
  const int i0 = blockIdx.x * PB + threadIdx.x;
  const bool act = i0 < nf;
  const int i = act ? i0 : nf - 1;
  const uint4 xi = R[i].x;
  const float4 bi = R[i].b;
  const int ncw = act ? NCW[i] : 0;
  const int phi = MULTI ? phase_of(xi) : 0;
  const float rho0i = p.rho0[phi], c2i = p.c2[phi], ci = p.c0[phi];
  const float rhoi = rho0i + bi.w, prsi = c2i * bi.w, ZL = rhoi * ci;
  KSum ax, ay, az;
  {
    auto body = make_body(R, [&](const uint4& xj, const float4& bj, const unsigned j) {
    const Geo g = geometry<DIM>(p, xi, xj);
    const float vd = fmaf(bi.z - bj.z, g.dz, fmaf(bi.y - bj.y, g.dy, (bi.x - bj.x) * g.dx));
    const float dU = -vd * g.rinv;  // U_L - U_R
    float coef;
    if (!MULTI) {
      // equal c: p*/rho_j = (rho_i p_j + rho_j p_i + rho_i rho_j beta dU) / ((rho_i + rho_j) rho_j)
      const float rhoj = rho0i + bj.w, prsj = c2i * bj.w;
      const float beta = fminf(3.0f * fmaxf(dU, 0.f), ci);
      const float num = fmaf(rhoi * rhoj, beta * dU, fmaf(rhoi, prsj, rhoj * prsi));
      coef = g.f * div_fast(num, (rhoi + rhoj) * rhoj);
    } else {
      const int phj = phase_of(xj);
      const float rhoj = p.rho0[phj] + bj.w, prsj = p.c2[phj] * bj.w, ZR = rhoj * p.c0[phj];
      const float izs = div_fast(1.0f, ZL + ZR);
      const float ctil = (ZL + ZR) * div_fast(1.0f, rhoi + rhoj);
      const float beta = fminf(3.0f * fmaxf(dU, 0.f), ctil);
      const float pstar = fmaf(ZL, prsj, ZR * prsi) * izs + ZL * ZR * izs * div_fast(beta, ctil) * dU;
      coef = g.f * div_fast(p.mass[phj] * pstar, rhoj);
    }
    ax.add(coef * g.dx); ay.add(coef * g.dy);
    if (DIM == 3) az.add(coef * g.dz);
    });
    walk_l(NL + (size_t)(i0 >> 5) * (caps >> 2) * 32 + (threadIdx.x & 31), act ? NC[i] : 0, body);
  }
  KSum wx, wy, wz;
  if (__any_sync(FULL, ncw > 0)) {
    const bool pen = (p.pen_mask >> phi) & 1u;
    {
      auto body = make_body(WR, [&](const uint4& xj, const float4& bj, const unsigned j) {
      const float pw = bj.w;
      const Geo g = geometry<DIM>(p, xi, xj);
      const float rhow = fmaf(pw, p.inv_c2[phi], rho0i);
      const float pstar = div_fast(fmaf(rhoi, pw, rhow * prsi), rhoi + rhow);  // Eq. 2.11
      const float coef = g.f * pstar;
      wx.add(coef * g.dx); wy.add(coef * g.dy);
      if (DIM == 3) wz.add(coef * g.dz);
      if (pen) {
        const float4 n = __ldg(WN + j);
        if (n.x != 0.f || n.y != 0.f || n.z != 0.f) {
          const float nd = n.x * g.dx + n.y * g.dy + n.z * g.dz;  // n_w . (r_i - r_w) / Q
          const float delta = nd * p.two_over_dp;                  // Eq. 2.15 (reading A9); two_over_dp holds 2 Q / dp
          if (delta < 1.0f && delta > -1.0f) {
            const float lam = (1.0f - delta) * (1.0f - delta);     // Eq. 2.14 (reading A8)
            const float Pn = p.gamma_p * lam * fabsf(prsi * nd * g.rinv);
            const float c = Pn * g.f * g.r;                        // Eq. 2.13, W' = (W'/r) r
            wx.add(c * n.x); wy.add(c * n.y);
            if (DIM == 3) wz.add(c * n.z);
          }
        }
      }
      });
      walk_l(NLW + (size_t)(i0 >> 5) * (capsw >> 2) * 32 + (threadIdx.x & 31), ncw, body);
    }
  }
  if (!act) return;
  const float sf = -2.0f * p.gradcQ / rhoi * (MULTI ? 1.0f : p.mass[0]);  // Eq. 2.10
  const float sw = -2.0f * p.gradcQ / rhoi * p.V0;
  // a = g + sf * fluid sum + sw * wall sum, combined in float64 once per particle (the two sums
  // nearly cancel against g in a resting column)
  const double sfd = (double)sf, swd = (double)sw;
  const float fx = (float)((double)S->g[0] + sfd * ((double)ax.s - (double)ax.c) + swd * ((double)wx.s - (double)wx.c));
  const float fy = (float)((double)S->g[1] + sfd * ((double)ay.s - (double)ay.c) + swd * ((double)wy.s - (double)wy.c));
  const float fz = DIM == 3 ? (float)((double)S->g[2] + sfd * ((double)az.s - (double)az.c) + swd * ((double)wz.s - (double)wz.c)) : 0.f;
  ACC[i] = make_float4(fx, fy, fz, 0.f);
  const float hdt = 0.5f * S->dt;
  Bout[i] = make_float4(fmaf(hdt, fx, bi.x), fmaf(hdt, fy, bi.y), fmaf(hdt, fz, bi.z), bi.w);  // Eq. 2.22
}
