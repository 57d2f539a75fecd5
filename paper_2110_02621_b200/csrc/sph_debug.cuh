// sph_debug.cuh — output, integral quantities and the integer-contract debug paths (not on the
// hot path).  Included by sph.cu only.  The contract (reading A24) is defined on the float32
// image of the master position: these kernels work on image arrays G = (xg, yg, zg, 0).
#pragma once
#include "sph_common.cuh"

__global__ void k_image(DP p, int n, const XB* __restrict__ R, float4* __restrict__ G) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 x = R[i].x;
  G[i] = make_float4(fx_image(p, x, 0), fx_image(p, x, 1), p.dim == 3 ? fx_image(p, x, 2) : 0.0f, 0.0f);
}

// ------------------------------------------------------------------------------------------
// Contract-exact stencil walk (debug paths): one warp per particle, lanes over the candidates of each x-row of the
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
  const int RC = p.reach, W = 2 * RC + 1;     // W * W <= 25 rows: one per lane
  const int nrow = p.dim == 3 ? W * W : W;
  int rs = 0, re = 0;
  if (lane < nrow) {
    int y = cy + (lane % W) - RC, z = cz + (lane / W) - RC;
    if (p.dim != 3) z = 0;
    if (y >= 0 && y < p.ny && z >= 0 && z < p.nz) {
      int rb = (z * p.ny + y) * p.nx;
      rs = lb[rb + max(cx - RC, 0)];
      re = lb[rb + min(cx + RC, p.nx - 1) + 1];
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

constexpr int PW = 8;  // warps per block in k_neigh


// ------------------------------------------------------------------------------------------
// Output
// ------------------------------------------------------------------------------------------
__global__ void k_get(DP p, int n, int is_wall, const XB* __restrict__ R, const float4* __restrict__ B,
                      const float4* __restrict__ ACC, const unsigned* __restrict__ ID, float* pos,
                      float* vel, float* rho, float* prs, float* acc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 x = R[i].x;
  const float4 b = B ? B[i] : R[i].b;
  const size_t o = ID[i];
  if (pos) {
    pos[3 * o] = fx_image(p, x, 0);
    pos[3 * o + 1] = fx_image(p, x, 1);
    pos[3 * o + 2] = p.dim == 3 ? fx_image(p, x, 2) : 0.0f;
  }
  if (vel) { vel[3 * o] = b.x; vel[3 * o + 1] = b.y; vel[3 * o + 2] = b.z; }
  if (is_wall) {  // B = (v_w, p_w)
    if (acc) { acc[3 * o] = 0.f; acc[3 * o + 1] = 0.f; acc[3 * o + 2] = 0.f; }
    if (rho) rho[o] = fmaf(b.w, p.inv_c2[0], p.rho0[0]);
    if (prs) prs[o] = b.w;
  } else {
    const int ph = phase_of(x);
    if (acc) { const float4 a = ACC[i]; acc[3 * o] = a.x; acc[3 * o + 1] = a.y; acc[3 * o + 2] = a.z; }
    if (rho) rho[o] = p.rho0[ph] + b.w;
    if (prs) prs[o] = p.c2[ph] * b.w;
  }
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
k_stats(DP p, int nf, const XB* __restrict__ R, const float4* __restrict__ B, StatAcc* out) {
  double ek = 0;
  unsigned cnt[SPH_MAX_PHASES] = {0, 0, 0, 0};
  float xf = -INFINITY;
  const int up = p.dim - 1;
  const float zlim = p.dmin[up] + 6.0f * (float)p.dpD;
  for (int i = blockIdx.x * 256 + threadIdx.x; i < nf; i += gridDim.x * 256) {
    const uint4 x = R[i].x;
    const float4 v = B[i];
    const int ph = phase_of(x);
    ek += 0.5 * p.massD[ph] * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
#pragma unroll
    for (int k = 0; k < SPH_MAX_PHASES; ++k) cnt[k] += (ph == k);
    const float zz = fx_image(p, x, up);
    if (ph == 0 && zz < zlim) xf = fmaxf(xf, fx_image(p, x, 0));
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

// sph_debug_list_check: every fluid neighbour of the float32 contract (reading A24) must be an entry
// of the step's neighbour list (the float16 / float32 candidate filters of k_build are conservative);
// out[0] += contract neighbours missing from the list, out[1] += list entries (self excluded) that
// are not contract neighbours, out[2] += list entries in total.
__global__ void __launch_bounds__(PW * 32)
k_list_check(DP p, int nf, const float4* __restrict__ P, const int* __restrict__ lbF,
             const uint4* __restrict__ NL, const int* __restrict__ NC, int caps, unsigned long long* out) {
  __shared__ unsigned qs[PW][64];
  const int i = blockIdx.x * PW + (threadIdx.x >> 5);
  if (i >= nf) return;
  const int lane = threadIdx.x & 31;
  const float4 pi = P[i];
  const unsigned* col = reinterpret_cast<const unsigned*>(NL + (size_t)(i >> 5) * (caps >> 2) * 32 + (i & 31));
  const int cnt = NC[i];
  int missing = 0, found = 0;
  walk(p, P, lbF, pi.x, pi.y, pi.z, i, qs[threadIdx.x >> 5], [&](int j) {
    bool in = false;
    for (int k = 0; k < cnt && !in; ++k) in = col[(size_t)(k >> 2) * 128 + (k & 3)] == (unsigned)j;
    if (in) ++found; else ++missing;
  });
  for (int o = 16; o > 0; o >>= 1) {
    missing += __shfl_xor_sync(FULL, missing, o);
    found += __shfl_xor_sync(FULL, found, o);
  }
  if (lane == 0) {
    if (missing) atomicAdd(out, (unsigned long long)missing);
    atomicAdd(out + 1, (unsigned long long)(cnt - 1 - found));
    atomicAdd(out + 2, (unsigned long long)cnt);
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

// contract_view (sph.cu): sort keys of the on-demand contract order
__global__ void k_dbg_idkeys(int n, const unsigned* __restrict__ ID, unsigned* __restrict__ keys, unsigned* __restrict__ vals) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  keys[i] = ID[i];
  vals[i] = (unsigned)i;
}
__global__ void k_dbg_cellkeys(DP p, int n, const float4* __restrict__ G, const unsigned* __restrict__ vals,
                               unsigned* __restrict__ keys) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const float4 r = G[vals[k]];
  keys[k] = cell_key(p, r.x, r.y, r.z);
}
__global__ void k_dbg_gather(int n, const unsigned* __restrict__ vals, const float4* __restrict__ G,
                             const unsigned* __restrict__ ID, float4* __restrict__ Gout, unsigned* __restrict__ IDout) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const unsigned v = vals[k];
  Gout[k] = G[v];
  IDout[k] = ID[v];
}

__global__ void k_dbg_ranges(int ncell, const int* __restrict__ lb, int* cs, int* ce) {
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  int s = lb[c], e = lb[c + 1];
  if (s == e) s = e = 0;
  cs[c] = s;
  ce[c] = e;
}

// sph_debug_step_lists: the neighbour lists the pair passes and the second wall pass actually READ
// (NL / NLW per fluid particle, NLF per wall particle), mapped to caller ids, for a host-side check
// against the oracle's float32 contract.  mode 0: cnt[caller id] = entries; mode 1: ids at off[caller id]
// (order of the lists: not sorted; the self entry of a fluid row is included).
__global__ void __launch_bounds__(256)
k_list_export(int n, int mode, const unsigned* __restrict__ IDrow,
              const uint4* __restrict__ L1, const int* __restrict__ C1, int cap1, const unsigned* __restrict__ ID1,
              const uint4* __restrict__ L2, const int* __restrict__ C2, int cap2, const unsigned* __restrict__ ID2,
              int* __restrict__ cnt, const long long* __restrict__ off, int* __restrict__ ids, long long cap) {
  const int s = blockIdx.x * 256 + threadIdx.x;
  if (s >= n) return;
  const unsigned me = IDrow[s];
  const int n1 = C1[s], n2 = L2 ? C2[s] : 0;
  if (!mode) { cnt[me] = n1 + n2; return; }
  long long o = off[me];
  const unsigned* c1 = reinterpret_cast<const unsigned*>(L1 + (size_t)(s >> 5) * (cap1 >> 2) * 32 + (s & 31));
  for (int k = 0; k < n1; ++k, ++o)
    if (o < cap) ids[o] = (int)ID1[c1[(size_t)(k >> 2) * 128 + (k & 3)]];
  if (n2) {
    const unsigned* c2 = reinterpret_cast<const unsigned*>(L2 + (size_t)(s >> 5) * (cap2 >> 2) * 32 + (s & 31));
    for (int k = 0; k < n2; ++k, ++o)
      if (o < cap) ids[o] = (int)ID2[c2[(size_t)(k >> 2) * 128 + (k & 3)]];
  }
}

// sph_debug_fma_peak: register-resident FP32 FMA loop (8 independent chains per thread, no memory
// traffic): the measured non-tensor FP32 peak that bench.py uses as the roofline denominator.
__global__ void __launch_bounds__(256)
k_fma_peak(float* __restrict__ out, int iters, float a, float b) {
  float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
      x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
    }
  }
  const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 12345.678f) out[0] = s;  // keeps the chains alive without a store in the common case
}

// sph_debug_gather_floor: the list walk of the pair passes (walk_l: one coalesced 16-byte list load, four 256-bit record
// gathers) with an empty pair body (every word of the record enters one XOR / ADD, nothing else), in the passes'
// launch configuration: what the passes' memory requests alone cost on this device, i.e. the roofline of the gather
// form.  MODE selects which record each lane asks for:
//   0  its own list entry (exactly the passes' requests),
//   1  the entry of the even lane of its lane pair   (what a list merged per lane pair would request),
//   2  the entry of the first lane of its quad       (a list merged per quad: 4 adjacent lanes, one record),
//   3  32 consecutive records from lane 0's entry on (the coalesced optimum: 8 lines, 1 KiB per request).
// HEAVY: a synthetic pair body of `fma` dependent-chain FFMAs per record (4 chains) on top of the XOR / ADD, to see how
// a pass with that much arithmetic per pair follows a cheaper walk (the real bodies issue 66-82 instructions per pair).
template <int MODE, bool HEAVY>
struct GatherBody {
  const XB* __restrict__ R;
  unsigned last, acc;
  int lane, fma;
  __device__ __forceinline__ XB load(unsigned j) const {
    if (MODE == 1) j = __shfl_sync(FULL, j, lane & ~1);
    if (MODE == 2) j = __shfl_sync(FULL, j, lane & ~3);
    if (MODE == 3) j = (__shfl_sync(FULL, j, 0) & ~31u) + (unsigned)lane;
    return ldg256(R + min(j, last));  // MODE > 0 also reads the slots behind a lane's own count: clamped
  }
  __device__ __forceinline__ void apply(const XB& r) {
    acc += (r.x.x ^ r.x.y) + (r.x.z ^ r.x.w) + (__float_as_uint(r.b.x) ^ __float_as_uint(r.b.y)) +
           (__float_as_uint(r.b.z) ^ __float_as_uint(r.b.w));
    if (HEAVY) {
      float a = r.b.x, b = r.b.y, c = r.b.z, d = r.b.w;
#pragma unroll 4
      for (int u = 0; u < fma; u += 4) { a = fmaf(a, 1.0001f, b); b = fmaf(b, 0.9999f, c); c = fmaf(c, 1.0002f, d); d = fmaf(d, 0.9998f, a); }
      acc += __float_as_uint((a + b) + (c + d));
    }
  }
};
template <int MODE, bool HEAVY>
__global__ void __launch_bounds__(PB, SPH_MINB)
k_gather_walk(const int nf, const XB* __restrict__ R, const uint4* __restrict__ NL, const int* __restrict__ NC,
              const int caps, unsigned* __restrict__ out, const int fma) {
  const int i0 = blockIdx.x * PB + threadIdx.x;
  const int lane = threadIdx.x & 31;
  GatherBody<MODE, HEAVY> body{R, (unsigned)(nf - 1), 0u, lane, fma};
  // MODE > 0 shuffles inside the loop, so every lane runs to the warp's largest count (32 active lanes, not ~30)
  const int cnt = i0 < nf ? NC[i0] : 0;
  walk_l(NL + (size_t)(i0 >> 5) * (caps >> 2) * 32 + lane, MODE ? __reduce_max_sync(FULL, cnt) : cnt, body);
  if (body.acc == 0x9e3779b9u) out[0] = body.acc;  // keeps the gathers alive without a store in the common case
}
// warp-wide gather requests of one list walk: sum over the warps of the largest count in the warp
__global__ void k_gather_requests(const int nf, const int* __restrict__ NC, unsigned long long* __restrict__ tot) {
  const int i0 = blockIdx.x * 256 + threadIdx.x;
  const int m = __reduce_max_sync(FULL, i0 < nf ? NC[i0] : 0);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(tot, (unsigned long long)m);
}

// Mode 4 of sph_debug_gather_floor: the same walk (mode 0) with the chunks (PB consecutive particles = one block's
// work) taken in an SM-AFFINE order: chunks are sorted by the blob of cells their first particle lies in (L cells along
// x by ry x rz cell rows), every SM owns a contiguous part of that order, and persistent blocks pop consecutive chunks
// from the counter of the SM they run on (%smid), so that the blocks sharing an L1 walk one neighbourhood together.
// Measures how much of the walk's time is L1 misses caused by the plain chunk = blockIdx.x mapping.
__global__ void k_chunk_keys(const DP p, const int nf, const unsigned* __restrict__ K, const int M, const int L,
                             const int ry, const int rz, unsigned* __restrict__ key, unsigned* __restrict__ val) {
  const int c = blockIdx.x * 256 + threadIdx.x;
  if (c >= M) return;
  int cx, cy, cz;
  cell_of_key(p, K[min(c * PB, nf - 1)] >> p.sub_bits, cx, cy, cz);
  const int nbx = (p.nx + L - 1) / L, nby = (p.ny + ry - 1) / ry;
  const int bx = cx / L, by = cy / ry, bz = cz / rz;
  key[c] = ((unsigned)((bz * nby + by) * nbx + bx) << 10) | ((unsigned)(cz - bz * rz) << 8) | ((unsigned)(cy - by * ry) << 6) |
           (unsigned)min(cx - bx * L, 63);
  val[c] = (unsigned)c;
}
template <bool HEAVY>
__global__ void __launch_bounds__(PB, SPH_MINB)
k_gather_walk_affine(const int nf, const XB* __restrict__ R, const uint4* __restrict__ NL, const int* __restrict__ NC,
                     const int caps, unsigned* __restrict__ out, const unsigned* __restrict__ CO, const int M,
                     unsigned* __restrict__ q, const int nq, const int fma) {
  __shared__ int chunk_s;
  unsigned smid;
  asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
  const int own = (int)(smid % (unsigned)nq), per = (M + nq - 1) / nq;
  const int lane = threadIdx.x & 31;
  GatherBody<0, HEAVY> body{R, (unsigned)(nf - 1), 0u, lane, fma};
  int cur = own;
#pragma unroll 1
  for (;;) {
    if (threadIdx.x < 32) {
      int ch = -1;
      for (;;) {
        int k = 0;
        if (lane == 0) k = (int)atomicAdd(q + cur, 1u);
        k = __shfl_sync(FULL, k, 0);
        const int pos = cur * per + k;
        if (k < per && pos < M) { ch = (int)CO[pos]; break; }
        // this queue is empty: the first one behind this SM's own that still holds chunks (32 queues per look)
        int found = -1;
        for (int t = 0; t < nq && found < 0; t += 32) {
          const int o = t + lane;
          int s = own + 1 + o;
          if (s >= nq) s -= nq;
          bool has = false;
          if (o < nq) has = (int)*(volatile unsigned*)(q + s) < min(per, M - s * per);
          const unsigned b = __ballot_sync(FULL, has);
          if (b) found = __shfl_sync(FULL, s, __ffs(b) - 1);
        }
        if (found < 0) break;
        cur = found;
      }
      if (lane == 0) chunk_s = ch;
    }
    __syncthreads();
    const int chunk = chunk_s;
    __syncthreads();
    if (chunk < 0) break;
    const int i0 = chunk * PB + threadIdx.x;
    walk_l(NL + (size_t)(i0 >> 5) * (caps >> 2) * 32 + lane, i0 < nf ? NC[i0] : 0, body);
  }
  if (body.acc == 0x9e3779b9u) out[0] = body.acc;
}

// sph_debug_gather_patterns: what a warp-wide gather of 32-byte records (one LDG.E.ENL2.256 per lane) costs in the L1
// as a function of the address pattern, records resident in L1 (a window of 512 records = 16 KiB per block, 8 blocks
// per SM).  PAT: 0 32 random records; 1 32 consecutive records (8 lines); 2 16 random lines, adjacent lane pairs in
// one line; 3 8 random lines, each read by 4 adjacent lanes (4 records); 4 8 records, each read by 4 adjacent lanes;
// 5 one record for all lanes; 6 32 different lines, one record of each; 7 32 random records of a 64-record window (16
// lines: lanes that share a line are not neighbours in the warp).  Addresses come from an integer hash of
// (block, warp, iteration, lane group), a handful of ALU instructions per request.
__device__ __forceinline__ unsigned mix32(unsigned x) {
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return x;
}
template <int PAT>
__global__ void __launch_bounds__(PB, SPH_MINB)
k_gather_patterns(const XB* __restrict__ R, const int iters, unsigned* __restrict__ out) {
  constexpr unsigned W = 512, NL = W / 4;
  const XB* base = R + (size_t)blockIdx.x * W;
  const unsigned lane = threadIdx.x & 31, seed = (blockIdx.x * 4u + (threadIdx.x >> 5)) * 0x9e3779b9u;
  unsigned acc = 0;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
    XB r[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const unsigned q = seed + (unsigned)(it * 4 + u) * 0x85ebca6bu;
      unsigned idx;
      if (PAT == 0) idx = mix32(q + lane) % W;
      else if (PAT == 1) idx = ((mix32(q) % (NL - 8)) << 2) + lane;
      else if (PAT == 2) { const unsigned h = mix32(q + (lane >> 1)); idx = ((h % NL) << 2) + ((h >> 20) & 2u) + (lane & 1u); }
      else if (PAT == 3) idx = ((mix32(q + (lane >> 2)) % NL) << 2) + (lane & 3u);
      else if (PAT == 4) idx = ((mix32(q + (lane >> 2)) % NL) << 2) + 1u;
      else if (PAT == 5) idx = mix32(q) % W;
      else if (PAT == 6) idx = (((mix32(q) + lane) % NL) << 2) + (mix32(q + lane) & 3u);
      else idx = ((mix32(q) % (NL - 16)) << 2) + (mix32(q + lane) & 63u);
      r[u] = ldg256(base + idx);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
      acc += (r[u].x.x ^ r[u].x.y) + (r[u].x.z ^ r[u].x.w) + (__float_as_uint(r[u].b.x) ^ __float_as_uint(r[u].b.y)) +
             (__float_as_uint(r[u].b.z) ^ __float_as_uint(r[u].b.w));
  }
  if (acc == 0x9e3779b9u) out[0] = acc;
}
