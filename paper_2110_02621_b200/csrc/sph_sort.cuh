// sph_sort.cuh — device radix sort of (cell id, index) and cell lower bounds.  Included by sph.cu.
#pragma once
// ------------------------------------------------------------------------------------------
// Device radix sort (stable LSD) of (cell id, index).  Digits of RB = 8 or 9 bits (ND = 256 / 512
// bins), whichever needs fewer passes for the grid's cell count: 17-18 bit cell ids (cfg1, cfg4 up
// to 4 M) sort in 2 passes of 9 bits instead of 3 of 8; a pass is 3 dependent launches and at
// these sizes latency-bound.  BASELINE.json north_star
// "cell hash, device radix sort"; the paper only names the step.
// Per pass: tile histograms (+ per-digit totals by atomics) -> scan -> stable scatter with warp match
// ranking: 3 dependent launches.
// ------------------------------------------------------------------------------------------
// Keys per thread: 16 (tile of 4096) for large inputs; 4 (tile of 1024) below RS_SMALL_N keys, where
// 4096-key tiles leave most SMs idle and every block runs a serial chain of 16 match rounds.
constexpr int RS_THREADS = 256, RS_WARPS = 8, RS_SMALL_N = 2 << 20;
inline int rs_items(size_t n) { return n < (size_t)RS_SMALL_N ? 4 : 16; }

template <int ND, int RS_ITEMS>
__global__ void __launch_bounds__(RS_THREADS)
k_radix_hist(const unsigned* __restrict__ keys, int n, int shift, unsigned* __restrict__ hist,
             int nblk, unsigned* __restrict__ rowsum) {
  __shared__ unsigned h[ND];
  for (int d = threadIdx.x; d < ND; d += RS_THREADS) h[d] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  constexpr int RS_TILE = RS_THREADS * RS_ITEMS;
  const int base = blockIdx.x * RS_TILE;
#pragma unroll 4
  for (int it = 0; it < RS_ITEMS; ++it) {
    int idx = base + it * RS_THREADS + threadIdx.x;
    bool ok = idx < n;
    unsigned d = ok ? ((keys[idx] >> shift) & (unsigned)(ND - 1)) : (unsigned)ND;
    unsigned peers = __match_any_sync(FULL, d);
    if (ok && lane == __ffs(peers) - 1) atomicAdd(&h[d], (unsigned)__popc(peers));
  }
  __syncthreads();
  for (int d = threadIdx.x; d < ND; d += RS_THREADS) {
    hist[d * nblk + blockIdx.x] = h[d];
    if (h[d]) atomicAdd(&rowsum[d], h[d]);  // per-digit totals (zeroed by the previous scatter): no separate row-sum launch
  }
}

// Exclusive scan of hist in (digit-major, block-minor) order, in place.
__global__ void __launch_bounds__(256)
k_scan_apply(unsigned* __restrict__ hist, int nblk, const unsigned* __restrict__ rowsum) {
  __shared__ unsigned sm[8];
  __shared__ unsigned carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // base = sum of rowsum[d'] for d' < digit
  unsigned b = 0u;
  for (int t = threadIdx.x; t < (int)blockIdx.x; t += 256) b += rowsum[t];
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

template <int ND, int RS_ITEMS>
__global__ void __launch_bounds__(RS_THREADS)
k_radix_scatter(const unsigned* __restrict__ keys, const unsigned* __restrict__ vals, int n, int shift,
                const unsigned* __restrict__ hist, int nblk, unsigned* __restrict__ keys_out,
                unsigned* __restrict__ vals_out, unsigned* __restrict__ rowsum) {
  if (blockIdx.x == 0)  // the scan has consumed the digit totals: clear them for the next pass's histogram
    for (int d = threadIdx.x; d < ND; d += RS_THREADS) rowsum[d] = 0;
  __shared__ unsigned wc[RS_WARPS][ND];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < RS_WARPS * ND; i += RS_THREADS) (&wc[0][0])[i] = 0;
  __syncthreads();
  constexpr int RS_TILE = RS_THREADS * RS_ITEMS;
  const int base = blockIdx.x * RS_TILE + wid * (RS_ITEMS * 32);
  unsigned k[RS_ITEMS], rank[RS_ITEMS];
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int it = 0; it < RS_ITEMS; ++it) {
    int idx = base + it * 32 + lane;  // warp-contiguous order keeps the sort stable
    bool ok = idx < n;
    k[it] = ok ? keys[idx] : 0xffffffffu;
    unsigned d = ok ? ((k[it] >> shift) & (unsigned)(ND - 1)) : (unsigned)ND;
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
  for (int d = threadIdx.x; d < ND; d += RS_THREADS) {  // exclusive prefix over warps per digit, plus the scanned global base of this tile
    unsigned run = hist[d * nblk + blockIdx.x];
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
      unsigned d = (k[it] >> shift) & (unsigned)(ND - 1);
      unsigned dst = wc[wid][d] + rank[it];
      keys_out[dst] = k[it];
      vals_out[dst] = vals[idx];
    }
  }
}

// lb[c] = number of sorted particles with key < c, c = 0..ncell (dense lower bounds: the three
// cells of an x-row of the stencil are one contiguous range [lb[c0], lb[c1+1])).  One thread per
// cell, binary search in the sorted keys (the tank may be mostly dry: no serial gap filling).
__global__ void __launch_bounds__(256)
k_cell_bounds(const unsigned* __restrict__ keys, int n, int ncell, int* __restrict__ lb, int sub_bits) {
  const int c = blockIdx.x * 256 + threadIdx.x;
  if (c > ncell) return;
  int lo = 0, hi = n;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if ((keys[mid] >> sub_bits) < (unsigned)c) lo = mid + 1; else hi = mid;
  }
  lb[c] = lo;
}
