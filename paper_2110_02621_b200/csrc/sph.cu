// paper_2110_02621_b200/csrc/sph.cu — libsph: the per-time-step SPH pipeline of
// arXiv 2110.02621 as hand-written CUDA for B200 (sm_100a) behind the C ABI of include/sph.h.
//
// Citations: PAPER.md:<line> / equation; readings Axx are listed in DESIGN.md §3.
// Nothing here is shared with oracle/ (the CPU checker); there is no CPU fallback.
//
// Kernels: sph_sort.cuh (radix sort, cell bounds), sph_aux.cuh (load, dt, predictor, reorder,
// normals), sph_pair.cuh (wall extrapolation, pass A, pass B), sph_debug.cuh (output, stats,
// integer-contract debug paths).  This file is the host side and the extern "C" entry points.
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <string>
#include <vector>

#include "sph.h"

namespace {
#include "sph_common.cuh"
#include "sph_sort.cuh"
#include "sph_aux.cuh"
#include "sph_pair.cuh"
#include "sph_debug.cuh"
#include "sph_probe.cuh"
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
  float sigma0 = 0.f;
  // fluid (cell-sorted): master position, filter image, (v, rho - rho0) x3, acceleration
  // R0: records after the reorder, R1: after pass A (density updated); TB: (v, rho - rho0) after pass B
  XB *R0 = nullptr, *R1 = nullptr;
  uint4* TX = nullptr;
  float4 *A = nullptr, *TB = nullptr, *ACC = nullptr;
  float *SIG = nullptr, *DRHO = nullptr;
  uint4* NL = nullptr;     // neighbour lists in groups of 4, per warp: [npad / 32][caps / 4][32] (caps % 4 == 0)
  int* NC = nullptr;       // neighbours per fluid particle
  int caps = 0;
  uint4* NLW = nullptr;    // fluid-wall neighbour lists, same layout with capsw slots
  int* NCW = nullptr;
  int capsw = 0;
  uint4* NLF = nullptr;    // wall-fluid neighbour lists (per wall particle, capsw slots), written by the first wall pass of a step
  int* NCF = nullptr;
  size_t npad = 0;
  unsigned *ID0 = nullptr, *ID1 = nullptr, *IDcur = nullptr, *IDnext = nullptr;
  unsigned *keyA = nullptr, *valA = nullptr, *keyB = nullptr, *valB = nullptr, *hist = nullptr,
           *rowsum = nullptr;
  const unsigned* K = nullptr;  // sorted cell keys of the current fluid order (one of keyA / keyB)
  int *lbF = nullptr, *lbW = nullptr;
  // wall (static)
  XB* WR = nullptr;
  float4 *WA = nullptr, *WN = nullptr, *WG = nullptr;
  unsigned *WK = nullptr, *WID = nullptr;
  unsigned char* wnear = nullptr;
  SS* S = nullptr;
  double* dt_seq = nullptr;
  int64_t dt_seq_cap = 0;
  StatAcc* stat = nullptr;
  // NEXT-1 (moving walls): wall positions and caller ids in set-up order, sort buffers of the per-step re-sort
  int moving = 0;
  uint4* WX0 = nullptr;
  float4* WN0 = nullptr;   // wall normals in set-up order (translation-invariant)
  unsigned *WID0 = nullptr, *WkeyA = nullptr, *WkeyB = nullptr, *WvalA = nullptr, *WvalB = nullptr;
  // the re-sort runs on its own stream beside the fluid's predict / sort / reorder (it depends on k_dt only):
  // own scratch, fork / join events (captured into the step graph as a parallel branch)
  uint4* WTX = nullptr;
  float4* WTB = nullptr;
  unsigned *Whist = nullptr, *Wrowsum = nullptr;
  cudaStream_t wstream = nullptr;
  cudaEvent_t evFork = nullptr, evJoin = nullptr;
  std::map<void*, size_t> cap_bytes;  // dalloc: capacity of the buffer behind each pointer member
  // DEVICE staging of the host-pointer entry points (caller order), kept across calls
  float *stage_pos = nullptr, *stage_vel = nullptr, *stage_rho = nullptr;
  int32_t* stage_tag = nullptr;
  float* stage_out = nullptr;
  // device scratch of the classification in sph_set_particles (stable sort of (class, caller index))
  unsigned *clsKa = nullptr, *clsVa = nullptr, *clsKb = nullptr, *clsVb = nullptr, *clsHist = nullptr, *clsRow = nullptr;
  unsigned long long* clsCnt = nullptr;
  // PINNED host bounce buffer of the host-pointer entry points: pageable caller memory goes through it in two
  // halves (the copy of one half overlaps the memcpy of the other), so their speed does not depend on the
  // caller pinning its arrays; memory that is already pinned or registered is copied directly
  char* pin = nullptr;
  size_t pin_bytes = 0;
  cudaEvent_t pin_ev[2] = {nullptr, nullptr};
  // one step captured as a CUDA graph (launch-bound small configurations); rebuilt after sph_set_particles
  cudaGraphExec_t gexec = nullptr;
  cudaStream_t cap_stream = nullptr, cap_stream2 = nullptr;
  int64_t graph_launches = 0;  // kernel launches of a captured step that keeps its lists
  int64_t body_launches = 0;   // ... of its rebuild branch
  int64_t direct_rebuilds = 0;          // rebuild branches issued by plain launches (already in `launches`)
  int64_t graph_rebuilds_counted = 0;   // rebuild branches taken inside graph replays already added to `launches`
  int cell_bits = 1;           // significant bits of a cell id of the step's grid
  DP dpC;                      // the contract grid of reading A24 (cell edge 2h(1 + 2^-10)); = dp's grid when skin = 0
  int64_t ncellC = 0;
  uint4* WXB = nullptr;        // moving walls with kept lists: set-up positions in the current wall order
  // scratch of contract_view (debug entry points with skin > 0)
  unsigned *dKa = nullptr, *dVa = nullptr, *dKb = nullptr, *dVb = nullptr, *dID = nullptr, *dWID = nullptr;
  float4 *dG = nullptr, *dWG = nullptr;
  int *dlbF = nullptr, *dlbW = nullptr;
  bool ev_rebuilt[64] = {};
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

// Pair kernels are instantiated for DIM in {2,3} x MULTI x a third flag: EXACT (filter form) for the list
// builds, SUBQ (residuals in sigma) for pass A; pass B and the wall passes ignore it.
#define SEL3(c, third) (((c)->prm.dim == 3 ? 4 : 0) | ((c)->multi ? 2 : 0) | ((third) ? 1 : 0))
#define PAIR_DISPATCH(KERN, sel, grid, st, ...)                                       \
  switch (sel) {                                                                      \
    case 0: LAUNCH((KERN<2, false, false>), grid, PB, st, __VA_ARGS__); break;        \
    case 1: LAUNCH((KERN<2, false, true>), grid, PB, st, __VA_ARGS__); break;         \
    case 2: LAUNCH((KERN<2, true, false>), grid, PB, st, __VA_ARGS__); break;         \
    case 3: LAUNCH((KERN<2, true, true>), grid, PB, st, __VA_ARGS__); break;          \
    case 4: LAUNCH((KERN<3, false, false>), grid, PB, st, __VA_ARGS__); break;        \
    case 5: LAUNCH((KERN<3, false, true>), grid, PB, st, __VA_ARGS__); break;         \
    case 6: LAUNCH((KERN<3, true, false>), grid, PB, st, __VA_ARGS__); break;         \
    default: LAUNCH((KERN<3, true, true>), grid, PB, st, __VA_ARGS__); break;         \
  }
// list builds: DIM x EXACT
#define BUILD_DISPATCH(KERN, grid, st, ...)                                           \
  switch (((c)->prm.dim == 3 ? 2 : 0) | ((c)->dp.exact_filter ? 1 : 0)) {             \
    case 0: LAUNCH((KERN<2, false>), grid, PB, st, __VA_ARGS__); break;               \
    case 1: LAUNCH((KERN<2, true>), grid, PB, st, __VA_ARGS__); break;                \
    case 2: LAUNCH((KERN<3, false>), grid, PB, st, __VA_ARGS__); break;               \
    default: LAUNCH((KERN<3, true>), grid, PB, st, __VA_ARGS__); break;               \
  }

inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// Device buffer of at least `count` elements; a buffer that is already large enough is kept (a second
// sph_set_particles of the same size allocates nothing: cudaMalloc / cudaFree cost more than the set-up kernels).
template <typename T>
int dalloc(sph_ctx* c, T** p, size_t count) {
  if (count == 0) count = 1;
  const size_t bytes = count * sizeof(T);
  auto it = c->cap_bytes.find((void*)p);
  if (*p && it != c->cap_bytes.end() && it->second >= bytes) return SPH_OK;
  if (*p) { cudaFree(*p); *p = nullptr; }
  c->cap_bytes.erase((void*)p);
  CK(cudaMalloc((void**)p, bytes));
  c->cap_bytes[(void*)p] = bytes;
  return SPH_OK;
}

void free_all(sph_ctx* c) {
  void* ptrs[] = {c->R0, c->R1, c->TX, c->A, c->TB, c->ACC, c->SIG, c->DRHO, c->NL, c->NC, c->NLW, c->NCW, c->NLF, c->NCF, c->ID0, c->ID1,
                  c->keyA, c->valA, c->keyB, c->valB, c->hist, c->rowsum, c->lbF, c->lbW, c->WR,
                  c->WA, c->WN, c->WG, c->WK, c->WID, c->wnear, c->S, c->dt_seq, c->stat,
                  c->stage_pos, c->stage_vel, c->stage_rho, c->stage_tag, c->stage_out, c->clsKa, c->clsVa, c->clsKb, c->clsVb, c->clsHist, c->clsRow, c->clsCnt,
                  c->WX0, c->WXB, c->WN0, c->WID0, c->dKa, c->dVa, c->dKb, c->dVb, c->dID, c->dWID, c->dG, c->dWG, c->dlbF, c->dlbW, c->WkeyA, c->WkeyB, c->WvalA, c->WvalB,
                  c->WTX, c->WTB, c->Whist, c->Wrowsum};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (auto e : c->ev) cudaEventDestroy(e);
  if (c->gexec) cudaGraphExecDestroy(c->gexec);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  if (c->cap_stream2) cudaStreamDestroy(c->cap_stream2);
  if (c->evFork) cudaEventDestroy(c->evFork);
  if (c->evJoin) cudaEventDestroy(c->evJoin);
  if (c->wstream) cudaStreamDestroy(c->wstream);
  if (c->pin) cudaFreeHost(c->pin);
  for (int k = 0; k < 2; ++k) if (c->pin_ev[k]) cudaEventDestroy(c->pin_ev[k]);
}

// Digits of 9 bits when that saves a pass over 8-bit digits (sph_sort.cuh).
inline void radix_plan(int bits, int* digit_bits, int* passes) {
  *digit_bits = (bits + 8) / 9 < (bits + 7) / 8 ? 9 : 8;
  *passes = (bits + *digit_bits - 1) / *digit_bits;
}
inline int bits_for(int64_t count) {
  int bits = 1;
  while ((1ll << bits) < count) ++bits;
  return bits;
}

// Stable radix sort of (keys, vals) on keys of `bits` significant bits; result pointers returned in *ko, *vo.
int radix_sort(sph_ctx* c, cudaStream_t st, int n, int bits, unsigned* kA, unsigned* vA, unsigned* kB, unsigned* vB,
               unsigned** ko, unsigned** vo, unsigned* hist = nullptr, unsigned* rowsum = nullptr) {
  if (!hist) { hist = c->hist; rowsum = c->rowsum; }
  unsigned *ki = kA, *vi = vA, *kt = kB, *vt = vB;
  int dbits, passes;
  radix_plan(bits, &dbits, &passes);
  if (n > 0) {
    const int items = rs_items((size_t)n), nblk = cdiv(n, RS_THREADS * items);
    for (int pass = 0; pass < passes; ++pass) {
      int shift = dbits * pass;
#define RS_PASS(ND, IT)                                                                                   \
  do {                                                                                                    \
    LAUNCH((k_radix_hist<ND, IT>), nblk, RS_THREADS, st, ki, n, shift, hist, nblk, rowsum);               \
    LAUNCH(k_scan_apply, ND, 256, st, hist, nblk, rowsum);                                                \
    LAUNCH((k_radix_scatter<ND, IT>), nblk, RS_THREADS, st, ki, vi, n, shift, hist, nblk, kt, vt, rowsum); \
  } while (0)
      if (dbits == 9) { if (items == 4) RS_PASS(512, 4); else RS_PASS(512, 16); }
      else { if (items == 4) RS_PASS(256, 4); else RS_PASS(256, 16); }
#undef RS_PASS
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
  bool on;
  Prof(sph_ctx* c_, cudaStream_t s) : c(c_), st(s) {
    on = c->prof && c->ev_steps < sph_ctx::EV_MAX_STEPS;
  }
  // marks: 0 start, 1 predict, 2 sort, 3 reorder, 4 list build (wall + fluid), 5 wall 1, 6 pass A, 7 wall 2, 8 pass B
  void mark(int slot) {
    if (!on) return;
    cudaEventRecord(c->ev[c->ev_steps * sph_ctx::EV_PER_STEP + slot], st);
  }
  void done(bool rebuilt) {
    if (!on) return;
    c->ev_rebuilt[c->ev_steps] = rebuilt;
    c->ev_steps++;
  }
};

// Eq. 2.12 for every wall particle from its wall-fluid list (R = the fluid records the pressures are read from)
void launch_wall(sph_ctx* c, cudaStream_t st, bool with_vel, const XB* R) {
  if (c->nw == 0 || c->nf == 0) return;
  const int grid = cdiv(c->nw, PB), nw = (int)c->nw;
  if (with_vel) {
    PAIR_DISPATCH(k_wall, SEL3(c, 1), grid, st, c->dp, c->S, nw, c->WR, R, c->NLF, c->NCF, c->capsw);
  } else {
    PAIR_DISPATCH(k_wall, SEL3(c, 0), grid, st, c->dp, c->S, nw, c->WR, R, c->NLF, c->NCF, c->capsw);
  }
}

// NEXT-1 (moving walls): the walls at their positions of t^{n+1}, re-sorted into the cell grid (the
// same kernels as the set-up, on scratch of their own: `st` is the wall stream, which runs beside the
// fluid's sort / reorder inside the rebuild branch).
int wall_rebuild(sph_ctx* c, cudaStream_t st) {
  const int nw = (int)c->nw;
  if (nw == 0) return SPH_OK;
  LAUNCH(k_wall_shift, cdiv(nw, 256), 256, st, c->dp, c->S, nw, c->WX0, c->WTX, c->WTB, c->WkeyA, c->WvalA);
  unsigned *ks, *vs;
  int rc = radix_sort(c, st, nw, c->cell_bits, c->WkeyA, c->WvalA, c->WkeyB, c->WvalB, &ks, &vs, c->Whist, c->Wrowsum);
  if (rc) return rc;
  // gather + wall cell lower bounds in one launch, as for the fluid
  LAUNCH(k_reorder, std::max(cdiv(nw, 256), cdiv(c->ncell + 1, 256)), 256, st, c->dp, nw, vs, c->WTX, c->WTB, c->WID0,
         c->WR, c->WA, c->WID, ks, (int)c->ncell, c->lbW);
  CK(cudaMemcpyAsync(c->WK, ks, sizeof(unsigned) * nw, cudaMemcpyDeviceToDevice, st));
  LAUNCH(k_gather4, cdiv(nw, 256), 256, st, nw, vs, c->WN0, c->WN);  // normals: translation-invariant
  LAUNCH(k_gatherx, cdiv(nw, 256), 256, st, nw, vs, c->WX0, c->WXB); // set-up positions in the new order (k_wall_move)
  LAUNCH(k_wnear, cdiv(c->ncell, 256), 256, st, c->dp, (int)c->ncell, c->lbW, c->wnear);
  return SPH_OK;
}

// The rebuild branch of a step (and the set-up): radix sort of the cell keys, gather into cell order with the
// cell bounds, wall re-sort (moving walls, on the wall stream beside the fluid's), wall-fluid lists, fluid lists.
// Input: TX / TB (positions, (v, rho - rho0)) and keyA / valA in the current order; output: R0, A, IDcur, lbF,
// NL / NLW / NLF in the new order.
int rebuild_body(sph_ctx* c, cudaStream_t st, int init, Prof& pf) {
  const int nf = (int)c->nf;
  const bool wall_branch = c->moving && !init && c->nw > 0;
  if (wall_branch) {
    CK(cudaEventRecord(c->evFork, st));
    CK(cudaStreamWaitEvent(c->wstream, c->evFork, 0));
    int rcw = wall_rebuild(c, c->wstream);
    if (rcw) return rcw;
    CK(cudaEventRecord(c->evJoin, c->wstream));
  }
  unsigned *ks, *vs;
  int rc = radix_sort(c, st, nf, c->cell_bits, c->keyA, c->valA, c->keyB, c->valB, &ks, &vs);
  if (rc) return rc;
  c->K = ks;
  pf.mark(2);  // end sort
  if (nf > 0) {
    // no pointer ping-pong: every rebuild issues the same launches with the same arguments (CUDA graph);
    // k_build copies IDnext back to IDcur
    LAUNCH(k_reorder, std::max(cdiv(nf, 256), cdiv(c->ncell + 1, 256)), 256, st, c->dp, nf, vs, c->TX, c->TB, c->IDcur,
           c->R0, c->A, c->IDnext, ks, (int)c->ncell, c->lbF);
  } else {
    LAUNCH(k_cell_bounds, cdiv(c->ncell + 1, 256), 256, st, ks, nf, (int)c->ncell, c->lbF, c->dp.sub_bits);
  }
  if (wall_branch) CK(cudaStreamWaitEvent(st, c->evJoin, 0));
  pf.mark(3);  // end reorder
  if (c->nw > 0 && nf > 0)
    BUILD_DISPATCH(k_wall_build, cdiv(c->nw, PB), st, c->dp, c->S, (int)c->nw, c->WA, c->WK, c->A, c->lbF, c->NLF,
                   c->NCF, c->capsw);
  if (nf > 0)
    BUILD_DISPATCH(k_build, cdiv(nf, PB), st, c->dp, c->S, nf, c->A, c->K, c->lbF, c->NL, c->NC, c->caps, c->WA,
                   c->lbW, c->wnear, c->NLW, c->NCW, c->capsw, c->IDcur, c->IDnext);
  pf.mark(4);  // end list build
  CK(cudaGetLastError());
  return SPH_OK;
}

// The part of a step every step runs: wall pass, pass A, wall pass, pass B (R0 -> R1 -> TB, ACC).
int pass_tail(sph_ctx* c, cudaStream_t st, int init, Prof& pf) {
  const int nf = (int)c->nf;
  if (c->moving && !init && c->nw > 0 && c->dp.skin > 0.0)  // kept lists: the walls move inside their cell order
    LAUNCH(k_wall_move, cdiv(c->nw, 256), 256, st, c->dp, c->S, (int)c->nw, c->WXB, c->WR);
  launch_wall(c, st, true, c->R0);
  pf.mark(5);  // end wall 1
  if (nf > 0) {
    PAIR_DISPATCH(k_pass_a, SEL3(c, c->dp.subq), cdiv(nf, PB), st, c->dp, c->S, nf, init, c->R0, c->WR, c->R1, c->SIG,
                  c->DRHO, c->NL, c->NC, c->caps, c->NLW, c->NCW, c->capsw);
  }
  pf.mark(6);  // end pass A
  launch_wall(c, st, false, c->R1);
  pf.mark(7);  // end wall 2
  if (nf > 0) {
    PAIR_DISPATCH(k_pass_b, SEL3(c, 0), cdiv(nf, PB), st, c->dp, c->S, nf, c->R1, c->WR, c->WN, c->TB, c->ACC, c->NL,
                  c->NC, c->caps, c->NLW, c->NCW, c->capsw);
  }
  pf.mark(8);  // end pass B
  CK(cudaGetLastError());
  return SPH_OK;
}

// k_dt + k_predict: the head of a step.  cond / use_cond: the IF node of the step graph (0: plain launches).
int step_head(sph_ctx* c, cudaStream_t q, const double* seq, int s, cudaGraphConditionalHandle cond, int use_cond) {
  const int nf = (int)c->nf;
  const int dt_grid = std::max(1, std::min(cdiv(nf, 256), 148 * 4));
  LAUNCH(k_dt, dt_grid, 256, q, c->dp, c->S, nf, c->TB, seq, s);
  if (nf > 0)
    LAUNCH((k_predict<true, true>), cdiv(nf, 256), 256, q, c->dp, c->S, nf, c->R1, c->TB, c->ACC, c->SIG, c->TX, c->R0,
           c->keyA, c->valA, cond, use_cond, 1);
  CK(cudaGetLastError());
  return SPH_OK;
}

// One step as a CUDA graph: head (k_dt, k_predict) -> IF node (rebuild branch, taken when k_predict's last
// block says so through cudaGraphSetConditional) -> tail (wall, pass A, wall, pass B).
int build_step_graph(sph_ctx* c) {
  if (!c->cap_stream) CK(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
  if (!c->cap_stream2) CK(cudaStreamCreateWithFlags(&c->cap_stream2, cudaStreamNonBlocking));
  const int64_t l0 = c->launches;
  cudaGraph_t g = nullptr;
  CK(cudaGraphCreate(&g, 0));
  cudaGraphConditionalHandle cond = 0;
  const bool use_cond = c->nf > 0;
  int rc = SPH_OK;
  cudaError_t e = cudaSuccess;
  Prof pf(c, c->cap_stream);
  pf.on = false;
  do {
    if (use_cond) {
      e = cudaGraphConditionalHandleCreate(&cond, g, 0, cudaGraphCondAssignDefault);
      if (e != cudaSuccess) break;
    }
    e = cudaStreamBeginCaptureToGraph(c->cap_stream, g, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) break;
    rc = step_head(c, c->cap_stream, nullptr, 0, cond, use_cond ? 1 : 0);
    const int64_t l_head = c->launches;
    if (!rc && use_cond) {
      cudaStreamCaptureStatus cs;
      const cudaGraphNode_t* deps = nullptr;
      size_t nd = 0;
      e = cudaStreamGetCaptureInfo_v2(c->cap_stream, &cs, nullptr, nullptr, &deps, &nd);
      if (e != cudaSuccess) break;
      cudaGraphNodeParams np = {};
      np.type = cudaGraphNodeTypeConditional;
      np.conditional.handle = cond;
      np.conditional.type = cudaGraphCondTypeIf;
      np.conditional.size = 1;
      cudaGraphNode_t cn;
      e = cudaGraphAddNode(&cn, g, deps, nd, &np);
      if (e != cudaSuccess) break;
      cudaGraph_t body = np.conditional.phGraph_out[0];
      e = cudaStreamBeginCaptureToGraph(c->cap_stream2, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
      if (e != cudaSuccess) break;
      pf.st = c->cap_stream2;
      rc = rebuild_body(c, c->cap_stream2, 0, pf);
      cudaError_t e2 = cudaStreamEndCapture(c->cap_stream2, nullptr);
      c->body_launches = c->launches - l_head;
      if (e2 != cudaSuccess) { e = e2; break; }
      e = cudaStreamUpdateCaptureDependencies(c->cap_stream, &cn, 1, cudaStreamSetCaptureDependencies);
      if (e != cudaSuccess) break;
    }
    pf.st = c->cap_stream;
    if (!rc) rc = pass_tail(c, c->cap_stream, 0, pf);
  } while (0);
  cudaGraph_t gout = nullptr;
  cudaStreamCaptureStatus cst = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(c->cap_stream, &cst);
  if (cst != cudaStreamCaptureStatusNone) {
    cudaError_t e3 = cudaStreamEndCapture(c->cap_stream, &gout);
    if (e == cudaSuccess) e = e3;
  }
  c->graph_launches = c->launches - l0 - c->body_launches;  // launches of a step that keeps its lists
  c->launches = l0;
  if (rc || e != cudaSuccess) {
    cudaGraphDestroy(g);
    if (!rc) { c->err = std::string("step graph: ") + cudaGetErrorString(e); rc = SPH_ECUDA; }
    return rc;
  }
  e = cudaGraphInstantiate(&c->gexec, g, 0);
  cudaGraphDestroy(g);
  if (e != cudaSuccess) { c->gexec = nullptr; c->err = std::string("graph instantiate: ") + cudaGetErrorString(e); return SPH_ECUDA; }
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
  // Device-computed dt, no per-stage events: every step is the same launch sequence with the same
  // arguments, so it is captured once (on private streams) and replayed as a CUDA graph.
  const bool use_graph = !dt_host && !c->prof && !(c->prm.flags & SPH_FLAG_NO_GRAPH) && n_steps > 0;
  if (use_graph && !c->gexec) {
    CK(cudaStreamSynchronize(st));  // the capture streams are not ordered after st: drain st once
    int rc = build_step_graph(c);
    if (rc) return rc;
  }
  for (int s = 0; s < n_steps; ++s) {
    if (use_graph) {
      CK(cudaGraphLaunch(c->gexec, st));
      c->launches += c->graph_launches;   // + body_launches on the steps that rebuild: added from S->rebuilds at the next stats read
      continue;
    }
    // plain launches: the host reads the rebuild decision of k_predict (one 4-byte copy and a sync per step)
    Prof pf(c, st);
    pf.mark(0);
    int rc = step_head(c, st, dt_host ? c->dt_seq : nullptr, s, 0, 0);
    if (rc) return rc;
    pf.mark(1);
    int rb = 1;
    if (c->nf > 0 && c->dp.skin > 0.0) {
      CK(cudaMemcpyAsync(&rb, (char*)c->S + offsetof(SS, rebuild), sizeof(int), cudaMemcpyDeviceToHost, st));
      CK(cudaStreamSynchronize(st));
    }
    if (rb) {
      rc = rebuild_body(c, st, 0, pf);
      if (rc) return rc;
      c->direct_rebuilds++;
    } else {
      pf.mark(2); pf.mark(3); pf.mark(4);
    }
    rc = pass_tail(c, st, 0, pf);
    if (rc) return rc;
    pf.done(rb != 0);
  }
  return SPH_OK;
}

// float32 images of the current fluid positions for the contract-exact debug walks (scratch: TX)
float4* fluid_images(sph_ctx* c, cudaStream_t st) {
  float4* G = reinterpret_cast<float4*>(c->TX);
  if (c->nf) LAUNCH(k_image, cdiv(c->nf, 256), 256, st, c->dp, (int)c->nf, c->R1, G);
  return G;
}

// What the integer-contract debug entry points walk: float32 images and caller ids of the fluid and wall
// particles in the cell order of the CONTRACT grid (reading A24) at the current positions, with its cell bounds.
// skin = 0: the step's own structures (its grid is the contract grid and it is rebuilt every step).
// skin > 0: the step's grid has a larger cell edge and is only rebuilt now and then, so the contract order is
// produced on demand with the step's sort kernels on scratch of its own: a stable sort by caller id, then by
// contract cell id, i.e. the (unique) order the oracle's std::stable_sort from id order gives (reading A25).
struct View {
  DP dp;
  const float4 *G = nullptr, *WG = nullptr;
  const unsigned *ID = nullptr, *WID = nullptr;
  const int *lb = nullptr, *lbW = nullptr;
};

int contract_order(sph_ctx* c, cudaStream_t st, int n, const float4* G, const unsigned* ID, float4* Gout,
                   unsigned* IDout, int* lb) {
  const int nc = (int)c->ncellC;
  if (n == 0) {
    LAUNCH(k_cell_bounds, cdiv(nc + 1, 256), 256, st, c->dKa, 0, nc, lb, 0);
    return SPH_OK;
  }
  unsigned *ks, *vs;
  LAUNCH(k_dbg_idkeys, cdiv(n, 256), 256, st, n, ID, c->dKa, c->dVa);
  int rc = radix_sort(c, st, n, bits_for(c->n), c->dKa, c->dVa, c->dKb, c->dVb, &ks, &vs);
  if (rc) return rc;
  unsigned *k2 = ks == c->dKa ? c->dKb : c->dKa, *v2 = vs == c->dVa ? c->dVb : c->dVa;
  LAUNCH(k_dbg_cellkeys, cdiv(n, 256), 256, st, c->dpC, n, G, vs, ks);   // keys of the id-ordered sequence, in place of the ids
  rc = radix_sort(c, st, n, bits_for(c->ncellC), ks, vs, k2, v2, &ks, &vs);
  if (rc) return rc;
  LAUNCH(k_dbg_gather, cdiv(n, 256), 256, st, n, vs, G, ID, Gout, IDout);
  LAUNCH(k_cell_bounds, cdiv(nc + 1, 256), 256, st, ks, n, nc, lb, 0);
  return SPH_OK;
}

int contract_view(sph_ctx* c, cudaStream_t st, View* v) {
  const float4* G = fluid_images(c, st);
  if (c->moving && c->nw) LAUNCH(k_image, cdiv(c->nw, 256), 256, st, c->dp, (int)c->nw, c->WR, c->WG);
  v->dp = c->dpC;
  if (c->dp.skin <= 0.0) {
    v->G = G; v->ID = c->IDcur; v->lb = c->lbF; v->WG = c->WG; v->WID = c->WID; v->lbW = c->lbW;
    return SPH_OK;
  }
  const size_t cap = (size_t)std::max<int64_t>(std::max(c->nf, c->nw), 1);
  int rc = dalloc(c, &c->dKa, cap) | dalloc(c, &c->dVa, cap) | dalloc(c, &c->dKb, cap) | dalloc(c, &c->dVb, cap) |
           dalloc(c, &c->dG, (size_t)c->nf) | dalloc(c, &c->dID, (size_t)c->nf) | dalloc(c, &c->dWG, (size_t)c->nw) |
           dalloc(c, &c->dWID, (size_t)c->nw) | dalloc(c, &c->dlbF, (size_t)c->ncellC + 1) |
           dalloc(c, &c->dlbW, (size_t)c->ncellC + 1);
  if (rc) return SPH_ENOMEM;
  rc = contract_order(c, st, (int)c->nf, G, c->IDcur, c->dG, c->dID, c->dlbF);
  if (rc) return rc;
  rc = contract_order(c, st, (int)c->nw, c->WG, c->WID, c->dWG, c->dWID, c->dlbW);
  if (rc) return rc;
  v->G = c->dG; v->ID = c->dID; v->lb = c->dlbF; v->WG = c->dWG; v->WID = c->dWID; v->lbW = c->dlbW;
  return SPH_OK;
}

bool is_pinned(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeHost || a.type == cudaMemoryTypeManaged;
}

int pin_init(sph_ctx* c) {
  if (c->pin) return SPH_OK;
  const size_t bytes = (size_t)32 << 20;
  if (cudaMallocHost((void**)&c->pin, bytes) != cudaSuccess) { cudaGetLastError(); c->pin = nullptr; c->err = "pinned staging allocation failed"; return SPH_ENOMEM; }
  c->pin_bytes = bytes;
  for (int k = 0; k < 2; ++k) CK(cudaEventCreateWithFlags(&c->pin_ev[k], cudaEventDisableTiming));
  return SPH_OK;
}

// host -> device / device -> host through the pinned bounce buffer (or directly when the caller's memory is pinned)
int h2d(sph_ctx* c, void* dst, const void* src, size_t bytes, cudaStream_t st) {
  if (!bytes) return SPH_OK;
  if (is_pinned(src)) { CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st)); return SPH_OK; }
  int rc = pin_init(c);
  if (rc) return rc;
  const size_t half = c->pin_bytes / 2;
  int k = 0;
  for (size_t off = 0; off < bytes; off += half, k ^= 1) {
    const size_t m = std::min(half, bytes - off);
    CK(cudaEventSynchronize(c->pin_ev[k]));  // the previous copy out of this half is done
    memcpy(c->pin + k * half, (const char*)src + off, m);
    CK(cudaMemcpyAsync((char*)dst + off, c->pin + k * half, m, cudaMemcpyHostToDevice, st));
    CK(cudaEventRecord(c->pin_ev[k], st));
  }
  return SPH_OK;
}

int d2h(sph_ctx* c, void* dst, const void* src, size_t bytes, cudaStream_t st) {
  if (!bytes) return SPH_OK;
  if (is_pinned(dst)) { CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st)); return SPH_OK; }
  int rc = pin_init(c);
  if (rc) return rc;
  const size_t half = c->pin_bytes / 2;
  size_t pend_off[2] = {0, 0}, pend_m[2] = {0, 0};
  int k = 0;
  for (size_t off = 0; off < bytes; off += half, k ^= 1) {
    const size_t m = std::min(half, bytes - off);
    if (pend_m[k]) {  // drain the chunk that sits in this half
      CK(cudaEventSynchronize(c->pin_ev[k]));
      memcpy((char*)dst + pend_off[k], c->pin + k * half, pend_m[k]);
    }
    CK(cudaMemcpyAsync(c->pin + k * half, (const char*)src + off, m, cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(c->pin_ev[k], st));
    pend_off[k] = off; pend_m[k] = m;
  }
  for (int j = 0; j < 2; ++j, k ^= 1)
    if (pend_m[k]) {
      CK(cudaEventSynchronize(c->pin_ev[k]));
      memcpy((char*)dst + pend_off[k], c->pin + k * half, pend_m[k]);
      pend_m[k] = 0;
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
  const double h = prm->h, dp = prm->dp, rc = 2.0 * h;
  // Verlet skin: the step's lists hold every pair within 2h(1 + s) at the last build
  double skin = prm->list_skin;
  if (!(skin >= 0.0)) skin = 0.1;  // library default
  if (getenv("SPH_SKIN")) skin = atof(getenv("SPH_SKIN"));   // measurement switch (profiles/): not part of the interface
  if (!(skin >= 0.0) || skin > 0.5) { delete c; return SPH_EINVAL; }
  const double rl = rc * (1.0 + skin);  // list radius
  d.dim = prm->dim; d.n_phases = prm->n_phases;
  d.rc2 = (float)(4.0 * h * h);
  const double alpha = prm->dim == 2 ? 7.0 / (4.0 * PI * h * h) : 21.0 / (16.0 * PI * h * h * h);
  d.alpha = (float)alpha;
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
    c->sigma0 = (float)s;
    d.a_over_s0 = alpha / s;
  }
  // fixed-point frame: Q = 2^-k with 2^32 Q >= 1.5 Lmax + 16 h, domain centred in the span
  {
    double Lmax = 0, R2 = 0;
    for (int k = 0; k < prm->dim; ++k) {
      const double L = prm->domain_max[k] - prm->domain_min[k];
      Lmax = std::max(Lmax, L);
      R2 += 0.25 * L * L;
    }
    const double need = 1.5 * Lmax + 16.0 * h;
    int e = 0;
    frexp(need, &e);            // need = m 2^e, 0.5 <= m < 1  ->  2^e >= need
    d.Q = ldexp(1.0, e - 32);   // span 2^32 Q = 2^e
    for (int k = 0; k < 3; ++k) {
      if (k < prm->dim) {
        const double mid = 0.5 * (prm->domain_min[k] + prm->domain_max[k]);
        d.O[k] = d.Q * floor((mid - ldexp(1.0, e - 1)) / d.Q);
        d.C[k] = mid;
      } else {
        d.O[k] = 0.0; d.C[k] = 0.0;
      }
    }
    d.sub_per_m = 1024.0 / d.Q;
    d.Qs = d.Q / 1024.0;
    // pair unit Qp = Q / 2^mbits (sph_common.cuh "fixed-point master positions"): the largest mbits <= 10 for which
    // 2.5 list radii — more than any two particles of one stencil are apart along an axis — stay below 2^30 Qp, so
    // that a wrapping 32-bit subtraction is their exact separation and the 64-bit integer r^2 cannot overflow
    d.mbits = 0;
    while (d.mbits < 10 && 2.5 * rl / (d.Q / (double)(2 << d.mbits)) < 1073741824.0) ++d.mbits;
    if (getenv("SPH_MBITS")) d.mbits = std::min(d.mbits, std::max(0, atoi(getenv("SPH_MBITS"))));   // measurement switch
    d.lobits = 10 - d.mbits;
    d.Qp = d.Q / (double)(1 << d.mbits);
    d.sub_scale = (float)(1 << d.lobits); d.sub_half_inv = 0.5f / (float)(1 << d.lobits);
    d.Qf = (float)d.Qp; d.qh = (float)(d.Qp / h); d.qhD = d.Qp / h;
    d.mhqD[0] = -0.5 * d.qhD; d.mhqD[1] = -0.5 * d.Qs / h; d.tqD[0] = 2.0 * d.qhD; d.tqD[1] = 2.0 * d.Qs / h;
    // sigma from separations that include the bits below the record's word (k_pass_a<.., SUBQ>, +15 % on pass A) when
    // the pair unit is coarse for the case: positions rounded to a unit U leave about 15 (U / h) (L_g / h) |g| in the
    // acceleration, L_g the extent of the domain along gravity (measured with U = Q: 5.5e-4 |g| at config 4's 16.8 M
    // size, Q / h = 1.4e-7, L_g / h = 200); the 1e-4 bar decides.  With the pair unit Qp = Q / 2^mbits this is off for
    // every single-phase configuration of BASELINE.json; multi-phase runs always take it.
    {
      double gn = 0, Lg = 0;
      for (int k = 0; k < prm->dim; ++k) gn += prm->g[k] * prm->g[k];
      for (int k = 0; k < prm->dim; ++k)
        Lg += (gn > 0 ? fabs(prm->g[k]) / sqrt(gn) : 0.0) * (prm->domain_max[k] - prm->domain_min[k]);
      if (!(gn > 0)) Lg = Lmax;
      d.subq = (prm->n_phases > 1 || 15.0 * (d.Qp / h) * (Lg / h) > 1e-4) ? 1 : 0;
      if (getenv("SPH_FORCE_SUBQ")) d.subq = 1;   // measurement switches (profiles/): not part of the interface
      if (getenv("SPH_NO_SUBQ") && prm->n_phases == 1) d.subq = 0;
    }
    d.gradcQ = (float)(-5.0 * alpha / (h * h) * d.Qp);
    d.two_over_dp = (float)(2.0 * d.Qp / dp);
    // candidate filter margin: rounding of the expanded form |xj|^2 - 2 xi.xj + |xi|^2 on images
    // of magnitude <= R, plus the rounding of the images themselves
    const double R = sqrt(R2), u = ldexp(1.0, -24);
    const double err_expanded = 16.0 * u * R2 + 8.0 * u * R * rl;
    const double err_diff = 16.0 * u * R * rl;
    d.exact_filter = 2.0 * err_expanded > 0.08 * rc * rc ? 1 : 0;
    d.marg32 = 2.0 * (d.exact_filter ? err_diff : err_expanded);
    d.marg16 = 2.0 * err_diff / (h * h);
    d.rc2m = (float)(rl * rl + d.marg32);   // thresholds at the largest skin: the first build's (SS::rl2m / thr_h2 later)
    {  // float16 filter of k_build (sph_pair.cuh): threshold rounded up to the next half; the margin analysis
       // there is relative to the radius, so the 4.08 of r = 2 becomes 4.08 (1 + s)^2 at the list radius
      d.inv_h = (float)(1.0 / h);
      const double thr = 4.08 * (1.0 + skin) * (1.0 + skin) + 2.0 * err_diff / (h * h);
      __half th = __double2half(thr);
      if ((double)__half2float(th) < thr) th = __ushort_as_half((unsigned short)(__half_as_ushort(th) + 1));
      d.thr_h2 = (unsigned)__half_as_ushort(th) * 0x10001u;
    }
  }
  d.gamma_p = (float)prm->penalty_strength;
  d.pen_mask = (prm->flags & SPH_FLAG_WALL_ADAMI_ONLY) ? 0u : prm->penalty_phase_mask; d.fs_mask = prm->free_surface_mask; d.flags = prm->flags;
  d.skin = skin;
  d.skin_min = std::min(skin, 0.002);
  // contract grid (reading A24: cell edge 2h(1 + 2^-10)) and the step's grid (cell edge that times 1 + s)
  d.ox = (float)prm->domain_min[0]; d.oy = (float)prm->domain_min[1]; d.oz = (float)prm->domain_min[2];
  for (int k = 0; k < 3; ++k) {
    d.dmin[k] = (float)prm->domain_min[k]; d.dmax[k] = (float)prm->domain_max[k];
    d.g[k] = prm->g[k]; d.gamp[k] = prm->g_osc_amp[k];
  }
  auto set_grid = [&](DP& q, double edge, int64_t* ncell) {
    q.inv_edge = (float)(1.0 / edge);
    int nc[3] = {1, 1, 1};
    for (int k = 0; k < prm->dim; ++k)
      nc[k] = std::max(1, (int)ceil((prm->domain_max[k] - prm->domain_min[k]) / edge));
    q.nx = nc[0]; q.ny = nc[1]; q.nz = nc[2];
    *ncell = (int64_t)nc[0] * nc[1] * nc[2];
  };
  const double edgeC = 2.0 * h * (1.0 + 1.0 / 1024.0);  // reading A24
  // NEXT-4: cell edge = half the list radius with a 125 / 25-cell walk, measured against the 27 / 9-cell walk
  // (profiles/r02_README.md); only with kept lists (the contract grid stays the 27-cell one)
  d.reach = 1;
  if (skin > 0.0 && getenv("SPH_REACH")) d.reach = atoi(getenv("SPH_REACH")) == 2 ? 2 : 1;   // measurement switch
  set_grid(d, edgeC * (1.0 + skin) / d.reach, &c->ncell);
  for (int k = 0; k < 3; ++k) d.wamp[k] = k < prm->dim ? prm->wall_osc_amp[k] : 0.0;
  d.womega = 6.283185307179586476925286766559 * prm->wall_osc_freq;
  c->moving = prm->wall_osc_freq > 0.0 && (d.wamp[0] != 0.0 || d.wamp[1] != 0.0 || d.wamp[2] != 0.0);
  if (!c->moving) { d.womega = 0.0; d.wamp[0] = d.wamp[1] = d.wamp[2] = 0.0; }
  d.gperiod = prm->g_osc_period; d.cmax = cmax; d.cfl = prm->cfl; d.hD = h; d.dpD = dp;
  c->dpC = d;
  set_grid(c->dpC, edgeC, &c->ncellC);
  if (c->ncell >= (1ll << 31) - 2 || c->ncellC >= (1ll << 31) - 2) { delete c; return SPH_EINVAL; }
  // sub-cell Morton bits in the sort key (possible when the lists are kept, skin > 0: the contract's id order inside
  // a cell is then produced on demand by contract_view).  Measured (profiles/r02_README.md): 1 or 2 bits per axis
  // change the pair passes by less than 1 % and cost a radix pass, so the default is 0.
  d.sub_bits = 0;
  if (skin > 0.0) {
    int b = 0;
    if (getenv("SPH_SUB_BITS")) b = atoi(getenv("SPH_SUB_BITS"));   // measurement switch (profiles/): not part of the interface
    while (b > 0 && bits_for(c->ncell) + b * prm->dim > 31) --b;
    d.sub_bits = b * prm->dim;
  }
  c->dpC.sub_bits = 0; c->dpC.reach = 1;
  c->cell_bits = bits_for(c->ncell) + d.sub_bits;
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
int64_t sph_num_cells(const sph_ctx* c) { return c ? c->ncellC : 0; }

int sph_set_particles(sph_ctx* c, int64_t n, const float* pos, const float* vel, const float* rho,
                      const int32_t* tag, void* stream) {
  if (!c) return SPH_EINVAL;
  if (n < 0 || n >= (1ll << 31) - 64 || (n > 0 && (!pos || !vel || !rho || !tag))) {
    c->err = "bad arguments to sph_set_particles";
    return SPH_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)stream;
  c->loaded = false;
  if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }  // buffers are reallocated below
  // classify on the device (one-off): caller indices of the fluid entries, then of the wall entries, each in
  // ascending order: a stable one-pass radix sort of (class, index); only the three class counts come to the host
  unsigned* cls_idx = nullptr;
  {
    const size_t m = (size_t)std::max<int64_t>(n, 1);
    int rc0 = dalloc(c, &c->clsKa, m);
    if (!rc0) rc0 = dalloc(c, &c->clsVa, m);
    if (!rc0) rc0 = dalloc(c, &c->clsKb, m);
    if (!rc0) rc0 = dalloc(c, &c->clsVb, m);
    if (!rc0) rc0 = dalloc(c, &c->clsHist, (size_t)512 * cdiv(m, RS_THREADS * rs_items(m)));
    if (!rc0) rc0 = dalloc(c, &c->clsRow, 512);
    if (rc0) return rc0;
    CK(cudaMemsetAsync(c->clsRow, 0, 512 * sizeof(unsigned), st));
    unsigned long long hcnt[3] = {0, 0, 0};
    if (dalloc(c, &c->clsCnt, 3)) return SPH_ENOMEM;
    unsigned long long* counts = c->clsCnt;
    CK(cudaMemsetAsync(counts, 0, 3 * sizeof(unsigned long long), st));
    unsigned *ks = c->clsKa, *vs = c->clsVa;
    if (n) {
      LAUNCH(k_classify, cdiv(n, 256), 256, st, (int)n, c->prm.n_phases, tag, c->clsKa, c->clsVa, counts);
      int rcs = radix_sort(c, st, (int)n, 2, c->clsKa, c->clsVa, c->clsKb, c->clsVb, &ks, &vs, c->clsHist, c->clsRow);
      if (rcs) return rcs;
    }
    CK(cudaMemcpyAsync(hcnt, counts, sizeof(hcnt), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (hcnt[2]) { c->err = "tag out of range"; return SPH_EINVAL; }
    c->n = n; c->nf = (int64_t)hcnt[0]; c->nw = (int64_t)hcnt[1];
    cls_idx = vs;
  }
  const int nf = (int)c->nf, nw = (int)c->nw;
  const size_t cap = (size_t)std::max(nf, nw);
  int rc = SPH_OK;
  // every allocation is attempted only while the previous ones succeeded; the first failing code is returned
#define TRY(call) do { if (rc == SPH_OK) rc = (call); } while (0)
  TRY(dalloc(c, &c->R0, nf)); TRY(dalloc(c, &c->R1, nf)); TRY(dalloc(c, &c->TX, cap)); TRY(dalloc(c, &c->A, (size_t)nf + 16));
  TRY(dalloc(c, &c->TB, cap));
  TRY(dalloc(c, &c->ACC, nf)); TRY(dalloc(c, &c->SIG, nf)); TRY(dalloc(c, &c->DRHO, nf));
  c->npad = ((size_t)nf + PB - 1) / PB * PB;
  c->caps = c->prm.max_neighbours ? (int)((c->prm.max_neighbours + 3u) & ~3u) : (c->prm.dim == 3 ? 160 : 64);
  TRY(dalloc(c, &c->NL, c->npad * (size_t)(c->caps >> 2))); TRY(dalloc(c, &c->NC, nf));
  c->capsw = (c->caps * 3 / 4 + 3) & ~3;  // a particle in a corner of three walls has 7/8 of its (then smaller) support in them
  TRY(dalloc(c, &c->NLW, c->npad * (size_t)(c->capsw >> 2))); TRY(dalloc(c, &c->NCW, nf));
  TRY(dalloc(c, &c->NLF, ((size_t)nw + PB - 1) / PB * PB * (size_t)(c->capsw >> 2))); TRY(dalloc(c, &c->NCF, nw));
  TRY(dalloc(c, &c->ID0, cap)); TRY(dalloc(c, &c->ID1, cap));
  TRY(dalloc(c, &c->keyA, cap)); TRY(dalloc(c, &c->valA, cap)); TRY(dalloc(c, &c->keyB, cap));
  TRY(dalloc(c, &c->valB, cap));
  TRY(dalloc(c, &c->hist, (size_t)512 * std::max(cdiv(std::max(nf, 1), RS_THREADS * rs_items((size_t)nf)),
                                                  cdiv(std::max(nw, 1), RS_THREADS * rs_items((size_t)nw)))));
  TRY(dalloc(c, &c->rowsum, 512));
  if (rc == SPH_OK) CK(cudaMemsetAsync(c->rowsum, 0, 512 * sizeof(unsigned), (cudaStream_t)stream));  // radix digit totals: zero between passes
  TRY(dalloc(c, &c->lbF, c->ncell + 1)); TRY(dalloc(c, &c->lbW, c->ncell + 1));
  TRY(dalloc(c, &c->wnear, c->ncell));
  TRY(dalloc(c, &c->WR, nw)); TRY(dalloc(c, &c->WA, (size_t)nw + 16));
  TRY(dalloc(c, &c->WN, nw)); TRY(dalloc(c, &c->WG, nw)); TRY(dalloc(c, &c->WK, nw));
  TRY(dalloc(c, &c->WID, nw));
  TRY(dalloc(c, &c->S, 1)); TRY(dalloc(c, &c->stat, 1));
#undef TRY
  if (rc) return rc;
  c->IDcur = c->ID0; c->IDnext = c->ID1;
  CK(cudaMemsetAsync(c->S, 0, sizeof(SS), st));
  {  // the first build takes the largest skin; k_predict adapts it from the displacements it sees
    SS h0;
    memset(&h0, 0, sizeof(h0));
    h0.skin_cur = c->dp.skin; h0.budget = 2.0 * c->dp.hD * c->dp.skin * (1.0 - 1e-6);
    h0.rl2m = c->dp.rc2m; h0.thr_h2 = c->dp.thr_h2;
    CK(cudaMemcpyAsync(c->S, &h0, sizeof(SS), cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
  }
  CK(cudaMemsetAsync(c->A + nf, 0, 16 * sizeof(float4), st));   // padding read by the chunked candidate loads
  CK(cudaMemsetAsync(c->WA + nw, 0, 16 * sizeof(float4), st));
  CK(cudaMemsetAsync(c->ACC, 0, sizeof(float4) * std::max(nf, 1), st));
  {  // gravity at t = 0 (sin(0) = 0)
    float g0[3] = {(float)c->prm.g[0], (float)c->prm.g[1], (float)c->prm.g[2]};
    CK(cudaMemcpyAsync((char*)c->S + offsetof(SS, g), g0, sizeof(g0), cudaMemcpyHostToDevice, st));
    // walls at t = 0: no displacement, a_w = 0, v_wall = A omega
    CK(cudaMemcpyAsync((char*)c->S + offsetof(SS, gw), g0, sizeof(g0), cudaMemcpyHostToDevice, st));
    float v0[3] = {(float)(c->dp.wamp[0] * c->dp.womega), (float)(c->dp.wamp[1] * c->dp.womega), (float)(c->dp.wamp[2] * c->dp.womega)};
    CK(cudaMemcpyAsync((char*)c->S + offsetof(SS, vwall), v0, sizeof(v0), cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync((char*)c->S + offsetof(SS, sq), 0, 3 * sizeof(int), st));
    CK(cudaStreamSynchronize(st));  // g0 / v0 are stack variables
  }
  const int* idx_f = reinterpret_cast<const int*>(cls_idx);            // fluid caller ids, ascending
  const int* idx_w = reinterpret_cast<const int*>(cls_idx) + c->nf;    // wall caller ids, ascending
  // ---- wall structure, built once ----
  if (nw > 0) {
    LAUNCH(k_load, cdiv(nw, 256), 256, st, c->dp, nw, 1, idx_w, pos, vel, rho, tag, c->TX, c->TB, c->ID0, c->keyA, c->valA);
    if (c->moving) {  // NEXT-1: keep the set-up order for the per-step re-sort
      rc = dalloc(c, &c->WX0, nw);
      if (!rc) rc = dalloc(c, &c->WXB, nw);
      if (!rc) rc = dalloc(c, &c->WN0, nw);
      if (!rc) rc = dalloc(c, &c->WID0, nw);
      if (!rc) rc = dalloc(c, &c->WkeyA, nw);
      if (!rc) rc = dalloc(c, &c->WkeyB, nw);
      if (!rc) rc = dalloc(c, &c->WvalA, nw);
      if (!rc) rc = dalloc(c, &c->WvalB, nw);
      if (!rc) rc = dalloc(c, &c->WTX, nw);
      if (!rc) rc = dalloc(c, &c->WTB, nw);
      if (!rc) rc = dalloc(c, &c->Whist, (size_t)512 * cdiv(nw, RS_THREADS * rs_items((size_t)nw)));
      if (!rc) rc = dalloc(c, &c->Wrowsum, 512);
      if (rc) return rc;
      CK(cudaMemsetAsync(c->Wrowsum, 0, 512 * sizeof(unsigned), st));
      if (!c->wstream) CK(cudaStreamCreateWithFlags(&c->wstream, cudaStreamNonBlocking));
      if (!c->evFork) CK(cudaEventCreateWithFlags(&c->evFork, cudaEventDisableTiming));
      if (!c->evJoin) CK(cudaEventCreateWithFlags(&c->evJoin, cudaEventDisableTiming));
      CK(cudaMemcpyAsync(c->WX0, c->TX, sizeof(uint4) * nw, cudaMemcpyDeviceToDevice, st));
      CK(cudaMemcpyAsync(c->WID0, c->ID0, sizeof(unsigned) * nw, cudaMemcpyDeviceToDevice, st));
    }
    unsigned *ks, *vs;
    rc = radix_sort(c, st, nw, c->cell_bits, c->keyA, c->valA, c->keyB, c->valB, &ks, &vs);
    if (rc) return rc;
    LAUNCH(k_reorder, cdiv(nw, 256), 256, st, c->dp, nw, vs, c->TX, c->TB, c->ID0, c->WR, c->WA, c->WID,
           (const unsigned*)nullptr, -1, (int*)nullptr);
    CK(cudaMemcpyAsync(c->WK, ks, sizeof(unsigned) * nw, cudaMemcpyDeviceToDevice, st));
    LAUNCH(k_image, cdiv(nw, 256), 256, st, c->dp, nw, c->WR, c->WG);
    LAUNCH(k_cell_bounds, cdiv(c->ncell + 1, 256), 256, st, ks, nw, (int)c->ncell, c->lbW, c->dp.sub_bits);
    if (c->prm.dim == 3) LAUNCH(k_normals<3>, cdiv(nw, 128), 128, st, c->dp, nw, c->WR, c->WK, c->lbW, c->WN);
    else LAUNCH(k_normals<2>, cdiv(nw, 128), 128, st, c->dp, nw, c->WR, c->WK, c->lbW, c->WN);
    if (c->moving) {
      LAUNCH(k_unsort4, cdiv(nw, 256), 256, st, nw, vs, c->WN, c->WN0);
      LAUNCH(k_gatherx, cdiv(nw, 256), 256, st, nw, vs, c->WX0, c->WXB);
    }
  } else {
    LAUNCH(k_cell_bounds, cdiv(c->ncell + 1, 256), 256, st, c->keyA, 0, (int)c->ncell, c->lbW, 0);
  }
  LAUNCH(k_wnear, cdiv(c->ncell, 256), 256, st, c->dp, (int)c->ncell, c->lbW, c->wnear);
  // ---- fluid: load, then the common pipeline in init mode (dt = 0: sigma_i, p_w, (dv/dt)^0) ----
  if (nf > 0) {
    LAUNCH(k_load, cdiv(nf, 256), 256, st, c->dp, nf, 0, idx_f, pos, vel, rho, tag, c->TX, c->TB, c->IDcur, c->keyA, c->valA);
  }
  Prof pf(c, st);
  pf.on = false;
  rc = rebuild_body(c, st, 1, pf);
  if (!rc) rc = pass_tail(c, st, 1, pf);
  c->direct_rebuilds = 0; c->graph_rebuilds_counted = 0;
  cudaError_t e = cudaStreamSynchronize(st);
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
  size_t m = (size_t)std::max<int64_t>(n, 1);
  int rc = dalloc(c, &c->stage_pos, m * 3);
  if (!rc) rc = dalloc(c, &c->stage_vel, m * 3);
  if (!rc) rc = dalloc(c, &c->stage_rho, m);
  if (!rc) rc = dalloc(c, &c->stage_tag, m);
  if (rc) return rc;
  float *dpos = c->stage_pos, *dvel = c->stage_vel, *drho = c->stage_rho;
  int32_t* dtag = c->stage_tag;
  if (n) {
    rc = h2d(c, dpos, pos, (size_t)n * 12, st);
    if (!rc) rc = h2d(c, dvel, vel, (size_t)n * 12, st);
    if (!rc) rc = h2d(c, drho, rho, (size_t)n * 4, st);
    if (!rc) rc = h2d(c, dtag, tag, (size_t)n * 4, st);
  }
  if (rc == SPH_OK) rc = sph_set_particles(c, n, dpos, dvel, drho, dtag, stream);
  cudaStreamSynchronize(st);
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
  if (c->nf) LAUNCH(k_get, cdiv(c->nf, 256), 256, st, c->dp, (int)c->nf, 0, c->R1, c->TB, c->ACC, c->IDcur, pos, vel, rho, p, acc);
  if (c->nw) LAUNCH(k_get, cdiv(c->nw, 256), 256, st, c->dp, (int)c->nw, 1, c->WR, (const float4*)nullptr, (const float4*)nullptr, c->WID, pos, vel, rho, p, acc);
  CK(cudaGetLastError());
  return SPH_OK;
}

int sph_get_fields_host(sph_ctx* c, float* pos, float* vel, float* rho, float* p, float* acc, void* stream) {
  if (!c) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)std::max<int64_t>(c->n, 1);
  if (dalloc(c, &c->stage_out, n * 11)) return SPH_ECUDA;  // kept across calls
  float* buf = c->stage_out;
  float *dpos = buf, *dvel = buf + 3 * n, *dacc = buf + 6 * n, *drho = buf + 9 * n, *dp = buf + 10 * n;
  int rc = sph_get_fields(c, pos ? dpos : nullptr, vel ? dvel : nullptr, rho ? drho : nullptr,
                          p ? dp : nullptr, acc ? dacc : nullptr, stream);
  if (rc == SPH_OK && c->n) {
    if (pos) rc = d2h(c, pos, dpos, (size_t)c->n * 12, st);
    if (vel && !rc) rc = d2h(c, vel, dvel, (size_t)c->n * 12, st);
    if (acc && !rc) rc = d2h(c, acc, dacc, (size_t)c->n * 12, st);
    if (rho && !rc) rc = d2h(c, rho, drho, (size_t)c->n * 4, st);
    if (p && !rc) rc = d2h(c, p, dp, (size_t)c->n * 4, st);
  }
  cudaError_t e2 = cudaStreamSynchronize(st);
  if (rc) return rc;
  if (e2 != cudaSuccess) {
    c->err = cudaGetErrorString(e2);
    return SPH_ECUDA;
  }
  return SPH_OK;
}

int sph_get_stats(sph_ctx* c, sph_stats* out, void* stream) { return sph_get_stats_ex(c, out, 1, stream); }

int sph_get_stats_ex(sph_ctx* c, sph_stats* out, int32_t with_pairs, void* stream) {
  if (!c || !out) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  StatAcc z;
  memset(&z, 0, sizeof(z));
  CK(cudaMemcpyAsync(c->stat, &z, sizeof(z), cudaMemcpyHostToDevice, st));
  const int nf = (int)c->nf;
  if (nf) {
    LAUNCH(k_stats, std::min(cdiv(nf, 256), 1184), 256, st, c->dp, nf, c->R1, c->TB, c->stat);
    if (with_pairs) {
      View v;
      int rc = contract_view(c, st, &v);
      if (rc) return rc;
      LAUNCH(k_neigh, cdiv(nf, PW), PW * 32, st, v.dp, nf, 0, 0, v.G, v.ID, v.G, v.ID, v.lb, v.WG,
             v.WID, v.lbW, (int*)nullptr, (const long long*)nullptr, (int*)nullptr, 0ll, &c->stat->pairs);
    }
  }
  SS hs;
  CK(cudaMemcpyAsync(&z, c->stat, sizeof(z), cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(&hs, c->S, sizeof(hs), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  out->t = hs.t; out->dt = hs.dt_d; out->steps = hs.steps; out->n_fluid = c->nf; out->n_wall = c->nw;
  out->n_pairs = with_pairs ? (int64_t)z.pairs : -1; out->e_kin = z.ek;
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
  out->rebuilds = (int64_t)hs.rebuilds + 1;  // + the set-up's
  out->list_skin = hs.skin_cur;
  {  // rebuild branches taken inside graph replays: their kernels were launched by the graph, count them now
    const int64_t in_graph = (int64_t)hs.rebuilds - c->direct_rebuilds;
    if (in_graph > c->graph_rebuilds_counted) {
      c->launches += (in_graph - c->graph_rebuilds_counted) * c->body_launches;
      c->graph_rebuilds_counted = in_graph;
    }
  }
  if (hs.nonfinite) { c->err = "non-finite particle state"; return SPH_ENONFINITE; }
  if (hs.list_overflow) {
    c->err = "a particle has " + std::to_string(hs.list_overflow) + " neighbours, the lists hold " +
             std::to_string(c->caps) + " fluid and " + std::to_string(c->capsw) +
             " wall entries: set sph_params.max_neighbours";
    return SPH_ENEIGHBOURS;
  }
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

int sph_get_timings(sph_ctx* c, float* ms, int32_t* n_steps, int32_t* n_rebuilds) {
  if (!c || !ms || !n_steps) return SPH_EINVAL;
  for (int k = 0; k < SPH_STAGE_COUNT; ++k) ms[k] = 0.f;
  *n_steps = c->ev_steps;
  if (n_rebuilds) *n_rebuilds = 0;
  if (c->ev_steps == 0) return SPH_OK;
  CK(cudaEventSynchronize(c->ev[(c->ev_steps - 1) * sph_ctx::EV_PER_STEP + 8]));
  // marks per step: 0 start, 1 predict, 2 sort, 3 reorder, 4 list build, 5 wall 1, 6 pass A, 7 wall 2, 8 pass B
  static const int stage_of[8] = {SPH_STAGE_PREDICT, SPH_STAGE_SORT, SPH_STAGE_REORDER, SPH_STAGE_BUILD, SPH_STAGE_WALL,
                                  SPH_STAGE_PASS_A, SPH_STAGE_WALL, SPH_STAGE_PASS_B};
  for (int s = 0; s < c->ev_steps; ++s) {
    if (n_rebuilds && c->ev_rebuilt[s]) ++*n_rebuilds;
    for (int k = 0; k < 8; ++k) {
      float t = 0.f;
      CK(cudaEventElapsedTime(&t, c->ev[s * sph_ctx::EV_PER_STEP + k], c->ev[s * sph_ctx::EV_PER_STEP + k + 1]));
      ms[stage_of[k]] += t;
    }
  }
  c->ev_steps = 0;
  return SPH_OK;
}

int sph_debug_cells(sph_ctx* c, int32_t* cell_id, int32_t* perm, int32_t* cs, int32_t* ce, void* stream) {
  if (!c) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)std::max<int64_t>(c->n, 1), nc = (size_t)c->ncellC;
  int *dcid = nullptr, *dperm = nullptr, *dcs = nullptr, *dce = nullptr;
  CK(cudaMalloc((void**)&dcid, n * 4)); CK(cudaMalloc((void**)&dperm, n * 4));
  CK(cudaMalloc((void**)&dcs, 2 * nc * 4)); CK(cudaMalloc((void**)&dce, 2 * nc * 4));
  View v;
  int rcv = contract_view(c, st, &v);
  if (rcv) { cudaFree(dcid); cudaFree(dperm); cudaFree(dcs); cudaFree(dce); return rcv; }
  if (c->nf) LAUNCH(k_dbg_cells, cdiv(c->nf, 256), 256, st, v.dp, (int)c->nf, v.G, v.ID, dcid, dperm, 0);
  if (c->nw) LAUNCH(k_dbg_cells, cdiv(c->nw, 256), 256, st, v.dp, (int)c->nw, v.WG, v.WID, dcid, dperm, (int)c->nf);
  LAUNCH(k_dbg_ranges, cdiv(nc, 256), 256, st, (int)nc, v.lb, dcs, dce);
  LAUNCH(k_dbg_ranges, cdiv(nc, 256), 256, st, (int)nc, v.lbW, dcs + nc, dce + nc);
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
  View v;
  int rcv = contract_view(c, st, &v);
  if (rcv) { cudaFree(dcnt); return rcv; }
  auto run = [&](int mode, const long long* doff, int* dids, long long dcap) {
    if (c->nf)
      LAUNCH(k_neigh, cdiv(c->nf, PW), PW * 32, st, v.dp, (int)c->nf, 0, mode, v.G, v.ID, v.G, v.ID, v.lb,
             v.WG, v.WID, v.lbW, dcnt, doff, dids, dcap, (unsigned long long*)nullptr);
    if (c->nw && c->nf)
      LAUNCH(k_neigh, cdiv(c->nw, PW), PW * 32, st, v.dp, (int)c->nw, 1, mode, v.WG, v.WID, v.G, v.ID, v.lb,
             v.WG, v.WID, v.lbW, dcnt, doff, dids, dcap, (unsigned long long*)nullptr);
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

static int probe_common(sph_ctx* c, int32_t m, const float* xyz, float* o1, float* o2, int gauge, void* stream) {
  if (!c || m < 0 || (m > 0 && (!xyz || !o1 || (!gauge && !o2)))) { if (c) c->err = "bad arguments"; return SPH_EINVAL; }
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  if (m == 0) return SPH_OK;
  cudaStream_t st = (cudaStream_t)stream;
  float* d = nullptr;
  CK(cudaMalloc((void**)&d, (size_t)m * 5 * sizeof(float)));
  cudaError_t e = cudaMemcpyAsync(d, xyz, (size_t)m * 12, cudaMemcpyHostToDevice, st);
  const int nf = (int)c->nf;
  if (gauge) LAUNCH(k_probe_gauge, m, 256, st, c->dp, nf, m, d, c->R1, d + 3 * m);
  else LAUNCH(k_probe_pressure, m, 32, st, c->dp, nf, m, d, c->R1, c->lbF, d + 3 * m, d + 4 * m);
  if (e == cudaSuccess) e = cudaMemcpyAsync(o1, d + 3 * m, (size_t)m * 4, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && !gauge) e = cudaMemcpyAsync(o2, d + 4 * m, (size_t)m * 4, cudaMemcpyDeviceToHost, st);
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(d);
  if (e != cudaSuccess || e2 != cudaSuccess) { c->err = cudaGetErrorString(e != cudaSuccess ? e : e2); return SPH_ECUDA; }
  return SPH_OK;
}

int sph_probe_pressure(sph_ctx* c, int32_t m, const float* xyz, float* p_out, float* wsum_out, void* stream) {
  return probe_common(c, m, xyz, p_out, wsum_out, 0, stream);
}

int sph_probe_gauge(sph_ctx* c, int32_t m, const float* xyz, float* eta_out, void* stream) {
  return probe_common(c, m, xyz, eta_out, nullptr, 1, stream);
}

int sph_debug_list_check(sph_ctx* c, int64_t* out3, void* stream) {
  if (!c || !out3) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  out3[0] = out3[1] = out3[2] = 0;
  if (!c->nf) return SPH_OK;
  unsigned long long* d = nullptr;
  CK(cudaMalloc((void**)&d, 24));
  CK(cudaMemsetAsync(d, 0, 24, st));
  const float4* G = fluid_images(c, st);
  LAUNCH(k_list_check, cdiv(c->nf, PW), PW * 32, st, c->dp, (int)c->nf, G, c->lbF, c->NL, c->NC, c->caps, d);
  unsigned long long h[3];
  cudaError_t e = cudaMemcpyAsync(h, d, 24, cudaMemcpyDeviceToHost, st);
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(d);
  if (e != cudaSuccess || e2 != cudaSuccess) { c->err = cudaGetErrorString(e != cudaSuccess ? e : e2); return SPH_ECUDA; }
  for (int k = 0; k < 3; ++k) out3[k] = (int64_t)h[k];
  return SPH_OK;
}

int sph_debug_step_lists(sph_ctx* c, int64_t* offsets, int32_t* ids, int64_t cap, int64_t* total, void* stream) {
  if (!c || !offsets || !total) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = c->n;
  int* dcnt = nullptr;
  CK(cudaMalloc((void**)&dcnt, std::max<int64_t>(n, 1) * 4));
  CK(cudaMemsetAsync(dcnt, 0, std::max<int64_t>(n, 1) * 4, st));
  auto run = [&](int mode, const long long* doff, int* dids, long long dcap) {
    if (c->nf)
      LAUNCH(k_list_export, cdiv(c->nf, 256), 256, st, (int)c->nf, mode, c->IDcur, c->NL, c->NC, c->caps, c->IDcur,
             c->NLW, c->NCW, c->capsw, c->WID, dcnt, doff, dids, dcap);
    if (c->nw && c->nf)
      LAUNCH(k_list_export, cdiv(c->nw, 256), 256, st, (int)c->nw, mode, c->WID, c->NLF, c->NCF, c->capsw, c->IDcur,
             (const uint4*)nullptr, (const int*)nullptr, 0, (const unsigned*)nullptr, dcnt, doff, dids, dcap);
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

int sph_debug_time_pointwise(sph_ctx* c, float* ms, void* stream) {
  if (!c || !ms) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  ms[0] = ms[1] = ms[2] = 0.f;
  const int nf = (int)c->nf;
  if (!nf) return SPH_OK;
  // scratch outputs: the state (R1, TB, ACC, SIG, R0, keyA / valA of the step) is read, never written
  float4* B2 = nullptr; uint4* X2 = nullptr; XB* R2 = nullptr; unsigned *k2 = nullptr, *v2 = nullptr;
  CK(cudaMalloc((void**)&B2, sizeof(float4) * nf)); CK(cudaMalloc((void**)&X2, sizeof(uint4) * nf));
  CK(cudaMalloc((void**)&R2, sizeof(XB) * nf)); CK(cudaMalloc((void**)&k2, 4 * (size_t)nf)); CK(cudaMalloc((void**)&v2, 4 * (size_t)nf));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = cdiv(nf, 256);
  for (int which = 0; which < 3; ++which) {
    float tot = 0.f;
    for (int rep = 0; rep < 6; ++rep) {
      CK(cudaMemcpyAsync(B2, c->TB, sizeof(float4) * nf, cudaMemcpyDeviceToDevice, st));  // the kernels update (v, rho) in place
      cudaEventRecord(e0, st);
      if (which == 0) LAUNCH((k_predict<true, false>), grid, 256, st, c->dp, c->S, nf, c->R1, B2, c->ACC, c->SIG, X2, R2, k2, v2, 0ull, 0, 0);
      else if (which == 1) LAUNCH((k_predict<false, true>), grid, 256, st, c->dp, c->S, nf, c->R1, B2, c->ACC, c->SIG, X2, R2, k2, v2, 0ull, 0, 0);
      else LAUNCH((k_predict<true, true>), grid, 256, st, c->dp, c->S, nf, c->R1, B2, c->ACC, c->SIG, X2, R2, k2, v2, 0ull, 0, 0);
      cudaEventRecord(e1, st);
      cudaError_t e = cudaEventSynchronize(e1);
      if (e != cudaSuccess) { c->err = cudaGetErrorString(e); return SPH_ECUDA; }
      float t = 0.f;
      cudaEventElapsedTime(&t, e0, e1);
      if (rep) tot += t;
    }
    ms[which] = tot / 5.f;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(B2); cudaFree(X2); cudaFree(R2); cudaFree(k2); cudaFree(v2);
  return SPH_OK;
}

int sph_debug_fma_peak(double* tflops_host, void* stream) {
  if (!tflops_host) return SPH_EINVAL;
  *tflops_host = 0.0;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, nsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return SPH_ECUDA;
  float* d = nullptr;
  if (cudaMalloc((void**)&d, 4) != cudaSuccess) return SPH_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = nsm * 8, iters = 4096;   // 8 blocks of 256 threads per SM: 2048 resident threads
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {  // the first repetitions warm the clocks up; best of the rest
    cudaEventRecord(e0, st);
    k_fma_peak<<<blocks, 256, 0, st>>>(d, iters, 0.999f, 0.001f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return SPH_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = (double)blocks * 256.0 * (double)iters * 64.0 * 2.0;
    if (rep >= 2 && ms > 0.f) best = std::max(best, flop / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d);
  *tflops_host = best;
  return SPH_OK;
}

int sph_debug_gather_floor(sph_ctx* c, int32_t body_fma, float* ms, int64_t* requests, void* stream) {
  if (!c || !ms || body_fma < 0 || body_fma > 4096) return SPH_EINVAL;
  if (!c->loaded) { c->err = "no particles"; return SPH_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  for (int m = 0; m < 5; ++m) ms[m] = 0.f;
  if (requests) *requests = 0;
  const int nf = (int)c->nf;
  if (!nf) return SPH_OK;
  const int M = cdiv(nf, PB);
  int dev = 0, nsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1)
    return SPH_ECUDA;
  const int nq = std::min(nsm, 1000);
  // scratch: [0] request count, [1] the kernels' never-written output word, then the queue counters of mode 4;
  // chunk keys / values of mode 4 (two ping-pong pairs)
  unsigned long long* d = nullptr;   // one allocation: 16 bytes, then nq counters (padded to 16 bytes), then 4 M words
  const size_t qwords = ((size_t)nq + 3) & ~(size_t)3;
  CK(cudaMalloc((void**)&d, 16 + 4 * qwords + 16 * (size_t)M));
  unsigned* q = reinterpret_cast<unsigned*>(d + 2);
  unsigned* ck = q + qwords;
  if (cudaMemsetAsync(d, 0, 16, st) != cudaSuccess) { cudaFree(d); c->err = "cudaMemsetAsync"; return SPH_ECUDA; }
  LAUNCH(k_gather_requests, cdiv(nf, 256), 256, st, nf, c->NC, d);
  // mode 4: blobs of one chunk length along x by 4 x 4 cell rows (best of 1 x 1 ... 16 x 16, profiles/r02_README.md)
  const double edge_dp = 1.0 / ((double)c->dp.inv_edge * c->prm.dp);
  const int L = std::max(1, std::min(63, (int)lrint((double)PB / (c->prm.dim == 3 ? edge_dp * edge_dp * edge_dp : edge_dp * edge_dp))));
  const int ry = std::min(4, c->dp.ny), rz = std::min(4, c->dp.nz);
  const int cobits = bits_for((int64_t)cdiv(c->dp.nx, L) * cdiv(c->dp.ny, ry) * cdiv(c->dp.nz, rz)) + 10;
  unsigned *ko = nullptr, *vo = nullptr;
  int rc = SPH_OK;
  if (cobits <= 32) {
    LAUNCH(k_chunk_keys, cdiv(M, 256), 256, st, c->dp, nf, c->K, M, L, ry, rz, ck, ck + M);
    rc = radix_sort(c, st, M, cobits, ck, ck + M, ck + 2 * (size_t)M, ck + 3 * (size_t)M, &ko, &vo);
  }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = cdiv(nf, PB);
  // R1 = the records pass B gathers (the state after pass A); the lists are the ones the passes read
  for (int mode = 0; mode < 5 && rc == SPH_OK; ++mode) {
    if (mode == 4 && !vo) break;
    float best = 0.f;
    for (int rep = 0; rep < 4; ++rep) {   // one warm-up launch, best of three
      if (mode == 4) cudaMemsetAsync(q, 0, 4 * (size_t)nq, st);
      cudaEventRecord(e0, st);
#define GW(MODE)                                                                                                              \
  do {                                                                                                                        \
    if (body_fma) LAUNCH((k_gather_walk<MODE, true>), grid, PB, st, nf, c->R1, c->NL, c->NC, c->caps, (unsigned*)(d + 1), body_fma); \
    else LAUNCH((k_gather_walk<MODE, false>), grid, PB, st, nf, c->R1, c->NL, c->NC, c->caps, (unsigned*)(d + 1), 0);       \
  } while (0)
      switch (mode) {
        case 0: GW(0); break;
        case 1: GW(1); break;
        case 2: GW(2); break;
        case 3: GW(3); break;
        default:
          if (body_fma) LAUNCH(k_gather_walk_affine<true>, std::min(M, nq * SPH_MINB), PB, st, nf, c->R1, c->NL, c->NC, c->caps, (unsigned*)(d + 1), vo, M, q, nq, body_fma);
          else LAUNCH(k_gather_walk_affine<false>, std::min(M, nq * SPH_MINB), PB, st, nf, c->R1, c->NL, c->NC, c->caps, (unsigned*)(d + 1), vo, M, q, nq, 0);
          break;
      }
#undef GW
      cudaEventRecord(e1, st);
      cudaError_t e = cudaEventSynchronize(e1);
      if (e != cudaSuccess) { c->err = cudaGetErrorString(e); rc = SPH_ECUDA; break; }
      float t = 0.f;
      cudaEventElapsedTime(&t, e0, e1);
      if (rep && (best == 0.f || t < best)) best = t;
    }
    ms[mode] = best;
  }
  unsigned long long h = 0;
  if (rc == SPH_OK && cudaMemcpy(&h, d, 8, cudaMemcpyDeviceToHost) != cudaSuccess) { c->err = "request count read-back"; rc = SPH_ECUDA; }
  if (requests) *requests = (int64_t)h;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d);
  return rc;
}

int sph_debug_gather_patterns(double* cycles, void* stream) {
  if (!cycles) return SPH_EINVAL;
  for (int k = 0; k < 8; ++k) cycles[k] = 0.0;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, nsm = 0, khz = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev) != cudaSuccess)
    return SPH_ECUDA;
  const int blocks = nsm * SPH_MINB, iters = 1024;
  XB* R = nullptr;
  if (cudaMalloc((void**)&R, (size_t)blocks * 512 * sizeof(XB) + 16) != cudaSuccess) return SPH_ENOMEM;
  cudaMemsetAsync(R, 1, (size_t)blocks * 512 * sizeof(XB) + 16, st);
  unsigned* out = reinterpret_cast<unsigned*>(R + (size_t)blocks * 512);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  int rc = SPH_OK;
  for (int pat = 0; pat < 8 && rc == SPH_OK; ++pat) {
    float best = 0.f;
    for (int rep = 0; rep < 4; ++rep) {   // one warm-up launch, best of three
      cudaEventRecord(e0, st);
      switch (pat) {
        case 0: k_gather_patterns<0><<<blocks, PB, 0, st>>>(R, iters, out); break;
        case 1: k_gather_patterns<1><<<blocks, PB, 0, st>>>(R, iters, out); break;
        case 2: k_gather_patterns<2><<<blocks, PB, 0, st>>>(R, iters, out); break;
        case 3: k_gather_patterns<3><<<blocks, PB, 0, st>>>(R, iters, out); break;
        case 4: k_gather_patterns<4><<<blocks, PB, 0, st>>>(R, iters, out); break;
        case 5: k_gather_patterns<5><<<blocks, PB, 0, st>>>(R, iters, out); break;
        case 6: k_gather_patterns<6><<<blocks, PB, 0, st>>>(R, iters, out); break;
        default: k_gather_patterns<7><<<blocks, PB, 0, st>>>(R, iters, out); break;
      }
      cudaEventRecord(e1, st);
      if (cudaEventSynchronize(e1) != cudaSuccess) { rc = SPH_ECUDA; break; }
      float t = 0.f;
      cudaEventElapsedTime(&t, e0, e1);
      if (rep && (best == 0.f || t < best)) best = t;
    }
    // SM cycles at the device's maximum clock per warp-wide gather request (SPH_MINB blocks x PB / 32 warps per SM)
    const double requests_per_sm = (double)SPH_MINB * (PB / 32) * iters * 4.0;
    cycles[pat] = best * 1e-3 * (double)khz * 1e3 / requests_per_sm;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(R);
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
    LAUNCH(k_scatter_f, cdiv(c->nf, 256), 256, st, (int)c->nf, c->SIG, c->IDcur, d, c->sigma0, 1.0f);
    LAUNCH(k_scatter_f, cdiv(c->nf, 256), 256, st, (int)c->nf, c->DRHO, c->IDcur, d + n, 1.0f, 0.0f);
  }
  cudaError_t e = cudaMemcpyAsync(sigma, d, c->n * 4, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(sigma + c->n, d + n, c->n * 4, cudaMemcpyDeviceToHost, st);
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(d);
  if (e != cudaSuccess || e2 != cudaSuccess) { c->err = cudaGetErrorString(e != cudaSuccess ? e : e2); return SPH_ECUDA; }
  return SPH_OK;
}

}  // extern "C"

// ============================================================================================
// sph_cell_sort_static: the cell-list radix sort with its scratch in a static device array
// (include/sph.h; for callers that must not allocate).  Same kernels as radix_sort() above.
// ============================================================================================
namespace {

// n <= SPH_STATIC_SORT_MAX_KEYS < RS_SMALL_N: tiles of RS_THREADS * 4 keys, as rs_items() picks for these sizes
constexpr int SSO_ITEMS = 4;
constexpr int SSO_MAX_BLOCKS = SPH_STATIC_SORT_MAX_KEYS / (RS_THREADS * SSO_ITEMS);
static_assert(SPH_STATIC_SORT_MAX_KEYS < RS_SMALL_N && SPH_STATIC_SORT_MAX_KEYS % (RS_THREADS * SSO_ITEMS) == 0,
              "the static sort uses the small-input tile size");
// layout of the array in 32-bit words: digit totals | tile histograms (digit-major) | keys | values
constexpr size_t SSO_ROWSUM = 0, SSO_HIST = 512, SSO_KEYS = SSO_HIST + (size_t)512 * SSO_MAX_BLOCKS,
                 SSO_VALS = SSO_KEYS + SPH_STATIC_SORT_MAX_KEYS, SSO_WORDS = SSO_VALS + SPH_STATIC_SORT_MAX_KEYS;

// In HOST code this name is a host-side stand-in for the symbol, not a device address: the kernels get the
// address cudaGetSymbolAddress returns for the current device (sso_scratch below).
static __device__ __align__(256) unsigned g_sso_scratch[SSO_WORDS];

constexpr int SSO_MAX_DEVICES = 64;
unsigned* g_sso_ptr[SSO_MAX_DEVICES] = {};  // per device: address of g_sso_scratch, looked up once with that device current
char g_sso_err[192] = "";

int sso_fail(int code, const char* fmt, long long a = 0, long long b = 0) {
  snprintf(g_sso_err, sizeof g_sso_err, fmt, a, b);
  return code;
}
int sso_fail_cuda(const char* what, cudaError_t e) {
  snprintf(g_sso_err, sizeof g_sso_err, "sph_cell_sort_static: %s: %s", what, cudaGetErrorString(e));
  cudaGetLastError();
  return SPH_ECUDA;
}

// Device address of the scratch array on the CURRENT device.  Two threads making the first call at once both
// get the same address from the runtime and store the same value.
int sso_scratch(unsigned** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return sso_fail_cuda("cudaGetDevice", e);
  if (dev < 0 || dev >= SSO_MAX_DEVICES) return sso_fail(SPH_EINVAL, "sph_cell_sort_static: device ordinal %lld is beyond the %lld this entry point keeps addresses for", dev, SSO_MAX_DEVICES);
  unsigned* p = __atomic_load_n(&g_sso_ptr[dev], __ATOMIC_ACQUIRE);
  if (!p) {
    e = cudaGetSymbolAddress((void**)&p, g_sso_scratch);
    if (e != cudaSuccess) return sso_fail_cuda("cudaGetSymbolAddress", e);
    if (!p) return sso_fail(SPH_ECUDA, "sph_cell_sort_static: cudaGetSymbolAddress returned a null address");
    __atomic_store_n(&g_sso_ptr[dev], p, __ATOMIC_RELEASE);
  }
  *out = p;
  return SPH_OK;
}

__global__ void __launch_bounds__(256) k_sso_iota(unsigned* __restrict__ v, int n) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i < n) v[i] = (unsigned)i;
}

template <int ND>
void sso_pass(cudaStream_t st, const unsigned* ki, const unsigned* vi, int n, int shift, unsigned* hist, int nblk,
              unsigned* rowsum, unsigned* kt, unsigned* vt) {
  k_radix_hist<ND, SSO_ITEMS><<<nblk, RS_THREADS, 0, st>>>(ki, n, shift, hist, nblk, rowsum);
  k_scan_apply<<<ND, 256, 0, st>>>(hist, nblk, rowsum);
  k_radix_scatter<ND, SSO_ITEMS><<<nblk, RS_THREADS, 0, st>>>(ki, vi, n, shift, hist, nblk, kt, vt, rowsum);
}

}  // namespace

extern "C" {

const char* sph_cell_sort_static_error(void) { return g_sso_err; }

int sph_cell_sort_static(int32_t n, const uint32_t* keys, const uint32_t* vals, int32_t key_bits, uint32_t* keys_out,
                         uint32_t* vals_out, void* stream) {
  if (n < 0) return sso_fail(SPH_EINVAL, "sph_cell_sort_static: n = %lld is negative", n);
  if (n > SPH_STATIC_SORT_MAX_KEYS)
    return sso_fail(SPH_EINVAL, "sph_cell_sort_static: n = %lld exceeds SPH_STATIC_SORT_MAX_KEYS = %lld (the static scratch array holds no more; use a context)",
                    n, SPH_STATIC_SORT_MAX_KEYS);
  if (key_bits < 1 || key_bits > 32) return sso_fail(SPH_EINVAL, "sph_cell_sort_static: key_bits = %lld is outside 1..32", key_bits);
  if (n == 0) return SPH_OK;
  if (!keys || !keys_out || !vals_out) return sso_fail(SPH_EINVAL, "sph_cell_sort_static: NULL keys or output pointer");
  cudaStream_t st = (cudaStream_t)stream;
  unsigned* scratch = nullptr;
  int rc = sso_scratch(&scratch);
  if (rc) return rc;
  unsigned *rowsum = scratch + SSO_ROWSUM, *hist = scratch + SSO_HIST, *ktmp = scratch + SSO_KEYS, *vtmp = scratch + SSO_VALS;
  // the array keeps what the last call left: the digit totals must start at zero (an interrupted call leaves them set)
  cudaError_t e = cudaMemsetAsync(rowsum, 0, 512 * sizeof(unsigned), st);
  if (e != cudaSuccess) return sso_fail_cuda("cudaMemsetAsync", e);
  int dbits, passes;
  radix_plan(key_bits, &dbits, &passes);
  const int nblk = cdiv(n, RS_THREADS * SSO_ITEMS);
  // pass p writes the caller's outputs when an even number of passes follows it, else the scratch pair: the last
  // pass lands in the outputs and no pass reads the buffer it writes
  auto to_out = [&](int p) { return ((passes - 1 - p) & 1) == 0; };
  const unsigned *ki = keys, *vi = vals;
  if (!vi) {  // indices 0..n-1, into the value buffer that pass 0 does not write
    unsigned* v0 = to_out(0) ? vtmp : vals_out;
    k_sso_iota<<<cdiv(n, 256), 256, 0, st>>>(v0, n);
    vi = v0;
  }
  for (int p = 0; p < passes; ++p) {
    unsigned *kt = to_out(p) ? keys_out : ktmp, *vt = to_out(p) ? vals_out : vtmp;
    if (dbits == 9) sso_pass<512>(st, ki, vi, n, dbits * p, hist, nblk, rowsum, kt, vt);
    else sso_pass<256>(st, ki, vi, n, dbits * p, hist, nblk, rowsum, kt, vt);
    ki = kt;
    vi = vt;
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return sso_fail_cuda("kernel launch", e);
  return SPH_OK;
}

}  // extern "C"
