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
  int sort_passes = 1, sort_bits = 8;
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
  float *hpos = nullptr, *hvel = nullptr, *hrho = nullptr;  // staging of sph_set_particles_host
  int32_t* htagd = nullptr;
  float* hout = nullptr;   // staging of sph_get_fields_host
  int* hidx = nullptr;     // caller indices of one class during sph_set_particles
  // one step captured as a CUDA graph (launch-bound small configurations); rebuilt after sph_set_particles
  cudaGraphExec_t gexec = nullptr;
  cudaStream_t cap_stream = nullptr;
  int64_t graph_launches = 0;  // kernel launches inside the captured step
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

// Pair kernels are instantiated for DIM in {2,3} x MULTI x EXACT (filter form).
#define PAIR_SEL(c) (((c)->prm.dim == 3 ? 4 : 0) | ((c)->multi ? 2 : 0) | ((c)->dp.exact_filter ? 1 : 0))
#define PAIR_DISPATCH(KERN, grid, st, ...)                                            \
  switch (PAIR_SEL(c)) {                                                              \
    case 0: LAUNCH((KERN<2, false, false>), grid, PB, st, __VA_ARGS__); break;        \
    case 1: LAUNCH((KERN<2, false, true>), grid, PB, st, __VA_ARGS__); break;         \
    case 2: LAUNCH((KERN<2, true, false>), grid, PB, st, __VA_ARGS__); break;         \
    case 3: LAUNCH((KERN<2, true, true>), grid, PB, st, __VA_ARGS__); break;          \
    case 4: LAUNCH((KERN<3, false, false>), grid, PB, st, __VA_ARGS__); break;        \
    case 5: LAUNCH((KERN<3, false, true>), grid, PB, st, __VA_ARGS__); break;         \
    case 6: LAUNCH((KERN<3, true, false>), grid, PB, st, __VA_ARGS__); break;         \
    default: LAUNCH((KERN<3, true, true>), grid, PB, st, __VA_ARGS__); break;         \
  }
#define WALL_DISPATCH(VEL, grid, st, ...)                                             \
  switch (PAIR_SEL(c)) {                                                              \
    case 0: LAUNCH((k_wall<2, false, false, VEL>), grid, PB, st, __VA_ARGS__); break; \
    case 1: LAUNCH((k_wall<2, false, true, VEL>), grid, PB, st, __VA_ARGS__); break;  \
    case 2: LAUNCH((k_wall<2, true, false, VEL>), grid, PB, st, __VA_ARGS__); break;  \
    case 3: LAUNCH((k_wall<2, true, true, VEL>), grid, PB, st, __VA_ARGS__); break;   \
    case 4: LAUNCH((k_wall<3, false, false, VEL>), grid, PB, st, __VA_ARGS__); break; \
    case 5: LAUNCH((k_wall<3, false, true, VEL>), grid, PB, st, __VA_ARGS__); break;  \
    case 6: LAUNCH((k_wall<3, true, false, VEL>), grid, PB, st, __VA_ARGS__); break;  \
    default: LAUNCH((k_wall<3, true, true, VEL>), grid, PB, st, __VA_ARGS__); break;  \
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
                  c->hpos, c->hvel, c->hrho, c->htagd, c->hout, c->hidx,
                  c->WX0, c->WN0, c->WID0, c->WkeyA, c->WkeyB, c->WvalA, c->WvalB,
                  c->WTX, c->WTB, c->Whist, c->Wrowsum};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (auto e : c->ev) cudaEventDestroy(e);
  if (c->gexec) cudaGraphExecDestroy(c->gexec);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  if (c->evFork) cudaEventDestroy(c->evFork);
  if (c->evJoin) cudaEventDestroy(c->evJoin);
  if (c->wstream) cudaStreamDestroy(c->wstream);
}

// Stable radix sort of (keys, vals); result pointers returned in *ko, *vo.
int radix_sort(sph_ctx* c, cudaStream_t st, int n, unsigned* kA, unsigned* vA, unsigned* kB, unsigned* vB,
               unsigned** ko, unsigned** vo, unsigned* hist = nullptr, unsigned* rowsum = nullptr) {
  if (!hist) { hist = c->hist; rowsum = c->rowsum; }
  unsigned *ki = kA, *vi = vA, *kt = kB, *vt = vB;
  if (n > 0) {
    const int items = rs_items((size_t)n), nblk = cdiv(n, RS_THREADS * items);
    for (int pass = 0; pass < c->sort_passes; ++pass) {
      int shift = c->sort_bits * pass;
#define RS_PASS(ND, IT)                                                                                   \
  do {                                                                                                    \
    LAUNCH((k_radix_hist<ND, IT>), nblk, RS_THREADS, st, ki, n, shift, hist, nblk, rowsum);               \
    LAUNCH(k_scan_apply, ND, 256, st, hist, nblk, rowsum);                                                \
    LAUNCH((k_radix_scatter<ND, IT>), nblk, RS_THREADS, st, ki, vi, n, shift, hist, nblk, kt, vt, rowsum); \
  } while (0)
      if (c->sort_bits == 9) { if (items == 4) RS_PASS(512, 4); else RS_PASS(512, 16); }
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

// wall extrapolation launcher (B = the fluid (v, rho - rho0) array the pressures are read from)
void launch_wall(sph_ctx* c, cudaStream_t st, bool with_vel, const XB* R) {
  if (c->nw == 0 || c->nf == 0) return;
  const int grid = cdiv(c->nw, PB), nw = (int)c->nw;
  if (with_vel) {
    WALL_DISPATCH(true, grid, st, c->dp, c->S, nw, c->WA, c->WR, c->WK, c->A, R, c->lbF, c->NLF, c->NCF, c->capsw);
  } else {
    WALL_DISPATCH(false, grid, st, c->dp, c->S, nw, c->WA, c->WR, c->WK, c->A, R, c->lbF, c->NLF, c->NCF, c->capsw);
  }
}

// NEXT-1 (moving walls): the walls at their positions of t^{n+1}, re-sorted into the cell grid (the
// same kernels as the set-up, on scratch of their own: `st` is the wall stream, which runs beside the
// fluid's predict / sort / reorder).
int wall_rebuild(sph_ctx* c, cudaStream_t st) {
  const int nw = (int)c->nw;
  if (nw == 0) return SPH_OK;
  LAUNCH(k_wall_shift, cdiv(nw, 256), 256, st, c->dp, c->S, nw, c->WX0, c->WTX, c->WTB, c->WkeyA, c->WvalA);
  unsigned *ks, *vs;
  int rc = radix_sort(c, st, nw, c->WkeyA, c->WvalA, c->WkeyB, c->WvalB, &ks, &vs, c->Whist, c->Wrowsum);
  if (rc) return rc;
  // gather + wall cell lower bounds in one launch, as for the fluid
  LAUNCH(k_reorder, std::max(cdiv(nw, 256), cdiv(c->ncell + 1, 256)), 256, st, c->dp, nw, vs, c->WTX, c->WTB, c->WID0,
         c->WR, c->WA, c->WID, ks, (int)c->ncell, c->lbW);
  CK(cudaMemcpyAsync(c->WK, ks, sizeof(unsigned) * nw, cudaMemcpyDeviceToDevice, st));
  LAUNCH(k_image, cdiv(nw, 256), 256, st, c->dp, nw, c->WR, c->WG);
  LAUNCH(k_gather4, cdiv(nw, 256), 256, st, nw, vs, c->WN0, c->WN);  // normals: translation-invariant
  LAUNCH(k_wnear, cdiv(c->ncell, 256), 256, st, c->dp, (int)c->ncell, c->lbW, c->wnear);
  return SPH_OK;
}

// Everything after the drift: sort, reorder, cell ranges, wall pass, pass A, wall pass, pass B.
int pipeline_after_hash(sph_ctx* c, cudaStream_t st, int init, Prof& pf) {
  const int nf = (int)c->nf;
  unsigned *ks, *vs;
  int rc = radix_sort(c, st, nf, c->keyA, c->valA, c->keyB, c->valB, &ks, &vs);
  if (rc) return rc;
  c->K = ks;
  pf.mark();  // end sort
  if (nf > 0) {
    // reorder + cell lower bounds in one launch; no pointer ping-pong: every step issues the same launches
    // with the same arguments (CUDA graph), k_build copies IDnext back to IDcur
    LAUNCH(k_reorder, std::max(cdiv(nf, 256), cdiv(c->ncell + 1, 256)), 256, st, c->dp, nf, vs, c->TX, c->TB, c->IDcur,
           c->R0, c->A, c->IDnext, ks, (int)c->ncell, c->lbF);
  } else {
    LAUNCH(k_cell_bounds, cdiv(c->ncell + 1, 256), 256, st, ks, nf, (int)c->ncell, c->lbF);
  }
  if (c->moving && !init && c->nw > 0) CK(cudaStreamWaitEvent(st, c->evJoin, 0));  // join the wall branch of one_step
  pf.mark();  // end reorder
  launch_wall(c, st, true, c->R0);
  pf.mark();  // end wall 1
  if (nf > 0) {
    switch (PAIR_SEL(c) & 5) {  // DIM x EXACT
      case 0: LAUNCH((k_build<2, false>), cdiv(nf, PB), PB, st, c->dp, c->S, nf, c->A, c->K, c->lbF, c->NL, c->NC, c->caps, c->WA, c->lbW, c->wnear, c->NLW, c->NCW, c->capsw, c->IDcur, c->IDnext); break;
      case 1: LAUNCH((k_build<2, true>), cdiv(nf, PB), PB, st, c->dp, c->S, nf, c->A, c->K, c->lbF, c->NL, c->NC, c->caps, c->WA, c->lbW, c->wnear, c->NLW, c->NCW, c->capsw, c->IDcur, c->IDnext); break;
      case 4: LAUNCH((k_build<3, false>), cdiv(nf, PB), PB, st, c->dp, c->S, nf, c->A, c->K, c->lbF, c->NL, c->NC, c->caps, c->WA, c->lbW, c->wnear, c->NLW, c->NCW, c->capsw, c->IDcur, c->IDnext); break;
      default: LAUNCH((k_build<3, true>), cdiv(nf, PB), PB, st, c->dp, c->S, nf, c->A, c->K, c->lbF, c->NL, c->NC, c->caps, c->WA, c->lbW, c->wnear, c->NLW, c->NCW, c->capsw, c->IDcur, c->IDnext); break;
    }
  }
  pf.mark();  // end list build
  if (nf > 0) {
    // third template parameter of k_pass_a: SUBQ (residuals in sigma), not the filter form
#undef PAIR_SEL
#define PAIR_SEL(c) (((c)->prm.dim == 3 ? 4 : 0) | ((c)->multi ? 2 : 0) | ((c)->dp.subq ? 1 : 0))
    PAIR_DISPATCH(k_pass_a, cdiv(nf, PB), st, c->dp, c->S, nf, init, c->A, c->R0, c->K, c->lbF, c->WA, c->WR,
                  c->lbW, c->wnear, c->R1, c->SIG, c->DRHO, c->NL, c->NC, c->caps, c->NLW, c->NCW, c->capsw);
  }
#undef PAIR_SEL
#define PAIR_SEL(c) (((c)->prm.dim == 3 ? 4 : 0) | ((c)->multi ? 2 : 0) | ((c)->dp.exact_filter ? 1 : 0))
  pf.mark();  // end pass A
  launch_wall(c, st, false, c->R1);
  pf.mark();  // end wall 2
  if (nf > 0) {
    PAIR_DISPATCH(k_pass_b, cdiv(nf, PB), st, c->dp, c->S, nf, c->A, c->R1, c->K, c->lbF, c->WA, c->WR,
                  c->WN, c->lbW, c->wnear, c->TB, c->ACC, c->NL, c->NC, c->caps, c->NLW, c->NCW, c->capsw);
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
  auto one_step = [&](cudaStream_t q, const double* seq, int s, Prof& pf) -> int {
    pf.mark();  // start
    LAUNCH(k_dt, dt_grid, 256, q, c->dp, c->S, nf, c->TB, seq, s);
    if (c->moving && c->nw > 0) {
      // NEXT-1: the wall re-sort needs the displacement of t^{n+1} (k_dt) and nothing of the fluid: fork
      // it onto the wall stream; pipeline_after_hash joins before the first wall pass.  Under capture
      // the events make it a parallel branch of the step graph.
      CK(cudaEventRecord(c->evFork, q));
      CK(cudaStreamWaitEvent(c->wstream, c->evFork, 0));
      int rcw = wall_rebuild(c, c->wstream);
      if (rcw) return rcw;
      CK(cudaEventRecord(c->evJoin, c->wstream));
    }
    if (nf > 0)
      LAUNCH(k_predict, cdiv(nf, 256), 256, q, c->dp, c->S, nf, c->R1, c->TB, c->ACC, c->SIG, c->TX, c->keyA, c->valA);
    pf.mark();  // end predict
    return pipeline_after_hash(c, q, 0, pf);
  };
  // Device-computed dt, no per-stage events: every step is the same launch sequence with the same
  // arguments, so it is captured once (on a private stream) and replayed as a CUDA graph.
  const bool use_graph = !dt_host && !c->prof && !(c->prm.flags & SPH_FLAG_NO_GRAPH) && n_steps > 0;
  if (use_graph && !c->gexec) {
    if (!c->cap_stream) CK(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
    CK(cudaStreamSynchronize(st));  // the capture stream is not ordered after st: drain st once
    const int64_t l0 = c->launches;
    CK(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    Prof pf(c, c->cap_stream);
    pf.on = false;
    int rc = one_step(c->cap_stream, nullptr, 0, pf);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
    c->graph_launches = c->launches - l0;
    c->launches = l0;
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) { c->err = std::string("graph capture: ") + cudaGetErrorString(e); return SPH_ECUDA; }
    e = cudaGraphInstantiate(&c->gexec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { c->gexec = nullptr; c->err = std::string("graph instantiate: ") + cudaGetErrorString(e); return SPH_ECUDA; }
  }
  for (int s = 0; s < n_steps; ++s) {
    if (use_graph) {
      CK(cudaGraphLaunch(c->gexec, st));
      c->launches += c->graph_launches;
      continue;
    }
    Prof pf(c, st);
    int rc = one_step(st, dt_host ? c->dt_seq : nullptr, s, pf);
    if (rc) return rc;
    pf.done();
  }
  return SPH_OK;
}

// float32 images of the current fluid positions for the contract-exact debug walks (scratch: TX)
float4* fluid_images(sph_ctx* c, cudaStream_t st) {
  float4* G = reinterpret_cast<float4*>(c->TX);
  if (c->nf) LAUNCH(k_image, cdiv(c->nf, 256), 256, st, c->dp, (int)c->nf, c->R1, G);
  return G;
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
    d.Qf = (float)d.Q; d.qh = (float)(d.Q / h); d.qhD = d.Q / h;
    d.mhqD[0] = -0.5 * d.qhD; d.mhqD[1] = d.mhqD[0] / 1024.0; d.tqD[0] = 2.0 * d.qhD; d.tqD[1] = d.tqD[0] / 1024.0;
    // sigma from residual-exact separations (k_pass_a<.., SUBQ>) when the quantum is coarse for the case: the
    // acceleration error from positions rounded to Q is about 15 (Q / h) (L / h) g (measured: 5.5e-4 g at
    // config 4's 16.8 M size, Q / h = 1.4e-7, L / h = 200), so the 1e-4 bar needs (Q / h)(L / h) < 2e-6
    d.subq = (prm->n_phases > 1 || (d.Q / h) * (Lmax / h) > 2e-6 || getenv("SPH_FORCE_SUBQ")) ? 1 : 0;
    if (getenv("SPH_NO_SUBQ") && prm->n_phases == 1) d.subq = 0;
    d.gradcQ = (float)(-5.0 * alpha / (h * h) * d.Q);
    d.two_over_dp = (float)(2.0 * d.Q / dp);
    // candidate filter margin: rounding of the expanded form |xj|^2 - 2 xi.xj + |xi|^2 on images
    // of magnitude <= R, plus the rounding of the images themselves
    const double R = sqrt(R2), u = ldexp(1.0, -24);
    const double err_expanded = 16.0 * u * R2 + 8.0 * u * R * rc;
    const double err_diff = 16.0 * u * R * rc;
    d.exact_filter = 2.0 * err_expanded > 0.08 * rc * rc ? 1 : 0;
    d.rc2m = (float)(rc * rc + 2.0 * (d.exact_filter ? err_diff : err_expanded));
    {  // float16 filter of k_build (sph_pair.cuh): threshold rounded up to the next half
      d.inv_h = (float)(1.0 / h);
      const double thr = 4.08 + 2.0 * err_diff / (h * h);
      __half th = __double2half(thr);
      if ((double)__half2float(th) < thr) th = __ushort_as_half((unsigned short)(__half_as_ushort(th) + 1));
      d.thr_h2 = (unsigned)__half_as_ushort(th) * 0x10001u;
    }
  }
  d.gamma_p = (float)prm->penalty_strength;
  d.pen_mask = (prm->flags & SPH_FLAG_WALL_ADAMI_ONLY) ? 0u : prm->penalty_phase_mask; d.fs_mask = prm->free_surface_mask; d.flags = prm->flags;
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
  for (int k = 0; k < 3; ++k) d.wamp[k] = k < prm->dim ? prm->wall_osc_amp[k] : 0.0;
  d.womega = 6.283185307179586476925286766559 * prm->wall_osc_freq;
  c->moving = prm->wall_osc_freq > 0.0 && (d.wamp[0] != 0.0 || d.wamp[1] != 0.0 || d.wamp[2] != 0.0);
  if (!c->moving) { d.womega = 0.0; d.wamp[0] = d.wamp[1] = d.wamp[2] = 0.0; }
  d.gperiod = prm->g_osc_period; d.cmax = cmax; d.cfl = prm->cfl; d.hD = h; d.dpD = dp;
  c->ncell = (int64_t)nc[0] * nc[1] * nc[2];
  if (c->ncell >= (1ll << 31) - 2) { delete c; return SPH_EINVAL; }
  int bits = 1;
  while ((1ll << bits) < c->ncell) ++bits;
  c->sort_bits = (bits + 8) / 9 < (bits + 7) / 8 ? 9 : 8;
  c->sort_passes = (bits + c->sort_bits - 1) / c->sort_bits;
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
  if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }  // buffers are reallocated below
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
  rc |= dalloc(c, &c->R0, nf); rc |= dalloc(c, &c->R1, nf); rc |= dalloc(c, &c->TX, cap); rc |= dalloc(c, &c->A, (size_t)nf + 16);
  rc |= dalloc(c, &c->TB, cap);
  rc |= dalloc(c, &c->ACC, nf); rc |= dalloc(c, &c->SIG, nf); rc |= dalloc(c, &c->DRHO, nf);
  c->npad = ((size_t)nf + PB - 1) / PB * PB;
  c->caps = c->prm.max_neighbours ? (int)((c->prm.max_neighbours + 3u) & ~3u) : (c->prm.dim == 3 ? 160 : 64);
  rc |= dalloc(c, &c->NL, c->npad * (size_t)(c->caps >> 2)); rc |= dalloc(c, &c->NC, nf);
  c->capsw = (c->caps * 3 / 4 + 3) & ~3;  // a particle in a corner of three walls has 7/8 of its (then smaller) support in them
  rc |= dalloc(c, &c->NLW, c->npad * (size_t)(c->capsw >> 2)); rc |= dalloc(c, &c->NCW, nf);
  rc |= dalloc(c, &c->NLF, ((size_t)nw + PB - 1) / PB * PB * (size_t)(c->capsw >> 2)); rc |= dalloc(c, &c->NCF, nw);
  rc |= dalloc(c, &c->ID0, cap); rc |= dalloc(c, &c->ID1, cap);
  rc |= dalloc(c, &c->keyA, cap); rc |= dalloc(c, &c->valA, cap); rc |= dalloc(c, &c->keyB, cap);
  rc |= dalloc(c, &c->valB, cap);
  rc |= dalloc(c, &c->hist, (size_t)512 * std::max(cdiv(std::max(nf, 1), RS_THREADS * rs_items((size_t)nf)),
                                                  cdiv(std::max(nw, 1), RS_THREADS * rs_items((size_t)nw))));
  rc |= dalloc(c, &c->rowsum, 512);
  if (!rc) CK(cudaMemsetAsync(c->rowsum, 0, 512 * sizeof(unsigned), (cudaStream_t)stream));  // radix digit totals: zero between passes
  rc |= dalloc(c, &c->lbF, c->ncell + 1); rc |= dalloc(c, &c->lbW, c->ncell + 1);
  rc |= dalloc(c, &c->wnear, c->ncell);
  rc |= dalloc(c, &c->WR, nw); rc |= dalloc(c, &c->WA, (size_t)nw + 16);
  rc |= dalloc(c, &c->WN, nw); rc |= dalloc(c, &c->WG, nw); rc |= dalloc(c, &c->WK, nw);
  rc |= dalloc(c, &c->WID, nw);
  rc |= dalloc(c, &c->S, 1); rc |= dalloc(c, &c->stat, 1);
  if (rc) return c->err.find("out of memory") != std::string::npos ? SPH_ENOMEM : SPH_ECUDA;
  c->IDcur = c->ID0; c->IDnext = c->ID1;
  CK(cudaMemsetAsync(c->S, 0, sizeof(SS), st));
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
  if (dalloc(c, &c->hidx, std::max<size_t>(cap, 1))) return SPH_ECUDA;  // kept across calls
  int* idx = c->hidx;
  // ---- wall structure, built once ----
  if (nw > 0) {
    CK(cudaMemcpyAsync(idx, wid.data(), sizeof(int) * nw, cudaMemcpyHostToDevice, st));
    LAUNCH(k_load, cdiv(nw, 256), 256, st, c->dp, nw, 1, idx, pos, vel, rho, tag, c->TX, c->TB, c->ID0, c->keyA, c->valA);
    if (c->moving) {  // NEXT-1: keep the set-up order for the per-step re-sort
      rc = dalloc(c, &c->WX0, nw) | dalloc(c, &c->WN0, nw) | dalloc(c, &c->WID0, nw) | dalloc(c, &c->WkeyA, nw) | dalloc(c, &c->WkeyB, nw) |
           dalloc(c, &c->WvalA, nw) | dalloc(c, &c->WvalB, nw) | dalloc(c, &c->WTX, nw) | dalloc(c, &c->WTB, nw) |
           dalloc(c, &c->Whist, (size_t)512 * cdiv(nw, RS_THREADS * rs_items((size_t)nw))) | dalloc(c, &c->Wrowsum, 512);
      if (rc) return rc;
      CK(cudaMemsetAsync(c->Wrowsum, 0, 512 * sizeof(unsigned), st));
      if (!c->wstream) CK(cudaStreamCreateWithFlags(&c->wstream, cudaStreamNonBlocking));
      if (!c->evFork) CK(cudaEventCreateWithFlags(&c->evFork, cudaEventDisableTiming));
      if (!c->evJoin) CK(cudaEventCreateWithFlags(&c->evJoin, cudaEventDisableTiming));
      CK(cudaMemcpyAsync(c->WX0, c->TX, sizeof(uint4) * nw, cudaMemcpyDeviceToDevice, st));
      CK(cudaMemcpyAsync(c->WID0, c->ID0, sizeof(unsigned) * nw, cudaMemcpyDeviceToDevice, st));
    }
    unsigned *ks, *vs;
    rc = radix_sort(c, st, nw, c->keyA, c->valA, c->keyB, c->valB, &ks, &vs);
    if (rc) return rc;
    LAUNCH(k_reorder, cdiv(nw, 256), 256, st, c->dp, nw, vs, c->TX, c->TB, c->ID0, c->WR, c->WA, c->WID,
           (const unsigned*)nullptr, -1, (int*)nullptr);
    CK(cudaMemcpyAsync(c->WK, ks, sizeof(unsigned) * nw, cudaMemcpyDeviceToDevice, st));
    LAUNCH(k_image, cdiv(nw, 256), 256, st, c->dp, nw, c->WR, c->WG);
    LAUNCH(k_cell_bounds, cdiv(c->ncell + 1, 256), 256, st, ks, nw, (int)c->ncell, c->lbW);
    if (c->prm.dim == 3) LAUNCH(k_normals<3>, cdiv(nw, 128), 128, st, c->dp, nw, c->WR, c->WK, c->lbW, c->WN);
    else LAUNCH(k_normals<2>, cdiv(nw, 128), 128, st, c->dp, nw, c->WR, c->WK, c->lbW, c->WN);
    if (c->moving) LAUNCH(k_unsort4, cdiv(nw, 256), 256, st, nw, vs, c->WN, c->WN0);
  } else {
    LAUNCH(k_cell_bounds, cdiv(c->ncell + 1, 256), 256, st, c->keyA, 0, (int)c->ncell, c->lbW);
  }
  LAUNCH(k_wnear, cdiv(c->ncell, 256), 256, st, c->dp, (int)c->ncell, c->lbW, c->wnear);
  CK(cudaStreamSynchronize(st));  // wid host buffer / idx reuse
  // ---- fluid: load, then the common pipeline in init mode (dt = 0: sigma_i, p_w, (dv/dt)^0) ----
  if (nf > 0) {
    CK(cudaMemcpyAsync(idx, fid.data(), sizeof(int) * nf, cudaMemcpyHostToDevice, st));
    LAUNCH(k_load, cdiv(nf, 256), 256, st, c->dp, nf, 0, idx, pos, vel, rho, tag, c->TX, c->TB, c->IDcur, c->keyA, c->valA);
  }
  Prof pf(c, st);
  pf.on = false;
  rc = pipeline_after_hash(c, st, 1, pf);
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
  int rc = dalloc(c, &c->hpos, m * 3) | dalloc(c, &c->hvel, m * 3) | dalloc(c, &c->hrho, m) | dalloc(c, &c->htagd, m);
  if (rc) return rc;
  float *dpos = c->hpos, *dvel = c->hvel, *drho = c->hrho;
  int32_t* dtag = c->htagd;
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
  if (dalloc(c, &c->hout, n * 11)) return SPH_ECUDA;  // kept across calls
  float* buf = c->hout;
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
  if (rc) return rc;
  if (e != cudaSuccess || e2 != cudaSuccess) {
    c->err = cudaGetErrorString(e != cudaSuccess ? e : e2);
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
      const float4* G = fluid_images(c, st);
      LAUNCH(k_neigh, cdiv(nf, PW), PW * 32, st, c->dp, nf, 0, 0, G, c->IDcur, G, c->IDcur, c->lbF, c->WG,
             c->WID, c->lbW, (int*)nullptr, (const long long*)nullptr, (int*)nullptr, 0ll, &c->stat->pairs);
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

int sph_get_timings(sph_ctx* c, float* ms, int32_t* n_steps) {
  if (!c || !ms || !n_steps) return SPH_EINVAL;
  for (int k = 0; k < SPH_STAGE_COUNT; ++k) ms[k] = 0.f;
  *n_steps = c->ev_steps;
  if (c->ev_steps == 0) return SPH_OK;
  CK(cudaEventSynchronize(c->ev[(c->ev_steps - 1) * sph_ctx::EV_PER_STEP + 8]));
  // marks per step: 0 start, 1 predict, 2 sort, 3 reorder, 4 wall1, 5 list build, 6 passA, 7 wall2, 8 passB
  static const int stage_of[8] = {SPH_STAGE_PREDICT, SPH_STAGE_SORT, SPH_STAGE_REORDER, SPH_STAGE_WALL, SPH_STAGE_BUILD,
                                  SPH_STAGE_PASS_A, SPH_STAGE_WALL, SPH_STAGE_PASS_B};
  for (int s = 0; s < c->ev_steps; ++s)
    for (int k = 0; k < 8; ++k) {
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
  const float4* G = fluid_images(c, st);
  if (c->nf) LAUNCH(k_dbg_cells, cdiv(c->nf, 256), 256, st, c->dp, (int)c->nf, G, c->IDcur, dcid, dperm, 0);
  if (c->nw) LAUNCH(k_dbg_cells, cdiv(c->nw, 256), 256, st, c->dp, (int)c->nw, c->WG, c->WID, dcid, dperm, (int)c->nf);
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
  const float4* G = fluid_images(c, st);
  auto run = [&](int mode, const long long* doff, int* dids, long long dcap) {
    if (c->nf)
      LAUNCH(k_neigh, cdiv(c->nf, PW), PW * 32, st, c->dp, (int)c->nf, 0, mode, G, c->IDcur, G, c->IDcur, c->lbF,
             c->WG, c->WID, c->lbW, dcnt, doff, dids, dcap, (unsigned long long*)nullptr);
    if (c->nw && c->nf)
      LAUNCH(k_neigh, cdiv(c->nw, PW), PW * 32, st, c->dp, (int)c->nw, 1, mode, c->WG, c->WID, G, c->IDcur, c->lbF,
             c->WG, c->WID, c->lbW, dcnt, doff, dids, dcap, (unsigned long long*)nullptr);
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
