// =====================================================================================
// gfcc_lib.cu -- C ABI of the B200-native GFCCSD-IP hot path (see include/gfcc.h).
//
//   gfcc_create   : SURVEY.md 8a P1-P7  (one-time intermediates)
//   gfcc_sigma_ip : SURVEY.md 8a S1-S13 (batched sigma, Eq. 5, Alg. 1)
//   gfcc_solve_ip : SURVEY.md 8a G1-G6  (batched GMRES PAPER.md:136-138 + G assembly PAPER.md:89-94)
//
// Every O(N^5)/O(N^6) contraction is a real FP64 GEMM on the DMMA engine of gfcc_gemm.cuh with the RHS
// batch folded into N; the (ov x ov) ring/exchange integrals are streamed through bounded panels built
// on the fly from the Cholesky vectors (never stored; BASELINE.json configs[2..4]).  No CPU fallback.
// =====================================================================================
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <mutex>
#include <vector>
#include <algorithm>

#include "../../include/gfcc.h"
#include "gfcc_gemm.cuh"
#include "gfcc_gemm_ws.cuh"
#include "gfcc_kernels.cuh"
#include "gfcc_solve.cuh"
#include "gfcc_probe.cuh"
#include "gfcc_mor.cuh"
#include "gfcc_ozaki.cuh"
#include "gfcc_ea.cuh"

using namespace gfcc;

// NVTX range per sigma term / create phase / solver phase (the paper times get / compute / add per
// iteration, Table 4; here the phases are the rows of SURVEY.md 8a).  Header-only NVTX v3: a no-op unless a
// profiler is attached.
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};

static thread_local std::string g_create_error;

struct EaState;   // EA / advanced part (gfcc_ea_host.inl), created on first use
static void ea_destroy(struct gfcc_ctx* h);
static void ea_release_ws(struct gfcc_ctx* h);

struct gfcc_ctx {
  EaState* ea = nullptr;
  int o = 0, v = 0, Q = 0, N = 0;
  long long npair = 0, ntri = 0, nvec = 0;   // nvec = o + npair*v (rows of an internal vector)
  cudaStream_t stream = 0;
  cudaStream_t cur = 0;              // stream the next gemm()/kernel launch goes to (== stream outside sigma_internal)
  cudaStream_t sB = nullptr, sC = nullptr;   // side streams: K4/V panel chain, small sigma terms (overlap with the K2 chain)
  cudaEvent_t evFork = nullptr, evB = nullptr, evC = nullptr;
  std::string err;
  std::vector<void*> allocs;
  double bytes = 0;
  // ---- intermediates (device) ----
  double *Lov = nullptr, *LooT = nullptr, *Lvv = nullptr, *Lm = nullptr;   // [Q][o][v], [Q][i][m], [Q][a][e], [Q][i][a]
  double *Fme = nullptr, *Fmi = nullptr, *Fae = nullptr, *fdiag = nullptr;
  double *Wp = nullptr;    // W_mnij  packed [(i<j)][(m<n)]
  double *WB = nullptr;    // W_mbij  packed [(i<j)][a][m] = W[m,a,j,i]
  double *D = nullptr, *t1 = nullptr, *l1 = nullptr;
  const double *T2p = nullptr, *L2p = nullptr;   // borrowed
  long long* blk_tab = nullptr;   // [o][o] element offset of the T2 block of the pair {i,n}
  double* blk_sgn = nullptr;      // [o][o] +1 (i<n), -1 (i>n), 0 (i==n)
  // ---- workspace, sized for ws_nrhs ----
  int ws_nrhs = 0;
  double *XU = nullptr, *Z = nullptr, *V = nullptr, *Y = nullptr, *KP = nullptr, *KP2 = nullptr, *yv = nullptr, *part = nullptr, *d_omega = nullptr;
  double *vin = nullptr, *vout = nullptr;   // internal vectors for gfcc_sigma_ip
  long long part_elems = 0;
  int panel_ni = 1;
  // ---- INT8 tensor-core (Ozaki) engine for S8-S11 (gfcc_ozaki.cuh, gfcc_ozaki_host.inl; option "engine" = 1) ----
  int opt_engine = 0, opt_oz_slices = 7;
  OzSliced ozLvv, ozLooT, ozLov, ozXU, ozKP, ozWp;
  double* ozS6scale = nullptr; long long ozS6rows = 0;
  int* oz_fail = nullptr;
  bool oz_const_ready = false;
  int oz_ws_nrhs = 0, oz_ws_ni = 0;
  double st_oz_gemms = 0;
  // ---- options / stats ----
  double opt_m = 50, opt_maxit = 1000, opt_fixed = 0, opt_x0 = 1, opt_panel_bytes = 0 /* 0 = automatic, see panel_budget() */, opt_max_batch = 256, opt_overlap = 0;
  double opt_compact = 0.125, opt_poll = 0, opt_graph = -1, opt_dense = -1;
  // ---- dense Hbar_IP (n x n, row-major) for tiny systems: sigma inside the solver = one GEMM + a shift kernel ----
  double* Hd = nullptr; bool hd_ready = false;
  double st_dense_apps = 0;
  // ---- CUDA graphs of one sigma application for latency-bound (tiny) systems, keyed by the batch width ----
  struct SigmaGraph { int nrhs; const double* d_omega; double eta; cudaGraphExec_t exec; size_t nodes; };
  std::vector<SigmaGraph> graphs;
  double *gx = nullptr, *gy = nullptr; long long g_elems = 0;
  double st_graph_launches = 0;
  double st_iterations = 0, st_sigma_apps = 0, st_flops_sigma = 0, st_flops_create = 0, st_max_relres = 0, st_nunconv = 0;
  double st_gemm_launches = 0, st_kernel_launches = 0, st_flops_exec = 0;
  std::vector<double> last_relres;
  std::vector<int> last_iters;
  std::vector<std::vector<double>> last_hist;   // per right-hand side: relative residual after every sigma application
  SolveWs sw;
  // ---- MOR subspace: S, Hbar*S as [n_pad][cap] real, H^ as [cap][cap] ----
  int mor_cap = 0, mor_m = 0;
  long long mor_npad = 0;
  double *mor_S = nullptr, *mor_HS = nullptr, *mor_Hh = nullptr;
  double st_mor_dropped = 0, st_mor_sigma_cols = 0;
  // ---- optional per-launch timing of the GEMM engine (CUDA events on the handle's stream; bench.py roofline) ----
  bool prof = false;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;
  std::vector<double> ev_flops;   // flops of the launch bracketed by events (2k, 2k+1)
  std::vector<double> ev_ops8;    // int8 multiply-add operations x2 of that launch (0 for an FP64 DMMA launch)
};

#define CUDA_TRY(h, expr)                                                                      \
  do {                                                                                         \
    cudaError_t e__ = (expr);                                                                  \
    if (e__ != cudaSuccess) {                                                                  \
      char buf__[512];                                                                         \
      snprintf(buf__, sizeof buf__, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
      (h)->err = buf__;                                                                        \
      return (e__ == cudaErrorMemoryAllocation) ? GFCC_ENOMEM : GFCC_ECUDA;                    \
    }                                                                                          \
  } while (0)
#define TRY(expr) do { int rc__ = (expr); if (rc__ != GFCC_OK) return rc__; } while (0)
#define KLAUNCH(h) do { (h)->st_kernel_launches += 1; CUDA_TRY(h, cudaGetLastError()); } while (0)

static int dev_alloc(gfcc_ctx* h, double** p, long long elems) {
  if (elems <= 0) elems = 1;
  void* q = nullptr;
  cudaError_t e = cudaMalloc(&q, (size_t)elems * sizeof(double));
  if (e != cudaSuccess) {
    char buf[256];
    snprintf(buf, sizeof buf, "cudaMalloc of %.3f GB failed: %s", elems * 8e-9, cudaGetErrorString(e));
    h->err = buf;
    cudaGetLastError();
    return GFCC_ENOMEM;
  }
  h->allocs.push_back(q);
  h->bytes += (double)elems * 8;
  *p = (double*)q;
  return GFCC_OK;
}
static void dev_free(gfcc_ctx* h, double* p, long long elems) {
  if (!p) return;
  for (size_t k = 0; k < h->allocs.size(); ++k)
    if (h->allocs[k] == (void*)p) { h->allocs.erase(h->allocs.begin() + k); break; }
  cudaFree(p);
  h->bytes -= (double)std::max(elems, 1LL) * 8;
}

static int gemm(gfcc_ctx* h, const GemmDesc& d) {
  const bool timed = h->prof && d.M > 0 && d.N > 0 && d.K0 > 0;
  if (timed) {
    while (h->ev_pool.size() < h->ev_used + 2) { cudaEvent_t e; CUDA_TRY(h, cudaEventCreate(&e)); h->ev_pool.push_back(e); }
    CUDA_TRY(h, cudaEventRecord(h->ev_pool[h->ev_used], h->cur));
  }
  CUDA_TRY(h, launch_dgemm(d, h->cur));
  if (timed) {
    CUDA_TRY(h, cudaEventRecord(h->ev_pool[h->ev_used + 1], h->cur));
    h->ev_used += 2;
    h->ev_flops.push_back(2.0 * d.M * (double)d.N * (double)d.K1 * d.K0 * d.batch);
    h->ev_ops8.push_back(0.0);
  }
  h->st_gemm_launches += 1;
  h->st_kernel_launches += 1;
  h->st_flops_exec += 2.0 * d.M * (double)d.N * (double)d.K1 * d.K0 * d.batch;
  return GFCC_OK;
}

// split the K1 blocks of a GEMM over S batches, partial sums in h->part, deterministic reduction
static int gemm_splitk(gfcc_ctx* h, GemmDesc d, int S) {
  S = std::max(1, std::min(S, d.K1));
  const long long need = (long long)S * d.M * d.N;
  // (a short reduction gains nothing from the split and costs two more launches: the small systems are latency-bound)
  if (S == 1 || d.batch != 1 || d.tabA || d.tabB || d.sgn || need > h->part_elems || (long long)d.K1 * d.K0 <= 2048) return gemm(h, d);
  const int chunk = (d.K1 + S - 1) / S;
  // K1 blocks [z*chunk, min(K1,(z+1)*chunk)): launch full chunks as one batched GEMM, the ragged tail separately
  const int full = d.K1 / chunk;            // batches with exactly `chunk` blocks
  const int tail = d.K1 - full * chunk;     // blocks in the last partial batch
  GemmDesc g = d;
  g.C = h->part; g.sCm0 = d.N; g.sCm1 = 0; g.Md = d.M; g.sCn0 = 1; g.sCn1 = 0; g.Nd = d.N;
  g.alpha = 1.0; g.beta = 0.0;
  g.K1 = chunk; g.batch = full;
  g.bsA = (long long)chunk * d.sAk1; g.bsB = (long long)chunk * d.sBk1; g.bsC = (long long)d.M * d.N;
  if (full > 0) TRY(gemm(h, g));
  int nparts = full;
  if (tail > 0) {
    GemmDesc t = g;
    t.K1 = tail; t.batch = 1;
    t.A = d.A + (long long)full * chunk * d.sAk1;
    t.B = d.B + (long long)full * chunk * d.sBk1;
    t.C = h->part + (long long)full * d.M * d.N;
    TRY(gemm(h, t));
    ++nparts;
  }
  const long long tot = (long long)d.M * d.N;
  k_splitk_reduce<<<(unsigned)((tot + 255) / 256), 256, 0, h->cur>>>(d.C, h->part, nparts, d.M, d.N, d.alpha, d.beta, d.sCm0,
                                                                      d.sCm1, d.Md > 0 ? d.Md : d.M, d.sCn0, d.sCn1,
                                                                      d.Nd > 0 ? d.Nd : d.N);
  KLAUNCH(h);
  return GFCC_OK;
}

static inline unsigned nblk(long long n, int t = 256, long long cap = 148LL * 32) {
  long long b = (n + t - 1) / t;
  return (unsigned)std::max(1LL, std::min(b, cap));
}

// ------------------------------------------------------------------------------------------
// workspace for a batch of nrhs right-hand sides
// ------------------------------------------------------------------------------------------
#include "gfcc_ozaki_host.inl"

static void graphs_clear(gfcc_ctx* h) {
  for (auto& g : h->graphs) cudaGraphExecDestroy(g.exec);
  h->graphs.clear();
  dev_free(h, h->gx, h->g_elems); dev_free(h, h->gy, h->g_elems);
  h->gx = h->gy = nullptr; h->g_elems = 0;
}

static void free_workspace(gfcc_ctx* h) {
  const int o = h->o, v = h->v;
  graphs_clear(h);   // the captured launches hold pointers into this workspace
  oz_free_ws(h);
  const long long Nc = 2LL * h->ws_nrhs, big = (long long)o * v * o * Nc;
  dev_free(h, h->XU, big); dev_free(h, h->Z, big); dev_free(h, h->V, big);
  dev_free(h, h->Y, (long long)h->Q * o * Nc);
  dev_free(h, h->KP, (long long)h->panel_ni * v * o * v);
  dev_free(h, h->KP2, (long long)h->panel_ni * v * o * v);
  dev_free(h, h->yv, (long long)v * Nc);
  dev_free(h, h->d_omega, h->ws_nrhs);
  dev_free(h, h->vin, h->nvec * Nc); dev_free(h, h->vout, h->nvec * Nc);
  h->XU = h->Z = h->V = h->Y = h->KP = h->KP2 = h->yv = h->d_omega = h->vin = h->vout = nullptr;
  h->ws_nrhs = 0;
}

// byte budget of one panel scratch: the "panel_bytes" option when set, else 12.8 GB for the sigma workspace of the DMMA engine
// (20 occupied indices per panel at config 4: 33.9 TFLOP/s per step against 33.5 with 5 -- the K2 panel build then fills its
// 96-row tiles) and 3.2 GB for everything else (create-time scratch, EA panels, INT8 engine)
static double panel_budget(const gfcc_ctx* h, bool sigma_dmma) {
  return h->opt_panel_bytes > 0 ? h->opt_panel_bytes : (sigma_dmma ? 12.8e9 : 3.2e9);
}
// choose how many occupied indices one (ov x ov) panel covers: as many as the byte budget allows, preferring
// counts whose consuming GEMM fills whole waves of 148 CTAs.
static int choose_panel(int o, int v, long long ncols, double budget_bytes) {
  const double row_bytes = (double)o * v * 8.0;
  int nmax = (int)std::min<double>(o, std::floor(budget_bytes / (row_bytes * v)));
  if (nmax < 1) nmax = 1;
  int best = nmax; double best_eff = -1;
  const int tiles_n = (int)((ncols + GEMM_BN - 1) / GEMM_BN);
  for (int n = nmax; n >= std::max(1, nmax / 2); --n) {
    const int rows = n * v;
    const int bm = gemm_bm(rows, ncols);
    const long long tiles = (long long)((rows + bm - 1) / bm) * tiles_n;
    const long long waves = (tiles + 147) / 148;
    const double eff = (double)rows * ncols / ((double)waves * 148 * bm * GEMM_BN);
    if (eff > best_eff + 1e-9) { best_eff = eff; best = n; }
  }
  return best;
}

// The workspace holds room for ws_nrhs right-hand sides and serves every batch of at most that many (the solver shrinks
// its batch when right-hand sides converge).  ws_nrhs is committed only when every allocation has succeeded; a failed
// allocation releases whatever the call had obtained, so the handle never keeps a half-built workspace.
static int ensure_workspace(gfcc_ctx* h, int nrhs, bool need_abi_vecs) {
  const int o = h->o, v = h->v, Q = h->Q;
  if (h->ws_nrhs < nrhs) {
    if (h->ws_nrhs) { cudaStreamSynchronize(h->stream); free_workspace(h); }
    const long long Nc = 2LL * nrhs, big = (long long)o * v * o * Nc;
    h->panel_ni = h->opt_engine == 1 ? oz_choose_panel(o, v, (long long)o * Nc, panel_budget(h, false))
                                     : choose_panel(o, v, (long long)o * Nc, panel_budget(h, true));
    h->ws_nrhs = nrhs;   // free_workspace() sizes its bookkeeping with it; reset to 0 there if anything below fails
    int rc = GFCC_OK;
    do {
      if ((rc = dev_alloc(h, &h->XU, big))) break;
      if ((rc = dev_alloc(h, &h->Z, big))) break;
      if ((rc = dev_alloc(h, &h->V, big))) break;
      if ((rc = dev_alloc(h, &h->Y, (long long)Q * o * Nc))) break;
      if ((rc = dev_alloc(h, &h->KP, (long long)h->panel_ni * v * o * v))) break;
      if (h->opt_overlap != 0 && (rc = dev_alloc(h, &h->KP2, (long long)h->panel_ni * v * o * v))) break;
      if ((rc = dev_alloc(h, &h->yv, (long long)v * Nc))) break;
      if ((rc = dev_alloc(h, &h->d_omega, nrhs))) break;
    } while (0);
    if (rc != GFCC_OK) { free_workspace(h); return rc; }
  }
  if (need_abi_vecs && !h->vin) {
    const long long Nc = 2LL * h->ws_nrhs;
    double *a = nullptr, *b = nullptr;
    int rc = dev_alloc(h, &a, h->nvec * Nc);
    if (rc == GFCC_OK && (rc = dev_alloc(h, &b, h->nvec * Nc)) != GFCC_OK) dev_free(h, a, h->nvec * Nc);
    if (rc != GFCC_OK) return rc;
    h->vin = a; h->vout = b;
  }
  return GFCC_OK;
}

// ------------------------------------------------------------------------------------------
// sigma on internal vectors:  sout = (omega - i eta) xin + Hbar xin
// d_omega: device [nrhs].  xin, sout: [nvec][Nc].
// ------------------------------------------------------------------------------------------
static int sigma_internal(gfcc_ctx* h, int nrhs, const double* d_omega, double eta, const double* xin, double* sout) {
  const int o = h->o, v = h->v, Q = h->Q;
  const long long Nc = 2LL * nrhs, ld = (long long)o * Nc, ov = (long long)o * v;
  const double* x2 = xin + (long long)o * Nc;
  double* s2 = sout + (long long)o * Nc;
  // Three independent chains (the paper's "levelizer" exposes the same op-level parallelism):
  //   A (handle stream): S7, then K2 panels -> Z        B (side stream): K4 panels -> V
  //   C (side stream)  : sigma1, S6, S12, S5 -> sout
  // Every GEMM CTA owns a whole SM, so running the chains on separate streams lets the block scheduler fill the
  // ragged last wave of one panel GEMM with CTAs of another chain.  With per-launch GEMM timing on (profile_gemm)
  // the chains are serialised on the handle's stream so that the event brackets do not overlap.
  const bool oz = h->opt_engine == 1;
  const bool par = !oz && h->opt_overlap != 0 && !h->prof && h->sB && h->sC && h->KP2;
  cudaStream_t s0 = h->stream, sB = par ? h->sB : s0, sC = par ? h->sC : s0;
  double* KPb = par ? h->KP2 : h->KP;
  struct Restore { gfcc_ctx* h; ~Restore() { h->cur = h->stream; } } restore{h};

  NvtxRange nv_sigma("gfcc sigma (S1-S13)");
  h->cur = s0;
  // XU[m][e][j][c] = x2[m,j,e]
  k_unpack_xu<<<(unsigned)(h->npair + o), 256, 0, s0>>>(h->XU, xin, o, v, (int)Nc);
  KLAUNCH(h);
  // S1: Y[Q][(j,c)] = sum_(m,e) Lov[Q][(m,e)] XU[(m,e)][(j,c)]
  {
    NvtxRange nv("S1 Y = Lov XU");
    GemmDesc d; d.M = Q; d.N = (int)ld; d.K0 = (int)ov;
    d.A = h->Lov; d.sAm = ov; d.sAk0 = 1;
    d.B = h->XU; d.sBk0 = ld; d.sBn = 1;
    d.C = h->Y; d.sCm0 = ld;
    TRY(gemm(h, d));
  }
  if (par) {
    CUDA_TRY(h, cudaEventRecord(h->evFork, s0));
    CUDA_TRY(h, cudaStreamWaitEvent(sB, h->evFork, 0));
    CUDA_TRY(h, cudaStreamWaitEvent(sC, h->evFork, 0));
  }
  // S7: Z[(i,a)][(j,c)] = sum_Q Lm[Q][(i,a)] Y[Q][(j,c)]
  {
    NvtxRange nv("S7 Z13 = Lm^T Y");
    GemmDesc d; d.M = (int)ov; d.N = (int)ld; d.K0 = Q;
    d.A = h->Lm; d.sAm = 1; d.sAk0 = ov;
    d.B = h->Y; d.sBk0 = ld; d.sBn = 1;
    d.C = h->Z; d.sCm0 = ld;
    TRY(gemm(h, d));
  }
  if (oz) TRY(sigma_ring_ozaki(h, nrhs));
  for (int i0 = 0; i0 < o && !oz; i0 += h->panel_ni) {
    const int ni = std::min(h->panel_ni, o - i0);
    NvtxRange nv_panel("S8-S10 panel (K2 build, Z -= K2 XU, K4 build, V = K4 XU)");
    // ---- chain A: S8+S9 (+S3,S4 folded): panel of K2'[(i,a)][(m,e)], Z -= K2' XU
    h->cur = s0;
    {
      GemmDesc d; d.M = ni * o; d.N = v * v; d.K0 = Q;
      d.A = h->LooT + (long long)i0 * o; d.sAm = 1; d.sAk0 = (long long)o * o;
      d.B = h->Lvv; d.sBk0 = (long long)v * v; d.sBn = 1;
      d.C = h->KP; d.Md = o; d.sCm1 = (long long)v * ov; d.sCm0 = v; d.Nd = v; d.sCn1 = ov; d.sCn0 = 1;
      TRY(gemm(h, d));
    }
    k_k2_fixup<<<(unsigned)(ni * v), 128, 0, s0>>>(h->KP, h->Fmi, h->Fae, o, v, i0);
    KLAUNCH(h);
    {
      GemmDesc d; d.M = ni * v; d.N = (int)ld; d.K0 = (int)ov;
      d.A = h->KP; d.sAm = ov; d.sAk0 = 1;
      d.B = h->XU; d.sBk0 = ld; d.sBn = 1;
      d.C = h->Z + (long long)i0 * v * ld; d.sCm0 = ld;
      d.alpha = -1.0; d.beta = 1.0;
      TRY(gemm(h, d));
    }
    // ---- chain B: S10: panel of K4[(n,f)][(m,e)] = sum_Q L[Q,m,f] L[Q,n,e];  V = K4 XU
    h->cur = sB;
    {
      GemmDesc d; d.M = (int)ov; d.N = ni * v; d.K0 = Q;
      d.A = h->Lov; d.sAm = 1; d.sAk0 = ov;
      d.B = h->Lov + (long long)i0 * v; d.sBk0 = ov; d.sBn = 1;
      d.C = KPb; d.Md = v; d.sCm1 = v; d.sCm0 = ov; d.Nd = v; d.sCn1 = (long long)v * ov; d.sCn0 = 1;
      TRY(gemm(h, d));
    }
    {
      GemmDesc d; d.M = ni * v; d.N = (int)ld; d.K0 = (int)ov;
      d.A = KPb; d.sAm = ov; d.sAk0 = 1;
      d.B = h->XU; d.sBk0 = ld; d.sBn = 1;
      d.C = h->V + (long long)i0 * v * ld; d.sCm0 = ld;
      TRY(gemm(h, d));
    }
  }
  // ---- chain C: everything that goes straight to sout ----
  h->cur = sC;
  // S12a: yv[e][c] = - sum_(Q,m) Lov[Q][m][e] Y[Q][m][c]
  {
    NvtxRange nv("S12a yv");
    GemmDesc d; d.M = v; d.N = (int)Nc; d.K1 = Q; d.K0 = o;
    d.A = h->Lov; d.sAm = 1; d.sAk0 = v; d.sAk1 = ov;
    d.B = h->Y; d.sBk0 = Nc; d.sBk1 = ld; d.sBn = 1;
    d.C = h->yv; d.sCm0 = Nc; d.alpha = -1.0;
    TRY(gemm_splitk(h, d, 64));
  }
  // S2: sigma1[i][c] = sum_(Q,n) Loo[Q,n,i] Y[Q][n][c]  -  sum_(m,e) Fme[m,e] XU[(m,e)][(i,c)]  + small terms
  nvtxRangePushA("S2 sigma1");
  {
    GemmDesc d; d.M = o; d.N = (int)Nc; d.K1 = Q; d.K0 = o;
    d.A = h->LooT; d.sAm = o; d.sAk0 = 1; d.sAk1 = (long long)o * o;
    d.B = h->Y; d.sBk0 = Nc; d.sBk1 = ld; d.sBn = 1;
    d.C = sout; d.sCm0 = Nc;
    TRY(gemm_splitk(h, d, 64));
  }
  {
    // treat the (m,e) sum as K1 = o blocks of K0 = v so that it can be split
    GemmDesc d; d.M = 1; d.N = (int)ld; d.K1 = o; d.K0 = v;
    d.A = h->Fme; d.sAm = ov; d.sAk0 = 1; d.sAk1 = v;
    d.B = h->XU; d.sBk0 = ld; d.sBk1 = (long long)v * ld; d.sBn = 1;
    d.C = sout; d.sCm0 = ld; d.alpha = -1.0; d.beta = 1.0;
    TRY(gemm_splitk(h, d, 32));
  }
  k_sigma1_small<<<(unsigned)((o * nrhs + 127) / 128), 128, 0, sC>>>(sout, xin, h->Fmi, d_omega, eta, o, nrhs);
  nvtxRangePop();
  KLAUNCH(h);
  // S6 (D): s2[(i<j)][(a,c)] = sum_(m<n) W[(i<j)][(m<n)] x2[(m<n)][(a,c)]
  bool s6_done = false;
  if (oz) TRY(sigma_s6_ozaki(h, nrhs, x2, s2, &s6_done));
  if (!s6_done) {
    NvtxRange nv("S6 W_mnij x2");
    GemmDesc d; d.M = (int)h->npair; d.N = (int)(v * Nc); d.K0 = (int)h->npair;
    d.A = h->Wp; d.sAm = h->npair; d.sAk0 = 1;
    d.B = x2; d.sBk0 = v * Nc; d.sBn = 1;
    d.C = s2; d.sCm0 = v * Nc;
    TRY(gemm(h, d));
  }
  // S12b (F): s2[(pair,a)][c] += sum_e t[(pair),a,e] yv[e][c]
  {
    NvtxRange nv("S12b T2 yv");
    GemmDesc d; d.M = (int)(h->npair * v); d.N = (int)Nc; d.K0 = v;
    d.A = h->T2p; d.sAm = v; d.sAk0 = 1;
    d.B = h->yv; d.sBk0 = Nc; d.sBn = 1;
    d.C = s2; d.sCm0 = Nc; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  // S5 (C): s2[(pair,a)][c] += sum_m WB[(pair,a)][m] x1[m][c]
  {
    NvtxRange nv("S5 W_mbij x1");
    GemmDesc d; d.M = (int)(h->npair * v); d.N = (int)Nc; d.K0 = o;
    d.A = h->WB; d.sAm = o; d.sAk0 = 1;
    d.B = xin; d.sBk0 = Nc; d.sBn = 1;
    d.C = s2; d.sCm0 = Nc; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  // ---- join ----
  h->cur = s0;
  if (par) {
    CUDA_TRY(h, cudaEventRecord(h->evB, sB));
    CUDA_TRY(h, cudaEventRecord(h->evC, sC));
    CUDA_TRY(h, cudaStreamWaitEvent(s0, h->evB, 0));
    CUDA_TRY(h, cudaStreamWaitEvent(s0, h->evC, 0));
  }
  // S11: Z[i][a][(j,c)] += sum_(n,f) t[i,n,f,a] V[(n,f)][(j,c)]   (T2 blocks through the pair table, sign per block)
  if (!oz) {
    NvtxRange nv("S11 Z4 = T2 V");
    if ((v & 1) == 0) {
      // panels of panel_ni occupied indices i: ONE launch of ni*v rows whose K-block offsets and signs come from the pair table row
      // of each row's i (row-block mode of the GEMM engine) -- 128-row tiles and full waves like the S9 panels
      for (int i0 = 0; i0 < o; i0 += h->panel_ni) {
        const int ni = std::min(h->panel_ni, o - i0);
        GemmDesc d; d.M = ni * v; d.N = (int)ld; d.K1 = o; d.K0 = v;
        d.A = h->T2p; d.sAm = 1; d.sAk0 = v; d.tabA = h->blk_tab + (long long)i0 * o; d.sgn = h->blk_sgn + (long long)i0 * o;
        d.Rb = v; d.tabR = o; d.tabs_even = true;
        d.B = h->V; d.sBk1 = (long long)v * ld; d.sBk0 = ld; d.sBn = 1;
        d.C = h->Z + (long long)i0 * v * ld; d.sCm0 = ld; d.beta = 1.0;
        TRY(gemm(h, d));
      }
    } else {   // odd v: one batch entry per i (16-byte chunks would straddle row blocks)
      GemmDesc d; d.M = v; d.N = (int)ld; d.K1 = o; d.K0 = v;
      d.A = h->T2p; d.sAm = 1; d.sAk0 = v; d.tabA = h->blk_tab; d.sgn = h->blk_sgn; d.tab_batch_stride = o;
      d.tabs_even = ((long long)v * v) % 2 == 0;
      d.B = h->V; d.sBk1 = (long long)v * ld; d.sBk0 = ld; d.sBn = 1;
      d.C = h->Z; d.sCm0 = ld; d.bsC = (long long)v * ld;
      d.batch = o; d.beta = 1.0;
      TRY(gemm(h, d));
    }
  }
  // S13: shift + P(ij) ring
  NvtxRange nv_s13("S13 epilogue");
  k_sigma2_epilogue<<<(unsigned)h->npair, 256, 0, s0>>>(sout, xin, h->Z, d_omega, eta, o, v, nrhs);
  KLAUNCH(h);
  h->st_sigma_apps += 1;
  return GFCC_OK;
}

// executed FP64 flop model of one batched sigma application (GEMM M*N*K products, pair-packed o^4 term)
static double sigma_flops(const gfcc_ctx* h, int nrhs) {
  const double o = h->o, v = h->v, Q = h->Q, Nc = 2.0 * nrhs, ov = o * v, np_ = (double)h->npair;
  double f = 0;
  f += 2 * Q * ov * o * Nc * 2;              // S1, S7
  f += 2 * 2 * Q * ov * ov;                  // S8, S10 panel builds (independent of nrhs)
  f += 3 * 2 * ov * ov * o * Nc;             // S9, S10 (V), S11
  f += 2 * np_ * np_ * v * Nc;               // S6, pair-packed
  f += 2 * np_ * v * v * Nc + 2 * np_ * v * o * Nc;   // S12, S5
  f += 2 * Q * o * v * Nc + 2 * Q * o * o * Nc + 2 * ov * o * Nc;   // yv, sigma1
  return f;
}

// One sigma application through a CUDA graph (SURVEY.md section 7 "hard parts": config 0 is launch/latency-bound, ~2e8 flop per
// application in ~20 launches).  The graph is captured once per (batch width, omega array, eta) on fixed staging vectors gx -> gy;
// a replay costs two device copies and one graph launch on the host instead of ~20 kernel launches.
static int sigma_via_graph(gfcc_ctx* h, int nrhs, const double* d_omega, double eta, const double* xin, double* sout) {
  cudaStream_t st = h->stream;
  const long long need = h->nvec * 2LL * h->ws_nrhs, elems = h->nvec * 2LL * nrhs;
  if (h->g_elems < need) {
    CUDA_TRY(h, cudaStreamSynchronize(st));
    graphs_clear(h);
    TRY(dev_alloc(h, &h->gx, need));
    int rc = dev_alloc(h, &h->gy, need);
    if (rc) { dev_free(h, h->gx, need); h->gx = nullptr; return rc; }
    h->g_elems = need;
  }
  CUDA_TRY(h, cudaMemcpyAsync(h->gx, xin, (size_t)elems * 8, cudaMemcpyDeviceToDevice, st));
  const gfcc_ctx::SigmaGraph* found = nullptr;
  for (const auto& g : h->graphs) if (g.nrhs == nrhs && g.d_omega == d_omega && g.eta == eta) found = &g;
  if (found) {
    CUDA_TRY(h, cudaGraphLaunch(found->exec, st));
    h->st_sigma_apps += 1; h->st_graph_launches += 1; h->st_kernel_launches += (double)found->nodes;
  } else {
    TRY(sigma_internal(h, nrhs, d_omega, eta, h->gx, h->gy));       // eager: a valid result, and every kernel attribute gets configured
    const double k0 = h->st_kernel_launches, g0 = h->st_gemm_launches, f0 = h->st_flops_exec, a0 = h->st_sigma_apps;
    cudaGraph_t graph = nullptr;
    // the legacy default stream cannot be captured: record on a side stream then (the replay is launched on the handle's stream)
    cudaStream_t cap = (st == nullptr || st == cudaStreamLegacy || st == cudaStreamPerThread) ? h->sB : st;
    bool ok = cap != nullptr && cudaStreamBeginCapture(cap, cudaStreamCaptureModeRelaxed) == cudaSuccess;
    if (ok) {
      h->stream = cap;
      const int rc = sigma_internal(h, nrhs, d_omega, eta, h->gx, h->gy);
      h->stream = st; h->cur = st;
      ok = (cudaStreamEndCapture(cap, &graph) == cudaSuccess) && rc == GFCC_OK && graph != nullptr;
    }
    h->st_kernel_launches = k0; h->st_gemm_launches = g0; h->st_flops_exec = f0; h->st_sigma_apps = a0;
    gfcc_ctx::SigmaGraph g{nrhs, d_omega, eta, nullptr, 0};
    if (ok) ok = cudaGraphInstantiate(&g.exec, graph, 0) == cudaSuccess;
    if (ok) { cudaGraphGetNodes(graph, nullptr, &g.nodes); h->graphs.push_back(g); }
    else { cudaGetLastError(); h->opt_graph = 0; }                  // capture not possible here: stay on plain launches
    if (graph) cudaGraphDestroy(graph);
  }
  CUDA_TRY(h, cudaMemcpyAsync(sout, h->gy, (size_t)elems * 8, cudaMemcpyDeviceToDevice, st));
  return GFCC_OK;
}

// Latency path for tiny systems (SURVEY.md section 7 "hard parts": config 0 is ~2e8 flop per application in ~20 launches).  For
// n = o + o(o-1)/2*v <= DENSE_AUTO_MAX the real matrix Hbar_IP (n x n; 3.7 MB at config 0) is built ONCE per handle by applying the
// S1-S13 path to unit vectors (omega = eta = 0, all 2*nb real columns of a batch used: ceil(n / (2 nb)) applications), and a sigma
// application inside gfcc_solve_ip becomes sout = Hd * xin (one DMMA GEMM, 2 n^2 Nc flop -- FEWER than the factorised route at these
// sizes) plus the (omega - i eta) shift: 2 launches instead of ~20.  gfcc_sigma_ip itself always runs S1-S13.  Only for sizes where
// n^2 doubles are small; the "no o^2 v^2 intermediate" rule of BASELINE.json's configs 2-4 is about sizes where this is never used.
constexpr long long DENSE_AUTO_MAX = 2048, DENSE_HARD_MAX = 8192;
static bool dense_wanted(const gfcc_ctx* h) {
  if (h->opt_dense == 1) return h->nvec <= DENSE_HARD_MAX;
  return h->opt_dense < 0 && h->nvec <= DENSE_AUTO_MAX;
}
static int dense_build(gfcc_ctx* h) {
  if (h->hd_ready) return GFCC_OK;
  NvtxRange nv("gfcc dense Hbar build (tiny systems)");
  const long long n = h->nvec;
  const int nb = (int)std::max<long long>(1, std::min<long long>(128, (n + 1) / 2));
  TRY(ensure_workspace(h, std::max(nb, h->ws_nrhs), false));
  const long long Nc = 2LL * nb;
  cudaStream_t st = h->stream;
  double *vin = nullptr, *vout = nullptr, *zero = nullptr, *Hd = nullptr;
  int rc = GFCC_OK;
  do {
    if ((rc = dev_alloc(h, &Hd, n * n))) break;
    if ((rc = dev_alloc(h, &vin, n * Nc))) break;
    if ((rc = dev_alloc(h, &vout, n * Nc))) break;
    if ((rc = dev_alloc(h, &zero, nb))) break;
    if (cudaMemsetAsync(zero, 0, (size_t)nb * 8, st) != cudaSuccess) { h->err = "memset failed"; rc = GFCC_ECUDA; break; }
    for (long long c0 = 0; c0 < n && rc == GFCC_OK; c0 += Nc) {
      const int nc = (int)std::min<long long>(Nc, n - c0);
      k_unit_cols<<<nblk(n * Nc), 256, 0, st>>>(vin, n, (int)Nc, c0);
      h->st_kernel_launches += 1;
      rc = sigma_internal(h, nb, zero, 0.0, vin, vout);      // columns are independent real vectors: Hbar is real
      if (rc) break;
      k_store_cols<<<nblk(n * nc), 256, 0, st>>>(Hd, vout, n, (int)Nc, c0, nc);
      h->st_kernel_launches += 1;
    }
    if (rc) break;
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { h->err = "dense Hbar build failed"; rc = GFCC_ECUDA; break; }
  } while (0);
  cudaStreamSynchronize(st);
  dev_free(h, vin, n * Nc); dev_free(h, vout, n * Nc); dev_free(h, zero, nb);
  if (rc != GFCC_OK) { dev_free(h, Hd, n * n); return rc; }
  h->Hd = Hd; h->hd_ready = true;
  return GFCC_OK;
}
static int dense_apply(gfcc_ctx* h, int nrhs, const double* d_omega, double eta, const double* xin, double* sout) {
  const long long n = h->nvec, Nc = 2LL * nrhs;
  h->cur = h->stream;
  GemmDesc d; d.M = (int)n; d.N = (int)Nc; d.K0 = (int)n;
  d.A = h->Hd; d.sAm = n; d.sAk0 = 1;
  d.B = xin; d.sBk0 = Nc; d.sBn = 1;
  d.C = sout; d.sCm0 = Nc;
  TRY(gemm(h, d));
  k_dense_shift<<<nblk(n * nrhs), 256, 0, h->stream>>>(sout, xin, d_omega, eta, n, nrhs);
  KLAUNCH(h);
  h->st_sigma_apps += 1; h->st_dense_apps += 1;
  return GFCC_OK;
}

// ------------------------------------------------------------------------------------------
// gfcc_create
// ------------------------------------------------------------------------------------------
static int create_impl(gfcc_ctx* h, const double* fock, const double* T1, const double* L1, const double* Lchol) {
  const int o = h->o, v = h->v, Q = h->Q, N = h->N;
  const long long ov = (long long)o * v, npair = h->npair, vv = (long long)v * v;
  cudaStream_t st = h->stream;
  h->cur = st;
  const double flops0 = h->st_flops_exec;
  CUDA_TRY(h, cudaStreamCreateWithFlags(&h->sB, cudaStreamNonBlocking));
  CUDA_TRY(h, cudaStreamCreateWithFlags(&h->sC, cudaStreamNonBlocking));
  CUDA_TRY(h, cudaEventCreateWithFlags(&h->evFork, cudaEventDisableTiming));
  CUDA_TRY(h, cudaEventCreateWithFlags(&h->evB, cudaEventDisableTiming));
  CUDA_TRY(h, cudaEventCreateWithFlags(&h->evC, cudaEventDisableTiming));

  TRY(dev_alloc(h, &h->Lov, Q * ov)); TRY(dev_alloc(h, &h->LooT, (long long)Q * o * o));
  TRY(dev_alloc(h, &h->Lvv, Q * vv)); TRY(dev_alloc(h, &h->Lm, Q * ov));
  TRY(dev_alloc(h, &h->Fme, ov)); TRY(dev_alloc(h, &h->Fmi, (long long)o * o)); TRY(dev_alloc(h, &h->Fae, vv));
  TRY(dev_alloc(h, &h->fdiag, N)); TRY(dev_alloc(h, &h->D, (long long)o * o));
  TRY(dev_alloc(h, &h->t1, ov)); TRY(dev_alloc(h, &h->l1, ov));
  TRY(dev_alloc(h, &h->Wp, npair * npair)); TRY(dev_alloc(h, &h->WB, npair * v * o));
  // split-K partial buffer, sized for the largest user
  h->part_elems = std::max<long long>({64LL * v * 512, 64LL * o * 512, 32LL * o * 512, 32LL * vv, 32LL * o * o, 1LL << 20});
  TRY(dev_alloc(h, &h->part, h->part_elems));
  CUDA_TRY(h, cudaMemcpyAsync(h->t1, T1, ov * 8, cudaMemcpyDeviceToDevice, st));
  CUDA_TRY(h, cudaMemcpyAsync(h->l1, L1, ov * 8, cudaMemcpyDeviceToDevice, st));
  CUDA_TRY(h, cudaMemcpy2DAsync(h->fdiag, 8, fock, (size_t)(N + 1) * 8, 8, N, cudaMemcpyDeviceToDevice, st));
  {   // pair-block table for the T2 operand
    std::vector<long long> tab((size_t)o * o, 0);
    std::vector<double> sg((size_t)o * o, 0.0);
    for (int i = 0; i < o; ++i)
      for (int n = 0; n < o; ++n) {
        if (i == n) continue;
        tab[(size_t)i * o + n] = pair_index(std::min(i, n), std::max(i, n), o) * vv;
        sg[(size_t)i * o + n] = (i < n) ? 1.0 : -1.0;
      }
    double* tmp = nullptr;
    TRY(dev_alloc(h, &tmp, (long long)o * o)); h->blk_tab = (long long*)tmp;
    TRY(dev_alloc(h, &h->blk_sgn, (long long)o * o));
    CUDA_TRY(h, cudaMemcpyAsync(h->blk_tab, tab.data(), tab.size() * 8, cudaMemcpyHostToDevice, st));
    CUDA_TRY(h, cudaMemcpyAsync(h->blk_sgn, sg.data(), sg.size() * 8, cudaMemcpyHostToDevice, st));
    CUDA_TRY(h, cudaStreamSynchronize(st));   // host vectors go out of scope
  }
  auto copy_block = [&](double* dst, int R, int Cc, int row0, int col0, int transpose) {
    dim3 grid((Cc + 31) / 32, (R + 31) / 32, Q), blk(32, 8);
    k_copy_block<<<grid, blk, 0, st>>>(dst, Lchol, R, Cc, row0, col0, N, transpose);
  };
  // ---- P1: T1-dressed Cholesky blocks ----
  nvtxRangePushA("gfcc_create P1-P2 (dressing)");
  copy_block(h->Lov, o, v, 0, o, 0); KLAUNCH(h);          // Lov[Q][m][e] = L[Q][m][o+e]
  copy_block(h->LooT, o, o, 0, 0, 1); KLAUNCH(h);         // LooT[Q][i][m] = L[Q][m][i]
  copy_block(h->Lvv, v, v, o, o, 0); KLAUNCH(h);          // Lvv[Q][a][e] = L[Q][o+a][o+e]
  copy_block(h->Lm, o, v, o, 0, 1); KLAUNCH(h);           // Lm[Q][i][a] = L[Q][o+a][i]
  {   // LooT[Q][i][m] += sum_e t1[i,e] Lov[Q][m][e]
    GemmDesc d; d.M = o; d.N = o; d.K0 = v; d.batch = Q;
    d.A = h->t1; d.sAm = v; d.sAk0 = 1;
    d.B = h->Lov; d.sBk0 = 1; d.sBn = v; d.bsB = ov;
    d.C = h->LooT; d.sCm0 = o; d.bsC = (long long)o * o; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  {   // Lm[Q][i][a] -= sum_m L[Q][m][i] t1[m,a]      (uses the UNdressed L_mi)
    GemmDesc d; d.M = o; d.N = v; d.K0 = o; d.batch = Q;
    d.A = Lchol; d.sAm = 1; d.sAk0 = N; d.bsA = (long long)N * N;
    d.B = h->t1; d.sBk0 = v; d.sBn = 1;
    d.C = h->Lm; d.sCm0 = v; d.bsC = ov; d.alpha = -1.0; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  {   // Lvv[Q][a][e] -= sum_m t1[m,a] Lov[Q][m][e]
    GemmDesc d; d.M = v; d.N = v; d.K0 = o; d.batch = Q;
    d.A = h->t1; d.sAm = 1; d.sAk0 = v;
    d.B = h->Lov; d.sBk0 = v; d.sBn = 1; d.bsB = ov;
    d.C = h->Lvv; d.sCm0 = v; d.bsC = vv; d.alpha = -1.0; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  {   // Lm[Q][i][a] += sum_e t1[i,e] Lvv[Q][a][e]     (dressed Lvv)  -> Lm holds Ltilde_vo[Q,a,i]
    GemmDesc d; d.M = o; d.N = v; d.K0 = v; d.batch = Q;
    d.A = h->t1; d.sAm = v; d.sAk0 = 1;
    d.B = h->Lvv; d.sBk0 = 1; d.sBn = v; d.bsB = vv;
    d.C = h->Lm; d.sCm0 = v; d.bsC = ov; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  // ---- P2: dressed Fock  ft = A^T (f + J - K) B ----
  double *sq = nullptr, *U = nullptr, *Kmat = nullptr, *g = nullptr, *tmp = nullptr, *ft = nullptr;
  TRY(dev_alloc(h, &sq, Q)); TRY(dev_alloc(h, &U, (long long)Q * N * o));
  TRY(dev_alloc(h, &Kmat, (long long)N * N)); TRY(dev_alloc(h, &g, (long long)N * N));
  TRY(dev_alloc(h, &tmp, (long long)N * N)); TRY(dev_alloc(h, &ft, (long long)N * N));
  k_sq<<<Q, 256, 0, st>>>(sq, h->t1, h->Lov, (int)ov); KLAUNCH(h);
  {   // U[Q][p][k] = sum_c L[Q][p][o+c] t1[k,c]
    GemmDesc d; d.M = N; d.N = o; d.K0 = v; d.batch = Q;
    d.A = Lchol + o; d.sAm = N; d.sAk0 = 1; d.bsA = (long long)N * N;
    d.B = h->t1; d.sBk0 = 1; d.sBn = v;
    d.C = U; d.sCm0 = o; d.bsC = (long long)N * o;
    TRY(gemm(h, d));
  }
  {   // K[p][q] = sum_(Q,k) U[Q][p][k] L[Q][k][q]
    GemmDesc d; d.M = N; d.N = N; d.K1 = Q; d.K0 = o;
    d.A = U; d.sAm = o; d.sAk0 = 1; d.sAk1 = (long long)N * o;
    d.B = Lchol; d.sBk0 = N; d.sBk1 = (long long)N * N; d.sBn = 1;
    d.C = Kmat; d.sCm0 = N;
    const int S = (int)std::max<long long>(1, std::min<long long>(32, h->part_elems / ((long long)N * N)));
    TRY(gemm_splitk(h, d, S));
  }
  k_fock_jk<<<(unsigned)(((long long)N * N + 127) / 128), 128, 0, st>>>(g, fock, sq, Lchol, Kmat, N, Q); KLAUNCH(h);
  k_dress_left<<<(unsigned)(((long long)N * N + 127) / 128), 128, 0, st>>>(tmp, g, h->t1, o, v); KLAUNCH(h);
  k_dress_right<<<(unsigned)(((long long)N * N + 127) / 128), 128, 0, st>>>(ft, tmp, h->t1, o, v); KLAUNCH(h);
  k_fock_block<<<(unsigned)((ov + 127) / 128), 128, 0, st>>>(h->Fme, ft, o, v, 0, o, N); KLAUNCH(h);
  k_fock_block<<<(unsigned)(((long long)o * o + 127) / 128), 128, 0, st>>>(h->Fmi, ft, o, o, 0, 0, N); KLAUNCH(h);
  k_fock_block<<<(unsigned)((vv + 127) / 128), 128, 0, st>>>(h->Fae, ft, v, v, o, o, N); KLAUNCH(h);
  CUDA_TRY(h, cudaStreamSynchronize(st));
  dev_free(h, sq, Q); dev_free(h, U, (long long)Q * N * o); dev_free(h, Kmat, (long long)N * N);
  dev_free(h, g, (long long)N * N); dev_free(h, tmp, (long long)N * N); dev_free(h, ft, (long long)N * N);

  nvtxRangePop();
  NvtxRange nv_p37("gfcc_create P3-P7");
  // ---- P3: Mq[Q][i][a] = sum_(n,f) t[i,n,f,a] Lov[Q][n][f]   (batch over i, T2 blocks via the pair table on B)
  double* Mq = nullptr;
  TRY(dev_alloc(h, &Mq, Q * ov));
  {
    GemmDesc d; d.M = Q; d.N = v; d.K1 = o; d.K0 = v; d.batch = o;
    d.A = h->Lov; d.sAm = ov; d.sAk0 = 1; d.sAk1 = v;
    d.B = h->T2p; d.sBk0 = v; d.sBn = 1; d.tabB = h->blk_tab; d.sgn = h->blk_sgn; d.tab_batch_stride = o;
    d.tabs_even = (vv % 2) == 0;
    d.C = Mq; d.sCm0 = ov; d.bsC = v;
    TRY(gemm(h, d));
  }
  // ---- P4: F_mi -= sum_(Q,e) Lov[Q,m,e] M[Q,i,e];  F_ae += sum_(Q,m) M[Q,m,a] Lov[Q,m,e]
  {
    GemmDesc d; d.M = o; d.N = o; d.K1 = Q; d.K0 = v;
    d.A = h->Lov; d.sAm = v; d.sAk0 = 1; d.sAk1 = ov;
    d.B = Mq; d.sBk0 = 1; d.sBn = v; d.sBk1 = ov;
    d.C = h->Fmi; d.sCm0 = o; d.alpha = -1.0; d.beta = 1.0;
    TRY(gemm_splitk(h, d, 32));
  }
  {
    GemmDesc d; d.M = v; d.N = v; d.K1 = Q; d.K0 = o;
    d.A = Mq; d.sAm = 1; d.sAk0 = v; d.sAk1 = ov;
    d.B = h->Lov; d.sBk0 = v; d.sBk1 = ov; d.sBn = 1;
    d.C = h->Fae; d.sCm0 = v; d.alpha = 1.0; d.beta = 1.0;
    TRY(gemm_splitk(h, d, 32));
  }
  // Lm = Ltilde_vo - M
  k_sub<<<nblk(Q * ov), 256, 0, st>>>(h->Lm, Mq, Q * ov); KLAUNCH(h);
  CUDA_TRY(h, cudaStreamSynchronize(st));
  dev_free(h, Mq, Q * ov);

  // ---- create-time panel scratch ----
  const double budget = panel_budget(h, false);
  // ---- P5: W_mnij packed ----
  CUDA_TRY(h, cudaMemsetAsync(h->Wp, 0, (size_t)(npair * npair) * 8, st));
  {
    // term 1: sum_Q Loo[Q,m,i] Loo[Q,n,j] antisymmetrised in (i,j); panels over i
    const long long oo = (long long)o * o;
    int ni = (int)std::max<double>(1, std::min<double>(o, std::floor(budget / (8.0 * o * oo))));
    double* G1 = nullptr;
    TRY(dev_alloc(h, &G1, (long long)ni * o * oo));
    for (int i0 = 0; i0 < o; i0 += ni) {
      const int n_i = std::min(ni, o - i0);
      GemmDesc d; d.M = n_i * o; d.N = (int)oo; d.K0 = Q;
      d.A = h->LooT + (long long)i0 * o; d.sAm = 1; d.sAk0 = oo;
      d.B = h->LooT; d.sBk0 = oo; d.sBn = 1;
      d.C = G1; d.sCm0 = oo;
      TRY(gemm(h, d));
      for (int mode = 0; mode < 2; ++mode) {
        k_scatter_oooo<<<nblk((long long)n_i * o * npair), 256, 0, st>>>(h->Wp, G1, o, i0, n_i, mode);
        KLAUNCH(h);
      }
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, G1, (long long)ni * o * oo);
    // term 2: sum_ef t[i,j,e,f] <mn|ef>, <mn|ef> = sum_Q L[Q,m,e] L[Q,n,f]; panels over m, columns n >= m0 only
    int nm = (int)std::max<double>(1, std::min<double>(o, std::floor(budget / (8.0 * vv * o))));
    double *O = nullptr, *tmpw = nullptr;
    TRY(dev_alloc(h, &O, vv * nm * o)); TRY(dev_alloc(h, &tmpw, npair * nm * o));
    for (int m0 = 0; m0 < o; m0 += nm) {
      const int n_m = std::min(nm, o - m0);
      const int nlo = m0, ncols = o - nlo;       // only n >= m0 can satisfy m < n
      const long long ldO = (long long)n_m * ncols;
      {   // O[(e,f)][(m',n')] = sum_Q Lov[Q][(m,e)] Lov[Q][(n,f)]
        GemmDesc d; d.M = n_m * v; d.N = ncols * v; d.K0 = Q;
        d.A = h->Lov + (long long)m0 * v; d.sAm = 1; d.sAk0 = ov;
        d.B = h->Lov + (long long)nlo * v; d.sBk0 = ov; d.sBn = 1;
        d.C = O; d.Md = v; d.sCm1 = ncols; d.sCm0 = (long long)v * ldO; d.Nd = v; d.sCn1 = 1; d.sCn0 = ldO;
        TRY(gemm(h, d));
      }
      {   // tmpw[(i<j)][(m',n')] = sum_(e,f) T2p[(i<j)][(e,f)] O[(e,f)][(m',n')]
        GemmDesc d; d.M = (int)npair; d.N = (int)ldO; d.K0 = (int)vv;
        d.A = h->T2p; d.sAm = vv; d.sAk0 = 1;
        d.B = O; d.sBk0 = ldO; d.sBn = 1;
        d.C = tmpw; d.sCm0 = ldO;
        TRY(gemm(h, d));
      }
      k_pack_oooo_cols<<<nblk(npair * ldO), 256, 0, st>>>(h->Wp, tmpw, o, m0, n_m, nlo, 1.0);
      KLAUNCH(h);
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, O, vv * nm * o); dev_free(h, tmpw, npair * nm * o);
  }
  // ---- P6: W_mbij.  Wacc[(i<j)][b][m] accumulates W[m,b,i,j]; WB = -Wacc (= W[m,b,j,i]) ----
  CUDA_TRY(h, cudaMemsetAsync(h->WB, 0, (size_t)(npair * v * o) * 8, st));
  {
    // term A: P(ij) sum_Q Loo[Q,m,i] Lm[Q,j,b]; panels over i
    int ni = (int)std::max<double>(1, std::min<double>(o, std::floor(budget / (8.0 * o * ov))));
    double* X1 = nullptr;
    TRY(dev_alloc(h, &X1, (long long)ni * o * ov));
    for (int i0 = 0; i0 < o; i0 += ni) {
      const int n_i = std::min(ni, o - i0);
      GemmDesc d; d.M = n_i * o; d.N = (int)ov; d.K0 = Q;
      d.A = h->LooT + (long long)i0 * o; d.sAm = 1; d.sAk0 = (long long)o * o;
      d.B = h->Lm; d.sBk0 = ov; d.sBn = 1;
      d.C = X1; d.sCm0 = ov;
      TRY(gemm(h, d));
      for (int mode = 0; mode < 2; ++mode) {
        k_scatter_ovoo<<<nblk((long long)n_i * o * ov), 256, 0, st>>>(h->WB, X1, o, v, i0, n_i, mode);
        KLAUNCH(h);
      }
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, X1, (long long)ni * o * ov);
    // term B: - sum_e Fme[m,e] t[i,j,b,e]
    {
      GemmDesc d; d.M = (int)(npair * v); d.N = o; d.K0 = v;
      d.A = h->T2p; d.sAm = v; d.sAk0 = 1;
      d.B = h->Fme; d.sBk0 = 1; d.sBn = v;
      d.C = h->WB; d.sCm0 = o; d.alpha = -1.0; d.beta = 1.0;
      TRY(gemm(h, d));
    }
    // term C: sum_(e,f) t[i,j,e,f] R[(e,f)][(b,m)],  R = sum_Q Lov[Q,m,e] Lvv[Q,b,f]; panels over b
    int nb = (int)std::max<double>(1, std::min<double>(v, std::floor(budget / (8.0 * vv * o))));
    double* R = nullptr;
    TRY(dev_alloc(h, &R, vv * nb * o));
    for (int b0 = 0; b0 < v; b0 += nb) {
      const int n_b = std::min(nb, v - b0);
      const long long ldR = (long long)n_b * o;
      {
        GemmDesc d; d.M = (int)ov; d.N = n_b * v; d.K0 = Q;
        d.A = h->Lov; d.sAm = 1; d.sAk0 = ov;
        d.B = h->Lvv + (long long)b0 * v; d.sBk0 = vv; d.sBn = 1;
        d.C = R; d.Md = v; d.sCm1 = 1; d.sCm0 = (long long)v * ldR; d.Nd = v; d.sCn1 = o; d.sCn0 = ldR;
        TRY(gemm(h, d));
      }
      {
        GemmDesc d; d.M = (int)npair; d.N = (int)ldR; d.K0 = (int)vv;
        d.A = h->T2p; d.sAm = vv; d.sAk0 = 1;
        d.B = R; d.sBk0 = ldR; d.sBn = 1;
        d.C = h->WB + (long long)b0 * o; d.sCm0 = (long long)v * o; d.beta = 1.0;
        TRY(gemm(h, d));
      }
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, R, vv * nb * o);
    // term D: X2[m,b,i,j] = - sum_(n,e) S[(i,m)][(n,e)] t[j,n,b,e],  S = sum_Q Loo[Q,n,i] Lov[Q,m,e]; panels over i
    int ni2 = (int)std::max<double>(1, std::min<double>(o, std::floor(budget / (8.0 * (o * ov + (double)o * o * v)))));
    double *S = nullptr, *X2 = nullptr;
    TRY(dev_alloc(h, &S, (long long)ni2 * o * ov)); TRY(dev_alloc(h, &X2, (long long)o * ni2 * o * v));
    for (int i0 = 0; i0 < o; i0 += ni2) {
      const int n_i = std::min(ni2, o - i0);
      {   // S[(i',m)][(n,e)] : GEMM rows (i',n) from LooT, cols (m,e) from Lov
        GemmDesc d; d.M = n_i * o; d.N = (int)ov; d.K0 = Q;
        d.A = h->LooT + (long long)i0 * o; d.sAm = 1; d.sAk0 = (long long)o * o;
        d.B = h->Lov; d.sBk0 = ov; d.sBn = 1;
        d.C = S; d.Md = o; d.sCm1 = (long long)o * ov; d.sCm0 = v; d.Nd = v; d.sCn1 = ov; d.sCn0 = 1;
        TRY(gemm(h, d));
      }
      {   // batch j: X2[j][(i',m)][b] = - sum_(n,e) S[(i',m)][(n,e)] sgn(j,n) T2p[blk(j,n)][b][e]
        GemmDesc d; d.M = n_i * o; d.N = v; d.K1 = o; d.K0 = v; d.batch = o;
        d.A = S; d.sAm = ov; d.sAk0 = 1; d.sAk1 = v;
        d.B = h->T2p; d.sBk0 = 1; d.sBn = v; d.tabB = h->blk_tab; d.sgn = h->blk_sgn; d.tab_batch_stride = o;
        d.tabs_even = (vv % 2) == 0;
        d.C = X2; d.sCm0 = v; d.bsC = (long long)n_i * o * v; d.alpha = -1.0;
        TRY(gemm(h, d));
      }
      for (int mode = 0; mode < 2; ++mode) {
        k_scatter_ovoo_batched<<<nblk((long long)o * n_i * o * v), 256, 0, st>>>(h->WB, X2, o, v, i0, n_i, mode);
        KLAUNCH(h);
      }
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, S, (long long)ni2 * o * ov); dev_free(h, X2, (long long)o * ni2 * o * v);
    // WB[(i<j)][a][m] = W[m,a,j,i] = -W[m,a,i,j]
    k_scale<<<nblk(npair * v * o), 256, 0, st>>>(h->WB, -1.0, npair * v * o); KLAUNCH(h);
  }
  // ---- P7: D[k][i] = sum_a t1[k,a] l1[i,a] + 1/2 sum_(j,a,b) t[k,j,a,b] l[i,j,a,b] ----
  {
    k_D_singles<<<(o * o + 127) / 128, 128, 0, st>>>(h->D, h->t1, h->l1, o, v); KLAUNCH(h);
    double *TJ = nullptr, *LJ = nullptr;
    TRY(dev_alloc(h, &TJ, (long long)o * vv)); TRY(dev_alloc(h, &LJ, (long long)o * vv));
    for (int j = 0; j < o; ++j) {
      k_gather_t2_rows<<<nblk((long long)o * vv), 256, 0, st>>>(TJ, h->T2p, o, v, j); KLAUNCH(h);
      k_gather_l2_rows<<<nblk((long long)o * vv), 256, 0, st>>>(LJ, h->L2p, o, v, j); KLAUNCH(h);
      GemmDesc d; d.M = o; d.N = o; d.K1 = v; d.K0 = v;
      d.A = TJ; d.sAm = vv; d.sAk0 = 1; d.sAk1 = v;
      d.B = LJ; d.sBk0 = 1; d.sBn = vv; d.sBk1 = v;
      d.C = h->D; d.sCm0 = o; d.alpha = 0.5; d.beta = 1.0;
      TRY(gemm_splitk(h, d, 32));
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, TJ, (long long)o * vv); dev_free(h, LJ, (long long)o * vv);
  }
  CUDA_TRY(h, cudaStreamSynchronize(st));
  h->st_flops_create = h->st_flops_exec - flops0;
  return GFCC_OK;
}

static void free_side_streams(gfcc_ctx* h) {
  if (h->sB) { cudaStreamSynchronize(h->sB); cudaStreamDestroy(h->sB); }
  if (h->sC) { cudaStreamSynchronize(h->sC); cudaStreamDestroy(h->sC); }
  if (h->evFork) cudaEventDestroy(h->evFork);
  if (h->evB) cudaEventDestroy(h->evB);
  if (h->evC) cudaEventDestroy(h->evC);
  h->sB = h->sC = nullptr; h->evFork = h->evB = h->evC = nullptr;
}

extern "C" int gfcc_create(int o, int v, int Q, const double* fock, const double* T1, const double* T2, const double* L1,
                           const double* L2, const double* Lchol, gfcc_handle* out) {
  if (out) *out = nullptr;
  if (!out || !fock || !T1 || !T2 || !L1 || !L2 || !Lchol || o < 2 || v < 2 || Q < 1) {
    g_create_error = "gfcc_create: null pointer or invalid size (need o >= 2, v >= 2, Q >= 1)";
    return GFCC_EINVAL;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    g_create_error = "gfcc_create: no CUDA device (there is no CPU fallback)";
    cudaGetLastError();
    return GFCC_ECUDA;
  }
  gfcc_ctx* h = new gfcc_ctx();
  h->o = o; h->v = v; h->Q = Q; h->N = o + v;
  h->npair = (long long)o * (o - 1) / 2; h->ntri = (long long)v * (v - 1) / 2;
  h->nvec = o + h->npair * v;
  h->T2p = T2; h->L2p = L2;
  int rc = create_impl(h, fock, T1, L1, Lchol);
  if (rc != GFCC_OK) {
    g_create_error = h->err;
    free_side_streams(h);
    for (void* p : h->allocs) cudaFree(p);
    delete h;
    return rc;
  }
  *out = h;
  return GFCC_OK;
}

// Closed-shell (spin-restricted) entry: the spatial tensors are expanded to spin orbitals on the device and the spin-orbital
// intermediates are built from them (include/gfcc.h).  The expanded T2 / Lambda2 are owned by the handle.
extern "C" int gfcc_create_closed_shell(int no, int nv, int Q, const double* fock, const double* T1, const double* T2,
                                        const double* L1, const double* L2, const double* Lchol, gfcc_handle* out) {
  if (out) *out = nullptr;
  if (!out || !fock || !T1 || !T2 || !L1 || !L2 || !Lchol || no < 1 || nv < 1 || Q < 1) {
    g_create_error = "gfcc_create_closed_shell: null pointer or invalid size (need no >= 1, nv >= 1, Q >= 1)";
    return GFCC_EINVAL;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    g_create_error = "gfcc_create_closed_shell: no CUDA device (there is no CPU fallback)";
    cudaGetLastError();
    return GFCC_ECUDA;
  }
  const int o = 2 * no, v = 2 * nv, N = o + v;
  gfcc_ctx* h = new gfcc_ctx();
  h->o = o; h->v = v; h->Q = Q; h->N = N;
  h->npair = (long long)o * (o - 1) / 2; h->ntri = (long long)v * (v - 1) / 2;
  h->nvec = o + h->npair * v;
  double *f_so = nullptr, *t1_so = nullptr, *l1_so = nullptr, *L_so = nullptr, *t2p = nullptr, *l2p = nullptr;
  auto run = [&]() -> int {
    const long long NN = (long long)N * N, ov = (long long)o * v;
    TRY(dev_alloc(h, &t2p, h->npair * v * v)); TRY(dev_alloc(h, &l2p, h->npair * h->ntri));
    TRY(dev_alloc(h, &f_so, NN)); TRY(dev_alloc(h, &t1_so, ov)); TRY(dev_alloc(h, &l1_so, ov)); TRY(dev_alloc(h, &L_so, (long long)Q * NN));
    cudaStream_t st = h->stream;
    k_cs_expand_matrix<<<dim3(nblk(NN), 1, 1), 256, 0, st>>>(f_so, fock, no, nv);
    k_cs_expand_matrix<<<dim3(nblk(NN, 256, 4096), 1, Q), 256, 0, st>>>(L_so, Lchol, no, nv);
    k_cs_expand_t1<<<(unsigned)((ov + 127) / 128), 128, 0, st>>>(t1_so, T1, no, nv);
    k_cs_expand_t1<<<(unsigned)((ov + 127) / 128), 128, 0, st>>>(l1_so, L1, no, nv);
    k_cs_expand_doubles<<<nblk(h->npair * v * v), 256, 0, st>>>(t2p, T2, no, nv, 0);
    k_cs_expand_doubles<<<nblk(h->npair * h->ntri), 256, 0, st>>>(l2p, L2, no, nv, 1);
    h->st_kernel_launches += 6;
    CUDA_TRY(h, cudaGetLastError());
    h->T2p = t2p; h->L2p = l2p;
    TRY(create_impl(h, f_so, t1_so, l1_so, L_so));
    dev_free(h, f_so, NN); dev_free(h, t1_so, ov); dev_free(h, l1_so, ov); dev_free(h, L_so, (long long)Q * NN);
    return GFCC_OK;
  };
  const int rc = run();
  if (rc != GFCC_OK) {
    g_create_error = h->err;
    free_side_streams(h);
    for (void* p : h->allocs) cudaFree(p);
    delete h;
    return rc;
  }
  *out = h;
  return GFCC_OK;
}

extern "C" int gfcc_destroy(gfcc_handle h) {
  if (!h) return GFCC_EINVAL;
  cudaStreamSynchronize(h->stream);
  free_side_streams(h);
  graphs_clear(h);
  solve_free(h->sw);
  ea_destroy(h);
  for (void* p : h->allocs) cudaFree(p);
  for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
  delete h;
  return GFCC_OK;
}

extern "C" const char* gfcc_last_error(gfcc_handle h) { return h ? h->err.c_str() : g_create_error.c_str(); }

extern "C" int gfcc_set_stream(gfcc_handle h, void* s) {
  if (!h) return GFCC_EINVAL;
  h->stream = (cudaStream_t)s;
  h->cur = h->stream;
  return GFCC_OK;
}

extern "C" int gfcc_set_option(gfcc_handle h, const char* key, double val) {
  if (!h || !key) return GFCC_EINVAL;
  std::string k(key);
  if (k == "gmres_m" && val >= 1) h->opt_m = std::floor(val);
  else if (k == "gmres_maxit" && val >= 1) h->opt_maxit = std::floor(val);
  else if (k == "gmres_fixed" && val >= 0) h->opt_fixed = std::floor(val);
  else if (k == "x0" && (val == 0 || val == 1)) h->opt_x0 = val;
  else if (k == "panel_bytes" && val > 0) { h->opt_panel_bytes = val; if (h->ws_nrhs) { cudaStreamSynchronize(h->stream); free_workspace(h); } }
  else if (k == "max_batch" && val >= 1) h->opt_max_batch = std::floor(val);
  else if (k == "release_workspace") { cudaStreamSynchronize(h->stream); if (h->ws_nrhs) free_workspace(h); solve_free(h->sw); ea_release_ws(h); }
  else if (k == "compact" && val <= 1) h->opt_compact = val;
  else if (k == "graph" && (val == -1 || val == 0 || val == 1)) h->opt_graph = val;
  else if (k == "dense" && (val == -1 || val == 0 || val == 1)) h->opt_dense = val;
  else if (k == "gmres_poll" && val >= 0) h->opt_poll = std::floor(val);
  else if (k == "overlap" && (val == 0 || val == 1)) { h->opt_overlap = val; if (h->ws_nrhs) { cudaStreamSynchronize(h->stream); free_workspace(h); } }
  else if (k == "engine" && (val == 0 || val == 1)) { h->opt_engine = (int)val; if (h->ws_nrhs) { cudaStreamSynchronize(h->stream); free_workspace(h); } }
  else if (k == "ozaki_slices" && val >= 2 && val <= OZ_MAX_SLICES) {
    cudaStreamSynchronize(h->stream);
    if (h->ws_nrhs) free_workspace(h);
    oz_release(h, h->ozLvv); oz_release(h, h->ozLooT); oz_release(h, h->ozLov); oz_release(h, h->ozWp); h->oz_const_ready = false;
    h->opt_oz_slices = (int)val;
  }
  else if (k == "profile_gemm") { h->prof = (val != 0); h->ev_used = 0; h->ev_flops.clear(); h->ev_ops8.clear(); }
  else { h->err = "gfcc_set_option: unknown key or invalid value: " + k; return GFCC_EINVAL; }
  return GFCC_OK;
}

extern "C" int gfcc_get_stat(gfcc_handle h, const char* key, double* val) {
  if (!h || !key || !val) return GFCC_EINVAL;
  std::string k(key);
  if (k == "iterations") *val = h->st_iterations;
  else if (k == "sigma_applications") *val = h->st_sigma_apps;
  else if (k == "flops_sigma") *val = h->st_flops_sigma;
  else if (k == "flops_create") *val = h->st_flops_create;
  else if (k == "flops_executed") *val = h->st_flops_exec;
  else if (k == "bytes_device") *val = h->bytes + h->sw.bytes;
  else if (k == "max_relres") *val = h->st_max_relres;
  else if (k == "n_unconverged") *val = h->st_nunconv;
  else if (k == "gemm_launches") *val = h->st_gemm_launches;
  else if (k == "kernel_launches") *val = h->st_kernel_launches;
  else if (k == "panel_ni") *val = h->panel_ni;
  else if (k == "oz_gemms") *val = h->st_oz_gemms;
  else if (k == "oz_fail") {
    int hf = 0;
    if (h->oz_fail && (cudaStreamSynchronize(h->stream) != cudaSuccess ||
                       cudaMemcpy(&hf, h->oz_fail, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess)) { h->err = "sync failed"; return GFCC_ECUDA; }
    *val = hf;
  }
  else if (k == "gmres_m_used") *val = h->sw.m_run;
  else if (k == "gmres_m_cap") *val = h->sw.mcap;
  else if (k == "gmres_m_memory_limit") *val = solve_mmax(h->nvec, std::max(1, h->sw.cap > 0 ? h->sw.cap : (int)h->opt_max_batch)) + (h->sw.cap > 0 ? h->sw.mcap + 6 : 0);
  else if (k == "graph_launches") *val = h->st_graph_launches;
  else if (k == "dense_applications") *val = h->st_dense_apps;
  else if (k == "compactions") *val = (double)h->sw.compactions;
  else if (k == "refills") *val = (double)h->sw.refills;
  else if (k == "polls") *val = (double)h->sw.polls;
  else if (k == "active_col_steps") *val = h->sw.active_col_steps;
  else if (k == "lockstep_col_steps") *val = h->sw.full_col_steps;
  else if (k == "oz_time_ms" || k == "oz_ops_timed" || k == "oz_flops_timed" || k == "oz_launches_timed") {
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) { h->err = "sync failed"; return GFCC_ECUDA; }
    double ms = 0, ops = 0, fl = 0, n = 0;
    for (size_t q = 0; q < h->ev_flops.size(); ++q) {
      float t = 0;
      if (h->ev_ops8[q] > 0 && cudaEventElapsedTime(&t, h->ev_pool[2 * q], h->ev_pool[2 * q + 1]) == cudaSuccess) {
        ms += t; ops += h->ev_ops8[q]; fl += h->ev_flops[q]; n += 1;
      }
    }
    *val = (k == "oz_time_ms") ? ms : (k == "oz_ops_timed") ? ops : (k == "oz_flops_timed") ? fl : n;
  }
  else if (k == "gemm_time_ms" || k == "gemm_flops_timed" || k == "gemm_launches_timed" || k == "gemm_time_max_ms") {
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) { h->err = "sync failed"; return GFCC_ECUDA; }
    double ms = 0, fl = 0, mx = 0;
    for (size_t q = 0; q < h->ev_flops.size(); ++q) {
      float t = 0;
      if (cudaEventElapsedTime(&t, h->ev_pool[2 * q], h->ev_pool[2 * q + 1]) == cudaSuccess) { ms += t; fl += h->ev_flops[q]; mx = std::max(mx, (double)t); }
    }
    *val = (k == "gemm_time_ms") ? ms : (k == "gemm_flops_timed") ? fl : (k == "gemm_time_max_ms") ? mx : (double)h->ev_flops.size();
  }
  else if (k == "reset_counters") { h->ev_used = 0; h->ev_flops.clear(); h->ev_ops8.clear(); *val = 0; h->st_gemm_launches = h->st_kernel_launches = h->st_flops_exec = h->st_sigma_apps = h->st_graph_launches = h->st_dense_apps = 0; }
  else { h->err = "gfcc_get_stat: unknown key " + k; return GFCC_EINVAL; }
  return GFCC_OK;
}

extern "C" int gfcc_get_residuals(gfcc_handle h, int n, double* relres, int* iters) {
  if (!h || n < 0 || (size_t)n > h->last_relres.size()) return GFCC_EINVAL;
  for (int k = 0; k < n; ++k) {
    if (relres) relres[k] = h->last_relres[k];
    if (iters) iters[k] = h->last_iters[k];
  }
  return GFCC_OK;
}

extern "C" long long gfcc_get_intermediate(gfcc_handle h, const char* name, double* out) {
  if (!h || !name) return GFCC_EINVAL;
  const long long o = h->o, v = h->v, Q = h->Q, np_ = h->npair;
  std::string k(name);
  const double* src = nullptr; long long n = 0;
  if (k == "Fme") { src = h->Fme; n = o * v; }
  else if (k == "Fmi") { src = h->Fmi; n = o * o; }
  else if (k == "Fae") { src = h->Fae; n = v * v; }
  else if (k == "Wmnij") { src = h->Wp; n = np_ * np_; }
  else if (k == "Wmbij") { src = h->WB; n = np_ * v * o; }
  else if (k == "D") { src = h->D; n = o * o; }
  else if (k == "Lm") { src = h->Lm; n = Q * o * v; }
  else { h->err = "gfcc_get_intermediate: unknown name " + k; return GFCC_EINVAL; }
  if (out) {
    if (cudaMemcpyAsync(out, src, (size_t)n * 8, cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess) { h->err = "copy failed"; return GFCC_ECUDA; }
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) { h->err = "sync failed"; return GFCC_ECUDA; }
  }
  return n;
}

// ------------------------------------------------------------------------------------------
// gfcc_sigma_ip
// ------------------------------------------------------------------------------------------
static int sigma_abi(gfcc_handle h, int nrhs, const double* omega, double eta, const void* X1, const void* X2, void* S1, void* S2) {
  const int o = h->o, v = h->v;
  TRY(ensure_workspace(h, nrhs, true));
  cudaStream_t st = h->stream;
  CUDA_TRY(h, cudaMemcpyAsync(h->d_omega, omega, (size_t)nrhs * 8, cudaMemcpyHostToDevice, st));
  dim3 blk(32, 8), grid((unsigned)((h->nvec + 31) / 32), (unsigned)((nrhs + 31) / 32));
  k_abi_to_vec<<<grid, blk, 0, st>>>(h->vin, (const double2*)X1, (const double2*)X2, o, v, nrhs);
  KLAUNCH(h);
  TRY(sigma_internal(h, nrhs, h->d_omega, eta, h->vin, h->vout));
  k_vec_to_abi<<<grid, blk, 0, st>>>((double2*)S1, (double2*)S2, h->vout, o, v, nrhs);
  KLAUNCH(h);
  k_zero_diag<<<nblk((long long)nrhs * o * v), 256, 0, st>>>((double2*)S2, o, v, nrhs);
  KLAUNCH(h);
  h->st_flops_sigma = sigma_flops(h, nrhs);
  return GFCC_OK;
}

extern "C" int gfcc_sigma_ip(gfcc_handle h, int nrhs, const double* omega, double eta, const void* X1, const void* X2,
                             void* S1, void* S2) {
  if (!h) return GFCC_EINVAL;
  if (nrhs < 1 || !omega || !X1 || !X2 || !S1 || !S2) { h->err = "gfcc_sigma_ip: null pointer or nrhs < 1"; return GFCC_EINVAL; }
  return sigma_abi(h, nrhs, omega, eta, X1, X2, S1, S2);
}

extern "C" int gfcc_sigma_ip_host(gfcc_handle h, int nrhs, const double* omega, double eta, const void* X1, const void* X2,
                                  void* S1, void* S2) {
  if (!h) return GFCC_EINVAL;
  if (nrhs < 1 || !omega || !X1 || !X2 || !S1 || !S2) { h->err = "gfcc_sigma_ip_host: null pointer or nrhs < 1"; return GFCC_EINVAL; }
  const long long o = h->o, v = h->v;
  const long long n1 = (long long)nrhs * o * 2, n2 = (long long)nrhs * o * o * v * 2;
  TRY(ensure_workspace(h, nrhs, true));
  // stage the ABI-layout vectors in the Z and V scratch (each o*v*o*Nc doubles = exactly one X2 batch)
  double* dX2 = h->V;      // V is written late in sigma_internal, after vin has been built
  double* dS2 = h->XU;     // XU is dead when the result is unpacked
  double *dX1 = nullptr, *dS1 = nullptr;
  TRY(dev_alloc(h, &dX1, n1)); TRY(dev_alloc(h, &dS1, n1));
  cudaStream_t st = h->stream;
  int rc = GFCC_OK;
  do {
    if (cudaMemcpyAsync(dX1, X1, (size_t)n1 * 8, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(dX2, X2, (size_t)n2 * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) { h->err = "H2D copy failed"; rc = GFCC_ECUDA; break; }
    rc = sigma_abi(h, nrhs, omega, eta, dX1, dX2, dS1, dS2);
    if (rc) break;
    if (cudaMemcpyAsync(S1, dS1, (size_t)n1 * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(S2, dS2, (size_t)n2 * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) { h->err = "D2H copy failed"; rc = GFCC_ECUDA; break; }
    if (cudaStreamSynchronize(st) != cudaSuccess) { h->err = "sync failed"; rc = GFCC_ECUDA; }
  } while (0);
  cudaStreamSynchronize(st);
  dev_free(h, dX1, n1); dev_free(h, dS1, n1);
  return rc;
}

extern "C" int gfcc_dgemm(void* stream, int M, int N, int K, double alpha, const double* A, long long sAm, long long sAk,
                          const double* B, long long sBk, long long sBn, double beta, double* C, long long sCm, long long sCn) {
  if (M < 0 || N < 0 || K < 0 || !A || !B || !C) return GFCC_EINVAL;
  if ((sAm != 1 && sAk != 1) || (sBk != 1 && sBn != 1)) return GFCC_EINVAL;
  GemmDesc d; d.M = M; d.N = N; d.K0 = K;
  d.A = A; d.sAm = sAm; d.sAk0 = sAk; d.B = B; d.sBk0 = sBk; d.sBn = sBn;
  if (sAk == 1 && sAm == 1) d.sAm = (K > 1) ? K : 1;   // degenerate: treat as K-contiguous row
  d.C = C; d.sCm0 = sCm; d.sCn0 = sCn; d.alpha = alpha; d.beta = beta;
  if (K == 0) d.K0 = 0;
  cudaError_t e = launch_dgemm(d, (cudaStream_t)stream);
  return e == cudaSuccess ? GFCC_OK : GFCC_ECUDA;
}

// FP64-accurate GEMM on the INT8 tensor pipe (gfcc_ozaki.cuh): C = alpha*A*B + beta*C, same operand
// conventions as gfcc_dgemm.  Synchronous; temporary slices are allocated and freed inside.  ms_slice / ms_gemm (nullable)
// receive the CUDA-event times of the slicing pass and of the tensor-core kernel.
extern "C" int gfcc_dgemm_ozaki(void* stream, int M, int N, int K, double alpha, const double* A, long long sAm, long long sAk,
                                const double* B, long long sBk, long long sBn, double beta, double* C, long long sCm, long long sCn,
                                int nslices, double* ms_slice, double* ms_gemm) {
  if (M < 1 || N < 1 || K < 1 || !A || !B || !C || nslices < 1 || nslices > OZ_MAX_SLICES) return GFCC_EINVAL;
  if ((sAm != 1 && sAk != 1) || (sBk != 1 && sBn != 1)) return GFCC_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  OzOperand a, b;
  a.base = A; a.sR = sAm; a.sK0 = sAk; a.R = M; a.K0 = K;
  b.base = B; b.sR = sBn; b.sK0 = sBk; b.R = N; b.K0 = K;
  OzSliced sa, sb;
  oz_shape(sa, M, K, nslices); oz_shape(sb, N, K, nslices);
  int* fail = nullptr;
  cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
  int rc = GFCC_OK;
  auto cleanup = [&]() {
    cudaFree(sa.q); cudaFree(sa.scale); cudaFree(sa.amax); cudaFree(sb.q); cudaFree(sb.scale); cudaFree(sb.amax); cudaFree(fail);
    for (auto e : ev) if (e) cudaEventDestroy(e);
  };
  do {
    if (cudaMalloc(&sa.q, sa.bytes()) != cudaSuccess || cudaMalloc(&sb.q, sb.bytes()) != cudaSuccess ||
        cudaMalloc(&sa.scale, (size_t)M * 8) != cudaSuccess || cudaMalloc(&sb.scale, (size_t)N * 8) != cudaSuccess ||
        cudaMalloc(&sa.amax, (size_t)M * 8) != cudaSuccess || cudaMalloc(&sb.amax, (size_t)N * 8) != cudaSuccess ||
        cudaMalloc(&fail, 2 * sizeof(int)) != cudaSuccess) { rc = GFCC_ENOMEM; break; }
    for (auto& e : ev) if (cudaEventCreate(&e) != cudaSuccess) { rc = GFCC_ECUDA; break; }
    if (rc) break;
    cudaMemsetAsync(fail, 0, 2 * sizeof(int), st);
    cudaEventRecord(ev[0], st);
    if (oz_slice(a, sa, st) != cudaSuccess || oz_slice(b, sb, st) != cudaSuccess) { rc = GFCC_ECUDA; break; }
    cudaEventRecord(ev[1], st);
    OzCDesc c; c.C = C; c.sCm0 = sCm; c.sCn0 = sCn; c.alpha = alpha; c.beta = beta;
    if (oz_igemm(sa, sb, c, fail, st, 148, nullptr, reinterpret_cast<unsigned*>(fail) + 1) != cudaSuccess) { rc = GFCC_ECUDA; break; }
    cudaEventRecord(ev[2], st);
    if (cudaStreamSynchronize(st) != cudaSuccess) { rc = GFCC_ECUDA; break; }
    int hfail = 0;
    cudaMemcpy(&hfail, fail, sizeof(int), cudaMemcpyDeviceToHost);
    if (hfail) { rc = GFCC_ECUDA; break; }
    float t = 0;
    if (ms_slice) { cudaEventElapsedTime(&t, ev[0], ev[1]); *ms_slice = t; }
    if (ms_gemm) { cudaEventElapsedTime(&t, ev[1], ev[2]); *ms_gemm = t; }
  } while (0);
  if (rc != GFCC_OK) cudaGetLastError();
  cleanup();
  return rc;
}

// ------------------------------------------------------------------------------------------
// gfcc_dgemm_splitk_noalloc: split-K FP64 GEMM that allocates NOTHING (include/gfcc.h).
// The handle-based split-K path (gemm_splitk above) keeps its partial sums in h->part, a cudaMalloc'ed buffer.  Callers that must not
// call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it) get the same two kernels -- the DMMA
// GEMM writing one partial product per K chunk, then k_splitk_reduce -- with the partials in this file-scope device array.  Every GPU
// that loads the library holds the array (16 MiB) until the process exits.  In HOST code the name g_noalloc_scratch is only a stand-in
// for the symbol, NOT a device address: the address is fetched once per device with cudaGetSymbolAddress and that pointer goes to the
// kernels.
// ------------------------------------------------------------------------------------------
#define GFCC_NOALLOC_SCRATCH_DOUBLES (1LL << 21)   /* 2 097 152 doubles = 16 MiB; keep in step with include/gfcc.h */
static __device__ __align__(256) double g_noalloc_scratch[GFCC_NOALLOC_SCRATCH_DOUBLES];

static int noalloc_scratch_ptr(double** out) {
  constexpr int MAXDEV = 64;
  static double* ptr[MAXDEV] = {nullptr};
  static std::mutex mtx;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAXDEV) { cudaGetLastError(); return GFCC_ECUDA; }
  std::lock_guard<std::mutex> lock(mtx);
  if (!ptr[dev]) {   // once per device, with that device current
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      g_create_error = std::string("gfcc_dgemm_splitk_noalloc: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e);
      cudaGetLastError();
      return GFCC_ECUDA;
    }
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return GFCC_OK;
}

extern "C" int gfcc_dgemm_splitk_noalloc(void* stream, int M, int N, int K, double alpha, const double* A, long long sAm,
                                         long long sAk, const double* B, long long sBk, long long sBn, double beta, double* C,
                                         long long sCm, long long sCn, int splits) {
  if (M < 1 || N < 1 || K < 1 || splits < 1 || !A || !B || !C) {
    g_create_error = "gfcc_dgemm_splitk_noalloc: null pointer or non-positive size";
    return GFCC_EINVAL;
  }
  if ((sAm != 1 && sAk != 1) || (sBk != 1 && sBn != 1)) {
    g_create_error = "gfcc_dgemm_splitk_noalloc: one stride of A and one stride of B must be 1";
    return GFCC_EINVAL;
  }
  const int S = std::min(splits, K);
  const int chunk = (K + S - 1) / S;             // K elements per part; every part is non-empty
  const int full = K / chunk, tail = K - full * chunk;
  const int nparts = full + (tail > 0 ? 1 : 0);
  const long long need = (long long)nparts * M * N;
  if (need > GFCC_NOALLOC_SCRATCH_DOUBLES) {
    char buf[256];
    snprintf(buf, sizeof buf, "gfcc_dgemm_splitk_noalloc: %d parts x %d x %d = %lld doubles of partial sums exceed the built-in scratch "
             "of %lld doubles (16 MiB): use fewer splits or gfcc_dgemm", nparts, M, N, need, (long long)GFCC_NOALLOC_SCRATCH_DOUBLES);
    g_create_error = buf;
    return GFCC_EINVAL;
  }
  double* part = nullptr;
  const int rcp = noalloc_scratch_ptr(&part);
  if (rcp != GFCC_OK) return rcp;
  cudaStream_t st = (cudaStream_t)stream;
  // part[z][m][n] = sum over chunk z of A B.  beta = 0: every element of the parts in use is overwritten, nothing has to start at zero
  // (the array keeps the previous call's contents beyond them, which nothing reads).
  GemmDesc g; g.M = M; g.N = N; g.K0 = chunk;
  g.A = A; g.sAm = sAm; g.sAk0 = sAk; g.B = B; g.sBk0 = sBk; g.sBn = sBn;
  if (sAk == 1 && sAm == 1) g.sAm = (K > 1) ? K : 1;
  g.C = part; g.sCm0 = N; g.sCn0 = 1; g.alpha = 1.0; g.beta = 0.0;
  g.batch = full; g.bsA = (long long)chunk * sAk; g.bsB = (long long)chunk * sBk; g.bsC = (long long)M * N;
  if (full > 0 && launch_dgemm(g, st) != cudaSuccess) { g_create_error = "gfcc_dgemm_splitk_noalloc: GEMM launch failed"; cudaGetLastError(); return GFCC_ECUDA; }
  if (tail > 0) {
    GemmDesc t = g;
    t.K0 = tail; t.batch = 1;
    t.A = A + (long long)full * chunk * sAk; t.B = B + (long long)full * chunk * sBk; t.C = part + (long long)full * M * N;
    if (launch_dgemm(t, st) != cudaSuccess) { g_create_error = "gfcc_dgemm_splitk_noalloc: GEMM launch failed"; cudaGetLastError(); return GFCC_ECUDA; }
  }
  const long long tot = (long long)M * N;
  k_splitk_reduce<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(C, part, nparts, M, N, alpha, beta, sCm, 0, M, sCn, 0, N);
  if (cudaGetLastError() != cudaSuccess) { g_create_error = "gfcc_dgemm_splitk_noalloc: reduction launch failed"; return GFCC_ECUDA; }
  return GFCC_OK;
}

extern "C" int gfcc_probe_fp64_peak(void* stream, int iters, int reps, double* tflops) {
  if (!tflops || iters < 1 || reps < 1) return GFCC_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return GFCC_ECUDA; }
  const double t = dmma_peak_probe((cudaStream_t)stream, iters, reps);
  if (t < 0) return GFCC_ECUDA;
  *tflops = t;
  return GFCC_OK;
}

// ------------------------------------------------------------------------------------------
// gfcc_solve_ip : batched GMRES + G assembly (gfcc_solve.cuh holds the kernels and the driver loop)
// ------------------------------------------------------------------------------------------
extern "C" int gfcc_solve_ip_x(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol,
                               void* G, void* X1out, void* X2out) {
  if (!h) return GFCC_EINVAL;
  if (np < 1 || nw < 1 || !p || !omega || !G || !(tol > 0)) { h->err = "gfcc_solve_ip: null pointer, np/nw < 1 or tol <= 0"; return GFCC_EINVAL; }
  for (int k = 0; k < np; ++k)
    if (p[k] < 0 || p[k] >= h->N) { h->err = "gfcc_solve_ip: target orbital out of range"; return GFCC_EINVAL; }
  const int ntot = np * nw;
  h->last_relres.assign(ntot, 0.0);
  h->last_iters.assign(ntot, 0);
  h->last_hist.assign(ntot, std::vector<double>());
  h->st_iterations = 0;
  std::vector<SolveTask> tasks(ntot);
  for (int ip = 0; ip < np; ++ip)
    for (int iw = 0; iw < nw; ++iw) { tasks[ip * nw + iw].p = p[ip]; tasks[ip * nw + iw].omega = omega[iw]; }
  const int batch = std::max(1, std::min(ntot, (int)h->opt_max_batch));
  TRY(ensure_workspace(h, batch, false));
  double* Gq = nullptr;   // [ntot][np] complex
  TRY(dev_alloc(h, &Gq, (long long)ntot * np * 2));
  int* dq = nullptr;
  { double* t = nullptr; int rc = dev_alloc(h, &t, np); if (rc) { dev_free(h, Gq, (long long)ntot * np * 2); return rc; } dq = (int*)t; }
  int rc_final = GFCC_OK;
  do {
    if (cudaMemcpyAsync(dq, p, (size_t)np * sizeof(int), cudaMemcpyHostToDevice, h->stream) != cudaSuccess) { h->err = "H2D failed"; rc_final = GFCC_ECUDA; break; }
    SolveCfg cfg;
    cfg.o = h->o; cfg.v = h->v; cfg.nvec = h->nvec; cfg.npair = h->npair;
    cfg.m = (int)h->opt_m; cfg.maxit = (int)h->opt_maxit; cfg.fixed = (int)h->opt_fixed; cfg.x0 = (int)h->opt_x0;
    cfg.batch = batch; cfg.compact = h->opt_compact;
    // polling period of the device-side done flags: every step when one sigma application is long, every 4th for tiny systems
    cfg.poll = h->opt_poll > 0 ? (int)h->opt_poll : (sigma_flops(h, batch) < 5e9 ? 4 : 1);
    cfg.eta = eta; cfg.tol = tol;
    cfg.t1 = h->t1; cfg.l1 = h->l1; cfg.T2p = h->T2p; cfg.L2p = h->L2p; cfg.D = h->D; cfg.fdiag = h->fdiag;
    cfg.stream = h->stream;
    const bool tiny = sigma_flops(h, batch) < 5e9;
    const bool dense = dense_wanted(h);
    if (dense) { const int rcd = dense_build(h); if (rcd != GFCC_OK) { rc_final = rcd; break; } }
    SigmaFn apply = [&](int nrhs, const double* d_omega, const double* xin, double* sout) -> int {
      if (dense) return dense_apply(h, nrhs, d_omega, eta, xin, sout);
      const bool graph = (h->opt_graph == 1 || (h->opt_graph < 0 && tiny)) && !h->prof && h->opt_engine == 0 && h->opt_overlap == 0;
      return graph ? sigma_via_graph(h, nrhs, d_omega, eta, xin, sout) : sigma_internal(h, nrhs, d_omega, eta, xin, sout);
    };
    cudaStream_t st = h->stream;
    SolveHooks hooks;
    // G1: b_p and the zeroth-order guess for the batch columns [c0, A)
    hooks.init = [&](double* b, double* x, int A, int c0, const int* p_col, const double* omega_col, double* nl) -> int {
      const long long tot = h->nvec * (A - c0);
      k_build_rhs<<<nblk(tot, 256, 148LL * 16), 256, 0, st>>>(b, p_col, h->t1, h->T2p, h->o, h->v, A, h->nvec, c0);
      k_x0<<<(unsigned)(h->npair + 1), 256, 0, st>>>(x, b, omega_col, eta, h->fdiag, h->o, h->v, A, cfg.x0, c0);
      *nl += 2;
      return cudaGetLastError() == cudaSuccess ? 0 : GFCC_ECUDA;
    };
    // G6: g = Lambda2 . X2 and G_pq for the retired columns; optional X output in the C-ABI layout
    hooks.finish = [&](const double* xr, int ld, int nret, const int* ret_row, double* nl) -> int {
      SolveWs& s = h->sw;
      const int Nc = 2 * ld;
      dim3 grid((2 * nret + LG_CC - 1) / LG_CC, s.g_blocks);
      static bool attr_set = false;
      if (!attr_set) { cudaFuncSetAttribute(k_lambda2_g, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); attr_set = true; }
      k_lambda2_g<<<grid, 32 * LG_WARPS, lambda2_g_smem_bytes(h->v), st>>>(s.gpart, h->L2p, xr, h->o, h->v, Nc, h->npair);
      const long long n = (long long)h->v * Nc;
      k_g_reduce<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(s.gvec, s.gpart, s.g_blocks, n);
      dim3 gg(np, nret);
      k_assemble_G<<<gg, 256, 0, st>>>((double2*)Gq, dq, np, xr, s.gvec, h->D, h->t1, h->l1, h->o, h->v, ld, ret_row);
      *nl += 3;
      if (X1out && X2out) {
        dim3 blk(32, 8), g2((unsigned)((h->nvec + 31) / 32), (unsigned)((nret + 31) / 32));
        k_vec_to_abi<<<g2, blk, 0, st>>>((double2*)X1out, (double2*)X2out, xr, h->o, h->v, nret, ld, ret_row);
        const long long tot = (long long)nret * h->o * h->v;
        k_zero_diag<<<(unsigned)std::min<long long>(4096, (tot + 255) / 256), 256, 0, st>>>((double2*)X2out, h->o, h->v, nret, ret_row);
        *nl += 2;
      }
      return cudaGetLastError() == cudaSuccess ? 0 : GFCC_ECUDA;
    };
    std::string err;
    double nlaunch = 0;
    int rc = solve_run(h->sw, cfg, tasks, apply, hooks, &h->last_hist, &nlaunch, err);
    h->st_kernel_launches += nlaunch;
    if (rc == GFCC_ENOCONV) rc_final = GFCC_ENOCONV;
    else if (rc != GFCC_OK) { h->err = err; rc_final = rc; break; }
    // G[iw][ip][iq] <- Gq[(ip*nw+iw)][iq]
    std::vector<double> hostG((size_t)ntot * np * 2), outG((size_t)ntot * np * 2);
    if (cudaMemcpyAsync(hostG.data(), Gq, hostG.size() * 8, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaStreamSynchronize(h->stream) != cudaSuccess) { h->err = "D2H of G failed"; rc_final = GFCC_ECUDA; break; }
    for (int ip = 0; ip < np; ++ip)
      for (int iw = 0; iw < nw; ++iw)
        for (int iq = 0; iq < np; ++iq)
          for (int c = 0; c < 2; ++c)
            outG[(((size_t)iw * np + ip) * np + iq) * 2 + c] = hostG[(((size_t)ip * nw + iw) * np + iq) * 2 + c];
    if (cudaMemcpy(G, outG.data(), outG.size() * 8, cudaMemcpyDefault) != cudaSuccess) { h->err = "copy of G to the caller failed"; rc_final = GFCC_ECUDA; break; }
  } while (0);
  cudaStreamSynchronize(h->stream);
  dev_free(h, Gq, (long long)ntot * np * 2);
  dev_free(h, (double*)dq, np);
  h->st_max_relres = 0; h->st_nunconv = 0;
  for (int k = 0; k < ntot; ++k) {
    h->last_relres[k] = tasks[k].relres;
    h->last_iters[k] = tasks[k].iters;
    h->st_iterations = std::max(h->st_iterations, (double)tasks[k].iters);
    h->st_max_relres = std::max(h->st_max_relres, tasks[k].relres);
    if (h->opt_fixed == 0 && !tasks[k].converged) h->st_nunconv += 1;
  }
  h->st_flops_sigma = sigma_flops(h, batch);
  return rc_final;
}

extern "C" int gfcc_solve_ip(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol, void* G) {
  return gfcc_solve_ip_x(h, np, p, nw, omega, eta, tol, G, nullptr, nullptr);
}

// relative residual of right-hand side `rhs` of the last solve after each of its sigma applications
extern "C" int gfcc_get_residual_history(gfcc_handle h, int rhs, int cap, double* hist, int* n_out) {
  if (!h || rhs < 0 || (size_t)rhs >= h->last_hist.size() || cap < 0 || (cap > 0 && !hist)) return GFCC_EINVAL;
  const std::vector<double>& v = h->last_hist[rhs];
  if (n_out) *n_out = (int)v.size();
  for (int k = 0; k < cap && k < (int)v.size(); ++k) hist[k] = v[k];
  return GFCC_OK;
}

// G assembly of caller-provided vectors (first term of Eq. 7-8): Gout[r][iq] = c_{q[iq]} . X_r
extern "C" int gfcc_assemble_g(gfcc_handle h, int nrhs, const void* X1, const void* X2, int nq, const int* q, void* Gout) {
  if (!h) return GFCC_EINVAL;
  if (nrhs < 1 || nq < 1 || !X1 || !X2 || !q || !Gout) { h->err = "gfcc_assemble_g: null pointer or nrhs/nq < 1"; return GFCC_EINVAL; }
  for (int k = 0; k < nq; ++k)
    if (q[k] < 0 || q[k] >= h->N) { h->err = "gfcc_assemble_g: orbital out of range"; return GFCC_EINVAL; }
  const int o = h->o, v = h->v;
  const long long Nc = 2LL * nrhs;
  cudaStream_t st = h->stream;
  const int g_blocks = (int)std::min<long long>(296, h->npair);
  double *vec = nullptr, *gpart = nullptr, *gvec = nullptr, *Gq = nullptr, *dqd = nullptr;
  int rc = GFCC_OK;
  do {
    if ((rc = dev_alloc(h, &vec, h->nvec * Nc))) break;
    if ((rc = dev_alloc(h, &gpart, (long long)g_blocks * v * Nc))) break;
    if ((rc = dev_alloc(h, &gvec, (long long)v * Nc))) break;
    if ((rc = dev_alloc(h, &Gq, (long long)nrhs * nq * 2))) break;
    if ((rc = dev_alloc(h, &dqd, nq))) break;
    int* dq = (int*)dqd;
    rc = GFCC_ECUDA;
    if (cudaMemcpyAsync(dq, q, (size_t)nq * sizeof(int), cudaMemcpyHostToDevice, st) != cudaSuccess) { h->err = "H2D failed"; break; }
    dim3 blk(32, 8), grid((unsigned)((h->nvec + 31) / 32), (unsigned)((nrhs + 31) / 32));
    k_abi_to_vec<<<grid, blk, 0, st>>>(vec, (const double2*)X1, (const double2*)X2, o, v, nrhs);
    h->st_kernel_launches += 1;
    if (cudaFuncSetAttribute(k_lambda2_g, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess) { h->err = "smem attribute"; break; }
    dim3 lg((unsigned)((Nc + LG_CC - 1) / LG_CC), g_blocks);
    k_lambda2_g<<<lg, 32 * LG_WARPS, lambda2_g_smem_bytes(v), st>>>(gpart, h->L2p, vec, o, v, (int)Nc, h->npair);
    const long long n = (long long)v * Nc;
    k_g_reduce<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(gvec, gpart, g_blocks, n);
    dim3 gg(nq, nrhs);
    k_assemble_G<<<gg, 256, 0, st>>>((double2*)Gq, dq, nq, vec, gvec, h->D, h->t1, h->l1, o, v, nrhs, nullptr);
    h->st_kernel_launches += 3;
    if (cudaGetLastError() != cudaSuccess) { h->err = "gfcc_assemble_g: launch failed"; break; }
    if (cudaMemcpyAsync(Gout, Gq, (size_t)nrhs * nq * 16, cudaMemcpyDefault, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) { h->err = "gfcc_assemble_g: copy of G failed"; break; }
    rc = GFCC_OK;
  } while (0);
  cudaStreamSynchronize(st);
  dev_free(h, vec, h->nvec * Nc); dev_free(h, gpart, (long long)g_blocks * v * Nc); dev_free(h, gvec, (long long)v * Nc);
  dev_free(h, Gq, (long long)nrhs * nq * 2); dev_free(h, dqd, nq);
  return rc;
}

#include "gfcc_ea_host.inl"
#include "gfcc_mor_host.inl"
#include "gfcc_workflow_host.inl"
