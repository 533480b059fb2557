// =====================================================================================
// gfcc_solve.cuh -- batched GMRES with converged-RHS compaction and G_pq assembly.
//
// GMRES (Saad & Schultz, PAPER.md ref. 85) for a batch of right-hand sides in lockstep on the
// RHS-fastest internal vectors vec[n][2*A] (A = active columns):
//   Arnoldi with classical Gram-Schmidt + one re-orthogonalisation (CGS2): ONE block-dot launch and ONE block-axpy launch per
//   pass over the whole basis (each basis vector read once per pass, w read/written once by the axpy; HBM-bound, coalesced
//   along the RHS columns);
//   per-RHS complex Givens rotations / least squares in a tiny device kernel (one thread per RHS); the done flags stay on
//   the device and are polled every `poll` steps.
// Load balance ("convergence ... for different (omega,p) pairs would become different and lead to severe
// load imbalance"; PAPER.md:253 a group that finishes early "will be told to proceed to pick another orbital"; iteration
// counts 1-2 vs 5-40): the analogue of the paper's dynamic task pick on one GPU is
//   COMPACTION -- columns whose stop test has fired are finalised (x += V y), moved to a retirement buffer and dropped from
//                 every live vector, so the GEMM N dimension of the next sigma application shrinks with the active set;
//   REFILL     -- at every restart boundary the free columns are given to the next pending (p, omega) tasks.
// Per-RHS small arrays are addressed by the SLOT a task occupies for its life in the batch (stride = batch capacity), so
// only the big vectors move (one gather pass each).
// G assembly (Eq. 7-8 first term, cheap form of SURVEY.md 8c item 10) runs on the retirement buffer:
//   g[b] = sum_ija lambda[i,j,b,a] x2[i,j,a];   q=k occ: G = x1[k] - sum_i D[k,i] x1[i] + sum_ja l1[j,a] x2[k,j,a] - 1/2 sum_b t1[k,b] g[b]
//   q=o+c virt: G = sum_i l1[i,c] x1[i] + 1/2 g[c].
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <cmath>
#include <string>
#include <vector>
#include <functional>
#include <algorithm>
#include "gfcc_kernels.cuh"

namespace gfcc {

struct SolveCfg {
  int o, v; long long nvec, npair;
  int m, maxit, fixed, x0, poll, batch;   // batch: column capacity B
  double compact;                         // compact when at least max(1, compact*A) finished columns are still in the batch (<0: never)
  double eta, tol;
  const double *t1, *l1, *T2p, *L2p, *D, *fdiag;
  cudaStream_t stream;
};

struct SolveWs {
  int cap = 0, mcap = 0, histcap = 0; long long nvec = 0;
  double bytes = 0;
  std::vector<void*> allocs;
  std::vector<double*> V;                 // mcap + 1 basis vectors, each [nvec][2*cap]
  double *x = nullptr, *b = nullptr, *w = nullptr, *xr = nullptr, *spare = nullptr;
  double2 *H = nullptr, *R = nullptr, *cs = nullptr, *g = nullptr, *y = nullptr, *part = nullptr, *hn2 = nullptr, *bn2 = nullptr;
  double *sn = nullptr, *scale = nullptr, *res = nullptr, *gvec = nullptr, *gpart = nullptr, *hist = nullptr, *omega_col = nullptr;
  int *stat = nullptr;                    // [done(cap) | jstop(cap) | age(cap)]
  int *slot_col = nullptr, *p_col = nullptr, *map = nullptr, *ret_row = nullptr;
  const double** vptr = nullptr;          // device copy of {V_0..V_mcap, w, b}
  int dot_blocks = 0, g_blocks = 0;
  // statistics of the last run
  int m_run = 0; long long compactions = 0, refills = 0, polls = 0; double active_col_steps = 0, full_col_steps = 0;
};

inline void solve_free(SolveWs& s) {
  for (void* p : s.allocs) cudaFree(p);
  s = SolveWs();
}

// ---- right-hand sides b_p in the internal layout, columns [c0, nrhs); imaginary parts are zero ----
__global__ void k_build_rhs(double* __restrict__ b, const int* __restrict__ p_of_rhs, const double* __restrict__ t1,
                            const double* __restrict__ T2p, int o, int v, int nrhs, long long nvec, int c0 = 0) {
  const int nc = nrhs - c0;
  const long long total = nvec * nc;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long row = idx / nc;
    const int r = c0 + (int)(idx - row * nc);
    const int p = p_of_rhs[r];
    double val = 0.0;
    if (p < o) { if (row == p) val = 1.0; }
    else {
      const int c = p - o;
      if (row < o) val = t1[row * v + c];
      else {
        const long long q = row - o;
        const long long pr = q / v;
        const int a = q % v;
        val = T2p[(pr * v + c) * v + a];   // t[i,j,c,a]
      }
    }
    reinterpret_cast<double2*>(b)[row * nrhs + r] = make_double2(val, 0.0);
  }
}
// x0 = b / (omega - i eta + d),  d_i = -f_ii, d_ija = f_aa - f_ii - f_jj  (reading 11); kind 0: x0 = 0.
// Columns [c0, nrhs).  Block 0 handles the o singles rows, block 1 + pr the v rows of pair pr (decoded once per block);
// one reciprocal per element.
__global__ void __launch_bounds__(256) k_x0(double* __restrict__ x, const double* __restrict__ b, const double* __restrict__ omega,
                                            double eta, const double* __restrict__ fdiag, int o, int v, int nrhs, int kind, int c0) {
  const int nc = nrhs - c0;
  long long row0; int nrow; double dbase;
  if (blockIdx.x == 0) { row0 = 0; nrow = o; dbase = 0.0; }
  else {
    const long long pr = blockIdx.x - 1;
    int i, j;
    decode_pair(pr, o, i, j);
    row0 = (long long)o + pr * v; nrow = v; dbase = -fdiag[i] - fdiag[j];
  }
  const int total = nrow * nc;
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int a = t / nc, r = c0 + (t - a * nc);
    const long long idx = (row0 + a) * nrhs + r;
    double2 out = make_double2(0.0, 0.0);
    if (kind == 1) {
      const double d = blockIdx.x == 0 ? -fdiag[a] : dbase + fdiag[o + a];
      const double re = omega[r] + d;
      const double inv = 1.0 / (re * re + eta * eta);
      const double2 bb = reinterpret_cast<const double2*>(b)[idx];
      out.x = (bb.x * re - bb.y * eta) * inv;     // b / (re - i eta) = b (re + i eta) / (re^2 + eta^2)
      out.y = (bb.y * re + bb.x * eta) * inv;
    }
    reinterpret_cast<double2*>(x)[idx] = out;
  }
}

// start of a cycle: beta = sqrt(rn2), res = beta/bnorm; scale = done ? 0 : 1/beta; g[0] = beta.
// One thread per ACTIVE column r; every array is addressed by the column's slot s = slot[r] with stride ldc.
__global__ void k_cycle_start(const double2* __restrict__ rn2, const double2* __restrict__ bn2, double2* __restrict__ g,
                              double* __restrict__ scale, double* __restrict__ res, int* __restrict__ done,
                              int* __restrict__ jstop, int* __restrict__ age, double* __restrict__ hist, int histcap, int nrhs,
                              int mp1, double tol, int fixed, const int* __restrict__ slot, int ldc) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nrhs) return;
  const int s = slot[r];
  const double beta = sqrt(fmax(rn2[s].x, 0.0));
  const double bn = sqrt(fmax(bn2[s].x, 0.0));
  for (int k = 0; k < mp1; ++k) g[(long long)k * ldc + s] = make_double2(0.0, 0.0);
  jstop[s] = 0;
  if (done[s]) { scale[s] = 0.0; return; }
  const double rr = (bn > 0.0) ? beta / bn : 0.0;
  res[s] = rr;
  const int ag = age[s]++;
  if (ag < histcap) hist[(long long)ag * ldc + s] = rr;
  if ((!fixed && rr <= tol) || beta == 0.0) { done[s] = 1; scale[s] = 0.0; return; }
  g[s] = make_double2(beta, 0.0);
  scale[s] = 1.0 / beta;
}

// one Arnoldi column for every active RHS: H[0..j] (CGS2 coefficients), hn2 = ||w||^2.
// Applies the previous rotations, forms the new one, updates g, decides convergence, sets the scale of v_{j+1}.
// R is stored with the CAPACITY stride mcap + 1 per column.
__global__ void k_givens(int j, int mcap, int nrhs, double2* __restrict__ H, const double2* __restrict__ Hcorr, const double2* __restrict__ hn2,
                         double2* __restrict__ R, double2* __restrict__ cs, double* __restrict__ sn, double2* __restrict__ g,
                         double* __restrict__ res, const double2* __restrict__ bn2, double tol, int* __restrict__ done,
                         int* __restrict__ jstop, int* __restrict__ age, double* __restrict__ hist, int histcap,
                         double* __restrict__ scale, int fixed, const int* __restrict__ slot, int ldc) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nrhs) return;
  const int s = slot[r];
  if (done[s]) { scale[s] = 0.0; return; }
  const long long L = ldc;
  const double hn = sqrt(fmax(hn2[s].x, 0.0));
  for (int k = 0; k <= j; ++k) {   // CGS2: h = first-pass coefficients + re-orthogonalisation correction
    const double2 cr = Hcorr[k * L + s];
    H[k * L + s].x += cr.x; H[k * L + s].y += cr.y;
  }
  for (int k = 0; k < j; ++k) {
    const double2 a = H[k * L + s], b = H[(k + 1) * L + s];
    const double2 c = cs[k * L + s];
    const double sk = sn[k * L + s];
    // [ conj(c)  s ] [a]
    // [ -s       c ] [b]
    H[k * L + s] = make_double2(c.x * a.x + c.y * a.y + sk * b.x, c.x * a.y - c.y * a.x + sk * b.y);
    H[(k + 1) * L + s] = make_double2(-sk * a.x + c.x * b.x - c.y * b.y, -sk * a.y + c.x * b.y + c.y * b.x);
  }
  const double2 a = H[j * L + s];
  const double den = sqrt(a.x * a.x + a.y * a.y + hn * hn);
  const int ag = age[s]++;
  if (den == 0.0) {   // zero column: nothing left in the Krylov space
    done[s] = 1; scale[s] = 0.0; jstop[s] = j;
    if (ag < histcap) hist[(long long)ag * L + s] = res[s];
    return;
  }
  const double2 c = make_double2(a.x / den, a.y / den);
  const double sj = hn / den;
  cs[j * L + s] = c;
  sn[j * L + s] = sj;
  H[j * L + s] = make_double2(den, 0.0);
  for (int k = 0; k <= j; ++k) R[((long long)j * (mcap + 1) + k) * L + s] = H[k * L + s];
  const double2 gj = g[j * L + s];
  g[(j + 1) * L + s] = make_double2(-sj * gj.x, -sj * gj.y);
  g[j * L + s] = make_double2(c.x * gj.x + c.y * gj.y, c.x * gj.y - c.y * gj.x);
  const double bn = sqrt(fmax(bn2[s].x, 0.0));
  const double gn = sj * sqrt(gj.x * gj.x + gj.y * gj.y);
  const double rr = bn > 0.0 ? gn / bn : 0.0;
  res[s] = rr;
  if (ag < histcap) hist[(long long)ag * L + s] = rr;
  jstop[s] = j + 1;
  if ((!fixed && rr <= tol) || hn <= 1e-300) { done[s] = 1; scale[s] = 0.0; }
  else scale[s] = 1.0 / hn;
}

// y = R^-1 g (upper triangular, jstop columns), zero for k in [jstop, nk).  only_done: columns whose stop test has not fired
// get y = 0 (they are finalised later; used when finished columns are retired in the middle of a cycle).
__global__ void k_backsolve(int mcap, int nk, int nrhs, const double2* __restrict__ R, const double2* __restrict__ g,
                            const int* __restrict__ jstop, const int* __restrict__ done, int only_done, double2* __restrict__ y,
                            const int* __restrict__ slot, int ldc) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nrhs) return;
  const int s = slot[r];
  const long long L = ldc;
  const int js = (only_done && !done[s]) ? 0 : min(jstop[s], nk);
  for (int k = nk - 1; k >= js; --k) y[k * L + s] = make_double2(0.0, 0.0);
  for (int k = js - 1; k >= 0; --k) {
    double2 acc = g[k * L + s];
    for (int q = k + 1; q < js; ++q) {
      const double2 rv = R[((long long)q * (mcap + 1) + k) * L + s], yq = y[q * L + s];
      acc.x -= rv.x * yq.x - rv.y * yq.y;
      acc.y -= rv.x * yq.y + rv.y * yq.x;
    }
    const double2 d = R[((long long)k * (mcap + 1) + k) * L + s];
    const double den = d.x * d.x + d.y * d.y;
    y[k * L + s] = make_double2((acc.x * d.x + acc.y * d.y) / den, (acc.y * d.x - acc.x * d.y) / den);
  }
}

// ---- g[b][c] = sum_(i,j,a) lambda[i,j,b,a] x2[i,j,a][c] = 2 sum_(i<j) sum_a l_p[b,a] x_p[a][c]  (Lambda2 packed [pair][a<b]) ----
// grid (column chunks of LG_CC real columns, pair blocks); gpart[blk][v][Nc].
// The chunks of one pair stream are neighbours in launch order, run at the same time and share every Lambda2 block through L2 (one
// DRAM read of Lambda2 per batch).  Inside a block every warp OWNS 32-row blocks R of the output (R = warp, warp + 8, ...), so the
// sums live in registers across all pairs and nothing is accumulated with atomics:
//   g[b in R] -= sum_(a < b) U[a][b] x[a]   lane = b, walks DOWN column b of the packed triangle: every load is coalesced across b
//   g[a in R] += sum_(b > a) U[a][b] x[b]   lane = a, needs row a: 32 x 32 tiles are read coalesced (along b) into shared memory
//                                           and walked transposed
constexpr int LG_CC = 8;
constexpr int LG_WARPS = 8;
constexpr int LG_NQ = 4;                  // output row blocks per warp and pass (one pass covers v <= 32 * 8 * 4 = 1024)
constexpr int LG_TS = 33;                 // padded tile stride: the transposed walk is bank-conflict free
inline int lg_vpad(int v) { return (v + 31) / 32 * 32; }
inline size_t lambda2_g_smem_bytes(int v) {
  return ((size_t)lg_vpad(v) * LG_CC + (size_t)LG_WARPS * 32 * LG_TS) * sizeof(double);
}
__global__ void __launch_bounds__(32 * LG_WARPS) k_lambda2_g(double* __restrict__ gpart, const double* __restrict__ L2p,
                                                              const double* __restrict__ vec, int o, int v, int Nc, long long npair) {
  extern __shared__ double sm[];
  const int vpad = (v + 31) / 32 * 32, nt = vpad / 32;
  double* xs = sm;                                   // [vpad][LG_CC], rows >= v are zero
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* Ts = xs + (size_t)vpad * LG_CC + (size_t)warp * 32 * LG_TS;   // this warp's [32][LG_TS] tile
  const int c0 = blockIdx.x * LG_CC;
  const long long ntri = (long long)v * (v - 1) / 2;
  const double* x2 = vec + (long long)o * Nc;
  for (int rbase = 0; rbase < nt; rbase += LG_WARPS * LG_NQ) {
    double acc[LG_NQ][LG_CC];
#pragma unroll
    for (int q = 0; q < LG_NQ; ++q)
#pragma unroll
      for (int c = 0; c < LG_CC; ++c) acc[q][c] = 0.0;
    for (long long pr = blockIdx.y; pr < npair; pr += gridDim.y) {
      __syncthreads();
      for (int t = threadIdx.x; t < vpad * LG_CC; t += blockDim.x) {
        const int a = t / LG_CC, c = t % LG_CC;
        xs[t] = (a < v && c0 + c < Nc) ? x2[(pr * v + a) * Nc + c0 + c] : 0.0;
      }
      __syncthreads();
      const double* lp = L2p + pr * ntri;
#pragma unroll
      for (int q = 0; q < LG_NQ; ++q) {
        const int R = rbase + warp + LG_WARPS * q;
        if (R >= nt) continue;                       // warp-uniform
        const int me = R * 32 + lane;                // the output row this lane owns
        // lambda[b, a] = -U[a][b] for a < b: column walk, coalesced across the lanes (b)
        if (me < v) {
#pragma unroll 8
          for (int a = 0; a < me; ++a) {
            const double u = lp[tri_index(a, me, v)];
            const double* xr = xs + (size_t)a * LG_CC;
#pragma unroll
            for (int c = 0; c < LG_CC; ++c) acc[q][c] -= u * xr[c];
          }
        }
        // lambda[a, b] = U[a][b] for b > a: row walk through transposed tiles
        for (int tb = R; tb < nt; ++tb) {
          const int b = tb * 32 + lane;
          __syncwarp();
#pragma unroll 8
          for (int r = 0; r < 32; ++r) {
            const int a = R * 32 + r;
            Ts[r * LG_TS + lane] = (a < b && b < v) ? lp[tri_index(a, b, v)] : 0.0;
          }
          __syncwarp();
#pragma unroll 4
          for (int k = 0; k < 32; ++k) {
            const double u = Ts[lane * LG_TS + k];
            const double* xr = xs + (size_t)(tb * 32 + k) * LG_CC;
#pragma unroll
            for (int c = 0; c < LG_CC; ++c) acc[q][c] += u * xr[c];
          }
        }
      }
    }
#pragma unroll
    for (int q = 0; q < LG_NQ; ++q) {
      const int row = (rbase + warp + LG_WARPS * q) * 32 + lane;
      if (row < v) {
#pragma unroll
        for (int c = 0; c < LG_CC; ++c)
          if (c0 + c < Nc) gpart[((long long)blockIdx.y * v + row) * Nc + c0 + c] = acc[q][c];
      }
    }
  }
}
__global__ void k_g_reduce(double* __restrict__ gvec, const double* __restrict__ gpart, int nblk, long long n) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  double acc = 0;
  for (int b = 0; b < nblk; ++b) acc += gpart[(long long)b * n + idx];
  gvec[idx] = 2.0 * acc;
}
// Gq[out_row[r]][iq] for target q = qlist[iq] and column r of vec (row stride ld complex columns); one block per (iq, r)
__global__ void __launch_bounds__(256) k_assemble_G(double2* __restrict__ Gq, const int* __restrict__ qlist, int nq,
                                                     const double* __restrict__ vec, const double* __restrict__ gvec,
                                                     const double* __restrict__ D, const double* __restrict__ t1,
                                                     const double* __restrict__ l1, int o, int v, int ld,
                                                     const int* __restrict__ out_row = nullptr) {
  __shared__ double2 red[256];
  const int iq = blockIdx.x, r = blockIdx.y;
  const int q = qlist[iq];
  const double2* x = reinterpret_cast<const double2*>(vec);
  const double2* gq = reinterpret_cast<const double2*>(gvec);
  double2 acc = make_double2(0.0, 0.0);
  auto add = [&](double c, double2 val) { acc.x += c * val.x; acc.y += c * val.y; };
  if (q < o) {
    const int k = q;
    for (int t = threadIdx.x; t < o; t += blockDim.x) add((t == k ? 1.0 : 0.0) - D[(long long)k * o + t], x[(long long)t * ld + r]);
    for (int t = threadIdx.x; t < v; t += blockDim.x) add(-0.5 * t1[(long long)k * v + t], gq[(long long)t * ld + r]);
    for (long long t = threadIdx.x; t < (long long)o * v; t += blockDim.x) {
      const int j = t / v, a = t % v;
      if (j == k) continue;
      const long long row = o + (j > k ? pair_index(k, j, o) : pair_index(j, k, o)) * v + a;
      add((j > k ? 1.0 : -1.0) * l1[(long long)j * v + a], x[row * ld + r]);
    }
  } else {
    const int c = q - o;
    for (int t = threadIdx.x; t < o; t += blockDim.x) add(l1[(long long)t * v + c], x[(long long)t * ld + r]);
    if (threadIdx.x == 0) add(0.5, gq[(long long)c * ld + r]);
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) { red[threadIdx.x].x += red[threadIdx.x + s].x; red[threadIdx.x].y += red[threadIdx.x + s].y; }
    __syncthreads();
  }
  if (threadIdx.x == 0) Gq[(long long)(out_row ? out_row[r] : r) * nq + iq] = red[0];
}

// ------------------------------------------------------------------------------------------
#define S_CUDA(expr)                                                                              \
  do {                                                                                            \
    cudaError_t e__ = (expr);                                                                     \
    if (e__ != cudaSuccess) {                                                                     \
      err = std::string(#expr) + " failed: " + cudaGetErrorString(e__);                           \
      return (e__ == cudaErrorMemoryAllocation) ? -2 : -3;                                        \
    }                                                                                             \
  } while (0)
#define S_K() do { *nlaunch += 1; S_CUDA(cudaGetLastError()); } while (0)
#define S_TRY(expr) do { int rc__ = (expr); if (rc__) return rc__; } while (0)

template <typename T>
inline int s_alloc(SolveWs& s, T** p, long long elems, std::string& err) {
  void* q = nullptr;
  if (elems < 1) elems = 1;
  cudaError_t e = cudaMalloc(&q, (size_t)elems * sizeof(T));
  if (e != cudaSuccess) { err = std::string("cudaMalloc (solver workspace) failed: ") + cudaGetErrorString(e); cudaGetLastError(); return -2; }
  s.allocs.push_back(q);
  s.bytes += (double)elems * sizeof(T);
  *p = (T*)q;
  return 0;
}

// memory-limited restart length (SURVEY.md 8a memory budget): basis vectors that fit beside x, b, w, the retirement buffer and
// one spare vector, keeping 2 GB of headroom
inline int solve_mmax(long long nvec, int cap) {
  size_t fre = 0, tot = 0;
  cudaMemGetInfo(&fre, &tot);
  const double vecbytes = (double)nvec * 2.0 * cap * 8.0;
  return (int)std::floor(((double)fre - 2e9) / vecbytes) - 6;
}

static int solve_alloc(SolveWs& s, const SolveCfg& c, int mcap, std::string& err) {
  const long long vecel = c.nvec * 2LL * c.batch;
  const int nr = c.batch;
  // every batch vector is its own allocation: they trade places by pointer swap when the batch is compacted
  // (staggering their start addresses to de-correlate the low address bits was measured: slower, not faster)
  s.V.assign(mcap + 1, nullptr);
  for (int k = 0; k <= mcap; ++k) S_TRY(s_alloc(s, &s.V[k], vecel, err));
  S_TRY(s_alloc(s, &s.x, vecel, err)); S_TRY(s_alloc(s, &s.b, vecel, err)); S_TRY(s_alloc(s, &s.w, vecel, err));
  S_TRY(s_alloc(s, &s.xr, vecel, err)); S_TRY(s_alloc(s, &s.spare, vecel, err));
  s.dot_blocks = (int)std::min<long long>(592, std::max<long long>(1, c.nvec / 64));
  while (s.dot_blocks > 148 && (double)s.dot_blocks * (mcap + 1) * nr * 16.0 > 512e6) s.dot_blocks /= 2;   // bound the partial-sum buffer
  s.g_blocks = (int)std::min<long long>(296, c.npair);
  s.histcap = 8192;   // residual-history entries kept per right-hand side
  S_TRY(s_alloc(s, &s.H, (long long)(mcap + 2) * nr, err));
  S_TRY(s_alloc(s, &s.R, (long long)mcap * (mcap + 1) * nr, err));
  S_TRY(s_alloc(s, &s.cs, (long long)mcap * nr, err));
  S_TRY(s_alloc(s, &s.sn, (long long)mcap * nr, err));
  S_TRY(s_alloc(s, &s.g, (long long)(mcap + 1) * nr, err));
  S_TRY(s_alloc(s, &s.y, (long long)(mcap + 1) * nr, err));
  S_TRY(s_alloc(s, &s.part, (long long)s.dot_blocks * (mcap + 1) * nr, err));
  S_TRY(s_alloc(s, &s.hn2, nr, err)); S_TRY(s_alloc(s, &s.bn2, nr, err));
  S_TRY(s_alloc(s, &s.scale, nr, err)); S_TRY(s_alloc(s, &s.res, nr, err));
  S_TRY(s_alloc(s, &s.hist, (long long)s.histcap * nr, err));
  S_TRY(s_alloc(s, &s.omega_col, nr, err));
  S_TRY(s_alloc(s, &s.stat, 3LL * nr, err));
  S_TRY(s_alloc(s, &s.slot_col, nr, err)); S_TRY(s_alloc(s, &s.p_col, nr, err));
  S_TRY(s_alloc(s, &s.map, nr, err)); S_TRY(s_alloc(s, &s.ret_row, nr, err));
  S_TRY(s_alloc(s, &s.gvec, (long long)std::max(c.o, c.v) * 2 * nr, err));
  S_TRY(s_alloc(s, &s.gpart, (long long)s.g_blocks * c.v * 2 * nr, err));
  S_TRY(s_alloc(s, &s.vptr, mcap + 3, err));
  return 0;
}

// (Re)allocate the workspace for batch capacity c.batch and a basis of at least the requested length (clipped to memory).
// The ACTIVE restart length of a run is m_run = min(requested, mcap), recomputed on every call (a lowered gmres_m or a
// different gmres_fixed takes effect without reallocation).  Nothing is committed unless every allocation succeeded.
inline int solve_prepare(SolveWs& s, const SolveCfg& c, std::string& err) {
  const int want = c.fixed > 0 ? c.fixed : c.m;
  if (s.cap == c.batch && s.nvec == c.nvec && s.mcap >= want && !s.V.empty()) {
    s.m_run = want;
    return 0;
  }
  solve_free(s);
  int mmax = solve_mmax(c.nvec, c.batch);
  if (mmax < 1) { err = "not enough device memory for a GMRES basis"; return -2; }
  if (c.fixed > 0 && mmax < want) { err = "gmres_fixed exceeds the memory-limited basis size"; return -2; }
  const int mcap = std::min(want, mmax);
  int rc = solve_alloc(s, c, mcap, err);
  if (rc) { solve_free(s); return rc; }
  s.cap = c.batch; s.mcap = mcap; s.nvec = c.nvec; s.m_run = mcap;
  return 0;
}

// One (p, omega) task of a solve and what is known about it on the host
struct SolveTask {
  int p = 0; double omega = 0;
  int slot = -1, iters = 0, age = 0; bool finished = false, converged = false; double relres = 0;
};

// sigma(nrhs, d_omega, xin, sout): batched sigma on internal vectors with nrhs active columns (0 or a GFCC error code)
typedef std::function<int(int, const double*, const double*, double*)> SigmaFn;
// The solver core is agnostic of what a vector row means (IP: 1h + 2h1p rows, Eq. 5; EA: 1p + 2p1h rows, Eq. 6).  Two hooks
// supply the problem-specific pieces; both enqueue on the solver's stream and return 0 or a negative error code:
//   init(b, x, A, c0, p_col, omega_col): right-hand sides and initial guesses of the active columns [c0, A) (row stride A)
//   finish(xr, ld, nret, ret_row)      : G assembly (and optional X output) of the first nret columns of the retirement buffer
//                                        xr (row stride ld complex columns); column r belongs to task ret_row[r] (device)
struct SolveHooks {
  std::function<int(double*, double*, int, int, const int*, const double*, double*)> init;
  std::function<int(const double*, int, int, const int*, double*)> finish;
};

struct SolveRun {
  SolveWs& s; const SolveCfg& c; const SigmaFn& sigma; const SolveHooks& hooks; std::string& err; double* nlaunch;
  std::vector<SolveTask>& tasks;
  std::vector<std::vector<double>>* hist_out;
  cudaStream_t st;
  int B, A = 0, nret = 0;
  std::vector<int> col_task;            // active column -> task id
  std::vector<int> ret_task;            // retirement-buffer column -> task id
  std::vector<int> free_slots;
  std::vector<int> h_stat; std::vector<double> h_res;
  size_t next = 0;

  unsigned nbv(int ncols) const { return (unsigned)std::max<long long>(1, std::min<long long>(148LL * 16, (c.nvec * ncols + 255) / 256)); }

  int upload_ptrs(int nbasis) {
    std::vector<const double*> hp(s.mcap + 3, nullptr);
    for (int k = 0; k <= s.mcap; ++k) hp[k] = s.V[k];
    hp[s.mcap + 1] = s.w; hp[s.mcap + 2] = s.b;
    (void)nbasis;
    S_CUDA(cudaMemcpyAsync(s.vptr, hp.data(), hp.size() * sizeof(double*), cudaMemcpyHostToDevice, st));
    S_CUDA(cudaStreamSynchronize(st));   // hp goes out of scope
    return 0;
  }
  int upload_cols() {
    std::vector<int> sl(A), pp(A); std::vector<double> om(A);
    for (int r = 0; r < A; ++r) { const SolveTask& t = tasks[col_task[r]]; sl[r] = t.slot; pp[r] = t.p; om[r] = t.omega; }
    S_CUDA(cudaMemcpyAsync(s.slot_col, sl.data(), A * sizeof(int), cudaMemcpyHostToDevice, st));
    S_CUDA(cudaMemcpyAsync(s.p_col, pp.data(), A * sizeof(int), cudaMemcpyHostToDevice, st));
    S_CUDA(cudaMemcpyAsync(s.omega_col, om.data(), A * sizeof(double), cudaMemcpyHostToDevice, st));
    S_CUDA(cudaStreamSynchronize(st));
    return 0;
  }
  // h[k][slot] = <V_k, w> (+ add[k][slot]) for k in [0,nk): one launch over the whole basis + one small reduction
  int dots(const double* const* Vs, int nk, const double* w, double2* h, const double2* add = nullptr) {
    const int TX = A >= 64 ? 64 : A >= 32 ? 32 : (A >= 16 ? 16 : (A >= 8 ? 8 : 4));
    const int TY = 256 / TX;
    dim3 blk(TX, TY), grid(s.dot_blocks, (A + TX - 1) / TX);
    if (nk <= 2) { k_multi_dot<2, 4><<<grid, blk, (size_t)TX * TY * sizeof(double2), st>>>(s.part, Vs, w, c.nvec, A, nk); S_K(); }
    else { k_multi_dot<8, 1><<<grid, blk, (size_t)TX * TY * sizeof(double2), st>>>(s.part, Vs, w, c.nvec, A, nk); S_K(); }
    k_dot_finish<<<(nk * A + 127) / 128, 128, 0, st>>>(h, s.part, s.dot_blocks, nk, A, add, s.slot_col, B); S_K();
    return 0;
  }
  int axpy(double* w, const double* const* Vs, int nk, const double2* coef, double sign) {
    if (nk <= 0) return 0;
    const int TX = A >= 32 ? 32 : (A >= 16 ? 16 : (A >= 8 ? 8 : 4));
    const int TY = 256 / TX;
    const long long rb = (c.nvec + 4LL * TY - 1) / (4LL * TY);
    dim3 blk(TX, TY), grid((unsigned)std::max<long long>(1, std::min<long long>(148LL * 8, rb)), (A + TX - 1) / TX);
    k_multi_axpy<4><<<grid, blk, 0, st>>>(w, Vs, coef, c.nvec, A, nk, sign, s.slot_col, B); S_K();
    return 0;
  }
  // blocking poll of the device flags: h_stat = [done | jstop | age] by slot, h_res by slot
  int poll() {
    S_CUDA(cudaMemcpyAsync(h_stat.data(), s.stat, 3 * (size_t)B * sizeof(int), cudaMemcpyDeviceToHost, st));
    S_CUDA(cudaMemcpyAsync(h_res.data(), s.res, (size_t)B * sizeof(double), cudaMemcpyDeviceToHost, st));
    S_CUDA(cudaStreamSynchronize(st));
    s.polls += 1;
    return 0;
  }
  int* d_done() { return s.stat; }
  int* d_jstop() { return s.stat + B; }
  int* d_age() { return s.stat + 2 * B; }

  // G assembly + X output of the retirement buffer (problem-specific hook), then empty it
  int flush() {
    if (nret == 0) return 0;
    S_CUDA(cudaMemcpyAsync(s.ret_row, ret_task.data(), nret * sizeof(int), cudaMemcpyHostToDevice, st));
    int rc = hooks.finish(s.xr, B, nret, s.ret_row, nlaunch);
    if (rc) { err = "G assembly failed"; return rc; }
    S_CUDA(cudaStreamSynchronize(st));   // ret_task is reused
    nret = 0; ret_task.clear();
    return 0;
  }

  // Move the columns listed in `leave` (active column indices whose x is final) to the retirement buffer, then re-lay every
  // live vector (x, b and, inside a cycle, the basis V_0..V_nbasis-1) out with the surviving columns only.
  int retire_and_compact(const std::vector<int>& leave, int nbasis) {
    if (leave.empty()) return 0;
    if (nret + (int)leave.size() > B) S_TRY(flush());
    std::vector<int> mp(leave.begin(), leave.end());
    S_CUDA(cudaMemcpyAsync(s.map, mp.data(), mp.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    k_gather_cols<<<nbv((int)leave.size()), 256, 0, st>>>(s.xr, B, nret, s.x, A, s.map, (int)leave.size(), c.nvec); S_K();
    S_CUDA(cudaStreamSynchronize(st));
    std::vector<char> gone(A, 0);
    for (int r : leave) {
      gone[r] = 1;
      SolveTask& t = tasks[col_task[r]];
      ret_task.push_back(col_task[r]); ++nret;
      free_slots.push_back(t.slot);
      t.finished = true;
    }
    std::vector<int> keep, keep_task;
    for (int r = 0; r < A; ++r) if (!gone[r]) { keep.push_back(r); keep_task.push_back(col_task[r]); }
    const int A2 = (int)keep.size();
    if (A2 > 0) {
      S_CUDA(cudaMemcpyAsync(s.map, keep.data(), A2 * sizeof(int), cudaMemcpyHostToDevice, st));
      auto move = [&](double*& vec) -> int {
        k_gather_cols<<<nbv(A2), 256, 0, st>>>(s.spare, A2, 0, vec, A, s.map, A2, c.nvec); S_K();
        std::swap(vec, s.spare);
        return 0;
      };
      S_TRY(move(s.x)); S_TRY(move(s.b));
      for (int k = 0; k < nbasis; ++k) S_TRY(move(s.V[k]));
      S_CUDA(cudaStreamSynchronize(st));
    }
    col_task = keep_task; A = A2;
    if (A > 0) { S_TRY(upload_cols()); S_TRY(upload_ptrs(nbasis)); }
    s.compactions += 1;
    return 0;
  }

  // restart boundary: give the free columns to pending tasks (new width A + nnew), build their b and x0
  int refill() {
    const int nnew = (int)std::min<size_t>((size_t)(B - A), tasks.size() - next);
    if (nnew <= 0) return 0;
    const int A2 = A + nnew;
    if (A > 0) {   // widen x and b (new columns zero for now)
      std::vector<int> mp(A2, -1);
      for (int r = 0; r < A; ++r) mp[r] = r;
      S_CUDA(cudaMemcpyAsync(s.map, mp.data(), A2 * sizeof(int), cudaMemcpyHostToDevice, st));
      auto move = [&](double*& vec) -> int {
        k_gather_cols<<<nbv(A2), 256, 0, st>>>(s.spare, A2, 0, vec, A, s.map, A2, c.nvec); S_K();
        std::swap(vec, s.spare);
        return 0;
      };
      S_TRY(move(s.x)); S_TRY(move(s.b));
      S_CUDA(cudaStreamSynchronize(st));
      s.refills += 1;
    }
    std::vector<int> zero_slots;
    for (int k = 0; k < nnew; ++k) {
      SolveTask& t = tasks[next];
      t.slot = free_slots.back(); free_slots.pop_back();
      zero_slots.push_back(t.slot);
      col_task.push_back((int)next);
      ++next;
    }
    const int c0 = A;
    A = A2;
    S_TRY(upload_cols()); S_TRY(upload_ptrs(0));
    for (int sl : zero_slots) {   // done = 0, jstop = 0, age = 0 for the new slots
      S_CUDA(cudaMemsetAsync(s.stat + sl, 0, sizeof(int), st));
      S_CUDA(cudaMemsetAsync(s.stat + B + sl, 0, sizeof(int), st));
      S_CUDA(cudaMemsetAsync(s.stat + 2 * B + sl, 0, sizeof(int), st));
    }
    int rc = hooks.init(s.b, s.x, A, c0, s.p_col, s.omega_col, nlaunch);
    if (rc) { err = "right-hand side / initial guess failed"; return rc; }
    S_TRY(dots(s.vptr + s.mcap + 2, 1, s.b, s.bn2));   // ||b||^2 of every active column (the old ones are recomputed: same value)
    return 0;
  }

  int run() {
    B = c.batch; st = c.stream;
    const int m = s.m_run;
    const bool fixed = c.fixed > 0;
    h_stat.assign(3 * (size_t)B, 0); h_res.assign(B, 0.0);
    free_slots.clear();
    for (int k = B - 1; k >= 0; --k) free_slots.push_back(k);
    s.compactions = s.refills = s.polls = 0; s.active_col_steps = s.full_col_steps = 0;
    S_CUDA(cudaMemsetAsync(s.stat, 0, 3 * (size_t)B * sizeof(int), st));
    const int pollk = std::max(1, c.poll);
    auto record = [&](int r) {   // copy the polled device state of active column r to its task
      SolveTask& t = tasks[col_task[r]];
      t.relres = h_res[t.slot]; t.age = h_stat[2 * B + t.slot];
    };
    while (next < tasks.size() || A > 0) {
      S_TRY(refill());
      const int width0 = A;
      // ---- r = b - A x -> w, beta, v_0 (one batched sigma on every active column; x = 0 columns would not need it, but
      //      a uniform application keeps the batch one GEMM) ----
      bool all_zero_x = (c.x0 == 0);
      for (int r = 0; r < A && all_zero_x; ++r) if (tasks[col_task[r]].age > 0) all_zero_x = false;
      if (all_zero_x) { S_CUDA(cudaMemcpyAsync(s.w, s.b, (size_t)c.nvec * 2 * A * 8, cudaMemcpyDeviceToDevice, st)); }
      else {
        int rc = sigma(A, s.omega_col, s.x, s.w);
        if (rc) { err = "sigma failed inside GMRES"; return rc; }
        s.active_col_steps += A; s.full_col_steps += width0;
        k_residual<<<nbv(A), 256, 0, st>>>(s.w, s.b, s.w, c.nvec * 2LL * A); S_K();
      }
      S_TRY(dots(s.vptr + s.mcap + 1, 1, s.w, s.hn2));
      k_cycle_start<<<(A + 127) / 128, 128, 0, st>>>(s.hn2, s.bn2, s.g, s.scale, s.res, d_done(), d_jstop(), d_age(), s.hist, s.histcap,
                                                     A, s.mcap + 1, c.tol, fixed ? 1 : 0, s.slot_col, B); S_K();
      k_scale_cols<<<nbv(A), 256, 0, st>>>(s.V[0], s.w, s.scale, c.nvec, A, s.slot_col); S_K();
      // cycle length: no task may exceed its sigma-application budget
      int L = m;
      if (!fixed) {
        for (int r = 0; r < A; ++r) L = std::min(L, std::max(1, c.maxit - (tasks[col_task[r]].age + 1)));
        S_TRY(poll());
        std::vector<int> leave;   // converged before the first Arnoldi step of this cycle: x is already final
        for (int r = 0; r < A; ++r) if (h_stat[tasks[col_task[r]].slot]) { record(r); tasks[col_task[r]].converged = true; leave.push_back(r); }
        if (!leave.empty()) S_TRY(retire_and_compact(leave, 1));
        if (A == 0) continue;
      }
      int j = 0;
      for (; j < L; ++j) {
        int rc = sigma(A, s.omega_col, s.V[j], s.w);
        if (rc) { err = "sigma failed inside GMRES"; return rc; }
        s.active_col_steps += A; s.full_col_steps += width0;
        // CGS2
        S_TRY(dots(s.vptr, j + 1, s.w, s.H));
        S_TRY(axpy(s.w, s.vptr, j + 1, s.H, -1.0));
        S_TRY(dots(s.vptr, j + 1, s.w, s.y));   // y: the re-orthogonalisation correction
        S_TRY(axpy(s.w, s.vptr, j + 1, s.y, -1.0));
        S_TRY(dots(s.vptr + s.mcap + 1, 1, s.w, s.hn2));
        k_givens<<<(A + 127) / 128, 128, 0, st>>>(j, s.mcap, A, s.H, s.y, s.hn2, s.R, s.cs, s.sn, s.g, s.res, s.bn2, c.tol, d_done(), d_jstop(),
                                                  d_age(), s.hist, s.histcap, s.scale, fixed ? 1 : 0, s.slot_col, B); S_K();
        if (j + 1 <= s.mcap) { k_scale_cols<<<nbv(A), 256, 0, st>>>(s.V[j + 1], s.w, s.scale, c.nvec, A, s.slot_col); S_K(); }
        if (fixed) continue;
        if ((j + 1) % pollk != 0 && j + 1 < L) continue;
        S_TRY(poll());
        int ndone = 0;
        for (int r = 0; r < A; ++r) ndone += h_stat[tasks[col_task[r]].slot] ? 1 : 0;
        if (ndone == A) { ++j; break; }
        if (j + 1 == L) continue;
        if (c.compact >= 0 && ndone >= std::max(1, (int)std::ceil(c.compact * A))) {
          // finalise the finished columns (x += V y with y = 0 elsewhere), retire them, shrink the batch
          k_backsolve<<<(A + 127) / 128, 128, 0, st>>>(s.mcap, j + 1, A, s.R, s.g, d_jstop(), d_done(), 1, s.y, s.slot_col, B); S_K();
          S_TRY(axpy(s.x, s.vptr, j + 1, s.y, 1.0));
          std::vector<int> leave;
          for (int r = 0; r < A; ++r) {
            SolveTask& t = tasks[col_task[r]];
            if (h_stat[t.slot]) { record(r); t.iters += h_stat[B + t.slot]; t.converged = true; leave.push_back(r); }
          }
          S_TRY(retire_and_compact(leave, j + 2));
        }
      }
      // ---- end of the cycle: x += V y for every column still in the batch, retire what is finished ----
      const int nk = std::min(j, s.mcap);
      k_backsolve<<<(A + 127) / 128, 128, 0, st>>>(s.mcap, nk, A, s.R, s.g, d_jstop(), d_done(), 0, s.y, s.slot_col, B); S_K();
      S_TRY(axpy(s.x, s.vptr, nk, s.y, 1.0));
      S_TRY(poll());
      std::vector<int> leave;
      for (int r = 0; r < A; ++r) {
        SolveTask& t = tasks[col_task[r]];
        record(r);
        t.iters += h_stat[B + t.slot];
        if (fixed) { leave.push_back(r); continue; }
        if (h_stat[t.slot]) { t.converged = true; leave.push_back(r); }
        else if (t.age + 1 >= c.maxit) leave.push_back(r);   // sigma-application budget spent: retire unconverged
      }
      S_TRY(retire_and_compact(leave, 0));
    }
    // per-task residual histories (device hist is indexed by slot: copy before the slot is reused is not possible in general,
    // so histories are only guaranteed for tasks of the LAST occupancy of a slot; solves with ntot <= batch keep all)
    if (hist_out) {
      std::vector<double> hh((size_t)s.histcap * B);
      S_CUDA(cudaMemcpyAsync(hh.data(), s.hist, hh.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
      S_CUDA(cudaStreamSynchronize(st));
      hist_out->assign(tasks.size(), std::vector<double>());
      std::vector<int> last_of_slot(B, -1);
      for (size_t k = 0; k < tasks.size(); ++k) if (tasks[k].slot >= 0) last_of_slot[tasks[k].slot] = (int)k;
      for (int sl = 0; sl < B; ++sl) {
        const int k = last_of_slot[sl];
        if (k < 0) continue;
        const int n = std::min(tasks[k].age, s.histcap);
        (*hist_out)[k].resize(n);
        for (int q = 0; q < n; ++q) (*hist_out)[k][q] = hh[(size_t)q * B + sl];
      }
    }
    S_TRY(flush());
    return 0;
  }
};

// Solve all tasks; the hooks build the right-hand sides and consume the solutions.  Statistics in `s`.
// Returns 0, -4 (some task not converged) or a negative error code.
inline int solve_run(SolveWs& s, const SolveCfg& c, std::vector<SolveTask>& tasks, const SigmaFn& sigma, const SolveHooks& hooks,
                     std::vector<std::vector<double>>* hist_out, double* nlaunch, std::string& err) {
  int rc = solve_prepare(s, c, err);
  if (rc) return rc;
  SolveRun run{s, c, sigma, hooks, err, nlaunch, tasks, hist_out, c.stream, c.batch};
  rc = run.run();
  if (rc) return rc;
  bool conv = true;
  if (c.fixed == 0) for (const SolveTask& t : tasks) if (!t.converged) conv = false;
  return conv ? 0 : -4;
}

}  // namespace gfcc
