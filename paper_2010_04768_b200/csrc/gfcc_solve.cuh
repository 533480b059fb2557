// =====================================================================================
// gfcc_solve.cuh -- batched GMRES and G_pq assembly.
//
// GMRES (Saad & Schultz, PAPER.md ref. 85) for all right-hand sides of a batch in
// lockstep on the RHS-fastest internal vectors vec[n][2*nrhs]:
//   Arnoldi with classical Gram-Schmidt + one re-orthogonalisation (CGS2): block dots and block axpys
//   that read each basis vector once per pass (HBM-bound, coalesced along the RHS columns);
//   per-RHS complex Givens rotations / least squares in a tiny device kernel (one thread per RHS);
//   converged columns are masked (their next basis vector is zero), the host only reads the flags.
// G assembly (Eq. 7-8 first term, cheap form of SURVEY.md 8c item 10):
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
  int o, v, nrhs; long long nvec, npair;
  int m, maxit, fixed, x0;
  double eta, tol;
  const double *t1, *l1, *T2p, *L2p, *D, *fdiag;
  cudaStream_t stream;
};

struct SolveWs {
  int nrhs = 0, m = 0; long long nvec = 0;
  double bytes = 0;
  std::vector<void*> allocs;
  double *basis = nullptr, *x = nullptr, *b = nullptr, *w = nullptr;
  double2 *H = nullptr, *R = nullptr, *cs = nullptr, *g = nullptr, *y = nullptr, *part = nullptr, *hn2 = nullptr, *bn2 = nullptr;
  double *sn = nullptr, *scale = nullptr, *res = nullptr, *gvec = nullptr, *gpart = nullptr;
  int *done = nullptr, *jstop = nullptr, *d_p = nullptr;
  const double** vptr = nullptr;
  int dot_blocks = 0, g_blocks = 0;
};

inline void solve_free(SolveWs& s) {
  for (void* p : s.allocs) cudaFree(p);
  s.allocs.clear();
  s = SolveWs();
}

// ---- right-hand sides b_p in the internal layout; imaginary parts are zero ----
__global__ void k_build_rhs(double* __restrict__ b, const int* __restrict__ p_of_rhs, const double* __restrict__ t1,
                            const double* __restrict__ T2p, int o, int v, int nrhs, long long nvec) {
  const long long total = nvec * nrhs;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long row = idx / nrhs;
    const int r = idx % nrhs;
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
    reinterpret_cast<double2*>(b)[idx] = make_double2(val, 0.0);
  }
}
// x0 = b / (omega - i eta + d),  d_i = -f_ii, d_ija = f_aa - f_ii - f_jj  (reading 11); kind 0: x0 = 0
__global__ void k_x0(double* __restrict__ x, const double* __restrict__ b, const double* __restrict__ omega, double eta,
                     const double* __restrict__ fdiag, int o, int v, int nrhs, long long nvec, int kind) {
  const long long total = nvec * nrhs;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    double2 out = make_double2(0.0, 0.0);
    if (kind == 1) {
      const long long row = idx / nrhs;
      const int r = idx % nrhs;
      double d;
      if (row < o) d = -fdiag[row];
      else {
        const long long q = row - o;
        int i, j;
        decode_pair(q / v, o, i, j);
        d = fdiag[o + (int)(q % v)] - fdiag[i] - fdiag[j];
      }
      const double re = omega[r] + d, im = -eta;
      const double den = re * re + im * im;
      const double2 bb = reinterpret_cast<const double2*>(b)[idx];
      out.x = (bb.x * re + bb.y * im) / den;
      out.y = (bb.y * re - bb.x * im) / den;
    }
    reinterpret_cast<double2*>(x)[idx] = out;
  }
}

// start of a cycle: beta = sqrt(bn2), res = beta/bnorm; scale = done ? 0 : 1/beta; g[0] = beta
__global__ void k_cycle_start(const double2* __restrict__ rn2, const double2* __restrict__ bn2, double2* __restrict__ g,
                              double* __restrict__ scale, double* __restrict__ res, int* __restrict__ done,
                              int* __restrict__ jstop, int nrhs, int mp1, double tol, int fixed) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nrhs) return;
  const double beta = sqrt(fmax(rn2[r].x, 0.0));
  const double bn = sqrt(fmax(bn2[r].x, 0.0));
  for (int k = 0; k < mp1; ++k) g[(long long)k * nrhs + r] = make_double2(0.0, 0.0);
  jstop[r] = 0;
  if (done[r]) { scale[r] = 0.0; return; }
  const double rr = (bn > 0.0) ? beta / bn : 0.0;
  res[r] = rr;
  if ((!fixed && rr <= tol) || beta == 0.0) { done[r] = 1; scale[r] = 0.0; return; }
  g[r] = make_double2(beta, 0.0);
  scale[r] = 1.0 / beta;
}

// one Arnoldi column for every RHS: H[0..j] (CGS2 coefficients), hn2 = ||w||^2.
// Applies the previous rotations, forms the new one, updates g, decides convergence, sets the scale of v_{j+1}.
__global__ void k_givens(int j, int m, int nrhs, double2* __restrict__ H, const double2* __restrict__ hn2,
                         double2* __restrict__ R, double2* __restrict__ cs, double* __restrict__ sn, double2* __restrict__ g,
                         double* __restrict__ res, const double2* __restrict__ bn2, double tol, int* __restrict__ done,
                         int* __restrict__ jstop, double* __restrict__ scale, int fixed) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nrhs) return;
  if (done[r]) { scale[r] = 0.0; return; }
  const double hn = sqrt(fmax(hn2[r].x, 0.0));
  for (int k = 0; k < j; ++k) {
    const double2 a = H[(long long)k * nrhs + r], b = H[(long long)(k + 1) * nrhs + r];
    const double2 c = cs[(long long)k * nrhs + r];
    const double s = sn[(long long)k * nrhs + r];
    // [ conj(c)  s ] [a]
    // [ -s       c ] [b]
    H[(long long)k * nrhs + r] = make_double2(c.x * a.x + c.y * a.y + s * b.x, c.x * a.y - c.y * a.x + s * b.y);
    H[(long long)(k + 1) * nrhs + r] = make_double2(-s * a.x + c.x * b.x - c.y * b.y, -s * a.y + c.x * b.y + c.y * b.x);
  }
  const double2 a = H[(long long)j * nrhs + r];
  const double den = sqrt(a.x * a.x + a.y * a.y + hn * hn);
  if (den == 0.0) {   // zero column: nothing left in the Krylov space
    done[r] = 1; scale[r] = 0.0; jstop[r] = j;
    return;
  }
  const double2 c = make_double2(a.x / den, a.y / den);
  const double s = hn / den;
  cs[(long long)j * nrhs + r] = c;
  sn[(long long)j * nrhs + r] = s;
  H[(long long)j * nrhs + r] = make_double2(den, 0.0);
  for (int k = 0; k <= j; ++k) R[((long long)j * (m + 1) + k) * nrhs + r] = H[(long long)k * nrhs + r];
  const double2 gj = g[(long long)j * nrhs + r];
  g[(long long)(j + 1) * nrhs + r] = make_double2(-s * gj.x, -s * gj.y);
  g[(long long)j * nrhs + r] = make_double2(c.x * gj.x + c.y * gj.y, c.x * gj.y - c.y * gj.x);
  const double bn = sqrt(fmax(bn2[r].x, 0.0));
  const double gn = s * sqrt(gj.x * gj.x + gj.y * gj.y);
  const double rr = bn > 0.0 ? gn / bn : 0.0;
  res[r] = rr;
  jstop[r] = j + 1;
  if ((!fixed && rr <= tol) || hn <= 1e-300) { done[r] = 1; scale[r] = 0.0; }
  else scale[r] = 1.0 / hn;
}

// y = R^-1 g (upper triangular, jstop columns), zero beyond
__global__ void k_backsolve(int m, int nrhs, const double2* __restrict__ R, const double2* __restrict__ g,
                            const int* __restrict__ jstop, double2* __restrict__ y) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nrhs) return;
  const int js = jstop[r];
  for (int k = m - 1; k >= js; --k) y[(long long)k * nrhs + r] = make_double2(0.0, 0.0);
  for (int k = js - 1; k >= 0; --k) {
    double2 acc = g[(long long)k * nrhs + r];
    for (int q = k + 1; q < js; ++q) {
      const double2 rv = R[((long long)q * (m + 1) + k) * nrhs + r], yq = y[(long long)q * nrhs + r];
      acc.x -= rv.x * yq.x - rv.y * yq.y;
      acc.y -= rv.x * yq.y + rv.y * yq.x;
    }
    const double2 d = R[((long long)k * (m + 1) + k) * nrhs + r];
    const double den = d.x * d.x + d.y * d.y;
    y[(long long)k * nrhs + r] = make_double2((acc.x * d.x + acc.y * d.y) / den, (acc.y * d.x - acc.x * d.y) / den);
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
// Gq[r][iq] for target q = qlist[iq]; one block per (iq, r)
__global__ void __launch_bounds__(256) k_assemble_G(double2* __restrict__ Gq, const int* __restrict__ qlist, int nq,
                                                     const double* __restrict__ vec, const double* __restrict__ gvec,
                                                     const double* __restrict__ D, const double* __restrict__ t1,
                                                     const double* __restrict__ l1, int o, int v, int nrhs) {
  __shared__ double2 red[256];
  const int iq = blockIdx.x, r = blockIdx.y;
  const int q = qlist[iq];
  const double2* x = reinterpret_cast<const double2*>(vec);
  const double2* gq = reinterpret_cast<const double2*>(gvec);
  double2 acc = make_double2(0.0, 0.0);
  auto add = [&](double c, double2 val) { acc.x += c * val.x; acc.y += c * val.y; };
  if (q < o) {
    const int k = q;
    for (int t = threadIdx.x; t < o; t += blockDim.x) add((t == k ? 1.0 : 0.0) - D[(long long)k * o + t], x[(long long)t * nrhs + r]);
    for (int t = threadIdx.x; t < v; t += blockDim.x) add(-0.5 * t1[(long long)k * v + t], gq[(long long)t * nrhs + r]);
    for (long long t = threadIdx.x; t < (long long)o * v; t += blockDim.x) {
      const int j = t / v, a = t % v;
      if (j == k) continue;
      const long long row = o + (j > k ? pair_index(k, j, o) : pair_index(j, k, o)) * v + a;
      add((j > k ? 1.0 : -1.0) * l1[(long long)j * v + a], x[row * nrhs + r]);
    }
  } else {
    const int c = q - o;
    for (int t = threadIdx.x; t < o; t += blockDim.x) add(l1[(long long)t * v + c], x[(long long)t * nrhs + r]);
    if (threadIdx.x == 0) add(0.5, gq[(long long)c * nrhs + r]);
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) { red[threadIdx.x].x += red[threadIdx.x + s].x; red[threadIdx.x].y += red[threadIdx.x + s].y; }
    __syncthreads();
  }
  if (threadIdx.x == 0) Gq[(long long)r * nq + iq] = red[0];
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

inline int solve_prepare(SolveWs& s, const SolveCfg& c, std::string& err) {
  int m = c.fixed > 0 ? c.fixed : c.m;
  if (s.nrhs == c.nrhs && s.nvec == c.nvec && s.m >= m && s.basis) return 0;
  solve_free(s);
  const long long vecel = c.nvec * 2LL * c.nrhs;
  size_t fre = 0, tot = 0;
  cudaMemGetInfo(&fre, &tot);
  // memory-limited restart length (SURVEY.md 8a memory budget): keep 2 GB of headroom
  const double avail = (double)fre - 2e9 - 3.0 * vecel * 8.0;
  int mmax = (int)std::floor(avail / (vecel * 8.0)) - 1;
  if (mmax < 1) { err = "not enough device memory for a GMRES basis"; return -2; }
  if (c.fixed > 0 && mmax < m) { err = "gmres_fixed exceeds the memory-limited basis size"; return -2; }
  m = std::min(m, mmax);
  s.m = m; s.nrhs = c.nrhs; s.nvec = c.nvec;
  const int nr = c.nrhs;
  int rc;
  if ((rc = s_alloc(s, &s.basis, vecel * (m + 1), err))) return rc;
  if ((rc = s_alloc(s, &s.x, vecel, err))) return rc;
  if ((rc = s_alloc(s, &s.b, vecel, err))) return rc;
  if ((rc = s_alloc(s, &s.w, vecel, err))) return rc;
  s.dot_blocks = (int)std::min<long long>(592, std::max<long long>(1, c.nvec / 64));
  s.g_blocks = (int)std::min<long long>(296, c.npair);
  if ((rc = s_alloc(s, &s.H, (long long)(m + 2) * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.R, (long long)m * (m + 1) * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.cs, (long long)m * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.sn, (long long)m * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.g, (long long)(m + 1) * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.y, (long long)m * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.part, (long long)s.dot_blocks * 8 * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.hn2, nr, err))) return rc;
  if ((rc = s_alloc(s, &s.bn2, nr, err))) return rc;
  if ((rc = s_alloc(s, &s.scale, nr, err))) return rc;
  if ((rc = s_alloc(s, &s.res, nr, err))) return rc;
  if ((rc = s_alloc(s, &s.done, nr, err))) return rc;
  if ((rc = s_alloc(s, &s.jstop, nr, err))) return rc;
  if ((rc = s_alloc(s, &s.d_p, nr, err))) return rc;
  if ((rc = s_alloc(s, &s.gvec, (long long)c.v * 2 * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.gpart, (long long)s.g_blocks * c.v * 2 * nr, err))) return rc;
  if ((rc = s_alloc(s, &s.vptr, m + 3, err))) return rc;
  std::vector<const double*> hp(m + 3);
  for (int k = 0; k <= m; ++k) hp[k] = s.basis + (long long)k * vecel;
  hp[m + 1] = s.w; hp[m + 2] = s.b;
  if (cudaMemcpy(s.vptr, hp.data(), hp.size() * sizeof(double*), cudaMemcpyHostToDevice) != cudaSuccess) { err = "vptr copy failed"; return -3; }
  return 0;
}

// h[k][r] (+)= <V_k, w>  for k in [0,nk)   (groups of 8 basis vectors per pass over w)
inline int block_dots(SolveWs& s, const SolveCfg& c, const double* const* Vs, int nk, const double* w, double2* h, int accumulate,
                      double* nlaunch, std::string& err) {
  const int TX = std::min(32, c.nrhs >= 32 ? 32 : (c.nrhs >= 16 ? 16 : (c.nrhs >= 8 ? 8 : 4)));
  const int TY = 256 / TX;
  dim3 blk(TX, TY), grid(s.dot_blocks, (c.nrhs + TX - 1) / TX);
  for (int k0 = 0; k0 < nk; k0 += 8) {
    const int n = std::min(8, nk - k0);
    k_multi_dot<8><<<grid, blk, (size_t)TX * TY * sizeof(double2), c.stream>>>(s.part, Vs + k0, w, c.nvec, c.nrhs, n);
    S_K();
    k_dot_finish<<<(n * c.nrhs + 127) / 128, 128, 0, c.stream>>>(h + (long long)k0 * c.nrhs, s.part, s.dot_blocks, n, c.nrhs, accumulate);
    S_K();
  }
  return 0;
}
inline int block_axpy(SolveWs& s, const SolveCfg& c, double* w, const double* const* Vs, int nk, const double2* coef, double sign,
                      double* nlaunch, std::string& err) {
  const long long total = c.nvec * c.nrhs;
  const unsigned nb = (unsigned)std::min<long long>(148LL * 16, (total + 255) / 256);
  for (int k0 = 0; k0 < nk; k0 += 8) {
    const int n = std::min(8, nk - k0);
    k_multi_axpy<8><<<nb, 256, 0, c.stream>>>(w, Vs + k0, coef + (long long)k0 * c.nrhs, c.nvec, c.nrhs, n, sign);
    S_K();
  }
  return 0;
}

// apply(xin, sout) : batched sigma on internal vectors (returns 0 or a GFCC error code)
inline int solve_run(SolveWs& s, const SolveCfg& c, const int* p_of_rhs, const double* w_of_rhs, double* d_omega,
                     const std::function<int(const double*, double*)>& apply, double2* Gq, const int* qlist, int nq,
                     double* X1out, double* X2out, int rhs_offset, int nrhs_total, std::vector<double>& relres,
                     std::vector<int>& iters, double* iterations, double* nlaunch, std::string& err) {
  int rc = solve_prepare(s, c, err);
  if (rc) return rc;
  const int nr = c.nrhs, m = s.m;
  const long long vecel = c.nvec * 2LL * nr;
  cudaStream_t st = c.stream;
  const unsigned nbv = (unsigned)std::min<long long>(148LL * 16, (c.nvec * nr + 255) / 256);
  S_CUDA(cudaMemcpyAsync(d_omega, w_of_rhs, (size_t)nr * 8, cudaMemcpyHostToDevice, st));
  S_CUDA(cudaMemcpyAsync(s.d_p, p_of_rhs, (size_t)nr * sizeof(int), cudaMemcpyHostToDevice, st));
  S_CUDA(cudaMemsetAsync(s.done, 0, (size_t)nr * sizeof(int), st));
  k_build_rhs<<<nbv, 256, 0, st>>>(s.b, s.d_p, c.t1, c.T2p, c.o, c.v, nr, c.nvec); S_K();
  if ((rc = block_dots(s, c, s.vptr + m + 2, 1, s.b, s.bn2, 0, nlaunch, err))) return rc;
  k_x0<<<nbv, 256, 0, st>>>(s.x, s.b, d_omega, c.eta, c.fdiag, c.o, c.v, nr, c.nvec, c.x0); S_K();
  std::vector<int> h_done(nr, 0), h_js(nr, 0), it_acc(nr, 0);
  std::vector<double> h_res(nr, 1.0);
  const bool fixed = c.fixed > 0;
  int napply = 0;
  bool x_is_zero = (c.x0 == 0);
  bool all_done = false;
  double* V0 = s.basis;
  while (!all_done && (fixed ? napply == 0 : napply < c.maxit)) {
    // r = b - A x  -> w
    if (x_is_zero) { S_CUDA(cudaMemcpyAsync(s.w, s.b, (size_t)vecel * 8, cudaMemcpyDeviceToDevice, st)); }
    else {
      if ((rc = apply(s.x, s.w))) { err = "sigma failed inside GMRES"; return rc; }
      ++napply;
      k_residual<<<nbv, 256, 0, st>>>(s.w, s.b, s.w, vecel); S_K();
    }
    if ((rc = block_dots(s, c, s.vptr + m + 1, 1, s.w, s.hn2, 0, nlaunch, err))) return rc;
    k_cycle_start<<<(nr + 127) / 128, 128, 0, st>>>(s.hn2, s.bn2, s.g, s.scale, s.res, s.done, s.jstop, nr, m + 1, c.tol, fixed ? 1 : 0);
    S_K();
    k_scale_cols<<<nbv, 256, 0, st>>>(V0, s.w, s.scale, c.nvec, nr); S_K();
    if (!fixed) {
      S_CUDA(cudaMemcpyAsync(h_done.data(), s.done, (size_t)nr * sizeof(int), cudaMemcpyDeviceToHost, st));
      S_CUDA(cudaStreamSynchronize(st));
      all_done = std::all_of(h_done.begin(), h_done.end(), [](int d) { return d != 0; });
      if (all_done) break;
    }
    int j = 0;
    for (; j < m && (fixed || napply < c.maxit); ++j) {
      double* Vj = s.basis + (long long)j * vecel;
      double* Vn = s.basis + (long long)(j + 1) * vecel;
      if ((rc = apply(Vj, s.w))) { err = "sigma failed inside GMRES"; return rc; }
      ++napply;
      // CGS2
      if ((rc = block_dots(s, c, s.vptr, j + 1, s.w, s.H, 0, nlaunch, err))) return rc;
      if ((rc = block_axpy(s, c, s.w, s.vptr, j + 1, s.H, -1.0, nlaunch, err))) return rc;
      if ((rc = block_dots(s, c, s.vptr, j + 1, s.w, s.y, 0, nlaunch, err))) return rc;   // y used as scratch for the correction
      if ((rc = block_axpy(s, c, s.w, s.vptr, j + 1, s.y, -1.0, nlaunch, err))) return rc;
      k_cadd<<<((j + 1) * nr + 127) / 128, 128, 0, st>>>(s.H, s.y, (j + 1) * nr); S_K();
      if ((rc = block_dots(s, c, s.vptr + m + 1, 1, s.w, s.hn2, 0, nlaunch, err))) return rc;
      k_givens<<<(nr + 127) / 128, 128, 0, st>>>(j, m, nr, s.H, s.hn2, s.R, s.cs, s.sn, s.g, s.res, s.bn2, c.tol, s.done, s.jstop,
                                                 s.scale, fixed ? 1 : 0);
      S_K();
      k_scale_cols<<<nbv, 256, 0, st>>>(Vn, s.w, s.scale, c.nvec, nr); S_K();
      if (!fixed) {
        S_CUDA(cudaMemcpyAsync(h_done.data(), s.done, (size_t)nr * sizeof(int), cudaMemcpyDeviceToHost, st));
        S_CUDA(cudaStreamSynchronize(st));
        if (std::all_of(h_done.begin(), h_done.end(), [](int d) { return d != 0; })) { ++j; all_done = true; break; }
      }
    }
    // x += V y
    k_backsolve<<<(nr + 127) / 128, 128, 0, st>>>(m, nr, s.R, s.g, s.jstop, s.y); S_K();
    if ((rc = block_axpy(s, c, s.x, s.vptr, std::min(j, m), s.y, 1.0, nlaunch, err))) return rc;
    x_is_zero = false;
    S_CUDA(cudaMemcpyAsync(h_js.data(), s.jstop, (size_t)nr * sizeof(int), cudaMemcpyDeviceToHost, st));
    S_CUDA(cudaStreamSynchronize(st));
    for (int r = 0; r < nr; ++r) it_acc[r] += h_js[r];
    if (fixed) break;
  }
  S_CUDA(cudaMemcpyAsync(h_res.data(), s.res, (size_t)nr * 8, cudaMemcpyDeviceToHost, st));
  S_CUDA(cudaMemcpyAsync(h_done.data(), s.done, (size_t)nr * sizeof(int), cudaMemcpyDeviceToHost, st));
  // ---- G assembly ----
  {
    const int Nc = 2 * nr;
    dim3 grid((Nc + LG_CC - 1) / LG_CC, s.g_blocks);
    const size_t smem = lambda2_g_smem_bytes(c.v);
    static bool attr_set = false;
    if (!attr_set) { cudaFuncSetAttribute(k_lambda2_g, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); attr_set = true; }
    k_lambda2_g<<<grid, 32 * LG_WARPS, smem, st>>>(s.gpart, c.L2p, s.x, c.o, c.v, Nc, c.npair); S_K();
    const long long n = (long long)c.v * Nc;
    k_g_reduce<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(s.gvec, s.gpart, s.g_blocks, n); S_K();
    dim3 gg(nq, nr);
    k_assemble_G<<<gg, 256, 0, st>>>(Gq, qlist, nq, s.x, s.gvec, c.D, c.t1, c.l1, c.o, c.v, nr); S_K();
  }
  if (X1out && X2out) {
    dim3 blk(32, 8), grid((unsigned)((c.nvec + 31) / 32), (unsigned)((nr + 31) / 32));
    double2* x1o = (double2*)X1out + (long long)rhs_offset * c.o;
    double2* x2o = (double2*)X2out + (long long)rhs_offset * c.o * c.o * c.v;
    k_vec_to_abi<<<grid, blk, 0, st>>>(x1o, x2o, s.x, c.o, c.v, nr); S_K();
    const long long tot = (long long)nr * c.o * c.v;
    k_zero_diag<<<(unsigned)std::min<long long>(4096, (tot + 255) / 256), 256, 0, st>>>(x2o, c.o, c.v, nr); S_K();
  }
  S_CUDA(cudaStreamSynchronize(st));
  (void)nrhs_total;
  bool conv = true;
  int itmax = 0;
  for (int r = 0; r < nr; ++r) {
    relres[rhs_offset + r] = h_res[r];
    iters[rhs_offset + r] = it_acc[r];
    itmax = std::max(itmax, it_acc[r]);
    if (!fixed && !h_done[r]) conv = false;
  }
  *iterations = std::max(*iterations, (double)itmax);
  return conv ? 0 : -4;
}

}  // namespace gfcc
