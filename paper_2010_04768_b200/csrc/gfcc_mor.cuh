// =====================================================================================
// gfcc_mor.cuh -- kernels of the model-order-reduction step.
//
// Paper: Eq. 10 and Alg. 1 lines 18-21:
//   Gram-Schmidt of the new X_p(omega) against the orthonormal subspace S (O(m^2 O^2 V)),
//   projection H^ = S^T Hbar_N S (O(m O^3 V^2): one batched sigma application per block of new vectors),
//   b^ = S^T b, c^ = S^T c, then for every omega of a fine grid (omega - i eta + H^) X^ = b^,
//   G^ = c^^T X^ and the spectral function A(omega) = (1/pi) sum_p Im G^_pp (Eq. 9; sign: DESIGN.md
//   reading 25).  S is REAL (Eq. 10 writes transposes; Hbar, b, c are real; reading 24): every complex X
//   contributes Re X and Im X, which are exactly the two real columns of the internal RHS-fastest layout.
//
// The tall-skinny products (S^T V, V -= S C, S^T (Hbar S)) run on the FP64 DMMA GEMM engine (split-K over the
// row dimension); this file holds the bandwidth-bound helpers and the batched dense complex LU of the reduced
// systems (one CTA per frequency).
// =====================================================================================
#pragma once
#include <cuda_runtime.h>

namespace gfcc {

// partial[blk][c] = sum over this block's rows of V[r][c]^2      (V row-major, leading dimension ld)
__global__ void __launch_bounds__(256) k_mor_colsq_partial(double* __restrict__ partial, const double* __restrict__ V,
                                                            long long n, int k, long long ld) {
  __shared__ double red[8][33];
  const int tx = threadIdx.x, ty = threadIdx.y;   // (32, 8)
  const int c = blockIdx.y * 32 + tx;
  double acc = 0.0;
  if (c < k)
    for (long long r = (long long)blockIdx.x * 8 + ty; r < n; r += (long long)gridDim.x * 8) {
      const double x = V[r * ld + c];
      acc += x * x;
    }
  red[ty][tx] = acc;
  __syncthreads();
  if (ty == 0 && c < k) {
    double s = 0.0;
#pragma unroll
    for (int y = 0; y < 8; ++y) s += red[y][tx];
    partial[(long long)blockIdx.x * k + c] = s;
  }
}
// out[c] = sum_blk partial[blk][c];  inv[c] = out > 0 ? 1/sqrt(out) : 0
__global__ void k_mor_colsq_finish(double* __restrict__ sq, double* __restrict__ inv, const double* __restrict__ partial,
                                   int nblk, int k) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k) return;
  double s = 0.0;
  for (int b = 0; b < nblk; ++b) s += partial[(long long)b * k + c];
  sq[c] = s;
  if (inv) inv[c] = s > 0.0 ? 1.0 / sqrt(s) : 0.0;
}
// V[r][c] *= scale[c]
__global__ void k_mor_scale_cols(double* __restrict__ V, const double* __restrict__ scale, long long n, int k, long long ld) {
  const long long total = n * k;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long r = idx / k;
    const int c = (int)(idx % k);
    V[r * ld + c] *= scale[c];
  }
}
// dst[r*ldd] = s * src[r*lds]       (one column, strided on both sides)
__global__ void k_mor_copy_col(double* __restrict__ dst, long long ldd, const double* __restrict__ src, long long lds, long long n,
                               double s) {
  for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += (long long)gridDim.x * blockDim.x)
    dst[r * ldd] = s * src[r * lds];
}
// dst[r][0:cnt] = src[r][0:cnt], zero fill of dst[r][cnt:wd]     (column block between matrices of different widths)
__global__ void k_mor_copy_cols(double* __restrict__ dst, long long ldd, int wd, const double* __restrict__ src, long long lds,
                                long long n, int cnt) {
  const long long total = n * wd;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long r = idx / wd;
    const int c = (int)(idx % wd);
    dst[r * ldd + c] = c < cnt ? src[r * lds + c] : 0.0;
  }
}
// chat[(c0 + 2r + s)][iq] = (s == 0 ? Re : Im) Gq[r][iq]   for the valid columns only
__global__ void k_mor_store_chat(double* __restrict__ chat, const double2* __restrict__ Gq, int nb, int nq, int c0, int ncols) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nb * nq) return;
  const int r = idx / nq, iq = idx % nq;
  const double2 g = Gq[idx];
  if (2 * r < ncols) chat[(long long)(c0 + 2 * r) * nq + iq] = g.x;
  if (2 * r + 1 < ncols) chat[(long long)(c0 + 2 * r + 1) * nq + iq] = g.y;
}

// ---- reduced systems: one CTA per frequency ------------------------------------------------------------------
// (omega_w - i eta + H^) X^ = b^  by dense complex LU with partial pivoting in the CTA's own m x m scratch
// (global memory, L2-resident for the sizes MOR produces), then G^[w][ip][iq] = sum_j c^[j][iq] X^[j][ip] and
// A[w] = (1/pi) sum_p Im G^[w][p][p].   Hh: [m][ldh] real; bh2: [m][2*np] (even columns = b^, the odd ones are the
// zero imaginary parts of the RHS builder); chat: [m][nq].
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cinv(double2 a) {
  const double d = a.x * a.x + a.y * a.y;
  return make_double2(a.x / d, -a.y / d);
}

constexpr int MOR_LU_THREADS = 512;
__global__ void __launch_bounds__(MOR_LU_THREADS) k_mor_lu_solve(int m, int ldh, const double* __restrict__ Hh,
                                                                  const double* __restrict__ bh2, int np,
                                                                  const double* __restrict__ chat, int nq,
                                                                  const double* __restrict__ omega, double eta,
                                                                  double2* __restrict__ Awork, double2* __restrict__ Xwork,
                                                                  double2* __restrict__ G, double* __restrict__ Aspec,
                                                                  int* __restrict__ singular) {
  __shared__ double s_val[MOR_LU_THREADS];
  __shared__ int s_idx[MOR_LU_THREADS];
  __shared__ double2 s_inv;
  const int tid = threadIdx.x, nt = blockDim.x;
  const int w = blockIdx.x;
  double2* A = Awork + (size_t)w * m * m;
  double2* X = Xwork + (size_t)w * m * np;
  const double om = omega[w];
  for (long long idx = tid; idx < (long long)m * m; idx += nt) {
    const int i = (int)(idx / m), j = (int)(idx % m);
    A[idx] = make_double2(Hh[(long long)i * ldh + j] + (i == j ? om : 0.0), i == j ? -eta : 0.0);
  }
  for (int idx = tid; idx < m * np; idx += nt) X[idx] = make_double2(bh2[(long long)(idx / np) * 2 * np + 2 * (idx % np)], 0.0);
  __syncthreads();
  for (int k = 0; k < m; ++k) {
    // pivot search in column k
    double best = -1.0; int bi = k;
    for (int i = k + tid; i < m; i += nt) {
      const double2 a = A[(size_t)i * m + k];
      const double mag = a.x * a.x + a.y * a.y;
      if (mag > best) { best = mag; bi = i; }
    }
    s_val[tid] = best; s_idx[tid] = bi;
    __syncthreads();
    for (int s = nt / 2; s > 0; s >>= 1) {
      if (tid < s) {
        const double ov = s_val[tid + s]; const int oi = s_idx[tid + s];
        if (ov > s_val[tid] || (ov == s_val[tid] && oi < s_idx[tid])) { s_val[tid] = ov; s_idx[tid] = oi; }
      }
      __syncthreads();
    }
    const int piv = s_idx[0];
    if (s_val[0] <= 0.0) { if (tid == 0) singular[w] = 1; }
    if (piv != k) {
      for (int j = k + tid; j < m; j += nt) { const double2 t = A[(size_t)k * m + j]; A[(size_t)k * m + j] = A[(size_t)piv * m + j]; A[(size_t)piv * m + j] = t; }
      for (int p = tid; p < np; p += nt) { const double2 t = X[k * np + p]; X[k * np + p] = X[piv * np + p]; X[piv * np + p] = t; }
    }
    __syncthreads();
    if (tid == 0) s_inv = cinv(A[(size_t)k * m + k]);
    __syncthreads();
    const double2 inv = s_inv;
    for (int i = k + 1 + tid; i < m; i += nt) A[(size_t)i * m + k] = cmul(A[(size_t)i * m + k], inv);
    __syncthreads();
    const int rem = m - k - 1;
    // trailing update of A (columns k+1..m-1) and of the right-hand sides
    for (long long idx = tid; idx < (long long)rem * rem; idx += nt) {
      const int i = k + 1 + (int)(idx / rem), j = k + 1 + (int)(idx % rem);
      const double2 l = A[(size_t)i * m + k], u = A[(size_t)k * m + j];
      double2 a = A[(size_t)i * m + j];
      a.x -= l.x * u.x - l.y * u.y; a.y -= l.x * u.y + l.y * u.x;
      A[(size_t)i * m + j] = a;
    }
    for (int idx = tid; idx < rem * np; idx += nt) {
      const int i = k + 1 + idx / np, p = idx % np;
      const double2 l = A[(size_t)i * m + k], u = X[k * np + p];
      double2 a = X[i * np + p];
      a.x -= l.x * u.x - l.y * u.y; a.y -= l.x * u.y + l.y * u.x;
      X[i * np + p] = a;
    }
    __syncthreads();
  }
  // back substitution (column oriented)
  for (int k = m - 1; k >= 0; --k) {
    if (tid == 0) s_inv = cinv(A[(size_t)k * m + k]);
    __syncthreads();
    for (int p = tid; p < np; p += nt) X[k * np + p] = cmul(X[k * np + p], s_inv);
    __syncthreads();
    for (int idx = tid; idx < k * np; idx += nt) {
      const int i = idx / np, p = idx % np;
      const double2 u = A[(size_t)i * m + k], x = X[k * np + p];
      double2 a = X[i * np + p];
      a.x -= u.x * x.x - u.y * x.y; a.y -= u.x * x.y + u.y * x.x;
      X[i * np + p] = a;
    }
    __syncthreads();
  }
  // G^[w][ip][iq]
  for (int idx = tid; idx < np * nq; idx += nt) {
    const int ip = idx / nq, iq = idx % nq;
    double2 acc = make_double2(0.0, 0.0);
    for (int j = 0; j < m; ++j) {
      const double c = chat[(long long)j * nq + iq];
      const double2 x = X[j * np + ip];
      acc.x += c * x.x; acc.y += c * x.y;
    }
    G[((size_t)w * np + ip) * nq + iq] = acc;
  }
  __syncthreads();
  if (tid == 0 && Aspec) {
    double tr = 0.0;
    const int nd = np < nq ? np : nq;
    for (int p = 0; p < nd; ++p) tr += G[((size_t)w * np + p) * nq + p].y;
    Aspec[w] = tr / 3.14159265358979323846;
  }
}

}  // namespace gfcc
