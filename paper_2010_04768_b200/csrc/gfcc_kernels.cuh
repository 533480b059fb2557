// =====================================================================================
// gfcc_kernels.cuh -- bandwidth-bound and small kernels of the GFCCSD-IP path (sm_100a).
//
// Internal vector layout ("RHS-fastest"): a batch of nrhs complex vectors is a REAL matrix
//   vec[n][Nc],  Nc = 2*nrhs (column 2r = Re, 2r+1 = Im of right-hand side r),
//   rows 0..o-1 = x1[i], rows o + pair(i<j)*v + a = x2[i,j,a]   (n = o + npair*v).
// Because Hbar is real, every contraction acts on the Nc real columns independently
// ("complex-real mixed operations"; SURVEY.md 8c point 20).
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gfcc {

__host__ __device__ inline long long pair_index(int i, int j, int o) {
  return (long long)i * o - (long long)i * (i + 1) / 2 + (j - i - 1);
}
__host__ __device__ inline long long tri_index(int a, int b, int v) {
  return (long long)a * v - (long long)a * (a + 1) / 2 + (b - a - 1);
}

// inverse of pair_index: packed index pr -> (i<j)
__host__ __device__ inline void decode_pair(long long pr, int o, int& i, int& j) {
  const double t = 2.0 * o - 1.0;
  int ii = (int)((t - sqrt(t * t - 8.0 * (double)pr)) * 0.5);
  if (ii < 0) ii = 0;
  if (ii > o - 2) ii = o - 2;
  while (ii > 0 && pair_index(ii, ii + 1, o) > pr) --ii;
  while (ii + 2 < o && pair_index(ii + 1, ii + 2, o) <= pr) ++ii;
  i = ii;
  j = (int)(pr - pair_index(ii, ii + 1, o)) + ii + 1;
}

// ------------------------------------------------------------------------------------
// dst[q][r][c] = src[q][row0 + r][col0 + c]            (transpose == 0)
// dst[q][r][c] = src[q][row0 + c][col0 + r]            (transpose == 1)   src is [Q][N][N]
// 32x32 shared-memory tiles so that both sides are coalesced.
// ------------------------------------------------------------------------------------
__global__ void k_copy_block(double* __restrict__ dst, const double* __restrict__ src, int R, int Cc, int row0, int col0,
                             int N, int transpose) {
  __shared__ double tile[32][33];
  const int q = blockIdx.z;
  const double* s = src + (long long)q * N * N;
  double* d = dst + (long long)q * R * Cc;
  const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
  if (!transpose) {
    for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
      const int r = r0 + rr, c = c0 + threadIdx.x;
      if (r < R && c < Cc) d[(long long)r * Cc + c] = s[(long long)(row0 + r) * N + col0 + c];
    }
  } else {
    // read src rows (row0 + c) with r fastest: src[row0 + c][col0 + r]
    for (int cc = threadIdx.y; cc < 32; cc += blockDim.y) {
      const int c = c0 + cc, r = r0 + threadIdx.x;
      if (r < R && c < Cc) tile[cc][threadIdx.x] = s[(long long)(row0 + c) * N + col0 + r];
    }
    __syncthreads();
    for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
      const int r = r0 + rr, c = c0 + threadIdx.x;
      if (r < R && c < Cc) d[(long long)r * Cc + c] = tile[threadIdx.x][rr];
    }
  }
}

// s[q] = sum_{k,c} t1[k,c] Lov[q][k][c]
__global__ void k_sq(double* __restrict__ s, const double* __restrict__ t1, const double* __restrict__ Lov, int ov) {
  __shared__ double red[256];
  const int q = blockIdx.x;
  double acc = 0;
  for (int k = threadIdx.x; k < ov; k += blockDim.x) acc += t1[k] * Lov[(long long)q * ov + k];
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s2 = blockDim.x / 2; s2 > 0; s2 >>= 1) {
    if (threadIdx.x < s2) red[threadIdx.x] += red[threadIdx.x + s2];
    __syncthreads();
  }
  if (threadIdx.x == 0) s[q] = red[0];
}

// g[p][q] = f[p][q] + sum_Q s[Q] L[Q][p][q] - Kmat[p][q]
__global__ void k_fock_jk(double* __restrict__ g, const double* __restrict__ f, const double* __restrict__ s,
                          const double* __restrict__ L, const double* __restrict__ Kmat, int N, int Q) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)N * N) return;
  double acc = f[idx] - Kmat[idx];
  for (int q = 0; q < Q; ++q) acc += s[q] * L[(long long)q * N * N + idx];
  g[idx] = acc;
}

// tmp = A^T g ;  A = 1 - t1 on the [occ, virt] block   -> tmp[p][q] = g[p][q] - (p virtual) sum_m t1[m,a] g[m][q]
__global__ void k_dress_left(double* __restrict__ tmp, const double* __restrict__ g, const double* __restrict__ t1, int o,
                             int v) {
  const int N = o + v;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)N * N) return;
  const int p = idx / N, q = idx % N;
  double acc = g[idx];
  if (p >= o) {
    const int a = p - o;
    for (int m = 0; m < o; ++m) acc -= t1[(long long)m * v + a] * g[(long long)m * N + q];
  }
  tmp[idx] = acc;
}
// ft = tmp B ;  B = 1 + t1^T on the [virt, occ] block   -> ft[p][q] = tmp[p][q] + (q occupied) sum_e t1[q,e] tmp[p][o+e]
__global__ void k_dress_right(double* __restrict__ ft, const double* __restrict__ tmp, const double* __restrict__ t1, int o,
                              int v) {
  const int N = o + v;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)N * N) return;
  const int p = idx / N, q = idx % N;
  double acc = tmp[idx];
  if (q < o)
    for (int e = 0; e < v; ++e) acc += t1[(long long)q * v + e] * tmp[(long long)p * N + o + e];
  ft[idx] = acc;
}

// copy a block of the dressed Fock: dst[r][c] = ft[row0 + r][col0 + c]
__global__ void k_fock_block(double* __restrict__ dst, const double* __restrict__ ft, int R, int Cc, int row0, int col0,
                             int N) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)R * Cc) return;
  const int r = idx / Cc, c = idx % Cc;
  dst[idx] = ft[(long long)(row0 + r) * N + col0 + c];
}

// Lm[q][i][a] -= Mq[q][i][a]
__global__ void k_sub(double* __restrict__ dst, const double* __restrict__ src, long long n) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    dst[i] -= src[i];
}
__global__ void k_scale(double* __restrict__ dst, double s, long long n) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    dst[i] *= s;
}

// ------------------------------------------------------------------------------------
// split-K reduction: C(m,n) = alpha * sum_s part[s][m][n] + beta * C(m,n) with two-level scatter
// ------------------------------------------------------------------------------------
__global__ void k_splitk_reduce(double* __restrict__ C, const double* __restrict__ part, int S, int M, int N, double alpha,
                                double beta, long long sCm0, long long sCm1, int Md, long long sCn0, long long sCn1, int Nd) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)M * N) return;
  const int m = idx / N, n = idx % N;
  double acc = 0;
  for (int s = 0; s < S; ++s) acc += part[(long long)s * M * N + idx];
  double* p = C + (long long)(m / Md) * sCm1 + (long long)(m % Md) * sCm0 + (long long)(n / Nd) * sCn1 + (long long)(n % Nd) * sCn0;
  *p = alpha * acc + (beta != 0.0 ? beta * *p : 0.0);
}

// ------------------------------------------------------------------------------------
// P5/P6 scatter kernels (create)
// ------------------------------------------------------------------------------------
// G1p[(i',m)][(j,n)] for i = i0 + i' :  mode 0: Wp[(i<j)][(m<n)] += G1 (pairs with i<j);
//                                        mode 1: Wp[(j<i)][(m<n)] -= G1 (pairs with j<i).
// Two launches per panel so that no address is touched twice inside one launch (deterministic, race-free).
__global__ void k_scatter_oooo(double* __restrict__ Wp, const double* __restrict__ G1p, int o, int i0, int ni, int mode) {
  const long long npair = (long long)o * (o - 1) / 2;
  const long long total = (long long)ni * o * npair;   // (i', j, (m<n))
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long mn = idx % npair;
    const int j = (idx / npair) % o;
    const int ip = idx / (npair * o);
    const int i = i0 + ip;
    if (i == j || (mode == 0) != (i < j)) continue;
    int m, n;
    decode_pair(mn, o, m, n);
    const double val = G1p[((long long)ip * o + m) * ((long long)o * o) + (long long)j * o + n];
    if (i < j) Wp[pair_index(i, j, o) * npair + mn] += val;
    else Wp[pair_index(j, i, o) * npair + mn] -= val;
  }
}
// tmp[(i<j)][(m', n')] (m = m0+m', n = nlo + n', ncols = o - nlo) : Wp[(i<j)][(m<n)] += sign * tmp for m<n
__global__ void k_pack_oooo_cols(double* __restrict__ Wp, const double* __restrict__ tmp, int o, int m0, int nm, int nlo,
                                 double sign) {
  const long long npair = (long long)o * (o - 1) / 2;
  const int ncols = o - nlo;
  const long long total = npair * nm * ncols;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int np_ = idx % ncols;
    const int mp = (idx / ncols) % nm;
    const long long ij = idx / ((long long)ncols * nm);
    const int m = m0 + mp, n = nlo + np_;
    if (m < n) Wp[ij * npair + pair_index(m, n, o)] += sign * tmp[idx];
  }
}
// X1p[(i',m)][(j,b)] (i = i0+i'):  Wacc[(i<j)][b][m] += X (i<j);  Wacc[(j<i)][b][m] -= X (j<i)
__global__ void k_scatter_ovoo(double* __restrict__ Wacc, const double* __restrict__ Xp, int o, int v, int i0, int ni, int mode) {
  const long long total = (long long)ni * o * o * v;   // (i', j, b, m)  -- m fastest for coalesced writes
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int m = idx % o;
    const int b = (idx / o) % v;
    const int j = (idx / ((long long)o * v)) % o;
    const int ip = idx / ((long long)o * v * o);
    const int i = i0 + ip;
    if (i == j || (mode == 0) != (i < j)) continue;
    const double val = Xp[((long long)ip * o + m) * ((long long)o * v) + (long long)j * v + b];
    if (i < j) Wacc[(pair_index(i, j, o) * v + b) * o + m] += val;
    else Wacc[(pair_index(j, i, o) * v + b) * o + m] -= val;
  }
}
// X2p[j][(i',m)][b] (i = i0+i'): same scatter rule
__global__ void k_scatter_ovoo_batched(double* __restrict__ Wacc, const double* __restrict__ Xp, int o, int v, int i0, int ni, int mode) {
  const long long total = (long long)o * ni * o * v;   // (j, i', b, m)
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int m = idx % o;
    const int b = (idx / o) % v;
    const int ip = (idx / ((long long)o * v)) % ni;
    const int j = idx / ((long long)o * v * ni);
    const int i = i0 + ip;
    if (i == j || (mode == 0) != (i < j)) continue;
    const double val = Xp[(((long long)j * ni + ip) * o + m) * v + b];
    if (i < j) Wacc[(pair_index(i, j, o) * v + b) * o + m] += val;
    else Wacc[(pair_index(j, i, o) * v + b) * o + m] -= val;
  }
}

// gather rows for D: TJ[k][(a,b)] = t[k,j,a,b] (full v*v, from pair-packed T2), LJ[i][(a,b)] = lambda[i,j,a,b] (from [a<b] packed)
__global__ void k_gather_t2_rows(double* __restrict__ TJ, const double* __restrict__ T2p, int o, int v, int j) {
  const long long vv = (long long)v * v;
  const long long total = (long long)o * vv;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int k = idx / vv;
    const long long ab = idx % vv;
    double val = 0.0;
    if (k < j) val = T2p[pair_index(k, j, o) * vv + ab];
    else if (k > j) val = -T2p[pair_index(j, k, o) * vv + ab];
    TJ[idx] = val;
  }
}
__global__ void k_gather_l2_rows(double* __restrict__ LJ, const double* __restrict__ L2p, int o, int v, int j) {
  const long long vv = (long long)v * v, nt = (long long)v * (v - 1) / 2;
  const long long total = (long long)o * vv;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int i = idx / vv;
    const int a = (idx % vv) / v, b = idx % v;
    double val = 0.0;
    if (i != j && a != b) {
      double s = 1.0;
      int ii = i, jj = j, aa = a, bb = b;
      if (ii > jj) { int t = ii; ii = jj; jj = t; s = -s; }
      if (aa > bb) { int t = aa; aa = bb; bb = t; s = -s; }
      val = s * L2p[pair_index(ii, jj, o) * nt + tri_index(aa, bb, v)];
    }
    LJ[idx] = val;
  }
}
// D[k][i] = sum_a t1[k,a] l1[i,a]    (initialisation; the doubles part is accumulated by GEMMs)
__global__ void k_D_singles(double* __restrict__ D, const double* __restrict__ t1, const double* __restrict__ l1, int o, int v) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= o * o) return;
  const int k = idx / o, i = idx % o;
  double acc = 0;
  for (int a = 0; a < v; ++a) acc += t1[(long long)k * v + a] * l1[(long long)i * v + a];
  D[idx] = acc;
}

// ------------------------------------------------------------------------------------
// layout conversion between the C-ABI vectors and the internal RHS-fastest vectors
// ------------------------------------------------------------------------------------
// X1 [nrhs][o] complex, X2 [nrhs][o][o][v] complex  ->  vec[n][Nc]  (reads the i<j half of X2)
__global__ void k_abi_to_vec(double* __restrict__ vec, const double2* __restrict__ X1, const double2* __restrict__ X2, int o,
                             int v, int nrhs) {
  // one block per packed row block: blockIdx.x over rows (o singles rows + npair*v doubles rows) in chunks of 32 rows
  __shared__ double2 tile[32][33];
  const long long npair = (long long)o * (o - 1) / 2;
  const long long n = o + npair * v;
  const long long row0 = (long long)blockIdx.x * 32;
  const int r0 = blockIdx.y * 32;
  const int Nc = 2 * nrhs;
  // load: thread (x = row within 32 [contiguous in a for doubles rows], y = rhs)
  for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
    const int r = r0 + rr;
    const long long row = row0 + threadIdx.x;
    if (r < nrhs && row < n) {
      double2 val;
      if (row < o) val = X1[(long long)r * o + row];
      else {
        const long long q = row - o;
        const long long pr = q / v;
        const int a = q % v;
        int i, j;
        decode_pair(pr, o, i, j);
        val = X2[(((long long)r * o + i) * o + j) * v + a];
      }
      tile[rr][threadIdx.x] = val;
    }
  }
  __syncthreads();
  for (int rw = threadIdx.y; rw < 32; rw += blockDim.y) {
    const long long row = row0 + rw;
    const int r = r0 + threadIdx.x;
    if (r < nrhs && row < n) reinterpret_cast<double2*>(vec + row * Nc)[r] = tile[threadIdx.x][rw];
  }
}
// vec[n][ld] -> S1 [.][o], S2 [.][o][o][v] complex, antisymmetric fill (the diagonal blocks are zeroed by k_zero_diag).
// Column r of the first nrhs columns of vec goes to output vector out_row[r] (nullptr: r); ld = row stride of vec in
// complex columns (>= nrhs).
__global__ void k_vec_to_abi(double2* __restrict__ S1, double2* __restrict__ S2, const double* __restrict__ vec, int o, int v,
                             int nrhs, int ld = 0, const int* __restrict__ out_row = nullptr) {
  __shared__ double2 tile[32][33];
  const long long npair = (long long)o * (o - 1) / 2;
  const long long n = o + npair * v;
  const long long row0 = (long long)blockIdx.x * 32;
  const int r0 = blockIdx.y * 32;
  const long long Nc = 2LL * (ld > 0 ? ld : nrhs);
  for (int rw = threadIdx.y; rw < 32; rw += blockDim.y) {
    const long long row = row0 + rw;
    const int r = r0 + threadIdx.x;
    if (r < nrhs && row < n) tile[threadIdx.x][rw] = reinterpret_cast<const double2*>(vec + row * Nc)[r];
  }
  __syncthreads();
  for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
    const int r = r0 + rr;
    const long long row = row0 + threadIdx.x;
    if (r < nrhs && row < n) {
      const long long ro = out_row ? out_row[r] : r;
      const double2 val = tile[rr][threadIdx.x];
      if (row < o) S1[ro * o + row] = val;
      else {
        const long long q = row - o;
        const long long pr = q / v;
        const int a = q % v;
        int i, j;
        decode_pair(pr, o, i, j);
        S2[((ro * o + i) * o + j) * v + a] = val;
        S2[((ro * o + j) * o + i) * v + a] = make_double2(-val.x, -val.y);
      }
    }
  }
}
// zero the i == j blocks of output vectors out_row[r] (nullptr: r), r < nrhs
__global__ void k_zero_diag(double2* __restrict__ S2, int o, int v, int nrhs, const int* __restrict__ out_row = nullptr) {
  const long long total = (long long)nrhs * o * v;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int a = idx % v;
    const int i = (idx / v) % o;
    const int r = idx / ((long long)v * o);
    const long long ro = out_row ? out_row[r] : r;
    S2[((ro * o + i) * o + i) * v + a] = make_double2(0.0, 0.0);
  }
}

// XU[m][e][j][c] = x2[m,j,e,c]   from the packed vector (rows o + pair*v + e), antisymmetric fill.
// One block per pair (m<j): its v*Nc source doubles are contiguous and are read ONCE; both images XU[m][e][j][:] = +x and
// XU[j][e][m][:] = -x are written from registers (Nc-double pieces).  The earlier form (one block per destination row) read every x2
// element twice from DRAM -- once for (m,j), once for (j,m), in blocks far apart: ncu showed 2.04 GB read for 1.04 GB of x2 at config 2
// with the DRAM pipe saturated (6.6 TB/s of real traffic).  Blocks npair .. npair+o-1 zero the diagonal XU[m][e][m][:].
__global__ void __launch_bounds__(256) k_unpack_xu(double* __restrict__ XU, const double* __restrict__ vec, int o, int v, int Nc) {
  const int nr = Nc >> 1;                                             // complex columns
  const long long npair = (long long)o * (o - 1) / 2;
  double2* __restrict__ xu = reinterpret_cast<double2*>(XU);
  const int total = v * nr;
  if (blockIdx.x >= npair) {
    const long long m = blockIdx.x - npair;
    for (int t = threadIdx.x; t < total; t += blockDim.x) {
      const int e = t / nr, c = t - e * nr;
      xu[((m * v + e) * o + m) * nr + c] = make_double2(0.0, 0.0);
    }
    return;
  }
  int m, j;
  decode_pair(blockIdx.x, o, m, j);
  const double2* __restrict__ src = reinterpret_cast<const double2*>(vec + (long long)o * Nc) + (long long)blockIdx.x * total;
  double2* __restrict__ dmj = xu + ((long long)m * v * o + j) * nr;    // + e*o*nr + c
  double2* __restrict__ djm = xu + ((long long)j * v * o + m) * nr;
  const long long se = (long long)o * nr;
  for (int t0 = threadIdx.x; t0 < total; t0 += 4 * blockDim.x) {
    double2 val[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int t = t0 + u * blockDim.x;
      if (t < total) val[u] = src[t];
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int t = t0 + u * blockDim.x;
      if (t < total) {
        const int e = t / nr, c = t - e * nr;
        dmj[e * se + c] = val[u];
        djm[e * se + c] = make_double2(-val[u].x, -val[u].y);
      }
    }
  }
}

// K2P[(i',a)][(m,e)] += delta_ae Fmi[m][i] - 1/2 delta_im Fae[a][e]      (folds sigma2 terms A and B into the ring panel)
__global__ void k_k2_fixup(double* __restrict__ K2P, const double* __restrict__ Fmi, const double* __restrict__ Fae, int o, int v,
                           int i0) {
  const int row = blockIdx.x;   // (i', a)
  const int ip = row / v, a = row % v;
  const int i = i0 + ip;
  double* r = K2P + (long long)row * o * v;
  for (int t = threadIdx.x; t < o + v; t += blockDim.x) {
    if (t < o) {
      const int m = t;
      double add = Fmi[(long long)m * o + i];
      if (m == i) add -= 0.5 * Fae[(long long)a * v + a];
      r[(long long)m * v + a] += add;
    } else {
      const int e = t - o;
      if (e != a) r[(long long)i * v + e] -= 0.5 * Fae[(long long)a * v + e];
    }
  }
}

// sigma1 small terms: s1[i][c] += shift_c * x1[i][c] - sum_m Fmi[m][i] x1[m][c]
__global__ void k_sigma1_small(double* __restrict__ sout, const double* __restrict__ xin, const double* __restrict__ Fmi,
                               const double* __restrict__ omega, double eta, int o, int nrhs) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;   // (i, r)
  if (idx >= o * nrhs) return;
  const int i = idx / nrhs, r = idx % nrhs;
  const int Nc = 2 * nrhs;
  const double2 x = reinterpret_cast<const double2*>(xin + (long long)i * Nc)[r];
  const double w = omega[r];
  double re = w * x.x + eta * x.y, im = w * x.y - eta * x.x;
  for (int m = 0; m < o; ++m) {
    const double f = Fmi[(long long)m * o + i];
    const double2 xm = reinterpret_cast<const double2*>(xin + (long long)m * Nc)[r];
    re -= f * xm.x;
    im -= f * xm.y;
  }
  double2* out = reinterpret_cast<double2*>(sout + (long long)i * Nc) + r;
  double2 cur = *out;
  cur.x += re;
  cur.y += im;
  *out = cur;
}

// sigma2 epilogue: s2[(i<j)][a][c] += (w - i eta) x2 + Z[i][a][j][c] - Z[j][a][i][c]
// One block per pair (i<j): the pair is decoded once; the block's rows of x2 / s2 (v*Nc doubles) are contiguous, the two Z
// operands come as Nc-double pieces (one per a).  One thread per complex element, four elements (16 independent 16-byte
// loads) in flight per thread.
__global__ void __launch_bounds__(256) k_sigma2_epilogue(double* __restrict__ sout, const double* __restrict__ xin,
                                                         const double* __restrict__ Z, const double* __restrict__ omega, double eta,
                                                         int o, int v, int nrhs) {
  const long long pr = blockIdx.x;
  int i, j;
  decode_pair(pr, o, i, j);
  const long long row0 = (long long)o + pr * v;
  const double2* __restrict__ x = reinterpret_cast<const double2*>(xin) + row0 * nrhs;
  double2* __restrict__ s = reinterpret_cast<double2*>(sout) + row0 * nrhs;
  const double2* __restrict__ zij = reinterpret_cast<const double2*>(Z) + ((long long)i * v * o + j) * nrhs;   // + a*o*nrhs + r
  const double2* __restrict__ zji = reinterpret_cast<const double2*>(Z) + ((long long)j * v * o + i) * nrhs;
  const long long za = (long long)o * nrhs;
  const int total = v * nrhs;
  for (int t0 = threadIdx.x; t0 < total; t0 += 4 * blockDim.x) {
    double2 xv[4], cur[4], p[4], q[4];
    double w[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int t = t0 + u * blockDim.x;
      if (t < total) {
        const int a = t / nrhs, r = t - a * nrhs;
        xv[u] = x[t]; cur[u] = s[t]; p[u] = zij[a * za + r]; q[u] = zji[a * za + r]; w[u] = omega[r];
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int t = t0 + u * blockDim.x;
      if (t < total) {
        cur[u].x += w[u] * xv[u].x + eta * xv[u].y + p[u].x - q[u].x;
        cur[u].y += w[u] * xv[u].y - eta * xv[u].x + p[u].y - q[u].y;
        s[t] = cur[u];
      }
    }
  }
}

// ------------------------------------------------------------------------------------
// GMRES building blocks on vec[n][Nc] matrices (complex columns = double2 per active right-hand side).
// Vectors are indexed by the ACTIVE column r in [0, nrhs) (compact layout, row stride nrhs complex numbers); the small
// per-RHS arrays of the solver (Hessenberg columns, rotations, scales, flags) are indexed by the SLOT the right-hand side
// occupies for its whole life in the batch: element (k, r) lives at [k*ldc + slot[r]] (slot == nullptr: slot[r] = r), so
// that dropping converged columns from the vectors (gfcc_solve.cuh) never moves the small arrays.
// ------------------------------------------------------------------------------------
// partial[blk][k][r] = sum over this block's rows of conj(V_k[row][r]) * w[row][r] for ALL k in [0,nk) in one launch: the basis is
// walked in groups of NK vectors (NK complex accumulators per thread), w is re-read once per group (it stays in L2 for the small
// systems where launch count matters, and costs 1/NK of the basis traffic for the large ones).
// blockDim = (TX rhs lanes, TY row lanes); gridDim = (row blocks, ceil(nrhs/TX)); dynamic smem TX*TY double2.
template <int NK, int UR>
__global__ void __launch_bounds__(256, 4) k_multi_dot(   // 4 CTAs per SM: the solver's 592-block grids are exactly one wave
double2* __restrict__ partial, const double* const* __restrict__ Vs, const double* __restrict__ w,
                            long long n, int nrhs, int nk) {
  extern __shared__ double2 sred[];
  // rows are dealt to the blocks round-robin (grid-stride), so that at any moment all blocks read NEIGHBOURING rows of each vector:
  // 1 + NK sequential DRAM streams for the whole GPU instead of (1 + NK) x gridDim.x scattered ones
  const long long rbeg = (long long)blockIdx.x * blockDim.y, rstep = (long long)gridDim.x * blockDim.y, rend = n;
  const int r = blockIdx.y * blockDim.x + threadIdx.x;
  const bool ok = r < nrhs;
  for (int k0 = 0; k0 < nk; k0 += NK) {
    const int ng = min(NK, nk - k0);
    double2 acc[NK];
#pragma unroll
    for (int k = 0; k < NK; ++k) acc[k] = make_double2(0.0, 0.0);
    if (ok && UR == 1) {   // 1 + ng loads in flight per thread (measured best for ng > 2: 6.0 TB/s at 20 vectors)
      const double2* vq[NK];   // basis pointers read once per group, not once per row (no pointer -> data dependent load in the loop)
#pragma unroll
      for (int k = 0; k < NK; ++k) vq[k] = reinterpret_cast<const double2*>(Vs[k0 + min(k, ng - 1)]);
      for (long long row = rbeg + threadIdx.y; row < rend; row += rstep) {
        const double2 wv = reinterpret_cast<const double2*>(w)[row * nrhs + r];
#pragma unroll
        for (int k = 0; k < NK; ++k)
          if (k < ng) {
            const double2 vv = vq[k][row * nrhs + r];
            acc[k].x += vv.x * wv.x + vv.y * wv.y;   // conj(v) * w
            acc[k].y += vv.x * wv.y - vv.y * wv.x;
          }
      }
    } else if (ok) {       // few vectors (norms, first steps): UR rows per trip keep UR * (NK + 1) independent 16-byte loads in flight
      const double2* vp[NK];
#pragma unroll
      for (int k = 0; k < NK; ++k) vp[k] = reinterpret_cast<const double2*>(Vs[k0 + min(k, ng - 1)]);
#pragma unroll 1
      for (long long row = rbeg + threadIdx.y; row < rend; row += (long long)UR * rstep) {
        double2 wv[UR], vv[UR][NK];
#pragma unroll
        for (int u = 0; u < UR; ++u) {
          const long long rw = row + (long long)u * rstep;
          const bool in = rw < rend;
          wv[u] = in ? reinterpret_cast<const double2*>(w)[rw * nrhs + r] : make_double2(0.0, 0.0);
#pragma unroll
          for (int k = 0; k < NK; ++k) vv[u][k] = (in && k < ng) ? vp[k][rw * nrhs + r] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int u = 0; u < UR; ++u)
#pragma unroll
          for (int k = 0; k < NK; ++k) {
            acc[k].x += vv[u][k].x * wv[u].x + vv[u][k].y * wv[u].y;   // conj(v) * w
            acc[k].y += vv[u][k].x * wv[u].y - vv[u][k].y * wv[u].x;
          }
      }
    }
#pragma unroll
    for (int k = 0; k < NK; ++k) {
      if (k < ng) {   // ng is block-uniform
        sred[threadIdx.y * blockDim.x + threadIdx.x] = acc[k];
        __syncthreads();
        if (threadIdx.y == 0 && ok) {
          double2 s = sred[threadIdx.x];
          for (int yy = 1; yy < blockDim.y; ++yy) {
            const double2 t = sred[yy * blockDim.x + threadIdx.x];
            s.x += t.x;
            s.y += t.y;
          }
          partial[((long long)blockIdx.x * nk + k0 + k) * nrhs + r] = s;
        }
        __syncthreads();
      }
    }
  }
}
// h[k*ldc + slot[r]] = sum_blk partial[blk][k][r]  (+ add[k*ldc + slot[r]] if add != nullptr)
__global__ void k_dot_finish(double2* __restrict__ h, const double2* __restrict__ partial, int nblk, int nk, int nrhs,
                             const double2* __restrict__ add, const int* __restrict__ slot, int ldc) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nk * nrhs) return;
  double2 s = make_double2(0.0, 0.0);
  for (int b = 0; b < nblk; ++b) {
    const double2 t = partial[(long long)b * nk * nrhs + idx];
    s.x += t.x;
    s.y += t.y;
  }
  const int k = idx / nrhs, r = idx - k * nrhs;
  const long long out = (long long)k * ldc + (slot ? slot[r] : r);
  if (add) { s.x += add[out].x; s.y += add[out].y; }
  h[out] = s;
}
// w[row][r] += sign * sum_(k < nk) coef[k*ldc + slot[r]] * V_k[row][r]    all nk basis vectors in ONE launch: w is read and written
// once.  blockDim = (TX rhs lanes, TY row lanes): a thread owns ONE column r (its coefficient of vector k is one load per k, not per
// element) and UR rows at a time, whose sums live in registers; the k loop is unrolled so that 4*UR independent 16-byte basis loads
// are in flight per thread.  gridDim = (row blocks, ceil(nrhs/TX)).
template <int UR>
__global__ void __launch_bounds__(256) k_multi_axpy(double* __restrict__ w, const double* const* __restrict__ Vs,
                                                    const double2* __restrict__ coef, long long n, int nrhs, int nk, double sign,
                                                    const int* __restrict__ slot, int ldc) {
  const int r = blockIdx.y * blockDim.x + threadIdx.x;
  if (r >= nrhs) return;
  const long long sl = slot ? slot[r] : r;
  const long long TY = blockDim.y;
  double2* __restrict__ wp = reinterpret_cast<double2*>(w);
  for (long long row0 = (long long)blockIdx.x * UR * TY + threadIdx.y; row0 < n; row0 += (long long)gridDim.x * UR * TY) {
    double2 acc[UR];
#pragma unroll
    for (int u = 0; u < UR; ++u) {
      const long long row = row0 + u * TY;
      acc[u] = row < n ? wp[row * nrhs + r] : make_double2(0.0, 0.0);
    }
#pragma unroll 4
    for (int k = 0; k < nk; ++k) {
      const double2* __restrict__ vp = reinterpret_cast<const double2*>(Vs[k]);
      double2 c = coef[(long long)k * ldc + sl];
      c.x *= sign; c.y *= sign;
#pragma unroll
      for (int u = 0; u < UR; ++u) {
        const long long row = row0 + u * TY;
        if (row < n) {
          const double2 vv = vp[row * nrhs + r];
          acc[u].x += c.x * vv.x - c.y * vv.y;
          acc[u].y += c.x * vv.y + c.y * vv.x;
        }
      }
    }
#pragma unroll
    for (int u = 0; u < UR; ++u) {
      const long long row = row0 + u * TY;
      if (row < n) wp[row * nrhs + r] = acc[u];
    }
  }
}
// out[row][r] = scale[slot[r]] * in[row][r]   (real scale per rhs; scale 0 masks a converged / broken-down column)
__global__ void k_scale_cols(double* __restrict__ out, const double* __restrict__ in, const double* __restrict__ scale,
                             long long n, int nrhs, const int* __restrict__ slot) {
  const long long total = n * nrhs;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int r = idx % nrhs;
    const double s = scale[slot ? slot[r] : r];
    double2 x = reinterpret_cast<const double2*>(in)[idx];
    x.x *= s;
    x.y *= s;
    reinterpret_cast<double2*>(out)[idx] = x;
  }
}
// r = b - Ax
__global__ void k_residual(double* __restrict__ r, const double* __restrict__ b, const double* __restrict__ ax, long long n2) {
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n2; idx += (long long)gridDim.x * blockDim.x)
    r[idx] = b[idx] - ax[idx];
}
// column gather between two batch layouts (converged-RHS compaction, refill, retirement; gfcc_solve.cuh):
//   dst[row][dcol0 + c] = src[row][src_col[c]]  for c < ncopy  (src_col[c] < 0: zero);  row strides ldd / lds complex columns
__global__ void k_gather_cols(double* __restrict__ dst, int ldd, int dcol0, const double* __restrict__ src, int lds,
                              const int* __restrict__ src_col, int ncopy, long long n) {
  const long long total = n * ncopy;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long row = idx / ncopy;
    const int c = idx - row * ncopy;
    const int sc = src_col[c];
    reinterpret_cast<double2*>(dst)[row * ldd + dcol0 + c] =
        sc >= 0 ? reinterpret_cast<const double2*>(src)[row * lds + sc] : make_double2(0.0, 0.0);
  }
}

// ------------------------------------------------------------------------------------
// dense latency path for tiny systems (gfcc_lib.cu dense_build / dense_apply)
// ------------------------------------------------------------------------------------
// vec[row][c] = (row == c0 + c) ? 1 : 0      n x Nc real unit columns
__global__ void k_unit_cols(double* __restrict__ vec, long long n, int Nc, long long c0) {
  const long long total = n * Nc;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x)
    vec[idx] = (idx / Nc == c0 + idx % Nc) ? 1.0 : 0.0;
}
// H[row][c0 + c] = src[row][c] for c < nc   (H is n x n row-major, src is n x Nc)
__global__ void k_store_cols(double* __restrict__ H, const double* __restrict__ src, long long n, int Nc, long long c0, int nc) {
  const long long total = n * nc;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long row = idx / nc;
    const int c = (int)(idx - row * nc);
    H[row * n + c0 + c] = src[row * Nc + c];
  }
}
// s[row][r] += (omega[r] - i eta) x[row][r]     (complex columns)
__global__ void k_dense_shift(double* __restrict__ sout, const double* __restrict__ xin, const double* __restrict__ omega, double eta,
                              long long n, int nrhs) {
  const long long total = n * nrhs;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const double w = omega[idx % nrhs];
    const double2 x = reinterpret_cast<const double2*>(xin)[idx];
    double2 s = reinterpret_cast<double2*>(sout)[idx];
    s.x += w * x.x + eta * x.y;
    s.y += w * x.y - eta * x.x;
    reinterpret_cast<double2*>(sout)[idx] = s;
  }
}

// ------------------------------------------------------------------------------------
// closed-shell (spin-restricted) inputs -> spin-orbital tensors (gfcc_create_closed_shell).
// Spin-orbital ordering: occupied alpha (no), occupied beta (no), virtual alpha (nv), virtual beta (nv).
//   f[ps,qs'] = d(s,s') f[p,q]  (same for every Cholesky vector);  t[is,as'] = d(s,s') t1[i,a]
//   t[is,jt,as',bt'] = d(s,s') d(t,t') t2[i,j,a,b] - d(s,t') d(t,s') t2[i,j,b,a]     (same for Lambda)
// ------------------------------------------------------------------------------------
__device__ __forceinline__ void cs_split(int P, int no, int nv, int& spin, int& p) {   // spin-orbital -> (spin, spatial index)
  const int o = 2 * no;
  if (P < o) { spin = P / no; p = P - spin * no; }
  else { const int A = P - o; spin = A / nv; p = no + (A - spin * nv); }
}
// dst[q][P][R] = same spin ? src[q][p][r] : 0      grid.z = number of matrices
__global__ void k_cs_expand_matrix(double* __restrict__ dst, const double* __restrict__ src, int no, int nv) {
  const int Ns = no + nv, N = 2 * Ns;
  const long long total = (long long)N * N;
  const double* s = src + (long long)blockIdx.z * Ns * Ns;
  double* d = dst + (long long)blockIdx.z * total;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    int sp, p, sr, r;
    cs_split((int)(idx / N), no, nv, sp, p);
    cs_split((int)(idx % N), no, nv, sr, r);
    d[idx] = sp == sr ? s[(long long)p * Ns + r] : 0.0;
  }
}
__global__ void k_cs_expand_t1(double* __restrict__ dst, const double* __restrict__ src, int no, int nv) {
  const int o = 2 * no, v = 2 * nv;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= o * v) return;
  const int I = idx / v, A = idx % v;
  const int si = I / no, sa = A / nv;
  dst[idx] = si == sa ? src[(long long)(I - si * no) * nv + (A - sa * nv)] : 0.0;
}
// pair-packed [I<J][A][B] (tri == 0) or fully packed [I<J][A<B] (tri == 1) spin-orbital doubles from spatial x[i][j][a][b]
__global__ void k_cs_expand_doubles(double* __restrict__ dst, const double* __restrict__ x, int no, int nv, int tri) {
  const int o = 2 * no, v = 2 * nv;
  const long long npair = (long long)o * (o - 1) / 2, per = tri ? (long long)v * (v - 1) / 2 : (long long)v * v;
  const long long total = npair * per;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long pr = idx / per, ab = idx - pr * per;
    int I, J, A, B;
    decode_pair(pr, o, I, J);
    if (tri) decode_pair(ab, v, A, B);
    else { A = (int)(ab / v); B = (int)(ab % v); }
    const int si = I / no, sj = J / no, sa = A / nv, sb = B / nv;
    const long long i = I - si * no, j = J - sj * no, a = A - sa * nv, b = B - sb * nv;
    double val = 0.0;
    if (si == sa && sj == sb) val += x[((i * no + j) * nv + a) * nv + b];
    if (si == sb && sj == sa) val -= x[((i * no + j) * nv + b) * nv + a];
    dst[idx] = val;
  }
}

}  // namespace gfcc
