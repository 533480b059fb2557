// =====================================================================================
// gfcc_ea.cuh -- bandwidth-bound and small kernels of the EA / advanced part.
//
// PAPER.md:78 Eq. 4  Y_q = sum_a y1[a] a+_a + sum_{j, a<b} y2[j,a,b] a+_a a+_b a_j,
// PAPER.md:84 Eq. 6  (omega - Hbar_N + i eta) Y_q |Phi> = abar_q^+ |Phi>,
// PAPER.md:89-94     second terms of Eq. 7-8: G^A_pq = <Phi|(1+Lambda1+Lambda2) abar_p (Y_q1 + Y_q2)|Phi>.
// Working equations: DESIGN.md section 6.8 (derived from the operator definitions, pinned by the Fock-space brute force).
//
// Internal vector layout ("RHS-fastest", as for the IP part): vec[nE][Nc], Nc = 2*nrhs,
//   rows 0..v-1 = y1[a], row v + j*ntri + tri(a<b) = y2[j,a,b]   (nE = v + o*ntri).
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include "gfcc_kernels.cuh"

namespace gfcc {

// inverse of tri_index: packed index -> (a<b)
__host__ __device__ inline void decode_tri(long long t, int v, int& a, int& b) { decode_pair(t, v, a, b); }

// signed element t[k,j,a,b] of the pair-packed T2 / lambda[k,j,a<b] of the fully packed Lambda2
__device__ __forceinline__ double t2_signed(const double* __restrict__ T2p, int k, int j, long long ab, int o, long long vv) {
  if (k == j) return 0.0;
  return k < j ? T2p[pair_index(k, j, o) * vv + ab] : -T2p[pair_index(j, k, o) * vv + ab];
}

// ---- layout conversion: Y1 [nrhs][v], Y2 [nrhs][o][v][v] complex <-> vec[nE][Nc] (32 x 32 tiles, both sides coalesced) ----
__global__ void k_ea_abi_to_vec(double* __restrict__ vec, const double2* __restrict__ Y1, const double2* __restrict__ Y2, int o,
                                int v, int nrhs) {
  __shared__ double2 tile[32][33];
  const long long ntri = (long long)v * (v - 1) / 2, n = v + (long long)o * ntri;
  const long long row0 = (long long)blockIdx.x * 32;
  const int r0 = blockIdx.y * 32;
  for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
    const int r = r0 + rr;
    const long long row = row0 + threadIdx.x;
    if (r < nrhs && row < n) {
      double2 val;
      if (row < v) val = Y1[(long long)r * v + row];
      else {
        const long long q = row - v;
        const int j = (int)(q / ntri);
        int a, b;
        decode_tri(q - (long long)j * ntri, v, a, b);
        val = Y2[(((long long)r * o + j) * v + a) * v + b];
      }
      tile[rr][threadIdx.x] = val;
    }
  }
  __syncthreads();
  for (int rw = threadIdx.y; rw < 32; rw += blockDim.y) {
    const long long row = row0 + rw;
    const int r = r0 + threadIdx.x;
    if (r < nrhs && row < n) reinterpret_cast<double2*>(vec + row * 2 * nrhs)[r] = tile[threadIdx.x][rw];
  }
}
// vec (row stride ld complex columns, 0: nrhs) -> S1, S2 of output vector out_row[r] (nullptr: r); antisymmetric fill, zero diagonal
__global__ void k_ea_vec_to_abi(double2* __restrict__ S1, double2* __restrict__ S2, const double* __restrict__ vec, int o, int v,
                                int nrhs, int ld, const int* __restrict__ out_row) {
  __shared__ double2 tile[32][33];
  const long long ntri = (long long)v * (v - 1) / 2, n = v + (long long)o * ntri;
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
      if (row < v) S1[ro * v + row] = val;
      else {
        const long long q = row - v;
        const int j = (int)(q / ntri);
        int a, b;
        decode_tri(q - (long long)j * ntri, v, a, b);
        S2[((ro * o + j) * v + a) * v + b] = val;
        S2[((ro * o + j) * v + b) * v + a] = make_double2(-val.x, -val.y);
      }
    }
  }
}
__global__ void k_ea_zero_diag(double2* __restrict__ S2, int o, int v, int nrhs, const int* __restrict__ out_row) {
  const long long total = (long long)nrhs * o * v;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int a = idx % v;
    const int j = (idx / v) % o;
    const int r = idx / ((long long)v * o);
    const long long ro = out_row ? out_row[r] : r;
    S2[((ro * o + j) * v + a) * v + a] = make_double2(0.0, 0.0);
  }
}

// YU[l][d][a][c] = y2[l,a,d,c]  (B operand of the ring / exchange panels: rows (l,d), columns (a,c)); one block per (l,d)
__global__ void __launch_bounds__(256) k_ea_unpack_yu(double* __restrict__ YU, const double* __restrict__ vec, int o, int v, int Nc) {
  const int l = blockIdx.x / v, d = blockIdx.x % v;
  const int nr = Nc >> 1;
  const long long ntri = (long long)v * (v - 1) / 2;
  double2* __restrict__ dst = reinterpret_cast<double2*>(YU + (long long)blockIdx.x * v * Nc);
  const double2* __restrict__ y2 = reinterpret_cast<const double2*>(vec + (long long)v * Nc) + (long long)l * ntri * nr;
  const int total = v * nr;
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int a = t / nr, c = t - a * nr;
    double2 val = make_double2(0.0, 0.0);
    if (a < d) val = y2[tri_index(a, d, v) * nr + c];
    else if (a > d) { const double2 q = y2[tri_index(d, a, v) * nr + c]; val = make_double2(-q.x, -q.y); }
    dst[t] = val;
  }
}
// YV[c][d][j][cc] = y2[j,c,d,cc]  (B operand of the particle-particle ladder: rows (c,d), columns (j,cc)); one block per (c,d)
__global__ void __launch_bounds__(256) k_ea_unpack_yv(double* __restrict__ YV, const double* __restrict__ vec, int o, int v, int Nc) {
  const int c = blockIdx.x / v, d = blockIdx.x % v;
  const int nr = Nc >> 1;
  const long long ntri = (long long)v * (v - 1) / 2;
  double2* __restrict__ dst = reinterpret_cast<double2*>(YV + (long long)blockIdx.x * o * Nc);
  const double2* __restrict__ y2 = reinterpret_cast<const double2*>(vec + (long long)v * Nc);
  const int total = o * nr;
  const double sg = c < d ? 1.0 : -1.0;
  const long long tr = c == d ? 0 : (c < d ? tri_index(c, d, v) : tri_index(d, c, v));
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int j = t / nr, cc = t - j * nr;
    double2 val = make_double2(0.0, 0.0);
    if (c != d) { const double2 q = y2[((long long)j * ntri + tr) * nr + cc]; val = make_double2(sg * q.x, sg * q.y); }
    dst[t] = val;
  }
}
// Upair[(m<n)][(j,cc)] = U[m][n][(j,cc)] from the panel result Up[(m',n)][(j,cc)], m = m0 + m'
__global__ void k_ea_pack_u(double* __restrict__ Upair, const double* __restrict__ Up, int o, int m0, int nm, long long ld) {
  const long long total = (long long)nm * o * ld;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long col = idx % ld;
    const int n = (idx / ld) % o;
    const int m = m0 + (int)(idx / (ld * o));
    if (m < n) Upair[pair_index(m, n, o) * ld + col] = Up[idx];
  }
}
// hy2[(j, a<b)][cc] -= sum_k t[k,j,a,b] w[k][cc]     (three-body term of Hbar_EA); one block per (j, tri) row
__global__ void __launch_bounds__(64) k_ea_wt2(double* __restrict__ hy, const double* __restrict__ T2p, const double* __restrict__ w,
                                               int o, int v, int Nc) {
  const long long ntri = (long long)v * (v - 1) / 2, vv = (long long)v * v;
  const long long q = blockIdx.x;
  const int j = (int)(q / ntri);
  int a, b;
  decode_tri(q - (long long)j * ntri, v, a, b);
  const long long ab = (long long)a * v + b;
  double* out = hy + ((long long)v + q) * Nc;
  for (int c = threadIdx.x; c < Nc; c += blockDim.x) {
    double acc = 0.0;
    for (int k = 0; k < o; ++k) acc += t2_signed(T2p, k, j, ab, o, vv) * w[(long long)k * Nc + c];
    out[c] -= acc;
  }
}
// K2P[(j',b)][(l,d)] += cFmi * delta_bd Fmi[l][j] + cFae * delta_lj Fae[b][d]   (Fock terms folded into the ring panel;
// IP: cFmi = 1, cFae = -1/2 (k_k2_fixup); EA: cFmi = 1/2, cFae = -1)
__global__ void k_k2_fixup_general(double* __restrict__ K2P, const double* __restrict__ Fmi, const double* __restrict__ Fae, int o,
                                   int v, int j0, double cFmi, double cFae) {
  const int row = blockIdx.x;   // (j', b)
  const int jp = row / v, b = row % v;
  const int j = j0 + jp;
  double* r = K2P + (long long)row * o * v;
  for (int t = threadIdx.x; t < o + v; t += blockDim.x) {
    if (t < o) {
      const int l = t;
      double add = cFmi * Fmi[(long long)l * o + j];
      if (l == j) add += cFae * Fae[(long long)b * v + b];
      r[(long long)l * v + b] += add;
    } else {
      const int d = t - o;
      if (d != b) r[(long long)j * v + d] += cFae * Fae[(long long)b * v + d];
    }
  }
}
// sigma_EA epilogue: s[row] = (w + i eta) y[row] - hy[row] for the v singles rows, and for the doubles rows (j, a<b):
//   s = (w + i eta) y - ( hy + ZP[a][b][j][c] + R[j][b][a][c] - R[j][a][b][c] )       one block per (j, tri) row / per singles row
__global__ void __launch_bounds__(64) k_ea_epilogue(double* __restrict__ sout, const double* __restrict__ yin, const double* __restrict__ ZP,
                                                    const double* __restrict__ R, const double* __restrict__ omega, double eta, int o,
                                                    int v, int nrhs) {
  const long long ntri = (long long)v * (v - 1) / 2;
  const long long row = blockIdx.x;
  const double2* y = reinterpret_cast<const double2*>(yin) + row * nrhs;
  double2* s = reinterpret_cast<double2*>(sout) + row * nrhs;
  const double2 *zp = nullptr, *rba = nullptr, *rab = nullptr;
  if (row >= v) {
    const long long q = row - v;
    const int j = (int)(q / ntri);
    int a, b;
    decode_tri(q - (long long)j * ntri, v, a, b);
    zp = reinterpret_cast<const double2*>(ZP) + (((long long)a * v + b) * o + j) * nrhs;
    rba = reinterpret_cast<const double2*>(R) + (((long long)j * v + b) * v + a) * nrhs;
    rab = reinterpret_cast<const double2*>(R) + (((long long)j * v + a) * v + b) * nrhs;
  }
  for (int r = threadIdx.x; r < nrhs; r += blockDim.x) {
    const double w = omega[r];
    const double2 yv = y[r];
    double2 h = s[r];
    if (zp) { h.x += zp[r].x + rba[r].x - rab[r].x; h.y += zp[r].y + rba[r].y - rab[r].y; }
    s[r] = make_double2(w * yv.x - eta * yv.y - h.x, w * yv.y + eta * yv.x - h.y);
  }
}

// ---- right-hand sides of Eq. 6, columns [c0, nrhs): q = o+c: b1[a] = delta_ac; q = k occupied: b1[a] = -t[k,a], b2[j,a<b] = -t[k,j,a,b]
__global__ void k_ea_build_rhs(double* __restrict__ b, const int* __restrict__ q_of_rhs, const double* __restrict__ t1,
                               const double* __restrict__ T2p, int o, int v, int nrhs, long long nE, int c0) {
  const int nc = nrhs - c0;
  const long long total = nE * nc, ntri = (long long)v * (v - 1) / 2, vv = (long long)v * v;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long row = idx / nc;
    const int r = c0 + (int)(idx - row * nc);
    const int q = q_of_rhs[r];
    double val = 0.0;
    if (q >= o) { if (row == q - o) val = 1.0; }
    else if (row < v) val = -t1[(long long)q * v + row];
    else {
      const long long t = row - v;
      const int j = (int)(t / ntri);
      int a, bb;
      decode_tri(t - (long long)j * ntri, v, a, bb);
      val = -t2_signed(T2p, q, j, (long long)a * v + bb, o, vv);
    }
    reinterpret_cast<double2*>(b)[row * nrhs + r] = make_double2(val, 0.0);
  }
}
// y0 = b / (omega + i eta - d), d_a = f_aa, d_jab = f_aa + f_bb - f_jj (zeroth order); kind 0: y0 = 0.  Columns [c0, nrhs).
__global__ void k_ea_x0(double* __restrict__ x, const double* __restrict__ b, const double* __restrict__ omega, double eta,
                        const double* __restrict__ fdiag, int o, int v, int nrhs, long long nE, int kind, int c0) {
  const int nc = nrhs - c0;
  const long long total = nE * nc, ntri = (long long)v * (v - 1) / 2;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const long long row = idx / nc;
    const int r = c0 + (int)(idx - row * nc);
    double2 out = make_double2(0.0, 0.0);
    if (kind == 1) {
      double d;
      if (row < v) d = fdiag[o + row];
      else {
        const long long t = row - v;
        const int j = (int)(t / ntri);
        int a, bb;
        decode_tri(t - (long long)j * ntri, v, a, bb);
        d = fdiag[o + a] + fdiag[o + bb] - fdiag[j];
      }
      const double re = omega[r] - d;
      const double inv = 1.0 / (re * re + eta * eta);
      const double2 bv = reinterpret_cast<const double2*>(b)[row * nrhs + r];
      out.x = (bv.x * re + bv.y * eta) * inv;      // b / (re + i eta) = b (re - i eta) / (re^2 + eta^2)
      out.y = (bv.y * re - bv.x * eta) * inv;
    }
    reinterpret_cast<double2*>(x)[row * nrhs + r] = out;
  }
}

// ---- G^A assembly ----
// Dv[e][a] = sum_i l[i,a] t[i,e] + 1/2 sum_ijb l[i,j,a,b] t[i,j,e,b]    (one-time; v x v)
__global__ void k_ea_Dv(double* __restrict__ Dv, const double* __restrict__ t1, const double* __restrict__ l1,
                        const double* __restrict__ T2p, const double* __restrict__ L2p, int o, int v) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= v * v) return;
  const int e = idx / v, a = idx % v;
  const long long npair = (long long)o * (o - 1) / 2, ntri = (long long)v * (v - 1) / 2, vv = (long long)v * v;
  double acc = 0.0;
  for (int i = 0; i < o; ++i) acc += l1[(long long)i * v + a] * t1[(long long)i * v + e];
  for (long long pr = 0; pr < npair; ++pr)          // 1/2 sum_ij = sum_(i<j)
    for (int b = 0; b < v; ++b) {
      if (b == a) continue;
      const double l = a < b ? L2p[pr * ntri + tri_index(a, b, v)] : -L2p[pr * ntri + tri_index(b, a, v)];
      acc += l * T2p[pr * vv + (long long)e * v + b];
    }
  Dv[idx] = acc;
}
// g2[i][r] = sum_j sum_(b<c) lambda[i,j,b,c] y2[j,b,c][r]     grid (o, ceil(nrhs/32)); vec row stride ld complex columns
__global__ void __launch_bounds__(256) k_ea_g2(double2* __restrict__ g2, const double* __restrict__ L2p, const double* __restrict__ vec,
                                               int o, int v, int ld, int ncol) {
  __shared__ double2 red[8][32];
  const int i = blockIdx.x, r = blockIdx.y * 32 + threadIdx.x;
  const long long ntri = (long long)v * (v - 1) / 2;
  const double2* y2 = reinterpret_cast<const double2*>(vec) + (long long)v * ld;
  double2 acc = make_double2(0.0, 0.0);
  if (r < ncol)
    for (int j = 0; j < o; ++j) {
      if (j == i) continue;
      const double sg = i < j ? 1.0 : -1.0;
      const double* lp = L2p + (i < j ? pair_index(i, j, o) : pair_index(j, i, o)) * ntri;
      const double2* yj = y2 + (long long)j * ntri * ld + r;
      for (long long t = threadIdx.y; t < ntri; t += 8) {
        const double l = sg * lp[t];
        const double2 yv = yj[t * ld];
        acc.x += l * yv.x; acc.y += l * yv.y;
      }
    }
  red[threadIdx.y][threadIdx.x] = acc;
  __syncthreads();
  if (threadIdx.y == 0 && r < ncol) {
    for (int k = 1; k < 8; ++k) { acc.x += red[k][threadIdx.x].x; acc.y += red[k][threadIdx.x].y; }
    g2[(long long)i * ld + r] = acc;
  }
}
// Gq[out_row[r]][ip] = c_p . y_r for p = plist[ip]; one block per (ip, r)
//   p = k occupied : - sum_a l1[k,a] y1[a] - g2[k]
//   p = o+e virtual: sum_a (delta_ea - Dv[e][a]) y1[a] + sum_(j,b) l1[j,b] y2[j,e,b] - sum_i t1[i,e] g2[i]
__global__ void __launch_bounds__(256) k_ea_assemble_G(double2* __restrict__ Gq, const int* __restrict__ plist, int np,
                                                        const double* __restrict__ vec, const double2* __restrict__ g2,
                                                        const double* __restrict__ Dv, const double* __restrict__ t1,
                                                        const double* __restrict__ l1, int o, int v, int ld,
                                                        const int* __restrict__ out_row) {
  __shared__ double2 red[256];
  const int ip = blockIdx.x, r = blockIdx.y;
  const int p = plist[ip];
  const long long ntri = (long long)v * (v - 1) / 2;
  const double2* y = reinterpret_cast<const double2*>(vec);
  double2 acc = make_double2(0.0, 0.0);
  auto add = [&](double c, double2 val) { acc.x += c * val.x; acc.y += c * val.y; };
  if (p < o) {
    for (int a = threadIdx.x; a < v; a += blockDim.x) add(-l1[(long long)p * v + a], y[(long long)a * ld + r]);
    if (threadIdx.x == 0) add(-1.0, g2[(long long)p * ld + r]);
  } else {
    const int e = p - o;
    for (int a = threadIdx.x; a < v; a += blockDim.x) add((a == e ? 1.0 : 0.0) - Dv[(long long)e * v + a], y[(long long)a * ld + r]);
    for (int i = threadIdx.x; i < o; i += blockDim.x) add(-t1[(long long)i * v + e], g2[(long long)i * ld + r]);
    for (long long t = threadIdx.x; t < (long long)o * v; t += blockDim.x) {
      const int j = t / v, b = t % v;
      if (b == e) continue;
      const long long row = v + (long long)j * ntri + (e < b ? tri_index(e, b, v) : tri_index(b, e, v));
      add((e < b ? 1.0 : -1.0) * l1[(long long)j * v + b], y[row * ld + r]);
    }
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) { red[threadIdx.x].x += red[threadIdx.x + s].x; red[threadIdx.x].y += red[threadIdx.x + s].y; }
    __syncthreads();
  }
  if (threadIdx.x == 0) Gq[(long long)(out_row ? out_row[r] : r) * np + ip] = red[0];
}

// ---- create-time scatter kernels for W_abej (stored packed: WV[(j, a<b)][e]) ----
// WV[(j,a<b)][e] += sign * ( X[j][(a,e)][b]-type panel results ); the layouts are described at the call sites in gfcc_ea_host.inl.
// X1[(a',e)][(j,b)] for a = a0 + a':  WV[(j, a<b)][e] += X1 (a<b);  WV[(j, b<a)][e] -= X1 (b<a)      [antisymmetrised pair term]
__global__ void k_ea_scatter_aebj(double* __restrict__ WV, const double* __restrict__ X, int o, int v, int a0, int na, int mode) {
  const long long total = (long long)na * v * v * o, ntri = (long long)v * (v - 1) / 2;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int e = idx % v;                              // e fastest: coalesced writes of WV rows
    const int b = (idx / v) % v;
    const int j = (idx / ((long long)v * v)) % o;
    const int ap = idx / ((long long)v * v * o);
    const int a = a0 + ap;
    if (a == b || (mode == 0) != (a < b)) continue;
    const double val = X[((long long)ap * v + e) * ((long long)v * o) + (long long)j * v + b];
    if (a < b) WV[((long long)j * ntri + tri_index(a, b, v)) * v + e] += val;
    else WV[((long long)j * ntri + tri_index(b, a, v)) * v + e] -= val;
  }
}
// Xj[j][(b',e)][a] for b = b0 + b':  WV[(j, a<b)][e] -= Xj;  WV[(j, b<a)][e] += Xj      [ -P(ab) X[a,b,e,j] ]
__global__ void k_ea_scatter_jbea(double* __restrict__ WV, const double* __restrict__ X, int o, int v, int b0, int nb, int mode) {
  const long long total = (long long)o * nb * v * v, ntri = (long long)v * (v - 1) / 2;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int e = idx % v;
    const int a = (idx / v) % v;
    const int bp = (idx / ((long long)v * v)) % nb;
    const int j = idx / ((long long)v * v * nb);
    const int b = b0 + bp;
    if (a == b || (mode == 0) != (a < b)) continue;
    const double val = X[(((long long)j * nb + bp) * v + e) * v + a];
    if (a < b) WV[((long long)j * ntri + tri_index(a, b, v)) * v + e] -= val;
    else WV[((long long)j * ntri + tri_index(b, a, v)) * v + e] += val;
  }
}
// WV[(j, a<b)][e] += T[(a,b)][(e,j)] for a<b   (T = full v*v rows)
__global__ void k_ea_pack_abej(double* __restrict__ WV, const double* __restrict__ T, int o, int v, double sign) {
  const long long ntri = (long long)v * (v - 1) / 2, total = ntri * o * v;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int e = idx % v;
    const long long t = (idx / v) % ntri;
    const int j = idx / ((long long)v * ntri);
    int a, b;
    decode_tri(t, v, a, b);
    WV[idx] += sign * T[((long long)a * v + b) * ((long long)v * o) + (long long)e * o + j];
  }
}
// WV[(j, a<b)][e] -= sum_m Fme[m][e] t[m,j,a,b]
__global__ void k_ea_fme_t2(double* __restrict__ WV, const double* __restrict__ Fme, const double* __restrict__ T2p, int o, int v) {
  const long long ntri = (long long)v * (v - 1) / 2, total = ntri * o * v, vv = (long long)v * v;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int e = idx % v;
    const long long t = (idx / v) % ntri;
    const int j = idx / ((long long)v * ntri);
    int a, b;
    decode_tri(t, v, a, b);
    double acc = 0.0;
    for (int m = 0; m < o; ++m) acc += Fme[(long long)m * v + e] * t2_signed(T2p, m, j, (long long)a * v + b, o, vv);
    WV[idx] -= acc;
  }
}
// OOVO[(m<n)][(e,j)] = <mn||ej>~ from G[(m,e)][(j,n)] = sum_Q Lov[Q,m,e] Loo~[Q,n,j]:  G[(m,e)][(j,n)] - G[(n,e)][(j,m)]
__global__ void k_ea_oovo(double* __restrict__ out, const double* __restrict__ G, int o, int v) {
  const long long npair = (long long)o * (o - 1) / 2, total = npair * v * o;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
    const int j = idx % o;
    const int e = (idx / o) % v;
    const long long pr = idx / ((long long)o * v);
    int m, n;
    decode_pair(pr, o, m, n);
    out[idx] = G[((long long)m * v + e) * ((long long)o * o) + (long long)j * o + n] -
               G[((long long)n * v + e) * ((long long)o * o) + (long long)j * o + m];
  }
}
// dst += src (element-wise)
__global__ void k_ea_addto(double* __restrict__ dst, const double* __restrict__ src, long long n) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) dst[i] += src[i];
}

}  // namespace gfcc
