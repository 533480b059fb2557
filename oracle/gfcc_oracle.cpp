// =====================================================================================
// gfcc_oracle.cpp -- CPU ORACLE for the GFCCSD-IP hot path.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may load this library.  It shares no code, header, table or helper with the CUDA path
// (paper_2010_04768_b200/csrc) and never calls it.
//
// What it computes (all FP64, plain loops, OpenMP only over *output* elements):
//   * the spin-orbital similarity-transformed Hamiltonian elements F, W,
//     with the antisymmetrised <pq||rs> = <pq|rs> - <pq|sr>, <pq|rs> = sum_Q L[Q,p,r] L[Q,q,s]
//     formed EXPLICITLY from the Cholesky vectors (BASELINE.json north_star);
//   * sigma = (omega - i eta) X + Hbar X for X = (x1[i], x2[i,j,a])  -- PAPER.md:82 Eq. (5),
//     operator convention X = sum_i x_i a_i + sum_{i<j,a} x_ija a+_a a_j a_i, Eq. (3);
//   * right-hand sides b_p (Eq. 5 rhs) and bra vectors c_q (Eq. 7-8 first term);
//   * GMRES (Saad-Schultz, ref. 85) per right-hand side, modified Gram-Schmidt;
//   * a "row-sampled" sigma for large sizes that uses L-factorised sums of the T1-dressed forms
//     (SURVEY.md 8c item 8); its equality with the definition form is pinned in tests/.
//
// The paper prints none of the working equations (only Fig. 1); the readings
// are listed in DESIGN.md section "Readings".  Every function below is pinned by tests/test_oracle_*.py
// (Fock-space brute force, closed form, shift identity, 4-index route, dense LU) -- nothing is
// "parity unpinned".
//
// Array conventions (host, row-major, double; complex = interleaved re,im):
//   fock [N][N], N=o+v, occupied first.   T1, L1: [o][v].
//   T2p : pair-packed [i<j][a][b] (v*v per pair), pair(i,j)= i*o - i(i+1)/2 + (j-i-1).
//   L2p : fully packed [i<j][a<b], tri(a,b) = a*v - a(a+1)/2 + (b-a-1).
//   Lchol [Q][N][N].   X1 [nrhs][o], X2 [nrhs][o][o][v] (antisymmetric in i,j).
// =====================================================================================
#include <complex>
#include <vector>
#include <cmath>
#include <cstring>
#include <cstdio>
#include <cstdint>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
typedef long long i64;

namespace {

struct Ctx {
  int o, v, Q, N;
  i64 npair, ntri;
  std::vector<double> f, t1, l1;
  const double *T2p, *L2p, *L;     // borrowed from the caller (kept alive by the Python wrapper)
  // ---- definition form (mode 0) ----
  bool has_def = false;
  std::vector<double> t2, l2;                                     // full [o][o][v][v]
  std::vector<double> Lt;                                         // [p][r][Q]
  std::vector<double> oooo, ooov, oovv, ovvo, ovvv, ovoo;         // <pq||rs> blocks
  std::vector<double> Fme, Fmi, Fae, Wmnij, Wmnie, Wmbej, Wmbij;  // items 1-7
  // ---- EA / advanced part, definition form (mode bit 2) ----
  bool has_ea = false;
  std::vector<double> vvvv, vvvo;                 // <ab||ef>, <ab||ei>
  std::vector<double> Wamef, Wabef, Wabei;        // EA intermediates (build_ea)
  // ---- sampled (factorised, T1-dressed) form ----
  bool has_dressed = false;
  std::vector<double> Loo, Lov, Lvv, Lvo;  // dressed blocks, layout [m][i][Q], [m][e][Q], [a][e][Q], [a][i][Q]
  std::vector<double> ft;                  // dressed Fock [N][N]
};

inline i64 pairidx(int i, int j, int o) { return (i64)i * o - (i64)i * (i + 1) / 2 + (j - i - 1); }
inline i64 triidx(int a, int b, int v) { return (i64)a * v - (i64)a * (a + 1) / 2 + (b - a - 1); }

// t[i,j,a,b] from the pair-packed array (antisymmetric in ij; the ab antisymmetry is in the data)
inline double t2p_at(const Ctx& c, int i, int j, int a, int b) {
  if (i == j) return 0.0;
  if (i < j) return c.T2p[(pairidx(i, j, c.o) * c.v + a) * c.v + b];
  return -c.T2p[(pairidx(j, i, c.o) * c.v + a) * c.v + b];
}
inline double l2p_at(const Ctx& c, int i, int j, int a, int b) {
  if (i == j || a == b) return 0.0;
  double s = 1.0;
  if (i > j) { std::swap(i, j); s = -s; }
  if (a > b) { std::swap(a, b); s = -s; }
  return s * c.L2p[pairidx(i, j, c.o) * c.ntri + triidx(a, b, c.v)];
}

// index helpers for the definition-form arrays
#define IDX4(a, b, c_, d, nb, nc, nd) ((((i64)(a) * (nb) + (b)) * (nc) + (c_)) * (nd) + (d))

// <pq||rs> for global spin-orbital indices, from Lt[p][r][Q]
inline double asym_int(const Ctx& c, int p, int q, int r, int s) {
  const int Q = c.Q, N = c.N;
  const double* pr = &c.Lt[((i64)p * N + r) * Q];
  const double* qs = &c.Lt[((i64)q * N + s) * Q];
  const double* ps = &c.Lt[((i64)p * N + s) * Q];
  const double* qr = &c.Lt[((i64)q * N + r) * Q];
  double acc = 0.0;
  for (int k = 0; k < Q; ++k) acc += pr[k] * qs[k] - ps[k] * qr[k];
  return acc;
}

// block of antisymmetrised integrals over ranges [p0,p0+np) x ... (global indices)
void build_block(const Ctx& c, std::vector<double>& out, int p0, int np, int q0, int nq, int r0, int nr, int s0, int ns) {
  out.assign((size_t)np * nq * nr * ns, 0.0);
#pragma omp parallel for collapse(2) schedule(static)
  for (int p = 0; p < np; ++p)
    for (int q = 0; q < nq; ++q)
      for (int r = 0; r < nr; ++r)
        for (int s = 0; s < ns; ++s)
          out[IDX4(p, q, r, s, nq, nr, ns)] = asym_int(c, p0 + p, q0 + q, r0 + r, s0 + s);
}

// ------------------------------------------------------------------------------------
// Definition form: SURVEY.md 8c items 1-7 (spin-orbital Hbar elements).
// ------------------------------------------------------------------------------------
void build_def(Ctx& c) {
  const int o = c.o, v = c.v, Q = c.Q, N = c.N;
  // transposed Cholesky vectors Lt[p][r][Q]
  c.Lt.resize((size_t)N * N * Q);
#pragma omp parallel for collapse(2)
  for (int p = 0; p < N; ++p)
    for (int r = 0; r < N; ++r)
      for (int k = 0; k < Q; ++k) c.Lt[((i64)p * N + r) * Q + k] = c.L[((i64)k * N + p) * N + r];
  // full amplitudes
  c.t2.assign((size_t)o * o * v * v, 0.0);
  c.l2.assign((size_t)o * o * v * v, 0.0);
#pragma omp parallel for collapse(2)
  for (int i = 0; i < o; ++i)
    for (int j = 0; j < o; ++j)
      for (int a = 0; a < v; ++a)
        for (int b = 0; b < v; ++b) {
          c.t2[IDX4(i, j, a, b, o, v, v)] = t2p_at(c, i, j, a, b);
          c.l2[IDX4(i, j, a, b, o, v, v)] = l2p_at(c, i, j, a, b);
        }
  build_block(c, c.oooo, 0, o, 0, o, 0, o, 0, o);
  build_block(c, c.ooov, 0, o, 0, o, 0, o, o, v);
  build_block(c, c.oovv, 0, o, 0, o, o, v, o, v);
  build_block(c, c.ovvo, 0, o, o, v, o, v, 0, o);
  build_block(c, c.ovvv, 0, o, o, v, o, v, o, v);
  build_block(c, c.ovoo, 0, o, o, v, 0, o, 0, o);

  const std::vector<double>&t1 = c.t1, &t2 = c.t2, &f = c.f;
  auto T1 = [&](int i, int a) { return t1[(i64)i * v + a]; };
  auto T2 = [&](int i, int j, int a, int b) { return t2[IDX4(i, j, a, b, o, v, v)]; };
  auto TAU = [&](int i, int j, int a, int b) { return T2(i, j, a, b) + T1(i, a) * T1(j, b) - T1(i, b) * T1(j, a); };
  auto Foo = [&](int m, int i) { return f[(i64)m * N + i]; };
  auto Fov = [&](int m, int e) { return f[(i64)m * N + o + e]; };
  auto Fvv = [&](int a, int e) { return f[(i64)(o + a) * N + o + e]; };
  auto mnij = [&](int m, int n, int i, int j) { return c.oooo[IDX4(m, n, i, j, o, o, o)]; };
  auto mnie = [&](int m, int n, int i, int e) { return c.ooov[IDX4(m, n, i, e, o, o, v)]; };
  auto mnef = [&](int m, int n, int e, int g) { return c.oovv[IDX4(m, n, e, g, o, v, v)]; };
  auto mbej = [&](int m, int b, int e, int j) { return c.ovvo[IDX4(m, b, e, j, v, v, o)]; };
  auto mbef = [&](int m, int b, int e, int g) { return c.ovvv[IDX4(m, b, e, g, v, v, v)]; };
  auto mbij = [&](int m, int b, int i, int j) { return c.ovoo[IDX4(m, b, i, j, v, o, o)]; };
  auto amef = [&](int a, int m, int e, int g) { return -mbef(m, a, e, g); };   // <am||ef> = -<ma||ef>
  auto mnej = [&](int m, int n, int e, int j) { return -mnie(m, n, j, e); };   // <mn||ej> = -<mn||je>

  // item 1: F_me = f_me + sum_nf t[n,f] <mn||ef>
  c.Fme.assign((size_t)o * v, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int e = 0; e < v; ++e) {
      double acc = Fov(m, e);
      for (int n = 0; n < o; ++n)
        for (int g = 0; g < v; ++g) acc += T1(n, g) * mnef(m, n, e, g);
      c.Fme[(i64)m * v + e] = acc;
    }
  // item 2: F_mi = f_mi + sum_e f_me t[i,e] + sum_ne t[n,e]<mn||ie> + 1/2 sum_nef <mn||ef> tau[i,n,e,f]
  c.Fmi.assign((size_t)o * o, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int i = 0; i < o; ++i) {
      double acc = Foo(m, i);
      for (int e = 0; e < v; ++e) acc += Fov(m, e) * T1(i, e);
      for (int n = 0; n < o; ++n)
        for (int e = 0; e < v; ++e) acc += T1(n, e) * mnie(m, n, i, e);
      for (int n = 0; n < o; ++n)
        for (int e = 0; e < v; ++e)
          for (int g = 0; g < v; ++g) acc += 0.5 * mnef(m, n, e, g) * TAU(i, n, e, g);
      c.Fmi[(i64)m * o + i] = acc;
    }
  // item 3: F_ae = f_ae - sum_m f_me t[m,a] + sum_mf t[m,f]<am||ef> - 1/2 sum_mnf tau[m,n,a,f]<mn||ef>
  c.Fae.assign((size_t)v * v, 0.0);
#pragma omp parallel for collapse(2)
  for (int a = 0; a < v; ++a)
    for (int e = 0; e < v; ++e) {
      double acc = Fvv(a, e);
      for (int m = 0; m < o; ++m) acc -= Fov(m, e) * T1(m, a);
      for (int m = 0; m < o; ++m)
        for (int g = 0; g < v; ++g) acc += T1(m, g) * amef(a, m, e, g);
      for (int m = 0; m < o; ++m)
        for (int n = 0; n < o; ++n)
          for (int g = 0; g < v; ++g) acc -= 0.5 * TAU(m, n, a, g) * mnef(m, n, e, g);
      c.Fae[(i64)a * v + e] = acc;
    }
  // item 4: W_mnij = <mn||ij> + P(ij) sum_e t[j,e]<mn||ie> + 1/2 sum_ef tau[i,j,e,f]<mn||ef>
  c.Wmnij.assign((size_t)o * o * o * o, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int n = 0; n < o; ++n)
      for (int i = 0; i < o; ++i)
        for (int j = 0; j < o; ++j) {
          double acc = mnij(m, n, i, j);
          for (int e = 0; e < v; ++e) acc += T1(j, e) * mnie(m, n, i, e) - T1(i, e) * mnie(m, n, j, e);
          for (int e = 0; e < v; ++e)
            for (int g = 0; g < v; ++g) acc += 0.5 * TAU(i, j, e, g) * mnef(m, n, e, g);
          c.Wmnij[IDX4(m, n, i, j, o, o, o)] = acc;
        }
  // item 5: W_mnie = <mn||ie> + sum_f t[i,f]<mn||fe>
  c.Wmnie.assign((size_t)o * o * o * v, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int n = 0; n < o; ++n)
      for (int i = 0; i < o; ++i)
        for (int e = 0; e < v; ++e) {
          double acc = mnie(m, n, i, e);
          for (int g = 0; g < v; ++g) acc += T1(i, g) * mnef(m, n, g, e);
          c.Wmnie[IDX4(m, n, i, e, o, o, v)] = acc;
        }
  // item 6: W_mbej = <mb||ej> + sum_f t[j,f]<mb||ef> - sum_n t[n,b]<mn||ej>
  //                  - sum_nf (t[j,n,f,b] + t[j,f] t[n,b]) <mn||ef>
  c.Wmbej.assign((size_t)o * v * v * o, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int b = 0; b < v; ++b)
      for (int e = 0; e < v; ++e)
        for (int j = 0; j < o; ++j) {
          double acc = mbej(m, b, e, j);
          for (int g = 0; g < v; ++g) acc += T1(j, g) * mbef(m, b, e, g);
          for (int n = 0; n < o; ++n) acc -= T1(n, b) * mnej(m, n, e, j);
          for (int n = 0; n < o; ++n)
            for (int g = 0; g < v; ++g) acc -= (T2(j, n, g, b) + T1(j, g) * T1(n, b)) * mnef(m, n, e, g);
          c.Wmbej[IDX4(m, b, e, j, v, v, o)] = acc;
        }
  // item 7: W_mbij = <mb||ij> - sum_e F_me t[i,j,b,e] - sum_n t[n,b] W_mnij + 1/2 sum_ef <mb||ef> tau[i,j,e,f]
  //                  + P(ij) sum_ne <mn||ie> t[j,n,b,e]
  //                  + P(ij) sum_e t[i,e] ( <mb||ej> - sum_nf t[n,j,b,f] <mn||ef> )
  // the parenthesis of the last line is an array in (m,b,e,j):
  std::vector<double> par((size_t)o * v * v * o, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int b = 0; b < v; ++b)
      for (int e = 0; e < v; ++e)
        for (int j = 0; j < o; ++j) {
          double acc = mbej(m, b, e, j);
          for (int n = 0; n < o; ++n)
            for (int g = 0; g < v; ++g) acc -= T2(n, j, b, g) * mnef(m, n, e, g);
          par[IDX4(m, b, e, j, v, v, o)] = acc;
        }
  c.Wmbij.assign((size_t)o * v * o * o, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int b = 0; b < v; ++b)
      for (int i = 0; i < o; ++i)
        for (int j = 0; j < o; ++j) {
          double acc = mbij(m, b, i, j);
          for (int e = 0; e < v; ++e) acc -= c.Fme[(i64)m * v + e] * T2(i, j, b, e);
          for (int n = 0; n < o; ++n) acc -= T1(n, b) * c.Wmnij[IDX4(m, n, i, j, o, o, o)];
          for (int e = 0; e < v; ++e)
            for (int g = 0; g < v; ++g) acc += 0.5 * mbef(m, b, e, g) * TAU(i, j, e, g);
          for (int n = 0; n < o; ++n)
            for (int e = 0; e < v; ++e) acc += mnie(m, n, i, e) * T2(j, n, b, e) - mnie(m, n, j, e) * T2(i, n, b, e);
          for (int e = 0; e < v; ++e)
            acc += T1(i, e) * par[IDX4(m, b, e, j, v, v, o)] - T1(j, e) * par[IDX4(m, b, e, i, v, v, o)];
          c.Wmbij[IDX4(m, b, i, j, v, o, o)] = acc;
        }
  c.has_def = true;
}

// ------------------------------------------------------------------------------------
// sigma, definition form (SURVEY.md 8c "sigma"; operator order a+_a a_j a_i of PAPER.md:75 Eq. 3)
//  s1[i]     = (w - i eta) x1[i] - sum_m F_mi x1[m] - sum_me F_me x2[m,i,e] + 1/2 sum_mne W_nmie x2[m,n,e]
//  s2[i,j,a] = (w - i eta) x2[i,j,a] + sum_e F_ae x2[i,j,e] - P(ij) sum_m F_mi x2[m,j,a] + sum_m W_maji x1[m]
//              + 1/2 sum_mn W_mnij x2[m,n,a] + P(ij) sum_me W_maei x2[m,j,e]
//              + 1/2 sum_mnef <mn||ef> x2[m,n,f] t[i,j,a,e]
// ------------------------------------------------------------------------------------
void sigma_def_one(const Ctx& c, double omega, double eta, const cd* x1, const cd* x2, cd* s1, cd* s2) {
  const int o = c.o, v = c.v;
  const cd shift(omega, -eta);
  auto X2 = [&](int i, int j, int a) { return x2[((i64)i * o + j) * v + a]; };
  // y[e] = 1/2 sum_mnf <mn||ef> x2[m,n,f]
  std::vector<cd> y(v);
#pragma omp parallel for
  for (int e = 0; e < v; ++e) {
    cd acc = 0.0;
    for (int m = 0; m < o; ++m)
      for (int n = 0; n < o; ++n)
        for (int g = 0; g < v; ++g) acc += 0.5 * c.oovv[IDX4(m, n, e, g, o, v, v)] * X2(m, n, g);
    y[e] = acc;
  }
#pragma omp parallel for
  for (int i = 0; i < o; ++i) {
    cd acc = shift * x1[i];
    for (int m = 0; m < o; ++m) acc -= c.Fmi[(i64)m * o + i] * x1[m];
    for (int m = 0; m < o; ++m)
      for (int e = 0; e < v; ++e) acc -= c.Fme[(i64)m * v + e] * X2(m, i, e);
    for (int m = 0; m < o; ++m)
      for (int n = 0; n < o; ++n)
        for (int e = 0; e < v; ++e) acc += 0.5 * c.Wmnie[IDX4(n, m, i, e, o, o, v)] * X2(m, n, e);
    s1[i] = acc;
  }
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
  for (int i = 0; i < o; ++i)
    for (int j = 0; j < o; ++j)
      for (int a = 0; a < v; ++a) {
        cd acc = shift * X2(i, j, a);
        for (int e = 0; e < v; ++e) acc += c.Fae[(i64)a * v + e] * X2(i, j, e);
        for (int m = 0; m < o; ++m) acc -= c.Fmi[(i64)m * o + i] * X2(m, j, a) - c.Fmi[(i64)m * o + j] * X2(m, i, a);
        for (int m = 0; m < o; ++m) acc += c.Wmbij[IDX4(m, a, j, i, v, o, o)] * x1[m];
        for (int m = 0; m < o; ++m)
          for (int n = 0; n < o; ++n) acc += 0.5 * c.Wmnij[IDX4(m, n, i, j, o, o, o)] * X2(m, n, a);
        for (int m = 0; m < o; ++m)
          for (int e = 0; e < v; ++e)
            acc += c.Wmbej[IDX4(m, a, e, i, v, v, o)] * X2(m, j, e) - c.Wmbej[IDX4(m, a, e, j, v, v, o)] * X2(m, i, e);
        for (int e = 0; e < v; ++e) acc += c.t2[IDX4(i, j, a, e, o, v, v)] * y[e];
        s2[((i64)i * o + j) * v + a] = acc;
      }
}

// ------------------------------------------------------------------------------------
// T1-dressed Cholesky blocks and dressed Fock; used only by the
// row-sampled sigma.   Ltilde = A^T L B,  A = 1 - t1 (occ,virt block), B = 1 + t1^T (virt,occ block).
// Layouts put Q fastest so that every sum over Q below is a contiguous dot product.
// ------------------------------------------------------------------------------------
void build_dressed(Ctx& c) {
  const int o = c.o, v = c.v, Q = c.Q, N = c.N;
  auto Lg = [&](int k, int p, int q) { return c.L[((i64)k * N + p) * N + q]; };
  auto T1 = [&](int i, int a) { return c.t1[(i64)i * v + a]; };
  c.Lov.resize((size_t)o * v * Q); c.Loo.resize((size_t)o * o * Q);
  c.Lvv.resize((size_t)v * v * Q); c.Lvo.resize((size_t)v * o * Q);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int e = 0; e < v; ++e)
      for (int k = 0; k < Q; ++k) c.Lov[((i64)m * v + e) * Q + k] = Lg(k, m, o + e);
  // Loo[m,i] = L_mi + sum_e t[i,e] L_me
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int i = 0; i < o; ++i)
      for (int k = 0; k < Q; ++k) {
        double acc = Lg(k, m, i);
        for (int e = 0; e < v; ++e) acc += T1(i, e) * Lg(k, m, o + e);
        c.Loo[((i64)m * o + i) * Q + k] = acc;
      }
  // Lvv[a,e] = L_ae - sum_m t[m,a] L_me
#pragma omp parallel for collapse(2)
  for (int a = 0; a < v; ++a)
    for (int e = 0; e < v; ++e)
      for (int k = 0; k < Q; ++k) {
        double acc = Lg(k, o + a, o + e);
        for (int m = 0; m < o; ++m) acc -= T1(m, a) * Lg(k, m, o + e);
        c.Lvv[((i64)a * v + e) * Q + k] = acc;
      }
  // Lvo[a,i] = L_ai - sum_m t[m,a] L_mi + sum_e t[i,e] L_ae - sum_me t[m,a] t[i,e] L_me
  //          = L_ai - sum_m t[m,a] L_mi + sum_e t[i,e] ( L_ae - sum_m t[m,a] L_me )      [ (A^T L) B, SURVEY.md 8a P1 ]
  //          = L_ai - sum_m t[m,a] L_mi + sum_e t[i,e] Lvv[a,e]        with the dressed Lvv computed just above
  // (the bracketed sum is taken once per (a,e) instead of once per (a,i,e): same terms, O(Q v o (o+v)) work)
#pragma omp parallel for collapse(2)
  for (int a = 0; a < v; ++a)
    for (int i = 0; i < o; ++i) {
      double* dst = &c.Lvo[((i64)a * o + i) * Q];
      for (int k = 0; k < Q; ++k) dst[k] = Lg(k, o + a, i);
      for (int m = 0; m < o; ++m) {
        const double t = T1(m, a);
        for (int k = 0; k < Q; ++k) dst[k] -= t * Lg(k, m, i);
      }
      for (int e = 0; e < v; ++e) {
        const double t = T1(i, e);
        const double* lv = &c.Lvv[((i64)a * v + e) * Q];
        for (int k = 0; k < Q; ++k) dst[k] += t * lv[k];
      }
    }
  // dressed Fock: ft = A^T ( f + J - K ) B,  (f+J-K)_pq = f_pq + sum_kc t[k,c] <pk||qc>
  std::vector<double> s(Q, 0.0), g((size_t)N * N, 0.0), U((size_t)Q * N * o, 0.0);
  for (int k = 0; k < Q; ++k) {
    double acc = 0;
    for (int m = 0; m < o; ++m)
      for (int e = 0; e < v; ++e) acc += T1(m, e) * Lg(k, m, o + e);
    s[k] = acc;
  }
  // U[Q,p,k] = sum_c L[Q,p,c] t[k,c]
#pragma omp parallel for collapse(2)
  for (int k = 0; k < Q; ++k)
    for (int p = 0; p < N; ++p)
      for (int m = 0; m < o; ++m) {
        double acc = 0;
        for (int e = 0; e < v; ++e) acc += Lg(k, p, o + e) * T1(m, e);
        U[((i64)k * N + p) * o + m] = acc;
      }
#pragma omp parallel for collapse(2)
  for (int p = 0; p < N; ++p)
    for (int q = 0; q < N; ++q) {
      double acc = c.f[(i64)p * N + q];
      for (int k = 0; k < Q; ++k) {
        acc += s[k] * Lg(k, p, q);
        for (int m = 0; m < o; ++m) acc -= U[((i64)k * N + p) * o + m] * Lg(k, m, q);
      }
      g[(i64)p * N + q] = acc;
    }
  // A^T g B
  std::vector<double> Am((size_t)N * N, 0.0), Bm((size_t)N * N, 0.0), tmp((size_t)N * N, 0.0);
  for (int p = 0; p < N; ++p) Am[(i64)p * N + p] = Bm[(i64)p * N + p] = 1.0;
  for (int m = 0; m < o; ++m)
    for (int a = 0; a < v; ++a) { Am[(i64)m * N + o + a] -= T1(m, a); Bm[(i64)(o + a) * N + m] += T1(m, a); }
  for (int p = 0; p < N; ++p)
    for (int q = 0; q < N; ++q) {
      double acc = 0;
      for (int r = 0; r < N; ++r) acc += Am[(i64)r * N + p] * g[(i64)r * N + q];
      tmp[(i64)p * N + q] = acc;
    }
  c.ft.assign((size_t)N * N, 0.0);
  for (int p = 0; p < N; ++p)
    for (int q = 0; q < N; ++q) {
      double acc = 0;
      for (int r = 0; r < N; ++r) acc += tmp[(i64)p * N + r] * Bm[(i64)r * N + q];
      c.ft[(i64)p * N + q] = acc;
    }
  c.has_dressed = true;
}

inline double dotQ(const double* a, const double* b, int Q) {
  double acc = 0;
  for (int k = 0; k < Q; ++k) acc += a[k] * b[k];
  return acc;
}

// ------------------------------------------------------------------------------------
// EA / advanced part (Eq. 4, Eq. 6, second terms of Eq. 7-8), definition form.
// Operator Y = sum_a y1[a] a+_a + sum_{j, a<b} y2[j,a,b] a+_a a+_b a_j  (Eq. 4 order; y2 antisymmetric in a,b).
// The paper prints no working equations (reading 28); these are the spin-orbital EA-EOM-CCSD-type
// equations for the connected action <mu|[Hbar_N, Y]|Phi>, pinned by the Fock-space brute force in tests/:
//   W_amef = <am||ef> - sum_n t[n,a] <nm||ef>
//   W_abef = <ab||ef> - P(ab) sum_m t[m,b] <am||ef> + 1/2 sum_mn tau[m,n,a,b] <mn||ef>
//   W_abei = <ab||ei> + 1/2 sum_mn <mn||ei> tau[m,n,a,b] - sum_m F_me t[m,i,a,b] + sum_f W_abef t[i,f]
//            - P(ab) sum_mf <mb||ef> t[m,i,a,f] - P(ab) sum_m t[m,a] ( <mb||ei> - sum_nf t[n,i,b,f] <mn||ef> )
//   (Hbar y)1[a]     = sum_c F_ac y1[c] + sum_ld F_ld y2[l,a,d] + 1/2 sum_lcd W_alcd y2[l,c,d]
//   (Hbar y)2[j,a,b] = sum_c W_abcj y1[c] + P(ab) sum_c F_ac y2[j,c,b] - sum_l F_lj y2[l,a,b] + P(ab) sum_ld W_lbdj y2[l,a,d]
//                      + 1/2 sum_cd W_abcd y2[j,c,d] - 1/2 sum_klcd <kl||cd> y2[l,c,d] t[k,j,a,b]
//   sigma_EA = (omega + i eta) y - Hbar y                                                      (Eq. 6)
// ------------------------------------------------------------------------------------
void build_ea(Ctx& c) {
  const int o = c.o, v = c.v;
  build_block(c, c.vvvv, o, v, o, v, o, v, o, v);
  build_block(c, c.vvvo, o, v, o, v, o, v, 0, o);
  const std::vector<double>&t1 = c.t1, &t2 = c.t2;
  auto T1 = [&](int i, int a) { return t1[(i64)i * v + a]; };
  auto T2 = [&](int i, int j, int a, int b) { return t2[IDX4(i, j, a, b, o, v, v)]; };
  auto TAU = [&](int i, int j, int a, int b) { return T2(i, j, a, b) + T1(i, a) * T1(j, b) - T1(i, b) * T1(j, a); };
  auto mnef = [&](int m, int n, int e, int g) { return c.oovv[IDX4(m, n, e, g, o, v, v)]; };
  auto mbef = [&](int m, int b, int e, int g) { return c.ovvv[IDX4(m, b, e, g, v, v, v)]; };
  auto amef = [&](int a, int m, int e, int g) { return -mbef(m, a, e, g); };          // <am||ef> = -<ma||ef>
  auto mbei = [&](int m, int b, int e, int i) { return c.ovvo[IDX4(m, b, e, i, v, v, o)]; };
  auto mnei = [&](int m, int n, int e, int i) { return -c.ooov[IDX4(m, n, i, e, o, o, v)]; };   // <mn||ei> = -<mn||ie>
  c.Wamef.assign((size_t)v * o * v * v, 0.0);
#pragma omp parallel for collapse(2)
  for (int a = 0; a < v; ++a)
    for (int m = 0; m < o; ++m)
      for (int e = 0; e < v; ++e)
        for (int g = 0; g < v; ++g) {
          double acc = amef(a, m, e, g);
          for (int n = 0; n < o; ++n) acc -= T1(n, a) * mnef(n, m, e, g);
          c.Wamef[IDX4(a, m, e, g, o, v, v)] = acc;
        }
  c.Wabef.assign((size_t)v * v * v * v, 0.0);
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int a = 0; a < v; ++a)
    for (int b = 0; b < v; ++b)
      for (int e = 0; e < v; ++e)
        for (int g = 0; g < v; ++g) {
          double acc = c.vvvv[IDX4(a, b, e, g, v, v, v)];
          for (int m = 0; m < o; ++m) acc -= T1(m, b) * amef(a, m, e, g) - T1(m, a) * amef(b, m, e, g);
          for (int m = 0; m < o; ++m)
            for (int n = 0; n < o; ++n) acc += 0.5 * TAU(m, n, a, b) * mnef(m, n, e, g);
          c.Wabef[IDX4(a, b, e, g, v, v, v)] = acc;
        }
  // the P(ab) pieces of W_abei as arrays in (a,b,e,i)
  std::vector<double> tmp1((size_t)v * v * v * o, 0.0), tmp2((size_t)v * v * v * o, 0.0), par((size_t)o * v * v * o, 0.0);
#pragma omp parallel for collapse(2)
  for (int m = 0; m < o; ++m)
    for (int b = 0; b < v; ++b)
      for (int e = 0; e < v; ++e)
        for (int i = 0; i < o; ++i) {
          double acc = mbei(m, b, e, i);
          for (int n = 0; n < o; ++n)
            for (int g = 0; g < v; ++g) acc -= T2(n, i, b, g) * mnef(m, n, e, g);
          par[IDX4(m, b, e, i, v, v, o)] = acc;
        }
#pragma omp parallel for collapse(2)
  for (int a = 0; a < v; ++a)
    for (int b = 0; b < v; ++b)
      for (int e = 0; e < v; ++e)
        for (int i = 0; i < o; ++i) {
          double x1 = 0.0, x2 = 0.0;
          for (int m = 0; m < o; ++m)
            for (int g = 0; g < v; ++g) x1 += mbef(m, b, e, g) * T2(m, i, a, g);
          for (int m = 0; m < o; ++m) x2 += T1(m, a) * par[IDX4(m, b, e, i, v, v, o)];
          tmp1[IDX4(a, b, e, i, v, v, o)] = x1;
          tmp2[IDX4(a, b, e, i, v, v, o)] = x2;
        }
  c.Wabei.assign((size_t)v * v * v * o, 0.0);
#pragma omp parallel for collapse(2)
  for (int a = 0; a < v; ++a)
    for (int b = 0; b < v; ++b)
      for (int e = 0; e < v; ++e)
        for (int i = 0; i < o; ++i) {
          double acc = c.vvvo[IDX4(a, b, e, i, v, v, o)];
          for (int m = 0; m < o; ++m)
            for (int n = 0; n < o; ++n) acc += 0.5 * mnei(m, n, e, i) * TAU(m, n, a, b);
          for (int m = 0; m < o; ++m) acc -= c.Fme[(i64)m * v + e] * T2(m, i, a, b);
          for (int g = 0; g < v; ++g) acc += c.Wabef[IDX4(a, b, e, g, v, v, v)] * T1(i, g);
          acc -= tmp1[IDX4(a, b, e, i, v, v, o)] - tmp1[IDX4(b, a, e, i, v, v, o)];
          acc -= tmp2[IDX4(a, b, e, i, v, v, o)] - tmp2[IDX4(b, a, e, i, v, v, o)];
          c.Wabei[IDX4(a, b, e, i, v, v, o)] = acc;
        }
  c.has_ea = true;
}

// sigma_EA for one right-hand side.  y1 [v], y2 [o][v][v] (antisymmetric in a,b); s1, s2 same shapes.
void sigma_ea_one(const Ctx& c, double omega, double eta, const cd* y1, const cd* y2, cd* s1, cd* s2) {
  const int o = c.o, v = c.v;
  const cd shift(omega, eta);
  auto Y2 = [&](int j, int a, int b) { return y2[((i64)j * v + a) * v + b]; };
  // w[k] = 1/2 sum_lcd <kl||cd> y2[l,c,d]
  std::vector<cd> w(o);
  for (int k = 0; k < o; ++k) {
    cd acc = 0.0;
    for (int l = 0; l < o; ++l)
      for (int cc = 0; cc < v; ++cc)
        for (int d = 0; d < v; ++d) acc += 0.5 * c.oovv[IDX4(k, l, cc, d, o, v, v)] * Y2(l, cc, d);
    w[k] = acc;
  }
#pragma omp parallel for
  for (int a = 0; a < v; ++a) {
    cd acc = 0.0;
    for (int cc = 0; cc < v; ++cc) acc += c.Fae[(i64)a * v + cc] * y1[cc];
    for (int l = 0; l < o; ++l)
      for (int d = 0; d < v; ++d) acc += c.Fme[(i64)l * v + d] * Y2(l, a, d);
    for (int l = 0; l < o; ++l)
      for (int cc = 0; cc < v; ++cc)
        for (int d = 0; d < v; ++d) acc += 0.5 * c.Wamef[IDX4(a, l, cc, d, o, v, v)] * Y2(l, cc, d);
    s1[a] = shift * y1[a] - acc;
  }
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
  for (int j = 0; j < o; ++j)
    for (int a = 0; a < v; ++a)
      for (int b = 0; b < v; ++b) {
        cd acc = 0.0;
        for (int cc = 0; cc < v; ++cc) acc += c.Wabei[IDX4(a, b, cc, j, v, v, o)] * y1[cc];
        for (int cc = 0; cc < v; ++cc) acc += c.Fae[(i64)a * v + cc] * Y2(j, cc, b) - c.Fae[(i64)b * v + cc] * Y2(j, cc, a);
        for (int l = 0; l < o; ++l) acc -= c.Fmi[(i64)l * o + j] * Y2(l, a, b);
        for (int l = 0; l < o; ++l)
          for (int d = 0; d < v; ++d)
            acc += c.Wmbej[IDX4(l, b, d, j, v, v, o)] * Y2(l, a, d) - c.Wmbej[IDX4(l, a, d, j, v, v, o)] * Y2(l, b, d);
        for (int cc = 0; cc < v; ++cc)
          for (int d = 0; d < v; ++d) acc += 0.5 * c.Wabef[IDX4(a, b, cc, d, v, v, v)] * Y2(j, cc, d);
        for (int k = 0; k < o; ++k) acc -= w[k] * c.t2[IDX4(k, j, a, b, o, v, v)];
        s2[((i64)j * v + a) * v + b] = shift * Y2(j, a, b) - acc;
      }
}

// ------------------------------------------------------------------------------------
// GMRES(m) iteration shared by the IP system (Eq. 5) and the EA system (Eq. 6): Saad & Schultz 1986 (PAPER.md ref. 85;
// PAPER.md:136-138), modified Gram-Schmidt Arnoldi in the plain Euclidean metric of the PACKED vector, complex Givens
// rotations, stop when the rotated residual |g_{j+1}| <= tol * ||b||.  apply(z, Az) is the operator; x holds x0 on entry
// and the iterate on exit.  Returns the number of operator applications; res = final relative residual (estimate).
// hist (nullable): hist[k] = residual estimate after application k+1 (an output only).
// ------------------------------------------------------------------------------------
template <class Apply>
int gmres_core(i64 n, Apply&& apply, const std::vector<cd>& b, std::vector<cd>& x, double tol, int m, int maxit, double& res_out,
               double* hist, int nhist) {
  auto dot = [&](const std::vector<cd>& a, const std::vector<cd>& bb) {
    cd acc = 0.0;
    for (i64 k = 0; k < n; ++k) acc += std::conj(a[k]) * bb[k];
    return acc;
  };
  std::vector<cd> r, w;
  const double bnorm = std::sqrt(std::real(dot(b, b)));
  int napply = 0;
  double res = 1.0;
  while (napply < maxit) {
    apply(x, w); ++napply;
    r.resize(n);
    for (i64 k = 0; k < n; ++k) r[k] = b[k] - w[k];
    const double beta = std::sqrt(std::real(dot(r, r)));
    res = beta / bnorm;
    if (hist && napply - 1 < nhist) hist[napply - 1] = res;
    if (res <= tol) break;
    std::vector<std::vector<cd>> V(1, r);
    for (auto& e : V[0]) e /= beta;
    std::vector<std::vector<cd>> H(m + 1, std::vector<cd>(m, 0.0));
    std::vector<cd> cs(m), sn(m), g(m + 1, 0.0);
    g[0] = beta;
    int j = 0;
    for (; j < m && napply < maxit; ++j) {
      apply(V[j], w); ++napply;
      for (int k = 0; k <= j; ++k) {
        H[k][j] = dot(V[k], w);
        for (i64 q = 0; q < n; ++q) w[q] -= H[k][j] * V[k][q];
      }
      const double hn = std::sqrt(std::real(dot(w, w)));
      H[j + 1][j] = hn;
      for (int k = 0; k < j; ++k) {   // previous rotations
        cd a = H[k][j], bb = H[k + 1][j];
        H[k][j] = std::conj(cs[k]) * a + std::conj(sn[k]) * bb;
        H[k + 1][j] = -sn[k] * a + cs[k] * bb;
      }
      {   // new rotation annihilating H[j+1][j]
        cd a = H[j][j]; double bb = hn;
        double den = std::sqrt(std::norm(a) + bb * bb);
        cs[j] = a / den; sn[j] = bb / den;
        H[j][j] = std::conj(cs[j]) * a + std::conj(sn[j]) * bb;
        H[j + 1][j] = 0.0;
        g[j + 1] = -sn[j] * g[j];
        g[j] = std::conj(cs[j]) * g[j];
      }
      res = std::abs(g[j + 1]) / bnorm;
      if (hist && napply - 1 < nhist) hist[napply - 1] = res;
      if (res <= tol || hn == 0.0) { ++j; break; }
      V.push_back(w);
      for (auto& e : V.back()) e /= hn;
    }
    // back substitution and update
    std::vector<cd> yv(j);
    for (int k = j - 1; k >= 0; --k) {
      cd acc = g[k];
      for (int q = k + 1; q < j; ++q) acc -= H[k][q] * yv[q];
      yv[k] = acc / H[k][k];
    }
    for (int k = 0; k < j; ++k)
      for (i64 q = 0; q < n; ++q) x[q] += yv[k] * V[k][q];
    if (res <= tol) break;
  }
  res_out = res;
  return napply;
}

}  // namespace

extern "C" {

// mode bit 0: build the definition-form arrays (items 1-7; needs O(o v^3) memory);
// mode bit 1: build the T1-dressed blocks for the row-sampled sigma;
// mode bit 2 (with bit 0): build the EA intermediates W_amef, W_abef, W_abei (needs O(v^4) memory).
void* orc_create(int o, int v, int Q, const double* fock, const double* T1, const double* T2p, const double* L1,
                 const double* L2p, const double* Lchol, int mode) {
  Ctx* c = new Ctx();
  c->o = o; c->v = v; c->Q = Q; c->N = o + v;
  c->npair = (i64)o * (o - 1) / 2; c->ntri = (i64)v * (v - 1) / 2;
  c->f.assign(fock, fock + (size_t)c->N * c->N);
  c->t1.assign(T1, T1 + (size_t)o * v);
  c->l1.assign(L1, L1 + (size_t)o * v);
  c->T2p = T2p; c->L2p = L2p; c->L = Lchol;
  if (mode & 1) build_def(*c);
  if (mode & 2) build_dressed(*c);
  if ((mode & 4) && c->has_def) build_ea(*c);
  return c;
}
void orc_destroy(void* h) { delete (Ctx*)h; }

int orc_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// copy out an intermediate of the definition form (tests): returns element count or -1
i64 orc_get(void* h, const char* name, double* out) {
  Ctx& c = *(Ctx*)h;
  const std::vector<double>* src = nullptr;
  std::string n(name);
  if (n == "Fme") src = &c.Fme; else if (n == "Fmi") src = &c.Fmi; else if (n == "Fae") src = &c.Fae;
  else if (n == "Wmnij") src = &c.Wmnij; else if (n == "Wmnie") src = &c.Wmnie; else if (n == "Wmbej") src = &c.Wmbej;
  else if (n == "Wmbij") src = &c.Wmbij; else if (n == "oovv") src = &c.oovv; else if (n == "ft") src = &c.ft;
  else if (n == "Wamef") src = &c.Wamef; else if (n == "Wabef") src = &c.Wabef; else if (n == "Wabei") src = &c.Wabei;
  if (!src) return -1;
  if (out) std::memcpy(out, src->data(), src->size() * sizeof(double));
  return (i64)src->size();
}

// batched definition-form sigma. X1 [nrhs][o], X2 [nrhs][o][o][v] complex; omega[nrhs].
int orc_sigma(void* h, int nrhs, const double* omega, double eta, const cd* X1, const cd* X2, cd* S1, cd* S2) {
  Ctx& c = *(Ctx*)h;
  if (!c.has_def) return -1;
  const i64 n2 = (i64)c.o * c.o * c.v;
  for (int r = 0; r < nrhs; ++r) sigma_def_one(c, omega[r], eta, X1 + (i64)r * c.o, X2 + r * n2, S1 + (i64)r * c.o, S2 + r * n2);
  return 0;
}

// Right-hand side b_p (projections of abar_p|Phi>, Eq. 5):
//   p = k occupied: b1[i] = delta_ik, b2 = 0;   p = o+c virtual: b1[i] = t[i,c], b2[i,j,a] = t[i,j,c,a].
int orc_rhs(void* h, int p, cd* b1, cd* b2) {
  Ctx& c = *(Ctx*)h;
  const int o = c.o, v = c.v;
  if (p < 0 || p >= c.N) return -1;
  for (int i = 0; i < o; ++i) b1[i] = 0.0;
  for (i64 k = 0; k < (i64)o * o * v; ++k) b2[k] = 0.0;
  if (p < o) { b1[p] = 1.0; return 0; }
  const int cc = p - o;
  for (int i = 0; i < o; ++i) b1[i] = c.t1[(i64)i * v + cc];
  for (int i = 0; i < o; ++i)
    for (int j = 0; j < o; ++j)
      for (int a = 0; a < v; ++a) b2[((i64)i * o + j) * v + a] = t2p_at(c, i, j, cc, a);
  return 0;
}

// Bra vector c_q (<Phi|(1+Lambda) abar_q^+ ..., Eq. 7-8 first term), real.
//   q = k occ: c1[i] = delta_ki - sum_a t[k,a] l[i,a] - 1/2 sum_jab t[k,j,a,b] l[i,j,a,b]
//              c2[i,j,a] = delta_ki l[j,a] - delta_kj l[i,a] - sum_b t[k,b] l[i,j,b,a]
//   q = o+c  : c1[i] = l[i,c];  c2[i,j,a] = l[i,j,c,a]
// G_pq = sum_i c1[i] x1[i] + sum_{i<j,a} c2[i,j,a] x2[i,j,a].
int orc_bra(void* h, int q, double* c1, double* c2) {
  Ctx& c = *(Ctx*)h;
  const int o = c.o, v = c.v;
  if (q < 0 || q >= c.N) return -1;
  if (q < o) {
    const int k = q;
#pragma omp parallel for
    for (int i = 0; i < o; ++i) {
      double acc = (i == k) ? 1.0 : 0.0;
      for (int a = 0; a < v; ++a) acc -= c.t1[(i64)k * v + a] * c.l1[(i64)i * v + a];
      for (int j = 0; j < o; ++j)
        for (int a = 0; a < v; ++a)
          for (int b = 0; b < v; ++b) acc -= 0.5 * t2p_at(c, k, j, a, b) * l2p_at(c, i, j, a, b);
      c1[i] = acc;
    }
#pragma omp parallel for collapse(2)
    for (int i = 0; i < o; ++i)
      for (int j = 0; j < o; ++j)
        for (int a = 0; a < v; ++a) {
          double acc = 0.0;
          if (i == k) acc += c.l1[(i64)j * v + a];
          if (j == k) acc -= c.l1[(i64)i * v + a];
          for (int b = 0; b < v; ++b) acc -= c.t1[(i64)k * v + b] * l2p_at(c, i, j, b, a);
          c2[((i64)i * o + j) * v + a] = acc;
        }
  } else {
    const int cc = q - o;
    for (int i = 0; i < o; ++i) c1[i] = c.l1[(i64)i * v + cc];
    for (int i = 0; i < o; ++i)
      for (int j = 0; j < o; ++j)
        for (int a = 0; a < v; ++a) c2[((i64)i * o + j) * v + a] = l2p_at(c, i, j, cc, a);
  }
  return 0;
}

// G_pq = c_q . x in the packed (i<j) metric (reading 9 of DESIGN.md)
void orc_bra_dot(void* h, const double* c1, const double* c2, const cd* x1, const cd* x2, cd* out) {
  Ctx& c = *(Ctx*)h;
  const int o = c.o, v = c.v;
  cd acc = 0.0;
  for (int i = 0; i < o; ++i) acc += c1[i] * x1[i];
  for (int i = 0; i < o; ++i)
    for (int j = i + 1; j < o; ++j)
      for (int a = 0; a < v; ++a) acc += c2[((i64)i * o + j) * v + a] * x2[((i64)i * o + j) * v + a];
  *out = acc;
}

// ------------------------------------------------------------------------------------
// GMRES(m) for one right-hand side (Saad & Schultz 1986, PAPER.md ref. 85):
// modified Gram-Schmidt Arnoldi in the packed metric, complex Givens rotations, stop when the
// rotated residual |g_{j+1}| <= tol * ||b||.  x0kind 0: x0 = 0;  1: x0 = b / (omega - i eta + d),
// d_i = -f_ii, d_ija = f_aa - f_ii - f_jj (zeroth order; reading 11).
// Works on the packed vector z = (x1[i], x2[i<j,a]); sigma is applied through sigma_def_one.
// Returns the number of sigma applications; relres = final |g| / ||b||.
// hist (nullable, nhist entries): hist[k] = the residual estimate after sigma application k+1, i.e. ||b - A x|| / ||b|| for the
// application that starts a cycle and |g_{j+1}| / ||b|| for an Arnoldi step (an output only; the iteration does not read it).
// ------------------------------------------------------------------------------------
int orc_gmres_hist(void* h, int p, double omega, double eta, double tol, int m, int maxit, int x0kind, cd* x1out,
                   cd* x2out, double* relres, double* hist, int nhist) {
  Ctx& c = *(Ctx*)h;
  if (!c.has_def) return -1;
  const int o = c.o, v = c.v, N = c.N;
  const i64 n2 = (i64)o * o * v, np_ = c.npair * v, n = o + np_;
  auto pack = [&](const cd* a1, const cd* a2, std::vector<cd>& z) {
    z.resize(n);
    for (int i = 0; i < o; ++i) z[i] = a1[i];
    i64 k = o;
    for (int i = 0; i < o; ++i)
      for (int j = i + 1; j < o; ++j)
        for (int a = 0; a < v; ++a) z[k++] = a2[((i64)i * o + j) * v + a];
  };
  auto unpack = [&](const std::vector<cd>& z, cd* a1, cd* a2) {
    for (int i = 0; i < o; ++i) a1[i] = z[i];
    for (i64 k = 0; k < n2; ++k) a2[k] = 0.0;
    i64 k = o;
    for (int i = 0; i < o; ++i)
      for (int j = i + 1; j < o; ++j)
        for (int a = 0; a < v; ++a) {
          a2[((i64)i * o + j) * v + a] = z[k];
          a2[((i64)j * o + i) * v + a] = -z[k];
          ++k;
        }
  };
  std::vector<cd> t1b(o), t2b(n2), s1b(o), s2b(n2);
  auto apply = [&](const std::vector<cd>& z, std::vector<cd>& Az) {
    unpack(z, t1b.data(), t2b.data());
    sigma_def_one(c, omega, eta, t1b.data(), t2b.data(), s1b.data(), s2b.data());
    pack(s1b.data(), s2b.data(), Az);
  };
  std::vector<cd> b, x(n, 0.0);
  {
    std::vector<cd> b1(o), b2(n2);
    orc_rhs(h, p, b1.data(), b2.data());
    pack(b1.data(), b2.data(), b);
  }
  if (x0kind == 1) {
    const cd shift(omega, -eta);
    auto F = [&](int q) { return c.f[(i64)q * N + q]; };
    for (int i = 0; i < o; ++i) x[i] = b[i] / (shift - F(i));
    i64 k = o;
    for (int i = 0; i < o; ++i)
      for (int j = i + 1; j < o; ++j)
        for (int a = 0; a < v; ++a) { x[k] = b[k] / (shift + F(o + a) - F(i) - F(j)); ++k; }
  }
  double res = 1.0;
  const int napply = gmres_core(n, apply, b, x, tol, m, maxit, res, hist, nhist);
  unpack(x, x1out, x2out);
  *relres = res;
  return napply;
}

int orc_gmres(void* h, int p, double omega, double eta, double tol, int m, int maxit, int x0kind, cd* x1out,
              cd* x2out, double* relres) {
  return orc_gmres_hist(h, p, omega, eta, tol, m, maxit, x0kind, x1out, x2out, relres, nullptr, 0);
}

// ------------------------------------------------------------------------------------
// Row-sampled sigma for large sizes (SURVEY.md 8c "large configs"): exact sigma1[i] for the listed
// i and sigma2[i,j,a] at the listed triples, through L-factorised sums of the T1-dressed forms
// (8c item 8).  No o^2 v^2 array is formed.  X1 [nrhs][o], X2 [nrhs][o][o][v].
//   s1_idx [n1], S1out [n1][nrhs];  s2_idx [n2][3], S2out [n2][nrhs].
// ------------------------------------------------------------------------------------
int orc_sigma_rows(void* h, int nrhs, const double* omega, double eta, const cd* X1, const cd* X2, int n1,
                   const int* s1_idx, cd* S1out, int n2s, const int* s2_idx, cd* S2out) {
  Ctx& c = *(Ctx*)h;
  if (!c.has_dressed) return -1;
  const int o = c.o, v = c.v, Q = c.Q, N = c.N;
  const i64 nx2 = (i64)o * o * v;
  auto X2at = [&](int r, int i, int j, int a) { return X2[r * nx2 + ((i64)i * o + j) * v + a]; };
  auto Loo = [&](int m, int i) { return &c.Loo[((i64)m * o + i) * Q]; };
  auto Lov = [&](int m, int e) { return &c.Lov[((i64)m * v + e) * Q]; };
  auto Lvv = [&](int a, int e) { return &c.Lvv[((i64)a * v + e) * Q]; };
  auto Lvo = [&](int a, int i) { return &c.Lvo[((i64)a * o + i) * Q]; };
  auto FT = [&](int p, int q) { return c.ft[(i64)p * N + q]; };

  // Y[r][j][Q] = sum_me L[Q,m,e] x2[m,j,e]     (8a S1)
  std::vector<cd> Y((size_t)nrhs * o * Q);
#pragma omp parallel for collapse(2)
  for (int r = 0; r < nrhs; ++r)
    for (int j = 0; j < o; ++j) {
      cd* y = &Y[((i64)r * o + j) * Q];
      for (int k = 0; k < Q; ++k) y[k] = 0.0;
      for (int m = 0; m < o; ++m)
        for (int e = 0; e < v; ++e) {
          const cd x = X2at(r, m, j, e);
          const double* l = Lov(m, e);
          for (int k = 0; k < Q; ++k) y[k] += l[k] * x;
        }
    }
  // yv[r][e] = 1/2 sum_mnf <mn||ef> x2[m,n,f] = -sum_Q sum_m L[Q,m,e] Y[Q,m]   (8a S12)
  std::vector<cd> yv((size_t)nrhs * v);
#pragma omp parallel for collapse(2)
  for (int r = 0; r < nrhs; ++r)
    for (int e = 0; e < v; ++e) {
      cd acc = 0.0;
      for (int m = 0; m < o; ++m) {
        const double* l = Lov(m, e);
        const cd* y = &Y[((i64)r * o + m) * Q];
        for (int k = 0; k < Q; ++k) acc -= l[k] * y[k];
      }
      yv[(i64)r * v + e] = acc;
    }
  // M_i[e][Q] = sum_nf t[i,n,f,e] L[Q,n,f]  for one occupied i   (8a P3)
  auto build_Mi = [&](int i, std::vector<double>& Mi) {
    Mi.assign((size_t)v * Q, 0.0);
#pragma omp parallel for
    for (int e = 0; e < v; ++e) {
      double* mq = &Mi[(i64)e * Q];
      for (int n = 0; n < o; ++n)
        for (int g = 0; g < v; ++g) {
          const double t = t2p_at(c, i, n, g, e);
          if (t == 0.0) continue;
          const double* l = Lov(n, g);
          for (int k = 0; k < Q; ++k) mq[k] += t * l[k];
        }
    }
  };
  // column i of F_mi:  F_mi = ft_mi + 1/2 sum_nef <mn||ef> t[i,n,e,f] = ft_mi - sum_Q sum_e L[Q,m,e] M_i[Q,e]  (8a P4)
  auto Fmi_col = [&](int i, const std::vector<double>& Mi, std::vector<double>& col) {
    col.assign(o, 0.0);
    for (int m = 0; m < o; ++m) {
      double acc = FT(m, i);
      for (int e = 0; e < v; ++e) acc -= dotQ(Lov(m, e), &Mi[(i64)e * Q], Q);
      col[m] = acc;
    }
  };
  // row a of F_ae: F_ae = ft_ae - 1/2 sum_mnf t[m,n,a,f]<mn||ef> = ft_ae + sum_Q sum_m L[Q,m,e] Mq[m][Q], Mq[m] = sum_nf t[m,n,f,a] L[Q,n,f]
  auto Fae_row = [&](int a, std::vector<double>& row) {
    std::vector<double> Ma((size_t)o * Q, 0.0);
#pragma omp parallel for
    for (int m = 0; m < o; ++m) {
      double* mq = &Ma[(i64)m * Q];
      for (int n = 0; n < o; ++n)
        for (int g = 0; g < v; ++g) {
          const double t = t2p_at(c, m, n, g, a);
          if (t == 0.0) continue;
          const double* l = Lov(n, g);
          for (int k = 0; k < Q; ++k) mq[k] += t * l[k];
        }
    }
    row.assign(v, 0.0);
#pragma omp parallel for
    for (int e = 0; e < v; ++e) {
      double acc = FT(o + a, o + e);
      for (int m = 0; m < o; ++m) acc += dotQ(Lov(m, e), &Ma[(i64)m * Q], Q);
      row[e] = acc;
    }
  };

  // ---- sigma1 rows:  s1[i] = (w - i eta) x1[i] - sum_m F_mi x1[m] - sum_me F_me x2[m,i,e] + sum_Q sum_n Loo[Q,n,i] Y[Q,n]
  for (int s = 0; s < n1; ++s) {
    const int i = s1_idx[s];
    std::vector<double> Mi, col;
    build_Mi(i, Mi);
    Fmi_col(i, Mi, col);
#pragma omp parallel for
    for (int r = 0; r < nrhs; ++r) {
      cd acc = cd(omega[r], -eta) * X1[(i64)r * o + i];
      for (int m = 0; m < o; ++m) acc -= col[m] * X1[(i64)r * o + m];
      for (int m = 0; m < o; ++m)
        for (int e = 0; e < v; ++e) acc -= FT(m, o + e) * X2at(r, m, i, e);
      for (int n = 0; n < o; ++n) {
        const double* l = Loo(n, i);
        const cd* y = &Y[((i64)r * o + n) * Q];
        for (int k = 0; k < Q; ++k) acc += l[k] * y[k];
      }
      S1out[(i64)s * nrhs + r] = acc;
    }
  }

  // ---- sigma2 samples
  for (int s = 0; s < n2s; ++s) {
    const int i = s2_idx[3 * s], j = s2_idx[3 * s + 1], a = s2_idx[3 * s + 2];
    std::vector<double> Mi, Mj, Fi, Fj, Fa;
    build_Mi(i, Mi); build_Mi(j, Mj);
    Fmi_col(i, Mi, Fi); Fmi_col(j, Mj, Fj);
    Fae_row(a, Fa);
    // W_mnij[m,n] for this (i,j):  <mn||ij>~ + sum_ef t[i,j,e,f] <mn|ef>
    std::vector<double> U((size_t)o * v * Q, 0.0);   // U[m][f][Q] = sum_e L[Q,m,e] t[i,j,e,f]
#pragma omp parallel for collapse(2)
    for (int m = 0; m < o; ++m)
      for (int g = 0; g < v; ++g) {
        double* u = &U[((i64)m * v + g) * Q];
        for (int e = 0; e < v; ++e) {
          const double t = t2p_at(c, i, j, e, g);
          const double* l = Lov(m, e);
          for (int k = 0; k < Q; ++k) u[k] += t * l[k];
        }
      }
    std::vector<double> Wmn((size_t)o * o, 0.0);
#pragma omp parallel for collapse(2)
    for (int m = 0; m < o; ++m)
      for (int n = 0; n < o; ++n) {
        double acc = dotQ(Loo(m, i), Loo(n, j), Q) - dotQ(Loo(m, j), Loo(n, i), Q);
        for (int g = 0; g < v; ++g) acc += dotQ(&U[((i64)m * v + g) * Q], Lov(n, g), Q);
        Wmn[(i64)m * o + n] = acc;
      }
    // ring block W_mbej[m,b,e,jj] for fixed (b,jj), all (m,e):
    //   <mb||e jj>~ - sum_nf t[jj,n,f,b] <mn||ef>
    //   = sum_Q ( L[m,e] Lvo[b,jj] - Loo[m,jj] Lvv[b,e] ) - sum_Q L[Q,m,e] M_jj[Q,b] + sum_Q sum_n (sum_f t[jj,n,f,b] L[Q,m,f]) L[Q,n,e]
    auto ring_block = [&](int b, int jj, const std::vector<double>& Mjj, std::vector<double>& Wme) {
      std::vector<double> Bq((size_t)o * o * Q, 0.0);   // Bq[n][m][Q] = sum_f t[jj,n,f,b] L[Q,m,f]
#pragma omp parallel for collapse(2)
      for (int n = 0; n < o; ++n)
        for (int m = 0; m < o; ++m) {
          double* bq = &Bq[((i64)n * o + m) * Q];
          for (int g = 0; g < v; ++g) {
            const double t = t2p_at(c, jj, n, g, b);
            if (t == 0.0) continue;
            const double* l = Lov(m, g);
            for (int k = 0; k < Q; ++k) bq[k] += t * l[k];
          }
        }
      Wme.assign((size_t)o * v, 0.0);
#pragma omp parallel for collapse(2)
      for (int m = 0; m < o; ++m)
        for (int e = 0; e < v; ++e) {
          double acc = dotQ(Lov(m, e), Lvo(b, jj), Q) - dotQ(Loo(m, jj), Lvv(b, e), Q) - dotQ(Lov(m, e), &Mjj[(i64)b * Q], Q);
          for (int n = 0; n < o; ++n) acc += dotQ(&Bq[((i64)n * o + m) * Q], Lov(n, e), Q);
          Wme[(i64)m * v + e] = acc;
        }
    };
    std::vector<double> Rai, Raj;
    ring_block(a, i, Mi, Rai);
    ring_block(a, j, Mj, Raj);
    // W_mbij[m, b=a, I=j, J=i] for all m (dressed item 8):
    //  <mb||IJ>~ - sum_e ft_me t[I,J,b,e] + sum_ef <mb|ef>~ t[I,J,e,f] + P(IJ) sum_ne <mn||Ie>~ t[J,n,b,e]
    std::vector<double> Wm(o, 0.0);
    {
      const int I = j, J = i, b = a;
      std::vector<double> Cq((size_t)v * Q, 0.0);   // Cq[e][Q] = sum_f Lvv[Q,b,f] t[I,J,e,f]
#pragma omp parallel for
      for (int e = 0; e < v; ++e)
        for (int g = 0; g < v; ++g) {
          const double t = t2p_at(c, I, J, e, g);
          const double* l = Lvv(b, g);
          for (int k = 0; k < Q; ++k) Cq[(i64)e * Q + k] += t * l[k];
        }
      // for the P(IJ) term:  sum_ne (Loo[m,I] L[n,e] - L[m,e] Loo[n,I]) t[J,n,b,e]
      auto pterm = [&](int I_, int J_, std::vector<double>& out) {
        std::vector<double> sQ(Q, 0.0);              // sum_ne L[Q,n,e] t[J,n,b,e]
        std::vector<double> Dq((size_t)v * Q, 0.0);  // Dq[e][Q] = sum_n Loo[Q,n,I] t[J,n,b,e]
        for (int n = 0; n < o; ++n)
          for (int e = 0; e < v; ++e) {
            const double t = t2p_at(c, J_, n, b, e);
            if (t == 0.0) continue;
            const double *l = Lov(n, e), *lo = Loo(n, I_);
            for (int k = 0; k < Q; ++k) { sQ[k] += t * l[k]; Dq[(i64)e * Q + k] += t * lo[k]; }
          }
        out.assign(o, 0.0);
        for (int m = 0; m < o; ++m) {
          double acc = dotQ(Loo(m, I_), sQ.data(), Q);
          for (int e = 0; e < v; ++e) acc -= dotQ(Lov(m, e), &Dq[(i64)e * Q], Q);
          out[m] = acc;
        }
      };
      std::vector<double> pIJ, pJI;
      pterm(I, J, pIJ); pterm(J, I, pJI);
      for (int m = 0; m < o; ++m) {
        double acc = dotQ(Loo(m, I), Lvo(b, J), Q) - dotQ(Loo(m, J), Lvo(b, I), Q);
        for (int e = 0; e < v; ++e) acc -= FT(m, o + e) * t2p_at(c, I, J, b, e);
        for (int e = 0; e < v; ++e) acc += dotQ(Lov(m, e), &Cq[(i64)e * Q], Q);
        acc += pIJ[m] - pJI[m];
        Wm[m] = acc;
      }
    }
#pragma omp parallel for
    for (int r = 0; r < nrhs; ++r) {
      cd acc = cd(omega[r], -eta) * X2at(r, i, j, a);
      for (int e = 0; e < v; ++e) acc += Fa[e] * X2at(r, i, j, e);
      for (int m = 0; m < o; ++m) acc -= Fi[m] * X2at(r, m, j, a) - Fj[m] * X2at(r, m, i, a);
      for (int m = 0; m < o; ++m) acc += Wm[m] * X1[(i64)r * o + m];
      for (int m = 0; m < o; ++m)
        for (int n = 0; n < o; ++n) acc += 0.5 * Wmn[(i64)m * o + n] * X2at(r, m, n, a);
      for (int m = 0; m < o; ++m)
        for (int e = 0; e < v; ++e) acc += Rai[(i64)m * v + e] * X2at(r, m, j, e) - Raj[(i64)m * v + e] * X2at(r, m, i, e);
      for (int e = 0; e < v; ++e) acc += t2p_at(c, i, j, a, e) * yv[(i64)r * v + e];
      S2out[(i64)s * nrhs + r] = acc;
    }
  }
  return 0;
}

// ------------------------------------------------------------------------------------
// EA / advanced part: C entry points (Eq. 6; second terms of Eq. 7-8).
// Y1 [nrhs][v], Y2 [nrhs][o][v][v] (index order j, a, b; antisymmetric in a,b), complex interleaved.
// ------------------------------------------------------------------------------------
int orc_sigma_ea(void* h, int nrhs, const double* omega, double eta, const cd* Y1, const cd* Y2, cd* S1, cd* S2) {
  Ctx& c = *(Ctx*)h;
  if (!c.has_ea) return -1;
  const i64 n2 = (i64)c.o * c.v * c.v;
  for (int r = 0; r < nrhs; ++r) sigma_ea_one(c, omega[r], eta, Y1 + (i64)r * c.v, Y2 + r * n2, S1 + (i64)r * c.v, S2 + r * n2);
  return 0;
}

// Right-hand side of Eq. 6: projections of abar_q^+ |Phi> on the 1p and 2p1h determinants.
//   q = o+c virtual: b1[a] = delta_ac, b2 = 0;   q = k occupied: b1[a] = -t[k,a], b2[j,a,b] = -t[k,j,a,b].
int orc_rhs_ea(void* h, int q, cd* b1, cd* b2) {
  Ctx& c = *(Ctx*)h;
  const int o = c.o, v = c.v;
  if (q < 0 || q >= c.N) return -1;
  for (int a = 0; a < v; ++a) b1[a] = 0.0;
  for (i64 k = 0; k < (i64)o * v * v; ++k) b2[k] = 0.0;
  if (q >= o) { b1[q - o] = 1.0; return 0; }
  for (int a = 0; a < v; ++a) b1[a] = -c.t1[(i64)q * v + a];
  for (int j = 0; j < o; ++j)
    for (int a = 0; a < v; ++a)
      for (int b = 0; b < v; ++b) b2[((i64)j * v + a) * v + b] = -t2p_at(c, q, j, a, b);
  return 0;
}

// Bra vector of the second term of Eq. 7-8: c_p[nu] = <Phi|(1 + Lambda1 + Lambda2) abar_p tau_nu|Phi>, real.
//   p = k occupied : c1[a] = -l[k,a];  c2[j,a,b] = -l[k,j,a,b]
//   p = o+e virtual: c1[a] = delta_ea - sum_i l[i,a] t[i,e] - 1/2 sum_ijb l[i,j,a,b] t[i,j,e,b]
//                    c2[j,a,b] = delta_ea l[j,b] - delta_eb l[j,a] - sum_i t[i,e] l[i,j,a,b]
// G^A_pq = sum_a c1[a] y1[a] + sum_{j, a<b} c2[j,a,b] y2[j,a,b].
int orc_bra_ea(void* h, int p, double* c1, double* c2) {
  Ctx& c = *(Ctx*)h;
  const int o = c.o, v = c.v;
  if (p < 0 || p >= c.N) return -1;
  if (p < o) {
    for (int a = 0; a < v; ++a) c1[a] = -c.l1[(i64)p * v + a];
    for (int j = 0; j < o; ++j)
      for (int a = 0; a < v; ++a)
        for (int b = 0; b < v; ++b) c2[((i64)j * v + a) * v + b] = -l2p_at(c, p, j, a, b);
    return 0;
  }
  const int e = p - o;
#pragma omp parallel for
  for (int a = 0; a < v; ++a) {
    double acc = (a == e) ? 1.0 : 0.0;
    for (int i = 0; i < o; ++i) acc -= c.l1[(i64)i * v + a] * c.t1[(i64)i * v + e];
    for (int i = 0; i < o; ++i)
      for (int j = 0; j < o; ++j)
        for (int b = 0; b < v; ++b) acc -= 0.5 * l2p_at(c, i, j, a, b) * t2p_at(c, i, j, e, b);
    c1[a] = acc;
  }
#pragma omp parallel for collapse(2)
  for (int j = 0; j < o; ++j)
    for (int a = 0; a < v; ++a)
      for (int b = 0; b < v; ++b) {
        double acc = 0.0;
        if (a == e) acc += c.l1[(i64)j * v + b];
        if (b == e) acc -= c.l1[(i64)j * v + a];
        for (int i = 0; i < o; ++i) acc -= c.t1[(i64)i * v + e] * l2p_at(c, i, j, a, b);
        c2[((i64)j * v + a) * v + b] = acc;
      }
  return 0;
}

void orc_bra_dot_ea(void* h, const double* c1, const double* c2, const cd* y1, const cd* y2, cd* out) {
  Ctx& c = *(Ctx*)h;
  const int o = c.o, v = c.v;
  cd acc = 0.0;
  for (int a = 0; a < v; ++a) acc += c1[a] * y1[a];
  for (int j = 0; j < o; ++j)
    for (int a = 0; a < v; ++a)
      for (int b = a + 1; b < v; ++b) acc += c2[((i64)j * v + a) * v + b] * y2[((i64)j * v + a) * v + b];
  *out = acc;
}

// GMRES(m) for Eq. 6 with target q, packed vector z = (y1[a], y2[j, a<b]) (j slowest).
// x0kind 1: y0 = b / (omega + i eta - d), d_a = f_aa, d_jab = f_aa + f_bb - f_jj (zeroth order of Hbar on 1p / 2p1h).
int orc_gmres_ea(void* h, int q, double omega, double eta, double tol, int m, int maxit, int x0kind, cd* y1out, cd* y2out,
                 double* relres, double* hist, int nhist) {
  Ctx& c = *(Ctx*)h;
  if (!c.has_ea) return -1;
  const int o = c.o, v = c.v, N = c.N;
  const i64 n2 = (i64)o * v * v, n = v + (i64)o * c.ntri;
  auto pack = [&](const cd* a1, const cd* a2, std::vector<cd>& z) {
    z.resize(n);
    for (int a = 0; a < v; ++a) z[a] = a1[a];
    i64 k = v;
    for (int j = 0; j < o; ++j)
      for (int a = 0; a < v; ++a)
        for (int b = a + 1; b < v; ++b) z[k++] = a2[((i64)j * v + a) * v + b];
  };
  auto unpack = [&](const std::vector<cd>& z, cd* a1, cd* a2) {
    for (int a = 0; a < v; ++a) a1[a] = z[a];
    for (i64 k = 0; k < n2; ++k) a2[k] = 0.0;
    i64 k = v;
    for (int j = 0; j < o; ++j)
      for (int a = 0; a < v; ++a)
        for (int b = a + 1; b < v; ++b) {
          a2[((i64)j * v + a) * v + b] = z[k];
          a2[((i64)j * v + b) * v + a] = -z[k];
          ++k;
        }
  };
  std::vector<cd> t1b(v), t2b(n2), s1b(v), s2b(n2);
  auto apply = [&](const std::vector<cd>& z, std::vector<cd>& Az) {
    unpack(z, t1b.data(), t2b.data());
    sigma_ea_one(c, omega, eta, t1b.data(), t2b.data(), s1b.data(), s2b.data());
    pack(s1b.data(), s2b.data(), Az);
  };
  std::vector<cd> b, x(n, 0.0);
  {
    std::vector<cd> b1(v), b2(n2);
    orc_rhs_ea(h, q, b1.data(), b2.data());
    pack(b1.data(), b2.data(), b);
  }
  if (x0kind == 1) {
    const cd shift(omega, eta);
    auto F = [&](int r) { return c.f[(i64)r * N + r]; };
    for (int a = 0; a < v; ++a) x[a] = b[a] / (shift - F(o + a));
    i64 k = v;
    for (int j = 0; j < o; ++j)
      for (int a = 0; a < v; ++a)
        for (int bb = a + 1; bb < v; ++bb) { x[k] = b[k] / (shift - F(o + a) - F(o + bb) + F(j)); ++k; }
  }
  double res = 1.0;
  const int napply = gmres_core(n, apply, b, x, tol, m, maxit, res, hist, nhist);
  unpack(x, y1out, y2out);
  *relres = res;
  return napply;
}

}  // extern "C"
