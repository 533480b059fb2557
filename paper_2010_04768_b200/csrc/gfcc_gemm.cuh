// =====================================================================================
// gfcc_gemm.cuh -- the FP64 tensor-core GEMM engine (sm_100a).
//
// Every large contraction of the GFCCSD-IP sigma build (SURVEY.md 8a S1,S6-S11; Eq. 11)
// is a REAL FP64 GEMM (Hbar is real, X complex: the RHS batch is folded into N as 2*nrhs real columns;
// PAPER.md:155 "complex-real mixed operations").  tcgen05 has no f64 kind, so the tensor path on
// sm_100a is DMMA: mma.sync.aligned.m8n8k4.f64 (SASS DMMA.8x8x4; the m16n8k{4,8,16} PTX shapes are
// split into 8x8x4 by ptxas on this target).  Measured issue-rate ceiling on B200: 36.95 TFLOP/s.
//
// Kernel: CTA tile BM x 128 x 16 with BM = WGM*8*WMF (WMF = m8 fragments per warp, chosen per problem
// to avoid ragged-M waste), WGM x 4 warps (default WGM = 2: 8 warps, warp tile up to 64 x 32), accumulators in
// registers, fragments double-buffered in registers across k4 steps and across tiles, 4-stage cp.async
// (LDGSTS) shared-memory pipeline with padded, bank-conflict-free tiles.
//
// Operand addressing (element strides, FP64):
//   A(m, k1, k0) = A + offA(k1) + m*sAm + k0*sAk0      B(k1, k0, n) = B + offB(k1) + k0*sBk0 + n*sBn
//   offX(k1) = tabX ? tabX[k1] : k1*sXk1.   K = K1 blocks of length K0 (each zero-padded to BK tiles).
//   Optional sgn[k1] in {+1,-1,0}: the block's contribution is multiplied by it (0 = skipped).
//   Exactly one of (sAm, sAk0) and one of (sBk0, sBn) is 1 (template flags A_KC / B_NC).
//   C(m, n) = C + (m/Md)*sCm1 + (m%Md)*sCm0 + (n/Nd)*sCn1 + (n%Nd)*sCn0   (two-level output scatter)
//   batch index z: A += z*bsA (tabA/sgn += z*K1), B += z*bsB, C += z*bsC.
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

namespace gfcc {

struct GemmParams {
  int M, N, K1, K0;
  const double* A; long long sAm, sAk0, sAk1; const long long* tabA;
  const double* B; long long sBn, sBk0, sBk1; const long long* tabB;
  const double* sgn;
  double* C; long long sCm0, sCm1; int Md; long long sCn0, sCn1; int Nd;
  double alpha, beta;
  int batch; long long bsA, bsB, bsC; int tab_batch_stride;   // tabA/tabB/sgn advance by this per batch
  int tiles_m, tiles_n, group_m;
  int vecA, vecB;   // 1: 16-byte cp.async legal for this operand (alignment checked on the host)
};

constexpr int GEMM_BN = 128;
constexpr int GEMM_BK = 16;
constexpr int GEMM_STAGES = 4;
constexpr int GEMM_PAD = 4;   // doubles; makes every fragment load bank-conflict free (ld % 16 == 4)

template <int WGM, int WMF> struct GemmTile {
  static constexpr int THREADS = WGM * 4 * 32;
  static constexpr int BM = WGM * 8 * WMF;
  static constexpr int LDK = GEMM_BK + GEMM_PAD;             // K-contiguous tiles: [rows][LDK]
  static constexpr int LDA_M = BM + GEMM_PAD;                // M-contiguous A tile: [BK][LDA_M]
  static constexpr int LDB_N = GEMM_BN + GEMM_PAD;           // N-contiguous B tile: [BK][LDB_N]
  static constexpr int A_ELEMS = (BM * LDK > GEMM_BK * LDA_M) ? BM * LDK : GEMM_BK * LDA_M;
  static constexpr int B_ELEMS = (GEMM_BN * LDK > GEMM_BK * LDB_N) ? GEMM_BN * LDK : GEMM_BK * LDB_N;
  static constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
  static constexpr size_t SMEM_BYTES = (size_t)GEMM_STAGES * STAGE_ELEMS * sizeof(double);
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// copy one 2-double chunk (contiguous in global memory) into shared memory with zero fill.
// nvalid in {0,1,2}: number of in-range elements of the chunk.
// `safe` is any valid address of the operand (used when the chunk is entirely out of range: src-size 0).
__device__ __forceinline__ void load_chunk(double* sdst, const double* gsrc, int nvalid, int vec, const double* safe) {
  if (vec) {
    cp_async16(sdst, nvalid > 0 ? gsrc : safe, nvalid > 0 ? nvalid * 8 : 0);
  } else {
    cp_async8(sdst, nvalid > 0 ? gsrc : safe, nvalid > 0 ? 8 : 0);
    cp_async8(sdst + 1, nvalid > 1 ? gsrc + 1 : safe, nvalid > 1 ? 8 : 0);
  }
}

__device__ __forceinline__ double flip_sign(double x, unsigned mask) {
  return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));   // integer pipe, not the FP64 pipe
}

template <int WGM, int WMF, bool A_KC, bool B_NC, bool HAS_SIGN>
__global__ void __launch_bounds__(WGM * 128, 1) dgemm_dmma_kernel(const GemmParams p) {
  using T = GemmTile<WGM, WMF>;
  constexpr int BM = T::BM, BN = GEMM_BN, BK = GEMM_BK, GEMM_THREADS = T::THREADS;
  extern __shared__ __align__(16) double smem[];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 2, wn = warp & 3;   // 2 x 4 warps
  const int z = blockIdx.z;

  // ---- tile rasterisation: groups of group_m M-tiles, M fastest inside a group (L2 reuse of B panels)
  int tm, tn;
  {
    const int t = blockIdx.x;
    const int per_group = p.group_m * p.tiles_n;
    const int g = t / per_group;
    const int first = g * p.group_m;
    const int gsz = min(p.group_m, p.tiles_m - first);
    const int r = t - g * per_group;
    tm = first + r % gsz;
    tn = r / gsz;
  }
  const int m0 = tm * BM, n0 = tn * BN;

  const double* __restrict__ Ab = p.A + (long long)z * p.bsA;
  const double* __restrict__ Bb = p.B + (long long)z * p.bsB;
  const long long* tabA = p.tabA ? p.tabA + (long long)z * p.tab_batch_stride : nullptr;
  const long long* tabB = p.tabB ? p.tabB + (long long)z * p.tab_batch_stride : nullptr;
  const double* sgn = HAS_SIGN ? p.sgn + (long long)z * p.tab_batch_stride : nullptr;

  const int KT0 = (p.K0 + BK - 1) / BK;
  int nblocks = 0;   // number of non-skipped k1 blocks
  if (HAS_SIGN) { for (int k1 = 0; k1 < p.K1; ++k1) nblocks += (sgn[k1] != 0.0) ? 1 : 0; }
  else nblocks = p.K1;
  const int total = nblocks * KT0;

  // ---- loader state: (k1, kt) of the next tile to fetch
  int ld_k1 = 0, ld_kt = 0, ld_count = 0;
  auto skip_zero = [&](int& k1) { if (HAS_SIGN) { while (k1 < p.K1 && sgn[k1] == 0.0) ++k1; } };
  skip_zero(ld_k1);

  auto issue_load = [&](int stage) {
    double* As = smem + (size_t)stage * T::STAGE_ELEMS;
    double* Bs = As + T::A_ELEMS;
    const long long offA = tabA ? tabA[ld_k1] : (long long)ld_k1 * p.sAk1;
    const long long offB = tabB ? tabB[ld_k1] : (long long)ld_k1 * p.sBk1;
    const int k0 = ld_kt * BK;
    if (A_KC) {   // As[BM][LDK], chunks along k
      constexpr int CPR = BK / 2;
#pragma unroll
      for (int c = tid; c < BM * CPR; c += GEMM_THREADS) {
        const int row = c / CPR, kc = (c % CPR) * 2;
        const int gm = m0 + row, gk = k0 + kc;
        int nv = (gm < p.M) ? min(2, max(0, p.K0 - gk)) : 0;
        load_chunk(As + row * T::LDK + kc, Ab + offA + (long long)gm * p.sAm + gk, nv, p.vecA, p.A);
      }
    } else {      // As[BK][LDA_M], chunks along m
      constexpr int CPR = BM / 2;
#pragma unroll
      for (int c = tid; c < BK * CPR; c += GEMM_THREADS) {
        const int kr = c / CPR, mc = (c % CPR) * 2;
        const int gm = m0 + mc, gk = k0 + kr;
        int nv = (gk < p.K0) ? min(2, max(0, p.M - gm)) : 0;
        load_chunk(As + kr * T::LDA_M + mc, Ab + offA + (long long)gk * p.sAk0 + gm, nv, p.vecA, p.A);
      }
    }
    if (B_NC) {   // Bs[BK][LDB_N], chunks along n
      constexpr int CPR = BN / 2;
#pragma unroll
      for (int c = tid; c < BK * CPR; c += GEMM_THREADS) {
        const int kr = c / CPR, nc = (c % CPR) * 2;
        const int gn = n0 + nc, gk = k0 + kr;
        int nv = (gk < p.K0) ? min(2, max(0, p.N - gn)) : 0;
        load_chunk(Bs + kr * T::LDB_N + nc, Bb + offB + (long long)gk * p.sBk0 + gn, nv, p.vecB, p.B);
      }
    } else {      // Bs[BN][LDK], chunks along k
      constexpr int CPR = BK / 2;
#pragma unroll
      for (int c = tid; c < BN * CPR; c += GEMM_THREADS) {
        const int col = c / CPR, kc = (c % CPR) * 2;
        const int gn = n0 + col, gk = k0 + kc;
        int nv = (gn < p.N) ? min(2, max(0, p.K0 - gk)) : 0;
        load_chunk(Bs + col * T::LDK + kc, Bb + offB + (long long)gn * p.sBn + gk, nv, p.vecB, p.B);
      }
    }
    // advance loader
    ++ld_count;
    if (++ld_kt == KT0) { ld_kt = 0; ++ld_k1; skip_zero(ld_k1); }
  };

  double acc[WMF][4][2];
#pragma unroll
  for (int f = 0; f < WMF; ++f)
#pragma unroll
    for (int g = 0; g < 4; ++g) acc[f][g][0] = acc[f][g][1] = 0.0;

  // ---- prologue
#pragma unroll
  for (int s = 0; s < GEMM_STAGES - 1; ++s) {
    if (ld_count < total) issue_load(s);
    cp_async_commit();
  }

  // compute-side block tracking (for the sign)
  int c_k1 = 0, c_kt = 0;
  skip_zero(c_k1);

  const int arow = wm * (8 * WMF) + (lane >> 2);   // + 8 f
  const int bcol = wn * 32 + (lane >> 2);          // + 8 g
  const int kl = lane & 3;

  // register double buffer of fragments: the fragments of k4-step kk+1 (or of step 0 of the NEXT tile) are
  // loaded while the DMMAs of step kk issue, so that neither LDS latency nor the per-tile barrier leaves the
  // DMMA pipe idle.  Requires tiles `it` and `it+1` to be resident at the top of iteration `it`.
  double fa[2][WMF], fb[2][4];
  auto load_frags = [&](int buf, int stage, int kk, unsigned smask) {
    const double* As = smem + (size_t)stage * T::STAGE_ELEMS;
    const double* Bs = As + T::A_ELEMS;
    const int k = kk * 4 + kl;
#pragma unroll
    for (int f = 0; f < WMF; ++f)
      fa[buf][f] = A_KC ? As[(arow + 8 * f) * T::LDK + k] : As[k * T::LDA_M + arow + 8 * f];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const double bv = B_NC ? Bs[k * T::LDB_N + bcol + 8 * g] : Bs[(bcol + 8 * g) * T::LDK + k];
      fb[buf][g] = HAS_SIGN ? flip_sign(bv, smask) : bv;
    }
  };
  auto mask_of = [&](int k1) -> unsigned { return (HAS_SIGN && k1 < p.K1 && sgn[k1] < 0.0) ? 0x80000000u : 0u; };

  cp_async_wait<GEMM_STAGES - 3>();
  __syncthreads();
  if (total > 0) load_frags(0, 0, 0, mask_of(c_k1));

  for (int it = 0; it < total; ++it) {
    if (it > 0) {
      cp_async_wait<GEMM_STAGES - 3>();   // tiles it and it+1 have landed
      __syncthreads();                    // ... for every thread; and everyone is done with tile it-1
    }
    {   // prefetch tile it + STAGES - 1 into the stage consumed in iteration it-1
      if (ld_count < total) issue_load((it + GEMM_STAGES - 1) % GEMM_STAGES);
      cp_async_commit();
    }
    // (k1, kt) of the next tile, for the sign of the prefetched fragments
    int n_k1 = c_k1, n_kt = c_kt + 1;
    if (n_kt == KT0) { n_kt = 0; ++n_k1; skip_zero(n_k1); }
    const unsigned cur_mask = mask_of(c_k1), nxt_mask = mask_of(n_k1);
    const int stage = it % GEMM_STAGES;
#pragma unroll
    for (int kk = 0; kk < BK / 4; ++kk) {
      const int cur = kk & 1, nxt = cur ^ 1;
      if (kk + 1 < BK / 4) load_frags(nxt, stage, kk + 1, cur_mask);
      else if (it + 1 < total) load_frags(nxt, (it + 1) % GEMM_STAGES, 0, nxt_mask);
#pragma unroll
      for (int f = 0; f < WMF; ++f)
#pragma unroll
        for (int g = 0; g < 4; ++g) dmma884(acc[f][g][0], acc[f][g][1], fa[cur][f], fb[cur][g]);
    }
    c_k1 = n_k1; c_kt = n_kt;
  }
  cp_async_wait<0>();

  // ---- epilogue: C = alpha*acc + beta*C with two-level scatter
  double* __restrict__ Cb = p.C + (long long)z * p.bsC;
  long long coff[4][2];
  bool cok[4][2];
#pragma unroll
  for (int g = 0; g < 4; ++g)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int n = n0 + wn * 32 + 8 * g + 2 * kl + e;
      cok[g][e] = n < p.N;
      coff[g][e] = (long long)(n / p.Nd) * p.sCn1 + (long long)(n % p.Nd) * p.sCn0;
    }
#pragma unroll
  for (int f = 0; f < WMF; ++f) {
    const int m = m0 + arow + 8 * f;
    if (m >= p.M) continue;
    const long long roff = (long long)(m / p.Md) * p.sCm1 + (long long)(m % p.Md) * p.sCm0;
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      if (cok[g][0] && cok[g][1] && coff[g][1] == coff[g][0] + 1 && (((roff + coff[g][0]) & 1) == 0) &&
          ((reinterpret_cast<uintptr_t>(Cb) & 15) == 0)) {
        double2* ptr = reinterpret_cast<double2*>(Cb + roff + coff[g][0]);
        double2 o;
        if (p.beta != 0.0) {
          double2 old = *ptr;
          o.x = p.alpha * acc[f][g][0] + p.beta * old.x;
          o.y = p.alpha * acc[f][g][1] + p.beta * old.y;
        } else {
          o.x = p.alpha * acc[f][g][0];
          o.y = p.alpha * acc[f][g][1];
        }
        *ptr = o;
      } else {
#pragma unroll
        for (int e = 0; e < 2; ++e)
          if (cok[g][e]) {
            double* ptr = Cb + roff + coff[g][e];
            double val = p.alpha * acc[f][g][e];
            if (p.beta != 0.0) val += p.beta * *ptr;
            *ptr = val;
          }
      }
    }
  }
}

// ---- host side -------------------------------------------------------------------------
struct GemmDesc {
  int M = 0, N = 0, K1 = 1, K0 = 0;
  const double* A = nullptr; long long sAm = 0, sAk0 = 0, sAk1 = 0; const long long* tabA = nullptr;
  const double* B = nullptr; long long sBn = 0, sBk0 = 0, sBk1 = 0; const long long* tabB = nullptr;
  const double* sgn = nullptr;
  double* C = nullptr; long long sCm0 = 0, sCm1 = 0; int Md = 0; long long sCn0 = 1, sCn1 = 0; int Nd = 0;
  double alpha = 1.0, beta = 0.0;
  int batch = 1; long long bsA = 0, bsB = 0, bsC = 0; int tab_batch_stride = 0;
  bool tabs_even = true;   // caller's promise that every table offset is even (16-byte alignment)
};

// warp-grid rows: 2 (8 warps per CTA, WMF in 4..8; measured 31.0 TFLOP/s on 8192^3) by default;
// GFCC_GEMM_WGM=4 selects the 16-warp variant (WMF 2..4; measured 28.9 TFLOP/s) for experiments.
inline int gemm_wgm() {
  static int w = -1;
  if (w < 0) { const char* e = getenv("GFCC_GEMM_WGM"); w = (e && e[0] == '4') ? 4 : 2; }
  return w;
}
// choose the m8-fragment count per warp (BM = WGM*8*WMF): the kernel runs one CTA per SM, so the launch takes
// ceil(tiles / 148) waves of time ~ BM each; pick the BM with the smallest waves*BM (this covers both ragged-M padding
// and the partially filled last wave), with a mild penalty for small tiles (more shared-memory traffic per flop).
constexpr int GEMM_NUM_SMS = 148;
inline int pick_wmf(int M, long long N = 0, int batch = 1, int wgm = gemm_wgm()) {
  const int hi = (wgm == 4) ? 4 : 8, lo = (wgm == 4) ? 2 : 4;
  const long long tiles_n = (N > 0) ? (N + GEMM_BN - 1) / GEMM_BN : 0;
  int best = hi; double bestcost = -1;
  for (int w = hi; w >= lo; --w) {
    const int bm = wgm * 8 * w;
    const long long tiles_m = (M + bm - 1) / bm;
    double cost;
    if (tiles_n > 0) {
      const long long tiles = tiles_m * tiles_n * (batch > 0 ? batch : 1);
      const long long waves = (tiles + GEMM_NUM_SMS - 1) / GEMM_NUM_SMS;
      cost = (double)waves * bm;
    } else {
      cost = (double)tiles_m * bm;   // N unknown: padded rows only
    }
    cost *= 1.0 + 0.01 * (hi - w);
    if (bestcost < 0 || cost < bestcost) { bestcost = cost; best = w; }
  }
  return best;
}
inline int gemm_bm(int M, long long N = 0, int batch = 1) { return gemm_wgm() * 8 * pick_wmf(M, N, batch); }

// engine selection: the warp-specialised kernel (gfcc_gemm_ws.cuh; 34.4 TFLOP/s on 8192^3 = 93 % of the DMMA ceiling,
// GPU parity suite green) is the default; GFCC_GEMM_ENGINE=v1 selects the single-role kernel of this file
// (31.0 TFLOP/s) for comparison.  The WGM=4 experiment implies v1.
inline bool gemm_use_ws() {
  static int w = -1;
  if (w < 0) { const char* e = getenv("GFCC_GEMM_ENGINE"); w = (e && e[0] == 'v' && e[1] == '1') ? 0 : 1; }
  return w == 1 && gemm_wgm() == 2;
}
cudaError_t launch_dgemm_ws(const GemmParams& p, bool a_kc, bool b_nc, bool sign, int wmf, cudaStream_t st);

template <int WGM, int WMF, bool A_KC, bool B_NC, bool HAS_SIGN>
inline cudaError_t launch_dgemm_t(const GemmParams& p, cudaStream_t st) {
  using T = GemmTile<WGM, WMF>;
  auto kern = dgemm_dmma_kernel<WGM, WMF, A_KC, B_NC, HAS_SIGN>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((unsigned)(p.tiles_m * p.tiles_n), 1, (unsigned)p.batch);
  kern<<<grid, T::THREADS, T::SMEM_BYTES, st>>>(p);
  return cudaGetLastError();
}

template <bool A_KC, bool B_NC, bool HAS_SIGN>
inline cudaError_t launch_dgemm_w(int wgm, int wmf, const GemmParams& p, cudaStream_t st) {
  if (wgm == 4) {
    switch (wmf) {
      case 4: return launch_dgemm_t<4, 4, A_KC, B_NC, HAS_SIGN>(p, st);
      case 3: return launch_dgemm_t<4, 3, A_KC, B_NC, HAS_SIGN>(p, st);
      default: return launch_dgemm_t<4, 2, A_KC, B_NC, HAS_SIGN>(p, st);
    }
  }
  switch (wmf) {
    case 8: return launch_dgemm_t<2, 8, A_KC, B_NC, HAS_SIGN>(p, st);
    case 7: return launch_dgemm_t<2, 7, A_KC, B_NC, HAS_SIGN>(p, st);
    case 6: return launch_dgemm_t<2, 6, A_KC, B_NC, HAS_SIGN>(p, st);
    case 5: return launch_dgemm_t<2, 5, A_KC, B_NC, HAS_SIGN>(p, st);
    default: return launch_dgemm_t<2, 4, A_KC, B_NC, HAS_SIGN>(p, st);
  }
}
template <bool A_KC, bool B_NC>
inline cudaError_t launch_dgemm_s(bool sign, int wgm, int wmf, const GemmParams& p, cudaStream_t st) {
  return sign ? launch_dgemm_w<A_KC, B_NC, true>(wgm, wmf, p, st) : launch_dgemm_w<A_KC, B_NC, false>(wgm, wmf, p, st);
}

inline cudaError_t launch_dgemm(const GemmDesc& d, cudaStream_t st) {
  if (d.M <= 0 || d.N <= 0 || d.K0 <= 0 || d.K1 <= 0 || d.batch <= 0) return cudaSuccess;   // empty: nothing to do
  const bool a_kc = (d.sAk0 == 1);
  const bool b_nc = (d.sBn == 1);
  if (!a_kc && d.sAm != 1) return cudaErrorInvalidValue;
  if (!b_nc && d.sBk0 != 1) return cudaErrorInvalidValue;
  GemmParams p;
  p.M = d.M; p.N = d.N; p.K1 = d.K1; p.K0 = d.K0;
  p.A = d.A; p.sAm = d.sAm; p.sAk0 = d.sAk0; p.sAk1 = d.sAk1; p.tabA = d.tabA;
  p.B = d.B; p.sBn = d.sBn; p.sBk0 = d.sBk0; p.sBk1 = d.sBk1; p.tabB = d.tabB;
  p.sgn = d.sgn;
  p.C = d.C; p.sCm0 = d.sCm0; p.sCm1 = d.sCm1; p.Md = d.Md > 0 ? d.Md : (d.M > 0 ? d.M : 1);
  p.sCn0 = d.sCn0; p.sCn1 = d.sCn1; p.Nd = d.Nd > 0 ? d.Nd : (d.N > 0 ? d.N : 1);
  p.alpha = d.alpha; p.beta = d.beta;
  p.batch = d.batch; p.bsA = d.bsA; p.bsB = d.bsB; p.bsC = d.bsC; p.tab_batch_stride = d.tab_batch_stride;
  const int wgm = gemm_wgm();
  const int wmf = pick_wmf(d.M, d.N, d.batch, wgm);
  const int bm = wgm * 8 * wmf;
  p.tiles_m = (d.M + bm - 1) / bm;
  p.tiles_n = (d.N + GEMM_BN - 1) / GEMM_BN;
  p.group_m = 8;
  auto even = [](long long x) { return (x & 1LL) == 0; };
  auto al16 = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; };
  // 16-byte cp.async needs: aligned base, even strides along every non-contiguous direction, even offsets
  p.vecA = al16(d.A) && even(a_kc ? d.sAm : d.sAk0) && even(d.bsA) && (d.tabA ? d.tabs_even : even(d.sAk1));
  p.vecB = al16(d.B) && even(b_nc ? d.sBk0 : d.sBn) && even(d.bsB) && (d.tabB ? d.tabs_even : even(d.sBk1));
  const bool sign = d.sgn != nullptr;
  if (gemm_use_ws()) return launch_dgemm_ws(p, a_kc, b_nc, sign, wmf, st);
  if (a_kc) return b_nc ? launch_dgemm_s<true, true>(sign, wgm, wmf, p, st) : launch_dgemm_s<true, false>(sign, wgm, wmf, p, st);
  return b_nc ? launch_dgemm_s<false, true>(sign, wgm, wmf, p, st) : launch_dgemm_s<false, false>(sign, wgm, wmf, p, st);
}

}  // namespace gfcc
