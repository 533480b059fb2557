// =====================================================================================
// gfcc_gemm.cuh -- the FP64 tensor-core GEMM engine (sm_100a).
//
// Every large contraction of the GFCCSD-IP sigma build (SURVEY.md 8a S1,S6-S11; Eq. 11)
// is a REAL FP64 GEMM (Hbar is real, X complex: the RHS batch is folded into N as 2*nrhs real columns;
// PAPER.md:155 "complex-real mixed operations").  tcgen05 has no f64 kind, so the tensor path on
// sm_100a is DMMA: mma.sync.aligned.m8n8k4.f64 (SASS DMMA.8x8x4; the m16n8k{4,8,16} PTX shapes are
// split into 8x8x4 by ptxas on this target).  Measured issue-rate ceiling on B200: 36.95 TFLOP/s.
//
// Kernel (gfcc_gemm_ws.cuh, warp-specialised): CTA tile BM x 128 x 16 with BM = 16*WMF (WMF = m8 fragments per warp,
// chosen per problem to avoid ragged-M waste), 2 x 4 consumer warps (warp tile up to 64 x 32) + one producer warpgroup,
// accumulators in registers, fragments double-buffered in registers across k4 steps and across tiles, multi-stage
// cp.async (LDGSTS) shared-memory ring with padded, bank-conflict-free tiles.  This header holds the operand
// description, the tile geometry, the PTX helpers and the host-side launch logic.
//
// Operand addressing (element strides, FP64):
//   A(m, k1, k0) = A + offA(k1) + m*sAm + k0*sAk0      B(k1, k0, n) = B + offB(k1) + k0*sBk0 + n*sBn
//   offX(k1) = tabX ? tabX[k1] : k1*sXk1.   K = K1 blocks of length K0 (each zero-padded to BK tiles).
//   Optional sgn[k1] in {+1,-1,0}: the block's contribution is multiplied by it (0 = skipped).
//   Exactly one of (sAm, sAk0) and one of (sBk0, sBn) is 1 (template flags A_KC / B_NC).
//   C(m, n) = C + (m/Md)*sCm1 + (m%Md)*sCm0 + (n/Nd)*sCn1 + (n%Nd)*sCn0   (two-level output scatter)
//   batch index z: A += z*bsA (tabA/sgn += z*K1), B += z*bsB, C += z*bsC.
//   Row-block mode (Rb > 0; A m-contiguous with tabA and sgn): A(m, k1, k0) = A + tabA[(m/Rb)*tabR + k1] + (m%Rb) + k0*sAk0 and the
//   sign sgn[(m/Rb)*tabR + k1] is applied per row (0: the rows of that block are zero-filled).
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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
  int Rb, tabR;     // row-block mode of the A operand (Rb > 0): row m belongs to block rb = m / Rb, its local row is m % Rb, and the
                    // K-block offset and sign are tabA[rb*tabR + k1], sgn[rb*tabR + k1] (several signed pair-packed T2 row blocks in
                    // ONE launch: S11 as 3300-row panels instead of 660-row batches)
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
  int Rb = 0, tabR = 0;    // row-block mode of the A operand (see GemmParams)
};

// choose the m8-fragment count per warp (BM = 16*WMF, WMF in 4..8): the kernel runs one CTA per SM, so the launch takes
// ceil(tiles / 148) waves of time ~ BM each; pick the BM with the smallest waves*BM (this covers both ragged-M padding
// and the partially filled last wave), with a mild penalty for small tiles (more shared-memory traffic per flop).
constexpr int GEMM_NUM_SMS = 148;
constexpr int GEMM_WGM = 2;
inline int pick_wmf(int M, long long N = 0, int batch = 1) {
  const int hi = 8, lo = 4;
  const long long tiles_n = (N > 0) ? (N + GEMM_BN - 1) / GEMM_BN : 0;
  int best = hi; double bestcost = -1;
  for (int w = hi; w >= lo; --w) {
    const int bm = GEMM_WGM * 8 * w;
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
inline int gemm_bm(int M, long long N = 0, int batch = 1) { return GEMM_WGM * 8 * pick_wmf(M, N, batch); }

cudaError_t launch_dgemm_ws(const GemmParams& p, bool a_kc, bool b_nc, bool sign, int wmf, cudaStream_t st);
cudaError_t launch_dgemm_ws_rowblk(const GemmParams& p, bool b_nc, int wmf, cudaStream_t st);

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
  // row-block mode: only tile heights whose BM/2 chunks per tile row divide the 128 producer threads keep the producer on its fast
  // path (a thread then loads the same two rows in every tile and caches their block's table entry): 128 or 64 rows
  const int wmf = (d.Rb > 0) ? (d.M > 64 ? 8 : 4) : pick_wmf(d.M, d.N, d.batch);
  const int bm = GEMM_WGM * 8 * wmf;
  p.Rb = d.Rb; p.tabR = d.tabR;
  if (d.Rb > 0 && (a_kc || !d.tabA || !d.sgn || d.batch != 1 || (d.Rb & 1))) return cudaErrorInvalidValue;
  p.tiles_m = (d.M + bm - 1) / bm;
  p.tiles_n = (d.N + GEMM_BN - 1) / GEMM_BN;
  p.group_m = 8;
  auto even = [](long long x) { return (x & 1LL) == 0; };
  auto al16 = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; };
  // 16-byte cp.async needs: aligned base, even strides along every non-contiguous direction, even offsets
  p.vecA = al16(d.A) && even(a_kc ? d.sAm : d.sAk0) && even(d.bsA) && (d.tabA ? d.tabs_even : even(d.sAk1));
  p.vecB = al16(d.B) && even(b_nc ? d.sBk0 : d.sBn) && even(d.bsB) && (d.tabB ? d.tabs_even : even(d.sBk1));
  const bool sign = d.sgn != nullptr;
  if (d.Rb > 0) return launch_dgemm_ws_rowblk(p, b_nc, wmf, st);
  return launch_dgemm_ws(p, a_kc, b_nc, sign, wmf, st);
}

}  // namespace gfcc
