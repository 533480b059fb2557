// =====================================================================================
// gfcc_gemm_ws.cuh -- the warp-specialised kernel of the FP64 DMMA GEMM engine (sm_100a).
//
// Contraction, operand addressing and tile shapes as described in gfcc_gemm.cuh (SURVEY.md 8a
// S1,S6-S11, Eq. 11); pipeline:
//   * one PRODUCER warpgroup (4 warps) does nothing but address arithmetic + cp.async (LDGSTS) into a
//     WS_STAGES-deep ring of padded shared-memory tiles and signals "full" mbarriers through
//     cp.async.mbarrier.arrive (completion of the copies, not their issue);
//   * two CONSUMER warpgroups (2 x 4 warps, warp tile (8*WMF) x 32) only wait on "full", load fragments
//     (LDS.64, register double-buffered across k4 steps and across tiles) and issue DMMA.8x8x4; one lane per
//     warp releases the stage on an "empty" mbarrier.
// No CTA-wide barrier in the main loop, no integer address work between a barrier and the first DMMA of a
// tile (the bubble ncu showed in the single-role kernel), and registers are moved from the producer to the
// consumers with setmaxnreg (56 / 224 per thread: 128*56 + 256*224 = 64512 <= 65536).
// =====================================================================================
#pragma once
#include "gfcc_gemm.cuh"

namespace gfcc {

constexpr int WS_STAGES = 5;
constexpr int WS_CONSUMER_THREADS = 256;
constexpr int WS_PRODUCER_THREADS = 128;
constexpr int WS_THREADS = WS_CONSUMER_THREADS + WS_PRODUCER_THREADS;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WS_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra WS_DONE;\n"
      "bra WS_WAIT;\n"
      "WS_DONE:\n"
      "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
// arrive on `b` once every cp.async previously issued by this thread has landed (count pre-charged at init)
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t* b) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(smem_u32(b)) : "memory");
}

template <int WMF> struct GemmTileWS {
  using T = GemmTile<2, WMF>;
  static constexpr size_t SMEM_BYTES = (size_t)WS_STAGES * T::STAGE_ELEMS * sizeof(double) + 2 * WS_STAGES * sizeof(uint64_t);
};

template <int WMF, bool A_KC, bool B_NC, bool HAS_SIGN, bool ROWBLK = false>
__global__ void __launch_bounds__(WS_THREADS, 1) dgemm_ws_kernel(const GemmParams p) {
  static_assert(!ROWBLK || (!A_KC && HAS_SIGN), "row-block mode: m-contiguous A with table and sign");
  using T = GemmTile<2, WMF>;
  constexpr int BM = T::BM, BN = GEMM_BN, BK = GEMM_BK, S = WS_STAGES;
  extern __shared__ __align__(16) double smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)S * T::STAGE_ELEMS);
  uint64_t* empty = full + S;

  const int tid = threadIdx.x;
  const int z = blockIdx.z;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < S; ++s) { mbar_init(&full[s], WS_PRODUCER_THREADS); mbar_init(&empty[s], WS_CONSUMER_THREADS / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();

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
  const double* sgn = HAS_SIGN ? p.sgn + (long long)z * p.tab_batch_stride : nullptr;
  const int KT0 = (p.K0 + BK - 1) / BK;
  int nblocks = 0;   // number of non-skipped k1 blocks
  if (HAS_SIGN && !ROWBLK) { for (int k1 = 0; k1 < p.K1; ++k1) nblocks += (sgn[k1] != 0.0) ? 1 : 0; }
  else nblocks = p.K1;   // row-block mode: a K block is zero only for SOME rows of the tile, so none is skipped
  const int total = nblocks * KT0;
  auto skip_zero = [&](int& k1) { if (HAS_SIGN && !ROWBLK) { while (k1 < p.K1 && sgn[k1] == 0.0) ++k1; } };

  if (tid >= WS_CONSUMER_THREADS) {
    // ================================ producer warpgroup ================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;\n");
    const int ptid = tid - WS_CONSUMER_THREADS;
    const double* __restrict__ Ab = p.A + (long long)z * p.bsA;
    const double* __restrict__ Bb = p.B + (long long)z * p.bsB;
    const long long* tabA = p.tabA ? p.tabA + (long long)z * p.tab_batch_stride : nullptr;
    const long long* tabB = p.tabB ? p.tabB + (long long)z * p.tab_batch_stride : nullptr;
    int ld_k1 = 0, ld_kt = 0;
    skip_zero(ld_k1);
    // row-block mode: with BM/2 chunks per tile row dividing the producer thread count, a thread loads the same two rows in every tile
    constexpr bool RB_FIXED = ROWBLK && (WS_PRODUCER_THREADS % (BM / 2) == 0);
    int rb_fix = 0, lr_fix = 0, rb_k1 = -1;
    long long rb_off = 0;
    bool rb_nz = false;
    if (RB_FIXED) {
      const int gm = min(m0 + (ptid % (BM / 2)) * 2, p.M - 1);
      rb_fix = gm / p.Rb; lr_fix = (m0 + (ptid % (BM / 2)) * 2) - rb_fix * p.Rb;
    }
    int stage = 0;
    unsigned phase = 1;   // waiting on parity 1 of a fresh mbarrier returns immediately (first pass over the ring)
    for (int it = 0; it < total; ++it) {
      mbar_wait(&empty[stage], phase);
      double* As = smem + (size_t)stage * T::STAGE_ELEMS;
      double* Bs = As + T::A_ELEMS;
      const long long offA = ROWBLK ? 0 : (tabA ? tabA[ld_k1] : (long long)ld_k1 * p.sAk1);
      const long long offB = tabB ? tabB[ld_k1] : (long long)ld_k1 * p.sBk1;
      const int k0 = ld_kt * BK;
      if (A_KC) {   // As[BM][LDK], chunks along k
        constexpr int CPR = BK / 2;
#pragma unroll
        for (int c = ptid; c < BM * CPR; c += WS_PRODUCER_THREADS) {
          const int row = c / CPR, kc = (c % CPR) * 2;
          const int gm = m0 + row, gk = k0 + kc;
          const int nv = (gm < p.M) ? min(2, max(0, p.K0 - gk)) : 0;
          load_chunk(As + row * T::LDK + kc, Ab + offA + (long long)gm * p.sAm + gk, nv, p.vecA, p.A);
        }
      } else if (ROWBLK) {   // As[BK][LDA_M], chunks along m; a chunk's rows lie in ONE row block (Rb is even)
        constexpr int CPR = BM / 2;
        if (RB_FIXED) {        // this thread always loads the same two rows: block, local row and (per K block) offset / sign are cached
          if (rb_k1 != ld_k1) {
            const long long t = (long long)rb_fix * p.tabR + ld_k1;
            rb_nz = sgn[t] != 0.0;
            rb_off = rb_nz ? tabA[t] : 0;
            rb_k1 = ld_k1;
          }
#pragma unroll
          for (int c = ptid; c < BK * CPR; c += WS_PRODUCER_THREADS) {
            const int kr = c / CPR, mc = (c % CPR) * 2;
            const int gk = k0 + kr;
            const int nv = (gk < p.K0 && rb_nz) ? min(2, max(0, p.M - (m0 + mc))) : 0;
            load_chunk(As + kr * T::LDA_M + mc, Ab + rb_off + (long long)gk * p.sAk0 + lr_fix, nv, p.vecA, p.A);
          }
        } else {
#pragma unroll
          for (int c = ptid; c < BK * CPR; c += WS_PRODUCER_THREADS) {
            const int kr = c / CPR, mc = (c % CPR) * 2;
            const int gm = m0 + mc, gk = k0 + kr;
            int nv = (gk < p.K0) ? min(2, max(0, p.M - gm)) : 0;
            const int rb = gm / p.Rb, lr = gm - rb * p.Rb;
            long long off = 0;
            if (nv > 0) {
              const long long t = (long long)rb * p.tabR + ld_k1;
              if (sgn[t] == 0.0) nv = 0;               // zero-filled rows: this K block does not couple to the row block
              else off = tabA[t];
            }
            load_chunk(As + kr * T::LDA_M + mc, Ab + off + (long long)gk * p.sAk0 + lr, nv, p.vecA, p.A);
          }
        }
      } else {      // As[BK][LDA_M], chunks along m
        constexpr int CPR = BM / 2;
#pragma unroll
        for (int c = ptid; c < BK * CPR; c += WS_PRODUCER_THREADS) {
          const int kr = c / CPR, mc = (c % CPR) * 2;
          const int gm = m0 + mc, gk = k0 + kr;
          const int nv = (gk < p.K0) ? min(2, max(0, p.M - gm)) : 0;
          load_chunk(As + kr * T::LDA_M + mc, Ab + offA + (long long)gk * p.sAk0 + gm, nv, p.vecA, p.A);
        }
      }
      if (B_NC) {   // Bs[BK][LDB_N], chunks along n
        constexpr int CPR = BN / 2;
#pragma unroll
        for (int c = ptid; c < BK * CPR; c += WS_PRODUCER_THREADS) {
          const int kr = c / CPR, nc = (c % CPR) * 2;
          const int gn = n0 + nc, gk = k0 + kr;
          const int nv = (gk < p.K0) ? min(2, max(0, p.N - gn)) : 0;
          load_chunk(Bs + kr * T::LDB_N + nc, Bb + offB + (long long)gk * p.sBk0 + gn, nv, p.vecB, p.B);
        }
      } else {      // Bs[BN][LDK], chunks along k
        constexpr int CPR = BK / 2;
#pragma unroll
        for (int c = ptid; c < BN * CPR; c += WS_PRODUCER_THREADS) {
          const int col = c / CPR, kc = (c % CPR) * 2;
          const int gn = n0 + col, gk = k0 + kc;
          const int nv = (gn < p.N) ? min(2, max(0, p.K0 - gk)) : 0;
          load_chunk(Bs + col * T::LDK + kc, Bb + offB + (long long)gn * p.sBn + gk, nv, p.vecB, p.B);
        }
      }
      cp_async_mbar_arrive(&full[stage]);
      if (++ld_kt == KT0) { ld_kt = 0; ++ld_k1; skip_zero(ld_k1); }
      if (++stage == S) { stage = 0; phase ^= 1u; }
    }
    // the copies must have landed before the CTA's shared memory is released
    asm volatile("cp.async.wait_all;\n" ::: "memory");
    return;
  }

  // ================================== consumer warpgroups ==================================
  asm volatile("setmaxnreg.inc.sync.aligned.u32 224;\n");
  const int lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 2, wn = warp & 3;   // 2 x 4 warps

  double acc[WMF][4][2];
#pragma unroll
  for (int f = 0; f < WMF; ++f)
#pragma unroll
    for (int g = 0; g < 4; ++g) acc[f][g][0] = acc[f][g][1] = 0.0;

  int c_k1 = 0, c_kt = 0;   // block tracking for the sign
  skip_zero(c_k1);
  const int arow = wm * (8 * WMF) + (lane >> 2);   // + 8 f
  const int bcol = wn * 32 + (lane >> 2);          // + 8 g
  const int kl = lane & 3;

  double fa[2][WMF], fb[2][4];
  // row-block mode: the sign belongs to the ROW (block rb_f of fragment row f) and is applied to the A fragments; two masks per
  // fragment row (current / next K block) are refreshed when the K block changes
  int rbt[ROWBLK ? WMF : 1];
  unsigned rm_cur[ROWBLK ? WMF : 1], rm_nxt[ROWBLK ? WMF : 1];
  if (ROWBLK) {
#pragma unroll
    for (int f = 0; f < WMF; ++f) rbt[f] = min((m0 + arow + 8 * f) / p.Rb, (p.M - 1) / p.Rb) * p.tabR;
  }
  auto row_mask = [&](int f, int k1) -> unsigned { return (k1 < p.K1 && sgn[rbt[f] + k1] < 0.0) ? 0x80000000u : 0u; };
  auto load_frags = [&](int buf, int stage, int kk, unsigned smask, const unsigned* rm) {
    const double* As = smem + (size_t)stage * T::STAGE_ELEMS;
    const double* Bs = As + T::A_ELEMS;
    const int k = kk * 4 + kl;
#pragma unroll
    for (int f = 0; f < WMF; ++f) {
      const double av = A_KC ? As[(arow + 8 * f) * T::LDK + k] : As[k * T::LDA_M + arow + 8 * f];
      fa[buf][f] = ROWBLK ? flip_sign(av, rm[f]) : av;
    }
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const double bv = B_NC ? Bs[k * T::LDB_N + bcol + 8 * g] : Bs[(bcol + 8 * g) * T::LDK + k];
      fb[buf][g] = (HAS_SIGN && !ROWBLK) ? flip_sign(bv, smask) : bv;
    }
  };
  auto mask_of = [&](int k1) -> unsigned { return (HAS_SIGN && !ROWBLK && k1 < p.K1 && sgn[k1] < 0.0) ? 0x80000000u : 0u; };

  int stage = 0;
  unsigned phase = 0;
  const int tail4 = (p.K0 - (KT0 - 1) * BK + 3) / 4;   // k4 steps that hold data in the last tile of a K block (1..4)
  if (total > 0) {
    if (ROWBLK) {   // masks of the current K block and, one block AHEAD, of the next (their global loads are never waited for)
#pragma unroll
      for (int f = 0; f < WMF; ++f) { rm_cur[f] = row_mask(f, c_k1); rm_nxt[f] = row_mask(f, c_k1 + 1); }
    }
    mbar_wait(&full[0], 0);
    load_frags(0, 0, 0, mask_of(c_k1), rm_cur);
  }
  for (int it = 0; it < total; ++it) {
    int n_k1 = c_k1, n_kt = c_kt + 1;
    if (n_kt == KT0) { n_kt = 0; ++n_k1; skip_zero(n_k1); }
    const unsigned cur_mask = mask_of(c_k1), nxt_mask = mask_of(n_k1);
    int nstage = stage + 1;
    unsigned nphase = phase;
    if (nstage == S) { nstage = 0; nphase ^= 1u; }
    const int nk4 = (c_kt == KT0 - 1) ? tail4 : BK / 4;
#pragma unroll
    for (int kk = 0; kk < BK / 4; ++kk) {
      const int cur = kk & 1, nxt = cur ^ 1;
      if (kk + 1 < BK / 4) load_frags(nxt, stage, kk + 1, cur_mask, rm_cur);
      else if (it + 1 < total) {
        mbar_wait(&full[nstage], nphase);
        // first fragments of the next tile: its K block's row masks (rm_nxt only if that tile starts a new block; warp-uniform)
        if (ROWBLK && n_k1 != c_k1) load_frags(nxt, nstage, 0, nxt_mask, rm_nxt);
        else load_frags(nxt, nstage, 0, nxt_mask, rm_cur);
      }
      if (!ROWBLK || kk < nk4) {   // row-block mode (short K blocks: 660 = 41.25 tiles): skip the zero-padded k4 steps of a block's
                                   // last tile (warp-uniform); elsewhere the test costs more than the padding (measured)
#pragma unroll
        for (int f = 0; f < WMF; ++f)
#pragma unroll
          for (int g = 0; g < 4; ++g) dmma884(acc[f][g][0], acc[f][g][1], fa[cur][f], fb[cur][g]);
      }
    }
    // every fragment of this stage has been consumed by an issued DMMA: hand the stage back to the producer
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[stage]);
    if (ROWBLK && n_k1 != c_k1) {   // block change (no block is skipped in row-block mode: n_k1 == c_k1 + 1)
#pragma unroll
      for (int f = 0; f < WMF; ++f) { rm_cur[f] = rm_nxt[f]; rm_nxt[f] = row_mask(f, n_k1 + 1); }
    }
    c_k1 = n_k1; c_kt = n_kt;
    stage = nstage; phase = nphase;
  }

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

template <int WMF, bool A_KC, bool B_NC, bool HAS_SIGN>
inline cudaError_t launch_dgemm_ws_t(const GemmParams& p, cudaStream_t st) {
  auto kern = dgemm_ws_kernel<WMF, A_KC, B_NC, HAS_SIGN>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GemmTileWS<WMF>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((unsigned)(p.tiles_m * p.tiles_n), 1, (unsigned)p.batch);
  kern<<<grid, WS_THREADS, GemmTileWS<WMF>::SMEM_BYTES, st>>>(p);
  return cudaGetLastError();
}

template <bool A_KC, bool B_NC, bool HAS_SIGN>
inline cudaError_t launch_dgemm_ws_w(int wmf, const GemmParams& p, cudaStream_t st) {
  switch (wmf) {
    case 8: return launch_dgemm_ws_t<8, A_KC, B_NC, HAS_SIGN>(p, st);
    case 7: return launch_dgemm_ws_t<7, A_KC, B_NC, HAS_SIGN>(p, st);
    case 6: return launch_dgemm_ws_t<6, A_KC, B_NC, HAS_SIGN>(p, st);
    case 5: return launch_dgemm_ws_t<5, A_KC, B_NC, HAS_SIGN>(p, st);
    default: return launch_dgemm_ws_t<4, A_KC, B_NC, HAS_SIGN>(p, st);
  }
}

template <int WMF, bool B_NC>
inline cudaError_t launch_dgemm_ws_rb_t(const GemmParams& p, cudaStream_t st) {
  auto kern = dgemm_ws_kernel<WMF, false, B_NC, true, true>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GemmTileWS<WMF>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((unsigned)(p.tiles_m * p.tiles_n), 1, 1);
  kern<<<grid, WS_THREADS, GemmTileWS<WMF>::SMEM_BYTES, st>>>(p);
  return cudaGetLastError();
}
template <bool B_NC>
inline cudaError_t launch_dgemm_ws_rb_w(int wmf, const GemmParams& p, cudaStream_t st) {
  switch (wmf) {
    case 8: return launch_dgemm_ws_rb_t<8, B_NC>(p, st);
    case 7: return launch_dgemm_ws_rb_t<7, B_NC>(p, st);
    case 6: return launch_dgemm_ws_rb_t<6, B_NC>(p, st);
    case 5: return launch_dgemm_ws_rb_t<5, B_NC>(p, st);
    default: return launch_dgemm_ws_rb_t<4, B_NC>(p, st);
  }
}
inline cudaError_t launch_dgemm_ws_rowblk(const GemmParams& p, bool b_nc, int wmf, cudaStream_t st) {
  return b_nc ? launch_dgemm_ws_rb_w<true>(wmf, p, st) : launch_dgemm_ws_rb_w<false>(wmf, p, st);
}

inline cudaError_t launch_dgemm_ws(const GemmParams& p, bool a_kc, bool b_nc, bool sign, int wmf, cudaStream_t st) {
  if (a_kc) {
    if (b_nc) return sign ? launch_dgemm_ws_w<true, true, true>(wmf, p, st) : launch_dgemm_ws_w<true, true, false>(wmf, p, st);
    return sign ? launch_dgemm_ws_w<true, false, true>(wmf, p, st) : launch_dgemm_ws_w<true, false, false>(wmf, p, st);
  }
  if (b_nc) return sign ? launch_dgemm_ws_w<false, true, true>(wmf, p, st) : launch_dgemm_ws_w<false, true, false>(wmf, p, st);
  return sign ? launch_dgemm_ws_w<false, false, true>(wmf, p, st) : launch_dgemm_ws_w<false, false, false>(wmf, p, st);
}

}  // namespace gfcc
