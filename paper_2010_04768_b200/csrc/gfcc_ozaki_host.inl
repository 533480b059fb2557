// =====================================================================================
// gfcc_ozaki_host.inl -- the INT8 tensor-core (Ozaki) engine inside the sigma driver (included by gfcc_lib.cu).
//
// S6 and S8-S11 (panel builds from the Cholesky vectors, the two (ov x ov) panel contractions and the
// T2 contraction -- 97 % of the flops of an application at config 4) on tcgen05.mma kind::i8 with FP64 accuracy.
// Option "engine" = 1 selects it; the graded default (engine 0) is the FP64 DMMA engine.
//   constant operands (sliced once per handle):  Lvv [(a,e)][Q], LooT [(i,m)][Q], Lov [(m,e)][Q]
//   per application: XU [(j,c)][(m,e)] (shared B operand of S9 and S10), then V [(j,c)][(n,f)] in the same buffer
//   per panel: K2' / K4 panel [(i,a)][(m,e)] and the T2 row batch [(i,a)][(n,f)] in one buffer
// =====================================================================================

static int oz_alloc(gfcc_ctx* h, OzSliced& s, int R, int K) {
  oz_shape(s, R, K, h->opt_oz_slices);
  double* p = nullptr;
  TRY(dev_alloc(h, &p, (long long)((s.bytes() + 7) / 8))); s.q = reinterpret_cast<int8_t*>(p);
  TRY(dev_alloc(h, &p, R)); s.scale = p;
  TRY(dev_alloc(h, &p, R)); s.amax = reinterpret_cast<unsigned long long*>(p);
  return GFCC_OK;
}
static void oz_release(gfcc_ctx* h, OzSliced& s) {
  if (s.q) dev_free(h, reinterpret_cast<double*>(s.q), (long long)((s.bytes() + 7) / 8));
  if (s.scale) dev_free(h, s.scale, s.R);
  if (s.amax) dev_free(h, reinterpret_cast<double*>(s.amax), s.R);
  s = OzSliced();
}
static void oz_free_ws(gfcc_ctx* h) {
  oz_release(h, h->ozXU); oz_release(h, h->ozKP);
  h->oz_ws_nrhs = 0; h->oz_ws_ni = 0;
}
// rows [r0, r0 + nr) of a sliced operand (same slice stride)
static OzSliced oz_rows(const OzSliced& s, long long r0, int nr) {
  OzSliced w = s;
  w.q = s.q + r0 * s.Kpad; w.scale = s.scale + r0; w.amax = s.amax + r0; w.R = nr;
  return w;
}
static int oz_do_slice(gfcc_ctx* h, const OzOperand& a, OzSliced& s) {
  CUDA_TRY(h, oz_slice(a, s, h->cur));
  h->st_kernel_launches += 3;
  return GFCC_OK;
}
// C (+)= alpha A B^T on the INT8 pipe; accounted (launch counters, FP64-equivalent flops 2MNK, optional event timing) like gemm()
static int oz_gemm(gfcc_ctx* h, const OzSliced& A, const OzSliced& B, const OzCDesc& c) {
  const double fl = 2.0 * A.R * (double)B.R * (double)A.K;
  const bool timed = h->prof;
  if (timed) {
    while (h->ev_pool.size() < h->ev_used + 2) { cudaEvent_t e; CUDA_TRY(h, cudaEventCreate(&e)); h->ev_pool.push_back(e); }
    CUDA_TRY(h, cudaEventRecord(h->ev_pool[h->ev_used], h->cur));
  }
  CUDA_TRY(h, oz_igemm(A, B, c, h->oz_fail, h->cur, 148, nullptr, reinterpret_cast<unsigned*>(h->oz_fail) + 1));
  if (timed) {
    CUDA_TRY(h, cudaEventRecord(h->ev_pool[h->ev_used + 1], h->cur));
    h->ev_used += 2;
    h->ev_flops.push_back(fl);
    h->ev_ops8.push_back(fl * (A.S * (A.S + 1) / 2));
  }
  h->st_gemm_launches += 1; h->st_kernel_launches += 1; h->st_oz_gemms += 1; h->st_flops_exec += fl;
  return GFCC_OK;
}

// panel height for the INT8 engine: as many occupied indices as the byte budget allows, preferring whole waves of 128 x 256 tiles
static int oz_choose_panel(int o, int v, long long ncols, double budget_bytes) {
  const double row_bytes = (double)o * v * 8.0;
  int nmax = (int)std::min<double>(o, std::floor(budget_bytes / (row_bytes * v)));
  if (nmax < 1) nmax = 1;
  int best = nmax; double best_eff = -1;
  const long long tiles_n = (ncols + OZ_BN - 1) / OZ_BN;
  for (int n = nmax; n >= std::max(1, nmax / 2); --n) {
    const long long rows = (long long)n * v;
    const long long tiles = ((rows + OZ_BM - 1) / OZ_BM) * tiles_n;
    const long long waves = (tiles + 147) / 148;
    const double eff = (double)rows * ncols / ((double)waves * 148 * OZ_BM * OZ_BN);
    if (eff > best_eff + 1e-9) { best_eff = eff; best = n; }
  }
  return best;
}

// constants once per handle, application buffers per (nrhs, panel height)
static int oz_prepare(gfcc_ctx* h, int nrhs) {
  const int o = h->o, v = h->v, Q = h->Q;
  const long long Nc = 2LL * nrhs, ld = (long long)o * Nc, ov = (long long)o * v, vv = (long long)v * v;
  if (ld > 2147483647LL || vv > 2147483647LL) { h->err = "ozaki engine: operand has more than 2^31 rows"; return GFCC_EINVAL; }
  if (!h->oz_fail) {
    double* p = nullptr;
    TRY(dev_alloc(h, &p, 1));
    h->oz_fail = reinterpret_cast<int*>(p);
    CUDA_TRY(h, cudaMemsetAsync(h->oz_fail, 0, 8, h->cur));
  }
  if (!h->oz_const_ready) {
    TRY(oz_alloc(h, h->ozLvv, (int)vv, Q)); TRY(oz_alloc(h, h->ozLooT, o * o, Q)); TRY(oz_alloc(h, h->ozLov, (int)ov, Q));
    OzOperand a;
    a.base = h->Lvv; a.sR = 1; a.sK0 = vv; a.R = (int)vv; a.K0 = Q;              TRY(oz_do_slice(h, a, h->ozLvv));
    a.base = h->LooT; a.sR = 1; a.sK0 = (long long)o * o; a.R = o * o; a.K0 = Q;  TRY(oz_do_slice(h, a, h->ozLooT));
    a.base = h->Lov; a.sR = 1; a.sK0 = ov; a.R = (int)ov; a.K0 = Q;               TRY(oz_do_slice(h, a, h->ozLov));
    h->oz_const_ready = true;
  }
  if (h->oz_ws_nrhs < nrhs || h->oz_ws_ni != h->panel_ni) {   // capacity semantics, like ensure_workspace()
    oz_release(h, h->ozXU); oz_release(h, h->ozKP);
    h->oz_ws_nrhs = 0; h->oz_ws_ni = 0;
    const int cap = std::max(nrhs, h->ws_nrhs);
    const long long ldcap = (long long)o * 2 * cap;
    if (ldcap > 2147483647LL) { h->err = "ozaki engine: operand has more than 2^31 rows"; return GFCC_EINVAL; }
    int rc = oz_alloc(h, h->ozXU, (int)ldcap, (int)ov);
    if (rc == GFCC_OK) rc = oz_alloc(h, h->ozKP, h->panel_ni * v, (int)ov);
    if (rc != GFCC_OK) { oz_release(h, h->ozXU); oz_release(h, h->ozKP); return rc; }
    h->oz_ws_nrhs = cap; h->oz_ws_ni = h->panel_ni;
  }
  return GFCC_OK;
}

// S8-S11 of one application on the INT8 engine.  On entry XU is unpacked and Z holds S7's result; on exit Z holds the whole
// ring/exchange term that k_sigma2_epilogue antisymmetrises, exactly as after the DMMA branch.
static int sigma_ring_ozaki(gfcc_ctx* h, int nrhs) {
  const int o = h->o, v = h->v;
  const long long Nc = 2LL * nrhs, ld = (long long)o * Nc, ov = (long long)o * v;
  cudaStream_t st = h->cur;
  TRY(oz_prepare(h, nrhs));
  {   // a pipeline time-out of an earlier launch (never seen; the waits are bounded so that a bug cannot hang the device)
    int hf = 0;
    CUDA_TRY(h, cudaMemcpyAsync(&hf, h->oz_fail, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(h, cudaStreamSynchronize(st));
    if (hf) { h->err = "ozaki engine: tensor-core pipeline wait timed out"; return GFCC_ECUDA; }
  }
  // XU as B operand: rows (j,c), K = (m,e); the slice buffer may have room for a wider batch
  OzSliced xu = oz_rows(h->ozXU, 0, (int)ld);
  {
    OzOperand x; x.base = h->XU; x.sR = 1; x.sK0 = ld; x.R = (int)ld; x.K0 = (int)ov;
    TRY(oz_do_slice(h, x, xu));
  }
  for (int i0 = 0; i0 < o; i0 += h->panel_ni) {
    const int ni = std::min(h->panel_ni, o - i0);
    OzSliced kp = oz_rows(h->ozKP, 0, ni * v);
    OzOperand kpo; kpo.base = h->KP; kpo.sR = ov; kpo.sK0 = 1; kpo.R = ni * v; kpo.K0 = (int)ov;
    // S8: K2[(i,a)][(m,e)] = sum_Q LooT[Q][(i,m)] Lvv[Q][(a,e)], written in the consumer's order; S3, S4 folded by the fix-up
    {
      OzCDesc c; c.C = h->KP; c.Md = o; c.sCm1 = (long long)v * ov; c.sCm0 = v; c.Nd = v; c.sCn1 = ov; c.sCn0 = 1;
      TRY(oz_gemm(h, oz_rows(h->ozLooT, (long long)i0 * o, ni * o), h->ozLvv, c));
    }
    k_k2_fixup<<<(unsigned)(ni * v), 128, 0, st>>>(h->KP, h->Fmi, h->Fae, o, v, i0);
    KLAUNCH(h);
    TRY(oz_do_slice(h, kpo, kp));
    // S9: Z[(i,a)][(j,c)] -= K2' XU
    {
      OzCDesc c; c.C = h->Z + (long long)i0 * v * ld; c.sCm0 = ld; c.alpha = -1.0; c.beta = 1.0;
      TRY(oz_gemm(h, kp, xu, c));
    }
    // S10: K4[(n,f)][(m,e)] = sum_Q L[Q,m,f] L[Q,n,e];  V[(n,f)][(j,c)] = K4 XU
    {
      OzCDesc c; c.C = h->KP; c.Md = v; c.sCm1 = v; c.sCm0 = ov; c.Nd = v; c.sCn1 = (long long)v * ov; c.sCn0 = 1;
      TRY(oz_gemm(h, h->ozLov, oz_rows(h->ozLov, (long long)i0 * v, ni * v), c));
    }
    TRY(oz_do_slice(h, kpo, kp));
    {
      OzCDesc c; c.C = h->V + (long long)i0 * v * ld; c.sCm0 = ld;
      TRY(oz_gemm(h, kp, xu, c));
    }
  }
  // S11: Z[(i,a)][(j,c)] += sum_(n,f) t[i,n,f,a] V[(n,f)][(j,c)]; V takes XU's slice buffer, T2 rows come in batches of panel_ni i's
  {
    OzOperand x; x.base = h->V; x.sR = 1; x.sK0 = ld; x.R = (int)ld; x.K0 = (int)ov;
    TRY(oz_do_slice(h, x, xu));
  }
  for (int i0 = 0; i0 < o; i0 += h->panel_ni) {
    const int ni = std::min(h->panel_ni, o - i0);
    OzSliced tb = oz_rows(h->ozKP, 0, ni * v);
    OzOperand t; t.base = h->T2p; t.sR = 1; t.sK0 = v; t.K0 = v; t.K1 = o; t.R = ni * v;
    t.tab = h->blk_tab + (long long)i0 * o; t.sgn = h->blk_sgn + (long long)i0 * o; t.Rb = v; t.tabR = o;
    TRY(oz_do_slice(h, t, tb));
    OzCDesc c; c.C = h->Z + (long long)i0 * v * ld; c.sCm0 = ld; c.beta = 1.0;
    TRY(oz_gemm(h, tb, xu, c));
  }
  return GFCC_OK;
}

// S6 on the INT8 engine: s2[(i<j)][(a,c)] = sum_(m<n) W[(i<j)][(m<n)] x2[(m<n)][(a,c)].  W's digit slices are made once per handle;
// x2's go into the panel slice buffer, which is idle outside the panel loop (if they do not fit, *done stays false and the caller
// uses the DMMA engine).
static int sigma_s6_ozaki(gfcc_ctx* h, int nrhs, const double* x2, double* s2, bool* done) {
  *done = false;
  const long long npair = h->npair, cols = (long long)h->v * 2 * nrhs;
  if (npair < 1 || cols > 2147483647LL || !h->ozKP.q) return GFCC_OK;
  OzSliced xb;
  oz_shape(xb, (int)cols, (int)npair, h->opt_oz_slices);
  if (xb.bytes() > h->ozKP.bytes()) return GFCC_OK;
  if (!h->ozWp.q) {
    TRY(oz_alloc(h, h->ozWp, (int)npair, (int)npair));
    OzOperand a; a.base = h->Wp; a.sR = npair; a.sK0 = 1; a.R = (int)npair; a.K0 = (int)npair;
    TRY(oz_do_slice(h, a, h->ozWp));
  }
  if (h->ozS6rows < cols) {
    if (h->ozS6scale) { CUDA_TRY(h, cudaStreamSynchronize(h->cur)); dev_free(h, h->ozS6scale, 2 * h->ozS6rows); h->ozS6scale = nullptr; }
    TRY(dev_alloc(h, &h->ozS6scale, 2 * cols));
    h->ozS6rows = cols;
  }
  xb.q = h->ozKP.q; xb.scale = h->ozS6scale; xb.amax = reinterpret_cast<unsigned long long*>(h->ozS6scale + cols);
  OzOperand x; x.base = x2; x.sR = 1; x.sK0 = cols; x.R = (int)cols; x.K0 = (int)npair;
  TRY(oz_do_slice(h, x, xb));
  OzCDesc c; c.C = s2; c.sCm0 = cols;
  TRY(oz_gemm(h, h->ozWp, xb, c));
  *done = true;
  return GFCC_OK;
}
