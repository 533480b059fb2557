// =====================================================================================
// gfcc_ea_host.inl -- EA / advanced part of the GFCCSD matrix, included by gfcc_lib.cu.
//
// PAPER.md:78 Eq. 4 (Y_q), Eq. 6 ((omega - Hbar_N + i eta) Y_q|Phi> = abar_q^+|Phi>), second terms of Eq. 7-8
// (PAPER.md:89-94): G^A_pq = <Phi|(1+Lambda1+Lambda2) abar_p (Y_q1 + Y_q2)|Phi>.  Working equations: DESIGN.md section 6.8
// (T1-dressed, Cholesky-factorised; every term checked against a Fock-space brute force in tests/).
//
//   sigma_EA = (omega + i eta) y - Hbar y,  with y1[a], y2[j,a,b] (antisymmetric in a,b), L~ = T1-dressed Cholesky blocks:
//   Yq[Q,a]      = sum_ld L_ov[Q,l,d] y2[l,a,d]                       w[k] = sum_Qc L_ov[Q,k,c] Yq[Q,c]
//   (Hy)1[a]     = sum_c F_ac y1[c] + sum_ld F_ld y2[l,a,d] + sum_Qc L~vv[Q,a,c] Yq[Q,c]
//   R[j,b,a]     = sum_Q (L~vo[Q,b,j] - M[Q,j,b]) Yq[Q,a] - sum_ld K2'[(j,b),(l,d)] y2[l,a,d] + sum_nf t[j,n,f,b] V[n,f,a]
//                  K2'[(j,b),(l,d)] = sum_Q L~oo[Q,l,j] L~vv[Q,b,d] - delta_lj F_bd + 1/2 delta_bd F_lj   (Fock terms folded in)
//                  V[n,f,a] = sum_ld (sum_Q L_ov[Q,l,f] L_ov[Q,n,d]) y2[l,a,d]
//   ZP[a,b,j]    = sum_cd (sum_Q L~vv[Q,a,c] L~vv[Q,b,d]) y2[j,c,d] + sum_(m<n) t[m,n,a,b] U[m,n,j],
//                  U[m,n,j] = sum_cd (sum_Q L_ov[Q,m,c] L_ov[Q,n,d]) y2[j,c,d]
//   (Hy)2[j,a,b] = sum_c W_abcj y1[c] - sum_k t[k,j,a,b] w[k] + ZP[a,b,j] + R[j,b,a] - R[j,a,b]
// The (ov x ov) ring / exchange panels and the (vv x vv) ladder panels are built on the fly from the Cholesky vectors and
// streamed through the same bounded scratch as the IP part; W_abcj (v^3 o / 2 doubles, packed a<b) is the one stored EA
// intermediate, which bounds this part to sizes where it fits (configs 0-1: 0.65 GB at config 1).
// Everything runs on the FP64 DMMA GEMM engine (the INT8 engine is not used here).
// =====================================================================================

struct EaState {
  bool ready = false;
  long long ntri = 0, nE = 0;
  double *WV = nullptr;     // W_abej packed [(j, a<b)][e]
  double *Dv = nullptr;     // [e][a]
  // per-batch workspace (capacity ws_nrhs right-hand sides)
  int ws_nrhs = 0, ni = 1, na = 1, nm = 1;
  double *YU = nullptr, *YV = nullptr, *R = nullptr, *V = nullptr, *ZP = nullptr, *Yq = nullptr, *KP = nullptr, *PP = nullptr;
  double *Up = nullptr, *Upair = nullptr, *w = nullptr, *d_omega = nullptr, *vin = nullptr, *vout = nullptr;
  SolveWs sw;
  std::vector<double> last_relres;
  std::vector<int> last_iters;
  std::vector<std::vector<double>> last_hist;
};

static void ea_free_ws(gfcc_ctx* h, EaState& e) {
  const long long o = h->o, v = h->v, Q = h->Q, Nc = 2LL * e.ws_nrhs, ldE = v * Nc, ldO = o * Nc, ov = o * v, vv = v * v;
  dev_free(h, e.YU, ov * ldE); dev_free(h, e.R, ov * ldE); dev_free(h, e.V, ov * ldE);
  dev_free(h, e.YV, vv * ldO); dev_free(h, e.ZP, vv * ldO);
  dev_free(h, e.Yq, Q * ldE);
  dev_free(h, e.KP, (long long)e.ni * v * ov); dev_free(h, e.PP, (long long)e.na * v * vv);
  dev_free(h, e.Up, (long long)e.nm * o * ldO); dev_free(h, e.Upair, std::max<long long>(1, h->npair) * ldO);
  dev_free(h, e.w, o * Nc); dev_free(h, e.d_omega, e.ws_nrhs);
  dev_free(h, e.vin, e.nE * Nc); dev_free(h, e.vout, e.nE * Nc);
  e.YU = e.R = e.V = e.YV = e.ZP = e.Yq = e.KP = e.PP = e.Up = e.Upair = e.w = e.d_omega = e.vin = e.vout = nullptr;
  e.ws_nrhs = 0;
}

static int ea_ensure_ws(gfcc_ctx* h, EaState& e, int nrhs) {
  if (e.ws_nrhs >= nrhs) return GFCC_OK;
  if (e.ws_nrhs) { cudaStreamSynchronize(h->stream); ea_free_ws(h, e); }
  const long long o = h->o, v = h->v, Q = h->Q, Nc = 2LL * nrhs, ldE = v * Nc, ldO = o * Nc, ov = o * v, vv = v * v;
  const double budget = panel_budget(h, false);
  e.ni = (int)std::max<double>(1, std::min<double>((double)o, std::floor(budget / (8.0 * v * ov))));
  e.na = (int)std::max<double>(1, std::min<double>((double)v, std::floor(budget / (8.0 * v * vv))));
  e.nm = (int)std::max<long long>(1, std::min<long long>(o, (long long)e.na * v / o));   // the (m',n) x (c,d) panel of U lives in PP
  e.nm = (int)std::max<double>(1, std::min<double>((double)e.nm, std::floor(budget / (8.0 * o * ldO))));
  e.ws_nrhs = nrhs;
  int rc = GFCC_OK;
  do {
    if ((rc = dev_alloc(h, &e.YU, ov * ldE))) break;
    if ((rc = dev_alloc(h, &e.R, ov * ldE))) break;
    if ((rc = dev_alloc(h, &e.V, ov * ldE))) break;
    if ((rc = dev_alloc(h, &e.YV, vv * ldO))) break;
    if ((rc = dev_alloc(h, &e.ZP, vv * ldO))) break;
    if ((rc = dev_alloc(h, &e.Yq, Q * ldE))) break;
    if ((rc = dev_alloc(h, &e.KP, (long long)e.ni * v * ov))) break;
    if ((rc = dev_alloc(h, &e.PP, (long long)e.na * v * vv))) break;
    if ((rc = dev_alloc(h, &e.Up, (long long)e.nm * o * ldO))) break;
    if ((rc = dev_alloc(h, &e.Upair, std::max<long long>(1, h->npair) * ldO))) break;
    if ((rc = dev_alloc(h, &e.w, o * Nc))) break;
    if ((rc = dev_alloc(h, &e.d_omega, nrhs))) break;
    if ((rc = dev_alloc(h, &e.vin, e.nE * Nc))) break;
    if ((rc = dev_alloc(h, &e.vout, e.nE * Nc))) break;
  } while (0);
  if (rc != GFCC_OK) ea_free_ws(h, e);
  return rc;
}

// One-time EA intermediates: W_abej (dressed form) and Dv.
//   W_abej = <ab||ej>~ - sum_m F_me t[m,j,a,b] + sum_(m<n) <mn||ej>~ t[m,n,a,b] - P(ab) sum_mf <mb||ef>~ t[m,j,a,f]
static int ea_prepare(gfcc_ctx* h, EaState& e) {
  if (e.ready) return GFCC_OK;
  NvtxRange nv("gfcc EA prepare (W_abej, Dv)");
  const int o = h->o, v = h->v, Q = h->Q;
  const long long ov = (long long)o * v, vv = (long long)v * v, npair = h->npair, oo = (long long)o * o;
  e.ntri = h->ntri; e.nE = v + (long long)o * e.ntri;
  cudaStream_t st = h->stream;
  h->cur = st;
  const long long nWV = (long long)o * e.ntri * v;
  TRY(dev_alloc(h, &e.WV, nWV)); TRY(dev_alloc(h, &e.Dv, vv));
  CUDA_TRY(h, cudaMemsetAsync(e.WV, 0, (size_t)std::max<long long>(nWV, 1) * 8, st));
  k_ea_Dv<<<(unsigned)((vv + 127) / 128), 128, 0, st>>>(e.Dv, h->t1, h->l1, h->T2p, h->L2p, o, v); KLAUNCH(h);
  // L~vo[Q][j][b] = Lm + M  (gfcc_create keeps only Lm = L~vo - M): M[Q][i][a] = sum_(n,f) t[i,n,f,a] Lov[Q][n][f]  (P3's GEMM)
  double* Lvo = nullptr;
  TRY(dev_alloc(h, &Lvo, Q * ov));
  {
    GemmDesc d; d.M = Q; d.N = v; d.K1 = o; d.K0 = v; d.batch = o;
    d.A = h->Lov; d.sAm = ov; d.sAk0 = 1; d.sAk1 = v;
    d.B = h->T2p; d.sBk0 = v; d.sBn = 1; d.tabB = h->blk_tab; d.sgn = h->blk_sgn; d.tab_batch_stride = o;
    d.tabs_even = (vv % 2) == 0;
    d.C = Lvo; d.sCm0 = ov; d.bsC = v;
    TRY(gemm(h, d));
  }
  k_ea_addto<<<nblk(Q * ov), 256, 0, st>>>(Lvo, h->Lm, Q * ov); KLAUNCH(h);
  const double budget = panel_budget(h, false);
  // ---- T_a: X1[(a',e)][(j,b)] = sum_Q Lvv[Q][a][e] L~vo[Q][j][b], antisymmetrised in (a,b) by the scatter; panels over a
  {
    int na = (int)std::max<double>(1, std::min<double>(v, std::floor(budget / (8.0 * v * ov))));
    double* X1 = nullptr;
    TRY(dev_alloc(h, &X1, (long long)na * v * ov));
    for (int a0 = 0; a0 < v; a0 += na) {
      const int n_a = std::min(na, v - a0);
      GemmDesc d; d.M = n_a * v; d.N = (int)ov; d.K0 = Q;
      d.A = h->Lvv + (long long)a0 * v; d.sAm = 1; d.sAk0 = vv;
      d.B = Lvo; d.sBk0 = ov; d.sBn = 1;
      d.C = X1; d.sCm0 = ov;
      TRY(gemm(h, d));
      for (int mode = 0; mode < 2; ++mode) {
        k_ea_scatter_aebj<<<nblk((long long)n_a * v * ov), 256, 0, st>>>(e.WV, X1, o, v, a0, n_a, mode); KLAUNCH(h);
      }
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, X1, (long long)na * v * ov);
  }
  dev_free(h, Lvo, Q * ov);
  // ---- T_b: - sum_m F_me t[m,j,a,b]
  k_ea_fme_t2<<<nblk(nWV), 256, 0, st>>>(e.WV, h->Fme, h->T2p, o, v); KLAUNCH(h);
  // ---- T_c: sum_(m<n) <mn||ej>~ t[m,n,a,b]
  if (npair > 0) {
    double *G = nullptr, *OOVO = nullptr, *T = nullptr;
    TRY(dev_alloc(h, &G, ov * oo)); TRY(dev_alloc(h, &OOVO, npair * v * o)); TRY(dev_alloc(h, &T, vv * v * o));
    {   // G[(m,e)][(j,n)] = sum_Q Lov[Q][(m,e)] LooT[Q][(j,n)]      (LooT[Q][j][n] = L~oo[Q,n,j])
      GemmDesc d; d.M = (int)ov; d.N = (int)oo; d.K0 = Q;
      d.A = h->Lov; d.sAm = 1; d.sAk0 = ov;
      d.B = h->LooT; d.sBk0 = oo; d.sBn = 1;
      d.C = G; d.sCm0 = oo;
      TRY(gemm(h, d));
    }
    k_ea_oovo<<<nblk(npair * v * o), 256, 0, st>>>(OOVO, G, o, v); KLAUNCH(h);
    {   // T[(a,b)][(e,j)] = sum_(m<n) T2p[(m<n)][(a,b)] OOVO[(m<n)][(e,j)]
      GemmDesc d; d.M = (int)vv; d.N = v * o; d.K0 = (int)npair;
      d.A = h->T2p; d.sAm = 1; d.sAk0 = vv;
      d.B = OOVO; d.sBk0 = (long long)v * o; d.sBn = 1;
      d.C = T; d.sCm0 = (long long)v * o;
      TRY(gemm(h, d));
    }
    k_ea_pack_abej<<<nblk(nWV), 256, 0, st>>>(e.WV, T, o, v, 1.0); KLAUNCH(h);
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, G, ov * oo); dev_free(h, OOVO, npair * v * o); dev_free(h, T, vv * v * o);
  }
  // ---- T_d: - P(ab) X[a,b,e,j],  X = sum_mf <mb||ef>~ t[m,j,a,f];  panels over b
  {
    int nb = (int)std::max<double>(1, std::min<double>(v, std::floor(budget / (8.0 * v * (ov + (double)o * v)))));
    double *P = nullptr, *X = nullptr;
    TRY(dev_alloc(h, &P, (long long)nb * v * ov)); TRY(dev_alloc(h, &X, (long long)o * nb * vv));
    for (int b0 = 0; b0 < v; b0 += nb) {
      const int n_b = std::min(nb, v - b0);
      {   // P[(b',e)][(m,f)] = sum_Q Lvv[Q][b][f] Lov[Q][m][e]      GEMM rows (b',f), columns (m,e), scattered
        GemmDesc d; d.M = n_b * v; d.N = (int)ov; d.K0 = Q;
        d.A = h->Lvv + (long long)b0 * v; d.sAm = 1; d.sAk0 = vv;
        d.B = h->Lov; d.sBk0 = ov; d.sBn = 1;
        d.C = P; d.Md = v; d.sCm1 = (long long)v * ov; d.sCm0 = 1; d.Nd = v; d.sCn1 = v; d.sCn0 = ov;
        TRY(gemm(h, d));
      }
      {   // P[(b',e)][(m,f)] -= sum_Q Lvv[Q][b][e] Lov[Q][m][f]
        GemmDesc d; d.M = n_b * v; d.N = (int)ov; d.K0 = Q;
        d.A = h->Lvv + (long long)b0 * v; d.sAm = 1; d.sAk0 = vv;
        d.B = h->Lov; d.sBk0 = ov; d.sBn = 1;
        d.C = P; d.sCm0 = ov; d.alpha = -1.0; d.beta = 1.0;
        TRY(gemm(h, d));
      }
      {   // batch j: X[j][(b',e)][a] = sum_(m,f) P[(b',e)][(m,f)] t[m,j,a,f] = - sum P sgn(j,m) T2p[blk(j,m)][a][f]
        GemmDesc d; d.M = n_b * v; d.N = v; d.K1 = o; d.K0 = v; d.batch = o;
        d.A = P; d.sAm = ov; d.sAk0 = 1; d.sAk1 = v;
        d.B = h->T2p; d.sBk0 = 1; d.sBn = v; d.tabB = h->blk_tab; d.sgn = h->blk_sgn; d.tab_batch_stride = o;
        d.tabs_even = (vv % 2) == 0;
        d.C = X; d.sCm0 = v; d.bsC = (long long)n_b * vv; d.alpha = -1.0;
        TRY(gemm(h, d));
      }
      for (int mode = 0; mode < 2; ++mode) {
        k_ea_scatter_jbea<<<nblk((long long)o * n_b * vv), 256, 0, st>>>(e.WV, X, o, v, b0, n_b, mode); KLAUNCH(h);
      }
    }
    CUDA_TRY(h, cudaStreamSynchronize(st));
    dev_free(h, P, (long long)nb * v * ov); dev_free(h, X, (long long)o * nb * vv);
  }
  CUDA_TRY(h, cudaStreamSynchronize(st));
  e.ready = true;
  return GFCC_OK;
}

// ------------------------------------------------------------------------------------------
// sigma_EA on internal vectors: sout = (omega + i eta) yin - Hbar yin.   d_omega: device [nrhs].  yin, sout: [nE][Nc].
// ------------------------------------------------------------------------------------------
static int ea_sigma_internal(gfcc_ctx* h, EaState& e, int nrhs, const double* d_omega, double eta, const double* yin, double* sout) {
  NvtxRange nv_sigma("gfcc sigma_EA");
  const int o = h->o, v = h->v, Q = h->Q;
  const long long Nc = 2LL * nrhs, ldE = (long long)v * Nc, ldO = (long long)o * Nc, ov = (long long)o * v, vv = (long long)v * v;
  const long long npair = h->npair, ntri = e.ntri;
  cudaStream_t st = h->stream;
  h->cur = st;
  const double* y1 = yin;
  double* hy2 = sout + (long long)v * Nc;
  k_ea_unpack_yu<<<(unsigned)ov, 256, 0, st>>>(e.YU, yin, o, v, (int)Nc); KLAUNCH(h);
  k_ea_unpack_yv<<<(unsigned)vv, 256, 0, st>>>(e.YV, yin, o, v, (int)Nc); KLAUNCH(h);
  {   // Yq[Q][(a,c)] = sum_(l,d) Lov[Q][(l,d)] YU[(l,d)][(a,c)]
    GemmDesc d; d.M = Q; d.N = (int)ldE; d.K0 = (int)ov;
    d.A = h->Lov; d.sAm = ov; d.sAk0 = 1;
    d.B = e.YU; d.sBk0 = ldE; d.sBn = 1;
    d.C = e.Yq; d.sCm0 = ldE;
    TRY(gemm(h, d));
  }
  {   // R[(j,b)][(a,c)] = sum_Q Lm[Q][(j,b)] Yq[Q][(a,c)]
    GemmDesc d; d.M = (int)ov; d.N = (int)ldE; d.K0 = Q;
    d.A = h->Lm; d.sAm = 1; d.sAk0 = ov;
    d.B = e.Yq; d.sBk0 = ldE; d.sBn = 1;
    d.C = e.R; d.sCm0 = ldE;
    TRY(gemm(h, d));
  }
  for (int j0 = 0; j0 < o; j0 += e.ni) {
    const int ni = std::min(e.ni, o - j0);
    NvtxRange nvp("EA ring / exchange panel");
    {   // K2[(j',b)][(l,d)] = sum_Q LooT[Q][j][l] Lvv[Q][b][d]
      GemmDesc d; d.M = ni * o; d.N = v * v; d.K0 = Q;
      d.A = h->LooT + (long long)j0 * o; d.sAm = 1; d.sAk0 = (long long)o * o;
      d.B = h->Lvv; d.sBk0 = vv; d.sBn = 1;
      d.C = e.KP; d.Md = o; d.sCm1 = (long long)v * ov; d.sCm0 = v; d.Nd = v; d.sCn1 = ov; d.sCn0 = 1;
      TRY(gemm(h, d));
    }
    k_k2_fixup_general<<<(unsigned)(ni * v), 128, 0, st>>>(e.KP, h->Fmi, h->Fae, o, v, j0, 0.5, -1.0); KLAUNCH(h);
    {   // R[(j,b)] -= K2' YU
      GemmDesc d; d.M = ni * v; d.N = (int)ldE; d.K0 = (int)ov;
      d.A = e.KP; d.sAm = ov; d.sAk0 = 1;
      d.B = e.YU; d.sBk0 = ldE; d.sBn = 1;
      d.C = e.R + (long long)j0 * v * ldE; d.sCm0 = ldE; d.alpha = -1.0; d.beta = 1.0;
      TRY(gemm(h, d));
    }
    {   // K4[(n,f)][(l,d)] = sum_Q Lov[Q,l,f] Lov[Q,n,d] for the panel's n
      GemmDesc d; d.M = (int)ov; d.N = ni * v; d.K0 = Q;
      d.A = h->Lov; d.sAm = 1; d.sAk0 = ov;
      d.B = h->Lov + (long long)j0 * v; d.sBk0 = ov; d.sBn = 1;
      d.C = e.KP; d.Md = v; d.sCm1 = v; d.sCm0 = ov; d.Nd = v; d.sCn1 = (long long)v * ov; d.sCn0 = 1;
      TRY(gemm(h, d));
    }
    {   // V[(n,f)][(a,c)] = K4 YU
      GemmDesc d; d.M = ni * v; d.N = (int)ldE; d.K0 = (int)ov;
      d.A = e.KP; d.sAm = ov; d.sAk0 = 1;
      d.B = e.YU; d.sBk0 = ldE; d.sBn = 1;
      d.C = e.V + (long long)j0 * v * ldE; d.sCm0 = ldE;
      TRY(gemm(h, d));
    }
  }
  {   // R[j][b][(a,c)] += sum_(n,f) t[j,n,f,b] V[(n,f)][(a,c)]
    GemmDesc d; d.M = v; d.N = (int)ldE; d.K1 = o; d.K0 = v;
    d.A = h->T2p; d.sAm = 1; d.sAk0 = v; d.tabA = h->blk_tab; d.sgn = h->blk_sgn; d.tab_batch_stride = o;
    d.tabs_even = (vv % 2) == 0;
    d.B = e.V; d.sBk1 = (long long)v * ldE; d.sBk0 = ldE; d.sBn = 1;
    d.C = e.R; d.sCm0 = ldE; d.bsC = (long long)v * ldE;
    d.batch = o; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  // ---- particle-particle ladder: ZP[(a,b)][(j,cc)] = sum_(c,d) PP[(a,b)][(c,d)] YV[(c,d)][(j,cc)], panels over a
  for (int a0 = 0; a0 < v; a0 += e.na) {
    const int na = std::min(e.na, v - a0);
    NvtxRange nvp("EA pp-ladder panel");
    {   // PP[(a',b)][(c,d)] = sum_Q Lvv[Q][a][c] Lvv[Q][b][d]: GEMM rows (a',c), columns (b,d), scattered
      GemmDesc d; d.M = na * v; d.N = (int)vv; d.K0 = Q;
      d.A = h->Lvv + (long long)a0 * v; d.sAm = 1; d.sAk0 = vv;
      d.B = h->Lvv; d.sBk0 = vv; d.sBn = 1;
      d.C = e.PP; d.Md = v; d.sCm1 = (long long)v * vv; d.sCm0 = v; d.Nd = v; d.sCn1 = vv; d.sCn0 = 1;
      TRY(gemm(h, d));
    }
    {
      GemmDesc d; d.M = na * v; d.N = (int)ldO; d.K0 = (int)vv;
      d.A = e.PP; d.sAm = vv; d.sAk0 = 1;
      d.B = e.YV; d.sBk0 = ldO; d.sBn = 1;
      d.C = e.ZP + (long long)a0 * v * ldO; d.sCm0 = ldO;
      TRY(gemm(h, d));
    }
  }
  // ---- U[m,n,j] = sum_(c,d) (mc|nd) y2[j,c,d] (antisymmetric in m,n), then ZP += sum_(m<n) t[m,n,a,b] U[(m<n)]
  if (npair > 0) {
    NvtxRange nvp("EA U term");
    for (int m0 = 0; m0 < o; m0 += e.nm) {
      const int nm = std::min(e.nm, o - m0);
      {   // OO[(m',n)][(c,d)] = sum_Q Lov[Q][m][c] Lov[Q][n][d]: GEMM rows (m',c), columns (n,d), scattered; lives in PP
        GemmDesc d; d.M = nm * v; d.N = (int)ov; d.K0 = Q;
        d.A = h->Lov + (long long)m0 * v; d.sAm = 1; d.sAk0 = ov;
        d.B = h->Lov; d.sBk0 = ov; d.sBn = 1;
        d.C = e.PP; d.Md = v; d.sCm1 = (long long)o * vv; d.sCm0 = v; d.Nd = v; d.sCn1 = vv; d.sCn0 = 1;
        TRY(gemm(h, d));
      }
      {
        GemmDesc d; d.M = nm * o; d.N = (int)ldO; d.K0 = (int)vv;
        d.A = e.PP; d.sAm = vv; d.sAk0 = 1;
        d.B = e.YV; d.sBk0 = ldO; d.sBn = 1;
        d.C = e.Up; d.sCm0 = ldO;
        TRY(gemm(h, d));
      }
      k_ea_pack_u<<<nblk((long long)nm * o * ldO), 256, 0, st>>>(e.Upair, e.Up, o, m0, nm, ldO); KLAUNCH(h);
    }
    GemmDesc d; d.M = (int)vv; d.N = (int)ldO; d.K0 = (int)npair;
    d.A = h->T2p; d.sAm = 1; d.sAk0 = vv;
    d.B = e.Upair; d.sBk0 = ldO; d.sBn = 1;
    d.C = e.ZP; d.sCm0 = ldO; d.beta = 1.0;
    TRY(gemm(h, d));
  }
  // ---- direct terms into sout ----
  {   // (Hy)2[(j,a<b)][cc] = sum_e WV[(j,a<b)][e] y1[e][cc]
    GemmDesc d; d.M = (int)(o * ntri); d.N = (int)Nc; d.K0 = v;
    d.A = e.WV; d.sAm = v; d.sAk0 = 1;
    d.B = y1; d.sBk0 = Nc; d.sBn = 1;
    d.C = hy2; d.sCm0 = Nc;
    if (ntri > 0) TRY(gemm(h, d));
  }
  {   // w[k][cc] = sum_(Q,c) Lov[Q][k][c] Yq[Q][c][cc]
    GemmDesc d; d.M = o; d.N = (int)Nc; d.K1 = Q; d.K0 = v;
    d.A = h->Lov; d.sAm = v; d.sAk0 = 1; d.sAk1 = ov;
    d.B = e.Yq; d.sBk0 = Nc; d.sBk1 = ldE; d.sBn = 1;
    d.C = e.w; d.sCm0 = Nc;
    TRY(gemm_splitk(h, d, 64));
  }
  if (ntri > 0) { k_ea_wt2<<<(unsigned)(o * ntri), 64, 0, st>>>(sout, h->T2p, e.w, o, v, (int)Nc); KLAUNCH(h); }
  {   // (Hy)1[a][cc] = sum_c Fae[a][c] y1[c][cc]
    GemmDesc d; d.M = v; d.N = (int)Nc; d.K0 = v;
    d.A = h->Fae; d.sAm = v; d.sAk0 = 1;
    d.B = y1; d.sBk0 = Nc; d.sBn = 1;
    d.C = sout; d.sCm0 = Nc;
    TRY(gemm(h, d));
  }
  {   // += sum_(l,d) Fme[(l,d)] YU[(l,d)][(a,cc)]
    GemmDesc d; d.M = 1; d.N = (int)ldE; d.K1 = o; d.K0 = v;
    d.A = h->Fme; d.sAm = ov; d.sAk0 = 1; d.sAk1 = v;
    d.B = e.YU; d.sBk0 = ldE; d.sBk1 = (long long)v * ldE; d.sBn = 1;
    d.C = sout; d.sCm0 = ldE; d.beta = 1.0;
    TRY(gemm_splitk(h, d, 32));
  }
  {   // += sum_(Q,c) Lvv[Q][a][c] Yq[Q][c][cc]
    GemmDesc d; d.M = v; d.N = (int)Nc; d.K1 = Q; d.K0 = v;
    d.A = h->Lvv; d.sAm = v; d.sAk0 = 1; d.sAk1 = vv;
    d.B = e.Yq; d.sBk0 = Nc; d.sBk1 = ldE; d.sBn = 1;
    d.C = sout; d.sCm0 = Nc; d.beta = 1.0;
    TRY(gemm_splitk(h, d, 64));
  }
  k_ea_epilogue<<<(unsigned)e.nE, 64, 0, st>>>(sout, yin, e.ZP, e.R, d_omega, eta, o, v, nrhs); KLAUNCH(h);
  h->st_sigma_apps += 1;
  return GFCC_OK;
}

static EaState& ea_state(gfcc_ctx* h);

static int ea_sigma_abi(gfcc_ctx* h, int nrhs, const double* omega, double eta, const void* Y1, const void* Y2, void* S1, void* S2) {
  EaState& e = ea_state(h);
  TRY(ea_prepare(h, e));
  TRY(ea_ensure_ws(h, e, nrhs));
  cudaStream_t st = h->stream;
  CUDA_TRY(h, cudaMemcpyAsync(e.d_omega, omega, (size_t)nrhs * 8, cudaMemcpyHostToDevice, st));
  dim3 blk(32, 8), grid((unsigned)((e.nE + 31) / 32), (unsigned)((nrhs + 31) / 32));
  k_ea_abi_to_vec<<<grid, blk, 0, st>>>(e.vin, (const double2*)Y1, (const double2*)Y2, h->o, h->v, nrhs); KLAUNCH(h);
  TRY(ea_sigma_internal(h, e, nrhs, e.d_omega, eta, e.vin, e.vout));
  k_ea_vec_to_abi<<<grid, blk, 0, st>>>((double2*)S1, (double2*)S2, e.vout, h->o, h->v, nrhs, 0, nullptr); KLAUNCH(h);
  k_ea_zero_diag<<<nblk((long long)nrhs * h->o * h->v), 256, 0, st>>>((double2*)S2, h->o, h->v, nrhs, nullptr); KLAUNCH(h);
  return GFCC_OK;
}

extern "C" int gfcc_sigma_ea(gfcc_handle h, int nrhs, const double* omega, double eta, const void* Y1, const void* Y2, void* S1,
                             void* S2) {
  if (!h) return GFCC_EINVAL;
  if (nrhs < 1 || !omega || !Y1 || !Y2 || !S1 || !S2) { h->err = "gfcc_sigma_ea: null pointer or nrhs < 1"; return GFCC_EINVAL; }
  return ea_sigma_abi(h, nrhs, omega, eta, Y1, Y2, S1, S2);
}

// G^A assembly of the first ncol columns of `vec` (row stride ld complex columns): Gq[out_row[r]][ip] = c_{p[ip]} . y_r
static int ea_assemble(gfcc_ctx* h, EaState& e, const double* vec, int ld, int ncol, const int* d_plist, int np, double2* Gq,
                       const int* out_row, double2* g2, double* nl) {
  cudaStream_t st = h->stream;
  dim3 blk(32, 8), grid(h->o, (ncol + 31) / 32);
  k_ea_g2<<<grid, blk, 0, st>>>(g2, h->L2p, vec, h->o, h->v, ld, ncol);
  dim3 gg(np, ncol);
  k_ea_assemble_G<<<gg, 256, 0, st>>>(Gq, d_plist, np, vec, g2, e.Dv, h->t1, h->l1, h->o, h->v, ld, out_row);
  *nl += 2;
  return cudaGetLastError() == cudaSuccess ? GFCC_OK : GFCC_ECUDA;
}

extern "C" int gfcc_assemble_g_ea(gfcc_handle h, int nrhs, const void* Y1, const void* Y2, int np, const int* p, void* Gout) {
  if (!h) return GFCC_EINVAL;
  if (nrhs < 1 || np < 1 || !Y1 || !Y2 || !p || !Gout) { h->err = "gfcc_assemble_g_ea: null pointer or nrhs/np < 1"; return GFCC_EINVAL; }
  for (int k = 0; k < np; ++k)
    if (p[k] < 0 || p[k] >= h->N) { h->err = "gfcc_assemble_g_ea: orbital out of range"; return GFCC_EINVAL; }
  EaState& e = ea_state(h);
  TRY(ea_prepare(h, e));
  const long long Nc = 2LL * nrhs;
  cudaStream_t st = h->stream;
  double *vec = nullptr, *g2 = nullptr, *Gq = nullptr, *dpd = nullptr;
  int rc = GFCC_OK;
  do {
    if ((rc = dev_alloc(h, &vec, e.nE * Nc))) break;
    if ((rc = dev_alloc(h, &g2, (long long)h->o * Nc))) break;
    if ((rc = dev_alloc(h, &Gq, (long long)nrhs * np * 2))) break;
    if ((rc = dev_alloc(h, &dpd, np))) break;
    rc = GFCC_ECUDA;
    if (cudaMemcpyAsync(dpd, p, (size_t)np * sizeof(int), cudaMemcpyHostToDevice, st) != cudaSuccess) { h->err = "H2D failed"; break; }
    dim3 blk(32, 8), grid((unsigned)((e.nE + 31) / 32), (unsigned)((nrhs + 31) / 32));
    k_ea_abi_to_vec<<<grid, blk, 0, st>>>(vec, (const double2*)Y1, (const double2*)Y2, h->o, h->v, nrhs);
    double nl = 1;
    if (ea_assemble(h, e, vec, nrhs, nrhs, (const int*)dpd, np, (double2*)Gq, nullptr, (double2*)g2, &nl) != GFCC_OK) { h->err = "gfcc_assemble_g_ea: launch failed"; break; }
    h->st_kernel_launches += nl;
    if (cudaMemcpyAsync(Gout, Gq, (size_t)nrhs * np * 16, cudaMemcpyDefault, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) { h->err = "gfcc_assemble_g_ea: copy of G failed"; break; }
    rc = GFCC_OK;
  } while (0);
  cudaStreamSynchronize(st);
  dev_free(h, vec, e.nE * Nc); dev_free(h, g2, (long long)h->o * Nc); dev_free(h, Gq, (long long)nrhs * np * 2); dev_free(h, dpd, np);
  return rc;
}

// Solve Eq. 6 for every (q = p[iq], omega[iw]) with the batched GMRES of gfcc_solve.cuh (same core, compaction and refill as the
// IP part; tasks r = iq*nw + iw) and assemble the advanced part G^A[iw][ip][iq] = c_{p[ip]} . Y_{p[iq]}(omega_iw).
extern "C" int gfcc_solve_ea_x(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol, void* G,
                               void* Y1out, void* Y2out) {
  if (!h) return GFCC_EINVAL;
  if (np < 1 || nw < 1 || !p || !omega || !G || !(tol > 0)) { h->err = "gfcc_solve_ea: null pointer, np/nw < 1 or tol <= 0"; return GFCC_EINVAL; }
  for (int k = 0; k < np; ++k)
    if (p[k] < 0 || p[k] >= h->N) { h->err = "gfcc_solve_ea: target orbital out of range"; return GFCC_EINVAL; }
  EaState& e = ea_state(h);
  TRY(ea_prepare(h, e));
  const int ntot = np * nw;
  e.last_relres.assign(ntot, 0.0); e.last_iters.assign(ntot, 0); e.last_hist.assign(ntot, std::vector<double>());
  std::vector<SolveTask> tasks(ntot);
  for (int iq = 0; iq < np; ++iq)
    for (int iw = 0; iw < nw; ++iw) { tasks[iq * nw + iw].p = p[iq]; tasks[iq * nw + iw].omega = omega[iw]; }
  const int batch = std::max(1, std::min(ntot, (int)h->opt_max_batch));
  TRY(ea_ensure_ws(h, e, batch));
  double *Gq = nullptr, *dpd = nullptr, *g2 = nullptr;   // Gq [ntot][np] complex: Gq[task (iq,iw)][ip]
  int rc_final = GFCC_OK;
  cudaStream_t st = h->stream;
  do {
    if ((rc_final = dev_alloc(h, &Gq, (long long)ntot * np * 2))) break;
    if ((rc_final = dev_alloc(h, &dpd, np))) break;
    if ((rc_final = dev_alloc(h, &g2, (long long)h->o * 2 * batch))) break;
    const int* dp = (const int*)dpd;
    if (cudaMemcpyAsync(dpd, p, (size_t)np * sizeof(int), cudaMemcpyHostToDevice, st) != cudaSuccess) { h->err = "H2D failed"; rc_final = GFCC_ECUDA; break; }
    SolveCfg cfg;
    cfg.o = h->o; cfg.v = h->v; cfg.nvec = e.nE; cfg.npair = h->npair;
    cfg.m = (int)h->opt_m; cfg.maxit = (int)h->opt_maxit; cfg.fixed = (int)h->opt_fixed; cfg.x0 = (int)h->opt_x0;
    cfg.batch = batch; cfg.compact = h->opt_compact;
    cfg.poll = h->opt_poll > 0 ? (int)h->opt_poll : 1;
    cfg.eta = eta; cfg.tol = tol;
    cfg.t1 = h->t1; cfg.l1 = h->l1; cfg.T2p = h->T2p; cfg.L2p = h->L2p; cfg.D = h->D; cfg.fdiag = h->fdiag;
    cfg.stream = st;
    SigmaFn apply = [&](int nrhs, const double* d_omega, const double* yin, double* sout) -> int {
      return ea_sigma_internal(h, e, nrhs, d_omega, eta, yin, sout);
    };
    SolveHooks hooks;
    hooks.init = [&](double* b, double* x, int A, int c0, const int* q_col, const double* omega_col, double* nl) -> int {
      const long long tot = e.nE * (A - c0);
      k_ea_build_rhs<<<nblk(tot, 256, 148LL * 16), 256, 0, st>>>(b, q_col, h->t1, h->T2p, h->o, h->v, A, e.nE, c0);
      k_ea_x0<<<nblk(tot, 256, 148LL * 16), 256, 0, st>>>(x, b, omega_col, eta, h->fdiag, h->o, h->v, A, e.nE, cfg.x0, c0);
      *nl += 2;
      return cudaGetLastError() == cudaSuccess ? 0 : GFCC_ECUDA;
    };
    hooks.finish = [&](const double* xr, int ld, int nret, const int* ret_row, double* nl) -> int {
      int rc = ea_assemble(h, e, xr, ld, nret, dp, np, (double2*)Gq, ret_row, (double2*)g2, nl);
      if (rc) return rc;
      if (Y1out && Y2out) {
        dim3 blk(32, 8), g3((unsigned)((e.nE + 31) / 32), (unsigned)((nret + 31) / 32));
        k_ea_vec_to_abi<<<g3, blk, 0, st>>>((double2*)Y1out, (double2*)Y2out, xr, h->o, h->v, nret, ld, ret_row);
        const long long tot = (long long)nret * h->o * h->v;
        k_ea_zero_diag<<<(unsigned)std::min<long long>(4096, (tot + 255) / 256), 256, 0, st>>>((double2*)Y2out, h->o, h->v, nret, ret_row);
        *nl += 2;
      }
      return cudaGetLastError() == cudaSuccess ? 0 : GFCC_ECUDA;
    };
    std::string err;
    double nlaunch = 0;
    int rc = solve_run(e.sw, cfg, tasks, apply, hooks, &e.last_hist, &nlaunch, err);
    h->st_kernel_launches += nlaunch;
    if (rc == GFCC_ENOCONV) rc_final = GFCC_ENOCONV;
    else if (rc != GFCC_OK) { h->err = err; rc_final = rc; break; }
    // G[iw][ip][iq] <- Gq[(iq*nw+iw)][ip]
    std::vector<double> hostG((size_t)ntot * np * 2), outG((size_t)ntot * np * 2);
    if (cudaMemcpyAsync(hostG.data(), Gq, hostG.size() * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) { h->err = "D2H of G failed"; rc_final = GFCC_ECUDA; break; }
    for (int iq = 0; iq < np; ++iq)
      for (int iw = 0; iw < nw; ++iw)
        for (int ip = 0; ip < np; ++ip)
          for (int c = 0; c < 2; ++c)
            outG[(((size_t)iw * np + ip) * np + iq) * 2 + c] = hostG[(((size_t)iq * nw + iw) * np + ip) * 2 + c];
    if (cudaMemcpy(G, outG.data(), outG.size() * 8, cudaMemcpyDefault) != cudaSuccess) { h->err = "copy of G to the caller failed"; rc_final = GFCC_ECUDA; break; }
  } while (0);
  cudaStreamSynchronize(st);
  dev_free(h, Gq, (long long)ntot * np * 2); dev_free(h, dpd, np); dev_free(h, g2, (long long)h->o * 2 * batch);
  h->st_max_relres = 0; h->st_nunconv = 0; h->st_iterations = 0;
  for (int k = 0; k < ntot; ++k) {
    e.last_relres[k] = tasks[k].relres; e.last_iters[k] = tasks[k].iters;
    h->st_iterations = std::max(h->st_iterations, (double)tasks[k].iters);
    h->st_max_relres = std::max(h->st_max_relres, tasks[k].relres);
    if (h->opt_fixed == 0 && !tasks[k].converged) h->st_nunconv += 1;
  }
  // the per-RHS getters (gfcc_get_residuals, gfcc_get_residual_history) report the LAST solve, IP or EA
  h->last_relres = e.last_relres; h->last_iters = e.last_iters; h->last_hist = e.last_hist;
  return rc_final;
}

extern "C" int gfcc_solve_ea(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol, void* G) {
  return gfcc_solve_ea_x(h, np, p, nw, omega, eta, tol, G, nullptr, nullptr);
}

static EaState& ea_state(gfcc_ctx* h) {
  if (!h->ea) h->ea = new EaState();
  return *h->ea;
}
static void ea_destroy(gfcc_ctx* h) {
  if (!h->ea) return;
  solve_free(h->ea->sw);
  delete h->ea;
  h->ea = nullptr;
}
static void ea_release_ws(gfcc_ctx* h) {
  if (!h->ea) return;
  if (h->ea->ws_nrhs) ea_free_ws(h, *h->ea);
  solve_free(h->ea->sw);
}
