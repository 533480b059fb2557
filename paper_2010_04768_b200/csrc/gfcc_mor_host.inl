// =====================================================================================
// gfcc_mor_host.inl -- host drivers of the MOR calls of include/gfcc.h (included by gfcc_lib.cu, which provides
// gfcc_ctx, gemm(), gemm_splitk(), dev_alloc(), sigma_internal(), ensure_workspace() and the error macros).
//
//   gfcc_mor_reset  : allocate / clear the subspace
//   gfcc_mor_extend : Alg. 1 line 18 (Gram-Schmidt, O(m^2 O^2 V)) + line 19 (projection, O(m O^3 V^2))
//   gfcc_mor_solve  : Eq. 10 reduced systems on a frequency grid + Eq. 9 spectral function (Alg. 1 line 20-21)
// =====================================================================================

static constexpr int MOR_KSPLIT = 128;     // row chunks of the tall-skinny S^T V products (K1 blocks of the split-K GEMM)

static int mor_ensure_part(gfcc_ctx* h, long long elems) {
  if (elems <= h->part_elems) return GFCC_OK;
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  dev_free(h, h->part, h->part_elems);
  h->part = nullptr; h->part_elems = 0;
  TRY(dev_alloc(h, &h->part, elems));
  h->part_elems = elems;
  return GFCC_OK;
}

// C[ma][nb] (leading dimension ldc) = A[:, 0:ma]^T B[:, 0:nb] over the n_pad rows; A, B row-major with leading dims lda, ldb
static int mor_atb(gfcc_ctx* h, const double* A, long long lda, int ma, const double* B, long long ldb, int nb, double* C,
                   long long ldc) {
  if (ma <= 0 || nb <= 0) return GFCC_OK;
  const long long K0 = h->mor_npad / MOR_KSPLIT;
  GemmDesc d; d.M = ma; d.N = nb; d.K1 = MOR_KSPLIT; d.K0 = (int)K0;
  d.A = A; d.sAm = 1; d.sAk0 = lda; d.sAk1 = K0 * lda;
  d.B = B; d.sBk0 = ldb; d.sBn = 1; d.sBk1 = K0 * ldb;
  d.C = C; d.sCm0 = ldc;
  const long long tiles = (long long)((ma + 127) / 128) * ((nb + 127) / 128);
  int S = (int)std::max<long long>(1, std::min<long long>(MOR_KSPLIT, 296 / tiles));
  while (MOR_KSPLIT % S) --S;                       // equal chunks: no ragged tail launch
  TRY(mor_ensure_part(h, (long long)S * ma * nb));
  return gemm_splitk(h, d, S);
}

// V[:, 0:nb] -= A[:, 0:ma] C[0:ma][0:nb]
static int mor_sub_ac(gfcc_ctx* h, double* V, long long ldv, int nb, const double* A, long long lda, int ma, const double* C,
                      long long ldc) {
  if (ma <= 0 || nb <= 0) return GFCC_OK;
  GemmDesc d; d.M = (int)h->nvec; d.N = nb; d.K0 = ma;
  d.A = A; d.sAm = lda; d.sAk0 = 1;
  d.B = C; d.sBk0 = ldc; d.sBn = 1;
  d.C = V; d.sCm0 = ldv; d.alpha = -1.0; d.beta = 1.0;
  return gemm(h, d);
}

extern "C" int gfcc_mor_reset(gfcc_handle h, int m_cap) {
  if (!h) return GFCC_EINVAL;
  if (m_cap < 0) { h->err = "gfcc_mor_reset: m_cap < 0"; return GFCC_EINVAL; }
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  if (h->mor_S) {
    dev_free(h, h->mor_S, h->mor_npad * h->mor_cap); dev_free(h, h->mor_HS, h->mor_npad * h->mor_cap);
    dev_free(h, h->mor_Hh, (long long)h->mor_cap * h->mor_cap);
    h->mor_S = h->mor_HS = h->mor_Hh = nullptr;
  }
  h->mor_cap = h->mor_m = 0; h->st_mor_dropped = 0; h->st_mor_sigma_cols = 0;
  if (m_cap == 0) return GFCC_OK;
  const int cap = (int)std::min<long long>((m_cap + 1) & ~1, (h->nvec + 1) & ~1LL);   // even; never more than the dimension
  h->mor_npad = ((h->nvec + 2 * MOR_KSPLIT - 1) / (2 * MOR_KSPLIT)) * (2 * MOR_KSPLIT);   // K0 even: 16-byte cp.async stays legal
  TRY(dev_alloc(h, &h->mor_S, h->mor_npad * cap)); TRY(dev_alloc(h, &h->mor_HS, h->mor_npad * cap));
  TRY(dev_alloc(h, &h->mor_Hh, (long long)cap * cap));
  CUDA_TRY(h, cudaMemsetAsync(h->mor_S, 0, (size_t)(h->mor_npad * cap) * 8, h->stream));
  CUDA_TRY(h, cudaMemsetAsync(h->mor_HS, 0, (size_t)(h->mor_npad * cap) * 8, h->stream));
  CUDA_TRY(h, cudaMemsetAsync(h->mor_Hh, 0, (size_t)cap * cap * 8, h->stream));
  h->mor_cap = cap;
  return GFCC_OK;
}

extern "C" int gfcc_mor_extend(gfcc_handle h, int nx, const void* X1, const void* X2, double droptol, int* m_out) {
  if (!h) return GFCC_EINVAL;
  if (nx < 1 || !X1 || !X2 || !(droptol >= 0)) { h->err = "gfcc_mor_extend: null pointer, nx < 1 or droptol < 0"; return GFCC_EINVAL; }
  if (!h->mor_S) { h->err = "gfcc_mor_extend: no subspace (call gfcc_mor_reset(h, m_cap) first)"; return GFCC_EINVAL; }
  const int o = h->o, v = h->v, cap = h->mor_cap, k = 2 * nx;
  const long long n = h->nvec, npad = h->mor_npad;
  cudaStream_t st = h->stream;
  h->cur = st;
  const int nblk_n = (int)std::min<long long>(592, (n + 7) / 8);
  double *V = nullptr, *partial = nullptr, *sq = nullptr, *inv = nullptr, *Cbuf = nullptr;
  struct Scratch { gfcc_ctx* h; double** p; long long n; ~Scratch() { cudaStreamSynchronize(h->stream); dev_free(h, *p, n); } };
  TRY(dev_alloc(h, &V, npad * k));                        Scratch f1{h, &V, npad * k};
  TRY(dev_alloc(h, &partial, (long long)nblk_n * k));     Scratch f2{h, &partial, (long long)nblk_n * k};
  TRY(dev_alloc(h, &sq, k));                              Scratch f3{h, &sq, k};
  TRY(dev_alloc(h, &inv, k));                             Scratch f4{h, &inv, k};
  TRY(dev_alloc(h, &Cbuf, (long long)cap * k));           Scratch f5{h, &Cbuf, (long long)cap * k};
  CUDA_TRY(h, cudaMemsetAsync(V, 0, (size_t)(npad * k) * 8, st));
  {
    dim3 blk(32, 8), grid((unsigned)((n + 31) / 32), (unsigned)((nx + 31) / 32));
    k_abi_to_vec<<<grid, blk, 0, st>>>(V, (const double2*)X1, (const double2*)X2, o, v, nx); KLAUNCH(h);
  }
  auto colsq = [&](const double* M, int ncols, long long ld, double* invp) -> int {
    dim3 blk(32, 8), grid((unsigned)nblk_n, (unsigned)((ncols + 31) / 32));
    k_mor_colsq_partial<<<grid, blk, 0, st>>>(partial, M, n, ncols, ld); KLAUNCH(h);
    k_mor_colsq_finish<<<(ncols + 127) / 128, 128, 0, st>>>(sq, invp, partial, nblk_n, ncols); KLAUNCH(h);
    return GFCC_OK;
  };
  // every candidate (Re X_r, Im X_r) is normalised first: the drop test is relative to its own length
  TRY(colsq(V, k, k, inv));
  k_mor_scale_cols<<<nblk(n * k), 256, 0, st>>>(V, inv, n, k, k); KLAUNCH(h);
  const int m0 = h->mor_m;
  // block CGS2 against the previous orthonormal vectors
  for (int pass = 0; pass < 2 && m0 > 0; ++pass) {
    TRY(mor_atb(h, h->mor_S, cap, m0, V, k, k, Cbuf, k));
    TRY(mor_sub_ac(h, V, k, k, h->mor_S, cap, m0, Cbuf, k));
  }
  // sequential CGS2 inside the block, in the order Re X_0, Im X_0, Re X_1, ...
  int m1 = m0, dropped = 0;
  for (int j = 0; j < k; ++j) {
    if (m1 >= cap) { dropped += k - j; break; }
    double* vj = V + j;
    for (int pass = 0; pass < 2 && m1 > m0; ++pass) {
      TRY(mor_atb(h, h->mor_S + m0, cap, m1 - m0, vj, k, 1, Cbuf, 1));
      TRY(mor_sub_ac(h, vj, k, 1, h->mor_S + m0, cap, m1 - m0, Cbuf, 1));
    }
    TRY(colsq(vj, 1, k, nullptr));
    double hsq = 0.0;
    CUDA_TRY(h, cudaMemcpyAsync(&hsq, sq, 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(h, cudaStreamSynchronize(st));
    const double nrm = std::sqrt(hsq);
    if (nrm > droptol && nrm > 0.0) {
      k_mor_copy_col<<<nblk(n), 256, 0, st>>>(h->mor_S + m1, cap, vj, k, n, 1.0 / nrm); KLAUNCH(h);
      ++m1;
    } else ++dropped;
  }
  h->st_mor_dropped += dropped;
  // projection: Hbar S_new by batched sigma at omega = eta = 0 (two real columns ride as one complex RHS), then H^
  const int knew = m1 - m0;
  if (knew > 0) {
    const int nb = h->ws_nrhs > 0 ? h->ws_nrhs : std::max(1, std::min((int)h->opt_max_batch, (knew + 1) / 2));
    TRY(ensure_workspace(h, nb, true));
    CUDA_TRY(h, cudaMemsetAsync(h->d_omega, 0, (size_t)nb * 8, st));
    for (int c0 = m0; c0 < m1; c0 += 2 * nb) {
      const int cnt = std::min(2 * nb, m1 - c0);
      k_mor_copy_cols<<<nblk(n * 2 * nb), 256, 0, st>>>(h->vin, 2 * nb, 2 * nb, h->mor_S + c0, cap, n, cnt); KLAUNCH(h);
      TRY(sigma_internal(h, nb, h->d_omega, 0.0, h->vin, h->vout));
      k_mor_copy_cols<<<nblk(n * cnt), 256, 0, st>>>(h->mor_HS + c0, cap, cnt, h->vout, 2 * nb, n, cnt); KLAUNCH(h);
      h->st_mor_sigma_cols += cnt;
    }
    TRY(mor_atb(h, h->mor_S, cap, m1, h->mor_HS + m0, cap, knew, h->mor_Hh + m0, cap));                       // new columns
    TRY(mor_atb(h, h->mor_S + m0, cap, knew, h->mor_HS, cap, m0, h->mor_Hh + (long long)m0 * cap, cap));       // new rows
  }
  h->mor_m = m1;
  CUDA_TRY(h, cudaStreamSynchronize(st));
  if (m_out) *m_out = m1;
  return GFCC_OK;
}

// Eq. 10 reduced systems on a frequency grid + Eq. 9.  G: [nw][np][np] complex (G[w][ip][iq], q over the same list),
// Aspec: [nw] or null; both may be host or device pointers (copied with cudaMemcpyDefault).
extern "C" int gfcc_mor_solve(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, void* G, double* Aspec) {
  if (!h) return GFCC_EINVAL;
  if (np < 1 || nw < 1 || !p || !omega || !G) { h->err = "gfcc_mor_solve: null pointer or np/nw < 1"; return GFCC_EINVAL; }
  for (int k = 0; k < np; ++k)
    if (p[k] < 0 || p[k] >= h->N) { h->err = "gfcc_mor_solve: target orbital out of range"; return GFCC_EINVAL; }
  if (!h->mor_S || h->mor_m < 1) { h->err = "gfcc_mor_solve: empty subspace (gfcc_mor_reset + gfcc_mor_extend first)"; return GFCC_EINVAL; }
  const int o = h->o, v = h->v, cap = h->mor_cap, m = h->mor_m;
  const long long n = h->nvec, npad = h->mor_npad;
  cudaStream_t st = h->stream;
  h->cur = st;
  // chunk of S columns pushed through the G assembly at a time (pairs of real columns = one complex "RHS")
  const int nbc = std::max(1, std::min(16, (m + 1) / 2));
  const int Ncc = 2 * nbc;
  const int g_blocks = (int)std::min<long long>(296, h->npair);
  // frequencies per LU launch: bounded scratch (<= 2 GB)
  const long long per_w = ((long long)m * m + (long long)m * np) * 2;
  const int nwc = (int)std::max<long long>(1, std::min<long long>(nw, (long long)(2e9 / 8) / std::max<long long>(per_w, 1)));
  double *B = nullptr, *bh2 = nullptr, *chat = nullptr, *vec = nullptr, *gvec = nullptr, *gpart = nullptr, *Gq = nullptr;
  double *dq = nullptr, *dom = nullptr, *Aw = nullptr, *Xw = nullptr, *dG = nullptr, *dA = nullptr, *dsing = nullptr;
  struct Scratch { gfcc_ctx* h; double** p; long long n; ~Scratch() { cudaStreamSynchronize(h->stream); dev_free(h, *p, n); } };
#define MOR_ALLOC(ptr, elems, tag) TRY(dev_alloc(h, &ptr, (elems))); Scratch tag{h, &ptr, (elems)}
  MOR_ALLOC(B, npad * 2 * np, s01);
  MOR_ALLOC(bh2, (long long)m * 2 * np, s02);
  MOR_ALLOC(chat, (long long)(m + 1) * np, s03);
  MOR_ALLOC(vec, n * Ncc, s04);
  MOR_ALLOC(gvec, (long long)v * Ncc, s05);
  MOR_ALLOC(gpart, (long long)g_blocks * v * Ncc, s06);
  MOR_ALLOC(Gq, (long long)nbc * np * 2, s07);
  MOR_ALLOC(dq, np, s08);
  MOR_ALLOC(dom, nw, s09);
  MOR_ALLOC(Aw, (long long)nwc * m * m * 2, s10);
  MOR_ALLOC(Xw, (long long)nwc * m * np * 2, s11);
  MOR_ALLOC(dG, (long long)nw * np * np * 2, s12);
  MOR_ALLOC(dA, nw, s13);
  MOR_ALLOC(dsing, nw, s14);
#undef MOR_ALLOC
  int* dqi = (int*)dq;
  int* dsi = (int*)dsing;
  CUDA_TRY(h, cudaMemcpyAsync(dqi, p, (size_t)np * sizeof(int), cudaMemcpyHostToDevice, st));
  CUDA_TRY(h, cudaMemcpyAsync(dom, omega, (size_t)nw * 8, cudaMemcpyHostToDevice, st));
  CUDA_TRY(h, cudaMemsetAsync(dsi, 0, (size_t)nw * sizeof(int), st));
  // b^ = S^T b_p   (b_p through the RHS builder of the solver: complex [n][np] with zero imaginary parts)
  CUDA_TRY(h, cudaMemsetAsync(B, 0, (size_t)(npad * 2 * np) * 8, st));
  k_build_rhs<<<nblk(n * np), 256, 0, st>>>(B, dqi, h->t1, h->T2p, o, v, np, n); KLAUNCH(h);
  TRY(mor_atb(h, h->mor_S, cap, m, B, 2 * np, 2 * np, bh2, 2 * np));
  // c^ = S^T c_q   through the G assembly (cheap form of SURVEY.md 8c item 10), which is linear in x
  {
    static bool attr_set = false;
    if (!attr_set) { cudaFuncSetAttribute(k_lambda2_g, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); attr_set = true; }
    const size_t smem = lambda2_g_smem_bytes(v);
    for (int c0 = 0; c0 < m; c0 += Ncc) {
      const int cnt = std::min(Ncc, m - c0);
      k_mor_copy_cols<<<nblk(n * Ncc), 256, 0, st>>>(vec, Ncc, Ncc, h->mor_S + c0, cap, n, cnt); KLAUNCH(h);
      dim3 grid((Ncc + LG_CC - 1) / LG_CC, g_blocks);
      k_lambda2_g<<<grid, 32 * LG_WARPS, smem, st>>>(gpart, h->L2p, vec, o, v, Ncc, h->npair); KLAUNCH(h);
      const long long ng = (long long)v * Ncc;
      k_g_reduce<<<(unsigned)((ng + 127) / 128), 128, 0, st>>>(gvec, gpart, g_blocks, ng); KLAUNCH(h);
      dim3 gg(np, nbc);
      k_assemble_G<<<gg, 256, 0, st>>>((double2*)Gq, dqi, np, vec, gvec, h->D, h->t1, h->l1, o, v, nbc); KLAUNCH(h);
      k_mor_store_chat<<<(nbc * np + 127) / 128, 128, 0, st>>>(chat, (const double2*)Gq, nbc, np, c0, cnt); KLAUNCH(h);
    }
  }
  // reduced systems, one CTA per frequency
  for (int w0 = 0; w0 < nw; w0 += nwc) {
    const int nwn = std::min(nwc, nw - w0);
    k_mor_lu_solve<<<nwn, MOR_LU_THREADS, 0, st>>>(m, cap, h->mor_Hh, bh2, np, chat, np, dom + w0, eta, (double2*)Aw, (double2*)Xw,
                                                   (double2*)dG + (long long)w0 * np * np, dA + w0, dsi + w0);
    KLAUNCH(h);
  }
  std::vector<int> hs(nw, 0);
  CUDA_TRY(h, cudaMemcpyAsync(hs.data(), dsi, (size_t)nw * sizeof(int), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(h, cudaStreamSynchronize(st));
  CUDA_TRY(h, cudaMemcpy(G, dG, (size_t)nw * np * np * 16, cudaMemcpyDefault));
  if (Aspec) CUDA_TRY(h, cudaMemcpy(Aspec, dA, (size_t)nw * 8, cudaMemcpyDefault));
  for (int w = 0; w < nw; ++w)
    if (hs[w]) { h->err = "gfcc_mor_solve: singular reduced system at some frequency"; return GFCC_ENOCONV; }
  return GFCC_OK;
}

// parity hooks: name = "Hhat" -> [m][m], "S" -> [n][m], "HS" -> [n][m]; out may be host or device; out == null returns the count
extern "C" long long gfcc_mor_get(gfcc_handle h, const char* name, double* out) {
  if (!h || !name) return GFCC_EINVAL;
  const std::string k(name);
  const int m = h->mor_m, cap = h->mor_cap;
  if (k == "m") return m;
  if (k == "cap") return cap;
  const double* src = nullptr; long long rows = 0;
  if (k == "Hhat") { src = h->mor_Hh; rows = m; }
  else if (k == "S") { src = h->mor_S; rows = h->nvec; }
  else if (k == "HS") { src = h->mor_HS; rows = h->nvec; }
  else { h->err = "gfcc_mor_get: unknown name " + k; return GFCC_EINVAL; }
  if (!out || m == 0) return rows * m;
  cudaStreamSynchronize(h->stream);
  if (cudaMemcpy2D(out, (size_t)m * 8, src, (size_t)cap * 8, (size_t)m * 8, (size_t)rows, cudaMemcpyDefault) != cudaSuccess) {
    h->err = "gfcc_mor_get: copy failed"; cudaGetLastError(); return GFCC_ECUDA;
  }
  return rows * m;
}
