// =====================================================================================
// gfcc_workflow_host.inl -- the level loop of the retarded GFCCSD workflow (included at the end of gfcc_lib.cu).
//
// Alg. 1: levels -> frequencies of the level -> (omega, p) solves -> Gram-Schmidt -> projection ->
// spectral function on the fine grid -> frequencies of the next level; frequencies by adaptive midpoint refinement with the
// counts of Eq. 12-13.  Readings: DESIGN.md section 2, items 26-27.  Host-side control only (SURVEY.md
// 8f row 3): every numerical step is one of the library's own calls (gfcc_solve_ip_x, gfcc_mor_extend, gfcc_mor_solve).
// =====================================================================================

extern "C" int gfcc_spectral_adaptive(gfcc_handle h, int np, const int* p, double wmin, double wmax, double dw, double eta,
                                      double tol, double spec_tol, int max_levels, double droptol, int n_fine, double* A,
                                      void* G, int* level_of, int* levels_out, int* m_out) {
  if (!h) return GFCC_EINVAL;
  if (np < 1 || !p || !(wmax > wmin) || !(dw > 0) || !(tol > 0) || !(spec_tol >= 0) || !(droptol >= 0) || !A || !level_of) {
    h->err = "gfcc_spectral_adaptive: null pointer, np < 1, empty window or bad tolerance"; return GFCC_EINVAL;
  }
  const int N = (int)std::llround((wmax - wmin) / dw) + 1;                 // N_tot
  if (N < 3 || n_fine != N) { h->err = "gfcc_spectral_adaptive: n_fine must be round((wmax-wmin)/dw)+1 >= 3"; return GFCC_EINVAL; }
  for (int k = 0; k < np; ++k)
    if (p[k] < 0 || p[k] >= h->N) { h->err = "gfcc_spectral_adaptive: target orbital out of range"; return GFCC_EINVAL; }
  int lmax = std::max(1, (int)std::floor(std::log2((wmax - wmin) / dw) + 1e-12));   // Eq. 13
  if (max_levels > 0) lmax = std::min(lmax, max_levels);
  std::vector<double> w(N), Anew(N, 0.0), Aold;
  for (int k = 0; k < N; ++k) w[k] = wmin + dw * k;
  std::vector<int> lev(N, 0);
  // the subspace can take two real vectors per solution; at most 3 + sum_{L=2}^{lmax} 2^(L-1) frequencies are ever sampled (Eq. 12)
  long long nsamp_max = 3;
  for (int L = 2; L <= lmax; ++L) nsamp_max += 1LL << (L - 1);
  nsamp_max = std::min<long long>(nsamp_max, N);
  const long long cap = std::min<long long>(h->nvec + 1, 2LL * np * nsamp_max);
  TRY(gfcc_mor_reset(h, (int)std::min<long long>(cap, 2147483646LL)));
  std::vector<int> cur = {0, (N - 1) / 2, N - 1};
  std::sort(cur.begin(), cur.end());
  cur.erase(std::unique(cur.begin(), cur.end()), cur.end());
  const long long n1 = (long long)h->o * 2, n2 = (long long)h->o * h->o * h->v * 2;
  int level = 0, rc_final = GFCC_OK, m = 0;
  std::vector<double> Ghost((size_t)N * np * np * 2);
  while (!cur.empty()) {
    ++level;
    const int nw = (int)cur.size();
    std::vector<double> om(nw);
    for (int q = 0; q < nw; ++q) { om[q] = w[cur[q]]; lev[cur[q]] = level; }
    // Alg. 1 lines 4-16: all (omega, p) tasks of the level as one batched solve; solutions stay on the device
    double *X1 = nullptr, *X2 = nullptr;
    const long long nx = (long long)np * nw;
    TRY(dev_alloc(h, &X1, nx * n1));
    int rc = dev_alloc(h, &X2, nx * n2);
    if (rc) { dev_free(h, X1, nx * n1); return rc; }
    std::vector<double> Glev((size_t)nw * np * np * 2);
    rc = gfcc_solve_ip_x(h, np, p, nw, om.data(), eta, tol, Glev.data(), X1, X2);
    if (rc == GFCC_ENOCONV) { rc_final = GFCC_ENOCONV; rc = GFCC_OK; }     // keep going with the best iterates; reported at the end
    if (rc == GFCC_OK) rc = gfcc_mor_extend(h, (int)nx, X1, X2, droptol, &m);          // lines 18-19
    dev_free(h, X1, nx * n1); dev_free(h, X2, nx * n2);
    if (rc) return rc;
    if (m < 1) { h->err = "gfcc_spectral_adaptive: empty subspace (all solutions are zero)"; return GFCC_EINVAL; }
    TRY(gfcc_mor_solve(h, np, p, N, w.data(), eta, Ghost.data(), Anew.data()));         // line 20
    if (level >= lmax) break;
    // line 21: intervals whose spectral function still moves get their middle grid point, at most 2^level of them (Eq. 12)
    std::vector<int> sampled;
    for (int k = 0; k < N; ++k) if (lev[k]) sampled.push_back(k);
    double scale = 0.0;
    for (int k = 0; k < N; ++k) scale = std::max(scale, std::fabs(Anew[k]));
    scale = std::max(scale, 1e-300);
    struct Cand { double d; int a, b; };
    std::vector<Cand> cand;
    for (size_t q = 0; q + 1 < sampled.size(); ++q) {
      const int a = sampled[q], b = sampled[q + 1];
      if (b - a < 2) continue;
      double d = INFINITY;
      if (!Aold.empty()) {
        d = 0.0;
        for (int k = a; k <= b; ++k) d = std::max(d, std::fabs(Anew[k] - Aold[k]));
        d /= scale;
        if (d <= spec_tol) continue;
      }
      cand.push_back({d, a, b});
    }
    std::stable_sort(cand.begin(), cand.end(), [](const Cand& x, const Cand& y) { return x.d > y.d || (x.d == y.d && x.a < y.a); });
    const size_t keep = std::min<size_t>(cand.size(), (size_t)1 << level);
    cur.clear();
    for (size_t q = 0; q < keep; ++q) cur.push_back((cand[q].a + cand[q].b) / 2);
    std::sort(cur.begin(), cur.end());
    Aold = Anew;
  }
  std::memcpy(A, Anew.data(), (size_t)N * 8);
  std::memcpy(level_of, lev.data(), (size_t)N * sizeof(int));
  if (G) CUDA_TRY(h, cudaMemcpy(G, Ghost.data(), Ghost.size() * 8, cudaMemcpyDefault));
  if (levels_out) *levels_out = level;
  if (m_out) *m_out = m;
  return rc_final;
}
