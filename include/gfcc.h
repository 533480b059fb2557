/* =====================================================================================
 * gfcc.h -- C ABI of the B200-native GFCCSD-IP hot path (libgfcc_b200.so).
 *
 * The library computes, entirely in hand-written CUDA kernels for sm_100a:
 *   gfcc_create    one-time similarity-transformed-Hamiltonian intermediates
 *                  ("constant intermediate tensors ... pre-computed")
 *   gfcc_sigma_ip  the batched complex matvec  sigma = (omega + Hbar_N - i eta) X  on IP-type
 *                  vectors X_p(omega) = (X1_i, X2_ija)            (Eq. 3, Eq. 5;
 *                  "GFCC singles / doubles equations", Alg. 1)
 *   gfcc_solve_ip  batched GMRES for Eq. 5 (Alg. 1) and the assembly
 *                  G_pq(omega) = <Phi|(1+Lambda1+Lambda2) abar_q^+ (X_p1 + X_p2)|Phi>
 *                  (first, IP term of Eq. 7-8)
 * The working equations (the paper prints none) are SURVEY.md section 8(c); readings are in DESIGN.md.
 *
 * Conventions
 *   spin-orbitals, N = o + v, occupied first.  i,j,m,n occupied in [0,o); a,b,e,f virtual in [0,v).
 *   <pq|rs> = sum_Q L[Q,p,r] L[Q,q,s];  all of fock, T1, T2, Lambda1, Lambda2, L are REAL FP64.
 *   complex = interleaved (re, im) pairs of FP64 (layout of cuDoubleComplex / std::complex<double>).
 *   pair(i<j)  = i*o - i*(i+1)/2 + (j-i-1)          (npair = o(o-1)/2)
 *   tri(a<b)   = a*v - a*(a+1)/2 + (b-a-1)          (ntri  = v(v-1)/2)
 *
 * Pointers: every array argument is a DEVICE pointer unless marked [host].  The *_host entry points
 * take HOST pointers for the vectors and do the host<->device copies themselves.
 * Ownership: inputs are read-only.  gfcc_create copies or derives everything it needs EXCEPT T2 and
 * L2, which are BORROWED: they must stay valid and unmodified until gfcc_destroy (T2 is 56 GB and
 * Lambda2 28 GB at config 4; they are not duplicated).  fock, T1, L1, Lchol may be freed when
 * gfcc_create returns.  Outputs are caller-allocated and fully overwritten.
 * Errors: every call returns 0 on success or a negative GFCC_E* code; no exception or abort crosses
 * the boundary.  gfcc_last_error(h) gives a message for the last failing call on that handle
 * (gfcc_last_error(NULL): last failure of gfcc_create on this thread).
 * Streams: work is enqueued on the handle's stream (default: the legacy default stream; see
 * gfcc_set_stream).  gfcc_create and gfcc_solve_ip synchronise that stream before returning;
 * gfcc_sigma_ip is asynchronous with respect to the host.
 * There is no CPU fallback: without a CUDA device every call fails with GFCC_ECUDA.
 * ===================================================================================== */
#ifndef GFCC_H_
#define GFCC_H_

#ifdef __cplusplus
extern "C" {
#endif

#define GFCC_OK       0
#define GFCC_EINVAL  -1   /* null pointer, non-positive size, index out of range, unknown option */
#define GFCC_ENOMEM  -2   /* device allocation failed */
#define GFCC_ECUDA   -3   /* CUDA runtime error (message in gfcc_last_error) */
#define GFCC_ENOCONV -4   /* GMRES hit max iterations for at least one right-hand side; G is still written */

typedef struct gfcc_ctx* gfcc_handle;

/* Build the one-time intermediates on the device:
 *   T1-dressed Cholesky blocks, dressed Fock, F_mi, F_ae, F_me, M^Q_ia, W_mnij (o^4, pair-packed),
 *   W_mbij (o^3 v, pair-packed), D_ki for the G assembly.
 * fock  [N][N] row-major (general: f_ov may be non-zero)
 * T1,L1 [o][v]
 * T2    pair-packed [npair][v][v]:  T2[pair(i,j)][a][b] = t[i,j,a,b], i<j  (antisymmetric in a,b)   BORROWED
 * L2    fully packed [npair][ntri]: L2[pair(i,j)][tri(a,b)] = lambda[i,j,a,b], i<j, a<b               BORROWED
 * Lchol [Q][N][N]
 * o >= 2, v >= 2, Q >= 1.                                                                            */
int gfcc_create(int o, int v, int Q, const double* fock, const double* T1, const double* T2, const double* L1,
                const double* L2, const double* Lchol, gfcc_handle* out);

/* Closed-shell (spin-restricted) inputs (Table 2 note: the paper's production code is the closed-shell one and "only
 * deals with the alpha electrons").  SPATIAL tensors of an RHF-based CCSD calculation, no occupied / nv virtual orbitals, Ns = no+nv:
 *   fock [Ns][Ns], T1, L1 [no][nv], T2, L2 [no][no][nv][nv] with x[i,j,a,b] = x[j,i,b,a]  (T = sum t1 E_ai + 1/2 sum t2 E_ai E_bj,
 *   E_pq = sum_s a+_ps a_qs; same form for Lambda), Lchol [Q][Ns][Ns].  All device pointers; NONE is borrowed.
 * The tensors are expanded to spin orbitals ON THE DEVICE (t[is,jt,as',bt'] = d(s,s')d(t,t') t2[i,j,a,b] - d(s,t')d(t,s') t2[i,j,b,a],
 * ...) and the handle is an ordinary spin-orbital handle with o = 2 no, v = 2 nv in the ordering occupied alpha, occupied beta,
 * virtual alpha, virtual beta: spatial orbital p with alpha spin is spin-orbital p (p < no) or 2 no + (p - no) (p >= no).  For alpha
 * targets gfcc_solve_ip / gfcc_solve_ea return the closed-shell G_pq; G_{p beta, q beta} = G_{p alpha, q alpha}, mixed-spin elements
 * vanish.  This entry gives the closed-shell WORKFLOW through the spin-orbital kernels; it does not realise the flop saving of a
 * spin-adapted formulation.                                                                              */
int gfcc_create_closed_shell(int no, int nv, int Q, const double* fock, const double* T1, const double* T2, const double* L1,
                             const double* L2, const double* Lchol, gfcc_handle* out);

/* sigma_r = (omega[r] - i eta) X_r + Hbar X_r for r = 0..nrhs-1.
 * omega [host][nrhs];  X1,S1 complex [nrhs][o];  X2,S2 complex [nrhs][o][o][v].
 * Precondition (unchecked): X2[r][i][j][a] = -X2[r][j][i][a].  S2 is returned antisymmetric.        */
int gfcc_sigma_ip(gfcc_handle h, int nrhs, const double* omega, double eta, const void* X1, const void* X2,
                  void* S1, void* S2);
/* same, X1,X2,S1,S2 are HOST pointers (pinned or pageable); copies are part of the call; synchronous. */
int gfcc_sigma_ip_host(gfcc_handle h, int nrhs, const double* omega, double eta, const void* X1, const void* X2,
                       void* S1, void* S2);

/* Solve (omega_w + Hbar - i eta) X = b_p for every (p[ip], omega[iw]) with batched GMRES
 * (classical Gram-Schmidt with re-orthogonalisation, complex Givens least squares; restart length,
 * max iterations and initial guess are options) and assemble
 *   G[iw][ip][iq] = G_{p[ip], q = p[iq]}(omega[iw])       complex [nw][np][np]
 * p [host][np] spin-orbital indices in [0,N) (occupied or virtual);  omega [host][nw].
 * Right-hand sides are ordered r = ip*nw + iw.  G may be a device or a host pointer.
 * Stop test: |rotated residual| <= tol * ||b||.  Returns GFCC_ENOCONV if some RHS did not converge
 * (statistics tell which).  X1out/X2out of gfcc_solve_ip_x (nullable, device, layouts of gfcc_sigma_ip
 * with nrhs = np*nw) receive the solutions.                                                          */
int gfcc_solve_ip(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol, void* G);
int gfcc_solve_ip_x(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol,
                    void* G, void* X1out, void* X2out);

/* stream is a cudaStream_t passed as void* (e.g. torch.cuda.current_stream().cuda_stream). */
int gfcc_set_stream(gfcc_handle h, void* cuda_stream);

/* Options (double-valued):
 *   "gmres_m"      restart length (default 50; clipped to what device memory allows)
 *   "gmres_maxit"  maximum number of sigma applications per solve (default 1000)
 *   "gmres_fixed"  if > 0: run exactly this many Arnoldi steps in ONE cycle, no stop test, no compaction (timing mode);
 *                  takes effect on every call (a later smaller value is honoured without reallocation)
 *   "x0"           0: zero initial guess, 1: zeroth-order guess b/(omega - i eta + d) (default 1)
 *   "panel_bytes"  upper bound for one (ov x ov) integral panel scratch.  Default (option never set): 12.8e9 for the sigma workspace of
 *                  the DMMA engine (20 occupied indices per panel at config 4) and 3.2e9 for the create-time scratch, the EA panels and
 *                  the INT8 engine; a value set here applies to all of them
 *   "max_batch"    largest number of right-hand sides processed at once by gfcc_solve_ip (default 256)
 *   "compact"      converged-RHS compaction (iteration counts differ between (omega,p) tasks): when at least
 *                  max(1, compact * active columns) right-hand sides of the batch have met the stop test they are finalised and
 *                  dropped from every live vector, so the GEMM N dimension of the following sigma applications shrinks; free
 *                  columns are refilled from the pending (p,omega) list at the next restart boundary.  Default 0.125; < 0: never
 *                  (lock-step batch with a done mask; same G)
 *   "graph"        CUDA graph of one sigma application inside gfcc_solve_ip (captured once per batch width, replayed afterwards):
 *                  -1 (default) only for latency-bound systems (< 5 GFLOP per application), 0 never, 1 always; the statistic
 *                  "graph_launches" counts replays and "kernel_launches" still counts every kernel a replay runs
 *   "dense"        latency path for tiny systems inside gfcc_solve_ip: the real matrix Hbar_IP (n x n, n = o + o(o-1)/2*v) is built once
 *                  per handle by applying S1-S13 to unit vectors and a sigma application becomes ONE GEMM + a shift kernel.
 *                  -1 (default): when n <= 2048 (33 MB); 0 never; 1 whenever n <= 8192.  gfcc_sigma_ip always runs S1-S13.
 *                  Statistic "dense_applications" counts them.  Takes precedence over "graph".
 *   "release_workspace"  (any value) free the per-batch sigma workspace and the GMRES basis now; they are re-allocated on demand
 *   "gmres_poll"   the done flags live on the device; the host reads them every gmres_poll Arnoldi steps (0 = default: every step
 *                  when one sigma application is >= 5 GFLOP, else every 4th step)
 *   "overlap"      1: the K2 chain, the K4 chain and the small sigma terms run on three streams so that
 *                  CTAs of one chain fill the ragged last wave of another; 0 (default): everything on the handle's stream
 *   "profile_gemm" 1: bracket every GEMM-engine launch with CUDA events on the handle's stream (statistics
 *                  "gemm_time_ms", "gemm_flops_timed", "gemm_launches_timed"; implies overlap = 0 while it is on); 0: off (default)
 *   "engine"       0 (default): every contraction on the FP64 tensor-core (DMMA) engine; 1: S6 and S8-S11 on the INT8 tensor pipe
 *                  with FP64 accuracy (gfcc_dgemm_ozaki's scheme; needs ~22 GB more device memory at config 4), the rest on DMMA
 *   "ozaki_slices" digit slices of the INT8 engine, 2..8 (default 7: ~1e-13 per contraction; 6: ~1e-11)
 * Statistics of the INT8 engine: "oz_gemms" (launches), "oz_fail" (1 if a bounded pipeline wait ever timed out; the call that
 * notices it returns GFCC_ECUDA), "oz_time_ms" / "oz_ops_timed" / "oz_flops_timed" / "oz_launches_timed" (with profile_gemm). */
int gfcc_set_option(gfcc_handle h, const char* key, double val);

/* Statistics of the last call (double-valued): "iterations" (Arnoldi steps of the last solve),
 * "sigma_applications", "flops_sigma" (executed FP64 flop model of ONE batched application),
 * "flops_create", "bytes_device" (device memory owned by the handle), "max_relres", "n_unconverged",
 * "gemm_launches", "kernel_launches" (since create or the last reset by reading "reset_counters"),
 * "gmres_m_used" (active restart length of the last solve), "gmres_m_cap" (allocated basis length), "gmres_m_memory_limit"
 * (largest basis the free device memory would allow for the current batch width),
 * "compactions", "refills", "polls", "active_col_steps" (sum over sigma applications of the last solve of the number of
 * right-hand-side columns in the batch) and "lockstep_col_steps" (the same sum had every column stayed until its cycle ended). */
int gfcc_get_stat(gfcc_handle h, const char* key, double* val);
/* per right-hand-side results of the last solve: relres [host][n], iters [host][n], n = np*nw.        */
int gfcc_get_residuals(gfcc_handle h, int n, double* relres, int* iters);

/* relative residual |rotated residual| / ||b|| of right-hand side `rhs` (r = ip*nw + iw) of the last solve after each of
 * its sigma applications: hist[0] = ||b - A x0|| / ||b||, hist[k] after Arnoldi step k (a restart contributes the true residual
 * of its first application).  *n_out [host, nullable] = number of entries available (at most 8192 are kept); the first
 * min(cap, n) are copied to hist [host].  When the solve had more right-hand sides than "max_batch", histories are kept for the
 * tasks that were the last occupants of their batch column.                                                              */
int gfcc_get_residual_history(gfcc_handle h, int rhs, int cap, double* hist, int* n_out);

/* G assembly alone (first, IP term of Eq. 7-8) for caller-provided vectors:
 *   Gout[r][iq] = <Phi|(1+Lambda1+Lambda2) abar_{q[iq]}^+ (X1_r + X2_r)|Phi> = c_q . X_r   complex [nrhs][nq]
 * X1 [nrhs][o], X2 [nrhs][o][o][v] device, layouts of gfcc_sigma_ip (only the i<j half of X2 is read); q [host][nq] in [0,N);
 * Gout host or device.  Linear in X: gfcc_solve_ip's G is this map applied to the solutions.  Synchronous.             */
int gfcc_assemble_g(gfcc_handle h, int nrhs, const void* X1, const void* X2, int nq, const int* q, void* Gout);

/* ---- EA / advanced part (Eq. 4, Eq. 6, second terms of Eq. 7-8) ----
 * Y_q = sum_a y1[a] a+_a + sum_{j, a<b} y2[j,a,b] a+_a a+_b a_j solves (omega - Hbar_N + i eta) Y_q |Phi> = abar_q^+ |Phi>, and
 * G^A_pq = <Phi|(1+Lambda1+Lambda2) abar_p (Y_q1 + Y_q2)|Phi> is the second term of Eq. 8 (the full GFCCSD matrix element is
 * gfcc_solve_ip's G + this G^A).  Working equations: DESIGN.md section 6.8.  Vector layouts: Y1 complex [nrhs][v],
 * Y2 complex [nrhs][o][v][v] with index order (j, a, b), antisymmetric in (a, b) (precondition for inputs, guaranteed for outputs).
 * The first EA call on a handle builds the stored intermediate W_abcj (o v^3 / 2 doubles: this part is meant for sizes where
 * that fits, BASELINE.json configs 0-1) -- GFCC_ENOMEM otherwise.
 *   gfcc_sigma_ea      sigma_r = (omega[r] + i eta) Y_r - Hbar Y_r,  r < nrhs; omega [host]; asynchronous like gfcc_sigma_ip
 *   gfcc_solve_ea(_x)  batched GMRES (the solver of gfcc_solve_ip: CGS2, device Givens, compaction, refill, same options and
 *                      statistics) for every (q = p[iq], omega[iw]), tasks r = iq*nw + iw, and
 *                      G[iw][ip][iq] = G^A_{p[ip], p[iq]}(omega[iw])  complex [nw][np][np] (host or device);
 *                      Y1out/Y2out (nullable, device) receive the solutions in task order
 *   gfcc_assemble_g_ea Gout[r][ip] = c_{p[ip]} . Y_r for caller-provided vectors (complex [nrhs][np], host or device)      */
int gfcc_sigma_ea(gfcc_handle h, int nrhs, const double* omega, double eta, const void* Y1, const void* Y2, void* S1, void* S2);
int gfcc_solve_ea(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol, void* G);
int gfcc_solve_ea_x(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, double tol, void* G,
                    void* Y1out, void* Y2out);
int gfcc_assemble_g_ea(gfcc_handle h, int nrhs, const void* Y1, const void* Y2, int np, const int* p, void* Gout);

/* Copy a named intermediate to a caller buffer (device pointer, FP64), for parity tests:
 *   "Fme" [o][v], "Fmi" [o][o], "Fae" [v][v], "Wmnij" packed [npair(i<j)][npair(m<n)],
 *   "Wmbij" packed [npair(i<j)][v][o] holding W_mbij[m,a,j,i] at [pair(i,j)][a][m], "D" [o][o],
 *   "Lm" [Q][o][v].  Returns the element count (>0), or <0 on error; out may be NULL to query size.   */
long long gfcc_get_intermediate(gfcc_handle h, const char* name, double* out);

/* ---- Model-order reduction (Eq. 9-10, Alg. 1 lines 18-21 PAPER.md:225-228) ----
 * The subspace S = {v_1..v_m} is a REAL orthonormal basis in the packed 1h + 2h1p(i<j) metric, owned by the handle
 * (Eq. 10 writes transposes and Hbar, b, c are real: every complex X contributes Re X and Im X; reading 24).
 *
 * gfcc_mor_reset : (re)allocate an empty subspace with room for m_cap vectors (rounded up to even, at most the
 *   dimension o + o(o-1)/2*v); m_cap = 0 frees it.  Device memory: 2*n*m_cap + m_cap^2 doubles.
 * gfcc_mor_extend: Gram-Schmidt (Alg. 1 line 18) of nx new solutions X1 [nx][o], X2 [nx][o][o][v] (device, complex,
 *   layouts of gfcc_sigma_ip, e.g. the output of gfcc_solve_ip_x) against S, in the order Re X_0, Im X_0, Re X_1, ...;
 *   each candidate is normalised, orthogonalised twice (classical Gram-Schmidt with re-orthogonalisation) and DROPPED
 *   if what is left of its unit norm is <= droptol (or if the subspace is full); then the projection (line 19):
 *   Hbar*v for the accepted vectors by batched sigma at omega = eta = 0 and H^ = S^T Hbar S (new rows and columns).
 *   *m_out [host, nullable] receives the new dimension m.  Synchronous.
 * gfcc_mor_solve : b^ = S^T b_p, c^ = S^T c_q (q over the same list), then for every omega[iw] of the (fine) grid the
 *   reduced system (omega - i eta + H^) X^ = b^ by dense complex LU with partial pivoting (one CTA per frequency),
 *   G[iw][ip][iq] = c^_q^T X^_p  complex [nw][np][np]  and  A[iw] = (1/pi) sum_p Im G[iw][p][p]  (Eq. 9; sign: DESIGN.md
 *   reading 25).  p, omega host; G and A (nullable) may be host or device pointers.  Returns GFCC_ENOCONV if a reduced
 *   matrix is exactly singular.  Synchronous.
 * gfcc_mor_get   : parity hooks.  "m", "cap" return the value; "Hhat" [m][m], "S" [n][m], "HS" (= Hbar S) [n][m] are
 *   copied to `out` (host or device; NULL queries the element count).  Returns the count or a negative error code.    */
int gfcc_mor_reset(gfcc_handle h, int m_cap);
int gfcc_mor_extend(gfcc_handle h, int nx, const void* X1, const void* X2, double droptol, int* m_out);
int gfcc_mor_solve(gfcc_handle h, int np, const int* p, int nw, const double* omega, double eta, void* G, double* A);
long long gfcc_mor_get(gfcc_handle h, const char* name, double* out);

/* ---- Level loop of the retarded GFCCSD workflow (Alg. 1, Eq. 12-13) ----
 * Fine grid w_k = wmin + k*dw, k = 0..n_fine-1 with n_fine = round((wmax-wmin)/dw)+1 (the caller passes it; checked).
 * Level 1 solves Eq. 5 at 3 grid points (both ends and the middle, Eq. 12) for every target p [host][np] with the batched
 * GMRES of gfcc_solve_ip (stop test tol), orthogonalises the solutions into the MOR subspace (droptol), projects, and
 * evaluates G^ and A on the whole fine grid (gfcc_mor_*).  Level L > 1 adds the middle grid points of at most 2^(L-1)
 * intervals between sampled points (Eq. 12): all of them at level 2, afterwards those on which A moved by more than
 * spec_tol * max|A| between the two latest models, largest change first (readings 26-27; the paper cites Ref. 100
 * for the strategy and prints only the counts).  Stops when no interval qualifies, after L_max = floor(log2((wmax-wmin)/dw))
 * levels (Eq. 13) or after max_levels (> 0) levels.  The handle's MOR subspace is reset and left holding the final model.
 * Outputs (host): A [n_fine] spectral function, G [n_fine][np][np] complex (nullable; host or device), level_of [n_fine]
 * (level at which the grid point was sampled, 0 = never), *levels_out, *m_out (nullable).  Synchronous.
 * Returns GFCC_ENOCONV if some GMRES solve stopped at its iteration limit (results are still written).                   */
int gfcc_spectral_adaptive(gfcc_handle h, int np, const int* p, double wmin, double wmax, double dw, double eta,
                           double tol, double spec_tol, int max_levels, double droptol, int n_fine, double* A,
                           void* G, int* level_of, int* levels_out, int* m_out);

const char* gfcc_last_error(gfcc_handle h);
int gfcc_destroy(gfcc_handle h);

/* The FP64 tensor-core GEMM engine every large contraction goes through (exported for unit tests):
 *   C[m,n] = alpha * sum_k A[m,k] B[k,n] + beta * C[m,n],  element addresses
 *   A + m*sAm + k*sAk,  B + k*sBk + n*sBn,  C + m*sCm + n*sCn   (exactly one of sAm/sAk and one of
 *   sBk/sBn must be 1).  DMMA m8n8k4 (mma.sync f64), cp.async multi-stage shared-memory pipeline.     */
int gfcc_dgemm(void* cuda_stream, int M, int N, int K, double alpha, const double* A, long long sAm, long long sAk,
               const double* B, long long sBk, long long sBn, double beta, double* C, long long sCm, long long sCn);

/* Split-K variant of gfcc_dgemm that ALLOCATES NOTHING: for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same product and operand conventions as gfcc_dgemm; K is cut into `splits` chunks
 * (>= 1; more parallelism for tall-skinny-K products such as the sigma1 / Fock-type reductions), each chunk's partial product goes
 * to a scratch buffer and a second kernel reduces them into C = alpha * sum + beta * C (deterministic summation order).
 * The scratch is a file-scope `static __device__` array inside the library of GFCC_NOALLOC_SCRATCH_DOUBLES doubles (16 MiB, held by
 * every GPU that loads the library until the process exits): the call needs  ceil(K / ceil(K/splits)) * M * N  <= that many doubles
 * and returns GFCC_EINVAL with a message in gfcc_last_error(NULL) otherwise (as for any other invalid argument).  It calls no
 * cudaMalloc / cudaFree / allocating library routine; the caller passes inputs and outputs (device pointers) and a stream.
 * EVERY call on a device shares the one array: calls whose kernels may overlap on the GPU (different streams, or graphs replayed
 * concurrently) race on it -- serialise them.  Nothing in the array has to start at zero (every partial element that is read was
 * written by the same call); it keeps the last call's contents.  Asynchronous with respect to the host.                      */
#define GFCC_NOALLOC_SCRATCH_DOUBLES (1LL << 21)
int gfcc_dgemm_splitk_noalloc(void* cuda_stream, int M, int N, int K, double alpha, const double* A, long long sAm, long long sAk,
                              const double* B, long long sBk, long long sBn, double beta, double* C, long long sCm, long long sCn,
                              int splits);

/* FP64-accurate GEMM on the INT8 tensor pipe ("Ozaki-style FP64-accurate GEMM on the low-precision
 * tensor pipes"; the contraction is Eq. 11's pattern).  Same operand conventions as gfcc_dgemm.
 * A's rows and B's columns are scaled by powers of two and cut into `nslices` (1..8) signed 7-bit digit matrices
 * (error-free, int8, K-major); all digit-matrix products of order s+t < nslices run on tcgen05.mma kind::i8 with exact
 * int32 accumulation in TMEM and are added into C in FP64.  Truncation error <= ~2^(-7*nslices) * max|A row| * max|B col|
 * per term (nslices = 7: 2^-49).  Synchronous; scratch is allocated and freed inside.  ms_slice / ms_gemm [host,
 * nullable] receive the CUDA-event times of the slicing passes and of the tensor-core kernel.
 * Returns GFCC_EINVAL (bad sizes/strides), GFCC_ENOMEM, GFCC_ECUDA (launch failure or pipeline time-out).            */
int gfcc_dgemm_ozaki(void* cuda_stream, int M, int N, int K, double alpha, const double* A, long long sAm, long long sAk,
                     const double* B, long long sBk, long long sBn, double beta, double* C, long long sCm, long long sCn,
                     int nslices, double* ms_slice, double* ms_gemm);

/* Roofline denominator of the sigma contractions: measured issue-rate ceiling of the FP64 tensor-pipe instruction
 * the GEMM engine is built on (mma.sync m8n8k4 f64 = SASS DMMA), register-only loop on every SM, CUDA events on
 * `cuda_stream`.  iters: DMMAs per accumulator chain (>= 1; 20000 gives a ~30 ms launch); reps: timed launches
 * (best is returned).  *tflops [host] receives TFLOP/s.  The sigma path of BASELINE.json north_star is a dense FP64
 * contraction, MEASURED_PEAKS.json has no FP64 entry, hence this probe.                 */
int gfcc_probe_fp64_peak(void* cuda_stream, int iters, int reps, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* GFCC_H_ */
