/* wpcd.h -- C ABI of the B200-native (sm_100a) WPCD hot path.
 *
 * Method: wave-packet continuum discretisation for NN scattering, Miller, Ekstrom, Forssen, arXiv:2106.00454
 * (cited below as PAPER.md:<line>, the text under /root/reference).  The four compute calls are the steps (i)-(v)
 * of the paper's recipe:
 *
 *   wpcd_build_channels : steps (i)+V  -- free wave-packet energies (Eqs. 17-19) and the bin-averaged potential
 *                          <x_i|v|x_j> of Eq. 29, H = H0 + V per channel and potential sample
 *   wpcd_diag_batched   : step (ii)    -- H = C D C^T, Eq. 21, batched block-Jacobi
 *   wpcd_onshell_T      : steps (iii)-(v) -- pseudostate bin edges Eq. 23, analytic resolvent
 *                          Eqs. B.3-B.6, on-shell T of Eq. 32/39/27
 *   wpcd_phase_shifts   : S = 1 - 2 pi i T/dE (Eq. A.3 with the wave-packet normalisation of Eq. 25, PAPER.md:490,
 *                          196, 257), phase shifts by Eqs. A.4-A.5
 *
 * Conventions
 *   - fp64 everywhere.  Momenta fm^-1, energies MeV.  E = cE p^2, cE = hbarc^2/(2 mu)  (E = p^2/m_N).
 *   - Bins are 0-based: bin i = [p_i, p_{i+1}], i = 0..N-1.  Momentum wave packets f(k)=1, N_i = Delta k_i.
 *   - Matrices are row-major, batches are strided ("stored congruently"): element (b,i,j) at
 *     base[(b*n + i)*n + j].  Uncoupled channels have n = N; coupled channels n = 2N with row index alpha*N + i,
 *     alpha = 0 for l = J-1 and 1 for l = J+1, the SAME H0 in both blocks (degenerate bases).
 *   - Pointers named d_* are DEVICE pointers, h_* (and all struct members) are HOST pointers.  Every buffer is
 *     caller-allocated and caller-owned; the library allocates nothing after wpcd_create (workspace is passed in,
 *     its size comes from the *_workspace_bytes queries).  Device buffers must be 16-byte aligned.
 *   - Every compute call is asynchronous on `stream` (a cudaStream_t passed as void*, NULL = default stream) and
 *     does not synchronise with the host.  Host-side tables in the structs are read before the call returns.
 *   - Return value: WPCD_OK or a negative error code; argument errors are detected before any launch.
 *     No exceptions, no errno, no global state.  There is no CPU fallback anywhere in this library.
 */
#ifndef WPCD_H
#define WPCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WPCD_OK 0
#define WPCD_EINVAL (-1) /* bad argument (NULL pointer, non-positive size, unsorted edges, ...) */
#define WPCD_ESIZE (-2)  /* size not supported (n < 2, too many channels/terms for the tables) */
#define WPCD_EWORK (-3)  /* workspace too small */
#define WPCD_ECUDA (-4)  /* CUDA runtime / launch failure (see wpcd_last_cuda_error) */

#define WPCD_MAX_CHANNELS 16
#define WPCD_MAX_TERMS 4
#define WPCD_MAX_L 6 /* largest orbital angular momentum l (coupled channels use l = J+1): the range over which the Q_l
                        evaluation is held to 1e-12 of an independent one (reading C7); beyond: WPCD_ESIZE */

/* Local potential = sum of Yukawas V(r) = sum_t V0_t exp(-mu_t r)/r, projected on partial wave l with the Legendre
 * function of the second kind: <k'|v_l|k> = (1/pi) sum_t V0_t Q_l(z_t)/(k'k), z_t = (k'^2+k^2+mu_t^2)/(2k'k)
 * (convention B of DESIGN.md reading C1).  Coupled channels add the symmetric off-diagonal block
 * (1/pi) VT Q_J(z_T)/(k'k) (reading C8).  kind 1: separable Yamaguchi <k'|v|k> = -lambda g(k')g(k),
 * g = 1/(k^2+beta^2) (uncoupled only; lambda in convention B, MeV fm^-1). */
typedef struct {
  int kind;             /* 0 = Yukawa sum, 1 = Yamaguchi */
  int n_terms;          /* kind 0: number of Yukawa terms, 1..WPCD_MAX_TERMS */
  const double* V0;     /* [n_terms] strengths, MeV fm (sign included: repulsive > 0) */
  const double* mu;     /* [n_terms] ranges, fm^-1 */
  const int* scale_idx; /* [n_terms] column of d_scales multiplying V0_t for each sample, or -1 (NULL = all -1) */
  double VT, muT;       /* coupled-channel off-diagonal Yukawa: strength MeV fm, range fm^-1 */
  int VT_scale_idx;     /* column of d_scales multiplying VT, or -1 */
  double lambda, beta;  /* kind 1 */
} wpcd_potential;

typedef struct {
  int coupled; /* 0: uncoupled channel of orbital angular momentum lJ; 1: coupled l = J-1, J+1 with J = lJ >= 1 */
  int lJ;
} wpcd_channel;

typedef struct {
  int N;                 /* number of wave packets */
  const double* h_edges; /* [N+1] bin edges p_0 < p_1 < ... < p_N, fm^-1, p_0 >= 0 */
  double hbarc, mu;      /* MeV fm, MeV (reduced mass) */
  int n_gl;              /* Gauss-Legendre points per bin for Eq. 29, 1..16 (BASELINE configs: 8; 1 = mid-point rule, Eq. 30) */
  int wp_kind;           /* 0: momentum wave packets f(k) = 1, N_i = Delta k_i (the configs, the paper's choice);
                            1: energy wave packets f(k) = hbarc sqrt(k/mu), N_i = Delta E_i: H0 is Eq. 18
                               exactly, e_i = E_i + dE_i/2, and Eq. 29 carries the extra factor f(k')f(k) */
} wpcd_grid;

/* Handle: owns only immutable device tables.  One handle per host thread/stream.  device = CUDA ordinal.
 * Every compute call launches on the CALLER's current device and stream: the current device (cudaGetDevice) must be the
 * handle's device, else the call returns WPCD_EINVAL before any launch. */
int wpcd_create(void** handle, int device);
void wpcd_destroy(void* handle);
const char* wpcd_strerror(int code);
const char* wpcd_last_cuda_error(void* handle); /* text of the last CUDA error seen by this handle ("" if none) */
int wpcd_num_sms(void* handle);

/* Workspace sizes in bytes (0 is a valid answer). */
size_t wpcd_build_workspace_bytes(void* handle, int N, int n_chan);
size_t wpcd_diag_workspace_bytes(void* handle, int n, int batch);
size_t wpcd_onshell_workspace_bytes(void* handle, int N, int coupled, int batch, int nE);

/* Steps (i) + Eq. 29.  For every sample s = 0..S-1 and channel c of the list builds H = H0 + V.
 *   d_scales : [S][P] per-sample multiplicative scales (reading C14), or NULL with P = 0 (then S must be 1 or all
 *              samples are identical).  Strength t of sample s is V0_t * d_scales[s][scale_idx[t]].
 *   d_H_unc  : [S][n_unc][N][N]   (n_unc = number of uncoupled channels, list order), may be NULL if n_unc = 0
 *   d_H_cpl  : [S][n_cpl][2N][2N] (n_cpl = number of coupled channels, list order),   may be NULL if n_cpl = 0
 *   d_e0     : [N]   FWP kinetic energies e_i = cE (p_i^2 + p_i p_{i+1} + p_{i+1}^2)/3 (reading C4; energy packets:
 *                      cE (p_i^2 + p_{i+1}^2)/2, Eq. 18)
 *   d_dE     : [N]   FWP bin energy widths,  d_Eedge : [N+1] bin edges in energy (cE p_i^2)
 * The basis matrices (one per distinct (l, mu_t)) are built in the workspace by an 8x8-point (n_gl x n_gl)
 * Gauss-Legendre rule per bin pair and combined per sample with coalesced, vectorised stores.  H is exactly
 * symmetric.  V is not stored: V = H - diag(e0) (wpcd_onshell_T recomputes it on the fly). */
int wpcd_build_channels(void* handle, const wpcd_grid* grid, const wpcd_potential* pot, const wpcd_channel* chan,
                        int n_chan, const double* d_scales, int S, int P, double* d_H_unc, double* d_H_cpl,
                        double* d_e0, double* d_dE, double* d_Eedge, void* d_work, size_t work_bytes, void* stream);

/* Step (ii), Eq. 21.  Batched real-symmetric eigendecomposition by two-sided block-Jacobi, one CTA per matrix: 8-wide
 * blocks paired in a round-robin tournament; each 16x16 pivot sub-problem gets one parallel-ordered (Brent-Luk) Jacobi
 * sweep inside one warp -- all 120 pairs at about three steps per sweep, the 64 pairs between the two blocks otherwise; the
 * accumulated rotations are applied to H and C as fp64 tensor-core (DMMA) tile products; the pivots of the next step
 * are solved while the current step's updates run.  Rows and columns are taken in the order of descending diagonal
 * entries (a relabelling; one to two sweeps fewer on these graded matrices).  n <= 200: the matrix (upper 8x8 blocks) in shared memory, the
 * eigenvectors in an L2-resident workspace, 1-4 matrices in flight per SM; 200 < n <= 848: the matrix through L2, the
 * eigenvectors not accumulated during the sweeps at all -- the 16x16 rotation products are logged (workspace) and replayed
 * panel by panel in shared memory into d_C by the same persistent launch (bit-identical to the accumulation in place, a
 * tenth of its DRAM traffic; the workspace then holds two log regions per SM: ~3 GB at n = 300, ~20 GB at n = 800);
 * larger n: matrix and eigenvectors through the workspace.
 *   d_A    : [batch][n][n] input (only read; must be symmetric)
 *   d_W    : [batch][n] eigenvalues ascending
 *   d_C    : [batch][n][n] eigenvectors, column k belongs to d_W[k]  (C_ij = <x_i|z_j>)
 *   d_info : [batch] sweeps used (>= 1), or -1 if not converged in max_sweeps (-2 for every matrix: the scheduler of the
 *            200 < n <= 848 path gave up waiting -- a safety net that has never been seen to fire; the results are then invalid)
 *   tol    : a pivot is rotated iff |a_pq| > tol sqrt(|a_pp a_qq|); convergence = a full sweep without rotation.
 *            tol <= 0 selects the default 2^-52.
 *   h_rows : optional HOST array of n_ranges (<= 4) half-open row ranges [lo, hi) of C that the caller needs (NULL,
 *            0 = all rows).  C <- C J acts on the rows independently, so rows that share no 8-row block of the
 *            internal ordering with a wanted row are not updated; every row outside the ranges is returned as ZEROS;
 *            the eigenvalues and the wanted rows are unaffected (bit-identical to the full run).  The on-shell T of
 *            the n <= 200 path only reads the rows of the on-shell bins.
 *   d_work : wpcd_diag_workspace_bytes(n, batch) bytes (never 0: the schedule tables live there; gigabytes for 200 < n <= 848)
 * Test hook (csrc/jacobi.cu): the environment variable WPCD_JACOBI_LOG_SWEEPS, read at every call of this function and of
 * wpcd_diag_workspace_bytes, sets the capacity of a log region in sweeps (default 7; 0 = the 200 < n <= 848 path accumulates the
 * eigenvectors in the workspace as the larger sizes do, 1 = every matrix overflows its log and is redone by the fallback launch).
 * The results do not depend on it (bit-identical, tests/test_gpu_parity.py). */
int wpcd_diag_batched(void* handle, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                      double tol, int max_sweeps, const int* h_rows, int n_ranges, void* d_work, size_t work_bytes,
                      void* stream);

/* wpcd_diag_batched for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same kernels on the same arguments, Eq. 21, with the workspace taken from a
 * file-scope device array of WPCD_STATIC_WORK_BYTES inside the library instead of d_work.  The call allocates nothing
 * (no cudaMalloc / cudaFree / allocating library routine; the array's device address is looked up once per device, at
 * the first call on that device).  Every GPU that loads the library holds the array until the process exits.
 *   - sizes: wpcd_diag_workspace_bytes(handle, n, batch) must be <= WPCD_STATIC_WORK_BYTES, else WPCD_ESIZE before any
 *     launch (wpcd_last_cuda_error then holds the sizes).  16 MiB cover n <= 32 at any batch, n = 100 up to batch 193,
 *     n = 200 up to batch 52 -- one potential sample of the paper's channel list -- not the production batches.
 *   - ALL calls on a device share the one array: two calls that overlap on the GPU (different streams, or graphs replayed
 *     concurrently) race and give wrong results; calls in one stream are ordered and safe.  The array keeps the previous
 *     call's contents; nothing in it needs clearing by the caller: the schedule tables and the work counter are rewritten
 *     by the first kernel of every call and each CTA initialises its own eigenvector workspace per matrix.
 *   - results are those of wpcd_diag_batched (same grid, same kernels); all other arguments as there. */
#define WPCD_STATIC_WORK_BYTES (16u << 20)
int wpcd_diag_batched_static(void* handle, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                             double tol, int max_sweeps, const int* h_rows, int n_ranges, void* stream);

/* Steps (iii)-(v).  For every matrix b and energy e: FWP bin i(e) with Eedge_i <= E_e < Eedge_{i+1}, then
 *   uncoupled: T_ii(E) = V_ii + sum_b (VC)_ib^2/(E - eps_b) + sum_k (VC)_ik^2 g_k(E)
 *   coupled  : T^{ab}(E) = V_{(a i)(b i)} + sum_k (VC)_{(a i)k} g_k(E) (VC)_{(b i)k},  a,b in {0,1}
 * with g_k(E) = [ln|(E-lo_k)/(E-hi_k)| - i pi 1{lo_k <= E < hi_k}]/(hi_k - lo_k) (readings G2, C11), edges from
 * Eq. 23 as printed (C5), negative eigenvalues = bound states, positive eigenvalues of coupled channels alternate
 * between two branches by rank (C6).  VC = (H - diag(e0)) C is formed for the on-shell rows only; for n <= 200 through
 * the identity (VC)_ik = C_ik (eps_k - e_i) (H C = C D, H0 diagonal), which needs no product at all.
 *   d_H, d_W, d_C : as given to / returned by wpcd_diag_batched (n = N or 2N)
 *   d_Ecm  : [nE] c.m. energies, MeV
 *   mode   : 0 = point-wise resolvent g_k(E) above;
 *            1 = energy-averaged resolvent, Eq. 28 and B.7-B.8 (sign per reading G3): ONE T per
 *                on-shell FWP bin i, returned for every energy of that bin.  State k of branch beta is
 *                averaged over the pseudostate bin [a,b] of the i-th positive state of the same branch:
 *                Re = W/((b-a)(hi_k-lo_k)), W = (b-lo)ln|b-lo| - (b-hi)ln|b-hi| - (a-lo)ln|a-lo| + (a-hi)ln|a-hi|,
 *                Im = -pi/(hi_k-lo_k) for that i-th state only; bound states ln|(b-eps)/(a-eps)|/(b-a) over branch 0's
 *                bin; T = 0 if a branch has no i-th state (readings A1-A3)
 *   d_T    : [batch][nE][2] (re,im) or [batch][nE][2][2][2] for coupled;  zero where E is outside the grid
 *   d_bin  : [nE] FWP bin of each energy (-1 if outside the grid) */
int wpcd_onshell_T(void* handle, int N, int coupled, int batch, const double* d_e0, const double* d_Eedge,
                   const double* d_H, const double* d_W, const double* d_C, const double* d_Ecm, int nE, int mode,
                   double* d_T, int* d_bin, void* d_work, size_t work_bytes, void* stream);

/* Eqs. A.3-A.5.  S = 1 - 2 pi i T/dE_bin.  Uncoupled: delta = atan2(Im S, Re S)/2 in degrees, (-90, 90].
 * Coupled (Stapp): delta_- = arg(S_11)/2, delta_+ = arg(S_22)/2, eps = atan2(Re[-i S_12 e^{-i(d- + d+)}], |S_11|)/2.
 *   d_delta : [batch][nE] or [batch][nE][3] = (delta_-, delta_+, eps), degrees
 *   d_S     : optional (may be NULL) S-matrix, same layout as d_T */
int wpcd_phase_shifts(void* handle, int coupled, int batch, int nE, const double* d_T, const int* d_bin,
                      const double* d_dE, double* d_delta, double* d_S, void* stream);

/* Host helper (no GPU work): the row ranges of C that wpcd_onshell_T will read for the c.m. energies h_Ecm [nE] (HOST
 * array) on this grid, to be handed to wpcd_diag_batched as h_rows.  h_rows must hold 8 ints; *n_ranges comes back as
 * 0 when all rows are needed (the direct-product path of large n). */
int wpcd_onshell_rows(const wpcd_grid* grid, int coupled, const double* h_Ecm, int nE, int* h_rows, int* n_ranges);

/* Eq. 42, the second half of the paper's production variant (energy-averaged T per bin, then linear
 * interpolation between the bin mid-points): phase shifts at arbitrary momenta from the mid-point values.
 *   d_pedge     : [N+1] momentum bin edges, fm^-1 (device);  mid-points qbar_i = (p_i + p_{i+1})/2 (Eq. 43, n = m/2)
 *   d_delta_mid : [batch][N] or [batch][N][3] phases at the mid-points, degrees -- e.g. wpcd_onshell_T(mode 1) and
 *                 wpcd_phase_shifts evaluated at the N energies cE qbar_i^2
 *   d_q         : [nq] target momenta, fm^-1;  d_out : [batch][nq] or [batch][nq][3], degrees, delta in (-90, 90]
 * For q in bin i the line through the mid-points of bins i-1 and i, as printed (bin 0: bins 0 and 1); q outside the grid
 * gives NaN.  The mid-point phases are first made continuous: delta_i is shifted by the multiple of 180 degrees that
 * brings it within 90 degrees of delta_{i-1}, eps_J changes sign with every odd shift (readings I1-I2). */
int wpcd_interp_phases(void* handle, int coupled, int batch, int N, const double* d_pedge, const double* d_delta_mid,
                       const double* d_q, int nq, double* d_out, void* stream);

/* Total neutron-proton cross section from the on-shell T of all partial waves, Appendix A
 * (PAPER.md:473-537): S = 1 - 2 pi i T/dE_bin (Eq. A.3), spin-scattering matrix at theta = 0 (Eq. A.2), Saclay amplitudes
 * a, b (Eq. A.9), sigma_tot = (2 pi/p) Im(a + b) (Eq. A.11).  At theta = 0 the spin trace a + b collapses the
 * Clebsch-Gordan sums, so the kernel evaluates the equivalent partial-wave sum
 *   sigma_tot(E) = (pi/(2 p^2)) sum_channels (2J+1) sum_l Re(1 - S_ll),   p^2 = E_cm/cE,
 * every Pauli-allowed partial wave with weight 1 (np scattering, reading X1).
 *   h_J_unc : [n_unc] HOST, total angular momentum J of every uncoupled channel (e.g. 3P0: J = 0), list order
 *   h_J_cpl : [n_cpl] HOST, J >= 1 of every coupled channel
 *   d_T_unc : [S][n_unc][nE][2], d_T_cpl : [S][n_cpl][nE][2][2][2] -- as written by wpcd_onshell_T for batch = S x channels
 *             (NULL allowed when the count is 0);  d_bin, d_dE, d_Ecm as for wpcd_phase_shifts / wpcd_onshell_T.
 *             d_bin = d_dE = NULL: the two arrays hold S-MATRICES instead (same layout, e.g. from wpcd_mi_solve) and
 *             Re(1 - S_ll) is taken from them directly (no energy is then outside a grid)
 *   d_sigma : [S][nE] millibarn (1 fm^2 = 10 mb); NaN where the energy is outside the grid
 * n_unc, n_cpl <= WPCD_MAX_CHANNELS. */
int wpcd_sigma_tot(void* handle, int S, int nE, int n_unc, const int* h_J_unc, const double* d_T_unc, int n_cpl,
                   const int* h_J_cpl, const double* d_T_cpl, const int* d_bin, const double* d_dE, const double* d_Ecm,
                   double hbarc, double mu, double* d_sigma, void* stream);

/* The matrix-inversion (MI) method of Sec. 2.1 batched over (sample, channel, energy) -- the paper's
 * comparison method as a second workload.  One CTA per Lippmann-Schwinger system:
 * basis {k_1..k_NQ, p} with Gauss-Legendre nodes mapped k_j = cmap tan(pi(1+x_j)/4) (Eq. 4), propagator vector D derived
 * from Eqs. 2-4 (reading C3), F = 1 - V diag(D) (Eq. 7), F T = V (Eq. 6) solved in the K-matrix form the paper
 * recommends (Eq. 38): the principal-value part F_r K = V in REAL arithmetic by Gauss elimination with partial
 * pivoting in shared memory, then T_on = K_on (1 + i f p K_on)^-1 and S = 1 - 2 i f p T, f = 2 mu/hbarc^2.  The potential is the same wpcd_potential as for
 * wpcd_build_channels, used in convention A: v_l = sum_t V0_t Q_l(z_t)/(2k'k) (Yamaguchi: lambda_A = (pi/2) lambda).
 *   NQ      : quadrature points; the system has NQ+1 (coupled: 2(NQ+1)) real rows, one thread per row: NQ <= 255
 *             uncoupled, NQ <= 127 coupled, else WPCD_ESIZE.  Up to NQ = 164 / 81 it lives in one CTA's shared memory,
 *             above in an L2-resident region of the workspace per CTA (a fixed grid of CTAs loops over the systems)
 *   d_Ecm   : [nE] c.m. energies, MeV (p = sqrt(E_cm/cE))
 *   d_S_unc : [S][n_unc][nE][2]        S-matrix (re,im), list order of the uncoupled channels
 *   d_S_cpl : [S][n_cpl][nE][2][2][2]  S-matrix of the coupled channels
 *   d_work  : wpcd_mi_workspace_bytes(NQ) bytes */
size_t wpcd_mi_workspace_bytes(void* handle, int NQ);
int wpcd_mi_solve(void* handle, const wpcd_potential* pot, const wpcd_channel* chan, int n_chan, const double* d_scales, int S,
                  int P, int NQ, double cmap, double hbarc, double mu, const double* d_Ecm, int nE, double* d_S_unc,
                  double* d_S_cpl, void* d_work, size_t work_bytes, void* stream);

/* Measurement aid (bench.py "roofline.peak_measured"): one launch of register-only fp64 chains on every SM -- kind 0: eight
 * independent DFMA chains per thread, kind 1: eight independent mma.sync.m8n8k4.f64 accumulator chains per warp --
 * `iters` dependent steps each, 2 CTAs of 512 threads per SM.  The caller times the launch with events on `stream`.
 *   d_sink  : [wpcd_probe_sink_elems(handle)] doubles, written once at the end (keeps the chains alive)
 *   h_flops : host out, flops executed by the launch (FMA = 2) */
size_t wpcd_probe_sink_elems(void* handle);
int wpcd_probe_fp64(void* handle, int kind, int iters, double* d_sink, double* h_flops, void* stream);

/* Test hooks (host only, no GPU needed): the block tournament that wpcd_diag_batched runs (csrc/jacobi_schedule.cuh).
 * m = number of players (8-wide blocks, even, >= 6; players >= nb are padding), a sweep has m-1 steps of m/2 slots.
 *   wpcd_jacobi_schedule      : blocks (I < J) of slot s at step t; J = -1 single block, I = J = -1 empty slot.
 *   wpcd_jacobi_critical_slot : if the tile of slots (s1 < s2) at step t holds the off-diagonal block of a real
 *                               pivot of step tn, that pivot's slot at step tn, else -1 (WPCD_EINVAL on bad input).
 * Invariants (tests/test_abi_cpu.py): every pair of blocks meets exactly once per sweep; at most one pivot per tile. */
int wpcd_jacobi_schedule(int m, int nb, int t, int s, int* I, int* J);
int wpcd_jacobi_critical_slot(int m, int nb, int t, int tn, int s1, int s2);

#ifdef __cplusplus
}
#endif
#endif /* WPCD_H */
