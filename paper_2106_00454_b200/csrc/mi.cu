// mi.cu -- the matrix-inversion (MI) method of Sec. 2.1 on the GPU, batched over
// (sample, channel, energy): the second workload of SURVEY 8(f)-4 ("the MI method ... can be parallelised over the
// on-shell energies").  One CTA per Lippmann-Schwinger system:
//   basis q = {k_1..k_NQ, p}: Gauss-Legendre nodes mapped k_j = c tan(pi(1+x_j)/4), w_j -> c (pi/4) w_j/cos^2(.), plus the
//   on-shell momentum p = sqrt(E_cm/cE)                                                    (Eq. 4)
//   D_j = (2/pi) w_j k_j^2 f/(p^2-k_j^2),  D_{NQ+1} = -(2/pi) f p^2 sum_j w_j/(p^2-k_j^2) - i f p,  f = 2 mu/hbarc^2
//   (derived from Eqs. 2-4, reading C3: the printed Eq. 5 is inconsistent)
//   F = 1 - V diag(D) (Eq. 7), F T = V (Eq. 6), solved as the real K-matrix system plus the on-shell rank-nc correction
//   (Eq. 38; see k_mi_solve), S = 1 - 2 i f p T_onshell (convention A, reading C2).
// Potential in convention A: v_l(k',k) = sum_t V0_t Q_l(z_t)/(2k'k); coupled channels: blocks l = J-1, J+1 and the
// off-diagonal Yukawa V_T Q_J(z_T)/(2k'k) (reading C8); Yamaguchi -lambda_A g(k')g(k).
#include <math.h>
#include "legendre_q.cuh"
#include "wpcd_internal.cuh"

namespace {

constexpr int kMiThreads = 256;
constexpr int kMiWarps = kMiThreads / 32;   // one thread per row in the panel factorisation: n <= 166 < 256

struct MiParams {
  const double* kq;      // [NQ] grid momenta
  const double* wq;      // [NQ] grid weights
  const double* Ecm;     // [nE]
  const double* scales;  // [S][P] or nullptr
  double* Sout;          // [S][nch][nE][nc][nc][2]
  int NQ, nE, P, nch, coupled;
  int lJ[WPCD_MAX_CHANNELS];
  int kind, nterms;
  double V0[WPCD_MAX_TERMS], mu[WPCD_MAX_TERMS];
  int sidx[WPCD_MAX_TERMS];
  double VT, muT;
  int VT_sidx;
  double lambdaA, beta;
  double hbarc, mured;
  const double* basis;                                   // [nbasis][NQ][NQ]: Q_l(z(k_i,k_j))/(2 k_i k_j) per distinct (l, mu)
  const double* onb;                                     // [chunk energies][nbasis][NQ+1]: the same for (p, k_j), j = NQ: (p, p)
  int nbasis, e_first;                                   // this launch covers energies e_first .. e_first + gridDim.x - 1
  int id_mm[WPCD_MAX_CHANNELS][WPCD_MAX_TERMS];           // basis matrix of term t in the block l = lJ (uncoupled) / J-1
  int id_pp[WPCD_MAX_CHANNELS][WPCD_MAX_TERMS];           // ... in the block l = J+1
  int id_mp[WPCD_MAX_CHANNELS];                           // ... of the off-diagonal Yukawa
  double* fwork;                                         // L2 variant: [gridDim.x][n][ld] systems of the CTAs (else unused)
  int ne, S;                                             // energies of this launch, samples
};

struct MiBasisTable { int n; int l[WPCD_MAX_CHANNELS * (2 * WPCD_MAX_TERMS + 1)]; double mu[WPCD_MAX_CHANNELS * (2 * WPCD_MAX_TERMS + 1)]; };

// The grid x grid part of V does not depend on the energy or the sample: one matrix per distinct (l, mu), computed once
// per call; only the on-shell row and column are evaluated per system.
__global__ void k_mi_basis(int NQ, MiBasisTable tab, const double* __restrict__ kq, double* __restrict__ basis) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= NQ * NQ) return;
  const int i = idx / NQ, j = idx - i * NQ;
  const double kp = kq[i], k = kq[j], mu = tab.mu[blockIdx.y];
  const double diff = kp - k;
  const double zm1 = fma(diff, diff, mu * mu) / (2.0 * kp * k);
  basis[(size_t)blockIdx.y * NQ * NQ + idx] = legendre_q(tab.l[blockIdx.y], zm1) / (2.0 * kp * k);
}

// The on-shell row/column of V depends on the energy but not on the sample or the channel beyond (l, mu): one table per
// (energy of the chunk, distinct (l, mu)), entries j < NQ for (p, k_j), entry NQ for (p, p).  grid (chunk, nbasis).
__global__ void k_mi_onbasis(int NQ, MiBasisTable tab, const double* __restrict__ kq, const double* __restrict__ Ecm, int e_first,
                             double cE, double* __restrict__ onb) {
  const int j = threadIdx.x, b = blockIdx.y;
  if (j > NQ) return;
  const double p = sqrt(Ecm[e_first + blockIdx.x] / cE), k = j < NQ ? kq[j] : p, mu = tab.mu[b];
  const double diff = p - k;
  const double zm1 = fma(diff, diff, mu * mu) / (2.0 * p * k);
  onb[((size_t)blockIdx.x * gridDim.y + b) * (NQ + 1) + j] = legendre_q(tab.l[b], zm1) / (2.0 * p * k);
}

// k_j, w_j of the MI grid: root a of P_NQ by Newton, mapped with c tan(pi(1+x)/4)
__global__ void k_mi_grid(int NQ, double cmap, double* __restrict__ kq, double* __restrict__ wq) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= NQ) return;
  double x = -cos(WPCD_PI * (a + 0.75) / (NQ + 0.5)), dp = 1.0;
  for (int it = 0; it < 100; ++it) {
    double pm = 1.0, pc = x;
    for (int k = 2; k <= NQ; ++k) { double pn = ((2 * k - 1) * x * pc - (k - 1) * pm) / k; pm = pc; pc = pn; }
    dp = NQ * (x * pc - pm) / (x * x - 1.0);
    const double dx = pc / dp;
    x -= dx;
    if (fabs(dx) < 1e-16) break;
  }
  {
    double pm = 1.0, pc = x;
    for (int k = 2; k <= NQ; ++k) { double pn = ((2 * k - 1) * x * pc - (k - 1) * pm) / k; pm = pc; pc = pn; }
    dp = NQ * (x * pc - pm) / (x * x - 1.0);
  }
  const double w = 2.0 / ((1.0 - x * x) * dp * dp);
  const double ang = WPCD_PI * (1.0 + x) / 4.0, c = cos(ang);
  kq[a] = cmap * tan(ang);
  wq[a] = cmap * (WPCD_PI / 4.0) * w / (c * c);
}

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {  // D (8x8) += A (8x4, row) B (4x8, col), fp64 tensor core
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cdiv(double2 a, double2 b) {
  const double d = b.x * b.x + b.y * b.y;
  return make_double2((a.x * b.x + a.y * b.y) / d, (a.y * b.x - a.x * b.y) / d);
}

// grid (nE, nch, S); dynamic shared memory: F [n][ld] (ld = n + nc: the right-hand sides ride along), q [M], D [M], row flags.
//
// K-matrix form ("it is numerically more stable to first introduce the K-matrix as the principal value part of the
// LS equation ... a set of purely real matrix-equations", Eq. 38: a quarter of the complex flops).  The only
// complex entry of D is the on-shell one, D_{NQ+1} = D_r - i f p (reading C3), so F = F_r + i f p u e^T with F_r = 1 - V diag(D_r)
// real and u the on-shell column(s) of V: solve F_r K = u in real arithmetic (Gauss elimination with partial pivoting, the
// pivoting implicit through row flags: no row swaps, two barriers per column), then T_on = K_on (1 + i f p K_on)^-1
// (Sherman-Morrison for the rank-nc term) and S = 1 - 2 i f p T_on.  Same S as the complex elimination of Eqs. 6-7, which the
// oracle performs, up to rounding.  The unknowns are ordered grid points first (block by block), on-shell points last, so that
// K_on falls out of the last nc pivots without a back substitution over the grid.
// kGlob: systems too large for shared memory (coupled N_Q > 81, uncoupled N_Q > 164; n <= 256 rows: one thread per row)
// keep F in a per-CTA region of the workspace that stays in L2; the grid is then a fixed number of CTAs that loop over the
// systems.  Same code otherwise (the barriers of a CTA order its global accesses too).
template <bool kGlob>
__global__ void __launch_bounds__(kMiThreads) k_mi_solve(MiParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = blockDim.x, nwarps = nthr >> 5;  // nthr >= n (mi_threads)
  const int NQ = P.NQ, M = NQ + 1, nc = P.coupled ? 2 : 1, n = nc * M, ld = (n + nc + 1) & ~1, ng = nc * NQ;  // ld even: 16-byte row pairs
  double* F = kGlob ? P.fwork + (size_t)blockIdx.x * n * ld : reinterpret_cast<double*>(smem_raw);       // [n][ld]
  double* q = kGlob ? reinterpret_cast<double*>(smem_raw) : F + (size_t)n * ld;                         // [M]
  double* D = q + M;                                      // [M] real parts (principal value)
  int* prow = reinterpret_cast<int*>(D + M);              // [n] pivot row of column c
  int* lst = prow + n;                                    // [2][n] rows not yet used as a pivot (double buffered)
  __shared__ double sV0[WPCD_MAX_TERMS], sVT;
  __shared__ unsigned ckey[2 * kMiWarps];                 // pivot candidate of every warp (double buffered over the columns): its key,
  __shared__ int cpos[2 * kMiWarps];
  __shared__ double pb[2 * kMiWarps * 8];                 // ... and the panel entries of that row
  __shared__ int pivpos[8];                               // list positions of the panel's pivot rows
  const int nsys = kGlob ? P.ne * P.nch * P.S : 1;
  for (int sys = kGlob ? blockIdx.x : 0; sys < nsys; sys += gridDim.x) {
  const int el = kGlob ? sys % P.ne : blockIdx.x;                       // energy within the launch's chunk
  const int ch = kGlob ? (sys / P.ne) % P.nch : blockIdx.y;
  const size_t smp = kGlob ? sys / (P.ne * P.nch) : blockIdx.z;
  const int e = P.e_first + el;
  const double cE = P.hbarc * P.hbarc / (2.0 * P.mured), f = 2.0 * P.mured / (P.hbarc * P.hbarc);
  const double p = sqrt(P.Ecm[e] / cE);
  if (tid < P.nterms) {
    double v = P.V0[tid];
    if (P.scales && P.sidx[tid] >= 0) v *= P.scales[smp * P.P + P.sidx[tid]];
    sV0[tid] = v;
  }
  if (tid == 0) {
    double v = P.VT;
    if (P.scales && P.VT_sidx >= 0) v *= P.scales[smp * P.P + P.VT_sidx];
    sVT = v;
    q[NQ] = p;
  }
  for (int j = tid; j < NQ; j += nthr) {
    const double k = P.kq[j];
    q[j] = k;
    D[j] = (2.0 / WPCD_PI) * P.wq[j] * k * k * f / (p * p - k * k);
  }
  __syncthreads();
  if (tid == 0) {
    double ssum = 0.0;
    for (int j = 0; j < NQ; ++j) ssum += P.wq[j] / (p * p - q[j] * q[j]);
    D[NQ] = -(2.0 / WPCD_PI) * f * p * p * ssum;   // the principal-value part; the -i f p part enters after the solve
  }
  __syncthreads();
  // V on the basis, F_r = 1 - V diag(D_r), right-hand sides = on-shell columns of V.  Index r < ng: grid point r % NQ of
  // block r / NQ; r >= ng: on-shell point of block r - ng.
  // A warp per row, lanes along the columns; every Yukawa element comes from the tables (grid x grid: basis, per call;
  // row/column of the on-shell point: onb, per energy), scaled by this sample's strengths.
  const double* onb = P.onb + (size_t)el * P.nbasis * M;
  const size_t nn = (size_t)NQ * NQ;
  for (int r = warp; r < n; r += nwarps) {
    const int a = r < ng ? r / NQ : r - ng, i = r < ng ? r - a * NQ : NQ;
    double* Fr = F + (size_t)r * ld;
    for (int c = lane; c < n; c += 32) {
      const int b = c < ng ? c / NQ : c - ng, j = c < ng ? c - b * NQ : NQ;
      double v;
      if (P.kind == 1) {
        v = -P.lambdaA / ((q[i] * q[i] + P.beta * P.beta) * (q[j] * q[j] + P.beta * P.beta));
      } else {
        const bool gg = i < NQ && j < NQ;
        const size_t o = gg ? (size_t)i * NQ + j : (size_t)(i < j ? i : j);   // on-shell tables: index of the grid point (NQ: p itself)
        v = 0.0;
        if (a == b) {
          const int* id = (P.coupled && a == 1) ? P.id_pp[ch] : P.id_mm[ch];
          for (int t = 0; t < P.nterms; ++t) v += sV0[t] * (gg ? P.basis[id[t] * nn + o] : onb[id[t] * M + o]);
        } else {
          v = sVT * (gg ? P.basis[P.id_mp[ch] * nn + o] : onb[P.id_mp[ch] * M + o]);
        }
      }
      Fr[c] = (r == c ? 1.0 : 0.0) - v * D[j];
      if (j == NQ) Fr[n + b] = v;
    }
    if (lane == 0 && ld > n + nc) Fr[ld - 1] = 0.0;   // padding column
  }
  __syncthreads();
  // Blocked Gauss elimination with partial pivoting (right-looking, panels of 8 columns):
  //   (1) the panel is factorised in registers, one thread per row still to be eliminated, one barrier per column (the
  //       arg-max candidates of the warps travel with their rows' panel entries); multipliers stored in place -- the same
  //       pivot sequence as column-by-column partial pivoting;
  //   (2) the pivot rows' entries right of the panel get the panel's unit-lower-triangular solve (one thread per column),
  //       while another warp removes the pivot rows from the compact list of active rows;
  //   (3) trailing update A22 -= L21 U12 as fp64 tensor-core products (mma.sync m8n8k4, two per 8x8 tile).
  for (int j = tid; j < n; j += nthr) lst[j] = j;
  __syncthreads();
  for (int c0 = 0, m = n, lb = 0; c0 < n; c0 += 8, lb ^= 1) {
    const int w = n - c0 < 8 ? n - c0 : 8;   // panel width
    const int* la = lst + lb * n;            // active rows before this panel (m of them)
    int* ln = lst + (lb ^ 1) * n;            // ... after it (m - w)
    {
      // (1) panel factorisation: thread j < m holds the 8 panel entries of active row j.  Per column ONE barrier: every
      // warp publishes its best candidate TOGETHER with that row's panel entries, after the barrier all threads pick the
      // winner among the warps and eliminate their own row.
      const bool mine = tid < m;
      double a[8];
      {
        const double* src = F + (size_t)(mine ? la[tid] : 0) * ld + c0;
#pragma unroll
        for (int x = 0; x < 8; ++x) a[x] = (mine && x < w) ? src[x] : 0.0;
      }
      bool used = !mine;
      const int nrw = (m + 31) >> 5;   // warps that hold rows
#pragma unroll
      for (int x = 0; x < 8; ++x) {
        if (x < w) {
          const int cb = x & 1;
          // arg-max of the warp by the high words of |a| (redux.sync; the order of positive doubles is that of their bit
          // patterns): the row taken is within 2^-20 of the largest, which is all that partial pivoting needs
          const double best = used ? -1.0 : fabs(a[x]);
          const unsigned key = used ? 0u : (unsigned)__double2hiint(best) + 1u;
          const unsigned kmax = __reduce_max_sync(0xffffffffu, key);
          const int bj = (tid & ~31) + __ffs(__ballot_sync(0xffffffffu, key == kmax)) - 1;
          if (warp < nrw && bj == tid) {
            ckey[cb * kMiWarps + warp] = kmax;
            cpos[cb * kMiWarps + warp] = tid;
#pragma unroll
            for (int x2 = 0; x2 < 8; ++x2) pb[(cb * kMiWarps + warp) * 8 + x2] = a[x2];
          }
          __syncthreads();
          const unsigned wk = lane < nrw ? ckey[cb * kMiWarps + lane] : 0u;   // the winner among the warps, the same way
          const unsigned wmax = __reduce_max_sync(0xffffffffu, wk);
          const int gw = __ffs(__ballot_sync(0xffffffffu, wk == wmax)) - 1;
          const int gpos = cpos[cb * kMiWarps + gw];
          double pr[8];
#pragma unroll
          for (int x2 = 0; x2 < 8; ++x2) pr[x2] = pb[(cb * kMiWarps + gw) * 8 + x2];
          if (tid == gpos) {
            used = true;
            prow[c0 + x] = la[tid];
            pivpos[x] = tid;
          }
          if (!used) {
            const double mlt = a[x] / pr[x];
            a[x] = mlt;
#pragma unroll
            for (int x2 = x + 1; x2 < 8; ++x2) a[x2] = fma(-mlt, pr[x2], a[x2]);
          }
        }
      }
      if (mine) {
        double* dst = F + (size_t)la[tid] * ld + c0;
#pragma unroll
        for (int x = 0; x < 8; ++x)
          if (x < w) dst[x] = a[x];
      }
    }
    __syncthreads();
    // (2) U12 = L11^-1 A12 on the pivot rows (thread per column right of the panel), and the new list of active rows
    if (tid < ld - c0 - w) {
      const int k = c0 + w + tid;
      double u[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) u[i] = i < w ? F[(size_t)prow[c0 + i] * ld + k] : 0.0;
#pragma unroll
      for (int i = 1; i < 8; ++i)
        if (i < w) {
          const double* li = F + (size_t)prow[c0 + i] * ld + c0;   // multipliers of pivot row i (columns c0 .. c0+i-1)
          double acc = u[i];
#pragma unroll
          for (int j = 0; j < 8; ++j)
            if (j < i) acc = fma(-li[j], u[j], acc);
          u[i] = acc;
        }
#pragma unroll
      for (int i = 1; i < 8; ++i)
        if (i < w) F[(size_t)prow[c0 + i] * ld + k] = u[i];
    }
    if (warp == nwarps - 1) {
      int base = 0;
      for (int j0 = 0; j0 < m; j0 += 32) {
        const int j = j0 + lane;
        bool keep = j < m;
#pragma unroll
        for (int x = 0; x < 8; ++x) keep = keep && !(x < w && pivpos[x] == j);
        const unsigned bal = __ballot_sync(0xffffffffu, keep);
        if (keep) ln[base + __popc(bal & ((1u << lane) - 1u))] = la[j];
        base += __popc(bal);
      }
    }
    __syncthreads();
    // (3) trailing update of the remaining rows, columns right of the panel (right-hand sides included)
    const int mr = m - w, ncol = ld - c0 - w;
    if (mr > 0 && ncol > 0) {
      const int g = lane >> 2, t = lane & 3;
      const int rt_n = (mr + 7) >> 3, ct_n = (ncol + 7) >> 3;
      for (int tile = warp; tile < rt_n * ct_n; tile += nwarps) {
        const int rt = tile / ct_n, ct = tile - rt * ct_n;
        const int jr = 8 * rt + g < mr ? 8 * rt + g : mr - 1;        // (a short tail repeats the last row: same values twice)
        double* rowp = F + (size_t)ln[jr] * ld;
        const int k0 = c0 + w + 8 * ct;
        const int kb = k0 + g < ld ? k0 + g : ld - 1;
        double cfr[2];
        const bool cin = k0 + 2 * t < ld;                            // ld and k0 are even: both columns of the pair or none
        const double2 cc = cin ? *reinterpret_cast<const double2*>(rowp + k0 + 2 * t) : make_double2(0.0, 0.0);
        cfr[0] = cc.x; cfr[1] = cc.y;
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const int x = 4 * hh + t;
          const double av = x < w ? -rowp[c0 + x] : 0.0;
          const double bv = x < w ? F[(size_t)prow[c0 + x] * ld + kb] : 0.0;
          dmma(cfr, av, bv);
        }
        if (cin && 8 * rt + g < mr) *reinterpret_cast<double2*>(rowp + k0 + 2 * t) = make_double2(cfr[0], cfr[1]);
      }
    }
    m = mr;
    __syncthreads();
  }
  // the on-shell unknowns are the last nc columns: K_on from the last nc pivot rows (upper triangular in pivot order)
  if (tid == 0) {
    double K[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
    const double* r1 = F + (size_t)prow[n - 1] * ld;
    if (nc == 1) {
      K[0][0] = r1[n] / r1[n - 1];
    } else {
      const double* r0 = F + (size_t)prow[n - 2] * ld;
      for (int b = 0; b < 2; ++b) {
        K[1][b] = r1[n + b] / r1[n - 1];
        K[0][b] = (r0[n + b] - r0[n - 1] * K[1][b]) / r0[n - 2];
      }
    }
    // T_on = K_on (1 + i g K_on)^-1, S = 1 - 2 i g T_on, g = f p
    const double g = f * p;
    double* o = P.Sout + ((smp * P.nch + ch) * P.nE + e) * (size_t)(nc * nc * 2);
    if (nc == 1) {
      const double x = g * K[0][0], den = 1.0 + x * x;
      o[0] = (1.0 - x * x) / den;
      o[1] = -2.0 * x / den;
    } else {
      // M = 1 + i g K;  M^-1 = adj(M)/det(M)
      const double2 m00 = make_double2(1.0, g * K[0][0]), m01 = make_double2(0.0, g * K[0][1]);
      const double2 m10 = make_double2(0.0, g * K[1][0]), m11 = make_double2(1.0, g * K[1][1]);
      const double2 d1 = cmul(m00, m11), d2 = cmul(m01, m10);
      const double2 det = make_double2(d1.x - d2.x, d1.y - d2.y);
      const double2 one = make_double2(1.0, 0.0);
      const double2 idet = cdiv(one, det);
      const double2 i00 = cmul(m11, idet), i11 = cmul(m00, idet);
      const double2 i01 = cmul(make_double2(-m01.x, -m01.y), idet), i10 = cmul(make_double2(-m10.x, -m10.y), idet);
      const double2 inv[2][2] = {{i00, i01}, {i10, i11}};
      for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
          // T_ab = sum_c K_ac inv_cb (K real)
          const double tr = K[a][0] * inv[0][b].x + K[a][1] * inv[1][b].x;
          const double ti = K[a][0] * inv[0][b].y + K[a][1] * inv[1][b].y;
          // -2 i g (tr + i ti) = 2 g ti - 2 i g tr
          o[(a * 2 + b) * 2] = (a == b ? 1.0 : 0.0) + 2.0 * g * ti;
          o[(a * 2 + b) * 2 + 1] = -2.0 * g * tr;
        }
    }
  }
  __syncthreads();   // the next system of this CTA (kGlob) reuses q, D and the lists
  }
}

// threads of a CTA (>= one per row of the system): two warps for n <= 64 (many CTAs per SM; measured N_Q = 24: 0.42 -> 0.23 ms
// per sample), the full 256 above, where the assembly and the trailing updates use them (N_Q = 96: 1.61 ms against 1.91 with 128)
int mi_threads(int NQ, int coupled) {
  const int n = (coupled ? 2 : 1) * (NQ + 1);
  return n <= 64 ? 64 : kMiThreads;
}

size_t mi_smem(int NQ, int coupled) {
  const int M = NQ + 1, nc = coupled ? 2 : 1, n = nc * M, ld = (n + nc + 1) & ~1;
  return (size_t)n * ld * 8 + (size_t)2 * M * 8 + (size_t)3 * n * 4 + 16;
}
// the L2 variant: F lives in the workspace, only the vectors and lists in shared memory
size_t mi_smem_glob(int NQ, int coupled) {
  const int M = NQ + 1, nc = coupled ? 2 : 1, n = nc * M;
  return (size_t)2 * M * 8 + (size_t)3 * n * 4 + 16;
}
size_t mi_fbytes(int NQ, int coupled) {
  const int M = NQ + 1, nc = coupled ? 2 : 1, n = nc * M, ld = (n + nc + 1) & ~1;
  return (((size_t)n * ld * 8) + 255) & ~(size_t)255;
}
constexpr int kMiGlobCtas = 320;   // CTAs of the L2 variant (2 per SM on 148 SMs, rounded up): each owns one F region

}  // namespace

constexpr int kMiMaxBasis = WPCD_MAX_CHANNELS * (2 * WPCD_MAX_TERMS + 1);
constexpr int kMiEChunk = 128;   // energies per launch: the on-shell tables of one chunk live in the workspace
static size_t mi_tables_bytes(int NQ) {
  return (((size_t)2 * ((NQ * 8 + 255) & ~255) + (size_t)kMiMaxBasis * NQ * NQ * 8 + (size_t)kMiEChunk * kMiMaxBasis * (NQ + 1) * 8) + 255) & ~(size_t)255;
}
// does the system of this kind fit one CTA's shared memory?  (227 KB opt-in on sm_100a: N_Q <= 164 uncoupled, <= 81 coupled)
static bool mi_in_smem(int NQ, int coupled) { return mi_smem(NQ, coupled) + 4096 <= (size_t)232448; }
size_t wpcd_mi_workspace(int NQ) {
  size_t f = 0;   // F regions of the L2 variant, for the larger of the two kinds that needs them
  for (int coupled = 0; coupled < 2; ++coupled)
    if (!mi_in_smem(NQ, coupled) && (coupled ? 2 : 1) * (NQ + 1) <= kMiThreads) {
      const size_t b = (size_t)kMiGlobCtas * mi_fbytes(NQ, coupled);
      f = b > f ? b : f;
    }
  return mi_tables_bytes(NQ) + f;
}

// is the system of this kind supported?  One thread per row: n <= 256 (N_Q <= 255 uncoupled, <= 127 coupled)
bool wpcd_mi_fits(const WpcdHandle* h, int NQ, int coupled) {
  if (mi_smem(NQ, coupled) + 4096 <= (size_t)h->max_smem_optin) return true;
  return (coupled ? 2 : 1) * (NQ + 1) <= kMiThreads;
}

int wpcd_mi_launch(WpcdHandle* h, const wpcd_potential* pot, const wpcd_channel* chan, int n_chan, const double* d_scales,
                   int S, int P, int NQ, double cmap, double hbarc, double mu, const double* d_Ecm, int nE, double* d_S_unc,
                   double* d_S_cpl, void* d_work, cudaStream_t st) {
  double* kq = static_cast<double*>(d_work);
  double* wq = reinterpret_cast<double*>(static_cast<char*>(d_work) + ((NQ * 8 + 255) & ~255));
  double* basis = reinterpret_cast<double*>(static_cast<char*>(d_work) + 2 * ((NQ * 8 + 255) & ~255));
  double* onb = basis + (size_t)kMiMaxBasis * NQ * NQ;
  const double cE = hbarc * hbarc / (2.0 * mu);
  k_mi_grid<<<(NQ + 127) / 128, 128, 0, st>>>(NQ, cmap, kq, wq);
  // distinct (l, mu) of all channel blocks
  MiBasisTable bt; bt.n = 0;
  auto find_or_add = [&](int l, double mu_) {
    for (int b = 0; b < bt.n; ++b) if (bt.l[b] == l && bt.mu[b] == mu_) return b;
    bt.l[bt.n] = l; bt.mu[bt.n] = mu_;
    return bt.n++;
  };
  int ids_mm[WPCD_MAX_CHANNELS][WPCD_MAX_TERMS] = {}, ids_pp[WPCD_MAX_CHANNELS][WPCD_MAX_TERMS] = {}, ids_mp[WPCD_MAX_CHANNELS] = {};
  if (pot->kind == 0) {
    for (int c = 0; c < n_chan; ++c)
      for (int t = 0; t < pot->n_terms; ++t) {
        if (!chan[c].coupled) ids_mm[c][t] = find_or_add(chan[c].lJ, pot->mu[t]);
        else { ids_mm[c][t] = find_or_add(chan[c].lJ - 1, pot->mu[t]); ids_pp[c][t] = find_or_add(chan[c].lJ + 1, pot->mu[t]); }
      }
    for (int c = 0; c < n_chan; ++c) if (chan[c].coupled) ids_mp[c] = find_or_add(chan[c].lJ, pot->muT);
    k_mi_basis<<<dim3((NQ * NQ + 255) / 256, bt.n), 256, 0, st>>>(NQ, bt, kq, basis);
  }
  for (int e_first = 0; e_first < nE; e_first += kMiEChunk) {
  const int ne = nE - e_first < kMiEChunk ? nE - e_first : kMiEChunk;
  if (pot->kind == 0) k_mi_onbasis<<<dim3(ne, bt.n), (NQ + 1 + 31) / 32 * 32, 0, st>>>(NQ, bt, kq, d_Ecm, e_first, cE, onb);
  for (int coupled = 0; coupled < 2; ++coupled) {
    MiParams Q;
    Q.kq = kq; Q.wq = wq; Q.Ecm = d_Ecm; Q.scales = d_scales; Q.Sout = coupled ? d_S_cpl : d_S_unc;
    Q.NQ = NQ; Q.nE = nE; Q.P = P; Q.coupled = coupled; Q.nch = 0; Q.basis = basis; Q.onb = onb; Q.nbasis = bt.n; Q.e_first = e_first;
    for (int c = 0; c < n_chan; ++c)
      if ((chan[c].coupled ? 1 : 0) == coupled) {
        for (int t = 0; t < WPCD_MAX_TERMS; ++t) { Q.id_mm[Q.nch][t] = ids_mm[c][t]; Q.id_pp[Q.nch][t] = ids_pp[c][t]; }
        Q.id_mp[Q.nch] = ids_mp[c];
        Q.lJ[Q.nch++] = chan[c].lJ;
      }
    if (!Q.nch) continue;
    Q.kind = pot->kind; Q.nterms = pot->kind == 0 ? pot->n_terms : 0;
    for (int t = 0; t < WPCD_MAX_TERMS; ++t) {
      Q.V0[t] = t < Q.nterms ? pot->V0[t] : 0.0;
      Q.mu[t] = t < Q.nterms ? pot->mu[t] : 1.0;
      Q.sidx[t] = (t < Q.nterms && pot->scale_idx) ? pot->scale_idx[t] : -1;
    }
    Q.VT = pot->VT; Q.muT = pot->muT; Q.VT_sidx = pot->VT_scale_idx;
    Q.lambdaA = pot->lambda * (WPCD_PI / 2.0);  // wpcd_potential.lambda is convention B: lambda_B = (2/pi) lambda_A (reading C15)
    Q.beta = pot->beta; Q.hbarc = hbarc; Q.mured = mu;
    Q.ne = ne; Q.S = S; Q.fwork = nullptr;
    if (mi_smem(NQ, coupled) + 4096 <= (size_t)h->max_smem_optin) {
      const size_t smem = mi_smem(NQ, coupled);
      int rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_mi_solve<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "mi attr");
      if (rc) return rc;
      k_mi_solve<false><<<dim3(ne, Q.nch, S), mi_threads(NQ, coupled), smem, st>>>(Q);
    } else {
      // L2 variant: a fixed grid of CTAs, each with its own F region behind the tables, loops over the systems
      Q.fwork = reinterpret_cast<double*>(static_cast<char*>(d_work) + mi_tables_bytes(NQ));
      const long long nsys = (long long)ne * Q.nch * S;
      int grid = 2 * h->num_sms < kMiGlobCtas ? 2 * h->num_sms : kMiGlobCtas;
      if (nsys < grid) grid = (int)nsys;
      k_mi_solve<true><<<grid, kMiThreads, mi_smem_glob(NQ, coupled), st>>>(Q);
    }
  }
  }
  return wpcd_check_cuda(h, cudaGetLastError(), "mi_solve launch");
}
