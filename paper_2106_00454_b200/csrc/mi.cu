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
  int id_mm[WPCD_MAX_CHANNELS][WPCD_MAX_TERMS];           // basis matrix of term t in the block l = lJ (uncoupled) / J-1
  int id_pp[WPCD_MAX_CHANNELS][WPCD_MAX_TERMS];           // ... in the block l = J+1
  int id_mp[WPCD_MAX_CHANNELS];                           // ... of the off-diagonal Yukawa
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
  basis[(size_t)blockIdx.y * NQ * NQ + idx] = legendre_q(tab.l[blockIdx.y], zm1);
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

__device__ __forceinline__ double yukawa_A(int l, int nterms, const double* V0, const double* mu, double kp, double k) {
  double s = 0.0;
  for (int t = 0; t < nterms; ++t) {
    const double diff = kp - k;
    const double zm1 = fma(diff, diff, mu[t] * mu[t]) / (2.0 * kp * k);
    s += V0[t] * legendre_q(l, zm1);
  }
  return s / (2.0 * kp * k);
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
__global__ void __launch_bounds__(kMiThreads) k_mi_solve(MiParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = kMiThreads / 32;
  const int NQ = P.NQ, M = NQ + 1, nc = P.coupled ? 2 : 1, n = nc * M, ld = n + nc, ng = nc * NQ;
  double* F = reinterpret_cast<double*>(smem_raw);       // [n][ld]
  double* q = F + (size_t)n * ld;                         // [M]
  double* D = q + M;                                      // [M] real parts (principal value)
  int* prow = reinterpret_cast<int*>(D + M);              // [n] pivot row of column c
  int* lst = prow + n;                                    // [2][n] rows not yet used as a pivot (double buffered)
  __shared__ double sV0[WPCD_MAX_TERMS], sVT;
  __shared__ double cval[2 * (kMiThreads / 32)];         // pivot candidates per warp (double buffered)
  __shared__ int cpos[2 * (kMiThreads / 32)];
  const int e = blockIdx.x, ch = blockIdx.y;
  const size_t smp = blockIdx.z;
  const double cE = P.hbarc * P.hbarc / (2.0 * P.mured), f = 2.0 * P.mured / (P.hbarc * P.hbarc);
  const double p = sqrt(P.Ecm[e] / cE);
  const int lJ = P.lJ[ch];
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
  for (int j = tid; j < NQ; j += kMiThreads) {
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
  for (int idx = tid; idx < n * n; idx += kMiThreads) {
    const int r = idx / n, c = idx - r * n;
    const int a = r < ng ? r / NQ : r - ng, i = r < ng ? r - a * NQ : NQ;
    const int b = c < ng ? c / NQ : c - ng, j = c < ng ? c - b * NQ : NQ;
    double v;
    if (P.kind == 1) {
      v = -P.lambdaA / ((q[i] * q[i] + P.beta * P.beta) * (q[j] * q[j] + P.beta * P.beta));
    } else if (i < NQ && j < NQ) {  // grid x grid: tabulated Q_l, same arithmetic as yukawa_A
      const size_t o = (size_t)i * NQ + j, nn = (size_t)NQ * NQ;
      double sacc = 0.0;
      if (a == b) {
        const int* id = (P.coupled && a == 1) ? P.id_pp[ch] : P.id_mm[ch];
        for (int t = 0; t < P.nterms; ++t) sacc += sV0[t] * P.basis[id[t] * nn + o];
      } else {
        sacc += sVT * P.basis[P.id_mp[ch] * nn + o];
      }
      v = sacc / (2.0 * q[i] * q[j]);
    } else if (!P.coupled) v = yukawa_A(lJ, P.nterms, sV0, P.mu, q[i], q[j]);
    else if (a == b) v = yukawa_A(a == 0 ? lJ - 1 : lJ + 1, P.nterms, sV0, P.mu, q[i], q[j]);
    else v = yukawa_A(lJ, 1, &sVT, &P.muT, q[i], q[j]);
    F[(size_t)r * ld + c] = (r == c ? 1.0 : 0.0) - v * D[j];
    if (j == NQ) F[(size_t)r * ld + n + b] = v;
  }
  __syncthreads();
  // Gauss elimination with partial pivoting, ONE barrier per column.  The rows still to be eliminated are kept as a
  // compact list (double buffered: a column reads list b and writes the list without its pivot row into b^1); the
  // pivot of column c+1 is found while column c is being eliminated (the lanes that update the entries of column c+1
  // keep the largest one per warp; double buffered candidates), so there is no separate search phase; a warp updates
  // four rows at a time with the pivot row's entries loaded once.
  {
    double best = -1.0;
    int bpos = 0;
    for (int j = tid; j < n; j += kMiThreads) {
      lst[j] = j;
      const double v = fabs(F[(size_t)j * ld]);
      if (v > best) { best = v; bpos = j; }
    }
    for (int o = 16; o > 0; o >>= 1) {
      const double ob = __shfl_xor_sync(0xffffffffu, best, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bpos, o);
      if (ob > best || (ob == best && oi < bpos)) { best = ob; bpos = oi; }
    }
    if (lane == 0) { cval[warp] = best; cpos[warp] = bpos; }
  }
  for (int c = 0; c < n; ++c) {
    __syncthreads();
    const int b = c & 1, nact = n - c;
    const int* lb = lst + b * n;
    int* ln = lst + (b ^ 1) * n;
    double best = cval[b * nwarps];
    int pos = cpos[b * nwarps];
    for (int w = 1; w < nwarps; ++w) {
      const double ob = cval[b * nwarps + w];
      const int oi = cpos[b * nwarps + w];
      if (ob > best || (ob == best && oi < pos)) { best = ob; pos = oi; }
    }
    const int piv = lb[pos], lastr = lb[nact - 1];
    if (tid == 0) prow[c] = piv;
    for (int j = tid; j < nact - 1; j += kMiThreads) ln[j] = j == pos ? lastr : lb[j];
    const double* prw = F + (size_t)piv * ld;
    const double rp = 1.0 / prw[c];
    double wbest = -1.0;
    int wpos = 0;
    for (int j0 = 4 * warp; j0 < nact - 1; j0 += 4 * nwarps) {
      double* row[4];
      double mlt[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        const int j = j0 + x < nact - 1 ? j0 + x : j0;   // (a short tail repeats row j0: same values written twice)
        row[x] = F + (size_t)(j == pos ? lastr : lb[j]) * ld;
        mlt[x] = row[x][c] * rp;
      }
      for (int k = c + 1 + lane; k < ld; k += 32) {
        const double pk = prw[k];
        double v[4];
#pragma unroll
        for (int x = 0; x < 4; ++x) v[x] = fma(-mlt[x], pk, row[x][k]);
#pragma unroll
        for (int x = 0; x < 4; ++x) row[x][k] = v[x];
        if (k == c + 1) {
#pragma unroll
          for (int x = 0; x < 4; ++x)
            if (j0 + x < nact - 1 && fabs(v[x]) > wbest) { wbest = fabs(v[x]); wpos = j0 + x; }
        }
      }
    }
    // lane 0 of a warp saw column c+1 of all its rows
    wbest = __shfl_sync(0xffffffffu, wbest, 0);
    wpos = __shfl_sync(0xffffffffu, wpos, 0);
    if (lane == 0) { cval[(b ^ 1) * nwarps + warp] = wbest; cpos[(b ^ 1) * nwarps + warp] = wpos; }
  }
  __syncthreads();
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
}

size_t mi_smem(int NQ, int coupled) {
  const int M = NQ + 1, nc = coupled ? 2 : 1, n = nc * M, ld = n + nc;
  return (size_t)n * ld * 8 + (size_t)2 * M * 8 + (size_t)3 * n * 4 + 16;
}

}  // namespace

constexpr int kMiMaxBasis = WPCD_MAX_CHANNELS * (2 * WPCD_MAX_TERMS + 1);
size_t wpcd_mi_workspace(int NQ) { return (size_t)2 * ((NQ * 8 + 255) & ~255) + (size_t)kMiMaxBasis * NQ * NQ * 8; }

// does the system of this kind fit one CTA's shared memory?
bool wpcd_mi_fits(const WpcdHandle* h, int NQ, int coupled) { return mi_smem(NQ, coupled) + 4096 <= (size_t)h->max_smem_optin; }

int wpcd_mi_launch(WpcdHandle* h, const wpcd_potential* pot, const wpcd_channel* chan, int n_chan, const double* d_scales,
                   int S, int P, int NQ, double cmap, double hbarc, double mu, const double* d_Ecm, int nE, double* d_S_unc,
                   double* d_S_cpl, void* d_work, cudaStream_t st) {
  double* kq = static_cast<double*>(d_work);
  double* wq = reinterpret_cast<double*>(static_cast<char*>(d_work) + ((NQ * 8 + 255) & ~255));
  double* basis = reinterpret_cast<double*>(static_cast<char*>(d_work) + 2 * ((NQ * 8 + 255) & ~255));
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
  for (int coupled = 0; coupled < 2; ++coupled) {
    MiParams Q;
    Q.kq = kq; Q.wq = wq; Q.Ecm = d_Ecm; Q.scales = d_scales; Q.Sout = coupled ? d_S_cpl : d_S_unc;
    Q.NQ = NQ; Q.nE = nE; Q.P = P; Q.coupled = coupled; Q.nch = 0; Q.basis = basis;
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
    const size_t smem = mi_smem(NQ, coupled);
    int rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_mi_solve, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "mi attr");
    if (rc) return rc;
    k_mi_solve<<<dim3(nE, Q.nch, S), kMiThreads, smem, st>>>(Q);
  }
  return wpcd_check_cuda(h, cudaGetLastError(), "mi_solve launch");
}
