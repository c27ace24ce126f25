// mi.cu -- the matrix-inversion (MI) method of Sec. 2.1 on the GPU, batched over
// (sample, channel, energy): the second workload of SURVEY 8(f)-4 ("the MI method ... can be parallelised over the
// on-shell energies").  One CTA per Lippmann-Schwinger system:
//   basis q = {k_1..k_NQ, p}: Gauss-Legendre nodes mapped k_j = c tan(pi(1+x_j)/4), w_j -> c (pi/4) w_j/cos^2(.), plus the
//   on-shell momentum p = sqrt(E_cm/cE)                                                    (Eq. 4)
//   D_j = (2/pi) w_j k_j^2 f/(p^2-k_j^2),  D_{NQ+1} = -(2/pi) f p^2 sum_j w_j/(p^2-k_j^2) - i f p,  f = 2 mu/hbarc^2
//   (derived from Eqs. 2-4, reading C3: the printed Eq. 5 is inconsistent)
//   F = 1 - V diag(D) (Eq. 7), F T = V (Eq. 6) by complex Gauss elimination with partial pivoting in shared memory,
//   S = 1 - 2 i f p T_onshell (convention A, reading C2).
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
};

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

// grid (nE, nch, S); dynamic shared memory: F [n][ld] complex (ld = n + nc: the right-hand sides ride along), q [M],
// D [M] complex.
__global__ void __launch_bounds__(kMiThreads) k_mi_solve(MiParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x;
  const int NQ = P.NQ, M = NQ + 1, nc = P.coupled ? 2 : 1, n = nc * M, ld = n + nc;
  double2* F = reinterpret_cast<double2*>(smem_raw);
  double* q = reinterpret_cast<double*>(F + (size_t)n * ld);
  double2* D = reinterpret_cast<double2*>(q + M + (M & 1));
  __shared__ double s_red[kMiThreads];
  __shared__ int s_idx[kMiThreads];
  __shared__ double sV0[WPCD_MAX_TERMS], sVT;
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
    D[j] = make_double2((2.0 / WPCD_PI) * P.wq[j] * k * k * f / (p * p - k * k), 0.0);
  }
  __syncthreads();
  if (tid == 0) {
    double ssum = 0.0;
    for (int j = 0; j < NQ; ++j) ssum += P.wq[j] / (p * p - q[j] * q[j]);
    D[NQ] = make_double2(-(2.0 / WPCD_PI) * f * p * p * ssum, -f * p);
  }
  __syncthreads();
  // V on the basis, F = 1 - V diag(D), right-hand sides = on-shell columns of V
  for (int idx = tid; idx < n * n; idx += kMiThreads) {
    const int r = idx / n, c = idx - r * n;
    const int a = r / M, i = r - a * M, b = c / M, j = c - b * M;
    double v;
    if (P.kind == 1) v = -P.lambdaA / ((q[i] * q[i] + P.beta * P.beta) * (q[j] * q[j] + P.beta * P.beta));
    else if (!P.coupled) v = yukawa_A(lJ, P.nterms, sV0, P.mu, q[i], q[j]);
    else if (a == b) v = yukawa_A(a == 0 ? lJ - 1 : lJ + 1, P.nterms, sV0, P.mu, q[i], q[j]);
    else v = yukawa_A(lJ, 1, &sVT, &P.muT, q[i], q[j]);
    const double2 d = D[j];
    F[(size_t)r * ld + c] = make_double2((r == c ? 1.0 : 0.0) - v * d.x, -v * d.y);
    if (j == NQ) F[(size_t)r * ld + n + b] = make_double2(v, 0.0);
  }
  __syncthreads();
  // Gauss elimination with partial pivoting
  for (int c = 0; c < n; ++c) {
    double best = -1.0;
    int bi = c;
    for (int r = c + tid; r < n; r += kMiThreads) {
      const double2 x = F[(size_t)r * ld + c];
      const double v = hypot(x.x, x.y);
      if (v > best) { best = v; bi = r; }
    }
    s_red[tid] = best; s_idx[tid] = bi;
    __syncthreads();
    for (int s = kMiThreads / 2; s > 0; s >>= 1) {
      if (tid < s) {
        const double o = s_red[tid + s];
        const int oi = s_idx[tid + s];
        if (o > s_red[tid] || (o == s_red[tid] && oi < s_idx[tid])) { s_red[tid] = o; s_idx[tid] = oi; }
      }
      __syncthreads();
    }
    const int piv = s_idx[0];
    if (piv != c)
      for (int k = c + tid; k < ld; k += kMiThreads) {
        const double2 t = F[(size_t)c * ld + k];
        F[(size_t)c * ld + k] = F[(size_t)piv * ld + k];
        F[(size_t)piv * ld + k] = t;
      }
    __syncthreads();
    const double2 dcc = F[(size_t)c * ld + c];
    for (int r = c + 1 + tid; r < n; r += kMiThreads) F[(size_t)r * ld + c] = cdiv(F[(size_t)r * ld + c], dcc);  // multiplier
    __syncthreads();
    const int w = ld - (c + 1), rows = n - (c + 1);
    for (int idx = tid; idx < rows * w; idx += kMiThreads) {
      const int r = c + 1 + idx / w, k = c + 1 + idx % w;
      const double2 m = F[(size_t)r * ld + c];
      const double2 x = cmul(m, F[(size_t)c * ld + k]);
      double2 y = F[(size_t)r * ld + k];
      y.x -= x.x; y.y -= x.y;
      F[(size_t)r * ld + k] = y;
    }
    __syncthreads();
  }
  // back substitution, column oriented: x_r = b_r / F_rr, then b_r' -= F_r'r x_r for the rows above
  for (int r = n - 1; r >= 0; --r) {
    if (tid < nc) F[(size_t)r * ld + n + tid] = cdiv(F[(size_t)r * ld + n + tid], F[(size_t)r * ld + r]);
    __syncthreads();
    for (int idx = tid; idx < r * nc; idx += kMiThreads) {
      const int rr = idx / nc, b = idx - rr * nc;
      const double2 x = cmul(F[(size_t)rr * ld + r], F[(size_t)r * ld + n + b]);
      double2 y = F[(size_t)rr * ld + n + b];
      y.x -= x.x; y.y -= x.y;
      F[(size_t)rr * ld + n + b] = y;
    }
    __syncthreads();
  }
  // S = 1 - 2 i f p T_onshell
  if (tid < nc * nc) {
    const int a = tid / nc, b = tid - a * nc;
    const double2 t = F[(size_t)(a * M + NQ) * ld + n + b];
    const double g = 2.0 * f * p;  // -i g t = (g t.y, -g t.x)
    double* o = P.Sout + (((smp * P.nch + ch) * P.nE + e) * nc * nc + tid) * 2;
    o[0] = (a == b ? 1.0 : 0.0) + g * t.y;
    o[1] = -g * t.x;
  }
}

size_t mi_smem(int NQ, int coupled) {
  const int M = NQ + 1, nc = coupled ? 2 : 1, n = nc * M, ld = n + nc;
  return (size_t)n * ld * 16 + (size_t)(M + (M & 1)) * 8 + (size_t)M * 16;
}

}  // namespace

size_t wpcd_mi_workspace(int NQ) { return (size_t)2 * ((NQ * 8 + 255) & ~255); }

// does the system of this kind fit one CTA's shared memory?
bool wpcd_mi_fits(const WpcdHandle* h, int NQ, int coupled) { return mi_smem(NQ, coupled) + 4096 <= (size_t)h->max_smem_optin; }

int wpcd_mi_launch(WpcdHandle* h, const wpcd_potential* pot, const wpcd_channel* chan, int n_chan, const double* d_scales,
                   int S, int P, int NQ, double cmap, double hbarc, double mu, const double* d_Ecm, int nE, double* d_S_unc,
                   double* d_S_cpl, void* d_work, cudaStream_t st) {
  double* kq = static_cast<double*>(d_work);
  double* wq = reinterpret_cast<double*>(static_cast<char*>(d_work) + ((NQ * 8 + 255) & ~255));
  k_mi_grid<<<(NQ + 127) / 128, 128, 0, st>>>(NQ, cmap, kq, wq);
  for (int coupled = 0; coupled < 2; ++coupled) {
    MiParams Q;
    Q.kq = kq; Q.wq = wq; Q.Ecm = d_Ecm; Q.scales = d_scales; Q.Sout = coupled ? d_S_cpl : d_S_unc;
    Q.NQ = NQ; Q.nE = nE; Q.P = P; Q.coupled = coupled; Q.nch = 0;
    for (int c = 0; c < n_chan; ++c)
      if ((chan[c].coupled ? 1 : 0) == coupled) Q.lJ[Q.nch++] = chan[c].lJ;
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
