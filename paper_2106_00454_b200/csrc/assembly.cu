// assembly.cu -- steps (i) and Eq. 29 of the WPCD recipe: H = H0 + V for every channel
// and potential sample.  Three kernels:
//   k_grid    : bin quantities (e0, dE, Eedge) and the n_gl-point Gauss-Legendre nodes/weights of every bin
//   k_basis   : one "basis matrix" per distinct (l, mu):  B[i][j] = (1/(pi sqrt(Dk_i Dk_j))) sum_ab w_ia w_jb Q_l(z)
//               (n_gl x n_gl rule per bin pair, 8 threads per element; FP64/SFU bound, done once per grid)
//   k_combine : H[s][c] = diag(e0) + sum_t V0_t scale[s][t] B_t   -- HBM-write bound: 8 B written per element,
//               double2 stores, the basis matrices stay L2-resident.
// Strengths enter linearly, so the per-sample work is the combine only.
#include <math.h>
#include "wpcd_internal.cuh"
#include "legendre_q.cuh"

#define MAX_BASIS (WPCD_MAX_CHANNELS * (2 * WPCD_MAX_TERMS + 1))

struct BasisDesc { int l; int kind; double mu; double beta; };  // kind 0: Yukawa Q_l, 1: Yamaguchi G_i G_j
struct BasisTable { int nbasis; BasisDesc d[MAX_BASIS]; };

struct BlockTerms { int nterms; int basis[WPCD_MAX_TERMS]; int sidx[WPCD_MAX_TERMS]; double V0[WPCD_MAX_TERMS]; };
struct ChanDesc { int coupled; int slot; BlockTerms mm, pp, mp; };
struct ChanTable { int nchan; int n_unc; int n_cpl; ChanDesc c[WPCD_MAX_CHANNELS]; };

// ------------------------------------------------------------------------------------------------ k_grid
// thread (i, a): Newton iteration for the a-th root of P_ngl, then maps it into bin i.
// wp_kind 1 (energy wave packets, f(k) = hbarc sqrt(k/mu), N_i = dE_i): e0 = E_i + dE_i/2 (Eq. 18), the node weights
// carry sqrt(k) and norm_i = sqrt(mu dE_i)/hbarc, so that (1/(norm_i norm_j)) sum_ab w_ia w_jb ... is Eq. 29 with
// f(k')f(k)/sqrt(N_i N_j); momentum packets: norm_i = sqrt(Dk_i).
__global__ void k_grid(int N, int ngl, int wp_kind, double hbarc, double mu, const double* __restrict__ p,
                       double* __restrict__ e0, double* __restrict__ dE, double* __restrict__ Eedge,
                       double* __restrict__ knode, double* __restrict__ wnode, double* __restrict__ norm) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  double cE = hbarc * hbarc / (2.0 * mu);
  if (idx <= N) Eedge[idx] = cE * p[idx] * p[idx];
  if (idx < N) {
    double a = p[idx], b = p[idx + 1];
    const double w = cE * b * b - cE * a * a;
    e0[idx] = wp_kind ? cE * a * a + 0.5 * w : cE * (a * a + a * b + b * b) / 3.0;
    dE[idx] = w;
    norm[idx] = wp_kind ? sqrt(mu * w) / hbarc : sqrt(b - a);
  }
  if (idx < N * ngl) {
    int i = idx / ngl, a = idx % ngl;
    // root a (ascending) of the Legendre polynomial P_ngl
    double x = -cos(WPCD_PI * (a + 0.75) / (ngl + 0.5));
    double dp = 1.0;
    for (int it = 0; it < 50; ++it) {
      double pm = 1.0, pc = x;
      for (int k = 2; k <= ngl; ++k) {
        double pn = ((2 * k - 1) * x * pc - (k - 1) * pm) / k;
        pm = pc; pc = pn;
      }
      if (ngl == 1) { pm = 1.0; pc = x; }
      dp = ngl * (x * pc - pm) / (x * x - 1.0);
      double dx = pc / dp;
      x -= dx;
      if (fabs(dx) < 1e-16) break;
    }
    {  // derivative at the converged root
      double pm = 1.0, pc = x;
      for (int k = 2; k <= ngl; ++k) {
        double pn = ((2 * k - 1) * x * pc - (k - 1) * pm) / k;
        pm = pc; pc = pn;
      }
      dp = ngl * (x * pc - pm) / (x * x - 1.0);
    }
    double w = 2.0 / ((1.0 - x * x) * dp * dp);
    double lo = p[i], hi = p[i + 1], half = 0.5 * (hi - lo);
    const double kn = 0.5 * (lo + hi) + half * x;
    knode[idx] = kn;
    wnode[idx] = wp_kind ? half * w * sqrt(kn) : half * w;
  }
}

// ------------------------------------------------------------------------------------------------ k_basis
// grid (ceil(8 ntri/128), nbasis); 8 threads per upper-triangle element (i <= j), each taking the quadrature rows
// a = sub, sub + 8, ... of the bin pair, summed over the 8 lanes by shuffles; mirrored store keeps B symmetric.
__global__ void __launch_bounds__(128) k_basis(int N, int ngl, int wp_kind, BasisTable tab, const double* __restrict__ p,
                                               const double* __restrict__ knode, const double* __restrict__ wnode,
                                               const double* __restrict__ norm, double* __restrict__ basis) {
  const int gt = blockIdx.x * blockDim.x + threadIdx.x;
  const int sub = gt & 7;
  int e = gt >> 3;
  const int ntri = N * (N + 1) / 2;
  const bool live = e < ntri;
  if (!live) e = ntri - 1;  // keeps the whole warp in the shuffles below
  // row i of the upper triangle: first element index i*N - i(i-1)/2
  int i = (int)((2.0 * N + 1.0 - sqrt((2.0 * N + 1.0) * (2.0 * N + 1.0) - 8.0 * e)) * 0.5);
  while (i * N - i * (i - 1) / 2 > e) --i;
  while ((i + 1) * N - (i + 1) * i / 2 <= e) ++i;
  int j = i + (e - (i * N - i * (i - 1) / 2));
  BasisDesc d = tab.d[blockIdx.y];
  double* B = basis + (size_t)blockIdx.y * N * N;
  double dki = p[i + 1] - p[i], dkj = p[j + 1] - p[j];
  double v;
  if (d.kind == 1 && wp_kind) {
    // Yamaguchi form factor of an energy packet: G_i = N_i^{-1/2} int k f(k) g(k) dk by the bin's quadrature rule
    double b2 = d.beta * d.beta, gi = 0.0, gj = 0.0;
    for (int a = 0; a < ngl; ++a) {
      double ki = knode[i * ngl + a], kj = knode[j * ngl + a];
      gi = fma(wnode[i * ngl + a], ki / (ki * ki + b2), gi);
      gj = fma(wnode[j * ngl + a], kj / (kj * kj + b2), gj);
    }
    v = (gi / norm[i]) * (gj / norm[j]);
  } else if (d.kind == 1) {
    // Yamaguchi form factor, closed form of int k/(k^2+beta^2) dk over the bin (reading C15)
    double b2 = d.beta * d.beta;
    double gi = 0.5 * log((p[i + 1] * p[i + 1] + b2) / (p[i] * p[i] + b2)) / sqrt(dki);
    double gj = 0.5 * log((p[j + 1] * p[j + 1] + b2) / (p[j] * p[j] + b2)) / sqrt(dkj);
    v = gi * gj;
  } else {
    double mu2 = d.mu * d.mu, acc = 0.0;
    for (int a = sub; a < ngl; a += 8) {
      double kp = knode[i * ngl + a], wa = wnode[i * ngl + a];
      double row = 0.0;
      for (int b = 0; b < ngl; ++b) {
        double k = knode[j * ngl + b];
        double diff = kp - k;
        double zm1 = fma(diff, diff, mu2) / (2.0 * kp * k);
        row = fma(wnode[j * ngl + b], legendre_q(d.l, zm1), row);
      }
      acc = fma(wa, row, acc);
    }
    acc += __shfl_xor_sync(0xffffffffu, acc, 1);
    acc += __shfl_xor_sync(0xffffffffu, acc, 2);
    acc += __shfl_xor_sync(0xffffffffu, acc, 4);
    v = wp_kind ? acc / (WPCD_PI * norm[i] * norm[j]) : acc / (WPCD_PI * sqrt(dki * dkj));
  }
  if (live && sub == 0) {
    B[(size_t)i * N + j] = v;
    B[(size_t)j * N + i] = v;
  }
}

// ------------------------------------------------------------------------------------------------ k_combine
__device__ __forceinline__ double combine_elem(const ChanDesc& c, int N, int i, int j, const double* __restrict__ basis,
                                               const double* __restrict__ e0, const double* __restrict__ scale, int P) {
  int bi = 0, bj = 0, ii = i, jj = j;
  if (c.coupled) { bi = i >= N; bj = j >= N; ii = i - bi * N; jj = j - bj * N; }
  const BlockTerms& bt = (bi == bj) ? (bi ? c.pp : c.mm) : c.mp;
  double v = (i == j) ? e0[ii] : 0.0;
  double acc = 0.0;
  for (int t = 0; t < bt.nterms; ++t) {
    double coef = bt.V0[t];
    if (bt.sidx[t] >= 0) coef *= scale[bt.sidx[t]];
    acc = fma(coef, basis[(size_t)bt.basis[t] * N * N + (size_t)ii * N + jj], acc);
  }
  return v + acc;
}

// grid: (ceil(n*n/4/256), nchan_of_kind, S).  N % 4 == 0 (the configs): each thread writes four adjacent elements of a
// row -- same block of the channel, same terms, 32-byte aligned loads of the basis rows and stores of H, 32-bit index
// arithmetic.  Other N: two elements per thread through combine_elem.
__global__ void __launch_bounds__(256) k_combine(int N, int coupled, ChanTable tab, const double* __restrict__ basis,
                                                 const double* __restrict__ e0, const double* __restrict__ scales, int P,
                                                 double* __restrict__ Hout) {
  const unsigned n = coupled ? 2 * N : N;
  const int nkind = coupled ? tab.n_cpl : tab.n_unc;
  // find the channel with this slot
  int ci = 0;
  for (int c = 0; c < tab.nchan; ++c)
    if (tab.c[c].coupled == coupled && tab.c[c].slot == (int)blockIdx.y) ci = c;
  const ChanDesc& cd = tab.c[ci];
  const double* scale = scales ? scales + (size_t)blockIdx.z * P : nullptr;
  double* H = Hout + ((size_t)blockIdx.z * nkind + blockIdx.y) * (size_t)n * n;
  const unsigned total = n * n;  // n <= 8192
  if ((N & 3) == 0) {
    const unsigned e = (blockIdx.x * blockDim.x + threadIdx.x) * 4u;
    if (e >= total) return;
    const unsigned i = e / n, j = e - i * n;
    const unsigned bi = coupled && i >= (unsigned)N, bj = coupled && j >= (unsigned)N;
    const unsigned ii = i - bi * N, jj = j - bj * N;
    const BlockTerms& bt = (bi == bj) ? (bi ? cd.pp : cd.mm) : cd.mp;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int t = 0; t < bt.nterms; ++t) {
      double coef = bt.V0[t];
      if (bt.sidx[t] >= 0) coef *= scale[bt.sidx[t]];
      const double2* b = reinterpret_cast<const double2*>(basis + (size_t)bt.basis[t] * N * N + (size_t)ii * N + jj);
      const double2 x0 = b[0], x1 = b[1];
      acc[0] = fma(coef, x0.x, acc[0]); acc[1] = fma(coef, x0.y, acc[1]);
      acc[2] = fma(coef, x1.x, acc[2]); acc[3] = fma(coef, x1.y, acc[3]);
    }
    const double d = e0[ii];
#pragma unroll
    for (int k = 0; k < 4; ++k) acc[k] = ((j + k == i) ? d : 0.0) + acc[k];
    double2* out = reinterpret_cast<double2*>(H + e);
    out[0] = make_double2(acc[0], acc[1]);
    out[1] = make_double2(acc[2], acc[3]);
    return;
  }
  const unsigned e = (blockIdx.x * blockDim.x + threadIdx.x) * 4u;
  for (unsigned k = e; k < e + 4 && k < total; ++k) H[k] = combine_elem(cd, N, (int)(k / n), (int)(k % n), basis, e0, scale, P);
}

// ------------------------------------------------------------------------------------------------ host side
static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

size_t wpcd_build_workspace(int N, int n_chan) {
  size_t nb = (size_t)n_chan * (2 * WPCD_MAX_TERMS + 1);
  if (nb > MAX_BASIS) nb = MAX_BASIS;
  return 2 * align256((size_t)(N + 1) * 8) + 2 * align256((size_t)N * 16 * 8) + nb * align256((size_t)N * N * 8);
}

static int find_or_add(BasisTable& t, int l, int kind, double mu, double beta) {
  for (int b = 0; b < t.nbasis; ++b)
    if (t.d[b].l == l && t.d[b].kind == kind && t.d[b].mu == mu && t.d[b].beta == beta) return b;
  if (t.nbasis >= MAX_BASIS) return -1;
  t.d[t.nbasis].l = l; t.d[t.nbasis].kind = kind; t.d[t.nbasis].mu = mu; t.d[t.nbasis].beta = beta;
  return t.nbasis++;
}

int wpcd_build_launch(WpcdHandle* h, const wpcd_grid* grid, const wpcd_potential* pot, const wpcd_channel* chan,
                      int n_chan, const double* d_scales, int S, int P, double* d_H_unc, double* d_H_cpl, double* d_e0,
                      double* d_dE, double* d_Eedge, void* d_work, size_t work_bytes, cudaStream_t st) {
  const int N = grid->N, ngl = grid->n_gl;
  BasisTable bt; bt.nbasis = 0;
  ChanTable ct; ct.nchan = n_chan; ct.n_unc = 0; ct.n_cpl = 0;
  for (int c = 0; c < n_chan; ++c) {
    ChanDesc& cd = ct.c[c];
    cd.coupled = chan[c].coupled ? 1 : 0;
    cd.slot = cd.coupled ? ct.n_cpl++ : ct.n_unc++;
    cd.mm.nterms = cd.pp.nterms = cd.mp.nterms = 0;
    auto fill_central = [&](BlockTerms& b, int l) -> int {
      b.nterms = pot->n_terms;
      for (int t = 0; t < pot->n_terms; ++t) {
        int id = find_or_add(bt, l, 0, pot->mu[t], 0.0);
        if (id < 0) return WPCD_ESIZE;
        b.basis[t] = id; b.V0[t] = pot->V0[t]; b.sidx[t] = pot->scale_idx ? pot->scale_idx[t] : -1;
      }
      return WPCD_OK;
    };
    int rc = WPCD_OK;
    if (pot->kind == 1) {
      int id = find_or_add(bt, 0, 1, 0.0, pot->beta);
      if (id < 0) return WPCD_ESIZE;
      cd.mm.nterms = 1; cd.mm.basis[0] = id; cd.mm.V0[0] = -pot->lambda; cd.mm.sidx[0] = -1;
    } else if (!cd.coupled) {
      rc = fill_central(cd.mm, chan[c].lJ);
    } else {
      rc = fill_central(cd.mm, chan[c].lJ - 1);
      if (rc == WPCD_OK) rc = fill_central(cd.pp, chan[c].lJ + 1);
      int id = find_or_add(bt, chan[c].lJ, 0, pot->muT, 0.0);
      if (id < 0) return WPCD_ESIZE;
      cd.mp.nterms = 1; cd.mp.basis[0] = id; cd.mp.V0[0] = pot->VT; cd.mp.sidx[0] = pot->VT_scale_idx;
    }
    if (rc != WPCD_OK) return rc;
  }
  char* w = static_cast<char*>(d_work);
  double* d_p = reinterpret_cast<double*>(w); w += align256((size_t)(N + 1) * 8);
  double* d_norm = reinterpret_cast<double*>(w); w += align256((size_t)(N + 1) * 8);
  double* d_k = reinterpret_cast<double*>(w); w += align256((size_t)N * 16 * 8);
  double* d_w = reinterpret_cast<double*>(w); w += align256((size_t)N * 16 * 8);
  double* d_basis = reinterpret_cast<double*>(w);
  if ((size_t)(w - static_cast<char*>(d_work)) + (size_t)bt.nbasis * N * N * 8 > work_bytes) return WPCD_EWORK;

  int rc = wpcd_check_cuda(h, cudaMemcpyAsync(d_p, grid->h_edges, (size_t)(N + 1) * 8, cudaMemcpyHostToDevice, st), "edges H2D");
  if (rc) return rc;
  int tot = N * ngl > N + 1 ? N * ngl : N + 1;
  k_grid<<<(tot + 127) / 128, 128, 0, st>>>(N, ngl, grid->wp_kind, grid->hbarc, grid->mu, d_p, d_e0, d_dE, d_Eedge, d_k, d_w, d_norm);
  int ntri = N * (N + 1) / 2;
  k_basis<<<dim3((8 * ntri + 127) / 128, bt.nbasis), 128, 0, st>>>(N, ngl, grid->wp_kind, bt, d_p, d_k, d_w, d_norm, d_basis);
  if (ct.n_unc) {
    size_t quarter = ((size_t)N * N + 3) / 4;
    k_combine<<<dim3((unsigned)((quarter + 255) / 256), ct.n_unc, S), 256, 0, st>>>(N, 0, ct, d_basis, d_e0, d_scales, P, d_H_unc);
  }
  if (ct.n_cpl) {
    size_t quarter = ((size_t)4 * N * N + 3) / 4;
    k_combine<<<dim3((unsigned)((quarter + 255) / 256), ct.n_cpl, S), 256, 0, st>>>(N, 1, ct, d_basis, d_e0, d_scales, P, d_H_cpl);
  }
  return wpcd_check_cuda(h, cudaGetLastError(), "build_channels launch");
}
