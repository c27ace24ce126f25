// onshell.cu -- steps (iii)-(v) of the WPCD recipe and the S-matrix / phase-shift conversion.
//   k_bins   : FWP bin of every on-shell energy (Eedge_i <= E < Eedge_{i+1}) and the range of bins in use
//   k_onshell: one CTA per matrix.  Pseudostate bin edges from the sorted eigenvalues (Eq. 23 as printed,
//              PAPER.md:166-173; bound states eps < 0 separate; coupled channels: two branches by rank parity),
//              then for chunks of 32 or 16 on-shell rows: VC = (H - diag e0) C as fp64 tensor-core products (mma.sync
//              m8n8k4; A fragments from shared memory, B fragments straight from C), and for every energy in the chunk
//              (one warp per energy, lanes over eigenstates) T = V_ii + sum_k (VC)_ik (VC)_i'k g_k(E) with the
//              analytic resolvent g_k of Eqs. B.3-B.6 (sign of the printed last line corrected).
//   k_phase  : S = 1 - 2 pi i T/dE_i, Eqs. A.3-A.5.
// HBM traffic per matrix: C and the on-shell rows of H are read (C once per chunk, from L2 after the first pass).
#include <math.h>
#include "wpcd_internal.cuh"

namespace {

constexpr int kOnThreads = 256;
constexpr int kOnGemmThreads = 512;  // k_onshell (direct product, n > kI1MaxN)

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {  // fp64 tensor-core MMA, D (8x8) += A (8x4) B (4x8)
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

__device__ __forceinline__ double xlnx(double x) { return x == 0.0 ? 0.0 : x * log(fabs(x)); }

// Resolvent of state k for the on-shell bin `b` / energy E.
//   mode 0: point-wise, Eqs. B.5-B.6 (sign per DESIGN.md reading G2); bound states 1/(E - eps).
//   mode 1: averaged over the pseudostate bin [lo_ki, hi_ki] of the b-th positive state ki of k's own branch, Eq. 28 and
//           B.7-B.8 (sign per reading G3): W/((hi_ki-lo_ki)(hi_k-lo_k)) - i pi/(hi_k-lo_k) [k = ki];
//           bound states averaged over branch 0's bin (readings A1-A3).  The caller has checked that every branch has a
//           b-th state.
__device__ __forceinline__ void resolvent_k(int mode, double E, int b, int k, int nbd, int nc, const double* sW,
                                            const double* sLo, const double* sHi, double& gr, double& gi) {
  gi = 0.0;
  if (mode == 0) {
    if (k < nbd) { gr = 1.0 / (E - sW[k]); return; }
    const double lo = sLo[k], hi = sHi[k], wdt = hi - lo;
    gr = log(fabs((E - lo) / (E - hi))) / wdt;
    if (E >= lo && E < hi) gi = -WPCD_PI / wdt;
    return;
  }
  if (k < nbd) {
    const int k0 = nbd + nc * b;
    const double A = sLo[k0], B = sHi[k0], w = sW[k];
    gr = log(fabs((B - w) / (A - w))) / (B - A);
    return;
  }
  const int ki = nbd + (k - nbd) % nc + nc * b;
  const double A = sLo[ki], B = sHi[ki], lo = sLo[k], hi = sHi[k];
  gr = (xlnx(B - lo) - xlnx(B - hi) - xlnx(A - lo) + xlnx(A - hi)) / ((B - A) * (hi - lo));
  if (k == ki) gi = -WPCD_PI / (hi - lo);
}

__global__ void k_bins(int N, int nE, const double* __restrict__ Eedge, const double* __restrict__ Ecm,
                       int* __restrict__ bin, int* __restrict__ range) {
  __shared__ int smin, smax;
  if (threadIdx.x == 0) { smin = 1 << 30; smax = -1; }
  __syncthreads();
  for (int e = threadIdx.x; e < nE; e += blockDim.x) {
    double E = Ecm[e];
    int b = -1;
    if (E >= Eedge[0] && E < Eedge[N]) {
      int lo = 0, hi = N;  // invariant Eedge[lo] <= E < Eedge[hi]
      while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (E >= Eedge[mid]) lo = mid; else hi = mid;
      }
      b = lo;
      atomicMin(&smin, b);
      atomicMax(&smax, b);
    }
    bin[e] = b;
  }
  __syncthreads();
  if (threadIdx.x == 0) { range[0] = smin; range[1] = smax; }
}

// Rows of VC for one chunk: sVC[nrows x n] = sV[nrows x n] (row stride ldv) times C (n x n) as fp64 tensor-core products
// (mma.sync m8n8k4).  A warp takes 8 NT columns at a time (MT x NT accumulator tiles: 2 x 4 for chunks of 16 rows, 4 x 2
// for chunks of 32 rows, which halve the passes over C where shared memory allows them, n <= ~430); A fragments from
// shared memory (row stride ldv = 4 mod 16: conflict-free), B fragments straight from global memory (lane (g, t) reads
// C[j0 + t][k0 + 8q + g]: four 64-byte row segments per load), unrolled so that 4 NT loads per warp are in flight.
template <int MT, int NT>
__device__ __forceinline__ void vc_rows_mma(const double* __restrict__ sV, int ldv, const double* __restrict__ C, int n,
                                            int nrows, double* __restrict__ sVC, int warp, int nwarps, int lane) {
  const int g = lane >> 2, t = lane & 3, mt = (nrows + 7) >> 3, nfull = n & ~3;
  constexpr int kCols = 8 * NT;
  for (int grp = warp; grp < (n + kCols - 1) / kCols; grp += nwarps) {
    const int k0 = grp * kCols;
    double acc[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
      for (int q = 0; q < NT; ++q) acc[i][q][0] = acc[i][q][1] = 0.0;
    const double* a0 = sV + (size_t)g * ldv + t;
    const double* bp = C + (size_t)t * n + k0 + g;
    bool kin[NT];
#pragma unroll
    for (int q = 0; q < NT; ++q) kin[q] = k0 + 8 * q + g < n;
#pragma unroll 4
    for (int j0 = 0; j0 < nfull; j0 += 4) {
      double b[NT], av[MT];
#pragma unroll
      for (int q = 0; q < NT; ++q) b[q] = kin[q] ? __ldg(bp + (size_t)j0 * n + 8 * q) : 0.0;
#pragma unroll
      for (int i = 0; i < MT; ++i) av[i] = i < mt ? a0[(size_t)8 * i * ldv + j0] : 0.0;
#pragma unroll
      for (int q = 0; q < NT; ++q)
#pragma unroll
        for (int i = 0; i < MT; ++i)
          if (i < mt) dmma(acc[i][q], av[i], b[q]);
    }
    if (nfull < n) {  // ragged tail of the contraction index
      const bool jin = nfull + t < n;
      double av[MT];
#pragma unroll
      for (int i = 0; i < MT; ++i) av[i] = (jin && i < mt) ? a0[(size_t)8 * i * ldv + nfull] : 0.0;
#pragma unroll
      for (int q = 0; q < NT; ++q) {
        const double b = (jin && kin[q]) ? __ldg(bp + (size_t)nfull * n + 8 * q) : 0.0;
#pragma unroll
        for (int i = 0; i < MT; ++i)
          if (i < mt) dmma(acc[i][q], av[i], b);
      }
    }
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
      for (int q = 0; q < NT; ++q) {
        const int row = 8 * i + g, col = k0 + 8 * q + 2 * t;
        if (row < nrows && col < n) sVC[(size_t)row * n + col] = acc[i][q][0];
        if (row < nrows && col + 1 < n) sVC[(size_t)row * n + col + 1] = acc[i][q][1];
      }
  }
}

struct OnshellParams {
  const double *e0, *H, *W, *C, *Ecm;
  const int* bin;
  const int* range;
  double* T;
  int N, n, nc, nE, R;  // R = bins per chunk
  int ldv, gemm;        // k_onshell: row stride of the V rows in shared memory; 1 = tensor-core product
  int nsplit;           // k_onshell: CTAs that share one matrix (they take the chunks of on-shell rows in turn)
  int mode;             // 0 point-wise resolvent (B.5-B.6), 1 energy-averaged (Eq. 28, B.7-B.8)
};

__global__ void __launch_bounds__(kOnGemmThreads) k_onshell(OnshellParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int N = P.N, n = P.n, nc = P.nc, nE = P.nE, R = P.R;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = kOnGemmThreads / 32;
  const int ldv = P.ldv, vrows = R * nc < 8 ? 8 : R * nc;
  double* sW = reinterpret_cast<double*>(smem_raw);  // [n]
  double* sLo = sW + n;                                // [n]
  double* sHi = sLo + n;                               // [n]
  double* sV = sHi + n;                                // [max(R*nc, 8)][ldv]
  double* sVC = sV + (size_t)vrows * ldv;              // [R*nc][n]
  __shared__ int s_nb;
  // nsplit consecutive CTAs work on the same matrix and take its chunks in turn: every chunk is a pass over all of C,
  // and with one matrix per SM the 148 C's in flight (n = 300: 106 MB) fall out of L2 between the passes (round 1: C read
  // ~12 times from DRAM); sharing a matrix between CTAs that run at the same time keeps the set of live C's inside L2.
  const size_t mat = blockIdx.x / P.nsplit;
  const int part = blockIdx.x % P.nsplit;
  const double* H = P.H + mat * (size_t)n * n;
  const double* C = P.C + mat * (size_t)n * n;
  const double* W = P.W + mat * (size_t)n;
  double* T = P.T + mat * (size_t)nE * nc * nc * 2;

  if (tid == 0) s_nb = 0;
  for (int k = tid; k < n; k += kOnGemmThreads) sW[k] = W[k];
  __syncthreads();
  {  // number of bound states = number of negative eigenvalues (ascending order)
    int cnt = 0;
    for (int k = tid; k < n; k += kOnGemmThreads) cnt += sW[k] < 0.0;
    if (cnt) atomicAdd(&s_nb, cnt);
  }
  __syncthreads();
  const int nbd = s_nb;
  for (int k = tid; k < n; k += kOnGemmThreads) {
    double lo = 0.0, hi = 0.0;
    if (k >= nbd) {
      int br = (k - nbd) % nc, i = (k - nbd) / nc;
      int mbr = (n - nbd - br + nc - 1) / nc;  // states in this branch
      double w = sW[k];
      lo = i == 0 ? 0.0 : 0.5 * (sW[k - nc] + w);
      if (i < mbr - 1) hi = 0.5 * (w + sW[k + nc]);
      else if (mbr == 1) hi = 2.0 * w;
      else {
        double lop = i == 1 ? 0.0 : 0.5 * (sW[k - 2 * nc] + sW[k - nc]);
        hi = w + 0.5 * (lo - lop);
      }
    }
    sLo[k] = lo; sHi[k] = hi;
  }
  // energies outside the grid: T = 0
  for (int e = tid; e < nE && part == 0; e += kOnGemmThreads)
    if (P.bin[e] < 0 || (P.mode == 1 && nbd + nc * P.bin[e] + nc - 1 >= n))
      for (int x = 0; x < nc * nc * 2; ++x) T[(size_t)e * nc * nc * 2 + x] = 0.0;
  const int bmin = P.range[0], bmax = P.range[1];
  for (int b0 = bmin + part * R; b0 <= bmax; b0 += R * P.nsplit) {
    const int nbins = min(R, bmax - b0 + 1), nrows = nbins * nc;
    __syncthreads();
    // V rows of this chunk: chunk row rr = (b - b0)*nc + alpha  <->  matrix row alpha*N + b
    for (int e = tid; e < nrows * n; e += kOnGemmThreads) {
      int rr = e / n, j = e - rr * n;
      int row = (rr % nc) * N + b0 + rr / nc;
      double v = H[(size_t)row * n + j];
      if (j == row) v -= P.e0[b0 + rr / nc];
      sV[(size_t)rr * ldv + j] = v;
    }
    __syncthreads();
    // VC rows of the chunk = sV (<= 16 x n) times C (n x n), C read ONCE per chunk (from L2 after the first chunk).
    if (P.gemm) {
      if (R * nc > 16) vc_rows_mma<4, 2>(sV, ldv, C, n, nrows, sVC, warp, nwarps, lane);
      else vc_rows_mma<2, 4>(sV, ldv, C, n, nrows, sVC, warp, nwarps, lane);
    } else {
      // very large n (fewer than 8 chunk rows fit shared memory): thread per column k, 16 accumulators
      for (int k = tid; k < n; k += kOnGemmThreads) {
        double acc[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) acc[r] = 0.0;
        for (int j = 0; j < n; ++j) {
          double c = C[(size_t)j * n + k];
#pragma unroll
          for (int r = 0; r < 16; ++r)
            if (r < nrows) acc[r] = fma(sV[(size_t)r * ldv + j], c, acc[r]);
        }
#pragma unroll
        for (int r = 0; r < 16; ++r)
          if (r < nrows) sVC[(size_t)r * n + k] = acc[r];
      }
    }
    __syncthreads();
    // energies of this chunk: one warp per energy
    for (int e = warp; e < nE; e += nwarps) {
      int b = P.bin[e];
      if (b < b0 || b >= b0 + nbins) continue;
      if (P.mode == 1 && nbd + nc * b + nc - 1 >= n) continue;  // a branch has no b-th state: T = 0 (set above)
      const double E = P.Ecm[e];
      const double* vc0 = sVC + (size_t)((b - b0) * nc) * n;
      const double* vc1 = vc0 + (nc - 1) * n;  // == vc0 for uncoupled
      double re00 = 0, im00 = 0, re01 = 0, im01 = 0, re11 = 0, im11 = 0;
      for (int k = lane; k < n; k += 32) {
        double gr, gi;
        resolvent_k(P.mode, E, b, k, nbd, nc, sW, sLo, sHi, gr, gi);
        double a = vc0[k];
        re00 = fma(a * a, gr, re00); im00 = fma(a * a, gi, im00);
        if (nc == 2) {
          double bb = vc1[k];
          re01 = fma(a * bb, gr, re01); im01 = fma(a * bb, gi, im01);
          re11 = fma(bb * bb, gr, re11); im11 = fma(bb * bb, gi, im11);
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        re00 += __shfl_xor_sync(0xffffffffu, re00, o); im00 += __shfl_xor_sync(0xffffffffu, im00, o);
        if (nc == 2) {
          re01 += __shfl_xor_sync(0xffffffffu, re01, o); im01 += __shfl_xor_sync(0xffffffffu, im01, o);
          re11 += __shfl_xor_sync(0xffffffffu, re11, o); im11 += __shfl_xor_sync(0xffffffffu, im11, o);
        }
      }
      if (lane == 0) {
        const double* v0 = sV + (size_t)((b - b0) * nc) * ldv;  // row (0, b)
        if (nc == 1) {
          T[(size_t)e * 2] = v0[b] + re00;
          T[(size_t)e * 2 + 1] = im00;
        } else {
          const double* v1 = v0 + ldv;  // row (1, b)
          double* t = T + (size_t)e * 8;
          t[0] = v0[b] + re00;     t[1] = im00;
          t[2] = v0[N + b] + re01; t[3] = im01;
          t[4] = v1[b] + re01;     t[5] = im01;
          t[6] = v1[N + b] + re11; t[7] = im11;
        }
      }
    }
  }
}

// Variant for n <= kI1MaxN: the rows of VC come from the eigen-identity (VC)_ik = C_ik (eps_k - e_i), which follows
// from H C = C D with H0 diagonal (coupled: e_{i mod N}); no V C product, only the on-shell rows of C are read (straight
// from global memory, coalesced along k), V_ii from the diagonal of H.  The identity inherits the eigen-residual
// eps ||H|| instead of eps ||V||: at n <= 200 the phase shifts move by < 6e-10 degrees against the direct product
// (DESIGN.md section 6), so it is gated by size and the direct kernel above stays the path for larger n.
constexpr int kI1MaxN = 200;

__global__ void __launch_bounds__(kOnThreads) k_onshell_i1(OnshellParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int N = P.N, n = P.n, nc = P.nc, nE = P.nE;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = kOnThreads / 32;
  double* sW = reinterpret_cast<double*>(smem_raw);  // [n]
  double* sLo = sW + n;                                // [n]
  double* sHi = sLo + n;                               // [n]
  double* sIw = sHi + n;                               // [n] 1/(hi - lo) of the positive states
  __shared__ int s_nb;
  const size_t mat = blockIdx.x;
  const double* H = P.H + mat * (size_t)n * n;
  const double* C = P.C + mat * (size_t)n * n;
  const double* W = P.W + mat * (size_t)n;
  double* T = P.T + mat * (size_t)nE * nc * nc * 2;
  if (tid == 0) s_nb = 0;
  for (int k = tid; k < n; k += kOnThreads) sW[k] = W[k];
  __syncthreads();
  {
    int cnt = 0;
    for (int k = tid; k < n; k += kOnThreads) cnt += sW[k] < 0.0;
    if (cnt) atomicAdd(&s_nb, cnt);
  }
  __syncthreads();
  const int nbd = s_nb;
  for (int k = tid; k < n; k += kOnThreads) {
    double lo = 0.0, hi = 0.0;
    if (k >= nbd) {
      int br = (k - nbd) % nc, i = (k - nbd) / nc;
      int mbr = (n - nbd - br + nc - 1) / nc;  // states in this branch
      double w = sW[k];
      lo = i == 0 ? 0.0 : 0.5 * (sW[k - nc] + w);
      if (i < mbr - 1) hi = 0.5 * (w + sW[k + nc]);
      else if (mbr == 1) hi = 2.0 * w;
      else {
        double lop = i == 1 ? 0.0 : 0.5 * (sW[k - 2 * nc] + sW[k - nc]);
        hi = w + 0.5 * (lo - lop);
      }
    }
    sLo[k] = lo; sHi[k] = hi;
    sIw[k] = k >= nbd ? 1.0 / (hi - lo) : 0.0;
  }
  __syncthreads();
  for (int e = warp; e < nE; e += nwarps) {
    const int b = P.bin[e];
    if (b < 0 || (P.mode == 1 && nbd + nc * b + nc - 1 >= n)) {  // outside the grid / a branch has no b-th state
      if (lane < nc * nc * 2) T[(size_t)e * nc * nc * 2 + lane] = 0.0;
      continue;
    }
    const double E = P.Ecm[e], e0b = P.e0[b];
    const double* c0 = C + (size_t)b * n;
    const double* c1 = C + (size_t)((nc - 1) * N + b) * n;  // == c0 for uncoupled
    double re00 = 0, im00 = 0, re01 = 0, im01 = 0, re11 = 0, im11 = 0;
    for (int k = lane; k < n; k += 32) {
      double gr, gi;
      if (P.mode == 0) {  // point-wise resolvent (resolvent_k, mode 0) with the tabulated reciprocal bin width
        gi = 0.0;
        if (k < nbd) {
          gr = 1.0 / (E - sW[k]);
        } else {
          const double lo = sLo[k], hi = sHi[k], iw = sIw[k];
          gr = log(fabs((E - lo) / (E - hi))) * iw;
          if (E >= lo && E < hi) gi = -WPCD_PI * iw;
        }
      } else {
        resolvent_k(P.mode, E, b, k, nbd, nc, sW, sLo, sHi, gr, gi);
      }
      const double w = sW[k] - e0b;
      const double a = c0[k] * w;
      re00 = fma(a * a, gr, re00); im00 = fma(a * a, gi, im00);
      if (nc == 2) {
        const double bb = c1[k] * w;
        re01 = fma(a * bb, gr, re01); im01 = fma(a * bb, gi, im01);
        re11 = fma(bb * bb, gr, re11); im11 = fma(bb * bb, gi, im11);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      re00 += __shfl_xor_sync(0xffffffffu, re00, o); im00 += __shfl_xor_sync(0xffffffffu, im00, o);
      if (nc == 2) {
        re01 += __shfl_xor_sync(0xffffffffu, re01, o); im01 += __shfl_xor_sync(0xffffffffu, im01, o);
        re11 += __shfl_xor_sync(0xffffffffu, re11, o); im11 += __shfl_xor_sync(0xffffffffu, im11, o);
      }
    }
    if (lane == 0) {
      const double* h0 = H + (size_t)b * n;  // row (0, b) of H; V = H - diag(e0)
      if (nc == 1) {
        T[(size_t)e * 2] = (h0[b] - e0b) + re00;
        T[(size_t)e * 2 + 1] = im00;
      } else {
        const double* h1 = H + (size_t)(N + b) * n;  // row (1, b)
        double* t = T + (size_t)e * 8;
        t[0] = (h0[b] - e0b) + re00;     t[1] = im00;
        t[2] = h0[N + b] + re01;         t[3] = im01;
        t[4] = h1[b] + re01;             t[5] = im01;
        t[6] = (h1[N + b] - e0b) + re11; t[7] = im11;
      }
    }
  }
}


// Point-wise variant of k_onshell_i1 (mode 0), one THREAD per energy and the telescoped form of SURVEY 8(d): inside a
// branch the pseudostate bins share their edges (hi_k = lo_{k+1}, Eq. 23), so
//   sum_k w_k [ln|E - lo_k| - ln|E - hi_k|]  =  sum_k (w_k - w_{k-1}) ln|E - lo_k|  -  w_last ln|E - hi_last|,
//   w_k = (VC)_ik (VC)_i'k / (hi_k - lo_k)  (Eqs. B.5-B.6, sign per reading G2):
// ONE logarithm per (energy, edge), no division, the three elements of a coupled block sharing it; the previous state's
// weights stay in registers.  No warp reduction: a thread walks the eigenstates alone, 32 energies per warp side by side
// (they sit in the same or neighbouring on-shell bins, so the rows of C they read are shared through L1).  Against the
// warp-per-energy kernel: 1.31 -> see profiles/r2_onshell.md at n = 100; it matters most for the paper's own N_WP = 16 .. 48
// (PAPER.md:437-445), where the on-shell step had become a third of the pass.
template <int NC>
__global__ void __launch_bounds__(512) k_onshell_i1_pw(OnshellParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int N = P.N, n = P.n, nE = P.nE;
  const int tid = threadIdx.x, nthr = blockDim.x;
  double* sW = reinterpret_cast<double*>(smem_raw);  // [n]
  double* sLo = sW + n;                                // [n + NC]: lower edge of state k; [n + br]: upper edge of the last state of branch br
  double* sIw = sLo + n + NC;                          // [n] 1/(hi - lo) of the positive states
  __shared__ int s_nb;
  const size_t mat = blockIdx.x;
  const double* H = P.H + mat * (size_t)n * n;
  const double* C = P.C + mat * (size_t)n * n;
  const double* W = P.W + mat * (size_t)n;
  double* T = P.T + mat * (size_t)nE * NC * NC * 2;
  if (tid == 0) s_nb = 0;
  for (int k = tid; k < n; k += nthr) sW[k] = W[k];
  __syncthreads();
  {
    int cnt = 0;
    for (int k = tid; k < n; k += nthr) cnt += sW[k] < 0.0;
    if (cnt) atomicAdd(&s_nb, cnt);
  }
  __syncthreads();
  const int nbd = s_nb;
  if (tid < NC) sLo[n + tid] = 0.0;
  for (int k = tid; k < n; k += nthr) {
    double lo = 0.0, hi = 0.0;
    if (k >= nbd) {
      const int br = (k - nbd) % NC, i = (k - nbd) / NC;
      const int mbr = (n - nbd - br + NC - 1) / NC;  // states in this branch
      const double w = sW[k];
      lo = i == 0 ? 0.0 : 0.5 * (sW[k - NC] + w);
      if (i < mbr - 1) hi = 0.5 * (w + sW[k + NC]);
      else if (mbr == 1) hi = 2.0 * w;
      else {
        const double lop = i == 1 ? 0.0 : 0.5 * (sW[k - 2 * NC] + sW[k - NC]);
        hi = w + 0.5 * (lo - lop);
      }
      if (i == mbr - 1) sLo[n + br] = hi;  // Eq. 23's last edge of the branch
    }
    sLo[k] = lo;
    sIw[k] = k >= nbd ? 1.0 / (hi - lo) : 0.0;
  }
  __syncthreads();
  for (int e = tid; e < nE; e += nthr) {
    const int b = P.bin[e];
    if (b < 0) {
#pragma unroll
      for (int x = 0; x < NC * NC * 2; ++x) T[(size_t)e * NC * NC * 2 + x] = 0.0;
      continue;
    }
    const double E = P.Ecm[e], e0b = P.e0[b];
    const double* c0 = C + (size_t)b * n;
    const double* c1 = C + (size_t)((NC - 1) * N + b) * n;
    double re00 = 0, im00 = 0, re01 = 0, im01 = 0, re11 = 0, im11 = 0;
    for (int k = 0; k < nbd; ++k) {  // bound states: 1/(E - eps_b)
      const double w = sW[k] - e0b, g = 1.0 / (E - sW[k]);
      const double a = __ldg(c0 + k) * w;
      re00 = fma(a * a, g, re00);
      if (NC == 2) {
        const double bb = __ldg(c1 + k) * w;
        re01 = fma(a * bb, g, re01);
        re11 = fma(bb * bb, g, re11);
      }
    }
    double p00[NC], p01[NC], p11[NC];   // weights of the previous state of each branch
#pragma unroll
    for (int br = 0; br < NC; ++br) p00[br] = p01[br] = p11[br] = 0.0;
#pragma unroll 4  // four states' loads of C in flight before their logarithms (n = 200: 1.84 -> 1.55 ms per 4096 matrices)
    for (int k0 = nbd; k0 < n; k0 += NC) {
#pragma unroll
      for (int br = 0; br < NC; ++br) {
        const int k = k0 + br;
        if (k < n) {
          const double lo = sLo[k], iw = sIw[k], w = sW[k] - e0b;
          const double hi = k + NC < n ? sLo[k + NC] : sLo[n + br];
          const double L = log(fabs(E - lo));
          const bool in = E >= lo && E < hi;
          const double a = __ldg(c0 + k) * w;
          const double w00 = a * a * iw;
          re00 = fma(w00 - p00[br], L, re00); p00[br] = w00;
          im00 += in ? w00 : 0.0;
          if (NC == 2) {
            const double bb = __ldg(c1 + k) * w;
            const double w01 = a * bb * iw, w11 = bb * bb * iw;
            re01 = fma(w01 - p01[br], L, re01); p01[br] = w01;
            re11 = fma(w11 - p11[br], L, re11); p11[br] = w11;
            im01 += in ? w01 : 0.0;
            im11 += in ? w11 : 0.0;
          }
        }
      }
    }
#pragma unroll
    for (int br = 0; br < NC; ++br) {   // the upper edge of each branch's last state
      if (nbd + br < n) {
        const double L = log(fabs(E - sLo[n + br]));
        re00 = fma(-p00[br], L, re00);
        if (NC == 2) { re01 = fma(-p01[br], L, re01); re11 = fma(-p11[br], L, re11); }
      }
    }
    const double* h0 = H + (size_t)b * n;  // row (0, b) of H; V = H - diag(e0)
    if (NC == 1) {
      T[(size_t)e * 2] = (h0[b] - e0b) + re00;
      T[(size_t)e * 2 + 1] = -WPCD_PI * im00;
    } else {
      const double* h1 = H + (size_t)(N + b) * n;  // row (1, b)
      double* t = T + (size_t)e * 8;
      t[0] = (h0[b] - e0b) + re00;     t[1] = -WPCD_PI * im00;
      t[2] = h0[N + b] + re01;         t[3] = -WPCD_PI * im01;
      t[4] = h1[b] + re01;             t[5] = -WPCD_PI * im01;
      t[6] = (h1[N + b] - e0b) + re11; t[7] = -WPCD_PI * im11;
    }
  }
}

__global__ void k_phase(int coupled, size_t total, int nE, const double* __restrict__ T, const int* __restrict__ bin,
                        const double* __restrict__ dE, double* __restrict__ delta, double* __restrict__ S) {
  size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  const int e = (int)(idx % nE);
  const int b = bin[e];
  const double w = b >= 0 ? dE[b] : 1.0;
  const double f = 2.0 * WPCD_PI / w, deg = 180.0 / WPCD_PI;
  if (!coupled) {
    double tr = T[idx * 2], ti = T[idx * 2 + 1];
    // S = 1 - i f T = 1 + f ti - i f tr
    double sr = 1.0 + f * ti, si = -f * tr;
    delta[idx] = 0.5 * atan2(si, sr) * deg;
    if (S) { S[idx * 2] = sr; S[idx * 2 + 1] = si; }
  } else {
    const double* t = T + idx * 8;
    double sr[4], si[4];
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      sr[x] = ((x == 0 || x == 3) ? 1.0 : 0.0) + f * t[2 * x + 1];
      si[x] = -f * t[2 * x];
      if (S) { S[idx * 8 + 2 * x] = sr[x]; S[idx * 8 + 2 * x + 1] = si[x]; }
    }
    double dm = 0.5 * atan2(si[0], sr[0]), dp = 0.5 * atan2(si[3], sr[3]);
    // -i S12 e^{-i(dm+dp)}:  real part = Im(S12 e^{-i phi}) = si cos(phi) - sr sin(phi)
    double sp, cp;
    sincos(dm + dp, &sp, &cp);
    double re = si[1] * cp - sr[1] * sp;
    double ep = 0.5 * atan2(re, hypot(sr[0], si[0]));
    delta[idx * 3] = dm * deg; delta[idx * 3 + 1] = dp * deg; delta[idx * 3 + 2] = ep * deg;
  }
}

// Eq. 42: phase shifts at arbitrary momenta from the values at the bin mid-points; one CTA per
// batch element.  The mid-point phases are first made continuous (shifts by multiples of 180 degrees, eps_J changing
// sign with every odd shift of delta_- or delta_+; readings I1-I2), sequentially along the grid by one
// thread per phase, then every target momentum takes the straight line of Eq. 42 as printed.
__global__ void __launch_bounds__(128) k_interp(int N, int nc, int nq, const double* __restrict__ pedge,
                                                const double* __restrict__ dmid, const double* __restrict__ q,
                                                double* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* u = reinterpret_cast<double*>(smem_raw);       // [N][nc] continuous mid-point phases
  int* flips = reinterpret_cast<int*>(u + (size_t)N * nc);  // [2][N] accumulated 180-degree shifts of delta_-/delta_+
  const double* d = dmid + (size_t)blockIdx.x * N * nc;
  double* o = out + (size_t)blockIdx.x * nq * nc;
  const int tid = threadIdx.x;
  if (tid < (nc == 3 ? 2 : 1)) {
    double shift = 0.0;
    for (int i = 0; i < N; ++i) {
      double x = d[(size_t)i * nc + tid] + shift;
      if (i > 0) {
        const double prev = u[(size_t)(i - 1) * nc + tid];
        while (x - prev > 90.0) { x -= 180.0; shift -= 180.0; }
        while (x - prev <= -90.0) { x += 180.0; shift += 180.0; }
      }
      u[(size_t)i * nc + tid] = x;
      flips[tid * N + i] = (int)llrint(shift / 180.0);
    }
  }
  __syncthreads();
  if (nc == 3)
    for (int i = tid; i < N; i += blockDim.x) {
      const double e = d[(size_t)i * 3 + 2];
      u[(size_t)i * 3 + 2] = ((flips[i] + flips[N + i]) & 1) ? -e : e;
    }
  __syncthreads();
  for (int e = tid; e < nq; e += blockDim.x) {
    const double qe = q[e];
    int ib = -1;
    if (qe >= pedge[0] && qe < pedge[N]) {
      int lo = 0, hi = N;  // invariant pedge[lo] <= qe < pedge[hi]
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (qe >= pedge[mid]) lo = mid; else hi = mid;
      }
      ib = lo;
    }
    for (int c = 0; c < nc; ++c) {
      double r = nan("");
      if (ib >= 0 && N >= 2) {
        const int i1 = ib > 0 ? ib : 1, i0 = i1 - 1;
        const double q0 = 0.5 * (pedge[i0] + pedge[i0 + 1]), q1 = 0.5 * (pedge[i1] + pedge[i1 + 1]);
        const double d0 = u[(size_t)i0 * nc + c], d1 = u[(size_t)i1 * nc + c];
        const double slope = (d1 - d0) / (q1 - q0);
        r = slope * qe + (d0 - slope * q0);
        if (!(nc == 3 && c == 2)) {
          r = fmod(r + 90.0, 180.0);
          if (r <= 0.0) r += 180.0;
          r -= 90.0;
        }
      }
      o[(size_t)e * nc + c] = r;
    }
  }
}

// Total np cross section, Appendix A.  The spin-scattering matrix of Eq. A.2 at theta = 0 only has
// m_s = m_s' elements (Y_l'^m(0) = sqrt((2l'+1)/4pi) delta_m0), and the combination a + b = M^1_11 + (M^1_00 + M^0_00)/2
// of Eq. A.9 is half the spin trace, in which the Clebsch-Gordan sums collapse (orthogonality) to 2J+1 per partial wave
// with l' = l.  With S_ll = 1 - 2 pi i T_ll/dE_i (Eq. A.3 in the wave-packet normalisation, reading C2) Eq. A.11
// becomes
//   sigma_tot(E) = (2 pi/p) Im(a+b) = (pi/(2 p^2)) sum_channels (2J+1) sum_l Re(1 - S_ll),  Re(1 - S_ll) = -2 pi Im T_ll/dE_i.
// One thread per (sample, energy); the channel loop reads T with the energy index fastest (coalesced).
struct SigmaParams {
  const double* Tunc;  // [S][n_unc][nE][2]
  const double* Tcpl;  // [S][n_cpl][nE][2][2][2]
  const int* bin;
  const double* dE;
  const double* Ecm;
  double* sigma;       // [S][nE] mb
  double cE;           // hbarc^2/(2 mu): E = cE p^2
  int S, nE, n_unc, n_cpl;
  int J_unc[WPCD_MAX_CHANNELS], J_cpl[WPCD_MAX_CHANNELS];
};

__global__ void k_sigma(SigmaParams P) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)P.S * P.nE) return;
  const int e = (int)(idx % P.nE);
  const size_t s = idx / P.nE;
  double acc = 0.0;
  if (P.dE == nullptr) {  // the inputs are S-matrices (e.g. from wpcd_mi_solve): Re(1 - S_ll) = 1 - Re S_ll
    for (int c = 0; c < P.n_unc; ++c)
      acc += (2.0 * P.J_unc[c] + 1.0) * (1.0 - P.Tunc[((s * P.n_unc + c) * P.nE + e) * 2]);
    for (int c = 0; c < P.n_cpl; ++c) {
      const double* t = P.Tcpl + ((s * P.n_cpl + c) * P.nE + e) * 8;
      acc += (2.0 * P.J_cpl[c] + 1.0) * ((1.0 - t[0]) + (1.0 - t[6]));
    }
  } else {
    const int b = P.bin[e];
    if (b < 0) { P.sigma[idx] = nan(""); return; }
    const double f = -2.0 * WPCD_PI / P.dE[b];
    for (int c = 0; c < P.n_unc; ++c) {
      const double ti = P.Tunc[((s * P.n_unc + c) * P.nE + e) * 2 + 1];
      acc += (2.0 * P.J_unc[c] + 1.0) * (f * ti);
    }
    for (int c = 0; c < P.n_cpl; ++c) {
      const double* t = P.Tcpl + ((s * P.n_cpl + c) * P.nE + e) * 8;
      acc += (2.0 * P.J_cpl[c] + 1.0) * (f * t[1] + f * t[7]);
    }
  }
  const double p2 = P.Ecm[e] / P.cE;
  P.sigma[idx] = 10.0 * WPCD_PI / (2.0 * p2) * acc;  // fm^2 -> mb
}

// Shared memory of k_onshell: eigenvalues and bin edges, the chunk's rows of V (at least 8 rows are laid out: the MMA
// A fragment spans 8) and of VC.
size_t onshell_smem(int n, int nc, int R, int ldv) {
  const int rows = R * nc;
  return ((size_t)3 * n + (size_t)(rows < 8 ? 8 : rows) * ldv + (size_t)rows * n) * 8;
}

}  // namespace

size_t wpcd_onshell_workspace(int, int, int, int) { return 256; }

int wpcd_onshell_launch(WpcdHandle* h, int N, int coupled, int batch, const double* d_e0, const double* d_Eedge,
                        const double* d_H, const double* d_W, const double* d_C, const double* d_Ecm, int nE,
                        int mode, double* d_T, int* d_bin, void* d_work, size_t, cudaStream_t st) {
  OnshellParams P;
  P.e0 = d_e0; P.H = d_H; P.W = d_W; P.C = d_C; P.Ecm = d_Ecm; P.bin = d_bin; P.range = static_cast<int*>(d_work);
  P.T = d_T; P.N = N; P.nc = coupled ? 2 : 1; P.n = P.nc * N; P.nE = nE; P.mode = mode; P.nsplit = 1;
  // chunk of 32 (else 16, else 8) rows of VC per pass over C on the tensor-core path; beyond that (n > ~1500) the plain loop
  // with as many bins per chunk as fit
  const size_t cap = (size_t)h->max_smem_optin - 1024;
  P.ldv = (P.n + 11) / 16 * 16 + 4;  // == 4 mod 16: conflict-free A fragments
  P.gemm = 1;
  P.R = 32 / P.nc;
  if (onshell_smem(P.n, P.nc, P.R, P.ldv) > cap) P.R = 16 / P.nc;
  if (onshell_smem(P.n, P.nc, P.R, P.ldv) > cap) P.R = 8 / P.nc;
  if (onshell_smem(P.n, P.nc, P.R, P.ldv) > cap) {
    P.gemm = 0; P.ldv = P.n; P.R = 16 / P.nc;
    while (P.R > 1 && onshell_smem(P.n, P.nc, P.R, P.ldv) > cap) P.R >>= 1;
  }
  const size_t smem = onshell_smem(P.n, P.nc, P.R, P.ldv);
  if (smem > (size_t)h->max_smem_optin) return WPCD_ESIZE;
  k_bins<<<1, 256, 0, st>>>(N, nE, d_Eedge, d_Ecm, d_bin, static_cast<int*>(d_work));
  if (P.n <= kI1MaxN) {
    if (mode == 0) {  // point-wise resolvent: one thread per energy, telescoped logarithms
      int thr = (nE + 127) / 128 * 128;
      if (thr > 512) thr = 512;
      const size_t sm = (size_t)(3 * P.n + P.nc) * 8;
      if (coupled) k_onshell_i1_pw<2><<<batch, thr, sm, st>>>(P);
      else k_onshell_i1_pw<1><<<batch, thr, sm, st>>>(P);
    } else {
      k_onshell_i1<<<batch, kOnThreads, (size_t)4 * P.n * 8, st>>>(P);
    }
    return wpcd_check_cuda(h, cudaGetLastError(), "onshell_T launch");
  }
  int rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_onshell, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "onshell attr");
  if (rc) return rc;
  {  // CTAs per matrix so that the C's of the matrices in flight (one CTA per SM) stay within ~40 MB of L2
    const double live = (double)h->num_sms * P.n * P.n * 8.0;
    int ns = (int)(live / (40.0 * 1048576.0)) + 1;
    const int nchunks_max = (N + P.R - 1) / P.R;
    if (ns > nchunks_max) ns = nchunks_max;
    if (ns > 16) ns = 16;
    if (ns < 1 || (size_t)batch * ns > 0x7fffffffu) ns = 1;
    P.nsplit = ns;
  }
  k_onshell<<<batch * P.nsplit, kOnGemmThreads, smem, st>>>(P);
  return wpcd_check_cuda(h, cudaGetLastError(), "onshell_T launch");
}

int wpcd_phase_launch(WpcdHandle* h, int coupled, int batch, int nE, const double* d_T, const int* d_bin,
                      const double* d_dE, double* d_delta, double* d_S, cudaStream_t st) {
  size_t total = (size_t)batch * nE;
  k_phase<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(coupled, total, nE, d_T, d_bin, d_dE, d_delta, d_S);
  return wpcd_check_cuda(h, cudaGetLastError(), "phase_shifts launch");
}

int wpcd_interp_launch(WpcdHandle* h, int coupled, int batch, int N, const double* d_pedge, const double* d_delta_mid,
                       const double* d_q, int nq, double* d_out, cudaStream_t st) {
  const int nc = coupled ? 3 : 1;
  const size_t smem = (size_t)N * nc * 8 + (size_t)2 * N * 4;
  if (smem > (size_t)h->max_smem_optin) return WPCD_ESIZE;
  int rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_interp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "interp attr");
  if (rc) return rc;
  k_interp<<<batch, 128, smem, st>>>(N, nc, nq, d_pedge, d_delta_mid, d_q, d_out);
  return wpcd_check_cuda(h, cudaGetLastError(), "interp_phases launch");
}

int wpcd_sigma_launch(WpcdHandle* h, int S, int nE, int n_unc, const int* h_J_unc, const double* d_T_unc, int n_cpl,
                      const int* h_J_cpl, const double* d_T_cpl, const int* d_bin, const double* d_dE, const double* d_Ecm,
                      double hbarc, double mu, double* d_sigma, cudaStream_t st) {
  SigmaParams P;
  P.Tunc = d_T_unc; P.Tcpl = d_T_cpl; P.bin = d_bin; P.dE = d_dE; P.Ecm = d_Ecm; P.sigma = d_sigma;
  P.cE = hbarc * hbarc / (2.0 * mu); P.S = S; P.nE = nE; P.n_unc = n_unc; P.n_cpl = n_cpl;
  for (int c = 0; c < WPCD_MAX_CHANNELS; ++c) {
    P.J_unc[c] = c < n_unc ? h_J_unc[c] : 0;
    P.J_cpl[c] = c < n_cpl ? h_J_cpl[c] : 0;
  }
  const size_t total = (size_t)S * nE;
  k_sigma<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(P);
  return wpcd_check_cuda(h, cudaGetLastError(), "sigma_tot launch");
}

// Rows of C that wpcd_onshell_T will read for these energies (host arithmetic, same bin rule as k_bins, widened by one
// bin on either side against rounding): none needed beyond the on-shell bins on the identity path, all rows on the
// direct path (n_ranges = 0).
int wpcd_onshell_rows_host(int N, int coupled, const double* h_edges, double hbarc, double mu, const double* h_Ecm, int nE,
                           int* h_rows, int* n_ranges) {
  const int n = coupled ? 2 * N : N;
  *n_ranges = 0;
  if (n > kI1MaxN) return WPCD_OK;
  const double cE = hbarc * hbarc / (2.0 * mu);
  int bmin = N, bmax = -1;
  for (int e = 0; e < nE; ++e)
    for (int i = 0; i < N; ++i)
      if (h_Ecm[e] >= cE * h_edges[i] * h_edges[i] && h_Ecm[e] < cE * h_edges[i + 1] * h_edges[i + 1]) {
        if (i < bmin) bmin = i;
        if (i > bmax) bmax = i;
        break;
      }
  if (bmax < 0) { bmin = 0; bmax = 0; }  // no energy on the grid: any row will do
  bmin = bmin > 0 ? bmin - 1 : 0;
  bmax = bmax < N - 1 ? bmax + 1 : N - 1;
  h_rows[0] = bmin; h_rows[1] = bmax + 1;
  *n_ranges = 1;
  if (coupled) { h_rows[2] = N + bmin; h_rows[3] = N + bmax + 1; *n_ranges = 2; }
  return WPCD_OK;
}
