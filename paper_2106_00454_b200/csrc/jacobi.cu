// jacobi.cu -- step (ii) of the WPCD recipe: H = C D C^T (Eq. 21), batched, fp64.
//
// Two-sided BLOCK Jacobi, one CTA per matrix.
//   * The n x n matrix is cut into 8-wide blocks.  A round-robin tournament pairs the blocks; each pair (I,J) is a
//     "slot" with a 16x16 symmetric pivot sub-problem S = A[IJ,IJ].
//   * Phase 1 (one warp per slot): one parallel-ordered Jacobi sweep of S (15 rounds of 8 disjoint rotations) with
//     the textbook rotation (theta, t, c, s; Rutishauser diagonal update), accumulating the 16x16 orthogonal Q.
//   * Phase 2 (all warps, dynamic work queue): A <- Q^T A Q tile by tile (only the upper slot-triangle is computed,
//     the mirror image is stored) and V <- V Q, as fp64 tensor-core products (mma.sync m8n8k4 = DMMA, which runs
//     at the full FP64 rate of the SM, 64 FMA/clk, with operands distributed over the warp).  The accumulator
//     fragment of the first product is re-used directly as the B fragment of the second one (the k index of an
//     MMA may be permuted freely), so a two-sided tile update needs no shuffle and no shared-memory round trip.
//   * A sweep = m-1 steps (m = number of blocks rounded up to even).  Converged when a whole sweep rotates nothing
//     (pivot test |a_pq| > tol sqrt(|a_pp a_qq|)).
// n <= 112: A and V live in shared memory (XOR-swizzled so that every fragment load/store pattern used below is
// bank-conflict free).  Larger n: same code on a per-CTA global workspace (L2 resident for moderate n).
//
// The rotation arithmetic follows the classical Jacobi method the paper names for this step ("parallel cyclic-order
// Jacobi"); blocking, tensor-core application and the schedule are this library's design.
#include <math.h>
#include "wpcd_internal.cuh"

namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int LDQ = 20;   // row stride of a slot's Q (doubles); == 4 mod 16 -> conflict-free fragment loads
constexpr int LDSS = 17;  // row stride of the warp-private 16x16 pivot block

// XOR swizzle of the column index (bits 2,3) by the row index; row stride must be a multiple of 16 doubles.
__device__ __forceinline__ int swz(int r, int c) { return c ^ (((r & 6) << 1) ^ ((r & 1) << 3)); }

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

// storage row of logical row k inside a slot's Q: within each group of 8 rows the order is 0,2,4,6,1,3,5,7 so that
// the k-chunks {8c+2t+r : t=0..3} used by the MMAs are 4 consecutive storage rows.
__device__ __forceinline__ int qrow(int k) { return (k & 8) | ((k & 1) << 2) | ((k >> 1) & 3); }

// Round-robin tournament (circle method) for m players, step t in [0,m-1), slot s in [0,m/2).
__device__ __forceinline__ void rr_pair(int m, int t, int s, int& a, int& b) {
  if (s == 0) { a = m - 1; b = t; }
  else { a = (t + s) % (m - 1); b = (t - s + (m - 1)) % (m - 1); }
}

struct Smem {
  double* A;     // [np][ld] swizzled (shared or global)
  double* V;     // [np][ld] swizzled
  double* Q;     // [nslots][16][LDQ]
  double* S;     // [kWarps][16][LDSS]
  double* wsort; // [np]
  int* slotI;    // [nslots]
  int* slotJ;    // [nslots]
  int* rot;      // [nslots]
  int* src;      // [np]
  int* ctr;      // [4]: 0 = work queue, 1 = rotations this sweep
  uchar2* pq;    // [15*8] pair table of the pivot sweep
};

// ---------------------------------------------------------------------------------------------- phase 1
// Pair table of one full sweep of a 16x16 pivot: 15 rounds of 8 disjoint pairs (p < q).  Rounds 0..7 take the 64
// "cross" pairs (i in block I, j in block J), rounds 8..14 the pairs inside I and inside J (two 8-player round-robin
// tournaments side by side), so every pair is met exactly once.
__device__ __forceinline__ void pivot_pair(int r, int j, int& p, int& q) {
  if (r < 8) { p = j; q = 8 + ((j + r) & 7); return; }
  int a, b;
  rr_pair(8, r - 8, j >> 1, a, b);
  const int off = (j & 1) << 3;
  p = off + (a < b ? a : b);
  q = off + (a < b ? b : a);
}

// Jacobi rotation annihilating a_pq (classical choice |angle| <= pi/4, "Jacobi method"), written with two
// reciprocal square roots and no division:  with d = a_qq - a_pp, b = 2 a_pq, h = sqrt(d^2 + b^2):
//   cos 2phi = |d|/h,  c = sqrt((1 + cos 2phi)/2),  s = sgn(d) (b/h)/(2c),  t = s/c.
__device__ __forceinline__ void rotation(double app, double aqq, double apq, double& c, double& s, double& t) {
  const double d = aqq - app, b = apq + apq;
  const double rh = rsqrt(fma(d, d, b * b));
  const double c2 = fma(0.5 * fabs(d), rh, 0.5);
  const double rc = rsqrt(c2);
  c = c2 * rc;
  s = copysign(0.5, d) * b * rh * rc;
  t = s * rc;
}

// One warp: load S = A[IJ,IJ], run one full sweep (15 rounds of 8 simultaneous rotations), write S back, leave the
// accumulated 16x16 rotation product in the slot's Q.  Lane (k0 = lane>>3, j = lane&7) owns the 2x2 blocks
// (row pair k0, column pair j) and (row pair k0+4, column pair j) of S and rows k0, k0+4, k0+8, k0+12 of Q; one
// round = S <- R^T S R, Q <- Q R with R the product of the round's 8 disjoint rotations, one __syncwarp per round.
__device__ void inner_solve(const Smem& sm, int ld, int slot, int I, int J, double tol, int lane, int warp) {
  double* S = sm.S + warp * 16 * LDSS;  // warp < min(nslots, kWarps)
  double* Q = sm.Q + slot * 16 * LDQ;
  for (int e = lane; e < 256; e += 32) {
    int a = e >> 4, b = e & 15;
    int r = 8 * (a < 8 ? I : J) + (a & 7), c = 8 * (b < 8 ? I : J) + (b & 7);
    S[a * LDSS + b] = sm.A[(size_t)r * ld + swz(r, c)];
  }
  __syncwarp();
  const int j = lane & 7, k0 = lane >> 3;
  const double tol2 = tol * tol;
  bool any = false;
#pragma unroll 1
  for (int r = 0; r < 15; ++r) {
    const uchar2 pj = sm.pq[r * 8 + j], pa = sm.pq[r * 8 + k0], pb = sm.pq[r * 8 + k0 + 4];
    const int p = pj.x, q = pj.y;
    const double app = S[p * LDSS + p], aqq = S[q * LDSS + q], apq = S[p * LDSS + q];
    double ba[4], bb[4], qx[4], qy[4];
    ba[0] = S[pa.x * LDSS + p]; ba[1] = S[pa.x * LDSS + q]; ba[2] = S[pa.y * LDSS + p]; ba[3] = S[pa.y * LDSS + q];
    bb[0] = S[pb.x * LDSS + p]; bb[1] = S[pb.x * LDSS + q]; bb[2] = S[pb.y * LDSS + p]; bb[3] = S[pb.y * LDSS + q];
#pragma unroll
    for (int u = 0; u < 4; ++u) { qx[u] = Q[(k0 + 4 * u) * LDQ + p]; qy[u] = Q[(k0 + 4 * u) * LDQ + q]; }
    // pivot test |a_pq| > tol sqrt(|a_pp a_qq|), squared
    const bool doit = apq * apq > tol2 * fabs(app * aqq);
    double c, s, t;
    rotation(app, aqq, apq, c, s, t);
    if (!doit) { c = 1.0; s = 0.0; t = 0.0; }
    any |= doit;
    const double ca = __shfl_sync(0xffffffffu, c, k0), sa = __shfl_sync(0xffffffffu, s, k0);
    const double cb = __shfl_sync(0xffffffffu, c, k0 + 4), sb = __shfl_sync(0xffffffffu, s, k0 + 4);
    {  // block (k0, j)
      double x00 = c * ba[0] - s * ba[1], x01 = s * ba[0] + c * ba[1];
      double x10 = c * ba[2] - s * ba[3], x11 = s * ba[2] + c * ba[3];
      double y00 = ca * x00 - sa * x10, y10 = sa * x00 + ca * x10;
      double y01 = ca * x01 - sa * x11, y11 = sa * x01 + ca * x11;
      if (k0 == j && doit) { y00 = app - t * apq; y11 = aqq + t * apq; y01 = 0.0; y10 = 0.0; }
      S[pa.x * LDSS + p] = y00; S[pa.x * LDSS + q] = y01; S[pa.y * LDSS + p] = y10; S[pa.y * LDSS + q] = y11;
    }
    {  // block (k0 + 4, j)
      double x00 = c * bb[0] - s * bb[1], x01 = s * bb[0] + c * bb[1];
      double x10 = c * bb[2] - s * bb[3], x11 = s * bb[2] + c * bb[3];
      double y00 = cb * x00 - sb * x10, y10 = sb * x00 + cb * x10;
      double y01 = cb * x01 - sb * x11, y11 = sb * x01 + cb * x11;
      if (k0 + 4 == j && doit) { y00 = app - t * apq; y11 = aqq + t * apq; y01 = 0.0; y10 = 0.0; }
      S[pb.x * LDSS + p] = y00; S[pb.x * LDSS + q] = y01; S[pb.y * LDSS + p] = y10; S[pb.y * LDSS + q] = y11;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      Q[(k0 + 4 * u) * LDQ + p] = c * qx[u] - s * qy[u];
      Q[(k0 + 4 * u) * LDQ + q] = s * qx[u] + c * qy[u];
    }
    __syncwarp();
  }
  const bool anyw = __any_sync(0xffffffffu, any);
  if (anyw) {
    for (int e = lane; e < 256; e += 32) {  // symmetric write-back (upper triangle is the master copy)
      int a = e >> 4, b = e & 15;
      int r = 8 * (a < 8 ? I : J) + (a & 7), c = 8 * (b < 8 ? I : J) + (b & 7);
      sm.A[(size_t)r * ld + swz(r, c)] = a <= b ? S[a * LDSS + b] : S[b * LDSS + a];
    }
  }
  if (lane == 0) {
    sm.rot[slot] = anyw ? 1 : 0;
    if (anyw) atomicAdd(&sm.ctr[1], 1);
  }
}

// ---------------------------------------------------------------------------------------------- phase 2
// T = A[P1,P2] <- Q1^T T Q2 (P = rows/cols of the slot's one or two blocks), mirrored into A[P2,P1].
__device__ __forceinline__ void apply_tile(double* __restrict__ A, int ld, const double* __restrict__ Q1,
                                           const double* __restrict__ Q2, int I1, int J1, int I2, int J2, int lane) {
  const int g = lane >> 2, t = lane & 3;
  const int n1 = J1 >= 0 ? 2 : 1, n2 = J2 >= 0 ? 2 : 1;
  const int rb[2] = {I1, J1}, cb[2] = {I2, J2};
  double2 tf[2][2];
#pragma unroll
  for (int ni = 0; ni < 2; ++ni)
#pragma unroll
    for (int c = 0; c < 2; ++c)
      if (ni < n1 && c < n2) {
        int r = 8 * rb[ni] + g, col = 8 * cb[c] + 2 * t;
        tf[ni][c] = *reinterpret_cast<const double2*>(A + (size_t)r * ld + swz(r, col));
      }
  // step A: U^T = Q2^T T^T ;  ut[mi][ni] holds U[8ni+2t+{0,1}][8mi+g]
  double ut[2][2][2];
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 2; ++ni) { ut[mi][ni][0] = 0.0; ut[mi][ni][1] = 0.0; }
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
    if (mi < n2) {
#pragma unroll
      for (int c = 0; c < 2; ++c)
        if (c < n2) {
#pragma unroll
          for (int r = 0; r < 2; ++r) {
            double a = Q2[(8 * c + 4 * r + t) * LDQ + 8 * mi + g];
#pragma unroll
            for (int ni = 0; ni < 2; ++ni)
              if (ni < n1) dmma(ut[mi][ni], a, r ? tf[ni][c].y : tf[ni][c].x);
          }
        }
    }
  // step B: T' = Q1^T U ;  out[mi][nj] = T'[8mi+g][8nj+2t+{0,1}]
  double out[2][2][2];
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int nj = 0; nj < 2; ++nj) { out[mi][nj][0] = 0.0; out[mi][nj][1] = 0.0; }
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
    if (mi < n1) {
#pragma unroll
      for (int c = 0; c < 2; ++c)
        if (c < n1) {
#pragma unroll
          for (int r = 0; r < 2; ++r) {
            double a = Q1[(8 * c + 4 * r + t) * LDQ + 8 * mi + g];
#pragma unroll
            for (int nj = 0; nj < 2; ++nj)
              if (nj < n2) dmma(out[mi][nj], a, ut[nj][c][r]);
          }
        }
    }
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int nj = 0; nj < 2; ++nj)
      if (mi < n1 && nj < n2) {
        int r = 8 * rb[mi] + g, col = 8 * cb[nj] + 2 * t;
        *reinterpret_cast<double2*>(A + (size_t)r * ld + swz(r, col)) = make_double2(out[mi][nj][0], out[mi][nj][1]);
        A[(size_t)col * ld + swz(col, r)] = out[mi][nj][0];
        A[(size_t)(col + 1) * ld + swz(col + 1, r)] = out[mi][nj][1];
      }
}

// V[rows of row-blocks rb0..rb1-1][P] <- V[..][P] Q
__device__ __forceinline__ void apply_V(double* __restrict__ V, int ld, const double* __restrict__ Q, int I, int J,
                                        int rb0, int rb1, int lane) {
  const int g = lane >> 2, t = lane & 3;
  const int nbk = J >= 0 ? 2 : 1;
  const int cb[2] = {I, J};
  double bq[2][2][2];
#pragma unroll
  for (int c = 0; c < 2; ++c)
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int ni = 0; ni < 2; ++ni) bq[c][r][ni] = (c < nbk && ni < nbk) ? Q[(8 * c + 4 * r + t) * LDQ + 8 * ni + g] : 0.0;
  for (int rb = rb0; rb < rb1; ++rb) {
    const int row = 8 * rb + g;
    double2 vf[2];
#pragma unroll
    for (int c = 0; c < 2; ++c)
      if (c < nbk) {
        int col = 8 * cb[c] + 2 * t;
        vf[c] = *reinterpret_cast<const double2*>(V + (size_t)row * ld + swz(row, col));
      }
    double out[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
    for (int c = 0; c < 2; ++c)
      if (c < nbk) {
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
          for (int ni = 0; ni < 2; ++ni)
            if (ni < nbk) dmma(out[ni], r ? vf[c].y : vf[c].x, bq[c][r][ni]);
      }
#pragma unroll
    for (int ni = 0; ni < 2; ++ni)
      if (ni < nbk) {
        int col = 8 * cb[ni] + 2 * t;
        *reinterpret_cast<double2*>(V + (size_t)row * ld + swz(row, col)) = make_double2(out[ni][0], out[ni][1]);
      }
  }
}

// ---------------------------------------------------------------------------------------------- the kernel
struct JacobiParams {
  const double* H;
  double* W;
  double* C;
  int* info;
  double* gwork;  // kGlobal: per-CTA workspace 2*np*ld doubles
  int n, batch, nb, np, ld, m, nslots, max_sweeps;
  double tol;
};

constexpr int kVRowBlocksPerItem = 2;

template <bool kGlobal>
__global__ void __launch_bounds__(kThreads, 1) k_jacobi(JacobiParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = P.n, np = P.np, ld = P.ld, nslots = P.nslots, m = P.m;
  Smem sm;
  {
    double* d = reinterpret_cast<double*>(smem_raw);
    if (kGlobal) {
      sm.A = P.gwork + (size_t)blockIdx.x * 2 * np * ld;
      sm.V = sm.A + (size_t)np * ld;
    } else {
      sm.A = d; d += (size_t)np * ld;
      sm.V = d; d += (size_t)np * ld;
    }
    sm.Q = d; d += (size_t)nslots * 16 * LDQ;
    sm.S = d; d += (nslots < kWarps ? nslots : kWarps) * 16 * LDSS;
    sm.wsort = d; d += np;
    int* ip = reinterpret_cast<int*>(d);
    sm.slotI = ip; ip += nslots;
    sm.slotJ = ip; ip += nslots;
    sm.rot = ip; ip += nslots;
    sm.src = ip; ip += np;
    sm.ctr = ip; ip += 4;
    sm.pq = reinterpret_cast<uchar2*>(ip);
  }
  if (tid < 120) {
    int p, q;
    pivot_pair(tid >> 3, tid & 7, p, q);
    sm.pq[tid] = make_uchar2((unsigned char)p, (unsigned char)q);
  }
  const int ntiles = nslots * (nslots - 1) / 2;
  const int nvgrp = (P.nb + kVRowBlocksPerItem - 1) / kVRowBlocksPerItem;
  const int nitems = ntiles + nslots * nvgrp;

  for (int mat = blockIdx.x; mat < P.batch; mat += gridDim.x) {
    const double* H = P.H + (size_t)mat * n * n;
    __syncthreads();
    for (int e = tid; e < np * np; e += kThreads) {
      int r = e / np, c = e - r * np;
      double a = (r < n && c < n) ? H[(size_t)r * n + c] : 0.0;
      sm.A[(size_t)r * ld + swz(r, c)] = a;
      sm.V[(size_t)r * ld + swz(r, c)] = (r == c) ? 1.0 : 0.0;
    }
    int sweeps = 0;
    bool converged = false;
    while (sweeps < P.max_sweeps) {
      __syncthreads();
      if (tid == 0) sm.ctr[1] = 0;
      for (int step = 0; step < m - 1; ++step) {
        // slots of this step, Q = identity
        for (int s = tid; s < nslots; s += kThreads) {
          int a, b;
          rr_pair(m, step, s, a, b);
          int I = a < b ? a : b, J = a < b ? b : a;
          if (J >= P.nb) J = -1;
          if (I >= P.nb) { I = J; J = -1; }  // cannot happen for m <= nb+1, kept for safety
          sm.slotI[s] = I; sm.slotJ[s] = J; sm.rot[s] = 0;
        }
        for (int e = tid; e < nslots * 16 * LDQ; e += kThreads) {
          int rr = (e / LDQ) & 15, cc = e % LDQ;
          sm.Q[e] = (cc < 16 && qrow(cc) == rr) ? 1.0 : 0.0;
        }
        if (tid == 0) sm.ctr[0] = 0;
        __syncthreads();
        for (int s = warp; s < nslots; s += kWarps)
          if (sm.slotJ[s] >= 0) inner_solve(sm, ld, s, sm.slotI[s], sm.slotJ[s], P.tol, lane, warp);
        __syncthreads();
        // dynamic queue over tiles (s1 < s2) and V items
        for (;;) {
          int it = 0;
          if (lane == 0) it = atomicAdd(&sm.ctr[0], 1);
          it = __shfl_sync(0xffffffffu, it, 0);
          if (it >= nitems) break;
          if (it < ntiles) {
            // unrank (s1 < s2)
            int s1 = 0, rem = it;
            while (rem >= nslots - 1 - s1) { rem -= nslots - 1 - s1; ++s1; }
            int s2 = s1 + 1 + rem;
            if (sm.rot[s1] | sm.rot[s2])
              apply_tile(sm.A, ld, sm.Q + s1 * 16 * LDQ, sm.Q + s2 * 16 * LDQ, sm.slotI[s1], sm.slotJ[s1], sm.slotI[s2],
                         sm.slotJ[s2], lane);
          } else {
            int v = it - ntiles;
            int s = v / nvgrp, grp = v - s * nvgrp;
            if (sm.rot[s]) {
              int rb0 = grp * kVRowBlocksPerItem, rb1 = rb0 + kVRowBlocksPerItem;
              if (rb1 > P.nb) rb1 = P.nb;
              apply_V(sm.V, ld, sm.Q + s * 16 * LDQ, sm.slotI[s], sm.slotJ[s], rb0, rb1, lane);
            }
          }
        }
        __syncthreads();
      }
      ++sweeps;
      if (sm.ctr[1] == 0) { converged = true; break; }
    }
    // eigenvalues = diagonal; rank sort ascending (ties by index); gather columns
    __syncthreads();
    for (int k = tid; k < n; k += kThreads) sm.wsort[k] = sm.A[(size_t)k * ld + swz(k, k)];
    __syncthreads();
    for (int k = tid; k < n; k += kThreads) {
      double wk = sm.wsort[k];
      int rank = 0;
      for (int j = 0; j < n; ++j) {
        double wj = sm.wsort[j];
        rank += (wj < wk) || (wj == wk && j < k);
      }
      sm.src[rank] = k;
    }
    __syncthreads();
    double* Wo = P.W + (size_t)mat * n;
    double* Co = P.C + (size_t)mat * n * n;
    for (int k = tid; k < n; k += kThreads) Wo[k] = sm.wsort[sm.src[k]];
    for (int e = tid; e < n * n; e += kThreads) {
      int i = e / n, k = e - i * n;
      int c = sm.src[k];
      Co[e] = sm.V[(size_t)i * ld + swz(i, c)];
    }
    if (tid == 0) P.info[mat] = converged ? sweeps : -1;
  }
}

struct Geometry { int nb, np, ld, m, nslots; size_t smem_fixed, smem_mat; };

Geometry geometry(int n) {
  Geometry g;
  g.nb = (n + 7) / 8;
  if (g.nb < 2) g.nb = 2;
  g.np = 8 * g.nb;
  g.ld = (g.np + 15) / 16 * 16;
  g.m = (g.nb & 1) ? g.nb + 1 : g.nb;
  g.nslots = g.m / 2;
  g.smem_fixed = (size_t)g.nslots * 16 * LDQ * 8 + (size_t)(g.nslots < kWarps ? g.nslots : kWarps) * 16 * LDSS * 8 + (size_t)g.np * 8 +
                 (size_t)(3 * g.nslots + g.np + 4) * 4 + 240 + 64;
  g.smem_mat = (size_t)2 * g.np * g.ld * 8;
  return g;
}

// CTAs of the global-workspace path: two per SM while all their workspaces together stay well inside the 126 MB L2.
int global_grid(const WpcdHandle* h, const Geometry& g, int batch) {
  int per_sm = ((size_t)2 * h->num_sms * g.smem_mat <= ((size_t)80 << 20)) ? 2 : 1;
  int grid = per_sm * h->num_sms;
  return batch < grid ? batch : grid;
}

}  // namespace

size_t wpcd_jacobi_workspace(const WpcdHandle* h, int n, int batch) {
  Geometry g = geometry(n);
  if (g.smem_fixed + g.smem_mat <= (size_t)h->max_smem_optin) return 0;
  int grid = global_grid(h, g, batch);
  return (size_t)grid * g.smem_mat;
}

int wpcd_jacobi_launch(WpcdHandle* h, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                       double tol, int max_sweeps, void* d_work, size_t work_bytes, cudaStream_t st) {
  Geometry g = geometry(n);
  JacobiParams P;
  P.H = d_A; P.W = d_W; P.C = d_C; P.info = d_info; P.gwork = static_cast<double*>(d_work);
  P.n = n; P.batch = batch; P.nb = g.nb; P.np = g.np; P.ld = g.ld; P.m = g.m; P.nslots = g.nslots;
  P.max_sweeps = max_sweeps;
  P.tol = tol > 0.0 ? tol : 2.220446049250313e-16;
  const bool in_smem = g.smem_fixed + g.smem_mat <= (size_t)h->max_smem_optin;
  int rc;
  if (in_smem) {
    size_t smem = g.smem_fixed + g.smem_mat;
    rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_jacobi<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "jacobi attr");
    if (rc) return rc;
    k_jacobi<false><<<batch, kThreads, smem, st>>>(P);
  } else {
    if (g.smem_fixed > (size_t)h->max_smem_optin) return WPCD_ESIZE;
    int grid = global_grid(h, g, batch);
    if (work_bytes < (size_t)grid * g.smem_mat) return WPCD_EWORK;
    rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_jacobi<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g.smem_fixed), "jacobi attr");
    if (rc) return rc;
    k_jacobi<true><<<grid, kThreads, g.smem_fixed, st>>>(P);
  }
  return wpcd_check_cuda(h, cudaGetLastError(), "diag_batched launch");
}
