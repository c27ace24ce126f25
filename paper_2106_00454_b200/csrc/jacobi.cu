// jacobi.cu -- step (ii) of the WPCD recipe: H = C D C^T (Eq. 21), batched, fp64.
//
// Two-sided BLOCK Jacobi, one CTA per matrix, software-pipelined over the steps of the block tournament.
//   * The n x n matrix is cut into 8-wide blocks.  A round-robin tournament (jacobi_schedule.cuh; tables written once
//     per launch by k_schedule) pairs the blocks; each pair (I,J) is a "slot" with a 16x16 symmetric pivot
//     sub-problem S = A[IJ,IJ].
//   * Pivot solve (one warp per slot): one Brent-Luk sweep of S -- all 120 pairs (15 rounds of 8 disjoint rotations)
//     at about three steps per tournament sweep, the 64 pairs between the two blocks (8 rounds) otherwise -- with the
//     classical rotation angle, division-free, accumulating the 16x16 orthogonal Q in registers.  A serial chain of rounds: latency/issue bound.
//   * Apply (all warps, dynamic work queue): A <- Q^T A Q tile by tile (one tile per slot pair) and V <- V Q, as fp64
//     tensor-core products (mma.sync m8n8k4 = DMMA, same flop rate as DFMA on B200 but operands distributed over the
//     warp).  The accumulator fragment of the first product is re-used directly as the B fragment of the second one
//     (the k index of an MMA may be permuted freely): no shuffle, no shared-memory round trip between the two sides.
//   * Pipeline: the pivot of a slot of step g+1 only needs ONE tile of step g (its "critical" tile) besides the
//     diagonal blocks.  In phase g a warp updates its critical tile and goes straight on to the pivot solve of step
//     g+1 (into the other Q buffer), then joins the queue of the other tiles and the V updates of step g; one
//     __syncthreads per step.
//   * A sweep = m-1 steps.  Converged when a whole sweep rotates nothing (pivot test |a_pq| > tol sqrt(|a_pp a_qq|)).
//   * Matrices are handed out to the CTAs dynamically (global counter): they need 6-8 sweeps each.
//   * Rows/columns are relabelled in the order of descending diagonal entries (de Rijk): on the graded WPCD Hamiltonians
//     the sweeps converge faster than in the natural ascending order (n=200: 7.0 -> 6.3 sweeps).
// n <= 200: A (upper 8x8 blocks) and Q in shared memory, V in a per-CTA global workspace that stays L2 resident; for
// n <= 104 with 320 threads (n <= 56: 160) so that 2 (4) matrices share an SM.
// 200 < n <= 848 (A does not fit shared memory, the Q buffers do): LOG MODE.  V <- V Q never feeds back into the sweeps, and
// with A and V both streaming through L2/DRAM every step the launch was DRAM-bound (174 GB per 592 matrices at n = 300).
// So the sweeps run on A alone (through L2), every rotating slot appends its 16x16 product to a log region, and the same
// persistent launch later REPLAYS the log: a CTA takes a panel of <= 64 rows of the identity into shared memory, applies
// the logged products in order (one barrier per tournament step) and writes the rows of C.  Solve jobs and replay units
// are handed out by a small scheduler in global memory (replay first, so that the two log regions of every CTA drain).
// Same products in the same order: bit-identical to the accumulation in place; a tenth of the DRAM traffic.
// Larger n (the Q buffers do not fit either): A, V and Q in the workspace.
//
// The rotation arithmetic follows the classical Jacobi method the paper names for this step ("parallel cyclic-order
// Jacobi"); blocking, tensor-core application, pipelining and the schedule are this library's.
#include <math.h>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <type_traits>
#include "jacobi_rotation.cuh"
#include "jacobi_schedule.cuh"
#include "wpcd_internal.cuh"

namespace {

// Optional cycle counters (only in profiling builds, -DWPCD_PROFILE), accumulated by CTA 0:
//   [0] whole steps (thread 0), [1] critical tile + pivot solve of warp 1, [2] number of steps,
//   [3] queue part of warp 15, [4] queue part of warp 1, [5] whole matrices (load, ordering, sweeps, write-back; thread 0),
//   [6] load + ordering + V = 1 part, [7] sort + write-back part
#ifdef WPCD_PROFILE
__device__ long long wpcd_prof[8];
#define WPCD_PROF_ADD(k, v) atomicAdd((unsigned long long*)&wpcd_prof[k], (unsigned long long)(v))
#endif

constexpr int LDQ = 16;   // row stride of a slot's Q (doubles), column pairs XOR-swizzled by the storage row
constexpr int kQSlot = 16 * LDQ;

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

// Q layout: logical row k sits in storage row qrow(k) -- within each group of 8 rows the order is 0,2,4,6,1,3,5,7 so
// that the k-chunks {8c+2t+r : t=0..3} used by the MMAs are 4 consecutive storage rows -- and column c of storage
// row sr sits at 2 ((c & 7) ^ 2 (sr & 3)) + (c >> 3): columns g and 8+g are adjacent (one 16-byte load feeds both
// column blocks of an MMA step) and the fragment loads are bank-conflict free with LDQ = 16.
__device__ __forceinline__ int qoff(int sr, int c) { return sr * LDQ + 2 * ((c & 7) ^ (2 * (sr & 3))) + (c >> 3); }
__device__ __forceinline__ int qrow(int k) { return (k & 8) | ((k & 1) << 2) | ((k >> 1) & 3); }

// View of the symmetric working matrix A (shared memory in mode 1, global workspace in modes 2 and 3): only the 8x8
// blocks (rb <= cb) are stored, 64 contiguous doubles each; a block below the diagonal is read/written through its
// transpose.  Half the footprint of a full mirrored array (which the workspace modes used at first: 20 % slower):
// n = 200 fits shared memory.  Inside a block row r sits in row slot prow(r) = 0,4,1,5,2,6,3,7: a row is 8 doubles = half
// the banks, and with this order the transposed fragment access (rows 2t resp. 2t+1, t = 0..3, column g) spreads over
// both halves -- 2 wavefronts instead of 4-6 -- while the direct access stays conflict free.
__device__ __forceinline__ int prow(int r) { return ((r & 1) << 2) | (r >> 1); }

struct AView {
  double* p;
  int nb;
  __device__ __forceinline__ size_t blk(int rb, int cb) const { return (size_t)(rb * nb - ((rb * (rb - 1)) >> 1) + (cb - rb)) << 6; }
  __device__ __forceinline__ double get(int r, int c) const {
    const int rb = r >> 3, cb = c >> 3;
    return rb <= cb ? p[blk(rb, cb) + (prow(r & 7) << 3) + (c & 7)] : p[blk(cb, rb) + (prow(c & 7) << 3) + (r & 7)];
  }
  // element (r,c) of a symmetric update where the caller visits BOTH (r,c) and (c,r)
  __device__ __forceinline__ void put(int r, int c, double v) const {
    const int rb = r >> 3, cb = c >> 3;
    if (rb <= cb) p[blk(rb, cb) + (prow(r & 7) << 3) + (c & 7)] = v;
  }
  // fragment of the off-diagonal block (rb != cb): rows 8rb+g, columns 8cb+2t, 8cb+2t+1
  __device__ __forceinline__ double2 load_frag(int rb, int cb, int g, int t) const {
    if (rb < cb) return *reinterpret_cast<const double2*>(p + blk(rb, cb) + (prow(g) << 3) + 2 * t);
    const double* q = p + blk(cb, rb) + (t << 3) + g;  // rows 2t, 2t+1 of the stored block: slots t, 4+t
    return make_double2(q[0], q[32]);
  }
  __device__ __forceinline__ void store_frag(int rb, int cb, int g, int t, double v0, double v1) const {
    if (rb < cb) { *reinterpret_cast<double2*>(p + blk(rb, cb) + (prow(g) << 3) + 2 * t) = make_double2(v0, v1); return; }
    double* q = p + blk(cb, rb) + (t << 3) + g;
    q[0] = v0; q[32] = v1;
  }
};

struct Smem {
  double* A;     // upper 8x8 blocks of the symmetric working matrix, see AView (shared or global)
  double* V;     // [nb][nb] blocks of 8x8 (64 contiguous doubles, row-major inside), global workspace: see vidx
  double* Q;     // [2][nslots][16][LDQ] (shared or global), double buffered over the steps
  double* wsort; // [np]
  int* rot;      // [2][nslots] slot rotated something
  int* src;      // [np]
  int* ctr;      // [0..1] work queues (step parity), [2..3] rotations per sweep (sweep parity)
  int* act;      // [nb] active row blocks of V (those that hold wanted rows of C)
  int* perm;     // [np] internal row/column i holds original index perm[i] & 0xFFFF; bit 16: row i of C is wanted
  const int* tab; // slot and feed tables [2][m-1][nslots]: shared-memory copy (modes 0, 1) or k_schedule's global ones
  // log mode: the log region of the matrix being solved (ctr[4] = entries so far, ctr[5] = overflow)
  double* logq;   // [log_cap][256] rotation products in the layout of a slot's Q
  int* logtag;    // [log_cap] I | J << 16
  int logcap;
};

// ---------------------------------------------------------------------------------------------- pivot solve
// Tournament of one full sweep of a 16x16 pivot (Brent-Luk): positions 0..15, pair j = positions (2j, 2j+1); after
// every round the data moves to position kPi(x) (position 0 stays, the other 15 rotate), so that after 15 rounds every
// pair has met exactly once and everything is back where it started.  The addressing of a round is therefore static.
__device__ __forceinline__ int kPi(int x) {
  if (x == 0) return 0;
  if (x == 1) return 2;
  if (x == 14) return 15;
  return (x & 1) ? x - 2 : x + 2;
}

// Cross-only tournament: the even positions (block I) stay, the odd ones (block J) move on by one pair, so that 8
// rounds meet the 64 pairs (i in I, j in J) exactly once and everything is back where it started.
__device__ __forceinline__ int kPiCross(int x) { return (x & 1) ? (((x >> 1) + 1) & 7) * 2 + 1 : x; }

// Pivot solve.  One warp: load S = A[IJ,IJ] into the scratch (position 2i = i-th index of block I, 2i+1 = i-th of J),
// run one sweep -- full: 15 rounds of 8 simultaneous rotations over all 120 pairs (Brent-Luk); cross: 8 rounds over
// the 64 pairs between the two blocks -- write S back, and write the accumulated 16x16 rotation product over the
// scratch (which is the slot's Q array) in the layout of the DMMA B fragments.  Returns (warp-uniform) whether
// anything was rotated.  Lane (k0 = lane>>3, j = lane&7) owns the 2x2 blocks (row pair k0, column pair j) and (row
// pair k0+4, column pair j) of S, which go through shared memory every round (static addresses: the data moves to the
// next round's positions, not the pairing), and storage rows k0, k0+4, k0+8, k0+12 of Q at column pair j, which stay
// in registers (the columns travel between the lanes of a k0 group by shuffle).  One round = S <- R^T S R, Q <- Q R
// with R the product of the round's 8 disjoint rotations.  The next round's pivots (a_pp, a_qq, a_pq) are fetched by
// shuffle right after the update, so that the next rotation (a long dependent chain) overlaps this round's stores.
__device__ __forceinline__ bool inner_solve(const AView& A, double* __restrict__ S, int I, int J, double tol,
                                            bool full, int lane) {
  constexpr int LDS_ = 16;  // S is the slot's 16 x LDQ array: a row = all 32 banks
  const int j = lane & 7, k0 = lane >> 3;
  const double tol2 = tol * tol;
  bool need = false;  // early exit: no pair of this sweep passes the rotation test (the usual case in the last sweeps)
  // Lane (h = lane >> 4, gam = lane & 15) moves column gam of the rows 2k + h of S: always the same block of A.
  const int h = lane >> 4, gam = lane & 15, bet = gam & 1;
  {
    const int b = gam >> 1;
    const double* src;
    int stride = 8;
    if (h == 0) src = A.p + A.blk(I, bet ? J : I) + b;                 // (I,I) or (I,J): element [k][b]
    else if (bet) src = A.p + A.blk(J, J) + b;                          // (J,J)
    else { src = A.p + A.blk(I, J) + 8 * prow(b); stride = 1; }         // (J,I) = transpose of (I,J): element [b][k]
#pragma unroll 4
    for (int k = 0; k < 8; ++k) S[(2 * k + h) * LDS_ + gam] = src[(stride == 8 ? prow(k) : k) * stride];
    __syncwarp();
    const double dg = S[gam * (LDS_ + 1)];
    const bool par = full || (h != bet);
#pragma unroll 4
    for (int k = 0; k < 8; ++k) {
      const int rho = 2 * k + h;
      const double x = S[rho * LDS_ + gam];
      need |= par && (rho < gam) && (x * x > tol2 * fabs(S[rho * (LDS_ + 1)] * dg));
    }
  }
  need = __any_sync(0xffffffffu, need);
  // static addresses: loads at (row pair, column pair), stores at the permuted positions
  const double* ldA = S + (2 * k0) * LDS_ + 2 * j;
  const double* ldB = S + (2 * k0 + 8) * LDS_ + 2 * j;
  const int cp = full ? kPi(2 * j) : kPiCross(2 * j), cq = full ? kPi(2 * j + 1) : kPiCross(2 * j + 1);
  double* stA0 = S + (full ? kPi(2 * k0) : kPiCross(2 * k0)) * LDS_;
  double* stA1 = S + (full ? kPi(2 * k0 + 1) : kPiCross(2 * k0 + 1)) * LDS_;
  double* stB0 = S + (full ? kPi(2 * k0 + 8) : kPiCross(2 * k0 + 8)) * LDS_;
  double* stB1 = S + (full ? kPi(2 * k0 + 9) : kPiCross(2 * k0 + 9)) * LDS_;
  // Look-ahead sources.  Full tournament: the next pivot of pair j sits, before the move, at rows/columns
  //   j:      0      1      2..6            7
  //   x, y:   0,3    1,5    2j-2, 2j+3      12,14
  // (diagonal entries from the rotations of pairs x/2, y/2; off-diagonal entry owned by lanes 1,2,11,20,29,6,15,23).
  // Cross tournament: x = 2j (own pair), y = 2((j-1)&7)+1: entry (0,1) of block (row pair j, column pair j-1).
  const int grp = lane & ~7;
  const int src_pp = full ? (j > 0 ? j - 1 : 0) : j;
  const int src_qq = full ? (j < 7 ? j + 1 : 7) : ((j + 7) & 7);
  const bool fix0 = full && j == 0, fix7 = full && j == 7;
  const int own_src = full ? (int)((0x170F061D140B0201ull >> (8 * j)) & 0xff) : 8 * (j & 3) + ((j + 7) & 7);
  int own_sel;  // which of its entries a lane supplies: 0 yA01, 1 yA11, 2 yB01, 3 yB00
  if (full) own_sel = lane == 2 ? 1 : ((lane == 6 || lane == 15) ? 2 : (lane == 23 ? 3 : 0));
  else own_sel = (((j + 1) & 7) < 4) ? 0 : 2;
  // Q[storage row k0 + 4u][position 2j], [position 2j + 1]; identity: local row k sits in storage row qrow(k), and
  // position 2i (2i+1) is local column i (8+i)
  double qt[4], qb[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    qt[u] = (qrow(j) == k0 + 4 * u) ? 1.0 : 0.0;
    qb[u] = (qrow(8 + j) == k0 + 4 * u) ? 1.0 : 0.0;
  }
  double app = 1.0, aqq = 1.0, apq = 0.0, c, s, t;
  if (need) {
    const double2 d0 = *reinterpret_cast<const double2*>(S + (2 * j) * LDS_ + 2 * j);
    const double2 d1 = *reinterpret_cast<const double2*>(S + (2 * j + 1) * LDS_ + 2 * j);
    app = d0.x; apq = d0.y; aqq = d1.y;
  }
  bool doit = rotation(app, aqq, apq, tol2, c, s, t);
  bool any = false;
  // The round loop, compiled twice: in the cross tournament the even positions never move, so the pivot's a_pp, the
  // first Q column of a pair and the exceptions of positions 0 and 15 need no shuffle and no select.
  auto rounds = [&](auto full_c) {
    constexpr bool kFull = decltype(full_c)::value;
    constexpr int nrounds = kFull ? 15 : 8;
    const bool f0 = kFull && fix0, f7 = kFull && fix7;
#pragma unroll 1
    for (int r = 0; r < nrounds; ++r) {
      const double2 a0 = *reinterpret_cast<const double2*>(ldA);
      const double2 a1 = *reinterpret_cast<const double2*>(ldA + LDS_);
      const double2 b0 = *reinterpret_cast<const double2*>(ldB);
      const double2 b1 = *reinterpret_cast<const double2*>(ldB + LDS_);
      __syncwarp();  // every lane has read its inputs before anybody stores
      any |= doit;
      const double ca = __shfl_sync(0xffffffffu, c, k0), sa = __shfl_sync(0xffffffffu, s, k0);
      const double cb = __shfl_sync(0xffffffffu, c, k0 + 4), sb = __shfl_sync(0xffffffffu, s, k0 + 4);
      const double dtop = app - t * apq, dbot = aqq + t * apq;  // rotated diagonal of pair j (t = 0: unchanged)
      // block (k0, j)
      const double xa00 = c * a0.x - s * a0.y, xa01 = s * a0.x + c * a0.y;
      const double xa10 = c * a1.x - s * a1.y, xa11 = s * a1.x + c * a1.y;
      const double ya00 = ca * xa00 - sa * xa10, ya10 = sa * xa00 + ca * xa10;
      const double ya01 = ca * xa01 - sa * xa11, ya11 = sa * xa01 + ca * xa11;
      // block (k0 + 4, j)
      const double xb00 = c * b0.x - s * b0.y, xb01 = s * b0.x + c * b0.y;
      const double xb10 = c * b1.x - s * b1.y, xb11 = s * b1.x + c * b1.y;
      const double yb00 = cb * xb00 - sb * xb10, yb10 = sb * xb00 + cb * xb10;
      const double yb01 = cb * xb01 - sb * xb11, yb11 = sb * xb01 + cb * xb11;
      // next round's pivot by shuffle
      double zsel;
      if (kFull) zsel = own_sel == 0 ? ya01 : (own_sel == 1 ? ya11 : (own_sel == 2 ? yb01 : yb00));
      else zsel = own_sel == 0 ? ya01 : yb01;
      double appn = dtop;
      if (kFull) appn = __shfl_sync(0xffffffffu, f0 ? dbot : dtop, src_pp);
      double aqqn = __shfl_sync(0xffffffffu, dbot, src_qq);
      const double apqn = __shfl_sync(0xffffffffu, zsel, own_src);
      if (f0) appn = dtop;
      if (f7) aqqn = dtop;
      // this round's stores, at the positions of the next round
      stA0[cp] = ya00; stA0[cq] = ya01; stA1[cp] = ya10; stA1[cq] = ya11;
      stB0[cp] = yb00; stB0[cq] = yb01; stB1[cp] = yb10; stB1[cq] = yb11;
      // Q <- Q R, then the columns move like the positions
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const double nt = c * qt[u] - s * qb[u], nb = s * qt[u] + c * qb[u];
        double mt = nt;
        if (kFull) mt = __shfl_sync(0xffffffffu, f0 ? nb : nt, grp | src_pp);
        const double mb = __shfl_sync(0xffffffffu, nb, grp | src_qq);
        qt[u] = f0 ? nt : mt;
        qb[u] = f7 ? nt : mb;
      }
      app = appn; aqq = aqqn; apq = apqn;
      doit = rotation(app, aqq, apq, tol2, c, s, t);  // independent of the stores above: overlaps them
      __syncwarp();
    }
  };
  if (need) {
    if (full) rounds(std::true_type{});
    else rounds(std::false_type{});
  }
  const bool anyw = __any_sync(0xffffffffu, any);
  if (anyw) {
    for (int e = lane; e < 256; e += 32) {
      const int a = e >> 4, b = e & 15;
      const int r = 8 * ((a & 1) ? J : I) + (a >> 1), c2 = 8 * ((b & 1) ? J : I) + (b >> 1);
      A.put(r, c2, a <= b ? S[a * LDS_ + b] : S[b * LDS_ + a]);
    }
  }
  __syncwarp();
  // Q over the scratch (layout qoff): position 2j -> local column j, 2j+1 -> 8+j, which are adjacent
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    *reinterpret_cast<double2*>(S + qoff(k0 + 4 * u, j)) = make_double2(qt[u], qb[u]);
  }
  return anyw;
}

// ---------------------------------------------------------------------------------------------- apply
// T = A[P1,P2] <- Q1^T T Q2 (P = rows/cols of the slot's one or two blocks), mirrored into A[P2,P1].
template <int n1, int n2>
__device__ __forceinline__ void apply_tile_n(const AView& A, const double* __restrict__ Q1,
                                             const double* __restrict__ Q2, int I1, int J1, int I2, int J2, int lane) {
  const int g = lane >> 2, t = lane & 3;
  const int rb[2] = {I1, J1}, cb[2] = {I2, J2};
  double2 tf[2][2];
#pragma unroll
  for (int ni = 0; ni < 2; ++ni)
#pragma unroll
    for (int c = 0; c < 2; ++c)
      if (ni < n1 && c < n2) tf[ni][c] = A.load_frag(rb[ni], cb[c], g, t);
  // Q fragments: one 16-byte load gives the entries of columns g and 8+g of storage row 8c+4r+t
  double2 q2[2][2], q1[2][2];
#pragma unroll
  for (int c = 0; c < 2; ++c)
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      if (c < n2) q2[c][r] = *reinterpret_cast<const double2*>(Q2 + qoff(8 * c + 4 * r + t, g));
      if (c < n1) q1[c][r] = *reinterpret_cast<const double2*>(Q1 + qoff(8 * c + 4 * r + t, g));
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
            const double a = mi ? q2[c][r].y : q2[c][r].x;
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
            const double a = mi ? q1[c][r].y : q1[c][r].x;
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
      if (mi < n1 && nj < n2) A.store_frag(rb[mi], cb[nj], g, t, out[mi][nj][0], out[mi][nj][1]);
}

// the usual case (two full slots) gets code without predication
__device__ __forceinline__ void apply_tile(const AView& A, const double* __restrict__ Q1,
                                           const double* __restrict__ Q2, int I1, int J1, int I2, int J2, int lane) {
  if (J1 >= 0 && J2 >= 0) apply_tile_n<2, 2>(A, Q1, Q2, I1, J1, I2, J2, lane);
  else if (J1 >= 0) apply_tile_n<2, 1>(A, Q1, Q2, I1, J1, I2, J2, lane);
  else if (J2 >= 0) apply_tile_n<1, 2>(A, Q1, Q2, I1, J1, I2, J2, lane);
  else apply_tile_n<1, 1>(A, Q1, Q2, I1, J1, I2, J2, lane);
}

// V (the accumulated eigenvectors) is kept block-wise: element (r, c) of block (r/8, c/8) at 8 (r%8) + c%8 inside 64
// contiguous doubles.  An update item then reads and writes whole 512-byte blocks instead of 64-byte pieces of rows
// 8 ld bytes apart (what the DRAM-bound workspace modes want; the L2-resident shared-memory mode does not care).
__device__ __forceinline__ size_t vidx(int nb, int r, int c) {
  return ((size_t)((r >> 3) * nb + (c >> 3)) << 6) + ((r & 7) << 3) + (c & 7);
}

// V[rows of the given row blocks][P] <- V[..][P] Q (V lives in global memory in every mode: L2 latency, so all loads of
// a pair of row blocks are in flight before the first product).
// One V item: row blocks rb[0..nrb-1] of V times the same Q, two row blocks at a time; the Q fragments are loaded once.
// Items of 4 row blocks (half the queue traffic and Q loads of items of 2: n=200 6 % faster; with A's upper-block layout
// in the workspace modes too: n=300 3 % faster, together with the interleaved queue order 11 %; items of 8: slower).

template <int nbk, bool kQcg = false>
__device__ __forceinline__ void apply_V_item(double* __restrict__ V, int nb, const double* __restrict__ Q, int I, int J,
                                             const int* __restrict__ rb, int nrb, int lane, bool kStream) {
  const int g = lane >> 2, t = lane & 3;
  const int cb[2] = {I, J};
  double2 bq[2][2];
#pragma unroll
  for (int c = 0; c < nbk; ++c)
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      if (kQcg) bq[c][r] = __ldcg(reinterpret_cast<const double2*>(Q + qoff(8 * c + 4 * r + t, g)));  // written by another CTA: L2 only
      else bq[c][r] = *reinterpret_cast<const double2*>(Q + qoff(8 * c + 4 * r + t, g));
    }
#pragma unroll 1
  for (int k = 0; k < nrb; k += 2) {
    const bool two = k + 1 < nrb;
    double* v0 = V + ((size_t)(rb[k] * nb) << 6) + 8 * g + 2 * t;
    double* v1 = V + ((size_t)(rb[two ? k + 1 : k] * nb) << 6) + 8 * g + 2 * t;
    double2 f0[2], f1[2];
#pragma unroll
    for (int c = 0; c < nbk; ++c) {
      if (kStream) {  // workspace modes, while all CTAs' A blocks together fit L2: V streams through L2 (evict first) and A stays resident
        f0[c] = __ldcs(reinterpret_cast<const double2*>(v0 + 64 * cb[c]));
        f1[c] = __ldcs(reinterpret_cast<const double2*>(v1 + 64 * cb[c]));
      } else {
        f0[c] = *reinterpret_cast<const double2*>(v0 + 64 * cb[c]);
        f1[c] = *reinterpret_cast<const double2*>(v1 + 64 * cb[c]);
      }
    }
    double o0[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, o1[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
    for (int c = 0; c < nbk; ++c)
#pragma unroll
      for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int ni = 0; ni < nbk; ++ni) {
          const double q = ni ? bq[c][r].y : bq[c][r].x;
          dmma(o0[ni], r ? f0[c].y : f0[c].x, q);
          dmma(o1[ni], r ? f1[c].y : f1[c].x, q);
        }
#pragma unroll
    for (int ni = 0; ni < nbk; ++ni) {
      if (kStream) {
        __stcs(reinterpret_cast<double2*>(v0 + 64 * cb[ni]), make_double2(o0[ni][0], o0[ni][1]));
        if (two) __stcs(reinterpret_cast<double2*>(v1 + 64 * cb[ni]), make_double2(o1[ni][0], o1[ni][1]));
      } else {
        *reinterpret_cast<double2*>(v0 + 64 * cb[ni]) = make_double2(o0[ni][0], o0[ni][1]);
        if (two) *reinterpret_cast<double2*>(v1 + 64 * cb[ni]) = make_double2(o1[ni][0], o1[ni][1]);
      }
    }
  }
}

// The same product for the replay of the log mode, with the B fragments of Q already in registers (they are loaded, through
// L2 only, before the warp waits for its item's turn).  Same arithmetic and order as apply_V_item<2>.
__device__ __forceinline__ void load_bq_cg(const double* __restrict__ Q, int lane, double2 (&bq)[2][2]) {
  const int g = lane >> 2, t = lane & 3;
#pragma unroll
  for (int c = 0; c < 2; ++c)
#pragma unroll
    for (int r = 0; r < 2; ++r) bq[c][r] = __ldcg(reinterpret_cast<const double2*>(Q + qoff(8 * c + 4 * r + t, g)));
}
__device__ __forceinline__ void apply_V_bq(double* __restrict__ V, int nb, const double2 (&bq)[2][2], int I, int J,
                                           const int* __restrict__ rb, int nrb, int lane) {
  const int g = lane >> 2, t = lane & 3;
  const int cb[2] = {I, J};
#pragma unroll 1
  for (int k = 0; k < nrb; k += 2) {
    const bool two = k + 1 < nrb;
    double* v0 = V + ((size_t)(rb[k] * nb) << 6) + 8 * g + 2 * t;
    double* v1 = V + ((size_t)(rb[two ? k + 1 : k] * nb) << 6) + 8 * g + 2 * t;
    double2 f0[2], f1[2];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      f0[c] = *reinterpret_cast<const double2*>(v0 + 64 * cb[c]);
      f1[c] = *reinterpret_cast<const double2*>(v1 + 64 * cb[c]);
    }
    double o0[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, o1[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
      for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int ni = 0; ni < 2; ++ni) {
          const double q = ni ? bq[c][r].y : bq[c][r].x;
          dmma(o0[ni], r ? f0[c].y : f0[c].x, q);
          dmma(o1[ni], r ? f1[c].y : f1[c].x, q);
        }
#pragma unroll
    for (int ni = 0; ni < 2; ++ni) {
      *reinterpret_cast<double2*>(v0 + 64 * cb[ni]) = make_double2(o0[ni][0], o0[ni][1]);
      if (two) *reinterpret_cast<double2*>(v1 + 64 * cb[ni]) = make_double2(o1[ni][0], o1[ni][1]);
    }
  }
}

// ---------------------------------------------------------------------------------------------- the kernel
struct JacobiParams {
  const double* H;
  double* W;
  double* C;
  int* info;
  double* gwork;   // per-CTA global workspace: [A nb(nb+1)/2 blocks of 64] (modes 2,3) [V np*np, blocked] (modes 1,2,3) [Q 2*nslots*16*LDQ] (mode 3)
  size_t gstride;  // doubles per CTA
  const int* tab;  // schedule tables written by k_schedule: [m-1][nslots] slots, [m-1][nslots] feeds, [m-1][ntiles] tiles
  int* next;       // global counter of the next matrix to hand out (behind the tables; k_schedule sets it to the grid size)
  int n, batch, nb, np, m, nslots, max_sweeps;
  int nranges, row_lo[4], row_hi[4];  // rows of C that are wanted (nranges = 0: all); the others are returned as zeros
  int stream_v;    // workspace modes: 1 = V accesses carry the evict-first hint (see wpcd_jacobi_launch)
  int full_every;  // a full 16x16 pivot sweep every full_every-th step of the tournament, cross-only sweeps between
  double tol;
  // fallback launches (matrices whose log overflowed): the matrices are list[0 .. *nlist) instead of 0 .. batch-1
  const int* list;
  const int* nlist;
  // log mode (kMode 4, see k_jacobi): scheduler block, log regions (two per CTA) and their geometry
  int* sched;
  char* logbase;
  size_t region_bytes;
  int log_cap, log_steps;  // capacity of a region in entries (rotating slots) and in tournament steps
  int rbp, npanels;        // row blocks of C per replay unit, replay units per matrix
  int nsolvers;            // CTAs that own log regions and an A workspace (the others only replay)
  int ready_off, fb_off;   // offsets (ints) of the ready list and of the fallback list inside the scheduler block
};

// Scheduler block of the log mode (ints): [0] next matrix, [1] matrices published for replay, [2] replay units claimed,
// [3] replay units done, [4] matrices solved (published or sent to the fallback list), [5] length of the fallback list,
// [6] watchdog flag, [kSchedDone + r] replay units done of log region r; then the ready list (region of the k-th published
// matrix, -1 = not written yet) and the fallback list.
constexpr int kSchedDone = 16;
__global__ void k_sched_init(int* __restrict__ sched, int nzero, int nneg) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nzero + nneg; i += gridDim.x * blockDim.x) sched[i] = i < nzero ? 0 : -1;
}
__global__ void k_set_counter(int* p, int v) { *p = v; }
// the watchdog of the log mode fired (a wait that should never be that long): no result of the launch can be trusted
__global__ void k_log_watchdog(const int* __restrict__ sched, int* __restrict__ info, int batch) {
  if (sched[6] == 0) return;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < batch; i += gridDim.x * blockDim.x) info[i] = -2;
}


// Schedule tables (one copy per launch, read through the L1): the tournament needs integer divisions that would
// otherwise be redone for every work item.
//   slot[t][s]  = I | J << 16                 blocks of slot s at step t (0xFFFF = none)
//   feed[t][s]  = s1 | s2 << 16               slots (s1 < s2) of the PREVIOUS step whose tile feeds the pivot of slot s
//   tile[t][k]  = s1 | s2 << 12 | crit << 24  k-th tile of step t (s1 < s2); crit: it feeds a pivot of the next step
__global__ void k_schedule(int m, int nb, int* __restrict__ tab, int* __restrict__ next, int first) {
  const int nslots = m / 2, ntiles = nslots * (nslots - 1) / 2, t = blockIdx.x;
  if (t == 0 && threadIdx.x == 0) *next = first;
  const int tp = (t + m - 2) % (m - 1), tn = (t + 1) % (m - 1);
  int* slot = tab + t * nslots;
  int* feed = tab + (m - 1) * nslots + t * nslots;
  int* tile = tab + 2 * (m - 1) * nslots + t * ntiles;
  for (int s = threadIdx.x; s < nslots; s += blockDim.x) {
    int I, J;
    slot_blocks(m, nb, t, s, I, J);
    slot[s] = (I & 0xFFFF) | ((J & 0xFFFF) << 16);
    int f = 0;
    if (J >= 0) {
      int s1 = rr_slot_of(m, tp, I), s2 = rr_slot_of(m, tp, J);
      if (s1 > s2) { int x = s1; s1 = s2; s2 = x; }
      f = s1 | (s2 << 16);
    }
    feed[s] = f;
  }
  for (int k = threadIdx.x; k < ntiles; k += blockDim.x) {
    int s1 = 0, rem = k;  // unrank (s1 < s2)
    while (rem >= nslots - 1 - s1) { rem -= nslots - 1 - s1; ++s1; }
    const int s2 = s1 + 1 + rem;
    const int crit = critical_slot(m, nb, t, tn, s1, s2) >= 0 ? 1 : 0;
    tile[k] = s1 | (s2 << 12) | (crit << 24);
  }
}

__device__ __forceinline__ void decode_slot(int x, int& I, int& J) {
  I = x & 0xFFFF; J = (x >> 16) & 0xFFFF;
  if (I == 0xFFFF) I = -1;
  if (J == 0xFFFF) J = -1;
}


// One warp prepares slot sn of step tn: identity into its Q (buffer bn), and for a real pair the critical tile of the
// running step t (buffer bc) followed by the pivot solve.
template <int kMode>
__device__ __forceinline__ void prepare_slot(const Smem& sm, const JacobiParams& P, int tn, int sn, int bn, bool has_cur,
                                             int t, int bc, int parity, int lane, int widx) {
  const AView A{sm.A, P.nb};
  const int m = P.m, nslots = P.nslots;
  double* Qn = sm.Q + (size_t)(bn * nslots + sn) * kQSlot;
  int I, J;
  decode_slot(sm.tab[tn * nslots + sn], I, J);
  if (J < 0)  // no pivot: identity (a pivot solve writes its own Q)
    for (int e = lane; e < 256; e += 32) {
      const int sr = e >> 4, c = e & 15;
      Qn[qoff(sr, c)] = (qrow(c) == sr) ? 1.0 : 0.0;
    }
  bool rotated = false;
  if (J >= 0) {
    if (has_cur) {
      const int f = sm.tab[(m - 1) * nslots + tn * nslots + sn];
      const int s1 = f & 0xFFFF, s2 = f >> 16;
      if (sm.rot[bc * nslots + s1] | sm.rot[bc * nslots + s2]) {
        int I1, J1, I2, J2;
        decode_slot(sm.tab[t * nslots + s1], I1, J1);
        decode_slot(sm.tab[t * nslots + s2], I2, J2);
        const double* Qc = sm.Q + (size_t)bc * nslots * kQSlot;
        apply_tile(A, Qc + (size_t)s1 * kQSlot, Qc + (size_t)s2 * kQSlot, I1, J1, I2, J2, lane);
      }
    }
    __syncwarp();
    // full sweep of the pivot every full_every-th step (every block then sits in a pivot at >= 1 full step per sweep,
    // so every pair is still met in every sweep); always for small matrices, where padding leaves few real pivots
    // nb >= 5 with two full steps per sweep (wpcd_jacobi_launch): a block is idle (paired with the one padding player of
    // nb = 5, 7) at most once per sweep, so it sits in a full real pivot in at least one of them
    const bool full = (tn % P.full_every) == 0 || P.nb < 5;
    rotated = inner_solve(A, Qn, I, J, P.tol, full, lane);
    if (kMode == 4 && rotated) {  // log mode: the eigenvectors are accumulated later, by a replay of these products
      int idx = 0;
      if (lane == 0) idx = atomicAdd(&sm.ctr[4], 1);
      idx = __shfl_sync(0xffffffffu, idx, 0);
      __syncwarp();
      if (idx < sm.logcap) {
        double2* dst = reinterpret_cast<double2*>(sm.logq + (size_t)idx * kQSlot);
        const double2* src = reinterpret_cast<const double2*>(Qn);
#pragma unroll
        for (int u = 0; u < kQSlot / 64; ++u) __stcs(dst + lane + 32 * u, src[lane + 32 * u]);  // streaming: A stays in L2
        if (lane == 0) {
          sm.logtag[idx] = (I & 0xFFFF) | ((J & 0xFFFF) << 16);
          // per-block sequence numbers for the replay's dataflow order (sm.act doubles as the counters in the log mode;
          // a block sits in one slot per step and the steps are barrier-separated: no race)
          sm.logtag[sm.logcap + idx] = (sm.act[I] & 0xFFFF) | ((sm.act[J] & 0xFFFF) << 16);
          ++sm.act[I]; ++sm.act[J];
        }
      } else if (lane == 0) {
        sm.ctr[5] = 1;
      }
    }
  }
  if (lane == 0) {
    sm.rot[bn * nslots + sn] = rotated ? 1 : 0;
    if (rotated) atomicAdd(&sm.ctr[2 + parity], 1);
  }
}

// ---------------------------------------------------------------------------------------------- log mode
// Layout of a log region (ints, then the products): [0] entries, [1] steps, [2] overflow, [3] matrix, [8 ..) perm[np],
// src[np], step_start[log_steps + 2], tags[log_cap] (I | J << 16), seq[log_cap] (how many earlier entries touched block I |
// the same for J << 16); the products [log_cap][256] doubles follow, 256-byte aligned.
__host__ __device__ inline int log_perm_off() { return 8; }
__host__ __device__ inline int log_src_off(int np) { return 8 + np; }
__host__ __device__ inline int log_step_off(int np) { return 8 + 2 * np; }
__host__ __device__ inline int log_tag_off(int np, int steps) { return 8 + 2 * np + steps + 2; }
__host__ __device__ inline size_t log_q_off(int np, int steps, int cap) {
  return (((size_t)(log_tag_off(np, steps) + 2 * cap) * 4) + 255) & ~(size_t)255;   // tags[cap], then seq[cap]
}
constexpr int kJobWait = 0, kJobSolve = 1, kJobReplay = 2, kJobExit = 3;

// Replay unit: rows [8 rbp panel, 8 rbp (panel + 1)) (internal order) of the eigenvector matrix of the matrix logged in
// `region`.  The panel starts as rows of the identity in shared memory (blocked like V: vidx with local row blocks), takes
// V <- V Q for every logged product in order -- the products of one tournament step touch disjoint column blocks, so the
// warps share them out and meet at one barrier per step -- and is written to its rows of C.  Same arithmetic, in the
// same order, as the V items of the workspace modes (apply_V_item), but V never leaves the SM and the products are read
// once per panel from L2: the DRAM traffic of the large-n path drops from ~200x to ~10x the algorithmic bytes.
template <int kThreads>
__device__ __forceinline__ void replay_panel(const JacobiParams& P, int region, int panel, double* Vp) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = P.n, np = P.np, nb = P.nb;
  const int* hdr = reinterpret_cast<const int*>(P.logbase + (size_t)region * P.region_bytes);
  const int* perm = hdr + log_perm_off();
  const int* src = hdr + log_src_off(np);
  const int* step_start = hdr + log_step_off(np);
  const int* tags = hdr + log_tag_off(np, P.log_steps);
  const double* logq = reinterpret_cast<const double*>(reinterpret_cast<const char*>(hdr) + log_q_off(np, P.log_steps, P.log_cap));
  const int nsteps = __ldcg(hdr + 1), mat = __ldcg(hdr + 3);
  const int rb0 = panel * P.rbp;
  const int nrbp = nb - rb0 < P.rbp ? nb - rb0 : P.rbp;
  int* srcs = reinterpret_cast<int*>(Vp + (size_t)P.rbp * nb * 64);  // [np] sort permutation, [rbp] local row blocks
  int* rbl = srcs + np;
  for (int e = tid; e < nrbp * nb * 64; e += kThreads) {
    const int blk = e >> 6, r = (e >> 3) & 7, c = e & 7;
    const int lr = blk / nb, cb = blk - lr * nb;
    Vp[e] = (8 * (rb0 + lr) + r == 8 * cb + c) ? 1.0 : 0.0;
  }
  for (int k = tid; k < n; k += kThreads) srcs[k] = __ldcg(src + k);
  if (tid < P.rbp) rbl[tid] = tid;
  __syncthreads();
  // Items = (log entry, pair of row blocks of the panel), in log order, dealt round-robin to the warps.  No barrier per
  // tournament step: an item may run as soon as the two column blocks of its entry have received all earlier products in
  // its rows -- dn[pr][block] counts them, the entry carries the counts it must see (seq).  Log order is a topological
  // order and every warp works through its items in that order, so the first unfinished item can always run.
  const int nper = (nrbp + 1) >> 1;  // items of two row blocks
  volatile int* dn = rbl + P.rbp;    // [nper][nb]
  const int* seqs = tags + P.log_cap;
  const int nent = __ldcg(hdr);
  for (int x = tid; x < nper * nb; x += kThreads) dn[x] = 0;
  __syncthreads();
  constexpr int kWarps = kThreads / 32;
  for (int itm = warp; itm < nent * nper; itm += kWarps) {
    const int e = itm / nper, pr = itm - e * nper;
    const int tag = __ldcg(tags + e), sq = __ldcg(seqs + e);
    const int I = tag & 0xFFFF, J = tag >> 16;
    {  // this warp's next product on its way from DRAM to L2 meanwhile
      const int en = (itm + kWarps) / nper;
      if (en < nent && lane < kQSlot * 8 / 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(logq + (size_t)en * kQSlot) + lane * 128));
    }
    double2 bq[2][2];
    load_bq_cg(logq + (size_t)e * kQSlot, lane, bq);  // in flight while the warp waits for its turn
    if (lane == 0) {
      volatile int* d = dn + pr * nb;
      int spins = 0;
      while ((d[I] != (sq & 0xFFFF) || d[J] != (sq >> 16)) && ++spins < (1 << 26)) __nanosleep(32);
    }
    __syncwarp();
    const int nrb = nrbp - 2 * pr < 2 ? nrbp - 2 * pr : 2;
    apply_V_bq(Vp, nb, bq, I, J, rbl + 2 * pr, nrb, lane);
    __threadfence_block();
    __syncwarp();
    if (lane == 0) { dn[pr * nb + I] = (sq & 0xFFFF) + 1; dn[pr * nb + J] = (sq >> 16) + 1; }
  }
  __syncthreads();
  double* Co = P.C + (size_t)mat * n * n;
  for (int lr = 0; lr < 8 * nrbp; ++lr) {
    const int i = 8 * rb0 + lr;
    if (i >= n) break;
    const int pi = __ldcg(perm + i);
    double* row = Co + (size_t)(pi & 0xFFFF) * n;
    const double* vrow = Vp + ((size_t)((lr >> 3) * nb) << 6) + ((lr & 7) << 3);
    for (int k = tid; k < n; k += kThreads) {
      const int c = srcs[k];
      row[k] = (pi >> 16) ? vrow[((size_t)(c >> 3) << 6) + (c & 7)] : 0.0;
    }
  }
}

// kMode 1: A (upper blocks only) and Q in shared memory, V in the global workspace (n <= 200)
//       2: A (upper blocks only, same layout as in mode 1) and V in the global workspace, Q in shared memory
//          (measured against the full mirrored array this path started with: 25 % less traffic per step, n = 300
//          522 -> 429 ms, n = 800 11.7 -> 9.5 s per 4096 matrices)
//       3: as 2 with Q in the global workspace too (very large n)
// The pivot scratch is always the slot's own Q array.
// kThr: 640 threads (one CTA per SM; 20 warps at 96 registers measured faster than 16 at 128 or 24 at 80), or 320 /
// 160 / 128 (two / four / five CTAs per SM; 128 for n <= 64: 1.45 -> 1.31 ms at n=32, 2.52 -> 2.20 at n=48, 3.28 -> 3.09
// at n=64 per 4096 matrices) where shared memory allows and a step has no more pivots than the CTA has warps:
// several matrices in flight per SM fill each other's pivot-chain bubbles.
template <int kMode, int kThr>
__global__ void __launch_bounds__(kThr, kThr == 128 ? 5 : 640 / kThr) k_jacobi(JacobiParams P) {
  constexpr int kThreads = kThr, kPivotWarps = kThr / 32;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = P.n, np = P.np, nslots = P.nslots, m = P.m, nb = P.nb;
  Smem sm;
  {
    double* d = reinterpret_cast<double*>(smem_raw);
    double* g = P.gwork + (size_t)blockIdx.x * P.gstride;
    if (kMode == 1) {
      sm.A = d; d += (size_t)(nb * (nb + 1) / 2) * 64;
      sm.V = g; g += (size_t)np * np;
    } else if (kMode == 4) {
      sm.A = g; g += (size_t)(nb * (nb + 1) / 2) * 64;
      sm.V = nullptr;
    } else {
      sm.A = g; g += (size_t)(nb * (nb + 1) / 2) * 64;
      sm.V = g; g += (size_t)np * np;
    }
    if (kMode == 3) sm.Q = g;
    else { sm.Q = d; d += (size_t)2 * nslots * kQSlot; }
    sm.wsort = d; d += np;
    int* ip = reinterpret_cast<int*>(d);
    sm.rot = ip; ip += 2 * nslots;
    sm.src = ip; ip += np;
    sm.ctr = ip; ip += 8;
    sm.act = ip; ip += 2 * nb;  // list of active row blocks, then a flag per row block
    sm.perm = ip; ip += np;
    if (kMode == 1) {  // small tables: keep the slot and feed tables of all steps in shared memory
      for (int e = tid; e < 2 * (m - 1) * nslots; e += kThreads) ip[e] = P.tab[e];
      sm.tab = ip;
    } else {
      sm.tab = P.tab;
    }
  }
  __syncthreads();
  // (Keeping the pivot solves on the warps of two SM sub-partitions and the update queue on the other two was measured
  // slower: the pivots then contend with each other for issue slots and the fp64 pipe.)
  const int widx = warp;  // every warp first solves pivots (slot widx, widx + kPivotWarps, ...), then joins the queue
  const AView Av{sm.A, nb};
  const int ntiles = nslots * (nslots - 1) / 2;
  constexpr int kVRowBlocksPerItem = 4;

  // matrices are handed out dynamically (they need 6-8 sweeps each): the first one is the CTA's own index, the next ones
  // come from a global counter that k_schedule set to gridDim.x
  __shared__ int s_next;
  __shared__ int s_job[4];
  constexpr bool kList = kMode == 2 || kMode == 3;  // only the workspace modes serve as the fallback launch of the log mode
  // log mode, used by thread 0 only: [0], [1] own log regions that wait for their replay, [2] consecutive waits
  __shared__ int s_state[4];
  if (kMode == 4 && tid == 0) { s_state[0] = 0; s_state[1] = 0; s_state[2] = 0; }
  for (int it = blockIdx.x;;) {
    int mat, region = 0;
    if (kMode == 4) {
      // Log mode: one persistent loop over three kinds of work, decided by thread 0.  (a) A replay unit (a panel of rows
      // of the eigenvector matrix of a solved matrix, see replay_panel) if one is published and unclaimed -- first, so
      // that the log regions drain; (b) else the next matrix, if one of this CTA's two log regions is free; (c) else wait.
      __syncthreads();
      if (tid == 0) {
        volatile int* sc = P.sched;
        int kind = kJobWait, a = 0, b = 0;
        int c = sc[2];
        for (;;) {
          const int pub = sc[1];
          if (c >= pub * P.npanels) break;
          const int old = atomicCAS(P.sched + 2, c, c + 1);
          if (old == c) { kind = kJobReplay; a = c / P.npanels; b = c - a * P.npanels; break; }
          c = old;
        }
        if (kind == kJobReplay) {  // the publisher's ticket may precede its list entry by a few cycles
          volatile int* rl = P.sched + P.ready_off;
          int spins = 0, r;
          while ((r = rl[a]) < 0 && ++spins < (1 << 24)) __nanosleep(64);
          if (r < 0) { P.sched[6] = 1; kind = kJobExit; }
          a = r;
        } else {
          int* done = P.sched + kSchedDone + 2 * blockIdx.x;
          if (s_state[0] && sc[kSchedDone + 2 * blockIdx.x] >= P.npanels) { done[0] = 0; s_state[0] = 0; }
          if (s_state[1] && sc[kSchedDone + 2 * blockIdx.x + 1] >= P.npanels) { done[1] = 0; s_state[1] = 0; }
          if ((int)blockIdx.x < P.nsolvers && !(s_state[0] && s_state[1]) && sc[0] < P.batch) {
            const int mnew = atomicAdd(P.sched, 1);
            if (mnew < P.batch) {
              kind = kJobSolve; a = mnew; b = s_state[0] ? 1 : 0;
              s_state[b] = 1;
            }
          }
          if (kind == kJobWait && sc[0] >= P.batch && sc[4] >= P.batch) {
            __threadfence();
            if (sc[3] >= sc[1] * P.npanels) kind = kJobExit;
          }
          if (kind == kJobWait && ++s_state[2] > (1 << 23)) { P.sched[6] = 1; kind = kJobExit; }  // watchdog: never hang the GPU
        }
        if (kind != kJobWait) s_state[2] = 0;
        s_job[0] = kind; s_job[1] = a; s_job[2] = b;
      }
      __syncthreads();
      const int kind = s_job[0];
      if (kind == kJobExit) break;
      if (kind == kJobWait) { __nanosleep(256); continue; }
      if (kind == kJobReplay) {
        replay_panel<kThreads>(P, s_job[1], s_job[2], reinterpret_cast<double*>(smem_raw));
        __syncthreads();
        if (tid == 0) {  // all reads of the region and all writes of C are done
          __threadfence();
          atomicAdd(P.sched + kSchedDone + s_job[1], 1);
          atomicAdd(P.sched + 3, 1);
        }
        continue;
      }
      mat = s_job[1];
      region = 2 * blockIdx.x + s_job[2];
    } else {
      if (it >= ((kList && P.nlist) ? *P.nlist : P.batch)) break;
      mat = (kList && P.list) ? P.list[it] : it;
    }
    int* const lhdr = kMode == 4 ? reinterpret_cast<int*>(P.logbase + (size_t)region * P.region_bytes) : nullptr;
    if (kMode == 4) {
      sm.logtag = lhdr + log_tag_off(np, P.log_steps);
      sm.logq = reinterpret_cast<double*>(reinterpret_cast<char*>(lhdr) + log_q_off(np, P.log_steps, P.log_cap));
      sm.logcap = P.log_cap;
    }
    const double* H = P.H + (size_t)mat * n * n;
    __syncthreads();
#ifdef WPCD_PROFILE
    const long long tm0 = clock64();
#endif
    // Ordering (de Rijk): the rows/columns are taken in the order of DESCENDING diagonal entries.  On these graded
    // Hamiltonians (kinetic energies from 1e-3 to 1e5 MeV along the diagonal) the cyclic sweeps then converge in one to
    // two sweeps fewer than in the natural ascending order (oracle: 7 -> 5-6 sweeps at N = 100).  Pure relabelling:
    // internal index i <-> original index perm[i]; eigenvalues are sorted at the end anyway, rows of C are written back
    // to their original places.
    for (int k = tid; k < n; k += kThreads) sm.wsort[k] = H[(size_t)k * n + k];
    __syncthreads();
    for (int k = tid; k < np; k += kThreads) {
      if (k < n) {
        const double dk = sm.wsort[k];
        int rank = 0;
        for (int j = 0; j < n; ++j) {
          const double dj = sm.wsort[j];
          rank += (dj > dk) || (dj == dk && j < k);
        }
        bool want = P.nranges == 0;
        for (int r = 0; r < P.nranges; ++r) want |= (k >= P.row_lo[r]) && (k < P.row_hi[r]);
        sm.perm[rank] = k | (want ? 0x10000 : 0);
      } else {
        sm.perm[k] = k;  // padding stays behind the matrix, never wanted
      }
    }
    __syncthreads();
    if (tid == 0) {  // row blocks of V that hold wanted rows of C (all of them unless row ranges were given)
      int na = 0;
      for (int rb = 0; rb < nb; ++rb) {
        int want = 0;
        for (int i = 0; i < 8; ++i) want |= sm.perm[8 * rb + i] >> 16;
        if (want) sm.act[na++] = rb;
        sm.act[nb + rb] = want;
      }
      sm.ctr[0] = na;
    }
    __syncthreads();
    const int nact = sm.ctr[0];
    const int nvgrp = (nact + kVRowBlocksPerItem - 1) / kVRowBlocksPerItem;
    const int nitems = kMode == 4 ? ntiles : ntiles + nslots * nvgrp;  // log mode: no eigenvector items
    const float rnvgrp = 1.0f / (float)(nvgrp > 0 ? nvgrp : 1);
    if (kMode == 4)  // the list of active row blocks is not used in the log mode: its place holds the per-block entry counters
      for (int rb = tid; rb < nb; rb += kThreads) sm.act[rb] = 0;
    __syncthreads();
    for (int e = tid; e < np * np; e += kThreads) {
      int r = e / np, c = e - r * np;
      double a = (r < n && c < n) ? H[(size_t)(sm.perm[r] & 0xFFFF) * n + (sm.perm[c] & 0xFFFF)] : 0.0;
      Av.put(r, c, a);
      if (kMode != 4) sm.V[vidx(nb, r, c)] = (r == c) ? 1.0 : 0.0;
    }
    if (tid < 8) sm.ctr[tid] = 0;
    __syncthreads();
#ifdef WPCD_PROFILE
    if (blockIdx.x == 0 && tid == 0) WPCD_PROF_ADD(6, clock64() - tm0);
#endif
    // prologue: pivots of (sweep 0, step 0) into Q buffer 0
    if (widx >= 0)
      for (int sn = widx; sn < nslots; sn += kPivotWarps) prepare_slot<kMode>(sm, P, 0, sn, 0, false, 0, 0, 0, lane, widx);
    __syncthreads();
    int sweeps = 0, buf = 0, gstep = 0;
    bool converged = false;
    // log mode: entries [step_start[k], step_start[k+1]) are the products applied at global step k; nprep steps prepared
    int nprep = 1;
    if (kMode == 4 && tid == 0) { lhdr[log_step_off(np)] = 0; lhdr[log_step_off(np) + 1] = sm.ctr[4]; }
    for (;;) {
      const int par = sweeps & 1;
      for (int step = 0; step < m - 1; ++step, ++gstep) {
        const bool last = (step == m - 2);
        if (last && sm.ctr[2 + par] == 0) { converged = true; break; }  // nothing rotated in this sweep
        const bool do_next = !(last && sweeps + 1 >= P.max_sweeps);
        const int tn = last ? 0 : step + 1;
        const int parn = last ? (par ^ 1) : par;
        if (tid == 0) {
          sm.ctr[(gstep + 1) & 1] = 0;
          if (step == 0) sm.ctr[2 + (par ^ 1)] = 0;
        }
#ifdef WPCD_PROFILE
        long long tk0 = clock64();
#endif
        // pivots of the next step (critical tile first), overlapped with the rest of this step's updates
        if (do_next && widx >= 0)
          for (int sn = widx; sn < nslots; sn += kPivotWarps) prepare_slot<kMode>(sm, P, tn, sn, buf ^ 1, true, step, buf, parn, lane, widx);
#ifdef WPCD_PROFILE
        if (blockIdx.x == 0 && tid == 32) WPCD_PROF_ADD(1, clock64() - tk0);
        long long tk1 = clock64();
#endif
        const int* rot = sm.rot + buf * nslots;
        const double* Qc = sm.Q + (size_t)buf * nslots * kQSlot;
        int* queue = sm.ctr + (gstep & 1);
        const int* tab_slot = sm.tab + step * nslots;
        const int* tab_tile = P.tab + 2 * (m - 1) * nslots + step * ntiles;
        for (;;) {
          int it = 0;
          if (lane == 0) it = atomicAdd(queue, 1);
          it = __shfl_sync(0xffffffffu, it, 0);
          if (it >= nitems) break;
          {  // interleave the (L2/DRAM-latency bound) V items with the tiles (all modes: n=300 6 % faster than tiles first)
            const int nv = nitems - ntiles, nmix = 2 * (ntiles < nv ? ntiles : nv);
            if (it < nmix) it = (it & 1) ? ntiles + (it >> 1) : (it >> 1);
            else if (nv < ntiles) it -= nv;  // the remaining tiles (remaining V items keep their index)
          }
          if (it < ntiles) {
            const int e = __ldg(tab_tile + it);
            const int s1 = e & 0xFFF, s2 = (e >> 12) & 0xFFF;
            if (!(rot[s1] | rot[s2])) continue;
            if (do_next && (e >> 24)) continue;  // feeds a pivot of the next step: done by that pivot's warp
            int I1, J1, I2, J2;
            decode_slot(tab_slot[s1], I1, J1);
            decode_slot(tab_slot[s2], I2, J2);
            if (I1 < 0 || I2 < 0) continue;
            apply_tile(Av, Qc + (size_t)s1 * kQSlot, Qc + (size_t)s2 * kQSlot, I1, J1, I2, J2, lane);
          } else {
            const int v = it - ntiles;
            const int s = (int)(((float)v + 0.5f) * rnvgrp), grp = v - s * nvgrp;
            if (!rot[s]) continue;
            int I, J;
            decode_slot(tab_slot[s], I, J);
            const int r0 = kVRowBlocksPerItem * grp;
            const int nrb = nact - r0 < kVRowBlocksPerItem ? nact - r0 : kVRowBlocksPerItem;
            if (J >= 0) apply_V_item<2>(sm.V, nb, Qc + (size_t)s * kQSlot, I, J, sm.act + r0, nrb, lane, kMode != 1 && P.stream_v);
            else apply_V_item<1>(sm.V, nb, Qc + (size_t)s * kQSlot, I, J, sm.act + r0, nrb, lane, kMode != 1 && P.stream_v);
          }
        }
#ifdef WPCD_PROFILE
        if (blockIdx.x == 0 && tid == 480) WPCD_PROF_ADD(3, clock64() - tk1);
        if (blockIdx.x == 0 && tid == 32) WPCD_PROF_ADD(4, clock64() - tk1);
#endif
        __syncthreads();
#ifdef WPCD_PROFILE
        if (blockIdx.x == 0 && tid == 0) { WPCD_PROF_ADD(0, clock64() - tk0); WPCD_PROF_ADD(2, 1); }
#endif
        if (kMode == 4 && do_next) {
          nprep = gstep + 2;
          if (tid == 0) {
            if (nprep <= P.log_steps) lhdr[log_step_off(np) + nprep] = sm.ctr[4];
            else sm.ctr[5] = 1;
          }
        }
        buf ^= 1;
      }
      ++sweeps;
      if (converged || sweeps >= P.max_sweeps) break;
    }
    // eigenvalues = diagonal; rank sort ascending (ties by index); gather columns
    __syncthreads();
#ifdef WPCD_PROFILE
    const long long tm1 = clock64();
#endif
    for (int k = tid; k < n; k += kThreads) sm.wsort[k] = Av.get(k, k);
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
    if (kMode != 4) {
      for (int e = tid; e < n * n; e += kThreads) {  // internal row i goes back to row perm[i]; unwanted rows: zeros
        int i = e / n, k = e - i * n;
        int c = sm.src[k];
        const int pi = sm.perm[i];
        Co[(size_t)(pi & 0xFFFF) * n + k] = (pi >> 16) ? sm.V[vidx(nb, i, c)] : 0.0;
      }
      if (tid == 0) {
        P.info[mat] = converged ? sweeps : -1;
        s_next = atomicAdd(P.next, 1);
      }
    } else {
      // log mode: what the replay needs besides the products -- the ordering, the sort, the step table -- then publish
      for (int k = tid; k < np; k += kThreads) {
        lhdr[log_perm_off() + k] = sm.perm[k];
        lhdr[log_src_off(np) + k] = k < n ? sm.src[k] : 0;
      }
      __threadfence();  // every thread's log and header writes, before thread 0 publishes the region
      __syncthreads();
      if (tid == 0) {
        const bool ovf = sm.ctr[5] != 0 || sm.ctr[4] > P.log_cap;
        P.info[mat] = converged ? sweeps : -1;
        lhdr[0] = sm.ctr[4]; lhdr[1] = nprep; lhdr[2] = ovf ? 1 : 0; lhdr[3] = mat;
        __threadfence();
        if (!ovf) {
          const int ticket = atomicAdd(P.sched + 1, 1);
          P.sched[P.ready_off + ticket] = region;
        } else {  // too many rotations for the log region: the matrix is redone by the fallback launch (workspace mode)
          P.sched[P.fb_off + atomicAdd(P.sched + 5, 1)] = mat;
          s_state[region & 1] = 0;
        }
        __threadfence();
        atomicAdd(P.sched + 4, 1);
      }
    }
    __syncthreads();
#ifdef WPCD_PROFILE
    if (blockIdx.x == 0 && tid == 0) { WPCD_PROF_ADD(5, clock64() - tm0); WPCD_PROF_ADD(7, clock64() - tm1); }
#endif
    it = s_next;
  }
}

struct Geometry {
  size_t tab_bytes;  // schedule tables at the head of the workspace
  int nb, np, m, nslots;
  int mode;        // k_jacobi<mode, threads>
  int threads;
  size_t gstride;  // doubles of global workspace per CTA
  size_t smem;     // dynamic shared memory of the launch (bytes)
};

Geometry geometry(const WpcdHandle* h, int n) {
  Geometry g;
  g.nb = (n + 7) / 8;
  if (g.nb < 2) g.nb = 2;
  g.np = 8 * g.nb;
  g.m = (g.nb & 1) ? g.nb + 1 : g.nb;
  if (g.m < 6) g.m = 6;  // the pipeline needs >= 3 slots (distinct critical tiles)
  g.nslots = g.m / 2;
  g.tab_bytes = ((((size_t)(g.m - 1) * (2 * g.nslots + g.nslots * (g.nslots - 1) / 2) * 4) + 255) & ~(size_t)255) + 256;  // + counter
  const size_t misc = (size_t)g.np * 8 + (size_t)(2 * g.nslots + 2 * g.np + 8 + 2 * g.nb) * 4 + 64;
  const size_t tabs = (size_t)2 * (g.m - 1) * g.nslots * 4;  // shared-memory copy of the slot and feed tables (modes 0, 1)
  const size_t q = (size_t)2 * g.nslots * kQSlot * 8;
  const size_t a_half = (size_t)(g.nb * (g.nb + 1) / 2) * 512, v = (size_t)g.np * g.np * 8;
  const size_t cap = (size_t)h->max_smem_optin;
  g.threads = 640;
  const size_t smem1 = misc + tabs + q + a_half;
  if (g.nslots <= 4 && 5 * (smem1 + 1024) <= cap) { g.mode = 1; g.threads = 128; g.smem = smem1; g.gstride = v / 8; }
  else if (g.nslots <= 5 && 4 * (smem1 + 1024) <= cap) { g.mode = 1; g.threads = 160; g.smem = smem1; g.gstride = v / 8; }
  else if (g.nslots <= 10 && 2 * (smem1 + 1024) <= cap) { g.mode = 1; g.threads = 320; g.smem = smem1; g.gstride = v / 8; }
  else if (misc + tabs + q + a_half <= cap) { g.mode = 1; g.smem = misc + tabs + q + a_half; g.gstride = v / 8; }
  else if (misc + q <= cap) { g.mode = 2; g.smem = misc + q; g.gstride = (a_half + v) / 8; }
  else { g.mode = 3; g.smem = misc; g.gstride = (a_half + v + q) / 8; }
  return g;
}

// CTAs of the workspace paths: as many as fit an SM (640 / threads: 96 registers per thread), each with its own
// workspace.  All workspaces together must stay inside L2 (measured: a 100 MB working set already spills to HBM -- the
// 126 MB L2 is split over two dies); the mode-1 sets are 25-50 MB.
int global_grid(const WpcdHandle* h, const Geometry& g, int batch) {
  const int grid = (g.threads == 128 ? 5 : 640 / g.threads) * h->num_sms;
  return batch < grid ? batch : grid;
}

template <int kMode, int kThr>
int launch_mode(WpcdHandle* h, const JacobiParams& P, int grid, size_t smem, cudaStream_t st) {
  int rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_jacobi<kMode, kThr>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "jacobi attr");
  if (rc) return rc;
  k_jacobi<kMode, kThr><<<grid, kThr, smem, st>>>(P);
  return WPCD_OK;
}

// Log mode (k_jacobi<4>): used where the workspace mode 2 would run (A does not fit shared memory, Q does: 200 < n <= 848).
// Capacity of a log region: kLogSweeps sweeps' worth of rotating slots (measured need: 5-6; more goes to the fallback
// launch) and 16 sweeps' worth of steps.  WPCD_JACOBI_LOG_SWEEPS in the environment overrides kLogSweeps (a test hook:
// 0 disables the log mode, 1 forces matrices into the fallback launch).
constexpr int kLogSweeps = 7;
struct LogGeometry {
  bool use;
  int grid, nsolvers, cap, steps, rbp, npanels, ready_off, fb_off;
  size_t region_bytes, smem, sched_bytes, a_bytes, off_sched, off_a, off_log, off_fb, total;
};

LogGeometry log_geometry(const WpcdHandle* h, const Geometry& g, int batch) {
  LogGeometry L{};
  int sweeps = kLogSweeps;
  if (const char* e = getenv("WPCD_JACOBI_LOG_SWEEPS")) sweeps = atoi(e);
  const size_t cap_smem = (size_t)h->max_smem_optin;
  const size_t per_rb = (size_t)g.nb * 512;
  size_t avail = cap_smem > 2048 + 4 * (size_t)(g.np + 4 * g.nb) ? cap_smem - 2048 - 4 * (size_t)(g.np + 4 * g.nb) : 0;
  int rbp = (int)(avail / per_rb);
  if (rbp > 8) rbp = 8;
  if (rbp > 2) rbp &= ~1;
  L.use = g.mode == 2 && sweeps > 0 && rbp >= 1;
  if (!L.use) return L;
  L.grid = h->num_sms;  // small batches: the CTAs beyond the batch take replay units only
  L.nsolvers = batch < h->num_sms ? batch : h->num_sms;
  L.cap = sweeps * (g.m - 1) * g.nslots;
  L.steps = 16 * (g.m - 1);
  L.rbp = rbp;
  L.npanels = (g.nb + rbp - 1) / rbp;
  L.region_bytes = (log_q_off(g.np, L.steps, L.cap) + (size_t)L.cap * kQSlot * 8 + 255) & ~(size_t)255;
  const size_t smem_b = (size_t)rbp * per_rb + 4 * (size_t)(g.np + 8 + 4 * g.nb);
  L.smem = g.smem > smem_b ? g.smem : smem_b;
  L.ready_off = kSchedDone + 2 * L.nsolvers;
  L.fb_off = L.ready_off + batch;
  L.sched_bytes = (((size_t)(L.fb_off + batch) * 4) + 255) & ~(size_t)255;
  L.a_bytes = (size_t)(g.nb * (g.nb + 1) / 2) * 512;
  L.off_sched = g.tab_bytes;
  L.off_a = L.off_sched + L.sched_bytes;
  L.off_log = L.off_a + (size_t)L.nsolvers * L.a_bytes;
  L.off_fb = L.off_log + (size_t)2 * L.nsolvers * L.region_bytes;
  L.total = L.off_fb + 256 + (size_t)L.nsolvers * g.gstride * 8;  // fallback: its own counter and mode-2 workspaces
  return L;
}

}  // namespace

size_t wpcd_jacobi_workspace(const WpcdHandle* h, int n, int batch) {
  if (n <= WPCD_SMALL_N_MAX) return wpcd_jacobi_small_workspace();
  Geometry g = geometry(h, n);
  const LogGeometry L = log_geometry(h, g, batch);
  if (L.use) return L.total;
  return g.tab_bytes + (size_t)global_grid(h, g, batch) * g.gstride * 8;
}

int wpcd_jacobi_launch(WpcdHandle* h, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                       double tol, int max_sweeps, const int* h_rows, int n_ranges, void* d_work, size_t work_bytes,
                       cudaStream_t st) {
  // the paper's own size regime: element-wise parallel Jacobi, one small CTA per matrix (jacobi_small.cu)
  if (n <= WPCD_SMALL_N_MAX)
    return wpcd_jacobi_small_launch(h, n, batch, d_A, d_W, d_C, d_info, tol, max_sweeps, h_rows, n_ranges, d_work, work_bytes, st);
  Geometry g = geometry(h, n);
  if (g.smem > (size_t)h->max_smem_optin) return WPCD_ESIZE;
  JacobiParams P;
  P.H = d_A; P.W = d_W; P.C = d_C; P.info = d_info; P.gstride = g.gstride;
  P.tab = static_cast<const int*>(d_work);
  P.gwork = reinterpret_cast<double*>(static_cast<char*>(d_work) + g.tab_bytes);
  P.n = n; P.batch = batch; P.nb = g.nb; P.np = g.np; P.m = g.m; P.nslots = g.nslots;
  P.max_sweeps = max_sweeps;
  P.nranges = n_ranges;
  for (int r = 0; r < 4; ++r) { P.row_lo[r] = r < n_ranges ? h_rows[2 * r] : 0; P.row_hi[r] = r < n_ranges ? h_rows[2 * r + 1] : 0; }
  // full pivot sweeps per sweep of the tournament (measured: fewer cost extra sweeps, more cost pivot time): about three
  // on the shared-memory path (n = 75 .. 300: periods 5, 5, 7, 9, 13 are the measured optima), about four where A goes
  // through L2 (n = 400: 13 beats 17)
  if (g.mode == 1) P.full_every = (g.m - 1 + 2) / 3 > 5 ? (g.m - 1 + 2) / 3 : 5;
  else P.full_every = (g.m - 1 + 3) / 4 > 4 ? (g.m - 1 + 3) / 4 : 4;
  if (g.m == 6) P.full_every = 3;  // n = 33 .. 48 (5 steps per sweep, steps 0 and 3 full): n = 48: 7.06 -> 6.02 sweeps, 1.81 -> 1.72 ms;
                                   // n = 33 .. 40 had full pivots in every step: n = 40 1.65 -> 1.48 ms
  if (g.m == 8) P.full_every = 4;  // n = 49 .. 64 (7 steps): n = 56 2.73 -> 2.65 ms, n = 64 unchanged
  P.tol = tol > 0.0 ? tol : 2.220446049250313e-16;
  P.list = nullptr; P.nlist = nullptr; P.sched = nullptr; P.logbase = nullptr;
  P.region_bytes = 0; P.log_cap = P.log_steps = P.rbp = P.npanels = P.nsolvers = P.ready_off = P.fb_off = 0;
  const LogGeometry L = log_geometry(h, g, batch);
  if (L.use) {
    // Log mode: one persistent launch solves the matrices without their eigenvectors (A through L2, as in mode 2),
    // logs the rotation products and replays them panel by panel into C (k_jacobi<4>, replay_panel); a second launch
    // of the workspace mode redoes the matrices whose log overflowed (normally none: its CTAs exit at once).
    if (work_bytes < L.total) return WPCD_EWORK;
    char* w = static_cast<char*>(d_work);
    P.next = reinterpret_cast<int*>(w + g.tab_bytes - 256);
    k_schedule<<<g.m - 1, 128, 0, st>>>(g.m, g.nb, static_cast<int*>(d_work), P.next, L.grid);
    JacobiParams P4 = P;
    P4.sched = reinterpret_cast<int*>(w + L.off_sched);
    P4.gwork = reinterpret_cast<double*>(w + L.off_a);
    P4.gstride = L.a_bytes / 8;
    P4.logbase = w + L.off_log;
    P4.region_bytes = L.region_bytes;
    P4.log_cap = L.cap; P4.log_steps = L.steps; P4.rbp = L.rbp; P4.npanels = L.npanels; P4.nsolvers = L.nsolvers;
    P4.ready_off = L.ready_off; P4.fb_off = L.fb_off;
    P4.stream_v = 0;
    k_sched_init<<<64, 256, 0, st>>>(P4.sched, L.ready_off, 2 * batch);
    int rc = launch_mode<4, 640>(h, P4, L.grid, L.smem, st);
    if (rc) return rc;
    JacobiParams P2 = P;
    P2.list = P4.sched + L.fb_off;
    P2.nlist = P4.sched + 5;
    P2.next = reinterpret_cast<int*>(w + L.off_fb);
    P2.gwork = reinterpret_cast<double*>(w + L.off_fb + 256);
    P2.stream_v = (size_t)L.nsolvers * L.a_bytes <= ((size_t)96 << 20);
    k_set_counter<<<1, 1, 0, st>>>(P2.next, L.nsolvers);
    rc = launch_mode<2, 640>(h, P2, L.nsolvers, g.smem, st);
    if (rc) return rc;
    k_log_watchdog<<<8, 256, 0, st>>>(P4.sched, d_info, batch);
    return wpcd_check_cuda(h, cudaGetLastError(), "diag_batched launch (log mode)");
  }
  const int grid = global_grid(h, g, batch);
  // Workspace modes: while the A blocks of all CTAs together fit L2 (n <= ~390 with 148 CTAs) V is streamed through it
  // with the evict-first hint and A stays resident: a third less DRAM traffic (n=300: 320 -> 280 ms per 4096 matrices;
  // n=600, where A does not fit either, was 4 % slower with the hint).
  P.stream_v = (size_t)grid * (size_t)(g.nb * (g.nb + 1) / 2) * 512 <= ((size_t)96 << 20);
  if (work_bytes < g.tab_bytes + (size_t)grid * g.gstride * 8) return WPCD_EWORK;
  P.next = reinterpret_cast<int*>(static_cast<char*>(d_work) + g.tab_bytes - 256);
  k_schedule<<<g.m - 1, 128, 0, st>>>(g.m, g.nb, static_cast<int*>(d_work), P.next, grid);
  int rc;
  switch (g.mode) {
    case 1:
      rc = g.threads == 128   ? launch_mode<1, 128>(h, P, grid, g.smem, st)
           : g.threads == 160 ? launch_mode<1, 160>(h, P, grid, g.smem, st)
           : g.threads == 320 ? launch_mode<1, 320>(h, P, grid, g.smem, st)
                              : launch_mode<1, 640>(h, P, grid, g.smem, st);
      break;
    case 2: rc = launch_mode<2, 640>(h, P, grid, g.smem, st); break;
    default: rc = launch_mode<3, 640>(h, P, grid, g.smem, st); break;
  }
  if (rc) return rc;
  return wpcd_check_cuda(h, cudaGetLastError(), "diag_batched launch");
}

// ------------------------------------------------------------------------- wpcd_diag_batched_static (include/wpcd.h)
// The workspace of the launch above -- schedule tables, work counter, per-CTA eigenvector blocks -- in a file-scope
// device array, for callers that must not allocate.  Every device that loads the library holds the array until exit.
// In host code the NAME of the array is a host-side stand-in, not a device address: the address the kernels get is
// looked up with cudaGetSymbolAddress, once per device, with that device current (the entry point has checked that the
// current device is the handle's).  All calls on a device share the array: overlapping calls race (see the header).
static __device__ __align__(256) unsigned char wpcd_static_work[WPCD_STATIC_WORK_BYTES];

namespace {
constexpr int kMaxStaticDevices = 64;
std::mutex s_static_mutex;
void* s_static_ptr[kMaxStaticDevices];  // device address of wpcd_static_work per CUDA ordinal, nullptr = not looked up yet
}  // namespace

int wpcd_jacobi_static_launch(WpcdHandle* h, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                              double tol, int max_sweeps, const int* h_rows, int n_ranges, cudaStream_t st) {
  if (h->device < 0 || h->device >= kMaxStaticDevices) return WPCD_EINVAL;
  const size_t need = wpcd_jacobi_workspace(h, n, batch);
  if (need > (size_t)WPCD_STATIC_WORK_BYTES) {
    snprintf(h->cuda_err, sizeof(h->cuda_err),
             "wpcd_diag_batched_static: n = %d, batch = %d needs %zu bytes of workspace, the static array holds %zu "
             "(use wpcd_diag_batched with a caller-allocated workspace)",
             n, batch, need, (size_t)WPCD_STATIC_WORK_BYTES);
    return WPCD_ESIZE;
  }
  void* ptr = nullptr;
  {
    std::lock_guard<std::mutex> lock(s_static_mutex);
    ptr = s_static_ptr[h->device];
    if (!ptr) {
      if (int rc = wpcd_check_cuda(h, cudaGetSymbolAddress(&ptr, wpcd_static_work), "cudaGetSymbolAddress(wpcd_static_work)")) return rc;
      if (!ptr) return WPCD_ECUDA;
      s_static_ptr[h->device] = ptr;
    }
  }
  // nothing to clear: k_schedule / k_small_counter rewrite the tables and the counter, the CTAs initialise their V blocks
  return wpcd_jacobi_launch(h, n, batch, d_A, d_W, d_C, d_info, tol, max_sweeps, h_rows, n_ranges, ptr,
                            (size_t)WPCD_STATIC_WORK_BYTES, st);
}

// Test hooks (host only): the block tournament of jacobi_schedule.cuh, see include/wpcd.h.
extern "C" int wpcd_jacobi_schedule(int m, int nb, int t, int s, int* I, int* J) {
  if (m < 6 || (m & 1) || t < 0 || t >= m - 1 || s < 0 || s >= m / 2 || !I || !J) return WPCD_EINVAL;
  slot_blocks(m, nb, t, s, *I, *J);
  return WPCD_OK;
}
extern "C" int wpcd_jacobi_critical_slot(int m, int nb, int t, int tn, int s1, int s2) {
  if (m < 6 || (m & 1) || s1 < 0 || s2 <= s1 || s2 >= m / 2) return WPCD_EINVAL;
  return critical_slot(m, nb, t, tn, s1, s2);
}

#ifdef WPCD_PROFILE
extern "C" int wpcd_debug_read_prof(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, wpcd_prof, sizeof(long long) * 8);
}
extern "C" int wpcd_debug_clear_prof() {
  long long z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  return (int)cudaMemcpyToSymbol(wpcd_prof, z, sizeof(z));
}
#endif
