// jacobi_small.cu -- step (ii) of the WPCD recipe, H = C D C^T (Eq. 21), for the paper's own size regime
// n <= 64 (N_WP = 16 ... 96 in Table 1; "32 x 32 ... fit entirely on the GPU shared memory",
// PAPER.md:418): element-wise parallel two-sided Jacobi, one small CTA (n threads, rounded up to 16/32/48/64) per matrix
// and many CTAs per SM, instead of the block tournament of jacobi.cu whose 16x16 pivot chain leaves the fp64 pipe idle
// at these sizes (7 % of peak at n = 32, profiles/r1_size_sweep.md).
//
//   * Ordering: odd-even transposition with swaps (the parallel cyclic-order Jacobi the paper names, in the
//     form that needs no data movement): positions 0..NP-1 on a line; even rounds pair (0,1),(2,3),..., odd rounds
//     (1,2),(3,4),...; every rotation is followed by the exchange of its two positions, so that in NP rounds every pair
//     of indices has met exactly once (the line ends up reversed).  The pairing is STATIC: a thread keeps its row of the
//     eigenvector matrix in registers for the whole solve and never exchanges it.
//   * A (upper triangle, row stride NP+2) lives in shared memory and is updated in place, 2x2 block (pair a) x (pair b)
//     by 2x2 block: T' = R_a^T T R_b with R = [[s, c], [c, -s]] (rotation, then swap).  Every element is loaded and stored
//     once per round; the blocks are dealt to the threads along the super-diagonals of the block grid, which makes the
//     128-bit accesses of the even rounds bank-conflict free.  The diagonal blocks are the pivots: one thread per pair
//     computes (c, s) division-free (jacobi_rotation.cuh), sets the annihilated element to exactly 0 and publishes (c, s).
//   * V <- V R: thread i owns row i (NP doubles in registers); (c, s) of the NP/2 pairs come as broadcast loads.
//   * In odd rounds the two ends of the line idle; they are treated as one more "pair" (NP-1, 0) with c = 0, s = 1, i.e.
//     R = diag(1, -1): no exchange, the sign of one eigenvector flips (reading C13: signs are not unique).
//   * Converged when no pair passes the rotation test |a_pq| > tol sqrt(|a_pp a_qq|); from the fourth sweep on the test is
//     also run directly over the upper triangle after a sweep, which replaces the rotation-free verification sweep.
//     info = rotating sweeps + 1, as in jacobi.cu.
//   * Padding (n < NP) sits behind the matrix as zero rows and columns: never rotated, carried along by the swaps.
//   * The next matrix of a CTA is fetched into a staging buffer with a bulk asynchronous copy (cp.async.bulk, the TMA
//     engine) while the current one is being diagonalised; matrices are handed out by a global counter.
#include <cuda.h>
#include "jacobi_rotation.cuh"
#include "wpcd_internal.cuh"

namespace {

struct SmallParams {
  const double* H;
  double* W;
  double* C;
  int* info;
  int* next;  // global counter of the next matrix to hand out (set to the grid size before the launch)
  int n, batch, max_sweeps;
  int nranges, row_lo[4], row_hi[4];
  double tol;
};

__global__ void k_small_counter(int* next, int first) { *next = first; }

// ---- mbarrier + bulk copy (global -> shared), single CTA
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned phase) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(phase)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

template <int T>
__device__ __forceinline__ void cta_sync() {
  if (T <= 32) __syncwarp();
  else __syncthreads();
}
template <int T>
__device__ __forceinline__ bool cta_any(bool x) {
  if (T <= 32) return __any_sync(0xffffffffu, x);
  return __syncthreads_or(x) != 0;
}

// Deal of the off-diagonal blocks (a < b) of a round to the threads.  The first element of block (a, b) sits (16-byte
// units modulo 8, row stride NP + 2) at bank group (2a + b + const) mod 8 =: its class.  Thread tid only takes blocks of
// class tid & 7, so that the eight threads of a quarter warp (128-bit accesses of the even rounds) always hit eight
// different bank groups; in the odd rounds (64-bit accesses, 16 threads per wavefront) the upper eight threads of a half
// warp start with the block's second column, which moves them to the other eight 8-byte banks.  Within a class the
// blocks go round-robin to the T/8 threads of that class; slots needed: ceil(largest class / (T/8)).
__host__ __device__ constexpr int class_slots(int pairs, int threads) {
  int cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int a = 0; a < pairs; ++a)
    for (int b = a + 1; b < pairs; ++b) ++cnt[(2 * a + b) & 7];
  int mx = 0;
  for (int c = 0; c < 8; ++c) mx = cnt[c] > mx ? cnt[c] : mx;
  const int ranks = threads / 8;
  return (mx + ranks - 1) / ranks;
}

// blocks of thread tid: out[k] = first-element offset | a << 16 | b << 24, 0xFFFFFFFF = none; odd: pairs (2j+1, 2j+2)
template <int K>
__device__ __forceinline__ void deal_blocks(int pairs, int threads, int tid, int LD, int odd, unsigned (&out)[K]) {
  const int cls = tid & 7, rank = tid >> 3, ranks = threads >> 3;
#pragma unroll
  for (int k = 0; k < K; ++k) out[k] = 0xFFFFFFFFu;
  int i = 0;
  for (int a = 0; a < pairs; ++a)
    for (int b = a + 1; b < pairs; ++b) {
      if (((2 * a + b) & 7) != cls) continue;
      if (i % ranks == rank) {
        const int slot = i / ranks;
        const unsigned w = (unsigned)((2 * a + odd) * LD + 2 * b + odd) | (a << 16) | (b << 24);
#pragma unroll
        for (int k = 0; k < K; ++k)
          if (k == slot) out[k] = w;
      }
      ++i;
    }
}

// NP: padded size (16, 24, 32; 48 and 64 compile too but the block kernel of jacobi.cu is faster there); one thread per row.
template <int NP>
__global__ void __launch_bounds__(NP <= 32 ? 32 : 64, NP <= 16 ? 16 : (NP <= 32 ? 12 : 1)) k_jacobi_small(SmallParams prm) {
  constexpr int T = NP <= 32 ? 32 : 64;       // threads of the CTA (rows >= NP idle in the V phase, work in the A phase)
  constexpr int P = NP / 2;                   // pairs of an even round
  constexpr int LD = NP + 2;                  // row stride of A (doubles): rows are 16 bytes apart modulo 128
  // off-diagonal blocks: P (P - 1) / 2 in even rounds; odd rounds have P - 1 real pairs (the end pair is handled apart)
  constexpr int K0 = class_slots(P, T), K1 = class_slots(P - 1, T);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* A = reinterpret_cast<double*>(smem_raw);       // [NP][LD], upper triangle
  double* cs = A + NP * LD;                              // [P] (c, s)
  double* stage = cs + 2 * P;                            // [n*n] the next matrix (bulk copy target)
  double* wsort = stage + NP * NP;                       // [NP]
  int* real = reinterpret_cast<int*>(wsort + NP);        // [NP] position holds a real (not padding) index
  int* src = real + NP;                                  // [NP]
  int* flags = src + NP;                                 // [4]: rotations of this sweep, scan result, next matrix
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(flags + 4);
  const int tid = threadIdx.x, n = prm.n;
  const double tol2 = prm.tol * prm.tol;

  // static work lists: blocks of the even and odd rounds as byte offsets of the block's first element and of the two
  // (c, s) entries: off | a << 16 | b << 24
  unsigned blk0[K0], blk1[K1];
  deal_blocks<K0>(P, T, tid, LD, 0, blk0);
  deal_blocks<K1>(P - 1, T, tid, LD, 1, blk1);
  // odd rounds: the upper eight threads of every half warp work on the column-swapped block (see deal_blocks):
  // [x1 x0] R(c, s) = [y1 y0] with R(c, -s)
  const int swp = (tid >> 3) & 1;
  const double sgn = swp ? -1.0 : 1.0;

  // bulk copies need 16-byte sizes and addresses: n even; odd n (never a config size) reads H with plain loads
  const bool bulk = (n & 1) == 0;
  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  cta_sync<T>();
  unsigned phase = 0;
  int mat = blockIdx.x;
  if (bulk && mat < prm.batch && tid == 0) {
    mbar_expect_tx(bar, (unsigned)(n * n * 8));
    bulk_g2s(stage, prm.H + (size_t)mat * n * n, (unsigned)(n * n * 8), bar);
  }
  while (mat < prm.batch) {
    // ---- H (staged by the bulk copy) -> upper triangle of A; V = 1
    for (int e = tid; e < NP * LD; e += T) A[e] = 0.0;
    if (tid < NP) real[tid] = tid < n;
    if (bulk) {
      mbar_wait(bar, phase);
      phase ^= 1;
    }
    cta_sync<T>();
    {
      const double* Hs = bulk ? stage : prm.H + (size_t)mat * n * n;
      for (int e = tid; e < n * n; e += T) {
        const int r = e / n, c = e - r * n;
        if (r <= c) A[r * LD + c] = Hs[e];
      }
    }
    cta_sync<T>();
    // the next matrix of this CTA: taken now, copied in the background
    if (tid == 0) {
      const int nx = atomicAdd(prm.next, 1);
      flags[2] = nx;
      if (bulk && nx < prm.batch) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the generic-proxy reads of stage come first
        mbar_expect_tx(bar, (unsigned)(n * n * 8));
        bulk_g2s(stage, prm.H + (size_t)nx * n * n, (unsigned)(n * n * 8), bar);
      }
    }
    double v[NP];
#pragma unroll
    for (int k = 0; k < NP; ++k) v[k] = (k == tid) ? 1.0 : 0.0;

    int sweeps = 0;
    bool converged = false;
    while (sweeps < prm.max_sweeps) {
      bool rotated = false;
#pragma unroll 1
      for (int rr = 0; rr < NP; rr += 2) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          // ---------------------------------------------------------------- pivots: one thread per pair
          if (tid < P) {
            const int p = 2 * tid + e, q = (e && tid == P - 1) ? 0 : p + 1;
            if (e && tid == P - 1) {  // the two ends of the line idle: R = diag(1, -1)
              A[NP - 1] = -A[NP - 1];    // element (0, NP-1)
              *reinterpret_cast<double2*>(cs + 2 * tid) = make_double2(0.0, 1.0);
            } else {
              const double app = A[p * LD + p], apq = A[p * LD + q], aqq = A[q * LD + q];
              double c, s, t;
              const bool doit = rotation(app, aqq, apq, tol2, c, s, t);
              rotated |= doit;
              // rotated diagonal, then the exchange of the two positions
              A[p * LD + p] = aqq + t * apq;
              A[q * LD + q] = app - t * apq;
              if (doit) A[p * LD + q] = 0.0;
              *reinterpret_cast<double2*>(cs + 2 * tid) = make_double2(c, s);
              if (n < NP) {  // padding travels with the positions
                const int rp = real[p], rq = real[q];
                real[p] = rq; real[q] = rp;
              }
            }
          }
          cta_sync<T>();
          // ---------------------------------------------------------------- eigenvectors: V <- V R, row tid
          if (tid < NP) {
#pragma unroll
            for (int j = 0; j < P; ++j) {
              const double2 g = *reinterpret_cast<const double2*>(cs + 2 * j);
              const int i0 = 2 * j + e, i1 = (2 * j + 1 + e) % NP;
              const double x0 = v[i0], x1 = v[i1];
              v[i0] = g.y * x0 + g.x * x1;
              v[i1] = g.x * x0 - g.y * x1;
            }
          }
          // ---------------------------------------------------------------- A <- R^T A R, off-diagonal blocks
          if (e == 0) {
#pragma unroll
            for (int k = 0; k < K0; ++k) {
              const unsigned w = blk0[k];
              if (w != 0xFFFFFFFFu) {
                double* x = A + (w & 0xFFFFu);
                const double2 ga = *reinterpret_cast<const double2*>(cs + 2 * ((w >> 16) & 0xFFu));
                const double2 gb = *reinterpret_cast<const double2*>(cs + 2 * (w >> 24));
                const double2 r0 = *reinterpret_cast<const double2*>(x), r1 = *reinterpret_cast<const double2*>(x + LD);
                const double y00 = gb.y * r0.x + gb.x * r0.y, y01 = gb.x * r0.x - gb.y * r0.y;
                const double y10 = gb.y * r1.x + gb.x * r1.y, y11 = gb.x * r1.x - gb.y * r1.y;
                *reinterpret_cast<double2*>(x) = make_double2(ga.y * y00 + ga.x * y10, ga.y * y01 + ga.x * y11);
                *reinterpret_cast<double2*>(x + LD) = make_double2(ga.x * y00 - ga.y * y10, ga.x * y01 - ga.y * y11);
              }
            }
          } else {
#pragma unroll
            for (int k = 0; k < K1; ++k) {
              const unsigned w = blk1[k];
              if (w != 0xFFFFFFFFu) {
                double* x = A + (w & 0xFFFFu);
                const double2 ga = *reinterpret_cast<const double2*>(cs + 2 * ((w >> 16) & 0xFFu));
                const double2 gb = *reinterpret_cast<const double2*>(cs + 2 * (w >> 24));
                double* xa = x + swp;        // first-loaded column of the block (the second one for the swapped threads)
                double* xb = x + 1 - swp;
                const double sb = sgn * gb.y;
                const double x00 = xa[0], x01 = xb[0], x10 = xa[LD], x11 = xb[LD];
                const double y00 = sb * x00 + gb.x * x01, y01 = gb.x * x00 - sb * x01;
                const double y10 = sb * x10 + gb.x * x11, y11 = gb.x * x10 - sb * x11;
                xa[0] = ga.y * y00 + ga.x * y10; xb[0] = ga.y * y01 + ga.x * y11;
                xa[LD] = ga.x * y00 - ga.y * y10; xb[LD] = ga.x * y01 - ga.y * y11;
              }
            }
            // the idle ends: row 0 gets the column rotations, column NP-1 the row rotations of the P-1 real pairs; the
            // sign flip of position 0 (R = diag(1,-1) of the end pair) applies to row 0
            if (tid < P - 1) {
              const double2 g = *reinterpret_cast<const double2*>(cs + 2 * tid);
              double* x = A + 2 * tid + 1;                       // (0, 2j+1), (0, 2j+2)
              const double x0 = -x[0], x1 = -x[1];
              x[0] = g.y * x0 + g.x * x1; x[1] = g.x * x0 - g.y * x1;
              double* y = A + (2 * tid + 1) * LD + NP - 1;       // (2j+1, NP-1), (2j+2, NP-1)
              const double y0 = y[0], y1 = y[LD];
              y[0] = g.y * y0 + g.x * y1; y[LD] = g.x * y0 - g.y * y1;
            }
          }
          cta_sync<T>();
        }
      }
      ++sweeps;
      if (!cta_any<T>(rotated)) { converged = true; break; }
      if (sweeps >= 3) {
        // direct test of every pair on the upper triangle: if none would rotate, the next sweep is the verification sweep
        // of jacobi.cu with nothing to do -- count it and stop
        bool any = false;
        for (int ee = tid; ee < NP * NP; ee += T) {
          const int r = ee / NP, c = ee - r * NP;
          if (r < c) {
            const double x = A[r * LD + c];
            any |= x * x > tol2 * fabs(A[r * LD + r] * A[c * LD + c]);
          }
        }
        if (!cta_any<T>(any)) { ++sweeps; converged = true; break; }
      }
    }
    // ---- eigenvalues = diagonal at the real positions, ascending (ties by position); C = V with sorted columns
    cta_sync<T>();
    if (tid < NP) wsort[tid] = A[tid * LD + tid];
    cta_sync<T>();
    if (tid < NP && real[tid]) {
      const double wk = wsort[tid];
      int rank = 0;
      for (int j = 0; j < NP; ++j) {
        const double wj = wsort[j];
        rank += real[j] && ((wj < wk) || (wj == wk && j < tid));
      }
      src[rank] = tid;
    }
    cta_sync<T>();
    // stage V through shared memory (A is free now): row i at i*(NP+1)
    double* vs = A;
    if (tid < NP) {
      bool want = prm.nranges == 0;
      for (int r = 0; r < prm.nranges; ++r) want |= (tid >= prm.row_lo[r]) && (tid < prm.row_hi[r]);
#pragma unroll
      for (int k = 0; k < NP; ++k) vs[tid * (NP + 1) + k] = want ? v[k] : 0.0;
    }
    cta_sync<T>();
    double* Wo = prm.W + (size_t)mat * n;
    double* Co = prm.C + (size_t)mat * n * n;
    for (int k = tid; k < n; k += T) Wo[k] = wsort[src[k]];
    for (int e = tid; e < n * n; e += T) {
      const int i = e / n, k = e - i * n;
      Co[e] = vs[i * (NP + 1) + src[k]];
    }
    if (tid == 0) prm.info[mat] = converged ? sweeps : -1;
    cta_sync<T>();
    mat = flags[2];
    cta_sync<T>();
  }
}

template <int NP>
size_t small_smem() {
  return (size_t)(NP * (NP + 2) + NP + NP * NP + NP) * 8 + (size_t)(2 * NP + 4) * 4 + 16;
}

template <int NP>
int launch_small(WpcdHandle* h, const SmallParams& prm, int ctas_per_sm, cudaStream_t st) {
  const size_t smem = small_smem<NP>();
  int rc = wpcd_check_cuda(h, cudaFuncSetAttribute(k_jacobi_small<NP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "jacobi_small attr");
  if (rc) return rc;
  int grid = ctas_per_sm * h->num_sms;
  if (grid > prm.batch) grid = prm.batch;
  k_small_counter<<<1, 1, 0, st>>>(prm.next, grid);
  k_jacobi_small<NP><<<grid, NP <= 32 ? 32 : 64, smem, st>>>(prm);
  return wpcd_check_cuda(h, cudaGetLastError(), "diag_batched (small) launch");
}

}  // namespace

size_t wpcd_jacobi_small_workspace() { return 256; }

int wpcd_jacobi_small_launch(WpcdHandle* h, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                             double tol, int max_sweeps, const int* h_rows, int n_ranges, void* d_work, size_t work_bytes,
                             cudaStream_t st) {
  if (work_bytes < wpcd_jacobi_small_workspace()) return WPCD_EWORK;
  SmallParams prm;
  prm.H = d_A; prm.W = d_W; prm.C = d_C; prm.info = d_info;
  prm.next = static_cast<int*>(d_work);
  prm.n = n; prm.batch = batch; prm.max_sweeps = max_sweeps;
  prm.nranges = n_ranges;
  for (int r = 0; r < 4; ++r) { prm.row_lo[r] = r < n_ranges ? h_rows[2 * r] : 0; prm.row_hi[r] = r < n_ranges ? h_rows[2 * r + 1] : 0; }
  prm.tol = tol > 0.0 ? tol : 2.220446049250313e-16;
  // CTAs per SM: bounded by registers (one row of V per thread) and by the 32-CTA limit
  if (n <= 16) return launch_small<16>(h, prm, 16, st);
  if (n <= 24) return launch_small<24>(h, prm, 12, st);
  return launch_small<32>(h, prm, 12, st);
}
