// jacobi_schedule.cuh -- the block tournament of the batched block-Jacobi eigensolver (jacobi.cu), as small
// host+device functions so that the CPU tests can check its invariants through the C ABI test hook
// wpcd_jacobi_schedule (every block pair met exactly once per sweep; the "critical" tiles that feed the next
// step's pivots are distinct).
//
// m players (blocks; m even, >= 6; players >= nb are dummies), m-1 steps per sweep, m/2 slots per step.
// Circle method: player m-1 stays, the others rotate:  slot 0 = (m-1, t),  slot s = ((t+s) mod (m-1), (t-s) mod (m-1)).
#pragma once

#ifdef __CUDACC__
#define WPCD_HD __host__ __device__ __forceinline__
#else
#define WPCD_HD inline
#endif

// the two players of slot s at step t
WPCD_HD void rr_pair(int m, int t, int s, int& a, int& b) {
  if (s == 0) { a = m - 1; b = t; }
  else { a = (t + s) % (m - 1); b = (t - s + (m - 1)) % (m - 1); }
}

// the player that meets x at step t
WPCD_HD int rr_partner(int m, int t, int x) {
  if (x == m - 1) return t;
  if (x == t) return m - 1;
  return (2 * t - x + 2 * (m - 1)) % (m - 1);
}

// the slot in which player x sits at step t
WPCD_HD int rr_slot_of(int m, int t, int x) {
  if (x == m - 1) return 0;
  const int u = (x - t + (m - 1)) % (m - 1);
  return u < m / 2 ? u : (m - 1) - u;
}

// Blocks (I < J) of slot s at step t with dummies removed: J = -1 for a single block, I = J = -1 for an empty slot.
WPCD_HD void slot_blocks(int m, int nb, int t, int s, int& I, int& J) {
  int a, b;
  rr_pair(m, t, s, a, b);
  I = a < b ? a : b;
  J = a < b ? b : a;
  if (J >= nb) J = -1;
  if (I >= nb) { I = -1; J = -1; }
}

// Is the tile (slots s1 < s2 of step t) the one that holds the off-diagonal block of a (real) pivot of step tn?
// If so returns that pivot's slot at step tn, else -1.
WPCD_HD int critical_slot(int m, int nb, int t, int tn, int s1, int s2) {
  int a1, b1, a2, b2;
  rr_pair(m, t, s1, a1, b1);
  rr_pair(m, t, s2, a2, b2);
  int x = -1;
  int p = rr_partner(m, tn, a1);
  if (p == a2 || p == b2) x = a1;
  p = rr_partner(m, tn, b1);
  if (x < 0 && (p == a2 || p == b2)) x = b1;
  if (x < 0) return -1;
  const int y = rr_partner(m, tn, x);
  if (x >= nb || y >= nb) return -1;
  return rr_slot_of(m, tn, x);
}
