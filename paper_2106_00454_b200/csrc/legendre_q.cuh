// legendre_q.cuh -- Legendre function of the second kind Q_l(z), z > 1, for the partial-wave projection of Yukawa
// potentials (reading C7); shared by the assembly kernels (Eq. 29) and the MI kernels (Eq. 2).  CUDA side only.
#pragma once
#include <math.h>

// Legendre function of the second kind for z > 1 given z-1 (reading C7): log1p form for Q_0, upward
// recurrence below z = 1.1, Gauss hypergeometric series in 1/z^2 above.
__device__ __forceinline__ double legendre_q(int l, double zm1) {
  double z = 1.0 + zm1;
  double q0 = 0.5 * log1p(2.0 / zm1);
  if (l == 0) return q0;
  if (z < 1.1) {
    double qa = q0, qb = fma(z, q0, -1.0);
    for (int k = 1; k < l; ++k) {
      double qn = ((2 * k + 1) * z * qb - k * qa) / (k + 1);
      qa = qb; qb = qn;
    }
    return qb;
  }
  double pref = 1.0, zi = 1.0 / z, zp = zi;
  for (int k = 1; k <= l; ++k) { pref *= (double)k / (double)(2 * k + 1); zp *= zi; }
  double x = zi * zi, a = 0.5 * (l + 1), b = 0.5 * (l + 2), c = l + 1.5;
  double term = 1.0, sum = 1.0;
  for (int k = 0; k < 1000; ++k) {
    term *= (a + k) * (b + k) / ((c + k) * (k + 1.0)) * x;
    sum += term;
    if (term < 1e-18 * sum) break;
  }
  return pref * zp * sum;
}

