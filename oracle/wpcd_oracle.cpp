// wpcd_oracle.cpp -- CPU ORACLE for the WPCD hot path (arXiv:2106.00454).  TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, fp64, obviously-correct restatement of what the hot path computes, written from
// /root/reference/PAPER.md (cited as PAPER.md:<line>) and the readings C1..C16 / G1..G3 of SURVEY.md section 8(c)
// (restated in DESIGN.md).  It shares NO code with the CUDA library under paper_2106_00454_b200/csrc and must only
// be imported / linked / executed by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs.  No BLAS, no LAPACK, no blocking, no fusion: every function follows the paper's order and notation.
//
// Parity pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
//   gl_rule          : weights sum to 2, exact on monomials to degree 2n-1, vs numpy.polynomial.legendre.leggauss
//   legendre_Q       : vs mpmath.legenq (independent arbitrary-precision evaluation) and the Neumann integral
//   V_yukawa         : vs adaptive quadrature of the radial (r-space) definition on tiny grids
//   jacobi           : closed-form 2x2/3x3, rank-one secular equation by bisection (Yamaguchi), invariants, mpmath
//   jacobi_ld        : (the 80-bit arbiter of the GPU parity tests) eigenvalues vs mpmath.eigsy at 50 digits on the config
//                      and Chebyshev grids up to N = 100, secular equation, eigenvectors vs mpmath and the residual in
//                      extended precision (tests/test_oracle_pins_arbiter.py)
//   V_yukawa (z-1)   : the cancellation-free argument on the high-momentum diagonal (z - 1 < 1e-5) vs mpmath with z formed
//                      in 50-digit arithmetic, 1e-13
//   onshell_T_avg    : coupled branch (readings A1-A3): two-branch toy spectrum with a bound state enumerated by hand,
//                      coupled averaged WPCD -> coupled MI decreasing with N
//   resolvent / T    : limits of Eq. B.3-B.6, sum rule, hand-evaluated tiny cases; energy-averaged variant (B.7-B.8)
//                      against numerical quadrature of the point-wise resolvent and the Yamaguchi closed form
//   phases           : closed forms of Eqs. A.3-A.5 (unit-modulus S built from known angles)
//   MI solver        : Yamaguchi analytic phase shifts; unitarity
//   whole WPCD chain : converges to MI as N grows, also on the paper's Chebyshev grid (Eq. 31)
//   sigma_tot        : Clebsch-Gordan vs sympy, Y_lm vs scipy, single-wave closed forms, partial-wave sum, optical
//                      theorem (angular integral of Eq. A.6), Yamaguchi closed form, WPCD -> MI convergence
//   The paper prints no matrix, eigenvalue or phase shift for a reproducible input (its potential, NNLO_opt, is
//   not available), so no value of the chain is pinned to a PAPER-PRINTED number: "parity unpinned by the paper
//   itself"; the pins above are closed forms / independent evaluations instead.
//
// Units: momenta fm^-1, energies MeV, hbarc = 197.327 MeV fm, mu = 469.46 MeV; E = cE p^2, cE = hbarc^2/(2 mu).
// Bins are 0-based: bin i spans [p_i, p_{i+1}], i = 0..N-1.  All matrices row-major.

#include <cmath>
#include <complex>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;

extern "C" {

// ---------------------------------------------------------------------------------------------------------------
// Gauss-Legendre rule on [-1,1]: nodes = roots of P_n by Newton, weights 2/((1-x^2) P_n'(x)^2).
// Used for the bin integrals of Eq. 29 (the paper only says "quadrature", PAPER.md:229;
// BASELINE.json fixes 8 points per bin) and for the MI grid.
void orc_gl_rule(int n, double* x, double* w) {
  for (int i = 0; i < n; ++i) {
    double z = std::cos(PI * (i + 0.75) / (n + 0.5));  // Tricomi-type initial guess
    double pp = 0.0;
    for (int it = 0; it < 100; ++it) {
      double p0 = 1.0, p1 = z;  // P_0, P_1
      for (int k = 2; k <= n; ++k) {
        double pk = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
        p0 = p1; p1 = pk;
      }
      if (n == 0) p1 = 1.0;
      pp = n * (z * p1 - p0) / (z * z - 1.0);  // P_n'(z)
      double dz = p1 / pp;
      z -= dz;
      if (std::fabs(dz) < 1e-16) break;
    }
    // recompute derivative at the converged node
    double p0 = 1.0, p1 = z;
    for (int k = 2; k <= n; ++k) {
      double pk = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
      p0 = p1; p1 = pk;
    }
    pp = n * (z * p1 - p0) / (z * z - 1.0);
    x[n - 1 - i] = z;  // ascending
    w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Legendre function of the second kind Q_l(z), z > 1, l >= 0 (reading C7; not in the paper, which defers the
// partial-wave projection to its ref. [26]).  int_0^inf r^2 dr j_l(k'r) (e^{-mu r}/r) j_l(kr)
// = Q_l(z)/(2k'k), z = (k'^2+k^2+mu^2)/(2k'k).
//   z <= zstar : Q_0 = 0.5*log1p(2/(z-1)),  Q_1 = z Q_0 - 1,  (l+1) Q_{l+1} = (2l+1) z Q_l - l Q_{l-1}   (upward)
//   z >  zstar : Q_l = sqrt(pi) Gamma(l+1)/(Gamma(l+3/2) (2z)^{l+1}) * 2F1((l+1)/2,(l+2)/2; l+3/2; z^-2)  (series)
// zstar = 1.1 (SURVEY proposed 1.5; 1.1 keeps the upward recurrence's error growth below ~1e-14 for l <= 5 while
// the series still converges geometrically with ratio z^-2 <= 0.83; reading C7).
// zm1 = z - 1 is passed separately so that callers can form it without cancellation:
//   z - 1 = ((k'-k)^2 + mu^2)/(2k'k)   (z itself is within 1e-5 of 1 on the high-momentum diagonal).
double orc_legendre_Qz(int l, double z, double zm1) {
  const double zstar = 1.1;
  double q0 = 0.5 * std::log1p(2.0 / zm1);
  if (l == 0) return q0;
  if (z <= zstar) {
    double qm = q0, q = z * q0 - 1.0;
    for (int k = 1; k < l; ++k) {
      double qn = ((2.0 * k + 1.0) * z * q - k * qm) / (k + 1.0);
      qm = q; q = qn;
    }
    return q;
  }
  // prefactor sqrt(pi) Gamma(l+1)/Gamma(l+3/2) = 2^{l+1} l! / (2l+1)!!  ->  pref/(2z)^{l+1} = l!/((2l+1)!! z^{l+1})
  double pref = 1.0;
  for (int k = 1; k <= l; ++k) pref *= (double)k / (2.0 * k + 1.0);
  double a = 0.5 * (l + 1.0), b = 0.5 * (l + 2.0), c = l + 1.5, x = 1.0 / (z * z);
  double term = 1.0, sum = 1.0;
  for (int k = 0; k < 2000; ++k) {
    term *= (a + k) * (b + k) / ((c + k) * (k + 1.0)) * x;
    sum += term;
    if (term < 1e-18 * sum) break;
  }
  return pref * sum / std::pow(z, l + 1);
}
double orc_legendre_Q(int l, double z) { return orc_legendre_Qz(l, z, z - 1.0); }

// z and z-1 of a Yukawa of range mu between momenta kp, k.
static inline void yukawa_z(double kp, double k, double mu, double* z, double* zm1) {
  *zm1 = ((kp - k) * (kp - k) + mu * mu) / (2.0 * kp * k);
  *z = 1.0 + *zm1;
}

// ---------------------------------------------------------------------------------------------------------------
// Step (i).  Config grid of BASELINE.json: p_i = alpha tan(pi i/(2N+1)), i = 0..N (row a0).
void orc_grid_tan(int N, double alpha, double* p) {
  for (int i = 0; i <= N; ++i) p[i] = alpha * std::tan(PI * i / (2.0 * N + 1.0));
}

// The paper's own bin distribution, Eq. 31: y_0 = 0, y_j = alpha tan^t((2j-1) pi/(4 N)), j = 1..N
// ("sparseness degree" t, scale alpha; the paper uses momentum bins with t = 2 and alpha = 100 MeV, i.e.
// alpha = 100/hbarc fm^-1).  SURVEY 8(f)-3.
void orc_grid_chebyshev(int N, double t, double alpha, double* p) {
  p[0] = 0.0;
  for (int j = 1; j <= N; ++j) p[j] = alpha * std::pow(std::tan((2.0 * j - 1.0) * PI / (4.0 * N)), t);
}

// Free wave-packet (f(k)=1, N_i = Delta k_i, Eq. 17) kinetic energies and bin energy widths.
// Reading C4: exact matrix element <x_i|h0|x_i> = cE (p_i^2 + p_i p_{i+1} + p_{i+1}^2)/3, not Eq. 18's midpoint.
// Eedge_i = cE p_i^2 (E = p^2/m_N, m_N = 2 mu), dE_i = Eedge_{i+1} - Eedge_i.
void orc_fwp(int N, const double* p, double hbarc, double mu, double* e0, double* dE, double* Eedge) {
  double cE = hbarc * hbarc / (2.0 * mu);
  for (int i = 0; i <= N; ++i) Eedge[i] = cE * p[i] * p[i];
  for (int i = 0; i < N; ++i) {
    e0[i] = cE * (p[i] * p[i] + p[i] * p[i + 1] + p[i + 1] * p[i + 1]) / 3.0;
    dE[i] = Eedge[i + 1] - Eedge[i];
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Eq. 29 with f=1, N_i = Delta k_i, convention B (reading C1):
//   <k'|v_l|k>_B = (1/pi) sum_t V0_t Q_l(z_t)/(k'k),  z_t = (k'^2+k^2+mu_t^2)/(2k'k)
//   V_ij = (1/(pi sqrt(Dk_i Dk_j))) sum_ab w_ia w_jb sum_t V0_t Q_l(z_t(k_ia,k_jb)),  n_gl points per bin.
// Upper triangle computed, mirrored (bit-symmetric).
void orc_V_yukawa(int N, const double* p, int l, int nterms, const double* V0, const double* mu, int ngl, double* V) {
  std::vector<double> x(ngl), w(ngl);
  orc_gl_rule(ngl, x.data(), w.data());
  std::vector<double> k(N * ngl), om(N * ngl);
  for (int i = 0; i < N; ++i)
    for (int a = 0; a < ngl; ++a) {
      double dk = p[i + 1] - p[i];
      k[i * ngl + a] = 0.5 * (p[i] + p[i + 1]) + 0.5 * dk * x[a];
      om[i * ngl + a] = 0.5 * dk * w[a];
    }
  for (int i = 0; i < N; ++i)
    for (int j = i; j < N; ++j) {
      double acc = 0.0;
      for (int a = 0; a < ngl; ++a)
        for (int b = 0; b < ngl; ++b) {
          double kp = k[i * ngl + a], kk = k[j * ngl + b];
          double s = 0.0;
          for (int t = 0; t < nterms; ++t) {
            double z, zm1;
            yukawa_z(kp, kk, mu[t], &z, &zm1);
            s += V0[t] * orc_legendre_Qz(l, z, zm1);
          }
          acc += om[i * ngl + a] * om[j * ngl + b] * s;
        }
      double v = acc / (PI * std::sqrt((p[i + 1] - p[i]) * (p[j + 1] - p[j])));
      V[i * N + j] = v;
      V[j * N + i] = v;
    }
}

// Separable Yamaguchi potential (reading C15): <k'|v|k>_B = -lambdaB g(k') g(k), g(k) = 1/(k^2+beta^2)
//   V_ij = -lambdaB G_i G_j,  G_i = Dk_i^{-1/2} int_{D_i} k g(k) dk.
// closed_form != 0: G_i = 0.5 ln((p_{i+1}^2+beta^2)/(p_i^2+beta^2))/sqrt(Dk_i); else n_gl-point Gauss-Legendre.
void orc_V_yamaguchi(int N, const double* p, double lambdaB, double beta, int ngl, int closed_form, double* V, double* G) {
  std::vector<double> x(ngl), w(ngl);
  orc_gl_rule(ngl, x.data(), w.data());
  for (int i = 0; i < N; ++i) {
    double dk = p[i + 1] - p[i];
    if (closed_form) {
      G[i] = 0.5 * std::log((p[i + 1] * p[i + 1] + beta * beta) / (p[i] * p[i] + beta * beta)) / std::sqrt(dk);
    } else {
      double acc = 0.0;
      for (int a = 0; a < ngl; ++a) {
        double k = 0.5 * (p[i] + p[i + 1]) + 0.5 * dk * x[a];
        acc += 0.5 * dk * w[a] * k / (k * k + beta * beta);
      }
      G[i] = acc / std::sqrt(dk);
    }
  }
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) V[i * N + j] = -lambdaB * G[i] * G[j];
}

// ---------------------------------------------------------------------------------------------------------------
// NEXT-4: ENERGY wave packets, Eq. 17 with the weighting function f(k) = hbarc sqrt(k/mu) (PAPER.md:143:
// "sqrt(k/mu)", hbar restored so that k dk f^2 = k dE) and N_i = Delta E_i.
//   <x_i|h0|x_i> = (1/dE_i) int_{D_i} E dE = E_i + dE_i/2                       -- Eq. 18, exact for these packets
//   <x_i|v|x_j>  = (1/sqrt(dE_i dE_j)) int int k'k dk'dk f(k')f(k) <k'|v|k>      -- Eq. 29
//               = (hbarc^2/(pi mu sqrt(dE_i dE_j))) sum_ab w_ia w_jb sqrt(k_ia k_jb) sum_t V0_t Q_l(z_t)   (Yukawa)
// The S-matrix relation S = 1 - 2 pi i T_ii/dE_i (reading C2) holds for them at every q of the bin: Eq. 20 gives
// <E|T|E> = (mu q/hbarc^2) f(q)^2/(N_i q^2) T_ii = T_ii/dE_i.  Steps (ii)-(v) are unchanged.
void orc_fwp_energy(int N, const double* p, double hbarc, double mu, double* e0, double* dE, double* Eedge) {
  double cE = hbarc * hbarc / (2.0 * mu);
  for (int i = 0; i <= N; ++i) Eedge[i] = cE * p[i] * p[i];
  for (int i = 0; i < N; ++i) {
    dE[i] = Eedge[i + 1] - Eedge[i];
    e0[i] = Eedge[i] + 0.5 * dE[i];
  }
}

void orc_V_yukawa_energy(int N, const double* p, int l, int nterms, const double* V0, const double* mu, int ngl,
                         double hbarc, double mured, double* V) {
  std::vector<double> x(ngl), w(ngl);
  orc_gl_rule(ngl, x.data(), w.data());
  double cE = hbarc * hbarc / (2.0 * mured);
  for (int i = 0; i < N; ++i)
    for (int j = i; j < N; ++j) {
      double dki = p[i + 1] - p[i], dkj = p[j + 1] - p[j];
      double acc = 0.0;
      for (int a = 0; a < ngl; ++a)
        for (int b = 0; b < ngl; ++b) {
          double kp = 0.5 * (p[i] + p[i + 1]) + 0.5 * dki * x[a], kk = 0.5 * (p[j] + p[j + 1]) + 0.5 * dkj * x[b];
          double s = 0.0;
          for (int t = 0; t < nterms; ++t) {
            double z, zm1;
            yukawa_z(kp, kk, mu[t], &z, &zm1);
            s += V0[t] * orc_legendre_Qz(l, z, zm1);
          }
          // k'k dk'dk f(k')f(k) <k'|v|k> = (hbarc^2/mu) sqrt(k'k) (1/pi) s dk'dk
          acc += (0.5 * dki * w[a]) * (0.5 * dkj * w[b]) * std::sqrt(kp * kk) * s;
        }
      double dEi = cE * (p[i + 1] * p[i + 1] - p[i] * p[i]), dEj = cE * (p[j + 1] * p[j + 1] - p[j] * p[j]);
      double v = hbarc * hbarc / mured * acc / (PI * std::sqrt(dEi * dEj));
      V[i * N + j] = v;
      V[j * N + i] = v;
    }
}

// Yamaguchi with energy packets: V_ij = -lambdaB G_i G_j, G_i = dE_i^{-1/2} int_{D_i} k f(k) g(k) dk by n_gl-point GL.
void orc_V_yamaguchi_energy(int N, const double* p, double lambdaB, double beta, int ngl, double hbarc, double mured,
                            double* V, double* G) {
  std::vector<double> x(ngl), w(ngl);
  orc_gl_rule(ngl, x.data(), w.data());
  double cE = hbarc * hbarc / (2.0 * mured);
  for (int i = 0; i < N; ++i) {
    double dk = p[i + 1] - p[i], acc = 0.0;
    for (int a = 0; a < ngl; ++a) {
      double k = 0.5 * (p[i] + p[i + 1]) + 0.5 * dk * x[a];
      acc += 0.5 * dk * w[a] * k * (hbarc * std::sqrt(k / mured)) / (k * k + beta * beta);
    }
    G[i] = acc / std::sqrt(cE * (p[i + 1] * p[i + 1] - p[i] * p[i]));
  }
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) V[i * N + j] = -lambdaB * G[i] * G[j];
}

// H = H0 + V.  Uncoupled: n = N, H = diag(e0) + Vmm.  Coupled (degenerate FWP bases,
// the same H0 in both blocks): n = 2N, H = [[H0 + Vmm, Vmp],[Vmp^T, H0 + Vpp]].  Also returns V (same layout).
void orc_assemble_H(int N, int coupled, const double* e0, const double* Vmm, const double* Vpp, const double* Vmp,
                    double* H, double* V) {
  int n = coupled ? 2 * N : N;
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      int bi = i / N, bj = j / N, ii = i % N, jj = j % N;
      double v;
      if (bi == 0 && bj == 0) v = Vmm[ii * N + jj];
      else if (bi == 1 && bj == 1) v = Vpp[ii * N + jj];
      else if (bi == 0 && bj == 1) v = Vmp[ii * N + jj];
      else v = Vmp[jj * N + ii];
      V[i * n + j] = v;
      H[i * n + j] = v + ((i == j) ? e0[ii] : 0.0);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Step (ii), Eq. 21: H = C D C^T by cyclic-by-row two-sided Jacobi (oracle step 4 of SURVEY 8(c)):
//   theta = (a_qq - a_pp)/(2 a_pq), t = sgn(theta)/(|theta| + sqrt(theta^2+1)), c = 1/sqrt(t^2+1), s = t c;
//   stop when a sweep starts with off(A) <= tol * ||A||_F  (tol = 1e-15 by default), eigenvalues = diagonal,
//   sorted ascending together with the columns of C.  Returns the number of sweeps done (or -1 if max_sweeps hit).
}  // extern "C" (template below has C++ linkage)
template <typename R>
static int jacobi_impl(int n, const double* Ain, double* W, double* C, double tol, int max_sweeps) {
  std::vector<R> A(Ain, Ain + (size_t)n * n), V((size_t)n * n, R(0));
  for (int i = 0; i < n; ++i) V[(size_t)i * n + i] = R(1);
  int sweeps = 0;
  bool converged = false;
  for (;;) {
    R off = 0, fro = 0;
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        R a = A[(size_t)i * n + j];
        fro += a * a;
        if (i != j) off += a * a;
      }
    if (std::sqrt(off) <= R(tol) * std::sqrt(fro)) { converged = true; break; }
    if (sweeps >= max_sweeps) break;
    for (int p = 0; p < n - 1; ++p)
      for (int q = p + 1; q < n; ++q) {
        R apq = A[(size_t)p * n + q];
        if (apq == 0) continue;
        R app = A[(size_t)p * n + p], aqq = A[(size_t)q * n + q];
        R theta = (aqq - app) / (R(2) * apq);
        R t = (theta >= 0 ? R(1) : R(-1)) / (std::fabs(theta) + std::sqrt(theta * theta + R(1)));
        R c = R(1) / std::sqrt(t * t + R(1)), s = t * c;
        for (int k = 0; k < n; ++k) {  // columns p,q:  A <- A J
          R akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
          A[(size_t)k * n + p] = c * akp - s * akq;
          A[(size_t)k * n + q] = s * akp + c * akq;
        }
        for (int k = 0; k < n; ++k) {  // rows p,q:  A <- J^T A
          R apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
          A[(size_t)p * n + k] = c * apk - s * aqk;
          A[(size_t)q * n + k] = s * apk + c * aqk;
        }
        // the rotated pivot is zero by construction; diagonal by the stable update
        A[(size_t)p * n + p] = app - t * apq;
        A[(size_t)q * n + q] = aqq + t * apq;
        A[(size_t)p * n + q] = 0;
        A[(size_t)q * n + p] = 0;
        for (int k = 0; k < n; ++k) {  // eigenvectors: V <- V J
          R vkp = V[(size_t)k * n + p], vkq = V[(size_t)k * n + q];
          V[(size_t)k * n + p] = c * vkp - s * vkq;
          V[(size_t)k * n + q] = s * vkp + c * vkq;
        }
      }
    ++sweeps;
  }
  std::vector<int> idx(n);
  for (int i = 0; i < n; ++i) idx[i] = i;
  std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return A[(size_t)a * n + a] < A[(size_t)b * n + b]; });
  for (int k = 0; k < n; ++k) {
    W[k] = (double)A[(size_t)idx[k] * n + idx[k]];
    for (int i = 0; i < n; ++i) C[(size_t)i * n + k] = (double)V[(size_t)i * n + idx[k]];
  }
  return converged ? sweeps : -1;
}

extern "C" {
int orc_jacobi(int n, const double* Ain, double* W, double* C, double tol, int max_sweeps) {
  return jacobi_impl<double>(n, Ain, W, C, tol, max_sweeps);
}
// The same algorithm in x87 extended precision (64-bit mantissa): a pin for the fp64 run, never timed.
int orc_jacobi_ld(int n, const double* Ain, double* W, double* C, double tol, int max_sweeps) {
  return jacobi_impl<long double>(n, Ain, W, C, tol, max_sweeps);
}

// ---------------------------------------------------------------------------------------------------------------
// Step (iii), Eq. 23, taken as printed (reading C5), for one branch of m positive eigenvalues
// eps[0..m-1] (ascending): edge[0] = 0, edge[i] = (eps[i-1]+eps[i])/2, edge[m] = eps[m-1] + (edge[m-1]-edge[m-2])/2.
// (m == 1: edge[1] = 2 eps[0], so that Eq. 22 holds.)
void orc_swp_edges(int m, const double* eps, double* edge) {
  if (m <= 0) return;
  edge[0] = 0.0;
  for (int i = 1; i < m; ++i) edge[i] = 0.5 * (eps[i - 1] + eps[i]);
  if (m == 1) edge[1] = 2.0 * eps[0];
  else edge[m] = eps[m - 1] + 0.5 * (edge[m - 1] - edge[m - 2]);
}

// Appendix B, Eqs. B.3-B.6 with the sign of the printed last line corrected (reading G2):
//   Re g_k(E) = ln|(E - lo)/(E - hi)|/(hi - lo),  Im g_k(E) = -pi/(hi - lo) iff lo <= E < hi  (half-open, C11).
cplx orc_resolvent(double E, double lo, double hi) {
  double w = hi - lo;
  double re = std::log(std::fabs((E - lo) / (E - hi))) / w;
  double im = (E >= lo && E < hi) ? -PI / w : 0.0;
  return cplx(re, im);
}
void orc_resolvent_c(double E, double lo, double hi, double* out) {
  cplx g = orc_resolvent(E, lo, hi);
  out[0] = g.real(); out[1] = g.imag();
}

// Steps (iv)-(v): Eq. 32 / Eq. 39 / Eq. 27, point-wise resolvent.
//   uncoupled: T_ii(E) = V_ii + sum_b (VC)_ib^2/(E-eps_b) + sum_k (VC)_ik^2 g_k(E),  i = FWP bin with
//              Eedge_i <= E < Eedge_{i+1};   out T[e] (re,im), bin[e] = i (or -1 if E is outside the grid: T = 0)
//   coupled  : rows (alpha,i) -> alpha*N+i; T^{ab} = V_{(a i)(b i)} + sum_k (VC)_{(a i)k} g_k (VC)_{(b i)k};
//              positive eigenvalues alternate between two branches by rank (reading C6), each branch with its own
//              Eq. 23 edges; out T[e][a][b] (re,im).
// W ascending, C columns = eigenvectors (as returned by orc_jacobi).  VC by the plain triple loop.
void orc_onshell_T(int N, int coupled, const double* Eedge, const double* V, const double* W, const double* C,
                   const double* Ecm, int nE, double* T, int* bin) {
  int n = coupled ? 2 * N : N;
  std::vector<double> VC((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i)
    for (int k = 0; k < n; ++k) {
      double s = 0.0;
      for (int j = 0; j < n; ++j) s += V[(size_t)i * n + j] * C[(size_t)j * n + k];
      VC[(size_t)i * n + k] = s;
    }
  int nb = 0;
  while (nb < n && W[nb] < 0.0) ++nb;
  int nbranch = coupled ? 2 : 1;
  std::vector<std::vector<int>> members(nbranch);
  for (int k = nb; k < n; ++k) members[(k - nb) % nbranch].push_back(k);
  std::vector<double> lo(n, 0.0), hi(n, 0.0);
  for (int br = 0; br < nbranch; ++br) {
    int m = (int)members[br].size();
    if (m == 0) continue;
    std::vector<double> eps(m), edge(m + 1);
    for (int i = 0; i < m; ++i) eps[i] = W[members[br][i]];
    orc_swp_edges(m, eps.data(), edge.data());
    for (int i = 0; i < m; ++i) { lo[members[br][i]] = edge[i]; hi[members[br][i]] = edge[i + 1]; }
  }
  int nc = coupled ? 2 : 1;
  for (int e = 0; e < nE; ++e) {
    double E = Ecm[e];
    int ib = -1;
    for (int i = 0; i < N; ++i)
      if (E >= Eedge[i] && E < Eedge[i + 1]) { ib = i; break; }
    bin[e] = ib;
    for (int a = 0; a < nc; ++a)
      for (int b = 0; b < nc; ++b) {
        cplx t(0.0, 0.0);
        if (ib >= 0) {
          int ra = a * N + ib, rb = b * N + ib;
          t = cplx(V[(size_t)ra * n + rb], 0.0);
          for (int k = 0; k < nb; ++k) t += VC[(size_t)ra * n + k] * VC[(size_t)rb * n + k] / (E - W[k]);
          for (int k = nb; k < n; ++k) t += VC[(size_t)ra * n + k] * VC[(size_t)rb * n + k] * orc_resolvent(E, lo[k], hi[k]);
        }
        size_t o = ((size_t)e * nc * nc + a * nc + b) * 2;
        T[o] = t.real(); T[o + 1] = t.imag();
      }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// NEXT-1: energy-averaged resolvent, Eq. 28 and Eqs. B.7-B.8.
// The average of g_k(E) (state bin [lo,hi]) over an averaging bin [a,b]:
//   Re gbar = W/((b-a)(hi-lo)),  W = (b-lo)ln|b-lo| - (b-hi)ln|b-hi| - (a-lo)ln|a-lo| + (a-hi)ln|a-hi|,  x ln|x| -> 0 at 0
//   Im gbar = -pi/(hi-lo) iff the averaging bin IS the state's bin
// W is the antiderivative (E-c)ln|E-c| - (E-c) of ln|E-c| taken between a and b for c = lo minus the same for c = hi;
// it is Eq. B.8 with the overall sign of the printed formula corrected (reading G3: the printed B.7 carries the same
// sign slip as B.5/B.6, reading G2).
static double xlnx(double x) { return x == 0.0 ? 0.0 : x * std::log(std::fabs(x)); }
cplx orc_resolvent_avg(double a, double b, double lo, double hi, int same_bin) {
  double W = xlnx(b - lo) - xlnx(b - hi) - xlnx(a - lo) + xlnx(a - hi);
  return cplx(W / ((b - a) * (hi - lo)), same_bin ? -PI / (hi - lo) : 0.0);
}
void orc_resolvent_avg_c(double a, double b, double lo, double hi, int same_bin, double* out) {
  cplx g = orc_resolvent_avg(a, b, lo, hi, same_bin);
  out[0] = g.real(); out[1] = g.imag();
}

// Energy-averaged on-shell T: ONE value per on-shell FWP bin i ("if we use energy averaging we only require a single
// evaluation for each on-shell wave packet"), returned for every requested energy of that bin.
//   T_ii = V_ii + sum_b (VC)_ib^2 gbar_b + sum_k (VC)_ik^2 gbar_k   (coupled: the 2x2 block as in orc_onshell_T)
// Readings (A1-A3): the averaging bin of a state of branch beta is the pseudostate bin of the i-th
// positive state of the SAME branch (k(i) = i in the positive spectrum, Eq. 39 "g_jj(E in D_i)"); only
// that state gets the -i pi term; a bound state's 1/(E - eps_b) is averaged over branch 0's bin:
// ln|(b-eps_b)/(a-eps_b)|/(b-a).  If a branch has no i-th state the bin is treated as outside the grid (T = 0).
void orc_onshell_T_avg(int N, int coupled, const double* Eedge, const double* V, const double* W, const double* C,
                       const double* Ecm, int nE, double* T, int* bin) {
  int n = coupled ? 2 * N : N;
  std::vector<double> VC((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i)
    for (int k = 0; k < n; ++k) {
      double s = 0.0;
      for (int j = 0; j < n; ++j) s += V[(size_t)i * n + j] * C[(size_t)j * n + k];
      VC[(size_t)i * n + k] = s;
    }
  int nb = 0;
  while (nb < n && W[nb] < 0.0) ++nb;
  int nbranch = coupled ? 2 : 1;
  std::vector<std::vector<int>> members(nbranch);
  for (int k = nb; k < n; ++k) members[(k - nb) % nbranch].push_back(k);
  std::vector<double> lo(n, 0.0), hi(n, 0.0);
  for (int br = 0; br < nbranch; ++br) {
    int m = (int)members[br].size();
    if (m == 0) continue;
    std::vector<double> eps(m), edge(m + 1);
    for (int i = 0; i < m; ++i) eps[i] = W[members[br][i]];
    orc_swp_edges(m, eps.data(), edge.data());
    for (int i = 0; i < m; ++i) { lo[members[br][i]] = edge[i]; hi[members[br][i]] = edge[i + 1]; }
  }
  int nc = coupled ? 2 : 1;
  for (int e = 0; e < nE; ++e) {
    double E = Ecm[e];
    int ib = -1;
    for (int i = 0; i < N; ++i)
      if (E >= Eedge[i] && E < Eedge[i + 1]) { ib = i; break; }
    bin[e] = ib;
    bool ok = ib >= 0;
    for (int br = 0; br < nbranch && ok; ++br) ok = ib < (int)members[br].size();
    for (int a = 0; a < nc; ++a)
      for (int b = 0; b < nc; ++b) {
        cplx t(0.0, 0.0);
        if (ok) {
          int ra = a * N + ib, rb = b * N + ib;
          t = cplx(V[(size_t)ra * n + rb], 0.0);
          int k0 = members[0][ib];
          for (int k = 0; k < nb; ++k)
            t += VC[(size_t)ra * n + k] * VC[(size_t)rb * n + k] *
                 (std::log(std::fabs((hi[k0] - W[k]) / (lo[k0] - W[k]))) / (hi[k0] - lo[k0]));
          for (int k = nb; k < n; ++k) {
            int ki = members[(k - nb) % nbranch][ib];  // the i-th state of k's branch: its bin is the averaging bin
            t += VC[(size_t)ra * n + k] * VC[(size_t)rb * n + k] * orc_resolvent_avg(lo[ki], hi[ki], lo[k], hi[k], k == ki);
          }
        }
        size_t o = ((size_t)e * nc * nc + a * nc + b) * 2;
        T[o] = t.real(); T[o + 1] = t.imag();
      }
  }
}

// Eqs. A.3-A.5 with the wave-packet normalisation of readings C2/A20:
//   S = 1 - 2 pi i T_ii(E)/dE_i  (dE_i = FWP bin energy width)
//   uncoupled: delta = 0.5 atan2(Im S, Re S) in degrees, in (-90, 90]; absS = |S|
//   coupled (Stapp): delta_- = 0.5 arg S_11, delta_+ = 0.5 arg S_22,
//                    sin 2eps = Re[-i S_12 e^{-i(delta_- + delta_+)}], cos 2eps = |S_11|, eps = 0.5 atan2(sin, cos)
//   out delta[e] or delta[e][3] = (delta_-, delta_+, eps) in degrees; S[e] or S[e][2][2] (re,im) if S != NULL.
void orc_phase_shifts(int coupled, int nE, const double* T, const int* bin, const double* dE, double* delta, double* S) {
  const double deg = 180.0 / PI;
  int nc = coupled ? 2 : 1;
  for (int e = 0; e < nE; ++e) {
    cplx s[2][2];
    double w = (bin[e] >= 0) ? dE[bin[e]] : 1.0;
    for (int a = 0; a < nc; ++a)
      for (int b = 0; b < nc; ++b) {
        size_t o = ((size_t)e * nc * nc + a * nc + b) * 2;
        cplx t(T[o], T[o + 1]);
        s[a][b] = (a == b ? 1.0 : 0.0) - cplx(0.0, 2.0 * PI) * t / w;
        if (S) { S[o] = s[a][b].real(); S[o + 1] = s[a][b].imag(); }
      }
    if (!coupled) {
      delta[e] = 0.5 * std::atan2(s[0][0].imag(), s[0][0].real()) * deg;
    } else {
      double dm = 0.5 * std::atan2(s[0][0].imag(), s[0][0].real());
      double dp = 0.5 * std::atan2(s[1][1].imag(), s[1][1].real());
      cplx r = cplx(0.0, -1.0) * s[0][1] * std::exp(cplx(0.0, -(dm + dp)));
      double ep = 0.5 * std::atan2(r.real(), std::abs(s[0][0]));
      delta[3 * e] = dm * deg; delta[3 * e + 1] = dp * deg; delta[3 * e + 2] = ep * deg;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Independent matrix-inversion (MI) Lippmann-Schwinger solver, Sec. 2.1, Eqs. 2-7 with D derived
// from Eqs. 2-4 directly (reading C3/G1: the printed Eq. 5 is inconsistent):
//   grid: GL nodes x_j on [-1,1] mapped k_j = c tan(pi(1+x_j)/4), w_j -> c (pi/4) w_j / cos^2(pi(1+x_j)/4), c = 1
//   f = 2 mu/hbarc^2;   D_j = (2/pi) w_j k_j^2 f/(p^2-k_j^2);   D_{NQ+1} = -(2/pi) f p^2 sum_j w_j/(p^2-k_j^2) - i f p
//   F = 1 - V diag(D)  (Eq. 7), solve F T = V (Eq. 6) by complex Gauss elimination with partial pivoting,
//   on-shell T = element(s) at the on-shell index;  S = 1 - 2 i f p T  (conv. A, reading C2).
// The potential is given by callback-free tables: vtab[(a*nc+b)][i][j] = v_A^{ab}(q_i,q_j) on the basis
// q = {k_1..k_NQ, p}, prepared by orc_mi_potential_* below (convention A: v = sum_t V0_t Q_l(z_t)/(2k'k)).
static void gauss_solve(int n, std::vector<cplx>& A, std::vector<cplx>& B, int nrhs) {
  for (int c = 0; c < n; ++c) {
    int piv = c; double best = std::abs(A[(size_t)c * n + c]);
    for (int r = c + 1; r < n; ++r) { double v = std::abs(A[(size_t)r * n + c]); if (v > best) { best = v; piv = r; } }
    if (piv != c) {
      for (int k = 0; k < n; ++k) std::swap(A[(size_t)c * n + k], A[(size_t)piv * n + k]);
      for (int k = 0; k < nrhs; ++k) std::swap(B[(size_t)c * nrhs + k], B[(size_t)piv * nrhs + k]);
    }
    for (int r = c + 1; r < n; ++r) {
      cplx m = A[(size_t)r * n + c] / A[(size_t)c * n + c];
      if (m == cplx(0.0, 0.0)) continue;
      for (int k = c; k < n; ++k) A[(size_t)r * n + k] -= m * A[(size_t)c * n + k];
      for (int k = 0; k < nrhs; ++k) B[(size_t)r * nrhs + k] -= m * B[(size_t)c * nrhs + k];
    }
  }
  for (int r = n - 1; r >= 0; --r)
    for (int k = 0; k < nrhs; ++k) {
      cplx s = B[(size_t)r * nrhs + k];
      for (int c = r + 1; c < n; ++c) s -= A[(size_t)r * n + c] * B[(size_t)c * nrhs + k];
      B[(size_t)r * nrhs + k] = s / A[(size_t)r * n + r];
    }
}

void orc_mi_grid(int NQ, double cmap, double* k, double* w) {
  std::vector<double> x(NQ), wx(NQ);
  orc_gl_rule(NQ, x.data(), wx.data());
  for (int j = 0; j < NQ; ++j) {
    double ang = PI * (1.0 + x[j]) / 4.0;
    k[j] = cmap * std::tan(ang);
    w[j] = cmap * (PI / 4.0) * wx[j] / (std::cos(ang) * std::cos(ang));
  }
}

// potential kinds for MI:  kind 0 = Yukawa sum (central terms V0/mu for block l; coupled: blocks l=J-1, J+1 with the
// same central terms and the off-diagonal block V_T Q_J(z)/(2k'k), reading C8);  kind 1 = Yamaguchi -lambdaA g g.
static double vA_yukawa(int l, int nterms, const double* V0, const double* mu, double kp, double k) {
  double s = 0.0;
  for (int t = 0; t < nterms; ++t) {
    double z, zm1;
    yukawa_z(kp, k, mu[t], &z, &zm1);
    s += V0[t] * orc_legendre_Qz(l, z, zm1);
  }
  return s / (2.0 * kp * k);
}

// Solve at one lab energy.  out S (nc x nc complex, re/im interleaved), T likewise.
void orc_mi_solve(int kind, int coupled, int l_or_J, int nterms, const double* V0, const double* mu, double VT, double muT,
                  double lambdaA, double beta, double hbarc, double mured, int NQ, double Tlab, double* Sout, double* Tout) {
  double p = std::sqrt(mured * Tlab) / hbarc;  // p = sqrt(mu T_lab)/hbarc (equal masses), E_cm = T_lab/2
  double f = 2.0 * mured / (hbarc * hbarc);
  std::vector<double> k(NQ), w(NQ);
  orc_mi_grid(NQ, 1.0, k.data(), w.data());
  int M = NQ + 1, nc = coupled ? 2 : 1, n = nc * M;
  std::vector<double> q(M);
  for (int j = 0; j < NQ; ++j) q[j] = k[j];
  q[NQ] = p;
  std::vector<cplx> D(M);
  double ssum = 0.0;
  for (int j = 0; j < NQ; ++j) {
    D[j] = (2.0 / PI) * w[j] * k[j] * k[j] * f / (p * p - k[j] * k[j]);
    ssum += w[j] / (p * p - k[j] * k[j]);
  }
  D[NQ] = cplx(-(2.0 / PI) * f * p * p * ssum, -f * p);
  std::vector<cplx> Vm((size_t)n * n), F((size_t)n * n), B((size_t)n * nc);
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b)
      for (int i = 0; i < M; ++i)
        for (int j = 0; j < M; ++j) {
          double v;
          if (kind == 1) v = -lambdaA / ((q[i] * q[i] + beta * beta) * (q[j] * q[j] + beta * beta));
          else if (!coupled) v = vA_yukawa(l_or_J, nterms, V0, mu, q[i], q[j]);
          else if (a == b) v = vA_yukawa(a == 0 ? l_or_J - 1 : l_or_J + 1, nterms, V0, mu, q[i], q[j]);
          else v = vA_yukawa(l_or_J, 1, &VT, &muT, q[i], q[j]);
          Vm[(size_t)(a * M + i) * n + (b * M + j)] = v;
        }
  for (int r = 0; r < n; ++r)
    for (int c = 0; c < n; ++c) F[(size_t)r * n + c] = (r == c ? 1.0 : 0.0) - Vm[(size_t)r * n + c] * D[c % M];
  for (int r = 0; r < n; ++r)
    for (int b = 0; b < nc; ++b) B[(size_t)r * nc + b] = Vm[(size_t)r * n + (b * M + NQ)];
  gauss_solve(n, F, B, nc);
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b) {
      cplx t = B[(size_t)(a * M + NQ) * nc + b];
      cplx s = (a == b ? 1.0 : 0.0) - cplx(0.0, 2.0 * f * p) * t;
      Tout[(a * nc + b) * 2] = t.real(); Tout[(a * nc + b) * 2 + 1] = t.imag();
      Sout[(a * nc + b) * 2] = s.real(); Sout[(a * nc + b) * 2 + 1] = s.imag();
    }
}

// ---------------------------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------------------------
// NEXT-1, second half: linear interpolation of the phase shifts between the bin mid-points, Eq. 42.
//   pedge[N+1]   momentum bin edges q_0..q_N (fm^-1); mid-points qbar_i = (q_i + q_{i+1})/2 (Eq. 43 with n = m/2)
//   dmid[N][nc]  phase shifts at the mid-points in degrees, nc = 1 (delta) or 3 (delta_-, delta_+, eps_J)
//   q[nq]        target momenta; out[nq][nc] in degrees, principal value (-90, 90]; q outside the grid: NaN
// As printed: for q in bin i the straight line through (qbar_{i-1}, delta_{i-1}) and (qbar_i, delta_i) (so the upper
// half of a bin is an extrapolation of that line); bin 0 uses the line of bins 0 and 1 (reading I1).  Before that the
// mid-point phases are made continuous (reading I2): delta_i is shifted by the multiple of 180 degrees that brings it
// within 90 degrees of delta_{i-1} (the principal value jumps by 180 at a bound-state transition), and
// eps_J changes sign with every odd shift of delta_- or delta_+ (S_12 = i sin 2eps e^{i(delta_- + delta_+)}, Eq. A.5).
static double wrap90(double d) {
  double r = std::fmod(d + 90.0, 180.0);
  if (r <= 0.0) r += 180.0;
  return r - 90.0;  // in (-90, 90]
}
void orc_interp_phases(int N, int nc, const double* pedge, const double* dmid, const double* q, int nq, double* out) {
  std::vector<double> u((size_t)N * nc);
  std::vector<int> flips(N, 0);
  for (int c = 0; c < (nc == 3 ? 2 : 1); ++c) {
    double shift = 0.0;
    for (int i = 0; i < N; ++i) {
      double d = dmid[(size_t)i * nc + c] + shift;
      if (i > 0) {
        double prev = u[(size_t)(i - 1) * nc + c];
        while (d - prev > 90.0) { d -= 180.0; shift -= 180.0; }
        while (d - prev <= -90.0) { d += 180.0; shift += 180.0; }
      }
      u[(size_t)i * nc + c] = d;
      flips[i] += (int)std::llround(shift / 180.0);
    }
  }
  if (nc == 3)
    for (int i = 0; i < N; ++i) u[(size_t)i * 3 + 2] = (flips[i] & 1) ? -dmid[(size_t)i * 3 + 2] : dmid[(size_t)i * 3 + 2];
  for (int e = 0; e < nq; ++e) {
    int ib = -1;
    for (int i = 0; i < N; ++i)
      if (q[e] >= pedge[i] && q[e] < pedge[i + 1]) { ib = i; break; }
    for (int c = 0; c < nc; ++c) {
      double r = std::nan("");
      if (ib >= 0 && N >= 2) {
        int i1 = ib > 0 ? ib : 1, i0 = i1 - 1;
        double q0 = 0.5 * (pedge[i0] + pedge[i0 + 1]), q1 = 0.5 * (pedge[i1] + pedge[i1 + 1]);
        double d0 = u[(size_t)i0 * nc + c], d1 = u[(size_t)i1 * nc + c];
        double slope = (d1 - d0) / (q1 - q0);
        r = slope * q[e] + (d0 - slope * q0);                     // Eq. 42 as printed
        if (!(nc == 3 && c == 2)) r = wrap90(r);
      }
      out[(size_t)e * nc + c] = r;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// NEXT-2: total cross section from the partial-wave S-matrix, Appendix A, followed
// step by step: spin-scattering matrix M (Eq. A.2) at theta = 0 -> Saclay amplitudes a, b (Eq. A.9) ->
// sigma_tot = (2 pi/p) Im(a + b) (Eq. A.11).
//
// Clebsch-Gordan coefficient <j1 m1 j2 m2 | J M> for INTEGER angular momenta (l, s in {0,1}, J), Racah's formula.
static double factorial(int n) { double f = 1.0; for (int i = 2; i <= n; ++i) f *= i; return f; }
double orc_clebsch_gordan(int j1, int m1, int j2, int m2, int J, int M) {
  if (m1 + m2 != M || J < std::abs(j1 - j2) || J > j1 + j2) return 0.0;
  if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(M) > J) return 0.0;
  double pre = (2.0 * J + 1.0) * factorial(J + j1 - j2) * factorial(J - j1 + j2) * factorial(j1 + j2 - J) / factorial(j1 + j2 + J + 1);
  pre *= factorial(J + M) * factorial(J - M) * factorial(j1 - m1) * factorial(j1 + m1) * factorial(j2 - m2) * factorial(j2 + m2);
  double sum = 0.0;
  for (int k = 0; k <= j1 + j2 - J; ++k) {
    int a = j1 + j2 - J - k, b = j1 - m1 - k, c = j2 + m2 - k, d = J - j2 + m1 + k, e = J - j1 - m2 + k;
    if (a < 0 || b < 0 || c < 0 || d < 0 || e < 0) continue;
    double term = 1.0 / (factorial(k) * factorial(a) * factorial(b) * factorial(c) * factorial(d) * factorial(e));
    sum += (k & 1) ? -term : term;
  }
  return std::sqrt(pre) * sum;
}

// Spherical harmonic Y_l^m(theta, phi = 0) (real; Condon-Shortley phase), by the upward recurrence of P_l^m(cos theta).
double orc_sph_harm(int l, int m, double theta) {
  int am = std::abs(m);
  if (am > l) return 0.0;
  double x = std::cos(theta), sx = std::sin(theta);
  double pmm = 1.0;
  for (int i = 1; i <= am; ++i) pmm *= -(2.0 * i - 1.0) * sx;  // P_m^m = (-1)^m (2m-1)!! sin^m
  double plm = pmm;
  if (l > am) {
    double pm1 = x * (2.0 * am + 1.0) * pmm;  // P_{m+1}^m
    plm = pm1;
    double pm2 = pmm;
    for (int ll = am + 2; ll <= l; ++ll) {
      plm = (x * (2.0 * ll - 1.0) * pm1 - (ll + am - 1.0) * pm2) / (ll - am);
      pm2 = pm1; pm1 = plm;
    }
  }
  double y = std::sqrt((2.0 * l + 1.0) / (4.0 * PI) * factorial(l - am) / factorial(l + am)) * plm;
  if (m < 0 && (am & 1)) y = -y;  // Y_l^{-m} = (-1)^m conj(Y_l^m)
  return y;
}


// Eq. A.2 for neutron-proton scattering at angle theta (phi = 0):
//   M^s_{m_s, m_s'} = (2 pi/(i p)) sum_{J,l,l'} sqrt((2l+1)/(4 pi)) Y_{l'}^{m_s - m_s'}(theta)
//                     <l' (m_s - m_s'), s m_s' | J m_s> <l 0, s m_s | J m_s> [S^{sJ}_{l'l} - delta_{l'l}]
// m_s = spin projection of the incoming state (beam along z: m_l = 0), m_s' of the outgoing one.
// Readings (X1-X2): the printed isospin factor [1 - (-1)^{l+s+T_Z}] would remove 1S0 from np scattering; it
// is the antisymmetrisation factor 1 - (-1)^{l+s+T} with the total isospin T, and the np amplitude is the mean of the
// T = 0 and T = 1 amplitudes, which gives weight 1 to every Pauli-allowed partial wave (each (l,s) has one T).  The
// second Clebsch-Gordan coefficient is printed with its projections in the order (m_s, 0); it couples (l, m_l = 0)
// with (s, m_s).  No factor i^{l-l'} (as printed; it does not affect sigma_tot).
// Partial waves: pw = 0..npw-1 with quantum numbers s[pw], J[pw], lp[pw] (outgoing l'), l[pw] (incoming l) and
// Spw[pw] = (re, im) of S^{sJ}_{l'l}.  Mout[s][m_s + 1][m_s' + 1] (re, im): 2 x 3 x 3 x 2 doubles.
void orc_spin_scattering_M(int npw, const int* s, const int* J, const int* lp, const int* l, const double* Spw, double p,
                           double theta, double* Mout) {
  for (int i = 0; i < 2 * 3 * 3 * 2; ++i) Mout[i] = 0.0;
  for (int ss = 0; ss <= 1; ++ss)
    for (int ms = -ss; ms <= ss; ++ms)
      for (int msp = -ss; msp <= ss; ++msp) {
        cplx tot(0.0, 0.0);
        for (int w = 0; w < npw; ++w) {
          if (s[w] != ss) continue;
          double y = orc_sph_harm(lp[w], ms - msp, theta);
          double c1 = orc_clebsch_gordan(lp[w], ms - msp, ss, msp, J[w], ms);
          double c2 = orc_clebsch_gordan(l[w], 0, ss, ms, J[w], ms);
          cplx Sm(Spw[2 * w] - (lp[w] == l[w] ? 1.0 : 0.0), Spw[2 * w + 1]);
          tot += std::sqrt((2.0 * l[w] + 1.0) / (4.0 * PI)) * y * c1 * c2 * Sm;
        }
        cplx M = cplx(2.0 * PI / p, 0.0) / cplx(0.0, 1.0) * tot;
        size_t o = ((size_t)(ss * 3 + (ms + 1)) * 3 + (msp + 1)) * 2;
        Mout[o] = M.real(); Mout[o + 1] = M.imag();
      }
}

// Eqs. A.9 and A.11 at theta = 0:
//   a = (M^1_{11} + M^1_{00} + M^1_{1,-1})/2,  b = (M^1_{11} + M^0_{00} + M^1_{1,-1})/2,  sigma_tot = (2 pi/p) Im(a + b)
// p in fm^-1; returns sigma_tot in millibarn (1 fm^2 = 10 mb).
double orc_sigma_tot(int npw, const int* s, const int* J, const int* lp, const int* l, const double* Spw, double p) {
  double M[2 * 3 * 3 * 2];
  orc_spin_scattering_M(npw, s, J, lp, l, Spw, p, 0.0, M);
  auto el = [&](int ss, int ms, int msp) { size_t o = ((size_t)(ss * 3 + (ms + 1)) * 3 + (msp + 1)) * 2; return cplx(M[o], M[o + 1]); };
  cplx a = 0.5 * (el(1, 1, 1) + el(1, 0, 0) + el(1, 1, -1));
  cplx b = 0.5 * (el(1, 1, 1) + el(0, 0, 0) + el(1, 1, -1));
  return 10.0 * (2.0 * PI / p) * (a + b).imag();
}

// Whole chain for a batch of (sample, channel) solves, OpenMP over the batch (used only for timing the oracle as the
// reported CPU baseline and by tests that need many solves).  Per solve b: H_b (n x n) and V_b are given
// (assembled by orc_V_yukawa/orc_assemble_H), outputs W, C, T, delta.  Returns max sweeps (or -1).
int orc_solve_batch(int N, int coupled, int batch, const double* Eedge, const double* dE, const double* H, const double* V,
                    const double* Ecm, int nE, double tol, int max_sweeps, double* W, double* C, double* T, int* bin,
                    double* delta, double* S, int* sweeps_out) {
  int n = coupled ? 2 * N : N, nc = coupled ? 2 : 1, worst = 0;
#pragma omp parallel for schedule(dynamic) reduction(max : worst)
  for (int b = 0; b < batch; ++b) {
    std::vector<int> binl(nE);
    int sw = orc_jacobi(n, H + (size_t)b * n * n, W + (size_t)b * n, C + (size_t)b * n * n, tol, max_sweeps);
    orc_onshell_T(N, coupled, Eedge, V + (size_t)b * n * n, W + (size_t)b * n, C + (size_t)b * n * n, Ecm, nE,
                  T + (size_t)b * nE * nc * nc * 2, binl.data());
    orc_phase_shifts(coupled, nE, T + (size_t)b * nE * nc * nc * 2, binl.data(), dE,
                     delta + (size_t)b * nE * (coupled ? 3 : 1), S ? S + (size_t)b * nE * nc * nc * 2 : nullptr);
    if (b == 0) std::memcpy(bin, binl.data(), sizeof(int) * nE);
    if (sweeps_out) sweeps_out[b] = sw;
    int swv = sw < 0 ? 1000000 : sw;
    if (swv > worst) worst = swv;
  }
  return worst >= 1000000 ? -1 : worst;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
