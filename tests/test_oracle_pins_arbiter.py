"""Round-2 pins of the oracle parts that round 1 left "parity unpinned":

  * orc_jacobi_ld -- the 80-bit arbiter of the GPU parity tests: eigenvalues against mpmath at 50
    digits on the graded Hamiltonians where the arbitration is used (config grid and the paper's Chebyshev grid), the
    rank-one secular equation (P2), eigenvectors against mpmath and through the residual in extended precision;
  * the COUPLED branch of orc_onshell_T_avg (readings A1-A3, C6): a two-branch toy spectrum with one bound state assembled
    by hand from orc_resolvent_avg with the branch membership written out explicitly, and convergence of the coupled
    averaged WPCD S-matrix towards coupled MI with N;
  * orc_V_yukawa on the high-momentum diagonal (reading C7: z - 1 ~ 1e-5 formed without cancellation) against mpmath
    with the argument z formed in 50-digit arithmetic;
  * reading C6 for the point-wise coupled T: the distance to coupled MI decreases with N.

None of these re-types the oracle's formulas: references are mpmath, bisection, quadrature, MI, or hand-enumerated cases.
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

from oracle import oracle as o
from paper_2106_00454_b200 import inputs as inp

MT = dict(V0=inp.MT_V0, mu=inp.MT_MU)


def _mt_H(p, l=0, ngl=8):
    e0, dE, Ee = o.fwp(p)
    H, Vf = o.assemble_H(e0, o.V_yukawa(p, l, ngl=ngl, **MT))
    return H


def _mp_eigs(H, vectors=False):
    mp.mp.dps = 50
    M = mp.matrix(H.tolist())
    if not vectors:
        return sorted(mp.eigsy(M, eigvals_only=True)), None
    E, Q = mp.eigsy(M)
    order = sorted(range(len(E)), key=lambda i: E[i])
    return [E[i] for i in order], [[Q[r, i] for r in range(H.shape[0])] for i in order]


def _rel_err_mp(W, ref):
    return max(abs(float((mp.mpf(float(a)) - b) / b)) for a, b in zip(W, ref))


# ------------------------------------------------------------------------------------- orc_jacobi_ld (the arbiter)
@pytest.mark.parametrize("grid,N,ngl,tol_ld", [("tan", 24, 8, 3e-16), ("cheb", 24, 1, 3e-16), ("cheb", 48, 1, 5e-14),
                                              ("cheb", 96, 1, 3e-16), ("tan", 100, 8, 3e-16)])
def test_jacobi_ld_eigenvalues_vs_mpmath(grid, N, ngl, tol_ld):
    """PAPER.md:158-160 (Eq. 21).  The long-double run must be componentwise accurate far below the 1e-11 parity
    tolerance on exactly the matrices where it arbitrates: the config grid (n up to 800: the same grading law) and the
    Chebyshev grid of Eq. 31, whose H spans 1e9 ... 1e-8 MeV.  Reference: mpmath.eigsy at 50 digits on the same fp64
    matrix.  fp64 storage of the result allows 1.1e-16; the one case that stops a sweep early (norm-wise stop rule,
    Chebyshev N = 48) still holds 5e-14."""
    p = inp.grid_edges(N) if grid == "tan" else inp.grid_chebyshev(N)
    H = _mt_H(p, 0, ngl)
    ref, _ = _mp_eigs(H)
    W_ld, C_ld, sw = o.jacobi_ld(H)
    assert 1 <= sw <= 12 and np.all(np.diff(W_ld) >= 0)
    err_ld = _rel_err_mp(W_ld, ref)
    assert err_ld <= tol_ld, (grid, N, err_ld)
    # and it is the better of the two runs wherever the fp64 oracle is off by more than a few ulps (why it may arbitrate)
    err_64 = _rel_err_mp(o.jacobi(H)[0], ref)
    assert err_ld <= max(err_64, 3e-16), (err_ld, err_64)
    if grid == "cheb" and N in (24, 96):
        assert err_64 > 1e-11       # the fp64 oracle (norm-wise stop) is NOT within the parity tolerance here: DESIGN.md section 3


def test_jacobi_ld_eigenvectors_vs_mpmath_and_extended_residual():
    """The phase arbitration uses the arbiter's eigenvectors too: columns against mpmath's (up to sign) on a graded H,
    C^T C = 1 and H C = C D evaluated in extended precision (numpy longdouble, not the oracle's code)."""
    N = 24
    H = _mt_H(inp.grid_chebyshev(N), 0, 1)
    ref, vec = _mp_eigs(H, vectors=True)
    W, C, _ = o.jacobi_ld(H)
    for k in range(N):
        v = np.array([float(x) for x in vec[k]])
        v /= np.linalg.norm(v)
        assert min(np.abs(C[:, k] - v).max(), np.abs(C[:, k] + v).max()) < 1e-13, k
    for Hm in (H, _mt_H(inp.grid_edges(60), 0, 8)):
        W, C, _ = o.jacobi_ld(Hm)
        n = Hm.shape[0]
        Hl, Cl, Wl = Hm.astype(np.longdouble), C.astype(np.longdouble), W.astype(np.longdouble)
        assert np.abs(Cl.T @ Cl - np.eye(n)).max() < 5e-16
        R = Hl @ Cl - Cl * Wl
        # column-wise: the residual of eigenpair k is small against |eps_k| + the rounding of the fp64-stored vector times ||H||
        assert np.abs(R).max() < 4e-16 * np.abs(Hm).max()


def test_jacobi_ld_rank_one_secular_P2():
    """Yamaguchi H = diag(e) - lam G G^T; its eigenvalues are the roots of 1 = lam sum_i G_i^2/(e_i - x), found
    by bisection in 60-digit arithmetic -- no eigensolver involved.  The arbiter must match them to fp64 rounding."""
    N = 40
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    lamA, lamB = inp.yamaguchi_lambda()
    V, G = o.V_yamaguchi(p, lamB * 1.5, inp.YAMAGUCHI_BETA)
    H, _ = o.assemble_H(e0, V)
    # the secular equation of the fp64 matrix that was actually stored: use H's own entries (diag and rank-one part)
    mp.mp.dps = 60
    e = [mp.mpf(float(x)) for x in e0]
    g2 = [mp.mpf(float(x)) ** 2 for x in G]
    lam = mp.mpf(float(lamB * 1.5))
    f = lambda x: 1 - lam * sum(gi / (ei - x) for gi, ei in zip(g2, e))
    roots = []
    for lo, hi in [(e[0] - 1e6, e[0])] + [(e[i - 1], e[i]) for i in range(1, N)]:
        w = hi - lo
        a, b = lo + w * mp.mpf(10) ** -40, hi - w * mp.mpf(10) ** -40
        fa = f(a)
        for _ in range(220):
            m = (a + b) / 2
            fm = f(m)
            if fa * fm <= 0: b = m
            else: a, fa = m, fm
        roots.append((a + b) / 2)
    W_ld = o.jacobi_ld(H)[0]
    # H's entries e_i - lam G_i G_j are rounded to fp64 when stored, which moves the eigenvalues by ~1e-16 ||H||-relative
    # parts of the rank-one term: compare at 2e-14 (the fp64 oracle's pin in test_oracle_pins.py holds 1e-13)
    assert _rel_err_mp(W_ld, sorted(roots)) < 2e-14
    assert roots[0] < 0 < roots[1]


# ------------------------------------------------------------------------------------- coupled energy-averaged T
def test_coupled_T_avg_two_branch_toy_by_hand():
    """Readings A1-A3 and C6 for a coupled channel, on a toy spectrum small enough to enumerate by hand:
    N = 3 (n = 6), eigenvalues (-1.5 | 0.6, 1.1, 2.2, 3.0, 5.1): one bound state; positive states alternate by rank, so
    branch 0 = states {1, 3, 5} (0.6, 2.2, 5.1) and branch 1 = states {2, 4} (1.1, 3.0) -- written out here, not computed
    from an index rule.  For on-shell bin i the averaging bin of a state is the bin of the i-th state of ITS branch, only
    that state gets -i pi, the bound state is averaged over branch 0's bin; bin 2 has no third state in branch 1, so it
    counts as outside the grid (A3)."""
    N, n = 3, 6
    Ee = np.array([0.0, 1.0, 3.0, 7.0])
    rng = np.random.default_rng(11)
    W = np.array([-1.5, 0.6, 1.1, 2.2, 3.0, 5.1])
    Cm = np.linalg.qr(rng.standard_normal((n, n)))[0]
    V = rng.standard_normal((n, n)); V = V + V.T
    Ecm = np.array([0.3, 0.8, 2.0, 5.0, 9.0])
    T, b = o.onshell_T(N, True, Ee, V, W, Cm, Ecm, averaged=True)
    assert list(b) == [0, 0, 1, 2, -1]
    assert np.array_equal(T[0], T[1])                       # one value per on-shell bin
    assert np.all(T[3] == 0) and np.all(T[4] == 0)          # A3 (branch 1 has no third state) and outside the grid
    branch = {0: [1, 3, 5], 1: [2, 4]}                      # state indices, by hand
    edges = {0: o.swp_edges(np.array([0.6, 2.2, 5.1])), 1: o.swp_edges(np.array([1.1, 3.0]))}
    assert np.allclose(edges[0], [0.0, 1.4, 3.65, 6.225]) and np.allclose(edges[1], [0.0, 2.05, 4.025])   # Eq. 23 by hand
    VC = V @ Cm
    for e, i in ((0, 0), (2, 1)):
        for al in range(2):
            for be in range(2):
                ra, rb = al * N + i, be * N + i
                t = complex(V[ra, rb])
                a0, b0 = edges[0][i], edges[0][i + 1]       # A2: the bound state is averaged over branch 0's bin
                gb = integrate.quad(lambda E: 1.0 / (E + 1.5), a0, b0, epsabs=1e-14, epsrel=1e-14)[0] / (b0 - a0)
                t += VC[ra, 0] * VC[rb, 0] * gb
                for br in (0, 1):
                    a_, b_ = edges[br][i], edges[br][i + 1]          # averaging bin: i-th bin of the state's own branch
                    for pos, k in enumerate(branch[br]):
                        g = o.resolvent_avg(a_, b_, edges[br][pos], edges[br][pos + 1], pos == i)
                        t += VC[ra, k] * VC[rb, k] * g
                assert abs(T[e][al, be] - t) < 1e-12 * max(1.0, abs(t)), (e, al, be, T[e][al, be], t)
        # Im T: exactly one state per branch contributes -pi/(bin width)
        im = -math.pi * sum(VC[i, branch[br][i]] ** 2 / (edges[br][i + 1] - edges[br][i]) for br in (0, 1))
        assert abs(T[e][0, 0].imag - im) < 1e-12
    # the averaged real part is the bin average of the point-wise one, branch by branch: with the point-wise T of the same
    # spectrum integrated over branch 0's bin alone the two differ (branch 1 is averaged over ITS bin) -- guards against
    # an implementation that averages every state over one common bin
    Tp = lambda E: o.onshell_T(N, True, Ee, V, W, Cm, np.array([E]))[0][0][0, 0].real
    a0, b0 = edges[0][0], edges[0][1]
    common = integrate.quad(Tp, a0, b0, points=[0.6, 1.1], limit=400)[0] / (b0 - a0)
    assert abs(common - T[0][0, 0].real) > 1e-3


def _coupled_chain(N, J, averaged, tlab=None):
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    Vmm = o.V_yukawa(p, J - 1, **MT); Vpp = o.V_yukawa(p, J + 1, **MT)
    Vmp = o.V_yukawa(p, J, [inp.TENSOR_V], [inp.TENSOR_MU])
    H, V = o.assemble_H(e0, Vmm, Vpp, Vmp)
    W, C, _ = o.jacobi(H)
    if tlab is None:   # bin mid-points inside 20..350 MeV (the averaged variant is defined there, Eq. 42)
        cE = inp.HBARC ** 2 / (2 * inp.MU)
        Em = cE * (0.5 * (p[:-1] + p[1:])) ** 2
        Ecm = Em[(2 * Em >= 20.0) & (2 * Em <= 350.0)]
    else:
        Ecm = np.asarray(tlab) / 2
    T, b = o.onshell_T(N, True, Ee, V, W, C, Ecm, averaged=averaged)
    d, S = o.phase_shifts(True, T, b, dE)
    return 2 * Ecm, S


def _mi_S(tlab, J):
    return np.array([o.mi_solve(t, coupled=True, l_or_J=J, V0=inp.MT_V0, mu=inp.MT_MU, VT=inp.TENSOR_V, muT=inp.TENSOR_MU)[0]
                     for t in tlab])


def test_coupled_T_avg_converges_to_coupled_MI():
    """Coupled energy-averaged WPCD (3S1-3D1-like, J = 1) against coupled MI at the bin mid-points: the largest |dS| over
    20..350 MeV decreases N = 50 -> 100 -> 200.  A wrong branch member or averaging bin
    destroys the convergence."""
    errs = []
    for N in (50, 100, 200):
        tl, S = _coupled_chain(N, 1, averaged=True)
        errs.append(np.abs(S - _mi_S(tl, 1)).max())
    assert errs[0] > errs[1] > errs[2], errs
    assert errs[2] < 0.03 and errs[0] < 0.2, errs


def test_coupled_pointwise_wpcd_converges_to_MI_reading_C6():
    """Reading C6 (branch assignment by rank) for the point-wise T: median |dS| against coupled MI over 20..350 MeV
    decreases with N (the point-wise variant spikes near bin edges, so the median is the monotone statistic)."""
    tl = np.linspace(20, 350, 23)
    Smi = _mi_S(tl, 1)
    errs = []
    for N in (50, 100, 200):
        _, S = _coupled_chain(N, 1, averaged=False, tlab=tl)
        errs.append(np.median(np.abs(S - Smi).reshape(len(tl), -1).max(axis=1)))
    assert errs[0] > errs[1] > errs[2], errs
    assert errs[2] < 0.03, errs


# ------------------------------------------------------------------------------------- V_ij on the high-momentum diagonal
@pytest.mark.parametrize("l", [0, 2, 5])
def test_V_yukawa_high_momentum_diagonal_vs_mpmath(l):
    """Reading C7: on the top bins of the N = 400 grid (k' ~ k ~ 300-500 fm^-1) z - 1 = ((k'-k)^2 + mu^2)/(2k'k) ~ 1e-5 and
    forming z first loses 5 digits of Q_l's argument.  Reference: Eq. 29's quadrature sum with numpy's
    Gauss-Legendre nodes, every z formed in 50-digit arithmetic from the fp64 nodes and Q_l by mpmath.legenq -- no
    cancellation anywhere.  The oracle must agree to 1e-13."""
    p = inp.grid_edges(400)[-5:]        # the top four bins of config 5's largest grid (edges are an input: a sub-grid is a grid)
    N = len(p) - 1
    V = o.V_yukawa(p, l, **MT)
    mp.mp.dps = 50
    x, w = np.polynomial.legendre.leggauss(8)
    for i, j in [(N - 1, N - 1), (N - 2, N - 1), (N - 3, N - 3), (N - 1, N - 4)]:
        ki = 0.5 * (p[i] + p[i + 1]) + 0.5 * (p[i + 1] - p[i]) * x; wi = 0.5 * (p[i + 1] - p[i]) * w
        kj = 0.5 * (p[j] + p[j + 1]) + 0.5 * (p[j + 1] - p[j]) * x; wj = 0.5 * (p[j + 1] - p[j]) * w
        s = mp.mpf(0)
        zmin = None
        for a in range(8):
            for b in range(8):
                kp, k = mp.mpf(float(ki[a])), mp.mpf(float(kj[b]))
                for V0, mu in zip(inp.MT_V0, inp.MT_MU):
                    z = (kp * kp + k * k + mp.mpf(float(mu)) ** 2) / (2 * kp * k)
                    zmin = z if zmin is None or z < zmin else zmin
                    s += mp.mpf(float(wi[a])) * mp.mpf(float(wj[b])) * mp.mpf(float(V0)) * mp.legenq(l, 0, z, type=3).real
        ref = s / (mp.pi * mp.sqrt(mp.mpf(float(p[i + 1] - p[i])) * mp.mpf(float(p[j + 1] - p[j]))))
        if i == j == N - 1:
            assert float(zmin) - 1 < 1e-5          # the regime the reading is about
        assert abs(float(V[i, j] / ref) - 1) < 1e-13, (l, i, j, V[i, j], float(ref))
