"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types the oracle's own formula: each compares against an independent evaluation (mpmath arbitrary
precision, scipy adaptive quadrature of the defining integral, closed forms, bisection of a secular equation,
invariants, limits).
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

from oracle import oracle as o
from paper_2106_00454_b200 import inputs as inp

MT = dict(V0=inp.MT_V0, mu=inp.MT_MU)


# ---------------------------------------------------------------- P7: Gauss-Legendre rule
@pytest.mark.parametrize("n", [1, 2, 5, 8, 24, 96])
def test_gl_rule(n):
    x, w = o.gl_rule(n)
    assert abs(w.sum() - 2.0) < 1e-14
    for d in range(0, 2 * n):  # exact for monomials up to degree 2n-1
        exact = 0.0 if d % 2 else 2.0 / (d + 1)
        assert abs(np.dot(w, x ** d) - exact) < 2e-14
    xr, wr = np.polynomial.legendre.leggauss(n)
    assert np.abs(x - xr).max() < 1e-14 and np.abs(w - wr).max() < 1e-14


# ---------------------------------------------------------------- P8: Legendre Q_l (reading C7)
def test_legendre_Q_vs_mpmath():
    mp.mp.dps = 40
    zs = np.concatenate([1.0 + np.logspace(-5, 7, 61), [1.0999999, 1.1, 1.1000001, 1.5]])
    for l in range(0, 7):
        for z in zs:
            ref = float(mp.legenq(l, 0, mp.mpf(float(z)), type=3).real)
            assert abs(o.legendre_Q(l, float(z)) / ref - 1.0) < 1e-12, (l, z)


def test_legendre_Q_neumann_integral():
    # Neumann's formula Q_l(z) = 1/2 int_{-1}^{1} P_l(t)/(z-t) dt, by scipy adaptive quadrature
    from scipy.special import eval_legendre
    for l in range(0, 6):
        for z in [1.05, 1.3, 2.0, 7.0]:
            val, _ = integrate.quad(lambda t: 0.5 * eval_legendre(l, t) / (z - t), -1, 1, epsabs=1e-14, epsrel=1e-13, limit=200)
            assert abs(o.legendre_Q(l, z) - val) < 1e-11 * max(1.0, abs(val)), (l, z)


def test_Q_is_the_yukawa_partial_wave():
    # int_0^inf r^2 dr j_l(k'r) e^{-mu r}/r j_l(kr) = Q_l(z)/(2k'k)   (defining relation used by reading C7/C1)
    mp.mp.dps = 30
    for l, kp, k, mu in [(0, 0.7, 1.3, 1.55), (1, 0.5, 0.9, 3.11), (2, 1.1, 0.8, 2.0)]:
        f = lambda r: r * mp.exp(-mu * r) * mp.besselj(l + 0.5, kp * r) * mp.besselj(l + 0.5, k * r) * mp.pi / (2 * mp.sqrt(kp * k) * r)
        val = mp.quad(f, mp.linspace(0, 40, 81))
        z = (kp * kp + k * k + mu * mu) / (2 * kp * k)
        assert abs(o.legendre_Q(l, z) / (2 * kp * k) - float(val)) < 1e-10


# ---------------------------------------------------------------- a0: grid and free wave packets
def test_grid_and_fwp():
    N = 50
    p = o.grid_tan(N, 1.0)
    assert np.abs(p - inp.grid_edges(N)).max() < 1e-13 * p[-1]
    assert abs(p[50] - 64.29) < 0.01          # p_50 = 64.29 fm^-1
    e0, dE, Ee = o.fwp(p)
    cE = inp.HBARC ** 2 / (2 * inp.MU)
    # <x_i|h0|x_i> = (1/Dk) int_{D_i} cE k^2 dk  (Eq. 17 with f=1) by adaptive quadrature
    for i in [0, 7, 49]:
        val, _ = integrate.quad(lambda k: cE * k * k, p[i], p[i + 1])
        assert abs(e0[i] - val / (p[i + 1] - p[i])) < 1e-12 * e0[i]
    assert np.allclose(np.cumsum(dE), Ee[1:], rtol=1e-13)


# ---------------------------------------------------------------- a1: bin-averaged potential, Eq. 29
def test_V_yukawa_vs_adaptive_double_integral():
    # tiny grid, smooth region: 8x8 GL must agree with scipy's adaptive dblquad of Eq. 29 (conv. B, f=1, N_i=Dk_i)
    p = np.array([0.4, 0.9, 1.5, 2.4])
    for l in (0, 2):
        V = o.V_yukawa(p, l, **MT)
        assert np.array_equal(V, V.T)
        for i, j in [(0, 0), (0, 2), (1, 2)]:
            def integrand(k, kp):
                s = 0.0
                for V0, mu in zip(inp.MT_V0, inp.MT_MU):
                    z = (kp * kp + k * k + mu * mu) / (2 * kp * k)
                    s += V0 * float(mp.legenq(l, 0, z, type=3).real)
                return s / math.pi
            val, _ = integrate.dblquad(integrand, p[i], p[i + 1], p[j], p[j + 1], epsabs=1e-10, epsrel=1e-10)
            ref = val / math.sqrt((p[i + 1] - p[i]) * (p[j + 1] - p[j]))
            assert abs(V[i, j] - ref) < 2e-6 * abs(ref), (l, i, j, V[i, j], ref)


def test_V_yamaguchi_closed_form_vs_gl():
    p = inp.grid_edges(50)
    lamA, lamB = inp.yamaguchi_lambda()
    assert abs(lamA - 238.3487) < 1e-3 and abs(lamB - 151.7375) < 1e-3
    V1, G1 = o.V_yamaguchi(p, lamB, inp.YAMAGUCHI_BETA, closed_form=True)
    V2, G2 = o.V_yamaguchi(p, lamB, inp.YAMAGUCHI_BETA, closed_form=False)
    assert np.abs(G1 - G2).max() < 1e-8
    for i in (0, 10, 49):
        val, _ = integrate.quad(lambda k: k / (k * k + inp.YAMAGUCHI_BETA ** 2), p[i], p[i + 1])
        assert abs(G1[i] - val / math.sqrt(p[i + 1] - p[i])) < 1e-13
    assert np.allclose(V1, -lamB * np.outer(G1, G1), rtol=1e-15)


def test_assemble_coupled_layout():
    N = 3
    e0 = np.array([1.0, 2.0, 3.0])
    Vmm = np.arange(9.0).reshape(3, 3); Vmm = Vmm + Vmm.T
    Vpp = 10 + Vmm
    Vmp = np.arange(9.0).reshape(3, 3) * 0.1
    H, V = o.assemble_H(e0, Vmm, Vpp, Vmp)
    ref = np.block([[Vmm, Vmp], [Vmp.T, Vpp]])
    assert np.array_equal(V, ref)
    assert np.array_equal(H, ref + np.diag(np.concatenate([e0, e0])))


# ---------------------------------------------------------------- a2: Jacobi (P2, P3, P10)
def test_jacobi_2x2_and_3x3_closed_form():
    W, C, sw = o.jacobi(np.array([[2.0, 1.0], [1.0, 2.0]]))
    assert np.allclose(W, [1.0, 3.0], atol=1e-15) and sw >= 1
    assert np.allclose(np.abs(C), 1 / math.sqrt(2), atol=1e-15)
    # tridiagonal Toeplitz (2,-1): eigenvalues 2 - 2 cos(k pi/(n+1))
    n = 3
    A = 2 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)
    W, C, _ = o.jacobi(A)
    assert np.allclose(W, 2 - 2 * np.cos(np.arange(1, n + 1) * math.pi / (n + 1)), atol=1e-15)
    n = 12
    A = 2 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)
    W, C, _ = o.jacobi(A)
    assert np.allclose(W, 2 - 2 * np.cos(np.arange(1, n + 1) * math.pi / (n + 1)), atol=4e-15)
    # eigenvector k of the Toeplitz matrix is sin(i k pi/(n+1)) up to sign/norm: pins the column <-> eigenvalue order
    for k in range(n):
        v = np.sin(np.arange(1, n + 1) * (k + 1) * math.pi / (n + 1)); v /= np.linalg.norm(v)
        assert min(np.abs(C[:, k] - v).max(), np.abs(C[:, k] + v).max()) < 1e-14


def _mt_H(N, l=0):
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    V = o.V_yukawa(p, l, **MT)
    H, Vf = o.assemble_H(e0, V)
    return p, e0, dE, Ee, H, Vf


def test_jacobi_invariants_P3():
    for N in (50, 100):
        p, e0, dE, Ee, H, V = _mt_H(N)
        W, C, sw = o.jacobi(H)
        assert 1 <= sw <= 12
        assert np.all(np.diff(W) >= 0)
        assert np.abs(C.T @ C - np.eye(N)).max() < 1e-12
        assert abs(np.trace(H) - W.sum()) < 1e-13 * np.abs(W).sum()
        assert abs((H * H).sum() - (W * W).sum()) < 1e-13 * (W * W).sum()
        assert np.abs(H @ C - C * W).max() < 1e-13 * np.abs(W).max()


def test_jacobi_componentwise_vs_mpmath():
    # reading C12: componentwise accuracy on a strongly graded H (N=24, MT potential), 50-digit reference
    N = 24
    p, e0, dE, Ee, H, V = _mt_H(N)
    mp.mp.dps = 50
    ref = sorted(float(x) for x in mp.eigsy(mp.matrix(H.tolist()), eigvals_only=True))
    W, C, _ = o.jacobi(H)
    assert np.abs(W / np.array(ref) - 1).max() < 1e-13


def test_jacobi_rank_one_secular_P2():
    # Yamaguchi H = diag(e) - lamB G G^T: eigenvalues are the roots of 1 = lamB sum_i G_i^2/(e_i - x); the bound
    # state lies below e_0 and one root lies in each (e_{i-1}, e_i): bisection in 60-digit arithmetic.
    N = 40
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    lamA, lamB = inp.yamaguchi_lambda()
    V, G = o.V_yamaguchi(p, lamB * 1.5, inp.YAMAGUCHI_BETA)  # x1.5: make it bind, so the x < e_0 root is exercised
    H, _ = o.assemble_H(e0, V)
    W, C, _ = o.jacobi(H)
    mp.mp.dps = 60
    e = [mp.mpf(float(x)) for x in e0]; g2 = [mp.mpf(float(x)) ** 2 for x in G]; lam = mp.mpf(float(lamB * 1.5))
    f = lambda x: 1 - lam * sum(gi / (ei - x) for gi, ei in zip(g2, e))
    roots = []
    brackets = [(e[0] - 1e6, e[0])] + [(e[i - 1], e[i]) for i in range(1, N)]
    for lo, hi in brackets:
        w = hi - lo
        a, b = lo + w * mp.mpf(10) ** -40, hi - w * mp.mpf(10) ** -40
        fa, fb = f(a), f(b)
        if fa * fb > 0:
            continue
        for _ in range(200):
            m = (a + b) / 2
            fm = f(m)
            if fa * fm <= 0: b, fb = m, fm
            else: a, fa = m, fm
        roots.append(float((a + b) / 2))
    assert len(roots) == N
    assert roots[0] < 0 < roots[1]
    assert np.abs(W / np.array(sorted(roots)) - 1).max() < 1e-13


# ---------------------------------------------------------------- a3: Eq. 23
def test_swp_edges_hand_values():
    e = o.swp_edges(np.array([1.0, 3.0, 7.0]))
    # E1=0, E2=(1+3)/2, E3=(3+7)/2, E4 = 7 + (E3-E2)/2 as printed (reading C5)
    assert np.allclose(e, [0.0, 2.0, 5.0, 8.5], atol=0)
    assert np.allclose(o.swp_edges(np.array([2.0])), [0.0, 4.0])
    assert np.allclose(o.swp_edges(np.array([2.0, 4.0])), [0.0, 3.0, 5.5])


# ---------------------------------------------------------------- a4: resolvent limits (P6) and T
def test_resolvent_limits_P6():
    lo, hi = 10.0, 10.5
    g = o.resolvent(10.2, lo, hi)
    assert abs(g.imag + math.pi / 0.5) < 1e-14          # Im g = -pi/width inside
    assert o.resolvent(9.9, lo, hi).imag == 0.0 and o.resolvent(10.5, lo, hi).imag == 0.0  # half-open
    assert o.resolvent(10.0, lo, hi + 1).imag != 0.0
    # far away: narrow bin -> 1/(E - eps)   (from B.3 with the integrand constant over the bin)
    for E in (200.0, -50.0, 0.3):
        g = o.resolvent(E, lo, hi)
        assert abs(g.real - 1 / (E - 10.25)) < 2e-3 * abs(1 / (E - 10.25)) ** 2 + 1e-6
        assert abs(g.real * (E - 10.25) - 1) < 1e-3
    # B.3 by adaptive principal-value-free quadrature for E outside the bin: (1/w) int_lo^hi dE'/(E - E')
    for E in (3.0, 11.0, 40.0):
        val, _ = integrate.quad(lambda x: 1 / (E - x), lo, hi)
        assert abs(o.resolvent(E, lo, hi).real - val / 0.5) < 1e-12
    # inside the bin: principal value
    val, _ = integrate.quad(lambda x: 1.0, lo, hi, weight="cauchy", wvar=10.2)
    assert abs(o.resolvent(10.2, lo, hi).real - (-val) / 0.5) < 1e-10


def test_T_sum_rule_and_ImT():
    N = 50
    p, e0, dE, Ee, H, V = _mt_H(N)
    W, C, _ = o.jacobi(H)
    tl, Ecm = inp.energies(100)
    T, b = o.onshell_T(N, False, Ee, V, W, C, Ecm)
    assert b.min() == 3 and b.max() == 35      # on-shell bins 3..35 at N=50
    nb = int((W < 0).sum()); assert nb == 1
    edges = o.swp_edges(W[nb:])
    VC = V @ C
    for e in (0, 17, 99):
        E = Ecm[e]
        k = np.searchsorted(edges, E, side="right") - 1      # SWP bin containing E
        # Im T = -pi (VC)_ik^2/width_k : only the bin containing E contributes an imaginary part
        assert abs(T[e].imag - (-math.pi * VC[b[e], nb + k] ** 2 / (edges[k + 1] - edges[k]))) < 1e-12 * abs(T[e].imag)
        # sum rule: sum_k width_k Im g_k(E) = -pi
        s = sum((edges[j + 1] - edges[j]) * o.resolvent(E, edges[j], edges[j + 1]).imag for j in range(len(edges) - 1))
        assert abs(s + math.pi) < 1e-12


def test_T_tiny_case_by_hand():
    # N=2, diagonal V => C = 1, eigenvalues = H diagonal; T_ii = V_ii + V_ii^2 g_i(E): checked with python complex math
    Ee = np.array([0.0, 4.0, 10.0])
    V = np.diag([0.5, -0.25]); H = np.diag([2.0, 7.0]) + V
    W, C, _ = o.jacobi(H)
    assert np.allclose(W, [2.5, 6.75]) and np.allclose(np.abs(C), np.eye(2))
    T, b = o.onshell_T(2, False, Ee, V, W, C, np.array([1.0, 5.0, 12.0]))
    assert list(b) == [0, 1, -1] and T[2] == 0
    ed = [0.0, (2.5 + 6.75) / 2, 6.75 + ((2.5 + 6.75) / 2 - 0.0) / 2]
    g0 = math.log(abs((1.0 - ed[0]) / (1.0 - ed[1]))) / (ed[1] - ed[0]) - 1j * math.pi / (ed[1] - ed[0])
    assert abs(T[0] - (0.5 + 0.25 * g0)) < 1e-15
    g1 = math.log(abs((5.0 - ed[1]) / (5.0 - ed[2]))) / (ed[2] - ed[1]) - 1j * math.pi / (ed[2] - ed[1])
    assert abs(T[1] - (-0.25 + 0.0625 * g1)) < 1e-15


def test_identity_I1_P4():
    # (VC)_ik = C_ik (eps_k - e_i)  because H C = C D and H0 is diagonal
    N = 50
    p, e0, dE, Ee, H, V = _mt_H(N)
    W, C, _ = o.jacobi(H)
    VC = V @ C
    I1 = C * (W[None, :] - e0[:, None])
    assert np.abs(VC - I1).max() < 1e-13 * np.abs(VC).max()


# ---------------------------------------------------------------- a5: S-matrix and phases
def test_phase_shifts_from_known_angles():
    rng = np.random.default_rng(3)
    dE = np.array([0.7, 1.9])
    bins = np.array([0, 1, 1, 0], dtype=np.int32)
    d = np.array([-80.0, -10.0, 33.0, 89.0])
    S = np.exp(2j * np.radians(d))
    T = (1 - S) * dE[bins] / (2j * math.pi)            # invert S = 1 - 2 pi i T/dE
    out, S2 = o.phase_shifts(False, T, bins, dE)
    assert np.abs(out - d).max() < 1e-12 and np.abs(S2 - S).max() < 1e-14
    # coupled, Stapp (Eq. A.4)
    dm, dp, ep = np.radians([25.0, -7.0, 3.5])
    S = np.array([[math.cos(2 * ep) * np.exp(2j * dm), 1j * math.sin(2 * ep) * np.exp(1j * (dm + dp))],
                  [1j * math.sin(2 * ep) * np.exp(1j * (dm + dp)), math.cos(2 * ep) * np.exp(2j * dp)]])
    T = (np.eye(2) - S) * dE[1] / (2j * math.pi)
    out, S2 = o.phase_shifts(True, T[None], np.array([1], dtype=np.int32), dE)
    assert np.abs(out[0] - [25.0, -7.0, 3.5]).max() < 1e-12


# ---------------------------------------------------------------- MI solver: P1, P5
def _yamaguchi_S_exact(tlab):
    beta = inp.YAMAGUCHI_BETA
    lamA, _ = inp.yamaguchi_lambda()
    lp = lamA * inp.MU / inp.HBARC ** 2
    p = math.sqrt(inp.MU * tlab) / inp.HBARC
    g2 = 1.0 / (p * p + beta * beta) ** 2
    # T = -lam g^2/(1 - lam' /(beta (beta - i p)^2)),  S = 1 - 2 i f p T,  f lam = 2 lam'
    return 1 + 4j * lp * p * g2 / (1 - lp / (beta * (beta - 1j * p) ** 2))


def test_mi_yamaguchi_analytic_P1():
    lamA, _ = inp.yamaguchi_lambda()
    for NQ in (48, 96):
        for tlab in (1.0, 10.0, 50.0, 150.0, 350.0):
            S, T = o.mi_solve(tlab, kind=1, lambdaA=lamA, beta=inp.YAMAGUCHI_BETA, NQ=NQ)
            Sx = _yamaguchi_S_exact(tlab)
            assert abs(abs(Sx) - 1) < 1e-14
            d = 0.5 * math.degrees(math.atan2(S.imag, S.real)); dx = 0.5 * math.degrees(math.atan2(Sx.imag, Sx.real))
            assert abs(d - dx) < 1e-9, (NQ, tlab, d, dx)
    # SURVEY C15 probe values of the exact phase: 63.3159 / 45.8472 / 14.9765 deg at 1 / 50 / 350 MeV
    for tlab, ref in ((1.0, 63.3159), (50.0, 45.8472), (350.0, 14.9765)):
        Sx = _yamaguchi_S_exact(tlab)
        assert abs(0.5 * math.degrees(math.atan2(Sx.imag, Sx.real)) - ref) < 1e-3
    # effective-range expansion: p cot(delta) -> -1/a as p -> 0
    tl = 1e-4
    Sx = _yamaguchi_S_exact(tl); p = math.sqrt(inp.MU * tl) / inp.HBARC
    dl = 0.5 * math.atan2(Sx.imag, Sx.real)
    assert abs(p / math.tan(dl) + 1 / inp.YAMAGUCHI_A) < 1e-5


def test_mi_unitarity_P5():
    for l in (0, 1, 2):
        for tlab in (1.0, 100.0, 350.0):
            S, T = o.mi_solve(tlab, V0=inp.MT_V0, mu=inp.MT_MU, l_or_J=l)
            assert abs(abs(S) - 1) < 1e-12
    for J in (1, 2, 4):
        for tlab in (5.0, 200.0):
            S, T = o.mi_solve(tlab, coupled=True, l_or_J=J, V0=inp.MT_V0, mu=inp.MT_MU, VT=inp.TENSOR_V, muT=inp.TENSOR_MU)
            assert np.abs(S @ S.conj().T - np.eye(2)).max() < 1e-12
            assert abs(S[0, 1] - S[1, 0]) < 1e-12


# ---------------------------------------------------------------- whole chain: P9 and WPCD -> MI
def _wpcd_phases(N, l=0, nE=11):
    p, e0, dE, Ee, H, V = _mt_H(N, l)
    W, C, _ = o.jacobi(H)
    tl = np.linspace(1, 350, nE)
    T, b = o.onshell_T(N, False, Ee, V, W, C, tl / 2)
    d, S = o.phase_shifts(False, T, b, dE)
    return tl, d, W


def _dist180(a, b):
    d = (a - b + 90.0) % 180.0 - 90.0
    return np.abs(d)


def test_bound_state_P9_and_convergence_to_MI():
    tl = np.linspace(1, 350, 11)
    mi = np.array([0.5 * math.degrees(np.angle(o.mi_solve(t, V0=inp.MT_V0, mu=inp.MT_MU)[0])) for t in tl])
    errs, eb = [], []
    for N in (50, 100, 200):
        _, d, W = _wpcd_phases(N)
        assert (W < 0).sum() == 1
        eb.append(W[0])
        errs.append(np.median(_dist180(d, mi)))
    # SURVEY P9 probe: -2.19 / -2.22 / -2.228 MeV
    assert abs(eb[0] + 2.19) < 0.01 and abs(eb[1] + 2.22) < 0.01 and abs(eb[2] + 2.228) < 0.002
    assert errs[0] > errs[1] > errs[2] and errs[2] < 1.0, errs


def test_wpcd_yamaguchi_converges_to_exact():
    lamA, lamB = inp.yamaguchi_lambda()
    tl = np.linspace(1, 350, 25)
    exact = np.array([0.5 * math.degrees(np.angle(_yamaguchi_S_exact(t))) for t in tl])
    errs = []
    for N in (50, 200):
        p = inp.grid_edges(N)
        e0, dE, Ee = o.fwp(p)
        V, G = o.V_yamaguchi(p, lamB, inp.YAMAGUCHI_BETA)
        H, Vf = o.assemble_H(e0, V)
        W, C, _ = o.jacobi(H)
        T, b = o.onshell_T(N, False, Ee, Vf, W, C, tl / 2)
        d, S = o.phase_shifts(False, T, b, dE)
        errs.append(np.median(_dist180(d, exact)))
    assert errs[1] < errs[0] and errs[1] < 1.0, errs


def test_coupled_wpcd_vs_mi():
    # reading C6 (branch assignment) and C8 (coupling): coupled WPCD S-matrix approaches the coupled MI S-matrix
    N, J = 100, 1
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    Vmm = o.V_yukawa(p, J - 1, **MT); Vpp = o.V_yukawa(p, J + 1, **MT)
    Vmp = o.V_yukawa(p, J, [inp.TENSOR_V], [inp.TENSOR_MU])
    H, V = o.assemble_H(e0, Vmm, Vpp, Vmp)
    W, C, _ = o.jacobi(H)
    tl = np.linspace(20, 350, 7)
    T, b = o.onshell_T(N, True, Ee, V, W, C, tl / 2)
    d, S = o.phase_shifts(True, T, b, dE)
    worst = 0.0
    for e, t in enumerate(tl):
        Smi, _ = o.mi_solve(t, coupled=True, l_or_J=J, V0=inp.MT_V0, mu=inp.MT_MU, VT=inp.TENSOR_V, muT=inp.TENSOR_MU)
        worst = max(worst, np.abs(S[e] - Smi).max())
    assert worst < 0.15, worst      # |dS| ~ 2 sin(d delta): a few degrees at N=100


def test_solve_batch_matches_single_calls():
    N = 32
    p, e0, dE, Ee, H, V = _mt_H(N)
    tl, Ecm = inp.energies(20)
    r = o.solve_batch(N, False, Ee, dE, np.stack([H, H]), np.stack([V, V]), Ecm)
    W, C, _ = o.jacobi(H)
    T, b = o.onshell_T(N, False, Ee, V, W, C, Ecm)
    d, S = o.phase_shifts(False, T, b, dE)
    assert np.array_equal(r["W"][1], W) and np.array_equal(r["delta"][0], d) and np.array_equal(r["bin"], b)


# ---------------------------------------------------------------- NEXT-1: energy-averaged resolvent (Eqs. 28, B.7-B.8)
def test_resolvent_avg_vs_quadrature_of_pointwise():
    """Reading G3 (sign of B.8): the averaged resolvent is the bin average of the point-wise one, checked by adaptive
    quadrature of the point-wise real part (integrable log singularities at shared edges) -- not by re-typing W."""
    cases = [(10.0, 11.0, 100.0, 103.0),    # far below the state
             (100.0, 103.0, 10.0, 11.0),    # far above
             (5.0, 7.0, 7.0, 8.5),          # adjacent: shares the edge 7
             (7.0, 8.5, 5.0, 7.0),          # adjacent on the other side
             (5.0, 7.0, 5.0, 7.0),          # the state's own bin
             (0.0, 0.4, 0.4, 1.1),          # first bin starts at 0
             (6.0, 9.0, 7.0, 8.0)]          # averaging bin covers the state's bin (not used by WPCD, still an average)
    for a, b, lo, hi in cases:
        f = lambda E: o.resolvent(E, lo, hi).real
        pts = sorted({x for x in (lo, hi) if a <= x <= b})
        val, err = integrate.quad(f, a, b, points=pts or None, limit=400, epsabs=1e-13, epsrel=1e-13)
        g = o.resolvent_avg(a, b, lo, hi, (a, b) == (lo, hi))
        assert abs(g.real - val / (b - a)) < 5e-10 * max(1.0, abs(g.real)), (a, b, lo, hi, g.real, val / (b - a))
        assert g.imag == (-math.pi / (hi - lo) if (a, b) == (lo, hi) else 0.0)
    # far apart, narrow bins: -> 1/(E - eps) at the bin centres; equal bins a distance L apart give 1/L
    g = o.resolvent_avg(1000.0, 1000.1, 10.0, 10.1, False)
    assert abs(g.real * 990.0 - 1.0) < 1e-6
    g = o.resolvent_avg(10.0, 10.1, 1000.0, 1000.1, False)
    assert abs(g.real * 990.0 + 1.0) < 1e-6
    assert abs(o.resolvent_avg(5.0, 7.0, 5.0, 7.0, True).real) < 1e-15       # own bin: the real part averages to zero


def test_T_avg_tiny_case_by_hand_and_bins():
    """orc_onshell_T_avg on a 3-state toy spectrum: one value per FWP bin, assembled by hand from resolvent_avg."""
    N = 3
    Ee = np.array([0.0, 1.0, 3.0, 7.0])
    rng = np.random.default_rng(5)
    W = np.array([0.6, 2.2, 5.1])
    Cm = np.linalg.qr(rng.standard_normal((3, 3)))[0]
    V = rng.standard_normal((3, 3)); V = V + V.T
    ed = o.swp_edges(W)
    Ecm = np.array([0.2, 0.9, 1.5, 2.9, 6.0, 8.0])
    T, b = o.onshell_T(N, False, Ee, V, W, Cm, Ecm, averaged=True)
    assert list(b) == [0, 0, 1, 1, 2, -1] and T[5] == 0
    assert T[0] == T[1] and T[2] == T[3]                                 # constant over a bin
    VC = V @ Cm
    for e, i in ((0, 0), (2, 1), (4, 2)):
        t = V[i, i] + sum(VC[i, k] ** 2 * o.resolvent_avg(ed[i], ed[i + 1], ed[k], ed[k + 1], k == i) for k in range(3))
        assert abs(T[e] - t) < 1e-13
        assert abs(T[e].imag + math.pi * VC[i, i] ** 2 / (ed[i + 1] - ed[i])) < 1e-13
    # a bound state is averaged as ln|(b - eps)/(a - eps)|/(b - a): against quadrature of 1/(E - eps)
    W2 = np.array([-1.5, 2.2, 5.1])
    T2, _ = o.onshell_T(N, False, Ee, V, W2, Cm, Ecm[:1], averaged=True)
    ed2 = o.swp_edges(W2[1:])
    gb = integrate.quad(lambda E: 1 / (E + 1.5), ed2[0], ed2[1])[0] / (ed2[1] - ed2[0])
    t = V[0, 0] + VC[0, 0] ** 2 * gb + sum(VC[0, k] ** 2 * o.resolvent_avg(ed2[0], ed2[1], ed2[k - 1], ed2[k], k == 1)
                                            for k in (1, 2))
    assert abs(T2[0] - t) < 1e-12


def test_wpcd_avg_yamaguchi_converges_monotonically():
    """with the energy-averaged resolvent the phase at the bin mid-points converges smoothly to the
    closed form (survey probe: max error 0.86 deg at N=50 -> 0.14 deg at N=400); the point-wise variant does not."""
    lamA, lamB = inp.yamaguchi_lambda()
    cE = inp.HBARC ** 2 / (2 * inp.MU)
    errs = []
    for N in (50, 100, 200):
        p = inp.grid_edges(N)
        e0, dE, Ee = o.fwp(p)
        V, G = o.V_yamaguchi(p, lamB, inp.YAMAGUCHI_BETA)
        H, Vf = o.assemble_H(e0, V)
        W, C, _ = o.jacobi(H)
        qm = 0.5 * (p[:-1] + p[1:])
        Em = cE * qm ** 2                                   # c.m. energy at the bin mid-points (Eq. 42's q-bar)
        sel = (2 * Em >= 1.0) & (2 * Em <= 350.0)
        T, b = o.onshell_T(N, False, Ee, Vf, W, C, Em[sel], averaged=True)
        d, S = o.phase_shifts(False, T, b, dE)
        exact = np.array([0.5 * math.degrees(np.angle(_yamaguchi_S_exact(2 * E))) for E in Em[sel]])
        errs.append(_dist180(d, exact).max())
    assert errs[0] > errs[1] > errs[2] and errs[0] < 1.5 and errs[2] < 0.4, errs


# ---------------------------------------------------------------- NEXT-1: mid-point interpolation (Eqs. 42-43)
def test_interp_phases_lines_wraps_and_mixing_sign():
    p = np.array([0.0, 0.5, 1.2, 2.0, 3.5, 5.0])
    qm = 0.5 * (p[:-1] + p[1:])
    q = np.array([0.05, 0.3, 0.9, 1.9, 2.0, 3.4, 4.99])
    # (1) a straight line in q is reproduced exactly (interpolation and the printed extrapolation in the upper half bin)
    assert np.allclose(o.interp_phases(p, 12.0 - 7.0 * qm, q), 12.0 - 7.0 * q, atol=1e-12)
    assert np.isnan(o.interp_phases(p, qm, np.array([5.0, -0.1]))).all()           # outside the grid
    # (2) Eq. 42 by hand for q in bin 2 (0-based): line through the mid-points of bins 1 and 2
    d = np.array([3.0, -20.0, 35.0, 40.0, 10.0])
    want = d[1] + (d[2] - d[1]) / (qm[2] - qm[1]) * (1.9 - qm[1])
    assert abs(o.interp_phases(p, d, np.array([1.9]))[0] - want) < 1e-12
    want0 = d[0] + (d[1] - d[0]) / (qm[1] - qm[0]) * (0.05 - qm[0])                 # bin 0 uses bins 0 and 1 (reading I1)
    assert abs(o.interp_phases(p, d, np.array([0.05]))[0] - want0) < 1e-12
    # (3) a 180-degree branch jump of the principal value is not interpolated across (reading I2):
    true = 150.0 - 40.0 * qm                                                         # smooth, crosses +90 and -90... wrapped:
    wrapped = (true + 90.0) % 180.0 - 90.0
    got = o.interp_phases(p, wrapped, q)
    exact = ((150.0 - 40.0 * q) + 90.0) % 180.0 - 90.0
    assert np.allclose((got - exact + 90.0) % 180.0 - 90.0, 0.0, atol=1e-10)
    assert np.all((got > -90.0) & (got <= 90.0))
    # (4) coupled: eps_J flips sign with every odd 180-degree shift of delta_- or delta_+ (Eq. A.5)
    dm = (80.0 + 30.0 * qm + 90.0) % 180.0 - 90.0                                    # delta_- wraps once along the grid
    dp = 5.0 + 0.0 * qm
    eps_true = 2.0 + 0.5 * qm
    k = np.round((80.0 + 30.0 * qm - dm) / 180.0).astype(int)
    k = k - k[0]                                                                     # shifts relative to the first bin
    eps_given = np.where(k % 2 == 1, -eps_true, eps_true)
    out = o.interp_phases(p, np.stack([dm, dp, eps_given], axis=1), q)
    assert np.allclose(out[:, 2], eps_true[0] / eps_true[0] * (2.0 + 0.5 * q), atol=1e-10)
    assert np.allclose(out[:, 1], 5.0, atol=1e-12)


def test_interp_phases_yamaguchi_beats_the_steps():
    """Fig. 5 / PAPER.md:385: mid-point interpolation of the energy-averaged phases is close to the exact result at ANY
    energy, closer than the step-like bin values (whose error adds the half-bin variation of the phase)."""
    lamA, lamB = inp.yamaguchi_lambda()
    cE = inp.HBARC ** 2 / (2 * inp.MU)
    tl = np.linspace(5.0, 350.0, 70)
    q = np.sqrt(tl / 2 / cE)
    exact = np.array([0.5 * math.degrees(np.angle(_yamaguchi_S_exact(t))) for t in tl])
    errs = []
    for N in (50, 100):
        p = inp.grid_edges(N)
        e0, dE, Ee = o.fwp(p)
        V, G = o.V_yamaguchi(p, lamB, inp.YAMAGUCHI_BETA)
        H, Vf = o.assemble_H(e0, V)
        W, C, _ = o.jacobi(H)
        qm = 0.5 * (p[:-1] + p[1:])
        T, b = o.onshell_T(N, False, Ee, Vf, W, C, cE * qm ** 2, averaged=True)
        dmid, _ = o.phase_shifts(False, T, b, dE)
        Ts, bs = o.onshell_T(N, False, Ee, Vf, W, C, tl / 2, averaged=True)
        dstep, _ = o.phase_shifts(False, Ts, bs, dE)
        e_int = _dist180(o.interp_phases(p, dmid, q), exact).max()
        e_step = _dist180(dstep, exact).max()
        assert e_int < 0.9 * e_step, (N, e_int, e_step)
        errs.append(e_int)
    assert errs[1] < errs[0] < 1.5, errs


# ---------------------------------------------------------------- NEXT-2: total cross section (Eqs. A.2, A.9, A.11)
def _random_unitary_pw(rng, Jmax=3):
    """Unitary partial-wave S-matrices built from random angles: uncoupled e^{2i delta} (Eq. A.5), coupled Stapp (A.4)."""
    pw = []
    for (s, l, J) in [(0, 0, 0), (1, 1, 0), (0, 1, 1), (1, 1, 1), (0, 2, 2), (1, 2, 2), (0, 3, 3), (1, 3, 3)]:
        if J <= Jmax:
            pw.append((s, J, l, l, np.exp(2j * rng.uniform(-1.2, 1.2))))
    for J in range(1, Jmax + 1):
        dm, dp, ep = rng.uniform(-1.2, 1.2), rng.uniform(-1.2, 1.2), rng.uniform(-0.4, 0.4)
        off = 1j * math.sin(2 * ep) * np.exp(1j * (dm + dp))
        pw += [(1, J, J - 1, J - 1, math.cos(2 * ep) * np.exp(2j * dm)), (1, J, J + 1, J + 1, math.cos(2 * ep) * np.exp(2j * dp)),
               (1, J, J - 1, J + 1, off), (1, J, J + 1, J - 1, off)]
    return pw


def test_clebsch_gordan_vs_sympy_and_orthogonality():
    from sympy import S as Sy
    from sympy.physics.quantum.cg import CG
    for j1 in range(0, 6):
        for j2 in (0, 1):
            for J in range(abs(j1 - j2), j1 + j2 + 1):
                for m1 in range(-j1, j1 + 1):
                    for m2 in range(-j2, j2 + 1):
                        M = m1 + m2
                        if abs(M) > J:
                            continue
                        ref = float(CG(Sy(j1), Sy(m1), Sy(j2), Sy(m2), Sy(J), Sy(M)).doit())
                        assert abs(o.clebsch_gordan(j1, m1, j2, m2, J, M) - ref) < 1e-14
    # orthogonality: sum_{m1 m2} <j1 m1 j2 m2|J M><j1 m1 j2 m2|J' M> = delta_JJ'
    for J in (2, 3, 4):
        for Jp in (2, 3, 4):
            t = sum(o.clebsch_gordan(3, m1, 1, m2, J, 1) * o.clebsch_gordan(3, m1, 1, m2, Jp, 1)
                    for m1 in range(-3, 4) for m2 in (-1, 0, 1))
            assert abs(t - (1.0 if J == Jp else 0.0)) < 1e-14
    assert o.clebsch_gordan(1, 1, 1, 1, 1, 1) == 0.0 and o.clebsch_gordan(2, 0, 1, 0, 4, 0) == 0.0


def test_sph_harm_vs_scipy():
    from scipy.special import sph_harm_y
    for l in range(0, 7):
        for m in range(-l, l + 1):
            for th in (0.0, 0.3, 1.1, math.pi / 2, 2.9, math.pi):
                ref = complex(sph_harm_y(l, m, th, 0.0))
                assert abs(ref.imag) < 1e-15 and abs(o.sph_harm(l, m, th) - ref.real) < 1e-13


def test_sigma_tot_single_wave_closed_forms():
    # only 1S0: spin weight 1/4 of 4 pi sin^2(delta)/p^2;  only 3P0 (J = 0): the same weight 2J+1 = 1
    p, d = 0.9, 0.7
    ref = 10.0 * math.pi * math.sin(d) ** 2 / p ** 2
    assert abs(o.sigma_tot([(0, 0, 0, 0, np.exp(2j * d))], p) - ref) < 1e-13 * ref
    assert abs(o.sigma_tot([(1, 0, 1, 1, np.exp(2j * d))], p) - ref) < 1e-13 * ref
    # 3P1 alone: weight 2J+1 = 3;  S = 1 everywhere: nothing scatters
    assert abs(o.sigma_tot([(1, 1, 1, 1, np.exp(2j * d))], p) - 3 * ref) < 1e-13 * ref
    assert o.sigma_tot([(0, 0, 0, 0, 1.0), (1, 1, 1, 1, 1.0)], p) == 0.0
    # 1S0 alone is isotropic: M^0_00 = e^{i delta} sin(delta)/p at every angle
    for th in (0.0, 1.0, 2.5):
        M = o.spin_scattering_M([(0, 0, 0, 0, np.exp(2j * d))], p, th)
        assert abs(M[(0, 0, 0)] - np.exp(1j * d) * math.sin(d) / p) < 1e-15


def test_sigma_tot_partial_wave_sum_and_optical_theorem():
    """(2 pi/p) Im(a+b) equals the partial-wave sum (pi/2p^2) sum (2J+1) Re(1 - S_ll) for ANY S (the off-diagonal
    elements drop out of the spin trace), and, for unitary S, the angular integral of the unpolarised differential
    cross section (1/4) Tr(M M^dagger) of Eq. A.6 (optical theorem) -- which checks Y, the Clebsch-Gordan coefficients,
    the sqrt((2l+1)/4pi) and 2pi/(ip) factors of Eq. A.2 and the weights of Eqs. A.9/A.11 all at once."""
    rng = np.random.default_rng(5)
    x, w = np.polynomial.legendre.leggauss(24)
    for trial in range(3):
        pw = _random_unitary_pw(rng)
        p = rng.uniform(0.3, 2.0)
        sig = o.sigma_tot(pw, p)
        closed = 10.0 * math.pi / (2 * p * p) * sum((2 * J + 1) * (1 - complex(Sv).real) for (s, J, lp, l, Sv) in pw if lp == l)
        assert abs(sig - closed) < 1e-13 * abs(closed)
        integral = 0.0
        for xi, wi in zip(x, w):
            M = o.spin_scattering_M(pw, p, math.acos(xi))
            integral += 2 * math.pi * wi * 0.25 * sum(abs(v) ** 2 for v in M.values())
        assert abs(10.0 * integral - sig) < 1e-12 * sig
    # non-unitary S (as WPCD produces): the partial-wave sum still holds, off-diagonal elements do not contribute
    pw = [(s, J, lp, l, Sv * rng.uniform(0.9, 1.05)) for (s, J, lp, l, Sv) in _random_unitary_pw(rng)]
    closed = 10.0 * math.pi / (2 * 0.8 ** 2) * sum((2 * J + 1) * (1 - complex(Sv).real) for (s, J, lp, l, Sv) in pw if lp == l)
    assert abs(o.sigma_tot(pw, 0.8) - closed) < 1e-13 * abs(closed)


def test_sigma_tot_yamaguchi_1S0_against_closed_form_phase():
    """1S0 only, separable Yamaguchi potential: sigma_tot from the MI S-matrix equals pi sin^2(delta)/p^2 with the
    analytic phase shift (reading C15)."""
    lamA, _ = inp.yamaguchi_lambda()
    for tlab in (10.0, 100.0, 300.0):
        p = math.sqrt(inp.MU * tlab) / inp.HBARC
        Sx = _yamaguchi_S_exact(tlab)
        d = 0.5 * math.atan2(Sx.imag, Sx.real)
        S, _ = o.mi_solve(tlab, kind=1, lambdaA=lamA, beta=inp.YAMAGUCHI_BETA, NQ=96)
        ref = 10.0 * math.pi * math.sin(d) ** 2 / p ** 2
        assert abs(o.sigma_tot([(0, 0, 0, 0, S)], p) - ref) < 1e-9 * ref


def test_sigma_tot_wpcd_converges_to_MI():
    """Shape of PAPER.md:389-405 (Figs. 6-7) on the synthetic potential: the WPCD total cross section of all 14
    channels approaches the MI ("exact") one as the number of wave packets grows; method error of a few mb."""
    names = [c[0] for c in inp.CHANNELS_J4]; channels = [(c[1], c[2]) for c in inp.CHANNELS_J4]
    sJ = [inp.channel_sJ(nm) for nm in names]
    tl = np.linspace(5.0, 345.0, 18); Ecm = tl / 2
    exact = []
    for t in tl:
        Su = [o.mi_solve(t, V0=inp.MT_V0, mu=inp.MT_MU, l_or_J=lJ, NQ=64)[0] for (k, lJ) in channels if not k]
        Sc = [o.mi_solve(t, coupled=True, V0=inp.MT_V0, mu=inp.MT_MU, l_or_J=lJ, VT=inp.TENSOR_V, muT=inp.TENSOR_MU, NQ=64)[0]
              for (k, lJ) in channels if k]
        exact.append(o.sigma_tot(o.partial_waves(channels, sJ, Su, Sc), math.sqrt(inp.MU * t) / inp.HBARC))
    exact = np.array(exact)
    assert 1500 < exact[0] < 1800 and 50 < exact[-1] < 60 and (np.diff(exact) < 0).all()   # np-like: falls with energy
    mean_err = {}
    for N in (32, 64):
        p = inp.grid_edges(N); e0, dE, Ee = o.fwp(p)
        S_unc, S_cpl = [], []
        for (k, lJ) in channels:
            if not k:
                H, V = o.assemble_H(e0, o.V_yukawa(p, lJ, inp.MT_V0, inp.MT_MU))
            else:
                H, V = o.assemble_H(e0, o.V_yukawa(p, lJ - 1, inp.MT_V0, inp.MT_MU), o.V_yukawa(p, lJ + 1, inp.MT_V0, inp.MT_MU),
                                    o.V_yukawa(p, lJ, [inp.TENSOR_V], [inp.TENSOR_MU]))
            W, Cm, _ = o.jacobi(H)
            T, b = o.onshell_T(N, k, Ee, V, W, Cm, Ecm)
            _, S = o.phase_shifts(k, T, b, dE)
            (S_cpl if k else S_unc).append(S)
        sig = np.array([o.sigma_tot(o.partial_waves(channels, sJ, [S[e] for S in S_unc], [S[e] for S in S_cpl]),
                                    math.sqrt(2 * inp.MU * Ecm[e]) / inp.HBARC) for e in range(len(Ecm))])
        err = np.abs(sig - exact)
        mean_err[N] = err.mean()
        assert np.median(err) < (2.0 if N == 32 else 1.0), (N, np.median(err))
    assert mean_err[64] < 0.7 * mean_err[32], mean_err


# ---------------------------------------------------------------- NEXT-3: the paper's own discretisation (Eqs. 30-31)
def test_chebyshev_grid_eq31():
    N = 32
    p = o.grid_chebyshev(N)                       # t = 2, alpha = 100 MeV
    assert p[0] == 0.0 and (np.diff(p) > 0).all()
    assert np.abs(p - inp.grid_chebyshev(N)).max() < 1e-13 * p[-1]
    a = 100.0 / inp.HBARC
    # hand values: j = 1 and the middle point j = (N+1)/2 -> tan(pi/4 + pi/(4N)...) ; t = 1 reduces to a plain tan grid
    assert abs(p[1] - a * math.tan(math.pi / 128) ** 2) < 1e-16
    assert abs(p[N] - a / math.tan(math.pi / 128) ** 2) < 1e-9 * p[N]      # tan(pi/2 - x) = 1/tan(x)
    # symmetry of Eq. 31 about alpha: y_j y_{N+1-j} = alpha^2 for t-th powers of tan(x) tan(pi/2 - x) = 1
    assert np.allclose(p[1:] * p[1:][::-1], a * a, rtol=1e-12)
    p1 = o.grid_chebyshev(8, t=1.0, alpha=2.5)
    assert np.allclose(p1[1:], 2.5 * np.tan((2 * np.arange(1, 9) - 1) * np.pi / 32), rtol=1e-14)


def test_midpoint_potential_eq30_is_the_one_point_rule():
    """Eq. 30: <x_i|v|x_j> ~ kbar_i kbar_j sqrt(Dk_i Dk_j) <kbar_i|v|kbar_j> with the convention-B
    element <k'|v_l|k> = (1/pi) sum_t V0_t Q_l(z_t)/(k'k).  The n_gl = 1 Gauss-Legendre rule of Eq. 29 is exactly that."""
    p = o.grid_chebyshev(12)
    for l in (0, 2):
        V = o.V_yukawa(p, l, inp.MT_V0, inp.MT_MU, ngl=1)
        kb = 0.5 * (p[:-1] + p[1:]); dk = np.diff(p)
        ref = np.empty_like(V)
        for i in range(12):
            for j in range(12):
                el = sum(V0 * float(mp.legenq(l, 0, (kb[i] ** 2 + kb[j] ** 2 + m ** 2) / (2 * kb[i] * kb[j]), type=3).real)
                         for V0, m in zip(inp.MT_V0, inp.MT_MU)) / (math.pi * kb[i] * kb[j])
                ref[i, j] = kb[i] * kb[j] * math.sqrt(dk[i] * dk[j]) * el
        assert np.abs(V - ref).max() < 1e-11 * np.abs(ref).max()
    # and it approaches the 8-point bin average where the potential varies mildly over a bin
    pf = inp.grid_edges(60)
    V1, V8 = o.V_yukawa(pf, 0, inp.MT_V0, inp.MT_MU, ngl=1), o.V_yukawa(pf, 0, inp.MT_V0, inp.MT_MU, ngl=8)
    assert np.abs(V1 - V8)[:30, :30].max() < 2e-3 * np.abs(V8)[:30, :30].max()


def test_chebyshev_grid_chain_converges_to_MI():
    """The paper's set-up (Chebyshev momentum bins, t = 2, alpha = 100 MeV) on the synthetic 1S0 potential: phase shifts
    approach MI as N_WP grows over the paper's range 16..96, with Eq. 29 and with Eq. 30."""
    tl = np.linspace(10.0, 340.0, 12); Ecm = tl / 2
    exact = np.array([0.5 * math.degrees(math.atan2(S.imag, S.real)) for S in
                      (o.mi_solve(t, V0=inp.MT_V0, mu=inp.MT_MU, l_or_J=0, NQ=96)[0] for t in tl)])
    for ngl in (8, 1):
        med = {}
        for N in (16, 32, 96):
            p = o.grid_chebyshev(N); e0, dE, Ee = o.fwp(p)
            H, V = o.assemble_H(e0, o.V_yukawa(p, 0, inp.MT_V0, inp.MT_MU, ngl=ngl))
            W, Cm, _ = o.jacobi(H)
            T, b = o.onshell_T(N, 0, Ee, V, W, Cm, Ecm, averaged=True)
            d, _ = o.phase_shifts(0, T, b, dE)
            err = np.abs((d - exact + 90.0) % 180.0 - 90.0)
            med[N] = np.median(err)
        assert med[96] < med[32] < med[16] and med[96] < 2.0, (ngl, med)


# ---------------------------------------------------------------- NEXT-4: energy wave packets (Eqs. 17-18)
def test_energy_packets_h0_and_potential_vs_adaptive_integrals():
    p = np.array([0.4, 0.9, 1.5, 2.4])
    cE = inp.HBARC ** 2 / (2 * inp.MU)
    e0, dE, Ee = o.fwp(p, energy_packets=True)
    f = lambda k: inp.HBARC * math.sqrt(k / inp.MU)          # weighting function of the energy packets
    for i in range(3):
        # normalisation N_i = dE_i:  int k dk f(k) int k' dk' f(k') delta(k-k')/(k k') = int f^2 dk
        nrm, _ = integrate.quad(lambda k: f(k) ** 2, p[i], p[i + 1])
        assert abs(nrm - dE[i]) < 1e-12 * dE[i]
        # Eq. 18: <x_i|h0|x_i> = (1/N_i) int f^2 cE k^2 dk = E_i + dE_i/2
        val, _ = integrate.quad(lambda k: f(k) ** 2 * cE * k * k, p[i], p[i + 1])
        assert abs(e0[i] - val / dE[i]) < 1e-12 * e0[i] and abs(e0[i] - (Ee[i] + 0.5 * dE[i])) < 1e-13 * e0[i]
    for l in (0, 2):
        V = o.V_yukawa(p, l, energy_packets=True, **MT)
        assert np.array_equal(V, V.T)
        for i, j in [(0, 0), (0, 2), (1, 2)]:
            def integrand(k, kp):     # k'k f(k')f(k) <k'|v_l|k>_B
                s = sum(V0 * float(mp.legenq(l, 0, (kp * kp + k * k + mu * mu) / (2 * kp * k), type=3).real)
                        for V0, mu in zip(inp.MT_V0, inp.MT_MU))
                return f(kp) * f(k) * s / math.pi
            val, _ = integrate.dblquad(integrand, p[i], p[i + 1], p[j], p[j + 1], epsabs=1e-10, epsrel=1e-10)
            ref = val / math.sqrt(dE[i] * dE[j])
            assert abs(V[i, j] - ref) < 2e-6 * abs(ref), (l, i, j, V[i, j], ref)
    # Yamaguchi form factor G_i = dE_i^{-1/2} int k f(k) g(k) dk
    lamA, lamB = inp.yamaguchi_lambda()
    V, G = o.V_yamaguchi_energy(p, lamB, inp.YAMAGUCHI_BETA)
    for i in range(3):
        val, _ = integrate.quad(lambda k: k * f(k) / (k * k + inp.YAMAGUCHI_BETA ** 2), p[i], p[i + 1])
        assert abs(G[i] - val / math.sqrt(dE[i])) < 1e-10 * abs(G[i])
    assert np.allclose(V, -lamB * np.outer(G, G), rtol=1e-15)


def test_energy_packets_chain_agrees_with_momentum_packets_and_MI():
    """"we have implemented energy as well as momentum wave-packets, and have found no significant
    difference": the two bases give the same narrow-bin matrix elements, phase shifts that differ by less than the
    method error, and both approach MI / the Yamaguchi closed form as N grows."""
    p = inp.grid_edges(60)
    Vk = o.V_yukawa(p, 0, **MT); Ve = o.V_yukawa(p, 0, energy_packets=True, **MT)
    assert np.abs(Vk - Ve)[8:30, 8:30].max() < 5e-4 * np.abs(Vk)[8:30, 8:30].max()
    tl = np.linspace(10.0, 340.0, 12); Ecm = tl / 2
    lamA, lamB = inp.yamaguchi_lambda()
    exact = np.array([0.5 * math.degrees(math.atan2(S.imag, S.real)) for S in map(_yamaguchi_S_exact, tl)])
    med = {}
    for N in (50, 200):
        p = inp.grid_edges(N)
        d = {}
        for ep in (False, True):
            e0, dE, Ee = o.fwp(p, energy_packets=ep)
            V = o.V_yamaguchi_energy(p, lamB, inp.YAMAGUCHI_BETA)[0] if ep else o.V_yamaguchi(p, lamB, inp.YAMAGUCHI_BETA)[0]
            H, Vf = o.assemble_H(e0, V)
            W, Cm, _ = o.jacobi(H)
            T, b = o.onshell_T(N, 0, Ee, Vf, W, Cm, Ecm, averaged=True)
            d[ep], _ = o.phase_shifts(0, T, b, dE)
        err = {ep: np.abs((d[ep] - exact + 90.0) % 180.0 - 90.0) for ep in d}
        med[N] = np.median(err[True])
        # no significant difference: the two bases differ by less than either differs from the exact result
        assert np.abs((d[True] - d[False] + 90.0) % 180.0 - 90.0).max() < max(err[True].max(), err[False].max())
    assert med[200] < 0.5 * med[50] and med[200] < 0.3, med


def test_descending_diagonal_order_converges_faster_on_graded_H():
    """Why wpcd_diag_batched relabels rows/columns by descending diagonal: on the graded WPCD
    Hamiltonians the oracle's own cyclic Jacobi needs one to two sweeps fewer in that order than in the natural ascending
    one, with the same eigenvalues (a pure relabelling)."""
    from tests import helpers as hp
    for kind, lJ in ((0, 0), (1, 1)):
        ch = hp.oracle_channel(60, kind, lJ, (1.02, 0.97, 1.05))
        H = ch["H"]
        W_asc, _, sw_asc = o.jacobi(H)
        perm = np.argsort(-np.diag(H), kind="stable")
        W_desc, C_desc, sw_desc = o.jacobi(H[np.ix_(perm, perm)])
        assert sw_desc < sw_asc, (kind, sw_asc, sw_desc)
        assert np.abs(W_asc - W_desc).max() < 1e-11 * np.abs(W_asc).max()
        assert (np.abs(W_asc - W_desc) / np.abs(W_asc)).max() < 1e-10
        # eigenvector rows go back to their places: H C = C D in the original labelling
        C = np.empty_like(C_desc); C[perm, :] = C_desc
        assert np.abs(H @ C - C * W_desc).max() < 1e-10 * np.abs(H).max()
