"""ctypes front-end of oracle/wpcd_oracle.cpp (argument marshalling only; all arithmetic is in the C++ file).

TEST INFRASTRUCTURE ONLY: shares no code with paper_2106_00454_b200 and is never imported by it.
"""
import ctypes as C
import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())
_d = C.c_double
_i = C.c_int
_pd = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_pi = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_vp = C.c_void_p


def _sig(name, res, args):
    f = getattr(_lib, name)
    f.restype = res
    f.argtypes = args
    return f


_gl = _sig("orc_gl_rule", None, [_i, _pd, _pd])
_Q = _sig("orc_legendre_Q", _d, [_i, _d])
_grid = _sig("orc_grid_tan", None, [_i, _d, _pd])
_gridc = _sig("orc_grid_chebyshev", None, [_i, _d, _d, _pd])
_fwpE = _sig("orc_fwp_energy", None, [_i, _pd, _d, _d, _pd, _pd, _pd])
_VyukE = _sig("orc_V_yukawa_energy", None, [_i, _pd, _i, _i, _pd, _pd, _i, _d, _d, _pd])
_VyamE = _sig("orc_V_yamaguchi_energy", None, [_i, _pd, _d, _d, _i, _d, _d, _pd, _pd])
_fwp = _sig("orc_fwp", None, [_i, _pd, _d, _d, _pd, _pd, _pd])
_Vyuk = _sig("orc_V_yukawa", None, [_i, _pd, _i, _i, _pd, _pd, _i, _pd])
_Vyam = _sig("orc_V_yamaguchi", None, [_i, _pd, _d, _d, _i, _i, _pd, _pd])
_asm = _sig("orc_assemble_H", None, [_i, _i, _pd, _pd, _vp, _vp, _pd, _pd])
_jac = _sig("orc_jacobi", _i, [_i, _pd, _pd, _pd, _d, _i])
_jac_ld = _sig("orc_jacobi_ld", _i, [_i, _pd, _pd, _pd, _d, _i])
_edges = _sig("orc_swp_edges", None, [_i, _pd, _pd])
_res = _sig("orc_resolvent_c", None, [_d, _d, _d, _pd])
_onT = _sig("orc_onshell_T", None, [_i, _i, _pd, _pd, _pd, _pd, _pd, _i, _pd, _pi])
_onTavg = _sig("orc_onshell_T_avg", None, [_i, _i, _pd, _pd, _pd, _pd, _pd, _i, _pd, _pi])
_interp = _sig("orc_interp_phases", None, [_i, _i, _pd, _pd, _pd, _i, _pd])
_resavg = _sig("orc_resolvent_avg_c", None, [C.c_double, C.c_double, C.c_double, C.c_double, _i, _pd])
_ph = _sig("orc_phase_shifts", None, [_i, _i, _pd, _pi, _pd, _pd, _vp])
_migrid = _sig("orc_mi_grid", None, [_i, _d, _pd, _pd])
_mi = _sig("orc_mi_solve", None, [_i, _i, _i, _i, _pd, _pd, _d, _d, _d, _d, _d, _d, _i, _d, _pd, _pd])
_batch = _sig("orc_solve_batch", _i, [_i, _i, _i, _pd, _pd, _pd, _pd, _pd, _i, _d, _i, _pd, _pd, _pd, _pi, _pd, _vp, _vp])
_nthr = _sig("orc_num_threads", _i, [])
_cg = _sig("orc_clebsch_gordan", _d, [_i, _i, _i, _i, _i, _i])
_ylm = _sig("orc_sph_harm", _d, [_i, _i, _d])
_Mspin = _sig("orc_spin_scattering_M", None, [_i, _pi, _pi, _pi, _pi, _pd, _d, _d, _pd])
_sigtot = _sig("orc_sigma_tot", _d, [_i, _pi, _pi, _pi, _pi, _pd, _d])

HBARC = 197.327
MU = 469.46


def _f(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads():
    return int(_nthr())


def gl_rule(n):
    x = np.empty(n); w = np.empty(n)
    _gl(n, x, w)
    return x, w


def legendre_Q(l, z):
    return float(_Q(int(l), float(z)))


def grid_tan(N, alpha=1.0):
    p = np.empty(N + 1)
    _grid(N, alpha, p)
    return p


def grid_chebyshev(N, t=2.0, alpha=100.0 / HBARC):
    """Eq. 31: y_0 = 0, y_j = alpha tan^t((2j-1) pi/(4N)); defaults are the paper's (t = 2, alpha = 100 MeV)."""
    p = np.empty(N + 1)
    _gridc(N, t, alpha, p)
    return p


def fwp(p, hbarc=HBARC, mu=MU, energy_packets=False):
    """FWP kinetic energies, bin energy widths and energy edges; energy_packets: f = sqrt(k/mu), N_i = dE_i (Eq. 18)."""
    p = _f(p); N = len(p) - 1
    e0 = np.empty(N); dE = np.empty(N); Ee = np.empty(N + 1)
    (_fwpE if energy_packets else _fwp)(N, p, hbarc, mu, e0, dE, Ee)
    return e0, dE, Ee


def V_yukawa(p, l, V0, mu, ngl=8, energy_packets=False, hbarc=HBARC, mured=MU):
    p = _f(p); N = len(p) - 1
    V0 = _f(np.atleast_1d(V0)); mu = _f(np.atleast_1d(mu))
    V = np.empty((N, N))
    if energy_packets:
        _VyukE(N, p, int(l), len(V0), V0, mu, ngl, hbarc, mured, V)
    else:
        _Vyuk(N, p, int(l), len(V0), V0, mu, ngl, V)
    return V


def V_yamaguchi_energy(p, lambdaB, beta, ngl=8, hbarc=HBARC, mured=MU):
    p = _f(p); N = len(p) - 1
    V = np.empty((N, N)); G = np.empty(N)
    _VyamE(N, p, lambdaB, beta, ngl, hbarc, mured, V, G)
    return V, G


def V_yamaguchi(p, lambdaB, beta, ngl=8, closed_form=True):
    p = _f(p); N = len(p) - 1
    V = np.empty((N, N)); G = np.empty(N)
    _Vyam(N, p, lambdaB, beta, ngl, 1 if closed_form else 0, V, G)
    return V, G


def assemble_H(e0, Vmm, Vpp=None, Vmp=None):
    e0 = _f(e0); N = len(e0)
    coupled = Vpp is not None
    n = 2 * N if coupled else N
    H = np.empty((n, n)); V = np.empty((n, n))
    Vmm = _f(Vmm)
    if coupled:
        Vpp = _f(Vpp); Vmp = _f(Vmp)
        _asm(N, 1, e0, Vmm, Vpp.ctypes.data, Vmp.ctypes.data, H, V)
    else:
        _asm(N, 0, e0, Vmm, None, None, H, V)
    return H, V


def jacobi(A, tol=1e-15, max_sweeps=60):
    A = _f(A); n = A.shape[0]
    W = np.empty(n); Cm = np.empty((n, n))
    sw = _jac(n, A, W, Cm, tol, max_sweeps)
    return W, Cm, sw


def jacobi_ld(A, tol=1e-18, max_sweeps=60):
    """Same algorithm in 80-bit extended precision (pin for the fp64 oracle; results rounded to fp64)."""
    A = _f(A); n = A.shape[0]
    W = np.empty(n); Cm = np.empty((n, n))
    sw = _jac_ld(n, A, W, Cm, tol, max_sweeps)
    return W, Cm, sw


def swp_edges(eps):
    eps = _f(eps); m = len(eps)
    e = np.empty(m + 1)
    _edges(m, eps, e)
    return e


def resolvent(E, lo, hi):
    o = np.empty(2)
    _res(E, lo, hi, o)
    return complex(o[0], o[1])


def interp_phases(pedge, dmid, q):
    """Eq. 42: phases at momenta q from the mid-point phases dmid [N] or [N][3] (degrees)."""
    pedge = _f(pedge); dmid = _f(dmid); q = _f(q)
    N = len(pedge) - 1; nc = 1 if dmid.ndim == 1 else dmid.shape[1]
    out = np.empty((len(q), nc))
    _interp(N, nc, pedge, dmid, q, len(q), out)
    return out[:, 0] if nc == 1 else out


def resolvent_avg(a, b, lo, hi, same_bin):
    """Average of g(E; lo, hi) over E in [a, b] (Eqs. B.7-B.8, reading G3)."""
    o = np.empty(2)
    _resavg(a, b, lo, hi, 1 if same_bin else 0, o)
    return complex(o[0], o[1])


def onshell_T(N, coupled, Eedge, V, W, Cm, Ecm, averaged=False):
    Ecm = _f(Ecm); nE = len(Ecm); nc = 2 if coupled else 1
    T = np.empty((nE, nc, nc, 2)); b = np.empty(nE, dtype=np.int32)
    (_onTavg if averaged else _onT)(N, 1 if coupled else 0, _f(Eedge), _f(V), _f(W), _f(Cm), Ecm, nE, T, b)
    Tc = T[..., 0] + 1j * T[..., 1]
    return (Tc if coupled else Tc[:, 0, 0]), b


def phase_shifts(coupled, T, bins, dE):
    T = np.asarray(T, dtype=np.complex128); nE = T.shape[0]; nc = 2 if coupled else 1
    Tr = np.empty((nE, nc, nc, 2))
    Tr[..., 0] = T.real.reshape(nE, nc, nc); Tr[..., 1] = T.imag.reshape(nE, nc, nc)
    delta = np.empty((nE, 3) if coupled else (nE,))
    S = np.empty((nE, nc, nc, 2))
    _ph(1 if coupled else 0, nE, Tr, np.ascontiguousarray(bins, dtype=np.int32), _f(dE), delta, S.ctypes.data)
    Sc = S[..., 0] + 1j * S[..., 1]
    return delta, (Sc if coupled else Sc[:, 0, 0])


def mi_grid(NQ, cmap=1.0):
    k = np.empty(NQ); w = np.empty(NQ)
    _migrid(NQ, cmap, k, w)
    return k, w


def mi_solve(Tlab, kind=0, coupled=False, l_or_J=0, V0=(0.0,), mu=(1.0,), VT=0.0, muT=1.0, lambdaA=0.0, beta=1.0,
             NQ=96, hbarc=HBARC, mured=MU):
    V0 = _f(np.atleast_1d(V0)); mu = _f(np.atleast_1d(mu))
    nc = 2 if coupled else 1
    S = np.empty(nc * nc * 2); T = np.empty(nc * nc * 2)
    _mi(kind, 1 if coupled else 0, int(l_or_J), len(V0), V0, mu, VT, muT, lambdaA, beta, hbarc, mured, NQ, float(Tlab), S, T)
    Sc = (S[0::2] + 1j * S[1::2]).reshape(nc, nc)
    Tc = (T[0::2] + 1j * T[1::2]).reshape(nc, nc)
    return (Sc, Tc) if coupled else (Sc[0, 0], Tc[0, 0])


def solve_batch(N, coupled, Eedge, dE, H, V, Ecm, tol=1e-15, max_sweeps=60):
    """Whole chain (diag -> T -> phases) for H[b], V[b]; OpenMP over b.  Returns dict."""
    H = _f(H); V = _f(V); Ecm = _f(Ecm)
    batch = H.shape[0]; n = H.shape[1]; nE = len(Ecm); nc = 2 if coupled else 1
    W = np.empty((batch, n)); Cm = np.empty((batch, n, n)); T = np.empty((batch, nE, nc, nc, 2))
    b = np.empty(nE, dtype=np.int32)
    delta = np.empty((batch, nE, 3) if coupled else (batch, nE)); S = np.empty((batch, nE, nc, nc, 2))
    sw = np.empty(batch, dtype=np.int32)
    r = _batch(N, 1 if coupled else 0, batch, _f(Eedge), _f(dE), H, V, Ecm, nE, tol, max_sweeps, W, Cm, T, b, delta,
               S.ctypes.data, sw.ctypes.data)
    Tc = T[..., 0] + 1j * T[..., 1]; Sc = S[..., 0] + 1j * S[..., 1]
    if not coupled:
        Tc = Tc[:, :, 0, 0]; Sc = Sc[:, :, 0, 0]
    return dict(W=W, C=Cm, T=Tc, S=Sc, bin=b, delta=delta, sweeps=sw, worst=r)


def clebsch_gordan(j1, m1, j2, m2, J, M):
    return float(_cg(j1, m1, j2, m2, J, M))


def sph_harm(l, m, theta):
    return float(_ylm(l, m, float(theta)))


def _pw_arrays(pw):
    """pw: list of (s, J, l', l, S_{l'l}) -> int32 arrays and [npw][2] doubles."""
    i32 = lambda k: np.ascontiguousarray([w[k] for w in pw], dtype=np.int32)
    Sv = np.empty((len(pw), 2))
    Sv[:, 0] = [complex(w[4]).real for w in pw]; Sv[:, 1] = [complex(w[4]).imag for w in pw]
    return len(pw), i32(0), i32(1), i32(2), i32(3), Sv


def spin_scattering_M(pw, p, theta):
    """Eq. A.2: dict {(s, m_s, m_s'): M} for the partial waves pw = [(s, J, l', l, S_{l'l}), ...]."""
    n, s, J, lp, l, Sv = _pw_arrays(pw)
    M = np.empty((2, 3, 3, 2))
    _Mspin(n, s, J, lp, l, Sv, float(p), float(theta), M)
    Mc = M[..., 0] + 1j * M[..., 1]
    return {(ss, ms, msp): Mc[ss, ms + 1, msp + 1] for ss in (0, 1) for ms in range(-ss, ss + 1) for msp in range(-ss, ss + 1)}


def sigma_tot(pw, p):
    """Eqs. A.2, A.9, A.11: total np cross section in mb at c.m. momentum p (fm^-1)."""
    n, s, J, lp, l, Sv = _pw_arrays(pw)
    return float(_sigtot(n, s, J, lp, l, Sv, float(p)))


def partial_waves(channels, sJ, S_unc, S_cpl):
    """Partial-wave list for sigma_tot from channel S-matrices at ONE energy (index bookkeeping only).
    channels: [(coupled, lJ)] in list order; sJ: (s, J) of every channel (e.g. 3P0: l = 1, s = 1, J = 0);
    S_unc: complex per uncoupled channel (list order), S_cpl: complex 2x2 per coupled channel (list order)."""
    pw = []; iu = 0; ic = 0
    for (coupled, lJ), (s, J) in zip(channels, sJ):
        if not coupled:
            pw.append((s, J, lJ, lJ, S_unc[iu])); iu += 1
        else:
            ls = (J - 1, J + 1); Sm = np.asarray(S_cpl[ic]); ic += 1
            for a in range(2):
                for b in range(2):
                    pw.append((1, J, ls[a], ls[b], Sm[a, b]))
    return pw
