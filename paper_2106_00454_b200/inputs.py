"""Seeded synthetic inputs of the five BASELINE.json configs.

Holds NONE of the method's arithmetic: only constants, the config grids (bin edges are an *input* of the C ABI),
channel lists, energies and the seeded sample scales.  Both the CUDA path's tests/bench and the CPU oracle's tests
read their inputs from here; neither side's code is imported here.
"""
import numpy as np

HBARC = 197.327          # MeV fm
MU = 469.46              # MeV, reduced mass m_N/2
# Malfliet-Tjon-type two-Yukawa potential V(r) = V_R e^{-mu_R r}/r - V_A e^{-mu_A r}/r  (BASELINE.json config 1)
MT_V0 = np.array([1438.72, -626.885])   # MeV fm  (repulsive, attractive)
MT_MU = np.array([3.11, 1.55])          # fm^-1
TENSOR_V = 200.0         # MeV fm, "tensor-like" coupling l=J-1 <-> J+1 (config 2; reading C8)
TENSOR_MU = 2.0          # fm^-1
YAMAGUCHI_BETA = 1.4488  # fm^-1 (config 4)
YAMAGUCHI_A = -23.7      # fm, 1S0 scattering length


def grid_edges(N, alpha=1.0):
    """Config bin edges p_i = alpha tan(pi i/(2N+1)), i = 0..N, fm^-1 (BASELINE.json config 1)."""
    i = np.arange(N + 1, dtype=np.float64)
    return alpha * np.tan(np.pi * i / (2.0 * N + 1.0))


def grid_chebyshev(N, t=2.0, alpha=100.0 / HBARC):
    """The paper's own bin edges, Eq. 31: y_0 = 0, y_j = alpha tan^t((2j-1) pi/(4N)), j = 1..N, fm^-1;
    defaults t = 2, alpha = 100 MeV (an input of the C ABI like grid_edges)."""
    j = np.arange(1, N + 1, dtype=np.float64)
    return np.concatenate([[0.0], alpha * np.tan((2.0 * j - 1.0) * np.pi / (4.0 * N)) ** t])


def energies(nE):
    """nE lab energies uniform on 1..350 MeV; returns (T_lab, E_cm = T_lab/2)."""
    tlab = np.linspace(1.0, 350.0, nE)
    return tlab, tlab / 2.0


# np channels with J <= 4 (reading C9): (name, coupled, l or J)
CHANNELS_J4 = [
    ("1S0", 0, 0), ("3P0", 0, 1), ("1P1", 0, 1), ("3P1", 0, 1), ("1D2", 0, 2), ("3D2", 0, 2),
    ("1F3", 0, 3), ("3F3", 0, 3), ("1G4", 0, 4), ("3G4", 0, 4),
    ("3S1-3D1", 1, 1), ("3P2-3F2", 1, 2), ("3D3-3G3", 1, 3), ("3F4-3H4", 1, 4),
]


def channel_sJ(name):
    """(s, J) from the spectroscopic name 2s+1 L J of a channel ("3P0" -> (1, 0); "3S1-3D1" -> (1, 1))."""
    first = name.split("-")[0]
    return (int(first[0]) - 1) // 2, int(first[2])


def sample_scales(S, seed=0):
    """[S][3] multiplicative scales (V_R, V_A, V_T) = 1 + 0.1 N(0,1)  (config 3; reading C14)."""
    z = np.random.default_rng(seed).standard_normal((S, 3))
    return 1.0 + 0.1 * z


def yamaguchi_lambda(beta=YAMAGUCHI_BETA, a=YAMAGUCHI_A, hbarc=HBARC, mu=MU):
    """(lambda_A [MeV fm^-1], lambda_B = (2/pi) lambda_A) giving scattering length a (reading C15):
    lambda' = lambda_A mu/hbarc^2 = beta^4/(2 (beta/2 - 1/a))."""
    lam_p = beta ** 4 / (2.0 * (beta / 2.0 - 1.0 / a))
    lam_a = lam_p * hbarc * hbarc / mu
    return lam_a, 2.0 / np.pi * lam_a
