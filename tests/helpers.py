"""Shared helpers of the GPU parity tests: oracle-side references and comparison rules.

The oracle side (oracle.*) and the CUDA side (paper_2106_00454_b200.wpcd) are only ever combined here, in tests.
"""
import numpy as np

from oracle import oracle as o
from paper_2106_00454_b200 import inputs as inp

TOL_EIG_REL = 1e-11      # north_star: eigenvalues to relative error 1e-11 (componentwise, reading C12)
TOL_PHASE_DEG = 1e-8     # north_star: phase shifts to 1e-8 degrees absolute
TOL_S_ABS = 3.5e-10      # |dS| equivalent of 1e-8 deg (reading C10)
TOL_H_REL = 1e-12        # assembly gate: 1e-12 max|H|
EDGE_GUARD = 1e-9        # MeV: energies this close to a pseudostate bin edge are excluded (reading C11)


def oracle_channel(N, coupled, lJ, scale=(1.0, 1.0, 1.0), yamaguchi=None, edges=None, ngl=8, energy_packets=False):
    """Oracle H, V for one channel on the config grid (or the given bin edges).  scale = (V_R, V_A, V_T) multipliers."""
    p = inp.grid_edges(N) if edges is None else np.asarray(edges, dtype=np.float64)
    e0, dE, Ee = o.fwp(p, energy_packets=energy_packets)
    if yamaguchi is not None:
        if energy_packets:
            V, _ = o.V_yamaguchi_energy(p, yamaguchi[0], yamaguchi[1], ngl=ngl)
        else:
            V, _ = o.V_yamaguchi(p, yamaguchi[0], yamaguchi[1], closed_form=True)
        H, Vf = o.assemble_H(e0, V)
    else:
        V0 = inp.MT_V0 * np.array([scale[0], scale[1]])
        if not coupled:
            H, Vf = o.assemble_H(e0, o.V_yukawa(p, lJ, V0, inp.MT_MU, ngl=ngl, energy_packets=energy_packets))
        else:
            Vmm = o.V_yukawa(p, lJ - 1, V0, inp.MT_MU, ngl=ngl, energy_packets=energy_packets)
            Vpp = o.V_yukawa(p, lJ + 1, V0, inp.MT_MU, ngl=ngl, energy_packets=energy_packets)
            Vmp = o.V_yukawa(p, lJ, [inp.TENSOR_V * scale[2]], [inp.TENSOR_MU], ngl=ngl, energy_packets=energy_packets)
            H, Vf = o.assemble_H(e0, Vmm, Vpp, Vmp)
    return dict(p=p, e0=e0, dE=dE, Eedge=Ee, H=H, V=Vf)


def oracle_solve(N, coupled, ch, Ecm, averaged=False):
    W, C, sw = o.jacobi(ch["H"])
    T, b = o.onshell_T(N, coupled, ch["Eedge"], ch["V"], W, C, Ecm, averaged=averaged)
    d, S = o.phase_shifts(coupled, T, b, ch["dE"])
    return dict(W=W, C=C, sweeps=sw, T=T, bin=b, delta=d, S=S)


def swp_edge_distance(W, coupled, Ecm):
    """Distance of every energy to the nearest pseudostate bin edge (oracle edges), for the C11 exclusion."""
    nb = int((W < 0).sum())
    nbr = 2 if coupled else 1
    dist = np.full(len(Ecm), np.inf)
    for br in range(nbr):
        eps = W[nb + br::nbr]
        if len(eps) == 0:
            continue
        ed = o.swp_edges(eps)
        dist = np.minimum(dist, np.abs(Ecm[:, None] - ed[None, :]).min(axis=1))
    return dist


def dist180(a, b):
    return np.abs((np.asarray(a) - np.asarray(b) + 90.0) % 180.0 - 90.0)


def check_eig(W_gpu, W_ref, normH):
    W_gpu = np.asarray(W_gpu); W_ref = np.asarray(W_ref)
    small = np.abs(W_ref) < 1e-12 * normH
    rel = np.abs(W_gpu - W_ref) / np.where(small, normH, np.abs(W_ref))
    return rel.max()


def check_phases(coupled, delta_gpu, S_gpu, ref, Ecm):
    """Max phase error in degrees (mod 180) and max |dS| over energies not excluded by C11."""
    ok = swp_edge_distance(ref["W"], coupled, Ecm) > EDGE_GUARD
    ok &= ref["bin"] >= 0
    dmax = dist180(delta_gpu, ref["delta"])[ok]
    if coupled:
        dmax = dmax[:, :2]    # delta_-, delta_+; eps_J is compared through S (it flips sign with the branch, C10)
    smax = np.abs(np.asarray(S_gpu) - ref["S"])[ok]
    return (dmax.max() if dmax.size else 0.0), (smax.max() if smax.size else 0.0), int(ok.sum())
