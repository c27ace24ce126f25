"""Stored expected values (tests/golden/, written by tests/golden/make_golden.py from the oracle alone).

CPU: the Yamaguchi closed form (reading C15) and SURVEY's quoted numbers reproduce the stored MI values; the
oracle as it stands reproduces its stored config-1 chain.  GPU: the CUDA path reproduces the stored config-1 numbers."""
import math
import os

import numpy as np
import pytest

from paper_2106_00454_b200 import inputs as inp

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _yamaguchi_rows():
    return np.loadtxt(os.path.join(GOLD, "yamaguchi_1S0.txt"))


def _config1():
    out = dict(phase=[])
    for line in open(os.path.join(GOLD, "config1_1S0_N50.txt")):
        if line.startswith("#"):
            continue
        k, *v = line.split()
        if k == "phase":
            out["phase"].append((float(v[0]), int(v[1]), float(v[2])))
        else:
            out[k] = float(v[0])
    return out


def test_yamaguchi_closed_form_reproduces_stored_MI_values():
    beta = inp.YAMAGUCHI_BETA
    lp = beta ** 4 / (2 * (beta / 2 - 1 / inp.YAMAGUCHI_A))     # lambda' of reading C15
    assert abs(lp - 2.873679) < 1e-6
    for tlab, d, sig in _yamaguchi_rows():
        p = math.sqrt(inp.MU * tlab) / inp.HBARC
        pcot = (beta ** 4 - lp * beta + p * p * (2 * beta ** 2 + lp / beta) + p ** 4) / (2 * lp)
        dx = math.degrees(math.atan2(p, pcot))
        assert abs(dx - d) < 1e-9, (tlab, dx, d)
        assert abs(10 * math.pi * math.sin(math.radians(dx)) ** 2 / p ** 2 - sig) < 1e-9 * sig
    rows = {r[0]: r[1] for r in _yamaguchi_rows()}
    for tlab, ref in ((1.0, 63.3159), (50.0, 45.8472), (350.0, 14.9765)):   # SURVEY 8(c) C15 (probe values)
        assert abs(rows[tlab] - ref) < 1e-4


def test_oracle_reproduces_its_stored_config1_chain():
    from oracle import oracle as o
    g = _config1()
    N = 50
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    H, V = o.assemble_H(e0, o.V_yukawa(p, 0, inp.MT_V0, inp.MT_MU))
    W, Cm, sw = o.jacobi(H)
    assert sw == int(g["sweeps"])
    assert abs(W[0] - g["eig_min"]) < 1e-11 * abs(g["eig_min"]) and abs(W[-1] - g["eig_max"]) < 1e-11 * g["eig_max"]
    assert abs(W[1] - g["eig_second"]) < 1e-10 * g["eig_second"] and abs(W.sum() - g["trace"]) < 1e-11 * g["trace"]
    assert abs(g["eig_min"] + 2.19) < 0.01                       # bound state -2.19 MeV at N = 50
    tl, Ecm = inp.energies(100)
    T, b = o.onshell_T(N, 0, Ee, V, W, Cm, Ecm)
    d, _ = o.phase_shifts(0, T, b, dE)
    for tlab, bi, dg in g["phase"]:
        e = int(np.argmin(np.abs(tl - tlab)))
        assert b[e] == bi and abs(d[e] - dg) < 1e-8
    assert min(x[1] for x in g["phase"]) == 3 and max(x[1] for x in g["phase"]) == 35   # on-shell bins 3..35


@pytest.mark.gpu
def test_cuda_path_reproduces_stored_config1_values():
    import torch
    from paper_2106_00454_b200 import wpcd
    g = _config1()
    h = wpcd.Handle(0)
    N = 50
    tl, Ecm = inp.energies(100)
    out = h.build_channels(inp.grid_edges(N), [(0, 0)], V0=inp.MT_V0, mu=inp.MT_MU)
    Hb = out["H_unc"].reshape(-1, N, N)
    W, C, info = h.diag_batched(Hb)
    T, bins = h.onshell_T(N, 0, out["e0"], out["Eedge"], Hb, W, C, torch.as_tensor(Ecm, device="cuda:0"))
    delta, _ = h.phase_shifts(0, T, bins, out["dE"])
    W = W.cpu().numpy()[0]; d = delta.cpu().numpy()[0]; b = bins.cpu().numpy()
    assert abs(W[0] - g["eig_min"]) < 1e-11 * abs(g["eig_min"]) and abs(W[-1] - g["eig_max"]) < 1e-11 * g["eig_max"]
    assert abs(W[1] - g["eig_second"]) < 1e-11 * g["eig_second"]
    for tlab, bi, dg in g["phase"]:
        e = int(np.argmin(np.abs(tl - tlab)))
        assert b[e] == bi and abs((d[e] - dg + 90.0) % 180.0 - 90.0) < 1e-8
    h.close()
