"""GPU parity tests proper (-m gpu): the CUDA path, called through the C ABI (ctypes binding), against the CPU
oracle on the same seeded inputs.  Tolerances are north_star's: eigenvalues 1e-11 relative (componentwise),
phase shifts 1e-8 degrees absolute (mod 180; coupled channels also through |dS| <= 3.5e-10), H 1e-12 max|H|."""
import numpy as np
import pytest

from paper_2106_00454_b200 import inputs as inp
from tests import helpers as hp

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import torch
    from paper_2106_00454_b200 import wpcd
    h = wpcd.Handle(0)
    yield dict(torch=torch, wpcd=wpcd, h=h, dev=torch.device("cuda", 0))
    h.close()


def _to_dev(ctx, a, dtype=None):
    t = ctx["torch"].as_tensor(np.ascontiguousarray(a), device=ctx["dev"])
    return t if dtype is None else t.to(dtype)


def _gpu_pipeline(ctx, N, channels, Ecm, scales=None, S=1, yamaguchi=None, tol=0.0, edges=None, n_gl=8, mode=0,
                  energy_packets=False):
    """Full hot path on the GPU for a channel list; returns per-kind dicts of numpy arrays."""
    h, torch = ctx["h"], ctx["torch"]
    p = inp.grid_edges(N) if edges is None else edges
    d_scales = None if scales is None else _to_dev(ctx, scales)
    kw = dict(yamaguchi=yamaguchi) if yamaguchi is not None else dict(
        V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1] if scales is not None else None, VT=inp.TENSOR_V,
        muT=inp.TENSOR_MU, VT_scale_idx=2 if scales is not None else -1)
    out = h.build_channels(p, channels, scales=d_scales, S=S, n_gl=n_gl, energy_packets=energy_packets, **kw)
    d_E = _to_dev(ctx, Ecm)
    res = {}
    for kind, key in ((0, "H_unc"), (1, "H_cpl")):
        H = out[key]
        if H is None:
            continue
        n = H.shape[-1]
        Hb = H.reshape(-1, n, n)
        W, C, info = h.diag_batched(Hb, tol=tol)
        T, bins = h.onshell_T(N, kind, out["e0"], out["Eedge"], Hb, W, C, d_E, mode=mode)
        delta, Sm = h.phase_shifts(kind, T, bins, out["dE"])
        torch.cuda.synchronize()
        nch = H.shape[1]
        cplx = lambda x: x[..., 0].cpu().numpy() + 1j * x[..., 1].cpu().numpy()
        res[kind] = dict(H=H.cpu().numpy(), W=W.cpu().numpy().reshape(S, nch, n), C=C.cpu().numpy().reshape(S, nch, n, n),
                         info=info.cpu().numpy().reshape(S, nch), T=cplx(T).reshape((S, nch) + tuple(T.shape[1:-1])),
                         S=cplx(Sm).reshape((S, nch) + tuple(T.shape[1:-1])),
                         delta=delta.cpu().numpy().reshape((S, nch) + tuple(delta.shape[1:])), bin=bins.cpu().numpy())
    res["e0"] = out["e0"].cpu().numpy(); res["dE"] = out["dE"].cpu().numpy(); res["Eedge"] = out["Eedge"].cpu().numpy()
    return res


# Cases in which the 80-bit run of the oracle's Jacobi (orc_jacobi_ld, pinned in tests/test_oracle_pins_arbiter.py) had
# to arbitrate between the CUDA path and the fp64 oracle: (label, "eig" | "phase", N, custom grid?).
# names where that may happen -- n >= 600 or N >= 400 bins on the config grid (||H|| ~ p_N^2 grows with N, the rounding of
# the oracle's cyclic sweeps with n, while the smallest eigenvalues shrink: the fp64 oracle's own error on them is 1.6e-11
# at N = 300, n = 600, 1.6e-11 at N = 400, n = 800 and 2.0e-11 at N = 452, n = 452, measured against the 80-bit run, where
# the CUDA path is at 1e-13) and the paper's Chebyshev grid (norm-wise stop rule on a Hamiltonian graded over 13+ orders of
# magnitude); anywhere else it is a failure (test_zz_arbitration_only_where_design_allows, which runs last in this module).
ARBITRATED = []


def _arbitration_allowed(N, n, custom_grid):
    return custom_grid or N >= 400 or n >= 600


def _compare_channel(res, kind, s, c, N, lJ, Ecm, scale=(1.0, 1.0, 1.0), yamaguchi=None, label="", edges=None, ngl=8,
                     averaged=False, energy_packets=False):
    ch = hp.oracle_channel(N, kind, lJ, scale, yamaguchi, edges=edges, ngl=ngl, energy_packets=energy_packets)
    ref = hp.oracle_solve(N, kind, ch, Ecm, averaged=averaged)
    g = res[kind]
    n = ch["H"].shape[0]
    normH = np.abs(ch["H"]).max()
    errH = np.abs(g["H"][s, c] - ch["H"]).max() / normH
    assert errH <= hp.TOL_H_REL, (label, "H", errH)
    assert np.array_equal(g["H"][s, c], g["H"][s, c].T), (label, "H symmetric")
    assert g["info"][s, c] >= 1, (label, "info", g["info"][s, c])
    errW = hp.check_eig(g["W"][s, c], ref["W"], normH)
    if errW > hp.TOL_EIG_REL:
        # DESIGN.md section 3 "eigenvalue arbitration": at large n the fp64 oracle's own rounding error on the smallest
        # eigenvalues exceeds 1e-11; the 80-bit run of the same oracle algorithm decides.
        from oracle import oracle as o
        W_ld = o.jacobi_ld(ch["H"])[0]
        errW, err_oracle = hp.check_eig(g["W"][s, c], W_ld, normH), hp.check_eig(ref["W"], W_ld, normH)
        print(label, "eig arbitration vs long double: gpu", errW, "fp64 oracle", err_oracle)
        ARBITRATED.append((label, "eig", N, n, edges is not None))
        assert _arbitration_allowed(N, n, edges is not None), (label, "eig arbitration outside DESIGN.md's list", errW)
        assert err_oracle > errW, (label, "arbitration: the fp64 oracle must be the less accurate side", err_oracle, errW)
    assert errW <= hp.TOL_EIG_REL, (label, "eig", errW)
    C = g["C"][s, c]
    assert np.abs(C.T @ C - np.eye(n)).max() < 1e-12, (label, "orth")
    assert np.abs(ch["H"] @ C - C * g["W"][s, c]).max() < 1e-13 * n * normH, (label, "residual")
    assert np.array_equal(g["bin"], ref["bin"]), (label, "bins")
    dphi, dS, nok = hp.check_phases(kind, g["delta"][s, c], g["S"][s, c], ref, Ecm)
    assert nok > 0.9 * len(Ecm)
    if dphi > hp.TOL_PHASE_DEG or dS > hp.TOL_S_ABS:
        # DESIGN.md section 3 "arbitration": the fp64 oracle stops on a NORM-wise criterion (off(A) <= 1e-15 ||A||_F), so on
        # grids where ||H|| is 1e9 MeV (the paper's Chebyshev bins at N = 100) its small eigenpairs carry a relative error
        # that the log-singular resolvent amplifies near a bin edge.  The same chain with the eigenpairs of the oracle's
        # 80-bit Jacobi run (T and phases still fp64) decides.
        from oracle import oracle as o
        W_ld, C_ld, _ = o.jacobi_ld(ch["H"])
        T_ld, b_ld = o.onshell_T(N, kind, ch["Eedge"], ch["V"], W_ld, C_ld, Ecm, averaged=averaged)
        d_ld, S_ld = o.phase_shifts(kind, T_ld, b_ld, ch["dE"])
        ref_ld = dict(ref, W=W_ld, delta=d_ld, S=S_ld, bin=b_ld)
        dphi_o, dS_o, _ = hp.check_phases(kind, ref["delta"], ref["S"], ref_ld, Ecm)
        dphi, dS, nok = hp.check_phases(kind, g["delta"][s, c], g["S"][s, c], ref_ld, Ecm)
        print(label, "phase arbitration vs long-double eigenpairs: gpu", dphi, dS, "fp64 oracle", dphi_o, dS_o)
        ARBITRATED.append((label, "phase", N, n, edges is not None))
        assert _arbitration_allowed(N, n, edges is not None), (label, "phase arbitration outside DESIGN.md's list", dphi, dS)
        assert dphi_o > dphi or dS_o > dS, (label, "arbitration: the fp64 oracle must be the less accurate side")
    print("PARITY", label, "n", n, "eig", errW, "phase", dphi, "S", dS)
    assert dphi <= hp.TOL_PHASE_DEG, (label, "phase", dphi)
    assert dS <= hp.TOL_S_ABS, (label, "S", dS)
    return errH, errW, dphi, dS


# ----------------------------------------------------------------------------------------------- config 1
def test_config1_1S0_N50(ctx):
    tl, Ecm = inp.energies(100)
    res = _gpu_pipeline(ctx, 50, [(0, 0)], Ecm)
    errs = _compare_channel(res, 0, 0, 0, 50, 0, Ecm, label="cfg1")
    assert abs(res[0]["W"][0, 0, 0] + 2.19) < 0.01     # the bound state
    print("cfg1 errs (H, eig, phase, S):", errs)


# ----------------------------------------------------------------------------------------------- config 2
def test_config2_all_channels_N100(ctx):
    tl, Ecm = inp.energies(350)
    chans = [(c, l) for _, c, l in inp.CHANNELS_J4]
    res = _gpu_pipeline(ctx, 100, chans, Ecm)
    iu = ic = 0
    worst = np.zeros(4)
    for name, c, l in inp.CHANNELS_J4:
        idx = ic if c else iu
        worst = np.maximum(worst, _compare_channel(res, c, 0, idx, 100, l, Ecm, label=name))
        if c: ic += 1
        else: iu += 1
    print("cfg2 worst errs (H, eig, phase, S):", worst)


# ----------------------------------------------------------------------------------------------- config 3
def test_config3_sampled_batch(ctx):
    """1024 seeded samples on the GPU (full size); the oracle checks a seeded subsample of (sample, channel)."""
    S = 1024
    tl, Ecm = inp.energies(350)
    scales = inp.sample_scales(S, seed=0)
    assert np.allclose(scales[0], [1.012573, 0.986790, 1.064042], atol=1e-6)   # reading C14
    chans = [(c, l) for _, c, l in inp.CHANNELS_J4]
    res = _gpu_pipeline(ctx, 100, chans, Ecm, scales=scales, S=S)
    assert (res[0]["info"] >= 1).all() and (res[1]["info"] >= 1).all()
    nbound = (res[0]["W"][:, 0, :] < 0).sum(axis=1)          # 1S0: SURVEY 8(d): 957 samples bind, 67 do not
    assert set(np.unique(nbound)) == {0, 1} and (nbound == 1).sum() == 957
    rng = np.random.default_rng(1)
    picks = [(0, 0, 0, 0), (0, 1, 0, 1)] + [(int(rng.integers(S)), int(k), None, None) for k in rng.integers(0, 14, 6)]
    unc = [(i, l) for i, (_, c, l) in enumerate(inp.CHANNELS_J4) if not c]
    for s, k, _, _ in picks:
        name, c, l = inp.CHANNELS_J4[k % 14]
        idx = sum(1 for (_, cc, _) in inp.CHANNELS_J4[:k % 14] if cc == c)
        _compare_channel(res, c, s, idx, 100, l, Ecm, scale=tuple(scales[s]), label=f"cfg3 s={s} {name}")
    # a sample without an S-wave bound state must be among the checked ones (both n_b paths)
    s0 = int(np.where(nbound == 0)[0][0])
    _compare_channel(res, 0, s0, 0, 100, 0, Ecm, scale=tuple(scales[s0]), label=f"cfg3 unbound s={s0}")


# ----------------------------------------------------------------------------------------------- config 4
def test_config4_large_n_and_yamaguchi(ctx):
    """Config 4 at its stated size: 256 seeded samples x all 14 channels J <= 4 at N=200 (2560 matrices of 200^2 and 1024 of
    400^2: beyond shared memory -> the workspace path, every CTA takes several matrices) + the Yamaguchi analytic check.
    The oracle checks a seeded subsample of (sample, channel), among them matrices that a CTA takes second or later."""
    S = 256
    tl, Ecm = inp.energies(350)
    scales = inp.sample_scales(256, seed=0)
    chans = [(c, l) for _, c, l in inp.CHANNELS_J4]
    res = _gpu_pipeline(ctx, 200, chans, Ecm, scales=scales, S=S)
    assert (res[0]["info"] >= 1).all() and (res[1]["info"] >= 1).all()
    unc = [(nm, l) for nm, c, l in inp.CHANNELS_J4 if not c]
    cpl = [(nm, l) for nm, c, l in inp.CHANNELS_J4 if c]
    # (kind, sample, channel index within its kind): flat matrix index = sample * n_chan_of_kind + index
    for kind, s_, ci in ((0, 0, 0), (0, 255, 9), (0, 97, 4), (1, 1, 0), (1, 255, 3), (1, 140, 1)):
        nm, l = (cpl if kind else unc)[ci]
        _compare_channel(res, kind, s_, ci, 200, l, Ecm, scale=tuple(scales[s_]), label=f"cfg4 s={s_} {nm}")
    del res
    # Yamaguchi at N=200: GPU vs oracle, and GPU vs the closed-form phase shift (median error < 1 degree)
    lamA, lamB = inp.yamaguchi_lambda()
    yres = _gpu_pipeline(ctx, 200, [(0, 0)], Ecm, yamaguchi=(lamB, inp.YAMAGUCHI_BETA))
    _compare_channel(yres, 0, 0, 0, 200, 0, Ecm, yamaguchi=(lamB, inp.YAMAGUCHI_BETA), label="cfg4 yamaguchi")
    lp = lamA * inp.MU / inp.HBARC ** 2
    beta = inp.YAMAGUCHI_BETA
    pm = np.sqrt(inp.MU * tl) / inp.HBARC
    Sx = 1 + 4j * lp * pm / (pm * pm + beta * beta) ** 2 / (1 - lp / (beta * (beta - 1j * pm) ** 2))
    exact = 0.5 * np.degrees(np.angle(Sx))
    assert np.median(hp.dist180(yres[0]["delta"][0, 0], exact)) < 1.0


# ----------------------------------------------------------------------------------------------- config 5
@pytest.mark.parametrize("N", [32, 48, 64, 100, 150, 200, 300, 400])
def test_config5_size_sweep(ctx, N):
    """single (l=0, n=N) and coupled (J=1, n=2N) matrices at every N of the sweep, S seeded samples on the GPU, the
    oracle on one of them (cyclic Jacobi at n = 800 costs ~1e11 flops)."""
    S = 3
    tl, Ecm = inp.energies(350)
    scales = inp.sample_scales(4096, seed=0)[:S]
    res = _gpu_pipeline(ctx, N, [(0, 0), (1, 1)], Ecm, scales=scales, S=S)
    assert (res[0]["info"] >= 1).all() and (res[1]["info"] >= 1).all()
    _compare_channel(res, 0, 2, 0, N, 0, Ecm, scale=tuple(scales[2]), label=f"cfg5 N={N} single")
    _compare_channel(res, 1, 1, 0, N, 1, Ecm, scale=tuple(scales[1]), label=f"cfg5 N={N} coupled")


# ----------------------------------------------------------------------------------------------- edge cases
def _diag_check(ctx, A, tol_rel=1e-11):
    from oracle import oracle as o
    W, C, info = ctx["h"].diag_batched(_to_dev(ctx, A))
    ctx["torch"].cuda.synchronize()
    W = W.cpu().numpy(); C = C.cpu().numpy(); info = info.cpu().numpy()
    for b in range(A.shape[0]):
        Wr, Cr, _ = o.jacobi(A[b])
        n = A.shape[1]
        nrm = max(np.abs(A[b]).max(), 1e-300)
        assert info[b] >= 1
        assert np.abs(W[b] - Wr).max() <= tol_rel * nrm, (b, np.abs(W[b] - Wr).max() / nrm)
        assert np.abs(C[b].T @ C[b] - np.eye(n)).max() < 1e-12
        assert np.abs(A[b] @ C[b] - C[b] * W[b]).max() < 1e-13 * n * nrm
    return W, C, info


@pytest.mark.parametrize("n", [2, 3, 7, 8, 9, 16, 17, 31, 33, 36, 40, 41, 48, 49, 56, 63, 104, 105, 112, 113, 120, 129])
def test_diag_ragged_sizes_random(ctx, n):
    rng = np.random.default_rng(n)
    A = rng.standard_normal((5, n, n)); A = A + A.transpose(0, 2, 1)
    _diag_check(ctx, A)


def test_diag_largest_mode_q_in_workspace(ctx):
    """Maximum sizes: n = 904 (57 slots) no longer holds the Q buffers in shared memory -- the kernel mode with A, V and Q
    all in the global workspace.  The oracle's cyclic Jacobi needs minutes at this size, so the check is by what holds
    at any size: orthonormal C, small residual, trace and Frobenius norm, and the eigenvalues against
    LAPACK (normwise)."""
    n = 904
    rng = np.random.default_rng(n)
    A = rng.standard_normal((2, n, n)); A = A + A.transpose(0, 2, 1)
    A[1] *= np.geomspace(1e-3, 1e3, n)[:, None] * np.geomspace(1e-3, 1e3, n)[None, :]   # graded like the Hamiltonians
    W, C, info = ctx["h"].diag_batched(_to_dev(ctx, A))
    ctx["torch"].cuda.synchronize()
    W = W.cpu().numpy(); C = C.cpu().numpy(); info = info.cpu().numpy()
    for b in range(2):
        nrm = np.abs(A[b]).max()
        assert info[b] >= 1
        assert np.all(np.diff(W[b]) >= 0)
        assert np.abs(C[b].T @ C[b] - np.eye(n)).max() < 1e-12
        assert np.abs(A[b] @ C[b] - C[b] * W[b]).max() < 1e-13 * n * nrm
        assert abs(W[b].sum() - np.trace(A[b])) <= 1e-12 * n * nrm
        assert abs((W[b] ** 2).sum() - (A[b] ** 2).sum()) <= 1e-12 * (A[b] ** 2).sum()
        assert np.abs(W[b] - np.linalg.eigvalsh(A[b])).max() <= 1e-11 * np.abs(W[b]).max()


def test_diag_degenerate_cases(ctx):
    n = 24
    A = np.zeros((4, n, n))
    A[0] = np.diag(np.arange(n, 0, -1.0))                       # already diagonal, descending: pure sort
    A[1] = np.eye(n) * 3.0                                       # all eigenvalues equal
    A[2] = np.ones((n, n))                                       # rank one: eigenvalues {0 x23, 24}
    A[3][:] = 0.0                                                # zero matrix
    W, C, info = _diag_check(ctx, A)
    assert np.array_equal(W[0], np.arange(1.0, n + 1)) and info[0] == 1
    assert np.allclose(W[1], 3.0) and np.allclose(W[3], 0.0)
    assert abs(W[2][-1] - n) < 1e-12 and np.abs(W[2][:-1]).max() < 1e-12


def test_onshell_energy_outside_grid_and_empty_like_inputs(ctx):
    N = 16
    Ecm = np.array([-1.0, 0.5, 40.0, 1e9])      # below 0, inside, inside, above the last edge
    res = _gpu_pipeline(ctx, N, [(0, 0)], Ecm)
    ch = hp.oracle_channel(N, 0, 0)
    ref = hp.oracle_solve(N, 0, ch, Ecm)
    assert list(res[0]["bin"]) == list(ref["bin"]) and res[0]["bin"][0] == -1 and res[0]["bin"][3] == -1
    assert res[0]["T"][0, 0, 0] == 0 and res[0]["T"][0, 0, 3] == 0
    assert np.abs(res[0]["T"][0, 0, 1:3] - ref["T"][1:3]).max() < 1e-9 * np.abs(ref["T"][1:3]).max()


def test_onshell_largest_n_plain_loop_path(ctx):
    """Maximum sizes: beyond n ~ 1530 fewer than 8 rows of VC fit shared memory and wpcd_onshell_T leaves the tensor-core
    product for the plain loop.  The step only needs (H, W, C) of the right shapes, so the inputs are synthetic (no
    eigen-solve at this size); compared element by element with the oracle's on-shell T on identical inputs."""
    from oracle import oracle as o
    N = 1552
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    rng = np.random.default_rng(N)
    G = rng.standard_normal((N, N))
    H = np.diag(e0) + 20.0 * (G + G.T) / np.sqrt(N)
    V = H.copy(); V[np.arange(N), np.arange(N)] -= e0            # what the kernel forms: V = H - diag(e0)
    W = np.sort(e0 * (1.0 + 0.01 * rng.standard_normal(N))); W[0] = -2.2   # one bound state
    Cm = rng.standard_normal((N, N)) / np.sqrt(N)
    Ecm = np.array([-1.0, 20.0, 20.7, 21.3, 22.0, 1e12])
    T, bins = ctx["h"].onshell_T(N, False, _to_dev(ctx, e0), _to_dev(ctx, Ee), _to_dev(ctx, H[None]), _to_dev(ctx, W[None]),
                                 _to_dev(ctx, Cm[None]), _to_dev(ctx, Ecm))
    ctx["torch"].cuda.synchronize()
    T = T.cpu().numpy()[0]; T = T[:, 0] + 1j * T[:, 1]
    Tr, br = o.onshell_T(N, False, Ee, V, W, Cm, Ecm)
    assert list(bins.cpu().numpy()) == list(br) and br[0] == -1 and br[-1] == -1 and len(set(br[1:5])) == 4
    assert T[0] == 0 and T[-1] == 0
    ok = hp.swp_edge_distance(W, 0, Ecm) > hp.EDGE_GUARD
    ok[0] = ok[-1] = False
    assert ok.sum() >= 3
    assert np.abs(T[ok] - Tr[ok]).max() <= 1e-11 * np.abs(Tr[ok]).max()


def test_abi_argument_errors(ctx):
    import ctypes as C
    wp = ctx["wpcd"]
    lib = wp._lib
    h = ctx["h"]._h
    assert lib.wpcd_diag_batched(h, 1, 1, None, None, None, None, 0.0, 10, None, 0, None, 0, None) == -1      # NULL pointers
    t = ctx["torch"].zeros(16, dtype=ctx["torch"].float64, device=ctx["dev"])
    ti = ctx["torch"].zeros(4, dtype=ctx["torch"].int32, device=ctx["dev"])
    assert lib.wpcd_diag_batched(h, 1, 1, t.data_ptr(), t.data_ptr(), t.data_ptr(), ti.data_ptr(), 0.0, 10, None, 0, None, 0, None) == -2
    assert lib.wpcd_diag_batched(h, 200, 1, t.data_ptr(), t.data_ptr(), t.data_ptr(), ti.data_ptr(), 0.0, 10, None, 0, None, 0, None) == -3
    edges = (C.c_double * 3)(0.0, 2.0, 1.0)     # not increasing
    g = wp.Grid(2, edges, 197.327, 469.46, 8)
    assert lib.wpcd_build_channels(h, C.byref(g), None, None, 1, None, 1, 0, None, None, None, None, None, None, 0, None) == -1
    assert wp._lib.wpcd_strerror(-3) == b"workspace too small"


# ----------------------------------------------------------------------------------------------- NEXT-1: averaged resolvent
@pytest.mark.parametrize("N,kind,lJ", [(50, 0, 0), (100, 1, 1), (64, 1, 2), (120, 1, 1), (210, 0, 0)])
def test_energy_averaged_T_mode1(ctx, N, kind, lJ):
    """wpcd_onshell_T(mode=1) (Eq. 28, B.7-B.8) against the oracle's averaged T on the same eigenpairs' inputs:
    n <= 200 runs the identity kernel, n > 200 the direct one; uncoupled (with a bound state) and coupled channels."""
    h, torch = ctx["h"], ctx["torch"]
    tl, Ecm = inp.energies(120)
    out = h.build_channels(inp.grid_edges(N), [(kind, lJ)], S=1, V0=inp.MT_V0, mu=inp.MT_MU, VT=inp.TENSOR_V, muT=inp.TENSOR_MU)
    Hd = out["H_cpl" if kind else "H_unc"]
    n = Hd.shape[-1]
    Hb = Hd.reshape(-1, n, n)
    W, C, info = h.diag_batched(Hb)
    T, bins = h.onshell_T(N, kind, out["e0"], out["Eedge"], Hb, W, C, _to_dev(ctx, Ecm), mode=1)
    delta, Sm = h.phase_shifts(kind, T, bins, out["dE"])
    torch.cuda.synchronize()
    ch = hp.oracle_channel(N, kind, lJ)
    from oracle import oracle as o
    Wr, Cr, _ = o.jacobi(ch["H"])
    Tr, br = o.onshell_T(N, bool(kind), ch["Eedge"], ch["V"], Wr, Cr, Ecm, averaged=True)
    dr, Sr = o.phase_shifts(bool(kind), Tr, br, ch["dE"])
    assert np.array_equal(bins.cpu().numpy(), br)
    Tg = T.cpu().numpy()[0]; Tg = Tg[..., 0] + 1j * Tg[..., 1]
    Sg = Sm.cpu().numpy()[0]; Sg = Sg[..., 0] + 1j * Sg[..., 1]
    scale = np.abs(Tr).max()
    assert np.abs(Tg - Tr).max() <= 1e-10 * scale, np.abs(Tg - Tr).max() / scale
    assert np.abs(Sg - Sr).max() <= hp.TOL_S_ABS
    d = hp.dist180(delta.cpu().numpy()[0], dr)
    if kind:
        d = d[:, :2]
    assert d.max() <= hp.TOL_PHASE_DEG, d.max()
    # one value per on-shell bin
    bb = bins.cpu().numpy()
    for i in np.unique(bb[bb >= 0]):
        idx = np.where(bb == i)[0]
        assert np.all(Tg[idx] == Tg[idx[0]])


def test_diag_is_run_to_run_deterministic(ctx):
    """The pipelined kernel hands tiles to warps through a dynamic queue and overlaps the pivot solves of the next step
    with the updates of the running one; every item touches disjoint data, so repeated runs must agree BIT FOR BIT.
    (compute-sanitizer is closed on this pool; a data race would show up here as run-to-run differences.)"""
    h, torch = ctx["h"], ctx["torch"]
    # (150, coupled) = n = 300: the log mode (scheduler in global memory, dataflow replay), below and above the grid size
    for N, chans, S in ((100, [(0, 0)], 300), (100, [(1, 1)], 150), (24, [(0, 1)], 600), (150, [(1, 2)], 8), (150, [(1, 1)], 200)):
        scales = inp.sample_scales(S, seed=3)
        out = h.build_channels(inp.grid_edges(N), chans, scales=_to_dev(ctx, scales), S=S, V0=inp.MT_V0, mu=inp.MT_MU,
                               scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
        H = out["H_cpl" if chans[0][0] else "H_unc"]
        n = H.shape[-1]
        Hb = H.reshape(-1, n, n)
        ref = None
        for rep in range(4):
            W, C, info = h.diag_batched(Hb)
            torch.cuda.synchronize()
            cur = (W.clone(), C.clone(), info.clone())
            if ref is None:
                ref = cur
            else:
                assert torch.equal(cur[0], ref[0]) and torch.equal(cur[1], ref[1]) and torch.equal(cur[2], ref[2]), (N, chans, rep)
        assert (ref[2] >= 1).all()


@pytest.mark.parametrize("N,kind,lJ", [(50, 0, 0), (100, 1, 1), (40, 0, 2)])
def test_production_variant_averaged_T_then_interpolation(ctx, N, kind, lJ):
    """The paper's production chain: energy-averaged T at the bin mid-points, phases, then
    Eq. 42 at arbitrary energies -- GPU (wpcd_onshell_T mode 1 -> wpcd_phase_shifts -> wpcd_interp_phases) against the
    oracle's chain; plus synthetic mid-point phases with branch jumps fed to both interpolators."""
    from oracle import oracle as o
    h, torch = ctx["h"], ctx["torch"]
    p = inp.grid_edges(N)
    cE = inp.HBARC ** 2 / (2 * inp.MU)
    qm = 0.5 * (p[:-1] + p[1:])
    tl, Ecm = inp.energies(90)
    q = np.sqrt(Ecm / cE)
    out = h.build_channels(p, [(kind, lJ)], S=1, V0=inp.MT_V0, mu=inp.MT_MU, VT=inp.TENSOR_V, muT=inp.TENSOR_MU)
    Hd = out["H_cpl" if kind else "H_unc"]
    n = Hd.shape[-1]
    Hb = Hd.reshape(-1, n, n)
    W, C, info = h.diag_batched(Hb)
    T, bins = h.onshell_T(N, kind, out["e0"], out["Eedge"], Hb, W, C, _to_dev(ctx, cE * qm ** 2), mode=1)
    dmid, _ = h.phase_shifts(kind, T, bins, out["dE"])
    got = h.interp_phases(kind, _to_dev(ctx, p), dmid, _to_dev(ctx, q))
    torch.cuda.synchronize()
    ch = hp.oracle_channel(N, kind, lJ)
    Wr, Cr, _ = o.jacobi(ch["H"])
    Tr, br = o.onshell_T(N, bool(kind), ch["Eedge"], ch["V"], Wr, Cr, cE * qm ** 2, averaged=True)
    dr, _ = o.phase_shifts(bool(kind), Tr, br, ch["dE"])
    assert np.array_equal(bins.cpu().numpy(), br) and np.array_equal(br, np.arange(N))   # mid-point i lies in bin i
    # same mid-point inputs to both interpolators: agreement to rounding
    same = o.interp_phases(p, dmid.cpu().numpy()[0], q)
    g = got.cpu().numpy()[0]
    assert np.allclose(g, same, atol=1e-10, rtol=0, equal_nan=True)
    # whole chain against the oracle's chain, where the mid-point phases themselves agree to 1e-8 (top bins with no
    # i-th pseudostate give T = 0 on both sides)
    want = o.interp_phases(p, dr, q)
    d = hp.dist180(g, want)
    if kind:
        d = d[:, :2]
    assert np.nanmax(d) <= 5 * hp.TOL_PHASE_DEG, np.nanmax(d)
    # synthetic mid-point phases with principal-value jumps (and, coupled, mixing-angle sign flips)
    rng = np.random.default_rng(N)
    smooth = 150.0 * np.cos(3.0 * qm / qm[-1]) + 20.0
    wrapped = (smooth + 90.0) % 180.0 - 90.0
    dm = np.stack([wrapped, (0.5 * smooth + 90.0) % 180.0 - 90.0, rng.uniform(-5, 5, N)], axis=1) if kind else wrapped
    g2 = h.interp_phases(kind, _to_dev(ctx, p), _to_dev(ctx, dm[None]), _to_dev(ctx, q)).cpu().numpy()[0]
    assert np.allclose(g2, o.interp_phases(p, dm, q), atol=1e-10, rtol=0, equal_nan=True)


def test_diag_row_ranges_and_pipeline_rows(ctx):
    """wpcd_diag_batched with h_rows: same eigenvalues, the wanted rows of C bit-identical to the full run, the other
    rows zero; and the pipeline (which asks wpcd_onshell_rows for the rows) gives the same phases either way."""
    from paper_2106_00454_b200.pipeline import Pipeline
    h, torch = ctx["h"], ctx["torch"]
    N = 60
    out = h.build_channels(inp.grid_edges(N), [(1, 1)], S=3, scales=_to_dev(ctx, inp.sample_scales(3, seed=5)), V0=inp.MT_V0,
                           mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    Hb = out["H_cpl"].reshape(-1, 2 * N, 2 * N)
    W0, C0, i0 = h.diag_batched(Hb)
    rows = [(5, 41), (N + 5, N + 41)]
    W1, C1, i1 = h.diag_batched(Hb, rows=rows)
    torch.cuda.synchronize()
    assert torch.equal(W0, W1) and torch.equal(i0, i1)
    keep = np.zeros(2 * N, dtype=bool)
    for lo, hi in rows:
        keep[lo:hi] = True
    C0n, C1n = C0.cpu().numpy(), C1.cpu().numpy()
    assert np.array_equal(C1n[:, keep, :], C0n[:, keep, :]) and not C1n[:, ~keep, :].any() and (~keep).any()
    # argument errors
    with pytest.raises(Exception):
        h.diag_batched(Hb, rows=[(10, 5)])
    with pytest.raises(Exception):
        h.diag_batched(Hb, rows=[(0, 2 * N + 1)])
    # library-chosen rows: inside the grid for n <= 200, all rows beyond
    tl, Ecm = inp.energies(60)
    r = h.onshell_rows(inp.grid_edges(100), 1, Ecm)
    assert r is not None and len(r) == 2 and r[0][0] <= 6 and r[0][1] >= 72 and r[1] == (100 + r[0][0], 100 + r[0][1])
    assert h.onshell_rows(inp.grid_edges(150), 1, Ecm) is None and h.onshell_rows(inp.grid_edges(150), 0, Ecm) is not None
    pot = dict(V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    sc = inp.sample_scales(4, seed=2)
    res = []
    for flag in (True, False):
        pipe = Pipeline(inp.grid_edges(64), [(0, 0), (1, 1)], Ecm, 4, pot, device=0, onshell_rows_only=flag)
        d, info = pipe.solve_host(sc)
        res.append({k: v.clone() for k, v in d.items()})
    for k in res[0]:
        assert torch.equal(res[0][k], res[1][k])


def _oracle_sigma(N, channels, names, Ecm, scale):
    """Oracle chain per channel -> S-matrices -> Eqs. A.2/A.9/A.11 per energy.  Returns sigma [nE] (NaN off the grid),
    the oracle T per channel and the weight sum of (2J+1) over the diagonal partial waves."""
    sJ = [inp.channel_sJ(nm) for nm in names]
    refs = []
    for (kind, lJ) in channels:
        ch = hp.oracle_channel(N, kind, lJ, scale)
        refs.append((kind, hp.oracle_solve(N, kind, ch, Ecm), ch))
    sig = np.full(len(Ecm), np.nan)
    for e, E in enumerate(Ecm):
        if refs[0][1]["bin"][e] < 0:
            continue
        p = np.sqrt(E / (inp.HBARC ** 2 / (2 * inp.MU)))
        S_unc = [r["S"][e] for k, r, _ in refs if not k]
        S_cpl = [r["S"][e] for k, r, _ in refs if k]
        sig[e] = hp.o.sigma_tot(hp.o.partial_waves(channels, sJ, S_unc, S_cpl), p)
    wsum = sum((2 * J + 1) * (2 if k else 1) for (k, _), (_, J) in zip(channels, sJ))
    return sig, refs, wsum


def test_sigma_tot_all_channels(ctx):
    """NEXT-2: total cross section of all 14 channels, GPU chain (build -> diag -> T -> wpcd_sigma_tot) against the
    oracle chain (-> S -> Eq. A.2 with Clebsch-Gordan coefficients -> A.9 -> A.11).  Tolerance: the north_star S-matrix
    tolerance |dS| <= 3.5e-10 propagated through the partial-wave sum, (10 pi/(2 p^2)) sum (2J+1) |dS|."""
    h, torch = ctx["h"], ctx["torch"]
    N = 50
    names = [c[0] for c in inp.CHANNELS_J4]
    channels = [(c[1], c[2]) for c in inp.CHANNELS_J4]
    sJ = [inp.channel_sJ(nm) for nm in names]
    _, Ecm = inp.energies(40)
    Ecm = np.concatenate([Ecm, [1e9]])   # the last energy is outside the grid -> NaN
    scales = inp.sample_scales(2, seed=3)
    res = _gpu_pipeline(ctx, N, channels, Ecm, scales=scales, S=2)
    T_unc = _to_dev(ctx, np.stack([res[0]["T"].real, res[0]["T"].imag], axis=-1))
    T_cpl = _to_dev(ctx, np.stack([res[1]["T"].real, res[1]["T"].imag], axis=-1))
    J_unc = [J for (k, _), (_, J) in zip(channels, sJ) if not k]
    J_cpl = [J for (k, _), (_, J) in zip(channels, sJ) if k]
    bins, dE, dEcm = _to_dev(ctx, res[0]["bin"]), _to_dev(ctx, res["dE"]), _to_dev(ctx, Ecm)
    sig = h.sigma_tot(J_unc, T_unc, J_cpl, T_cpl, bins, dE, dEcm).cpu().numpy()
    assert sig.shape == (2, len(Ecm)) and np.isnan(sig[:, -1]).all()
    p2 = Ecm / (inp.HBARC ** 2 / (2 * inp.MU))
    worst = 0.0
    for s in range(2):
        ref, refs, wsum = _oracle_sigma(N, channels, names, Ecm, scales[s])
        ok = ~np.isnan(ref)
        for kind, r, _ in refs:
            ok &= hp.swp_edge_distance(r["W"], kind, Ecm) > hp.EDGE_GUARD
        assert ok.sum() >= 35 and np.isnan(ref[-1])
        bound = 10 * np.pi / (2 * p2) * wsum * hp.TOL_S_ABS
        err = np.abs(sig[s] - ref)
        assert (err[ok] <= bound[ok]).all(), (s, (err[ok] / bound[ok]).max())
        worst = max(worst, (err[ok] / np.abs(ref[ok])).max())
        assert (ref[ok] > 0).all()
    print("sigma_tot max relative deviation", worst)
    assert worst < 1e-9
    # the kernel alone, fed with the ORACLE's T (no eigen-solver differences): partial-wave sum vs the Clebsch-Gordan chain
    ref, refs, wsum = _oracle_sigma(N, channels, names, Ecm, scales[0])
    To_unc = np.stack([r["T"] for k, r, _ in refs if not k])[None]
    To_cpl = np.stack([r["T"] for k, r, _ in refs if k])[None]
    up = lambda T: _to_dev(ctx, np.stack([T.real, T.imag], axis=-1))
    sig1 = h.sigma_tot(J_unc, up(To_unc), J_cpl, up(To_cpl), bins, dE, dEcm).cpu().numpy()[0]
    ok = ~np.isnan(ref)
    assert (np.abs(sig1[ok] - ref[ok]) <= 2e-12 * np.abs(ref[ok]) + 1e-11).all()
    # subsets of the channel list: uncoupled only / coupled only add up to the total
    su = h.sigma_tot(J_unc, up(To_unc), [], None, bins, dE, dEcm).cpu().numpy()[0]
    sc = h.sigma_tot([], None, J_cpl, up(To_cpl), bins, dE, dEcm).cpu().numpy()[0]
    assert (np.abs(su[ok] + sc[ok] - sig1[ok]) <= 1e-12 * np.abs(sig1[ok])).all()
    # argument errors
    with pytest.raises(RuntimeError):
        h.sigma_tot([], None, [], None, bins, dE, dEcm, out=torch.empty((1, len(Ecm)), dtype=torch.float64, device=ctx["dev"]))
    with pytest.raises(RuntimeError):
        h.sigma_tot(J_unc, up(To_unc), [0], up(To_cpl[:, :1]), bins, dE, dEcm)   # coupled channels need J >= 1


def test_pipeline_sigma_tot_epilogue(ctx):
    """Pipeline(channel_J=...) appends wpcd_sigma_tot to the pass: same numbers as the oracle chain on sampled energies."""
    from paper_2106_00454_b200.pipeline import Pipeline
    N = 32
    names = [c[0] for c in inp.CHANNELS_J4]; channels = [(c[1], c[2]) for c in inp.CHANNELS_J4]
    _, Ecm = inp.energies(12)
    pot = dict(V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    pipe = Pipeline(inp.grid_edges(N), channels, Ecm, 3, pot, device=0, channel_J=[inp.channel_sJ(nm)[1] for nm in names])
    scales = inp.sample_scales(3, seed=11)
    pipe.scales.copy_(ctx["torch"].as_tensor(scales))
    pipe.solve_device(); ctx["torch"].cuda.synchronize()
    sig = pipe.sigma.cpu().numpy()
    assert pipe.launches_per_step == 15
    ref, refs, _ = _oracle_sigma(N, channels, names, Ecm, scales[2])
    ok = ~np.isnan(ref)
    for kind, r, _c in refs:
        ok &= hp.swp_edge_distance(r["W"], kind, Ecm) > hp.EDGE_GUARD
    assert ok.sum() >= 10 and (np.abs(sig[2][ok] - ref[ok]) < 1e-9 * ref[ok]).all()



@pytest.mark.parametrize("N", [16, 24, 32, 64, 96])
def test_paper_discretisation_chebyshev_midpoint(ctx, N):
    """NEXT-3: the paper's own set-up -- Chebyshev momentum bins of Eq. 31 (t = 2, alpha = 100 MeV), the
    mid-point potential of Eq. 30 (= the n_gl = 1 rule) and the 8-point bin average of Eq. 29, N_WP = 16..96 (the regime
    of PAPER.md:437-447, several matrices per SM), point-wise and energy-averaged T, uncoupled and coupled."""
    edges = inp.grid_chebyshev(N)
    tl, Ecm = inp.energies(60)
    scales = inp.sample_scales(3, seed=N)
    channels = [(0, 0), (0, 2), (1, 1)]
    for n_gl, mode in ((1, 1), (8, 0), (1, 0)):
        res = _gpu_pipeline(ctx, N, channels, Ecm, scales=scales, S=3, edges=edges, n_gl=n_gl, mode=mode)
        for s, c, kind, lJ in ((0, 0, 0, 0), (2, 1, 0, 2), (1, 0, 1, 1)):
            r = _compare_channel(res, kind, s, c, N, lJ, Ecm, scale=scales[s], label=f"cheb N={N} ngl={n_gl} mode={mode} kind={kind}",
                                 edges=edges, ngl=n_gl, averaged=bool(mode))
            print(f"cheb N={N} ngl={n_gl} mode={mode} kind={kind} lJ={lJ}: H {r[0]:.1e} eig {r[1]:.1e} phase {r[2]:.1e} S {r[3]:.1e}")



@pytest.mark.parametrize("N", [50, 100])
def test_energy_wave_packets(ctx, N):
    """NEXT-4: energy wave packets (wpcd_grid.wp_kind = 1; f = hbarc sqrt(k/mu), N_i = dE_i, Eq. 18 H0):
    same gates as the momentum packets of the configs -- H 1e-12, eigenvalues 1e-11, phases 1e-8 deg -- on the config
    grid and the Chebyshev grid, uncoupled and coupled, plus the Yamaguchi matrix (form factors by quadrature)."""
    tl, Ecm = inp.energies(50)
    scales = inp.sample_scales(2, seed=7)
    channels = [(0, 0), (0, 3), (1, 1), (1, 2)]
    for edges in (None, inp.grid_chebyshev(N)):
        res = _gpu_pipeline(ctx, N, channels, Ecm, scales=scales, S=2, edges=edges, energy_packets=True)
        for s, c, kind, lJ in ((0, 0, 0, 0), (1, 1, 0, 3), (1, 0, 1, 1), (0, 1, 1, 2)):
            r = _compare_channel(res, kind, s, c, N, lJ, Ecm, scale=scales[s], label=f"E-packets N={N} kind={kind} lJ={lJ}",
                                 edges=edges, energy_packets=True)
            print(f"E-packets N={N} cheb={edges is not None} kind={kind} lJ={lJ}: H {r[0]:.1e} eig {r[1]:.1e} phase {r[2]:.1e} S {r[3]:.1e}")
    lamA, lamB = inp.yamaguchi_lambda()
    res = _gpu_pipeline(ctx, N, [(0, 0)], Ecm, yamaguchi=(lamB, inp.YAMAGUCHI_BETA), energy_packets=True)
    _compare_channel(res, 0, 0, 0, N, 0, Ecm, yamaguchi=(lamB, inp.YAMAGUCHI_BETA), label="E-packets Yamaguchi", energy_packets=True)
    # the two kinds of packets really differ (e0 and V), so the test above is not vacuous
    res_k = _gpu_pipeline(ctx, N, [(0, 0)], Ecm)
    res_e = _gpu_pipeline(ctx, N, [(0, 0)], Ecm, energy_packets=True)
    assert np.abs(res_k["e0"] - res_e["e0"]).max() > 1e-3 and np.abs(res_k[0]["H"] - res_e[0]["H"]).max() > 1e-3


def test_pipeline_production_variant_options(ctx):
    """Pipeline(mode=1, n_gl=1, energy_packets=...) runs the paper's production variant (Chebyshev bins, mid-point V,
    energy-averaged T) end to end: phases and sigma_tot against the oracle chain with the same options."""
    from paper_2106_00454_b200.pipeline import Pipeline
    N = 24
    edges = inp.grid_chebyshev(N)
    names = [c[0] for c in inp.CHANNELS_J4]; channels = [(c[1], c[2]) for c in inp.CHANNELS_J4]
    sJ = [inp.channel_sJ(nm) for nm in names]
    _, Ecm = inp.energies(16)
    pot = dict(V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    scales = inp.sample_scales(2, seed=21)
    for ep in (False, True):
        pipe = Pipeline(edges, channels, Ecm, 2, pot, device=0, mode=1, n_gl=1, energy_packets=ep, channel_J=[J for _, J in sJ])
        delta, info = pipe.solve_host(scales)
        sig = pipe.sigma.cpu().numpy()
        s = 1
        S_unc, S_cpl = [], []
        iu = ic = 0
        for (kind, lJ) in channels:
            ch = hp.oracle_channel(N, kind, lJ, scales[s], edges=edges, ngl=1, energy_packets=ep)
            W, C, _ = hp.o.jacobi_ld(ch["H"])       # 80-bit eigenpairs: the arbiter on this grid
            T, b = hp.o.onshell_T(N, kind, ch["Eedge"], ch["V"], W, C, Ecm, averaged=True)
            d, Sm = hp.o.phase_shifts(kind, T, b, ch["dE"])
            g = delta[kind][s * (4 if kind else 10) + (ic if kind else iu)].numpy()
            err = hp.dist180(g, d)
            assert (err[:, :2] if kind else err).max() <= hp.TOL_PHASE_DEG, (ep, kind, lJ)
            (S_cpl if kind else S_unc).append(Sm)
            if kind: ic += 1
            else: iu += 1
        for e, E in enumerate(Ecm):
            p = np.sqrt(E / (inp.HBARC ** 2 / (2 * inp.MU)))
            ref = hp.o.sigma_tot(hp.o.partial_waves(channels, sJ, [S[e] for S in S_unc], [S[e] for S in S_cpl]), p)
            assert abs(sig[s, e] - ref) < 1e-9 * abs(ref), (ep, e, sig[s, e], ref)


def test_mi_solver_on_gpu(ctx):
    """NEXT-4, second half: wpcd_mi_solve (MI method of Sec. 2.1, one CTA per (sample, channel, energy)) against the
    oracle's MI solver: all 14 channels with seeded strength scales, and the Yamaguchi potential against its closed form.
    Tolerance: |dS| <= 1e-10 (both sides solve the same complex linear system in fp64; only the summation order differs)."""
    h, torch = ctx["h"], ctx["torch"]
    channels = [(c[1], c[2]) for c in inp.CHANNELS_J4]
    tl = np.array([1.0, 10.0, 50.0, 150.0, 350.0]); Ecm = tl / 2
    scales = inp.sample_scales(2, seed=4)
    dE = _to_dev(ctx, Ecm)
    for NQ in (24, 48):
        S_unc, S_cpl = h.mi_solve(channels, dE, NQ=NQ, V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V,
                                  muT=inp.TENSOR_MU, VT_scale_idx=2, scales=_to_dev(ctx, scales), S=2)
        torch.cuda.synchronize()
        Su = S_unc.cpu().numpy(); Sc = S_cpl.cpu().numpy()
        Su = Su[..., 0] + 1j * Su[..., 1]; Sc = Sc[..., 0] + 1j * Sc[..., 1]
        worst = 0.0
        for s in range(2):
            V0 = inp.MT_V0 * scales[s, :2]
            iu = ic = 0
            for (kind, lJ) in channels:
                for e, t in enumerate(tl):
                    if not kind:
                        ref, _ = hp.o.mi_solve(t, V0=V0, mu=inp.MT_MU, l_or_J=lJ, NQ=NQ)
                        worst = max(worst, abs(Su[s, iu, e] - ref))
                    else:
                        ref, _ = hp.o.mi_solve(t, coupled=True, V0=V0, mu=inp.MT_MU, l_or_J=lJ, VT=inp.TENSOR_V * scales[s, 2],
                                               muT=inp.TENSOR_MU, NQ=NQ)
                        worst = max(worst, np.abs(Sc[s, ic, e] - ref).max())
                        assert np.abs(Sc[s, ic, e] @ Sc[s, ic, e].conj().T - np.eye(2)).max() < 1e-11   # unitarity (P5)
                if kind: ic += 1
                else: iu += 1
        print(f"MI on the GPU, NQ={NQ}: max |dS| vs oracle {worst:.2e}")
        assert worst < 1e-10
        assert np.abs(np.abs(Su) - 1).max() < 1e-11
    # Yamaguchi: closed form (reading C15)
    lamA, lamB = inp.yamaguchi_lambda()
    S_unc, _ = h.mi_solve([(0, 0)], dE, NQ=96, yamaguchi=(lamB, inp.YAMAGUCHI_BETA))
    Su = S_unc.cpu().numpy(); Su = Su[0, 0, :, 0] + 1j * Su[0, 0, :, 1]
    beta = inp.YAMAGUCHI_BETA; lp = lamA * inp.MU / inp.HBARC ** 2
    for e, t in enumerate(tl):
        p = np.sqrt(inp.MU * t) / inp.HBARC
        Sx = 1 + 4j * lp * p / (p * p + beta * beta) ** 2 / (1 - lp / (beta * (beta - 1j * p) ** 2))
        assert abs(Su[e] - Sx) < 1e-11, (t, Su[e], Sx)
    # systems that do not fit one CTA's shared memory (coupled N_Q > 81, uncoupled N_Q > 164) run with F in an L2-resident
    # workspace region per CTA, a fixed grid looping over the systems: coupled N_Q = 96 and 120, uncoupled
    # N_Q = 200, more systems than CTAs (2 samples x 3 channels x 5 energies here; the loop is also taken with few systems)
    sc2 = inp.sample_scales(2, seed=6)
    for NQ, chans in ((96, [(1, 1), (1, 2), (0, 0)]), (120, [(1, 1)]), (200, [(0, 0), (0, 2)])):
        S_unc, S_cpl = h.mi_solve(chans, dE, NQ=NQ, V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V,
                                  muT=inp.TENSOR_MU, VT_scale_idx=2, scales=_to_dev(ctx, sc2), S=2)
        torch.cuda.synchronize()
        worst, iu, ic = 0.0, 0, 0
        for (kind, lJ) in chans:
            for s in range(2):
                V0 = inp.MT_V0 * sc2[s, :2]
                for e, t in enumerate(tl):
                    if kind:
                        got = S_cpl[s, ic, e].cpu().numpy(); got = got[..., 0] + 1j * got[..., 1]
                        ref, _ = hp.o.mi_solve(t, coupled=True, V0=V0, mu=inp.MT_MU, l_or_J=lJ, VT=inp.TENSOR_V * sc2[s, 2],
                                               muT=inp.TENSOR_MU, NQ=NQ)
                        worst = max(worst, np.abs(got - ref).max())
                    else:
                        got = S_unc[s, iu, e].cpu().numpy(); got = got[0] + 1j * got[1]
                        ref, _ = hp.o.mi_solve(t, V0=V0, mu=inp.MT_MU, l_or_J=lJ, NQ=NQ)
                        worst = max(worst, abs(got - ref))
            if kind: ic += 1
            else: iu += 1
        print(f"MI on the GPU (L2 variant), NQ={NQ}: max |dS| vs oracle {worst:.2e}")
        assert worst < 1e-10
    # more than one thread per row would be needed: refused
    with pytest.raises(RuntimeError):
        h.mi_solve([(1, 1)], dE, NQ=128, V0=inp.MT_V0, mu=inp.MT_MU, VT=inp.TENSOR_V, muT=inp.TENSOR_MU)
    with pytest.raises(RuntimeError):
        h.mi_solve([(0, 0)], dE, NQ=256, V0=inp.MT_V0, mu=inp.MT_MU)
    # wpcd_sigma_tot on S-matrices (d_bin = d_dE = NULL) against the oracle's Clebsch-Gordan chain on the oracle's MI S
    names = [c[0] for c in inp.CHANNELS_J4]; sJ = [inp.channel_sJ(nm) for nm in names]
    S_unc, S_cpl = h.mi_solve(channels, dE, NQ=24, V0=inp.MT_V0, mu=inp.MT_MU, VT=inp.TENSOR_V, muT=inp.TENSOR_MU)
    Ju = [J for (k, _), (_, J) in zip(channels, sJ) if not k]; Jc = [J for (k, _), (_, J) in zip(channels, sJ) if k]
    sig = h.sigma_tot(Ju, S_unc, Jc, S_cpl, None, None, dE).cpu().numpy()[0]
    for e, t in enumerate(tl):
        Su = [hp.o.mi_solve(t, V0=inp.MT_V0, mu=inp.MT_MU, l_or_J=lJ, NQ=24)[0] for (k, lJ) in channels if not k]
        Sc = [hp.o.mi_solve(t, coupled=True, V0=inp.MT_V0, mu=inp.MT_MU, l_or_J=lJ, VT=inp.TENSOR_V, muT=inp.TENSOR_MU, NQ=24)[0]
              for (k, lJ) in channels if k]
        ref = hp.o.sigma_tot(hp.o.partial_waves(channels, sJ, Su, Sc), np.sqrt(inp.MU * t) / inp.HBARC)
        assert abs(sig[e] - ref) < 1e-10 * ref, (t, sig[e], ref)


# ----------------------------------------------------------------------------------------------- large n at production batch
@pytest.mark.parametrize("N,S,picks", [(300, 450, (0, 161, 449)),        # n = 300 and n = 600: the workspace path
                                       (452, 300, (299,))])               # n = 452 / 904: the largest geometry
def test_large_n_batch_exceeds_grid(ctx, N, S, picks):
    """VERDICT r1 missing-5 / ADVICE: the n > 200 kernels at a batch larger than the grid, so that every CTA re-uses its
    global workspace for a second and third matrix (the hand-out counter), in the launch geometry the bench's size sweep
    uses (stored congruently).  All matrices: converged, ascending eigenvalues, trace; the oracle
    (cyclic Jacobi -> T -> phases) on matrices handed out first, second and last.  The coupled matrices (n = 2N) are
    checked by what holds at any size plus, at n = 600, the oracle on the last one."""
    torch, h = ctx["torch"], ctx["h"]
    tl, Ecm = inp.energies(350)
    scales = inp.sample_scales(S, seed=7)
    res = _gpu_pipeline(ctx, N, [(0, 0)], Ecm, scales=scales, S=S)
    g = res[0]
    assert (g["info"] >= 1).all()
    assert (np.diff(g["W"][:, 0, :], axis=1) >= 0).all()
    tr = np.trace(g["H"][:, 0], axis1=1, axis2=2)
    assert np.abs(g["W"][:, 0, :].sum(axis=1) - tr).max() <= 1e-12 * N * np.abs(g["H"]).max()
    for s in picks:
        _compare_channel(res, 0, s, 0, N, 0, Ecm, scale=tuple(scales[s]), label=f"batch>grid N={N} single s={s}")
    del res, g
    # coupled matrices of the same grid (n = 2N), fewer of them (memory: 8 n^2 bytes each for H and C)
    Sc = min(S, 320)
    res = _gpu_pipeline(ctx, N, [(1, 1)], Ecm, scales=scales[:Sc], S=Sc)
    g = res[1]
    n = 2 * N
    assert (g["info"] >= 1).all() and (np.diff(g["W"][:, 0, :], axis=1) >= 0).all()
    for s in (0, 150, Sc - 1):                       # invariants on first-, second- and last-round matrices
        Hs, C, W = g["H"][s, 0], g["C"][s, 0], g["W"][s, 0]
        nrm = np.abs(Hs).max()
        assert np.abs(C.T @ C - np.eye(n)).max() < 1e-12
        assert np.abs(Hs @ C - C * W).max() < 1e-13 * n * nrm
        assert abs(W.sum() - np.trace(Hs)) <= 1e-12 * n * nrm
    if n <= 600:
        _compare_channel(res, 1, Sc - 1, 0, N, 1, Ecm, scale=tuple(scales[Sc - 1]), label=f"batch>grid N={N} coupled s={Sc - 1}")


def test_log_mode_fallback_and_workspace_mode_are_bit_identical(ctx):
    """The three ways the large-n eigensolver can run give the same bits: the log mode (k_jacobi<4>: solve without
    eigenvectors, log the rotation products, replay them panel by panel into C), its fallback (a log region too small for
    the matrix: the matrix is redone by the workspace kernel) and the workspace mode alone.  Same rotations, same products,
    same order of the DMMA accumulations per column of C -- so W, C and info must agree exactly, with and without row
    ranges (rows outside the ranges: zeros).  WPCD_JACOBI_LOG_SWEEPS is the test hook of csrc/jacobi.cu."""
    import os
    torch, h = ctx["torch"], ctx["h"]
    N, S = 150, 40
    scales = torch.as_tensor(inp.sample_scales(S, seed=11), device=ctx["dev"])
    out = h.build_channels(inp.grid_edges(N), [(0, 0), (1, 1)], V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V,
                           muT=inp.TENSOR_MU, VT_scale_idx=2, scales=scales, S=S)
    H = out["H_cpl"].reshape(-1, 2 * N, 2 * N).contiguous()       # n = 300
    runs = {}
    old = os.environ.get("WPCD_JACOBI_LOG_SWEEPS")
    try:
        # capacities of 5 and 6 sweeps' worth sit at these matrices' need (5-6): some are replayed, the others fall back
        for name, val in (("log", None), ("fallback", "1"), ("mixed5", "5"), ("mixed6", "6"), ("workspace", "0")):
            if val is None:
                os.environ.pop("WPCD_JACOBI_LOG_SWEEPS", None)
            else:
                os.environ["WPCD_JACOBI_LOG_SWEEPS"] = val
            for rows in (None, [(10, 95), (160, 245)]):
                W, C, info = h.diag_batched(H, rows=rows)
                torch.cuda.synchronize()
                runs[(name, rows is None)] = (W.cpu().numpy(), C.cpu().numpy(), info.cpu().numpy())
    finally:
        if old is None:
            os.environ.pop("WPCD_JACOBI_LOG_SWEEPS", None)
        else:
            os.environ["WPCD_JACOBI_LOG_SWEEPS"] = old
    W0, C0, i0 = runs[("workspace", True)]
    assert (i0 >= 1).all() and np.abs(np.einsum("bik,bil->bkl", C0[:3], C0[:3]) - np.eye(2 * N)).max() < 1e-12
    for key, (W, C, info) in runs.items():
        assert np.array_equal(W, W0) and np.array_equal(info, i0), key
        if key[1]:
            assert np.array_equal(C, C0), key
        else:
            assert np.array_equal(C[:, 10:95], C0[:, 10:95]) and np.array_equal(C[:, 160:245], C0[:, 160:245]), key
            assert not C[:, :10].any() and not C[:, 95:160].any() and not C[:, 245:].any(), key


@pytest.mark.parametrize("n,batch,max_sweeps", [(201, 1, 30), (207, 3, 30), (333, 5, 30), (256, 2, 2), (505, 2, 30)])
def test_log_mode_edge_cases_against_the_oracle_and_the_workspace_mode(ctx, n, batch, max_sweeps):
    """Log mode at its edges: the smallest size it takes (n = 201), ragged sizes (padding rows in the last panel), batches
    smaller than the grid (every CTA but a few only replays), a sweep limit that stops before convergence (info = -1, the
    log is replayed all the same) and a log capacity of three sweeps' worth, where some matrices are replayed and the others
    go through the fallback launch.  Dense random symmetric matrices (the slowest to converge): invariants against the
    input and eigenvalues against the CPU oracle's Jacobi on the first matrix; every variant bit-identical to the workspace
    mode."""
    import os
    torch, h = ctx["torch"], ctx["h"]
    rng = np.random.default_rng(1000 + n)
    A = rng.standard_normal((batch, n, n)); A = A + A.transpose(0, 2, 1)
    d_A = _to_dev(ctx, A)
    old = os.environ.get("WPCD_JACOBI_LOG_SWEEPS")
    runs = {}
    try:
        for name, val in (("log", None), ("mixed", "3"), ("workspace", "0")):
            if val is None:
                os.environ.pop("WPCD_JACOBI_LOG_SWEEPS", None)
            else:
                os.environ["WPCD_JACOBI_LOG_SWEEPS"] = val
            W, C, info = h.diag_batched(d_A, max_sweeps=max_sweeps)
            torch.cuda.synchronize()
            runs[name] = (W.cpu().numpy(), C.cpu().numpy(), info.cpu().numpy())
    finally:
        if old is None:
            os.environ.pop("WPCD_JACOBI_LOG_SWEEPS", None)
        else:
            os.environ["WPCD_JACOBI_LOG_SWEEPS"] = old
    W0, C0, i0 = runs["workspace"]
    for name in ("log", "mixed"):
        W, C, info = runs[name]
        assert np.array_equal(W, W0) and np.array_equal(C, C0) and np.array_equal(info, i0), name
    W, C, info = runs["log"]
    if max_sweeps < 5:
        assert (info == -1).all()                       # stopped early: still an orthogonal similarity transform
        for b in range(batch):
            assert np.abs(C[b].T @ C[b] - np.eye(n)).max() < 1e-12
        return
    assert (info >= 1).all()
    for b in range(batch):
        nrm = np.abs(A[b]).max()
        assert np.abs(C[b].T @ C[b] - np.eye(n)).max() < 1e-12
        assert np.abs(A[b] @ C[b] - C[b] * W[b]).max() < 1e-13 * n * nrm
    if n <= 340:
        Wo = hp.o.jacobi(A[0])[0]
        assert np.abs(W[0] - Wo).max() <= 1e-12 * n * np.abs(A[0]).max()


def test_pipeline_cuda_graph_replay_and_fp64_probe(ctx):
    """Pipeline.capture(): the pass replayed as a CUDA graph gives bit-identical phase shifts for new inputs written into the
    pipeline's buffers; wpcd_probe_fp64 (the in-run FP64 peak measurement of bench.py) launches and reports its flop count."""
    torch = ctx["torch"]
    from paper_2106_00454_b200.pipeline import Pipeline
    tl, Ecm = inp.energies(50)
    pot = dict(V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    pipe = Pipeline(inp.grid_edges(24), [(0, 0), (1, 1)], Ecm, 3, pot, device=0)
    replay = pipe.capture()
    sc = torch.as_tensor(inp.sample_scales(3, seed=5), device=ctx["dev"])
    pipe.scales.copy_(sc)
    pipe.solve_device(); torch.cuda.synchronize()
    ref = {k: b["delta"].clone() for k, b in pipe.kind.items()}
    for b in pipe.kind.values():
        b["delta"].zero_()
    replay(); torch.cuda.synchronize()
    for k, b in pipe.kind.items():
        assert torch.equal(b["delta"], ref[k]) and bool((b["info"] >= 1).all())
    flops, sink = ctx["h"].probe_fp64(1, 200)
    torch.cuda.synchronize()
    assert flops == sink.numel() / 32 * 200 * 8 * 512 and bool(torch.isfinite(sink).all())


def test_zz_arbitration_only_where_design_allows():
    """Runs last in this module: every case that needed the 80-bit arbiter is on DESIGN.md section 3's list (n >= 600 or
    N >= 400 on the config grid, or the Chebyshev grid); the assertion at the point of use already failed otherwise -- this prints the
    list so that `pytest -q -rA` shows which cases were arbitrated."""
    for label, what, N, n, custom in ARBITRATED:
        assert _arbitration_allowed(N, n, custom), (label, what)
    print("arbitrated cases:", [(l, w) for l, w, _, _, _ in ARBITRATED])
