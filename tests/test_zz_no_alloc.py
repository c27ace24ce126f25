"""wpcd_diag_batched_static (include/wpcd.h): the Jacobi eigensolver of Eq. 21 with its workspace in the
library's file-scope device array, for callers that cannot allocate.  Checked against the existing entry point
wpcd_diag_batched (caller-allocated workspace) on the same WPCD Hamiltonians, within the parity tolerance of
tests/test_gpu_parity.py (eigenvalues 1e-11 relative, componentwise), on calls in a row that reuse the shared array with
different sizes and kernels.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2106_00454_b200 import inputs as inp

pytestmark = pytest.mark.gpu

EIG_RTOL = 1e-11      # north_star's eigenvalue tolerance, as in tests/test_gpu_parity.py
VEC_ATOL = 1e-10      # eigenvector columns (unit norm), up to sign


@pytest.fixture(scope="module")
def ctx():
    import torch
    from paper_2106_00454_b200 import wpcd
    h = wpcd.Handle(0)
    yield dict(torch=torch, wpcd=wpcd, h=h, dev=torch.device("cuda", 0))
    h.close()


def _hamiltonians(ctx, N, S, seed):
    """H of the np channel list (10 uncoupled, 4 coupled) for S potential samples on the config grid:
    ([S*10][N][N], [S*4][2N][2N])."""
    h, torch = ctx["h"], ctx["torch"]
    scales = torch.as_tensor(inp.sample_scales(S, seed=seed), device=ctx["dev"])
    chans = [(c, l) for _, c, l in inp.CHANNELS_J4]
    out = h.build_channels(inp.grid_edges(N), chans, V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V,
                           muT=inp.TENSOR_MU, VT_scale_idx=2, scales=scales, S=S)
    return out["H_unc"].reshape(-1, N, N).contiguous(), out["H_cpl"].reshape(-1, 2 * N, 2 * N).contiguous()


def _outputs(ctx, batch, n):
    torch, dev = ctx["torch"], ctx["dev"]
    # poisoned, so that an entry point that wrote nothing cannot pass
    return (torch.full((batch, n), float("nan"), dtype=torch.float64, device=dev),
            torch.full((batch, n, n), float("nan"), dtype=torch.float64, device=dev),
            torch.full((batch,), -7, dtype=torch.int32, device=dev))


def _compare(ctx, H, rows=None):
    """One call of the static entry point against the existing path on the same matrices."""
    h, torch = ctx["h"], ctx["torch"]
    batch, n = H.shape[0], H.shape[-1]
    assert h.diag_workspace_bytes(n, batch) <= h.STATIC_WORK_BYTES
    W1, C1, i1 = h.diag_batched_static(H, *_outputs(ctx, batch, n), rows=rows)
    W0, C0, i0 = h.diag_batched(H, rows=rows)
    torch.cuda.synchronize()
    W0, W1, C0, C1 = (x.cpu().numpy() for x in (W0, W1, C0, C1))
    assert np.array_equal(i0.cpu().numpy(), i1.cpu().numpy()) and (i1.cpu().numpy() >= 1).all()
    assert np.all(np.isfinite(W1)) and np.all(np.isfinite(C1))
    assert np.all(np.abs(W1 - W0) <= EIG_RTOL * np.abs(W0)), np.abs(W1 / W0 - 1).max()
    err = np.minimum(np.abs(C1 - C0).max(axis=1), np.abs(C1 + C0).max(axis=1))     # per (matrix, column), up to sign
    assert err.max() <= VEC_ATOL, err.max()
    return W1


def test_static_workspace_matches_existing_path_on_calls_in_a_row(ctx):
    """Calls in a row share the one array, which keeps the previous call's contents: block kernel n = 100 (10 matrices),
    then n = 200 (4: other tables, other per-CTA stride), then n = 100 again on OTHER matrices, then the small kernel
    (n = 24: only the work counter) and n = 48; every call must agree with the existing path."""
    Hu_a, Hc_a = _hamiltonians(ctx, 100, 1, seed=3)
    Hu_b, _ = _hamiltonians(ctx, 100, 2, seed=4)
    Wa = _compare(ctx, Hu_a)
    _compare(ctx, Hc_a)
    Wb = _compare(ctx, Hu_b[10:])
    assert not np.array_equal(Wa, Wb)                  # the second n = 100 call really had other inputs
    Hu_s, Hc_s = _hamiltonians(ctx, 24, 40, seed=5)    # 400 x (24 x 24), 160 x (48 x 48)
    _compare(ctx, Hu_s)
    _compare(ctx, Hc_s)
    # the same call twice: identical results (nothing left over from the first one matters)
    W1 = _compare(ctx, Hu_a)
    assert np.array_equal(W1, Wa)
    # the row-range variant of the on-shell path goes through the same workspace
    _compare(ctx, Hu_a, rows=[(0, 40)])


def test_static_workspace_rejects_sizes_beyond_the_array(ctx):
    """WPCD_ESIZE before any launch when wpcd_diag_workspace_bytes(n, batch) > WPCD_STATIC_WORK_BYTES, with the sizes in
    the error text; the outputs stay untouched."""
    h, torch, wpcd = ctx["h"], ctx["torch"], ctx["wpcd"]
    n, batch = 100, 512
    assert h.diag_workspace_bytes(n, batch) > h.STATIC_WORK_BYTES
    H = torch.zeros((batch, n, n), dtype=torch.float64, device=ctx["dev"])
    W, C, info = _outputs(ctx, batch, n)
    with pytest.raises(wpcd.WpcdError) as e:
        h.diag_batched_static(H, W, C, info)
    assert "unsupported size" in str(e.value) and "static array holds 16777216" in str(e.value)
    torch.cuda.synchronize()
    assert (info.cpu().numpy() == -7).all() and np.isnan(W.cpu().numpy()).all()
    # the largest batch that fits at this n is accepted (limit stated in include/wpcd.h)
    fit = max(b for b in range(1, 512) if h.diag_workspace_bytes(n, b) <= h.STATIC_WORK_BYTES)
    assert fit == 193
    assert max(b for b in range(1, 200) if h.diag_workspace_bytes(200, b) <= h.STATIC_WORK_BYTES) == 52
    assert h.diag_workspace_bytes(32, 1 << 20) <= h.STATIC_WORK_BYTES


def test_static_workspace_call_is_capturable(ctx):
    """The reason for the entry point: a cudaMalloc inside a stream capture fails the capture.  After one warm call (the
    array's device address is looked up once per device) the call is captured into a CUDA graph and replayed twice on
    new inputs written into the same buffers."""
    h, torch = ctx["h"], ctx["torch"]
    Hu, _ = _hamiltonians(ctx, 100, 2, seed=9)
    Hbuf = Hu[:10].clone()
    W, C, info = _outputs(ctx, 10, 100)
    h.diag_batched_static(Hbuf, W, C, info)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            h.diag_batched_static(Hbuf, W, C, info, stream=s)
    for part in (Hu[10:], Hu[:10]):
        Hbuf.copy_(part)
        W.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        W0, _, _ = h.diag_batched(part)
        torch.cuda.synchronize()
        W0, W1 = W0.cpu().numpy(), W.cpu().numpy()
        assert np.all(np.abs(W1 - W0) <= EIG_RTOL * np.abs(W0))
