"""Thin ctypes binding of libwpcd.so (include/wpcd.h): argument marshalling only -- every step runs in the CUDA
kernels.  torch is used for device memory and streams.  Fails loudly if the library is missing; no CPU fallback."""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# WPCD_LIBRARY selects another build of the same C ABI (e.g. one compiled with -DWPCD_PROFILE)
_LIBPATH = os.environ.get("WPCD_LIBRARY") or os.path.join(_HERE, "libwpcd.so")

MAX_TERMS = 4
MAX_CHANNELS = 16


class WpcdError(RuntimeError):
    pass


if not os.path.exists(_LIBPATH):
    raise WpcdError(f"{_LIBPATH} is missing: build it with `python -m paper_2106_00454_b200.build` "
                    "(or __graft_entry__.build()); there is no CPU fallback")
_lib = C.CDLL(_LIBPATH)


class Potential(C.Structure):
    _fields_ = [("kind", C.c_int), ("n_terms", C.c_int), ("V0", C.POINTER(C.c_double)), ("mu", C.POINTER(C.c_double)),
                ("scale_idx", C.POINTER(C.c_int)), ("VT", C.c_double), ("muT", C.c_double), ("VT_scale_idx", C.c_int),
                ("lambda_", C.c_double), ("beta", C.c_double)]


class Channel(C.Structure):
    _fields_ = [("coupled", C.c_int), ("lJ", C.c_int)]


class Grid(C.Structure):
    _fields_ = [("N", C.c_int), ("h_edges", C.POINTER(C.c_double)), ("hbarc", C.c_double), ("mu", C.c_double),
                ("n_gl", C.c_int), ("wp_kind", C.c_int)]


_vp, _sz, _i, _d = C.c_void_p, C.c_size_t, C.c_int, C.c_double
_lib.wpcd_create.argtypes = [C.POINTER(_vp), _i]; _lib.wpcd_create.restype = _i
_lib.wpcd_destroy.argtypes = [_vp]; _lib.wpcd_destroy.restype = None
_lib.wpcd_strerror.argtypes = [_i]; _lib.wpcd_strerror.restype = C.c_char_p
_lib.wpcd_last_cuda_error.argtypes = [_vp]; _lib.wpcd_last_cuda_error.restype = C.c_char_p
_lib.wpcd_num_sms.argtypes = [_vp]; _lib.wpcd_num_sms.restype = _i
_lib.wpcd_build_workspace_bytes.argtypes = [_vp, _i, _i]; _lib.wpcd_build_workspace_bytes.restype = _sz
_lib.wpcd_diag_workspace_bytes.argtypes = [_vp, _i, _i]; _lib.wpcd_diag_workspace_bytes.restype = _sz
_lib.wpcd_onshell_workspace_bytes.argtypes = [_vp, _i, _i, _i, _i]; _lib.wpcd_onshell_workspace_bytes.restype = _sz
_lib.wpcd_build_channels.argtypes = [_vp, C.POINTER(Grid), C.POINTER(Potential), C.POINTER(Channel), _i, _vp, _i, _i,
                                     _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.wpcd_build_channels.restype = _i
_lib.wpcd_diag_batched.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _d, _i, C.POINTER(_i), _i, _vp, _sz, _vp]
_lib.wpcd_diag_batched.restype = _i
_lib.wpcd_diag_batched_static.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _d, _i, C.POINTER(_i), _i, _vp]
_lib.wpcd_diag_batched_static.restype = _i
_lib.wpcd_onshell_T.argtypes = [_vp, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _i, _i, _vp, _vp, _vp, _sz, _vp]
_lib.wpcd_onshell_T.restype = _i
_lib.wpcd_phase_shifts.argtypes = [_vp, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.wpcd_phase_shifts.restype = _i
_lib.wpcd_interp_phases.argtypes = [_vp, _i, _i, _i, _vp, _vp, _vp, _i, _vp, _vp]
_lib.wpcd_interp_phases.restype = _i
_lib.wpcd_onshell_rows.argtypes = [C.POINTER(Grid), _i, C.POINTER(_d), _i, C.POINTER(_i), C.POINTER(_i)]
_lib.wpcd_onshell_rows.restype = _i
_lib.wpcd_sigma_tot.argtypes = [_vp, _i, _i, _i, C.POINTER(_i), _vp, _i, C.POINTER(_i), _vp, _vp, _vp, _vp, _d, _d, _vp, _vp]
_lib.wpcd_sigma_tot.restype = _i
_lib.wpcd_mi_workspace_bytes.argtypes = [_vp, _i]; _lib.wpcd_mi_workspace_bytes.restype = _sz
_lib.wpcd_mi_solve.argtypes = [_vp, C.POINTER(Potential), C.POINTER(Channel), _i, _vp, _i, _i, _i, _d, _d, _d, _vp, _i, _vp,
                               _vp, _vp, _sz, _vp]
_lib.wpcd_mi_solve.restype = _i

_lib.wpcd_probe_sink_elems.argtypes = [_vp]; _lib.wpcd_probe_sink_elems.restype = _sz
_lib.wpcd_probe_fp64.argtypes = [_vp, _i, _i, _vp, C.POINTER(_d), _vp]; _lib.wpcd_probe_fp64.restype = _i

# every symbol include/wpcd.h declares (tests/test_abi_cpu.py compares this list with the header and the library)
EXPORTS = ["wpcd_create", "wpcd_destroy", "wpcd_strerror", "wpcd_last_cuda_error", "wpcd_num_sms",
           "wpcd_build_workspace_bytes", "wpcd_diag_workspace_bytes", "wpcd_onshell_workspace_bytes",
           "wpcd_build_channels", "wpcd_diag_batched", "wpcd_diag_batched_static", "wpcd_onshell_T", "wpcd_phase_shifts", "wpcd_onshell_rows",
           "wpcd_interp_phases", "wpcd_sigma_tot", "wpcd_mi_workspace_bytes", "wpcd_mi_solve",
           "wpcd_probe_sink_elems", "wpcd_probe_fp64", "wpcd_jacobi_schedule", "wpcd_jacobi_critical_slot"]


def _ptr(t):
    return None if t is None else t.data_ptr()


def _stream(stream, device=None):
    s = stream if stream is not None else torch.cuda.current_stream(device)
    return s.cuda_stream


class Handle:
    """wpcd_create / wpcd_destroy."""

    def __init__(self, device=0):
        self._h = _vp()
        self.device = torch.device("cuda", device)
        rc = _lib.wpcd_create(C.byref(self._h), device)
        if rc != 0:
            raise WpcdError(f"wpcd_create failed: {_lib.wpcd_strerror(rc).decode()} (is a B200 visible?)")

    def close(self):
        if self._h:
            _lib.wpcd_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc != 0:
            raise WpcdError(f"{what}: {_lib.wpcd_strerror(rc).decode()} {_lib.wpcd_last_cuda_error(self._h).decode()}")

    def num_sms(self):
        return _lib.wpcd_num_sms(self._h)

    def probe_fp64(self, kind=1, iters=20000, stream=None, sink=None):
        """wpcd_probe_fp64: launches the register-only fp64 chain kernel (kind 0 DFMA, 1 DMMA); returns the flops of the
        launch.  The caller times it with CUDA events."""
        if sink is None:
            sink = torch.empty(_lib.wpcd_probe_sink_elems(self._h), dtype=torch.float64, device=self.device)
        fl = _d(0.0)
        self._check(_lib.wpcd_probe_fp64(self._h, kind, iters, _ptr(sink), C.byref(fl), _stream(stream, self.device)), "wpcd_probe_fp64")
        return fl.value, sink

    def _work(self, nbytes):
        return torch.empty(max(int(nbytes), 16), dtype=torch.uint8, device=self.device)

    # ------------------------------------------------------------------ wpcd_build_channels
    def build_channels(self, edges, channels, V0=None, mu=None, scale_idx=None, VT=0.0, muT=1.0, VT_scale_idx=-1,
                       yamaguchi=None, scales=None, S=1, hbarc=197.327, mured=469.46, n_gl=8, stream=None, out=None,
                       energy_packets=False):
        """edges: host sequence [N+1]; channels: list of (coupled, lJ); scales: device tensor [S][P] or None.
        Returns dict(H_unc, H_cpl, e0, dE, Eedge) of device tensors."""
        N = len(edges) - 1
        if hasattr(edges, "ctypes") and edges.dtype.name == "float64" and edges.flags["C_CONTIGUOUS"]:
            # the caller's array is used in place: the library copies it to the device asynchronously (a captured CUDA graph
            # replays that copy, so the array has to outlive the graph -- Pipeline keeps it)
            h_edges = edges.ctypes.data_as(C.POINTER(C.c_double))
        else:
            h_edges = (C.c_double * (N + 1))(*[float(x) for x in edges])
        grid = Grid(N, h_edges, hbarc, mured, n_gl, 1 if energy_packets else 0)
        pot = Potential()
        keep = []
        if yamaguchi is not None:
            pot.kind = 1; pot.n_terms = 0; pot.lambda_, pot.beta = float(yamaguchi[0]), float(yamaguchi[1])
            pot.VT_scale_idx = -1; pot.muT = 1.0
        else:
            nt = len(V0)
            a = (C.c_double * nt)(*[float(x) for x in V0]); b = (C.c_double * nt)(*[float(x) for x in mu])
            keep += [a, b]
            pot.kind = 0; pot.n_terms = nt; pot.V0 = a; pot.mu = b
            if scale_idx is not None:
                c = (C.c_int * nt)(*[int(x) for x in scale_idx]); keep.append(c); pot.scale_idx = c
            pot.VT, pot.muT, pot.VT_scale_idx = float(VT), float(muT), int(VT_scale_idx)
        nch = len(channels)
        ch = (Channel * nch)(*[Channel(int(c), int(l)) for c, l in channels])
        n_unc = sum(1 for c, _ in channels if not c); n_cpl = nch - n_unc
        P = 0 if scales is None else scales.shape[1]
        dev = self.device
        if out is None:
            out = dict(
                H_unc=torch.empty((S, n_unc, N, N), dtype=torch.float64, device=dev) if n_unc else None,
                H_cpl=torch.empty((S, n_cpl, 2 * N, 2 * N), dtype=torch.float64, device=dev) if n_cpl else None,
                e0=torch.empty(N, dtype=torch.float64, device=dev), dE=torch.empty(N, dtype=torch.float64, device=dev),
                Eedge=torch.empty(N + 1, dtype=torch.float64, device=dev))
        wb = _lib.wpcd_build_workspace_bytes(self._h, N, nch)
        work = out.get("work")
        if work is None or work.numel() < wb:
            work = self._work(wb); out["work"] = work
        rc = _lib.wpcd_build_channels(self._h, C.byref(grid), C.byref(pot), ch, nch, _ptr(scales), S, P,
                                      _ptr(out["H_unc"]), _ptr(out["H_cpl"]), _ptr(out["e0"]), _ptr(out["dE"]),
                                      _ptr(out["Eedge"]), _ptr(work), work.numel(), _stream(stream, self.device))
        self._check(rc, "wpcd_build_channels")
        return out

    # ------------------------------------------------------------------ wpcd_mi_solve
    def mi_solve(self, channels, Ecm, NQ=96, V0=None, mu=None, scale_idx=None, VT=0.0, muT=1.0, VT_scale_idx=-1,
                 yamaguchi=None, scales=None, S=1, cmap=1.0, hbarc=197.327, mured=469.46, stream=None):
        """MI method (Sec. 2.1) for every (sample, channel, energy); the potential arguments are those of build_channels
        (yamaguchi = (lambda_B, beta)).  Returns (S_unc [S][n_unc][nE][2], S_cpl [S][n_cpl][nE][2][2][2]) device tensors."""
        pot = Potential()
        keep = []
        if yamaguchi is not None:
            pot.kind = 1; pot.n_terms = 0; pot.lambda_, pot.beta = float(yamaguchi[0]), float(yamaguchi[1])
            pot.VT_scale_idx = -1; pot.muT = 1.0
        else:
            nt = len(V0)
            a = (C.c_double * nt)(*[float(x) for x in V0]); b = (C.c_double * nt)(*[float(x) for x in mu])
            keep += [a, b]
            pot.kind = 0; pot.n_terms = nt; pot.V0 = a; pot.mu = b
            if scale_idx is not None:
                c = (C.c_int * nt)(*[int(x) for x in scale_idx]); keep.append(c); pot.scale_idx = c
            pot.VT, pot.muT, pot.VT_scale_idx = float(VT), float(muT), int(VT_scale_idx)
        nch = len(channels)
        ch = (Channel * nch)(*[Channel(int(c), int(l)) for c, l in channels])
        n_unc = sum(1 for c, _ in channels if not c); n_cpl = nch - n_unc
        P = 0 if scales is None else scales.shape[1]
        nE = Ecm.shape[0]; dev = self.device
        S_unc = torch.empty((S, n_unc, nE, 2), dtype=torch.float64, device=dev) if n_unc else None
        S_cpl = torch.empty((S, n_cpl, nE, 2, 2, 2), dtype=torch.float64, device=dev) if n_cpl else None
        work = self._work(_lib.wpcd_mi_workspace_bytes(self._h, int(NQ)))
        rc = _lib.wpcd_mi_solve(self._h, C.byref(pot), ch, nch, _ptr(scales), S, P, int(NQ), float(cmap), float(hbarc),
                                float(mured), _ptr(Ecm), nE, _ptr(S_unc), _ptr(S_cpl), _ptr(work), work.numel(), _stream(stream, self.device))
        self._check(rc, "wpcd_mi_solve")
        return S_unc, S_cpl

    # ------------------------------------------------------------------ wpcd_diag_batched
    def diag_workspace_bytes(self, n, batch):
        return _lib.wpcd_diag_workspace_bytes(self._h, n, batch)

    def diag_batched(self, A, tol=0.0, max_sweeps=30, stream=None, W=None, Cm=None, info=None, work=None, rows=None):
        """A: device tensor [batch][n][n] (read only).  Returns (W [batch][n] ascending, C [batch][n][n], info).
        rows: optional list of up to 4 (lo, hi) row ranges of C that are needed (the other rows come back as zeros)."""
        batch, n = A.shape[0], A.shape[-1]
        dev = A.device
        W = torch.empty((batch, n), dtype=torch.float64, device=dev) if W is None else W
        Cm = torch.empty((batch, n, n), dtype=torch.float64, device=dev) if Cm is None else Cm
        info = torch.empty(batch, dtype=torch.int32, device=dev) if info is None else info
        wb = _lib.wpcd_diag_workspace_bytes(self._h, n, batch)
        if work is None or work.numel() < wb:
            work = self._work(wb)
        nr = 0 if rows is None else len(rows)
        h_rows = (_i * (2 * nr))(*[int(x) for r in rows for x in r]) if nr else None
        rc = _lib.wpcd_diag_batched(self._h, n, batch, _ptr(A), _ptr(W), _ptr(Cm), _ptr(info), float(tol), int(max_sweeps),
                                    h_rows, nr, _ptr(work), work.numel(), _stream(stream, self.device))
        self._check(rc, "wpcd_diag_batched")
        return W, Cm, info

    STATIC_WORK_BYTES = 16 << 20   # WPCD_STATIC_WORK_BYTES of include/wpcd.h

    def diag_batched_static(self, A, W, Cm, info, tol=0.0, max_sweeps=30, stream=None, rows=None):
        """wpcd_diag_batched_static: diag_batched with the workspace in the library's static device array -- the call
        allocates nothing, so the outputs W [batch][n], Cm [batch][n][n], info [batch] (int32) are the caller's.  Sizes with
        diag_workspace_bytes(n, batch) > STATIC_WORK_BYTES raise WpcdError; calls that overlap on the GPU race."""
        batch, n = A.shape[0], A.shape[-1]
        nr = 0 if rows is None else len(rows)
        h_rows = (_i * (2 * nr))(*[int(x) for r in rows for x in r]) if nr else None
        rc = _lib.wpcd_diag_batched_static(self._h, n, batch, _ptr(A), _ptr(W), _ptr(Cm), _ptr(info), float(tol),
                                           int(max_sweeps), h_rows, nr, _stream(stream, self.device))
        self._check(rc, "wpcd_diag_batched_static")
        return W, Cm, info

    # ------------------------------------------------------------------ wpcd_onshell_T
    def onshell_T(self, N, coupled, e0, Eedge, H, W, Cm, Ecm, stream=None, T=None, bins=None, work=None, mode=0):
        """mode 0: point-wise resolvent; mode 1: energy-averaged resolvent (one T per on-shell bin)."""
        batch = H.shape[0]; nE = Ecm.shape[0]; dev = H.device
        shape = (batch, nE, 2, 2, 2) if coupled else (batch, nE, 2)
        T = torch.empty(shape, dtype=torch.float64, device=dev) if T is None else T
        bins = torch.empty(nE, dtype=torch.int32, device=dev) if bins is None else bins
        wb = _lib.wpcd_onshell_workspace_bytes(self._h, N, int(coupled), batch, nE)
        if work is None or work.numel() < wb:
            work = self._work(wb)
        rc = _lib.wpcd_onshell_T(self._h, N, int(coupled), batch, _ptr(e0), _ptr(Eedge), _ptr(H), _ptr(W), _ptr(Cm),
                                 _ptr(Ecm), nE, int(mode), _ptr(T), _ptr(bins), _ptr(work), work.numel(), _stream(stream, self.device))
        self._check(rc, "wpcd_onshell_T")
        return T, bins

    # ------------------------------------------------------------------ wpcd_onshell_rows
    def onshell_rows(self, edges, coupled, Ecm, hbarc=197.327, mu=469.46):
        """Row ranges of C that onshell_T will read for the (host) energies Ecm; None = all rows."""
        import numpy as np
        e = np.ascontiguousarray(edges, dtype=np.float64); E = np.ascontiguousarray(Ecm, dtype=np.float64)
        g = Grid(len(e) - 1, e.ctypes.data_as(C.POINTER(_d)), hbarc, mu, 8)
        rows = (_i * 8)(); nr = _i(0)
        self._check(_lib.wpcd_onshell_rows(C.byref(g), int(coupled), E.ctypes.data_as(C.POINTER(_d)), len(E), rows, C.byref(nr)),
                    "wpcd_onshell_rows")
        return [(rows[2 * r], rows[2 * r + 1]) for r in range(nr.value)] or None

    # ------------------------------------------------------------------ wpcd_interp_phases
    def interp_phases(self, coupled, pedge, delta_mid, q, stream=None, out=None):
        """Eq. 42: delta_mid [batch][N] (or [batch][N][3]) at the bin mid-points -> phases at momenta q [nq]."""
        batch, N = delta_mid.shape[0], delta_mid.shape[1]; nq = q.shape[0]; dev = delta_mid.device
        shape = (batch, nq, 3) if coupled else (batch, nq)
        out = torch.empty(shape, dtype=torch.float64, device=dev) if out is None else out
        rc = _lib.wpcd_interp_phases(self._h, int(coupled), batch, N, _ptr(pedge), _ptr(delta_mid), _ptr(q), nq, _ptr(out),
                                     _stream(stream, self.device))
        self._check(rc, "wpcd_interp_phases")
        return out

    # ------------------------------------------------------------------ wpcd_sigma_tot
    def sigma_tot(self, J_unc, T_unc, J_cpl, T_cpl, bins, dE, Ecm, hbarc=197.327, mu=469.46, stream=None, out=None):
        """Eqs. A.2, A.9, A.11: total np cross section [S][nE] in mb from T_unc [S][n_unc][nE][2] and
        T_cpl [S][n_cpl][nE][2][2][2] (either may be None); J_unc / J_cpl: total J of every channel."""
        n_unc, n_cpl = len(J_unc), len(J_cpl)
        ref = T_unc if T_unc is not None else T_cpl
        nE = Ecm.shape[0]
        if ref is None:  # no channels at all: let the library report the argument error
            S = 1 if out is None else out.shape[0]
        else:
            S = ref.numel() // (max(n_unc if T_unc is not None else n_cpl, 1) * nE * (2 if T_unc is not None else 8))
        out = torch.empty((S, nE), dtype=torch.float64, device=Ecm.device) if out is None else out
        ju = (_i * max(n_unc, 1))(*[int(j) for j in J_unc]); jc = (_i * max(n_cpl, 1))(*[int(j) for j in J_cpl])
        rc = _lib.wpcd_sigma_tot(self._h, S, nE, n_unc, ju, _ptr(T_unc), n_cpl, jc, _ptr(T_cpl), _ptr(bins), _ptr(dE),
                                 _ptr(Ecm), float(hbarc), float(mu), _ptr(out), _stream(stream, self.device))
        self._check(rc, "wpcd_sigma_tot")
        return out

    # ------------------------------------------------------------------ wpcd_phase_shifts
    def phase_shifts(self, coupled, T, bins, dE, want_S=True, stream=None, delta=None, S=None):
        batch, nE = T.shape[0], T.shape[1]; dev = T.device
        shape = (batch, nE, 3) if coupled else (batch, nE)
        delta = torch.empty(shape, dtype=torch.float64, device=dev) if delta is None else delta
        if want_S and S is None:
            S = torch.empty_like(T)
        rc = _lib.wpcd_phase_shifts(self._h, int(coupled), batch, nE, _ptr(T), _ptr(bins), _ptr(dE), _ptr(delta),
                                    _ptr(S), _stream(stream, self.device))
        self._check(rc, "wpcd_phase_shifts")
        return delta, S
