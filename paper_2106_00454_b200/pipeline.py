"""Batched WPCD pipeline on one GPU: the four C-ABI calls in sequence with preallocated device buffers.

This is host orchestration only (buffer ownership, streams, events); every arithmetic step runs in the CUDA kernels
behind include/wpcd.h.  `solve_device` keeps inputs and outputs in HBM; `solve_host` is the end-to-end user call with
pinned host buffers (scales in, phase shifts out) and the copies inside.
"""
import numpy as np
import torch

from . import wpcd


class Pipeline:
    """Channels x samples -> phase shifts.  channels: list of (coupled, lJ); potential: dict for build_channels."""

    KERNELS_PER_STEP_FIXED = 2  # k_grid, k_basis

    def __init__(self, edges, channels, Ecm, S, potential, n_scale_cols=3, device=0, max_sweeps=30, tol=0.0,
                 onshell_rows_only=True, channel_J=None, mode=0, n_gl=8, energy_packets=False):
        self.h = wpcd.Handle(device)
        self.dev = self.h.device
        self.edges = np.ascontiguousarray(edges, dtype=np.float64)
        self.N = len(self.edges) - 1
        self.channels = list(channels)
        self.S = int(S)
        self.potential = dict(potential)
        self.max_sweeps, self.tol = max_sweeps, tol
        # mode 1: energy-averaged resolvent (the paper's production variant); n_gl = 1: mid-point potential (Eq. 30)
        self.mode, self.n_gl, self.energy_packets = int(mode), int(n_gl), bool(energy_packets)
        self.n_unc = sum(1 for c, _ in self.channels if not c)
        self.n_cpl = len(self.channels) - self.n_unc
        N, f64 = self.N, torch.float64
        self.nE = len(Ecm)
        # rows of C the on-shell kernel will read (library decides; None = all): C <- C J is row-independent, so the
        # eigenvector update can skip the rest (wpcd_diag_batched h_rows)
        self.rows = {k: (self.h.onshell_rows(self.edges, k, np.asarray(Ecm, dtype=np.float64)) if onshell_rows_only else None)
                     for k in (0, 1)}
        self.Ecm = torch.as_tensor(np.ascontiguousarray(Ecm, dtype=np.float64), device=self.dev)
        self.scales = torch.ones((self.S, n_scale_cols), dtype=f64, device=self.dev)
        self.geo = dict(e0=torch.empty(N, dtype=f64, device=self.dev), dE=torch.empty(N, dtype=f64, device=self.dev),
                        Eedge=torch.empty(N + 1, dtype=f64, device=self.dev), H_unc=None, H_cpl=None)
        self.kind = {}
        for kind, nch in ((0, self.n_unc), (1, self.n_cpl)):
            if not nch:
                continue
            n = (2 * N) if kind else N
            batch = self.S * nch
            H = torch.empty((self.S, nch, n, n), dtype=f64, device=self.dev)
            self.geo["H_cpl" if kind else "H_unc"] = H
            wb = self.h.diag_workspace_bytes(n, batch)
            self.kind[kind] = dict(
                n=n, batch=batch, nch=nch, H=H.view(batch, n, n),
                W=torch.empty((batch, n), dtype=f64, device=self.dev), C=torch.empty((batch, n, n), dtype=f64, device=self.dev),
                info=torch.empty(batch, dtype=torch.int32, device=self.dev),
                work=torch.empty(max(wb, 16), dtype=torch.uint8, device=self.dev),
                T=torch.empty((batch, self.nE, 2, 2, 2) if kind else (batch, self.nE, 2), dtype=f64, device=self.dev),
                bins=torch.empty(self.nE, dtype=torch.int32, device=self.dev),
                owork=torch.empty(256, dtype=torch.uint8, device=self.dev),
                delta=torch.empty((batch, self.nE, 3) if kind else (batch, self.nE), dtype=f64, device=self.dev))
        # optional epilogue: total cross section from all channels; channel_J = total J per channel
        self.J = None
        if channel_J is not None:
            self.J = {k: [int(J) for (c, _), J in zip(self.channels, channel_J) if bool(c) == bool(k)] for k in (0, 1)}
            self.sigma = torch.empty((self.S, self.nE), dtype=f64, device=self.dev)
        # pinned host buffers of the end-to-end call
        self.h_scales = torch.empty((self.S, n_scale_cols), dtype=f64).pin_memory()
        self.h_delta = {k: torch.empty(v["delta"].shape, dtype=f64).pin_memory() for k, v in self.kind.items()}
        self.h_info = {k: torch.empty(v["info"].shape, dtype=torch.int32).pin_memory() for k, v in self.kind.items()}
        # the device->host copies of one kind's results run on a side stream while the next kind is diagonalised
        self.copy_stream = torch.cuda.Stream(device=self.dev)
        self.done = {k: torch.cuda.Event() for k in self.kind}

    @property
    def channel_solves(self):
        return self.S * len(self.channels)

    @property
    def launches_per_step(self):
        # k_grid, k_basis, k_combine per kind; k_schedule, k_jacobi, k_bins, k_onshell, k_phase per kind; the eigensolver's
        # log mode (200 < n <= 848, csrc/jacobi.cu) adds k_sched_init, k_set_counter, the fallback launch of k_jacobi and
        # k_log_watchdog
        extra = sum(4 for b in self.kind.values() if 200 < b["n"] <= 848)
        return 2 + len(self.kind) * 6 + extra + (1 if self.J is not None else 0)

    def solve_device(self, events=None, to_host=False):
        """One pass of the whole hot path with inputs resident in HBM.  events: optional dict name -> (start, end)
        torch.cuda.Event pairs recorded on the current stream around each stage.  to_host: as soon as a kind's phase
        shifts are complete they are copied to the pinned host buffers on the side stream (overlapping the next kind)."""
        def rec(name, which):
            if events is not None:
                events[name][which].record()
        p = self.potential
        rec("build", 0)
        self.h.build_channels(self.edges, self.channels, scales=self.scales, S=self.S, out=self.geo, n_gl=self.n_gl,
                              energy_packets=self.energy_packets, **p)
        rec("build", 1)
        for kind, b in self.kind.items():
            tag = "cpl" if kind else "unc"
            rec("diag_" + tag, 0)
            self.h.diag_batched(b["H"], tol=self.tol, max_sweeps=self.max_sweeps, W=b["W"], Cm=b["C"], info=b["info"], work=b["work"],
                                rows=self.rows[kind])
            rec("diag_" + tag, 1)
            rec("onshell_" + tag, 0)
            self.h.onshell_T(self.N, kind, self.geo["e0"], self.geo["Eedge"], b["H"], b["W"], b["C"], self.Ecm,
                             T=b["T"], bins=b["bins"], work=b["owork"], mode=self.mode)
            self.h.phase_shifts(kind, b["T"], b["bins"], self.geo["dE"], want_S=False, delta=b["delta"])
            rec("onshell_" + tag, 1)
            if to_host:
                self.done[kind].record()
                with torch.cuda.stream(self.copy_stream):
                    self.copy_stream.wait_event(self.done[kind])
                    self.h_delta[kind].copy_(b["delta"], non_blocking=True)
                    self.h_info[kind].copy_(b["info"], non_blocking=True)
        if self.J is not None:
            any_kind = next(iter(self.kind.values()))
            self.h.sigma_tot(self.J[0], self.kind[0]["T"] if 0 in self.kind else None, self.J[1],
                             self.kind[1]["T"] if 1 in self.kind else None, any_kind["bins"], self.geo["dE"], self.Ecm,
                             out=self.sigma)

    def capture(self):
        """Captures one pass (solve_device) into a CUDA graph: the pass is a fixed sequence of 14-15 small launches on
        preallocated buffers, so for ONE potential sample (the paper's Table-1 use, latency bound) replaying the graph removes
        the launch overhead.  Returns a callable that replays it on the current stream."""
        for _ in range(2):
            self.solve_device()          # warm-up outside the capture (function attributes, lazy module loading)
        torch.cuda.synchronize(self.dev)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            self.solve_device()
        self.graph = graph
        return graph.replay

    def stage_names(self):
        names = ["build"]
        for kind in self.kind:
            tag = "cpl" if kind else "unc"
            names += ["diag_" + tag, "onshell_" + tag]
        return names

    def solve_host(self, scales_host):
        """End-to-end user call: host scales [S][P] -> host phase shifts (pinned buffers), copies included."""
        self.h_scales.copy_(torch.as_tensor(scales_host))
        self.scales.copy_(self.h_scales, non_blocking=True)
        self.solve_device(to_host=True)
        self.copy_stream.synchronize()
        torch.cuda.current_stream(self.dev).synchronize()
        return self.h_delta, self.h_info

    def h2d_bytes(self):
        return self.h_scales.numel() * 8

    def d2h_bytes(self):
        return sum(t.numel() * 8 for t in self.h_delta.values()) + sum(t.numel() * 4 for t in self.h_info.values())
