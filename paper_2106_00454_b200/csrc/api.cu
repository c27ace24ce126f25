// C-ABI entry points of libwpcd.so (see include/wpcd.h): argument checks, then kernel launches.  No CPU fallback.
#include <cstdio>
#include <cstring>
#include <new>
#include "wpcd_internal.cuh"

int wpcd_check_cuda(WpcdHandle* h, cudaError_t e, const char* where) {
  if (e == cudaSuccess) return WPCD_OK;
  if (h) snprintf(h->cuda_err, sizeof(h->cuda_err), "%s: %s", where, cudaGetErrorString(e));
  return WPCD_ECUDA;
}

extern "C" {

int wpcd_create(void** handle, int device) {
  if (!handle) return WPCD_EINVAL;
  *handle = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return WPCD_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return WPCD_ECUDA;
  if (prop.major < 10) return WPCD_ECUDA;  // sm_100a only
  WpcdHandle* h = new (std::nothrow) WpcdHandle();
  if (!h) return WPCD_EINVAL;
  h->device = device;
  h->num_sms = prop.multiProcessorCount;
  h->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
  h->cuda_err[0] = 0;
  *handle = h;
  return WPCD_OK;
}

void wpcd_destroy(void* handle) { delete static_cast<WpcdHandle*>(handle); }

const char* wpcd_strerror(int code) {
  switch (code) {
    case WPCD_OK: return "ok";
    case WPCD_EINVAL: return "invalid argument";
    case WPCD_ESIZE: return "unsupported size";
    case WPCD_EWORK: return "workspace too small";
    case WPCD_ECUDA: return "CUDA runtime or launch failure";
    default: return "unknown error";
  }
}

const char* wpcd_last_cuda_error(void* handle) { return handle ? static_cast<WpcdHandle*>(handle)->cuda_err : ""; }
int wpcd_num_sms(void* handle) { return handle ? static_cast<WpcdHandle*>(handle)->num_sms : 0; }

size_t wpcd_build_workspace_bytes(void* handle, int N, int n_chan) {
  if (!handle || N < 1 || n_chan < 1) return 0;
  return wpcd_build_workspace(N, n_chan);
}
size_t wpcd_diag_workspace_bytes(void* handle, int n, int batch) {
  if (!handle || n < 2 || batch < 1) return 0;
  return wpcd_jacobi_workspace(static_cast<WpcdHandle*>(handle), n, batch);
}
size_t wpcd_onshell_workspace_bytes(void* handle, int N, int coupled, int batch, int nE) {
  if (!handle || N < 1 || batch < 1 || nE < 1) return 0;
  return wpcd_onshell_workspace(N, coupled, batch, nE);
}

static bool aligned16(const void* p) { return (reinterpret_cast<size_t>(p) & 15) == 0; }

// Every compute call acts on the CALLER's current device (launches, function attributes, the caller's stream and
// buffers): it must be the device the handle was created for (include/wpcd.h, "Handle").
static bool on_handle_device(const WpcdHandle* h) {
  int cur = -1;
  return cudaGetDevice(&cur) == cudaSuccess && cur == h->device;
}

// Checks of a wpcd_potential and a channel list shared by wpcd_build_channels and wpcd_mi_solve, so that the same struct
// behaves the same way in both: term counts, positive ranges, scale columns inside [0, P) and backed by d_scales,
// partial waves inside the range the Q_l evaluation is pinned for (reading C7: l <= WPCD_MAX_L).
static int check_potential_channels(const wpcd_potential* pot, const wpcd_channel* chan, int n_chan, const double* d_scales,
                                    int P, int* n_unc_out, int* n_cpl_out) {
  if (!pot || !chan || n_chan < 1 || P < 0) return WPCD_EINVAL;
  if (n_chan > WPCD_MAX_CHANNELS) return WPCD_ESIZE;
  if (P > 0 && !d_scales) return WPCD_EINVAL;
  if (pot->kind != 0 && pot->kind != 1) return WPCD_EINVAL;
  if (pot->kind == 0) {
    if (pot->n_terms < 1 || !pot->V0 || !pot->mu) return WPCD_EINVAL;
    if (pot->n_terms > WPCD_MAX_TERMS) return WPCD_ESIZE;
    for (int t = 0; t < pot->n_terms; ++t) {
      if (!(pot->mu[t] > 0)) return WPCD_EINVAL;
      if (pot->scale_idx && (pot->scale_idx[t] >= P || (pot->scale_idx[t] >= 0 && !d_scales))) return WPCD_EINVAL;
    }
    if (pot->VT_scale_idx >= P || (pot->VT_scale_idx >= 0 && !d_scales)) return WPCD_EINVAL;
  } else {
    if (!(pot->beta > 0)) return WPCD_EINVAL;
  }
  int n_unc = 0, n_cpl = 0;
  for (int c = 0; c < n_chan; ++c) {
    if (chan[c].coupled) {
      if (chan[c].lJ < 1 || pot->kind == 1 || !(pot->muT > 0)) return WPCD_EINVAL;
      if (chan[c].lJ + 1 > WPCD_MAX_L) return WPCD_ESIZE;
      ++n_cpl;
    } else {
      if (chan[c].lJ < 0) return WPCD_EINVAL;
      if (chan[c].lJ > WPCD_MAX_L) return WPCD_ESIZE;
      ++n_unc;
    }
  }
  *n_unc_out = n_unc; *n_cpl_out = n_cpl;
  return WPCD_OK;
}

int wpcd_build_channels(void* handle, const wpcd_grid* grid, const wpcd_potential* pot, const wpcd_channel* chan,
                        int n_chan, const double* d_scales, int S, int P, double* d_H_unc, double* d_H_cpl,
                        double* d_e0, double* d_dE, double* d_Eedge, void* d_work, size_t work_bytes, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || !grid || !pot || !chan || !d_e0 || !d_dE || !d_Eedge) return WPCD_EINVAL;
  if (grid->N < 1 || !grid->h_edges || grid->n_gl < 1 || grid->n_gl > 16 || !(grid->hbarc > 0) || !(grid->mu > 0)) return WPCD_EINVAL;
  if (grid->wp_kind != 0 && grid->wp_kind != 1) return WPCD_EINVAL;
  if (grid->N > 4096) return WPCD_ESIZE;  // 32-bit element indices in the assembly kernels (n = 2N <= 8192)
  if (S < 1) return WPCD_EINVAL;
  if (!(grid->h_edges[0] >= 0)) return WPCD_EINVAL;
  for (int i = 0; i < grid->N; ++i)
    if (!(grid->h_edges[i + 1] > grid->h_edges[i])) return WPCD_EINVAL;
  int n_unc = 0, n_cpl = 0;
  if (int rc = check_potential_channels(pot, chan, n_chan, d_scales, P, &n_unc, &n_cpl)) return rc;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  if ((n_unc && !d_H_unc) || (n_cpl && !d_H_cpl)) return WPCD_EINVAL;
  if (!aligned16(d_H_unc) || !aligned16(d_H_cpl) || !aligned16(d_work)) return WPCD_EINVAL;
  if (work_bytes < wpcd_build_workspace(grid->N, n_chan) || (!d_work && wpcd_build_workspace(grid->N, n_chan))) return WPCD_EWORK;
  return wpcd_build_launch(h, grid, pot, chan, n_chan, d_scales, S, P, d_H_unc, d_H_cpl, d_e0, d_dE, d_Eedge, d_work,
                           work_bytes, static_cast<cudaStream_t>(stream));
}

int wpcd_diag_batched(void* handle, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                      double tol, int max_sweeps, const int* h_rows, int n_ranges, void* d_work, size_t work_bytes,
                      void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || !d_A || !d_W || !d_C || !d_info || batch < 1 || max_sweeps < 1) return WPCD_EINVAL;
  if (n_ranges < 0 || n_ranges > 4 || (n_ranges > 0 && !h_rows)) return WPCD_EINVAL;
  for (int r = 0; r < n_ranges; ++r)
    if (h_rows[2 * r] < 0 || h_rows[2 * r + 1] > n || h_rows[2 * r] >= h_rows[2 * r + 1]) return WPCD_EINVAL;
  if (n < 2 || n > 4096) return WPCD_ESIZE;
  if (!aligned16(d_A) || !aligned16(d_C) || !aligned16(d_work)) return WPCD_EINVAL;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  size_t need = wpcd_jacobi_workspace(h, n, batch);
  if (work_bytes < need || (need && !d_work)) return WPCD_EWORK;
  return wpcd_jacobi_launch(h, n, batch, d_A, d_W, d_C, d_info, tol, max_sweeps, h_rows, n_ranges, d_work, work_bytes,
                            static_cast<cudaStream_t>(stream));
}

int wpcd_diag_batched_static(void* handle, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                             double tol, int max_sweeps, const int* h_rows, int n_ranges, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || !d_A || !d_W || !d_C || !d_info || batch < 1 || max_sweeps < 1) return WPCD_EINVAL;
  if (n_ranges < 0 || n_ranges > 4 || (n_ranges > 0 && !h_rows)) return WPCD_EINVAL;
  for (int r = 0; r < n_ranges; ++r)
    if (h_rows[2 * r] < 0 || h_rows[2 * r + 1] > n || h_rows[2 * r] >= h_rows[2 * r + 1]) return WPCD_EINVAL;
  if (n < 2 || n > 4096) return WPCD_ESIZE;
  if (!aligned16(d_A) || !aligned16(d_C)) return WPCD_EINVAL;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  return wpcd_jacobi_static_launch(h, n, batch, d_A, d_W, d_C, d_info, tol, max_sweeps, h_rows, n_ranges,
                                   static_cast<cudaStream_t>(stream));
}

int wpcd_onshell_T(void* handle, int N, int coupled, int batch, const double* d_e0, const double* d_Eedge,
                   const double* d_H, const double* d_W, const double* d_C, const double* d_Ecm, int nE, int mode,
                   double* d_T, int* d_bin, void* d_work, size_t work_bytes, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || !d_e0 || !d_Eedge || !d_H || !d_W || !d_C || !d_Ecm || !d_T || !d_bin) return WPCD_EINVAL;
  if (N < 1 || batch < 1 || nE < 1 || (mode != 0 && mode != 1)) return WPCD_EINVAL;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  size_t need = wpcd_onshell_workspace(N, coupled, batch, nE);
  if (work_bytes < need || (need && !d_work)) return WPCD_EWORK;
  return wpcd_onshell_launch(h, N, coupled ? 1 : 0, batch, d_e0, d_Eedge, d_H, d_W, d_C, d_Ecm, nE, mode, d_T, d_bin,
                             d_work, work_bytes, static_cast<cudaStream_t>(stream));
}

int wpcd_phase_shifts(void* handle, int coupled, int batch, int nE, const double* d_T, const int* d_bin,
                      const double* d_dE, double* d_delta, double* d_S, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || !d_T || !d_bin || !d_dE || !d_delta || batch < 1 || nE < 1) return WPCD_EINVAL;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  return wpcd_phase_launch(h, coupled ? 1 : 0, batch, nE, d_T, d_bin, d_dE, d_delta, d_S,
                           static_cast<cudaStream_t>(stream));
}

int wpcd_interp_phases(void* handle, int coupled, int batch, int N, const double* d_pedge, const double* d_delta_mid,
                       const double* d_q, int nq, double* d_out, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || !d_pedge || !d_delta_mid || !d_q || !d_out || batch < 1 || N < 1 || nq < 1) return WPCD_EINVAL;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  return wpcd_interp_launch(h, coupled ? 1 : 0, batch, N, d_pedge, d_delta_mid, d_q, nq, d_out,
                            static_cast<cudaStream_t>(stream));
}

int wpcd_sigma_tot(void* handle, int S, int nE, int n_unc, const int* h_J_unc, const double* d_T_unc, int n_cpl,
                   const int* h_J_cpl, const double* d_T_cpl, const int* d_bin, const double* d_dE, const double* d_Ecm,
                   double hbarc, double mu, double* d_sigma, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || S < 1 || nE < 1 || n_unc < 0 || n_cpl < 0 || n_unc + n_cpl < 1 || !d_Ecm || !d_sigma) return WPCD_EINVAL;
  if ((d_bin == nullptr) != (d_dE == nullptr)) return WPCD_EINVAL;  // both given (inputs are T) or both NULL (inputs are S)
  if ((n_unc && (!h_J_unc || !d_T_unc)) || (n_cpl && (!h_J_cpl || !d_T_cpl)) || !(hbarc > 0) || !(mu > 0)) return WPCD_EINVAL;
  if (n_unc > WPCD_MAX_CHANNELS || n_cpl > WPCD_MAX_CHANNELS) return WPCD_ESIZE;
  for (int c = 0; c < n_unc; ++c) if (h_J_unc[c] < 0) return WPCD_EINVAL;
  for (int c = 0; c < n_cpl; ++c) if (h_J_cpl[c] < 1) return WPCD_EINVAL;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  return wpcd_sigma_launch(h, S, nE, n_unc, h_J_unc, d_T_unc, n_cpl, h_J_cpl, d_T_cpl, d_bin, d_dE, d_Ecm, hbarc, mu, d_sigma,
                           static_cast<cudaStream_t>(stream));
}

size_t wpcd_mi_workspace_bytes(void* handle, int NQ) {
  (void)handle;
  return NQ > 0 ? wpcd_mi_workspace(NQ) : 0;
}

int wpcd_mi_solve(void* handle, const wpcd_potential* pot, const wpcd_channel* chan, int n_chan, const double* d_scales, int S,
                  int P, int NQ, double cmap, double hbarc, double mu, const double* d_Ecm, int nE, double* d_S_unc,
                  double* d_S_cpl, void* d_work, size_t work_bytes, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || !pot || !chan || n_chan < 1 || S < 1 || nE < 1 || !d_Ecm || NQ < 2 || !(cmap > 0) || !(hbarc > 0) || !(mu > 0)) return WPCD_EINVAL;
  if (d_scales && P < 1) return WPCD_EINVAL;
  int n_unc = 0, n_cpl = 0;
  if (int rc = check_potential_channels(pot, chan, n_chan, d_scales, P, &n_unc, &n_cpl)) return rc;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  if ((n_unc && !d_S_unc) || (n_cpl && !d_S_cpl)) return WPCD_EINVAL;
  if ((n_unc && !wpcd_mi_fits(h, NQ, 0)) || (n_cpl && !wpcd_mi_fits(h, NQ, 1))) return WPCD_ESIZE;
  if (!d_work || work_bytes < wpcd_mi_workspace(NQ)) return WPCD_EWORK;
  return wpcd_mi_launch(h, pot, chan, n_chan, d_scales, S, P, NQ, cmap, hbarc, mu, d_Ecm, nE, d_S_unc, d_S_cpl, d_work,
                        static_cast<cudaStream_t>(stream));
}

size_t wpcd_probe_sink_elems(void* handle) { return handle ? wpcd_probe_sink(static_cast<WpcdHandle*>(handle)) : 0; }

int wpcd_probe_fp64(void* handle, int kind, int iters, double* d_sink, double* h_flops, void* stream) {
  WpcdHandle* h = static_cast<WpcdHandle*>(handle);
  if (!h || (kind != 0 && kind != 1) || iters < 1 || !d_sink || !h_flops) return WPCD_EINVAL;
  if (!on_handle_device(h)) return WPCD_EINVAL;
  return wpcd_probe_launch(h, kind, iters, d_sink, h_flops, static_cast<cudaStream_t>(stream));
}

int wpcd_onshell_rows(const wpcd_grid* grid, int coupled, const double* h_Ecm, int nE, int* h_rows, int* n_ranges) {
  if (!grid || !grid->h_edges || grid->N < 1 || !h_Ecm || nE < 1 || !h_rows || !n_ranges) return WPCD_EINVAL;
  return wpcd_onshell_rows_host(grid->N, coupled ? 1 : 0, grid->h_edges, grid->hbarc, grid->mu, h_Ecm, nE, h_rows, n_ranges);
}

}  // extern "C"
