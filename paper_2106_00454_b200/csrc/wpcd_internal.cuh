// Internal declarations shared by the translation units of libwpcd.so (CUDA side only; nothing here is used by
// the CPU oracle under /oracle).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include "../../include/wpcd.h"

#define WPCD_PI 3.14159265358979323846264338327950288

struct WpcdHandle {
  int device;
  int num_sms;
  int max_smem_optin;
  char cuda_err[256];
};

// Records a CUDA error text in the handle and returns WPCD_ECUDA (or WPCD_OK).
int wpcd_check_cuda(WpcdHandle* h, cudaError_t e, const char* where);

// jacobi.cu
size_t wpcd_jacobi_workspace(const WpcdHandle* h, int n, int batch);
int wpcd_jacobi_launch(WpcdHandle* h, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                       double tol, int max_sweeps, const int* h_rows, int n_ranges, void* d_work, size_t work_bytes,
                       cudaStream_t st);
// wpcd_diag_batched_static: the same launch with the workspace in jacobi.cu's file-scope device array
int wpcd_jacobi_static_launch(WpcdHandle* h, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                              double tol, int max_sweeps, const int* h_rows, int n_ranges, cudaStream_t st);
// jacobi_small.cu (n <= WPCD_SMALL_N_MAX)
#define WPCD_SMALL_N_MAX 32
size_t wpcd_jacobi_small_workspace();
int wpcd_jacobi_small_launch(WpcdHandle* h, int n, int batch, const double* d_A, double* d_W, double* d_C, int* d_info,
                             double tol, int max_sweeps, const int* h_rows, int n_ranges, void* d_work, size_t work_bytes,
                             cudaStream_t st);
// assembly.cu
size_t wpcd_build_workspace(int N, int n_chan);
int wpcd_build_launch(WpcdHandle* h, const wpcd_grid* grid, const wpcd_potential* pot, const wpcd_channel* chan,
                      int n_chan, const double* d_scales, int S, int P, double* d_H_unc, double* d_H_cpl, double* d_e0,
                      double* d_dE, double* d_Eedge, void* d_work, size_t work_bytes, cudaStream_t st);
// onshell.cu
size_t wpcd_onshell_workspace(int N, int coupled, int batch, int nE);
int wpcd_onshell_launch(WpcdHandle* h, int N, int coupled, int batch, const double* d_e0, const double* d_Eedge,
                        const double* d_H, const double* d_W, const double* d_C, const double* d_Ecm, int nE,
                        int mode, double* d_T, int* d_bin, void* d_work, size_t work_bytes, cudaStream_t st);
int wpcd_phase_launch(WpcdHandle* h, int coupled, int batch, int nE, const double* d_T, const int* d_bin,
                      const double* d_dE, double* d_delta, double* d_S, cudaStream_t st);
int wpcd_interp_launch(WpcdHandle* h, int coupled, int batch, int N, const double* d_pedge, const double* d_delta_mid,
                       const double* d_q, int nq, double* d_out, cudaStream_t st);
int wpcd_sigma_launch(WpcdHandle* h, int S, int nE, int n_unc, const int* h_J_unc, const double* d_T_unc, int n_cpl,
                      const int* h_J_cpl, const double* d_T_cpl, const int* d_bin, const double* d_dE, const double* d_Ecm,
                      double hbarc, double mu, double* d_sigma, cudaStream_t st);
int wpcd_onshell_rows_host(int N, int coupled, const double* h_edges, double hbarc, double mu, const double* h_Ecm, int nE,
                           int* h_rows, int* n_ranges);
// mi.cu
size_t wpcd_mi_workspace(int NQ);
bool wpcd_mi_fits(const WpcdHandle* h, int NQ, int coupled);
int wpcd_mi_launch(WpcdHandle* h, const wpcd_potential* pot, const wpcd_channel* chan, int n_chan, const double* d_scales,
                   int S, int P, int NQ, double cmap, double hbarc, double mu, const double* d_Ecm, int nE, double* d_S_unc,
                   double* d_S_cpl, void* d_work, cudaStream_t st);
// probe.cu
size_t wpcd_probe_sink(const WpcdHandle* h);
int wpcd_probe_launch(WpcdHandle* h, int kind, int iters, double* d_sink, double* h_flops, cudaStream_t st);
