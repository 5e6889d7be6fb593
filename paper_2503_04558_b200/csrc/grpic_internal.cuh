// Internal declarations shared by the translation units of libgrpic.so (CUDA, sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/grpic.h"

// Geometry + table pointers handed to every kernel by value.
struct GridDev {
  double a, M, a2, twoM;
  double xi_in, xi_out, dxi, dth, inv_dxi, inv_dth, dphi;
  int nr, nth, ng;
  int pitch, rows, i0, j0;  // element (i,j) at (j+j0)*pitch + (i+i0)
  // 1-D tables, index i+i0 (length pitch) / j+j0 (length rows)
  const double* r_n;    // r at node i
  const double* r_h;    // r at i+1/2
  const double* dr_n;   // r(i+1/2) - r(i-1/2): r-edge centred on node i
  const double* dr_h;   // r(i+1) - r(i):       r-edge centred on i+1/2
  const double* sin_n;  // sin(theta_j)
  const double* cos_n;
  const double* sin_h;  // sin(theta_{j+1/2})
  const double* cos_h;
  // area factors, grid layout.  iADr = dphi/A^D_r, iADth = dphi/A^D_th, iADph = 1/A^D_ph,
  // iABr = dphi/A^B_r, iABth = dphi/A^B_th, iABph = 1/A^B_ph; 0 where the area vanishes.
  const double *iADr, *iADth, *iADph, *iABr, *iABth, *iABph;
  __host__ __device__ __forceinline__ size_t idx(int i, int j) const {
    return (size_t)(j + j0) * (size_t)pitch + (size_t)(i + i0);
  }
  __host__ __device__ __forceinline__ size_t size() const { return (size_t)pitch * (size_t)rows; }
};

struct grpic_ctx {
  grpic_params p;
  GridDev g;
  double* tables;   // one allocation: 1-D tables + 6 raw area arrays + 6 area factors
  double* areas[6]; // raw A^D_r, A^D_th, A^D_ph, A^B_r, A^B_th, A^B_ph
  void* ws;
  size_t ws_bytes;
  int sm_count;
  unsigned long long* removed_counter;   // grpic_set_removed_counter (caller's device word, nullable)
  unsigned long long* clock_probe;       // grpic_set_clock_probe (caller's 4 device words, nullable)
  grpic_flux_exchange_fn flux_exchange;  // grpic_set_flux_exchange (multi-GPU sum of the fluxes in grpic_step_host)
  void* flux_exchange_user;
  void* host_step;  // staging buffers / streams of grpic_step_host (host_step.cu), lazily created
};

#define GRPIC_CUDA_OK(expr)                     \
  do {                                          \
    cudaError_t e__ = (expr);                   \
    if (e__ != cudaSuccess) return GRPIC_ERR_CUDA; \
  } while (0)

static inline int grpic_launch_ok() {
  return cudaGetLastError() == cudaSuccess ? GRPIC_OK : GRPIC_ERR_CUDA;
}

// Kerr-Schild building blocks shared by the device code (Appendix A).
// sqrt(gamma) = rho^2 sin(theta) sqrt(1+z)
__device__ __forceinline__ double ks_sqrtg(double a2, double M, double r, double s, double c) {
  const double rho2 = fma(a2 * c, c, r * r);
  return s * sqrt(rho2 * (rho2 + 2.0 * M * r));
}

// launch bookkeeping for bench.py's gpu_launches (api.cu)
void grpic_count_launches(int n);
// in-place exclusive scan of data[0..n) (sort.cu); scratch >= n/2048 + n/2048^2 + 8 words
int grpic_exclusive_scan(uint32_t* data, size_t n, uint32_t* scratch, cudaStream_t st);
// first-order shape + Vay pusher through the tuned kernel (push_deposit.cu); GRPIC_ERR_ARG if the arrays
// do not allow its bulk-TMA tiles
int grpic_push_deposit_cic_vay(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields, grpic_current* flux,
                               double dt, uint32_t* status, cudaStream_t st);
// frees the staging state of grpic_step_host (host_step.cu)
void grpic_host_step_release(grpic_ctx* ctx);
