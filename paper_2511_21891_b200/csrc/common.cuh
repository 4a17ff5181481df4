// common.cuh -- grid geometry shared by the kernels of the GANDALF hot path (device side only).
//
// Storage spaces (all complex fp64, kx fastest; "c" indices run over RETAINED modes only, i.e.
// the modes Eq. 20 keeps: 3|n| <= N):
//   compact  S[f][cz][cy][cx]   Kz*Ky*Kx per field   fully spectral state / RHS
//   hybrid   H[f][z ][cy][cx]   nz*Ky*Kx per field   z in real space, (kx,ky) spectral
//   xy-real  D[a][z ][y ][cx]   nz*ny*Kx per array   y,z real, kx spectral (retained kx only)
// cx = 0..Kx-1 is n_x = cx; cy = 0..Ky-1 is n_y = cy (cy <= hy3) or cy-Ky (negative modes);
// cz likewise.  The zeroed third is never stored or transformed.
#pragma once
#include <cuda_runtime.h>
#include "fft.cuh"

struct Dims {
  int nx, ny, nz, M, F;
  int hx;                 // nx/2+1 (boundary layout)
  int Kx, Ky, Kz;         // retained counts
  int hx3, hy3, hz3;      // floor(N/3)
  double kx0, ky0, kz0;   // 2 pi / L
  double inv_n;           // 1/(nx ny nz)
  size_t PS, PH, PD;      // per-field strides (complex elements) of the three spaces
};

__device__ __forceinline__ int c2n(int c, int h3, int K) { return c <= h3 ? c : c - K; }        // compact -> signed mode
// FFT index (0..N-1) -> compact index, or -1 if the mode is removed by the 2/3 rule
__device__ __forceinline__ int fft2c(int i, int N, int h3, int K) {
  if (i <= h3) return i;
  if (i >= N - h3) return i - N + K;
  return -1;
}
__device__ __forceinline__ int fft2n(int i, int N) { return i < N / 2 ? i : i - N; }

__device__ __forceinline__ cd ldg_cd(const cd* p) {
  const double2 v = __ldg(reinterpret_cast<const double2*>(p));
  return cmake(v.x, v.y);
}
__device__ __forceinline__ void st_cd(cd* p, cd v) { *reinterpret_cast<double2*>(p) = make_double2(v.x, v.y); }

struct PhysParams {
  double vA;
  double eta; int r; int eta_normalized;
  double eta_z; int r_z;
  double eta_g;
  double k2max_perp, kz2max;     // (pi nx/Lx)^2 + (pi ny/Ly)^2 ; (pi nz/Lz)^2
  int if_variant; int g_sign;
};

// device scalars owned by the context
enum { SC_DT = 0, SC_T = 1, SC_LASTDT = 2, SC_COUNT = 8 };

// Launch geometry shared by the FFT passes: THREADS lanes per CTA, THREADS/T lines per CTA.
#define GD_FFT_THREADS 128
