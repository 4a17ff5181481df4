// passes_zy.cu -- z transforms (compact <-> hybrid) and the y passes P1 / P3 of the RHS pipeline.
//
//   k_zinv : S[f][cz][cy][cx] -> H[f][z][cy][cx]      inverse c2c along z, zero-padded
//   k_zfwd : H -> S                                   forward c2c along z, kz part of Eq. 20, 1/N scale
//   k_yinv : P1.  H -> D: for w+- also xi = -w/kperp^2; for every source field f the
//            pair ( f , d f/dy = IFFT_y(i ky f) )  (Eq. 10), inverse c2c along y
//   k_yfwd : P3.  E -> H: forward c2c along y, ky part of Eq. 20; the Elsasser pair is assembled as
//            N+- = -1/2 A -+ 1/2 kperp^2 B  (Eq. 1 with Eq. 11)
// Every FFT is fft_lanes<N> (fft.cuh): T lanes of one warp per column, data in registers, one
// shared-memory exchange per stage boundary.  Adjacent lane groups take adjacent cx so that global
// accesses of a warp cover contiguous kx runs.
#include <vector>
#include "common.cuh"

template <int NZ, int DIR>
__global__ void __launch_bounds__(GD_FFT_THREADS) k_zfft(Dims d, const cd* __restrict__ in, cd* __restrict__ out,
                                                       const cd* __restrict__ tw, int ncols) {
  using G = FftGeom<NZ>;
  constexpr int T = G::T, E = G::E;
  extern __shared__ cd smem[];
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  const int gid = blockIdx.x * (GD_FFT_THREADS / T) + grp;
  cd* buf = smem + FftTw<NZ>::COUNT + (size_t)grp * (G::BUF + 1);
  fft_load_table<NZ>(smem, tw);
  const cd* tws = smem;
  const bool active = gid < ncols;
  const int plane = d.Ky * d.Kx;
  const int f = active ? gid / plane : 0, rem = active ? gid % plane : 0;
  cd v[E];
  if (DIR > 0) {   // compact -> hybrid
    const cd* src = in + (size_t)f * d.PS + rem;
#pragma unroll
    for (int q = 0; q < E; ++q) {
      const int cz = fft2c(t + T * q, NZ, d.hz3, d.Kz);
      v[q] = (active && cz >= 0) ? ldg_cd(src + (size_t)cz * plane) : cmake(0.0, 0.0);
    }
    fft_lanes<NZ, +1>(v, t, buf, tws);
    if (active) {
      cd* dst = out + (size_t)f * d.PH + rem;
#pragma unroll
      for (int q = 0; q < E; ++q) st_cd(dst + (size_t)(t + T * q) * plane, v[q]);
    }
  } else {         // hybrid -> compact, masked, scaled by 1/(nx ny nz)
    const cd* src = in + (size_t)f * d.PH + rem;
#pragma unroll
    for (int q = 0; q < E; ++q) v[q] = active ? ldg_cd(src + (size_t)(t + T * q) * plane) : cmake(0.0, 0.0);
    fft_lanes<NZ, -1>(v, t, buf, tws);
    if (active) {
      cd* dst = out + (size_t)f * d.PS + rem;
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int cz = fft2c(t + T * q, NZ, d.hz3, d.Kz);
        if (cz >= 0) st_cd(dst + (size_t)cz * plane, cscale(v[q], d.inv_n));
      }
    }
  }
}

// P1.  One lane group per (source field s, z, cx) column.  Sources: s = 0,1 -> w+, w-;  s = 2+m -> g_m.
// D array order: 0/1 xi+ , 2/3 xi- , 4/5 w+ , 6/7 w- , 8+2m / 9+2m g_m   (even: f, odd: df/dy).
template <int NY>
__global__ void __launch_bounds__(GD_FFT_THREADS) k_yinv(Dims d, const cd* __restrict__ H, cd* __restrict__ D,
                                                       const cd* __restrict__ tw, int ncols) {
  using G = FftGeom<NY>;
  constexpr int T = G::T, E = G::E;
  extern __shared__ cd smem[];
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  const int gid = blockIdx.x * (GD_FFT_THREADS / T) + grp;
  cd* buf = smem + FftTw<NY>::COUNT + (size_t)grp * (G::BUF + 1);
  fft_load_table<NY>(smem, tw);
  const cd* tws = smem;
  const bool active = gid < ncols;
  const int cx = active ? gid % d.Kx : 0;
  const int sz = active ? gid / d.Kx : 0;
  const int z = sz % d.nz, s = sz / d.nz;
  const cd* src = H + (size_t)s * d.PH + (size_t)z * d.Ky * d.Kx + cx;
  const double kx = d.kx0 * cx;
  cd v0[E], v[E];
  double ky[E];
#pragma unroll
  for (int q = 0; q < E; ++q) {
    const int iy = t + T * q;
    const int cy = fft2c(iy, NY, d.hy3, d.Ky);
    v0[q] = (active && cy >= 0) ? ldg_cd(src + (size_t)cy * d.Kx) : cmake(0.0, 0.0);
    ky[q] = d.ky0 * fft2n(iy, NY);
  }
  const size_t obase = (size_t)z * NY * d.Kx + cx;
  auto emit = [&](int a) {   // inverse transform v and write array a
    fft_lanes<NY, +1>(v, t, buf, tws);
    if (active) {
      cd* dst = D + (size_t)a * d.PD + obase;
#pragma unroll
      for (int q = 0; q < E; ++q) st_cd(dst + (size_t)(t + T * q) * d.Kx, v[q]);
    }
  };
  if (s < 2) {
    // potentials: xi = -w / kperp^2, zero at kperp = 0
#pragma unroll
    for (int q = 0; q < E; ++q) {
      const double k2 = kx * kx + ky[q] * ky[q];
      const double inv = k2 > 0.0 ? -1.0 / k2 : 0.0;
      v[q] = cscale(v0[q], inv);
    }
    emit(2 * s);
#pragma unroll
    for (int q = 0; q < E; ++q) {
      const double k2 = kx * kx + ky[q] * ky[q];
      const double inv = k2 > 0.0 ? -1.0 / k2 : 0.0;
      v[q] = cscale(mul_i(v0[q]), inv * ky[q]);
    }
    emit(2 * s + 1);
  }
  const int a0 = (s < 2) ? 4 + 2 * s : 8 + 2 * (s - 2);
#pragma unroll
  for (int q = 0; q < E; ++q) v[q] = v0[q];
  emit(a0);
#pragma unroll
  for (int q = 0; q < E; ++q) v[q] = cscale(mul_i(v0[q]), ky[q]);
  emit(a0 + 1);
}

// P3.  One lane group per (task e, z, cx): e = 0 handles A and B together, e = 1+m handles R_m.
// E array order: 0 A, 1 B, 2+m R_m.  Output hybrid fields: 0 N+, 1 N-, 2+m R_m.
template <int NY>
__global__ void __launch_bounds__(GD_FFT_THREADS) k_yfwd(Dims d, const cd* __restrict__ Ein, cd* __restrict__ Gh,
                                                       const cd* __restrict__ tw, int ncols) {
  using G = FftGeom<NY>;
  constexpr int T = G::T, E = G::E;
  extern __shared__ cd smem[];
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  const int gid = blockIdx.x * (GD_FFT_THREADS / T) + grp;
  cd* buf = smem + FftTw<NY>::COUNT + (size_t)grp * (G::BUF + 1);
  fft_load_table<NY>(smem, tw);
  const cd* tws = smem;
  const bool active = gid < ncols;
  const int cx = active ? gid % d.Kx : 0;
  const int ez = active ? gid / d.Kx : 0;
  const int z = ez % d.nz, e = ez / d.nz;
  const size_t ibase = (size_t)z * NY * d.Kx + cx;
  const size_t obase = (size_t)z * d.Ky * d.Kx + cx;
  cd v[E];
  auto load = [&](int a) {
    const cd* src = Ein + (size_t)a * d.PD + ibase;
#pragma unroll
    for (int q = 0; q < E; ++q) v[q] = active ? ldg_cd(src + (size_t)(t + T * q) * d.Kx) : cmake(0.0, 0.0);
    fft_lanes<NY, -1>(v, t, buf, tws);
  };
  if (e == 0) {
    cd va[E];
    load(0);
#pragma unroll
    for (int q = 0; q < E; ++q) va[q] = v[q];
    load(1);
    if (active) {
      const double kx = d.kx0 * cx;
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int iy = t + T * q;
        const int cy = fft2c(iy, NY, d.hy3, d.Ky);
        if (cy >= 0) {
          const double ky = d.ky0 * fft2n(iy, NY);
          const double hk2 = 0.5 * (kx * kx + ky * ky);
          // N+- = -1/2 A -+ 1/2 kperp^2 B
          const cd np = cmake(-0.5 * va[q].x - hk2 * v[q].x, -0.5 * va[q].y - hk2 * v[q].y);
          const cd nm = cmake(-0.5 * va[q].x + hk2 * v[q].x, -0.5 * va[q].y + hk2 * v[q].y);
          st_cd(Gh + obase + (size_t)cy * d.Kx, np);
          st_cd(Gh + d.PH + obase + (size_t)cy * d.Kx, nm);
        }
      }
    }
  } else {
    load(1 + e);
    if (active) {
      cd* dst = Gh + (size_t)(1 + e) * d.PH + obase;
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int cy = fft2c(t + T * q, NY, d.hy3, d.Ky);
        if (cy >= 0) st_cd(dst + (size_t)cy * d.Kx, v[q]);
      }
    }
  }
}

// ---- launchers ------------------------------------------------------------------------------------
template <int N> static size_t fft_smem() { return ((size_t)(GD_FFT_THREADS / FftGeom<N>::T) * (FftGeom<N>::BUF + 1) + FftTw<N>::COUNT) * sizeof(cd); }
template <int N> static int fft_blocks(long long ncols) { const int gpb = GD_FFT_THREADS / FftGeom<N>::T; return (int)((ncols + gpb - 1) / gpb); }

#define GD_DISPATCH(NVAL, MACRO)                                                      \
  switch (NVAL) {                                                                     \
    case 2: MACRO(2) break; case 4: MACRO(4) break; case 8: MACRO(8) break;           \
    case 16: MACRO(16) break; case 32: MACRO(32) break; case 64: MACRO(64) break;     \
    case 128: MACRO(128) break; case 256: MACRO(256) break; case 512: MACRO(512) break; \
    default: return cudaErrorInvalidValue;                                            \
  }

cudaError_t launch_zfft(const Dims& d, int dir, const cd* in, cd* out, const cd* tw, int nfields, cudaStream_t st) {
  const long long ncols = (long long)nfields * d.Ky * d.Kx;
#define ZCASE(NN)                                                                                         \
  if (dir > 0) k_zfft<NN, +1><<<fft_blocks<NN>(ncols), GD_FFT_THREADS, fft_smem<NN>(), st>>>(d, in, out, tw, (int)ncols); \
  else k_zfft<NN, -1><<<fft_blocks<NN>(ncols), GD_FFT_THREADS, fft_smem<NN>(), st>>>(d, in, out, tw, (int)ncols);
  GD_DISPATCH(d.nz, ZCASE)
  return cudaGetLastError();
}
cudaError_t launch_yinv(const Dims& d, const cd* H, cd* D, const cd* tw, cudaStream_t st) {
  const long long ncols = (long long)d.F * d.nz * d.Kx;
#define YICASE(NN) k_yinv<NN><<<fft_blocks<NN>(ncols), GD_FFT_THREADS, fft_smem<NN>(), st>>>(d, H, D, tw, (int)ncols);
  GD_DISPATCH(d.ny, YICASE)
  return cudaGetLastError();
}
cudaError_t launch_yfwd(const Dims& d, const cd* E, cd* Gh, const cd* tw, cudaStream_t st) {
  const long long ncols = (long long)(1 + d.M) * d.nz * d.Kx;
#define YFCASE(NN) k_yfwd<NN><<<fft_blocks<NN>(ncols), GD_FFT_THREADS, fft_smem<NN>(), st>>>(d, E, Gh, tw, (int)ncols);
  GD_DISPATCH(d.ny, YFCASE)
  return cudaGetLastError();
}

// Host: the stage twiddle table of length-n transforms (fft.cuh layout); empty for single-stage sizes.
int fft_stage_table_host(int n, std::vector<cd>& out) {
#define TCASE(NN) out.assign(FftTw<NN>::COUNT + 1, cmake(0.0, 0.0)); fft_fill_stage_table<NN>(out.data());
  switch (n) {
    case 2: TCASE(2) break; case 4: TCASE(4) break; case 8: TCASE(8) break; case 16: TCASE(16) break;
    case 32: TCASE(32) break; case 64: TCASE(64) break; case 128: TCASE(128) break; case 256: TCASE(256) break;
    case 512: TCASE(512) break;
    default: return -1;
  }
  return 0;
}
