// pointwise.cu -- the small kernels that are diagonal in k: per-step factor tables of the stage update (the update
// itself is fused with the z transforms, passes_zy.cu), boundary pack/unpack with projection, forcing, CFL dt,
// and the energy / shell-spectrum reductions.
#include "common.cuh"


__device__ __forceinline__ double ipow_d(double x, int n) { double r = 1.0; for (int i = 0; i < n; ++i) r *= x; return r; }

__device__ __forceinline__ double rate_perp_shape(const PhysParams& p, double k2) {
  return p.eta_normalized ? ipow_d(k2 / p.k2max_perp, p.r) : ipow_d(k2, p.r);     // Eq. 18 / Eq. 17
}

// Per-step factor tables of the fused stage update (k_zstep, passes_zy.cu), separable in (kz) and (kx,ky):
//   tabz[cz] = { cos th/2, sin th/2, cos th, sin th, fz, fzg },  th = kz vA dt (Eq. 13),
//              fz = exp(-eta_z (kz^2/kz,max^2)^r_z dt), fzg = fz if eta_g > 0 else 1
//   tabp[cy][cx] = { exp(-eta P_perp dt), exp(-eta_g P_perp dt) },  P_perp of Eq. 17 / Eq. 18
__global__ void __launch_bounds__(256) k_tables(Dims d, PhysParams p, const double* __restrict__ scal, double* __restrict__ tabz,
                                                double* __restrict__ tabp) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const double dt = scal[SC_DT];
  const int plane = d.Ky * d.Kx;
  if (i < plane) {
    const int cx = i % d.Kx, cy = i / d.Kx;
    const double kx = d.kx0 * cx, ky = d.ky0 * c2n(cy, d.hy3, d.Ky);
    const double shape = rate_perp_shape(p, kx * kx + ky * ky);
    tabp[2 * i] = exp(-(p.eta * shape) * dt);
    tabp[2 * i + 1] = (p.eta_g > 0.0) ? exp(-(p.eta_g * shape) * dt) : 1.0;
  }
  if (i < d.Kz) {
    const double kz = d.kz0 * c2n(i, d.hz3, d.Kz);
    const double th = kz * p.vA * dt;
    double s1, c1, sh, ch;
    sincos(th, &s1, &c1);
    sincos(0.5 * th, &sh, &ch);
    const double fz = (p.eta_z > 0.0) ? exp(-(p.eta_z * ipow_d(kz * kz / p.kz2max, p.r_z)) * dt) : 1.0;
    double* tz = tabz + 6 * i;
    tz[0] = ch; tz[1] = sh; tz[2] = c1; tz[3] = s1; tz[4] = fz; tz[5] = (p.eta_g > 0.0) ? fz : 1.0;
  }
}

// dt for this step and the per-moment collision factors exp(-nu (m/M)^(2p) dt) (Eq. 19).
// fixed_dt > 0: use it; else Eq. 16 from the max |grad Phi|^2 the x-pass left in maxbits, capped by dt_max (> 0).
// No flow and no dt_max: Eq. 16 gives no step -- dt = 0 makes this and every later step a no-op (the state survives, as
// in the oracle) and the sticky flag scal[SC_ERR] is reported by the next synchronising call (GANDALF_ERR_CFL).
__global__ void k_prepare_dt(double fixed_dt, double cfl_dxy, double dt_max, const unsigned long long* maxbits, double* scal,
                             const double* __restrict__ crate, double* __restrict__ collfac, int M) {
  __shared__ double sdt;
  if (threadIdx.x == 0) {
    double dt = fixed_dt;
    if (!(fixed_dt > 0.0)) {
      const double g2 = __longlong_as_double((long long)*maxbits);
      if (scal[SC_ERR] != 0.0) dt = 0.0;
      else if (g2 > 0.0) { dt = cfl_dxy / sqrt(g2); if (dt_max > 0.0 && dt > dt_max) dt = dt_max; }
      else if (dt_max > 0.0) dt = dt_max;
      else { dt = 0.0; scal[SC_ERR] = 1.0; }
    }
    scal[SC_DT] = dt;
    sdt = dt;
  }
  __syncthreads();
  for (int m = threadIdx.x; m < M; m += blockDim.x) collfac[m] = exp(-crate[m] * sdt);
}

__global__ void k_zero_u64(unsigned long long* p) { *p = 0ull; }

// ---- boundary layout <-> compact ---------------------------------------------------------------------
// pack: in[f][iz][iy][ix] half-plane (hx = nx/2+1) -> S[f][cz][cy][cx] with the projection of gandalf_set_state.
// Fields f < nzeta are potentials: stored as w = -kperp^2 zeta (zero at kperp = 0).
__global__ void __launch_bounds__(256) k_pack(Dims d, const cd* __restrict__ in, cd* __restrict__ S, int nfields, int nzeta) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= d.PS * (size_t)nfields) return;
  const int f = (int)(idx / d.PS);
  const size_t r = idx % d.PS;
  const int cx = (int)(r % d.Kx);
  const int cy = (int)((r / d.Kx) % d.Ky);
  const int cz = (int)(r / ((size_t)d.Kx * d.Ky));
  const int ny_ = c2n(cy, d.hy3, d.Ky), nz_ = c2n(cz, d.hz3, d.Kz);
  const int iy = (ny_ + d.ny) % d.ny, iz = (nz_ + d.nz) % d.nz;
  const size_t fb = (size_t)f * d.nz * d.ny * d.hx;
  cd v = in[fb + ((size_t)iz * d.ny + iy) * d.hx + cx];
  if (cx == 0) {
    const int jy = (d.ny - iy) % d.ny, jz = (d.nz - iz) % d.nz;
    const cd u = in[fb + ((size_t)jz * d.ny + jy) * d.hx];
    v = cmake(0.5 * (v.x + u.x), 0.5 * (v.y - u.y));
  }
  if (f < nzeta) {
    const double kx = d.kx0 * cx, ky = d.ky0 * ny_;
    v = cscale(v, -(kx * kx + ky * ky));
  }
  S[idx] = v;
}

// unpack: compact -> boundary layout with zeros at removed modes; potentials: zeta = -w/kperp^2.
__global__ void __launch_bounds__(256) k_unpack(Dims d, const cd* __restrict__ S, cd* __restrict__ out, int nfields, int nzeta) {
  const size_t hp = (size_t)d.nz * d.ny * d.hx;
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= hp * (size_t)nfields) return;
  const int f = (int)(idx / hp);
  const size_t r = idx % hp;
  const int ix = (int)(r % d.hx);
  const int iy = (int)((r / d.hx) % d.ny);
  const int iz = (int)(r / ((size_t)d.hx * d.ny));
  const int cy = fft2c(iy, d.ny, d.hy3, d.Ky), cz = fft2c(iz, d.nz, d.hz3, d.Kz);
  cd v = cmake(0.0, 0.0);
  if (ix <= d.hx3 && cy >= 0 && cz >= 0) {
    v = S[(size_t)f * d.PS + ((size_t)cz * d.Ky + cy) * d.Kx + ix];
    if (f < nzeta) {
      const double kx = d.kx0 * ix, ky = d.ky0 * fft2n(iy, d.ny);
      const double k2 = kx * kx + ky * ky;
      v = cscale(v, k2 > 0.0 ? -1.0 / k2 : 0.0);
    }
  }
  out[idx] = v;
}

// ---- forcing (Eq. 25; Q17) ---------------------------------------------------
__device__ __forceinline__ double rng_u01(unsigned long long seed, unsigned long long counter) {
  unsigned long long z = seed + 0x9E3779B97F4A7C15ULL * (counter + 1ULL);
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
  z ^= z >> 27; z *= 0x94D049BB133111EBULL;
  z ^= z >> 31;
  return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}
// pairs: int3 (nx >= 0, ny, nz) canonical members.  One thread per (field, pair).
__global__ void k_forcing(Dims d, cd* __restrict__ S, const int* __restrict__ pairs, int npairs, double amp,
                          unsigned long long seed, const double* __restrict__ scal) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 2 * npairs) return;
  const long long step = (long long)scal[SC_STEP];
  const int f = i / npairs, ip = i % npairs;
  const int nx_ = pairs[3 * ip], ny_ = pairs[3 * ip + 1], nz_ = pairs[3 * ip + 2];
  const unsigned long long base = (((unsigned long long)step * 2ULL + (unsigned long long)f) * (unsigned long long)npairs + (unsigned long long)ip) * 2ULL;
  const double u1 = rng_u01(seed, base), u2 = rng_u01(seed, base + 1ULL);
  const double rad = sqrt(-2.0 * log(1.0 - u1));
  double sn, cs;
  sincos(2.0 * 3.14159265358979323846 * u2, &sn, &cs);
  const double sc = amp * sqrt(scal[SC_DT]) * 0.70710678118654752440;
  const cd dxi = cmake(sc * rad * cs, sc * rad * sn);
  const double kx = d.kx0 * nx_, ky = d.ky0 * ny_;
  const double k2 = kx * kx + ky * ky;
  const int cy = ny_ >= 0 ? ny_ : ny_ + d.Ky, cz = nz_ >= 0 ? nz_ : nz_ + d.Kz;
  cd* w = S + (size_t)f * d.PS;
  const size_t i1 = ((size_t)cz * d.Ky + cy) * d.Kx + nx_;
  w[i1] = cmake(w[i1].x - k2 * dxi.x, w[i1].y - k2 * dxi.y);
  if (nx_ == 0) {   // the conjugate partner (0,-ny,-nz) lives in the stored half-plane too
    const int cy2 = (-ny_) >= 0 ? -ny_ : -ny_ + d.Ky, cz2 = (-nz_) >= 0 ? -nz_ : -nz_ + d.Kz;
    const size_t i2 = ((size_t)cz2 * d.Ky + cy2) * d.Kx;
    w[i2] = cmake(w[i2].x - k2 * dxi.x, w[i2].y + k2 * dxi.y);
  }
}

// g_0 forcing of the velocity-space benchmark (Q26): one thread.
__global__ void k_forcing_g(Dims d, cd* __restrict__ S, int nzf, double amp, unsigned long long seed,
                            const double* __restrict__ scal) {
  const long long step = (long long)scal[SC_STEP];
  const unsigned long long key = seed ^ 0xA5A5A5A5A5A5A5A5ULL;
  const double u1 = rng_u01(key, 2ULL * (unsigned long long)step), u2 = rng_u01(key, 2ULL * (unsigned long long)step + 1ULL);
  const double rad = sqrt(-2.0 * log(1.0 - u1));
  double sn, cs;
  sincos(2.0 * 3.14159265358979323846 * u2, &sn, &cs);
  const double sc = amp * sqrt(scal[SC_DT]) * 0.70710678118654752440;
  const cd dg = cmake(sc * rad * cs, sc * rad * sn);
  cd* g0 = S + (size_t)2 * d.PS;
  const size_t plane = (size_t)d.Ky * d.Kx;
  const size_t i1 = (size_t)nzf * plane, i2 = (size_t)(d.Kz - nzf) * plane;      // (kx, ky) = (0, 0); kz = +nzf, -nzf
  g0[i1] = cmake(g0[i1].x + dg.x, g0[i1].y + dg.y);
  g0[i2] = cmake(g0[i2].x + dg.x, g0[i2].y - dg.y);
}

// ---- energies (Q14): deterministic two-level reduction ---------------------------------------
// partial[b][5] = { E+, E-, E_kin, E_mag, W_g } of block b; half-plane weight 1 at kx = 0, else 2.
__global__ void __launch_bounds__(256) k_energy_partial(Dims d, const cd* __restrict__ S, double* __restrict__ partial) {
  double acc[5] = {0, 0, 0, 0, 0};
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < d.PS; idx += (size_t)gridDim.x * blockDim.x) {
    const int cx = (int)(idx % d.Kx);
    const int cy = (int)((idx / d.Kx) % d.Ky);
    const double kx = d.kx0 * cx, ky = d.ky0 * c2n(cy, d.hy3, d.Ky);
    const double k2 = kx * kx + ky * ky;
    const double wgt = cx == 0 ? 1.0 : 2.0;
    if (k2 > 0.0) {
      const cd wp = S[idx], wm = S[d.PS + idx];
      const double ik2 = 1.0 / k2;                       // k2 |xi|^2 = |w|^2 / k2
      const double ap = (wp.x * wp.x + wp.y * wp.y) * ik2, am = (wm.x * wm.x + wm.y * wm.y) * ik2;
      const cd sp = cmake(0.5 * (wp.x + wm.x), 0.5 * (wp.y + wm.y)), sm = cmake(0.5 * (wp.x - wm.x), 0.5 * (wp.y - wm.y));
      acc[0] += wgt * 0.25 * ap;
      acc[1] += wgt * 0.25 * am;
      acc[2] += wgt * 0.5 * (sp.x * sp.x + sp.y * sp.y) * ik2;
      acc[3] += wgt * 0.5 * (sm.x * sm.x + sm.y * sm.y) * ik2;
    }
    double g2 = 0.0;
    for (int m = d.own_lo; m < d.own_hi; ++m) {          // owned moments (a shard's halo copies belong to its neighbours)
      const cd g = S[(size_t)(2 + m) * d.PS + idx];
      g2 += g.x * g.x + g.y * g.y;
    }
    acc[4] += wgt * 0.5 * g2;
  }
  __shared__ double sh[8][5];
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double v = acc[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5][k] = v;
  }
  __syncthreads();
  if (threadIdx.x < 5) {
    double v = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += sh[w][threadIdx.x];
    partial[(size_t)blockIdx.x * 5 + threadIdx.x] = v;
  }
}
// Final sum in a fixed order (deterministic): warp k sums quantity k, lane l takes blocks l, l+32, ... then a shuffle tree.
// advance == 0: the record {t, E_A, E+, E-, Ekin, Emag, Wg} goes to rec.  advance != 0: t += dt, rec is the energy HISTORY and the
// record goes to its slot (step - hist_base), then the step number moves on -- all on the device, so that the launch has the same
// arguments every step (CUDA graph replay).
__global__ void __launch_bounds__(160) k_energy_final(const double* __restrict__ partial, int nblocks, double* __restrict__ rec, long long hist_base,
                                                      double* scal, int advance) {
  __shared__ double sh[5];
  const int k = threadIdx.x >> 5, l = threadIdx.x & 31;
  double v = 0.0;
  for (int b = l; b < nblocks; b += 32) v += partial[(size_t)b * 5 + k];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if (l == 0) sh[k] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    if (advance) {
      scal[SC_T] += scal[SC_DT]; scal[SC_LASTDT] = scal[SC_DT];
      rec += ((long long)scal[SC_STEP] - hist_base) * 7;
      scal[SC_STEP] += 1.0;
    }
    rec[0] = scal[SC_T];
    rec[1] = sh[0] + sh[1]; rec[2] = sh[0]; rec[3] = sh[1]; rec[4] = sh[2]; rec[5] = sh[3]; rec[6] = sh[4];
  }
}

// ---- shell spectrum (Eq. 26; Q15) -----------------------------------------------------------------------
// step 1: per (cy,cx) sum over cz of the mode energy (deterministic serial sum), with half-plane weight.
__global__ void __launch_bounds__(256) k_spec_columns(Dims d, const cd* __restrict__ S, double* __restrict__ col, int literal) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int plane = d.Ky * d.Kx;
  if (i >= plane) return;
  const int cx = i % d.Kx, cy = i / d.Kx;
  const double kx = d.kx0 * cx, ky = d.ky0 * c2n(cy, d.hy3, d.Ky);
  const double k2 = kx * kx + ky * ky;
  double e = 0.0;
  if (k2 > 0.0) {
    for (int cz = 0; cz < d.Kz; ++cz) {
      const cd wp = S[(size_t)cz * plane + i], wm = S[d.PS + (size_t)cz * plane + i];
      e += (wp.x * wp.x + wp.y * wp.y) + (wm.x * wm.x + wm.y * wm.y);
    }
    // |xi|^2 = |w|^2/k2^2 ; mode energy 1/4 k2 |xi|^2 = 1/4 |w|^2 / k2
    e *= literal ? 1.0 / (k2 * k2) : 0.25 / k2;
    e *= (cx == 0 ? 1.0 : 2.0);
  }
  col[i] = e;
}
// step 2: one block per bin j = floor(kperp/dk + 1/2); fixed-order strided loop + tree reduction.
__global__ void __launch_bounds__(256) k_spec_bins(Dims d, const double* __restrict__ col, double dk, double* __restrict__ out) {
  const int j = blockIdx.x;
  const int plane = d.Ky * d.Kx;
  double acc = 0.0;
  for (int i = threadIdx.x; i < plane; i += blockDim.x) {
    const int cx = i % d.Kx, cy = i / d.Kx;
    const double kx = d.kx0 * cx, ky = d.ky0 * c2n(cy, d.hy3, d.Ky);
    const int b = (int)floor(sqrt(kx * kx + ky * ky) / dk + 0.5);
    if (b == j) acc += col[i];
  }
  __shared__ double sh[256];
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[j] = sh[0];
}

// ---- Hermite spectrum C_m = <|g_m|^2> (Eq. 27) and parallel spectrum E(|n_z|) (Q25) ----
// One block per row r: a fixed-order strided sum and a tree reduction (deterministic).
//   kind 0: r = m,  C_m = sum_k |g_m(k)|^2 over the full spectrum (half-plane weight 1 at kx = 0, else 2)
//   kind 1: r = cz, the Alfvenic mode energy 1/4 |w+-|^2 / kperp^2 summed over the (kx,ky) plane of that kz
__global__ void __launch_bounds__(256) k_row_sums(Dims d, const cd* __restrict__ S, int kind, double* __restrict__ out) {
  const int r = blockIdx.x;
  const int plane = d.Ky * d.Kx;
  double acc = 0.0;
  if (kind == 0) {
    const cd* g = S + (size_t)(2 + r) * d.PS;
    for (size_t i = threadIdx.x; i < d.PS; i += blockDim.x) {
      const cd v = g[i];
      acc += ((int)(i % d.Kx) == 0 ? 1.0 : 2.0) * (v.x * v.x + v.y * v.y);
    }
  } else {
    for (int i = threadIdx.x; i < plane; i += blockDim.x) {
      const int cx = i % d.Kx, cy = i / d.Kx;
      const double kx = d.kx0 * cx, ky = d.ky0 * c2n(cy, d.hy3, d.Ky);
      const double k2 = kx * kx + ky * ky;
      if (k2 > 0.0) {
        const cd wp = S[(size_t)r * plane + i], wm = S[d.PS + (size_t)r * plane + i];
        acc += (cx == 0 ? 1.0 : 2.0) * 0.25 * ((wp.x * wp.x + wp.y * wp.y) + (wm.x * wm.x + wm.y * wm.y)) / k2;
      }
    }
  }
  __shared__ double sh[256];
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[r] = sh[0];
}
// bins j = |n_z|: out[j] = row(+j) + row(-j)
__global__ void k_kpar_bins(Dims d, const double* __restrict__ rows, int nbins, double* __restrict__ out) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nbins) return;
  double v = 0.0;
  if (j <= d.hz3) {
    v = rows[j];
    if (j > 0) v += rows[d.Kz - j];
  }
  out[j] = v;
}

// ---- launchers ---------------------------------------------------------------------------------------------
static inline int nblk(size_t n, int b) { return (int)((n + b - 1) / b); }

cudaError_t launch_tables(const Dims& d, const PhysParams& p, const double* scal, double* tabz, double* tabp, cudaStream_t st) {
  const int n = d.Ky * d.Kx > d.Kz ? d.Ky * d.Kx : d.Kz;
  k_tables<<<nblk((size_t)n, 256), 256, 0, st>>>(d, p, scal, tabz, tabp);
  return cudaGetLastError();
}
cudaError_t launch_prepare_dt(double fixed_dt, double cfl_dxy, double dt_max, const unsigned long long* maxbits, double* scal,
                              const double* crate, double* collfac, int M, cudaStream_t st) {
  k_prepare_dt<<<1, 128, 0, st>>>(fixed_dt, cfl_dxy, dt_max, maxbits, scal, crate, collfac, M);
  return cudaGetLastError();
}
cudaError_t launch_zero_u64(unsigned long long* p, cudaStream_t st) { k_zero_u64<<<1, 1, 0, st>>>(p); return cudaGetLastError(); }
cudaError_t launch_pack(const Dims& d, const cd* in, cd* S, int nfields, int nzeta, cudaStream_t st) {
  k_pack<<<nblk(d.PS * (size_t)nfields, 256), 256, 0, st>>>(d, in, S, nfields, nzeta);
  return cudaGetLastError();
}
cudaError_t launch_unpack(const Dims& d, const cd* S, cd* out, int nfields, int nzeta, cudaStream_t st) {
  const size_t hp = (size_t)d.nz * d.ny * d.hx;
  k_unpack<<<nblk(hp * (size_t)nfields, 256), 256, 0, st>>>(d, S, out, nfields, nzeta);
  return cudaGetLastError();
}
cudaError_t launch_forcing(const Dims& d, cd* S, const int* pairs, int npairs, double amp, unsigned long long seed,
                           const double* scal, cudaStream_t st) {
  k_forcing<<<nblk(2 * (size_t)npairs, 64), 64, 0, st>>>(d, S, pairs, npairs, amp, seed, scal);
  return cudaGetLastError();
}
cudaError_t launch_energy(const Dims& d, const cd* S, double* partial, int nblocks, double* rec, long long hist_base, double* scal, int advance,
                          cudaStream_t st) {
  k_energy_partial<<<nblocks, 256, 0, st>>>(d, S, partial);
  k_energy_final<<<1, 160, 0, st>>>(partial, nblocks, rec, hist_base, scal, advance);
  return cudaGetLastError();
}
cudaError_t launch_spectrum(const Dims& d, const cd* S, double* col, int nbins, int literal, double dk, double* out, cudaStream_t st) {
  k_spec_columns<<<nblk((size_t)d.Ky * d.Kx, 256), 256, 0, st>>>(d, S, col, literal);
  k_spec_bins<<<nbins, 256, 0, st>>>(d, col, dk, out);
  return cudaGetLastError();
}
cudaError_t launch_hermite_spectrum(const Dims& d, const cd* S, double* out, cudaStream_t st) {
  k_row_sums<<<d.M, 256, 0, st>>>(d, S, 0, out);
  return cudaGetLastError();
}
cudaError_t launch_kpar_spectrum(const Dims& d, const cd* S, double* rows, int nbins, double* out, cudaStream_t st) {
  k_row_sums<<<d.Kz, 256, 0, st>>>(d, S, 1, rows);
  k_kpar_bins<<<nblk((size_t)nbins, 128), 128, 0, st>>>(d, rows, nbins, out);
  return cudaGetLastError();
}
cudaError_t launch_forcing_g(const Dims& d, cd* S, int nzf, double amp, unsigned long long seed,
                             const double* scal, cudaStream_t st) {
  k_forcing_g<<<1, 1, 0, st>>>(d, S, nzf, amp, seed, scal);
  return cudaGetLastError();
}
