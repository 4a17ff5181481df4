// hermite.cu -- exact propagator of the Hermite streaming / phase-mixing operator (hermite_exact = 1; Q30).
//
// For one (kx, ky, kz) the linear part of Eq. 6 is  d g/dt = s i kz (I - T) g  over the moment index, T the
// symmetric tridiagonal coupling matrix T[m][m-1] = sqrt(m/2), T[m][m+1] = sqrt((m+1)/2) (absorbing closure g_M = 0) -- the
// Jacobi matrix of the Hermite functions.  With T = V diag(lambda) V^T (computed once on the host) the propagator over a
// time tau is   P(tau) = V diag( exp(s i kz (1 - lambda_j) tau) ) V^T,   a dense M x M complex matrix per kz:
//   k_hermite_propagator  builds P(dt/2) for every retained kz (and both species) from the device-resident dt,
//   k_hermite_apply       applies it to the moment vector of every retained mode -- a small dense contraction
//                         (M^2 complex multiply-adds per mode), optionally followed by the dissipation factors of Eq. 17-19.
// The paper advances g_m by plain RK2 (Alg. 1 l.4, l.9) and names exponential integrators as future work (PAPER.md:657,
// 829); this variant lifts the dt < dz/v_th constraint of PAPER.md:214.  It is not on the default path.
#include <cmath>
#include <vector>
#include "common.cuh"

// Host: eigen-decomposition of a real symmetric matrix by cyclic Jacobi rotations (A is destroyed; V columns = eigenvectors).
void jacobi_eigh(int n, std::vector<double>& A, std::vector<double>& V, std::vector<double>& lam) {
  V.assign((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) V[(size_t)i * n + i] = 1.0;
  for (int sweep = 0; sweep < 64; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) (i == j ? diag : off) += A[(size_t)i * n + j] * A[(size_t)i * n + j];
    if (off <= 1e-32 * (diag + 1e-300)) break;
    for (int p = 0; p < n - 1; ++p)
      for (int q = p + 1; q < n; ++q) {
        const double apq = A[(size_t)p * n + q];
        if (apq == 0.0) continue;
        const double theta = (A[(size_t)q * n + q] - A[(size_t)p * n + p]) / (2.0 * apq);
        const double t = (theta >= 0.0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
        const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
        for (int k = 0; k < n; ++k) {          // A <- A J
          const double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
          A[(size_t)k * n + p] = c * akp - s * akq; A[(size_t)k * n + q] = s * akp + c * akq;
        }
        for (int k = 0; k < n; ++k) {          // A <- J^T A
          const double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
          A[(size_t)p * n + k] = c * apk - s * aqk; A[(size_t)q * n + k] = s * apk + c * aqk;
        }
        for (int k = 0; k < n; ++k) {          // V <- V J
          const double vkp = V[(size_t)k * n + p], vkq = V[(size_t)k * n + q];
          V[(size_t)k * n + p] = c * vkp - s * vkq; V[(size_t)k * n + q] = s * vkp + c * vkq;
        }
      }
  }
  lam.resize(n);
  for (int i = 0; i < n; ++i) lam[i] = A[(size_t)i * n + i];
}

// P[sp][cz][m][k] = sum_j V[m][j] V[k][j] exp(i s_sp kz (1 - lambda_j) tau),  tau = frac * dt.  One block per (cz, sp).
__global__ void __launch_bounds__(256) k_hermite_propagator(Dims d, double skz_sign, double frac, const double* __restrict__ scal,
                                                            const double* __restrict__ V, const double* __restrict__ lam,
                                                            cd* __restrict__ P) {
  extern __shared__ cd ph[];                    // Msp phases
  const int M = d.Msp, cz = blockIdx.x, sp = blockIdx.y;
  const double tau = frac * scal[SC_DT];
  const double skz = (sp == 0 ? skz_sign : -skz_sign) * d.kz0 * c2n(cz, d.hz3, d.Kz);
  for (int j = threadIdx.x; j < M; j += blockDim.x) {
    double sn, cs;
    sincos(skz * (1.0 - lam[j]) * tau, &sn, &cs);
    ph[j] = cmake(cs, sn);
  }
  __syncthreads();
  cd* out = P + ((size_t)sp * d.Kz + cz) * M * M;
  for (int e = threadIdx.x; e < M * M; e += blockDim.x) {
    const int m = e / M, k = e % M;
    double ar = 0.0, ai = 0.0;
    for (int j = 0; j < M; ++j) {
      const double w = V[(size_t)m * M + j] * V[(size_t)k * M + j];
      ar = fma(w, ph[j].x, ar); ai = fma(w, ph[j].y, ai);
    }
    out[e] = cmake(ar, ai);
  }
}

// out[sp*Msp + m][cz][pt] = fac * sum_k P[sp][cz][m][k] in[sp*Msp + k][cz][pt]  for the moment fields of the compact arrays
// `in`, `out` (pointers to field 0 = w+; must not alias).  One block: 128 consecutive (cy,cx) points of one kz plane, one
// species, MO consecutive output moments; the MO rows of P sit in shared memory.  diss != 0: fac = collfac[m] * tabp[pt].g *
// tabz[cz].g, the exponential dissipation of Eq. 17-19 applied after the full step (Alg. 2 l.12-14).
#define GD_HX_MO 8
__global__ void __launch_bounds__(128) k_hermite_apply(Dims d, const cd* __restrict__ in, cd* __restrict__ out, const cd* __restrict__ P,
                                                       int diss, const double* __restrict__ collfac, const double* __restrict__ tabz,
                                                       const double* __restrict__ tabp) {
  extern __shared__ cd rows[];                  // [MO][Msp]
  const int M = d.Msp, plane = d.Ky * d.Kx;
  const int nchunk = (M + GD_HX_MO - 1) / GD_HX_MO;
  const int cz = blockIdx.y, sp = blockIdx.z / nchunk, m0 = (blockIdx.z % nchunk) * GD_HX_MO;
  const int nmo = min(GD_HX_MO, M - m0);
  const cd* Pz = P + ((size_t)sp * d.Kz + cz) * M * M + (size_t)m0 * M;
  for (int e = threadIdx.x; e < nmo * M; e += blockDim.x) rows[e] = Pz[e];
  __syncthreads();
  const int pt = blockIdx.x * blockDim.x + threadIdx.x;
  if (pt >= plane) return;
  const size_t idx = (size_t)cz * plane + pt;
  cd acc[GD_HX_MO];
#pragma unroll
  for (int o = 0; o < GD_HX_MO; ++o) acc[o] = cmake(0.0, 0.0);
  const cd* src = in + (size_t)(2 + sp * M) * d.PS + idx;
  for (int k = 0; k < M; ++k) {
    const cd x = ldg_cd(src + (size_t)k * d.PS);
#pragma unroll
    for (int o = 0; o < GD_HX_MO; ++o) {
      if (o < nmo) {
        const cd w = rows[o * M + k];
        acc[o].x = fma(w.x, x.x, fma(-w.y, x.y, acc[o].x));
        acc[o].y = fma(w.x, x.y, fma(w.y, x.x, acc[o].y));
      }
    }
  }
  const double fk = diss ? tabp[2 * pt + 1] * tabz[6 * cz + 5] : 1.0;
#pragma unroll
  for (int o = 0; o < GD_HX_MO; ++o) {
    if (o < nmo) {
      const int f = sp * M + m0 + o;
      const double fac = diss ? fk * collfac[f] : 1.0;
      st_cd(out + (size_t)(2 + f) * d.PS + idx, cscale(acc[o], fac));
    }
  }
}

cudaError_t launch_hermite_propagator(const Dims& d, int g_sign, double frac, const double* scal, const double* V, const double* lam,
                                      cd* P, cudaStream_t st) {
  const int nsp = d.M / d.Msp;
  k_hermite_propagator<<<dim3(d.Kz, nsp), 256, (size_t)d.Msp * sizeof(cd), st>>>(d, (double)g_sign, frac, scal, V, lam, P);
  return cudaGetLastError();
}
cudaError_t launch_hermite_apply(const Dims& d, const cd* in, cd* out, const cd* P, int diss, const double* collfac,
                                 const double* tabz, const double* tabp, cudaStream_t st) {
  const int nsp = d.M / d.Msp, plane = d.Ky * d.Kx;
  const int nchunk = (d.Msp + GD_HX_MO - 1) / GD_HX_MO;
  k_hermite_apply<<<dim3((plane + 127) / 128, d.Kz, nsp * nchunk), 128, (size_t)GD_HX_MO * d.Msp * sizeof(cd), st>>>(
      d, in, out, P, diss, collfac, tabz, tabp);
  return cudaGetLastError();
}
