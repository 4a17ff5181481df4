// gandalf_oracle.cpp -- CPU ORACLE for the GANDALF KRMHD hot path.  TEST INFRASTRUCTURE ONLY.
//
// This file is the plain, slow, obviously-correct restatement of what the hot path computes,
// written from /root/reference/PAPER.md (arXiv 2511.21891).  It is NOT part of the product:
// only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load it.  It shares no code, header, table or helper with paper_2511_21891_b200/csrc.
//
// What it follows (PAPER.md line numbers, section / equation):
//   * Fourier representation, f(x) = sum_k fhat(k) exp(+i k.x), k = 2 pi n / L   PAPER.md:125-128 (Eq. 9)
//   * spectral derivative  d/dx_j <-> i k_j, Laplacian <-> -kperp^2             PAPER.md:134-138 (Eq. 10-11)
//   * pseudo-spectral Poisson bracket {P,Q} = PxQy - PyQx                        PAPER.md:51, 140-142 (Sec. 3.1)
//   * 2/3 dealiasing (rectangular, strict ">")                                   PAPER.md:251-257 (Eq. 20)
//   * Elsasser RMHD equations                                                    PAPER.md:49 (Eq. 1), 154-156 (Eq. 12)
//   * Hermite hierarchy                                                          PAPER.md:89-93 (Eq. 6a-c), closure 105
//   * integrating-factor RK2 (midpoint) step                                     PAPER.md:164-208 (Eq. 14-15, Alg. 1)
//   * exponential dissipation                                                    PAPER.md:226-245 (Eq. 17-19)
//   * complete step                                                              PAPER.md:297-315 (Alg. 2)
//   * advective CFL                                                              PAPER.md:214-218 (Eq. 16)
//   * forcing                                                                    PAPER.md:560-564 (Eq. 25)
//   * shell spectrum                                                             PAPER.md:570-574 (Eq. 26)
// Readings of silent / ambiguous passages are the ones listed in DESIGN.md ("Readings", Q1-Q24).
//
// Data model: FULL complex spectrum fhat[nz][ny][nx] for every field (no half-plane packing,
// deliberately unlike the GPU path), physical normalisation fhat = (1/N) sum_x f exp(-i k.x).
// FFT: own iterative radix-2 with every twiddle from cos/sin (no recurrences); an O(N^2) DFT is
// exported to test it.  Everything is fp64 (complex128 in the paper).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): P0 FFT vs DFT; P1 Alfven wave exact phase; P2
// single-mode bracket closed form; P3 bracket = truncated convolution sum (brute force); P4
// ideal invariants per RHS; P5 Orszag-Tang energies and drift; P6 mask counts; P7 exact
// dissipation decay; P8 Hermite free streaming (Jacobi matrix / closed-form envelope);
// P10 spectrum sums to E_A; P11 forcing power and Hermitian consistency.
// Unpinned (stated here as required): the driven k^-5/3 slope, E_total~1.73e4 and the Hermite
// m^-1/2 slope of PAPER.md:575, 617 -- "parity unpinned" for those long-run statistics only.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;

extern "C" {

// Mirrors the fields a caller sets; the layout is private to the oracle (tests fill it by name
// through ctypes).  Meaning of each field: see include/gandalf.h in the product, which was
// written separately from the same DESIGN.md table.
struct oracle_params {
  int nx, ny, nz;
  int M;
  double Lx, Ly, Lz, vA;
  double eta; int r; int eta_normalized;
  double eta_z; int r_z;
  double eta_g;
  double nu_coll; double p;
  int closure;        // 0 absorbing, 1 reflecting
  int if_variant;     // 0 paper-literal double phase, 1 standard IF midpoint
  int g_sign;         // +1 / -1
  int nonlinear;      // 1 / 0
  int hermite_coeff;  // 0 uniform sqrt(m/2), sqrt((m+1)/2); 1 literal Eq. 6a/6b first coefficients
  double force_eps; int force_nperp_min, force_nperp_max, force_nz_max;
  unsigned long long seed;
  double cfl;
  double force_g_amp; int force_g_nz;   // g_0 forcing at k = (0,0,+-nz) (Q26)
  int nspecies;       // 1: g (sign g_sign);  2: g^+ (g_sign) then g^- (-g_sign), M moments each (Q27)
  double dt_max;      // > 0: upper bound of the CFL step of Eq. 16 (and the step taken when the flow vanishes); 0 = none (Q29)
  int hermite_exact;  // 1: exact propagator exp(s i kz (I - T) dt) for the streaming / phase-mixing terms of Eq. 6 (Q30)
  // Moment shard (Q31): this instance holds the moments m_offset .. m_offset+M-1 of a hierarchy of
  // M_global moments (0 = not sharded, M_global = M).  If m_offset > 0 its first field is a HALO copy of the neighbour's g_{m_offset}
  // and if m_offset+M < M_global its last field is one: halos are inputs (set by the caller after every stage), their own update
  // is meaningless, and they are left out of W_g.  The arithmetic of an owned moment is that of the unsharded run, operation by operation.
  int m_offset, M_global;
};

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// 1-D transforms.  sign = -1: forward kernel exp(-2 pi i jk/n); sign = +1: inverse kernel.
// Neither applies a 1/n factor.
// ---------------------------------------------------------------------------------------------
static void dft_naive(int n, int sign, const cplx* in, cplx* out) {
  for (int k = 0; k < n; ++k) {
    cplx acc(0.0, 0.0);
    for (int j = 0; j < n; ++j) {
      long long jk = ((long long)j * k) % n;
      double ang = sign * 2.0 * PI * (double)jk / (double)n;
      acc += in[j] * cplx(std::cos(ang), std::sin(ang));
    }
    out[k] = acc;
  }
}

// Iterative radix-2 decimation-in-time, in place, n a power of two (n >= 1).
static void fft_radix2(int n, int sign, cplx* a) {
  // bit reversal
  for (int i = 1, j = 0; i < n; ++i) {
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) std::swap(a[i], a[j]);
  }
  for (int len = 2; len <= n; len <<= 1) {
    int half = len >> 1;
    for (int base = 0; base < n; base += len) {
      for (int j = 0; j < half; ++j) {
        double ang = sign * 2.0 * PI * (double)j / (double)len;
        cplx w(std::cos(ang), std::sin(ang));
        cplx u = a[base + j];
        cplx v = a[base + j + half] * w;
        a[base + j] = u + v;
        a[base + j + half] = u - v;
      }
    }
  }
}

static bool is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

// ---------------------------------------------------------------------------------------------
// Context: grid, full-spectrum state (vorticities w+-, moments g_m), time, history.
// ---------------------------------------------------------------------------------------------
struct Field {               // one full complex spectrum or real-space complex array [nz][ny][nx]
  std::vector<cplx> a;
};

struct oracle_ctx {
  oracle_params p;
  int nx, ny, nz, M;                        // M = number of moment FIELDS = nspecies * Msp
  int Msp, nsp;                             // moments per species, species
  size_t N;                                 // nx*ny*nz
  std::vector<double> kx, ky, kz;           // physical wavenumbers per FFT index (Eq. 9 text)
  std::vector<int> mx, my, mz;              // signed integer mode numbers per FFT index
  std::vector<cplx> w[2];                   // w^+ , w^-  
  std::vector<std::vector<cplx>> g;         // g_0 .. g_{M-1}
  std::vector<double> coef_dn, coef_up;     // Eq. 6 coupling coefficients to g_{m-1}, g_{m+1}
  std::vector<cplx> hw[2];                  // half-step (stage) state of Alg. 1 l.3-4 between the two stages of a step
  std::vector<std::vector<cplx>> hg;
  double dt_cur;                            // the step's dt (fixed, or Eq. 16), set by the first stage
  bool stage_pending = false;               // between oracle_step_stage(.., 0) and (.., 1): (hw, hg) hold a half-step state
  int moff, Mg;                             // shard: global index of local moment 0, global moment count (Q31)
  int own_lo, own_hi;                       // owned local moments [own_lo, own_hi): the rest are halos
  double t; long long step; double last_dt;
  std::vector<double> hist;                 // 7 doubles per record: t, E_A, E+, E-, E_kin, E_mag, W_g
  std::string err;
};

static inline size_t IDX(const oracle_ctx* c, int iz, int iy, int ix) {
  return ((size_t)iz * c->ny + iy) * c->nx + ix;
}

static int signed_mode(int i, int n) { return (i < n / 2) ? i : i - n; }  // FFT order 0..n/2-1, -n/2..-1

// Eq. 20 with k_max = Nyquist = pi N / L: |k|/k_max = 2|n|/N > 2/3  <=>  3|n| > N.
static inline bool masked(const oracle_ctx* c, int iz, int iy, int ix) {
  int a = std::abs(c->mx[ix]), b = std::abs(c->my[iy]), d = std::abs(c->mz[iz]);
  return (3 * a > c->nx) || (3 * b > c->ny) || (3 * d > c->nz);
}

// 3-D transform of a full complex array, in place, axis by axis.  sign=-1 forward (and the caller
// applies 1/N), sign=+1 inverse.
static void fft3(const oracle_ctx* c, int sign, std::vector<cplx>& a) {
  const int nx = c->nx, ny = c->ny, nz = c->nz;
  // x lines
#pragma omp parallel for collapse(2) schedule(static)
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy) fft_radix2(nx, sign, &a[((size_t)iz * ny + iy) * nx]);
  // y lines
#pragma omp parallel
  {
    std::vector<cplx> line(ny);
#pragma omp for collapse(2) schedule(static)
    for (int iz = 0; iz < nz; ++iz)
      for (int ix = 0; ix < nx; ++ix) {
        for (int iy = 0; iy < ny; ++iy) line[iy] = a[((size_t)iz * ny + iy) * nx + ix];
        fft_radix2(ny, sign, line.data());
        for (int iy = 0; iy < ny; ++iy) a[((size_t)iz * ny + iy) * nx + ix] = line[iy];
      }
  }
  // z lines
#pragma omp parallel
  {
    std::vector<cplx> line(nz);
#pragma omp for collapse(2) schedule(static)
    for (int iy = 0; iy < ny; ++iy)
      for (int ix = 0; ix < nx; ++ix) {
        for (int iz = 0; iz < nz; ++iz) line[iz] = a[((size_t)iz * ny + iy) * nx + ix];
        fft_radix2(nz, sign, line.data());
        for (int iz = 0; iz < nz; ++iz) a[((size_t)iz * ny + iy) * nx + ix] = line[iz];
      }
  }
}

// Real-space derivative d f / d x_axis from a spectrum: IFFT3(i k f_hat) (Eq. 10).
// The result of a Hermitian spectrum is real; the imaginary part is checked and dropped.
static void deriv_real(const oracle_ctx* c, const std::vector<cplx>& fhat, int axis,
                       std::vector<double>& out, double* max_imag) {
  std::vector<cplx> tmp(c->N);
#pragma omp parallel for collapse(2) schedule(static)
  for (int iz = 0; iz < c->nz; ++iz)
    for (int iy = 0; iy < c->ny; ++iy)
      for (int ix = 0; ix < c->nx; ++ix) {
        double k = (axis == 0) ? c->kx[ix] : c->ky[iy];
        tmp[IDX(c, iz, iy, ix)] = cplx(0.0, k) * fhat[IDX(c, iz, iy, ix)];
      }
  fft3(c, +1, tmp);
  out.resize(c->N);
  double mi = 0.0;
#pragma omp parallel for reduction(max : mi) schedule(static)
  for (size_t i = 0; i < c->N; ++i) {
    out[i] = tmp[i].real();
    double im = std::fabs(tmp[i].imag());
    if (im > mi) mi = im;
  }
  if (max_imag && mi > *max_imag) *max_imag = mi;
}

struct Grad { std::vector<double> x, y; };

static void gradient(const oracle_ctx* c, const std::vector<cplx>& fhat, Grad& g) {
  deriv_real(c, fhat, 0, g.x, nullptr);
  deriv_real(c, fhat, 1, g.y, nullptr);
}

// Pseudo-spectral dealiased bracket (PAPER.md:140 then Eq. 20): FFT3(Px Qy - Py Qx)/N, masked.
static void bracket_from_grads(const oracle_ctx* c, const Grad& P, const Grad& Q, std::vector<cplx>& out) {
  out.assign(c->N, cplx(0.0, 0.0));
#pragma omp parallel for schedule(static)
  for (size_t i = 0; i < c->N; ++i) out[i] = cplx(P.x[i] * Q.y[i] - P.y[i] * Q.x[i], 0.0);
  fft3(c, -1, out);
  const double inv = 1.0 / (double)c->N;
#pragma omp parallel for collapse(2) schedule(static)
  for (int iz = 0; iz < c->nz; ++iz)
    for (int iy = 0; iy < c->ny; ++iy)
      for (int ix = 0; ix < c->nx; ++ix) {
        size_t i = IDX(c, iz, iy, ix);
        out[i] = masked(c, iz, iy, ix) ? cplx(0.0, 0.0) : out[i] * inv;
      }
}

// ---------------------------------------------------------------------------------------------
// RHS evaluation: oracle algorithm step 1 of DESIGN.md "Oracle algorithm" (Alg. 2 l.3-5, 7-9).
//   N^+-  = -1/2 A -+ 1/2 kperp^2 B,  A = {xi+,w-}^ + {xi-,w+}^,  B = {xi+,xi-}^      (Eq. 1 with Eq. 11)
//   H_m   = -{Phi,g_m}^ + a_m {Psi,g_{m-1}}^ + b_m {Psi,g_{m+1}}^
//           + s i kz [ g_m - a_m g_{m-1} - b_m g_{m+1} ]                               (Eq. 6a-c, v_A = 1)
// Each bracket is evaluated separately (no real-space combination).
// ---------------------------------------------------------------------------------------------
struct State {
  std::vector<cplx> w[2];
  std::vector<std::vector<cplx>> g;
};

static inline double kperp2(const oracle_ctx* c, int iy, int ix) { return c->kx[ix] * c->kx[ix] + c->ky[iy] * c->ky[iy]; }

static void potentials(const oracle_ctx* c, const std::vector<cplx>& w, std::vector<cplx>& xi) {
  xi.assign(c->N, cplx(0.0, 0.0));
#pragma omp parallel for collapse(2) schedule(static)
  for (int iz = 0; iz < c->nz; ++iz)
    for (int iy = 0; iy < c->ny; ++iy)
      for (int ix = 0; ix < c->nx; ++ix) {
        double k2 = kperp2(c, iy, ix);
        size_t i = IDX(c, iz, iy, ix);
        xi[i] = (k2 > 0.0) ? -w[i] / k2 : cplx(0.0, 0.0);   // xi = -w / kperp^2; 0 at kperp = 0 (Q22)
      }
}

// The neighbour g_{m} with the closure applied for m == M: absorbing -> none,
// reflecting -> g_{M-2}.  Returns -1 when the neighbour is identically zero.
static int neighbour_index(const oracle_ctx* c, int sp, int m) {   // field index of moment m of species sp, or -1
  const int M = c->Msp;
  if (m < 0) return -1;
  if (m < M) return sp * M + m;
  if (m == M && c->moff + M == c->Mg && c->p.closure == 1 && M >= 2) return sp * M + M - 2;   // the closure sits at the GLOBAL end (Q31)
  return -1;
}

static void rhs_eval(const oracle_ctx* c, const State& s, State& out, double* max_gradphi2, bool with_streaming = true) {
  const int M = c->M;
  out.w[0].assign(c->N, cplx(0, 0));
  out.w[1].assign(c->N, cplx(0, 0));
  out.g.assign(M, std::vector<cplx>());
  for (int m = 0; m < M; ++m) out.g[m].assign(c->N, cplx(0, 0));

  std::vector<cplx> xi[2], Phi(c->N), Psi(c->N);
  potentials(c, s.w[0], xi[0]);
  potentials(c, s.w[1], xi[1]);
#pragma omp parallel for schedule(static)
  for (size_t i = 0; i < c->N; ++i) {
    Phi[i] = 0.5 * (xi[0][i] + xi[1][i]);    // xi+- = Phi +- Psi
    Psi[i] = 0.5 * (xi[0][i] - xi[1][i]);
  }

  if (max_gradphi2) {   // Eq. 16: max |grad_perp Phi| over the real-space grid
    Grad gP;
    gradient(c, Phi, gP);
    double mx = 0.0;
    for (size_t i = 0; i < c->N; ++i) {
      double v = gP.x[i] * gP.x[i] + gP.y[i] * gP.y[i];
      if (v > mx) mx = v;
    }
    *max_gradphi2 = mx;
  }

  if (c->p.nonlinear) {
    Grad gxi[2], gw[2];
    for (int a = 0; a < 2; ++a) { gradient(c, xi[a], gxi[a]); gradient(c, s.w[a], gw[a]); }
    std::vector<cplx> b1, b2, B;
    bracket_from_grads(c, gxi[0], gw[1], b1);     // {xi+, w-}
    bracket_from_grads(c, gxi[1], gw[0], b2);     // {xi-, w+}
    bracket_from_grads(c, gxi[0], gxi[1], B);     // {xi+, xi-}
#pragma omp parallel for collapse(2) schedule(static)
    for (int iz = 0; iz < c->nz; ++iz)
      for (int iy = 0; iy < c->ny; ++iy)
        for (int ix = 0; ix < c->nx; ++ix) {
          size_t i = IDX(c, iz, iy, ix);
          double k2 = kperp2(c, iy, ix);
          cplx A = b1[i] + b2[i];
          // -1/2 [ A -+ lap B ],  lap -> -kperp^2
          out.w[0][i] = -0.5 * (A - (-k2) * B[i]);
          out.w[1][i] = -0.5 * (A + (-k2) * B[i]);
        }
    if (M > 0) {
      Grad gPhi, gPsi;
      gradient(c, Phi, gPhi);
      gradient(c, Psi, gPsi);
      std::vector<Grad> gg(M);
      for (int m = 0; m < M; ++m) gradient(c, s.g[m], gg[m]);
      std::vector<cplx> br;
      for (int sp = 0; sp < c->nsp; ++sp)                               // the bracket terms of Eq. 6 are the same for g^+ and g^-
        for (int m = 0; m < c->Msp; ++m) {
          const int fi = sp * c->Msp + m;
          bracket_from_grads(c, gPhi, gg[fi], br);                    // {Phi, g_m}
          for (size_t i = 0; i < c->N; ++i) out.g[fi][i] -= br[i];
          int lo = neighbour_index(c, sp, m - 1), hi = neighbour_index(c, sp, m + 1);
          const int gm = c->moff + m;                                 // global moment index (= m unless sharded, Q31)
          if (lo >= 0 && c->coef_dn[gm] != 0.0) {
            bracket_from_grads(c, gPsi, gg[lo], br);                  // {Psi, g_{m-1}}
            for (size_t i = 0; i < c->N; ++i) out.g[fi][i] += c->coef_dn[gm] * br[i];
          }
          if (hi >= 0) {
            bracket_from_grads(c, gPsi, gg[hi], br);                  // {Psi, g_{m+1}}
            for (size_t i = 0; i < c->N; ++i) out.g[fi][i] += c->coef_up[gm] * br[i];
          }
        }
    }
  }
  // linear streaming / phase-mixing terms of Eq. 6 (d/dz -> i kz), sign s = +1 for g^+ (upper signs)
  // (left out when the stepper integrates them exactly, hermite_exact = 1)
  for (int fi = 0; with_streaming && fi < M; ++fi) {
    const int sp = fi / c->Msp, m = fi % c->Msp;
    const double sgn = (sp == 0) ? (double)c->p.g_sign : -(double)c->p.g_sign;   // upper / lower signs of Eq. 6
    int lo = neighbour_index(c, sp, m - 1), hi = neighbour_index(c, sp, m + 1);
    const int gm = c->moff + m;
#pragma omp parallel for collapse(2) schedule(static)
    for (int iz = 0; iz < c->nz; ++iz)
      for (int iy = 0; iy < c->ny; ++iy)
        for (int ix = 0; ix < c->nx; ++ix) {
          size_t i = IDX(c, iz, iy, ix);
          cplx lin = s.g[fi][i];
          if (lo >= 0) lin -= c->coef_dn[gm] * s.g[lo][i];
          if (hi >= 0) lin -= c->coef_up[gm] * s.g[hi][i];
          out.g[fi][i] += cplx(0.0, sgn * c->kz[iz]) * lin;
        }
  }
}

// ---------------------------------------------------------------------------------------------
// Dissipation factors (Eq. 17-19; readings Q9, Q10 in DESIGN.md).
// ---------------------------------------------------------------------------------------------
static double ipow(double x, int n) { double r = 1.0; for (int i = 0; i < n; ++i) r *= x; return r; }

static double perp_rate_shape(const oracle_ctx* c, int iy, int ix) {
  double k2 = kperp2(c, iy, ix);
  if (c->p.eta_normalized) {
    double kxm = PI * c->nx / c->p.Lx, kym = PI * c->ny / c->p.Ly;   // Nyquist wavenumbers
    double k2max = kxm * kxm + kym * kym;                             // max(kx^2+ky^2)
    return ipow(k2 / k2max, c->p.r);                                  // Eq. 18
  }
  return ipow(k2, c->p.r);                                            // Eq. 17 generalised: eta kperp^(2r)
}
static double par_rate_shape(const oracle_ctx* c, int iz) {
  double kzm = PI * c->nz / c->p.Lz;
  return ipow(c->kz[iz] * c->kz[iz] / (kzm * kzm), c->p.r_z);
}

static void apply_dissipation(const oracle_ctx* c, State& s, double dt) {
  const oracle_params& p = c->p;
#pragma omp parallel for collapse(2) schedule(static)
  for (int iz = 0; iz < c->nz; ++iz)
    for (int iy = 0; iy < c->ny; ++iy)
      for (int ix = 0; ix < c->nx; ++ix) {
        size_t i = IDX(c, iz, iy, ix);
        double rate_w = p.eta * perp_rate_shape(c, iy, ix);
        if (p.eta_z > 0.0) rate_w += p.eta_z * par_rate_shape(c, iz);
        double fw = std::exp(-rate_w * dt);
        s.w[0][i] *= fw;
        s.w[1][i] *= fw;
        double rate_gk = 0.0;
        if (p.eta_g > 0.0) {
          rate_gk = p.eta_g * perp_rate_shape(c, iy, ix);
          if (p.eta_z > 0.0) rate_gk += p.eta_z * par_rate_shape(c, iz);
        }
        for (int fi = 0; fi < c->M; ++fi) {
          const int m = fi % c->Msp;
          double rate = rate_gk + p.nu_coll * std::pow((double)(c->moff + m) / (double)c->Mg, 2.0 * p.p);   // Eq. 19 (global m and M, Q31)
          s.g[fi][i] *= std::exp(-rate * dt);
        }
      }
}

// ---------------------------------------------------------------------------------------------
// Forcing (Eq. 25; reading Q17).  Counter-based RNG restated from DESIGN.md.
// ---------------------------------------------------------------------------------------------
static double rng_uniform(unsigned long long seed, unsigned long long counter) {
  unsigned long long z = seed + 0x9E3779B97F4A7C15ULL * (counter + 1ULL);
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
  z ^= z >> 27; z *= 0x94D049BB133111EBULL;
  z ^= z >> 31;
  return (double)(z >> 11) * (1.0 / 9007199254740992.0);   // 2^-53
}

struct ForcedPair { int nx, ny, nz; };

static std::vector<ForcedPair> forced_pairs(const oracle_ctx* c) {
  std::vector<ForcedPair> v;
  const oracle_params& p = c->p;
  int lo2 = p.force_nperp_min * p.force_nperp_min, hi2 = p.force_nperp_max * p.force_nperp_max;
  for (int nz = -p.force_nz_max; nz <= p.force_nz_max; ++nz)
    for (int ny = -p.force_nperp_max; ny <= p.force_nperp_max; ++ny)
      for (int nx = 0; nx <= p.force_nperp_max; ++nx) {
        int n2 = nx * nx + ny * ny;
        if (n2 < lo2 || n2 > hi2 || n2 == 0) continue;
        bool canonical = (nx > 0) || (nx == 0 && ny > 0);
        if (!canonical) continue;
        v.push_back({nx, ny, nz});
      }
  return v;
}

static inline int wrap(int n, int N) { return ((n % N) + N) % N; }

static void apply_forcing(oracle_ctx* c, State& s, double dt) {
  const oracle_params& p = c->p;
  if (!(p.force_eps > 0.0)) return;
  std::vector<ForcedPair> pairs = forced_pairs(c);
  if (pairs.empty()) return;
  double sumk2 = 0.0;
  for (const ForcedPair& q : pairs) {
    double kx = 2 * PI * q.nx / p.Lx, ky = 2 * PI * q.ny / p.Ly;
    sumk2 += 2.0 * (kx * kx + ky * ky);            // both members of the +-k pair
  }
  double a = std::sqrt(2.0 * p.force_eps / sumk2);
  unsigned long long np = pairs.size();
  for (int f = 0; f < 2; ++f)
    for (unsigned long long ip = 0; ip < np; ++ip) {
      const ForcedPair& q = pairs[ip];
      unsigned long long base = (((unsigned long long)c->step * 2ULL + (unsigned long long)f) * np + ip) * 2ULL;
      double u1 = rng_uniform(p.seed, base), u2 = rng_uniform(p.seed, base + 1ULL);
      double rad = std::sqrt(-2.0 * std::log(1.0 - u1));
      double er = rad * std::cos(2.0 * PI * u2), ei = rad * std::sin(2.0 * PI * u2);
      cplx dxi = a * std::sqrt(dt) * cplx(er, ei) / std::sqrt(2.0);
      double kx = 2 * PI * q.nx / p.Lx, ky = 2 * PI * q.ny / p.Ly;
      double k2 = kx * kx + ky * ky;
      size_t i1 = IDX(c, wrap(q.nz, c->nz), wrap(q.ny, c->ny), wrap(q.nx, c->nx));
      size_t i2 = IDX(c, wrap(-q.nz, c->nz), wrap(-q.ny, c->ny), wrap(-q.nx, c->nx));
      s.w[f][i1] += -k2 * dxi;                      // delta w = -kperp^2 delta xi
      s.w[f][i2] += -k2 * std::conj(dxi);
    }
}

// Velocity-space benchmark forcing ("single forced mode k=(0,0,1) in g_0"; reading Q26): after the
// dissipation step, delta g_0(0,0,n) = a_g sqrt(dt) (eta_r + i eta_i)/sqrt(2), the conjugate at (0,0,-n).
// RNG key seed ^ 0xA5A5A5A5A5A5A5A5, counters 2*step and 2*step+1; Box-Muller as in apply_forcing.
static void apply_forcing_g(oracle_ctx* c, State& s, double dt) {
  const oracle_params& p = c->p;
  if (!(p.force_g_amp > 0.0) || c->M < 1 || c->moff != 0) return;   // g_0 lives on the shard with m_offset = 0
  unsigned long long key = p.seed ^ 0xA5A5A5A5A5A5A5A5ULL;
  double u1 = rng_uniform(key, 2ULL * (unsigned long long)c->step), u2 = rng_uniform(key, 2ULL * (unsigned long long)c->step + 1ULL);
  double rad = std::sqrt(-2.0 * std::log(1.0 - u1));
  cplx dg = p.force_g_amp * std::sqrt(dt) * cplx(rad * std::cos(2.0 * PI * u2), rad * std::sin(2.0 * PI * u2)) / std::sqrt(2.0);
  s.g[0][IDX(c, wrap(p.force_g_nz, c->nz), 0, 0)] += dg;
  s.g[0][IDX(c, wrap(-p.force_g_nz, c->nz), 0, 0)] += std::conj(dg);
}

// ---------------------------------------------------------------------------------------------
// Diagnostics (Q14, Q15): sums over the full spectrum.
// ---------------------------------------------------------------------------------------------
static void energies(const oracle_ctx* c, const State& s, double out[6]) {
  double Ep = 0, Em = 0, Ek = 0, Eb = 0, Wg = 0;
  for (int iz = 0; iz < c->nz; ++iz)
    for (int iy = 0; iy < c->ny; ++iy)
      for (int ix = 0; ix < c->nx; ++ix) {
        double k2 = kperp2(c, iy, ix);
        if (!(k2 > 0.0)) continue;
        size_t i = IDX(c, iz, iy, ix);
        cplx xp = -s.w[0][i] / k2, xm = -s.w[1][i] / k2;
        cplx phi = 0.5 * (xp + xm), psi = 0.5 * (xp - xm);
        Ep += 0.25 * k2 * std::norm(xp);
        Em += 0.25 * k2 * std::norm(xm);
        Ek += 0.5 * k2 * std::norm(phi);
        Eb += 0.5 * k2 * std::norm(psi);
      }
  for (int m = c->own_lo; m < c->own_hi; ++m)            // owned moments (all of them unless sharded)
    for (size_t i = 0; i < c->N; ++i) Wg += 0.5 * std::norm(s.g[m][i]);
  out[0] = Ep + Em; out[1] = Ep; out[2] = Em; out[3] = Ek; out[4] = Eb; out[5] = Wg;
}

// ---------------------------------------------------------------------------------------------
// Exact treatment of the Hermite streaming / phase-mixing terms (hermite_exact = 1; Q30; the paper lists
// exponential integrators as future work, and the constraint it lifts at PAPER.md:214).
// For one (kx,ky,kz) the linear part of Eq. 6 is  d g/dt = s i kz (I - T) g  with T[m][m-1] = sqrt(m/2), T[m][m+1] =
// sqrt((m+1)/2) (closure folded in as in rhs_eval).  propagate() applies  exp(s i kz (I - T) tau)  to the moment vector of
// every mode; the matrix exponential is a plain scaling-and-squaring Taylor series.
// ---------------------------------------------------------------------------------------------
static void mat_mul(int n, const std::vector<cplx>& A, const std::vector<cplx>& B, std::vector<cplx>& C) {
  C.assign((size_t)n * n, cplx(0, 0));
  for (int i = 0; i < n; ++i)
    for (int k = 0; k < n; ++k) {
      const cplx a = A[(size_t)i * n + k];
      if (a == cplx(0, 0)) continue;
      for (int j = 0; j < n; ++j) C[(size_t)i * n + j] += a * B[(size_t)k * n + j];
    }
}

static void mat_expm(int n, const std::vector<cplx>& A, std::vector<cplx>& E) {
  double norm1 = 0.0;                                    // max column sum
  for (int j = 0; j < n; ++j) { double cs = 0; for (int i = 0; i < n; ++i) cs += std::abs(A[(size_t)i * n + j]); if (cs > norm1) norm1 = cs; }
  int nsq = 0;
  while (std::ldexp(norm1, -nsq) > 0.25) ++nsq;
  std::vector<cplx> As(A);
  for (auto& v : As) v = cplx(std::ldexp(v.real(), -nsq), std::ldexp(v.imag(), -nsq));
  E.assign((size_t)n * n, cplx(0, 0));
  std::vector<cplx> term((size_t)n * n, cplx(0, 0)), tmp;
  for (int i = 0; i < n; ++i) { E[(size_t)i * n + i] = 1.0; term[(size_t)i * n + i] = 1.0; }
  for (int k = 1; k <= 24; ++k) {                        // 0.25^25 / 25! is far below round-off
    mat_mul(n, term, As, tmp);
    for (size_t i = 0; i < tmp.size(); ++i) { term[i] = tmp[i] / (double)k; E[i] += term[i]; }
  }
  for (int q = 0; q < nsq; ++q) { mat_mul(n, E, E, tmp); E.swap(tmp); }
}

static void streaming_matrix(const oracle_ctx* c, std::vector<double>& T) {     // M_sp x M_sp, real
  const int M = c->Msp;
  T.assign((size_t)M * M, 0.0);
  for (int m = 0; m < M; ++m) {
    int lo = neighbour_index(c, 0, m - 1), hi = neighbour_index(c, 0, m + 1);
    if (lo >= 0) T[(size_t)m * M + lo] += c->coef_dn[m];
    if (hi >= 0) T[(size_t)m * M + hi] += c->coef_up[m];
  }
}

static void propagate(const oracle_ctx* c, std::vector<std::vector<cplx>>& g, double tau) {
  const int M = c->Msp;
  if (M == 0) return;
  std::vector<double> T;
  streaming_matrix(c, T);
  for (int iz = 0; iz < c->nz; ++iz) {
    for (int sp = 0; sp < c->nsp; ++sp) {
      const double sgn = (sp == 0) ? (double)c->p.g_sign : -(double)c->p.g_sign;
      std::vector<cplx> A((size_t)M * M), E;
      for (int i = 0; i < M; ++i)
        for (int j = 0; j < M; ++j) A[(size_t)i * M + j] = cplx(0.0, sgn * c->kz[iz] * tau) * ((i == j ? 1.0 : 0.0) - T[(size_t)i * M + j]);
      mat_expm(M, A, E);
#pragma omp parallel for collapse(2) schedule(static)
      for (int iy = 0; iy < c->ny; ++iy)
        for (int ix = 0; ix < c->nx; ++ix) {
          size_t i = IDX(c, iz, iy, ix);
          std::vector<cplx> in(M), out(M, cplx(0, 0));
          for (int m = 0; m < M; ++m) in[m] = g[sp * M + m][i];
          for (int m = 0; m < M; ++m)
            for (int k = 0; k < M; ++k) out[m] += E[(size_t)m * M + k] * in[k];
          for (int m = 0; m < M; ++m) g[sp * M + m][i] = out[m];
        }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// One complete step (Alg. 2; Alg. 1).
// ---------------------------------------------------------------------------------------------
// The step is written as two stages so that a moment-sharded run (Q31) can refresh its halo moments in between; step_once
// runs them back to back.  Stage 1: RHS at state_n, dt, half-step predictor -> (hw, hg).  Stage 2: midpoint RHS, corrector,
// dissipation, forcing, time and diagnostics.
static int step_stage1(oracle_ctx* c, double dt_in) {
  const int M = c->M;
  State sn; sn.w[0] = c->w[0]; sn.w[1] = c->w[1]; sn.g = c->g;
  State k1, sh;
  double dt = dt_in;
  double maxg2 = 0.0;
  // Alg. 2 l.2: CFL step from state_n (only when the caller asks for it: dt <= 0)
  const bool exact = (c->p.hermite_exact != 0) && M > 0;    // Q30: brackets by the midpoint rule, streaming terms exactly
  rhs_eval(c, sn, k1, (dt_in > 0.0) ? nullptr : &maxg2, !exact);
  if (!(dt_in > 0.0)) {
    double dxy = std::fmin(c->p.Lx / c->nx, c->p.Ly / c->ny);
    if (maxg2 > 0.0) {
      dt = c->p.cfl * dxy / std::sqrt(maxg2);                         // Eq. 16
      if (c->p.dt_max > 0.0 && dt > c->p.dt_max) dt = c->p.dt_max;    // Q29
    } else if (c->p.dt_max > 0.0) {
      dt = c->p.dt_max;                                               // no flow: Eq. 16 gives no bound (Q29)
    } else { c->err = "CFL: max|grad Phi| is zero"; return -1; }
  }
  // Alg. 1 l.3-4: half-step predictor (Eq. 15)
  sh.w[0].resize(c->N); sh.w[1].resize(c->N); sh.g.assign(M, std::vector<cplx>(c->N));
  for (int a = 0; a < 2; ++a) {
    double sg = (a == 0) ? +1.0 : -1.0;
#pragma omp parallel for collapse(2) schedule(static)
    for (int iz = 0; iz < c->nz; ++iz)
      for (int iy = 0; iy < c->ny; ++iy)
        for (int ix = 0; ix < c->nx; ++ix) {
          size_t i = IDX(c, iz, iy, ix);
          double th = c->kz[iz] * c->p.vA * dt;
          cplx ph = cplx(std::cos(0.5 * sg * th), std::sin(0.5 * sg * th));      // exp(+-i theta/2)
          cplx phN = (c->p.if_variant == 0) ? ph : cplx(1.0, 0.0);               // Q6
          sh.w[a][i] = ph * (sn.w[a][i] + phN * (0.5 * dt) * k1.w[a][i]);
        }
  }
  for (int m = 0; m < M; ++m)
    for (size_t i = 0; i < c->N; ++i) sh.g[m][i] = sn.g[m][i] + (0.5 * dt) * k1.g[m][i];
  if (exact) propagate(c, sh.g, 0.5 * dt);                  // g_{n+1/2} = P(dt/2) (g_n + dt/2 R_n),  P(tau) = exp(s i kz (I - T) tau)
  c->hw[0].swap(sh.w[0]); c->hw[1].swap(sh.w[1]); c->hg.swap(sh.g);
  c->dt_cur = dt;
  c->stage_pending = true;
  return 0;
}

static int step_stage2(oracle_ctx* c) {
  const int M = c->M;
  const bool exact = (c->p.hermite_exact != 0) && M > 0;
  const double dt = c->dt_cur;
  State sn; sn.w[0] = c->w[0]; sn.w[1] = c->w[1]; sn.g = c->g;
  State sh; sh.w[0] = c->hw[0]; sh.w[1] = c->hw[1]; sh.g = c->hg;
  State k2;
  // Alg. 1 l.6: midpoint RHS
  rhs_eval(c, sh, k2, nullptr, !exact);
  // Alg. 1 l.8-9: full-step corrector
  State s1; s1.w[0].resize(c->N); s1.w[1].resize(c->N); s1.g.assign(M, std::vector<cplx>(c->N));
  for (int a = 0; a < 2; ++a) {
    double sg = (a == 0) ? +1.0 : -1.0;
#pragma omp parallel for collapse(2) schedule(static)
    for (int iz = 0; iz < c->nz; ++iz)
      for (int iy = 0; iy < c->ny; ++iy)
        for (int ix = 0; ix < c->nx; ++ix) {
          size_t i = IDX(c, iz, iy, ix);
          double th = c->kz[iz] * c->p.vA * dt;
          cplx ph = cplx(std::cos(sg * th), std::sin(sg * th));                  // exp(+-i theta)
          cplx phN = (c->p.if_variant == 0) ? ph : cplx(std::cos(0.5 * sg * th), std::sin(0.5 * sg * th));
          if (c->p.if_variant == 0)
            s1.w[a][i] = ph * (sn.w[a][i] + phN * dt * k2.w[a][i]);
          else
            s1.w[a][i] = ph * sn.w[a][i] + phN * dt * k2.w[a][i];
        }
  }
  if (exact) {                                              // g_{n+1} = P(dt) g_n + P(dt/2) dt R_{n+1/2} = P(dt/2) (P(dt/2) g_n + dt R_{n+1/2})
    for (int m = 0; m < M; ++m) s1.g[m] = sn.g[m];
    propagate(c, s1.g, 0.5 * dt);
    for (int m = 0; m < M; ++m)
      for (size_t i = 0; i < c->N; ++i) s1.g[m][i] += dt * k2.g[m][i];
    propagate(c, s1.g, 0.5 * dt);
  } else {
    for (int m = 0; m < M; ++m)
      for (size_t i = 0; i < c->N; ++i) s1.g[m][i] = sn.g[m][i] + dt * k2.g[m][i];
  }
  // Alg. 2 l.12-14: dissipation with the full dt
  apply_dissipation(c, s1, dt);
  // forcing increment (Q17), then time and diagnostics
  apply_forcing(c, s1, dt);
  apply_forcing_g(c, s1, dt);
  c->w[0].swap(s1.w[0]); c->w[1].swap(s1.w[1]); c->g.swap(s1.g);
  c->t += dt; c->step += 1; c->last_dt = dt;
  c->stage_pending = false;
  State cur; cur.w[0] = c->w[0]; cur.w[1] = c->w[1]; cur.g = c->g;
  double e[6]; energies(c, cur, e);
  c->hist.push_back(c->t);
  for (int i = 0; i < 6; ++i) c->hist.push_back(e[i]);
  for (int i = 0; i < 6; ++i) if (!std::isfinite(e[i])) { c->err = "non-finite energy"; return -3; }
  return 0;
}

static int step_once(oracle_ctx* c, double dt_in) {
  int rc = step_stage1(c, dt_in);
  if (rc) return rc;
  return step_stage2(c);
}

// ---------------------------------------------------------------------------------------------
// Half-plane <-> full-spectrum conversion at the boundary.  Boundary layout (same arrays the
// product takes): [field][kz][ky][kx], kx = 0..nx/2 fastest, FFT order in ky,kz, (re,im) pairs.
// Projection applied on input: Hermitian completion, averaging
// of the self-conjugate kx=0 plane, Eq. 20 mask, and kperp=0 -> 0 for the potentials.
// ---------------------------------------------------------------------------------------------
static void half_to_full(const oracle_ctx* c, const double* in, std::vector<cplx>& full) {
  const int nx = c->nx, ny = c->ny, nz = c->nz, hx = nx / 2 + 1;
  full.assign(c->N, cplx(0, 0));
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy) {
      int jz = (nz - iz) % nz, jy = (ny - iy) % ny;
      for (int ix = 0; ix < hx; ++ix) {
        size_t h = (((size_t)iz * ny + iy) * hx + ix) * 2;
        cplx v(in[h], in[h + 1]);
        if (ix == 0) {
          size_t h2 = (((size_t)jz * ny + jy) * hx + 0) * 2;
          cplx v2(in[h2], in[h2 + 1]);
          full[IDX(c, iz, iy, 0)] = 0.5 * (v + std::conj(v2));
        } else if (ix < nx / 2) {
          full[IDX(c, iz, iy, ix)] = v;
          full[IDX(c, jz, jy, nx - ix)] = std::conj(v);
        }   // ix == nx/2 (Nyquist) is always removed by Eq. 20
      }
    }
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy)
      for (int ix = 0; ix < nx; ++ix)
        if (masked(c, iz, iy, ix)) full[IDX(c, iz, iy, ix)] = cplx(0, 0);
}

static void full_to_half(const oracle_ctx* c, const std::vector<cplx>& full, double* out) {
  const int nx = c->nx, ny = c->ny, nz = c->nz, hx = nx / 2 + 1;
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy)
      for (int ix = 0; ix < hx; ++ix) {
        size_t h = (((size_t)iz * ny + iy) * hx + ix) * 2;
        cplx v = full[IDX(c, iz, iy, ix % nx)];
        out[h] = v.real(); out[h + 1] = v.imag();
      }
}

extern "C" {

int oracle_create(const oracle_params* p, oracle_ctx** out) {
  if (!p || !out) return -1;
  if (!is_pow2(p->nx) || !is_pow2(p->ny) || !is_pow2(p->nz) || p->nx < 4 || p->ny < 4 || p->nz < 2) return -1;
  if (p->M < 0 || !(p->Lx > 0) || !(p->Ly > 0) || !(p->Lz > 0)) return -1;
  if (p->M > 0 && p->vA != 1.0) return -4;                 // Q12
  if (p->nspecies != 1 && p->nspecies != 2) return -1;
  if (p->hermite_exact != 0 && p->hermite_exact != 1) return -1;
  if (p->M_global != 0) {                                  // moment shard (Q31): one species, plain RK2 streaming
    if (p->M < 1 || p->m_offset < 0 || p->m_offset + p->M > p->M_global || p->nspecies != 1 || p->hermite_exact) return -1;
  } else if (p->m_offset != 0) return -1;
  oracle_ctx* c = new oracle_ctx();
  c->p = *p; c->nx = p->nx; c->ny = p->ny; c->nz = p->nz;
  c->Msp = p->M; c->nsp = p->nspecies; c->M = p->M * p->nspecies;
  c->moff = p->m_offset; c->Mg = p->M_global ? p->M_global : p->M;
  c->own_lo = (c->moff > 0) ? 1 : 0;
  c->own_hi = (p->M_global && c->moff + p->M < c->Mg) ? c->M - 1 : c->M;
  c->dt_cur = 0.0;
  c->N = (size_t)p->nx * p->ny * p->nz;
  c->kx.resize(c->nx); c->ky.resize(c->ny); c->kz.resize(c->nz);
  c->mx.resize(c->nx); c->my.resize(c->ny); c->mz.resize(c->nz);
  for (int i = 0; i < c->nx; ++i) { c->mx[i] = signed_mode(i, c->nx); c->kx[i] = 2 * PI * c->mx[i] / p->Lx; }
  for (int i = 0; i < c->ny; ++i) { c->my[i] = signed_mode(i, c->ny); c->ky[i] = 2 * PI * c->my[i] / p->Ly; }
  for (int i = 0; i < c->nz; ++i) { c->mz[i] = signed_mode(i, c->nz); c->kz[i] = 2 * PI * c->mz[i] / p->Lz; }
  c->w[0].assign(c->N, cplx(0, 0)); c->w[1].assign(c->N, cplx(0, 0));
  c->g.assign(c->M, std::vector<cplx>(c->N, cplx(0, 0)));
  c->coef_dn.resize(c->Mg + 1); c->coef_up.resize(c->Mg + 1);   // indexed by the GLOBAL moment number
  for (int m = 0; m <= c->Mg; ++m) {
    c->coef_dn[m] = std::sqrt(m / 2.0);                    // Eq. 6c
    c->coef_up[m] = std::sqrt((m + 1) / 2.0);
  }
  if (p->hermite_coeff == 1) {                             // literal Eq. 6a / 6b (Q24)
    if (c->Mg > 0) c->coef_up[0] = std::sqrt(2.0);
    if (c->Mg > 1) c->coef_up[1] = std::sqrt(1.5);
  }
  c->t = 0.0; c->step = 0; c->last_dt = 0.0;
  *out = c;
  return 0;
}

int oracle_destroy(oracle_ctx* c) { delete c; return 0; }

int oracle_set_state(oracle_ctx* c, const double* zeta_hat, const double* g_hat) {
  if (!c || !zeta_hat || (c->M > 0 && !g_hat)) return -1;
  c->stage_pending = false;                 // a new state abandons a half-done step (as gandalf_set_state)
  const size_t hp = (size_t)c->nz * c->ny * (c->nx / 2 + 1) * 2;
  for (int a = 0; a < 2; ++a) {
    std::vector<cplx> xi;
    half_to_full(c, zeta_hat + a * hp, xi);
    for (int iz = 0; iz < c->nz; ++iz)
      for (int iy = 0; iy < c->ny; ++iy)
        for (int ix = 0; ix < c->nx; ++ix) {
          size_t i = IDX(c, iz, iy, ix);
          c->w[a][i] = -kperp2(c, iy, ix) * xi[i];          // w = lap_perp xi; kperp=0 -> 0
        }
  }
  for (int m = 0; m < c->M; ++m) half_to_full(c, g_hat + m * hp, c->g[m]);
  return 0;
}

int oracle_get_state(const oracle_ctx* c, double* zeta_hat, double* g_hat) {
  if (!c || !zeta_hat || (c->M > 0 && !g_hat)) return -1;
  const size_t hp = (size_t)c->nz * c->ny * (c->nx / 2 + 1) * 2;
  for (int a = 0; a < 2; ++a) {
    std::vector<cplx> xi;
    potentials(c, c->w[a], xi);
    full_to_half(c, xi, zeta_hat + a * hp);
  }
  for (int m = 0; m < c->M; ++m) full_to_half(c, c->g[m], g_hat + m * hp);
  return 0;
}

int oracle_rhs(oracle_ctx* c, double* dw_hat, double* dg_hat) {
  if (!c || !dw_hat || (c->M > 0 && !dg_hat)) return -1;
  State s; s.w[0] = c->w[0]; s.w[1] = c->w[1]; s.g = c->g;
  State k; rhs_eval(c, s, k, nullptr);
  const size_t hp = (size_t)c->nz * c->ny * (c->nx / 2 + 1) * 2;
  for (int a = 0; a < 2; ++a) full_to_half(c, k.w[a], dw_hat + a * hp);
  for (int m = 0; m < c->M; ++m) full_to_half(c, k.g[m], dg_hat + m * hp);
  return 0;
}

int oracle_step(oracle_ctx* c, double dt, int nsteps) {
  if (!c || nsteps < 0) return -1;
  if (c->stage_pending) { c->err = "oracle_step: a step is half done (stage 0 without stage 1)"; return -1; }
  for (int i = 0; i < nsteps; ++i) { int rc = step_once(c, dt); if (rc) return rc; }
  return 0;
}

int oracle_energy(oracle_ctx* c, double out[6]) {
  if (!c || !out) return -1;
  State s; s.w[0] = c->w[0]; s.w[1] = c->w[1]; s.g = c->g;
  energies(c, s, out);
  return 0;
}

// Shell spectrum (Eq. 26; Q15): bin j = floor(kperp/dk + 1/2), dk = 2 pi / max(Lx,Ly).
// literal_eq26 = 0: mode energy 1/4 kperp^2 (|xi+|^2+|xi-|^2)  (sums to E_A);  1: |xi+|^2+|xi-|^2.
int oracle_kperp_spectrum(oracle_ctx* c, int nbins, int literal_eq26, double* out) {
  if (!c || !out || nbins <= 0) return -1;
  for (int j = 0; j < nbins; ++j) out[j] = 0.0;
  double dk = 2 * PI / std::fmax(c->p.Lx, c->p.Ly);
  for (int iz = 0; iz < c->nz; ++iz)
    for (int iy = 0; iy < c->ny; ++iy)
      for (int ix = 0; ix < c->nx; ++ix) {
        double k2 = kperp2(c, iy, ix);
        if (!(k2 > 0.0)) continue;
        size_t i = IDX(c, iz, iy, ix);
        cplx xp = -c->w[0][i] / k2, xm = -c->w[1][i] / k2;
        double e = std::norm(xp) + std::norm(xm);
        if (!literal_eq26) e *= 0.25 * k2;
        int j = (int)std::floor(std::sqrt(k2) / dk + 0.5);
        if (j >= 0 && j < nbins) out[j] += e;
      }
  return 0;
}

// Hermite spectrum (Eq. 27): C_m = <|g_m|^2> = sum over the FULL spectrum of |g_m(k)|^2 (Parseval with
// the physical normalisation of Eq. 9).  out: M doubles.
int oracle_hermite_spectrum(oracle_ctx* c, double* out) {
  if (!c || (c->M > 0 && !out)) return -1;
  for (int m = 0; m < c->M; ++m) {
    double s = 0.0;
    for (size_t i = 0; i < c->N; ++i) s += std::norm(c->g[m][i]);
    out[m] = s;
  }
  return 0;
}

// Truncation monitor (section 3.5: "the energy ratio E_M/E_total (energy in the single highest retained moment
// m = M relative to total energy)"; reading Q32): E_M = 1/2 sum_k |g_{M-1}|^2 summed over the species, E_total = E_A + W_g.
int oracle_truncation_ratio(oracle_ctx* c, double* out) {
  if (!c || !out || c->M < 1 || c->p.M_global != 0) return -1;
  double eM = 0.0;
  for (int sp = 0; sp < c->nsp; ++sp) {
    const std::vector<cplx>& g = c->g[sp * c->Msp + c->Msp - 1];
    for (size_t i = 0; i < c->N; ++i) eM += 0.5 * std::norm(g[i]);
  }
  State cur; cur.w[0] = c->w[0]; cur.w[1] = c->w[1]; cur.g = c->g;
  double e[6]; energies(c, cur, e);
  *out = eM / (e[0] + e[5]);
  return 0;
}

// Parallel spectrum (Q25): bin j = |n_z| of the Alfvenic mode energy 1/4 kperp^2 (|xi+|^2+|xi-|^2).
int oracle_kpar_spectrum(oracle_ctx* c, int nbins, double* out) {
  if (!c || !out || nbins <= 0) return -1;
  for (int j = 0; j < nbins; ++j) out[j] = 0.0;
  for (int iz = 0; iz < c->nz; ++iz)
    for (int iy = 0; iy < c->ny; ++iy)
      for (int ix = 0; ix < c->nx; ++ix) {
        double k2 = kperp2(c, iy, ix);
        if (!(k2 > 0.0)) continue;
        size_t i = IDX(c, iz, iy, ix);
        cplx xp = -c->w[0][i] / k2, xm = -c->w[1][i] / k2;
        int j = std::abs(c->mz[iz]);
        if (j < nbins) out[j] += 0.25 * k2 * (std::norm(xp) + std::norm(xm));
      }
  return 0;
}

int oracle_energy_history(oracle_ctx* c, int max_records, double* out, int* n) {
  if (!c || !n) return -1;
  int have = (int)(c->hist.size() / 7);
  int k = have < max_records ? have : max_records;
  if (out) std::memcpy(out, c->hist.data(), (size_t)k * 7 * sizeof(double));
  *n = k;
  return 0;
}

int oracle_get_time(const oracle_ctx* c, double* t, long long* step, double* last_dt) {
  if (!c) return -1;
  if (t) *t = c->t;
  if (step) *step = c->step;
  if (last_dt) *last_dt = c->last_dt;
  return 0;
}

// Restart support: time and step counter (the forcing RNG counters derive from the step number, Q17/Q26).
int oracle_set_time(oracle_ctx* c, double t, long long step) {
  if (!c || step < 0) return -1;
  c->t = t; c->step = step;
  return 0;
}

const char* oracle_last_error(const oracle_ctx* c) { return c ? c->err.c_str() : "null ctx"; }

// ---- helpers exported only so the pins can reach the building blocks ------------------------
void oracle_fft1d(int n, int sign, const double* in, double* out) {        // radix-2, no scaling
  std::vector<cplx> a(n);
  for (int i = 0; i < n; ++i) a[i] = cplx(in[2 * i], in[2 * i + 1]);
  fft_radix2(n, sign, a.data());
  for (int i = 0; i < n; ++i) { out[2 * i] = a[i].real(); out[2 * i + 1] = a[i].imag(); }
}
void oracle_dft1d(int n, int sign, const double* in, double* out) {        // O(n^2) definition
  std::vector<cplx> a(n), b(n);
  for (int i = 0; i < n; ++i) a[i] = cplx(in[2 * i], in[2 * i + 1]);
  dft_naive(n, sign, a.data(), b.data());
  for (int i = 0; i < n; ++i) { out[2 * i] = b[i].real(); out[2 * i + 1] = b[i].imag(); }
}
// Dealiased bracket of two FULL spectra [nz][ny][nx] (re,im), result full spectrum.
int oracle_bracket_full(oracle_ctx* c, const double* f_hat, const double* g_hat, double* out, double* max_imag) {
  if (!c) return -1;
  std::vector<cplx> f(c->N), g(c->N), b;
  for (size_t i = 0; i < c->N; ++i) { f[i] = cplx(f_hat[2 * i], f_hat[2 * i + 1]); g[i] = cplx(g_hat[2 * i], g_hat[2 * i + 1]); }
  Grad gf, gg; double mi = 0.0;
  deriv_real(c, f, 0, gf.x, &mi); deriv_real(c, f, 1, gf.y, &mi);
  deriv_real(c, g, 0, gg.x, &mi); deriv_real(c, g, 1, gg.y, &mi);
  bracket_from_grads(c, gf, gg, b);
  for (size_t i = 0; i < c->N; ++i) { out[2 * i] = b[i].real(); out[2 * i + 1] = b[i].imag(); }
  if (max_imag) *max_imag = mi;
  return 0;
}
// One stage of a step (stage 0: RHS at state_n + predictor; stage 1: midpoint RHS + corrector + dissipation + forcing + record).
// A moment-sharded run exchanges its halo moments between the stages (Q31); oracle_step(dt, 1) == stage 0 then stage 1.
int oracle_step_stage(oracle_ctx* c, double dt, int stage) {
  if (!c || (stage != 0 && stage != 1)) return -1;
  // the stages alternate 0, 1 (as gandalf_step_stage): stage 1 without a half-step state would read empty arrays
  if ((stage == 1) != c->stage_pending || (stage == 1 && c->hw[0].size() != c->N)) {
    c->err = "oracle_step_stage: stages must alternate 0, 1";
    return -1;
  }
  return stage == 0 ? step_stage1(c, dt) : step_stage2(c);
}
// Full-spectrum access to the half-step (stage) state, same field numbering as oracle_get_full.
int oracle_get_stage_full(const oracle_ctx* c, int field, double* out) {
  if (!c || field < 0 || field >= 2 + c->M || c->hw[0].size() != c->N) return -1;
  const std::vector<cplx>& a = (field < 2) ? c->hw[field] : c->hg[field - 2];
  for (size_t i = 0; i < c->N; ++i) { out[2 * i] = a[i].real(); out[2 * i + 1] = a[i].imag(); }
  return 0;
}
int oracle_set_stage_full(oracle_ctx* c, int field, const double* in) {
  if (!c || field < 0 || field >= 2 + c->M || c->hw[0].size() != c->N) return -1;
  std::vector<cplx>& a = (field < 2) ? c->hw[field] : c->hg[field - 2];
  for (size_t i = 0; i < c->N; ++i) a[i] = cplx(in[2 * i], in[2 * i + 1]);
  return 0;
}
// Full-spectrum access to the evolved vorticities / moments (field 0,1 = w+-, 2+m = g_m).
int oracle_get_full(const oracle_ctx* c, int field, double* out) {
  if (!c || field < 0 || field >= 2 + c->M) return -1;
  const std::vector<cplx>& a = (field < 2) ? c->w[field] : c->g[field - 2];
  for (size_t i = 0; i < c->N; ++i) { out[2 * i] = a[i].real(); out[2 * i + 1] = a[i].imag(); }
  return 0;
}
int oracle_set_full(oracle_ctx* c, int field, const double* in) {
  if (!c || field < 0 || field >= 2 + c->M) return -1;
  std::vector<cplx>& a = (field < 2) ? c->w[field] : c->g[field - 2];
  for (size_t i = 0; i < c->N; ++i) a[i] = cplx(in[2 * i], in[2 * i + 1]);
  return 0;
}
// Thread count of the OpenMP loops (bench.py times the oracle on all host cores and once single-threaded).
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n >= 1) omp_set_num_threads(n);
#else
  (void)n;
#endif
}
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
