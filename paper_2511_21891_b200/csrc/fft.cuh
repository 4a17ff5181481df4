// fft.cuh -- register-resident radix-2/4/8/16 butterflies and a lane-group cooperative FFT.
//
// One FFT of length N is computed by a group of T = N/E consecutive lanes of ONE warp; each lane
// keeps E complex doubles in registers.  Distribution contract (same on input and output):
//     lane t (0..T-1) holds   v[q] = x[t + T*q],  q = 0..E-1.
// The transform is a Stockham autosort with radices {r_1,..,r_S} (product N).  Between stages the
// data crosses lanes through a padded shared-memory line buffer; the last stage needs no exchange
// because its natural output index  j + i*N/r  is again  t + T*(b + i*E/r).  All synchronisation is
// __syncwarp(): every lane of the warp must call the routine (idle groups transform zeros).
//
// The phases (compute / scatter / gather) are separate HD functions so that a host test can
// emulate the T lanes sequentially (tests/test_fft_host.py compiles this header with g++).
//
// Sign convention: DIR = -1 forward kernel exp(-2 pi i jk/N), DIR = +1 inverse; no scaling.
#pragma once
#include <cmath>

#if defined(__CUDACC__)
#define GD_HD __host__ __device__ __forceinline__
#else
#define GD_HD inline
#endif

struct alignas(16) cd {   // complex double
  double x, y;
};

GD_HD cd cmake(double a, double b) { cd r; r.x = a; r.y = b; return r; }
GD_HD cd operator+(cd a, cd b) { return cmake(a.x + b.x, a.y + b.y); }
GD_HD cd operator-(cd a, cd b) { return cmake(a.x - b.x, a.y - b.y); }
GD_HD cd cmul(cd a, cd b) { return cmake(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
GD_HD cd cconj(cd a) { return cmake(a.x, -a.y); }
GD_HD cd cscale(cd a, double s) { return cmake(a.x * s, a.y * s); }
// multiply by DIR*i : forward (-1) -> -i, inverse (+1) -> +i
template <int DIR> GD_HD cd mul_dir_i(cd a) { return DIR < 0 ? cmake(a.y, -a.x) : cmake(-a.y, a.x); }
// multiply by i (always +i)
GD_HD cd mul_i(cd a) { return cmake(-a.y, a.x); }

#define GD_SQRT1_2 0.70710678118654752440
#define GD_COS_PI_8 0.92387953251128675613
#define GD_SIN_PI_8 0.38268343236508977173

// multiply by exp(DIR * 2 pi i * P / 16), P in 0..15, with the cheap cases special-cased
template <int P, int DIR> GD_HD cd mul_w16(cd a) {
  if constexpr (P == 0) return a;
  else if constexpr (P == 4) return mul_dir_i<DIR>(a);
  else if constexpr (P == 8) return cmake(-a.x, -a.y);
  else if constexpr (P == 12) return mul_dir_i<-DIR>(a);
  else if constexpr (P == 2) return cmake(GD_SQRT1_2 * (a.x - DIR * a.y), GD_SQRT1_2 * (DIR * a.x + a.y));
  else if constexpr (P == 6) return mul_w16<2, DIR>(mul_dir_i<DIR>(a));
  else if constexpr (P == 10) return mul_w16<2, DIR>(cmake(-a.x, -a.y));
  else if constexpr (P == 14) return mul_w16<2, DIR>(mul_dir_i<-DIR>(a));
  else {
    // odd P: general rotation by angle P*pi/8
    constexpr double c = (P == 1 || P == 15) ? GD_COS_PI_8 : (P == 3 || P == 13) ? GD_SIN_PI_8
                        : (P == 5 || P == 11) ? -GD_SIN_PI_8 : -GD_COS_PI_8;          // 7, 9
    constexpr double s0 = (P == 1 || P == 7) ? GD_SIN_PI_8 : (P == 3 || P == 5) ? GD_COS_PI_8
                         : (P == 9 || P == 15) ? -GD_SIN_PI_8 : -GD_COS_PI_8;        // 11, 13
    constexpr double s = DIR * s0;
    return cmake(a.x * c - a.y * s, a.x * s + a.y * c);
  }
}

// ---- in-register butterflies: natural order in, natural order out -----------------------------
template <int DIR> GD_HD void bf2(cd (&x)[2]) {
  cd a = x[0], b = x[1];
  x[0] = a + b; x[1] = a - b;
}
template <int DIR> GD_HD void bf4(cd& x0, cd& x1, cd& x2, cd& x3) {
  cd a0 = x0 + x2, a1 = x0 - x2, a2 = x1 + x3, a3 = mul_dir_i<DIR>(x1 - x3);
  x0 = a0 + a2; x1 = a1 + a3; x2 = a0 - a2; x3 = a1 - a3;
}
template <int DIR> GD_HD void bf4(cd (&x)[4]) { bf4<DIR>(x[0], x[1], x[2], x[3]); }
template <int DIR> GD_HD void bf8(cd (&x)[8]) {
  cd e0 = x[0], e1 = x[2], e2 = x[4], e3 = x[6];
  cd o0 = x[1], o1 = x[3], o2 = x[5], o3 = x[7];
  bf4<DIR>(e0, e1, e2, e3);
  bf4<DIR>(o0, o1, o2, o3);
  o1 = mul_w16<2, DIR>(o1);
  o2 = mul_w16<4, DIR>(o2);
  o3 = mul_w16<6, DIR>(o3);
  x[0] = e0 + o0; x[4] = e0 - o0;
  x[1] = e1 + o1; x[5] = e1 - o1;
  x[2] = e2 + o2; x[6] = e2 - o2;
  x[3] = e3 + o3; x[7] = e3 - o3;
}
#ifndef GD_FFT_FOLD
#define GD_FFT_FOLD 0     // 1: the 1/sqrt 2 of the w16^2, w16^6 twiddles is folded into the following additions as fused multiply-adds
#endif
// rotation by DIR*45 degrees WITHOUT its factor 1/sqrt 2:  sqrt(2) * exp(DIR i pi/4) * a
template <int DIR> GD_HD cd rot45u(cd a) { return cmake(a.x - DIR * a.y, DIR * a.x + a.y); }
GD_HD cd cfma(double s, cd a, cd b) { return cmake(fma(s, a.x, b.x), fma(s, a.y, b.y)); }   // s*a + b
template <int DIR> GD_HD void bf16(cd (&x)[16]) {
  // n = 4*n1 + n2 ; k = k1 + 4*k2.  Y[n2][k1] = FFT4 over n1; twiddle w16^(n2*k1); FFT4 over n2.
  cd y0[4] = {x[0], x[4], x[8], x[12]};
  cd y1[4] = {x[1], x[5], x[9], x[13]};
  cd y2[4] = {x[2], x[6], x[10], x[14]};
  cd y3[4] = {x[3], x[7], x[11], x[15]};
  bf4<DIR>(y0); bf4<DIR>(y1); bf4<DIR>(y2); bf4<DIR>(y3);
#if GD_FFT_FOLD
  // The twiddles w16^2, w16^6 carry a factor 1/sqrt 2: it is not applied to the operand but folded into the additions of the
  // second FFT4 as fused multiply-adds (8 fewer fp64 instructions per butterfly than scale-then-add).  Measured: no gain at
  // full clock (x-pass 1.388 -> 1.395 ms), DESIGN.md section 5.
  constexpr double H = GD_SQRT1_2;
  {
    cd a = y0[0], b = y1[0], c = y2[0], d = y3[0];
    bf4<DIR>(a, b, c, d);
    x[0] = a; x[4] = b; x[8] = c; x[12] = d;
  }
  {
    const cd a = y0[1], b = mul_w16<1, DIR>(y1[1]), cu = rot45u<DIR>(y2[1]), d = mul_w16<3, DIR>(y3[1]);
    const cd a0 = cfma(H, cu, a), a1 = cfma(-H, cu, a), a2 = b + d, a3 = mul_dir_i<DIR>(b - d);
    x[1] = a0 + a2; x[5] = a1 + a3; x[9] = a0 - a2; x[13] = a1 - a3;
  }
  {
    const cd a = y0[2], bu = rot45u<DIR>(y1[2]), c = mul_dir_i<DIR>(y2[2]), du = rot45u<DIR>(mul_dir_i<DIR>(y3[2]));
    const cd a0 = a + c, a1 = a - c, s2 = bu + du, s3 = mul_dir_i<DIR>(bu - du);
    x[2] = cfma(H, s2, a0); x[6] = cfma(H, s3, a1); x[10] = cfma(-H, s2, a0); x[14] = cfma(-H, s3, a1);
  }
  {
    const cd a = y0[3], b = mul_w16<3, DIR>(y1[3]), cu = rot45u<DIR>(mul_dir_i<DIR>(y2[3])), d = mul_w16<9, DIR>(y3[3]);
    const cd a0 = cfma(H, cu, a), a1 = cfma(-H, cu, a), a2 = b + d, a3 = mul_dir_i<DIR>(b - d);
    x[3] = a0 + a2; x[7] = a1 + a3; x[11] = a0 - a2; x[15] = a1 - a3;
  }
#else
  y1[1] = mul_w16<1, DIR>(y1[1]); y1[2] = mul_w16<2, DIR>(y1[2]); y1[3] = mul_w16<3, DIR>(y1[3]);
  y2[1] = mul_w16<2, DIR>(y2[1]); y2[2] = mul_w16<4, DIR>(y2[2]); y2[3] = mul_w16<6, DIR>(y2[3]);
  y3[1] = mul_w16<3, DIR>(y3[1]); y3[2] = mul_w16<6, DIR>(y3[2]); y3[3] = mul_w16<9, DIR>(y3[3]);
#pragma unroll
  for (int k1 = 0; k1 < 4; ++k1) {
    cd a = y0[k1], b = y1[k1], c = y2[k1], d = y3[k1];
    bf4<DIR>(a, b, c, d);
    x[k1] = a; x[k1 + 4] = b; x[k1 + 8] = c; x[k1 + 12] = d;
  }
#endif
}
template <int R, int DIR> GD_HD void butterfly(cd (&x)[R]) {
  if constexpr (R == 2) bf2<DIR>(x);
  else if constexpr (R == 4) bf4<DIR>(x);
  else if constexpr (R == 8) bf8<DIR>(x);
  else bf16<DIR>(x);
}

// ---- plan: N -> lanes per FFT, elements per lane, stage radices -------------------------------
// The template argument of every routine below is a plan ID: the transform length N, or N + GD_FFT_ALT for the alternative
// plan of that length (more lanes, fewer registers per lane: 256 = 8*8*4 on a whole warp, for kernels that want 16 warps per SM).
#define GD_FFT_ALT 4096
template <int N> struct FftPlan;
template <> struct FftPlan<2>   { static constexpr int T = 1,  E = 2,  S = 1, R0 = 2,  R1 = 1,  R2 = 1, PAD = R0; };
template <> struct FftPlan<4>   { static constexpr int T = 1,  E = 4,  S = 1, R0 = 4,  R1 = 1,  R2 = 1, PAD = R0; };
template <> struct FftPlan<8>   { static constexpr int T = 1,  E = 8,  S = 1, R0 = 8,  R1 = 1,  R2 = 1, PAD = R0; };
template <> struct FftPlan<16>  { static constexpr int T = 1,  E = 16, S = 1, R0 = 16, R1 = 1,  R2 = 1, PAD = R0; };
template <> struct FftPlan<32>  { static constexpr int T = 4,  E = 8,  S = 2, R0 = 8,  R1 = 4,  R2 = 1, PAD = R0; };
template <> struct FftPlan<64>  { static constexpr int T = 8,  E = 8,  S = 2, R0 = 8,  R1 = 8,  R2 = 1, PAD = R0; };
template <> struct FftPlan<128> { static constexpr int T = 8,  E = 16, S = 2, R0 = 16, R1 = 8,  R2 = 1, PAD = R0; };
template <> struct FftPlan<256> { static constexpr int T = 16, E = 16, S = 2, R0 = 16, R1 = 16, R2 = 1, PAD = R0; };
// 512 = 16*4*8: measured against 8*8*8, 16*16*2 and 16*8*4 at config 4b (P1 1.03 / 0.87 / 0.87 / 0.84 ms: the radix-16 first stage
// keeps k_yinv<512> from spilling and its split exchange is conflict-free, 2 wavefronts per 8-byte access instead of 3)
#ifndef GD_FFT512_R0
#define GD_FFT512_R0 16
#define GD_FFT512_R1 4
#define GD_FFT512_R2 8
#endif
template <> struct FftPlan<512> { static constexpr int T = 32, E = 16, S = 3, R0 = GD_FFT512_R0, R1 = GD_FFT512_R1, R2 = GD_FFT512_R2, PAD = R0; };
template <> struct FftPlan<256 + GD_FFT_ALT> { static constexpr int T = 32, E = 8, S = 3, R0 = 8, R1 = 8, R2 = 4, PAD = 16; };   // pad 16: 8-byte exchange conflict-free on 32 lanes

template <int ID> struct FftGeom {
  using P = FftPlan<ID>;
  static constexpr int N = ID % GD_FFT_ALT;                // transform length
  static constexpr int T = P::T, E = P::E, S = P::S;
  static_assert(T * E == N, "plan covers the transform");
  static constexpr int PADDIV = P::PAD;                    // pad(idx) = idx + idx / PAD (PAD = R0 unless the plan says otherwise)
  static constexpr int BUF = (S > 1) ? (N + N / PADDIV) : 0;  // complex entries of the line buffer
  GD_HD static int pad(int idx) { return idx + idx / PADDIV; }
  template <int s> static constexpr int radix() { return s == 0 ? P::R0 : (s == 1 ? P::R1 : P::R2); }
  template <int s> static constexpr int ns() { return s == 0 ? 1 : (s == 1 ? P::R0 : P::R0 * P::R1); }
};

// Stage twiddles live in a per-N "stage table" (copied to shared memory by every kernel): for each stage
// s >= 1 the entries  tws[OFF_s + (i-1)*NS_s + k] = exp(-2 pi i * i*k / (NS_s*R_s)),  i = 1..R_s-1, k = 0..NS_s-1,
// so that consecutive lanes (consecutive k) read consecutive 16-byte words: conflict-free LDS.128.
template <int N> struct FftTw {
  using G = FftGeom<N>;
  static constexpr int CNT1 = (G::S > 1) ? (G::template radix<1>() - 1) * G::template ns<1>() : 0;
  static constexpr int CNT2 = (G::S > 2) ? (G::template radix<2>() - 1) * G::template ns<2>() : 0;
  static constexpr int COUNT = CNT1 + CNT2;
  template <int s> static constexpr int off() { return s == 1 ? 0 : CNT1; }
};

template <int N> inline void fft_fill_stage_table(cd* out) {   // host side, libm cos/sin per entry
  using G = FftGeom<N>;
  const double PI2 = 6.28318530717958647692528676655900577;
  int o = 0;
  if constexpr (G::S > 1) {
    constexpr int R = G::template radix<1>(), NS = G::template ns<1>();
    for (int i = 1; i < R; ++i)
      for (int k = 0; k < NS; ++k) { const double a = PI2 * (double)(i * k) / (double)(NS * R); out[o++] = cmake(std::cos(a), -std::sin(a)); }
  }
  if constexpr (G::S > 2) {
    constexpr int R = G::template radix<2>(), NS = G::template ns<2>();
    for (int i = 1; i < R; ++i)
      for (int k = 0; k < NS; ++k) { const double a = PI2 * (double)(i * k) / (double)(NS * R); out[o++] = cmake(std::cos(a), -std::sin(a)); }
  }
}

// Stage s, compute phase: twiddle (stage table, conjugated for DIR=+1) and radix butterflies on the lane's
// own registers.  Results stay at v[b + i*B].
template <int N, int DIR, int s> GD_HD void fft_stage_compute(cd (&v)[FftPlan<N>::E], int t, const cd* __restrict__ tws) {
  using G = FftGeom<N>;
  constexpr int R = G::template radix<s>();
  constexpr int NS = G::template ns<s>();
  constexpr int B = G::E / R;                 // butterflies per lane in this stage
#pragma unroll
  for (int b = 0; b < B; ++b) {
    cd x[R];
#pragma unroll
    for (int i = 0; i < R; ++i) x[i] = v[b + i * B];
    if constexpr (NS > 1) {
      const int k = (t + G::T * b) % NS;
      const cd* tb = tws + FftTw<N>::template off<s>() + k;
#pragma unroll
      for (int i = 1; i < R; ++i) {
        cd w = tb[(i - 1) * NS];
        if (DIR > 0) w.y = -w.y;
        x[i] = cmul(x[i], w);
      }
    }
    butterfly<R, DIR>(x);
#pragma unroll
    for (int i = 0; i < R; ++i) v[b + i * B] = x[i];
  }
}

// Stage s, scatter phase: write the lane's results to the line buffer at the Stockham positions.
template <int N, int s> GD_HD void fft_stage_scatter(const cd (&v)[FftPlan<N>::E], int t, cd* buf) {
  using G = FftGeom<N>;
  constexpr int R = G::template radix<s>();
  constexpr int NS = G::template ns<s>();
  constexpr int B = G::E / R;
#pragma unroll
  for (int b = 0; b < B; ++b) {
    const int j = t + G::T * b;
    const int j0 = (j / NS) * NS * R + (j % NS);
#pragma unroll
    for (int i = 0; i < R; ++i) buf[G::pad(j0 + i * NS)] = v[b + i * B];
  }
}

// Gather phase: read back the lane's own distribution v[q] = buf[t + T q].
template <int N> GD_HD void fft_gather(cd (&v)[FftPlan<N>::E], int t, const cd* buf) {
  using G = FftGeom<N>;
#pragma unroll
  for (int q = 0; q < G::E; ++q) v[q] = buf[G::pad(t + G::T * q)];
}

// Stage-1 compute with the first NREG stage twiddles of this lane held in registers (twr[i-1] = table entry of
// input i; only for plans whose stage 1 has ONE butterfly per lane, so the twiddles depend on the lane alone):
// fewer shared-memory reads per transform for kernels that run many transforms per lane.  DIR = -1 only.
template <int N, int NREG> GD_HD void fft_stage1_compute_rt(cd (&v)[FftPlan<N>::E], int t, const cd* __restrict__ tws,
                                                            const cd (&twr)[NREG]) {
  using G = FftGeom<N>;
  constexpr int R = G::template radix<1>();
  constexpr int NS = G::template ns<1>();
  static_assert(G::E / R == 1 && G::S == 2, "one stage-1 butterfly per lane");
  cd x[R];
#pragma unroll
  for (int i = 0; i < R; ++i) x[i] = v[i];
  const cd* tb = tws + FftTw<N>::template off<1>() + (t % NS);
#pragma unroll
  for (int i = 1; i < R; ++i) {
    const cd w = (i - 1 < NREG) ? twr[(i - 1 < NREG) ? i - 1 : 0] : tb[(i - 1) * NS];
    x[i] = cmul(x[i], w);
  }
  butterfly<R, -1>(x);
#pragma unroll
  for (int i = 0; i < R; ++i) v[i] = x[i];
}
template <int N, int NREG> GD_HD void fft_load_stage1_twiddles(cd (&twr)[NREG], int t, const cd* __restrict__ tws) {
  using G = FftGeom<N>;
  constexpr int NS = G::template ns<1>();
#pragma unroll
  for (int i = 0; i < NREG; ++i) twr[i] = tws[FftTw<N>::template off<1>() + i * NS + (t % NS)];
}

// Split exchange: the real parts cross the lanes first, then the imaginary parts, through a buffer of doubles
// (FftGeom<N>::BUF entries of 8 bytes -- half the shared memory of the complex exchange; in place, because a lane's
// .x registers can be overwritten by the gather while its .y registers still wait to be scattered).
template <int N, int s, int C> GD_HD void fft_stage_scatter_c(const cd (&v)[FftPlan<N>::E], int t, double* buf) {
  using G = FftGeom<N>;
  constexpr int R = G::template radix<s>();
  constexpr int NS = G::template ns<s>();
  constexpr int B = G::E / R;
#pragma unroll
  for (int b = 0; b < B; ++b) {
    const int j = t + G::T * b;
    const int j0 = (j / NS) * NS * R + (j % NS);
#pragma unroll
    for (int i = 0; i < R; ++i) buf[G::pad(j0 + i * NS)] = C ? v[b + i * B].y : v[b + i * B].x;
  }
}
template <int N, int C> GD_HD void fft_gather_c(cd (&v)[FftPlan<N>::E], int t, const double* buf) {
  using G = FftGeom<N>;
#pragma unroll
  for (int q = 0; q < G::E; ++q) {
    if (C) v[q].y = buf[G::pad(t + G::T * q)];
    else v[q].x = buf[G::pad(t + G::T * q)];
  }
}

#if defined(__CUDACC__)
// The cooperative transform.  buf: this line's shared buffer (FftGeom<N>::BUF entries; unused if S==1);
// tws: the stage table (FftTw<N>::COUNT entries), normally in shared memory.
// Copy helper: all threads of the CTA, followed by __syncthreads().
template <int N> __device__ __forceinline__ void fft_load_table(cd* dst, const cd* __restrict__ src) {
  for (int i = threadIdx.x; i < FftTw<N>::COUNT; i += blockDim.x) dst[i] = src[i];
  __syncthreads();
}
template <int N, int DIR> __device__ __forceinline__ void fft_lanes(cd (&v)[FftPlan<N>::E], int t, cd* buf,
                                                                     const cd* __restrict__ tws) {
  using G = FftGeom<N>;
  fft_stage_compute<N, DIR, 0>(v, t, tws);
  if constexpr (G::S > 1) {
    fft_stage_scatter<N, 0>(v, t, buf);
    __syncwarp();
    fft_gather<N>(v, t, buf);
    __syncwarp();
    fft_stage_compute<N, DIR, 1>(v, t, tws);
  }
  if constexpr (G::S > 2) {
    fft_stage_scatter<N, 1>(v, t, buf);
    __syncwarp();
    fft_gather<N>(v, t, buf);
    __syncwarp();
    fft_stage_compute<N, DIR, 2>(v, t, tws);
  }
}
// Forward transform with register-held stage-1 twiddles (see fft_stage1_compute_rt).
template <int N, int NREG> __device__ __forceinline__ void fft_lanes_fwd_rt(cd (&v)[FftPlan<N>::E], int t, cd* buf,
                                                                            const cd* __restrict__ tws, const cd (&twr)[NREG]) {
  fft_stage_compute<N, -1, 0>(v, t, tws);
  fft_stage_scatter<N, 0>(v, t, buf);
  __syncwarp();
  fft_gather<N>(v, t, buf);
  __syncwarp();
  fft_stage1_compute_rt<N, NREG>(v, t, tws, twr);
}
template <int N, int s> __device__ __forceinline__ void fft_exchange_split(cd (&v)[FftPlan<N>::E], int t, double* buf) {
  fft_stage_scatter_c<N, s, 0>(v, t, buf);
  __syncwarp();
  fft_gather_c<N, 0>(v, t, buf);
  __syncwarp();
  fft_stage_scatter_c<N, s, 1>(v, t, buf);
  __syncwarp();
  fft_gather_c<N, 1>(v, t, buf);
  __syncwarp();
}
// Forward transform with the split exchange and register-held stage-1 twiddles.
template <int N, int NREG> __device__ __forceinline__ void fft_lanes_fwd_rt_split(cd (&v)[FftPlan<N>::E], int t, double* buf,
                                                                                  const cd* __restrict__ tws, const cd (&twr)[NREG]) {
  fft_stage_compute<N, -1, 0>(v, t, tws);
  fft_exchange_split<N, 0>(v, t, buf);
  fft_stage1_compute_rt<N, NREG>(v, t, tws, twr);
}
// Same transform with the split exchange; buf: FftGeom<N>::BUF doubles per lane group.
template <int N, int DIR> __device__ __forceinline__ void fft_lanes_split(cd (&v)[FftPlan<N>::E], int t, double* buf,
                                                                           const cd* __restrict__ tws) {
  using G = FftGeom<N>;
  fft_stage_compute<N, DIR, 0>(v, t, tws);
  if constexpr (G::S > 1) {
    fft_exchange_split<N, 0>(v, t, buf);
    fft_stage_compute<N, DIR, 1>(v, t, tws);
  }
  if constexpr (G::S > 2) {
    fft_exchange_split<N, 1>(v, t, buf);
    fft_stage_compute<N, DIR, 2>(v, t, tws);
  }
}
#endif
