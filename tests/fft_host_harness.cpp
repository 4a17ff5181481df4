// Host emulation of csrc/fft.cuh's lane-group FFT: the T lanes of one transform are run
// sequentially, phase by phase, exactly as the warp would run them between __syncwarp()s.
// Built by tests/test_fft_host.py with g++ (no CUDA needed); checks the product's FFT index
// logic and butterflies on the CPU box.  Not part of the product path.
#include <cmath>
#include <vector>
#include "../paper_2511_21891_b200/csrc/fft.cuh"

template <int N, int DIR> static void run(const double* in, double* out) {
  using G = FftGeom<N>;
  constexpr int T = G::T, E = G::E;
  std::vector<cd> tw(FftTw<N>::COUNT + 1);
  fft_fill_stage_table<N>(tw.data());
  std::vector<cd> buf(G::BUF + 1);
  cd v[T][E];
  for (int t = 0; t < T; ++t)
    for (int q = 0; q < E; ++q) v[t][q] = cmake(in[2 * (t + T * q)], in[2 * (t + T * q) + 1]);
  for (int t = 0; t < T; ++t) fft_stage_compute<N, DIR, 0>(v[t], t, tw.data());
  if constexpr (G::S > 1) {
    for (int t = 0; t < T; ++t) fft_stage_scatter<N, 0>(v[t], t, buf.data());
    for (int t = 0; t < T; ++t) fft_gather<N>(v[t], t, buf.data());
    for (int t = 0; t < T; ++t) fft_stage_compute<N, DIR, 1>(v[t], t, tw.data());
  }
  if constexpr (G::S > 2) {
    for (int t = 0; t < T; ++t) fft_stage_scatter<N, 1>(v[t], t, buf.data());
    for (int t = 0; t < T; ++t) fft_gather<N>(v[t], t, buf.data());
    for (int t = 0; t < T; ++t) fft_stage_compute<N, DIR, 2>(v[t], t, tw.data());
  }
  for (int t = 0; t < T; ++t)
    for (int q = 0; q < E; ++q) { out[2 * (t + T * q)] = v[t][q].x; out[2 * (t + T * q) + 1] = v[t][q].y; }
}

// Same transform with the split (real parts, then imaginary parts) exchange through a buffer of doubles.
template <int N, int s> static void exchange_split(cd (*v)[FftPlan<N>::E], double* buf) {
  constexpr int T = FftGeom<N>::T;
  for (int t = 0; t < T; ++t) fft_stage_scatter_c<N, s, 0>(v[t], t, buf);
  for (int t = 0; t < T; ++t) fft_gather_c<N, 0>(v[t], t, buf);
  for (int t = 0; t < T; ++t) fft_stage_scatter_c<N, s, 1>(v[t], t, buf);
  for (int t = 0; t < T; ++t) fft_gather_c<N, 1>(v[t], t, buf);
}
template <int N, int DIR> static void run_split(const double* in, double* out) {
  using G = FftGeom<N>;
  constexpr int T = G::T, E = G::E;
  std::vector<cd> tw(FftTw<N>::COUNT + 1);
  fft_fill_stage_table<N>(tw.data());
  std::vector<double> buf(G::BUF + 2);
  cd v[T][E];
  for (int t = 0; t < T; ++t)
    for (int q = 0; q < E; ++q) v[t][q] = cmake(in[2 * (t + T * q)], in[2 * (t + T * q) + 1]);
  for (int t = 0; t < T; ++t) fft_stage_compute<N, DIR, 0>(v[t], t, tw.data());
  if constexpr (G::S > 1) {
    exchange_split<N, 0>(v, buf.data());
    for (int t = 0; t < T; ++t) fft_stage_compute<N, DIR, 1>(v[t], t, tw.data());
  }
  if constexpr (G::S > 2) {
    exchange_split<N, 1>(v, buf.data());
    for (int t = 0; t < T; ++t) fft_stage_compute<N, DIR, 2>(v[t], t, tw.data());
  }
  for (int t = 0; t < T; ++t)
    for (int q = 0; q < E; ++q) { out[2 * (t + T * q)] = v[t][q].x; out[2 * (t + T * q) + 1] = v[t][q].y; }
}
extern "C" int host_fft_split(int n, int dir, const double* in, double* out) {
#define SCASE(NN) case NN: if (dir < 0) run_split<NN, -1>(in, out); else run_split<NN, +1>(in, out); return 0;
  switch (n) { SCASE(2) SCASE(4) SCASE(8) SCASE(16) SCASE(32) SCASE(64) SCASE(128) SCASE(256) SCASE(512) SCASE(256 + GD_FFT_ALT) }
  return -1;
}

extern "C" int host_fft(int n, int dir, const double* in, double* out) {
#define CASE(NN) case NN: if (dir < 0) run<NN, -1>(in, out); else run<NN, +1>(in, out); return 0;
  switch (n) { CASE(2) CASE(4) CASE(8) CASE(16) CASE(32) CASE(64) CASE(128) CASE(256) CASE(512) CASE(256 + GD_FFT_ALT) }
  return -1;
}
// bank-conflict audit: max number of lanes of one quarter-warp (8 lanes x 16 B) whose scatter
// addresses fall in the same 16-byte bank group, for stage s of length n.
template <int N, int s> static int conflicts() {
  using G = FftGeom<N>;
  constexpr int R = G::template radix<s>(), NS = G::template ns<s>(), B = G::E / R;
  int worst = 1;
  for (int b = 0; b < B; ++b)
    for (int i = 0; i < R; ++i)
      for (int q0 = 0; q0 < 32; q0 += 8) {      // a quarter warp: lanes q0..q0+7 (lane -> line l, lane-in-group t)
        int cnt[8] = {0};
        for (int lane = q0; lane < q0 + 8; ++lane) {
          int t = lane % G::T, line = lane / G::T;
          int j = t + G::T * b, j0 = (j / NS) * NS * R + (j % NS);
          int addr = line * G::BUF + G::pad(j0 + i * NS);
          cnt[addr % 8]++;
        }
        for (int k = 0; k < 8; ++k) if (cnt[k] > worst) worst = cnt[k];
      }
  return worst;
}
extern "C" int host_fft_scatter_conflicts(int n) {
  switch (n) {
    case 32: return conflicts<32, 0>();
    case 64: return conflicts<64, 0>();
    case 128: return conflicts<128, 0>();
    case 256: return conflicts<256, 0>();
    case 512: { int a = conflicts<512, 0>(), b = conflicts<512, 1>(); return a > b ? a : b; }
  }
  return 1;
}

// Split (8-byte) exchange audit for a whole warp: worst number of lanes of one warp-wide store / load that fall on the same
// 8-byte bank pair (16 of them), over all scatter and gather instructions of stage s.  32 lanes x 8 B = 2 wavefronts at best,
// so the ideal answer is 2.  The warp holds 32/T lane groups with buffers BUF+2 doubles apart (pass_x.cu, passes_zy.cu).
template <int ID, int s> static int split_conflicts() {
  using G = FftGeom<ID>;
  constexpr int R = G::template radix<s>(), NS = G::template ns<s>(), B = G::E / R;
  int worst = 0;
  for (int b = 0; b < B; ++b)
    for (int i = 0; i < R; ++i) {
      int cnt[16] = {0};
      for (int lane = 0; lane < 32; ++lane) {
        int t = lane % G::T, line = lane / G::T;
        int j = t + G::T * b, j0 = (j / NS) * NS * R + (j % NS);
        cnt[(line * (G::BUF + 2) + G::pad(j0 + i * NS)) % 16]++;
      }
      for (int k = 0; k < 16; ++k) if (cnt[k] > worst) worst = cnt[k];
    }
  for (int q = 0; q < G::E; ++q) {
    int cnt[16] = {0};
    for (int lane = 0; lane < 32; ++lane) {
      int t = lane % G::T, line = lane / G::T;
      cnt[(line * (G::BUF + 2) + G::pad(t + G::T * q)) % 16]++;
    }
    for (int k = 0; k < 16; ++k) if (cnt[k] > worst) worst = cnt[k];
  }
  return worst;
}
extern "C" int host_fft_split_conflicts(int id) {
  switch (id) {
    case 256: return split_conflicts<256, 0>();
    case 256 + GD_FFT_ALT: { int a = split_conflicts<256 + GD_FFT_ALT, 0>(), b = split_conflicts<256 + GD_FFT_ALT, 1>(); return a > b ? a : b; }
    case 512: { int a = split_conflicts<512, 0>(), b = split_conflicts<512, 1>(); return a > b ? a : b; }
  }
  return -1;
}
