// microbench.cu -- measured ceilings of the units the hot path leans on (instrumentation, not on the step path):
//   0  fp64 FMA issue rate (dependency-free DFMA chains on every SM)        -> the "alu" roof of the x-pass
//   1  lane-group FFT-256 rate (fft.cuh, split exchange, register twiddles)   -> what the transforms alone can do
//   2  tensor-memory load bandwidth (tcgen05.ld 32x32b.x8, the x-pass's Phi/Psi reads)
//   3  shared-memory load bandwidth (conflict-free LDS.128)
// Each test runs `reps` timed launches after one warm-up and reports the best one.  bench.py --microbench prints them
// and the main bench line carries the fp64 figure beside the HBM roofline (last paragraph).
#include <algorithm>
#include <cstdio>
#include <vector>
#include "../../include/gandalf.h"
#include "common.cuh"

// ---- 0: DFMA -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_mb_dfma(double* __restrict__ out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = (double)(threadIdx.x + i);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- 1: bare lane-group FFT-256 --------------------------------------------------------------------------------
template <int N, int NTWR, int THREADS>      // N: FFT plan ID (fft.cuh)
__global__ void __launch_bounds__(THREADS, 1) k_mb_fft(cd* __restrict__ out, const cd* __restrict__ tw, int reps) {
  using G = FftGeom<N>;
  constexpr int T = G::T, E = G::E;
  extern __shared__ cd smem[];
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  fft_load_table<N>(smem, tw);
  const cd* tws = smem;
  double* buf = reinterpret_cast<double*>(smem + FftTw<N>::COUNT) + (size_t)grp * (G::BUF + 2);
  cd v[E];
#pragma unroll
  for (int q = 0; q < E; ++q) v[q] = cmake(1.0 / (1 + t + T * q), 0.25 * grp);
  cd twr[NTWR > 0 ? NTWR : 1];
  if constexpr (NTWR > 0) fft_load_stage1_twiddles<N, NTWR>(twr, t, tws);
  for (int r = 0; r < reps; ++r) {
    if constexpr (NTWR > 0) fft_lanes_fwd_rt_split<N, NTWR>(v, t, buf, tws, twr);
    else fft_lanes_split<N, -1>(v, t, buf, tws);
    if ((r & 7) == 7) {                                             // 256^8 = 2^64: exact rescale, 4 DMUL per transform on average
#pragma unroll
      for (int q = 0; q < E; ++q) v[q] = cscale(v[q], 5.42101086242752217e-20);
    }
  }
  cd s = cmake(0.0, 0.0);
#pragma unroll
  for (int q = 0; q < E; ++q) s = s + v[q];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- 2: tensor-memory loads --------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 1) k_mb_tmem(unsigned* __restrict__ out, long long* __restrict__ cycles, int reps) {
  __shared__ unsigned s_base;
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(&s_base)), "r"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const unsigned tm = s_base + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * 256);
  // initialise this warp's 256 columns
  for (int c = 0; c < 256; c += 4)
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(tm + c), "r"(c), "r"(c + 1), "r"(c + 2), "r"(c + 3) : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  __syncthreads();
  unsigned acc = 0;
  const long long t0 = clock64();
  for (int r = 0; r < reps; ++r) {
#pragma unroll
    for (int c = 0; c < 256; c += 32) {          // 4 loads of 8 words in flight per wait, like the x-pass's batches
      unsigned w[32];
#pragma unroll
      for (int j = 0; j < 4; ++j)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=r"(w[8 * j]), "=r"(w[8 * j + 1]), "=r"(w[8 * j + 2]), "=r"(w[8 * j + 3]), "=r"(w[8 * j + 4]),
                       "=r"(w[8 * j + 5]), "=r"(w[8 * j + 6]), "=r"(w[8 * j + 7]) : "r"(tm + c + 8 * j) : "memory");
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
      for (int j = 0; j < 32; ++j) acc ^= w[j];
    }
  }
  const long long t1 = clock64();
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_base), "r"(512) : "memory");
}

// ---- 3: shared-memory loads ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 1) k_mb_lds(double* __restrict__ out, long long* __restrict__ cycles, int reps) {
  __shared__ double2 tile[2048];                 // 32 KB
  for (int i = threadIdx.x; i < 2048; i += blockDim.x) tile[i] = make_double2(i, -i);
  __syncthreads();
  double2 acc = make_double2(0.0, 0.0);
  const long long t0 = clock64();
  for (int r = 0; r < reps; ++r) {
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const double2 v = tile[(threadIdx.x + 256 * k + 17 * r) & 2047];     // consecutive lanes -> consecutive 16-byte words
      acc.x += v.x; acc.y += v.y;
    }
  }
  const long long t1 = clock64();
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc.x + acc.y;
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

int fft_stage_table_host(int n, std::vector<cd>& out);

template <class L> static float best_ms(int reps, L&& launch) {
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  launch();                                        // warm-up
  float best = 1e30f;
  for (int r = 0; r < reps; ++r) {
    cudaEventRecord(a);
    launch();
    cudaEventRecord(b);
    cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    best = std::min(best, ms);
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  return best;
}

extern "C" int gandalf_microbench(int which, int device, double* out, int nout) {
  if (!out || nout < 4) return GANDALF_ERR_INVALID;
  if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return GANDALF_ERR_CUDA; }
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
  if (sms <= 0) return GANDALF_ERR_CUDA;
  for (int i = 0; i < nout; ++i) out[i] = 0.0;
  void* buf = nullptr;
  long long* cyc = nullptr;
  const size_t nthreads = (size_t)sms * 8 * 256;
  if (cudaMalloc(&buf, nthreads * sizeof(cd)) != cudaSuccess || cudaMalloc((void**)&cyc, (size_t)sms * 8 * sizeof(long long)) != cudaSuccess) {
    cudaGetLastError(); if (buf) cudaFree(buf); return GANDALF_ERR_CUDA;
  }
  int rc = GANDALF_OK;
  if (which == 0) {
    const int iters = 4096, blocks = sms * 8;
    const float ms = best_ms(5, [&] { k_mb_dfma<<<blocks, 256>>>((double*)buf, iters, 1.0000001, 1e-9); });
    const double fma = (double)blocks * 256 * (double)iters * 32.0;
    out[0] = 2.0 * fma / (ms * 1e-3) / 1e12;      // TFLOP/s
    out[1] = fma / (ms * 1e-3) / 1e12;            // T fp64 instructions/s (thread level)
    out[2] = ms; out[3] = sms;
  } else if (which == 1) {
    std::vector<cd> h, ha;
    cd *tw = nullptr, *twa = nullptr;
    constexpr int ALT = 256 + GD_FFT_ALT;
    if (fft_stage_table_host(256, h) != 0 || fft_stage_table_host(ALT, ha) != 0 || cudaMalloc((void**)&tw, h.size() * sizeof(cd)) != cudaSuccess ||
        cudaMalloc((void**)&twa, ha.size() * sizeof(cd)) != cudaSuccess) rc = GANDALF_ERR_CUDA;
    else {
      cudaMemcpy(tw, h.data(), h.size() * sizeof(cd), cudaMemcpyHostToDevice);
      cudaMemcpy(twa, ha.data(), ha.size() * sizeof(cd), cudaMemcpyHostToDevice);
      using G = FftGeom<256>;
      using GA = FftGeom<ALT>;
      const size_t smem = (FftTw<256>::COUNT) * sizeof(cd) + (size_t)(256 / G::T) * (G::BUF + 2) * sizeof(double);
      const size_t smema = (FftTw<ALT>::COUNT) * sizeof(cd) + (size_t)(512 / GA::T) * (GA::BUF + 2) * sizeof(double);
      const int reps = 512;
      cudaFuncSetAttribute(k_mb_fft<256, 8, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      cudaFuncSetAttribute(k_mb_fft<256, 0, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      cudaFuncSetAttribute(k_mb_fft<ALT, 0, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smema);
      const float ms8 = best_ms(5, [&] { k_mb_fft<256, 8, 256><<<sms, 256, smem>>>((cd*)buf, tw, reps); });
      const float ms0 = best_ms(5, [&] { k_mb_fft<256, 0, 256><<<sms, 256, smem>>>((cd*)buf, tw, reps); });
      const float msa = best_ms(5, [&] { k_mb_fft<ALT, 0, 512><<<sms, 512, smema>>>((cd*)buf, twa, reps); });
      const double ntr = (double)sms * (256 / G::T) * reps;
      out[0] = ntr / (ms8 * 1e-3) / 1e9;          // G transforms/s, plan 16*16 on 16 lanes, 8 register twiddles, 8 warps per SM
      out[1] = ntr / (ms0 * 1e-3) / 1e9;          // same, all twiddles from shared memory
      out[2] = ntr / (msa * 1e-3) / 1e9;          // plan 8*8*4 on 32 lanes, 16 warps per SM (the x-pass's plan at nx = 256)
      out[3] = ms8;
    }
    if (tw) cudaFree(tw);
    if (twa) cudaFree(twa);
  } else if (which == 2 || which == 3) {
    const int reps = which == 2 ? 2048 : 4096;
    float ms;
    if (which == 2) ms = best_ms(3, [&] { k_mb_tmem<<<sms, 256>>>((unsigned*)buf, cyc, reps); });
    else ms = best_ms(3, [&] { k_mb_lds<<<sms, 256>>>((double*)buf, cyc, reps); });
    std::vector<long long> hc(sms);
    cudaMemcpy(hc.data(), cyc, sms * sizeof(long long), cudaMemcpyDeviceToHost);
    double mean = 0.0;
    for (long long v : hc) mean += (double)v;
    mean /= sms;
    const double bytes_per_sm = which == 2 ? 256.0 * 32.0 * 4.0 * 8.0 /* 8 warps x 32 lanes x 256 words */ * reps
                                           : 256.0 * 16.0 * 16.0 * reps;
    out[0] = bytes_per_sm / mean;                 // bytes per SM clock per SM
    out[1] = bytes_per_sm * sms / (ms * 1e-3) / 1e12;   // TB/s over the chip
    out[2] = ms; out[3] = mean;
  } else rc = GANDALF_ERR_INVALID;
  if (rc == GANDALF_OK && cudaDeviceSynchronize() != cudaSuccess) rc = GANDALF_ERR_CUDA;
  if (cudaGetLastError() != cudaSuccess) rc = GANDALF_ERR_CUDA;
  cudaFree(buf); cudaFree(cyc);
  return rc;
}
