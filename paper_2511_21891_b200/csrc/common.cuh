// common.cuh -- grid geometry shared by the kernels of the GANDALF hot path (device side only).
//
// Storage spaces (all complex fp64, kx fastest; "c" indices run over RETAINED modes only, i.e.
// the modes Eq. 20 keeps: 3|n| <= N):
//   compact  S[f][cz][cy][cx]   Kz*Ky*Kx per field   fully spectral state / RHS
//   hybrid   H[f][z ][cy][cx]   nz*Ky*Kxp per field  z in real space, (kx,ky) spectral; row stride Kxp (= Kx, see api.cu)
//   xy-real  D[a][lb][cx][xl]   y,z real, kx spectral (retained kx only); line = z*ny+y = lb*xl + li, stored at slot
//                               li ^ (cx % xl): the tile of an x-pass CTA (xl lines) is one contiguous run (P1 -> P2)
//            E[a][z ][y ][cx]   nz*ny*Kxe per array  same space, kx fastest, rows padded to Kxe = 8*ceil(Kx/8) (P2 -> P3)
// cx = 0..Kx-1 is n_x = cx; cy = 0..Ky-1 is n_y = cy (cy <= hy3) or cy-Ky (negative modes);
// cz likewise.  The zeroed third is never stored or transformed.
#pragma once
#include <cuda.h>            // CUtensorMap (type only: the encoder is fetched through cudaGetDriverEntryPoint, api.cu)
#include <cuda_runtime.h>
#include "fft.cuh"

struct Dims {
  int nx, ny, nz, M, F;   // M = number of moment FIELDS (nspecies * Msp), F = 2 + M
  int Msp;                // moments per species
  int own_lo, own_hi;     // owned moment fields [own_lo, own_hi) (all of them unless the context is a moment shard with halos, Q31)
  int hx;                 // nx/2+1 (boundary layout)
  int Kx, Ky, Kz;         // retained counts
  int Kxp, Kxe;           // row strides (>= Kx) of the hybrid arrays H, Gh and of E
  int hx3, hy3, hz3;      // floor(N/3)
  double kx0, ky0, kz0;   // 2 pi / L
  double inv_n;           // 1/(nx ny nz)
  double bscale, inv_bscale;   // power of two ~ kperp,max^2/2: the x-pass transforms the pair (A, bscale*B) so that B's round-off
                          // floor is not set by A's magnitude before N+- = -1/2 A -+ 1/2 kperp^2 B amplifies it
  int xl, xlsh;           // lines per x-pass CTA (power of two) and its log2: block size of the D layout
  size_t PS, PH, PD, PE;  // per-field strides (complex elements): compact, hybrid, D (blocked, padded), E
};

// Row split of a tile of `rows` rows into boxes (a box has at most 256 rows; box starts stay multiples of 8 rows so that the
// swizzle phase of a row is its index & 7 throughout the sub-tile).  Used by the kernels (compile time) and by api.cu (maps).
constexpr int tma_nrb(int rows) { return (rows + 255) / 256; }
constexpr int tma_rb(int rows) { return tma_nrb(rows) == 1 ? rows : (((rows + tma_nrb(rows) - 1) / tma_nrb(rows) + 7) / 8 * 8); }
constexpr int tma_substr(int rows) {          // complex entries of one 8-column sub-tile, a multiple of 1024 bytes
  return (tma_nrb(rows) * tma_rb(rows) * 8 + 63) / 64 * 64;
}

// Tensor maps of the context's arrays (built once in gandalf_create, api.cu; passed to the kernels as __grid_constant__ params).
struct TMaps {
  CUtensorMap g_flat, h_flat;   // Gh, H as {2*Ky*Kx, nz, F}: the [nz][8 columns] boxes of P4 (load / store)
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

// ---- mbarrier + bulk async copy (TMA engine, 1-D form: no tensor map needed) -------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
               : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
// non-blocking probe of a phase: the result can be consumed much later, so its shared-memory round trip hides behind other work
__device__ __forceinline__ bool mbar_test_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  asm volatile("{\n .reg .pred p;\n mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
               : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
// try_wait is the suspending form: the hardware parks the thread for a bounded time before it returns false, so the
// retry loop does not burn issue slots.  -DGD_DEBUG_MBAR builds trap after ~2^26 retries (a faulted bulk copy then
// surfaces as a launch error instead of hanging the stream).
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
#ifdef GD_DEBUG_MBAR
  unsigned long long spins = 0;
#endif
  while (!mbar_try_wait(bar, parity)) {
#ifdef GD_DEBUG_MBAR
    if (++spins > (1ull << 26)) __trap();
#endif
  }
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completion counted on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// shared -> global (bulk group completion)
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src_smem, unsigned bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
}
// global -> L2 only (no shared-memory destination, no completion tracking): warms the lines a later load will ask for
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// ---- tiled bulk tensor copies (TMA, tensor-map form) for P4.  Its [nz][columns] tiles move with ONE instruction per 8-column
// sub-tile issued by one thread: per-row 1-D bulk copies cost a warp-serialised issue loop (ELECT/R2UR per lane: 20 % of P4's warp
// time in round 1).  The maps view the arrays as fp64 tensors (a complex entry = 2 elements); boxes are 8 complex columns wide
// (128 B) and land in shared memory with the 128-byte swizzle: element (row r, column c < 8) of a sub-tile sits at
// r*8 + (c ^ (r & 7)) (in complex entries; sub-tile base 1024-byte aligned), so the lanes of a transform, which read one column
// over consecutive rows, hit eight different 16-byte bank groups.  Measured at 4a: P4 0.816 -> 0.780 ms.  The same scheme on the
// y passes (P1, P3) was measured SLOWER than their per-row 1-D copies of 256 B (P1 0.869 -> 0.905 ms with two 8-column boxes,
// 0.924 ms with one row-major {16, 2, rows} box; P3 0.528 -> 0.542 / 0.566 ms), so they keep the 1-D form.
__device__ __forceinline__ int swz8(int r, int c) { return r * 8 + (c ^ (r & 7)); }
__device__ __forceinline__ void tma_load_3d(void* dst_smem, const CUtensorMap* m, int c0, int c1, int c2, unsigned long long* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(smem_u32(dst_smem)), "l"(m), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* m, int c0, int c1, int c2, const void* src_smem) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3}], [%4];"
               ::"l"(m), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(src_smem)) : "memory");
}
__device__ __forceinline__ cd* align1024(void* p) {           // dynamic shared memory is only 16-byte aligned by contract
  return reinterpret_cast<cd*>((reinterpret_cast<unsigned long long>(p) + 1023ull) & ~1023ull);
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

struct PhysParams {
  double vA;
  double eta; int r; int eta_normalized;
  double eta_z; int r_z;
  double eta_g;
  double k2max_perp, kz2max;     // (pi nx/Lx)^2 + (pi ny/Ly)^2 ; (pi nz/Lz)^2
  int if_variant; int g_sign;
};

// device scalars owned by the context
enum { SC_DT = 0, SC_T = 1, SC_LASTDT = 2, SC_ERR = 3, SC_STEP = 4, SC_COUNT = 8 };   // SC_ERR != 0: Eq. 16 had no flow to bound dt (sticky)
// SC_STEP: the step number (an exact integer in a double), advanced on the device with the time so that a captured CUDA graph of
// one step replays correctly: the forcing counters (Q17, Q26) and the slot of the energy record derive from it

// Launch geometry of the z transforms: GD_Z_THREADS lanes per CTA = GD_Z_THREADS/T adjacent (cy,cx) columns.
#define GD_Z_THREADS 128
