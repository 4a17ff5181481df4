// noalloc.cu -- gandalf_kperp_spectrum_noalloc (include/gandalf.h): the perpendicular shell spectrum of Eq. 26
// (Q15) for callers that must not allocate device memory.
//
// Who that is.  Every other entry point works on a gandalf_ctx, and gandalf_create / gandalf_kperp_spectrum obtain
// their buffers from cudaMalloc.  Some programs that want this diagnostic cannot do that at the point where they
// call it: a host application that handed the whole GPU to its own memory pool at start-up (a fresh cudaMalloc then
// fails, or forces the pool to give memory back), and monitoring hooks that run beside other streams' work and
// cannot afford the device-wide synchronisation cudaMalloc and cudaFree bring with them.  Such a caller owns the
// state array and the output array and hands both in; the only other memory the reduction needs -- one partial sum
// per retained (kx, ky) column -- lives in the fixed array below, which is part of the library image.
//
// What follows from a shared, fixed array:
//   * It has GANDALF_NOALLOC_MAX_COLUMNS entries (256 KB).  Every GPU on which this library's code gets loaded holds
//     that much until the process exits, whether or not the entry point is ever called.  Grids whose retained plane
//     (nx/3 + 1) * (2 (ny/3) + 1) is larger are refused with GANDALF_ERR_INVALID and a message; nothing is launched.
//   * All calls on one device use the same array, and it keeps whatever the previous call left there.  Nothing has to
//     start at zero: the first kernel writes entry i of every column i of THIS call's grid before the second kernel
//     reads exactly those entries, so leftovers from a larger earlier grid are never looked at.
//   * Two calls whose kernels can be on the GPU at the same time (different streams without an ordering between them,
//     or two host threads) overwrite each other's partial sums.  Order them: one stream, or an event between them.
//   * The first call on a device looks up the array's device address (cudaGetSymbolAddress, which may make the
//     driver load this library's code on that device).  Make that first call early -- before any stream capture is
//     begun -- so that later calls only validate and launch.
// The entry point calls no cudaMalloc, cudaFree or other allocating routine, and does not synchronise.
//
// The two kernels are variants of k_spec_columns / k_spec_bins (pointwise.cu): same arithmetic, same summation order.
#include <cstdio>
#include <mutex>

#include "../../include/gandalf.h"
#include "common.cuh"

// One partial sum per retained (ky, kx) column.  In HOST code this name is only a handle for the runtime (taking its
// address there does not give device memory); the device address comes from cudaGetSymbolAddress, per device.
static __device__ __align__(256) double g_noalloc_columns[GANDALF_NOALLOC_MAX_COLUMNS];

// step 1 (variant of k_spec_columns): col[cy][cx] = sum over cz of the mode energy, serial in cz, half-plane weight
__global__ void __launch_bounds__(256) k_noalloc_spec_columns(Dims d, const cd* __restrict__ W, double* __restrict__ col, int literal) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int plane = d.Ky * d.Kx;
  if (i >= plane) return;
  const int cx = i % d.Kx, cy = i / d.Kx;
  const double kx = d.kx0 * cx, ky = d.ky0 * c2n(cy, d.hy3, d.Ky);
  const double k2 = kx * kx + ky * ky;
  double e = 0.0;
  if (k2 > 0.0) {
    for (int cz = 0; cz < d.Kz; ++cz) {
      const cd wp = W[(size_t)cz * plane + i], wm = W[d.PS + (size_t)cz * plane + i];
      e += (wp.x * wp.x + wp.y * wp.y) + (wm.x * wm.x + wm.y * wm.y);
    }
    e *= literal ? 1.0 / (k2 * k2) : 0.25 / k2;     // |xi|^2 = |w|^2 / kperp^4 ; mode energy 1/4 kperp^2 |xi|^2
    e *= (cx == 0 ? 1.0 : 2.0);
  }
  col[i] = e;
}
// step 2 (variant of k_spec_bins): one block per bin j = floor(kperp/dk + 1/2); strided loop, then a tree
__global__ void __launch_bounds__(256) k_noalloc_spec_bins(Dims d, const double* __restrict__ col, double dk, double* __restrict__ out) {
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

// Device address of g_noalloc_columns on each device, looked up once per device with that device current.
static const int kMaxDevices = 64;
static std::mutex g_noalloc_mutex;
static double* g_noalloc_addr[kMaxDevices];

static cudaError_t noalloc_scratch(int device, double** out) {
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_addr[device]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_columns);     // the CURRENT device's copy
    if (e != cudaSuccess) return e;
    g_noalloc_addr[device] = static_cast<double*>(p);
  }
  *out = g_noalloc_addr[device];
  return cudaSuccess;
}

static int noalloc_fail(int code, char* err, int errlen, const char* msg) {
  if (err && errlen > 0) std::snprintf(err, (size_t)errlen, "%s", msg);
  return code;
}
static bool noalloc_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

extern "C" int gandalf_kperp_spectrum_noalloc(int device, void* stream, int nx, int ny, int nz, double Lx, double Ly,
                                              const double* w_raw, int nbins, int literal_eq26, double* out,
                                              char* err, int errlen) {
  if (err && errlen > 0) err[0] = '\0';
  char msg[256];
  // host-side checks first: nothing below this block runs for a bad argument
  if (!w_raw || !out) return noalloc_fail(GANDALF_ERR_INVALID, err, errlen, "gandalf_kperp_spectrum_noalloc: NULL array");
  if (!noalloc_pow2(nx) || !noalloc_pow2(ny) || !noalloc_pow2(nz) || nx < 8 || ny < 8 || nz < 2 || nx > 512 || ny > 512 || nz > 512)
    return noalloc_fail(GANDALF_ERR_INVALID, err, errlen,
                        "gandalf_kperp_spectrum_noalloc: grid must be powers of two with 8 <= nx, ny <= 512 and 2 <= nz <= 512");
  if (!(Lx > 0.0) || !(Ly > 0.0) || nbins <= 0 || nbins > 65535 || device < 0 || device >= kMaxDevices)
    return noalloc_fail(GANDALF_ERR_INVALID, err, errlen, "gandalf_kperp_spectrum_noalloc: bad box length, bin count or device");
  Dims d{};
  d.nx = nx; d.ny = ny; d.nz = nz;
  d.hx3 = nx / 3; d.hy3 = ny / 3; d.hz3 = nz / 3;
  d.Kx = d.hx3 + 1; d.Ky = 2 * d.hy3 + 1; d.Kz = 2 * d.hz3 + 1;
  const long long plane = (long long)d.Ky * d.Kx;
  if (plane > (long long)GANDALF_NOALLOC_MAX_COLUMNS) {
    std::snprintf(msg, sizeof(msg),
                  "gandalf_kperp_spectrum_noalloc: %d x %d has %lld retained (kx, ky) columns, the fixed scratch array holds "
                  "%d; use gandalf_kperp_spectrum (which allocates) for this grid", nx, ny, plane, GANDALF_NOALLOC_MAX_COLUMNS);
    return noalloc_fail(GANDALF_ERR_INVALID, err, errlen, msg);
  }
  const double kPi = 3.14159265358979323846264338327950288;
  d.kx0 = 2.0 * kPi / Lx; d.ky0 = 2.0 * kPi / Ly;
  d.PS = (size_t)d.Kz * d.Ky * d.Kx;
  const double dk = 2.0 * kPi / (Lx > Ly ? Lx : Ly);

  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
  double* col = nullptr;
  if (e == cudaSuccess) e = noalloc_scratch(device, &col);
  if (e == cudaSuccess) {
    cudaStream_t st = (cudaStream_t)stream;
    const cd* W = reinterpret_cast<const cd*>(w_raw);
    k_noalloc_spec_columns<<<(unsigned)((plane + 255) / 256), 256, 0, st>>>(d, W, col, literal_eq26);
    k_noalloc_spec_bins<<<nbins, 256, 0, st>>>(d, col, dk, out);
    e = cudaGetLastError();
  }
  if (prev >= 0 && prev != device) cudaSetDevice(prev);
  if (e != cudaSuccess) {
    std::snprintf(msg, sizeof(msg), "gandalf_kperp_spectrum_noalloc: %s", cudaGetErrorString(e));
    return noalloc_fail(GANDALF_ERR_CUDA, err, errlen, msg);
  }
  return GANDALF_OK;
}
