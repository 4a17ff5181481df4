// api.cu -- the C ABI of include/gandalf.h: context, buffers, and the step driver that enqueues the
// fixed kernel sequence of Algorithm 2 on one CUDA stream.  No host
// synchronisation inside gandalf_step: dt (also the CFL one), time and the energy records live
// on the device.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <new>
#include <string>
#include <vector>

#include "../../include/gandalf.h"
#include "common.cuh"

// ---- kernels' launchers (defined in passes_zy.cu, pass_x.cu, pointwise.cu) --------------------------------
cudaError_t launch_zfft(const Dims& d, const cd* in, cd* out, const cd* tw, int nfields, cudaStream_t st);
cudaError_t launch_yinv(const Dims& d, const cd* H, cd* D, const cd* tw, int num_sms, cudaStream_t st);
cudaError_t launch_yfwd(const Dims& d, const cd* E, cd* Gh, const cd* tw, int num_sms, cudaStream_t st);
cudaError_t prepare_passes_zy(int ny, int nz);
int xpass_lines_per_cta(int nx);
int xpass_fft_plan_id(int nx);
cudaError_t launch_xpass(const Dims& d, const cd* D, cd* Eo, const cd* tw, const double* cdn, const double* cup,
                         unsigned long long* maxbits, int num_sms, cudaStream_t st, bool prepare_only);
cudaError_t launch_zstep(const Dims& d, const TMaps& tm, int mode, bool exact, int if_variant, int g_sign, bool have_G, const cd* Wn, const cd* Ws,
                         cd* Wout, bool want_H, const double* scal, const double* cdn, const double* cup, const double* collfac,
                         const double* tabz, const double* tabp, const cd* tw, cudaStream_t st);
void jacobi_eigh(int n, std::vector<double>& A, std::vector<double>& V, std::vector<double>& lam);
cudaError_t launch_hermite_propagator(const Dims& d, int g_sign, double frac, const double* scal, const double* V, const double* lam,
                                      cd* P, cudaStream_t st);
cudaError_t launch_hermite_apply(const Dims& d, const cd* in, cd* out, const cd* P, int diss, const double* collfac,
                                 const double* tabz, const double* tabp, cudaStream_t st);
cudaError_t launch_tables(const Dims& d, const PhysParams& p, const double* scal, double* tabz, double* tabp, cudaStream_t st);
cudaError_t launch_prepare_dt(double fixed_dt, double cfl_dxy, double dt_max, const unsigned long long* maxbits, double* scal,
                              const double* crate, double* collfac, int M, cudaStream_t st);
cudaError_t launch_zero_u64(unsigned long long* p, cudaStream_t st);
cudaError_t launch_pack(const Dims& d, const cd* in, cd* S, int nfields, int nzeta, cudaStream_t st);
cudaError_t launch_unpack(const Dims& d, const cd* S, cd* out, int nfields, int nzeta, cudaStream_t st);
cudaError_t launch_forcing(const Dims& d, cd* S, const int* pairs, int npairs, double amp, unsigned long long seed,
                           const double* scal, cudaStream_t st);
cudaError_t launch_forcing_g(const Dims& d, cd* S, int nzf, double amp, unsigned long long seed,
                             const double* scal, cudaStream_t st);
cudaError_t launch_energy(const Dims& d, const cd* S, double* partial, int nblocks, double* rec, long long hist_base, double* scal, int advance,
                          cudaStream_t st);
cudaError_t launch_spectrum(const Dims& d, const cd* S, double* col, int nbins, int literal, double dk, double* out, cudaStream_t st);
cudaError_t launch_hermite_spectrum(const Dims& d, const cd* S, double* out, cudaStream_t st);
cudaError_t launch_kpar_spectrum(const Dims& d, const cd* S, double* rows, int nbins, double* out, cudaStream_t st);

static const double kPi = 3.14159265358979323846264338327950288;
enum { KC_ZINV = 0, KC_YINV = 1, KC_XPASS = 2, KC_YFWD = 3, KC_ZSTEP = 4, KC_N = 5 };
static const int kEnergyBlocks = 592;   // 4 x 148 SMs

struct gandalf_ctx {
  gandalf_params p;
  Dims d;
  PhysParams ph;
  TMaps tm;
  cudaStream_t st;
  // device buffers
  cd *S0, *S1, *H, *Gh, *D, *E;
  cd *twx, *twy, *twz;
  double *cdn, *cup, *crate, *collfac, *scal, *partial, *hist, *rec_scratch, *spec_col, *spec_out, *tabz, *tabp;
  double *hxV, *hxLam; cd* hxP;      // hermite_exact: eigenvectors / eigenvalues of the coupling matrix, propagators P(dt/2) per kz
  unsigned long long* maxbits;
  int* pairs; int npairs; double force_amp;
  cd* io; size_t io_bytes;
  int spec_cap;
  long long hist_cap;
  // host bookkeeping
  long long step, hist_base; bool H_valid;   // history record i belongs to step hist_base + i
  bool stage_pending, need_h;                // between gandalf_step_stage(.., 0) and (.., 1); whether this step keeps the hybrid copy
  int num_sms;
  long long launches;
  long long h2d_bytes, d2h_bytes;            // bytes the host-pointer entry points moved over PCIe so far (gandalf_transfer_bytes)
  bool timing;
  // CUDA graph of ONE step (gandalf_step with a fixed dt or the CFL dt; DESIGN.md section 5 "launch path"): captured from the very
  // launches a plain step makes, replayed nsteps times.  Valid while the by-value launch arguments stay the same (key below).
  int graph_mode;                            // 1 (default): replay a graph when the stream allows capture; 0: plain launches
  cudaGraphExec_t gexec; double g_dt, g_last_dt; double* g_hist; long long g_hist_base; long long g_launches; long long graph_replays;
  struct Ev { cudaEvent_t a, b; int cls; };
  std::vector<Ev> evs;
  double t_ms[KC_N]; long long t_n[KC_N];
  std::string err;
};

#define GD_FAIL(ctx, code, msg) do { (ctx)->err = (msg); return (code); } while (0)
#define GD_CUDA(ctx, call)                                                                         \
  do {                                                                                             \
    cudaError_t e__ = (call);                                                                      \
    if (e__ != cudaSuccess) {                                                                      \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                            \
      return GANDALF_ERR_CUDA;                                                                     \
    }                                                                                              \
  } while (0)

static bool pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// canonical members (nx > 0, or nx = 0 and ny > 0) of the +-k pairs of the forced shell (Eq. 25; Q17)
static int count_forced_pairs(const gandalf_params* p) {
  const int lo2 = p->force_nperp_min * p->force_nperp_min, hi2 = p->force_nperp_max * p->force_nperp_max;
  int n = 0;
  for (int nz = -p->force_nz_max; nz <= p->force_nz_max; ++nz)
    for (int ny = -p->force_nperp_max; ny <= p->force_nperp_max; ++ny)
      for (int nx = 0; nx <= p->force_nperp_max; ++nx) {
        const int n2 = nx * nx + ny * ny;
        if (n2 < lo2 || n2 > hi2 || n2 == 0) continue;
        if ((nx > 0) || (nx == 0 && ny > 0)) ++n;
      }
  return n;
}

template <class T> static cudaError_t dalloc(T** p, size_t count) { return cudaMalloc((void**)p, count * sizeof(T)); }

int fft_stage_table_host(int n, std::vector<cd>& out);

static cudaError_t upload_twiddles(cd** dst, int n, cudaStream_t st) {
  std::vector<cd> h;
  if (fft_stage_table_host(n, h) != 0) return cudaErrorInvalidValue;
  cudaError_t e = dalloc(dst, h.size());
  if (e != cudaSuccess) return e;
  e = cudaMemcpyAsync(*dst, h.data(), h.size() * sizeof(cd), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return e;
  return cudaStreamSynchronize(st);
}

// ---- tensor maps (TMA descriptors) ---------------------------------------------------------------------------
// cuTensorMapEncodeTiled is a driver entry point; it is fetched through the runtime so the library links against cudart only.
#ifndef GD_TMA_L2PROMO
#define GD_TMA_L2PROMO 3      // CU_TENSOR_MAP_L2_PROMOTION_*: 0 none, 1 64 B, 2 128 B, 3 256 B
#endif
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess) return nullptr;
  return (EncodeTiledFn)fn;
}
// fp64 view of a complex array: dims[0] counts doubles; strides in complex entries (dims 1..rank-1); boxes of 8 complex columns
// (16 doubles = 128 B) x box_rows rows, 128-byte swizzle, out-of-range elements read as zeros / are not written.
static bool make_map(EncodeTiledFn enc, CUtensorMap* m, cd* base, int rank, const unsigned long long* dims, const unsigned long long* strides_cd,
                     int box_rows) {
  cuuint64_t gd[5], gs[4];
  cuuint32_t box[5], es[5];
  for (int i = 0; i < rank; ++i) { gd[i] = dims[i]; box[i] = 1; es[i] = 1; }
  for (int i = 0; i + 1 < rank; ++i) gs[i] = strides_cd[i] * sizeof(cd);
  box[0] = 16; box[1] = (cuuint32_t)box_rows;
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, base, gd, gs, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, (CUtensorMapL2promotion)GD_TMA_L2PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
static bool build_tmaps(gandalf_ctx* c) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const Dims& d = c->d;
  const unsigned long long plane = (unsigned long long)d.Ky * d.Kx;
  const int zrows = tma_rb(d.nz);
  {   // P4: (ky,kx) plane flattened (hybrid rows are unpadded: Kxp == Kx)
    const unsigned long long dims[3] = {2 * plane, (unsigned long long)d.nz, (unsigned long long)d.F};
    const unsigned long long str[2] = {plane, d.PH};
    if (!make_map(enc, &c->tm.g_flat, c->Gh, 3, dims, str, zrows)) return false;
    if (!make_map(enc, &c->tm.h_flat, c->H, 3, dims, str, zrows)) return false;
  }
  return true;
}

static void free_all(gandalf_ctx* c) {
  void* ptrs[] = {c->tabz, c->tabp, c->S0, c->S1, c->H, c->Gh, c->D, c->E, c->twx, c->twy, c->twz, c->cdn, c->cup, c->crate,
                  c->collfac, c->scal, c->partial, c->hist, c->rec_scratch, c->spec_col, c->spec_out, c->maxbits,
                  c->pairs, c->io, c->hxV, c->hxLam, c->hxP};
  for (void* q : ptrs) if (q) cudaFree(q);
  if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
  for (auto& e : c->evs) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
}

// timing-aware launch wrapper
template <class F> static cudaError_t timed(gandalf_ctx* c, int cls, int nlaunch, F&& f) {
  c->launches += nlaunch;
  if (!c->timing || cls < 0) return f();
  gandalf_ctx::Ev ev; ev.cls = cls;
  cudaEventCreate(&ev.a); cudaEventCreate(&ev.b);
  cudaEventRecord(ev.a, c->st);
  cudaError_t e = f();
  cudaEventRecord(ev.b, c->st);
  c->evs.push_back(ev);
  return e;
}

static void drain_events(gandalf_ctx* c) {
  for (auto& e : c->evs) {
    float ms = 0.f;
    if (cudaEventSynchronize(e.b) == cudaSuccess && cudaEventElapsedTime(&ms, e.a, e.b) == cudaSuccess) {
      c->t_ms[e.cls] += ms; c->t_n[e.cls] += 1;
    }
    cudaEventDestroy(e.a); cudaEventDestroy(e.b);
  }
  c->evs.clear();
}

extern "C" {

int gandalf_default_params(gandalf_params* p) {
  if (!p) return GANDALF_ERR_INVALID;
  std::memset(p, 0, sizeof(*p));
  p->nx = p->ny = 32; p->nz = 16; p->M = 0;
  p->Lx = p->Ly = p->Lz = 2.0 * kPi; p->vA = 1.0;
  p->r = 1; p->r_z = 1; p->p = 1.0;
  p->g_sign = 1; p->nonlinear = 1;
  p->force_nperp_min = 1; p->force_nperp_max = 2; p->force_nz_max = 1;
  p->cfl = 0.3;
  p->force_g_nz = 1;
  p->nspecies = 1;
  p->dt_max = 0.0; p->hermite_exact = 0;
  p->m_offset = 0; p->M_global = 0;
  return GANDALF_OK;
}

int gandalf_create(const gandalf_params* p, gandalf_ctx** out) {
  if (!p || !out) return GANDALF_ERR_INVALID;
  *out = nullptr;
  if (!pow2(p->nx) || !pow2(p->ny) || !pow2(p->nz)) return GANDALF_ERR_INVALID;
  if (p->nx < 8 || p->ny < 8 || p->nz < 2 || p->nx > 512 || p->ny > 512 || p->nz > 512) return GANDALF_ERR_INVALID;
  if (p->M < 0 || p->M > 4096 || !(p->Lx > 0) || !(p->Ly > 0) || !(p->Lz > 0)) return GANDALF_ERR_INVALID;
  if (p->r < 1 || p->r_z < 1 || !(p->p > 0) || (p->g_sign != 1 && p->g_sign != -1)) return GANDALF_ERR_INVALID;
  if (p->eta < 0 || p->eta_z < 0 || p->eta_g < 0 || p->nu_coll < 0 || p->force_eps < 0) return GANDALF_ERR_INVALID;
  if (p->closure != 0 && p->closure != 1) return GANDALF_ERR_INVALID;
  if (p->force_g_amp < 0 || (p->force_g_amp > 0 && (p->M < 1 || p->force_g_nz < 1 || p->force_g_nz > p->nz / 3))) return GANDALF_ERR_INVALID;
  if (p->nspecies != 1 && p->nspecies != 2) return GANDALF_ERR_INVALID;
  if (!(p->dt_max >= 0.0) || !(p->cfl > 0.0)) return GANDALF_ERR_INVALID;
  if (p->hermite_exact != 0 && p->hermite_exact != 1) return GANDALF_ERR_INVALID;
  if (p->force_eps > 0.0 && (p->force_nperp_min < 0 || p->force_nperp_max > p->nx / 3 || p->force_nperp_max > p->ny / 3 ||
                             p->force_nz_max > p->nz / 3 || count_forced_pairs(p) == 0)) return GANDALF_ERR_INVALID;   // empty / unresolved shell
  if (p->M_global != 0) {   // moment shard (Q31)
    if (p->M < 1 || p->m_offset < 0 || p->m_offset + p->M > p->M_global) return GANDALF_ERR_INVALID;
    if (p->nspecies != 1 || p->hermite_exact) return GANDALF_ERR_UNSUPPORTED;
    if (p->m_offset > 0 && p->M < 2) return GANDALF_ERR_INVALID;               // a halo and at least one owned moment
    if (p->m_offset + p->M < p->M_global && p->M < 2 + (p->m_offset > 0)) return GANDALF_ERR_INVALID;
  } else if (p->m_offset != 0) return GANDALF_ERR_INVALID;
  if (p->M > 0 && p->vA != 1.0) return GANDALF_ERR_UNSUPPORTED;
  if (p->hermite_exact && p->M > 0 && (p->closure != 0 || p->hermite_coeff != 0)) return GANDALF_ERR_UNSUPPORTED;   // symmetric coupling matrix only (Q30)
  // k_hermite_apply keeps 8 rows of the M x M propagator in the default 48 KB of dynamic shared memory (128 M bytes), and the
  // set-up diagonalises the coupling matrix on the host (O(M^3)) and stores Kz M^2 propagator entries: bounded here, not at the first step
  if (p->hermite_exact && p->M > GANDALF_HERMITE_EXACT_MAX_M) return GANDALF_ERR_UNSUPPORTED;
  if (cudaSetDevice(p->device) != cudaSuccess) { cudaGetLastError(); return GANDALF_ERR_CUDA; }

  gandalf_ctx* c = new (std::nothrow) gandalf_ctx();
  if (!c) return GANDALF_ERR_INVALID;
  c->p = *p;
  c->st = (cudaStream_t)p->stream;
  Dims& d = c->d;
  d.nx = p->nx; d.ny = p->ny; d.nz = p->nz;
  d.Msp = p->M; d.M = p->M * p->nspecies; d.F = 2 + d.M;     // d.M = number of moment FIELDS (species-major)
  const int moff = p->m_offset, Mg = p->M_global ? p->M_global : p->M;   // global numbering of the moments (Q31)
  const bool halo_lo = moff > 0, halo_hi = p->M_global != 0 && moff + p->M < Mg;
  d.own_lo = halo_lo ? 1 : 0; d.own_hi = d.M - (halo_hi ? 1 : 0);
  d.hx = p->nx / 2 + 1;
  d.hx3 = p->nx / 3; d.hy3 = p->ny / 3; d.hz3 = p->nz / 3;
  d.Kx = d.hx3 + 1; d.Ky = 2 * d.hy3 + 1; d.Kz = 2 * d.hz3 + 1;
  d.kx0 = 2.0 * kPi / p->Lx; d.ky0 = 2.0 * kPi / p->Ly; d.kz0 = 2.0 * kPi / p->Lz;
  d.inv_n = 1.0 / ((double)p->nx * p->ny * p->nz);
  {
    const double k2ret = std::pow(d.kx0 * d.hx3, 2) + std::pow(d.ky0 * d.hy3, 2);     // largest retained kperp^2
    int ex = 0;
    std::frexp(0.5 * k2ret, &ex);
    d.bscale = std::ldexp(1.0, ex - 1); d.inv_bscale = 1.0 / d.bscale;                // exact power of two
  }
  // Row strides.  E rows are padded to 128 B multiples (P3 then reads whole DRAM granules: 0.52 -> 0.50 ms at 4a); the same
  // padding on the hybrid arrays was measured SLOWER (P3 0.60, P4 1.05 ms: their lane-per-row stores then camp on few L2
  // slices), so H and Gh keep unpadded rows.
  d.Kxp = d.Kx; d.Kxe = (d.Kx + 7) / 8 * 8;
  d.PS = (size_t)d.Kz * d.Ky * d.Kx; d.PH = (size_t)d.nz * d.Ky * d.Kxp; d.PE = (size_t)d.nz * d.ny * d.Kxe;
  d.xl = xpass_lines_per_cta(d.nx);
  d.xlsh = 0; while ((1 << d.xlsh) < d.xl) ++d.xlsh;
  { const size_t nlb = ((size_t)d.ny * d.nz + d.xl - 1) / d.xl; d.PD = nlb * d.Kx * (size_t)d.xl; }
  PhysParams& ph = c->ph;
  ph.vA = p->vA; ph.eta = p->eta; ph.r = p->r; ph.eta_normalized = p->eta_normalized;
  ph.eta_z = p->eta_z; ph.r_z = p->r_z; ph.eta_g = p->eta_g;
  ph.k2max_perp = std::pow(kPi * p->nx / p->Lx, 2) + std::pow(kPi * p->ny / p->Ly, 2);
  ph.kz2max = std::pow(kPi * p->nz / p->Lz, 2);
  ph.if_variant = p->if_variant; ph.g_sign = p->g_sign;

  const int F = d.F, M = d.M;
  cudaError_t e = cudaSuccess;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  A(dalloc(&c->S0, F * d.PS)); A(dalloc(&c->S1, F * d.PS));
  A(dalloc(&c->tabz, (size_t)6 * d.Kz)); A(dalloc(&c->tabp, (size_t)2 * d.Ky * d.Kx));
  A(dalloc(&c->H, F * d.PH)); A(dalloc(&c->Gh, F * d.PH));
  A(dalloc(&c->D, (size_t)2 * (F + 2) * d.PD)); A(dalloc(&c->E, F * d.PE));
  A(dalloc(&c->cdn, (size_t)M + 1)); A(dalloc(&c->cup, (size_t)M + 1)); A(dalloc(&c->crate, (size_t)M + 1));
  A(dalloc(&c->collfac, (size_t)M + 1)); A(dalloc(&c->scal, (size_t)SC_COUNT));
  A(dalloc(&c->partial, (size_t)kEnergyBlocks * 5)); A(dalloc(&c->rec_scratch, (size_t)8));
  A(dalloc(&c->spec_col, (size_t)d.Ky * d.Kx)); A(dalloc(&c->maxbits, (size_t)1));
  c->hist_cap = 4096;
  A(dalloc(&c->hist, (size_t)c->hist_cap * 7));
  if (e == cudaSuccess) e = upload_twiddles(&c->twx, xpass_fft_plan_id(d.nx), c->st);
  if (e == cudaSuccess) e = upload_twiddles(&c->twy, d.ny, c->st);
  if (e == cudaSuccess) e = upload_twiddles(&c->twz, d.nz, c->st);
  if (e == cudaSuccess) e = launch_xpass(d, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, c->st, true);
  if (e == cudaSuccess) e = prepare_passes_zy(d.ny, d.nz);
  if (e == cudaSuccess && !build_tmaps(c)) e = cudaErrorUnknown;
  c->num_sms = 0;
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, p->device);
  if (c->num_sms <= 0) c->num_sms = 148;

  // Hermite coupling coefficients with the closure folded in (Q10, Q23, Q24)
  // The tables run over the moment FIELDS, species after species: dn = 0 at the first and up = 0 at the last moment of a
  // species, so neither the sliding window of the x-pass nor the streaming stencil of P4 couples the species (Q27).
  std::vector<double> dn(M + 1, 0.0), up(M + 1, 0.0), cr(M + 1, 0.0);
  const int Ms = d.Msp;
  for (int sp = 0; sp < p->nspecies; ++sp) {
    double* dns = dn.data() + sp * Ms; double* ups = up.data() + sp * Ms; double* crs = cr.data() + sp * Ms;
    for (int m = 0; m < Ms; ++m) { const int gm = moff + m; dns[m] = std::sqrt(gm / 2.0); ups[m] = std::sqrt((gm + 1) / 2.0); }
    if (p->hermite_coeff == 1) {
      for (int m = 0; m < Ms; ++m) { if (moff + m == 0) ups[m] = std::sqrt(2.0); if (moff + m == 1) ups[m] = std::sqrt(1.5); }
    }
    if (Ms > 0) {
      if (!halo_hi && p->closure == 1 && Ms >= 2) dns[Ms - 1] += ups[Ms - 1];   // g_M := g_{M-2}: the closure sits at the GLOBAL end
      ups[Ms - 1] = 0.0;                                            // g_M := 0 otherwise; a shard's upper halo has no neighbour here
      if (halo_lo) dns[0] = 0.0;                                    // the lower halo has none either (its own update is discarded)
    }
    for (int m = 0; m < Ms; ++m) crs[m] = p->nu_coll * std::pow((double)(moff + m) / (double)Mg, 2.0 * p->p);   // Eq. 19
  }
  // hermite_exact: T = V diag(lambda) V^T of the Msp x Msp coupling matrix (absorbing closure: symmetric tridiagonal)
  if (p->hermite_exact && Ms > 0) {
    std::vector<double> T((size_t)Ms * Ms, 0.0), V, lam;
    for (int m = 1; m < Ms; ++m) T[(size_t)m * Ms + m - 1] = T[(size_t)(m - 1) * Ms + m] = std::sqrt(m / 2.0);
    jacobi_eigh(Ms, T, V, lam);
    A(dalloc(&c->hxV, (size_t)Ms * Ms)); A(dalloc(&c->hxLam, (size_t)Ms));
    A(dalloc(&c->hxP, (size_t)p->nspecies * d.Kz * Ms * Ms));
    if (e == cudaSuccess) {
      A(cudaMemcpyAsync(c->hxV, V.data(), V.size() * sizeof(double), cudaMemcpyHostToDevice, c->st));
      A(cudaMemcpyAsync(c->hxLam, lam.data(), lam.size() * sizeof(double), cudaMemcpyHostToDevice, c->st));
      A(cudaStreamSynchronize(c->st));        // V, lam live on this stack frame
    }
  }
  // forcing pairs (Eq. 25; Q17): canonical members of each +-k pair in a fixed enumeration order
  std::vector<int> pr;
  double sumk2 = 0.0;
  if (p->force_eps > 0.0) {
    const int lo2 = p->force_nperp_min * p->force_nperp_min, hi2 = p->force_nperp_max * p->force_nperp_max;
    if (p->force_nperp_max > d.hx3 || p->force_nperp_max > d.hy3 || p->force_nz_max > d.hz3 || p->force_nperp_min < 0) {
      free_all(c); delete c; return GANDALF_ERR_INVALID;
    }
    for (int nz = -p->force_nz_max; nz <= p->force_nz_max; ++nz)
      for (int ny = -p->force_nperp_max; ny <= p->force_nperp_max; ++ny)
        for (int nx = 0; nx <= p->force_nperp_max; ++nx) {
          const int n2 = nx * nx + ny * ny;
          if (n2 < lo2 || n2 > hi2 || n2 == 0) continue;
          if (!((nx > 0) || (nx == 0 && ny > 0))) continue;
          pr.push_back(nx); pr.push_back(ny); pr.push_back(nz);
          const double kx = d.kx0 * nx, ky = d.ky0 * ny;
          sumk2 += 2.0 * (kx * kx + ky * ky);
        }
  }
  c->npairs = (int)(pr.size() / 3);
  c->force_amp = c->npairs ? std::sqrt(2.0 * p->force_eps / sumk2) : 0.0;
  if (c->npairs) A(dalloc(&c->pairs, pr.size()));
  if (e == cudaSuccess) {
    A(cudaMemcpyAsync(c->cdn, dn.data(), (M + 1) * sizeof(double), cudaMemcpyHostToDevice, c->st));
    A(cudaMemcpyAsync(c->cup, up.data(), (M + 1) * sizeof(double), cudaMemcpyHostToDevice, c->st));
    A(cudaMemcpyAsync(c->crate, cr.data(), (M + 1) * sizeof(double), cudaMemcpyHostToDevice, c->st));
    if (c->npairs) A(cudaMemcpyAsync(c->pairs, pr.data(), pr.size() * sizeof(int), cudaMemcpyHostToDevice, c->st));
    A(cudaMemsetAsync(c->S0, 0, F * d.PS * sizeof(cd), c->st));
    A(cudaMemsetAsync(c->H, 0, F * d.PH * sizeof(cd), c->st));
    A(cudaMemsetAsync(c->scal, 0, SC_COUNT * sizeof(double), c->st));
    A(cudaStreamSynchronize(c->st));
  }
  if (e != cudaSuccess) { cudaGetLastError(); free_all(c); delete c; return GANDALF_ERR_CUDA; }
  c->step = 0; c->hist_base = 0; c->H_valid = true; c->launches = 0; c->timing = false;
  c->graph_mode = 1; c->gexec = nullptr; c->g_launches = 0; c->graph_replays = 0; c->g_last_dt = -1.0;
  c->stage_pending = false; c->need_h = true;
  c->h2d_bytes = 0; c->d2h_bytes = 0;
  for (int i = 0; i < KC_N; ++i) { c->t_ms[i] = 0; c->t_n[i] = 0; }
  *out = c;
  return GANDALF_OK;
}

int gandalf_destroy(gandalf_ctx* c) {
  if (!c) return GANDALF_ERR_INVALID;
  cudaSetDevice(c->p.device);
  cudaStreamSynchronize(c->st);
  free_all(c);
  delete c;
  return GANDALF_OK;
}

const char* gandalf_last_error(const gandalf_ctx* c) { return c ? c->err.c_str() : "null context"; }
long long gandalf_launch_count(const gandalf_ctx* c) { return c ? c->launches : 0; }

}  // extern "C"

// ---- internals of the step driver ----------------------------------------------------------------------------
static int ensure_io(gandalf_ctx* c, size_t bytes) {
  if (c->io_bytes >= bytes) return GANDALF_OK;
  if (c->io) { GD_CUDA(c, cudaStreamSynchronize(c->st)); cudaFree(c->io); c->io = nullptr; c->io_bytes = 0; }
  GD_CUDA(c, cudaMalloc((void**)&c->io, bytes));
  c->io_bytes = bytes;
  return GANDALF_OK;
}

// Host -> device copy of `nfields` boundary-layout fields.  gandalf_set_state reads only the RETAINED modes of its input (Eq. 20:
// kx <= nx/3 and the two retained ranges of ky and of kz: 30 % of the half-plane array), so for large arrays only those
// sub-blocks cross PCIe: four pitched 3-D copies per field into the same layout on the device (the rest of the staging buffer is
// never read).  Small arrays go in one piece (fewer calls).
static int copy_boundary_h2d(gandalf_ctx* c, cd* dst, const cd* src, int nfields) {
  const Dims& d = c->d;
  const size_t hp = (size_t)d.nz * d.ny * d.hx;
  if ((size_t)nfields * hp * sizeof(cd) < ((size_t)64 << 20)) {
    GD_CUDA(c, cudaMemcpyAsync(dst, src, (size_t)nfields * hp * sizeof(cd), cudaMemcpyHostToDevice, c->st));
    c->h2d_bytes += (long long)((size_t)nfields * hp * sizeof(cd));
    return GANDALF_OK;
  }
  const int zr[2][2] = {{0, d.hz3 + 1}, {d.nz - d.hz3, d.hz3}}, yr[2][2] = {{0, d.hy3 + 1}, {d.ny - d.hy3, d.hy3}};   // {start, count}
  for (int f = 0; f < nfields; ++f)
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b) {
        if (zr[a][1] <= 0 || yr[b][1] <= 0) continue;
        cudaMemcpy3DParms p3;
        std::memset(&p3, 0, sizeof(p3));
        p3.srcPtr = make_cudaPitchedPtr(const_cast<cd*>(src), (size_t)d.hx * sizeof(cd), (size_t)d.hx * sizeof(cd), (size_t)d.ny);
        p3.dstPtr = make_cudaPitchedPtr(dst, (size_t)d.hx * sizeof(cd), (size_t)d.hx * sizeof(cd), (size_t)d.ny);
        p3.srcPos = make_cudaPos(0, (size_t)yr[b][0], (size_t)f * d.nz + zr[a][0]);
        p3.dstPos = p3.srcPos;
        p3.extent = make_cudaExtent((size_t)d.Kx * sizeof(cd), (size_t)yr[b][1], (size_t)zr[a][1]);
        p3.kind = cudaMemcpyHostToDevice;
        GD_CUDA(c, cudaMemcpy3DAsync(&p3, c->st));
        c->h2d_bytes += (long long)((size_t)d.Kx * sizeof(cd) * yr[b][1] * zr[a][1]);
      }
  return GANDALF_OK;
}

// hybrid copy of S0 (z in real space) -- the form the RHS pipeline consumes
static int make_hybrid(gandalf_ctx* c, const cd* S) {
  GD_CUDA(c, timed(c, KC_ZINV, 1, [&] { return launch_zfft(c->d, S, c->H, c->twz, c->d.F, c->st); }));
  return GANDALF_OK;
}

// bracket terms of the state whose hybrid copy is in H  ->  Gh (hybrid: z real, (kx,ky) spectral and masked): N+-, R_m
static int rhs_pipeline(gandalf_ctx* c, bool want_cfl) {
  const Dims& d = c->d;
  if (!c->p.nonlinear && !want_cfl) return GANDALF_OK;
  // nonlinear == 0 with the CFL dt: Eq. 16 still needs max|grad Phi|, so P1/P2 run and the brackets are discarded
  if (want_cfl) GD_CUDA(c, timed(c, -1, 1, [&] { return launch_zero_u64(c->maxbits, c->st); }));
  GD_CUDA(c, timed(c, KC_YINV, d.M > 0 ? 2 : 1, [&] { return launch_yinv(d, c->H, c->D, c->twy, c->num_sms, c->st); }));
  GD_CUDA(c, timed(c, KC_XPASS, 1, [&] {
    return launch_xpass(d, c->D, c->E, c->twx, c->cdn, c->cup, want_cfl ? c->maxbits : nullptr, c->num_sms, c->st, false);
  }));
  if (!c->p.nonlinear) return GANDALF_OK;
  GD_CUDA(c, timed(c, KC_YFWD, d.M > 0 ? 2 : 1, [&] { return launch_yfwd(d, c->E, c->Gh, c->twy, c->num_sms, c->st); }));
  return GANDALF_OK;
}

// P4: forward z transform of Gh + stage update (mode 0/1/2) + inverse z transform into the hybrid copy (if wanted)
static int stage_update(gandalf_ctx* c, int mode, const cd* Wn, const cd* Ws, cd* Wout, bool want_hybrid, bool exact = false) {
  GD_CUDA(c, timed(c, KC_ZSTEP, 1, [&] {
    return launch_zstep(c->d, c->tm, mode, exact, c->p.if_variant, c->p.g_sign, c->p.nonlinear != 0, Wn, Ws, Wout,
                        want_hybrid, c->scal, c->cdn, c->cup, c->collfac, c->tabz, c->tabp, c->twz, c->st);
  }));
  return GANDALF_OK;
}

static int ensure_hist(gandalf_ctx* c, long long need) {   // need: records, counted from hist_base
  if (need <= c->hist_cap) return GANDALF_OK;
  long long cap = c->hist_cap;
  while (cap < need) cap *= 2;
  double* nh = nullptr;
  GD_CUDA(c, cudaMalloc((void**)&nh, (size_t)cap * 7 * sizeof(double)));
  GD_CUDA(c, cudaMemcpyAsync(nh, c->hist, (size_t)(c->step - c->hist_base) * 7 * sizeof(double), cudaMemcpyDeviceToDevice, c->st));
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  cudaFree(c->hist);
  c->hist = nh; c->hist_cap = cap;
  return GANDALF_OK;
}

// sticky device-side error flag (Eq. 16 without a flow and without dt_max); call after the stream is synchronised
static int check_device_flags(gandalf_ctx* c) {
  double s[SC_COUNT];
  GD_CUDA(c, cudaMemcpyAsync(s, c->scal, sizeof(s), cudaMemcpyDeviceToHost, c->st));
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  if (s[SC_ERR] != 0.0) GD_FAIL(c, GANDALF_ERR_CFL, "CFL step (Eq. 16): max|grad Phi| is zero and dt_max is not set; the state was left untouched");
  return GANDALF_OK;
}

extern "C" {

int gandalf_state_raw_doubles(const gandalf_ctx* c, long long* n) {
  if (!c || !n) return GANDALF_ERR_INVALID;
  *n = 2LL * (long long)c->d.F * (long long)c->d.PS;
  return GANDALF_OK;
}

int gandalf_get_state_raw(gandalf_ctx* c, double* out, int on_device) {
  if (!c) return GANDALF_ERR_INVALID;
  if (!out) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_get_state_raw: NULL array");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  const size_t bytes = (size_t)c->d.F * c->d.PS * sizeof(cd);
  GD_CUDA(c, cudaMemcpyAsync(out, c->S0, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->st));
  if (!on_device) { c->d2h_bytes += (long long)bytes; GD_CUDA(c, cudaStreamSynchronize(c->st)); }
  return GANDALF_OK;
}

int gandalf_set_state_raw(gandalf_ctx* c, const double* in, int on_device) {
  if (!c) return GANDALF_ERR_INVALID;
  if (!in) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_set_state_raw: NULL array");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  const size_t bytes = (size_t)c->d.F * c->d.PS * sizeof(cd);
  GD_CUDA(c, cudaMemcpyAsync(c->S0, in, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->st));
  if (!on_device) c->h2d_bytes += (long long)bytes;
  GD_CUDA(c, cudaMemsetAsync(c->scal + SC_ERR, 0, sizeof(double), c->st));   // a new state: the sticky Eq. 16 flag of the old one goes
  c->stage_pending = false;
  int rc = make_hybrid(c, c->S0);
  if (rc) return rc;
  c->H_valid = true;
  if (!on_device) GD_CUDA(c, cudaStreamSynchronize(c->st));
  return GANDALF_OK;
}

int gandalf_set_time(gandalf_ctx* c, double t, long long step) {
  if (!c) return GANDALF_ERR_INVALID;
  if (step < 0 || step > (1LL << 52) || !std::isfinite(t)) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_set_time: bad time or step");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  const double dstep = (double)step;
  GD_CUDA(c, cudaMemcpyAsync(c->scal + SC_T, &t, sizeof(double), cudaMemcpyHostToDevice, c->st));
  GD_CUDA(c, cudaMemcpyAsync(c->scal + SC_STEP, &dstep, sizeof(double), cudaMemcpyHostToDevice, c->st));
  GD_CUDA(c, cudaMemsetAsync(c->scal + SC_ERR, 0, sizeof(double), c->st));   // a resumed run starts without the sticky Eq. 16 flag
  GD_CUDA(c, cudaStreamSynchronize(c->st));     // t, dstep live on this stack frame
  c->step = step; c->hist_base = step;          // the history restarts at the resumed step
  return GANDALF_OK;
}

int gandalf_set_state(gandalf_ctx* c, const double* zeta_hat, const double* g_hat, int on_device) {
  if (!c) return GANDALF_ERR_INVALID;
  if (!zeta_hat || (c->d.M > 0 && !g_hat)) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_set_state: NULL array");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  const Dims& d = c->d;
  const size_t hp = (size_t)d.nz * d.ny * d.hx;
  const cd* zin = reinterpret_cast<const cd*>(zeta_hat);
  const cd* gin = reinterpret_cast<const cd*>(g_hat);
  if (!on_device) {
    int rc = ensure_io(c, (size_t)d.F * hp * sizeof(cd));
    if (rc) return rc;
    rc = copy_boundary_h2d(c, c->io, zin, 2);
    if (rc) return rc;
    if (d.M > 0) { rc = copy_boundary_h2d(c, c->io + 2 * hp, gin, d.M); if (rc) return rc; }
    zin = c->io; gin = c->io + 2 * hp;
  }
  GD_CUDA(c, timed(c, -1, 1, [&] { return launch_pack(d, zin, c->S0, 2, 2, c->st); }));
  if (d.M > 0) GD_CUDA(c, timed(c, -1, 1, [&] { return launch_pack(d, gin, c->S0 + 2 * d.PS, d.M, 0, c->st); }));
  GD_CUDA(c, cudaMemsetAsync(c->scal, 0, SC_COUNT * sizeof(double), c->st));
  c->step = 0; c->hist_base = 0; c->stage_pending = false;
  int rc = make_hybrid(c, c->S0);
  if (rc) return rc;
  c->H_valid = true;
  if (!on_device) GD_CUDA(c, cudaStreamSynchronize(c->st));
  return GANDALF_OK;
}

static int export_fields(gandalf_ctx* c, const cd* S, double* a2, double* aM, int nzeta, int on_device) {
  const Dims& d = c->d;
  const size_t hp = (size_t)d.nz * d.ny * d.hx;
  cd* o2 = reinterpret_cast<cd*>(a2);
  cd* oM = reinterpret_cast<cd*>(aM);
  if (!on_device) {
    int rc = ensure_io(c, (size_t)d.F * hp * sizeof(cd));
    if (rc) return rc;
    o2 = c->io; oM = c->io + 2 * hp;
  }
  GD_CUDA(c, timed(c, -1, 1, [&] { return launch_unpack(d, S, o2, 2, nzeta, c->st); }));
  if (d.M > 0) GD_CUDA(c, timed(c, -1, 1, [&] { return launch_unpack(d, S + 2 * d.PS, oM, d.M, 0, c->st); }));
  if (!on_device) {
    GD_CUDA(c, cudaMemcpyAsync(a2, o2, 2 * hp * sizeof(cd), cudaMemcpyDeviceToHost, c->st));
    if (d.M > 0) GD_CUDA(c, cudaMemcpyAsync(aM, oM, (size_t)d.M * hp * sizeof(cd), cudaMemcpyDeviceToHost, c->st));
    c->d2h_bytes += (long long)((size_t)d.F * hp * sizeof(cd));
    GD_CUDA(c, cudaStreamSynchronize(c->st));
  }
  return GANDALF_OK;
}

int gandalf_get_state(gandalf_ctx* c, double* zeta_hat, double* g_hat, int on_device) {
  if (!c) return GANDALF_ERR_INVALID;
  if (!zeta_hat || (c->d.M > 0 && !g_hat)) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_get_state: NULL array");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  return export_fields(c, c->S0, zeta_hat, g_hat, 2, on_device);
}

int gandalf_rhs(gandalf_ctx* c, double* dw_hat, double* dg_hat, int on_device) {
  if (!c) return GANDALF_ERR_INVALID;
  if (!dw_hat || (c->d.M > 0 && !dg_hat)) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_rhs: NULL array");
  if (c->stage_pending) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_rhs: a step is half done (the stage state would be overwritten)");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  int rc;
  if (!c->H_valid) { rc = make_hybrid(c, c->S0); if (rc) return rc; c->H_valid = true; }
  rc = rhs_pipeline(c, false);
  if (rc) return rc;
  rc = stage_update(c, 0, c->S0, c->S0, c->S1, false);
  if (rc) return rc;
  return export_fields(c, c->S1, dw_hat, dg_hat, 0, on_device);
}

}  // extern "C"

// One step = two stages (a moment-sharded run refreshes its halo moments in between, Q31).
// Stage 0 (Alg. 2 l.2-6): RHS at t_n (its x-pass also yields max|grad Phi| for Eq. 16), dt, tables, half-step predictor.
static int step_stage0(gandalf_ctx* c, double dt) {
  const Dims& d = c->d;
  const bool adaptive = !(dt > 0.0);
  const double cfl_dxy = c->p.cfl * std::fmin(c->p.Lx / d.nx, c->p.Ly / d.ny);
  const bool exact = c->p.hermite_exact && d.M > 0;
  int rc = rhs_pipeline(c, adaptive);
  if (rc) return rc;
  GD_CUDA(c, timed(c, -1, 1, [&] {
    return launch_prepare_dt(adaptive ? 0.0 : dt, cfl_dxy, c->p.dt_max, c->maxbits, c->scal, c->crate, c->collfac, d.M, c->st);
  }));
  GD_CUDA(c, timed(c, -1, 1, [&] { return launch_tables(d, c->ph, c->scal, c->tabz, c->tabp, c->st); }));
  if (!exact) {
    rc = stage_update(c, 1, c->S0, c->S0, c->S1, c->p.nonlinear);
    if (rc) return rc;
  } else {
    // hermite_exact (Q30): with P = P(dt/2) = exp(s i kz (I - T) dt/2) per kz,
    //   g_{n+1/2} = P (g_n + dt/2 R_n),   g_{n+1} = P (P g_n + dt R_{n+1/2}),   R = the bracket terms of Eq. 6;
    // w+- exactly as above.  D is free between two RHS pipelines and serves as scratch for the propagated half-step state.
    GD_CUDA(c, timed(c, -1, 1, [&] { return launch_hermite_propagator(d, c->p.g_sign, 0.5, c->scal, c->hxV, c->hxLam, c->hxP, c->st); }));
    rc = stage_update(c, 1, c->S0, c->S0, c->S1, c->p.nonlinear, true);          // S1 = w_{n+1/2} | g_n + dt/2 R_n ; H(w+-)
    if (rc) return rc;
    GD_CUDA(c, timed(c, -1, 1, [&] { return launch_hermite_apply(d, c->S1, c->D, c->hxP, 0, c->collfac, c->tabz, c->tabp, c->st); }));
    if (c->p.nonlinear) GD_CUDA(c, timed(c, KC_ZINV, 1, [&] { return launch_zfft(d, c->D + 2 * d.PS, c->H + 2 * d.PH, c->twz, d.M, c->st); }));
  }
  c->need_h = c->p.nonlinear || adaptive;
  c->stage_pending = true;
  return GANDALF_OK;
}
// Stage 1 (Alg. 2 l.7-14): midpoint RHS, full-step corrector + dissipation (in place on S0: each mode reads only its own S0
// entry), forcing, energy record.
static int step_stage1(gandalf_ctx* c) {
  const Dims& d = c->d;
  const bool exact = c->p.hermite_exact && d.M > 0;
  const bool need_h = c->need_h;
  int rc = rhs_pipeline(c, false);
  if (rc) return rc;
  if (!exact) {
    rc = stage_update(c, 2, c->S0, c->S1, c->S0, need_h);
    if (rc) return rc;
  } else {
    GD_CUDA(c, timed(c, -1, 1, [&] { return launch_hermite_apply(d, c->S0, c->S1, c->hxP, 0, c->collfac, c->tabz, c->tabp, c->st); }));   // S1(g) = P g_n
    rc = stage_update(c, 2, c->S0, c->S1, c->S0, need_h, true);                   // S0(w) = w_{n+1};  S1(g) += dt R_{n+1/2}
    if (rc) return rc;
    GD_CUDA(c, timed(c, -1, 1, [&] { return launch_hermite_apply(d, c->S1, c->S0, c->hxP, 1, c->collfac, c->tabz, c->tabp, c->st); }));   // S0(g) = diss . P S1(g)
    if (need_h) GD_CUDA(c, timed(c, KC_ZINV, 1, [&] { return launch_zfft(d, c->S0 + 2 * d.PS, c->H + 2 * d.PH, c->twz, d.M, c->st); }));
  }
  if (c->npairs) {
    GD_CUDA(c, timed(c, -1, 1, [&] {
      return launch_forcing(d, c->S0, c->pairs, c->npairs, c->force_amp, c->p.seed, c->scal, c->st);
    }));
    // the forcing touches w+- only: refresh the hybrid copy of those two fields
    if (need_h) GD_CUDA(c, timed(c, KC_ZINV, 1, [&] { return launch_zfft(d, c->S0, c->H, c->twz, 2, c->st); }));
  }
  if (c->p.force_g_amp > 0.0 && c->p.m_offset == 0) {     // g_0 lives on the shard with m_offset = 0
    GD_CUDA(c, timed(c, -1, 1, [&] {
      return launch_forcing_g(d, c->S0, c->p.force_g_nz, c->p.force_g_amp, c->p.seed, c->scal, c->st);
    }));
    // the forcing touches g_0 only: refresh the hybrid copy of that field
    if (need_h) GD_CUDA(c, timed(c, KC_ZINV, 1, [&] { return launch_zfft(d, c->S0 + 2 * d.PS, c->H + 2 * d.PH, c->twz, 1, c->st); }));
  }
  GD_CUDA(c, timed(c, -1, 2, [&] {
    return launch_energy(d, c->S0, c->partial, kEnergyBlocks, c->hist, c->hist_base, c->scal, 1, c->st);   // slot (step - hist_base), step on the device
  }));
  c->step += 1;
  c->H_valid = need_h;
  c->stage_pending = false;
  return GANDALF_OK;
}

extern "C" {

int gandalf_step(gandalf_ctx* c, double dt, int nsteps) {
  if (!c) return GANDALF_ERR_INVALID;
  if (nsteps < 0 || !std::isfinite(dt)) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_step: bad dt or nsteps");
  if (c->stage_pending) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_step: a step is half done (gandalf_step_stage(.., 0) without stage 1)");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  int rc = ensure_hist(c, c->step - c->hist_base + nsteps);
  if (rc) return rc;
  if (!c->H_valid) { rc = make_hybrid(c, c->S0); if (rc) return rc; c->H_valid = true; }
  int done = 0;
  // Graph path: one step is the same launch sequence with the same arguments every time (dt and the step number are read from
  // device memory), so it is captured once and replayed.  Not with per-kernel event timing, not on the legacy default stream
  // (capture is not allowed there), not inside somebody else's capture.
  if (c->graph_mode && !c->timing && c->st != nullptr && nsteps > 0) {
    const double key_dt = dt > 0.0 ? dt : 0.0;
    const bool cached = c->gexec && c->g_dt == key_dt && c->g_hist == c->hist && c->g_hist_base == c->hist_base;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    const bool want = !cached && (nsteps >= 2 || c->g_last_dt == key_dt) && cudaStreamIsCapturing(c->st, &cs) == cudaSuccess &&
                      cs == cudaStreamCaptureStatusNone;
    if (want && c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }   // before the capture begins (deferred until its replays end)
    if (want && cudaStreamBeginCapture(c->st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      const long long l0 = c->launches, s0 = c->step;
      int rcc = step_stage0(c, dt);
      if (!rcc) rcc = step_stage1(c);
      cudaGraph_t g = nullptr;
      cudaError_t e = cudaStreamEndCapture(c->st, &g);
      const long long per_step = c->launches - l0;
      c->launches = l0; c->step = s0; c->stage_pending = false; c->H_valid = true;   // nothing ran: the capture only recorded
      if (!rcc && e == cudaSuccess && g && cudaGraphInstantiate(&c->gexec, g, 0) == cudaSuccess) {
        c->g_dt = key_dt; c->g_hist = c->hist; c->g_hist_base = c->hist_base; c->g_launches = per_step;
      } else {
        c->gexec = nullptr;
        cudaGetLastError();                        // a failed capture is not an error of the step: plain launches follow
      }
      if (g) cudaGraphDestroy(g);
    }
    if (c->gexec && c->g_dt == key_dt && c->g_hist == c->hist && c->g_hist_base == c->hist_base) {
      for (; done < nsteps; ++done) {
        GD_CUDA(c, cudaGraphLaunch(c->gexec, c->st));
        c->step += 1; c->launches += c->g_launches; c->graph_replays += 1;
      }
      c->H_valid = c->p.nonlinear || !(dt > 0.0);   // what step_stage1 leaves (need_h)
    }
    c->g_last_dt = key_dt;                          // a second call with the same dt is worth a capture even with nsteps = 1
  }
  for (int i = done; i < nsteps; ++i) {
    rc = step_stage0(c, dt);
    if (rc) return rc;
    rc = step_stage1(c);
    if (rc) return rc;
  }
  return GANDALF_OK;
}

int gandalf_graph_mode(gandalf_ctx* c, int enable, long long* replays) {
  if (!c) return GANDALF_ERR_INVALID;
  if (enable == 0 || enable == 1) c->graph_mode = enable;
  else if (enable != -1) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_graph_mode: enable must be 0, 1 or -1 (query)");
  if (replays) *replays = c->graph_replays;
  return GANDALF_OK;
}

int gandalf_step_stage(gandalf_ctx* c, double dt, int stage) {
  if (!c) return GANDALF_ERR_INVALID;
  if ((stage != 0 && stage != 1) || !std::isfinite(dt)) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_step_stage: bad dt or stage");
  if ((stage == 1) != c->stage_pending) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_step_stage: stages must alternate 0, 1");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  if (stage == 1) return step_stage1(c);
  int rc = ensure_hist(c, c->step - c->hist_base + 1);
  if (rc) return rc;
  if (!c->H_valid) { rc = make_hybrid(c, c->S0); if (rc) return rc; c->H_valid = true; }
  return step_stage0(c, dt);
}

int gandalf_field_ptr(gandalf_ctx* c, int state, int field, void** device_ptr, long long* ncomplex) {
  if (!c || !device_ptr) return GANDALF_ERR_INVALID;
  if ((state != 0 && state != 1) || field < 0 || field >= c->d.F) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_field_ptr: bad state or field");
  *device_ptr = (state == 0 ? c->S0 : c->S1) + (size_t)field * c->d.PS;
  if (ncomplex) *ncomplex = (long long)c->d.PS;
  return GANDALF_OK;
}

int gandalf_halo_refresh(gandalf_ctx* c, int state) {
  if (!c) return GANDALF_ERR_INVALID;
  if (state != 0 && state != 1) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_halo_refresh: bad state");
  GD_CUDA(c, cudaSetDevice(c->p.device));
  const Dims& d = c->d;
  const cd* S = state == 0 ? c->S0 : c->S1;
  if (d.own_lo > 0) GD_CUDA(c, timed(c, KC_ZINV, 1, [&] { return launch_zfft(d, S + 2 * d.PS, c->H + 2 * d.PH, c->twz, 1, c->st); }));
  if (d.own_hi < d.M) {
    const size_t f = (size_t)(2 + d.M - 1);
    GD_CUDA(c, timed(c, KC_ZINV, 1, [&] { return launch_zfft(d, S + f * d.PS, c->H + f * d.PH, c->twz, 1, c->st); }));
  }
  return GANDALF_OK;
}

int gandalf_energy(gandalf_ctx* c, double out[6]) {
  if (!c || !out) return GANDALF_ERR_INVALID;
  GD_CUDA(c, cudaSetDevice(c->p.device));
  GD_CUDA(c, timed(c, -1, 2, [&] { return launch_energy(c->d, c->S0, c->partial, kEnergyBlocks, c->rec_scratch, 0, c->scal, 0, c->st); }));
  double rec[7];
  GD_CUDA(c, cudaMemcpyAsync(rec, c->rec_scratch, sizeof(rec), cudaMemcpyDeviceToHost, c->st));
  c->d2h_bytes += (long long)sizeof(rec);
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  bool ok = true;
  for (int i = 0; i < 6; ++i) { out[i] = rec[i + 1]; ok = ok && std::isfinite(out[i]); }
  if (!ok) GD_FAIL(c, GANDALF_ERR_NONFINITE, "non-finite energy");
  return check_device_flags(c);
}

int gandalf_kperp_spectrum(gandalf_ctx* c, int nbins, int literal_eq26, double* out) {
  if (!c || !out || nbins <= 0 || nbins > 65535) return GANDALF_ERR_INVALID;
  GD_CUDA(c, cudaSetDevice(c->p.device));
  if (nbins > c->spec_cap) {
    if (c->spec_out) { GD_CUDA(c, cudaStreamSynchronize(c->st)); cudaFree(c->spec_out); c->spec_out = nullptr; c->spec_cap = 0; }
    GD_CUDA(c, cudaMalloc((void**)&c->spec_out, (size_t)nbins * sizeof(double)));
    c->spec_cap = nbins;
  }
  const double dk = 2.0 * kPi / std::fmax(c->p.Lx, c->p.Ly);
  GD_CUDA(c, timed(c, -1, 2, [&] { return launch_spectrum(c->d, c->S0, c->spec_col, nbins, literal_eq26, dk, c->spec_out, c->st); }));
  GD_CUDA(c, cudaMemcpyAsync(out, c->spec_out, (size_t)nbins * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  return GANDALF_OK;
}

static int ensure_spec(gandalf_ctx* c, int n) {
  if (n <= c->spec_cap) return GANDALF_OK;
  if (c->spec_out) { GD_CUDA(c, cudaStreamSynchronize(c->st)); cudaFree(c->spec_out); c->spec_out = nullptr; c->spec_cap = 0; }
  GD_CUDA(c, cudaMalloc((void**)&c->spec_out, (size_t)n * sizeof(double)));
  c->spec_cap = n;
  return GANDALF_OK;
}

int gandalf_hermite_spectrum(gandalf_ctx* c, double* out) {
  if (!c || (c->d.M > 0 && !out)) return GANDALF_ERR_INVALID;
  if (c->d.M == 0) return GANDALF_OK;
  GD_CUDA(c, cudaSetDevice(c->p.device));
  int rc = ensure_spec(c, c->d.M);
  if (rc) return rc;
  GD_CUDA(c, timed(c, -1, 1, [&] { return launch_hermite_spectrum(c->d, c->S0, c->spec_out, c->st); }));
  GD_CUDA(c, cudaMemcpyAsync(out, c->spec_out, (size_t)c->d.M * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  return GANDALF_OK;
}

int gandalf_truncation_ratio(gandalf_ctx* c, double* out) {
  if (!c || !out) return GANDALF_ERR_INVALID;
  if (c->d.M < 1) GD_FAIL(c, GANDALF_ERR_INVALID, "gandalf_truncation_ratio: no moments");
  if (c->p.M_global != 0) GD_FAIL(c, GANDALF_ERR_UNSUPPORTED, "gandalf_truncation_ratio: moment shard");
  std::vector<double> cm((size_t)c->d.M);
  int rc = gandalf_hermite_spectrum(c, cm.data());
  if (rc) return rc;
  double e[6];
  rc = gandalf_energy(c, e);
  if (rc) return rc;
  double eM = 0.0;
  for (int sp = 0; sp < c->p.nspecies; ++sp) eM += 0.5 * cm[(size_t)sp * c->d.Msp + c->d.Msp - 1];
  *out = eM / (e[0] + e[5]);
  return GANDALF_OK;
}

int gandalf_kpar_spectrum(gandalf_ctx* c, int nbins, double* out) {
  if (!c || !out || nbins <= 0 || nbins > 65535) return GANDALF_ERR_INVALID;
  GD_CUDA(c, cudaSetDevice(c->p.device));
  int rc = ensure_spec(c, nbins);
  if (rc) return rc;
  // spec_col (Ky*Kx doubles) has room for the Kz per-plane sums: Kz <= Ky*Kx because nx, ny >= 8 ... checked here
  if ((size_t)c->d.Kz > (size_t)c->d.Ky * c->d.Kx) GD_FAIL(c, GANDALF_ERR_UNSUPPORTED, "gandalf_kpar_spectrum: nz too large for this grid");
  GD_CUDA(c, timed(c, -1, 2, [&] { return launch_kpar_spectrum(c->d, c->S0, c->spec_col, nbins, c->spec_out, c->st); }));
  GD_CUDA(c, cudaMemcpyAsync(out, c->spec_out, (size_t)nbins * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  return GANDALF_OK;
}

int gandalf_energy_history(gandalf_ctx* c, int max_records, double* t_and_E, int* n) {
  if (!c || !n || max_records < 0 || (max_records > 0 && !t_and_E)) return GANDALF_ERR_INVALID;
  GD_CUDA(c, cudaSetDevice(c->p.device));
  const long long have = c->step - c->hist_base;
  const long long k = have < max_records ? have : max_records;
  if (k > 0) GD_CUDA(c, cudaMemcpyAsync(t_and_E, c->hist, (size_t)k * 7 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  c->d2h_bytes += (long long)(k * 7 * sizeof(double));
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  *n = (int)k;
  for (long long i = 0; i < k * 7; ++i)
    if (!std::isfinite(t_and_E[i])) GD_FAIL(c, GANDALF_ERR_NONFINITE, "non-finite value in the energy history");
  return check_device_flags(c);
}

int gandalf_get_time(gandalf_ctx* c, double* t, long long* step, double* last_dt) {
  if (!c) return GANDALF_ERR_INVALID;
  GD_CUDA(c, cudaSetDevice(c->p.device));
  double s[SC_COUNT];
  GD_CUDA(c, cudaMemcpyAsync(s, c->scal, sizeof(s), cudaMemcpyDeviceToHost, c->st));
  GD_CUDA(c, cudaStreamSynchronize(c->st));
  if (t) *t = s[SC_T];
  if (step) *step = c->step;
  if (last_dt) *last_dt = s[SC_LASTDT];
  if (!std::isfinite(s[SC_T])) GD_FAIL(c, GANDALF_ERR_NONFINITE, "non-finite time (CFL dt)");
  if (s[SC_ERR] != 0.0) GD_FAIL(c, GANDALF_ERR_CFL, "CFL step (Eq. 16): max|grad Phi| is zero and dt_max is not set; the state was left untouched");
  return GANDALF_OK;
}

int gandalf_transfer_bytes(const gandalf_ctx* c, long long* h2d, long long* d2h) {
  if (!c) return GANDALF_ERR_INVALID;
  if (h2d) *h2d = c->h2d_bytes;
  if (d2h) *d2h = c->d2h_bytes;
  return GANDALF_OK;
}

int gandalf_kernel_timing(gandalf_ctx* c, int enable) {
  if (!c) return GANDALF_ERR_INVALID;
  cudaSetDevice(c->p.device);
  drain_events(c);
  c->timing = enable != 0;
  for (int i = 0; i < KC_N; ++i) { c->t_ms[i] = 0; c->t_n[i] = 0; }
  return GANDALF_OK;
}

int gandalf_kernel_time_ms(gandalf_ctx* c, int which, double* avg_ms, long long* launches) {
  if (!c || which < 0 || which >= KC_N) return GANDALF_ERR_INVALID;
  cudaSetDevice(c->p.device);
  drain_events(c);
  if (avg_ms) *avg_ms = c->t_n[which] ? c->t_ms[which] / (double)c->t_n[which] : 0.0;
  if (launches) *launches = c->t_n[which];
  return GANDALF_OK;
}

}  // extern "C"
