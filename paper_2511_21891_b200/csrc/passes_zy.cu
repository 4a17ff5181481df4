// passes_zy.cu -- the z transforms and the y passes of the RHS pipeline.
//
//   k_zfft      : S[f][cz][cy][cx] -> H[f][z][cy][cx]  inverse c2c along z, zero-padded; only after
//                 set_state and after a forcing increment
//   k_zstep     : P4.  Gh -> S', H': forward z transform + stage update + inverse z transform in one kernel
//   k_yinv      : P1.  H -> D: for every source field the two arrays U = kx f + df/dy, V = df/dy - kx f (Eq. 10,
//                 PAPER.md:134; for w+- also of xi = -w/kperp^2), inverse c2c along y
//   k_yfwd(_pair): P3.  E -> Gh: forward c2c along y, ky part of Eq. 20; the Elsasser pair is assembled as
//                 N+- = -1/2 A -+ 1/2 kperp^2 B  (Eq. 1 with Eq. 11)
// Every FFT is the lane-group transform of fft.cuh: T lanes of one warp per column, data in registers, one
// shared-memory exchange per stage boundary.  The y passes stage their input tiles with per-row bulk async copies (TMA engine,
// mbarrier completion) so that global memory sees whole 256-byte row segments; P4 moves its tiles with tensor-map TMA
// (cp.async.bulk.tensor, one instruction per 8-column sub-tile, 128-byte swizzle; common.cuh); see DESIGN.md section 5.
#include <vector>
#include "common.cuh"

template <int NZ>
__global__ void __launch_bounds__(GD_Z_THREADS) k_zfft(Dims d, const cd* __restrict__ in, cd* __restrict__ out,
                                                       const cd* __restrict__ tw, int ncols) {
  using G = FftGeom<NZ>;
  constexpr int T = G::T, E = G::E;
  extern __shared__ cd smem[];
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  const int gid = blockIdx.x * (GD_Z_THREADS / T) + grp;
  cd* buf = smem + FftTw<NZ>::COUNT + (size_t)grp * (G::BUF + 1);
  fft_load_table<NZ>(smem, tw);
  const cd* tws = smem;
  const bool active = gid < ncols;
  const int plane = d.Ky * d.Kx;
  const int f = active ? gid / plane : 0, rem = active ? gid % plane : 0;
  const int planeH = d.Ky * d.Kxp, remH = (rem / d.Kx) * d.Kxp + rem % d.Kx;       // hybrid rows are padded to Kxp
  cd v[E];
  const cd* src = in + (size_t)f * d.PS + rem;
#pragma unroll
  for (int q = 0; q < E; ++q) {
    const int cz = fft2c(t + T * q, NZ, d.hz3, d.Kz);
    v[q] = (active && cz >= 0) ? ldg_cd(src + (size_t)cz * plane) : cmake(0.0, 0.0);
  }
  fft_lanes<NZ, +1>(v, t, buf, tws);
  if (active) {
    cd* dst = out + (size_t)f * d.PH + remH;
#pragma unroll
    for (int q = 0; q < E; ++q) st_cd(dst + (size_t)(t + T * q) * planeH, v[q]);
  }
}

// P4.  Fused forward z transform + stage update + inverse z transform: one lane group per (field f, (ky,kx) column).
//   1. R^(kz) = (1/N) FFT_z of the bracket term Gh[f] (N+-, R_m), kz part of Eq. 20 (only retained kz are used)
//   2. mode 0: out = RHS (N+-, H_m);  mode 1: half-step predictor (Eq. 15, Alg. 1 l.3-4);  mode 2: full-step corrector
//      (Alg. 1 l.8-9) followed by the exponential dissipation factors (Eq. 17-19, Alg. 2 l.12-14).
//      H_m = R_m + s i kz [ g_m - dn_m g_{m-1} - up_m g_{m+1} ]  (Eq. 6) reads the stage state Ws of the neighbours.
//   3. the new state goes to Wout (compact) and, through an inverse z transform of the same registers, to the hybrid
//      copy Hout that the next RHS evaluation consumes -- the spectral bracket terms never reach HBM.
// Tables (k_tables, once per step): tabz[cz] = {cos th/2, sin th/2, cos th, sin th, fz, fzg}, th = kz vA dt;
// tabp[col] = {fperp, fperp_g}: the separable factors of exp(-(eta P_perp + eta_z P_z) dt).
// Work items are ordered with f fastest so that the CTAs that read g_{m-1}, g_m, g_{m+1} of the same columns run together.
template <int NZ> struct ZStepGeom {
  using G = FftGeom<NZ>;
  // 16 columns (256 B per z row) up to nz = 256; at nz = 512 (one warp per column) 8 columns
#ifndef GD_ZS_THREADS
#define GD_ZS_THREADS 128
#endif
  static constexpr int THREADS = (G::T >= 16) ? 256 : GD_ZS_THREADS;
  static constexpr int GROUPS = THREADS / G::T;              // columns per CTA
  static constexpr int NSUB = (GROUPS + 7) / 8;              // 8-column sub-tiles (one TMA box each)
  static constexpr int SUBSTR = tma_substr(NZ);              // complex entries per sub-tile [NZ][8], a multiple of 1024 bytes
  static constexpr int KZ = 2 * (NZ / 3) + 1;                // retained kz (== Dims::Kz)
  static constexpr int LD = GROUPS + 1;                      // padded row of the [kz][column] tile
  static constexpr int XCH = GROUPS * (G::BUF + 1);          // FFT exchange buffers (alias the tiles)
  static constexpr int cmax(int a, int b) { return a > b ? a : b; }
  static constexpr int REGION = cmax(cmax(XCH, KZ * LD), NSUB * SUBSTR);
  static constexpr size_t SMEM = ((size_t)REGION + FftTw<NZ>::COUNT) * sizeof(cd) + 1024;   // + alignment slack
};
// EXACT (hermite_exact = 1, hermite.cu; Q30): the streaming term of H_m is left to the exact propagator -- the moment
// fields get only their bracket term (no neighbour reads), no dissipation here, and no hybrid copy (the propagated state's
// copy is made afterwards); in mode 2 they are updated in place on Ws (= P(dt/2) g_n), w+- as usual on Wn -> Wout.
// mapG / mapH: Gh and H viewed as fp64 tensors {2*Ky*Kx, nz, F} (the (ky,kx) plane flattened: hybrid rows are unpadded, so a
// block of columns is contiguous even across a ky row end), boxes {16 doubles, NZ, 1}, 128-byte swizzle (common.cuh).
template <int NZ, int MODE, bool EXACT>   // MODE 0 / 1 / 2 = RHS only / predictor / corrector + dissipation (compile time: fewer registers)
__global__ void __launch_bounds__(ZStepGeom<NZ>::THREADS, ZStepGeom<NZ>::THREADS > 128 ? 2 : (ZStepGeom<NZ>::THREADS > 64 ? 4 : 8)) k_zstep(Dims d, int if_variant, double skz_sign,
                                                      const __grid_constant__ CUtensorMap mapG, const __grid_constant__ CUtensorMap mapH,
                                                      bool have_G, bool want_H,
                                                      const cd* __restrict__ Wn, const cd* __restrict__ Ws, cd* __restrict__ Wout,
                                                      const double* __restrict__ scal,
                                                      const double* __restrict__ cdn, const double* __restrict__ cup,
                                                      const double* __restrict__ collfac, const double* __restrict__ tabz,
                                                      const double* __restrict__ tabp, const cd* __restrict__ tw) {
  using G = FftGeom<NZ>;
  using Z = ZStepGeom<NZ>;
  constexpr int mode = MODE;
  constexpr int T = G::T, E = G::E;
  constexpr int GROUPS = Z::GROUPS, KZ = Z::KZ, LD = Z::LD, THREADS = Z::THREADS;
  constexpr int RB = tma_rb(NZ), NRB = tma_nrb(NZ);            // a box has at most 256 rows
  extern __shared__ cd smem_raw[];
  __shared__ unsigned long long bar;
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  cd* tile = align1024(smem_raw);                              // region: TMA sub-tiles / [KZ][LD] tile / exchange buffers
  cd* tws_s = tile + Z::REGION;                                // stage twiddle table
  cd* buf = tile + (size_t)grp * (G::BUF + 1);
  cd* sub = tile + (size_t)(grp >> 3) * Z::SUBSTR;             // this group's 8-column sub-tile, column grp & 7
  const int subc = grp & 7;
  const cd* tws = tws_s;
  const int plane = d.Ky * d.Kx;
  const int f = blockIdx.x % d.F, cb = blockIdx.x / d.F;
  const int col0 = cb * GROUPS;
  const int col = col0 + grp;
  const bool active = col < plane;
  const int ncolv = min(GROUPS, plane - col0);
  const int nsubv = (ncolv + 7) >> 3;                          // sub-tiles with at least one valid column
  // the bracket tile and the twiddle table are requested first (one thread, three instructions), then the per-item scalars
  if (threadIdx.x == 0) {
    mbar_init(&bar, 1);
    unsigned bytes = (unsigned)(FftTw<NZ>::COUNT * sizeof(cd));
    if (have_G) bytes += (unsigned)(nsubv * NZ * 8 * sizeof(cd));   // a box always delivers its full size (out-of-range columns as zeros)
    if (bytes > 0) {
      mbar_arrive_expect_tx(&bar, bytes);
      if (have_G)
        for (int sidx = 0; sidx < nsubv; ++sidx)
          for (int rb = 0; rb < NRB; ++rb) tma_load_3d(tile + (size_t)sidx * Z::SUBSTR + rb * RB * 8, &mapG, 2 * (col0 + 8 * sidx), rb * RB, f, &bar);
      if (FftTw<NZ>::COUNT > 0) bulk_g2s(tws_s, tw, (unsigned)(FftTw<NZ>::COUNT * sizeof(cd)), &bar);
    } else {
      mbar_arrive(&bar);
    }
  }
  const double dt = scal[SC_DT];
  const int m = f - 2;
  const double dn = f >= 2 ? cdn[m] : 0.0, up = f >= 2 ? cup[m] : 0.0;
  const double cf = (mode == 2 && f >= 2) ? collfac[m] : 1.0;
  __syncthreads();                                             // barrier initialised before anybody waits on it
  mbar_wait(&bar, 0);
  // 1. forward z transform of the bracket term, retained kz -> tile (scaled by 1/N)
  if (have_G) {
    cd v[E];
#pragma unroll
    for (int q = 0; q < E; ++q) v[q] = active ? sub[swz8(t + T * q, subc)] : cmake(0.0, 0.0);
    __syncthreads();                                           // tile consumed: the exchange buffers may overwrite it
    fft_lanes<NZ, -1>(v, t, buf, tws);
    __syncthreads();                                           // every group is done with its exchange buffer
#pragma unroll
    for (int q = 0; q < E; ++q) {
      const int cz = fft2c(t + T * q, NZ, NZ / 3, KZ);
      if (cz >= 0) tile[cz * LD + grp] = cscale(v[q], d.inv_n);
    }
  } else {
    for (int e = threadIdx.x; e < KZ * LD; e += THREADS) tile[e] = cmake(0.0, 0.0);
  }
  __syncthreads();
  // 2. pointwise stage update on the tile: thread <-> (kz, column), columns fastest (row-contiguous global accesses);
  //    the loads of UB modes are issued together
  {
    const double c = (mode == 1) ? 0.5 * dt : dt;
    const bool lo = !EXACT && f > 2, hi = !EXACT && f + 1 < d.F, same = (EXACT || Ws == Wn || mode == 0);
    cd* const wout = (EXACT && mode == 2 && f >= 2) ? const_cast<cd*>(Ws) : Wout;
    constexpr int NEL = KZ * GROUPS, UB = 6;
    for (int e0 = threadIdx.x; e0 < NEL; e0 += UB * THREADS) {
      cd a0[UB], a1[UB], a2[UB], a3[UB];
      bool ok[UB];
#pragma unroll
      for (int u = 0; u < UB; ++u) {
        const int e = e0 + u * THREADS;
        const int cz = e / GROUPS, cl = e % GROUPS;
        ok[u] = e < NEL && cl < ncolv;
        const size_t idx = ok[u] ? (size_t)cz * plane + col0 + cl : 0;
        a0[u] = a1[u] = a2[u] = a3[u] = cmake(0.0, 0.0);
        if (mode != 0 || f >= 2) {
          if (f < 2) a0[u] = ldg_cd(Wn + (size_t)f * d.PS + idx);
          else {
            a0[u] = ldg_cd(Ws + (size_t)f * d.PS + idx);
            if (lo) a1[u] = ldg_cd(Ws + (size_t)(f - 1) * d.PS + idx);
            if (hi) a2[u] = ldg_cd(Ws + (size_t)(f + 1) * d.PS + idx);
            if (!same) a3[u] = ldg_cd(Wn + (size_t)f * d.PS + idx);   // (no copy of a0 here: it would wait on the load)
          }
        }
      }
#pragma unroll
      for (int u = 0; u < UB; ++u) {
        if (!ok[u]) continue;
        const int e = e0 + u * THREADS;
        const int cz = e / GROUPS, cl = e % GROUPS;
        const size_t idx = (size_t)cz * plane + col0 + cl;
        const cd Gv = tile[cz * LD + cl];
        const double* tz = tabz + 6 * cz;
        cd out;
        if (f < 2) {
          if (mode == 0) out = Gv;
          else {
            const double sg = f == 0 ? 1.0 : -1.0;
            const cd ph_half = cmake(tz[0], sg * tz[1]), ph_full = cmake(tz[2], sg * tz[3]);
            const cd wn = a0[u];
            const cd N = cscale(Gv, c);
            if (mode == 1) {
              const cd inner = (if_variant == 0) ? wn + cmul(ph_half, N) : wn + N;     // Eq. 15 / standard IF midpoint
              out = cmul(ph_half, inner);
            } else {
              if (if_variant == 0) out = cmul(ph_full, wn + cmul(ph_full, N));
              else out = cmul(ph_full, wn) + cmul(ph_half, N);
              out = cscale(out, tabp[2 * (col0 + cl)] * tz[4]);
            }
          }
        } else {
          const double skz = (m < d.Msp ? skz_sign : -skz_sign) * d.kz0 * c2n(cz, NZ / 3, KZ);   // g^+ : upper, g^- : lower signs of Eq. 6
          const cd lin = cmake(a0[u].x - dn * a1[u].x - up * a2[u].x, a0[u].y - dn * a1[u].y - up * a2[u].y);
          const cd Hm = EXACT ? Gv : cmake(Gv.x - skz * lin.y, Gv.y + skz * lin.x);    // + i s kz lin  (Eq. 6)
          if (mode == 0) out = Hm;
          else {
            const cd gn = same ? a0[u] : a3[u];
            out = cmake(gn.x + c * Hm.x, gn.y + c * Hm.y);
            if (mode == 2 && !EXACT) out = cscale(out, cf * tabp[2 * (col0 + cl) + 1] * tz[5]);
          }
        }
        st_cd(wout + (size_t)f * d.PS + idx, out);
        tile[cz * LD + cl] = out;
      }
    }
  }
  if (!want_H || (EXACT && f >= 2)) return;
  __syncthreads();
  // 3. inverse z transform of the new stage state (zero-padded) -> hybrid copy
  cd v[E];
#pragma unroll
  for (int q = 0; q < E; ++q) {
    const int cz = fft2c(t + T * q, NZ, NZ / 3, KZ);
    v[q] = (cz >= 0 && active) ? tile[cz * LD + grp] : cmake(0.0, 0.0);
  }
  __syncthreads();                                             // tile read by every group: the exchange may overwrite it
  fft_lanes<NZ, +1>(v, t, buf, tws);
  // the [nz][GROUPS] result goes through the (now free) region in the swizzled sub-tile layout and leaves by one tensor store
  // per sub-tile (columns beyond the plane are clipped by the map)
  __syncthreads();                                             // every group is done with its exchange buffer
#pragma unroll
  for (int q = 0; q < E; ++q) sub[swz8(t + T * q, subc)] = v[q];
  fence_proxy_async();                                         // generic-proxy writes -> visible to the async proxy
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int sidx = 0; sidx < nsubv; ++sidx)
      for (int rb = 0; rb < NRB; ++rb) tma_store_3d(&mapH, 2 * (col0 + 8 * sidx), rb * RB, f, tile + (size_t)sidx * Z::SUBSTR + rb * RB * 8);
    bulk_commit();
    bulk_wait_read0();                                         // shared memory must stay valid until the engine has read it
  }
}

// Geometry of the y passes: THREADS lanes per CTA = GROUPS lane groups = GROUPS adjacent columns of ONE array,
// so a CTA covers GROUPS*16 B contiguous per row (256 B at ny = 256: strided row segments narrower than that lose
// HBM efficiency: a round-1 copy probe with this row stride moved 4.2 / 5.0 / 5.3 TB/s at 64 / 128 / 256 B per row)
// and two CTAs fit on an SM (<= 128 registers per lane).
template <int NY> struct YGeom {
  using G = FftGeom<NY>;
  static constexpr int T = G::T, E = G::E;
  // ny = 512 (one warp per transform): 12 warps = 12 columns with 170 registers per lane (no spills)
#ifndef GD_Y512_THREADS
#define GD_Y512_THREADS 384
#endif
  // ny = 64, 128 (8 lanes per transform): 128-thread CTAs = 16 columns (256-byte rows, as at ny = 256), four per SM.  With 256 threads
  // a CTA spans 32 columns and Kx = 43 (nx = 128) leaves the second block two thirds empty: measured at BASELINE config 3
  // (128x128x64, M = 32) P1 0.163 -> 0.125 ms, P3 0.091 -> 0.080 ms, step 1.170 -> 1.067 ms; config 2 0.1637 -> 0.1597 ms
#ifndef GD_Y8_THREADS
#define GD_Y8_THREADS 128
#endif
  static constexpr int THREADS = (T >= 32) ? GD_Y512_THREADS : (T == 8 ? GD_Y8_THREADS : 256);
  static constexpr int CTAS = (THREADS > 256) ? 1 : (THREADS <= 128 ? 4 : 2);       // resident CTAs per SM
  static constexpr int PAIR_CTAS = (THREADS <= 128) ? 2 : 1;                        // of the register-heavy pair kernel
  static constexpr int GROUPS = THREADS / T;                 // columns per CTA
};

// P1.  Persistent CTAs over the work items (source field s, z, block of GROUPS columns).  Sources: s = 0,1 -> w+, w-;
// s = 2+m -> g_m.  D array order: 0/1 xi+ , 2/3 xi- , 4/5 w+ , 6/7 w- , 8+2m / 9+2m g_m  (even: U = kx f + df/dy,
// odd: V = df/dy - kx f: the two combinations the x-pass packs, pass_x.cu).
// The [Ky][GROUPS] tile of retained modes arrives by one bulk async copy per row (TMA engine) into a padded
// shared-memory tile; every lane group then reads its column once per output array (U, then V, Eq. 10; the
// Elsasser sources first give xi = -w/kperp^2, then w) -- no second copy of the column in registers.
// The next item's tile is requested as soon as the last read of the current one is done.
#ifndef GD_Y_PAIR_RAGGED
#define GD_Y_PAIR_RAGGED 1
#endif
// Work items of the persistent P1.  Classic enumeration: (array, z, column block), column block fastest; the last block of
// a plane is ragged when GROUPS does not divide Kx (6 of 16 columns at nx = 256) and costs a full item's time.  Paired
// enumeration (npf >= 0, the number of FULL blocks per plane; needs nz even and a remainder of at most GROUPS/2 columns): per
// (array, pair of planes z0, z0+1) the 2*npf full blocks, then ONE item that takes the remainder columns of BOTH planes -- lane
// groups [0, GROUPS/2) work on plane z0, [GROUPS/2, GROUPS) on plane z0+1, each on its own half of the tile.  At nx = 256 that is
// 5.5 instead of 6 items per plane (lane use 86/88 instead of 86/96).  Measured at 4a, same box: P1 0.842 -> 0.800 ms, step 6.96 ->
// 6.88 ms.  P3 keeps the classic enumeration: there the paired item doubles the per-row copy issue loop, which is what P3 waits
// on (0.505 -> 0.513 ms).
struct YItem { int arr, z0, cb; bool rag; };
__device__ __forceinline__ YItem y_item(int item, int ncb, int nz, int npf) {
  YItem it;
  if (npf < 0) { it.cb = item % ncb; const int az = item / ncb; it.z0 = az % nz; it.arr = az / nz; it.rag = false; }
  else {
    const int ipp = 2 * npf + 1, j = item % ipp, ap = item / ipp, nzp = nz >> 1;
    it.rag = (j == 2 * npf);
    it.arr = ap / nzp;
    it.z0 = 2 * (ap % nzp) + (it.rag ? 0 : j / (npf > 0 ? npf : 1));
    it.cb = it.rag ? npf : j % (npf > 0 ? npf : 1);
  }
  return it;
}
// host: full blocks per plane if the paired enumeration applies, else -1; and the item count per array
static inline int y_pair_mode(int Kx, int groups, int nz) {
  const int rem = Kx % groups;
  return (rem > 0 && 2 * rem <= groups && (nz & 1) == 0) ? Kx / groups : -1;
}
static inline int y_items_per_array(int Kx, int groups, int nz, int npf) {
  return npf < 0 ? nz * ((Kx + groups - 1) / groups) : (nz / 2) * (2 * npf + 1);
}
template <int NY> struct YInvGeom {
  using Y = YGeom<NY>;
  static constexpr int LD = Y::GROUPS + 1;
  static constexpr int KYMAX = 2 * (NY / 3) + 1;
  static constexpr int XB = (FftGeom<NY>::S > 1 ? FftGeom<NY>::BUF : 0) + 2;            // doubles per group
  static constexpr size_t SMEM = ((size_t)FftTw<NY>::COUNT + (size_t)KYMAX * LD) * sizeof(cd) + (size_t)Y::GROUPS * XB * sizeof(double);
};
template <int NY, bool ELS>   // ELS: the Elsasser sources s = 0, 1 (four outputs each, potentials first); else s = 2 + m
__global__ void __launch_bounds__(YGeom<NY>::THREADS, YGeom<NY>::CTAS) k_yinv(Dims d, const cd* __restrict__ H, cd* __restrict__ D,
                                                        const cd* __restrict__ tw, int ncb, int nitems, int npf) {
  using Y = YGeom<NY>;
  using G = FftGeom<NY>;
  using YI = YInvGeom<NY>;
  constexpr int HALF = Y::GROUPS / 2;
  constexpr int T = G::T, E = G::E, LD = YI::LD;
  extern __shared__ cd smem[];
  __shared__ unsigned long long bar;
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  cd* tile = smem + FftTw<NY>::COUNT;
  double* xbuf = reinterpret_cast<double*>(tile + (size_t)YI::KYMAX * LD) + (size_t)grp * YI::XB;
  if (threadIdx.x == 0) mbar_init(&bar, 1);
  fft_load_table<NY>(smem, tw);                  // ends with __syncthreads()
  const cd* tws = smem;
  auto issue = [&](int item) {                   // all threads: one bulk copy per tile row (row = retained ky)
    const YItem it = y_item(item, ncb, d.nz, npf);
    const int s = it.arr + (ELS ? 0 : 2);
    const int cx0 = it.cb * Y::GROUPS;
    const int ncol = min(Y::GROUPS, d.Kx - cx0);
    const cd* src = H + (size_t)s * d.PH + (size_t)it.z0 * d.Ky * d.Kxp + cx0;
    if (threadIdx.x == 0) mbar_arrive_expect_tx(&bar, (unsigned)((it.rag ? 2 : 1) * d.Ky * ncol * sizeof(cd)));
    for (int r = threadIdx.x; r < d.Ky; r += Y::THREADS) {
      bulk_g2s(tile + (size_t)r * LD, src + (size_t)r * d.Kxp, (unsigned)(ncol * sizeof(cd)), &bar);
      if (it.rag) bulk_g2s(tile + (size_t)r * LD + HALF, src + ((size_t)d.Ky + r) * d.Kxp, (unsigned)(ncol * sizeof(cd)), &bar);   // plane z0 + 1
    }
  };
  constexpr int HY3 = NY / 3, KY = 2 * HY3 + 1;   // == d.hy3, d.Ky: compile-time so that the per-q mode tests fold
  int item = blockIdx.x;
  if (item < nitems) issue(item);
  unsigned phase = 0;
  const double kyt = d.ky0 * t, kyT = d.ky0 * T;
  while (item < nitems) {
    const YItem it = y_item(item, ncb, d.nz, npf);
    const int s = it.arr + (ELS ? 0 : 2);
    const int gz = (it.rag && grp >= HALF) ? 1 : 0;          // ragged pair item: the upper half of the groups takes plane z0 + 1
    const int z = it.z0 + gz;
    const int cx = it.cb * Y::GROUPS + grp - gz * HALF;
    const bool active = cx < d.Kx;                           // (ragged: the remainder is at most HALF columns wide)
    const double kx = d.kx0 * cx;
    const int cxa = active ? cx : 0;
    constexpr int rounds = ELS ? 4 : 2;
    // D[a][line block][kx][xl], line = z*ny + y, slot (line % xl) ^ (kx % xl): the lanes of a group fill whole aligned
    // runs of one block row.  Offsets of element q: off0 + q*ostr when a block row holds at most T lines.
    const int lineb = z * NY + t;
    const bool lin_off = d.xl <= T;
    const int sw = cxa & (d.xl - 1);
    const int off0 = ((((lineb >> d.xlsh) * d.Kx + cxa)) << d.xlsh) + ((lineb & (d.xl - 1)) ^ sw);
    const int ostr = T * d.Kx;
    mbar_wait(&bar, phase);
    phase ^= 1u;
    item += gridDim.x;
    for (int r = 0; r < rounds; ++r) {
      const bool pot = ELS && (r < 2);           // rounds 0,1 of an Elsasser source: the potential xi = -w/kperp^2
      const int which = r & 1;                   // 0: U, 1: V
      const int a = (ELS ? (pot ? 2 * s : 4 + 2 * s) : 8 + 2 * (s - 2)) + which;
      cd v[E];
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int cy = fft2c(t + T * q, NY, HY3, KY);
        v[q] = (active && cy >= 0) ? tile[cy * LD + grp] : cmake(0.0, 0.0);
      }
      if (r == rounds - 1) {
        __syncthreads();                         // last read of the tile by every lane
        if (item < nitems) issue(item);          // prefetch: overlaps the transform and the stores below
      }
      // which = 0: U = kx f + df/dy -> multiplier (kx + i ky);  which = 1: V = df/dy - kx f -> multiplier (i ky - kx)  (Eq. 10)
      {
        const double skx = which ? -kx : kx;
#pragma unroll
        for (int q = 0; q < E; ++q) {
          if (T * q <= HY3 || T * q + T - 1 >= NY - HY3) {      // compile-time: some lane of this q holds a retained ky
            const double ky = fma(kyT, (double)(q < E / 2 ? q : q - E), kyt);     // ky0 * signed mode number of t + T q
            double ar = skx, ai = ky;
            if (pot) { const double k2 = kx * kx + ky * ky; const double f = k2 > 0.0 ? -__drcp_rn(k2) : 0.0; ar *= f; ai *= f; }   // xi = -w/kperp^2 (correctly rounded reciprocal == -1.0/k2)
            v[q] = cmake(ar * v[q].x - ai * v[q].y, ar * v[q].y + ai * v[q].x);
          }
        }
      }
      fft_lanes_split<NY, +1>(v, t, xbuf, tws);
      if (active) {
        cd* dst = D + (size_t)a * d.PD;
        if (lin_off) {
#pragma unroll
          for (int q = 0; q < E; ++q) st_cd(dst + (off0 + q * ostr), v[q]);
        } else {
#pragma unroll
          for (int q = 0; q < E; ++q) {
            const int line = lineb + T * q;
            st_cd(dst + (((line >> d.xlsh) * d.Kx + cxa) << d.xlsh) + ((line & (d.xl - 1)) ^ sw), v[q]);
          }
        }
      }
    }
  }
}

// P3.  E arrays: 0 A, 1 B, 2+m R_m.  Output hybrid fields: 0 N+, 1 N-, 2+m R_m.
// The [ny][GROUPS] input tile of a work item arrives by one bulk async copy per row (TMA engine, mbarrier
// completion) into a padded shared-memory tile, so the global side moves whole row segments and the lanes then read
// their own column conflict-free.
//
// k_yfwd_pair: persistent CTAs over the work items (z, block of GROUPS columns).  Every lane group transforms column A,
// keeps it in registers, transforms column B of the same kx and forms N+- = -1/2 A -+ 1/2 kperp^2 B  (Eq. 1 with
// Eq. 11).  One tile buffer: B's tile is in flight during A's transform, the next item's A tile
// during B's transform.  (Geometry and shared-memory layout of k_yfwd below.)
template <int NY> struct YFwdGeom;
template <int NY>
__global__ void __launch_bounds__(YGeom<NY>::THREADS, YGeom<NY>::PAIR_CTAS) k_yfwd_pair(Dims d, const cd* __restrict__ Ein, cd* __restrict__ Gh,
                                                                     const cd* __restrict__ tw, int ncb, int nitems);

// k_yfwd: persistent CTAs over the work items (array a >= 2, z, block of GROUPS columns).  The exchange uses its
// own (split, 8-byte) buffers, so the NEXT item's tile is in flight while the current one is transformed and stored.
template <int NY> struct YFwdGeom {
  using Y = YGeom<NY>;
  static constexpr int LD = Y::GROUPS + 1;
  static constexpr int XB = (FftGeom<NY>::S > 1 ? FftGeom<NY>::BUF : 0) + 2;            // doubles per group (even: 16-B alignment)
  static constexpr size_t SMEM = ((size_t)FftTw<NY>::COUNT + (size_t)NY * LD) * sizeof(cd) + (size_t)Y::GROUPS * XB * sizeof(double);
};
template <int NY>
__global__ void __launch_bounds__(YGeom<NY>::THREADS, YGeom<NY>::CTAS) k_yfwd(Dims d, const cd* __restrict__ Ein, cd* __restrict__ Gh,
                                                        const cd* __restrict__ tw, int ncb, int nitems) {
  using Y = YGeom<NY>;
  using G = FftGeom<NY>;
  using YF = YFwdGeom<NY>;
  constexpr int T = G::T, E = G::E, LD = YF::LD;
  constexpr int HY3 = NY / 3, KY = 2 * HY3 + 1;   // == d.hy3, d.Ky
  extern __shared__ cd smem[];
  __shared__ unsigned long long bar;
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  cd* tile = smem + FftTw<NY>::COUNT;
  double* xbuf = reinterpret_cast<double*>(tile + (size_t)NY * LD) + (size_t)grp * YF::XB;
  if (threadIdx.x == 0) mbar_init(&bar, 1);
  fft_load_table<NY>(smem, tw);                  // ends with __syncthreads()
  const cd* tws = smem;
  auto issue = [&](int item) {                   // all threads: one bulk copy per tile row
    const int cb = item % ncb, az = item / ncb;
    const int z = az % d.nz, a = 2 + az / d.nz;
    const int cx0 = cb * Y::GROUPS;
    const int ncol = min(Y::GROUPS, d.Kx - cx0);
    if (threadIdx.x == 0) mbar_arrive_expect_tx(&bar, (unsigned)(NY * ncol * sizeof(cd)));
    for (int r = threadIdx.x; r < NY; r += Y::THREADS)
      bulk_g2s(tile + (size_t)r * LD, Ein + (size_t)a * d.PE + ((size_t)z * NY + r) * d.Kxe + cx0, (unsigned)(ncol * sizeof(cd)), &bar);
  };
  int item = blockIdx.x;
  if (item < nitems) issue(item);
  unsigned phase = 0;
  while (item < nitems) {
    const int cb = item % ncb, az = item / ncb;
    const int z = az % d.nz, a = 2 + az / d.nz;
    const int cx = cb * Y::GROUPS + grp;
    const bool active = cx < d.Kx;
    mbar_wait(&bar, phase);
    phase ^= 1u;
    cd v[E];
#pragma unroll
    for (int q = 0; q < E; ++q) v[q] = active ? tile[(t + T * q) * LD + grp] : cmake(0.0, 0.0);
    __syncthreads();                             // tile consumed by every lane
    item += gridDim.x;
    if (item < nitems) issue(item);              // prefetch: overlaps the transform and the stores below
    fft_lanes_split<NY, -1>(v, t, xbuf, tws);
    if (active) {
      cd* dst = Gh + (size_t)a * d.PH + (size_t)z * KY * d.Kxp + cx;
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int cy = fft2c(t + T * q, NY, HY3, KY);
        if (cy >= 0) st_cd(dst + cy * d.Kxp, v[q]);
      }
    }
  }
}

template <int NY>
__global__ void __launch_bounds__(YGeom<NY>::THREADS, YGeom<NY>::PAIR_CTAS) k_yfwd_pair(Dims d, const cd* __restrict__ Ein, cd* __restrict__ Gh,
                                                                     const cd* __restrict__ tw, int ncb, int nitems) {
  using Y = YGeom<NY>;
  using G = FftGeom<NY>;
  using YF = YFwdGeom<NY>;
  constexpr int T = G::T, E = G::E, LD = YF::LD;
  constexpr int HY3 = NY / 3, KY = 2 * HY3 + 1;   // == d.hy3, d.Ky
  extern __shared__ cd smem[];
  __shared__ unsigned long long bar;
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  cd* tile = smem + FftTw<NY>::COUNT;
  double* xbuf = reinterpret_cast<double*>(tile + (size_t)NY * LD) + (size_t)grp * YF::XB;
  if (threadIdx.x == 0) mbar_init(&bar, 1);
  fft_load_table<NY>(smem, tw);                  // ends with __syncthreads()
  const cd* tws = smem;
  auto issue = [&](int item, int arr) {          // all threads: one bulk copy per tile row of E array `arr` (0: A, 1: B)
    const int cb = item % ncb, z = item / ncb;
    const int cx0 = cb * Y::GROUPS;
    const int ncol = min(Y::GROUPS, d.Kx - cx0);
    if (threadIdx.x == 0) mbar_arrive_expect_tx(&bar, (unsigned)(NY * ncol * sizeof(cd)));
    for (int r = threadIdx.x; r < NY; r += Y::THREADS)
      bulk_g2s(tile + (size_t)r * LD, Ein + (size_t)arr * d.PE + ((size_t)z * NY + r) * d.Kxe + cx0, (unsigned)(ncol * sizeof(cd)), &bar);
  };
  int item = blockIdx.x;
  if (item < nitems) issue(item, 0);
  unsigned phase = 0;
  while (item < nitems) {
    const int cb = item % ncb, z = item / ncb;
    const int cx = cb * Y::GROUPS + grp;
    const bool active = cx < d.Kx;
    cd va[E], v[E];
    mbar_wait(&bar, phase);
    phase ^= 1u;
#pragma unroll
    for (int q = 0; q < E; ++q) va[q] = active ? tile[(t + T * q) * LD + grp] : cmake(0.0, 0.0);
    __syncthreads();                             // A tile consumed by every lane
    issue(item, 1);                              // B's tile travels during A's transform
    fft_lanes_split<NY, -1>(va, t, xbuf, tws);
    mbar_wait(&bar, phase);
    phase ^= 1u;
#pragma unroll
    for (int q = 0; q < E; ++q) v[q] = active ? tile[(t + T * q) * LD + grp] : cmake(0.0, 0.0);
    __syncthreads();                             // B tile consumed
    item += gridDim.x;
    if (item < nitems) issue(item, 0);           // the next item's A tile travels during B's transform and the stores
    fft_lanes_split<NY, -1>(v, t, xbuf, tws);
    if (active) {
      const double kx = d.kx0 * cx;
      cd* dp = Gh + (size_t)z * KY * d.Kxp + cx;
      cd* dm = dp + d.PH;
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int cy = fft2c(t + T * q, NY, HY3, KY);
        if (cy >= 0) {
          const double ky = d.ky0 * fft2n(t + T * q, NY);
          const double hk2 = 0.5 * (kx * kx + ky * ky) * d.inv_bscale;     // the x-pass delivered bscale*B (exact power of two)
          st_cd(dp + cy * d.Kxp, cmake(-0.5 * va[q].x - hk2 * v[q].x, -0.5 * va[q].y - hk2 * v[q].y));
          st_cd(dm + cy * d.Kxp, cmake(-0.5 * va[q].x + hk2 * v[q].x, -0.5 * va[q].y + hk2 * v[q].y));
        }
      }
    }
  }
}


// ---- launchers ------------------------------------------------------------------------------------
template <int N> static size_t fft_smem() { return ((size_t)(GD_Z_THREADS / FftGeom<N>::T) * (FftGeom<N>::BUF + 1) + FftTw<N>::COUNT) * sizeof(cd); }
template <int N> static int fft_blocks(long long ncols) { const int gpb = GD_Z_THREADS / FftGeom<N>::T; return (int)((ncols + gpb - 1) / gpb); }

#define GD_DISPATCH(NVAL, MACRO)                                                      \
  switch (NVAL) {                                                                     \
    case 2: MACRO(2) break; case 4: MACRO(4) break; case 8: MACRO(8) break;           \
    case 16: MACRO(16) break; case 32: MACRO(32) break; case 64: MACRO(64) break;     \
    case 128: MACRO(128) break; case 256: MACRO(256) break; case 512: MACRO(512) break; \
    default: return cudaErrorInvalidValue;                                            \
  }

cudaError_t launch_zfft(const Dims& d, const cd* in, cd* out, const cd* tw, int nfields, cudaStream_t st) {
  const long long ncols = (long long)nfields * d.Ky * d.Kx;
#define ZCASE(NN) k_zfft<NN><<<fft_blocks<NN>(ncols), GD_Z_THREADS, fft_smem<NN>(), st>>>(d, in, out, tw, (int)ncols);
  GD_DISPATCH(d.nz, ZCASE)
  return cudaGetLastError();
}
cudaError_t launch_zstep(const Dims& d, const TMaps& tm, int mode, bool exact, int if_variant, int g_sign, bool have_G, const cd* Wn, const cd* Ws,
                         cd* Wout, bool want_H, const double* scal, const double* cdn, const double* cup, const double* collfac,
                         const double* tabz, const double* tabp, const cd* tw, cudaStream_t st) {
  const long long ncols = (long long)d.Ky * d.Kx;
#define ZSARGS d, if_variant, (double)g_sign, tm.g_flat, tm.h_flat, have_G, want_H, Wn, Ws, Wout, scal, cdn, cup, collfac, tabz, tabp, tw
#define ZSCASE(NN)                                                                                               \
  {                                                                                                              \
    using Z = ZStepGeom<NN>;                                                                                     \
    const int nb = (int)((ncols + Z::GROUPS - 1) / Z::GROUPS) * d.F;                                             \
    if (mode == 0) k_zstep<NN, 0, false><<<nb, Z::THREADS, Z::SMEM, st>>>(ZSARGS);                               \
    else if (mode == 1 && !exact) k_zstep<NN, 1, false><<<nb, Z::THREADS, Z::SMEM, st>>>(ZSARGS);                \
    else if (mode == 1) k_zstep<NN, 1, true><<<nb, Z::THREADS, Z::SMEM, st>>>(ZSARGS);                           \
    else if (!exact) k_zstep<NN, 2, false><<<nb, Z::THREADS, Z::SMEM, st>>>(ZSARGS);                             \
    else k_zstep<NN, 2, true><<<nb, Z::THREADS, Z::SMEM, st>>>(ZSARGS);                                          \
  }
  GD_DISPATCH(d.nz, ZSCASE)
  return cudaGetLastError();
}
cudaError_t launch_yinv(const Dims& d, const cd* H, cd* D, const cd* tw, int num_sms, cudaStream_t st) {   // persistent: CTAS per SM
#define YICASE(NN)                                                                                         \
  {                                                                                                        \
    const int ncb = (d.Kx + YGeom<NN>::GROUPS - 1) / YGeom<NN>::GROUPS;                                    \
    const int cap = YGeom<NN>::CTAS * num_sms;                                                           \
    const int npf = GD_Y_PAIR_RAGGED ? y_pair_mode(d.Kx, YGeom<NN>::GROUPS, d.nz) : -1;                    \
    const int ipa = y_items_per_array(d.Kx, YGeom<NN>::GROUPS, d.nz, npf);                                 \
    const int ne = 2 * ipa, nm = d.M * ipa;                                                                \
    k_yinv<NN, true><<<ne < cap ? ne : cap, YGeom<NN>::THREADS, YInvGeom<NN>::SMEM, st>>>(d, H, D, tw, ncb, ne, npf);                 \
    if (nm > 0) k_yinv<NN, false><<<nm < cap ? nm : cap, YGeom<NN>::THREADS, YInvGeom<NN>::SMEM, st>>>(d, H, D, tw, ncb, nm, npf);    \
  }
  GD_DISPATCH(d.ny, YICASE)
  return cudaGetLastError();
}
cudaError_t launch_yfwd(const Dims& d, const cd* E, cd* Gh, const cd* tw, int num_sms, cudaStream_t st) {
#define YFCASE(NN)                                                                                         \
  {                                                                                                        \
    const int ncb = (d.Kx + YGeom<NN>::GROUPS - 1) / YGeom<NN>::GROUPS;                                    \
    const int np = d.nz * ncb;                                                                             \
    k_yfwd_pair<NN><<<np < YGeom<NN>::PAIR_CTAS * num_sms ? np : YGeom<NN>::PAIR_CTAS * num_sms, YGeom<NN>::THREADS, YFwdGeom<NN>::SMEM, st>>>(d, E, Gh, tw, ncb, np);   \
    const int nitems = d.M * d.nz * ncb;                                                                   \
    if (d.M > 0) k_yfwd<NN><<<nitems < YGeom<NN>::CTAS * num_sms ? nitems : YGeom<NN>::CTAS * num_sms, YGeom<NN>::THREADS, YFwdGeom<NN>::SMEM, st>>>(d, E, Gh, tw, ncb, nitems); \
  }
  GD_DISPATCH(d.ny, YFCASE)
  return cudaGetLastError();
}
// opt-in dynamic shared memory above 48 KB for every instantiation
cudaError_t prepare_passes_zy(int ny, int nz) {
#define ZPCASE(NN)                                                                                                         \
  {                                                                                                                        \
    cudaError_t e = cudaFuncSetAttribute(k_zfft<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem<NN>());      \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_zstep<NN, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZStepGeom<NN>::SMEM); \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_zstep<NN, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZStepGeom<NN>::SMEM); \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_zstep<NN, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZStepGeom<NN>::SMEM); \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_zstep<NN, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZStepGeom<NN>::SMEM);  \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_zstep<NN, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZStepGeom<NN>::SMEM);  \
    if (e != cudaSuccess) return e;                                                                                        \
  }
  GD_DISPATCH(nz, ZPCASE)
#define YPCASE(NN)                                                                                                         \
  {                                                                                                                        \
    cudaError_t e = cudaFuncSetAttribute(k_yinv<NN, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)YInvGeom<NN>::SMEM); \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_yinv<NN, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)YInvGeom<NN>::SMEM);      \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_yfwd_pair<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)YFwdGeom<NN>::SMEM);             \
    if (e != cudaSuccess) return e;                                                                                        \
    e = cudaFuncSetAttribute(k_yfwd<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)YFwdGeom<NN>::SMEM);            \
    if (e != cudaSuccess) return e;                                                                                        \
  }
  GD_DISPATCH(ny, YPCASE)
  return cudaSuccess;
}

// Host: the stage twiddle table of FFT plan ID n (fft.cuh layout); empty for single-stage sizes.
int fft_stage_table_host(int n, std::vector<cd>& out) {
#define TCASE(NN) out.assign(FftTw<NN>::COUNT + 1, cmake(0.0, 0.0)); fft_fill_stage_table<NN>(out.data());
  switch (n) {
    case 2: TCASE(2) break; case 4: TCASE(4) break; case 8: TCASE(8) break; case 16: TCASE(16) break;
    case 32: TCASE(32) break; case 64: TCASE(64) break; case 128: TCASE(128) break; case 256: TCASE(256) break;
    case 512: TCASE(512) break; case 256 + GD_FFT_ALT: TCASE(256 + GD_FFT_ALT) break;
    default: return -1;
  }
  return 0;
}
