// pass_x.cu -- P2, the fused row pass of the RHS pipeline (one lane group per (y,z) line).
//
// For every source field f in {xi+, xi-, w+, w-, g_m} the pass reads the two half-lines
// U = kx f~ + (df/dy)~ and V = (df/dy)~ - kx f~ of (kx; y,z) that P1 wrote (retained kx only), forms
//     Z(kx) = i kx f~(kx) + i (df/dy)~(kx) = i U(kx)        for kx >= 0       (Eq. 10)
//     Z(-kx) = conj(i kx f~) + i conj((df/dy)~) = i conj(V(kx))               (Hermitian completion)
// and ONE complex inverse FFT of length nx returns (df/dx) + i (df/dy) on the real line -- the
// derivative fields exist only in registers.  Bracket products:
//     A = {xi+,w-} + {xi-,w+},  B = {xi+,xi-}                          (Eq. 1)
//     P_m = {Phi,g_m}, Q_m = {Psi,g_m},  R_m = -P_m + dn_m Q_{m-1} + up_m Q_{m+1}   (Eq. 6)
// with {P,Q} = Px Qy - Py Qx.  R_m is combined in real space with a sliding window over m (linear,
// so one forward transform per moment instead of two).  Pairs of real lines (A,B), (R_m,R_{m+1}) go
// through ONE complex forward FFT and are separated by Hermitian symmetry; only kx <= nx/3 is
// written (kx part of Eq. 20).  The CFL quantity max (dPhi/dx)^2+(dPhi/dy)^2
// (Eq. 16) rides on the Elsasser part.
#include "common.cuh"

#ifndef GD_X_SPLIT
#define GD_X_SPLIT 1
#endif
#ifndef GD_X_NTWR
#define GD_X_NTWR 8
#endif
#ifndef GD_X_STAGGER_NS
#define GD_X_STAGGER_NS 0
#endif
#ifndef GD_X_QRTM
#define GD_X_QRTM 1       // 1: the Hermite sliding-window state (Q_{m-1}, the running R_m) lives in tensor memory next to the Phi/Psi lines
                          // (one 16-word record per x-point) instead of 64 registers per lane: the transforms then run with ~190 registers
#endif
#ifndef GD_X_PROBE
#define GD_X_PROBE 0      // 1: the full barrier of the NEXT inverse job's tile is probed (mbarrier.test_wait) right after the current tile was
                          // packed and the answer consumed a whole transform later, to take the barrier round trip (6 % of the warp
                          // samples) off the critical path.  Measured SLOWER (1.403 vs 1.389 ms at 4a, 1.228 vs 1.217 at 4b): kept as an option
#endif
#ifndef GD_X_TMPIPE
#define GD_X_TMPIPE 0     // moment products (QRTM): 0 = batches of four records, load - wait - compute; B > 0 = batches of B records software-
                          // pipelined (the next batch's tcgen05.ld is issued before the current batch is computed), 1 also with the first
                          // batch requested BEFORE the transform of g_m (the records do not depend on it)
#endif
#ifndef GD_X_TMHOIST
#define GD_X_TMHOIST 0
#endif
#ifndef GD_X_ROTATE
#define GD_X_ROTATE 1     // 1: the tile request of job g (wait for the stage to be released, two bulk copies) is made by warp g % WARPS instead of
                          // always warp 0, so no warp runs systematically behind the others (they meet at every stage's empty barrier).
                          // Measured, same box: x-pass 1.354 -> 1.288 ms at 4a, 1.215 -> 1.124 ms at 4b
#endif
#ifndef GD_X_ALT
#define GD_X_ALT 0        // 1: nx = 256 on one WARP per line (plan 8*8*4, 8 points per lane, 16 warps per SM).  Measured SLOWER (1.72 vs 1.40 ms at 4a:
                          // the second exchange costs more than the extra warps hide; bare transform 1.35 vs 2.53 G/s) -- kept as a tested option
#endif
template <int NX>
struct XGeom {
  static constexpr int FID = (GD_X_ALT && NX == 256) ? NX + GD_FFT_ALT : NX;   // FFT plan ID (fft.cuh)
  static constexpr bool ALT = (FID != NX);
  using G = FftGeom<FID>;
  static constexpr int T = G::T, E = G::E;
  static constexpr int SPLITX = (GD_X_SPLIT && (G::S == 2 || ALT)) ? 1 : 0;   // split (8-byte) FFT exchange: half the buffer, one more stage in flight
                                                                     // (the three-stage plan of nx = 512 pays two split exchanges: measured slower)
  static constexpr int LB = SPLITX ? (NX + NX / G::PADDIV + 2) / 2 : NX + NX / G::PADDIV + 1;   // per-group FFT exchange buffer, complex entries
  static constexpr int KXP = NX / 3 + 1;                    // retained kx count (== Dims::Kx)
#ifndef GD_X_THREADS
#define GD_X_THREADS 256
#endif
  static constexpr int THREADS = ALT ? 512 : GD_X_THREADS;  // 256: one CTA per SM (it owns the SM's tensor memory); 128: two CTAs per SM, each
                                                            // with half the lines, tiles and tensor memory (independent tile rings, so the two
                                                            // warps of a scheduler are never phase-locked) -- measured SLOWER: 1.481 vs 1.424 ms
                                                            // at 4a, 1.301 vs 1.217 ms at 4b; ALT: 16 warps, 4 per scheduler
  static constexpr int CTAS = (THREADS <= 128) ? 2 : 1;     // resident CTAs per SM
  static constexpr int WARPS = THREADS / 32;
  static constexpr int GROUPS = THREADS / T;                // lines per CTA: consecutive (z,y), y fastest
  static constexpr int LD = GROUPS;                         // row of a staged tile [kx][line]; line slot XOR-swizzled with kx
  static constexpr int STAGE = 2 * KXP * LD;                // one stage: the tiles of U and V (P1) for all lines of the CTA
  static constexpr size_t SMEM_CAP = (CTAS == 2 ? 113 : 227) * 1024;   // per CTA
  static constexpr size_t smem_for(int nst) { return ((size_t)GROUPS * LB + (size_t)nst * STAGE + FftTw<FID>::COUNT) * sizeof(cd); }
  static constexpr int NST = (SPLITX && smem_for(4) <= SMEM_CAP) ? 4 : (smem_for(3) <= SMEM_CAP ? 3 : 2);                             // stages in flight (full/empty mbarrier ring), <= 5 (the first NST-1 are Elsasser arrays)
  static constexpr int AHEAD = NST - 1;                      // tiles are requested this many jobs ahead (one stage less -- so that the stage being refilled was
                                                            // released two jobs ago -- measured: no gain at 4a, 1.12 -> 1.18 ms at 4b)
  // stage-1 twiddles held in registers (plans with one stage-1 butterfly per lane): fewer shared-memory reads per transform
  static constexpr int NTWR = (G::S == 2 && E / FftPlan<FID>::R1 == 1) ? GD_X_NTWR : 0;
  static constexpr size_t SMEM = ((size_t)GROUPS * LB + (size_t)NST * STAGE + FftTw<FID>::COUNT) * sizeof(cd);
  // Tensor memory as a thread-private scratchpad (tcgen05.ld/st, shape 32x32b: lane i of a warp owns TMEM lane
  // 32*(warp%4)+i).  Per thread: 8 words per x-point for (Phi_x,Phi_y,Psi_x,Psi_y) and 2 words per x-point for the
  // parked R_{m-2}.  Warps sharing a lane quarter take consecutive column slots.
  // QRTM layout: one 16-word record per x-point, [Phi_x Phi_y Psi_x Psi_y | Ra Rd Qp -] (Ra: the running R_m, Rd: the parked
  // R_{m-2}, Qp: Q_{m-1}), so one x16 load brings everything a moment's products need and one x8 store puts the window back.
  static constexpr bool QRTM = GD_X_QRTM && (16 * E * (THREADS / 128) <= 512);
  static constexpr int TM_PSTR = QRTM ? 16 : 8;             // words per x-point record
  static constexpr int TM_PHI = 0, TM_RD = 8 * E, TM_SLOT = QRTM ? 16 * E : 10 * E;
  static_assert(TM_SLOT * (THREADS / 128) <= 512, "TMEM columns");
  // columns to allocate: the next power of two >= what the CTA uses (>= 32), so that small-nx CTAs sharing an SM, or other
  // tensor-memory users on the device, are not locked out by a 512-column allocation
  static constexpr int tm_pow2(int n) { int p = 32; while (p < n) p *= 2; return p; }
  static constexpr int TM_COLS = tm_pow2(TM_SLOT * (THREADS / 128));
};

// ---- tensor-memory helpers (b32 columns <-> doubles) ------------------------------------------------------
__device__ __forceinline__ void tm_st2(unsigned a, double x) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(a), "r"(__double2loint(x)), "r"(__double2hiint(x)) : "memory");
}
__device__ __forceinline__ void tm_st4(unsigned a, double x, double y) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(__double2loint(x)), "r"(__double2hiint(x)),
               "r"(__double2loint(y)), "r"(__double2hiint(y)) : "memory");
}
__device__ __forceinline__ void tm_st8(unsigned a, double x, double y, double z, double w) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(a), "r"(__double2loint(x)), "r"(__double2hiint(x)),
               "r"(__double2loint(y)), "r"(__double2hiint(y)), "r"(__double2loint(z)), "r"(__double2hiint(z)), "r"(__double2loint(w)), "r"(__double2hiint(w)) : "memory");
}
struct TmRaw16 { unsigned w[16]; };
__device__ __forceinline__ void tm_ld16(unsigned a, TmRaw16& r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]), "=r"(r.w[4]), "=r"(r.w[5]), "=r"(r.w[6]), "=r"(r.w[7]),
                 "=r"(r.w[8]), "=r"(r.w[9]), "=r"(r.w[10]), "=r"(r.w[11]), "=r"(r.w[12]), "=r"(r.w[13]), "=r"(r.w[14]), "=r"(r.w[15]) : "r"(a) : "memory");
}
struct TmRaw2 { unsigned w[2]; };
struct TmRaw4 { unsigned w[4]; };
struct TmRaw8 { unsigned w[8]; };
__device__ __forceinline__ void tm_ld2(unsigned a, TmRaw2& r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r.w[0]), "=r"(r.w[1]) : "r"(a) : "memory");
}
__device__ __forceinline__ void tm_ld4(unsigned a, TmRaw4& r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]) : "r"(a) : "memory");
}
__device__ __forceinline__ void tm_ld8(unsigned a, TmRaw8& r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]), "=r"(r.w[4]), "=r"(r.w[5]), "=r"(r.w[6]), "=r"(r.w[7]) : "r"(a) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ double tm_d(const unsigned* w) { return __hiloint2double((int)w[1], (int)w[0]); }

template <int NX>
__global__ void __launch_bounds__(XGeom<NX>::THREADS, XGeom<NX>::CTAS) k_xpass(Dims d, const cd* __restrict__ D, cd* __restrict__ Eo,
                                                           const cd* __restrict__ tw, const double* __restrict__ cdn,
                                                           const double* __restrict__ cup,
                                                           unsigned long long* __restrict__ maxbits, int nlines) {
  using X = XGeom<NX>;
  using G = FftGeom<X::FID>;
  constexpr int FID = X::FID;
  constexpr int T = X::T, E = X::E;
  constexpr int HX3 = NX / 3, KX = X::KXP;        // == d.hx3, d.Kx (compile-time so per-q range tests fold)
  extern __shared__ cd smem[];
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  const int nblocks = (nlines + X::GROUPS - 1) / X::GROUPS;   // line blocks; a CTA takes blocks blockIdx.x, + gridDim.x, ... (persistent when the grid is smaller)
  cd* buf = smem + FftTw<FID>::COUNT + (size_t)grp * X::LB;
  cd* stages = smem + FftTw<FID>::COUNT + (size_t)X::GROUPS * X::LB;   // NST x [2][KX][LD]: U and V tiles, [kx][line]
  __shared__ unsigned s_tmem_base;
  __shared__ unsigned long long s_full[X::NST], s_empty[X::NST];
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);     // warp-uniform for the compiler (uniform registers)
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < X::NST; ++i) { mbar_init(&s_full[i], 1); mbar_init(&s_empty[i], X::WARPS); }
    // the first NST-1 stages (xi+, xi-: arrays 0/1 and 2/3) are requested right away, by the thread that initialised
    // the barriers, so that they travel while tensor memory is allocated and the twiddle table is staged
    constexpr unsigned TILE_BYTES0 = (unsigned)(X::KXP * X::LD * sizeof(cd));
#pragma unroll
    for (int kn = 0; kn < X::AHEAD; ++kn) {
      const int a = kn == 0 ? 0 : kn == 1 ? 2 : kn == 2 ? 6 : 4;
      mbar_arrive_expect_tx(&s_full[kn], 2u * TILE_BYTES0);
      cd* st = stages + (size_t)kn * X::STAGE;
      const cd* src = D + (size_t)a * d.PD + (size_t)blockIdx.x * (X::KXP * X::LD);
      bulk_g2s(st, src, TILE_BYTES0, &s_full[kn]);
      bulk_g2s(st + X::KXP * X::LD, src + d.PD, TILE_BYTES0, &s_full[kn]);
    }
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(&s_tmem_base)), "r"(X::TM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  fft_load_table<FID>(smem, tw);     // ends with __syncthreads()
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const cd* tws = smem;
  // this warp's TMEM window: lane quarter warp%4, column slot warp/4
  const unsigned tm = __shfl_sync(0xffffffffu, s_tmem_base, 0) + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * X::TM_SLOT);
  const int M = d.M;
  const double bsc = d.bscale;
  cd v[E];
  constexpr bool QRTM = X::QRTM;
  constexpr int PSTR = X::TM_PSTR;
  double Qp[QRTM ? 1 : E], Ra[QRTM ? 1 : E];   // Hermite sliding window (registers unless QRTM); Qp doubles as the {xi+,w-} accumulator of the Elsasser part

  // Producer (lane 0 of warp 0): the tiles of arrays a, a+1 for the lines of this CTA.  D[a][line block][kx][LD] is laid
  // out so that a CTA's tile is ONE contiguous run (line slot XOR-swizzled with kx against bank conflicts): one bulk async copy (TMA engine) per array into
  // stage kn % NST; completion on s_full, reuse gated by s_empty.
  auto produce = [&](int kn, int a, int blk) {
    const int sn = kn % X::NST;
    if (kn >= X::NST) mbar_wait(&s_empty[sn], (unsigned)((kn / X::NST - 1) & 1));
    if ((threadIdx.x & 31) == 0) {
      constexpr unsigned TILE_BYTES = (unsigned)(KX * X::LD * sizeof(cd));
      mbar_arrive_expect_tx(&s_full[sn], 2u * TILE_BYTES);
      cd* st = stages + (size_t)sn * X::STAGE;
      const cd* src = D + (size_t)a * d.PD + (size_t)blk * (KX * X::LD);
      bulk_g2s(st, src, TILE_BYTES, &s_full[sn]);
      bulk_g2s(st + KX * X::LD, src + d.PD, TILE_BYTES, &s_full[sn]);
    }
    __syncwarp();
  };
  // Job list of one line.  Kinds 0..3 are the inverse transforms of xi+, xi-, w-, w+; kind 4+m that of g_m.
  // After kind 3 and after every second moment a forward job (pair of real lines) follows.  Inverse transforms
  // run as conj(FFT(conj Z)) so that ONE forward-FFT code instance serves every job (instruction cache).
  auto src_array = [&](int kind) { return kind == 0 ? 0 : kind == 1 ? 2 : kind == 2 ? 6 : kind == 3 ? 4 : 8 + 2 * (kind - 4); };
  const int nkinds = 4 + M;
  double gmax = 0.0;
  bool tile_ready = false;         // the next inverse job's tile was already seen complete (GD_X_PROBE)
  TmRaw16 pre[GD_X_TMPIPE > 0 ? GD_X_TMPIPE : 1];   // prefetched records of the moment products (GD_X_TMPIPE)
  bool hoisted = false;
  cd twr[X::NTWR > 0 ? X::NTWR : 1];
  if constexpr (X::NTWR > 0) fft_load_stage1_twiddles<FID, X::NTWR>(twr, t, tws);
#if GD_X_STAGGER_NS > 0
  if (warp >= X::WARPS / 2) __nanosleep(GD_X_STAGGER_NS);
#endif
  // Persistent form: the stage ring runs on across line blocks (global job index g0 + kind), so the first tiles of the next
  // block travel during the last jobs of the current one -- with few fields per line (RMHD only: 4 inverse + 1 forward job)
  // a CTA per block spends a third of its life on the start-up round trip (config 4b).
  for (int blk = blockIdx.x, g0 = 0; blk < nblocks; blk += gridDim.x, g0 += nkinds) {
  const int line = blk * X::GROUPS + grp;
  const bool active = line < nlines;
  const size_t base = (size_t)(active ? line : 0) * d.Kxe;    // (z*ny + y)*Kxp  (output arrays E, kx fastest, padded rows)
  int kind = 0;
  bool fwd = false;                // the job about to run is a forward transform of the pair held in v
  bool tail_done = (M == 0);
  int e0 = 0, e1 = 1;
  double gblk = 0.0;
  for (;;) {
    if (!fwd) {
      if (kind == nkinds) {
        if (tail_done) break;
        // R_{M-1} is complete (up_{M-1} = 0 after the closure was folded into dn): flush the last pair / single
        tail_done = true;
        fwd = true;
        const bool pair = (((M - 1) & 1) == 1);
        if constexpr (QRTM) {
          tm_wait_st();
#pragma unroll
          for (int q0 = 0; q0 < E; q0 += 4) {
            TmRaw4 rr[4];
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) tm_ld4(tm + PSTR * (q0 + jj) + 8, rr[jj]);       // (Ra, Rd)
            tm_wait_ld();
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) v[q0 + jj] = pair ? cmake(tm_d(rr[jj].w + 2), tm_d(rr[jj].w)) : cmake(tm_d(rr[jj].w), 0.0);
          }
        } else if (pair) {
          tm_wait_st();
#pragma unroll
          for (int q0 = 0; q0 < E; q0 += 4) {
            TmRaw2 rd[4];
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) tm_ld2(tm + X::TM_RD + 2 * (q0 + jj), rd[jj]);
            tm_wait_ld();
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) v[q0 + jj] = cmake(tm_d(rd[jj].w), Ra[q0 + jj]);
          }
        } else {
#pragma unroll
          for (int q = 0; q < E; ++q) v[q] = cmake(Ra[q], 0.0);
        }
        if (pair) { e0 = 2 + M - 2; e1 = 2 + M - 1; }
        else { e0 = 2 + M - 1; e1 = -1; }
      } else {
        // wait for the staged tiles and pack conj(Z), Z = Fx + i Fy.  P1 delivers U = kx f~ + (df/dy)~ and
        // V = (df/dy)~ - kx f~, so that Z(kx) = i U(kx) and Z(-kx) = i conj(V(kx)) (Hermitian completion) need no arithmetic
        const int g = g0 + kind;
        const int sc = g % X::NST;
        if (!tile_ready) mbar_wait(&s_full[sc], (unsigned)((g / X::NST) & 1));
        const cd* pU = stages + (size_t)sc * X::STAGE;            // element n of this line: pU[n * LD + (grp ^ (n & (LD-1)))]
        const cd* pV = pU + (size_t)KX * X::LD;
#pragma unroll
        for (int q = 0; q < E; ++q) {
          const int n = t + T * q;
          cd z = cmake(0.0, 0.0);
          if (T * q <= HX3 && n <= HX3) {                       // first test is compile-time per q
            const cd u = pU[n * X::LD + (grp ^ (n & (X::LD - 1)))];
            z = cmake(n == 0 ? 0.0 : -u.y, -u.x);               // conj(i U); the kx = 0 entry of a real line is real
          } else if (T * q + T - 1 >= NX - HX3 && n >= NX - HX3) {
            const int c = NX - n;
            const cd w = pV[c * X::LD + (grp ^ (c & (X::LD - 1)))];
            z = cmake(w.y, -w.x);                               // conj(i conj(V)) = -i V
          }
          v[q] = z;
        }
        __syncwarp();                   // every lane of the warp has consumed the stage
        if ((threadIdx.x & 31) == 0) mbar_arrive(&s_empty[sc]);
#if GD_X_PROBE
        // (this warp has seen the previous use of that stage complete, so the parity test cannot alias)
        tile_ready = mbar_test_wait(&s_full[(g + 1) % X::NST], (unsigned)(((g + 1) / X::NST) & 1));
#endif
        if (warp == (GD_X_ROTATE ? (g & (X::WARPS - 1)) : 0)) {   // the producer role rotates over the warps: no warp lags the others by the request's cost
          const int kn = kind + X::AHEAD;                       // job AHEAD ahead: of this block, or of the CTA's next one
          if (kn < nkinds) produce(g0 + kn, src_array(kn), blk);
          else if (blk + (int)gridDim.x < nblocks) produce(g0 + kn, src_array(kn - nkinds), blk + (int)gridDim.x);
        }
      }
    }

#if GD_X_TMPIPE > 0 && GD_X_TMHOIST
    if (QRTM && !fwd && kind >= 4) {       // the first records of this moment's products: requested now, they arrive during the transform
      tm_wait_st();
#pragma unroll
      for (int jj = 0; jj < GD_X_TMPIPE; ++jj) tm_ld16(tm + PSTR * jj, pre[jj]);
      hoisted = true;
    }
#endif
    if constexpr (X::SPLITX && X::NTWR > 0) fft_lanes_fwd_rt_split<FID, X::NTWR>(v, t, reinterpret_cast<double*>(buf), tws, twr);
    else if constexpr (X::SPLITX) fft_lanes_split<FID, -1>(v, t, reinterpret_cast<double*>(buf), tws);
    else if constexpr (X::NTWR > 0) fft_lanes_fwd_rt<FID, X::NTWR>(v, t, buf, tws, twr);
    else fft_lanes<FID, -1>(v, t, buf, tws);

    if (fwd) {
      // separate the two real lines' spectra by Hermitian symmetry, keep kx <= nx/3, store.  The partner X[nx - c] of
      // c = t + T q sits in lane (T - t) % T of the same group at register E-1-q (lane 0: its own register (E - q) % E),
      // so it comes by warp shuffles -- no shared-memory round trip.
      fwd = false;
      {
        cd* p0 = Eo + (size_t)e0 * d.PE + base;
        cd* p1 = Eo + (size_t)(e1 < 0 ? e0 : e1) * d.PE + base;
        const int partner = (T - t) & (T - 1);
#pragma unroll
        for (int q = 0; q < E; ++q) {
          if (T * q <= HX3) {                                   // compile-time: some lane of this q holds a retained kx
            const int c = t + T * q;
            cd z2;
            z2.x = __shfl_sync(0xffffffffu, v[E - 1 - q].x, partner, T);
            z2.y = __shfl_sync(0xffffffffu, v[E - 1 - q].y, partner, T);
            if (t == 0) z2 = v[(E - q) & (E - 1)];
            const cd z1 = v[q];
            if (active && c <= HX3) {
              st_cd(p0 + c, cmake(0.5 * (z1.x + z2.x), 0.5 * (z1.y - z2.y)));
              if (e1 >= 0) st_cd(p1 + c, cmake(0.5 * (z1.y + z2.y), -0.5 * (z1.x - z2.x)));
            }
          }
        }
      }
      continue;
    }

    // inverse job done: v[q] = (df/dx, -df/dy) at x = t + T q   (conjugated output)
    if (kind == 0 || kind == 1) {          // xi+ / xi-: park the derivative lines in tensor memory
#pragma unroll
      for (int q = 0; q < E; ++q) tm_st4(tm + X::TM_PHI + PSTR * q + 4 * kind, v[q].x, -v[q].y);
    } else if (kind == 2) {                // w-: {xi+, w-}
      tm_wait_st();
#pragma unroll
      for (int q0 = 0; q0 < E; q0 += 4) {
        TmRaw4 r[4];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) tm_ld4(tm + X::TM_PHI + PSTR * (q0 + jj), r[jj]);
        tm_wait_ld();
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          const double xpx = tm_d(r[jj].w), xpy = tm_d(r[jj].w + 2);
          const double acc = xpx * (-v[q0 + jj].y) - xpy * v[q0 + jj].x;
          if constexpr (QRTM) tm_st2(tm + PSTR * (q0 + jj) + 12, acc);
          else Qp[q0 + jj] = acc;
        }
      }
    } else if (kind == 3) {                // w+: A = {xi+,w-} + {xi-,w+}, B = {xi+,xi-}; Phi/Psi lines; CFL max
      if constexpr (QRTM) tm_wait_st();
#pragma unroll
      for (int q0 = 0; q0 < E; q0 += 4) {
        TmRaw8 r[4];
        TmRaw2 rq[4];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) tm_ld8(tm + X::TM_PHI + PSTR * (q0 + jj), r[jj]);
        if constexpr (QRTM) {
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) tm_ld2(tm + PSTR * (q0 + jj) + 12, rq[jj]);
        }
        tm_wait_ld();
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          const int q = q0 + jj;
          const cd xp = cmake(tm_d(r[jj].w), tm_d(r[jj].w + 2)), xm = cmake(tm_d(r[jj].w + 4), tm_d(r[jj].w + 6));
          double acc;
          if constexpr (QRTM) acc = tm_d(rq[jj].w); else acc = Qp[q];
          const double a = acc + (xm.x * (-v[q].y) - xm.y * v[q].x);
          const double b = xp.x * xm.y - xp.y * xm.x;
          v[q] = cmake(a, bsc * b);                                          // (A, bscale*B): see Dims::bscale
          const cd phi = cmake(0.5 * (xp.x + xm.x), 0.5 * (xp.y + xm.y));   // grad Phi, Phi = (xi+ + xi-)/2
          const cd psi = cmake(0.5 * (xp.x - xm.x), 0.5 * (xp.y - xm.y));   // grad Psi
          if constexpr (QRTM) {
            tm_st8(tm + PSTR * q, phi.x, phi.y, psi.x, psi.y);
            tm_st8(tm + PSTR * q + 8, 0.0, 0.0, 0.0, 0.0);                   // Ra = Rd = Qp = 0
          } else {
            tm_st4(tm + X::TM_PHI + 8 * q, phi.x, phi.y);
            tm_st4(tm + X::TM_PHI + 8 * q + 4, psi.x, psi.y);
            Qp[q] = 0.0; Ra[q] = 0.0;
          }
          gblk = fmax(gblk, phi.x * phi.x + phi.y * phi.y);
        }
      }
      fwd = true; e0 = 0; e1 = 1;
    } else {                               // g_m: P_m, Q_m and the sliding window R_m = -P_m + dn_m Q_{m-1} + up_m Q_{m+1}
      const int m = kind - 4;
      const double dn = cdn[m];
      const double upp = (m > 0) ? cup[m - 1] : 0.0;
      const bool emit = (m >= 1) && (((m - 1) & 1) == 1);     // R_{m-1} completes the pair (R_{m-2}, R_{m-1})
      tm_wait_st();
      if constexpr (QRTM && GD_X_TMPIPE > 0) {
        constexpr int B = GD_X_TMPIPE;
        if (!(GD_X_TMHOIST && hoisted)) {
#pragma unroll
          for (int jj = 0; jj < B; ++jj) tm_ld16(tm + PSTR * jj, pre[jj]);
        }
        hoisted = false;
#pragma unroll
        for (int q0 = 0; q0 < E; q0 += B) {
          TmRaw16 r[B];
          tm_wait_ld();
#pragma unroll
          for (int jj = 0; jj < B; ++jj) r[jj] = pre[jj];
          if (q0 + B < E) {
#pragma unroll
            for (int jj = 0; jj < B; ++jj) tm_ld16(tm + PSTR * (q0 + B + jj), pre[jj]);
          }
#pragma unroll
          for (int jj = 0; jj < B; ++jj) {
            const int q = q0 + jj;
            const double phx = tm_d(r[jj].w), phy = tm_d(r[jj].w + 2), psx = tm_d(r[jj].w + 4), psy = tm_d(r[jj].w + 6);
            const double ra = tm_d(r[jj].w + 8), rd = tm_d(r[jj].w + 10), qp = tm_d(r[jj].w + 12);
            const double gx = v[q].x, gy = -v[q].y;
            const double P = phx * gy - phy * gx;               // {Phi, g_m}
            const double Q = psx * gy - psy * gx;               // {Psi, g_m}
            const double rfin = ra + upp * Q;                   // R_{m-1} complete
            if (emit) v[q] = cmake(rd, rfin);
            tm_st8(tm + PSTR * q + 8, dn * qp - P, rfin, Q, 0.0);
          }
        }
      } else if constexpr (QRTM) {
#pragma unroll
        for (int q0 = 0; q0 < E; q0 += 4) {
          TmRaw16 r[4];
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) tm_ld16(tm + PSTR * (q0 + jj), r[jj]);
          tm_wait_ld();
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) {
            const int q = q0 + jj;
            const double phx = tm_d(r[jj].w), phy = tm_d(r[jj].w + 2), psx = tm_d(r[jj].w + 4), psy = tm_d(r[jj].w + 6);
            const double ra = tm_d(r[jj].w + 8), rd = tm_d(r[jj].w + 10), qp = tm_d(r[jj].w + 12);
            const double gx = v[q].x, gy = -v[q].y;
            const double P = phx * gy - phy * gx;               // {Phi, g_m}
            const double Q = psx * gy - psy * gx;               // {Psi, g_m}
            const double rfin = ra + upp * Q;                   // R_{m-1} complete
            if (emit) v[q] = cmake(rd, rfin);
            tm_st8(tm + PSTR * q + 8, dn * qp - P, rfin, Q, 0.0);   // (Ra, Rd, Qp): the window moves on; Rd is dead after an emit
          }
        }
      } else
#pragma unroll
      for (int q0 = 0; q0 < E; q0 += 4) {
        TmRaw8 r[4];
        TmRaw2 rd[4];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) tm_ld8(tm + X::TM_PHI + 8 * (q0 + jj), r[jj]);
        if (emit) {
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) tm_ld2(tm + X::TM_RD + 2 * (q0 + jj), rd[jj]);
        }
        tm_wait_ld();
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          const int q = q0 + jj;
          const double phx = tm_d(r[jj].w), phy = tm_d(r[jj].w + 2), psx = tm_d(r[jj].w + 4), psy = tm_d(r[jj].w + 6);
          const double gx = v[q].x, gy = -v[q].y;
          const double P = phx * gy - phy * gx;               // {Phi, g_m}
          const double Q = psx * gy - psy * gx;               // {Psi, g_m}
          const double rfin = Ra[q] + upp * Q;                // R_{m-1} complete
          Ra[q] = dn * Qp[q] - P;
          Qp[q] = Q;
          if (emit) v[q] = cmake(tm_d(rd[jj].w), rfin);
          else tm_st2(tm + X::TM_RD + 2 * q, rfin);
        }
      }
      if (emit) { fwd = true; e0 = 2 + m - 2; e1 = 2 + m - 1; }
    }
    ++kind;
  }
  if (active) gmax = fmax(gmax, gblk);
  }
  if (maxbits != nullptr) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) gmax = fmax(gmax, __shfl_xor_sync(0xffffffffu, gmax, o));
    if ((threadIdx.x & 31) == 0) atomicMax(maxbits, (unsigned long long)__double_as_longlong(gmax));
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem_base), "r"(X::TM_COLS) : "memory");
}

// FFT plan ID of the x transforms (selects the stage twiddle table api.cu uploads)
int xpass_fft_plan_id(int nx) {
  switch (nx) {
    case 8: return XGeom<8>::FID; case 16: return XGeom<16>::FID; case 32: return XGeom<32>::FID; case 64: return XGeom<64>::FID;
    case 128: return XGeom<128>::FID; case 256: return XGeom<256>::FID; case 512: return XGeom<512>::FID;
    default: return 0;
  }
}
// lines per x-pass CTA (the block size of the D layout)
int xpass_lines_per_cta(int nx) {
  switch (nx) {
    case 8: return XGeom<8>::GROUPS; case 16: return XGeom<16>::GROUPS; case 32: return XGeom<32>::GROUPS;
    case 64: return XGeom<64>::GROUPS; case 128: return XGeom<128>::GROUPS; case 256: return XGeom<256>::GROUPS;
    case 512: return XGeom<512>::GROUPS;
    default: return 0;
  }
}

#ifndef GD_X_PERSIST_MAX_KINDS
#define GD_X_PERSIST_MAX_KINDS 1000000   // persistent CTAs (one per SM) when a line has at most this many inverse jobs (4 + M).  Measured:
                                         // 4b (5 jobs per line) 1.44 -> 1.20 ms; 4a (53 jobs) 1.397 -> 1.386 ms -- so always on
#endif
cudaError_t launch_xpass(const Dims& d, const cd* D, cd* Eo, const cd* tw, const double* cdn, const double* cup,
                         unsigned long long* maxbits, int num_sms, cudaStream_t st, bool prepare_only) {
  const int nlines = d.ny * d.nz;
  const bool persist = 4 + d.M <= GD_X_PERSIST_MAX_KINDS;
#define XCASE(NN)                                                                                             \
  {                                                                                                           \
    using X = XGeom<NN>;                                                                                      \
    if (prepare_only) return cudaFuncSetAttribute(k_xpass<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)X::SMEM); \
    const int nb = (nlines + X::GROUPS - 1) / X::GROUPS;                                                        \
    const int cap = X::CTAS * num_sms;                                                                          \
    k_xpass<NN><<<(persist && nb > cap) ? cap : nb, X::THREADS, X::SMEM, st>>>(d, D, Eo, tw, cdn, cup, maxbits, nlines); \
  }
  switch (d.nx) {
    case 8: XCASE(8) break; case 16: XCASE(16) break; case 32: XCASE(32) break; case 64: XCASE(64) break;
    case 128: XCASE(128) break; case 256: XCASE(256) break; case 512: XCASE(512) break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}
