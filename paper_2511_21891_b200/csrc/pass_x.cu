// pass_x.cu -- P2, the fused row pass of the RHS pipeline (one lane group per (y,z) line).
//
// For every source field f in {xi+, xi-, w+, w-, g_m} the pass reads the two half-lines
// f~(kx; y,z) and (df/dy)~(kx; y,z) that P1 wrote (retained kx only), forms
//     Z(kx) = i kx f~(kx) + i (df/dy)~(kx)          for kx >= 0       (Eq. 10)
//     Z(-kx) = conj(i kx f~) + i conj((df/dy)~)                        (Hermitian completion)
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

template <int NX>
struct XGeom {
  using G = FftGeom<NX>;
  static constexpr int T = G::T, E = G::E;
  static constexpr int LB = NX + NX / G::PADDIV + 1;        // line buffer (FFT exchange + unpack), complex entries
  static constexpr int KXP = NX / 3 + 1;                    // retained kx count (== Dims::Kx)
  static constexpr int STG = 2 * KXP;                       // staging buffer: the two half-lines (f, df/dy) of the NEXT field
  static constexpr int PER_GROUP = LB + STG;
  static constexpr int THREADS = 256;                       // 8 warps, one CTA per SM (it owns all 512 TMEM columns)
  static constexpr int GROUPS = THREADS / T;
  static constexpr size_t SMEM = ((size_t)GROUPS * PER_GROUP + FftTw<NX>::COUNT) * sizeof(cd);
  // Tensor memory as a thread-private scratchpad (tcgen05.ld/st, shape 32x32b: lane i of a warp owns TMEM lane
  // 32*(warp%4)+i).  Per thread: 8 words per x-point for (Phi_x,Phi_y,Psi_x,Psi_y) and 2 words per x-point for the
  // parked R_{m-2}.  Warps sharing a lane quarter take consecutive column slots.
  static constexpr int TM_PHI = 0, TM_RD = 8 * E, TM_SLOT = 10 * E;
  static_assert(TM_SLOT * (THREADS / 128) <= 512, "TMEM columns");
};

// ---- tensor-memory helpers (b32 columns <-> doubles) ------------------------------------------------------
__device__ __forceinline__ void tm_st2(unsigned a, double x) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(a), "r"(__double2loint(x)), "r"(__double2hiint(x)) : "memory");
}
__device__ __forceinline__ void tm_st4(unsigned a, double x, double y) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(__double2loint(x)), "r"(__double2hiint(x)),
               "r"(__double2loint(y)), "r"(__double2hiint(y)) : "memory");
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
__global__ void __launch_bounds__(XGeom<NX>::THREADS, 1) k_xpass(Dims d, const cd* __restrict__ D, cd* __restrict__ Eo,
                                                        const cd* __restrict__ tw, const double* __restrict__ cdn,
                                                        const double* __restrict__ cup,
                                                        unsigned long long* __restrict__ maxbits, int nlines) {
  using X = XGeom<NX>;
  using G = FftGeom<NX>;
  constexpr int T = X::T, E = X::E;
  extern __shared__ cd smem[];
  const int grp = threadIdx.x / T, t = threadIdx.x % T;
  const int line = blockIdx.x * X::GROUPS + grp;
  cd* buf = smem + FftTw<NX>::COUNT + (size_t)grp * X::PER_GROUP;
  __shared__ unsigned s_tmem_base;
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(&s_tmem_base)), "r"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  fft_load_table<NX>(smem, tw);      // ends with __syncthreads()
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const cd* tws = smem;
  // this warp's TMEM window: lane quarter warp%4, column slot warp/4
  const unsigned tm = s_tmem_base + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * X::TM_SLOT);
  const bool active = line < nlines;
  const size_t base = (size_t)(active ? line : 0) * d.Kx;     // (z*ny + y)*Kx
  const int hx3 = d.hx3;
  cd v[E];

  cd* sStage = buf + X::LB;        // [0,Kx): f~(kx), [Kx,2Kx): (df/dy)~(kx) of the field being fetched
  // asynchronous fetch (cp.async, 16 B per lane) of the two half-lines of array a, a+1 into the staging buffer
  auto fetch = [&](int a) {
    if (active) {
      const cd* pf = D + (size_t)a * d.PD + base;
      const unsigned sbase = (unsigned)__cvta_generic_to_shared(sStage);
      for (int c = t; c < 2 * d.Kx; c += T) {
        const cd* src = (c < d.Kx) ? pf + c : pf + d.PD + (c - d.Kx);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sbase + 16u * (unsigned)c), "l"(src) : "memory");
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  // wait for the staged half-lines, pack Z = Fx + i Fy on the full kx line into v, then start fetching array `next`
  auto load_pack = [&](int next) {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();
    const cd* pf = sStage;
    const cd* pfy = sStage + d.Kx;
#pragma unroll
    for (int q = 0; q < E; ++q) {
      const int n = t + T * q;
      cd z = cmake(0.0, 0.0);
      if (active) {
        if (n <= hx3) {
          cd f = pf[n], fy = pfy[n];
          if (n == 0) { f.y = 0.0; fy.y = 0.0; }
          const double kx = d.kx0 * n;
          // Fx = i kx f = (-kx f.y, kx f.x);  Z = Fx + i Fy
          z = cmake(-kx * f.y - fy.y, kx * f.x + fy.x);
        } else if (n >= NX - hx3) {
          const int c = NX - n;
          const cd f = pf[c], fy = pfy[c];
          const double kx = d.kx0 * c;
          // conj(Fx) + i conj(Fy) = (-kx f.y + fy.y, -kx f.x + fy.x)
          z = cmake(-kx * f.y + fy.y, -kx * f.x + fy.x);
        }
      }
      v[q] = z;
    }
    __syncwarp();                   // every lane has consumed the staging buffer
    if (next >= 0) fetch(next);
  };
  // forward-transform v = (U + i V) of two real lines and store U~, V~ (kx <= nx/3) to arrays e0, e1 (e1 < 0: skip)
  auto fwd_store = [&](int e0, int e1) {
    fft_lanes<NX, -1>(v, t, buf, tws);
#pragma unroll
    for (int q = 0; q < E; ++q) buf[G::pad(t + T * q)] = v[q];
    __syncwarp();
    if (active) {
      cd* p0 = Eo + (size_t)e0 * d.PD + base;
      cd* p1 = Eo + (size_t)(e1 < 0 ? e0 : e1) * d.PD + base;
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int c = t + T * q;
        if (c <= hx3) {
          const cd z1 = buf[G::pad(c)], z2 = buf[G::pad((NX - c) & (NX - 1))];
          st_cd(p0 + c, cmake(0.5 * (z1.x + z2.x), 0.5 * (z1.y - z2.y)));
          if (e1 >= 0) st_cd(p1 + c, cmake(0.5 * (z1.y + z2.y), -0.5 * (z1.x - z2.x)));
        }
      }
    }
    __syncwarp();
  };

  // ---- Elsasser part: A, B --------------------------------------------------------------------
  fetch(0);
  load_pack(2);                                   // xi+   (and start fetching xi-)
  fft_lanes<NX, +1>(v, t, buf, tws);
#pragma unroll
  for (int q = 0; q < E; ++q) tm_st4(tm + X::TM_PHI + 8 * q, v[q].x, v[q].y);
  load_pack(6);                                   // xi-   (fetch w-)
  fft_lanes<NX, +1>(v, t, buf, tws);
#pragma unroll
  for (int q = 0; q < E; ++q) tm_st4(tm + X::TM_PHI + 8 * q + 4, v[q].x, v[q].y);
  double A[E];
  load_pack(4);                                   // w-    (fetch w+)
  fft_lanes<NX, +1>(v, t, buf, tws);
  tm_wait_st();
#pragma unroll
  for (int q0 = 0; q0 < E; q0 += 4) {
    TmRaw4 r[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) tm_ld4(tm + X::TM_PHI + 8 * (q0 + j), r[j]);
    tm_wait_ld();
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const double xpx = tm_d(r[j].w), xpy = tm_d(r[j].w + 2);
      A[q0 + j] = xpx * v[q0 + j].y - xpy * v[q0 + j].x;          // {xi+, w-}
    }
  }
  load_pack(d.M > 0 ? 8 : -1);                    // w+    (fetch g_0)
  fft_lanes<NX, +1>(v, t, buf, tws);
  double gmax = 0.0;
#pragma unroll
  for (int q0 = 0; q0 < E; q0 += 4) {
    TmRaw8 r[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) tm_ld8(tm + X::TM_PHI + 8 * (q0 + j), r[j]);
    tm_wait_ld();
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int q = q0 + j;
      const cd xp = cmake(tm_d(r[j].w), tm_d(r[j].w + 2)), xm = cmake(tm_d(r[j].w + 4), tm_d(r[j].w + 6));
      const double a = A[q] + (xm.x * v[q].y - xm.y * v[q].x);      // + {xi-, w+}
      const double b = xp.x * xm.y - xp.y * xm.x;                   // {xi+, xi-}
      v[q] = cmake(a, b);
      const cd phi = cmake(0.5 * (xp.x + xm.x), 0.5 * (xp.y + xm.y));   // grad Phi, Phi = (xi+ + xi-)/2
      const cd psi = cmake(0.5 * (xp.x - xm.x), 0.5 * (xp.y - xm.y));   // grad Psi
      tm_st4(tm + X::TM_PHI + 8 * q, phi.x, phi.y);
      tm_st4(tm + X::TM_PHI + 8 * q + 4, psi.x, psi.y);
      gmax = fmax(gmax, phi.x * phi.x + phi.y * phi.y);
    }
  }
  if (maxbits != nullptr) {
    if (!active) gmax = 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) gmax = fmax(gmax, __shfl_xor_sync(0xffffffffu, gmax, o));
    if ((threadIdx.x & 31) == 0) atomicMax(maxbits, (unsigned long long)__double_as_longlong(gmax));
  }
  fwd_store(0, 1);

  // ---- Hermite part: R_m with a sliding window over m ------------------------------------------
  const int M = d.M;
  if (M > 0) {
    double Qp[E], Ra[E];
#pragma unroll
    for (int q = 0; q < E; ++q) { Qp[q] = 0.0; Ra[q] = 0.0; }
    for (int m = 0; m < M; ++m) {
      load_pack(m + 1 < M ? 8 + 2 * (m + 1) : -1);  // g_m  (fetch g_{m+1})
      fft_lanes<NX, +1>(v, t, buf, tws);
      const double dn = cdn[m];
      const double upp = (m > 0) ? cup[m - 1] : 0.0;
      const bool emit = (m >= 1) && (((m - 1) & 1) == 1);     // R_{m-1} completes the pair (R_{m-2}, R_{m-1})
      tm_wait_st();                                           // earlier tensor-memory stores are visible
#pragma unroll
      for (int q0 = 0; q0 < E; q0 += 4) {
        TmRaw8 r[4];
        TmRaw2 rd[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) tm_ld8(tm + X::TM_PHI + 8 * (q0 + j), r[j]);
        if (emit) {
#pragma unroll
          for (int j = 0; j < 4; ++j) tm_ld2(tm + X::TM_RD + 2 * (q0 + j), rd[j]);
        }
        tm_wait_ld();
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int q = q0 + j;
          const double phx = tm_d(r[j].w), phy = tm_d(r[j].w + 2), psx = tm_d(r[j].w + 4), psy = tm_d(r[j].w + 6);
          const double gx = v[q].x, gy = v[q].y;
          const double P = phx * gy - phy * gx;               // {Phi, g_m}
          const double Q = psx * gy - psy * gx;               // {Psi, g_m}
          const double rfin = Ra[q] + upp * Q;                // R_{m-1} complete
          Ra[q] = dn * Qp[q] - P;
          Qp[q] = Q;
          if (emit) v[q] = cmake(tm_d(rd[j].w), rfin);
          else tm_st2(tm + X::TM_RD + 2 * q, rfin);
        }
      }
      if (emit) fwd_store(2 + m - 2, 2 + m - 1);
    }
    // R_{M-1} is complete (up_{M-1} = 0 after the closure was folded into dn)
    if (((M - 1) & 1) == 1) {
      tm_wait_st();
#pragma unroll
      for (int q0 = 0; q0 < E; q0 += 4) {
        TmRaw2 rd[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) tm_ld2(tm + X::TM_RD + 2 * (q0 + j), rd[j]);
        tm_wait_ld();
#pragma unroll
        for (int j = 0; j < 4; ++j) v[q0 + j] = cmake(tm_d(rd[j].w), Ra[q0 + j]);
      }
      fwd_store(2 + M - 2, 2 + M - 1);
    } else {
#pragma unroll
      for (int q = 0; q < E; ++q) v[q] = cmake(Ra[q], 0.0);
      fwd_store(2 + M - 1, -1);
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem_base), "r"(512) : "memory");
}

cudaError_t launch_xpass(const Dims& d, const cd* D, cd* Eo, const cd* tw, const double* cdn, const double* cup,
                         unsigned long long* maxbits, cudaStream_t st, bool prepare_only) {
  const int nlines = d.ny * d.nz;
#define XCASE(NN)                                                                                             \
  {                                                                                                           \
    using X = XGeom<NN>;                                                                                      \
    if (prepare_only) return cudaFuncSetAttribute(k_xpass<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)X::SMEM); \
    k_xpass<NN><<<(nlines + X::GROUPS - 1) / X::GROUPS, X::THREADS, X::SMEM, st>>>(d, D, Eo, tw, cdn, cup, maxbits, nlines); \
  }
  switch (d.nx) {
    case 8: XCASE(8) break; case 16: XCASE(16) break; case 32: XCASE(32) break; case 64: XCASE(64) break;
    case 128: XCASE(128) break; case 256: XCASE(256) break; case 512: XCASE(512) break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}
