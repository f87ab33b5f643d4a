// cspt_euler.cuh -- Eulerian stage: FGC (Eq. (8) + pressureless HLL flux) and SUE (Eq. (4)),
// PAPER.md:45-50, :70-78, :112-113; readings G9-G14, with the CFL signal speed of U^{n+1}
// (G15) as epilogue.
//
// One CTA owns a TX x TY column of cells (one thread per cell of a plane) and streams along z
// (2.5-D): per plane one TMA box of U^n (halo 2 in x/y) and one of (U~, xi) (halo 1) land in a
// 2-stage shared-memory ring.  Per cell and axis the two one-sided flux parts
//     FP_i = max(u^L_i,0) U^L_i   (leaves through the + face),   FM_i = min(u^R_i,0) U^R_i   (through the - face)
// are computed ONCE (F_{i+1/2} = FP_i + FM_{i+1}) and handed to the x and y neighbours through
// shared memory (the parts of the halo columns / rows are computed by the first / the last warps);
// along z the thread keeps FP of the previous plane in registers and finishes cell p-1 when FM of
// plane p is known.  The z+ neighbour U^n(p+1) of the own column is read from the other ring stage.
// This layout is the fp32 default for the HLL flux (4 CTAs of 64 registers per SM); fp64, and the LF / HLLC fluxes in
// both precisions, run the row layout of cspt_euler2.cuh (profiles/r2_kernels.md has the A/B numbers).
#pragma once
#include "cspt_kernels.cuh"
#include "cspt_tma.cuh"

namespace cspt {

// minmod(a, b) is the median of {a, b, 0}: four FMNMX in fp32 instead of two compares, two selects and a product
// (where a or b is zero, or the signs differ, the median is that zero)
template <class T>
__device__ __forceinline__ T minmod_fast(T a, T b) {
  return fmaxf(fminf(a, b), fminf(fmaxf(a, b), 0.f));
}
// fp64: the sign agreement is tested on the high words (integer pipe instead of a DMUL and a DSETP on the FP64
// pipe); where a or b is zero the smaller magnitude r is that zero, so the result is the same
template <>
__device__ __forceinline__ double minmod_fast<double>(double a, double b) {
  double r = fabs(a) < fabs(b) ? a : b;
  return (__double2hiint(a) ^ __double2hiint(b)) >= 0 ? r : 0.0;
}

// One-sided flux parts of one cell along axis d.  Uc/Um/Up: U^n of the cell and of its -/+
// neighbours; hf = U^{n+1/2} = (U^n + U~)/2 (G10); xi = xi_d of the cell.
// van Leer's harmonic limiter 2ab/(a+b) for ab > 0, else 0 ("different TVD-limiters").
template <class T>
__device__ __forceinline__ T vanleer_fast(T a, T b) {
  T ab = a * b, sum = a + b;
  bool ok = ab > (T)0 && fabs(sum) > (sizeof(T) == 8 ? (T)1e-300 : (T)1e-36);      // keeps the reciprocal seed finite
  T r = ((T)2 * ab) * Fast<T>::rcp(ok ? sum : (T)1);
  return ok ? r : (T)0;
}
// TVD slope of Eq. (8): LIM 0 = minmod (reading G12), 1 = van Leer
template <class T, int LIM>
__device__ __forceinline__ T tvd_slope(T a, T b) {
  return LIM == 1 ? vanleer_fast<T>(a, b) : minmod_fast<T>(a, b);
}

// sign tests on the high word (integer pipe instead of an FP64 compare); a subnormal double counts as zero
template <class T> __device__ __forceinline__ bool is_pos(T x) { return x > (T)0; }
template <class T> __device__ __forceinline__ bool is_neg(T x) { return x < (T)0; }
template <> __device__ __forceinline__ bool is_pos<double>(double x) { return __double2hiint(x) > 0; }
template <> __device__ __forceinline__ bool is_neg<double>(double x) { return __double2hiint(x) < 0; }

template <class T, int WANT, int LIM>   // WANT bit 0: FP, bit 1: FM
__device__ __forceinline__ void flux_parts(const Params<T>& P, int d, const T* Uc, const T* Um, const T* Up, const T* hf,
                                           T xi, T* FP, T* FM) {
  // (h -+ xi)/2 * (1/h) = 1/2 -+ xi/(2h): the slope of Eq. (8) is limiter(dU)/h
  const T h2 = (T)0.5 * P.inv_h;
  const T cP = fma(-h2, xi, (T)0.5), cM = fma(h2, xi, (T)0.5);
  T UL[5], UR[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    T mm = tvd_slope<T, LIM>(Uc[q] - Um[q], Up[q] - Uc[q]);      // G12
    if (WANT & 1) UL[q] = fma(cP, mm, hf[q]);
    if (WANT & 2) UR[q] = fma(-cM, mm, hf[q]);
  }
  if (WANT & 1) {
    // max(u^L, 0) with u^L = m_d / rho (0 in vacuum, G9)                                                  (G13)
    T u;
    if constexpr (sizeof(T) == 8) {            // rho > 0, so the sign is the momentum's: one integer test
      const bool ok = UL[0] > P.rho_vac && is_pos<T>(UL[1 + d]);
      const T r = UL[1 + d] * Fast<T>::rcp(ok ? UL[0] : (T)1);
      u = ok ? r : (T)0;
    } else {
      u = UL[0] > P.rho_vac ? UL[1 + d] * Fast<T>::rcp(UL[0]) : (T)0;
      u = u > (T)0 ? u : (T)0;
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) FP[q] = u * UL[q];
  }
  if (WANT & 2) {
    T u;
    if constexpr (sizeof(T) == 8) {
      const bool ok = UR[0] > P.rho_vac && is_neg<T>(UR[1 + d]);
      const T r = UR[1 + d] * Fast<T>::rcp(ok ? UR[0] : (T)1);
      u = ok ? r : (T)0;
    } else {
      u = UR[0] > P.rho_vac ? UR[1 + d] * Fast<T>::rcp(UR[0]) : (T)0;
      u = u < (T)0 ? u : (T)0;
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) FM[q] = u * UR[q];
  }
}

template <class T, int TX, int TY>
struct EulerSmem {
  // x halo of the boxes: 2 cells are needed; 16 bytes' worth are loaded so that every box row starts
  // on a 16-byte boundary in global memory (an 8-byte-aligned fp32 start raised "illegal instruction")
  static constexpr int HX = 16 / (int)sizeof(T) < 2 ? 2 : 16 / (int)sizeof(T);
  static constexpr int BX = TX + 2 * HX;
  static constexpr int UY = TY + 4, LY = TY + 2;
  static constexpr int U_ELEMS = 5 * UY * BX;
  static constexpr int L_ELEMS = 7 * LY * BX;
  static constexpr int U_STAGE = (U_ELEMS * (int)sizeof(T) + 127) / 128 * 128;    // bytes
  static constexpr int L_STAGE = (L_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int EX_ELEMS = 10 * (TX + 2) * (TY + 2) + 10 * TX;    // exchange buffer (x, then y) + y halo rows
  static constexpr int OFF_U = 0;
  static constexpr int OFF_L = OFF_U + 2 * U_STAGE;
  static constexpr int OFF_E = OFF_L + 2 * L_STAGE;
  static constexpr int OFF_BAR = OFF_E + (EX_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int BYTES = OFF_BAR + 64 + 128;  // + slack for the 128-byte alignment of the base
};

// VAC = 1: with the gas-vacuum shortcuts (chosen by the host from the hint of cspt_set_state; both variants are exact)
template <class T, int TX, int TY, int LIM, int VAC>
__global__ void __launch_bounds__(TX* TY, (sizeof(T) == 4 ? 1024 : 512) / (TX * TY))
k_euler_stream(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapL, Params<T> P,
               const DevScalars<T>* __restrict__ sc, const T* __restrict__ U, T* __restrict__ UN,
               typename Real<T>::bits_t* __restrict__ smax_out, int zchunk, BrickMap M) {
  typedef EulerSmem<T, TX, TY> S;
  extern __shared__ __align__(128) unsigned char sm[];
  uint64_t* bar = (uint64_t*)(sm + S::OFF_BAR);
  T* sE = (T*)(sm + S::OFF_E);
  T* sYH = sE + 10 * (TX + 2) * (TY + 2);           // FP of row -1, FM of row TY
  const Layout& L = P.L;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int z0 = blockIdx.z * zchunk, z1 = min(L.nz, z0 + zchunk);
  const int i = i0 + tx, j = j0 + ty;
  const bool inside = i < L.nx && j < L.ny;
  const long long fs = L.fstride;
  constexpr uint32_t TX_BYTES = (uint32_t)((S::U_ELEMS + S::L_ELEMS) * sizeof(T));

  // all of U^n within reach of this CTA exactly 0 (BrickMap): U^{n+1} of its cells is exactly 0, no signal speed
  if (VAC && M.raw && cta_region_dead(M, L, i0 + GX - 3, i0 + TX + GX + 3, j0 + NG - 3, j0 + TY + NG + 3, z0 + NG - 3, z1 + NG + 3)) {
    if (inside && M.zero_fill)
      for (int p = z0; p < z1; ++p) {
        const long long c = L.idx(i, j, p);
#pragma unroll
        for (int q = 0; q < 5; ++q) UN[c + q * fs] = (T)0;
      }
    return;
  }

  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    mbar_fence_init();
    prefetch_tmap(&mapU);
    prefetch_tmap(&mapL);
  }
  __syncthreads();
  auto issue = [&](int p, int s) {      // plane p -> stage s
    mbar_expect_tx(&bar[s], TX_BYTES);
    tma_load_4d(sm + S::OFF_U + s * S::U_STAGE, &mapU, &bar[s], i0 + GX - S::HX, j0 + NG - 2, p + NG, 0);
    tma_load_4d(sm + S::OFF_L + s * S::L_STAGE, &mapL, &bar[s], i0 + GX - S::HX, j0 + NG - 1, p + NG, 0);
  };
  if (tid == 0) {
    issue(z0 - 1, 0);
    issue(z0, 1);
  }

  const T dt = load_dt(sc);
  const T lam = dt * P.inv_h;
  T Um[5], FPzp[5], acc[5], Utp[5];
  // running maximum of the exact speeds seen by this thread, seeded with the global maximum so far (other
  // CTAs' exact speeds: a lower bound of the final maximum)
  T smax = Real<T>::from_bits(*(volatile typename Real<T>::bits_t*)smax_out);
  const T speed_margin = sizeof(T) == 8 ? (T)(1.0 + 1e-12) : (T)(1.0 + 1e-5);
  // U^n of plane z0-2 (own column) for the z slope of plane z0-1
  {
    long long c = L.idx(inside ? i : 0, inside ? j : 0, z0 - 2);
#pragma unroll
    for (int q = 0; q < 5; ++q) { Um[q] = inside ? U[c + q * fs] : (T)0; FPzp[q] = 0; acc[q] = 0; Utp[q] = 0; }
  }

  // The z+ neighbour of the own column (plane p+1) is read from the OTHER ring stage, which plane p+1 is
  // landing in while plane p is processed: the z parts are therefore formed last in the iteration, after
  // waiting for that stage (a global load here would share a scoreboard with the shared-memory loads
  // and expose the DRAM latency every plane).
  uint32_t phase = 0;        // bit s: parity to wait for on stage s
  mbar_wait(&bar[0], 0u);
  phase ^= 1u;
  for (int p = z0 - 1; p <= z1; ++p) {
    const int s = (p - (z0 - 1)) & 1;
    const T* sU = (const T*)(sm + S::OFF_U + s * S::U_STAGE);
    const T* sL = (const T*)(sm + S::OFF_L + s * S::L_STAGE);
    auto u_at = [&](int q, int y, int x) { return sU[(q * S::UY + (y + 2)) * S::BX + (x + S::HX)]; };   // tile coords
    auto l_at = [&](int q, int y, int x) { return sL[(q * S::LY + (y + 1)) * S::BX + (x + S::HX)]; };

    T U0[5], hf[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U0[q] = u_at(q, ty, tx);
    hf[0] = U0[0];                                              // rho~ = rho^n (G2)
#pragma unroll
    for (int q = 1; q < 5; ++q) hf[q] = (T)0.5 * (U0[q] + l_at(q - 1, ty, tx));

    const bool active = p >= z0 && p < z1;
    T a[5] = {0, 0, 0, 0, 0};
    if (active) {
      // halo rows y = -1 (FP only) and y = TY (FM only), by the last two warps.  In fp64 they are formed already in
      // the x phase (while the first warp does the halo columns) into a buffer of their own, which shortens the y
      // phase (5.55 -> 5.40 ms); in fp32 that order measured slower (2.59 -> 2.75 ms) and they stay in the y phase.
      constexpr bool YH_EARLY = sizeof(T) == 8;
      auto y_halo_rows = [&]() {
        if (tid >= TX * TY - 2 * TX) {               // halo rows y = -1 (FP only) and y = TY (FM only): last two warps,
          // already in the x phase (their own buffer), while the first warp does the halo columns
          int t = tid - (TX * TY - 2 * TX);
          int hx = t % TX, side = t / TX, hy = side ? TY : -1;
          T Hc[5], Hm[5], Hp[5], hh[5], HF[5];
#pragma unroll
          for (int q = 0; q < 5; ++q) { Hc[q] = u_at(q, hy, hx); Hm[q] = u_at(q, hy - 1, hx); Hp[q] = u_at(q, hy + 1, hx); }
          hh[0] = Hc[0];
#pragma unroll
          for (int q = 1; q < 5; ++q) hh[q] = (T)0.5 * (Hc[q] + l_at(q - 1, hy, hx));
          T hxi = l_at(5, hy, hx);
          if (side) {
            flux_parts<T, 2, LIM>(P, 1, Hc, Hm, Hp, hh, hxi, HF, HF);
#pragma unroll
            for (int q = 0; q < 5; ++q) (YH_EARLY ? sYH[(q + 5) * TX + hx] : sE[((q + 5) * (TY + 2) + TY + 1) * TX + hx]) = HF[q];
          } else {
            flux_parts<T, 1, LIM>(P, 1, Hc, Hm, Hp, hh, hxi, HF, HF);
#pragma unroll
            for (int q = 0; q < 5; ++q) (YH_EARLY ? sYH[q * TX + hx] : sE[(q * (TY + 2) + 0) * TX + hx]) = HF[q];
          }
                }
      };
      // Gas-vacuum handling (G9): where the cell and its two neighbours along an axis all have rho <= rho_vac, the
      // reconstructed densities lie between theirs, both face velocities are 0 and both flux parts vanish: a warp
      // whose whole in-plane stencil is vacuum skips the reconstruction (most of the 1024^3 disk volume).
      bool vac_xy = false;
      if (VAC) {
        const T rxy = fmax(fmax(fmax(u_at(0, ty, tx - 1), u_at(0, ty, tx + 1)), fmax(u_at(0, ty - 1, tx), u_at(0, ty + 1, tx))), U0[0]);
        vac_xy = __all_sync(0xffffffffu, !(rxy > P.rho_vac));
      }
      // ---- x axis -------------------------------------------------------------
      {
        T Ux0[5], Ux1[5], FP[5] = {0, 0, 0, 0, 0}, FM[5] = {0, 0, 0, 0, 0};
        if (!vac_xy) {
#pragma unroll
          for (int q = 0; q < 5; ++q) { Ux0[q] = u_at(q, ty, tx - 1); Ux1[q] = u_at(q, ty, tx + 1); }
          flux_parts<T, 3, LIM>(P, 0, U0, Ux0, Ux1, hf, l_at(4, ty, tx), FP, FM);
        }
        // exchange layout: [q][ty][tx+1], FP in 0..4, FM in 5..9, row pitch TX+2
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          sE[(q * TY + ty) * (TX + 2) + tx + 1] = FP[q];
          sE[((q + 5) * TY + ty) * (TX + 2) + tx + 1] = FM[q];
          a[q] = FP[q] - FM[q];
        }
        if (tid < 2 * TY) {                         // halo columns x = -1 (FP only) and x = TX (FM only)
          int hy = tid >> 1, side = tid & 1, hx = side ? TX : -1;
          T Hc[5], Hm[5], Hp[5], hh[5], HF[5];
#pragma unroll
          for (int q = 0; q < 5; ++q) { Hc[q] = u_at(q, hy, hx); Hm[q] = u_at(q, hy, hx - 1); Hp[q] = u_at(q, hy, hx + 1); }
          hh[0] = Hc[0];
#pragma unroll
          for (int q = 1; q < 5; ++q) hh[q] = (T)0.5 * (Hc[q] + l_at(q - 1, hy, hx));
          T hxi = l_at(4, hy, hx);
          if (side) {
            flux_parts<T, 2, LIM>(P, 0, Hc, Hm, Hp, hh, hxi, HF, HF);
#pragma unroll
            for (int q = 0; q < 5; ++q) sE[((q + 5) * TY + hy) * (TX + 2) + TX + 1] = HF[q];
          } else {
            flux_parts<T, 1, LIM>(P, 0, Hc, Hm, Hp, hh, hxi, HF, HF);
#pragma unroll
            for (int q = 0; q < 5; ++q) sE[(q * TY + hy) * (TX + 2) + 0] = HF[q];
          }
        }
        if (YH_EARLY) y_halo_rows();
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 5; ++q)
          a[q] += sE[((q + 5) * TY + ty) * (TX + 2) + tx + 2] - sE[(q * TY + ty) * (TX + 2) + tx];
        __syncthreads();
      }
      // ---- y axis -------------------------------------------------------------
      {
        T Uy0[5], Uy1[5], FP[5] = {0, 0, 0, 0, 0}, FM[5] = {0, 0, 0, 0, 0};
        if (!vac_xy) {
#pragma unroll
          for (int q = 0; q < 5; ++q) { Uy0[q] = u_at(q, ty - 1, tx); Uy1[q] = u_at(q, ty + 1, tx); }
          flux_parts<T, 3, LIM>(P, 1, U0, Uy0, Uy1, hf, l_at(5, ty, tx), FP, FM);
        }
        // exchange layout: [q][ty+1][tx], rows -1..TY, row pitch TX
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          sE[(q * (TY + 2) + ty + 1) * TX + tx] = FP[q];
          sE[((q + 5) * (TY + 2) + ty + 1) * TX + tx] = FM[q];
          a[q] += FP[q] - FM[q];
        }
        if (!YH_EARLY) y_halo_rows();
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 5; ++q)
          a[q] += ((YH_EARLY && ty == TY - 1) ? sYH[(q + 5) * TX + tx] : sE[((q + 5) * (TY + 2) + ty + 2) * TX + tx]) -
                  ((YH_EARLY && ty == 0) ? sYH[q * TX + tx] : sE[(q * (TY + 2) + ty) * TX + tx]);
      }
    }
    // z axis: both parts of plane p; U^n of plane p+1 from the other stage
    T Up[5], FPz[5], FMz[5];
    mbar_wait(&bar[s ^ 1], (phase >> (s ^ 1)) & 1u);
    phase ^= 1u << (s ^ 1);
    {
      const T* sU1 = (const T*)(sm + S::OFF_U + (s ^ 1) * S::U_STAGE);
#pragma unroll
      for (int q = 0; q < 5; ++q) Up[q] = sU1[(q * S::UY + (ty + 2)) * S::BX + (tx + S::HX)];
    }
    if (VAC && __all_sync(0xffffffffu, !(fmax(fmax(Um[0], Up[0]), U0[0]) > P.rho_vac))) {
#pragma unroll
      for (int q = 0; q < 5; ++q) FPz[q] = FMz[q] = (T)0;         // vacuum along z as well
    } else {
      flux_parts<T, 3, LIM>(P, 2, U0, Um, Up, hf, l_at(6, ty, tx), FPz, FMz);
    }
    // finish cell p-1 (SUE, Eq. (4))
    if (p - 1 >= z0) {
      T un[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) un[q] = Utp[q] - lam * (acc[q] + FMz[q]);
      if (inside) {
        long long c = L.idx(i, j, p - 1);
#pragma unroll
        for (int q = 0; q < 5; ++q) UN[c + q * fs] = un[q];
        if (VAC && M.raw) {                          // the map follows the gas: flag the brick of a non-zero result
          bool nz = false;
#pragma unroll
          for (int q = 0; q < 5; ++q) nz = nz || (un[q] != (T)0);
          if (nz) brick_flag(M, i + GX, j + NG, p - 1 + NG);
        }
        // CFL speed of U^{n+1} (G15): exactly rounded, but only for cells whose estimate comes within the
        // filter margin of a speed already known exactly (this thread's maximum or the global one so far);
        // the true maximum always passes the filter, so the result is the exact maximum
        T se = cell_speed_upper<T>(un[0], un[1], un[2], un[3], un[4], P.gamma, P.rho_vac);
        if (se * speed_margin >= smax) {
          T sp = cell_speed_exact<T>(un[0], un[1], un[2], un[3], un[4], P.gamma, P.rho_vac);
          smax = sp > smax ? sp : smax;
        }
      }
    }
    if (active) {
      // z: own parts of plane p, FP of plane p-1; FM of plane p+1 is added when it is known
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        acc[q] = a[q] + ((FPz[q] - FMz[q]) - FPzp[q]);
        Utp[q] = q == 0 ? U0[0] : l_at(q - 1, ty, tx);
      }
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) { FPzp[q] = FPz[q]; Um[q] = U0[q]; }
    __syncthreads();                                   // everyone is done with stage s and with sE
    if (tid == 0 && p + 2 <= z1 + 1) issue(p + 2, s);
  }
  block_max_to_global<T>(smax, smax_out);
}

}  // namespace cspt
