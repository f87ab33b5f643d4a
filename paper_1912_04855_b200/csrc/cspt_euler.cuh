// cspt_euler.cuh -- Eulerian stage: FGC (Eq. (8) + pressureless HLL flux) and SUE (Eq. (4)),
// PAPER.md:45-50, :70-78, :112-113; readings G9-G14, with the CFL signal speed of U^{n+1}
// (G15) as epilogue.
//
// One CTA owns a TX x TY column of cells and streams along z (2.5-D): per plane one TMA box
// of U^n (halo 2 in x/y) and one of (U~, xi) (halo 1) land in a 2-stage shared-memory ring.
// Per cell and axis the two one-sided flux parts
//     FP_i = max(u^L_i,0) U^L_i   (leaves through the + face),   FM_i = min(u^R_i,0) U^R_i   (through the - face)
// are computed ONCE (F_{i+1/2} = FP_i + FM_{i+1}).  The CTA has TY + 2 warps: warp r+1 owns row r of the
// tile (TX = 32 cells = its lanes); the two extra warps own the halo rows -1 and TY, of which only the
// y parts are needed, and use their spare time for the x parts of the halo columns -1 and TX.  Parts
// travel to the x neighbours by warp shuffles, to the y neighbours through shared memory (one
// barrier), and along z in registers: the thread keeps FP of the previous plane and finishes cell
// p-1 when FM of plane p is known.
#pragma once
#include "cspt_kernels.cuh"
#include "cspt_tma.cuh"

namespace cspt {

template <class T>
__device__ __forceinline__ T minmod_fast(T a, T b) {
  T r = fabs(a) < fabs(b) ? a : b;
  return a * b > (T)0 ? r : (T)0;
}

// One-sided flux parts of one cell along axis d.  Uc/Um/Up: U^n of the cell and of its -/+
// neighbours; hf = U^{n+1/2} = (U^n + U~)/2 (G10); xi = xi_d of the cell.
template <class T, int WANT>   // WANT bit 0: FP, bit 1: FM
__device__ __forceinline__ void flux_parts(const Params<T>& P, int d, const T* Uc, const T* Um, const T* Up, const T* hf,
                                           T xi, T* FP, T* FM) {
  T cP = ((T)0.5 * (P.h - xi)) * P.inv_h;      // (h - xi)/2 * (1/h): slope is minmod(dU)/h (Eq. (8))
  T cM = ((T)0.5 * (P.h + xi)) * P.inv_h;
  T UL[5], UR[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    T mm = minmod_fast<T>(Uc[q] - Um[q], Up[q] - Uc[q]);      // G12
    if (WANT & 1) UL[q] = hf[q] + cP * mm;
    if (WANT & 2) UR[q] = hf[q] - cM * mm;
  }
  if (WANT & 1) {
    T u = UL[0] > P.rho_vac ? UL[1 + d] * Fast<T>::rcp(UL[0]) : (T)0;       // G9
    u = u > (T)0 ? u : (T)0;                                   // G13
#pragma unroll
    for (int q = 0; q < 5; ++q) FP[q] = u * UL[q];
  }
  if (WANT & 2) {
    T u = UR[0] > P.rho_vac ? UR[1 + d] * Fast<T>::rcp(UR[0]) : (T)0;
    u = u < (T)0 ? u : (T)0;
#pragma unroll
    for (int q = 0; q < 5; ++q) FM[q] = u * UR[q];
  }
}

template <class T, int TX, int TY>
struct EulerSmem {
  static_assert(TX == 32, "a warp owns one row of the tile");
  // x halo of the boxes: 2 cells are needed; 16 bytes' worth are loaded so that every box row starts
  // on a 16-byte boundary in global memory (an 8-byte-aligned fp32 start raised "illegal instruction")
  static constexpr int HX = 16 / (int)sizeof(T) < 2 ? 2 : 16 / (int)sizeof(T);
  static constexpr int BX = TX + 2 * HX;
  static constexpr int UY = TY + 4, LY = TY + 2;
  static constexpr int U_ELEMS = 5 * UY * BX;
  static constexpr int L_ELEMS = 7 * LY * BX;
  static constexpr int U_STAGE = (U_ELEMS * (int)sizeof(T) + 127) / 128 * 128;    // bytes
  static constexpr int L_STAGE = (L_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  // y exchange: FP of rows -1..TY-1 and FM of rows 0..TY;  x halo columns: FP of x = -1, FM of x = TX
  static constexpr int EY_ELEMS = 10 * (TY + 1) * TX;
  static constexpr int EX_ELEMS = 10 * TY;
  static constexpr int OFF_U = 0;
  static constexpr int OFF_L = OFF_U + 2 * U_STAGE;
  static constexpr int OFF_EY = OFF_L + 2 * L_STAGE;
  static constexpr int OFF_EX = OFF_EY + (EY_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int OFF_BAR = OFF_EX + (EX_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int BYTES = OFF_BAR + 64;
  static constexpr int THREADS = TX * (TY + 2);
};

template <class T, int TX, int TY>
__global__ void __launch_bounds__(TX*(TY + 2), 2)
k_euler_stream(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapL, Params<T> P,
               const DevScalars<T>* __restrict__ sc, const T* __restrict__ U, T* __restrict__ UN,
               typename Real<T>::bits_t* __restrict__ smax_out, int zchunk) {
  typedef EulerSmem<T, TX, TY> S;
  extern __shared__ __align__(128) unsigned char sm[];
  uint64_t* bar = (uint64_t*)(sm + S::OFF_BAR);
  T* sEY = (T*)(sm + S::OFF_EY);
  T* sEX = (T*)(sm + S::OFF_EX);
  const Layout& L = P.L;
  const int tid = threadIdx.x, tx = tid % TX;
  const int ty = tid / TX - 1;                       // row of the tile: -1 and TY are the halo rows
  const bool main_row = ty >= 0 && ty < TY;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int z0 = blockIdx.z * zchunk, z1 = min(L.nz, z0 + zchunk);
  const int i = i0 + tx, j = j0 + ty;
  const bool inside = main_row && i < L.nx && j < L.ny;
  const long long fs = L.fstride;
  constexpr uint32_t TX_BYTES = (uint32_t)((S::U_ELEMS + S::L_ELEMS) * sizeof(T));

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
  T smax = 0;
  // own column of planes z0-2 (z slope of plane z0-1) and, one iteration ahead of its use, p+1: straight
  // from global memory (plane p+1 becomes a TMA box one iteration later)
  const long long c_col = L.idx(inside ? i : 0, inside ? j : 0, 0), szp = L.sz();
  T Unext[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    Um[q] = main_row ? __ldg(U + c_col + (long long)(z0 - 2) * szp + q * fs) : (T)0;
    Unext[q] = main_row ? __ldg(U + c_col + (long long)z0 * szp + q * fs) : (T)0;
    FPzp[q] = 0; acc[q] = 0; Utp[q] = 0;
  }

  uint32_t phase = 0;        // bit s: parity to wait for on stage s
  for (int p = z0 - 1; p <= z1; ++p) {
    const int K = (p - (z0 - 1)) & 1;
    T Up[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) Up[q] = Unext[q];
    if (p < z1 && main_row) {
#pragma unroll
      for (int q = 0; q < 5; ++q) Unext[q] = __ldg(U + c_col + (long long)(p + 2) * szp + q * fs);
    }
    mbar_wait(&bar[K], (phase >> K) & 1u);
    phase ^= 1u << K;
    const T* sU = (const T*)(sm + S::OFF_U + K * S::U_STAGE);
    const T* sL = (const T*)(sm + S::OFF_L + K * S::L_STAGE);
    auto u_at = [&](int q, int y, int x) { return sU[(q * S::UY + (y + 2)) * S::BX + (x + S::HX)]; };   // tile coords
    auto l_at = [&](int q, int y, int x) { return sL[(q * S::LY + (y + 1)) * S::BX + (x + S::HX)]; };
    // U^n, its two neighbours along axis d and U^{n+1/2} (G10; rho~ = rho^n, G2) of tile cell (x, y)
    auto gather = [&](int d, int y, int x, T* Uc, T* Ua, T* Ub, T* hf) {
      const int ax = d == 0, ay = d == 1;
#pragma unroll
      for (int q = 0; q < 5; ++q) { Uc[q] = u_at(q, y, x); Ua[q] = u_at(q, y - ay, x - ax); Ub[q] = u_at(q, y + ay, x + ax); }
      hf[0] = Uc[0];
#pragma unroll
      for (int q = 1; q < 5; ++q) hf[q] = (T)0.5 * (Uc[q] + l_at(q - 1, y, x));
    };
    const bool active = p >= z0 && p < z1;

    if (main_row) {
      T U0[5], hf[5], FPz[5], FMz[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) U0[q] = u_at(q, ty, tx);
      hf[0] = U0[0];
#pragma unroll
      for (int q = 1; q < 5; ++q) hf[q] = (T)0.5 * (U0[q] + l_at(q - 1, ty, tx));
      // z axis: both parts of plane p
      flux_parts<T, 3>(P, 2, U0, Um, Up, hf, l_at(6, ty, tx), FPz, FMz);
      // finish cell p-1 (SUE, Eq. (4))
      if (p - 1 >= z0) {
        T un[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) un[q] = Utp[q] - lam * (acc[q] + FMz[q]);
        if (inside) {
          long long c = L.idx(i, j, p - 1);
#pragma unroll
          for (int q = 0; q < 5; ++q) UN[c + q * fs] = un[q];
          T sp = cell_speed_exact<T>(un[0], un[1], un[2], un[3], un[4], P.gamma, P.rho_vac);
          smax = sp > smax ? sp : smax;
        }
      }
      if (active) {
        T Ua[5], Ub[5], FP[5], FM[5];
        // z: own parts of plane p, FP of plane p-1; FM of plane p+1 is added when it is known
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          acc[q] = (FPz[q] - FMz[q]) - FPzp[q];
          Utp[q] = q == 0 ? U0[0] : l_at(q - 1, ty, tx);
        }
        // x: own parts; the neighbours' parts come from lanes -1 / +1 (the first and the last lane
        // take theirs from the halo columns after the barrier)
#pragma unroll
        for (int q = 0; q < 5; ++q) { Ua[q] = u_at(q, ty, tx - 1); Ub[q] = u_at(q, ty, tx + 1); }
        flux_parts<T, 3>(P, 0, U0, Ua, Ub, hf, l_at(4, ty, tx), FP, FM);
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          T fpl = __shfl_up_sync(0xffffffffu, FP[q], 1);
          T fmr = __shfl_down_sync(0xffffffffu, FM[q], 1);
          if (tx == 0) fpl = (T)0;
          if (tx == TX - 1) fmr = (T)0;
          acc[q] += (FP[q] - FM[q]) + (fmr - fpl);
        }
        // y: own parts; FP of row r goes to [q][r+1], FM of row r to [5+q][r]
#pragma unroll
        for (int q = 0; q < 5; ++q) { Ua[q] = u_at(q, ty - 1, tx); Ub[q] = u_at(q, ty + 1, tx); }
        flux_parts<T, 3>(P, 1, U0, Ua, Ub, hf, l_at(5, ty, tx), FP, FM);
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          sEY[(q * (TY + 1) + ty + 1) * TX + tx] = FP[q];
          sEY[((q + 5) * (TY + 1) + ty) * TX + tx] = FM[q];
          acc[q] += FP[q] - FM[q];
        }
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) { FPzp[q] = FPz[q]; Um[q] = U0[q]; }
    } else if (active) {
      // halo rows: y part towards the tile, then the x part of one halo column towards the tile
      const bool lo = ty < 0;
      T Uc[5], Ua[5], Ub[5], hf[5], HF[5];
      gather(1, ty, tx, Uc, Ua, Ub, hf);
      if (lo) {
        flux_parts<T, 1>(P, 1, Uc, Ua, Ub, hf, l_at(5, ty, tx), HF, HF);
#pragma unroll
        for (int q = 0; q < 5; ++q) sEY[(q * (TY + 1) + 0) * TX + tx] = HF[q];
      } else {
        flux_parts<T, 2>(P, 1, Uc, Ua, Ub, hf, l_at(5, ty, tx), HF, HF);
#pragma unroll
        for (int q = 0; q < 5; ++q) sEY[((q + 5) * (TY + 1) + TY) * TX + tx] = HF[q];
      }
      if (tx < TY) {
        const int hx = lo ? -1 : TX;
        gather(0, tx, hx, Uc, Ua, Ub, hf);
        if (lo) {
          flux_parts<T, 1>(P, 0, Uc, Ua, Ub, hf, l_at(4, tx, hx), HF, HF);
#pragma unroll
          for (int q = 0; q < 5; ++q) sEX[q * TY + tx] = HF[q];
        } else {
          flux_parts<T, 2>(P, 0, Uc, Ua, Ub, hf, l_at(4, tx, hx), HF, HF);
#pragma unroll
          for (int q = 0; q < 5; ++q) sEX[(q + 5) * TY + tx] = HF[q];
        }
      }
    }
    __syncthreads();                                   // the parts of plane p are visible

    if (main_row && active) {
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        T fpd = sEY[(q * (TY + 1) + ty) * TX + tx];                  // FP of row ty-1
        T fmu = sEY[((q + 5) * (TY + 1) + ty + 1) * TX + tx];        // FM of row ty+1
        T e = fmu - fpd;
        if (tx == 0) e -= sEX[q * TY + ty];                          // FP of column -1
        if (tx == TX - 1) e += sEX[(q + 5) * TY + ty];               // FM of column TX
        acc[q] += e;
      }
    }
    __syncthreads();                                   // everyone is done with stage K and with the exchange buffers
    if (tid == 0 && p + 2 <= z1) issue(p + 2, K);
  }
  block_max_to_global<T>(smax, smax_out);
}

}  // namespace cspt
