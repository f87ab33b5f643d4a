// cspt_euler2.cuh -- Eulerian stage, second layout: FGC (Eq. (8) + Riemann flux) and SUE (Eq. (4)), PAPER.md:45-50,
// :70-78, :112-113; readings G9-G14, with the CFL signal speed of U^{n+1} (G15) as epilogue.
//
// What bounds this kernel on B200 is the instruction issue rate (one instruction per cycle and SM sub-partition; only a
// third of its instructions are FP64 arithmetic, profiles/r2_issue_model.md), so the layout minimises instructions per
// cell; the z loop is unrolled twice (UNR) so that the registers carried from plane to plane are renamed, not moved:
//   * one CTA = TY main warps (warp = one row of 32 cells, one cell per thread and plane) + ONE helper warp, streaming
//     along z (2.5-D) over a 2-stage TMA ring of U^n (halo 2) and (U~, xi) (halo 1);
//   * per cell and axis the two EDGE quantities are formed once:  P_i belongs to face i+1/2, M_i to face i-1/2, and the
//     face flux is F_{i+1/2} = combine(P_i, M_{i+1}).  With the pressureless HLL flux of reading G13 they are the
//     one-sided flux parts P = max(u^L,0) U^L, M = min(u^R,0) U^R and combine is a sum; for a solver that needs both
//     states at the face (LF, HLLC: reading G13b/c) they are the reconstructed states U^L, U^R themselves;
//   * x: M travels one lane down and the finished face flux one lane up by warp shuffles (each face flux is
//     formed once); y: P and M go through a small shared-memory buffer; z: P of the previous plane stays in
//     registers and cell p-1 is finished when M of plane p is known;
//   * the edge quantities of the cells just outside the tile (rows -1 and TY, columns -1 and 32) are formed by the
//     helper warp, so the main warps do no redundant work and there are two barriers per plane (one before the
//     exchanged values are read, one before the ring stage is refilled) instead of four.
#pragma once
#include "cspt_euler.cuh"

namespace cspt {

enum { RIEM_HLL = 0, RIEM_LF = 1, RIEM_HLLC = 2 };

// face velocity of a reconstructed state: m_d / rho with the vacuum guard of reading G9
template <class T>
__device__ __forceinline__ T face_velocity(const Params<T>& P, int d, const T* Us) {
  return Us[0] > P.rho_vac ? Us[1 + d] * Fast<T>::rcp(Us[0]) : (T)0;
}

// Edge quantities of one cell along axis d (WANT bit 0: P, bit 1: M).  Uc/Um/Up: U^n of the cell and of its -/+
// neighbours; hf = U^{n+1/2} = (U^n + U~)/2 (G10); xi = xi_d of the cell; Eq. (8).
template <class T, int WANT, int LIM, int RIEM>
__device__ __forceinline__ void edge_parts(const Params<T>& P, int d, const T* Uc, const T* Um, const T* Up, const T* hf,
                                           T xi, T* Pq, T* Mq) {
  if (RIEM == RIEM_HLL) {
    flux_parts<T, WANT, LIM>(P, d, Uc, Um, Up, hf, xi, Pq, Mq);
  } else {
    const T h2 = (T)0.5 * P.inv_h;
    const T cP = fma(-h2, xi, (T)0.5), cM = fma(h2, xi, (T)0.5);
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      const T mm = tvd_slope<T, LIM>(Uc[q] - Um[q], Up[q] - Uc[q]);
      if (WANT & 1) Pq[q] = fma(cP, mm, hf[q]);           // U^L of face i+1/2
      if (WANT & 2) Mq[q] = fma(-cM, mm, hf[q]);          // U^R of face i-1/2
    }
  }
}

// Face flux from the edge quantity of the cell on the left (Pl) and of the cell on the right (Mr).
template <class T, int RIEM>
__device__ __forceinline__ void face_flux(const Params<T>& P, int d, const T* Pl, const T* Mr, T* F) {
  if (RIEM == RIEM_HLL) {
#pragma unroll
    for (int q = 0; q < 5; ++q) F[q] = Pl[q] + Mr[q];
  } else {
    const T uL = face_velocity<T>(P, d, Pl), uR = face_velocity<T>(P, d, Mr);
    if (RIEM == RIEM_LF) {
      // local Lax-Friedrichs (Rusanov) flux of the advective system, a = max(|u^L|, |u^R|)   (reading G13b)
      const T a = fmax(fabs(uL), fabs(uR));
      const T cl = (T)0.5 * (uL + a), cr = (T)0.5 * (uR - a);
#pragma unroll
      for (int q = 0; q < 5; ++q) F[q] = cl * Pl[q] + cr * Mr[q];
    } else {
      // HLLC of the pressureless system (reading G13c): S_L = min(u^L,u^R), S_R = max(u^L,u^R), contact speed
      // S* = (rho^L u^L + rho^R u^R) / (rho^L + rho^R) between converging streams
      const T up = uL > (T)0 ? uL : (T)0, um = uR < (T)0 ? uR : (T)0;
      if (uL > uR && uR < (T)0 && uL > (T)0) {
        const T rs = Pl[0] + Mr[0];
        const T ss = (Pl[0] * uL + Mr[0] * uR) * Fast<T>::rcp(rs);
        const bool left = ss >= (T)0;
        const T* UK = left ? Pl : Mr;
        const T uK = left ? uL : uR, sK = left ? uR : uL;              // S_L = u^R, S_R = u^L here
        const T fac = (sK - uK) * Fast<T>::rcp(sK - ss);                // rho*_K / rho_K
        T Us[5];
        Us[0] = fac * UK[0];
#pragma unroll
        for (int q = 1; q < 4; ++q) Us[q] = fac * UK[q];
        Us[1 + d] = Us[0] * ss;
        Us[4] = fac * (UK[4] + UK[0] * ((ss - uK) * ss));
#pragma unroll
        for (int q = 0; q < 5; ++q) F[q] = uK * UK[q] + sK * (Us[q] - UK[q]);
      } else {
#pragma unroll
        for (int q = 0; q < 5; ++q) F[q] = up * Pl[q] + um * Mr[q];
      }
    }
  }
}

template <class T, int TY>
struct Euler2Smem {
  static constexpr int TX = 32;
  static constexpr int HX = 16 / (int)sizeof(T) < 2 ? 2 : 16 / (int)sizeof(T);     // x halo of the boxes (16 bytes)
  static constexpr int BX = TX + 2 * HX;
  static constexpr int UY = TY + 4, LY = TY + 2;
  static constexpr int U_ELEMS = 5 * UY * BX;
  static constexpr int L_ELEMS = 7 * LY * BX;
  static constexpr int U_STAGE = (U_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int L_STAGE = (L_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int Y_ELEMS = 2 * 5 * (TY + 2) * TX;          // P and M of rows -1 .. TY
  static constexpr int X_ELEMS = 2 * 5 * TY;                      // P of column -1, M of column TX
  static constexpr int NSU = 3;                                   // U^n ring: planes p, p+1 resident, p+2 in flight
  static constexpr int OFF_U = 0;
  static constexpr int OFF_L = OFF_U + NSU * U_STAGE;
  static constexpr int OFF_Y = OFF_L + 2 * L_STAGE;
  static constexpr int OFF_X = OFF_Y + (Y_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int OFF_BAR = OFF_X + (X_ELEMS * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int BYTES = OFF_BAR + 64 + 128;
  static constexpr int THREADS = TX * (TY + 1);
};

template <class T, int TY, int MINB, int LIM, int RIEM, int UNR = 1>
__global__ void __launch_bounds__(32 * (TY + 1), MINB)
k_euler_rows(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapL, Params<T> P,
             const DevScalars<T>* __restrict__ sc, const T* __restrict__ U, T* __restrict__ UN,
             typename Real<T>::bits_t* __restrict__ smax_out, int zchunk) {
  typedef Euler2Smem<T, TY> S;
  constexpr int TX = S::TX;
  extern __shared__ __align__(128) unsigned char sm[];
  uint64_t* bar = (uint64_t*)(sm + S::OFF_BAR);
  T* sYP = (T*)(sm + S::OFF_Y);                     // [q][row + 1][x]
  T* sYM = sYP + 5 * (TY + 2) * TX;
  T* sXP = (T*)(sm + S::OFF_X);                     // [row][q]: P of column -1
  T* sXM = sXP + 5 * TY;                            //           M of column TX
  const Layout& L = P.L;
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const bool helper = ty == TY;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int z0 = blockIdx.z * zchunk, z1 = min(L.nz, z0 + zchunk);
  const int i = i0 + tx, j = j0 + ty;
  const bool inside = !helper && i < L.nx && j < L.ny;
  const long long fs = L.fstride;
  constexpr uint32_t U_BYTES = (uint32_t)(S::U_ELEMS * sizeof(T)), L_BYTES = (uint32_t)(S::L_ELEMS * sizeof(T));
  uint64_t* barU = bar;                             // [NSU]
  uint64_t* barL = bar + S::NSU;                    // [2]

  if (tid == 0) {
#pragma unroll
    for (int k = 0; k < S::NSU + 2; ++k) mbar_init(&bar[k], 1);
    mbar_fence_init();
    prefetch_tmap(&mapU);
    prefetch_tmap(&mapL);
  }
  __syncthreads();
  // the U^n ring is one plane deeper than the (U~, xi) ring: the z stencil reads U^n of plane p+1 while plane p is
  // processed, and plane p+2 must already be in flight then (with two stages the kernel waited for it every plane)
  auto slotU = [&](int p) { return (p - (z0 - 1)) % S::NSU; };
  auto slotL = [&](int p) { return (p - (z0 - 1)) & 1; };
  auto issueU = [&](int p) {
    const int k = slotU(p);
    mbar_expect_tx(&barU[k], U_BYTES);
    tma_load_4d(sm + S::OFF_U + k * S::U_STAGE, &mapU, &barU[k], i0 + GX - S::HX, j0 + NG - 2, p + NG, 0);
  };
  auto issueL = [&](int p) {
    const int k = slotL(p);
    mbar_expect_tx(&barL[k], L_BYTES);
    tma_load_4d(sm + S::OFF_L + k * S::L_STAGE, &mapL, &barL[k], i0 + GX - S::HX, j0 + NG - 1, p + NG, 0);
  };
  if (tid == 0) {
    issueU(z0 - 1); issueU(z0); issueU(z0 + 1);
    issueL(z0 - 1); issueL(z0);
  }
  uint32_t phaseU = 0, phaseL = 0;
  auto waitU = [&](int p) { const int k = slotU(p); mbar_wait(&barU[k], (phaseU >> k) & 1u); phaseU ^= 1u << k; };
  auto waitL = [&](int p) { const int k = slotL(p); mbar_wait(&barL[k], (phaseL >> k) & 1u); phaseL ^= 1u << k; };

  const T dt = load_dt(sc);
  const T lam = dt * P.inv_h;
  T smax = Real<T>::from_bits(*(volatile typename Real<T>::bits_t*)smax_out);
  const T speed_margin = sizeof(T) == 8 ? (T)(1.0 + 1e-12) : (T)(1.0 + 1e-5);

  T Um[5], U0[5], Pzp[5], acc[5], Utp[5];
  {
    // U^n of plane z0-2 (own column) for the z slope of plane z0-1
    long long c = L.idx(inside ? i : 0, inside ? j : 0, z0 - 2);
#pragma unroll
    for (int q = 0; q < 5; ++q) { Um[q] = inside ? U[c + q * fs] : (T)0; Pzp[q] = 0; acc[q] = 0; Utp[q] = 0; }
  }
  waitU(z0 - 1);
  if (!helper) {
    const T* sU = (const T*)(sm + S::OFF_U + slotU(z0 - 1) * S::U_STAGE);
#pragma unroll
    for (int q = 0; q < 5; ++q) U0[q] = sU[(q * S::UY + (ty + 2)) * S::BX + (tx + S::HX)];
  }

#pragma unroll UNR
  for (int p = z0 - 1; p <= z1; ++p) {
    const T* sU = (const T*)(sm + S::OFF_U + slotU(p) * S::U_STAGE);
    const T* sL = (const T*)(sm + S::OFF_L + slotL(p) * S::L_STAGE);
    waitL(p);
    auto u_at = [&](int q, int y, int x) { return sU[(q * S::UY + (y + 2)) * S::BX + (x + S::HX)]; };   // tile coords
    auto l_at = [&](int q, int y, int x) { return sL[(q * S::LY + (y + 1)) * S::BX + (x + S::HX)]; };
    const bool active = p >= z0 && p < z1;

    if (helper) {
      // ---- cells just outside the tile, plane p: their edge quantities towards the tile -----------------
      if (active) {
        auto halo_cell = [&](int d, int hy, int hx, bool wantP, T* dst, int stride) {
          T Hc[5], Hm[5], Hp[5], hh[5], Pq[5], Mq[5];
          const int oy = d == 1, ox = d == 0;
#pragma unroll
          for (int q = 0; q < 5; ++q) { Hc[q] = u_at(q, hy, hx); Hm[q] = u_at(q, hy - oy, hx - ox); Hp[q] = u_at(q, hy + oy, hx + ox); }
          hh[0] = Hc[0];
#pragma unroll
          for (int q = 1; q < 5; ++q) hh[q] = (T)0.5 * (Hc[q] + l_at(q - 1, hy, hx));
          const T hxi = l_at(4 + d, hy, hx);
          if (wantP) edge_parts<T, 1, LIM, RIEM>(P, d, Hc, Hm, Hp, hh, hxi, Pq, Mq);
          else edge_parts<T, 2, LIM, RIEM>(P, d, Hc, Hm, Hp, hh, hxi, Pq, Mq);
#pragma unroll
          for (int q = 0; q < 5; ++q) dst[q * stride] = wantP ? Pq[q] : Mq[q];
        };
        halo_cell(1, -1, tx, true, sYP + tx, (TY + 2) * TX);                               // row -1: P
        halo_cell(1, TY, tx, false, sYM + (TY + 1) * TX + tx, (TY + 2) * TX);              // row TY: M
        if (tx < 2 * TY) {
          const int r = tx >> 1, side = tx & 1;
          if (side) halo_cell(0, r, TX, false, sXM + r * 5, 1);                          // column TX: M
          else halo_cell(0, r, -1, true, sXP + r * 5, 1);                                // column -1: P
        }
      }
      waitU(p + 1);                                      // the helper reads plane p+1 in the next iteration
      if (active) __syncthreads();
      __syncthreads();
      continue;
    }

    T hf[5];
    hf[0] = U0[0];                                              // rho~ = rho^n (G2)
#pragma unroll
    for (int q = 1; q < 5; ++q) hf[q] = (T)0.5 * (U0[q] + l_at(q - 1, ty, tx));

    T Py[5], My[5];
    if (active) {
      // ---- y: own edge quantities into the exchange buffer -----------------------------------------------
      T Uy0[5], Uy1[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) { Uy0[q] = u_at(q, ty - 1, tx); Uy1[q] = u_at(q, ty + 1, tx); }
      edge_parts<T, 3, LIM, RIEM>(P, 1, U0, Uy0, Uy1, hf, l_at(5, ty, tx), Py, My);
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        sYP[(q * (TY + 2) + ty + 1) * TX + tx] = Py[q];
        sYM[(q * (TY + 2) + ty + 1) * TX + tx] = My[q];
      }
    }

    // ---- z: edge quantities of plane p; U^n of plane p+1 from the other stage; finish cell p-1 -----------
    T Up[5], Pz[5], Mz[5], Fzm[5];
    waitU(p + 1);
    {
      const T* sU1 = (const T*)(sm + S::OFF_U + slotU(p + 1) * S::U_STAGE);
#pragma unroll
      for (int q = 0; q < 5; ++q) Up[q] = sU1[(q * S::UY + (ty + 2)) * S::BX + (tx + S::HX)];
    }
    edge_parts<T, 3, LIM, RIEM>(P, 2, U0, Um, Up, hf, l_at(6, ty, tx), Pz, Mz);
    face_flux<T, RIEM>(P, 2, Pzp, Mz, Fzm);                      // face p - 1/2
    if (p - 1 >= z0) {
      T un[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) un[q] = Utp[q] - lam * (acc[q] + Fzm[q]);       // SUE, Eq. (4)
      if (inside) {
        long long c = L.idx(i, j, p - 1);
#pragma unroll
        for (int q = 0; q < 5; ++q) UN[c + q * fs] = un[q];
        // CFL speed of U^{n+1} (G15): exactly rounded only where the cheap upper bound can still beat the running maximum
        T se = cell_speed_upper<T>(un[0], un[1], un[2], un[3], un[4], P.gamma, P.rho_vac);
        if (se * speed_margin >= smax) {
          T sp = cell_speed_exact<T>(un[0], un[1], un[2], un[3], un[4], P.gamma, P.rho_vac);
          smax = sp > smax ? sp : smax;
        }
      }
    }

    if (active) {
      __syncthreads();                                   // exchange buffers of plane p are complete
      T a[5];
      // ---- x: M one lane down, the finished face flux one lane up ------------------------------------------
      {
        T Ux0[5], Ux1[5], Px[5], Mx[5], Mr[5], Fx[5], Fl[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) { Ux0[q] = u_at(q, ty, tx - 1); Ux1[q] = u_at(q, ty, tx + 1); }
        edge_parts<T, 3, LIM, RIEM>(P, 0, U0, Ux0, Ux1, hf, l_at(4, ty, tx), Px, Mx);
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          Mr[q] = __shfl_down_sync(0xffffffffu, Mx[q], 1);
          if (tx == TX - 1) Mr[q] = sXM[ty * 5 + q];
        }
        face_flux<T, RIEM>(P, 0, Px, Mr, Fx);                    // face i + 1/2
        T Pl[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          Fl[q] = __shfl_up_sync(0xffffffffu, Fx[q], 1);
          Pl[q] = sXP[ty * 5 + q];
        }
        if (tx == 0) face_flux<T, RIEM>(P, 0, Pl, Mx, Fl);       // face -1/2 of the tile
#pragma unroll
        for (int q = 0; q < 5; ++q) a[q] = Fx[q] - Fl[q];
      }
      // ---- y: faces j + 1/2 and j - 1/2 from the exchanged quantities ---------------------------------------
      {
        T Mu[5], Pd[5], Fu[5], Fd[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          Mu[q] = sYM[(q * (TY + 2) + ty + 2) * TX + tx];
          Pd[q] = sYP[(q * (TY + 2) + ty) * TX + tx];
        }
        face_flux<T, RIEM>(P, 1, Py, Mu, Fu);
        face_flux<T, RIEM>(P, 1, Pd, My, Fd);
#pragma unroll
        for (int q = 0; q < 5; ++q) a[q] += Fu[q] - Fd[q];
      }
      // z: face p - 1/2 now, face p + 1/2 when plane p + 1 is known
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        acc[q] = a[q] - Fzm[q];
        Utp[q] = q == 0 ? U0[0] : l_at(q - 1, ty, tx);
      }
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) { Pzp[q] = Pz[q]; Um[q] = U0[q]; U0[q] = Up[q]; }
    __syncthreads();                                   // everyone is done with plane p and with the exchange buffers
    if (tid == 0) {
      if (p + S::NSU <= z1 + 1) issueU(p + S::NSU);
      if (p + 2 <= z1) issueL(p + 2);
    }
  }
  block_max_to_global<T>(helper ? (T)0 : smax, smax_out);
}

}  // namespace cspt
