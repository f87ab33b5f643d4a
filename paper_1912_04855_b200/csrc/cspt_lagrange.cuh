// cspt_lagrange.cuh -- Lagrangian stage: HFC{corrector} + SUL{corrector}, Eq. (7) at the displaced
// particle positions r* and Eq. (6) (readings G1-G9), as a TMA-fed
// z-streaming kernel.
//
// One CTA owns a TX x TY column of cells of the extended domain interior(+)1 (G16) and streams along
// z.  The seven per-particle quantities of U*, r* that a NEIGHBOUR contributes to Eq. (7)
//     phi*, u*, v*, w*, eta* = xi*/h (3 components)
// arrive per plane as one TMA box (halo 1 in x/y) in a 4-stage shared-memory ring: planes p-1, p,
// p+1 are resident while plane p is evaluated and plane p+2 is in flight.  A thread owns CY cells
// adjacent in y, so that a neighbour particle read from shared memory serves up to CY cells.
//
// Per neighbour (lengths in units of h):  d = (eta_i - o) - eta_j,  s = |d|^2,  y = 1/sqrt(s),
// q = s y,  g^(q) = -W'(q)/q of the cubic spline (G5):  3 - 2.25 q  (s < 1),
// 0.75 (2-q)^2 / q = 3 y - 3 + 0.75 q  (1 <= s < 4),  0 (s >= 4);  no division, no IEEE sqrt.
// Sum_j w_j (u_i + u_j).d is split as u_i . Sum_j w_j d + Sum_j w_j (u_j . d).
#pragma once
#include "cspt_kernels.cuh"
#include "cspt_tma.cuh"

namespace cspt {

// 1/sqrt(s) and sqrt(s) for s > 0, accurate to rounding level for the type.
template <class T> struct Fast;
template <> struct Fast<double> {
  // MUFU.RSQ64H seed (about 2^-20 relative) + one third-order step: y = y0 (1 + e/2 + 3e^2/8),
  // e = 1 - s y0^2;  sqrt(s) = s y0 (1 + e/2 + 3e^2/8).  Six FP64 instructions, no branches.
  static __device__ __forceinline__ void rsqrt_sqrt(double s, double& y, double& t) {
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(s));
    double t0 = s * y0;
    double e = fma(-t0, y0, 1.0);
    double ce = fma(0.375, e, 0.5) * e;
    y = fma(y0, ce, y0);
    t = fma(t0, ce, t0);
  }
  // comparisons of a positive double with 1 and 4 on the high word (integer pipe)
  static __device__ __forceinline__ bool lt1(double s) { return __double2hiint(s) < 0x3FF00000; }
  static __device__ __forceinline__ bool lt4(double s) { return __double2hiint(s) < 0x40100000; }
  static __device__ __forceinline__ double tiny() { return 1e-300; }
};
template <> struct Fast<float> {
  static __device__ __forceinline__ void rsqrt_sqrt(float s, float& y, float& t) {
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(s));
    t = s * y;
  }
  static __device__ __forceinline__ bool lt1(float s) { return s < 1.0f; }
  static __device__ __forceinline__ bool lt4(float s) { return s < 4.0f; }
  static __device__ __forceinline__ float tiny() { return 1e-30f; }
};

// Field order of the star group (slot S_ST): what the predictor hands to the corrector.
enum StarField { ST_PHI = 0, ST_U, ST_V, ST_W, ST_EX, ST_EY, ST_EZ, ST_E, ST_COUNT };

template <class T, int TX, int TY, int CY, int NST>
struct CorrSmem {
  // left x halo: 1 cell is needed; tiles start at cell i = -1 (padded index GX-1 = 3), so HXL = 1
  // (fp64) / 3 (fp32) puts every box row on a 16-byte boundary in global memory.
  static constexpr int HXL = sizeof(T) == 8 ? 1 : 3;
  static constexpr int BX = TX + HXL + 1;
  static constexpr int BY = TY + 2;
  static constexpr int NF = 7;                                   // phi*, u*, eta* (E* is read directly)
  static constexpr int PLANE = NF * BY * BX;                     // elements per stage
  static constexpr int STAGE = (PLANE * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int OFF_BAR = NST * STAGE;
  static constexpr int BYTES = OFF_BAR + 64 + 128;               // + slack for the 128-byte alignment
  static constexpr int THREADS = TX * (TY / CY);
  static_assert(TY % CY == 0, "TY must be a multiple of CY");
  static_assert((BX * sizeof(T)) % 16 == 0, "box rows must be multiples of 16 bytes");
};

template <class T, int TX, int TY, int CY, int NST>
__global__ void __launch_bounds__(TX*(TY / CY))
k_corrector_stream(const __grid_constant__ CUtensorMap mapS, Params<T> P, const DevScalars<T>* __restrict__ sc,
                   const T* __restrict__ U, const T* __restrict__ F, const T* __restrict__ ST, T* __restrict__ UT,
                   T* __restrict__ XI, int zchunk) {
  typedef CorrSmem<T, TX, TY, CY, NST> S;
  typedef Fast<T> FT;
  extern __shared__ __align__(128) unsigned char sm[];
  uint64_t* bar = (uint64_t*)(sm + S::OFF_BAR);
  const Layout& L = P.L;
  const int tid = threadIdx.x, tx = tid % TX, tq = tid / TX;
  const int i0 = -1 + (int)blockIdx.x * TX, j0 = -1 + (int)blockIdx.y * TY;
  // output planes [z0, z1) of the extended domain [-1, nz+1)
  const int z0 = -1 + (int)blockIdx.z * zchunk, z1 = min(L.nz + 1, z0 + zchunk);
  const int i = i0 + tx;
  const int ly0 = tq * CY;                          // first own row inside the tile
  const long long fs = L.fstride;
  constexpr uint32_t TX_BYTES = (uint32_t)(S::PLANE * sizeof(T));

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) mbar_init(&bar[s], 1);
    mbar_fence_init();
    prefetch_tmap(&mapS);
  }
  __syncthreads();
  auto slot_of = [&](int q) { return (q - (z0 - 1)) % NST; };
  auto issue = [&](int q) {              // plane q -> its ring slot
    int s = slot_of(q);
    mbar_expect_tx(&bar[s], TX_BYTES);
    tma_load_4d(sm + s * S::STAGE, &mapS, &bar[s], i0 + GX - S::HXL, j0 + NG - 1, q + NG, 0);
  };
  if (tid == 0) {
    for (int q = z0 - 1; q < z0 - 1 + NST && q <= z1; ++q) issue(q);
  }

  const T dt = load_dt(sc);
  const T hdt = (T)0.5 * dt, qdt = (T)0.25 * dt;
  const T pnorm = P.wnorm * P.h;                   // 1 / (S0' h): sums are in units of h
  uint32_t phase = 0;                              // bit s: parity to wait for on slot s
  auto wait_plane = [&](int q) {
    int s = slot_of(q);
    mbar_wait(&bar[s], (phase >> s) & 1u);
    phase ^= 1u << s;
  };
  wait_plane(z0 - 1);
  wait_plane(z0);

  for (int p = z0; p < z1; ++p) {
    wait_plane(p + 1);
    const T* pl[3] = {(const T*)(sm + slot_of(p - 1) * S::STAGE), (const T*)(sm + slot_of(p) * S::STAGE),
                      (const T*)(sm + slot_of(p + 1) * S::STAGE)};
    auto at = [&](const T* base, int f, int ly, int lx) { return base[(f * S::BY + (ly + 1)) * S::BX + (lx + S::HXL)]; };

    // own particles
    T phi_i[CY], ui[CY][3], ei[CY][3][3];        // ei[c][comp][o+1] = eta_i - o
    T sx[CY], sy[CY], sz[CY], se[CY];
    bool valid[CY];
#pragma unroll
    for (int c = 0; c < CY; ++c) {
      int ly = ly0 + c;
      valid[c] = i <= L.nx && (j0 + ly) <= L.ny;
      phi_i[c] = at(pl[1], ST_PHI, ly, tx);
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        ui[c][d] = at(pl[1], ST_U + d, ly, tx);
        T e = at(pl[1], ST_EX + d, ly, tx);
        ei[c][d][0] = e + (T)1; ei[c][d][1] = e; ei[c][d][2] = e - (T)1;
      }
      sx[c] = sy[c] = sz[c] = se[c] = (T)0;
    }
    bool any = false;
#pragma unroll
    for (int c = 0; c < CY; ++c) any = any || valid[c];

    if (any) {
#pragma unroll
      for (int oz = -1; oz <= 1; ++oz) {
        const T* sp = pl[oz + 1];
#pragma unroll
        for (int r = -1; r <= CY; ++r) {
#pragma unroll
          for (int ox = -1; ox <= 1; ++ox) {
            // is this neighbour particle used by any own cell?
            bool used = false;
#pragma unroll
            for (int c = 0; c < CY; ++c) {
              int oy = r - c;
              if (oy >= -1 && oy <= 1 && !(oz == 0 && oy == 0 && ox == 0)) used = true;
            }
            if (!used) continue;
            const int ly = ly0 + r, lx = tx + ox;
            const T pj = at(sp, ST_PHI, ly, lx);
            const T uj = at(sp, ST_U, ly, lx), vj = at(sp, ST_V, ly, lx), wj = at(sp, ST_W, ly, lx);
            const T exj = at(sp, ST_EX, ly, lx), eyj = at(sp, ST_EY, ly, lx), ezj = at(sp, ST_EZ, ly, lx);
#pragma unroll
            for (int c = 0; c < CY; ++c) {
              const int oy = r - c;
              if (oy < -1 || oy > 1 || (oz == 0 && oy == 0 && ox == 0)) continue;
              const T dx = ei[c][0][ox + 1] - exj, dy = ei[c][1][oy + 1] - eyj, dz = ei[c][2][oz + 1] - ezj;
              const T s = fma(dz, dz, fma(dy, dy, fma(dx, dx, FT::tiny())));
              T y, q;
              FT::rsqrt_sqrt(s, y, q);
              const T g1 = fma((T)-2.25, q, (T)3);
              const T g2 = fma((T)0.75, q, fma((T)3, y, (T)-3));
              const T g = FT::lt1(s) ? g1 : (FT::lt4(s) ? g2 : (T)0);
              const T w = pj * g;
              sx[c] = fma(w, dx, sx[c]); sy[c] = fma(w, dy, sy[c]); sz[c] = fma(w, dz, sz[c]);
              se[c] = fma(w, fma(wj, dz, fma(vj, dy, uj * dx)), se[c]);
            }
          }
        }
      }
    }

    // SUL{corrector}, Eq. (6)
#pragma unroll
    for (int c = 0; c < CY; ++c) {
      if (!valid[c]) continue;
      const int j = j0 + ly0 + c;
      const long long cc = L.idx(i, j, p);
      const T rho = U[cc], mxn = U[cc + fs], myn = U[cc + 2 * fs], mzn = U[cc + 3 * fs], En = U[cc + 4 * fs];
      const T fx = F[cc], fy = F[cc + fs], fz = F[cc + 2 * fs];
      const T Es = ST[cc + (long long)ST_E * fs];
      const bool ok = rho > P.rho_vac;
      const T ir = ok ? (T)1 / rho : (T)0;
      const T un = mxn * ir, vn = myn * ir, wn = mzn * ir;
      const T us = ui[c][0], vs = ui[c][1], ws = ui[c][2];
      // U* momentum: rho u* (a vacuum particle has phi = 0, so Q_m = rho f there)
      const T mxs = ok ? rho * us : fma(dt, rho * fx, mxn);
      const T mys = ok ? rho * vs : fma(dt, rho * fy, myn);
      const T mzs = ok ? rho * ws : fma(dt, rho * fz, mzn);
      const T pn = phi_i[c] * pnorm;
      const T set = se[c] + (us * sx[c] + vs * sy[c] + ws * sz[c]);
      const T qx = pn * sx[c] + rho * fx;
      const T qy = pn * sy[c] + rho * fy;
      const T qz = pn * sz[c] + rho * fz;
      const T qe = (T)0.5 * pn * set + rho * ((us * fx + vs * fy) + ws * fz);
      const T mx = (T)0.5 * (mxn + mxs) + hdt * qx;
      const T my = (T)0.5 * (myn + mys) + hdt * qy;
      const T mz = (T)0.5 * (mzn + mzs) + hdt * qz;
      const T E = (T)0.5 * (En + Es) + hdt * qe;
      UT[cc] = mx; UT[cc + fs] = my; UT[cc + 2 * fs] = mz; UT[cc + 3 * fs] = E;
      XI[cc] = (T)0.5 * (hdt * (un + us)) + qdt * (un + mx * ir);
      XI[cc + fs] = (T)0.5 * (hdt * (vn + vs)) + qdt * (vn + my * ir);
      XI[cc + 2 * fs] = (T)0.5 * (hdt * (wn + ws)) + qdt * (wn + mz * ir);
    }

    __syncthreads();                                 // everyone is done with plane p-1
    if (tid == 0 && p - 1 + NST <= z1) issue(p - 1 + NST);
  }
}

}  // namespace cspt
