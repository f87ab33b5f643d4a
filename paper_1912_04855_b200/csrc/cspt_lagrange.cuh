// cspt_lagrange.cuh -- Lagrangian stage (readings G1-G9) as two z-streaming kernels:
//   k_predictor_stream: primitives + HFC{predictor} + SUL{predictor}, Eq. (7) at the cell centres and Eq. (5);
//   k_corrector_stream: HFC{corrector} + SUL{corrector}, Eq. (7) at the displaced positions r* and Eq. (6).
//
// Corrector: one CTA owns a TX x TY column of cells of the extended domain interior(+)1 (G16) and streams
// along z.  The seven per-particle quantities of U*, r* that a NEIGHBOUR contributes to Eq. (7)
//     phi*, u*, v*, w*, eta* = xi*/h (3 components)
// (and E* of the own cell) arrive per plane as one TMA box of four pair arrays (halo 1 in x/y) in a 4-stage
// shared-memory ring: planes p-1, p, p+1 are resident while plane p is evaluated and plane p+2 is in flight.
// A thread owns CY cells adjacent in y, so that a neighbour particle read from shared memory serves up to CY
// cells; in fp32 the two cells share packed f32x2 arithmetic.
//
// Per neighbour (lengths in units of h):  d = (eta_i - o) - eta_j,  s = |d|^2,  y = 1/sqrt(s),
// q = s y,  g^(q) = -W'(q)/q of the cubic spline (G5):  3 - 2.25 q  (s < 1),
// 0.75 (2-q)^2 / q = 3 y - 3 + 0.75 q  (1 <= s < 4),  0 (s >= 4);  no division, no IEEE sqrt.
// Sum_j w_j (u_i + u_j).d is split as u_i . Sum_j w_j d + Sum_j w_j (u_j . d).
#pragma once
#include "cspt_kernels.cuh"
#include "cspt_tma.cuh"

namespace cspt {

// The star group (slot S_ST): what the predictor hands to the corrector.  The eight quantities are stored
// as four arrays of PAIRS interleaved along x,
//     (phi*, u*)  (v*, w*)  (eta*_x, eta*_y)  (eta*_z, E*)
// so that HBM sees four long streams instead of eight and a neighbour particle is four vector loads from
// shared memory.  Pair array k starts at element k * 2 * fstride; the pair of cell c sits at 2c, 2c+1.
enum StarPair { SP_PHI_U = 0, SP_V_W, SP_EX_EY, SP_EZ_E, SP_COUNT };
template <class T> struct Pair;
template <> struct Pair<double> { typedef double2 type; static __device__ __forceinline__ double2 make(double a, double b) { return make_double2(a, b); } };
template <> struct Pair<float> { typedef float2 type; static __device__ __forceinline__ float2 make(float a, float b) { return make_float2(a, b); } };

// ---- O1 + O3 + O4: primitives, HFC{predictor}, SUL{predictor} as one z-streaming kernel -------------
// Eq. (7) with the particles at the cell centres is the lattice operator
//   S_c = sum_o a(|o|^2) o_c phi_{i+o},   T = sum_c sum_o a(|o|^2) o_c (phi u_c)_{i+o}
// (Q_m = -phi_i S / h + rho f,  Q_E = -phi_i (u_i . S + T) / (2h) + rho u_i . f;  G1-G6).
// One CTA owns a TX x TY column of the extended domain interior(+)2 and streams along z.  Per plane q
// one TMA box of U^n (tile + halo 1) and one of f land in a two-stage shared-memory ring, two planes ahead of their
// use (PredRing; the earlier version loaded them into registers one plane ahead and spent 19 % of its warp cycles
// waiting for the first of them and 24 % at the barrier behind it); the threads turn them into phi, phi u, phi v,
// phi w of the (TX+2) x (TY+2) cells in a 2-slot shared-memory buffer; every thread then forms the IN-PLANE parts of the
// sums of plane q for its column: with the |o_z| = 1 weights they belong to the particles of planes
// q-1 and q+1 (sign of the z terms flipped), with the o_z = 0 weights to plane q.  The running sums
// of the two particles in flight live in registers; particle q-1 is finished (Eq. (5)) when plane q
// has been added.  Output: the star group the corrector reads (phi*, u*, eta*, E*).
template <class T>
__device__ __forceinline__ Prim<T> prim_quick(T rho, T mx, T my, T mz, T E, T gamma, T rho_vac) {
  typedef Fast<T> FT;
  Prim<T> q;
  q.ok = rho > rho_vac;
  T ir = q.ok ? FT::rcp(rho) : (T)0;
  q.u = mx * ir; q.v = my * ir; q.w = mz * ir;
  T ke2 = (mx * q.u + my * q.v) + mz * q.w;
  T pp = (gamma - (T)1) * (E - (T)0.5 * ke2);
  q.p = q.ok ? (pp > (T)0 ? pp : (T)0) : (T)0;
  q.phi = FT::sqrt0((T)2 * q.p);
  return q;
}

template <class T, int TX, int TY>
struct PredSmem {
  static constexpr int BX = TX + 2, BY = TY + 2;
  static constexpr int NHALO = BX * BY - TX * TY;
  static constexpr int PLANE = 4 * BY * BX;              // phi, phi u, phi v, phi w
  static_assert(NHALO <= TX * TY, "one halo cell per thread at most");
};

// TMA ring of the predictor's inputs (NSTG > 0): per plane one box of U^n (5 fields, tile + halo 1) and one of f (3
// fields, tile) land in a stage of dynamic shared memory, NSTG planes ahead of their use; the boxes start on a 16-byte
// boundary in x (A elements) and are wide enough for the tile whatever the remainder.
template <class T, int TX, int TY, int NSTG>
struct PredRing {
  static constexpr int A = 16 / (int)sizeof(T);
  static constexpr int BXT = sizeof(T) == 8 ? 36 : 40;
  static constexpr int U_ELEMS = 5 * (TY + 2) * BXT, F_ELEMS = 3 * TY * BXT;
  static constexpr int U_BYTES = U_ELEMS * (int)sizeof(T), F_BYTES = F_ELEMS * (int)sizeof(T);
  static constexpr int OFF_F = (U_BYTES + 127) / 128 * 128;
  static constexpr int STAGE = (OFF_F + F_BYTES + 127) / 128 * 128;
  static constexpr int OFF_BAR = NSTG * STAGE;
  static constexpr int BYTES = NSTG > 0 ? OFF_BAR + 8 * NSTG + 128 : 0;    // + slack for the 128-byte alignment
};

template <class T, int TX, int TY, int NSTG = 0>
__global__ void __launch_bounds__(TX* TY, (sizeof(T) == 4 ? 768 : 512) / (TX * TY))
k_predictor_stream(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapF, Params<T> P,
                   const DevScalars<T>* __restrict__ sc, const T* __restrict__ U, const T* __restrict__ F,
                   T* __restrict__ ST, int zchunk, int x0, int x1, BrickMap M) {      // particle columns [x0, x1)
  typedef PredSmem<T, TX, TY> S;
  typedef PredRing<T, TX, TY, NSTG> R;
  __shared__ T sbuf[2][S::PLANE];
  extern __shared__ unsigned char ring_raw[];
  unsigned char* ring = (unsigned char*)(((uintptr_t)ring_raw + 127) & ~(uintptr_t)127);
  uint64_t* bar = (uint64_t*)(ring + R::OFF_BAR);
  const Layout& L = P.L;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int i0 = x0 + (int)blockIdx.x * TX, j0 = -2 + (int)blockIdx.y * TY;
  const int z0 = -2 + (int)blockIdx.z * zchunk, z1 = min(L.nz + 2, z0 + zchunk);   // particle planes [z0, z1)
  const long long fs = L.fstride;
  // own cell: its primitives are needed up to ghost layer 3 (neighbour of the last particle), the
  // particle itself exists up to layer 2; beyond that the index is clamped and the result unused
  const int i = min(i0 + tx, L.nx + 2), j = min(j0 + ty, L.ny + 2);
  const bool valid = (i0 + tx) < x1 && (j0 + ty) <= L.ny + 1;
  // halo cell of this thread (tile coordinates -1..TX, -1..TY)
  const bool has_halo = tid < S::NHALO;
  int hx, hy;
  if (tid < S::BX) { hx = tid - 1; hy = -1; }
  else if (tid < 2 * S::BX) { hx = tid - S::BX - 1; hy = TY; }
  else { int t = tid - 2 * S::BX; hx = (t & 1) ? TX : -1; hy = t >> 1; }
  const int hi = min(i0 + hx, L.nx + 2), hj = min(j0 + hy, L.ny + 2);
  const long long c_own = L.idx(i, j, 0), c_halo = L.idx(hi, hj, 0), sz = L.sz();

  // all inputs within reach of this CTA exactly 0 (BrickMap): the star group of its particles is exactly 0
  if (M.raw && cta_region_dead(M, L, i0 + GX - 3, i0 + TX + GX + 3, j0 + NG - 3, j0 + TY + NG + 3, z0 + NG - 3, z1 + NG + 3)) {
    if (valid && M.zero_fill) {
      typedef typename Pair<T>::type V2;
      const V2 zero = Pair<T>::make((T)0, (T)0);
      for (int q = z0; q < z1; ++q) {
        V2* st2 = (V2*)ST + c_own + (long long)q * sz;
#pragma unroll
        for (int k = 0; k < 4; ++k) st2[k * fs] = zero;
#pragma unroll
        for (int g = 0; g < 4; ++g) {            // periodic x: the ghost columns this particle wraps onto
          const int xd = g < 2 ? g - 2 : L.nx + (g - 2);
          if (x0 == 0 && ((xd % L.nx) + L.nx) % L.nx == i0 + tx) {
#pragma unroll
            for (int k = 0; k < 4; ++k) st2[xd - (i0 + tx) + k * fs] = zero;
          }
        }
      }
    }
    return;
  }

  const T dt = load_dt(sc);
  const T he = (T)0.5 * dt * P.inv_h;
  const T a1 = P.a1, a2 = P.a2, a3 = P.a3;

  auto put = [&](T* sb, int ly, int lx, const Prim<T>& q) {
    int o = (ly + 1) * S::BX + (lx + 1);
    sb[o] = q.phi; sb[S::BY * S::BX + o] = q.phi * q.u; sb[2 * S::BY * S::BX + o] = q.phi * q.v;
    sb[3 * S::BY * S::BX + o] = q.phi * q.w;
  };

  // TMA ring: box start (padded x index rounded down to a 16-byte boundary) and this thread's columns inside the box
  const int bxs = ((i0 - 1 + GX) / R::A) * R::A, lxo = (i0 - 1 + GX) - bxs;
  auto slot_of = [&](int qq) { return (qq - (z0 - 1)) % (NSTG > 0 ? NSTG : 1); };
  auto issue = [&](int qq) {
    const int k = slot_of(qq);
    mbar_expect_tx(&bar[k], (uint32_t)(R::U_BYTES + R::F_BYTES));
    tma_load_4d(ring + k * R::STAGE, &mapU, &bar[k], bxs, j0 - 1 + NG, qq + NG, 0);
    tma_load_4d(ring + k * R::STAGE + R::OFF_F, &mapF, &bar[k], bxs, j0 + NG, qq + NG, 0);
  };
  uint32_t phase = 0;
  T Uo[5], Uh[5];                 // plane q: own and halo cell, loaded one iteration ahead
  if (NSTG == 0) {
    const long long co = c_own + (long long)(z0 - 1) * sz, ch = c_halo + (long long)(z0 - 1) * sz;
#pragma unroll
    for (int f = 0; f < 5; ++f) { Uo[f] = __ldg(U + co + f * fs); Uh[f] = has_halo ? __ldg(U + ch + f * fs) : (T)0; }
  } else {
    if (tid == 0) {
#pragma unroll
      for (int k = 0; k < NSTG; ++k) mbar_init(&bar[k], 1);
      mbar_fence_init();
      prefetch_tmap(&mapU);
      prefetch_tmap(&mapF);
    }
    __syncthreads();
    if (tid == 0)
      for (int qq = z0 - 1; qq < z0 - 1 + NSTG && qq <= z1; ++qq) issue(qq);
  }
  // periodic x (x0 == 0: interior columns only): the ghost columns -2, -1, nx, nx+1 hold what this kernel would
  // compute there, i.e. the value of the column they wrap onto (same inputs, same arithmetic); woff[g] is the
  // offset from this thread's particle to ghost column g if it wraps onto the particle, else 0
  int woff[4];
#pragma unroll
  for (int g = 0; g < 4; ++g) {
    const int xd = g < 2 ? g - 2 : L.nx + (g - 2);
    woff[g] = (x0 == 0 && ((xd % L.nx) + L.nx) % L.nx == i0 + tx) ? xd - (i0 + tx) : 0;
  }
  T fn[3] = {0, 0, 0};            // force of particle q, requested one iteration before it is needed
  T Uc[5] = {0, 0, 0, 0, 0};      // particle q-1: U^n and primitives
  Prim<T> pc; pc.u = pc.v = pc.w = pc.p = pc.phi = (T)0; pc.ok = false;
  T acc0[4] = {0, 0, 0, 0}, acc1[4] = {0, 0, 0, 0};

  for (int q = z0 - 1; q <= z1; ++q) {
    T* sb = sbuf[(q - (z0 - 1)) & 1];
    T fstage[3] = {0, 0, 0};
    if (NSTG > 0) {               // plane q has landed: own and halo cell of U^n, f of particle q
      const int k = slot_of(q);
      mbar_wait(&bar[k], (phase >> k) & 1u);
      phase ^= 1u << k;
      const T* sU = (const T*)(ring + k * R::STAGE);
      const T* sF = (const T*)(ring + k * R::STAGE + R::OFF_F);
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        Uo[f] = sU[(f * (TY + 2) + ty + 1) * R::BXT + lxo + 1 + tx];
        Uh[f] = has_halo ? sU[(f * (TY + 2) + hy + 1) * R::BXT + lxo + 1 + hx] : (T)0;
      }
#pragma unroll
      for (int f = 0; f < 3; ++f) fstage[f] = sF[(f * TY + ty) * R::BXT + lxo + 1 + tx];
    }
    // O1 for plane q
    Prim<T> po = prim_quick<T>(Uo[0], Uo[1], Uo[2], Uo[3], Uo[4], P.gamma, P.rho_vac);
    put(sb, ty, tx, po);
    if (has_halo) {
      Prim<T> ph = prim_quick<T>(Uh[0], Uh[1], Uh[2], Uh[3], Uh[4], P.gamma, P.rho_vac);
      put(sb, hy, hx, ph);
    }
    T Un[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) Un[f] = Uo[f];
    // request plane q+1 and the force of particle q (used in the next iteration)
    T fq[3];
#pragma unroll
    for (int f = 0; f < 3; ++f) fq[f] = fn[f];
    if (NSTG > 0) {
#pragma unroll
      for (int f = 0; f < 3; ++f) fn[f] = fstage[f];
    } else if (q < z1) {
      const long long co = c_own + (long long)(q + 1) * sz, ch = c_halo + (long long)(q + 1) * sz;
#pragma unroll
      for (int f = 0; f < 5; ++f) { Uo[f] = __ldg(U + co + f * fs); if (has_halo) Uh[f] = __ldg(U + ch + f * fs); }
      if (q >= z0) {
        const long long cf = c_own + (long long)q * sz;
#pragma unroll
        for (int f = 0; f < 3; ++f) fn[f] = __ldg(F + cf + f * fs);
      }
    }
    const long long cs = c_own + (long long)(q - 1) * sz;       // particle q-1
    __syncthreads();
    if (NSTG > 0 && tid == 0 && q + NSTG <= z1) issue(q + NSTG);   // everyone has read stage q

    // in-plane parts of the lattice sums of plane q (tile coordinates of the own column: tx, ty)
    auto at = [&](int f, int oy, int ox) { return sb[(f * S::BY + (ty + 1 + oy)) * S::BX + (tx + 1 + ox)]; };
    T A0x, A0y, T0, A1x, A1y, A1z, T1xy, T1z;
    {
      // phi: x and y differences, and the plain 3x3 sum
      T pmm = at(0, -1, -1), pm0 = at(0, -1, 0), pmp = at(0, -1, 1);
      T p0m = at(0, 0, -1), p00 = at(0, 0, 0), p0p = at(0, 0, 1);
      T ppm = at(0, 1, -1), pp0 = at(0, 1, 0), ppp = at(0, 1, 1);
      T dx0 = p0p - p0m, dxs = (pmp - pmm) + (ppp - ppm);        // o_y = 0; o_y = +-1
      T dy0 = pp0 - pm0, dys = (ppm - pmm) + (ppp - pmp);        // o_x = 0; o_x = +-1
      A0x = a1 * dx0 + a2 * dxs;  A1x = a2 * dx0 + a3 * dxs;
      A0y = a1 * dy0 + a2 * dys;  A1y = a2 * dy0 + a3 * dys;
      A1z = a1 * p00 + a2 * ((p0m + p0p) + (pm0 + pp0)) + a3 * ((pmm + pmp) + (ppm + ppp));
      // phi u: x differences;  phi v: y differences
      T ux0 = at(1, 0, 1) - at(1, 0, -1), uxs = (at(1, -1, 1) - at(1, -1, -1)) + (at(1, 1, 1) - at(1, 1, -1));
      T vy0 = at(2, 1, 0) - at(2, -1, 0), vys = (at(2, 1, -1) - at(2, -1, -1)) + (at(2, 1, 1) - at(2, -1, 1));
      T0 = a1 * (ux0 + vy0) + a2 * (uxs + vys);
      T1xy = a2 * (ux0 + vy0) + a3 * (uxs + vys);
      // phi w: plain 3x3 sum
      T1z = a1 * at(3, 0, 0) + a2 * ((at(3, 0, -1) + at(3, 0, 1)) + (at(3, -1, 0) + at(3, 1, 0))) +
            a3 * ((at(3, -1, -1) + at(3, -1, 1)) + (at(3, 1, -1) + at(3, 1, 1)));
    }

    // particle q-1: plane q is its o_z = +1 layer; Eq. (7) and Eq. (5)
    if (q - 1 >= z0 && valid) {
      const T Sx = acc0[0] + A1x, Sy = acc0[1] + A1y, Sz = acc0[2] + A1z, Tt = acc0[3] + (T1xy + T1z);
      const T rho = Uc[0];
      const T ui = pc.u, vi = pc.v, wi = pc.w;
      const T pn = pc.phi * P.inv_h;
      const T qx = rho * fq[0] - pn * Sx;
      const T qy = rho * fq[1] - pn * Sy;
      const T qz = rho * fq[2] - pn * Sz;
      const T qe = rho * ((ui * fq[0] + vi * fq[1]) + wi * fq[2]) - (T)0.5 * pn * (((ui * Sx + vi * Sy) + wi * Sz) + Tt);
      const T mx = Uc[1] + dt * qx, my = Uc[2] + dt * qy, mz = Uc[3] + dt * qz, E = Uc[4] + dt * qe;
      Prim<T> ps = prim_quick<T>(rho, mx, my, mz, E, P.gamma, P.rho_vac);
      typedef typename Pair<T>::type V2;
      V2* st2 = (V2*)ST + cs;                       // pair array k: + k * fs pairs
      const V2 o0 = Pair<T>::make(ps.phi, ps.u), o1 = Pair<T>::make(ps.v, ps.w);
      const V2 o2 = Pair<T>::make(he * (ui + ps.u), he * (vi + ps.v)), o3 = Pair<T>::make(he * (wi + ps.w), E);
      st2[0] = o0; st2[fs] = o1; st2[2 * fs] = o2; st2[3 * fs] = o3;
#pragma unroll
      for (int g = 0; g < 4; ++g)
        if (woff[g]) {                          // periodic x: the ghost column this particle wraps onto
          V2* w2 = st2 + woff[g];
          w2[0] = o0; w2[fs] = o1; w2[2 * fs] = o2; w2[3 * fs] = o3;
        }
    }
    // particle q: had plane q-1 as its o_z = -1 layer, plane q is its own layer
    acc0[0] = acc1[0] + A0x; acc0[1] = acc1[1] + A0y; acc0[2] = acc1[2]; acc0[3] = acc1[3] + T0;
    // particle q+1: plane q is its o_z = -1 layer
    acc1[0] = A1x; acc1[1] = A1y; acc1[2] = -A1z; acc1[3] = T1xy - T1z;
#pragma unroll
    for (int f = 0; f < 5; ++f) Uc[f] = Un[f];
    pc = po;
  }
}


// ---- fp32, two cells per thread: the neighbour sums of both cells in the two halves of packed f32x2 registers
// (FFMA2 / FADD2 / FMUL2, sm_100): lane x = own cell 0, lane y = own cell 1.  The fp32 corrector is bound by the
// instruction issue rate, and one packed evaluation replaces two scalar ones.  Rows 0 and 1 of the thread's
// neighbourhood serve both cells (the same particle, offsets o_y = r and r - 1); row -1 serves only cell 0 and
// row 2 only cell 1: those two particles share one packed evaluation.  The self term is evaluated too: its d is
// exactly 0, so it adds exactly 0.
template <int KERN>
__device__ __forceinline__ void pair_eval_f32x2(float2 dx, float2 dy, float2 dz, float2 pj, float2 uj, float2 vj,
                                                float2 wj, float2& sx, float2& sy, float2& sz, float2& se) {
  const float2 tiny = make_float2(1e-30f, 1e-30f);
  const float2 s = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __ffma2_rn(dx, dx, tiny)));
  float2 g;
  if (KERN == 1) {
    const float2 t = __ffma2_rn(make_float2(-0.25f, -0.25f), s, make_float2(1.f, 1.f));
    const float2 t2 = __fmul2_rn(t, t), t4 = __fmul2_rn(t2, t2);
    g.x = s.x < 4.f ? t4.x : 0.f;
    g.y = s.y < 4.f ? t4.y : 0.f;
  } else {
    float2 y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y.x) : "f"(s.x));
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y.y) : "f"(s.y));
    const float2 q = __fmul2_rn(s, y);
    const float2 g1 = __ffma2_rn(make_float2(-2.25f, -2.25f), q, make_float2(3.f, 3.f));
    const float2 g2 = __ffma2_rn(make_float2(0.75f, 0.75f), q,
                                 __ffma2_rn(make_float2(3.f, 3.f), y, make_float2(-3.f, -3.f)));
    g.x = s.x < 1.f ? g1.x : (s.x < 4.f ? g2.x : 0.f);
    g.y = s.y < 1.f ? g1.y : (s.y < 4.f ? g2.y : 0.f);
  }
  const float2 w = __fmul2_rn(pj, g);
  sx = __ffma2_rn(w, dx, sx); sy = __ffma2_rn(w, dy, sy); sz = __ffma2_rn(w, dz, sz);
  se = __ffma2_rn(w, __ffma2_rn(wj, dz, __ffma2_rn(vj, dy, __fmul2_rn(uj, dx))), se);
}

template <int KERN, class At>
__device__ __forceinline__ void neighbours_f32x2(const float2* const* pl, At at, int ly0, int tx, const float (*ei)[3][3],
                                                 float* sx, float* sy, float* sz, float* se) {
  float2 ex[3], ez[3];
#pragma unroll
  for (int o = 0; o < 3; ++o) { ex[o] = make_float2(ei[0][0][o], ei[1][0][o]); ez[o] = make_float2(ei[0][2][o], ei[1][2][o]); }
  // eta_y - o_y: row r is o_y = r for cell 0 and o_y = r - 1 for cell 1
  const float2 ey_r0 = make_float2(ei[0][1][1], ei[1][1][0]), ey_r1 = make_float2(ei[0][1][2], ei[1][1][1]);
  const float2 ey_edge = make_float2(ei[0][1][0], ei[1][1][2]);       // row -1 for cell 0, row 2 for cell 1
  float2 ax = make_float2(0.f, 0.f), ay = ax, az = ax, ae = ax;
  auto bc = [](float v) { return make_float2(v, v); };
#pragma unroll
  for (int oz = -1; oz <= 1; ++oz) {
    const float2* sp = pl[oz + 1];
#pragma unroll
    for (int ox = -1; ox <= 1; ++ox) {
      const int lx = tx + ox;
#pragma unroll
      for (int r = 0; r <= 1; ++r) {
        const float2 b0 = at(sp, SP_PHI_U, ly0 + r, lx), b1 = at(sp, SP_V_W, ly0 + r, lx);
        const float2 b2 = at(sp, SP_EX_EY, ly0 + r, lx), b3 = at(sp, SP_EZ_E, ly0 + r, lx);
        pair_eval_f32x2<KERN>(__fadd2_rn(ex[ox + 1], bc(-b2.x)), __fadd2_rn(r ? ey_r1 : ey_r0, bc(-b2.y)),
                              __fadd2_rn(ez[oz + 1], bc(-b3.x)), bc(b0.x), bc(b0.y), bc(b1.x), bc(b1.y), ax, ay, az, ae);
      }
      {
        const float2 a0 = at(sp, SP_PHI_U, ly0 - 1, lx), a1 = at(sp, SP_V_W, ly0 - 1, lx);
        const float2 a2 = at(sp, SP_EX_EY, ly0 - 1, lx), a3 = at(sp, SP_EZ_E, ly0 - 1, lx);
        const float2 c0 = at(sp, SP_PHI_U, ly0 + 2, lx), c1 = at(sp, SP_V_W, ly0 + 2, lx);
        const float2 c2 = at(sp, SP_EX_EY, ly0 + 2, lx), c3 = at(sp, SP_EZ_E, ly0 + 2, lx);
        pair_eval_f32x2<KERN>(__fadd2_rn(ex[ox + 1], make_float2(-a2.x, -c2.x)),
                              __fadd2_rn(ey_edge, make_float2(-a2.y, -c2.y)),
                              __fadd2_rn(ez[oz + 1], make_float2(-a3.x, -c3.x)), make_float2(a0.x, c0.x),
                              make_float2(a0.y, c0.y), make_float2(a1.x, c1.x), make_float2(a1.y, c1.y), ax, ay, az, ae);
      }
    }
  }
  sx[0] = ax.x; sx[1] = ax.y; sy[0] = ay.x; sy[1] = ay.y; sz[0] = az.x; sz[1] = az.y; se[0] = ae.x; se[1] = ae.y;
}

template <class T, int TX, int TY, int CY, int NST, int XP>
struct CorrSmem {
  // halo 1 in x and y.  XP = 0: tiles start at cell i = -1 (padded index GX-1 = 3) and the box one cell to the
  // left, pair index 2: a 16-byte boundary in global memory in both precisions.  XP = 1 (periodic x, interior
  // columns only): tiles start at i = 0; in fp32 the box then starts two cells to the left (pair index 2 again).
  static constexpr int X0 = XP ? 0 : -1;
  static constexpr int HXL = (XP && sizeof(T) == 4) ? 2 : 1;
  static constexpr int BX = TX + HXL + ((XP && sizeof(T) == 4) ? 2 : 1);
  static constexpr int BY = TY + 2;
  static constexpr int NF = SP_COUNT;                            // pair arrays
  static constexpr int PLANE = NF * BY * BX * 2;                 // elements per stage
  static constexpr int STAGE = (PLANE * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int OFF_BAR = NST * STAGE;
  static constexpr int BYTES = OFF_BAR + 64 + 128;               // + slack for the 128-byte alignment
  static constexpr int THREADS = TX * (TY / CY);
  static_assert(TY % CY == 0, "TY must be a multiple of CY");
  static_assert((2 * BX * sizeof(T)) % 16 == 0, "box rows must be multiples of 16 bytes");
};

template <class T, int TX, int TY, int CY, int NST, int MINB, int KERN, int XP>
__global__ void __launch_bounds__(TX*(TY / CY), MINB)
k_corrector_stream(const __grid_constant__ CUtensorMap mapS, Params<T> P, const DevScalars<T>* __restrict__ sc,
                   const T* __restrict__ U, const T* __restrict__ F, const T* __restrict__ ST, T* __restrict__ UT,
                   T* __restrict__ XI, int zchunk, BrickMap M) {
  typedef CorrSmem<T, TX, TY, CY, NST, XP> S;
  typedef Fast<T> FT;
  extern __shared__ __align__(128) unsigned char sm[];
  uint64_t* bar = (uint64_t*)(sm + S::OFF_BAR);
  const Layout& L = P.L;
  const int tid = threadIdx.x, tx = tid % TX, tq = tid / TX;
  const int i0 = S::X0 + (int)blockIdx.x * TX, j0 = -1 + (int)blockIdx.y * TY;
  // output planes [z0, z1) of the extended domain [-1, nz+1)
  const int z0 = -1 + (int)blockIdx.z * zchunk, z1 = min(L.nz + 1, z0 + zchunk);
  const int i = i0 + tx;
  const int ly0 = tq * CY;                          // first own row inside the tile
  const long long fs = L.fstride;
  constexpr uint32_t TX_BYTES = (uint32_t)(S::PLANE * sizeof(T));

  // all inputs within reach of this CTA exactly 0 (BrickMap): U~ and xi of its cells are exactly 0
  if (M.raw && cta_region_dead(M, L, i0 + GX - 3, i0 + TX + GX + 3, j0 + NG - 3, j0 + TY + NG + 3, z0 + NG - 3, z1 + NG + 3)) {
    for (int p = z0; p < z1 && M.zero_fill; ++p) {
#pragma unroll
      for (int c = 0; c < CY; ++c) {
        const int j = j0 + ly0 + c;
        if (!(i < L.nx + (XP ? 0 : 1) && j <= L.ny)) continue;
        const long long cc = L.idx(i, j, p);
#pragma unroll
        for (int f = 0; f < 4; ++f) UT[cc + f * fs] = (T)0;
#pragma unroll
        for (int f = 0; f < 3; ++f) XI[cc + f * fs] = (T)0;
        if (XP) {
#pragma unroll
          for (int g = 0; g < 2; ++g) {
            const int xd = g ? L.nx : -1;
            if (((xd % L.nx) + L.nx) % L.nx == i) {
              const long long cw = cc + (xd - i);
#pragma unroll
              for (int f = 0; f < 4; ++f) UT[cw + f * fs] = (T)0;
#pragma unroll
              for (int f = 0; f < 3; ++f) XI[cw + f * fs] = (T)0;
            }
          }
        }
      }
    }
    return;
  }

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
    tma_load_4d(sm + s * S::STAGE, &mapS, &bar[s], 2 * (i0 + GX - S::HXL), j0 + NG - 1, q + NG, 0);
  };
  if (tid == 0) {
    for (int q = z0 - 1; q < z0 - 1 + NST && q <= z1; ++q) issue(q);
  }

  // periodic x (XP: interior columns only): ghost columns -1 and nx hold the value of the column they wrap
  // onto; woff[g] = offset from this thread's cell to ghost column g if it wraps onto the cell, else 0
  int woff[2];
#pragma unroll
  for (int g = 0; g < 2; ++g) {
    const int xd = g ? L.nx : -1;
    woff[g] = (XP && ((xd % L.nx) + L.nx) % L.nx == i) ? xd - i : 0;
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
    typedef typename Pair<T>::type V2;
    const V2* pl[3] = {(const V2*)(sm + slot_of(p - 1) * S::STAGE), (const V2*)(sm + slot_of(p) * S::STAGE),
                       (const V2*)(sm + slot_of(p + 1) * S::STAGE)};
    auto at = [&](const V2* base, int k, int ly, int lx) { return base[(k * S::BY + (ly + 1)) * S::BX + (lx + S::HXL)]; };

    // own particles
    T phi_i[CY], ui[CY][3], ei[CY][3][3], Es_i[CY];        // ei[c][comp][o+1] = eta_i - o
    T sx[CY], sy[CY], sz[CY], se[CY];
    bool valid[CY];
#pragma unroll
    for (int c = 0; c < CY; ++c) {
      int ly = ly0 + c;
      valid[c] = i < L.nx + (XP ? 0 : 1) && (j0 + ly) <= L.ny;
      const V2 a0 = at(pl[1], SP_PHI_U, ly, tx), a1 = at(pl[1], SP_V_W, ly, tx);
      const V2 a2 = at(pl[1], SP_EX_EY, ly, tx), a3 = at(pl[1], SP_EZ_E, ly, tx);
      phi_i[c] = a0.x; ui[c][0] = a0.y; ui[c][1] = a1.x; ui[c][2] = a1.y;
      Es_i[c] = a3.y;
      const T ee[3] = {a2.x, a2.y, a3.x};
#pragma unroll
      for (int d = 0; d < 3; ++d) { ei[c][d][0] = ee[d] + (T)1; ei[c][d][1] = ee[d]; ei[c][d][2] = ee[d] - (T)1; }
      sx[c] = sy[c] = sz[c] = se[c] = (T)0;
    }
    // a particle with phi = 0 (vacuum, or p floored to 0) neither exerts nor feels the pressure force: all four
    // sums of such a cell are multiplied by phi_i = 0 in Eq. (7), so a warp whose own particles all have phi = 0
    // skips the neighbour loop (gas-vacuum workloads: most of the 1024^3 disk volume)
    bool any = false;
#pragma unroll
    for (int c = 0; c < CY; ++c) any = any || (valid[c] && phi_i[c] != (T)0);
    any = __any_sync(0xffffffffu, any);
    // own-cell operands of Eq. (6) straight from global memory, requested before the neighbour loop
    // so that their latency is hidden behind it
    T own[CY][8];
#pragma unroll
    for (int c = 0; c < CY; ++c) {
      const long long cc = L.idx(valid[c] ? i : 0, valid[c] ? j0 + ly0 + c : 0, p);
#pragma unroll
      for (int f = 0; f < 5; ++f) own[c][f] = __ldg(U + cc + f * fs);
#pragma unroll
      for (int f = 0; f < 3; ++f) own[c][5 + f] = __ldg(F + cc + f * fs);
    }

    if constexpr (sizeof(T) == 4 && CY == 2) {
      if (any) neighbours_f32x2<KERN>(pl, at, ly0, tx, ei, sx, sy, sz, se);
    } else if (any) {
#pragma unroll
      for (int oz = -1; oz <= 1; ++oz) {
        const V2* sp = pl[oz + 1];
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
            const V2 b0 = at(sp, SP_PHI_U, ly, lx), b1 = at(sp, SP_V_W, ly, lx);
            const V2 b2 = at(sp, SP_EX_EY, ly, lx), b3 = at(sp, SP_EZ_E, ly, lx);
            const T pj = b0.x, uj = b0.y, vj = b1.x, wj = b1.y, exj = b2.x, eyj = b2.y, ezj = b3.x;
#pragma unroll
            for (int c = 0; c < CY; ++c) {
              const int oy = r - c;
              if (oy < -1 || oy > 1 || (oz == 0 && oy == 0 && ox == 0)) continue;
              const T dx = ei[c][0][ox + 1] - exj, dy = ei[c][1][oy + 1] - eyj, dz = ei[c][2][oz + 1] - ezj;
              const T s = fma(dz, dz, fma(dy, dy, fma(dx, dx, FT::tiny())));
              T g;
              if (KERN == 1) {                       // W ~ (1 - q^2/4)^5: g^ = (1 - s/4)^4 on s < 4
                const T t = fma((T)-0.25, s, (T)1), t2 = t * t;
                g = FT::lt4(s) ? t2 * t2 : (T)0;
              } else {                               // cubic spline (G5)
                T y, q;
                FT::rsqrt_sqrt(s, y, q);
                const T g1 = fma((T)-2.25, q, (T)3);
                const T g2 = fma((T)0.75, q, fma((T)3, y, (T)-3));
                g = FT::lt1(s) ? g1 : (FT::lt4(s) ? g2 : (T)0);
              }
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
      const T rho = own[c][0], mxn = own[c][1], myn = own[c][2], mzn = own[c][3], En = own[c][4];
      const T fx = own[c][5], fy = own[c][6], fz = own[c][7];
      const T Es = Es_i[c];
      const bool ok = rho > P.rho_vac;
      const T ir = ok ? FT::rcp(rho) : (T)0;
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
      const T xo[3] = {(T)0.5 * (hdt * (un + us)) + qdt * (un + mx * ir), (T)0.5 * (hdt * (vn + vs)) + qdt * (vn + my * ir),
                       (T)0.5 * (hdt * (wn + ws)) + qdt * (wn + mz * ir)};
      UT[cc] = mx; UT[cc + fs] = my; UT[cc + 2 * fs] = mz; UT[cc + 3 * fs] = E;
      XI[cc] = xo[0]; XI[cc + fs] = xo[1]; XI[cc + 2 * fs] = xo[2];
      if (XP) {
#pragma unroll
        for (int g = 0; g < 2; ++g)
          if (woff[g]) {                        // periodic x: the ghost column this cell wraps onto
            const long long cw = cc + woff[g];
            UT[cw] = mx; UT[cw + fs] = my; UT[cw + 2 * fs] = mz; UT[cw + 3 * fs] = E;
            XI[cw] = xo[0]; XI[cw + fs] = xo[1]; XI[cw + 2 * fs] = xo[2];
          }
      }
    }

    __syncthreads();                                 // everyone is done with plane p-1
    if (tid == 0 && p - 1 + NST <= z1) issue(p - 1 + NST);
  }
}

}  // namespace cspt
