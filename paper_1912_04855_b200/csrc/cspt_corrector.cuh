// cspt_corrector.cuh -- HFC{corrector} + SUL{corrector} (Eq. (7) at the displaced
// positions r*, Eq. (6)) with PAIR-SYMMETRIC evaluation of the SPH sums.
//
// Eq. (7) sums over pairs of particles: for the pair (i, j), d = r_i - r_j, |d|^2, the square root and the kernel
// factor g^(|d|) = -W'(|d|)/|d| are the same for both ends; only phi, u and the sign of d differ,
//     S_i += phi_j g d,   SE_i += phi_j g (u_j . d);      S_j -= phi_i g d,   SE_j -= phi_i g (u_i . d).
// A pair whose two ends are held by the same warp is therefore evaluated ONCE ("shared pair").
//
// Layout: a warp owns 32 columns (lane = x) of a strip of two rows (y) and streams along z; a CTA stacks TY/2
// strips.  Per iteration p the warp holds the particles of its own cells of planes p ("cur") and p+1 ("nxt") in
// registers and evaluates every pair between planes p and p, and between planes p and p+1 (the pairs between p+1
// and p+1 follow in the next iteration), so that a plane of the star group is read from shared memory for two
// iterations instead of three and the sums of the plane p+1 cells are carried in registers:
//   * own-own pairs (same lane: 1 in plane p, 4 between the planes): shared, both ends in registers;
//   * pairs with the cells of the lane to the right (12): shared, the partner's part goes to lane + 1 by warp
//     shuffles; the pairs with the lane to the left arrive the same way.  Lane 0 has no sender, so it is a
//     helper column whose own result is dropped: a tile advances by 31 columns;
//   * pairs with the rows below / above the strip (18): evaluated for the own end only (the other end belongs to
//     another warp, which evaluates them for itself).
// Per two cells: 17 shared + 18 one-sided evaluations instead of 52 one-sided ones.
//
// Per evaluation (lengths in units of h): d = (eta_i - o) - eta_j,  s = |d|^2,  y0 ~ 1/sqrt(s) (MUFU seed),
// t0 = s y0, e = 1 - t0 y0, c = 1 + e/2 + 3e^2/8  (so sqrt(s) = t0 c, 1/sqrt(s) = y0 c to rounding), and with the
// cubic spline (G5)  g^ = 3 - 2.25 q (s < 1),  3/q - 3 + 0.75 q (1 <= s < 4),  0 (s >= 4)  becomes one
// g^ = A c + B,  A = al t0 + be y0,  (al, be, B) = (-2.25, 0, 3) | (0.75, 3, -3) | (0, 0, 0) chosen by integer
// compares of the high word of s.  No division, no IEEE square root, no branch.
#pragma once
#include "cspt_lagrange.cuh"

namespace cspt {

template <class T> struct Acc4 { T x, y, z, e; };
template <class T> struct Particle { T p, u, v, w, ex, ey, ez; };      // phi*, u*, eta* = xi*/h

// g^(sqrt(s)) of the chosen kernel, s = |d|^2 > 0
template <class T, int KERN> struct GHat;
template <int KERN> struct GHat<double, KERN> {
  static __device__ __forceinline__ double eval(double s) {
    if (KERN == 1) {                       // W ~ (1 - q^2/4)^5: g^ = (1 - s/4)^4 on s < 4
      const double t = fma(-0.25, s, 1.0), t2 = t * t;
      return Fast<double>::lt4(s) ? t2 * t2 : 0.0;
    }
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(s));
    const double t0 = s * y0;
    const double e = fma(-t0, y0, 1.0);
    const double c = fma(fma(0.375, e, 0.5), e, 1.0);
    const int hi = __double2hiint(s);
    const bool lt1 = hi < 0x3FF00000, lt4 = hi < 0x40100000;
    // constants whose low words are zero: only the high words are selected (integer pipe)
    const double al = __hiloint2double(lt1 ? (int)0xC0020000 : (lt4 ? 0x3FE80000 : 0), 0);     // -2.25 | 0.75 | 0
    const double be = __hiloint2double(lt1 ? 0 : (lt4 ? 0x40080000 : 0), 0);                   //  0    | 3    | 0
    const double B = __hiloint2double(lt1 ? 0x40080000 : (lt4 ? (int)0xC0080000 : 0), 0);      //  3    | -3   | 0
    return fma(fma(al, t0, be * y0), c, B);
  }
};
template <int KERN> struct GHat<float, KERN> {
  static __device__ __forceinline__ float eval(float s) {
    if (KERN == 1) {
      const float t = fmaf(-0.25f, s, 1.f), t2 = t * t;
      return s < 4.f ? t2 * t2 : 0.f;
    }
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(s));
    const float q = s * y;
    const bool lt1 = s < 1.f, lt4 = s < 4.f;
    const float al = lt1 ? -2.25f : (lt4 ? 0.75f : 0.f);
    const float be = lt1 ? 0.f : (lt4 ? 3.f : 0.f);
    const float B = lt1 ? 3.f : (lt4 ? -3.f : 0.f);
    return fmaf(al, q, be * y) + B;
  }
};

// own end only: particle i <- partner j (d = r_i - r_j in units of h)
template <class T, int KERN>
__device__ __forceinline__ void pair_one(T dx, T dy, T dz, const Particle<T>& j, Acc4<T>& ai) {
  const T s = fma(dz, dz, fma(dy, dy, fma(dx, dx, Fast<T>::tiny())));
  const T w = j.p * GHat<T, KERN>::eval(s);
  ai.x = fma(w, dx, ai.x); ai.y = fma(w, dy, ai.y); ai.z = fma(w, dz, ai.z);
  ai.e = fma(w, fma(j.w, dz, fma(j.v, dy, j.u * dx)), ai.e);
}
// both ends of the pair
template <class T, int KERN>
__device__ __forceinline__ void pair_both(T dx, T dy, T dz, const Particle<T>& i, const Particle<T>& j, Acc4<T>& ai,
                                          Acc4<T>& aj) {
  const T s = fma(dz, dz, fma(dy, dy, fma(dx, dx, Fast<T>::tiny())));
  const T g = GHat<T, KERN>::eval(s);
  const T w = j.p * g, wn = -(i.p * g);
  ai.x = fma(w, dx, ai.x); ai.y = fma(w, dy, ai.y); ai.z = fma(w, dz, ai.z);
  ai.e = fma(w, fma(j.w, dz, fma(j.v, dy, j.u * dx)), ai.e);
  aj.x = fma(wn, dx, aj.x); aj.y = fma(wn, dy, aj.y); aj.z = fma(wn, dz, aj.z);
  aj.e = fma(wn, fma(i.w, dz, fma(i.v, dy, i.u * dx)), aj.e);
}

template <class T> __device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// XS = 1: pairs with the neighbouring lanes are shared through warp shuffles (tiles advance by 31 columns, lane 0 is
// a helper column); XS = 0: they are evaluated for the own end only (tiles advance by 32 columns).
template <class T, int TY, int NST, int XS>
struct PairSmem {
  static constexpr int TXO = XS ? 31 : 32;                       // output columns per tile
  // box columns: lane l holds column c0 + l, its neighbours c0 + l +- 1; fp32 boxes start on an even pair index
  // (16-byte boundary in global memory) and may therefore begin one column further left
  static constexpr int BX = sizeof(T) == 8 ? 34 : 36;
  static constexpr int BY = TY + 2;
  static constexpr int NF = SP_COUNT;
  static constexpr int PLANE = NF * BY * BX * 2;                 // elements per stage
  static constexpr int STAGE = (PLANE * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int OFF_BAR = NST * STAGE;
  static constexpr int BYTES = OFF_BAR + 64 + 128;
  static constexpr int THREADS = 32 * (TY / 2);
  static_assert(TY % 2 == 0, "strips are two rows high");
  static_assert((2 * BX * sizeof(T)) % 16 == 0, "box rows must be multiples of 16 bytes");
};

template <class T, int TY, int NST, int MINB, int KERN, int XP, int XS>
__global__ void __launch_bounds__(32 * (TY / 2), MINB)
k_corrector_pairs(const __grid_constant__ CUtensorMap mapS, Params<T> P, const DevScalars<T>* __restrict__ sc,
                  const T* __restrict__ U, const T* __restrict__ F, T* __restrict__ UT, T* __restrict__ XI, int zchunk) {
  typedef PairSmem<T, TY, NST, XS> S;
  typedef Fast<T> FT;
  typedef typename Pair<T>::type V2;
  typedef Particle<T> Pt;
  typedef Acc4<T> Ac;
  extern __shared__ __align__(128) unsigned char sm[];
  uint64_t* bar = (uint64_t*)(sm + S::OFF_BAR);
  const Layout& L = P.L;
  const int tid = threadIdx.x, lane = tid & 31, strip = tid >> 5;
  // first output column of the tile; lane l holds column c0 + l
  const int i0 = (XP ? 0 : -1) + (int)blockIdx.x * S::TXO;
  const int c0 = XS ? i0 - 1 : i0;
  const int j0 = -1 + (int)blockIdx.y * TY;
  const int z0 = -1 + (int)blockIdx.z * zchunk, z1 = min(L.nz + 1, z0 + zchunk);     // output planes [z0, z1)
  const int i = c0 + lane;
  const int ly0 = strip * 2;
  const long long fs = L.fstride;
  constexpr uint32_t TX_BYTES = (uint32_t)(S::PLANE * sizeof(T));
  // box start: column c0 - 1, moved left to an even pair index in fp32
  const int bxs = c0 - 1 + GX;
  const int bx0 = sizeof(T) == 8 ? bxs : (bxs & ~1);
  const int lxo = bxs - bx0 + 1 + lane;                          // box column of the own cells

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) mbar_init(&bar[s], 1);
    mbar_fence_init();
    prefetch_tmap(&mapS);
  }
  __syncthreads();
  auto slot_of = [&](int q) { return (q - (z0 - 1)) % NST; };
  auto issue = [&](int q) {
    int s = slot_of(q);
    mbar_expect_tx(&bar[s], TX_BYTES);
    tma_load_4d(sm + s * S::STAGE, &mapS, &bar[s], 2 * bx0, j0 + NG - 1, q + NG, 0);
  };
  if (tid == 0) {
    for (int q = z0 - 1; q < z0 - 1 + NST && q <= z1; ++q) issue(q);
  }

  int woff[2];
#pragma unroll
  for (int g = 0; g < 2; ++g) {
    const int xd = g ? L.nx : -1;
    woff[g] = (XP && ((xd % L.nx) + L.nx) % L.nx == i) ? xd - i : 0;
  }
  const T dt = load_dt(sc);
  const T hdt = (T)0.5 * dt, qdt = (T)0.25 * dt;
  const T pnorm = P.wnorm * P.h;                   // 1 / (S0' h): sums are in units of h
  uint32_t phase = 0;
  auto wait_plane = [&](int q) {
    int s = slot_of(q);
    mbar_wait(&bar[s], (phase >> s) & 1u);
    phase ^= 1u << s;
  };
  auto stage = [&](int q) { return (const V2*)(sm + slot_of(q) * S::STAGE); };
  auto load_particle = [&](const V2* sp, int r, int lx, Pt& q) {          // row r of the strip (-1..2), box column lx
    const int o = (ly0 + r + 1) * S::BX + lx;
    const V2 b0 = sp[(SP_PHI_U * S::BY) * S::BX + o], b1 = sp[(SP_V_W * S::BY) * S::BX + o];
    const V2 b2 = sp[(SP_EX_EY * S::BY) * S::BX + o], b3 = sp[(SP_EZ_E * S::BY) * S::BX + o];
    q.p = b0.x; q.u = b0.y; q.v = b1.x; q.w = b1.y; q.ex = b2.x; q.ey = b2.y; q.ez = b3.x;
  };

  const bool col_ok = (!XS || lane >= 1) && i < L.nx + (XP ? 0 : 1) && i < i0 + S::TXO;
  const bool valid[2] = {col_ok && (j0 + ly0) <= L.ny, col_ok && (j0 + ly0 + 1) <= L.ny};
  const bool strip_live = (j0 + ly0) <= L.ny;                    // warp-uniform: any row of the strip in the domain

  Pt cur[2], nxt[2];
  Ac acur[2], anxt[2];
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    acur[c].x = acur[c].y = acur[c].z = acur[c].e = (T)0;
    cur[c].p = cur[c].u = cur[c].v = cur[c].w = cur[c].ex = cur[c].ey = cur[c].ez = (T)0;
  }
  wait_plane(z0 - 1);
  if (strip_live) {
#pragma unroll
    for (int c = 0; c < 2; ++c) load_particle(stage(z0 - 1), c, lxo, cur[c]);
  }

  for (int p = z0 - 1; p < z1; ++p) {
    wait_plane(p + 1);
    const V2* sp0 = stage(p);
    const V2* sp1 = stage(p + 1);
    const bool emit = p >= z0;
    // own-cell operands of Eq. (6) from global memory, requested before the pair loop hides their latency
    T own[2][8];
    if (emit) {
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const long long cc = L.idx(valid[c] ? i : 0, valid[c] ? j0 + ly0 + c : 0, p);
#pragma unroll
        for (int f = 0; f < 5; ++f) own[c][f] = __ldg(U + cc + f * fs);
#pragma unroll
        for (int f = 0; f < 3; ++f) own[c][5 + f] = __ldg(F + cc + f * fs);
      }
    }
#pragma unroll
    for (int c = 0; c < 2; ++c) anxt[c].x = anxt[c].y = anxt[c].z = anxt[c].e = (T)0;
    bool work = false;
    if (strip_live) {
#pragma unroll
      for (int c = 0; c < 2; ++c) load_particle(sp1, c, lxo, nxt[c]);
      // a particle with phi = 0 (vacuum, or p floored to 0) neither exerts nor feels the pressure force: if every
      // own particle of the warp has phi = 0 all four sums of all of them are multiplied by 0 in Eq. (7)
      const bool dead = cur[0].p == (T)0 && cur[1].p == (T)0 && nxt[0].p == (T)0 && nxt[1].p == (T)0;
      work = !__all_sync(0xffffffffu, dead);
    }
    if (work) {
      // eta_z - o_z of the own particles: cur pairs with plane p (o_z = 0) and p+1 (o_z = +1), nxt with plane p (-1)
      const T czm[2] = {cur[0].ez - (T)1, cur[1].ez - (T)1};
      const T nzp[2] = {nxt[0].ez + (T)1, nxt[1].ez + (T)1};

      // ---- own-own pairs (same lane) ---------------------------------------------------------------
      // in plane p: cell 0 and cell 1 (o = (0, +1, 0) seen from cell 0)
      pair_both<T, KERN>(cur[0].ex - cur[1].ex, (cur[0].ey - (T)1) - cur[1].ey, cur[0].ez - cur[1].ez, cur[0], cur[1],
                         acur[0], acur[1]);
      // between the planes: cur c (i) and nxt c' (j), o = (0, c' - c, +1)
#pragma unroll
      for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int cp = 0; cp < 2; ++cp) {
          const T ey = cp == c ? cur[c].ey : (cp > c ? cur[c].ey - (T)1 : cur[c].ey + (T)1);
          pair_both<T, KERN>(cur[c].ex - nxt[cp].ex, ey - nxt[cp].ey, czm[c] - nxt[cp].ez, cur[c], nxt[cp], acur[c],
                             anxt[cp]);
        }

      // ---- the cells of the neighbouring lanes in the strip's rows -------------------------------------
#pragma unroll
      for (int ox = XS ? 1 : -1; ox <= 1; ox += 2) {
#pragma unroll
        for (int r = 0; r < 2; ++r) {
          Pt q;
          // partner in plane p: pairs with cur (in plane) and with nxt (o_z = -1)
          load_particle(sp0, r, lxo + ox, q);
          {
            const T qx = q.ex + (T)ox;
            Ac out; out.x = out.y = out.z = out.e = (T)0;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              const T qy = r == c ? q.ey : (r > c ? q.ey + (T)1 : q.ey - (T)1);       // eta_j + o_y
              if (XS) {
                pair_both<T, KERN>(cur[c].ex - qx, cur[c].ey - qy, cur[c].ez - q.ez, cur[c], q, acur[c], out);
                pair_both<T, KERN>(nxt[c].ex - qx, nxt[c].ey - qy, nzp[c] - q.ez, nxt[c], q, anxt[c], out);
              } else {
                pair_one<T, KERN>(cur[c].ex - qx, cur[c].ey - qy, cur[c].ez - q.ez, q, acur[c]);
                pair_one<T, KERN>(nxt[c].ex - qx, nxt[c].ey - qy, nzp[c] - q.ez, q, anxt[c]);
              }
            }
            if (XS) {                       // the partner is cell (lane + 1, r, p): its part travels one lane up
              const T rx = shfl_up1(out.x), ry = shfl_up1(out.y), rz = shfl_up1(out.z), re = shfl_up1(out.e);
              acur[r].x += rx; acur[r].y += ry; acur[r].z += rz; acur[r].e += re;
            }
          }
          // partner in plane p+1: pairs with cur (o_z = +1)
          load_particle(sp1, r, lxo + ox, q);
          {
            const T qx = q.ex + (T)ox;
            Ac out; out.x = out.y = out.z = out.e = (T)0;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              const T qy = r == c ? q.ey : (r > c ? q.ey + (T)1 : q.ey - (T)1);
              if (XS) pair_both<T, KERN>(cur[c].ex - qx, cur[c].ey - qy, czm[c] - q.ez, cur[c], q, acur[c], out);
              else pair_one<T, KERN>(cur[c].ex - qx, cur[c].ey - qy, czm[c] - q.ez, q, acur[c]);
            }
            if (XS) {
              const T rx = shfl_up1(out.x), ry = shfl_up1(out.y), rz = shfl_up1(out.z), re = shfl_up1(out.e);
              anxt[r].x += rx; anxt[r].y += ry; anxt[r].z += rz; anxt[r].e += re;
            }
          }
        }
      }

      // ---- the rows below and above the strip: own end only ---------------------------------------------
#pragma unroll
      for (int side = 0; side < 2; ++side) {
        const int r = side ? 2 : -1, c = side;                    // row 2 pairs with cell 1, row -1 with cell 0
        const T oy = side ? (T)1 : (T)-1;
#pragma unroll
        for (int ox = -1; ox <= 1; ++ox) {
          Pt q;
          load_particle(sp0, r, lxo + ox, q);
          {
            const T qx = ox == 0 ? q.ex : q.ex + (T)ox, qy = q.ey + oy;
            pair_one<T, KERN>(cur[c].ex - qx, cur[c].ey - qy, cur[c].ez - q.ez, q, acur[c]);
            pair_one<T, KERN>(nxt[c].ex - qx, nxt[c].ey - qy, nzp[c] - q.ez, q, anxt[c]);
          }
          load_particle(sp1, r, lxo + ox, q);
          {
            const T qx = ox == 0 ? q.ex : q.ex + (T)ox, qy = q.ey + oy;
            pair_one<T, KERN>(cur[c].ex - qx, cur[c].ey - qy, czm[c] - q.ez, q, acur[c]);
          }
        }
      }
    }

    // ---- SUL{corrector}, Eq. (6), for the cells of plane p ---------------------------------------------
    if (emit) {
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        if (!valid[c]) continue;
        const int j = j0 + ly0 + c;
        const long long cc = L.idx(i, j, p);
        const T rho = own[c][0], mxn = own[c][1], myn = own[c][2], mzn = own[c][3], En = own[c][4];
        const T fx = own[c][5], fy = own[c][6], fz = own[c][7];
        const T Es = sp0[((SP_EZ_E * S::BY) + (ly0 + c + 1)) * S::BX + lxo].y;
        const bool ok = rho > P.rho_vac;
        const T ir = ok ? FT::rcp(rho) : (T)0;
        const T un = mxn * ir, vn = myn * ir, wn = mzn * ir;
        const T us = cur[c].u, vs = cur[c].v, ws = cur[c].w;
        // U* momentum: rho u* (a vacuum particle has phi = 0, so Q_m = rho f there)
        const T mxs = ok ? rho * us : fma(dt, rho * fx, mxn);
        const T mys = ok ? rho * vs : fma(dt, rho * fy, myn);
        const T mzs = ok ? rho * ws : fma(dt, rho * fz, mzn);
        const T pn = cur[c].p * pnorm;
        const T sx = acur[c].x, sy = acur[c].y, sz = acur[c].z;
        const T set = acur[c].e + (us * sx + vs * sy + ws * sz);
        const T qx = pn * sx + rho * fx;
        const T qy = pn * sy + rho * fy;
        const T qz = pn * sz + rho * fz;
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
    }
#pragma unroll
    for (int c = 0; c < 2; ++c) { cur[c] = nxt[c]; acur[c] = anxt[c]; }

    __syncthreads();                                 // everyone is done with plane p
    if (tid == 0 && p + NST <= z1) issue(p + NST);
  }
}

}  // namespace cspt
