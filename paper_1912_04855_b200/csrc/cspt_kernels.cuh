// cspt_kernels.cuh -- device code of the CSPH-TVD step (sm_100a).
// Citations are to /root/reference/PAPER.md (section 2.2) and to the readings
// G1..G23 of DESIGN.md section 3.
#pragma once
#include "cspt_common.cuh"

namespace cspt {

template <class T> struct Params {
  Layout L;
  T h, gamma, rho_vac;
  T inv_h;
  T a1, a2, a3;     // lattice weights a(|o|^2) of the undisplaced cubic-spline operator (G5)
  T wnorm;          // 1 / (S0' h^2): kernel weight normalisation (G5)
  int bc[6];
};

// ---- primitives of one cell (G7, G9) ----------------------------
template <class T> struct Prim { T u, v, w, p, phi; bool ok; };

// Exactly rounded version: every operation is a single IEEE rn operation in a fixed
// order, so that the CFL time step and the vacuum mask are bit-exact (G15).
template <class T>
__device__ __forceinline__ Prim<T> prim_exact(T rho, T mx, T my, T mz, T E, T gamma, T rho_vac) {
  typedef Real<T> R;
  Prim<T> q;
  q.ok = rho > rho_vac;
  T ir = q.ok ? R::div((T)1, rho) : (T)0;
  q.u = R::mul(mx, ir); q.v = R::mul(my, ir); q.w = R::mul(mz, ir);
  T ke2 = R::add(R::add(R::mul(mx, q.u), R::mul(my, q.v)), R::mul(mz, q.w));
  T pp = R::mul(R::sub(gamma, (T)1), R::sub(E, R::mul((T)0.5, ke2)));
  q.p = q.ok ? (pp > (T)0 ? pp : (T)0) : (T)0;
  q.phi = R::sqrt(R::mul((T)2, q.p));
  return q;
}

// ---- fast reciprocal / square roots of the step kernels (parity is to 1e-11 / 1e-4, not bit-exact) ----
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
  // 1/x for normal x > 0: MUFU.RCP64H seed + one third-order step, y = y0 (1 + e + e^2), e = 1 - x y0
  static __device__ __forceinline__ double rcp(double x) {
    double y0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    double e = fma(-x, y0, 1.0);
    return fma(y0, fma(e, e, e), y0);
  }
  // sqrt(x) for x >= 0; values below 1e-280 (phi < 1e-140) are flushed to 0
  static __device__ __forceinline__ double sqrt0(double x) {
    double y, t;
    rsqrt_sqrt(x, y, t);
    return x > 1e-280 ? t : 0.0;
  }
  // comparisons of a positive double with 1 and 4 on the high word (integer pipe)
  static __device__ __forceinline__ bool lt1(double s) { return __double2hiint(s) < 0x3FF00000; }
  static __device__ __forceinline__ bool lt4(double s) { return __double2hiint(s) < 0x40100000; }
  static __device__ __forceinline__ double tiny() { return 1e-300; }
  static __device__ __forceinline__ double cancel_eps() { return 1.8e-15; }     // 16 ulp: see cell_speed_upper
};
template <> struct Fast<float> {
  static __device__ __forceinline__ void rsqrt_sqrt(float s, float& y, float& t) {
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(s));
    t = s * y;
  }
  static __device__ __forceinline__ float rcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
  }
  static __device__ __forceinline__ float sqrt0(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
  }
  static __device__ __forceinline__ bool lt1(float s) { return s < 1.0f; }
  static __device__ __forceinline__ bool lt4(float s) { return s < 4.0f; }
  static __device__ __forceinline__ float tiny() { return 1e-30f; }
  static __device__ __forceinline__ float cancel_eps() { return 9.6e-7f; }
};

// ---- brick map (cspt_common.cuh, BrickMap) ------------------------------------------------------------------------
// (px, py, pz): padded coordinates of a cell
__device__ __forceinline__ void brick_flag(const BrickMap& M, int px, int py, int pz) {
  M.raw[((size_t)(pz / BRZ) * M.nby + (py / BRY)) * M.nbx + (px / BRX)] = 1;
}
// Called by EVERY thread of a 1-D CTA: true if no brick that overlaps the box [x0,x1) x [y0,y1) x [z0,z1) of padded
// coordinates (clamped to the array) is live.  Flags are only ever added, also while a kernel runs (the Euler stage
// flags U^{n+1}): a CTA that sees such a flag early merely evaluates zeros in full.
__device__ __forceinline__ bool cta_region_dead(const BrickMap& M, const Layout& L, int x0, int x1, int y0, int y1, int z0, int z1) {
  x0 = max(x0, 0); y0 = max(y0, 0); z0 = max(z0, 0);
  x1 = min(x1, L.px); y1 = min(y1, L.py); z1 = min(z1, L.pz);
  const int bx0 = x0 / BRX, by0 = y0 / BRY, bz0 = z0 / BRZ;
  const int ex = (x1 - 1) / BRX - bx0 + 1, ey = (y1 - 1) / BRY - by0 + 1, ez = (z1 - 1) / BRZ - bz0 + 1;
  int any = 0;
  if (ex > 0 && ey > 0 && ez > 0) {
    const int n = ex * ey * ez;
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
      const int bx = bx0 + t % ex, r = t / ex, by = by0 + r % ey, bz = bz0 + r / ey;
      any |= __ldg(M.raw + ((size_t)bz * M.nby + by) * M.nbx + bx);
    }
  }
  const bool dead = !__syncthreads_or(any);
  if (dead && threadIdx.x == 0) atomicAdd(M.dead, 1ULL);
  return dead;
}

// rebuilds the map from the current U over the cells a step can read: interior and the 3 ghost layers
template <class T>
__global__ void k_brick_scan(Layout L, const T* __restrict__ U, BrickMap M) {
  const int ex = L.nx + 2 * NG, ey = L.ny + 2 * NG, ez = L.nz + 2 * NG;
  const long long n = (long long)ex * ey * ez;
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(m % ex) - NG;
    const long long r = m / ex;
    const int j = (int)(r % ey) - NG, k = (int)(r / ey) - NG;
    const long long c = L.idx(i, j, k);
    bool nz = false;
#pragma unroll
    for (int f = 0; f < 5; ++f) nz = nz || (U[c + f * L.fstride] != (T)0);
    if (nz) brick_flag(M, i + GX, j + NG, k + NG);
  }
}

// ---- set_state: primitives -> conserved, psi into a scratch field ----
template <class T>
__global__ void k_set_state(Params<T> P, const T* __restrict__ rho, const T* __restrict__ u,
                            const T* __restrict__ v, const T* __restrict__ w, const T* __restrict__ p,
                            const T* __restrict__ psi, T* __restrict__ U, T* __restrict__ psi_pad, int* __restrict__ has_vac) {
  typedef Real<T> R;
  const Layout& L = P.L;
  long long n = (long long)L.nx * L.ny * L.nz;
  int vac = 0;
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
    int i = (int)(m % L.nx);
    long long r = m / L.nx;
    int j = (int)(r % L.ny), k = (int)(r / L.ny);
    long long c = L.idx(i, j, k);
    T ro = rho[m], uu = u[m], vv = v[m], ww = w[m];
    vac |= !(ro > P.rho_vac);
    U[c] = ro;
    U[c + L.fstride] = R::mul(ro, uu);
    U[c + 2 * L.fstride] = R::mul(ro, vv);
    U[c + 3 * L.fstride] = R::mul(ro, ww);
    T ke = R::add(R::add(R::mul(uu, uu), R::mul(vv, vv)), R::mul(ww, ww));
    U[c + 4 * L.fstride] = R::add(R::div(p[m], R::sub(P.gamma, (T)1)), R::mul(R::mul((T)0.5, ro), ke));
    if (psi_pad) psi_pad[c] = psi[m];
  }
  if (__syncthreads_or(vac) && threadIdx.x == 0) atomicOr(has_vac, 1);     // hint for the host: vacuum shortcuts pay
}

template <class T>
__global__ void k_put_field(Layout L, const T* __restrict__ src, T* __restrict__ dst) {
  long long n = (long long)L.nx * L.ny * L.nz;
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
    int i = (int)(m % L.nx);
    long long r = m / L.nx;
    dst[L.idx(i, (int)(r % L.ny), (int)(r / L.ny))] = src[m];
  }
}

template <class T>
__global__ void k_get_field(Layout L, const T* __restrict__ src, T* __restrict__ dst) {
  long long n = (long long)L.nx * L.ny * L.nz;
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
    int i = (int)(m % L.nx);
    long long r = m / L.nx;
    dst[m] = src[L.idx(i, (int)(r % L.ny), (int)(r / L.ny))];
  }
}

template <class T>
__global__ void k_get_state(Params<T> P, const T* __restrict__ U, T* __restrict__ rho, T* __restrict__ u,
                            T* __restrict__ v, T* __restrict__ w, T* __restrict__ p, unsigned char* __restrict__ mask) {
  const Layout& L = P.L;
  long long n = (long long)L.nx * L.ny * L.nz;
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
    int i = (int)(m % L.nx);
    long long r = m / L.nx;
    long long c = L.idx(i, (int)(r % L.ny), (int)(r / L.ny));
    T ro = U[c];
    if (mask) { mask[m] = ro > P.rho_vac ? 0 : 1; continue; }
    Prim<T> q = prim_exact<T>(ro, U[c + L.fstride], U[c + 2 * L.fstride], U[c + 3 * L.fstride], U[c + 4 * L.fstride], P.gamma, P.rho_vac);
    rho[m] = ro; u[m] = q.u; v[m] = q.v; w[m] = q.w; p[m] = q.p;
  }
}

// ---- O0: ghost layers along one axis (G16) ----------------------------------------
// mode 0: state fields (wrap / copy boundary cell / frozen inflow layer)
// mode 1: like 0 but INFLOW faces are filled like OUTFLOW and their layer is captured
// mode 2: potential (wrap / odd reflection about the boundary cell)
// Axes before `d` are traversed over their padded range, axes after it over the interior,
// so that x, y, z launches in this order fill edges and corners.
template <class T>
__global__ void k_ghost_axis(Layout L, int d, int mode, int bc_lo, int bc_hi, int nfields,
                             T* __restrict__ F, T* __restrict__ inflow_lo, T* __restrict__ inflow_hi,
                             long long inflow_plane, BrickMap M) {
  int n[3] = {L.nx, L.ny, L.nz};
  int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
  int lo1 = d1 < d ? -NG : 0, hi1 = d1 < d ? n[d1] + NG : n[d1];
  int lo2 = d2 < d ? -NG : 0, hi2 = d2 < d ? n[d2] + NG : n[d2];
  long long e1 = hi1 - lo1, e2 = hi2 - lo2;
  long long total = e1 * e2 * NG * 2;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
    // fastest index: along the axis that is contiguous in memory when possible
    long long r = t;
    int b, a, g, side;
    if (d == 0) { g = (int)(r % NG) + 1; r /= NG; side = (int)(r % 2); r /= 2; b = (int)(r % e1) + lo1; a = (int)(r / e1) + lo2; }
    else if (d == 1) { a = (int)(r % e2) + lo2; r /= e2; g = (int)(r % NG) + 1; r /= NG; side = (int)(r % 2); r /= 2; b = (int)r + lo1; }
    else { b = (int)(r % e1) + lo1; r /= e1; a = (int)(r % e2) + lo2; r /= e2; g = (int)(r % NG) + 1; side = (int)(r / NG); }
    int kind = side ? bc_hi : bc_lo;
    if (kind == CSPT_BC_EXTERNAL) continue;            // ghost planes of a slab face: written by cspt_halo_put
    int q[3], s[3], e0[3];
    q[d1] = b; q[d2] = a; s[d1] = b; s[d2] = a; e0[d1] = b; e0[d2] = a;
    q[d] = side ? n[d] - 1 + g : -g;
    e0[d] = side ? n[d] - 1 : 0;
    long long cq = L.idx(q[0], q[1], q[2]);
    if (kind == CSPT_BC_PERIODIC) {
      s[d] = side ? ((g - 1) % n[d]) : (n[d] - 1 - ((g - 1) % n[d]));
      long long cs = L.idx(s[0], s[1], s[2]);
      bool nz = false;
      for (int f = 0; f < nfields; ++f) { T val = F[cs + f * L.fstride]; F[cq + f * L.fstride] = val; nz = nz || (val != (T)0); }
      if (M.raw && nz) brick_flag(M, q[0] + GX, q[1] + NG, q[2] + NG);
    } else if (mode == 2) {
      s[d] = side ? n[d] - 1 - g : g;
      s[d] = max(0, min(n[d] - 1, s[d]));
      long long cs = L.idx(s[0], s[1], s[2]), ce = L.idx(e0[0], e0[1], e0[2]);
      F[cq] = (T)2 * F[ce] - F[cs];
    } else {
      long long ce = L.idx(e0[0], e0[1], e0[2]);
      // captured planes are indexed by the padded coordinates of the two other axes
      int pd1 = d1 == 0 ? L.px : (d1 == 1 ? L.py : L.pz);
      int off1 = d1 == 0 ? GX : NG, off2 = d2 == 0 ? GX : NG;
      long long pi = (long long)(a + off2) * pd1 + (b + off1);
      T* inf = side ? inflow_hi : inflow_lo;
      for (int f = 0; f < nfields; ++f) {
        T val;
        if (kind == CSPT_BC_INFLOW && mode == 0) val = inf[f * inflow_plane + pi];
        else val = F[ce + f * L.fstride];
        F[cq + f * L.fstride] = val;
        if (kind == CSPT_BC_INFLOW && mode == 1 && g == 1) inf[f * inflow_plane + pi] = val;
        if (M.raw && val != (T)0) brick_flag(M, q[0] + GX, q[1] + NG, q[2] + NG);
      }
    }
  }
}

// ---- O2: external force f = -D[psi] on interior(+)2 (G5, G6) -----
template <class T>
__global__ void k_force(Params<T> P, const T* __restrict__ psi, T* __restrict__ F) {
  const Layout& L = P.L;
  int ex = L.nx + 4, ey = L.ny + 4, ez = L.nz + 4;
  long long n = (long long)ex * ey * ez;
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
    int i = (int)(m % ex) - 2;
    long long r = m / ex;
    int j = (int)(r % ey) - 2, k = (int)(r / ey) - 2;
    long long c = L.idx(i, j, k);
    T s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
    for (int oz = -1; oz <= 1; ++oz)
#pragma unroll
      for (int oy = -1; oy <= 1; ++oy)
#pragma unroll
        for (int ox = -1; ox <= 1; ++ox) {
          int o2 = ox * ox + oy * oy + oz * oz;
          if (o2 == 0) continue;
          T a = o2 == 1 ? P.a1 : (o2 == 2 ? P.a2 : P.a3);
          T q = a * psi[c + oz * L.sz() + oy * L.sy() + ox];
          s0 += (T)ox * q; s1 += (T)oy * q; s2 += (T)oz * q;
        }
    F[c] = -(s0 / P.h);
    F[c + L.fstride] = -(s1 / P.h);
    F[c + 2 * L.fstride] = -(s2 / P.h);
  }
}

// ---- O9: CFL signal speed maximum (paper silent; G15) -----------------------------
// Per-thread max -> warp shuffle max -> block max -> integer atomicMax on the IEEE bit
// pattern (non-negative floats order like unsigned integers): bit-exact, order independent.
template <class T>
__device__ __forceinline__ T cell_speed_exact(T rho, T mx, T my, T mz, T E, T gamma, T rho_vac) {
  typedef Real<T> R;
  Prim<T> q = prim_exact<T>(rho, mx, my, mz, E, gamma, rho_vac);
  if (!q.ok) return (T)0;
  T cs = R::sqrt(R::div(R::mul(gamma, q.p), rho));
  T a = fabs(q.u), b = fabs(q.v), c = fabs(q.w);
  T m = a > b ? a : b;
  m = m > c ? m : c;
  return R::add(cs, m);
}

// Cheap UPPER BOUND of the same signal speed (fast reciprocal / square root).  Used only as a FILTER: a cell whose
// bound lies below a speed that is already known exactly cannot be the maximum, so the exactly rounded evaluation
// is skipped for it.  E - rho|u|^2/2 cancels in cold supersonic cells: the contracted (FMA) evaluation here and
// the separately rounded one of cell_speed_exact then differ by a few ulp of the OPERANDS (relative eps Mach^2 / 2
// of the result), so the internal energy is raised by 16 ulp of |E| + rho|u|^2 before the square root; the
// remaining relative errors (reciprocal and square-root seeds, a few ulp) are covered by the caller's margin.
template <class T>
__device__ __forceinline__ T cell_speed_upper(T rho, T mx, T my, T mz, T E, T gamma, T rho_vac) {
  typedef Fast<T> FT;
  if (!(rho > rho_vac)) return (T)0;
  T ir = FT::rcp(rho);
  T u = mx * ir, v = my * ir, w = mz * ir;
  T ke2 = (mx * u + my * v) + mz * w;
  T pp = (gamma - (T)1) * ((E - (T)0.5 * ke2) + FT::cancel_eps() * (fabs(E) + ke2));
  pp = pp > (T)0 ? pp : (T)0;
  T a = fabs(u), b = fabs(v), c = fabs(w);
  T m = a > b ? a : b;
  m = m > c ? m : c;
  return FT::sqrt0(gamma * pp * ir) + m;
}

template <class T>
__device__ __forceinline__ void block_max_to_global(T s, typename Real<T>::bits_t* out) {
  typedef typename Real<T>::bits_t bits_t;
  __shared__ bits_t sm[32];
  bits_t b = s > (T)0 ? Real<T>::bits(s) : (bits_t)0;      // NaN and 0 contribute nothing
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bits_t other = __shfl_xor_sync(0xffffffffu, b, o);
    b = other > b ? other : b;
  }
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) sm[wid] = b;
  __syncthreads();
  if (wid == 0) {
    int nw = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
    b = lane < nw ? sm[lane] : (bits_t)0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      bits_t other = __shfl_xor_sync(0xffffffffu, b, o);
      b = other > b ? other : b;
    }
    if (lane == 0 && b != 0) atomicMax(out, b);
  }
}

template <class T>
__global__ void k_speed_max(Params<T> P, const T* __restrict__ U, typename Real<T>::bits_t* out) {
  const Layout& L = P.L;
  long long n = (long long)L.nx * L.ny * L.nz;
  T smax = 0;
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
    int i = (int)(m % L.nx);
    long long r = m / L.nx;
    long long c = L.idx(i, (int)(r % L.ny), (int)(r / L.ny));
    T s = cell_speed_exact<T>(U[c], U[c + L.fstride], U[c + 2 * L.fstride], U[c + 3 * L.fstride], U[c + 4 * L.fstride], P.gamma, P.rho_vac);
    if (s > smax) smax = s;
  }
  block_max_to_global<T>(smax, out);
}

// dt = (cfl*h)/smax in T, one rn operation each: identical to the host formula.  The maximum is consumed here: it is
// reset for the Euler stage of this step, which leaves the maximum of U^{n+1} behind.
template <class T>
__global__ void k_dt_finalize(DevScalars<T>* sc, T cfl, T h) {
  typedef Real<T> R;
  T smax = R::from_bits(sc->smax_bits);
  T dt = smax > (T)0 ? R::div(R::mul(cfl, h), smax) : R::inf();
  sc->dt = dt;
  sc->smax_bits = 0;
  if (dt < R::inf()) sc->time += (double)dt;
}

template <class T>
__global__ void k_set_dt(DevScalars<T>* sc, T dt) {
  sc->dt = dt;
  sc->smax_bits = 0;
  sc->time += (double)dt;
}

template <class T>
__global__ void k_reset_smax(DevScalars<T>* sc, int reset_time) {
  sc->smax_bits = 0;
  if (reset_time) sc->time = 0.0;
}

// ---- roofline probe: the FMA rate of the plain FP64 / FP32 pipe, measured on the box the bench runs on ----------
// Eight independent FMA chains per thread; NI > 0 puts NI independent integer instructions (add / xor on eight
// chains of their own) behind every FMA, to show how other instructions share the issue port with the FMAs
// (profiles/r2_issue_model.md: an FP64 FMA holds its pipe for two cycles but ONE other instruction issues in its
// shadow; beyond that every instruction costs about 1.1 issue cycles).
// NI = -1: FMAs with THREE distinct register operands, x = y * z + x: in fp64 each operand is a register pair and the
// register file delivers two pairs per cycle and sub-partition, so such a DFMA issues every 3 cycles, not 2.
template <class T, int NI>
__global__ void k_probe_fma(T* out, unsigned cap, int iters, T a, T b, int m) {
  T x[8], y[8], z[8];
  int i[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    x[c] = (T)(threadIdx.x + c); i[c] = (int)threadIdx.x * (2 * c + 3);
    y[c] = a + (T)1e-9 * (T)(threadIdx.x + c); z[c] = b * (T)(threadIdx.x * 3 + c + 1);
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        x[c] = NI < 0 ? fma(y[c], z[c], x[c]) : fma(x[c], a, b);
#pragma unroll
        for (int q = 0; q < NI; ++q) i[c] = (q & 1) ? (i[c] ^ m) : (i[c] + m);
      }
    }
  }
  int isum = 0;
  T xsum = 0;
#pragma unroll
  for (int c = 0; c < 8; ++c) { isum += i[c]; xsum += x[c] + (NI < 0 ? y[c] + z[c] : (T)0); }
  out[(blockIdx.x * blockDim.x + threadIdx.x) % cap] = xsum + (T)isum;      // a sink only: small grids wrap around
}

template <class T>
__device__ __forceinline__ T load_dt(const DevScalars<T>* sc) {
  T dt = sc->dt;
  return dt < Real<T>::inf() ? dt : (T)0;       // all-vacuum grid: dt = +inf -> identity step
}

}  // namespace cspt
