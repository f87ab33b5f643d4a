// cspt_step.cuh -- helpers shared by the step kernels, and the straightforward (one thread per
// cell, operands through L1/L2) FGC+SUE kernel kept as a debugging cross-check (env CSPT_LEGACY_EULER).
// (Eq. (4)-(8)).
#pragma once
#include "cspt_kernels.cuh"

namespace cspt {

// decode a linear index over the box [-ext, n+ext)^3
__device__ __forceinline__ bool decode_ext(const Layout& L, int ext, long long m, int& i, int& j, int& k) {
  int ex = L.nx + 2 * ext, ey = L.ny + 2 * ext, ez = L.nz + 2 * ext;
  if (m >= (long long)ex * ey * ez) return false;
  i = (int)(m % ex) - ext;
  long long r = m / ex;
  j = (int)(r % ey) - ext;
  k = (int)(r / ey) - ext;
  return true;
}

template <class T>
__device__ __forceinline__ T load_dt(const DevScalars<T>* sc) {
  T dt = sc->dt;
  return dt < Real<T>::inf() ? dt : (T)0;       // all-vacuum grid: dt = +inf -> identity step
}

template <class T>
__device__ __forceinline__ T minmod(T a, T b) {
  if (a > (T)0 && b > (T)0) return a < b ? a : b;
  if (a < (T)0 && b < (T)0) return a > b ? a : b;
  return (T)0;
}

// O7: one face flux, Eq. (8) + pressureless HLL (G10-G13).  cL/cR: cells left/right of the
// face along axis d (stride sd); returns F[5].
template <class T>
__device__ __forceinline__ void face_flux(const Params<T>& P, const T* __restrict__ U, const T* __restrict__ UT,
                                          const T* __restrict__ XI, long long cL, long long sd, int d, T* Fl) {
  const long long fs = P.L.fstride;
  long long cR = cL + sd;
  T UL[5], UR[5];
  T xL = XI[cL + d * fs], xR = XI[cR + d * fs];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const T* Uq = U + q * fs;
    T a = Uq[cL - sd], b = Uq[cL], c = Uq[cR], e = Uq[cR + sd];
    T thL = minmod<T>((b - a) * P.inv_h, (c - b) * P.inv_h);
    T thR = minmod<T>((c - b) * P.inv_h, (e - c) * P.inv_h);
    T tL = q == 0 ? b : UT[cL + (q - 1) * fs];       // rho~ = rho^n (G2)
    T tR = q == 0 ? c : UT[cR + (q - 1) * fs];
    T hL = (T)0.5 * (b + tL), hR = (T)0.5 * (c + tR);  // U^{n+1/2} (G10)
    UL[q] = hL + (T)0.5 * (P.h - xL) * thL;
    UR[q] = hR - (T)0.5 * (P.h + xR) * thR;
  }
  T uL = UL[0] > P.rho_vac ? UL[1 + d] / UL[0] : (T)0;
  T uR = UR[0] > P.rho_vac ? UR[1 + d] / UR[0] : (T)0;
  T up = uL > (T)0 ? uL : (T)0, um = uR < (T)0 ? uR : (T)0;
#pragma unroll
  for (int q = 0; q < 5; ++q) Fl[q] = up * UL[q] + um * UR[q];
}

// O7+O8: FGC + SUE, Eq. (4) unsplit (G14), interior cells; epilogue: CFL speed of U^{n+1}.
template <class T>
__global__ void k_euler(Params<T> P, const DevScalars<T>* sc, const T* __restrict__ U, const T* __restrict__ UT,
                        const T* __restrict__ XI, T* __restrict__ UN, typename Real<T>::bits_t* smax_out) {
  const Layout& L = P.L;
  long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  int i, j, k;
  T s = 0;
  if (decode_ext(L, 0, m, i, j, k)) {
    T dt = load_dt(sc);
    long long c = L.idx(i, j, k), fs = L.fstride;
    T acc[5] = {0, 0, 0, 0, 0};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      long long sd = d == 0 ? 1 : (d == 1 ? L.sy() : L.sz());
      T Fp[5], Fm[5];
      face_flux<T>(P, U, UT, XI, c, sd, d, Fp);
      face_flux<T>(P, U, UT, XI, c - sd, sd, d, Fm);
#pragma unroll
      for (int q = 0; q < 5; ++q) acc[q] += Fp[q] - Fm[q];
    }
    T lam = dt * P.inv_h;
    T un[5];
    un[0] = U[c] - lam * acc[0];
#pragma unroll
    for (int q = 1; q < 5; ++q) un[q] = UT[c + (q - 1) * fs] - lam * acc[q];
#pragma unroll
    for (int q = 0; q < 5; ++q) UN[c + q * fs] = un[q];
    s = cell_speed_exact<T>(un[0], un[1], un[2], un[3], un[4], P.gamma, P.rho_vac);
  }
  block_max_to_global<T>(s, smax_out);
}

}  // namespace cspt
