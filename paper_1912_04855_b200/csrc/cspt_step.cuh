// cspt_step.cuh -- helpers shared by the step kernels (Eq. (4)-(8)).
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

}  // namespace cspt
