// cspt_noalloc.cu -- cspt_cfl_dt_noalloc: the CFL time step (reading G15; the paper is
// silent on it) of five dense conserved arrays the caller already holds, for callers that cannot allocate.
//
// Who this is for.  cspt_compute_dt works on a ctx, and a ctx borrows a workspace of 28 padded fields that somebody
// has to allocate first.  Some users of this library cannot do that, and cannot call cudaMalloc for anything else
// either: a host code that handed the whole of HBM to its own arena at start-up (a 1024^3 run leaves little of the
// 180 GB over); a time loop in which cudaMalloc / cudaFree would stall every stream of the device; an in-situ monitor
// or a coupled solver that is handed device pointers to (rho, rho u, rho v, rho w, E) and must return a common time
// step without owning any memory.  For them this file carries its own scratch: the per-CTA maxima of the signal speed
// live in the file-scope __device__ array g_partials below, which the driver places once per GPU when the library's
// device code is loaded and keeps until the process ends.  The entry point calls no cudaMalloc, cudaFree, cudaMallocHost or any
// library routine that allocates; it launches two kernels on the caller's stream and returns.
//
// Arithmetic: the same as the ctx path (k_speed_max + k_dt_finalize in cspt_kernels.cuh): cell_speed_exact per cell in
// single IEEE rn operations, maximum over the IEEE bit patterns, dt = (cfl*h)/smax as one rn multiply and one rn divide
// in T; the result is therefore bit-identical to cspt_compute_dt on the same state (tests/test_zz_no_alloc.py).
// Only the path of the maximum differs: that kernel folds the CTA maxima into one workspace word with atomicMax
// (which has to be cleared first); here every CTA stores its maximum into its own slot of g_partials and a second
// one-CTA kernel reduces exactly the slots this call wrote, so nothing has to start at zero.
#include <mutex>

#include "cspt_kernels.cuh"

namespace cspt {
namespace {

constexpr int NA_THREADS = 256;                 // threads per CTA of the speed kernel
constexpr int NA_CELLS_PER_THREAD = 16;
constexpr long long NA_CELLS_PER_CTA = (long long)NA_THREADS * NA_CELLS_PER_THREAD;      // 4096
constexpr int NA_MAX_CTAS = 65536;              // slots of the scratch array
constexpr long long NA_MAX_CELLS = NA_CELLS_PER_CTA * NA_MAX_CTAS;                        // 2^28 = 268 435 456
constexpr int NA_MAX_DEVICES = 64;

// The scratch: one 8-byte slot per CTA (fp32 uses the low half of the slots as 4-byte words).  512 KiB of every GPU
// that loads libcspt.so, held until the process exits.  Every call on a device shares it and finds the previous
// call's contents in it.
// In HOST code the name g_partials is a host-side stand-in of the symbol, NOT a device address: a kernel handed
// `g_partials` from the host would fault (or scribble on host memory where the GPU can reach it).  The device
// address comes from cudaGetSymbolAddress, once per device, below.
static __device__ __align__(256) unsigned long long g_partials[NA_MAX_CTAS];

// CTA b takes cells [b*4096, (b+1)*4096) of the dense arrays, coalesced (consecutive threads, consecutive cells),
// and stores the maximum signal speed of its cells, as IEEE bits, into partials[b] -- always, also when it is 0.
template <class T>
__global__ void __launch_bounds__(NA_THREADS)
k_speed_partials(const T* __restrict__ rho, const T* __restrict__ mx, const T* __restrict__ my,
                 const T* __restrict__ mz, const T* __restrict__ E, long long n, T gamma, T rho_vac,
                 typename Real<T>::bits_t* __restrict__ partials) {
  typedef typename Real<T>::bits_t bits_t;
  __shared__ bits_t sm[NA_THREADS / 32];
  long long base = (long long)blockIdx.x * NA_CELLS_PER_CTA + threadIdx.x;
  T smax = 0;
#pragma unroll 4
  for (int q = 0; q < NA_CELLS_PER_THREAD; ++q) {
    long long m = base + (long long)q * NA_THREADS;
    if (m < n) {
      T s = cell_speed_exact<T>(rho[m], mx[m], my[m], mz[m], E[m], gamma, rho_vac);
      if (s > smax) smax = s;
    }
  }
  bits_t b = smax > (T)0 ? Real<T>::bits(smax) : (bits_t)0;      // non-negative floats order like unsigned integers
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bits_t other = __shfl_xor_sync(0xffffffffu, b, o);
    b = other > b ? other : b;
  }
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = b;
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int w = 1; w < NA_THREADS / 32; ++w) b = sm[w] > b ? sm[w] : b;
    partials[blockIdx.x] = b;
  }
}

// One CTA: maximum of the first `count` slots (the ones this call wrote, never more), then the two rn operations of
// k_dt_finalize.  count = 0 (no cells) and an all-vacuum grid give +inf, as cspt_compute_dt does.
template <class T>
__global__ void __launch_bounds__(1024)
k_dt_from_partials(const typename Real<T>::bits_t* __restrict__ partials, int count, T cfl, T h, T* __restrict__ dt_out) {
  typedef typename Real<T>::bits_t bits_t;
  typedef Real<T> R;
  __shared__ bits_t sm[32];
  bits_t b = 0;
  for (int i = threadIdx.x; i < count; i += blockDim.x) {
    bits_t v = partials[i];
    b = v > b ? v : b;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bits_t other = __shfl_xor_sync(0xffffffffu, b, o);
    b = other > b ? other : b;
  }
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = b;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) b = sm[w] > b ? sm[w] : b;
    T smax = R::from_bits(b);
    *dt_out = smax > (T)0 ? R::div(R::mul(cfl, h), smax) : R::inf();
  }
}

// Device address of g_partials on the current device, looked up on the first call there and remembered.
std::mutex g_mu;
void* g_addr[NA_MAX_DEVICES] = {};

int scratch_of_current_device(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return CSPT_ECUDA;
  if (dev < 0 || dev >= NA_MAX_DEVICES) return CSPT_ELIMIT;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_addr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_partials) != cudaSuccess || !p) return CSPT_ECUDA;
    g_addr[dev] = p;
  }
  *out = g_addr[dev];
  return CSPT_OK;
}

template <class T>
int cfl_dt_noalloc_t(long long n, const void* rho, const void* mx, const void* my, const void* mz, const void* E,
                     double gamma, double h, double cfl, void* dt_out, cudaStream_t st, void* scratch) {
  typedef typename Real<T>::bits_t bits_t;
  int ctas = (int)((n + NA_CELLS_PER_CTA - 1) / NA_CELLS_PER_CTA);
  if (ctas > 0)
    k_speed_partials<T><<<ctas, NA_THREADS, 0, st>>>((const T*)rho, (const T*)mx, (const T*)my, (const T*)mz,
                                                     (const T*)E, n, (T)gamma, (T)1e-12, (bits_t*)scratch);
  k_dt_from_partials<T><<<1, 1024, 0, st>>>((const bits_t*)scratch, ctas, (T)cfl, (T)h, (T*)dt_out);
  return cudaPeekAtLastError() == cudaSuccess ? CSPT_OK : CSPT_ECUDA;
}

}  // namespace
}  // namespace cspt

extern "C" {

long long cspt_noalloc_max_cells(void) { return cspt::NA_MAX_CELLS; }

int cspt_cfl_dt_noalloc(int dtype, long long ncells, const void* rho, const void* mx, const void* my, const void* mz,
                        const void* E, double gamma, double h, double cfl, void* dt_device_out, void* cuda_stream) {
  if (dtype != CSPT_F64 && dtype != CSPT_F32) return CSPT_EINVAL;
  if (ncells < 0 || !dt_device_out) return CSPT_EINVAL;
  if (ncells > 0 && (!rho || !mx || !my || !mz || !E)) return CSPT_EINVAL;
  if (!(h > 0) || !isfinite(h) || !(gamma > 1) || !isfinite(gamma) || !(cfl > 0) || !isfinite(cfl)) return CSPT_EINVAL;
  if (ncells > cspt::NA_MAX_CELLS) return CSPT_ELIMIT;      // the scratch has one slot per 4096 cells and 65536 slots
  void* scratch = nullptr;
  int rc = cspt::scratch_of_current_device(&scratch);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  return dtype == CSPT_F64
             ? cspt::cfl_dt_noalloc_t<double>(ncells, rho, mx, my, mz, E, gamma, h, cfl, dt_device_out, st, scratch)
             : cspt::cfl_dt_noalloc_t<float>(ncells, rho, mx, my, mz, E, gamma, h, cfl, dt_device_out, st, scratch);
}

}  // extern "C"
