// cspt_common.cuh -- grid layout, context and small device helpers of the
// CUDA CSPH-TVD path (sm_100a).  No code is shared with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <math.h>

#include "cspt.h"

namespace cspt {

// Ghost layers per face: one full step reaches +-3 cells (predictor radius 1 ->
// corrector radius 1 -> TVD stage needs U~ at +-1 and U^n at +-2).
constexpr int NG = 3;
// Left pad along x is 4 elements so that interior cell i = 0 sits on a 16-byte
// (fp32) / 32-byte (fp64) boundary; the x pitch is a multiple of 16 elements.
constexpr int GX = 4;

struct Layout {
  int nx, ny, nz;      // interior
  int px, py, pz;      // padded (allocated) extents
  long long fstride;   // elements per padded field
  __host__ __device__ long long idx(int i, int j, int k) const {
    return ((long long)(k + NG) * py + (j + NG)) * px + (i + GX);
  }
  __host__ __device__ long long sy() const { return px; }
  __host__ __device__ long long sz() const { return (long long)px * py; }
};

inline Layout make_layout(int nx, int ny, int nz) {
  Layout L;
  L.nx = nx; L.ny = ny; L.nz = nz;
  // minimum extents so that every TMA box of the streaming kernels fits inside the tensor
  L.px = ((nx + GX + NG + 15) / 16) * 16;
  if (L.px < 64) L.px = 64;
  L.py = ny + 2 * NG;
  if (L.py < 32) L.py = 32;
  L.pz = nz + 2 * NG;
  long long n = (long long)L.px * L.py * L.pz;
  L.fstride = ((n + 63) / 64) * 64;
  return L;
}

// Gas-vacuum handling at CTA level (fp32 streaming kernels): a byte per BRX x BRY x BRZ brick of the PADDED array,
// non-zero once any of rho, m, E was non-zero in a cell of the brick since the map was last rebuilt (flags are only
// ever added: a brick that held gas stays "live").  One full step reaches 3 cells, so a CTA whose output footprint,
// widened by 3 cells, touches no live brick has inputs that are exactly 0 and outputs that are exactly 0: it writes
// those zeros and returns before its first load.  raw == nullptr: off.
constexpr int BRX = 32, BRY = 8, BRZ = 8;
struct BrickMap {
  unsigned char* raw;
  int nbx, nby, nbz;
  unsigned long long* dead;      // diagnostics: CTAs that returned early since the map was last rebuilt
  int zero_fill;                 // 1: a dead CTA writes its zeros; 0: they are known to be in place already (it was
                                 // dead in the last two steps too and nothing else has touched the buffers since)
};

// Field slots inside the workspace (each fstride elements of T).
enum Slot {
  S_U0 = 0,        // U buffer A: rho, mx, my, mz, E          (5)
  S_U1 = 5,        // U buffer B                                 (5)
  S_F = 10,        // f = -D[psi]                                (3)
  S_UT = 13,       // U~: mx, my, mz, E  (rho~ = rho^n, G2)      (4)
  S_XI = 17,       // xi^{n+1}                                   (3)
  S_ST = 20,       // star group: phi*, u*, v*, w*, eta* (3), E* (8); between steps: dense staging
                   // arrays of the *_host entry points
  S_COUNT = 28
};

template <class T> struct Real;
template <> struct Real<double> {
  typedef unsigned long long bits_t;
  static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
  static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
  static __device__ __forceinline__ double sub(double a, double b) { return __dadd_rn(a, -b); }
  static __device__ __forceinline__ double div(double a, double b) { return __ddiv_rn(a, b); }
  static __device__ __forceinline__ double sqrt(double a) { return __dsqrt_rn(a); }
  static __device__ __forceinline__ bits_t bits(double a) { return (bits_t)__double_as_longlong(a); }
  static __device__ __forceinline__ double from_bits(bits_t b) { return __longlong_as_double((long long)b); }
  static __host__ __device__ __forceinline__ double inf() { return HUGE_VAL; }
};
template <> struct Real<float> {
  typedef unsigned int bits_t;
  static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
  static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
  static __device__ __forceinline__ float sub(float a, float b) { return __fadd_rn(a, -b); }
  static __device__ __forceinline__ float div(float a, float b) { return __fdiv_rn(a, b); }
  static __device__ __forceinline__ float sqrt(float a) { return __fsqrt_rn(a); }
  static __device__ __forceinline__ bits_t bits(float a) { return __float_as_uint(a); }
  static __device__ __forceinline__ float from_bits(bits_t b) { return __uint_as_float(b); }
  static __host__ __device__ __forceinline__ float inf() { return HUGE_VALF; }
};

// Per-step scalars living on the device, so that a step never needs the host.
template <class T> struct DevScalars {
  T dt;                                  // time step of the step being enqueued
  typename Real<T>::bits_t smax_bits;    // max signal speed, IEEE bits (positive floats order like integers)
  double time;                           // sum of the time steps taken since cspt_set_state
  int has_vac;                           // did cspt_set_state see a cell with rho <= rho_vac (hint for the host, below)
};

// Kernel ids for cspt_profile_* (names in cspt_api.cu, same order).
enum KernelId { K_GHOST = 0, K_PREDICTOR, K_CORRECTOR, K_EULER, K_SPEED_MAX, K_SCALAR, K_IO, K_FORCE, K_COUNT };

}  // namespace cspt

struct cspt_ctx {
  cspt::Layout L;
  int dtype;
  int sm_count;            // multiprocessors of the device that was current in cspt_create
  int bc[6];
  double h, gamma;
  void* ws;
  size_t ws_bytes;
  cudaStream_t stream;
  int cur;                 // which U buffer holds U^n
  bool has_state;
  bool force_pending;      // cspt_set_state on a slab: psi is padded, f = -D[psi] waits for cspt_finish_state
  bool smax_valid;         // smax_bits on the device belongs to the current U^n
  bool ghosts_current;     // cspt_fill_ghosts ran on the current U^n (cspt_step_filled asks for it)
  bool halo_current[2];    // z-lo / z-hi ghost planes were written by cspt_halo_put(CSPT_HALO_U) for the current U^n
  int cuda_error;          // sticky
  long long launches;
  void* h_pinned;          // small pinned staging buffer (scalars; byte 32: has_vac of the last cspt_set_state)
  // Gas-vacuum hint (performance only, both kernel variants are exact): cspt_set_state counts nothing but notes whether
  // the state holds vacuum cells; the flag reaches the host asynchronously (vac_ev), and until it has, or after
  // cspt_set_conserved, the variant WITH the vacuum shortcuts runs.
  cudaEvent_t vac_ev;
  bool vac_pending;        // a copy of has_vac is in flight
  int vac_hint;            // 1: run the kernels with the shortcuts
  int vac_forced;          // cspt_debug_force_vacuum_variant: -1 = follow the hint, 0 / 1 = force the variant
  int step_vac;            // the hint the step being enqueued (or captured) uses
  bool capturing;          // inside cspt_run_cfl's stream capture
  size_t elem;             // sizeof(T)
  // workspace sub-buffers (byte offsets)
  size_t off_fields, off_inflow, off_scalars, off_map;
  size_t map_bytes;
  bool map_valid;          // the brick map covers every non-zero cell of the current U^n
  int tile_skip;           // cspt_debug_tile_skip: 1 (default) = dead CTAs may return early, 0 = never
  int zero_fill_steps;     // steps in which dead CTAs must still WRITE their zeros: 2 after the map was rebuilt or the
                           // intermediate slots served as staging (both U buffers and every intermediate get clean)
  long long inflow_plane;  // elements per captured plane
  // TMA views (x, y, z, field) of the two U buffers, of the (U~, xi) group and of the star group
  CUtensorMap mapU[2], mapL, mapS;
  CUtensorMap mapPU[2], mapPF;      // predictor: U^n (tile + halo 1) and f (tile)
  int pred_stages;                  // predictor: 0 = register prefetch, 2..4 = TMA ring of that many stages
  bool have_maps;
  int kernel;               // CSPT_KERNEL_*: smoothing kernel W of Eq. (7)
  int limiter;              // CSPT_LIMITER_*: TVD slope of Eq. (8) in the Euler stage
  int riemann;              // CSPT_RIEMANN_*: flux at the faces of the Euler stage
  int euler_variant;        // 0: one thread per cell with shared-memory flux exchange, 1: rows + helper warp
  int corr_variant;         // 0: 26-neighbour corrector, 1: pair-symmetric strips with shared x pairs (warp shuffles)
  // asynchronous host entry points (cspt_*_host_async): copy streams of their own, so that the device-to-host copy of
  // one result and the host-to-device copy of the next input use both directions of the link at once
  cudaStream_t h2d_stream, d2h_stream;
  cudaEvent_t ev_in_free, ev_in_ready, ev_out_ready, ev_out_done;
  bool out_pending;                 // a device-to-host copy may still read its staging slots (U~ / xi slots)
  // CUDA graphs of two consecutive cspt_step_cfl steps (cspt_run_cfl), one per parity of `cur` at entry
  cudaGraphExec_t graph[2];
  cudaStream_t gstream;             // capture / replay stream of a ctx that lives on the legacy default stream
  double graph_cfl;                 // the CFL number the graphs were captured with
  int graph_vac;                    // the vacuum hint the graphs were captured with
  // per-kernel device timing (cspt_profile_*): event pairs recorded around each launch
  bool prof_on;
  int prof_used;                    // pairs recorded since the last reset
  int prof_cap;                     // pairs allocated
  cudaEvent_t* prof_ev;             // 2 * prof_cap events
  int* prof_kid;                    // kernel id of each pair
};
