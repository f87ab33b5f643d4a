// cspt_api.cu -- the C ABI declared in include/cspt.h: argument checks, workspace
// carving and kernel launches.  All arithmetic of the method is in the kernels.
#include <new>
#include <stdlib.h>
#include <string.h>

#include "cspt_euler.cuh"
#include "cspt_lagrange.cuh"
#include "cspt_corrector.cuh"
#include "cspt_euler2.cuh"

using namespace cspt;

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

size_t elem_size(int dtype) { return dtype == CSPT_F64 ? 8 : 4; }

long long inflow_plane_elems(const Layout& L) {
  long long a = (long long)L.px * L.py, b = (long long)L.py * L.pz, c = (long long)L.px * L.pz;
  long long m = a > b ? a : b;
  return m > c ? m : c;
}

bool valid_dims(int nx, int ny, int nz, int dtype) {
  if (nx < 1 || ny < 1 || nz < 1) return false;
  if (dtype != CSPT_F64 && dtype != CSPT_F32) return false;
  Layout L = make_layout(nx, ny, nz);
  // 32-bit cell counts inside kernels are avoided, but keep the padded field below 2^40 elements
  return L.fstride < (1LL << 40);
}

void carve(cspt_ctx* c) {
  size_t e = c->elem;
  c->off_fields = 0;
  c->inflow_plane = inflow_plane_elems(c->L);
  c->off_inflow = align_up((size_t)S_COUNT * c->L.fstride * e, 256);
  c->off_scalars = align_up(c->off_inflow + (size_t)6 * 5 * c->inflow_plane * e, 256);
  c->off_map = c->off_scalars + 256;
  c->map_bytes = 256 + align_up((size_t)((c->L.px + BRX - 1) / BRX) * ((c->L.py + BRY - 1) / BRY) * ((c->L.pz + BRZ - 1) / BRZ), 256);
}

// the brick map of the CTA-level gas-vacuum shortcut (cspt_common.cuh); on = false: a map that switches it off
inline BrickMap brick_map(const cspt_ctx* c, bool on) {
  BrickMap M;
  M.raw = on ? (unsigned char*)c->ws + c->off_map + 256 : nullptr;      // first 256 bytes: the diagnostics counter
  M.dead = (unsigned long long*)((unsigned char*)c->ws + c->off_map);
  M.zero_fill = c->zero_fill_steps > 0 ? 1 : 0;
  M.nbx = (c->L.px + BRX - 1) / BRX; M.nby = (c->L.py + BRY - 1) / BRY; M.nbz = (c->L.pz + BRZ - 1) / BRZ;
  return M;
}

template <class T> T* field(cspt_ctx* c, int slot) { return (T*)((char*)c->ws + c->off_fields) + (long long)slot * c->L.fstride; }
template <class T> T* inflow(cspt_ctx* c, int face) { return (T*)((char*)c->ws + c->off_inflow) + (long long)face * 5 * c->inflow_plane; }
template <class T> DevScalars<T>* scalars(cspt_ctx* c) { return (DevScalars<T>*)((char*)c->ws + c->off_scalars); }

template <class T> Params<T> make_params(const cspt_ctx* c) {
  Params<T> P;
  P.L = c->L;
  P.h = (T)c->h;
  P.gamma = (T)c->gamma;
  P.rho_vac = (T)1e-12;
  P.inv_h = (T)1 / P.h;
  // g^(q) = -W'(q)/q at the lattice distances 1, sqrt 2, sqrt 3: Monaghan cubic spline with smoothing length h
  // (G5), or W ~ (1 - q^2/4)^5 for which g^ ~ (1 - q^2/4)^4
  double s2 = sqrt(2.0), s3 = sqrt(3.0);
  double g1 = 0.75, g2 = 0.75 * (2.0 - s2) * (2.0 - s2) / s2, g3 = 0.75 * (2.0 - s3) * (2.0 - s3) / s3;
  if (c->kernel == CSPT_KERNEL_POLY5) { g1 = 0.31640625; g2 = 0.0625; g3 = 0.00390625; }
  double S = 2.0 * g1 + 8.0 * g2 + 8.0 * g3;
  P.a1 = (T)(g1 / S); P.a2 = (T)(g2 / S); P.a3 = (T)(g3 / S);
  P.wnorm = (T)(1.0 / ((double)(T)S * (double)P.h * (double)P.h));
  for (int q = 0; q < 6; ++q) P.bc[q] = c->bc[q];
  return P;
}

inline int blocks_for(long long n, int threads, int cap = 0) {
  long long b = (n + threads - 1) / threads;
  if (b < 1) b = 1;
  if (cap > 0 && b > cap) b = cap;
  return (int)b;
}

constexpr int TPB = 256;
constexpr int STRIDE_CAP = 148 * 16;   // grid-stride kernels: 16 CTAs of 256 threads per SM

// Event pair around one launch when cspt_profile_enable is on (device time per kernel).
const char* const kKernelNames[K_COUNT] = {"ghost_fill", "predictor", "corrector", "euler", "speed_max",
                                           "scalar", "io", "force"};

inline int prof_open(cspt_ctx* c, int kid) {
  if (!c->prof_on || c->prof_used >= c->prof_cap) return -1;
  int s = c->prof_used++;
  c->prof_kid[s] = kid;
  cudaEventRecord(c->prof_ev[2 * s], c->stream);
  return s;
}
inline void prof_close(cspt_ctx* c, int s) {
  if (s >= 0) cudaEventRecord(c->prof_ev[2 * s + 1], c->stream);
}

#define LAUNCH(ctx, kid, kernel, grid, block, ...)                \
  do {                                                            \
    int ps_ = prof_open((ctx), (kid));                            \
    kernel<<<(grid), (block), 0, (ctx)->stream>>>(__VA_ARGS__);   \
    prof_close((ctx), ps_);                                       \
    (ctx)->launches++;                                            \
  } while (0)

int check(cspt_ctx* c) {
  if (c->cuda_error) return CSPT_ECUDA;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { c->cuda_error = (int)e; return CSPT_ECUDA; }
  return CSPT_OK;
}

int cuda_call(cspt_ctx* c, cudaError_t e) {
  if (e != cudaSuccess) { c->cuda_error = (int)e; return CSPT_ECUDA; }
  return CSPT_OK;
}

// ---- ghost layers, x then y then z (G16) ----------------------------------------------
template <class T>
void fill_ghosts(cspt_ctx* c, T* F, int nfields, int mode, BrickMap M = BrickMap{nullptr, 0, 0, 0, nullptr, 1}) {
  const Layout& L = c->L;
  int n[3] = {L.nx, L.ny, L.nz};
  for (int d = 0; d < 3; ++d) {
    int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    long long e1 = d1 < d ? n[d1] + 2 * NG : n[d1], e2 = d2 < d ? n[d2] + 2 * NG : n[d2];
    long long total = e1 * e2 * NG * 2;
    LAUNCH(c, K_GHOST, k_ghost_axis<T>, blocks_for(total, TPB, STRIDE_CAP), TPB, L, d, mode, c->bc[2 * d], c->bc[2 * d + 1],
           nfields, F, inflow<T>(c, 2 * d), inflow<T>(c, 2 * d + 1), c->inflow_plane, M);
  }
}

// the ghost layers of the current U (boundary rules and slab halos) no longer belong to it
inline void stale_ghosts(cspt_ctx* c) { c->ghosts_current = false; c->halo_current[0] = c->halo_current[1] = false; }

inline bool has_external(const cspt_ctx* c) { return c->bc[4] == CSPT_BC_EXTERNAL || c->bc[5] == CSPT_BC_EXTERNAL; }

// S2: f = -D[psi] on interior(+)2 from the padded psi (all ghost layers filled)
template <class T>
int finish_state_t(cspt_ctx* c) {
  Params<T> P = make_params<T>(c);
  T* psi_pad = field<T>(c, S_UT);          // scratch: U~ is dead between steps
  long long ne = (long long)(c->L.nx + 4) * (c->L.ny + 4) * (c->L.nz + 4);
  LAUNCH(c, K_FORCE, k_force<T>, blocks_for(ne, TPB, STRIDE_CAP), TPB, P, psi_pad, field<T>(c, S_F));
  c->force_pending = false;
  c->has_state = true;
  return check(c);
}

// z-slab halo: NG xy-padded planes are contiguous in a padded field.  get: the interior
// planes next to the face; put: the ghost planes of the face.
template <class T>
int halo_copy_t(cspt_ctx* c, int face, int what, void* buf, bool put) {
  const Layout& L = c->L;
  const long long plane = (long long)L.px * L.py, chunk = NG * plane;
  const int nf = what == CSPT_HALO_U ? 5 : 1;
  T* F = what == CSPT_HALO_U ? field<T>(c, c->cur ? S_U1 : S_U0) : field<T>(c, S_UT);
  // first padded plane of the region: ghost planes [0, NG) | [NG + nz, 2 NG + nz), interior planes [NG, 2 NG) | [nz, nz + NG)
  long long k0;
  if (put) k0 = face == 4 ? 0 : NG + L.nz;
  else k0 = face == 4 ? NG : L.nz;
  int ps_ = prof_open(c, K_IO);
  for (int f = 0; f < nf; ++f) {
    T* fld = F + f * L.fstride + k0 * plane;
    T* b = (T*)buf + f * chunk;
    cudaError_t e = put ? cudaMemcpyAsync(fld, b, chunk * sizeof(T), cudaMemcpyDeviceToDevice, c->stream)
                        : cudaMemcpyAsync(b, fld, chunk * sizeof(T), cudaMemcpyDeviceToDevice, c->stream);
    if (e != cudaSuccess) { c->cuda_error = (int)e; return CSPT_ECUDA; }
  }
  prof_close(c, ps_);
  return check(c);
}

template <class T>
int fill_ghosts_t(cspt_ctx* c) {
  // a valid brick map keeps following the gas (flags are only added; an invalid one is rebuilt from the filled array)
  fill_ghosts<T>(c, field<T>(c, c->cur ? S_U1 : S_U0), 5, 0, brick_map(c, c->dtype == CSPT_F32 && c->map_valid));
  c->ghosts_current = true;
  return check(c);
}

template <class T>
int set_state_t(cspt_ctx* c, const void* rho, const void* u, const void* v, const void* w, const void* p, const void* psi) {
  Params<T> P = make_params<T>(c);
  long long n = (long long)c->L.nx * c->L.ny * c->L.nz;
  T* U = field<T>(c, S_U0);
  T* psi_pad = field<T>(c, S_UT);          // scratch: U~ is dead between steps
  cudaMemsetAsync(&scalars<T>(c)->has_vac, 0, sizeof(int), c->stream);
  LAUNCH(c, K_IO, k_set_state<T>, blocks_for(n, TPB, STRIDE_CAP), TPB, P, (const T*)rho, (const T*)u, (const T*)v,
         (const T*)w, (const T*)p, (const T*)psi, U, psi_pad, &scalars<T>(c)->has_vac);
  // the hint travels to the host without a sync: until it has arrived the variant with the shortcuts runs
  cudaMemcpyAsync((char*)c->h_pinned + 32, &scalars<T>(c)->has_vac, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
  cudaEventRecord(c->vac_ev, c->stream);
  c->vac_pending = true;
  c->vac_hint = 1;
  fill_ghosts<T>(c, psi_pad, 1, 2);
  fill_ghosts<T>(c, U, 5, 1);
  LAUNCH(c, K_SCALAR, k_reset_smax<T>, 1, 1, scalars<T>(c), 1);
  c->cur = 0;
  c->smax_valid = false;
  c->has_state = false;
  c->force_pending = true;
  c->map_valid = false;
  stale_ghosts(c);
  // a slab (EXTERNAL z faces) needs the psi ghost planes of its neighbours before f = -D[psi] can be formed there:
  // cspt_halo_get/put(CSPT_HALO_PSI), then cspt_finish_state
  if (has_external(c)) return check(c);
  return finish_state_t<T>(c);
}

template <class T>
int set_conserved_t(cspt_ctx* c, const void* const in[5]) {
  long long n = (long long)c->L.nx * c->L.ny * c->L.nz;
  T* U = field<T>(c, c->cur ? S_U1 : S_U0);
  for (int f = 0; f < 5; ++f)
    LAUNCH(c, K_IO, k_put_field<T>, blocks_for(n, TPB, STRIDE_CAP), TPB, c->L, (const T*)in[f], U + f * c->L.fstride);
  c->vac_pending = false;        // the new state was not looked at: keep the shortcuts on
  c->vac_hint = 1;
  c->smax_valid = false;
  c->map_valid = false;
  stale_ghosts(c);
  return check(c);
}

template <class T>
int get_conserved_t(cspt_ctx* c, void* const out[5]) {
  long long n = (long long)c->L.nx * c->L.ny * c->L.nz;
  const T* U = field<T>(c, c->cur ? S_U1 : S_U0);
  for (int f = 0; f < 5; ++f)
    LAUNCH(c, K_IO, k_get_field<T>, blocks_for(n, TPB, STRIDE_CAP), TPB, c->L, U + f * c->L.fstride, (T*)out[f]);
  return check(c);
}

template <class T>
int get_state_t(cspt_ctx* c, void* rho, void* u, void* v, void* w, void* p, unsigned char* mask) {
  Params<T> P = make_params<T>(c);
  long long n = (long long)c->L.nx * c->L.ny * c->L.nz;
  const T* U = field<T>(c, c->cur ? S_U1 : S_U0);
  LAUNCH(c, K_IO, k_get_state<T>, blocks_for(n, TPB, STRIDE_CAP), TPB, P, U, (T*)rho, (T*)u, (T*)v, (T*)w, (T*)p, mask);
  return check(c);
}

template <class T>
void ensure_smax(cspt_ctx* c) {
  if (c->smax_valid) return;
  Params<T> P = make_params<T>(c);
  long long n = (long long)c->L.nx * c->L.ny * c->L.nz;
  LAUNCH(c, K_SCALAR, k_reset_smax<T>, 1, 1, scalars<T>(c), 0);
  LAUNCH(c, K_SPEED_MAX, k_speed_max<T>, blocks_for(n, TPB, STRIDE_CAP), TPB, P, field<T>(c, c->cur ? S_U1 : S_U0),
         &scalars<T>(c)->smax_bits);
  c->smax_valid = true;
}

template <class T>
int compute_dt_t(cspt_ctx* c, double cfl, double* out) {
  typedef typename Real<T>::bits_t bits_t;
  ensure_smax<T>(c);
  int rc = check(c);
  if (rc) return rc;
  bits_t* hb = (bits_t*)c->h_pinned;
  rc = cuda_call(c, cudaMemcpyAsync(hb, &scalars<T>(c)->smax_bits, sizeof(bits_t), cudaMemcpyDeviceToHost, c->stream));
  if (rc) return rc;
  rc = cuda_call(c, cudaStreamSynchronize(c->stream));
  if (rc) return rc;
  T smax;
  memcpy(&smax, hb, sizeof(T));
  // same two rn operations as k_dt_finalize and the oracle: (cfl*h)/smax in T
  volatile T num = (T)cfl * (T)c->h;
  T dt = smax > (T)0 ? (T)(num / smax) : Real<T>::inf();
  *out = (double)dt;
  return CSPT_OK;
}

// Euler-stage tile (threads = cells of one plane of the column)
constexpr int ETX = 32;
template <class T> struct EulerTile { static constexpr int TY = 8; };

// CTA-level gas-vacuum shortcut (BrickMap): only the fp32 streaming kernels carry it, the map follows the gas through
// the flags of the ghost fill and of the cell-per-thread Euler stage, and it pays only where the state holds vacuum
inline bool tile_skip_on(const cspt_ctx* c) {
  return c->dtype == CSPT_F32 && c->euler_variant == 0 && c->step_vac != 0 && c->tile_skip != 0 &&
         c->bc[4] != CSPT_BC_EXTERNAL && c->bc[5] != CSPT_BC_EXTERNAL;
}
inline BrickMap step_map(const cspt_ctx* c) { return brick_map(c, tile_skip_on(c)); }

// the map must cover every non-zero cell of the current U^n before a step may rely on it: rebuilt (one read of U) after
// cspt_set_state / cspt_set_conserved and after steps that ran without the flags
template <class T>
void ensure_map(cspt_ctx* c) {
  if (c->map_valid || !tile_skip_on(c)) return;
  BrickMap M = brick_map(c, true);
  cudaMemsetAsync(M.dead, 0, c->map_bytes, c->stream);      // counter and flags
  long long n = (long long)(c->L.nx + 2 * NG) * (c->L.ny + 2 * NG) * (c->L.nz + 2 * NG);
  LAUNCH(c, K_IO, k_brick_scan<T>, blocks_for(n, TPB, STRIDE_CAP), TPB, c->L, field<T>(c, c->cur ? S_U1 : S_U0), M);
  c->map_valid = true;
  c->zero_fill_steps = 2;
}

int pick_zchunk(int tiles, int nz) {
  // enough CTAs for ~8 waves of 2 CTAs per SM, at least 16 planes per CTA (2 extra planes per chunk) and at
  // most 64: CTAs of neighbouring tiles then stay close in z, so the halo rows they share are still in L2
  // (1024^3 fp32: corrector 41.5 -> 32.1 ms against one chunk per column)
  int want = (148 * 2 * 8 + tiles - 1) / tiles;
  int zc = (nz + want - 1) / want;
  if (zc < 16) zc = 16;
  if (zc > 64) zc = 64;
  if (zc > nz) zc = nz;
  return zc;
}

// Corrector variants: tile TX x TY cells per plane, CY cells (adjacent in y) per thread, NST ring
// stages, MINB resident CTAs per SM asked of the compiler.  P == nullptr: set the kernel up (TMA map of
// the star group, dynamic shared memory); otherwise launch it.
// Corrector: tile TX x TY cells per plane, CY cells (adjacent in y) per thread, NST ring stages, MINB resident
// CTAs per SM asked of the compiler, XP = 1 when x is periodic (interior columns only; the kernel also writes the ghost columns they wrap onto).
// P == nullptr: set the kernel up (TMA map of the star group, dynamic shared memory); otherwise launch it.
template <class T, int TX, int TY, int CY, int NST, int MINB, int XP>
bool corr_variant(cspt_ctx* c, const Params<T>* P, const T* U) {
  typedef CorrSmem<T, TX, TY, CY, NST, XP> SC;
  const Layout& L = c->L;
  auto kern0 = k_corrector_stream<T, TX, TY, CY, NST, MINB, 0, XP>;
  auto kern1 = k_corrector_stream<T, TX, TY, CY, NST, MINB, 1, XP>;
  if (!P) {
    // the star group as four pair arrays: inner dimension 2 px elements, 2 fstride elements per array
    return make_field_map(&c->mapS, field<T>(c, S_ST), (int)sizeof(T), 2 * L.px, L.py, L.pz, 2 * L.fstride, SC::NF,
                          2 * SC::BX, SC::BY, SC::NF) &&
           cudaFuncSetAttribute(kern0, cudaFuncAttributeMaxDynamicSharedMemorySize, SC::BYTES) == cudaSuccess &&
           cudaFuncSetAttribute(kern1, cudaFuncAttributeMaxDynamicSharedMemorySize, SC::BYTES) == cudaSuccess;
  }
  auto kern = c->kernel == CSPT_KERNEL_POLY5 ? kern1 : kern0;
  int nxe = XP ? L.nx : L.nx + 2;
  int gx = (nxe + TX - 1) / TX, gy = (L.ny + 2 + TY - 1) / TY;
  int zc = pick_zchunk(gx * gy, L.nz + 2);
  dim3 grid(gx, gy, (L.nz + 2 + zc - 1) / zc);
  int ps_ = prof_open(c, K_CORRECTOR);
  kern<<<grid, SC::THREADS, SC::BYTES, c->stream>>>(c->mapS, *P, scalars<T>(c), U, field<T>(c, S_F), field<T>(c, S_ST),
                                                     field<T>(c, S_UT), field<T>(c, S_XI), zc, step_map(c));
  prof_close(c, ps_);
  c->launches++;
  return true;
}

// 32 x 8 cells per plane, 2 cells per thread, 4 ring stages, 2 CTAs per SM (224 registers in fp64): the fastest of
// the tile shapes tried on B200 in round 1; the fp32 default (fp64 runs the pair-symmetric kernel below)
template <class T>
bool corr_dispatch(cspt_ctx* c, const Params<T>* P, const T* U) {
  return c->bc[0] == CSPT_BC_PERIODIC ? corr_variant<T, 32, 8, 2, 4, 2, 1>(c, P, U)
                                      : corr_variant<T, 32, 8, 2, 4, 2, 0>(c, P, U);
}

// Pair-symmetric corrector (cspt_corrector.cuh): strips of two rows, TY rows per CTA, NST ring stages, MINB CTAs per
// SM, XS = 1: pairs with the neighbouring lanes shared by warp shuffles (31 output columns per tile).
template <class T, int TY, int NST, int MINB, int XP, int XS>
bool pair_variant(cspt_ctx* c, const Params<T>* P, const T* U) {
  typedef PairSmem<T, TY, NST, XS> SC;
  const Layout& L = c->L;
  auto kern0 = k_corrector_pairs<T, TY, NST, MINB, 0, XP, XS>;
  auto kern1 = k_corrector_pairs<T, TY, NST, MINB, 1, XP, XS>;
  if (!P) {
    return make_field_map(&c->mapS, field<T>(c, S_ST), (int)sizeof(T), 2 * L.px, L.py, L.pz, 2 * L.fstride, SC::NF,
                          2 * SC::BX, SC::BY, SC::NF) &&
           cudaFuncSetAttribute(kern0, cudaFuncAttributeMaxDynamicSharedMemorySize, SC::BYTES) == cudaSuccess &&
           cudaFuncSetAttribute(kern1, cudaFuncAttributeMaxDynamicSharedMemorySize, SC::BYTES) == cudaSuccess;
  }
  auto kern = c->kernel == CSPT_KERNEL_POLY5 ? kern1 : kern0;
  int nxe = XP ? L.nx : L.nx + 2;
  int gx = (nxe + SC::TXO - 1) / SC::TXO, gy = (L.ny + 2 + TY - 1) / TY;
  int zc = pick_zchunk(gx * gy, L.nz + 2);
  dim3 grid(gx, gy, (L.nz + 2 + zc - 1) / zc);
  int ps_ = prof_open(c, K_CORRECTOR);
  kern<<<grid, SC::THREADS, SC::BYTES, c->stream>>>(c->mapS, *P, scalars<T>(c), U, field<T>(c, S_F), field<T>(c, S_UT),
                                                     field<T>(c, S_XI), zc);
  prof_close(c, ps_);
  c->launches++;
  return true;
}

template <class T>
bool corr_select(cspt_ctx* c, const Params<T>* P, const T* U) {
  // one layout per precision, each the fastest measured on B200 (profiles/r2_kernels.md); the other is not compiled
  if constexpr (sizeof(T) == 4) return corr_dispatch<T>(c, P, U);
  else {
    const bool xp = c->bc[0] == CSPT_BC_PERIODIC;
    return xp ? pair_variant<T, 8, 4, 2, 1, 1>(c, P, U) : pair_variant<T, 8, 4, 2, 0, 1>(c, P, U);
  }
}

// Euler stage, second layout (cspt_euler2.cuh): TY rows of 32 cells + one helper warp per CTA.
// P == nullptr: tensor maps and dynamic shared memory; otherwise launch.
template <class T, int TY, int MINB, int UNR, int LIM, int RIEM>
bool euler2_kernel(cspt_ctx* c, const Params<T>* P, const T* U, T* UN) {
  typedef Euler2Smem<T, TY> S;
  auto kern = k_euler_rows<T, TY, MINB, LIM, RIEM, UNR>;
  if (!P) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::BYTES) == cudaSuccess;
  const Layout& L = c->L;
  int gx = (L.nx + S::TX - 1) / S::TX, gy = (L.ny + TY - 1) / TY;
  int zc = pick_zchunk(gx * gy, L.nz);
  dim3 grid(gx, gy, (L.nz + zc - 1) / zc);
  DevScalars<T>* sc = scalars<T>(c);
  int ps_ = prof_open(c, K_EULER);
  kern<<<grid, S::THREADS, S::BYTES, c->stream>>>(c->mapU[c->cur], c->mapL, *P, sc, U, UN, &sc->smax_bits, zc);
  prof_close(c, ps_);
  c->launches++;
  return true;
}

template <class T, int TY, int MINB, int UNR>
bool euler2_variant(cspt_ctx* c, const Params<T>* P, const T* U, T* UN) {
  typedef Euler2Smem<T, TY> S;
  const Layout& L = c->L;
  if (!P) {
    bool ok = true;
    for (int b = 0; b < 2; ++b)
      ok = ok && make_field_map(&c->mapU[b], field<T>(c, b ? S_U1 : S_U0), (int)sizeof(T), L.px, L.py, L.pz, L.fstride, 5,
                                S::BX, S::UY, 5);
    ok = ok && make_field_map(&c->mapL, field<T>(c, S_UT), (int)sizeof(T), L.px, L.py, L.pz, L.fstride, 7, S::BX, S::LY, 7);
    return ok && euler2_kernel<T, TY, MINB, UNR, 0, 0>(c, P, U, UN) && euler2_kernel<T, TY, MINB, UNR, 1, 0>(c, P, U, UN) &&
           euler2_kernel<T, TY, MINB, UNR, 0, 1>(c, P, U, UN) && euler2_kernel<T, TY, MINB, UNR, 1, 1>(c, P, U, UN) &&
           euler2_kernel<T, TY, MINB, UNR, 0, 2>(c, P, U, UN) && euler2_kernel<T, TY, MINB, UNR, 1, 2>(c, P, U, UN);
  }
  const bool vl = c->limiter == CSPT_LIMITER_VANLEER;
  switch (c->riemann) {
    case CSPT_RIEMANN_LF: return vl ? euler2_kernel<T, TY, MINB, UNR, 1, 1>(c, P, U, UN) : euler2_kernel<T, TY, MINB, UNR, 0, 1>(c, P, U, UN);
    case CSPT_RIEMANN_HLLC: return vl ? euler2_kernel<T, TY, MINB, UNR, 1, 2>(c, P, U, UN) : euler2_kernel<T, TY, MINB, UNR, 0, 2>(c, P, U, UN);
    default: return vl ? euler2_kernel<T, TY, MINB, UNR, 1, 0>(c, P, U, UN) : euler2_kernel<T, TY, MINB, UNR, 0, 0>(c, P, U, UN);
  }
}

template <class T>
bool euler1_setup(cspt_ctx* c) {
  const Layout& L = c->L;
  typedef EulerSmem<T, ETX, EulerTile<T>::TY> S;
  constexpr int ETY = EulerTile<T>::TY;
  bool ok = true;
  for (int b = 0; b < 2; ++b)
    ok = ok && make_field_map(&c->mapU[b], field<T>(c, b ? S_U1 : S_U0), (int)sizeof(T), L.px, L.py, L.pz, L.fstride, 5,
                              S::BX, S::UY, 5);
  ok = ok && make_field_map(&c->mapL, field<T>(c, S_UT), (int)sizeof(T), L.px, L.py, L.pz, L.fstride, 7, S::BX, S::LY, 7);
  if (ok) {
    ok = cudaFuncSetAttribute(k_euler_stream<T, ETX, ETY, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::BYTES) == cudaSuccess &&
         cudaFuncSetAttribute(k_euler_stream<T, ETX, ETY, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::BYTES) == cudaSuccess &&
         cudaFuncSetAttribute(k_euler_stream<T, ETX, ETY, 0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::BYTES) == cudaSuccess &&
         cudaFuncSetAttribute(k_euler_stream<T, ETX, ETY, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::BYTES) == cudaSuccess;
  }
  return ok;
}

// Row layout: 7 rows + helper warp per CTA; fp64 at 2 CTAs per SM (128 registers) with the z loop unrolled twice,
// fp32 at 3 CTAs per SM (the fastest of the shapes measured, profiles/r2_kernels.md)
template <class T>
bool euler_select(cspt_ctx* c, const Params<T>* P, const T* U, T* UN) {
  if (c->euler_variant == 0) return false;
  if constexpr (sizeof(T) == 8) return euler2_variant<T, 7, 2, 2>(c, P, U, UN);
  else return euler2_variant<T, 7, 3, 1>(c, P, U, UN);
}

// tensor maps and shared-memory attributes of the Euler layout the ctx is on (the cell-per-thread layout exists in
// fp32 only)
template <class T>
bool euler_setup(cspt_ctx* c) {
  if constexpr (sizeof(T) == 4) { if (c->euler_variant == 0) return euler1_setup<T>(c); }
  return euler_select<T>(c, nullptr, nullptr, nullptr);
}

template <class T>
bool make_maps(cspt_ctx* c) {
  return euler_setup<T>(c) && corr_select<T>(c, nullptr, nullptr);
}

// primitives + HFC/SUL{predictor} over the extended domain interior(+)2: 32 x 4 tiles, inputs through a TMA ring of two
// stages (3.78 -> 3.14 ms in fp64, 2.04 -> 1.75 ms in fp32 against the register prefetch; deeper rings and 32 x 8 tiles
// measured slower, profiles/r2_kernels.md)
constexpr int PTX = 32, PTY = 4;
template <class T>
void launch_predictor(cspt_ctx* c, const Params<T>& P, const T* U) {
  const Layout& L = c->L;
  const bool xp = c->bc[0] == CSPT_BC_PERIODIC;        // periodic x: interior columns only, ghost columns copied
  int x0 = xp ? 0 : -2, x1 = xp ? L.nx : L.nx + 2;
  int gx = (x1 - x0 + PTX - 1) / PTX, gy = (L.ny + 4 + PTY - 1) / PTY;
  int zc = pick_zchunk(gx * gy, L.nz + 4);
  dim3 grid(gx, gy, (L.nz + 4 + zc - 1) / zc);
  int ps_ = prof_open(c, K_PREDICTOR);
  auto launch = [&](auto kern, int bytes) {
    kern<<<grid, PTX * PTY, bytes, c->stream>>>(c->mapPU[c->cur], c->mapPF, P, scalars<T>(c), U, field<T>(c, S_F),
                                                 field<T>(c, S_ST), zc, x0, x1, step_map(c));
  };
  launch(k_predictor_stream<T, PTX, PTY, 2>, PredRing<T, PTX, PTY, 2>::BYTES);
  prof_close(c, ps_);
  c->launches++;
}

// TMA views of the predictor's inputs (cspt_lagrange.cuh, PredRing) and the dynamic shared memory of its ring
template <class T>
bool predictor_setup(cspt_ctx* c) {
  const Layout& L = c->L;
  typedef PredRing<T, PTX, PTY, 2> R;
  bool ok = true;
  for (int b = 0; b < 2; ++b)
    ok = ok && make_field_map(&c->mapPU[b], field<T>(c, b ? S_U1 : S_U0), (int)sizeof(T), L.px, L.py, L.pz, L.fstride, 5,
                              R::BXT, PTY + 2, 5);
  ok = ok && make_field_map(&c->mapPF, field<T>(c, S_F), (int)sizeof(T), L.px, L.py, L.pz, L.fstride, 3, R::BXT, PTY, 3);
  ok = ok && cudaFuncSetAttribute(k_predictor_stream<T, PTX, PTY, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  PredRing<T, PTX, PTY, 2>::BYTES) == cudaSuccess;
  return ok;
}

// HFC/SUL{corrector} over the extended domain interior(+)1
template <class T>
void launch_corrector(cspt_ctx* c, const Params<T>& P, const T* U) {
  corr_select<T>(c, &P, U);
}

// 1: run the kernel variants with the gas-vacuum shortcuts (the state holds vacuum cells, or nobody has looked yet)
int vacuum_hint(cspt_ctx* c) {
  if (c->vac_forced >= 0) return c->vac_forced;
  if (c->vac_pending) {
    cudaError_t q = cudaEventQuery(c->vac_ev);
    if (q == cudaSuccess) {
      c->vac_hint = *(volatile int*)((char*)c->h_pinned + 32) != 0;
      c->vac_pending = false;
    } else if (q == cudaErrorNotReady) {
      (void)cudaGetLastError();  // "not ready" is not an error of the ctx; anything else stays pending for check()
    }
  }
  return c->vac_hint;
}

template <class T>
void launch_euler(cspt_ctx* c, const Params<T>& P, const T* U, T* UN) {
  if (sizeof(T) == 8 || c->euler_variant) { euler_select<T>(c, &P, U, UN); return; }
  if constexpr (sizeof(T) == 4) {
  typedef EulerSmem<T, ETX, EulerTile<T>::TY> S;
  constexpr int ETY = EulerTile<T>::TY;
  const Layout& L = c->L;
  int gx = (L.nx + ETX - 1) / ETX, gy = (L.ny + ETY - 1) / ETY;
  int zc = pick_zchunk(gx * gy, L.nz);
  dim3 grid(gx, gy, (L.nz + zc - 1) / zc);
  DevScalars<T>* sc = scalars<T>(c);
  int ps_ = prof_open(c, K_EULER);
  const bool vl = c->limiter == CSPT_LIMITER_VANLEER, vac = c->step_vac != 0;
  auto kern = vac ? (vl ? k_euler_stream<T, ETX, ETY, 1, 1> : k_euler_stream<T, ETX, ETY, 0, 1>)
                  : (vl ? k_euler_stream<T, ETX, ETY, 1, 0> : k_euler_stream<T, ETX, ETY, 0, 0>);
  kern<<<grid, ETX * ETY, S::BYTES, c->stream>>>(c->mapU[c->cur], c->mapL, P, sc, U, UN, &sc->smax_bits, zc, step_map(c));
  prof_close(c, ps_);
  c->launches++;
  }
}

// a result on its way to the host (cspt_get_conserved_host_async) is staged in the U~ / xi slots: a step waits for it
void wait_pending_output(cspt_ctx* c) {
  if (c->out_pending && !c->capturing) {
    cudaStreamWaitEvent(c->stream, c->ev_out_done, 0);
    c->out_pending = false;
  }
}

template <class T>
void run_step(cspt_ctx* c, bool fill = true) {
  wait_pending_output(c);
  if (!c->capturing) { c->step_vac = vacuum_hint(c); ensure_map<T>(c); }
  Params<T> P = make_params<T>(c);
  T* U = field<T>(c, c->cur ? S_U1 : S_U0);
  T* UN = field<T>(c, c->cur ? S_U0 : S_U1);
  if (fill) fill_ghosts<T>(c, U, 5, 0, step_map(c));                               // O0
  launch_predictor<T>(c, P, U);                                                    // O1, O3, O4
  launch_corrector<T>(c, P, U);                                                    // O5, O6
  launch_euler<T>(c, P, U, UN);                                                  // O7, O8 (+O9 epilogue)
  c->cur ^= 1;
  c->smax_valid = true;
  stale_ghosts(c);               // U^{n+1} has no ghost layers yet
  if (!tile_skip_on(c)) c->map_valid = false;      // this step did not flag where its gas went
  else if (c->zero_fill_steps > 0) c->zero_fill_steps--;
}

template <class T>
int step_t(cspt_ctx* c, double dt) {
  LAUNCH(c, K_SCALAR, k_set_dt<T>, 1, 1, scalars<T>(c), (T)dt);
  run_step<T>(c);
  return check(c);
}

template <class T>
int step_filled_t(cspt_ctx* c, double dt) {
  LAUNCH(c, K_SCALAR, k_set_dt<T>, 1, 1, scalars<T>(c), (T)dt);
  run_step<T>(c, false);
  return check(c);
}

// slab path: the signal-speed maximum stays on the device, the caller max-reduces it over the slabs in place
template <class T>
int smax_device_t(cspt_ctx* c, void** ptr) {
  ensure_smax<T>(c);
  *ptr = &scalars<T>(c)->smax_bits;
  return check(c);
}

template <class T>
int step_filled_cfl_t(cspt_ctx* c, double cfl, double* out) {
  LAUNCH(c, K_SCALAR, k_dt_finalize<T>, 1, 1, scalars<T>(c), (T)cfl, (T)c->h);
  run_step<T>(c, false);
  int rc = check(c);
  if (rc || !out) return rc;
  T* hb = (T*)c->h_pinned;
  rc = cuda_call(c, cudaMemcpyAsync(hb, &scalars<T>(c)->dt, sizeof(T), cudaMemcpyDeviceToHost, c->stream));
  if (rc) return rc;
  rc = cuda_call(c, cudaStreamSynchronize(c->stream));
  if (rc) return rc;
  *out = (double)*hb;
  return CSPT_OK;
}

template <class T>
int step_cfl_t(cspt_ctx* c, double cfl, double* out) {
  ensure_smax<T>(c);
  LAUNCH(c, K_SCALAR, k_dt_finalize<T>, 1, 1, scalars<T>(c), (T)cfl, (T)c->h);
  run_step<T>(c);
  int rc = check(c);
  if (rc || !out) return rc;
  T* hb = (T*)c->h_pinned;
  rc = cuda_call(c, cudaMemcpyAsync(hb, &scalars<T>(c)->dt, sizeof(T), cudaMemcpyDeviceToHost, c->stream));
  if (rc) return rc;
  rc = cuda_call(c, cudaStreamSynchronize(c->stream));
  if (rc) return rc;
  *out = (double)*hb;
  return CSPT_OK;
}

// ---- cspt_run_cfl: n steps of cspt_step_cfl replayed from a CUDA graph ------------------------------------------
// One graph holds TWO consecutive steps, so that the ping-pong of the U buffers is back where it started; there is
// one graph per parity of `cur` at entry.  Anything that changes what a step launches drops the graphs.
void drop_graphs(cspt_ctx* c) {
  for (int k = 0; k < 2; ++k)
    if (c->graph[k]) { cudaGraphExecDestroy(c->graph[k]); c->graph[k] = nullptr; }
}

// The legacy default stream cannot be captured: a ctx created on it captures and replays on a stream of its own, a
// BLOCKING one, which the default stream orders itself against implicitly.
cudaStream_t graph_stream(cspt_ctx* c) {
  if (c->stream) return c->stream;
  if (!c->gstream && cudaStreamCreate(&c->gstream) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
  return c->gstream;
}

template <class T>
int capture_two_steps(cspt_ctx* c, double cfl) {
  const int k = c->cur;
  cudaGraph_t g = nullptr;
  cudaStream_t gs = graph_stream(c), user = c->stream;
  if (!gs) { c->cuda_error = (int)cudaErrorUnknown; return CSPT_ECUDA; }
  c->step_vac = c->graph_vac = vacuum_hint(c);
  ensure_map<T>(c);                                  // on the ctx's stream, ahead of the capture (the graph only adds flags)
  int rc = cuda_call(c, cudaStreamBeginCapture(gs, cudaStreamCaptureModeThreadLocal));
  if (rc) return rc;
  c->capturing = true;
  const long long l0 = c->launches;
  c->stream = gs;
  for (int s = 0; s < 2; ++s) {
    LAUNCH(c, K_SCALAR, k_dt_finalize<T>, 1, 1, scalars<T>(c), (T)cfl, (T)c->h);
    run_step<T>(c);
  }
  c->stream = user;
  c->capturing = false;
  c->launches = l0;                                  // counted when the graph is launched
  cudaError_t e = cudaStreamEndCapture(gs, &g);
  if (e != cudaSuccess || !g) { (void)cudaGetLastError(); c->cuda_error = (int)(e ? e : cudaErrorUnknown); return CSPT_ECUDA; }
  e = cudaGraphInstantiate(&c->graph[k], g, 0);
  cudaGraphDestroy(g);
  if (e != cudaSuccess) { (void)cudaGetLastError(); c->cuda_error = (int)e; return CSPT_ECUDA; }
  c->graph_cfl = cfl;
  return CSPT_OK;
}

template <class T>
int run_cfl_t(cspt_ctx* c, double cfl, int nsteps, double* t_out) {
  wait_pending_output(c);
  ensure_smax<T>(c);
  int rc = check(c);
  if (rc) return rc;
  int left = nsteps;
  // CTA-level vacuum shortcut: the graphs bake in "the zeros of dead CTAs are in place", which holds once two plain
  // steps have written them (after the map was rebuilt or the intermediate slots served as staging)
  if (!c->prof_on && left >= 2) {
    c->step_vac = vacuum_hint(c);
    if (tile_skip_on(c)) {
      ensure_map<T>(c);
      for (; left > 0 && c->zero_fill_steps > 0; --left) {
        LAUNCH(c, K_SCALAR, k_dt_finalize<T>, 1, 1, scalars<T>(c), (T)cfl, (T)c->h);
        run_step<T>(c);
      }
    }
  }
  if (!c->prof_on && left >= 2) {                    // event pairs cannot be recorded inside a graph: plain loop then
    if ((c->graph[0] || c->graph[1]) && (c->graph_cfl != cfl || c->graph_vac != vacuum_hint(c))) drop_graphs(c);
    if (!c->graph[c->cur]) {
      rc = capture_two_steps<T>(c, cfl);
      if (rc) return rc;
    }
    c->step_vac = c->graph_vac;
    const long long per_pair = 2 * 7;                // 3 ghost fills, predictor, corrector, Euler stage, dt
    for (; left >= 2; left -= 2) {
      rc = cuda_call(c, cudaGraphLaunch(c->graph[c->cur], graph_stream(c)));
      if (rc) return rc;
      c->launches += per_pair;
    }
  }
  for (; left > 0; --left) {
    LAUNCH(c, K_SCALAR, k_dt_finalize<T>, 1, 1, scalars<T>(c), (T)cfl, (T)c->h);
    run_step<T>(c);
  }
  rc = check(c);
  if (rc || !t_out) return rc;
  double* hb = (double*)c->h_pinned;
  rc = cuda_call(c, cudaMemcpyAsync(hb, &scalars<T>(c)->time, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  if (rc) return rc;
  rc = cuda_call(c, cudaStreamSynchronize(c->stream));
  if (rc) return rc;
  *t_out = *hb;
  return CSPT_OK;
}

template <class T>
int probe_fma_t(cspt_ctx* c, int other_per_fma, double min_ms, double* fma_per_second) {
  // scratch: the star-group slots are dead between steps; the kernel's stores are a sink that wraps around it, so
  // the grid always fills the device (8 CTAs of 128 threads per SM), whatever the size of the ctx's grid
  T* out = field<T>(c, S_ST);
  c->zero_fill_steps = 2;          // the sink overwrites slots that dead CTAs rely on
  const int threads = 128, blocks = c->sm_count * 8, iters = other_per_fma ? 1500 : 4000;
  long long room = c->L.fstride * 8, want = (long long)threads * blocks;
  const unsigned cap = (unsigned)(room < want ? room : want);
  auto kern = other_per_fma < 0    ? k_probe_fma<T, -1>
              : other_per_fma == 0 ? k_probe_fma<T, 0>
              : other_per_fma == 1 ? k_probe_fma<T, 1>
              : other_per_fma == 2 ? k_probe_fma<T, 2>
              : other_per_fma == 4 ? k_probe_fma<T, 4>
                                   : k_probe_fma<T, 8>;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { (void)cudaGetLastError(); return CSPT_ECUDA; }
  kern<<<blocks, threads, 0, c->stream>>>(out, cap, 200, (T)1.0000001, (T)1e-9, 5);          // warm-up
  c->launches++;
  // one timed launch first; if the caller wants the probe to last min_ms (so that it runs in the power state a long
  // step runs in, and a clock sampler sees it), as many launches back to back as that takes are timed as one region
  int rc = 0, reps = 1;
  float ms = 0;
  for (int pass = 0; pass < 2 && !rc; ++pass) {
    cudaEventRecord(e0, c->stream);
    for (int r = 0; r < reps; ++r) kern<<<blocks, threads, 0, c->stream>>>(out, cap, iters, (T)1.0000001, (T)1e-9, 5);
    cudaEventRecord(e1, c->stream);
    c->launches += reps;
    rc = cuda_call(c, cudaEventSynchronize(e1));
    if (!rc) rc = cuda_call(c, cudaEventElapsedTime(&ms, e0, e1));
    if (rc || pass == 1 || !(min_ms > (double)ms) || !(ms > 0)) break;
    double need = min_ms / (double)ms;
    reps = need > 4096.0 ? 4096 : (int)need + 1;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (rc) return rc;
  *fma_per_second = (double)reps * iters * 64.0 * threads * blocks / ((double)ms * 1e-3);
  return check(c);
}

// dense staging arrays for the *_host entry points live in the (dead between steps)
// star-group slots S_ST.. (8 padded slots >= 6 dense arrays)
template <class T> T* staging(cspt_ctx* c, int f) { return field<T>(c, S_ST + f); }
// staging of cspt_get_conserved_host_async: the U~ (but the first, psi's scratch) and xi slots, dead between steps and
// untouched by cspt_set_state, so that the next input can be staged while the result is still on its way out
template <class T> T* staging_out(cspt_ctx* c, int f) { return field<T>(c, S_UT + 1 + f); }

bool ensure_copy_streams(cspt_ctx* c) {
  if (c->h2d_stream) return true;
  bool ok = cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking) == cudaSuccess;
  cudaEvent_t* ev[4] = {&c->ev_in_free, &c->ev_in_ready, &c->ev_out_ready, &c->ev_out_done};
  for (int k = 0; ok && k < 4; ++k) ok = cudaEventCreateWithFlags(ev[k], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) { (void)cudaGetLastError(); c->cuda_error = (int)cudaErrorUnknown; }
  return ok;
}

}  // namespace

#define DISPATCH(c, call) ((c)->dtype == CSPT_F64 ? call<double> : call<float>)

extern "C" {

size_t cspt_workspace_bytes(int nx, int ny, int nz, int dtype) {
  if (!valid_dims(nx, ny, nz, dtype)) return 0;
  cspt_ctx tmp;
  tmp.L = make_layout(nx, ny, nz);
  tmp.elem = elem_size(dtype);
  carve(&tmp);
  return tmp.off_map + tmp.map_bytes;
}

int cspt_create(cspt_ctx** out, int nx, int ny, int nz, double h, double gamma, const int bc[6], int dtype,
                void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return CSPT_EINVAL;
  *out = nullptr;
  if (!bc || !workspace || !valid_dims(nx, ny, nz, dtype)) return CSPT_EINVAL;
  if (!(h > 0) || !(gamma > 1) || !isfinite(h) || !isfinite(gamma)) return CSPT_EINVAL;
  int n[3] = {nx, ny, nz};
  for (int d = 0; d < 3; ++d) {
    int lo = bc[2 * d], hi = bc[2 * d + 1];
    const int kmax = d == 2 ? CSPT_BC_EXTERNAL : CSPT_BC_INFLOW;         // EXTERNAL: z faces only (slab decomposition)
    if (lo < 0 || lo > kmax || hi < 0 || hi > kmax) return CSPT_EINVAL;
    if ((lo == CSPT_BC_PERIODIC) != (hi == CSPT_BC_PERIODIC)) return CSPT_EINVAL;
    if (lo != CSPT_BC_PERIODIC && n[d] < 4) return CSPT_EINVAL;
  }
  if (((uintptr_t)workspace & 255) != 0) return CSPT_EINVAL;
  if (workspace_bytes < cspt_workspace_bytes(nx, ny, nz, dtype)) return CSPT_EINVAL;
  cspt_ctx* c = new (std::nothrow) cspt_ctx;
  if (!c) return CSPT_ENOMEM;
  memset(c, 0, sizeof(*c));
  c->L = make_layout(nx, ny, nz);
  c->dtype = dtype;
  c->elem = elem_size(dtype);
  for (int q = 0; q < 6; ++q) c->bc[q] = bc[q];
  c->h = h; c->gamma = gamma;
  c->ws = workspace; c->ws_bytes = workspace_bytes;
  c->stream = (cudaStream_t)cuda_stream;
  carve(c);
  // kernel layouts per precision, each the fastest measured on B200 (profiles/r2_kernels.md): fp64 is bound by
  // the FP64 pipe and the issue port (profiles/r2_issue_model.md) and runs the pair-symmetric corrector and the
  // row-per-warp Euler stage; fp32 keeps the packed-f32x2 corrector and the one-thread-per-cell Euler stage
  c->corr_variant = dtype == CSPT_F64 ? 1 : 0;
  c->euler_variant = dtype == CSPT_F64 ? 1 : 0;
  c->pred_stages = 2;
  c->vac_forced = -1;            // cspt_debug_force_vacuum_variant
  c->tile_skip = 1;              // cspt_debug_tile_skip
  if (cudaMallocHost(&c->h_pinned, 64) != cudaSuccess) { (void)cudaGetLastError(); delete c; return CSPT_ECUDA; }
  if (cudaEventCreateWithFlags(&c->vac_ev, cudaEventDisableTiming) != cudaSuccess) {
    (void)cudaGetLastError(); cudaFreeHost(c->h_pinned); delete c; return CSPT_ECUDA;
  }
  c->vac_hint = 1;
  {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
      (void)cudaGetLastError(); cudaEventDestroy(c->vac_ev); cudaFreeHost(c->h_pinned); delete c; return CSPT_ECUDA;
    }
    c->sm_count = sms;
  }
  c->have_maps = dtype == CSPT_F64 ? (make_maps<double>(c) && predictor_setup<double>(c))
                                   : (make_maps<float>(c) && predictor_setup<float>(c));
  if (!c->have_maps) { (void)cudaGetLastError(); cudaEventDestroy(c->vac_ev); cudaFreeHost(c->h_pinned); delete c; return CSPT_ECUDA; }

  *out = c;
  return CSPT_OK;
}

void cspt_destroy(cspt_ctx* c) {
  if (!c) return;
  drop_graphs(c);
  if (c->gstream) cudaStreamDestroy(c->gstream);
  if (c->h_pinned) cudaFreeHost(c->h_pinned);
  if (c->vac_ev) cudaEventDestroy(c->vac_ev);
  if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
  if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
  for (cudaEvent_t e : {c->ev_in_free, c->ev_in_ready, c->ev_out_ready, c->ev_out_done})
    if (e) cudaEventDestroy(e);
  for (int i = 0; i < 2 * c->prof_cap; ++i) cudaEventDestroy(c->prof_ev[i]);
  delete[] c->prof_ev;
  delete[] c->prof_kid;
  delete c;
}

int cspt_profile_enable(cspt_ctx* c, int on) {
  if (!c) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  if (on && !c->prof_ev) {
    const int cap = 8192;
    c->prof_ev = new (std::nothrow) cudaEvent_t[2 * cap];
    c->prof_kid = new (std::nothrow) int[cap];
    if (!c->prof_ev || !c->prof_kid) { delete[] c->prof_ev; delete[] c->prof_kid; c->prof_ev = nullptr; c->prof_kid = nullptr; return CSPT_ENOMEM; }
    for (int i = 0; i < 2 * cap; ++i) {
      int rc = cuda_call(c, cudaEventCreate(&c->prof_ev[i]));
      if (rc) { c->prof_cap = i / 2; return rc; }
    }
    c->prof_cap = cap;
  }
  c->prof_on = on != 0;
  if (on) c->prof_used = 0;
  return CSPT_OK;
}

int cspt_profile_kernel_count(void) { return K_COUNT; }

const char* cspt_profile_kernel_name(int kid) { return kid >= 0 && kid < K_COUNT ? kKernelNames[kid] : nullptr; }

int cspt_profile_read(cspt_ctx* c, int kid, double* total_ms, long long* launches) {
  if (!c || kid < 0 || kid >= K_COUNT || !total_ms || !launches) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  int rc = cuda_call(c, cudaStreamSynchronize(c->stream));
  if (rc) return rc;
  double ms = 0;
  long long n = 0;
  for (int s = 0; s < c->prof_used; ++s) {
    if (c->prof_kid[s] != kid) continue;
    float t = 0;
    rc = cuda_call(c, cudaEventElapsedTime(&t, c->prof_ev[2 * s], c->prof_ev[2 * s + 1]));
    if (rc) return rc;
    ms += t;
    ++n;
  }
  *total_ms = ms;
  *launches = n;
  return CSPT_OK;
}

int cspt_set_state(cspt_ctx* c, const void* rho, const void* u, const void* v, const void* w, const void* p,
                   const void* psi) {
  if (!c || !rho || !u || !v || !w || !p || !psi) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, set_state_t)(c, rho, u, v, w, p, psi);
}

int cspt_set_state_host(cspt_ctx* c, const void* rho, const void* u, const void* v, const void* w, const void* p,
                        const void* psi) {
  if (!c || !rho || !u || !v || !w || !p || !psi) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  const void* in[6] = {rho, u, v, w, p, psi};
  void* dev[6];
  size_t bytes = (size_t)c->L.nx * c->L.ny * c->L.nz * c->elem;
  for (int f = 0; f < 6; ++f) {
    dev[f] = c->dtype == CSPT_F64 ? (void*)staging<double>(c, f) : (void*)staging<float>(c, f);
    int rc = cuda_call(c, cudaMemcpyAsync(dev[f], in[f], bytes, cudaMemcpyHostToDevice, c->stream));
    if (rc) return rc;
  }
  int rc = DISPATCH(c, set_state_t)(c, dev[0], dev[1], dev[2], dev[3], dev[4], dev[5]);
  if (rc) return rc;
  return cuda_call(c, cudaStreamSynchronize(c->stream));
}

int cspt_set_state_host_async(cspt_ctx* c, const void* rho, const void* u, const void* v, const void* w, const void* p,
                              const void* psi) {
  if (!c || !rho || !u || !v || !w || !p || !psi) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  if (!ensure_copy_streams(c)) return CSPT_ECUDA;
  const void* in[6] = {rho, u, v, w, p, psi};
  void* dev[6];
  size_t bytes = (size_t)c->L.nx * c->L.ny * c->L.nz * c->elem;
  // the staging slots are the star group of the last step: the copies start when the work enqueued so far is done
  int rc = cuda_call(c, cudaEventRecord(c->ev_in_free, c->stream));
  if (!rc) rc = cuda_call(c, cudaStreamWaitEvent(c->h2d_stream, c->ev_in_free, 0));
  for (int f = 0; f < 6 && !rc; ++f) {
    dev[f] = c->dtype == CSPT_F64 ? (void*)staging<double>(c, f) : (void*)staging<float>(c, f);
    rc = cuda_call(c, cudaMemcpyAsync(dev[f], in[f], bytes, cudaMemcpyHostToDevice, c->h2d_stream));
  }
  if (!rc) rc = cuda_call(c, cudaEventRecord(c->ev_in_ready, c->h2d_stream));
  if (!rc) rc = cuda_call(c, cudaStreamWaitEvent(c->stream, c->ev_in_ready, 0));
  if (rc) return rc;
  return DISPATCH(c, set_state_t)(c, dev[0], dev[1], dev[2], dev[3], dev[4], dev[5]);
}

int cspt_compute_dt(cspt_ctx* c, double cfl, double* dt_host_out) {
  if (!c || !dt_host_out || !(cfl > 0) || !isfinite(cfl)) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, compute_dt_t)(c, cfl, dt_host_out);
}

int cspt_set_kernel(cspt_ctx* c, int kernel) {
  if (!c || (kernel != CSPT_KERNEL_CUBIC_SPLINE && kernel != CSPT_KERNEL_POLY5)) return CSPT_EINVAL;
  if (kernel != c->kernel) { c->has_state = false; drop_graphs(c); }     // f = -D[psi] was formed with the other lattice weights
  c->kernel = kernel;
  return CSPT_OK;
}

int cspt_set_limiter(cspt_ctx* c, int limiter) {
  if (!c || (limiter != CSPT_LIMITER_MINMOD && limiter != CSPT_LIMITER_VANLEER)) return CSPT_EINVAL;
  if (limiter != c->limiter) drop_graphs(c);
  c->limiter = limiter;
  return CSPT_OK;
}

int cspt_set_riemann(cspt_ctx* c, int riemann) {
  if (!c || (riemann != CSPT_RIEMANN_HLL && riemann != CSPT_RIEMANN_LF && riemann != CSPT_RIEMANN_HLLC)) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  // the LF and HLLC fluxes need both states at a face: only the row layout of the Euler stage exchanges states, so a
  // ctx on the cell-per-thread layout (fp32 default) moves to the row layout (new tensor maps, host side only)
  if (riemann != CSPT_RIEMANN_HLL && c->euler_variant == 0) {
    c->euler_variant = 1;
    bool ok = c->dtype == CSPT_F64 ? euler_select<double>(c, nullptr, nullptr, nullptr)
                                   : euler_select<float>(c, nullptr, nullptr, nullptr);
    if (!ok) { (void)cudaGetLastError(); c->cuda_error = (int)cudaErrorUnknown; return CSPT_ECUDA; }
  }
  // back to HLL: back to the layout a fresh ctx runs HLL on (fp32: cell per thread, with the vacuum shortcuts), so
  // that results and speed do not depend on which solvers were selected before
  const int fresh = c->dtype == CSPT_F64 ? 1 : 0;
  if (riemann == CSPT_RIEMANN_HLL && c->euler_variant != fresh) {
    c->euler_variant = fresh;
    bool ok = c->dtype == CSPT_F64 ? euler_setup<double>(c) : euler_setup<float>(c);
    if (!ok) { (void)cudaGetLastError(); c->cuda_error = (int)cudaErrorUnknown; return CSPT_ECUDA; }
    drop_graphs(c);
  }
  if (riemann != c->riemann) drop_graphs(c);
  c->riemann = riemann;
  return CSPT_OK;
}

int cspt_debug_dead_ctas(cspt_ctx* c, long long* count) {
  if (!c || !count) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  *count = 0;
  if (!c->map_valid) return CSPT_OK;
  unsigned long long* hb = (unsigned long long*)c->h_pinned;
  int rc = cuda_call(c, cudaMemcpyAsync(hb, (unsigned char*)c->ws + c->off_map, 8, cudaMemcpyDeviceToHost, c->stream));
  if (!rc) rc = cuda_call(c, cudaStreamSynchronize(c->stream));
  if (!rc) *count = (long long)*hb;
  return rc;
}

int cspt_debug_tile_skip(cspt_ctx* c, int on) {
  if (!c || (on != 0 && on != 1)) return CSPT_EINVAL;
  if (on != c->tile_skip) { drop_graphs(c); c->map_valid = false; }
  c->tile_skip = on;
  return CSPT_OK;
}

int cspt_debug_force_vacuum_variant(cspt_ctx* c, int force) {
  if (!c || force < -1 || force > 1) return CSPT_EINVAL;
  if (force != c->vac_forced) drop_graphs(c);
  c->vac_forced = force;
  return CSPT_OK;
}

int cspt_step(cspt_ctx* c, double dt) {
  if (!c || !(dt > 0) || !isfinite(dt)) return CSPT_EINVAL;
  if (!c->has_state || has_external(c)) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, step_t)(c, dt);
}

int cspt_step_cfl(cspt_ctx* c, double cfl, double* dt_host_out) {
  if (!c || !(cfl > 0) || !isfinite(cfl)) return CSPT_EINVAL;
  if (!c->has_state || has_external(c)) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, step_cfl_t)(c, cfl, dt_host_out);
}

int cspt_run_cfl(cspt_ctx* c, double cfl, int nsteps, double* t_host_out) {
  if (!c || !(cfl > 0) || !isfinite(cfl) || nsteps < 0) return CSPT_EINVAL;
  if (!c->has_state || has_external(c)) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, run_cfl_t)(c, cfl, nsteps, t_host_out);
}

// ---- z-slab decomposition ------------------------------------------
int cspt_halo_elems(const cspt_ctx* c, int what, long long* elems) {
  if (!c || !elems || (what != CSPT_HALO_U && what != CSPT_HALO_PSI)) return CSPT_EINVAL;
  *elems = (long long)(what == CSPT_HALO_U ? 5 : 1) * NG * c->L.px * c->L.py;
  return CSPT_OK;
}

int cspt_halo_get(cspt_ctx* c, int face, int what, void* buf) {
  if (!c || !buf || (face != 4 && face != 5) || (what != CSPT_HALO_U && what != CSPT_HALO_PSI)) return CSPT_EINVAL;
  if (c->L.nz < NG) return CSPT_EINVAL;
  if (what == CSPT_HALO_U ? !c->has_state : !c->force_pending) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return c->dtype == CSPT_F64 ? halo_copy_t<double>(c, face, what, buf, false) : halo_copy_t<float>(c, face, what, buf, false);
}

int cspt_halo_put(cspt_ctx* c, int face, int what, const void* buf) {
  if (!c || !buf || (face != 4 && face != 5) || (what != CSPT_HALO_U && what != CSPT_HALO_PSI)) return CSPT_EINVAL;
  if (c->bc[face] != CSPT_BC_EXTERNAL) return CSPT_EINVAL;
  if (what == CSPT_HALO_U ? !c->has_state : !c->force_pending) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  int rc = c->dtype == CSPT_F64 ? halo_copy_t<double>(c, face, what, (void*)buf, true)
                                : halo_copy_t<float>(c, face, what, (void*)buf, true);
  if (!rc && what == CSPT_HALO_U) c->halo_current[face - 4] = true;
  return rc;
}

int cspt_finish_state(cspt_ctx* c) {
  if (!c) return CSPT_EINVAL;
  if (!c->force_pending) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, finish_state_t)(c);
}

int cspt_fill_ghosts(cspt_ctx* c) {
  if (!c) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, fill_ghosts_t)(c);
}

int cspt_step_filled(cspt_ctx* c, double dt) {
  if (!c || !(dt > 0) || !isfinite(dt)) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  // the step reads the ghost layers as they are: refuse layers that belong to an earlier state
  if (!c->ghosts_current) return CSPT_ESTATE;
  for (int f = 4; f < 6; ++f)
    if (c->bc[f] == CSPT_BC_EXTERNAL && !c->halo_current[f - 4]) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, step_filled_t)(c, dt);
}

int cspt_smax_device(cspt_ctx* c, void** device_ptr) {
  if (!c || !device_ptr) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, smax_device_t)(c, device_ptr);
}

int cspt_step_filled_cfl(cspt_ctx* c, double cfl, double* dt_host_out) {
  if (!c || !(cfl > 0) || !isfinite(cfl)) return CSPT_EINVAL;
  if (!c->has_state || !c->smax_valid) return CSPT_ESTATE;      // cspt_smax_device first
  if (!c->ghosts_current) return CSPT_ESTATE;
  for (int f = 4; f < 6; ++f)
    if (c->bc[f] == CSPT_BC_EXTERNAL && !c->halo_current[f - 4]) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, step_filled_cfl_t)(c, cfl, dt_host_out);
}

int cspt_probe_fma_rate(cspt_ctx* c, int other_per_fma, double* fma_per_second) {
  if (!c || !fma_per_second) return CSPT_EINVAL;
  if (other_per_fma != -1 && other_per_fma != 0 && other_per_fma != 1 && other_per_fma != 2 && other_per_fma != 4 && other_per_fma != 8)
    return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, probe_fma_t)(c, other_per_fma, 0.0, fma_per_second);
}

int cspt_probe_fma_rate_ms(cspt_ctx* c, int other_per_fma, double min_ms, double* fma_per_second) {
  if (!c || !fma_per_second || !(min_ms >= 0) || !(min_ms <= 10000.0)) return CSPT_EINVAL;
  if (other_per_fma != -1 && other_per_fma != 0 && other_per_fma != 1 && other_per_fma != 2 && other_per_fma != 4 && other_per_fma != 8)
    return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, probe_fma_t)(c, other_per_fma, min_ms, fma_per_second);
}

int cspt_sm_count(const cspt_ctx* c) { return c ? c->sm_count : 0; }

int cspt_get_state(cspt_ctx* c, void* rho, void* u, void* v, void* w, void* p) {
  if (!c || !rho || !u || !v || !w || !p) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, get_state_t)(c, rho, u, v, w, p, nullptr);
}

int cspt_get_conserved(cspt_ctx* c, void* rho, void* mx, void* my, void* mz, void* E) {
  if (!c || !rho || !mx || !my || !mz || !E) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  void* out[5] = {rho, mx, my, mz, E};
  return DISPATCH(c, get_conserved_t)(c, out);
}

int cspt_get_conserved_host(cspt_ctx* c, void* rho, void* mx, void* my, void* mz, void* E) {
  if (!c || !rho || !mx || !my || !mz || !E) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  void* host[5] = {rho, mx, my, mz, E};
  void* dev[5];
  c->zero_fill_steps = 2;          // the staging arrays overwrite intermediate slots that dead CTAs rely on
  for (int f = 0; f < 5; ++f) dev[f] = c->dtype == CSPT_F64 ? (void*)staging<double>(c, f) : (void*)staging<float>(c, f);
  int rc = DISPATCH(c, get_conserved_t)(c, dev);
  if (rc) return rc;
  size_t bytes = (size_t)c->L.nx * c->L.ny * c->L.nz * c->elem;
  for (int f = 0; f < 5; ++f) {
    rc = cuda_call(c, cudaMemcpyAsync(host[f], dev[f], bytes, cudaMemcpyDeviceToHost, c->stream));
    if (rc) return rc;
  }
  return cuda_call(c, cudaStreamSynchronize(c->stream));
}

int cspt_get_conserved_host_async(cspt_ctx* c, void* rho, void* mx, void* my, void* mz, void* E) {
  if (!c || !rho || !mx || !my || !mz || !E) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  if (!ensure_copy_streams(c)) return CSPT_ECUDA;
  wait_pending_output(c);                     // an earlier result still leaving through the same staging slots
  void* host[5] = {rho, mx, my, mz, E};
  void* dev[5];
  c->zero_fill_steps = 2;          // the staging arrays overwrite intermediate slots that dead CTAs rely on
  for (int f = 0; f < 5; ++f) dev[f] = c->dtype == CSPT_F64 ? (void*)staging_out<double>(c, f) : (void*)staging_out<float>(c, f);
  int rc = DISPATCH(c, get_conserved_t)(c, dev);
  if (rc) return rc;
  rc = cuda_call(c, cudaEventRecord(c->ev_out_ready, c->stream));
  if (!rc) rc = cuda_call(c, cudaStreamWaitEvent(c->d2h_stream, c->ev_out_ready, 0));
  size_t bytes = (size_t)c->L.nx * c->L.ny * c->L.nz * c->elem;
  for (int f = 0; f < 5 && !rc; ++f)
    rc = cuda_call(c, cudaMemcpyAsync(host[f], dev[f], bytes, cudaMemcpyDeviceToHost, c->d2h_stream));
  if (!rc) rc = cuda_call(c, cudaEventRecord(c->ev_out_done, c->d2h_stream));
  c->out_pending = true;
  return rc;
}

int cspt_set_conserved(cspt_ctx* c, const void* rho, const void* mx, const void* my, const void* mz, const void* E) {
  if (!c || !rho || !mx || !my || !mz || !E) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  const void* in[5] = {rho, mx, my, mz, E};
  return DISPATCH(c, set_conserved_t)(c, in);
}

int cspt_get_vacuum_mask(cspt_ctx* c, unsigned char* mask) {
  if (!c || !mask) return CSPT_EINVAL;
  if (!c->has_state) return CSPT_ESTATE;
  if (c->cuda_error) return CSPT_ECUDA;
  return DISPATCH(c, get_state_t)(c, nullptr, nullptr, nullptr, nullptr, nullptr, mask);
}

long long cspt_launch_count(const cspt_ctx* c) { return c ? c->launches : 0; }

int cspt_cuda_error(const cspt_ctx* c) { return c ? c->cuda_error : 0; }

int cspt_sync(cspt_ctx* c) {
  if (!c) return CSPT_EINVAL;
  if (c->cuda_error) return CSPT_ECUDA;
  int rc = cuda_call(c, cudaStreamSynchronize(c->stream));
  if (!rc && c->h2d_stream) rc = cuda_call(c, cudaStreamSynchronize(c->h2d_stream));
  if (!rc && c->d2h_stream) rc = cuda_call(c, cudaStreamSynchronize(c->d2h_stream));
  return rc;
}

const char* cspt_strerror(int code) {
  switch (code) {
    case CSPT_OK: return "ok";
    case CSPT_EINVAL: return "invalid argument";
    case CSPT_ENOMEM: return "out of host memory";
    case CSPT_ECUDA: return "CUDA error (sticky until destroy)";
    case CSPT_ESTATE: return "no state set";
    case CSPT_ELIMIT: return "size beyond the fixed capacity of the built-in scratch (cspt_cfl_dt_noalloc)";
    default: return "unknown status";
  }
}

}  // extern "C"
