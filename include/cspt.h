/* cspt.h -- C ABI of the B200-native CSPH-TVD time step.
 *
 * One explicit CSPH-TVD step (Khrapov, Khoperskov & Khoperskov 2019; PAPER.md
 * section 2.2, Eq. (4)-(8)) on a uniform 3-D Cartesian grid for the ideal-gas
 * Euler equations with an external potential psi (Eq. (1)-(3)):
 * Lagrangian SPH-style predictor/corrector (Eq. (5)-(7)), Eulerian TVD stage
 * (Eq. (8), (4)), CFL time step, boundary and gas-vacuum handling.  The readings
 * of everything the paper leaves open are listed in DESIGN.md section 3.
 *
 * Conventions
 *  - Every function returns an int status (CSPT_OK = 0, negative = error) unless
 *    stated otherwise; nothing throws, aborts or prints.
 *  - Arrays are dense, x fastest: element (i,j,k) at [ (k*ny + j)*nx + i ],
 *    nx*ny*nz elements of the ctx's dtype (double for CSPT_F64, float for
 *    CSPT_F32).  "device" pointers are CUDA device memory of the current
 *    device, "host" pointers are ordinary (preferably pinned) host memory.
 *  - Ownership: the caller owns every buffer it passes.  Inputs are copied,
 *    outputs are written, the workspace is borrowed from cspt_create until
 *    cspt_destroy.  The library owns only the small host-side ctx.
 *  - All work is enqueued on the CUDA stream given to cspt_create; only the
 *    functions marked "syncs" wait for it.
 *  - There is no CPU fallback: without a CUDA device every call that needs one
 *    returns CSPT_ECUDA.
 */
#ifndef CSPT_H
#define CSPT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cspt_ctx cspt_ctx; /* opaque */

enum { CSPT_F64 = 0, CSPT_F32 = 1 };
/* boundary kind per face, order xlo,xhi,ylo,yhi,zlo,zhi (reading G16) */
enum { CSPT_BC_PERIODIC = 0, CSPT_BC_OUTFLOW = 1, CSPT_BC_INFLOW = 2,
       /* z faces only: the face borders another z slab of the same grid (multi-GPU decomposition);
        * its ghost planes are not filled by a boundary rule but written by cspt_halo_put */
       CSPT_BC_EXTERNAL = 3 };
/* what a z-slab halo message carries: the five conserved fields of the current state, or the potential psi */
enum { CSPT_HALO_U = 0, CSPT_HALO_PSI = 1 };
/* TVD slope limiter of Eq. (8): minmod is the default (reading G12) */
enum { CSPT_LIMITER_MINMOD = 0, CSPT_LIMITER_VANLEER = 1 };
/* approximate Riemann solver of the Euler stage: HLL is the default (readings G13, G13b, G13c) */
enum { CSPT_RIEMANN_HLL = 0, CSPT_RIEMANN_LF = 1, CSPT_RIEMANN_HLLC = 2 };
/* smoothing kernel W of Eq. (7) (PAPER.md:68 leaves it open, :133): the cubic spline is the default (reading G5) */
enum { CSPT_KERNEL_CUBIC_SPLINE = 0, CSPT_KERNEL_POLY5 = 1 };
enum { CSPT_OK = 0, CSPT_EINVAL = -1, CSPT_ENOMEM = -2, CSPT_ECUDA = -3, CSPT_ESTATE = -4,
       CSPT_ELIMIT = -5 /* a size beyond the fixed capacity of cspt_cfl_dt_noalloc's built-in scratch */ };

/* Bytes of device workspace cspt_create needs for this grid (0 if the arguments
 * are invalid).  The caller allocates it (256-byte aligned), e.g. with torch. */
size_t cspt_workspace_bytes(int nx, int ny, int nz, int dtype);

/* Creates a solver for an nx*ny*nz grid of step h, adiabatic
 * index gamma and the six boundary kinds.  workspace: device
 * memory of at least cspt_workspace_bytes(); cuda_stream: a cudaStream_t
 * (NULL = default stream).
 * EINVAL: null out/bc/workspace, n < 1, n < 4 on a non-periodic axis, h <= 0,
 * gamma <= 1, one face of an axis periodic and the other not, unknown dtype or
 * boundary kind, CSPT_BC_EXTERNAL on an x or y face, workspace too small or misaligned.  In CSPT_F32 mode h, gamma,
 * cfl and dt are rounded to float once at the API. */
int cspt_create(cspt_ctx** out, int nx, int ny, int nz, double h, double gamma, const int bc[6],
                int dtype, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Sets the state from primitives rho,u,v,w,p and the potential psi:
 * U = (rho, rho u, E = p/(gamma-1) + rho |u|^2/2), f = -grad psi
 * by the lattice SPH operator (reading G6), INFLOW faces capture their boundary
 * layer (reading G16).  Device pointers; copied in; asynchronous. */
int cspt_set_state(cspt_ctx*, const void* rho, const void* u, const void* v, const void* w,
                   const void* p, const void* psi);
/* Same, from HOST buffers (copied through the stream; syncs). */
int cspt_set_state_host(cspt_ctx*, const void* rho, const void* u, const void* v, const void* w,
                        const void* p, const void* psi);
/* The same without the final wait: the six copies run on a copy stream of the ctx, the kernels follow on the ctx's
 * stream.  The host arrays (pinned, else the copies are not asynchronous) must stay untouched until cspt_sync.  With
 * cspt_get_conserved_host_async this lets the result of one state leave while the next state arrives (both
 * directions of the host link at once).  Does not sync. */
int cspt_set_state_host_async(cspt_ctx*, const void* rho, const void* u, const void* v, const void* w,
                              const void* p, const void* psi);

/* CFL time step (paper silent; reading G15): dt = cfl*h / max_cells(c + max(|u|,|v|,|w|)),
 * c = sqrt(gamma p / rho), vacuum cells skipped; +inf if every cell is vacuum.
 * Bit-exact and order independent (warp-shuffle + block max + integer atomic max
 * of the IEEE bit pattern).  Writes *dt_host_out; syncs.  EINVAL: cfl <= 0. */
int cspt_compute_dt(cspt_ctx*, double cfl, double* dt_host_out);

/* Chooses the smoothing kernel W of the SPH sums of Eq. (7) ("different smoothing kernels can be
 * used"): CSPT_KERNEL_CUBIC_SPLINE (default; Monaghan M4 with smoothing length h) or
 * CSPT_KERNEL_POLY5, W ~ (1 - q^2/4)^5 on q = r/h < 2, whose -W'(q)/q ~ (1 - q^2/4)^4 needs no square root.
 * Both are normalised on the lattice so that the undisplaced operator is exact for linear fields (G5).
 * The external force f = -D[psi] depends on the kernel's lattice weights, so a CHANGE of kernel discards the
 * state: call it before cspt_set_state.  Host-side only.  EINVAL: null ctx or unknown kernel. */
int cspt_set_kernel(cspt_ctx*, int kernel);

/* Chooses the slope limiter Theta of the piecewise-linear reconstruction, Eq. (8) ("the slope
 * ... should satisfy the TVD-condition"; "different TVD-limiters"): CSPT_LIMITER_MINMOD (default)
 * or CSPT_LIMITER_VANLEER (2ab/(a+b) where the one-sided differences a, b agree in sign, else 0).  Takes effect
 * from the next step.  Host-side only, no device work.  EINVAL: null ctx or unknown limiter. */
int cspt_set_limiter(cspt_ctx*, int limiter);

/* Chooses the approximate Riemann solver that gives the face fluxes F, G, H of Eq. (4) at t_{n+1/2} (PAPER.md:70-72:
 * "the approximate methods of Lax-Friedrichs (LF), Harten-Lax-van Lier (HLL), and the modified Harten-Lax-van Lier
 * method (HLLC)").  The flux vectors of Eq. (4) are advective (the pressure acts in the Lagrangian stage), so the
 * signal speeds are the face velocities u^L, u^R of the states of Eq. (8):
 *   CSPT_RIEMANN_HLL  (default) S_L = min, S_R = max of (u^L,u^R):  F = max(u^L,0) U^L + min(u^R,0) U^R;
 *   CSPT_RIEMANN_LF   local Lax-Friedrichs, F = (u^L U^L + u^R U^R)/2 - max(|u^L|,|u^R|) (U^R - U^L)/2;
 *   CSPT_RIEMANN_HLLC contact speed S* = (rho^L u^L + rho^R u^R)/(rho^L + rho^R) between converging streams, star
 *                     state of Toro's HLLC with p = 0; equal to HLL at every other face.
 * Takes effect from the next step.  Host-side only (LF / HLLC move a CSPT_F32 ctx to the kernel layout that
 * exchanges face states; selecting HLL again moves it back, so a ctx set to HLL always runs the same kernels whatever
 * was selected before).  EINVAL: null ctx or unknown solver. */
int cspt_set_riemann(cspt_ctx*, int riemann);

/* One full step U^n -> U^{n+1} with time step dt (Eq. (4)-(8)): ghost fill,
 * HFC/SUL predictor, HFC/SUL corrector, FGC, SUE.
 * Asynchronous.  EINVAL: dt <= 0 or not finite.  ESTATE: no state set. */
int cspt_step(cspt_ctx*, double dt);

/* compute_dt followed by step with that dt, the time step staying on the
 * device (no host sync).  dt_host_out may be NULL; if not, it is written and
 * the call syncs.  A grid that is all vacuum (dt = +inf) is left unchanged. */
int cspt_step_cfl(cspt_ctx*, double cfl, double* dt_host_out);

/* nsteps steps of cspt_step_cfl, the launches of two consecutive steps replayed from a CUDA
 * graph so that small grids are not bound by launch latency; bit-identical to a loop of cspt_step_cfl.  The time
 * steps stay on the device; their sum since cspt_set_state is kept there too and, if t_host_out is not NULL, copied
 * to *t_host_out (then the call syncs).  nsteps = 0 only reads the time.  With cspt_profile_enable on, the steps
 * are launched one by one (event pairs cannot be recorded inside a graph).  EINVAL: cfl <= 0, nsteps < 0. */
int cspt_run_cfl(cspt_ctx*, double cfl, int nsteps, double* t_host_out);

/* Primitives rho,u,v,w,p of the current state (vacuum cells: u = v = w = p = 0).
 * Device pointers; asynchronous. */
int cspt_get_state(cspt_ctx*, void* rho, void* u, void* v, void* w, void* p);
/* Conserved variables rho, rho u, rho v, rho w, E (parity is checked on these). */
int cspt_get_conserved(cspt_ctx*, void* rho, void* mx, void* my, void* mz, void* E);
/* Same, into HOST buffers (syncs). */
int cspt_get_conserved_host(cspt_ctx*, void* rho, void* mx, void* my, void* mz, void* E);
/* The same without the final wait: the five fields are staged on the device and copied out on a second copy stream;
 * the host arrays hold the result after cspt_sync (which waits for the ctx's stream and both copy streams).  A later
 * step waits by itself until the staged result has left.  Does not sync. */
int cspt_get_conserved_host_async(cspt_ctx*, void* rho, void* mx, void* my, void* mz, void* E);
/* Overwrites the conserved variables, keeping psi/f and the captured inflow layers
 * (checkpoint restore).  Device pointers. */
int cspt_set_conserved(cspt_ctx*, const void* rho, const void* mx, const void* my, const void* mz,
                       const void* E);
/* mask[i] = 1 where rho <= rho_vac = 1e-12 (reading G9), else 0.  Device pointer. */
int cspt_get_vacuum_mask(cspt_ctx*, unsigned char* mask);

/* ---- DIAGNOSTICS (measurement aids of bench.py and the tests; not part of the method) --------------------------- */
/* Number of kernel launches issued by this ctx so far (for bench.py's gpu_launches). */
long long cspt_launch_count(const cspt_ctx*);
/* Per-kernel device timing.  While enabled, every kernel the ctx launches is bracketed
 * by a CUDA event pair on the ctx's stream (up to 8192 launches since the last enable;
 * later ones are not recorded).  on != 0 resets the record.  cspt_profile_read sums the
 * device time and counts the launches of kernel `kid` (0 <= kid < cspt_profile_kernel_count(),
 * named by cspt_profile_kernel_name); it syncs.  Used by bench.py for the roofline figure. */
int cspt_profile_enable(cspt_ctx*, int on);
int cspt_profile_kernel_count(void);
const char* cspt_profile_kernel_name(int kid);
int cspt_profile_read(cspt_ctx*, int kid, double* total_ms, long long* launches);
/* Roofline probe: runs a kernel of independent FMAs in the ctx's precision on every SM and
 * writes the measured rate, thread-level FMAs per second, to *fma_per_second (the denominator of bench.py's "alu"
 * roofline, taken on the same box under the same clocks as the timed steps).  other_per_fma = 0: FMAs only;
 * 1, 2, 4 or 8: that many independent integer instructions behind every FMA, which shows how the FMAs share the
 * issue port with everything else (an FP64 FMA holds its pipe for two cycles, one other instruction issues in its
 * shadow, every further one costs about one issue cycle: DESIGN.md section 7).  Uses workspace that is dead between
 * steps: call it between steps only.  Syncs.  other_per_fma = -1: FMAs with three DISTINCT register operands
 * (x = y * z + x): in fp64 each is a register pair and the register file delivers two pairs per cycle, so these issue
 * every 3 cycles.  EINVAL: other_per_fma not one of -1, 0, 1, 2, 4, 8. */
int cspt_probe_fma_rate(cspt_ctx*, int other_per_fma, double* fma_per_second);
/* The same probe (one launch lasts about 3 ms), repeated back to back until the timed region lasts at least min_ms
 * (0 <= min_ms <= 10000): long enough for the GPU to settle into the power state a long step runs in and for an NVML
 * clock sampler to see it, so that the rate can be quoted per clock.  The launch fills every SM the device has
 * (cspt_sm_count) on any grid size.  EINVAL as above, or min_ms out of range. */
int cspt_probe_fma_rate_ms(cspt_ctx*, int other_per_fma, double min_ms, double* fma_per_second);
/* Multiprocessors of the device the ctx was created on (0 for a null ctx). */
int cspt_sm_count(const cspt_ctx*);
/* The fp32 Euler stage exists with and without its gas-vacuum shortcuts; a hint from cspt_set_state picks one, and both
 * give the same bits.  force = 0 / 1 pins the variant without / with the shortcuts (the test of that equality),
 * -1 follows the hint again.  Host-side only.  EINVAL: null ctx, force not in {-1, 0, 1}. */
int cspt_debug_force_vacuum_variant(cspt_ctx*, int force);
/* CTA-level gas-vacuum shortcut of the fp32 kernels: a CTA whose inputs within the 3-cell reach
 * of a step are all exactly 0, according to a device-resident map of bricks that have held gas, writes its exactly-zero
 * results and returns before its first load.  on = 0 switches it off (the test of bit equality with the full
 * evaluation), 1 (default) on.  Host-side only.  EINVAL: null ctx, on not 0 or 1. */
int cspt_debug_tile_skip(cspt_ctx*, int on);
/* CTAs that took that early return since the map was last rebuilt (cspt_set_state, cspt_set_conserved, a switch of
 * variant), 0 if no map is in use.  Syncs. */
int cspt_debug_dead_ctas(cspt_ctx*, long long* count);
/* ---- end of diagnostics ------------------------------------------------------------------------------------------ */
/* ---- z-slab decomposition over several GPUs ("the computational domain is divided between GPUs",
 * :123).  One ctx per slab of nz_local planes; a z face that borders another slab has
 * kind CSPT_BC_EXTERNAL.  The dependence of one step reaches 3 cells (reading G16), and every intermediate
 * field is evaluated on the extended domain from the ghost layers of U^n, so ONE exchange of the 3 ghost planes of the 5
 * conserved fields per face and step (plus psi once per cspt_set_state, and one scalar min-reduction of the time step)
 * makes the slabs advance exactly as the undivided grid does.  Protocol per step, the transport between the two
 * calls being the caller's (NCCL send/recv, a peer copy, ...):
 *     cspt_fill_ghosts;  cspt_halo_get(face) -> neighbour's cspt_halo_put(opposite face);  dt = min over slabs of
 *     cspt_compute_dt;  cspt_step_filled(dt)
 * and after cspt_set_state (which on such a ctx pads psi and stops):  cspt_halo_get/put(CSPT_HALO_PSI);
 * cspt_finish_state.  cspt_step, cspt_step_cfl and cspt_run_cfl return ESTATE on a ctx with an EXTERNAL face.
 *
 * cspt_halo_elems: elements of one halo message: (5 | 1) fields x 3 planes x the xy-PADDED plane (the x and y ghost
 *   layers travel with the plane: the z fill of reading G16 runs over the xy-padded array).
 * cspt_halo_get: copies the 3 interior planes next to z face `face` (4: z-lo, 5: z-hi), field by field, plane index
 *   ascending, into the device buffer buf.  CSPT_HALO_U: call after cspt_fill_ghosts (x and y ghosts must be current);
 *   CSPT_HALO_PSI: between cspt_set_state and cspt_finish_state.  EINVAL: face not 4 or 5, nz < 3.
 * cspt_halo_put: writes such a message into the 3 ghost planes of `face`, which must be EXTERNAL (else EINVAL).
 * cspt_finish_state: forms f = -D[psi] (S2) once the psi ghost planes are in place; ESTATE if no cspt_set_state is
 *   pending.  cspt_fill_ghosts: S0 on every face that is not EXTERNAL.  cspt_step_filled: S1..S9 with the given dt on a
 *   state whose ghost layers are complete: ESTATE unless, since the state last changed (a step, cspt_set_state,
 *   cspt_set_conserved), cspt_fill_ghosts has run and every EXTERNAL face has received its cspt_halo_put(CSPT_HALO_U).
 *   All enqueue on the ctx's stream and do not sync. */
int cspt_halo_elems(const cspt_ctx*, int what, long long* elems);
int cspt_halo_get(cspt_ctx*, int face, int what, void* device_buf);
int cspt_halo_put(cspt_ctx*, int face, int what, const void* device_buf);
int cspt_finish_state(cspt_ctx*);
int cspt_fill_ghosts(cspt_ctx*);
int cspt_step_filled(cspt_ctx*, double dt);
/* The same protocol without the host in the time-step reduction (no sync per step):
 *     cspt_fill_ghosts;  halo exchange;  cspt_smax_device -> max-reduce that word over the slabs IN PLACE on the
 *     ctx's stream (e.g. ncclAllReduce, ncclMax);  cspt_step_filled_cfl(cfl)
 * cspt_smax_device: evaluates the maximum signal speed max_cells(c + max(|u|,|v|,|w|)) of this slab (reading G15) if
 *   it is not already known from the last step's Euler stage, and returns the DEVICE address of the word that holds it:
 *   one element of the ctx's dtype (double / float), non-negative, 0 for an all-vacuum slab, valid once the ctx's
 *   stream reaches this point.  The maximum over the slabs, written back to the same word, is what the undivided grid
 *   would hold: non-negative IEEE numbers order like their bit patterns, so a floating-point max-reduction is exact.
 *   The word lives in the ctx's workspace; it is consumed (reset) by the next step.
 * cspt_step_filled_cfl: dt = (cfl*h)/that word (+inf -> identity step), then S1..S9 as cspt_step_filled.
 *   dt_host_out may be NULL; if not, dt is written there and the call syncs.  ESTATE: as cspt_step_filled, or
 *   cspt_smax_device was not called for the current state.  EINVAL: cfl <= 0 or not finite. */
int cspt_smax_device(cspt_ctx*, void** device_ptr);
int cspt_step_filled_cfl(cspt_ctx*, double cfl, double* dt_host_out);
/* ---- CFL time step without a ctx, a workspace or any allocation ------------------------------------------------
 * For callers that cannot allocate device memory.  cspt_compute_dt needs a ctx, and a ctx needs a workspace of 28
 * padded fields that someone must allocate.  That is impossible for a host code that gave all of HBM to its own arena
 * at start-up, unwelcome inside a time loop (cudaMalloc / cudaFree stall the whole device), and not an option for an
 * in-situ monitor or a coupled solver that is merely handed device pointers to the conserved fields and has to answer
 * with a common time step.  This call serves them: it computes the same CFL time step (reading G15; the paper is
 * silent) from five DENSE device arrays rho, rho u, rho v, rho w, E of ncells elements each (any order: the result
 * does not depend on it; no ghost cells), in the arithmetic of cspt_compute_dt, bit for bit:
 *     *dt_device_out = (cfl*h) / max_cells(c + max(|u|,|v|,|w|)),  c = sqrt(gamma p / rho),  cells with rho <= 1e-12
 *     skipped (reading G9);  +inf if ncells = 0 or every cell is vacuum.
 * dtype: CSPT_F64 (double arrays, double result) or CSPT_F32 (float arrays, float result; h, gamma, cfl rounded to
 * float once).  dt_device_out: ONE element of that type in device memory, the caller's.  cuda_stream: a cudaStream_t
 * of the current device (NULL = default stream).  Two kernels are enqueued on it; the call does not sync, and it calls
 * no cudaMalloc, cudaFree or other allocating routine.
 *
 * Its scratch (one maximum per 4096 cells) is a fixed array inside the library's device code: 65536 slots = 512 KiB
 * on every GPU that loads libcspt.so, held until the process exits.  Hence the limit
 *     ncells <= CSPT_NOALLOC_MAX_CELLS = 65536 * 4096 = 268 435 456   (512^3 fits, 1024^3 does not);
 * beyond it the call does nothing and returns CSPT_ELIMIT ("beyond the fixed capacity of the built-in scratch").
 * All calls on one device share that array, whatever their stream, and each finds the previous call's values in
 * it.  Nothing in it has to be zero at entry (each call reads back only the slots it has just written), but two calls
 * whose kernels may overlap on the GPU -- different streams without an event between them, or several host threads --
 * race on it and may both return a wrong time step: keep calls on one device ordered.
 * The FIRST call on each device looks up the device address of the array (cudaGetSymbolAddress, with that device
 * current) and keeps it; make that first call with the right device current and before any stream capture begins.
 * EINVAL: unknown dtype, ncells < 0, a null array with ncells > 0, null dt_device_out, h <= 0, gamma <= 1, cfl <= 0
 * or not finite.  ELIMIT: ncells too large (or a device ordinal >= 64).  ECUDA: the address lookup or a launch failed
 * (cudaGetLastError tells which error). */
#define CSPT_NOALLOC_MAX_CELLS 268435456LL
long long cspt_noalloc_max_cells(void);      /* the same number, for bindings that cannot read macros */
int cspt_cfl_dt_noalloc(int dtype, long long ncells, const void* rho, const void* mx, const void* my, const void* mz,
                        const void* E, double gamma, double h, double cfl, void* dt_device_out, void* cuda_stream);
/* The cudaError_t value behind a CSPT_ECUDA status of this ctx (0 if none). */
int cspt_cuda_error(const cspt_ctx*);
/* Waits for the ctx's stream and for the copy streams of the *_host_async calls. */
int cspt_sync(cspt_ctx*);
/* Frees the ctx, never the workspace.  NULL is allowed. */
void cspt_destroy(cspt_ctx*);
/* Static string for a status code. */
const char* cspt_strerror(int);

#ifdef __cplusplus
}
#endif
#endif /* CSPT_H */
