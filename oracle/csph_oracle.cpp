// csph_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU statement of one CSPH-TVD time step
// (Khrapov, Khoperskov & Khoperskov 2019, section 2.2, Eq. (4)-(8)),
// under the readings G1-G23 listed in DESIGN.md.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may load this.  It shares no code with the CUDA path
// (paper_1912_04855_b200/csrc) and neither includes the other.
//
// Every stage is a full-array pass over padded arrays (3 ghost layers per
// face), in the paper's order HFC{p} SUL{p} HFC{c} SUL{c} FGC SUE
// (PAPER.md:108-113).  No blocking, no fusion, no reordering.  The optional
// OpenMP pragma only splits the outermost (z) loop of a pass; every cell is
// still computed by exactly the same expression, so results are bit-identical
// for any thread count.
//
// Pins (tests/test_oracle_*.py): exact Riemann solution for Sod along x,y,z;
// uniform flow; Gamma=2 discrete hydrostatic equilibrium; conservation;
// axis permutation / mirror; advected-sine convergence; vacuum fan closed
// form; brute-force all-pairs evaluation of Eq. (7); closed-form lattice
// weights; free fall in a linear potential; the ghost rules of every boundary
// kind on non-uniform states, the pressure floor, the LF / HLL / HLLC face
// fluxes against the textbook solvers; second order for the linear transfer of
// a smooth wave on N = 400, 800, 1600 (reading G23 (i)); the
// ballistic particle offsets of Eq. (5), (6) in uniform free fall and the
// vacuum threshold of reading G9 (tests/test_oracle_round3_pins.py).
// Parity that stays UNPINNED: agreement with the authors' own code
// (kernel, limiter, Riemann solver, CFL rule and boundary rules are readings,
// DESIGN.md section 3), second order on a nonlinear simple wave (reading
// G23 (ii): measured first order) and the Fig. 1 shock position (parameters
// missing from the paper).
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.sh).
// -ffp-contract=off matters: the CFL time step and the vacuum mask are
// compared bit-for-bit with the GPU, so no FMA contraction may happen here.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

const int G = 3;  // ghost layers per face: one full step reaches +-3 cells

enum { BC_PERIODIC = 0, BC_OUTFLOW = 1, BC_INFLOW = 2 };

int g_threads = 1;

template <class T>
struct Oracle {
  int n[3];       // nx, ny, nz
  int p[3];       // padded sizes
  T h, gamma, rho_vac;
  int bc[6];      // xlo,xhi,ylo,yhi,zlo,zhi
  bool has_state;
  size_t ncell_pad;

  // U^n: rho, mx, my, mz, E.  psi: potential.
  std::vector<T> U[5], psi;
  // frozen ghost planes of INFLOW faces, captured at set_state (reading G16)
  std::vector<T> inflow[6][5];

  // work arrays, all padded
  std::vector<T> phi, vel[3], f[3];            // primitives of U^n, force
  std::vector<T> Q[4];                          // Eq. (7): momentum x3, energy
  std::vector<T> Us[5], phis, vels[3], xis[3];  // U*, phi*, u*, xi*
  std::vector<T> Ut[5], xi[3];                  // U~, xi^{n+1}
  std::vector<T> F[3][5];                       // face fluxes, face i+1/2 stored at i
  std::vector<T> Unew[5];

  // cubic-spline lattice constants (reading G5)
  T a_shell[4];  // a(|o|^2), |o|^2 = 1,2,3
  T S0p;

  size_t idx(int i, int j, int k) const {
    return ((size_t)(k + G) * p[1] + (size_t)(j + G)) * p[0] + (size_t)(i + G);
  }

  Oracle(int nx, int ny, int nz, double h_, double gamma_, const int* bc_) {
    n[0] = nx; n[1] = ny; n[2] = nz;
    for (int d = 0; d < 3; ++d) p[d] = n[d] + 2 * G;
    h = (T)h_; gamma = (T)gamma_; rho_vac = (T)1e-12;
    for (int q = 0; q < 6; ++q) bc[q] = bc_[q];
    has_state = false;
    ncell_pad = (size_t)p[0] * p[1] * p[2];
    auto A = [&](std::vector<T>& v) { v.assign(ncell_pad, (T)0); };
    for (int c = 0; c < 5; ++c) { A(U[c]); A(Us[c]); A(Ut[c]); A(Unew[c]); }
    A(psi); A(phi); A(phis);
    for (int d = 0; d < 3; ++d) {
      A(vel[d]); A(f[d]); A(vels[d]); A(xis[d]); A(xi[d]);
      for (int c = 0; c < 5; ++c) A(F[d][c]);
    }
    for (int c = 0; c < 4; ++c) A(Q[c]);
    set_kernel(0);
  }

  // Smoothing kernel W (PAPER.md:68 leaves it open; :133 "different smoothing kernels can be used"):
  //   kernel 0 (reading G5, the default): Monaghan cubic spline with smoothing length h,
  //       g^(q) = -W'(q)/q = 3 - 2.25 q (q < 1),  0.75 (2-q)^2 / q (1 <= q < 2),  0 (q >= 2)
  //   kernel 1: W ~ (1 - q^2/4)^5 on q < 2, for which -W'(q)/q ~ (1 - q^2/4)^4
  //       needs no square root (any constant factor cancels against S0')
  // S0' = sum over the 26 lattice neighbours of g^(|o|) o_x^2, so that the undisplaced operator
  // reproduces linear fields exactly (reading G5).
  int kernel = 0;
  static double ghat_d(int kernel, double q) {
    if (kernel == 1) { double t = 1.0 - 0.25 * q * q; return q < 2.0 ? (t * t) * (t * t) : 0.0; }
    if (q < 1.0) return 3.0 - 2.25 * q;
    if (q < 2.0) return 0.75 * (2.0 - q) * (2.0 - q) / q;
    return 0.0;
  }
  void set_kernel(int k) {
    kernel = k;
    double g1 = ghat_d(k, 1.0), g2 = ghat_d(k, std::sqrt(2.0)), g3 = ghat_d(k, std::sqrt(3.0));
    double S = 2.0 * g1 + 8.0 * g2 + 8.0 * g3;
    S0p = (T)S;
    a_shell[0] = 0; a_shell[1] = (T)(g1 / S); a_shell[2] = (T)(g2 / S); a_shell[3] = (T)(g3 / S);
    if (has_state) force();          // f = -D[psi] uses the lattice weights
  }

  // ---- O0: ghost cells, axis by axis (reading G16) ---------------------------
  // `freeze` = true at set_state: INFLOW faces are filled like OUTFLOW once and
  // their first ghost plane is captured; later calls copy the captured plane.
  void fill_axis_U(int d, bool freeze) {
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) {
      // axes already filled are traversed over their padded range
      lo[e] = (e < d) ? -G : 0;
      hi[e] = (e < d) ? n[e] + G : n[e];
    }
    int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    for (int side = 0; side < 2; ++side) {
      int kind = bc[2 * d + side];
      for (int c = 0; c < 5; ++c) {
        if (freeze && kind == BC_INFLOW) inflow[2 * d + side][c].assign(ncell_pad / p[d], (T)0);
        for (int a = lo[d2]; a < hi[d2]; ++a)
          for (int b = lo[d1]; b < hi[d1]; ++b)
            for (int g = 1; g <= G; ++g) {
              int q[3], s[3];
              q[d1] = b; q[d2] = a; s[d1] = b; s[d2] = a;
              q[d] = side ? n[d] - 1 + g : -g;
              if (kind == BC_PERIODIC) s[d] = side ? ((g - 1) % n[d]) : (n[d] - 1 - ((g - 1) % n[d]));
              else s[d] = side ? n[d] - 1 : 0;
              size_t plane_i = (size_t)(a + G) * p[d1] + (size_t)(b + G);
              T val;
              if (kind == BC_INFLOW && !freeze) val = inflow[2 * d + side][c][plane_i];
              else val = U[c][idx(s[0], s[1], s[2])];
              U[c][idx(q[0], q[1], q[2])] = val;
              if (kind == BC_INFLOW && freeze && g == 1) inflow[2 * d + side][c][plane_i] = val;
            }
      }
    }
  }
  void fill_ghosts_U(bool freeze) { for (int d = 0; d < 3; ++d) fill_axis_U(d, freeze); }

  // psi ghosts: periodic wrap, otherwise odd reflection about the boundary cell
  // (linear extrapolation of the force, reading G16).
  void fill_ghosts_psi() {
    for (int d = 0; d < 3; ++d) {
      int lo[3], hi[3];
      for (int e = 0; e < 3; ++e) { lo[e] = (e < d) ? -G : 0; hi[e] = (e < d) ? n[e] + G : n[e]; }
      int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
      for (int side = 0; side < 2; ++side) {
        int kind = bc[2 * d + side];
        for (int a = lo[d2]; a < hi[d2]; ++a)
          for (int b = lo[d1]; b < hi[d1]; ++b)
            for (int g = 1; g <= G; ++g) {
              int q[3], s[3], e0[3];
              q[d1] = b; q[d2] = a; s[d1] = b; s[d2] = a; e0[d1] = b; e0[d2] = a;
              q[d] = side ? n[d] - 1 + g : -g;
              T val;
              if (kind == BC_PERIODIC) {
                s[d] = side ? ((g - 1) % n[d]) : (n[d] - 1 - ((g - 1) % n[d]));
                val = psi[idx(s[0], s[1], s[2])];
              } else {
                e0[d] = side ? n[d] - 1 : 0;
                s[d] = side ? n[d] - 1 - g : g;
                if (s[d] < 0) s[d] = 0;
                if (s[d] > n[d] - 1) s[d] = n[d] - 1;
                val = (T)2 * psi[idx(e0[0], e0[1], e0[2])] - psi[idx(s[0], s[1], s[2])];
              }
              psi[idx(q[0], q[1], q[2])] = val;
            }
      }
    }
  }

  // ---- O1: primitives of one cell (readings G7, G9) --------
  struct Prim { T u, v, w, p, phi; bool ok; };
  Prim prim_cell(T rho, T mx, T my, T mz, T E) const {
    Prim q;
    q.ok = rho > rho_vac;
    T ir = q.ok ? (T)1 / rho : (T)0;
    q.u = mx * ir; q.v = my * ir; q.w = mz * ir;
    T ke2 = (mx * q.u + my * q.v) + mz * q.w;
    T pp = (gamma - (T)1) * (E - (T)0.5 * ke2);
    q.p = q.ok ? (pp > (T)0 ? pp : (T)0) : (T)0;
    q.phi = std::sqrt((T)2 * q.p);
    return q;
  }

  // primitives of a whole padded field set -> phi, velocity
  void primitives(const std::vector<T>* W, const std::vector<T>& rho, std::vector<T>& ph,
                  std::vector<T>* ve, int ext) {
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int k = -ext; k < n[2] + ext; ++k)
      for (int j = -ext; j < n[1] + ext; ++j)
        for (int i = -ext; i < n[0] + ext; ++i) {
          size_t c = idx(i, j, k);
          Prim q = prim_cell(rho[c], W[1][c], W[2][c], W[3][c], W[4][c]);
          ph[c] = q.phi; ve[0][c] = q.u; ve[1][c] = q.v; ve[2][c] = q.w;
        }
  }

  // ---- O2: external force f = -D[psi] on interior(+)2 (G6) --
  void force() {
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int k = -2; k < n[2] + 2; ++k)
      for (int j = -2; j < n[1] + 2; ++j)
        for (int i = -2; i < n[0] + 2; ++i) {
          T s[3] = {0, 0, 0};
          for (int oz = -1; oz <= 1; ++oz)
            for (int oy = -1; oy <= 1; ++oy)
              for (int ox = -1; ox <= 1; ++ox) {
                int o2 = ox * ox + oy * oy + oz * oz;
                if (o2 == 0) continue;
                T q = a_shell[o2] * psi[idx(i + ox, j + oy, k + oz)];
                s[0] += (T)ox * q; s[1] += (T)oy * q; s[2] += (T)oz * q;
              }
          size_t c = idx(i, j, k);
          for (int d = 0; d < 3; ++d) f[d][c] = -(s[d] / h);
        }
  }

  // kernel weight w(r) = g^(r/h) / (S0' h^2)   (reading G5)
  T kernel_w(T r) const {
    T q = r / h, g;
    if (kernel == 1) {
      T t = (T)1 - (T)0.25 * q * q;
      g = q < (T)2 ? (t * t) * (t * t) : (T)0;
    } else if (q < (T)1) g = (T)3 - (T)2.25 * q;
    else if (q < (T)2) g = (T)0.75 * ((T)2 - q) * ((T)2 - q) / q;
    else g = (T)0;
    return g / (S0p * h * h);
  }

  // ---- O3: Q(U, xi), Eq. (7) (readings G1-G6) -------------------
  // ph, ve: phi and velocity of the state; xs: particle offsets from the cell
  // centres (null = particles at the centres); ext: how far beyond
  // the interior Q is evaluated ("extended domain", G16).
  void eval_Q(const std::vector<T>& ph, const std::vector<T>* ve, const std::vector<T>* xs,
              const std::vector<T>& rho, int ext) {
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int k = -ext; k < n[2] + ext; ++k)
      for (int j = -ext; j < n[1] + ext; ++j)
        for (int i = -ext; i < n[0] + ext; ++i) {
          size_t ci = idx(i, j, k);
          T Sm[3] = {0, 0, 0}, SE = 0;
          T ui[3] = {ve[0][ci], ve[1][ci], ve[2][ci]};
          T xi_i[3] = {0, 0, 0};
          if (xs) for (int d = 0; d < 3; ++d) xi_i[d] = xs[d][ci];
          for (int oz = -1; oz <= 1; ++oz)
            for (int oy = -1; oy <= 1; ++oy)
              for (int ox = -1; ox <= 1; ++ox) {
                if (ox == 0 && oy == 0 && oz == 0) continue;  // self term: grad W(0) = 0 (G4)
                size_t cj = idx(i + ox, j + oy, k + oz);
                int o[3] = {ox, oy, oz};
                T dv[3], r2 = 0;
                for (int d = 0; d < 3; ++d) {
                  // d = r_i - r_j = (x_i + xi_i) - (x_i + o h + xi_j)
                  T xj = xs ? xs[d][cj] : (T)0;
                  dv[d] = -(T)o[d] * h + xi_i[d] - xj;
                  r2 += dv[d] * dv[d];
                }
                T w = kernel_w(std::sqrt(r2));
                T pw = ph[cj] * w;
                T ud = 0;
                for (int d = 0; d < 3; ++d) {
                  Sm[d] += pw * dv[d];
                  ud += (T)0.5 * (ui[d] + ve[d][cj]) * dv[d];
                }
                SE += pw * ud;
              }
          // sign of the force terms: reading G1 (Eq. (2),(3): -(grad p - rho f))
          T uf = 0;
          for (int d = 0; d < 3; ++d) {
            Q[d][ci] = ph[ci] * Sm[d] + rho[ci] * f[d][ci];
            uf += ui[d] * f[d][ci];
          }
          Q[3][ci] = ph[ci] * SE + rho[ci] * uf;
        }
  }

  // ---- one full step ---------------------------------------
  void step(T dt) {
    fill_ghosts_U(false);                              // O0
    primitives(U, U[0], phi, vel, G);                  // O1 on the whole padded array
    // O3+O4: predictor, Eq. (5), on interior(+)2; particles at the centres
    eval_Q(phi, vel, nullptr, U[0], 2);
    for_ext(2, [&](size_t c) {
      Us[0][c] = U[0][c];                              // mass row of Q is zero (G2)
      for (int q = 0; q < 4; ++q) Us[q + 1][c] = U[q + 1][c] + dt * Q[q][c];
    });
    primitives(Us, U[0], phis, vels, 2);
    for_ext(2, [&](size_t c) {
      for (int d = 0; d < 3; ++d) xis[d][c] = (T)0.5 * dt * (vel[d][c] + vels[d][c]);
    });
    // O5/O6: corrector, Eq. (6), on interior(+)1
    eval_Q(phis, vels, xis, U[0], 1);
    for_ext(1, [&](size_t c) {
      Ut[0][c] = U[0][c];
      for (int q = 0; q < 4; ++q)
        Ut[q + 1][c] = (T)0.5 * (U[q + 1][c] + Us[q + 1][c]) + (T)0.5 * dt * Q[q][c];
      Prim pt = prim_cell(Ut[0][c], Ut[1][c], Ut[2][c], Ut[3][c], Ut[4][c]);
      T ut[3] = {pt.u, pt.v, pt.w};
      for (int d = 0; d < 3; ++d)
        xi[d][c] = (T)0.5 * xis[d][c] + (T)0.25 * dt * (vel[d][c] + ut[d]);
    });
    fluxes();                                          // O7
    // O8: Eq. (4), unsplit (G14)
    T lam = dt / h;
    for_ext(0, [&](size_t c) {
      size_t sx = 1, sy = p[0], sz = (size_t)p[0] * p[1];
      for (int q = 0; q < 5; ++q)
        Unew[q][c] = Ut[q][c] - lam * (((F[0][q][c] - F[0][q][c - sx]) + (F[1][q][c] - F[1][q][c - sy])) +
                                       (F[2][q][c] - F[2][q][c - sz]));
    });
    for (int q = 0; q < 5; ++q) U[q].swap(Unew[q]);
  }

  template <class Fn>
  void for_ext(int ext, Fn fn) {
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int k = -ext; k < n[2] + ext; ++k)
      for (int j = -ext; j < n[1] + ext; ++j)
        for (int i = -ext; i < n[0] + ext; ++i) fn(idx(i, j, k));
  }

  static T minmod(T a, T b) {
    if (a > (T)0 && b > (T)0) return a < b ? a : b;
    if (a < (T)0 && b < (T)0) return a > b ? a : b;
    return (T)0;
  }
  // van Leer's harmonic-mean limiter: 2ab/(a+b) where a and b have the same sign, else 0.
  static T vanleer(T a, T b) {
    if (a * b > (T)0) return ((T)2 * a * b) / (a + b);
    return (T)0;
  }
  // TVD slope Theta (PAPER.md:78 "should satisfy the TVD-condition"; :133 "different TVD-limiters"):
  // limiter 0 = minmod (reading G12, the default), 1 = van Leer.
  int limiter = 0;
  T slope(T a, T b) const { return limiter == 1 ? vanleer(a, b) : minmod(a, b); }

  // ---- O7: FGC, Eq. (8) + Riemann flux at the faces (G10-G13) ----
  void fluxes() {
    for (int d = 0; d < 3; ++d) {
      size_t sd = d == 0 ? 1 : d == 1 ? (size_t)p[0] : (size_t)p[0] * p[1];
      int lo[3] = {0, 0, 0}, hi[3] = {n[0], n[1], n[2]};
      lo[d] = -1;  // face i+1/2 for i = -1 .. n-1
#pragma omp parallel for num_threads(g_threads) schedule(static)
      for (int k = lo[2]; k < hi[2]; ++k)
        for (int j = lo[1]; j < hi[1]; ++j)
          for (int i = lo[0]; i < hi[0]; ++i) {
            size_t cL = idx(i, j, k), cR = cL + sd;
            T UL[5], UR[5];
            for (int q = 0; q < 5; ++q) {
              // TVD slope from U^n (G12: limiter on conserved variables)
              T thL = slope((U[q][cL] - U[q][cL - sd]) / h, (U[q][cL + sd] - U[q][cL]) / h);
              T thR = slope((U[q][cR] - U[q][cR - sd]) / h, (U[q][cR + sd] - U[q][cR]) / h);
              // U^{n+1/2} = (U^n + U~)/2 (G10)
              T hL = (T)0.5 * (U[q][cL] + Ut[q][cL]);
              T hR = (T)0.5 * (U[q][cR] + Ut[q][cR]);
              UL[q] = hL + (T)0.5 * (h - xi[d][cL]) * thL;   // Eq. (8)
              UR[q] = hR - (T)0.5 * (h + xi[d][cR]) * thR;
            }
            T uL = UL[0] > rho_vac ? UL[1 + d] / UL[0] : (T)0;   // G9
            T uR = UR[0] > rho_vac ? UR[1 + d] / UR[0] : (T)0;
            T Ff[5];
            riemann_flux(d, UL, UR, uL, uR, Ff);
            for (int q = 0; q < 5; ++q) F[d][q][cL] = Ff[q];
          }
    }
  }

  // Approximate Riemann solver at a face ("the approximate methods of Lax-Friedrichs (LF),
  // Harten-Lax-van Lier (HLL), and the modified Harten-Lax-van Lier method (HLLC) [14]").  The flux vectors of
  // Eq. (4) are purely advective, F = u U (reading G3): the pressure acts in the Lagrangian stage, so
  // the Riemann problem of the Euler stage is the one of the pressureless system, whose only signal speeds are
  // the velocities themselves.  UL, UR: reconstructed states of Eq. (8); uL, uR: their normal velocities (G9).
  //   riemann 0 (reading G13, the default): HLL with S_L = min(uL,uR), S_R = max(uL,uR), which is
  //       F = max(uL,0) UL + min(uR,0) UR in all four sign cases;
  //   riemann 1 (reading G13b): local Lax-Friedrichs (Rusanov), F = (F_L + F_R)/2 - a (UR - UL)/2 with the largest
  //       local signal speed a = max(|uL|,|uR|) (a global a = h/dt would not vanish for gas at rest);
  //   riemann 2 (reading G13c): HLLC, Toro [14] section 10.4 with p = 0 and the wave speeds of riemann 0: contact speed
  //       S* = [rhoR uR (S_R-uR) - rhoL uL (S_L-uL)] / [rhoR (S_R-uR) - rhoL (S_L-uL)], star states
  //       U*_K = rho_K (S_K-u_K)/(S_K-S*) [1, S* (normal), v_K, w_K (tangential), E_K/rho_K + (S*-u_K) S*],
  //       F = F_L | F_L + S_L (U*_L - U_L) | F_R + S_R (U*_R - U_R) | F_R.  Between diverging streams the denominator
  //       vanishes (no mass in the star region) and the flux through the face is zero.
  int riemann = 0;
  void riemann_flux(int d, const T* UL, const T* UR, T uL, T uR, T* Ff) const {
    if (riemann == 1) {
      T a = std::fabs(uL) > std::fabs(uR) ? std::fabs(uL) : std::fabs(uR);
      for (int q = 0; q < 5; ++q)
        Ff[q] = (T)0.5 * (uL * UL[q] + uR * UR[q]) - (T)0.5 * a * (UR[q] - UL[q]);
      return;
    }
    if (riemann == 2) {
      T SL = uL < uR ? uL : uR, SR = uL < uR ? uR : uL;
      if (SL >= (T)0) { for (int q = 0; q < 5; ++q) Ff[q] = uL * UL[q]; return; }
      if (SR <= (T)0) { for (int q = 0; q < 5; ++q) Ff[q] = uR * UR[q]; return; }
      T den = UR[0] * (SR - uR) - UL[0] * (SL - uL);
      if (!(den > (T)0)) { for (int q = 0; q < 5; ++q) Ff[q] = (T)0; return; }
      T Ss = (UR[0] * uR * (SR - uR) - UL[0] * uL * (SL - uL)) / den;
      const T* UK = Ss >= (T)0 ? UL : UR;
      T uK = Ss >= (T)0 ? uL : uR, SK = Ss >= (T)0 ? SL : SR;
      T rs = UK[0] * (SK - uK) / (SK - Ss);
      T Us[5];
      Us[0] = rs;
      for (int q = 1; q < 4; ++q) Us[q] = rs * (UK[q] / UK[0]);
      Us[1 + d] = rs * Ss;
      Us[4] = rs * (UK[4] / UK[0] + (Ss - uK) * Ss);
      for (int q = 0; q < 5; ++q) Ff[q] = uK * UK[q] + SK * (Us[q] - UK[q]);
      return;
    }
    T up = uL > (T)0 ? uL : (T)0, um = uR < (T)0 ? uR : (T)0;
    for (int q = 0; q < 5; ++q) Ff[q] = up * UL[q] + um * UR[q];   // G13
  }

  // ---- O9: CFL time step (silent in the paper; reading G15) ------------------
  T cell_speed(size_t c) const {
    Prim q = prim_cell(U[0][c], U[1][c], U[2][c], U[3][c], U[4][c]);
    if (!q.ok) return (T)0;
    T cs = std::sqrt(gamma * q.p / U[0][c]);
    T a = std::fabs(q.u), b = std::fabs(q.v), cc = std::fabs(q.w);
    T m = a > b ? a : b; m = m > cc ? m : cc;
    return cs + m;
  }
  T compute_dt(T cfl) const {
    T smax = 0;
    for (int k = 0; k < n[2]; ++k)
      for (int j = 0; j < n[1]; ++j)
        for (int i = 0; i < n[0]; ++i) { T s = cell_speed(idx(i, j, k)); if (s > smax) smax = s; }
    if (!(smax > (T)0)) return std::numeric_limits<T>::infinity();
    return (cfl * h) / smax;
  }

  // ---- state in / out -------------------------------------------------------
  void set_state(const T* rho, const T* u, const T* v, const T* w, const T* pr, const T* ps) {
    size_t m = 0;
    for (int k = 0; k < n[2]; ++k)
      for (int j = 0; j < n[1]; ++j)
        for (int i = 0; i < n[0]; ++i, ++m) {
          size_t c = idx(i, j, k);
          U[0][c] = rho[m];
          U[1][c] = rho[m] * u[m]; U[2][c] = rho[m] * v[m]; U[3][c] = rho[m] * w[m];
          T ke = (u[m] * u[m] + v[m] * v[m]) + w[m] * w[m];
          U[4][c] = pr[m] / (gamma - (T)1) + ((T)0.5 * rho[m]) * ke;
          psi[c] = ps[m];
        }
    fill_ghosts_U(true);
    fill_ghosts_psi();
    force();
    has_state = true;
  }
  void get_field(const std::vector<T>& src, T* out) const {
    size_t m = 0;
    for (int k = 0; k < n[2]; ++k)
      for (int j = 0; j < n[1]; ++j)
        for (int i = 0; i < n[0]; ++i, ++m) out[m] = src[idx(i, j, k)];
  }
  void put_field(std::vector<T>& dst, const T* in) {
    size_t m = 0;
    for (int k = 0; k < n[2]; ++k)
      for (int j = 0; j < n[1]; ++j)
        for (int i = 0; i < n[0]; ++i, ++m) dst[idx(i, j, k)] = in[m];
  }
};

struct Handle { int dtype; void* o; };

}  // namespace

#define DISPATCH(hd, expr64, expr32)                                         \
  do {                                                                       \
    if ((hd)->dtype == 0) { auto* o = (Oracle<double>*)(hd)->o; typedef double T; (void)sizeof(T); expr64; } \
    else { auto* o = (Oracle<float>*)(hd)->o; typedef float T; (void)sizeof(T); expr32; }                     \
  } while (0)

extern "C" {

void orc_set_threads(int t) { g_threads = t < 1 ? 1 : t; }

void* orc_create(int nx, int ny, int nz, double h, double gamma, const int* bc, int dtype) {
  if (nx < 1 || ny < 1 || nz < 1 || !(h > 0) || !(gamma > 1) || !bc) return nullptr;
  Handle* hd = new Handle;
  hd->dtype = dtype;
  if (dtype == 0) hd->o = new Oracle<double>(nx, ny, nz, h, gamma, bc);
  else hd->o = new Oracle<float>(nx, ny, nz, h, gamma, bc);
  return hd;
}

void orc_destroy(void* vh) {
  Handle* hd = (Handle*)vh;
  if (!hd) return;
  if (hd->dtype == 0) delete (Oracle<double>*)hd->o; else delete (Oracle<float>*)hd->o;
  delete hd;
}

void orc_set_state(void* vh, const void* rho, const void* u, const void* v, const void* w,
                   const void* p, const void* psi) {
  Handle* hd = (Handle*)vh;
#define BODY o->set_state((const T*)rho, (const T*)u, (const T*)v, (const T*)w, (const T*)p, (const T*)psi)
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

double orc_compute_dt(void* vh, double cfl) {
  Handle* hd = (Handle*)vh;
  double r = 0;
  DISPATCH(hd, r = (double)o->compute_dt((T)cfl), r = (double)o->compute_dt((T)cfl));
  return r;
}

void orc_step(void* vh, double dt) {
  Handle* hd = (Handle*)vh;
  DISPATCH(hd, o->step((T)dt), o->step((T)dt));
}

// smoothing kernel: 0 = cubic spline (default), 1 = (1 - q^2/4)^5; other values are ignored
void orc_set_kernel(void* vh, int kernel) {
  Handle* hd = (Handle*)vh;
  if (kernel != 0 && kernel != 1) return;
  DISPATCH(hd, o->set_kernel(kernel), o->set_kernel(kernel));
}

// limiter: 0 = minmod (default), 1 = van Leer; other values are ignored
void orc_set_limiter(void* vh, int limiter) {
  Handle* hd = (Handle*)vh;
  if (limiter != 0 && limiter != 1) return;
  DISPATCH(hd, o->limiter = limiter, o->limiter = limiter);
}

// Riemann solver of the Euler stage: 0 = HLL (default), 1 = Lax-Friedrichs, 2 = HLLC; other values are ignored
void orc_set_riemann(void* vh, int riemann) {
  Handle* hd = (Handle*)vh;
  if (riemann < 0 || riemann > 2) return;
  DISPATCH(hd, o->riemann = riemann, o->riemann = riemann);
}

void orc_get_conserved(void* vh, void* rho, void* mx, void* my, void* mz, void* E) {
  Handle* hd = (Handle*)vh;
  void* out[5] = {rho, mx, my, mz, E};
#define BODY for (int c = 0; c < 5; ++c) o->get_field(o->U[c], (T*)out[c])
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

// overwrite the conserved state directly (psi and the inflow planes are kept)
void orc_set_conserved(void* vh, const void* rho, const void* mx, const void* my, const void* mz,
                       const void* E) {
  Handle* hd = (Handle*)vh;
  const void* in[5] = {rho, mx, my, mz, E};
#define BODY for (int c = 0; c < 5; ++c) o->put_field(o->U[c], (const T*)in[c])
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

void orc_get_state(void* vh, void* rho, void* u, void* v, void* w, void* p) {
  Handle* hd = (Handle*)vh;
#define BODY                                                                         \
  {                                                                                  \
    size_t m = 0;                                                                    \
    for (int k = 0; k < o->n[2]; ++k)                                                \
      for (int j = 0; j < o->n[1]; ++j)                                              \
        for (int i = 0; i < o->n[0]; ++i, ++m) {                                     \
          size_t c = o->idx(i, j, k);                                                \
          auto q = o->prim_cell(o->U[0][c], o->U[1][c], o->U[2][c], o->U[3][c], o->U[4][c]); \
          ((T*)rho)[m] = o->U[0][c]; ((T*)u)[m] = q.u; ((T*)v)[m] = q.v;             \
          ((T*)w)[m] = q.w; ((T*)p)[m] = q.p;                                        \
        }                                                                            \
  }
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

void orc_get_vacuum_mask(void* vh, unsigned char* mask) {
  Handle* hd = (Handle*)vh;
#define BODY                                                                  \
  {                                                                           \
    size_t m = 0;                                                             \
    for (int k = 0; k < o->n[2]; ++k)                                         \
      for (int j = 0; j < o->n[1]; ++j)                                       \
        for (int i = 0; i < o->n[0]; ++i, ++m)                                \
          mask[m] = o->U[0][o->idx(i, j, k)] > o->rho_vac ? 0 : 1;            \
  }
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

// Test hooks -------------------------------------------------------------------
// f = -D[psi] on the interior.
void orc_eval_force(void* vh, void* fx, void* fy, void* fz) {
  Handle* hd = (Handle*)vh;
  void* out[3] = {fx, fy, fz};
#define BODY for (int d = 0; d < 3; ++d) o->get_field(o->f[d], (T*)out[d])
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

// Q(U^n, xi) of Eq. (7) on the interior, for caller-supplied particle offsets
// (interior arrays, ghosts filled by wrap on periodic axes and by the boundary
// value otherwise); xi pointers may all be null (particles at the centres).
void orc_eval_Q(void* vh, const void* xix, const void* xiy, const void* xiz, void* qmx, void* qmy,
                void* qmz, void* qE) {
  Handle* hd = (Handle*)vh;
  const void* xin[3] = {xix, xiy, xiz};
  void* out[4] = {qmx, qmy, qmz, qE};
#define BODY                                                                              \
  {                                                                                       \
    o->fill_ghosts_U(false);                                                              \
    o->primitives(o->U, o->U[0], o->phi, o->vel, G);                                      \
    bool have = xix && xiy && xiz;                                                        \
    if (have) {                                                                           \
      for (int d = 0; d < 3; ++d) {                                                       \
        o->put_field(o->xis[d], (const T*)xin[d]);                                        \
        for (int k = -1; k < o->n[2] + 1; ++k)                                            \
          for (int j = -1; j < o->n[1] + 1; ++j)                                          \
            for (int i = -1; i < o->n[0] + 1; ++i) {                                      \
              int s[3] = {i, j, k};                                                       \
              for (int e = 0; e < 3; ++e) {                                               \
                if (o->bc[2 * e] == BC_PERIODIC) s[e] = ((s[e] % o->n[e]) + o->n[e]) % o->n[e]; \
                else s[e] = s[e] < 0 ? 0 : (s[e] > o->n[e] - 1 ? o->n[e] - 1 : s[e]);     \
              }                                                                           \
              o->xis[d][o->idx(i, j, k)] = o->xis[d][o->idx(s[0], s[1], s[2])];           \
            }                                                                             \
      }                                                                                   \
    }                                                                                     \
    o->eval_Q(o->phi, o->vel, have ? o->xis : nullptr, o->U[0], 0);                       \
    for (int c = 0; c < 4; ++c) o->get_field(o->Q[c], (T*)out[c]);                        \
  }
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

// Padded U^n (component c = 0..4: rho, mx, my, mz, E) right after the ghost fill O0 of the next step, as a
// (nz+6, ny+6, nx+6) array, x fastest: lets a test state the boundary rules of reading G16 in its own indexing.
void orc_get_padded(void* vh, int c, void* out) {
  Handle* hd = (Handle*)vh;
  if (c < 0 || c > 4) return;
#define BODY { o->fill_ghosts_U(false); memcpy(out, o->U[c].data(), o->ncell_pad * sizeof(T)); }
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

// Particle offsets of the LAST step (read-only test hook): which = 0: xi* of Eq. (5), valid on
// interior(+)2; which = 1: xi^{n+1} of Eq. (6), valid on interior(+)1; component d = 0..2; padded
// (nz+6, ny+6, nx+6) array, x fastest.  Lets a test check the kinematics of Eq. (5), (6) directly: they are Heun's
// rule for dr/dt = u, which integrates a constant acceleration exactly.
void orc_get_offsets(void* vh, int which, int d, void* out) {
  Handle* hd = (Handle*)vh;
  if (d < 0 || d > 2 || which < 0 || which > 1) return;
#define BODY { memcpy(out, (which ? o->xi[d] : o->xis[d]).data(), o->ncell_pad * sizeof(T)); }
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

// lattice constants (a_f, a_e, a_c, S0') for the closed-form pin
void orc_lattice_constants(void* vh, double* out4) {
  Handle* hd = (Handle*)vh;
#define BODY { out4[0] = o->a_shell[1]; out4[1] = o->a_shell[2]; out4[2] = o->a_shell[3]; out4[3] = o->S0p; }
  DISPATCH(hd, BODY, BODY);
#undef BODY
}

}  // extern "C"
