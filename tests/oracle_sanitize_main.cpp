// Test driver (tests/test_oracle_sanitize.py): the CPU oracle compiled with -fsanitize=address,undefined and run on
// the 64x4x4 Sod tube (BASELINE.json configs[0]) and on a ragged grid with one boundary kind per axis (SURVEY.md
// section 5: "oracle under -fsanitize=address,undefined").  Test infrastructure only; it includes the oracle's
// source so that every pass, ghost fill and getter runs instrumented.
#include "../oracle/csph_oracle.cpp"

#include <cstdio>

static int run_case(const char* name, int nx, int ny, int nz, const int* bc, int dtype, int sod, int steps, int riemann,
                    int limiter, int kernel) {
  size_t n = (size_t)nx * ny * nz;
  std::vector<double> f64[6];
  std::vector<float> f32[6];
  for (int q = 0; q < 6; ++q) { f64[q].resize(n); f32[q].resize(n); }
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        size_t m = ((size_t)k * ny + j) * nx + i;
        double x = (i + 0.5) / nx, y = (j + 0.5) / ny, z = (k + 0.5) / nz, v[6];
        if (sod) {
          v[0] = i < nx / 2 ? 1.0 : 0.125; v[1] = v[2] = v[3] = 0; v[4] = i < nx / 2 ? 1.0 : 0.1; v[5] = 0;
        } else {
          v[0] = 1 + 0.3 * std::sin(6.28 * x) * std::cos(6.28 * y);
          v[1] = 0.4 * std::sin(6.28 * (y + z)); v[2] = -0.3 * std::cos(6.28 * x); v[3] = 0.2 * std::sin(6.28 * z);
          v[4] = 1 + 0.2 * std::cos(6.28 * (x - z)); v[5] = 0.1 * std::sin(6.28 * x) * std::sin(6.28 * y);
        }
        for (int q = 0; q < 6; ++q) { f64[q][m] = v[q]; f32[q][m] = (float)v[q]; }
      }
  void* h = orc_create(nx, ny, nz, 1.0 / nx, 1.4, bc, dtype);
  if (!h) return 1;
  orc_set_kernel(h, kernel);
  orc_set_limiter(h, limiter);
  orc_set_riemann(h, riemann);
  if (dtype == 0) orc_set_state(h, f64[0].data(), f64[1].data(), f64[2].data(), f64[3].data(), f64[4].data(), f64[5].data());
  else orc_set_state(h, f32[0].data(), f32[1].data(), f32[2].data(), f32[3].data(), f32[4].data(), f32[5].data());
  for (int s = 0; s < steps; ++s) {
    double dt = orc_compute_dt(h, 0.4);
    if (!(dt > 0) || !std::isfinite(dt)) { std::printf("%s: bad dt\n", name); return 1; }
    orc_step(h, dt);
  }
  std::vector<double> out(5 * n);
  std::vector<unsigned char> mask(n);
  std::vector<double> pad((size_t)(nx + 6) * (ny + 6) * (nz + 6));
  orc_get_conserved(h, &out[0], &out[n], &out[2 * n], &out[3 * n], &out[4 * n]);
  orc_get_state(h, &out[0], &out[n], &out[2 * n], &out[3 * n], &out[4 * n]);
  orc_get_vacuum_mask(h, mask.data());
  orc_get_padded(h, 0, pad.data());
  orc_eval_force(h, &out[0], &out[n], &out[2 * n]);
  orc_eval_Q(h, nullptr, nullptr, nullptr, &out[0], &out[n], &out[2 * n], &out[3 * n]);
  double sum = 0;
  if (dtype == 0) for (size_t m = 0; m < n; ++m) sum += out[m];
  orc_destroy(h);
  std::printf("%s: ok (%d steps, checksum %.6e)\n", name, steps, sum);
  return std::isfinite(sum) ? 0 : 1;
}

int main() {
  int rc = 0;
  const int sod_bc[6] = {1, 1, 0, 0, 0, 0};
  const int mix_bc[6] = {2, 1, 0, 0, 1, 2};
  const int per_bc[6] = {0, 0, 0, 0, 0, 0};
  orc_set_threads(2);
  rc |= run_case("sod 64x4x4 f64", 64, 4, 4, sod_bc, 0, 1, 12, 0, 0, 0);
  rc |= run_case("ragged 13x7x5 f64 inflow/outflow/periodic", 13, 7, 5, mix_bc, 0, 0, 6, 0, 0, 0);
  rc |= run_case("ragged 13x7x5 f32 van Leer, HLLC, poly5", 13, 7, 5, mix_bc, 1, 0, 6, 2, 1, 1);
  rc |= run_case("thin 5x1x3 f64 LF", 5, 1, 3, per_bc, 0, 0, 4, 1, 0, 0);
  return rc;
}
