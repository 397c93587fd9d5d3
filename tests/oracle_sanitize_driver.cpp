// Driver of tests/test_oracle_sanitizers.py: linked with oracle/hard_oracle.cpp, both compiled with
// -fsanitize=address,undefined -fno-sanitize-recover=all.  Runs one Heun step (and reads everything back) for every
// scheme x boundary condition x {5, 6 fields (+ source)} on a small ragged 3-D mesh, a 2-D and a 1-D mesh.  Any
// out-of-bounds access, use of freed memory, leak, signed overflow or misaligned access aborts with a report and a
// non-zero exit code.  Inputs: a fixed positive state from a small integer hash (no method arithmetic here).
#include <cstdio>
#include <cstdlib>
#include <vector>

extern "C" {
void* oracle_create(int, int, int, double, int);
int oracle_destroy(void*);
int oracle_set_spacing(void*, double, double, double);
int oracle_enable_radiation(void*);
int oracle_set_rad_energy(void*, const double*);
int oracle_get_rad_energy(void*, double*);
int oracle_set_source(void*, double, double, double, double);
int oracle_set_scheme(void*, int);
int oracle_set_state(void*, const double*, const double*, const double*, const double*, const double*);
int oracle_get_state(void*, double*, double*, double*, double*, double*);
int oracle_step(void*, double, int);
int oracle_step_dt(void*, double, int);
int oracle_max_dt(void*, double*);
int oracle_get_time(void*, double*, long long*);
long long oracle_fallback_count(void*);
int oracle_rhs(void*, double*);
}

static double unit(unsigned long long i, unsigned long long salt) {          // in [0, 1)
  unsigned long long z = (i + 1) * 0x9E3779B97F4A7C15ull + salt * 0xBF58476D1CE4E5B9ull;
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull; z ^= z >> 27; z *= 0x94D049BB133111EBull; z ^= z >> 31;
  return (double)(z >> 11) / 9007199254740992.0;
}

#define CHECK(x) do { int rc__ = (x); if (rc__ != 0) { fprintf(stderr, "%s -> %d (n=%d,%d,%d scheme %d bc %d rad %d)\n", #x, rc__, nx, ny, nz, scheme, bc, rad); return 1; } } while (0)

static int run(int nx, int ny, int nz, int scheme, int bc, int rad) {
  const size_t n = (size_t)nx * ny * nz;
  std::vector<double> f[6], out[6], rhs(6 * n);
  for (int v = 0; v < 6; ++v) { f[v].resize(n); out[v].resize(n); }
  for (size_t i = 0; i < n; ++i) {
    f[0][i] = 1.0 + 0.5 * unit(i, 1);
    for (int d = 0; d < 3; ++d) f[1 + d][i] = 0.4 * (unit(i, 2 + d) - 0.5);
    f[4][i] = 2.5 + unit(i, 5);
    f[5][i] = 0.1 + unit(i, 6);
  }
  void* h = oracle_create(nx, ny, nz, 1.4, bc);
  if (!h) { fprintf(stderr, "oracle_create failed\n"); return 1; }
  CHECK(oracle_set_scheme(h, scheme));
  if (rad) CHECK(oracle_enable_radiation(h));
  CHECK(oracle_set_spacing(h, 1.0 / nx, 1.0 / ny, 1.0 / nz));
  CHECK(oracle_set_state(h, f[0].data(), f[1].data(), f[2].data(), f[3].data(), f[4].data()));
  if (rad) {
    CHECK(oracle_set_rad_energy(h, f[5].data()));
    if (rad == 2) CHECK(oracle_set_source(h, 0.5, 3.0, 1.0, 1.5));
  }
  double dt = 0.0, t = 0.0;
  long long steps = 0;
  CHECK(oracle_max_dt(h, &dt));
  CHECK(oracle_rhs(h, rhs.data()));
  CHECK(oracle_step(h, 0.4, 1));
  CHECK(oracle_step_dt(h, 0.1 * dt, 1));
  CHECK(oracle_get_state(h, out[0].data(), out[1].data(), out[2].data(), out[3].data(), out[4].data()));
  if (rad) CHECK(oracle_get_rad_energy(h, out[5].data()));
  CHECK(oracle_get_time(h, &t, &steps));
  if (steps != 2 || !(t > 0.0) || oracle_fallback_count(h) < 0) { fprintf(stderr, "bad bookkeeping\n"); return 1; }
  CHECK(oracle_destroy(h));
  return 0;
}

int main() {
  const int meshes[3][3] = { { 11, 7, 6 }, { 13, 9, 1 }, { 23, 1, 1 } };
  int runs = 0;
  for (const auto& m : meshes)
    for (int scheme = 0; scheme < 2; ++scheme)
      for (int bc = 0; bc < 3; ++bc)
        for (int rad = 0; rad < 3; ++rad) {
          if (run(m[0], m[1], m[2], scheme, bc, rad)) return 1;
          ++runs;
        }
  printf("sanitized oracle: %d runs clean\n", runs);
  return 0;
}
