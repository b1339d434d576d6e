// oracle/rtvd_oracle_capi.cpp — TEST INFRASTRUCTURE. extern "C" face of the fp64 relaxing-TVD oracle
// (rtvd_oracle.hpp) for ctypes (oracle/rtvd_oracle.py). CUDA-free; shares no code with the GPU path.
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "counting_real.hpp"
#include "rtvd_oracle.hpp"

extern "C" {

// Batch of cubic patch groups: U_in [n_groups][5][N+6][N+6][N+6] -> U_out [n_groups][5][N][N][N]. Returns threads used.
int rtvd_oracle_step_groups(const double* U_in, int n_groups, int N, double dt, double dx, double gamma, int sweep,
                            double* U_out, int n_threads) {
  const size_t S = (size_t)N + 6;
  const size_t in_sz = 5 * S * S * S, out_sz = (size_t)5 * N * N * N;
  int used = 1;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
  used = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1)
#endif
  for (int g = 0; g < n_groups; ++g)
    rtvd_oracle::step_box<double>(U_in + g * in_sz, N, N, N, dt, dx, gamma, sweep, U_out + g * out_sz);
  return used < n_groups ? used : (n_groups > 0 ? n_groups : 1);
}

void rtvd_oracle_step_box(const double* U_in, int nx, int ny, int nz, double dt, double dx, double gamma, int sweep,
                          double* U_out) {
  rtvd_oracle::step_box<double>(U_in, nx, ny, nz, dt, dx, gamma, sweep, U_out);
}

void rtvd_oracle_sweep_line(double* u, int L, int d, double dt, double dx, double gamma) {
  std::vector<double> v(u, u + 5 * (size_t)L);
  rtvd_oracle::sweep_line<double>(v, L, d, dt, dx, gamma);
  for (size_t k = 0; k < v.size(); ++k) u[k] = v[k];
}

double rtvd_oracle_vanleer(double a, double b) { return rtvd_oracle::vanleer<double>(a, b); }

void rtvd_oracle_flux_and_speed(const double* u, int d, double gamma, double* F, double* c) {
  rtvd_oracle::flux_and_speed<double>(u, d, gamma, F, *c);
}

// Algorithmic FLOPs of one step on one N^3 group (values given in fp64), by category: counts[0..4] = add, mul, div,
// sqrt, minmax (the convention of counting_real.hpp: abs, negate, compare, select and copies cost nothing). The same
// text as above with T = CountingReal. The values steer only the limiter's zero branch (differences of opposite sign
// skip the van Leer quotient) and the pressure clamp: pass a field that is monotone along every axis.
void rtvd_oracle_count_flops(const double* U_in, int N, double dt, double dx, double gamma, int sweep,
                             unsigned long long* counts) {
  using mhm_oracle::CountingReal;
  const size_t S = (size_t)N + 6;
  std::vector<CountingReal> in(5 * S * S * S), out((size_t)5 * N * N * N);
  for (size_t i = 0; i < in.size(); ++i) in[i] = CountingReal(U_in[i]);
  mhm_oracle::tally() = mhm_oracle::FlopTally();
  rtvd_oracle::step_box<CountingReal>(in.data(), N, N, N, CountingReal(dt), CountingReal(dx), CountingReal(gamma), sweep,
                                      out.data());
  const mhm_oracle::FlopTally t = mhm_oracle::tally();
  counts[0] = t.add; counts[1] = t.mul; counts[2] = t.div; counts[3] = t.sqrt; counts[4] = t.minmax;
}

}  // extern "C"
