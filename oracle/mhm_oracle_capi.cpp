// oracle/mhm_oracle_capi.cpp — TEST INFRASTRUCTURE. extern "C" face of the fp64 oracle (mhm_oracle.hpp)
// for ctypes (oracle/mhm_oracle.py). CUDA-free; shares no code with the GPU path.
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "counting_real.hpp"
#include "mhm_oracle.hpp"

using namespace mhm_oracle;

extern "C" {

int mhm_oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// Batch of cubic patch groups (SURVEY.md §8(b) layouts, all fp64):
//   U_in [n_groups][5][S][S][S], S = N + 2*ghost;  U_out [n_groups][5][N][N][N];
//   bflux [n_groups][6][5][N][N] or NULL;  guard/margin [n_groups][N+2][N+2][N+2] or NULL.
// stats_out[0] = guard cells, [1] = non-positive outputs (summed over groups). Returns threads used.
int mhm_oracle_step_groups(const double* U_in, int n_groups, int N, int ghost, double dt, double dx,
                           double gamma, int limiter, double* U_out, double* bflux, unsigned char* guard,
                           double* margin, unsigned long long* stats_out, int n_threads) {
  const size_t S = (size_t)N + 2 * ghost;
  const size_t in_sz = 5 * S * S * S, out_sz = (size_t)5 * N * N * N, bf_sz = (size_t)30 * N * N;
  const size_t g_sz = (size_t)(N + 2) * (N + 2) * (N + 2);
  unsigned long long gc = 0, npo = 0;
  int used = 1;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
  used = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : gc, npo)
#endif
  for (int g = 0; g < n_groups; ++g) {
    StepStats st = step_box<double>(U_in + g * in_sz, N, N, N, ghost, dt, dx, gamma, limiter, U_out + g * out_sz,
                                    bflux ? bflux + g * bf_sz : nullptr, guard ? guard + g * g_sz : nullptr,
                                    margin ? margin + g * g_sz : nullptr);
    gc += st.guard_cells;
    npo += st.nonpositive_out;
  }
  if (stats_out) { stats_out[0] = gc; stats_out[1] = npo; }
  return used < n_groups ? used : (n_groups > 0 ? n_groups : 1);
}

// The same with the robustness variants: flags = RiemannFlags, midflux [n_groups][3][5][N][N] or NULL.
int mhm_oracle_step_groups_ex(const double* U_in, int n_groups, int N, int ghost, double dt, double dx, double gamma,
                              int limiter, int flags, double* U_out, double* bflux, double* midflux,
                              unsigned char* guard, unsigned long long* stats_out, int n_threads,
                              unsigned char* hlle_faces) {   // hlle_faces: [n_groups][3][N+1][N+1][N+1] or NULL
  const size_t S = (size_t)N + 2 * ghost;
  const size_t in_sz = 5 * S * S * S, out_sz = (size_t)5 * N * N * N, bf_sz = (size_t)30 * N * N, mf_sz = (size_t)15 * N * N;
  const size_t h_sz = (size_t)3 * (N + 1) * (N + 1) * (N + 1);
  const size_t g_sz = (size_t)(N + 2) * (N + 2) * (N + 2);
  unsigned long long gc = 0, npo = 0;
  int used = 1;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
  used = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : gc, npo)
#endif
  for (int g = 0; g < n_groups; ++g) {
    StepStats st = step_box<double>(U_in + g * in_sz, N, N, N, ghost, dt, dx, gamma, limiter, U_out + g * out_sz,
                                    bflux ? bflux + g * bf_sz : nullptr, guard ? guard + g * g_sz : nullptr, nullptr,
                                    flags, midflux ? midflux + g * mf_sz : nullptr,
                                    hlle_faces ? hlle_faces + g * h_sz : nullptr);
    gc += st.guard_cells;
    npo += st.nonpositive_out;
  }
  if (stats_out) { stats_out[0] = gc; stats_out[1] = npo; }
  return used < n_groups ? used : (n_groups > 0 ? n_groups : 1);
}

int mhm_oracle_roe_flux_ex(const double* UL, const double* UR, double gamma, int d, int flags, double* F) {
  bool hlle = false;
  roe_flux<double>(UL, UR, gamma, d, F, flags, &hlle);
  return hlle ? 1 : 0;
}

// One global box (O8): U_in [5][nz+2g][ny+2g][nx+2g] -> U_out [5][nz][ny][nx]. Serial.
void mhm_oracle_step_box(const double* U_in, int nx, int ny, int nz, int ghost, double dt, double dx, double gamma,
                         int limiter, double* U_out, double* bflux, unsigned char* guard, double* margin,
                         unsigned long long* stats_out) {
  StepStats st = step_box<double>(U_in, nx, ny, nz, ghost, dt, dx, gamma, limiter, U_out, bflux, guard, margin);
  if (stats_out) { stats_out[0] = st.guard_cells; stats_out[1] = st.nonpositive_out; }
}

void mhm_oracle_cons_to_prim(const double* U, double gamma, double* W) { cons_to_prim<double>(U, gamma, W); }
void mhm_oracle_prim_to_cons(const double* W, double gamma, double* U) { prim_to_cons<double>(W, gamma, U); }
double mhm_oracle_limited_slope(double dL, double dR, int limiter) { return limited_slope<double>(dL, dR, limiter); }

void mhm_oracle_phys_flux(const double* U, double gamma, int d, double* F) {
  double W[5];
  cons_to_prim<double>(U, gamma, W);
  phys_flux<double>(U, W, d, F);
}

void mhm_oracle_roe_flux(const double* UL, const double* UR, double gamma, int d, double* F) {
  roe_flux<double>(UL, UR, gamma, d, F);
}

// alpha[5], lambda[5], K[5][5] (K[i][c], rotated component order rho, m_n, m_t1, m_t2, E)
void mhm_oracle_roe_decompose(const double* UL, const double* UR, double gamma, int d, double* alpha, double* lambda,
                              double* K) {
  RoeDecomp<double> R;
  roe_decompose<double>(UL, UR, gamma, d, R);
  for (int i = 0; i < 5; ++i) {
    alpha[i] = R.alpha[i];
    lambda[i] = R.lambda[i];
    for (int c = 0; c < 5; ++c) K[i * 5 + c] = R.K[i][c];
  }
}

// Algorithmic FLOPs of one step on one N^3 group (input values given in fp64), by category:
// counts[0..4] = add, mul, div, sqrt, minmax. The values only steer the limiter's zero-slope branch
// (a zero slope skips min / the van Leer quotient) and the guard; pass a generic smooth field.
void mhm_oracle_count_flops(const double* U_in, int N, int ghost, double dt, double dx, double gamma, int limiter,
                            unsigned long long* counts) {
  const size_t S = (size_t)N + 2 * ghost;
  std::vector<CountingReal> in(5 * S * S * S), out((size_t)5 * N * N * N), bf((size_t)30 * N * N);
  for (size_t i = 0; i < in.size(); ++i) in[i] = CountingReal(U_in[i]);
  tally() = FlopTally();
  step_box<CountingReal>(in.data(), N, N, N, ghost, CountingReal(dt), CountingReal(dx), CountingReal(gamma), limiter,
                         out.data(), bf.data(), nullptr, nullptr);
  const FlopTally t = tally();
  counts[0] = t.add; counts[1] = t.mul; counts[2] = t.div; counts[3] = t.sqrt; counts[4] = t.minmax;
}

}  // extern "C"
