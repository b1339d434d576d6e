// oracle/rtvd_oracle.hpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU statement (fp64, CUDA-free) of the OTHER hydrodynamic solver the paper names
// (SURVEY.md §8(f) rank 3): the second-order relaxing total-variation-diminishing (TVD) scheme.
//
//   PAPER.md:13 (§2)  "... the second-order relaxing total variation diminishing (TVD) method (Trac & Pen 2003) ...
//                      [with] dimensional splitting"
//   PAPER.md:27 (§2)  the relaxing TVD scheme needs "seven points" per direction (=> 3 ghost cells), against five
//                      for MUSCL-Hancock.
//
// The paper prints no formula; the algorithm below is the published one of Trac & Pen (2003, "A primer on Eulerian
// computational fluid dynamics for astrophysics", their relaxing-TVD section; after Jin & Xin 1995), restated in my
// own code, with the readings RT1–RT8 of DESIGN.md §13:
//   RT1  relaxation system of one sweep along axis d: u = uR + uL, F(u) = c (uR - uL), i.e. the right- / left-moving
//        fluxes fr = (c u + F)/2 and fl = (c u - F)/2, with the freezing speed c = |v_d| + c_s PER CELL
//   RT2  second order in time: a half step with the first-order upwind fluxes of the relaxed system, then the full
//        step with second-order TVD fluxes evaluated on the half-step state
//   RT3  flux limiter: van Leer (harmonic mean) on the one-sided differences of fr and of fl; zero unless both
//        differences have the same sign
//   RT4  three dimensions by dimensional splitting; `sweep` = 0: x, y, z; 1: z, y, x (callers alternate)
//   RT5  3 ghost cells per side; a sweep along d updates every line whose other two indices are still valid (the
//        valid range shrinks by 3 per side along a swept axis only)
//   RT6  ideal gas; c_s = sqrt(gamma max(P, 0) / rho); no floors anywhere
//   RT7  layouts as the MUSCL-Hancock path with ghost = 3: U_in [5][nz+6][ny+6][nx+6] -> U_out [5][nz][ny][nx]
//   RT8  the update forms flux DIFFERENCES first and adds them to the state (a uniform state is preserved exactly)
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may use anything under oracle/. Shares no code
// with paper_1007_3818_b200/csrc/. Pins: tests/test_rtvd_oracle_pins.py (uniform state, conservation, Sod tube against
// the exact Riemann solution, second-order convergence, TVD, 1-D reduction and a periodic whole-box transcription with
// array shifts, decomposition invariance, axis-permutation symmetry of the two sweep orders).
#pragma once
#include <cmath>
#include <cstddef>
#include <vector>

namespace rtvd_oracle {

// The text below is templated on the scalar T ONLY so that the same lines also run with T = CountingReal
// (counting_real.hpp), which tallies their arithmetic: that tally is the FLOP numerator of bench.py's relaxing-TVD
// roofline. With T = double (everything else in this header's users) o_sqrt / o_abs / o_value are the plain functions.
inline double o_sqrt(double x) { return std::sqrt(x); }
inline double o_abs(double x) { return std::fabs(x); }
inline double o_value(double x) { return x; }

// physical flux along axis d and freezing speed of one cell (RT1, RT6)
template <class T>
inline void flux_and_speed(const T u[5], int d, T gamma, T F[5], T& c) {
  const T rho = u[0];
  const T v = u[1 + d] / rho;
  const T ke = T(0.5) * (u[1] * u[1] + u[2] * u[2] + u[3] * u[3]) / rho;
  const T P = (gamma - T(1.0)) * (u[4] - ke);
  F[0] = u[1 + d];
  F[1] = u[1] * v;
  F[2] = u[2] * v;
  F[3] = u[3] * v;
  F[1 + d] = F[1 + d] + P;
  F[4] = (u[4] + P) * v;
  const T Pc = o_value(P) > 0.0 ? P : T(0.0);
  c = o_abs(v) + o_sqrt(gamma * Pc / rho);
}

// van Leer limiter of two one-sided differences (RT3); the sign test is by comparison (no product underflow)
template <class T>
inline T vanleer(T a, T b) {
  const bool same = (o_value(a) > 0.0 && o_value(b) > 0.0) || (o_value(a) < 0.0 && o_value(b) < 0.0);
  return same ? T(2.0) * a * b / (a + b) : T(0.0);
}

// One sweep of one line of L cells along axis d (RT1–RT3, RT8). u: [L][5], updated in place for j = 3 .. L-4.
template <class T>
inline void sweep_line(std::vector<T>& u, int L, int d, T dt, T dx, T gamma) {
  const T lam = dt / dx;
  std::vector<T> fr(5 * L), fl(5 * L), u1(5 * L), fu(5 * L);
  // half step: first-order upwind fluxes of the relaxed system at the faces j+1/2, j = 0 .. L-2
  for (int j = 0; j < L; ++j) {
    T F[5], c;
    flux_and_speed(&u[5 * j], d, gamma, F, c);
    for (int q = 0; q < 5; ++q) {
      fr[5 * j + q] = T(0.5) * (c * u[5 * j + q] + F[q]);
      fl[5 * j + q] = T(0.5) * (c * u[5 * j + q] - F[q]);
    }
  }
  for (int j = 0; j + 1 < L; ++j)
    for (int q = 0; q < 5; ++q) fu[5 * j + q] = fr[5 * j + q] - fl[5 * (j + 1) + q];   // face j+1/2
  for (int j = 1; j + 1 < L; ++j)
    for (int q = 0; q < 5; ++q) u1[5 * j + q] = u[5 * j + q] - T(0.5) * lam * (fu[5 * j + q] - fu[5 * (j - 1) + q]);
  // full step: second-order TVD fluxes on the half-step state (cells 1 .. L-2)
  for (int j = 1; j + 1 < L; ++j) {
    T F[5], c;
    flux_and_speed(&u1[5 * j], d, gamma, F, c);
    for (int q = 0; q < 5; ++q) {
      fr[5 * j + q] = T(0.5) * (c * u1[5 * j + q] + F[q]);
      fl[5 * j + q] = T(0.5) * (c * u1[5 * j + q] - F[q]);
    }
  }
  for (int j = 2; j + 3 < L; ++j)   // faces j+1/2, j = 2 .. L-4
    for (int q = 0; q < 5; ++q) {
      const T FR = fr[5 * j + q] + vanleer(T(0.5) * (fr[5 * j + q] - fr[5 * (j - 1) + q]),
                                           T(0.5) * (fr[5 * (j + 1) + q] - fr[5 * j + q]));
      const T FL = fl[5 * (j + 1) + q] + vanleer(T(0.5) * (fl[5 * j + q] - fl[5 * (j + 1) + q]),
                                                 T(0.5) * (fl[5 * (j + 1) + q] - fl[5 * (j + 2) + q]));
      fu[5 * j + q] = FR - FL;
    }
  for (int j = 3; j + 3 < L; ++j)
    for (int q = 0; q < 5; ++q) u[5 * j + q] = u[5 * j + q] - lam * (fu[5 * j + q] - fu[5 * (j - 1) + q]);
}

// One time step of one box (RT4, RT5, RT7). U_in [5][nz+6][ny+6][nx+6] -> U_out [5][nz][ny][nx].
template <class T>
inline void step_box(const T* U_in, int nx, int ny, int nz, T dt, T dx, T gamma, int sweep, T* U_out) {
  const int G = 3;
  const int S[3] = {nx + 2 * G, ny + 2 * G, nz + 2 * G};   // stored extent along x, y, z
  const size_t vol = (size_t)S[0] * S[1] * S[2];
  std::vector<T> W(U_in, U_in + 5 * vol);
  int lo[3] = {0, 0, 0}, hi[3] = {S[0], S[1], S[2]};        // valid index range per axis
  const size_t stride[3] = {1, (size_t)S[0], (size_t)S[0] * S[1]};
  for (int pass = 0; pass < 3; ++pass) {
    const int d = sweep == 0 ? pass : 2 - pass;
    const int a = (d + 1) % 3, b = (d + 2) % 3;
    const int L = S[d];
    std::vector<T> line(5 * L);
    for (int ib = lo[b]; ib < hi[b]; ++ib)
      for (int ia = lo[a]; ia < hi[a]; ++ia) {
        const size_t base = ia * stride[a] + ib * stride[b];
        for (int j = 0; j < L; ++j)
          for (int q = 0; q < 5; ++q) line[5 * j + q] = W[q * vol + base + j * stride[d]];
        sweep_line(line, L, d, dt, dx, gamma);
        for (int j = G; j < L - G; ++j)
          for (int q = 0; q < 5; ++q) W[q * vol + base + j * stride[d]] = line[5 * j + q];
      }
    lo[d] = G;
    hi[d] = S[d] - G;
  }
  for (int q = 0; q < 5; ++q)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i)
          U_out[((size_t)(q * nz + k) * ny + j) * nx + i] = W[q * vol + (size_t)(k + G) * stride[2] + (j + G) * stride[1] + (i + G)];
}

}  // namespace rtvd_oracle
