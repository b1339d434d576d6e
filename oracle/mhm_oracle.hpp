// oracle/mhm_oracle.hpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU statement (fp64, CUDA-free) of the hot path of arXiv 1007.3818:
// the unsplit 3-D MUSCL-Hancock finite-volume update with Roe's Riemann solver.
//
//   PAPER.md:15 (§2)  "This approach contains four steps, namely, the spatial data reconstruction, the
//                      half-step prediction, the Riemann solver, and the full-step update. We apply the
//                      unsplit finite volume method for the three-dimensional evolution, and the Roe's
//                      solver is adopted for the Riemann problem."
//   PAPER.md:27 (§2)  "it requires only a five-point stencil in each spatial direction"
//   PAPER.md:9,59,65  cites Toro (2009) for MUSCL-Hancock and Roe (1981) for the solver.
//
// The paper prints no formulas; every numerical detail below is the reading fixed in SURVEY.md §8(c)
// (steps O0–O8, readings R1–R21) and restated in DESIGN.md §3. The result is *defined by* this algorithm,
// so the code follows it step by step, in the order and notation of §8(c), with no blocking, fusion or
// reordering. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may use anything in oracle/. It shares no code with paper_1007_3818_b200/csrc/.
//
// Parity status: every function here is pinned by tests/test_oracle_pins.py (P1–P16) except the two
// conventions that have no independent definition — "parity unpinned": the R7 guard rule (what to do
// when a predicted face state is non-physical) and the R12 boundary-flux layout. Both are pinned only by
// being written down; the layout is additionally cross-checked by the balance pin P11.
//
// Templated on the scalar T so that the same text runs with T = double (the oracle) and with
// T = CountingReal (oracle/counting_real.hpp), which tallies the algorithmic FLOPs of SURVEY.md §8(d).
#pragma once
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <vector>

namespace mhm_oracle {

enum Limiter { MINMOD = 0, VANLEER = 1, MC = 2 };
// Robustness variants of the Riemann step (readings R8b, R8c of DESIGN.md §14). PAPER.md:15
// names only "the Roe's solver": flags = 0 is that plain solver and the default everywhere.
enum RiemannFlags { ENTROPY_FIX = 1, HLLE_FALLBACK = 2 };

// scalar helpers, overloaded for CountingReal in counting_real.hpp
inline double o_sqrt(double x) { return std::sqrt(x); }
inline double o_abs(double x) { return std::fabs(x); }
inline double o_min(double a, double b) { return a < b ? a : b; }
inline double o_value(double x) { return x; }

// ---------------------------------------------------------------------------------------------------
// O1 (R1). Ideal gas, U = (rho, mx, my, mz, E), W = (rho, vx, vy, vz, P).
//   v = m / rho,  P = (gamma-1) * (E - 1/2 (mx vx + my vy + mz vz))
template <class T>
inline void cons_to_prim(const T U[5], T gamma, T W[5]) {
  W[0] = U[0];
  W[1] = U[1] / U[0];
  W[2] = U[2] / U[0];
  W[3] = U[3] / U[0];
  W[4] = (gamma - T(1.0)) * (U[4] - T(0.5) * (U[1] * W[1] + U[2] * W[2] + U[3] * W[3]));
}

// O4 (R1). m = rho v,  E = P/(gamma-1) + 1/2 rho |v|^2
template <class T>
inline void prim_to_cons(const T W[5], T gamma, T U[5]) {
  U[0] = W[0];
  U[1] = W[0] * W[1];
  U[2] = W[0] * W[2];
  U[3] = W[0] * W[3];
  U[4] = W[4] / (gamma - T(1.0)) + T(0.5) * W[0] * (W[1] * W[1] + W[2] * W[2] + W[3] * W[3]);
}

// O4. Physical flux density along axis d (0=x,1=y,2=z) of a state given both as conserved U and as
// primitive W (the caller holds both), components in the global order (rho, mx, my, mz, E):
//   F_d = (m_d, m_d v_d + P, m_t1 v_d, m_t2 v_d, (E+P) v_d).
template <class T>
inline void phys_flux(const T U[5], const T W[5], int d, T F[5]) {
  const T vd = W[1 + d];
  F[0] = U[1 + d];
  F[1] = U[1] * vd;
  F[2] = U[2] * vd;
  F[3] = U[3] * vd;
  F[1 + d] = F[1 + d] + W[4];
  F[4] = (U[4] + W[4]) * vd;
}

// O2 (R3, R4). Limited slope from the one-sided differences dL = W_c - W_{c-1}, dR = W_{c+1} - W_c.
//   zero when the signs differ or either difference is zero (sign test by comparison, not product);
//   MinMod:   sign(dL) * min(|dL|, |dR|)
//   van Leer: 2 dL dR / (dL + dR)               (harmonic mean)
//   MC:       sign(dL) * min(2|dL|, 2|dR|, |dL + dR| / 2)   (monotonized central)
template <class T>
inline T limited_slope(T dL, T dR, int limiter) {
  const bool same_sign = (o_value(dL) > 0.0 && o_value(dR) > 0.0) || (o_value(dL) < 0.0 && o_value(dR) < 0.0);
  if (!same_sign) return T(0.0);
  if (limiter == MINMOD) {
    const T m = o_min(o_abs(dL), o_abs(dR));
    return o_value(dL) > 0.0 ? m : -m;
  }
  if (limiter == MC) {
    const T m = o_min(o_min(T(2.0) * o_abs(dL), T(2.0) * o_abs(dR)), T(0.5) * o_abs(dL + dR));
    return o_value(dL) > 0.0 ? m : -m;
  }
  return T(2.0) * dL * dR / (dL + dR);
}

// O5 (R8, R9, R21). Roe's linearisation in the frame rotated so that axis d is "x".
// Component order in the rotated frame: (rho, m_n, m_t1, m_t2, E) with n = d, t1 = (d+1)%3, t2 = (d+2)%3.
template <class T>
struct RoeDecomp {
  T WL[5], WR[5];  // primitives of the two sides (global component order)
  T alpha[5];   // wave strengths
  T lambda[5];  // eigenvalues u-a, u, u, u, u+a
  T K[5][5];    // K[i][c]: component c (rotated order) of right eigenvector i
};

template <class T>
inline void roe_decompose(const T UL[5], const T UR[5], T gamma, int d, RoeDecomp<T>& R) {
  const int n = d, t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  T* WL = R.WL;
  T* WR = R.WR;
  cons_to_prim(UL, gamma, WL);
  cons_to_prim(UR, gamma, WR);
  const T HL = (UL[4] + WL[4]) / UL[0];
  const T HR = (UR[4] + WR[4]) / UR[0];
  const T sL = o_sqrt(UL[0]), sR = o_sqrt(UR[0]);
  const T den = sL + sR;
  // sqrt(rho)-weighted averages of u, v, w, H
  const T u = (sL * WL[1 + n] + sR * WR[1 + n]) / den;
  const T v = (sL * WL[1 + t1] + sR * WR[1 + t1]) / den;
  const T w = (sL * WL[1 + t2] + sR * WR[1 + t2]) / den;
  const T H = (sL * HL + sR * HR) / den;
  const T V2 = u * u + v * v + w * w;
  const T a2 = (gamma - T(1.0)) * (H - T(0.5) * V2);
  const T a = o_sqrt(a2);
  // jumps of the conserved variables in rotated order
  const T du1 = UR[0] - UL[0];
  const T du2 = UR[1 + n] - UL[1 + n];
  const T du3 = UR[1 + t1] - UL[1 + t1];
  const T du4 = UR[1 + t2] - UL[1 + t2];
  const T du5 = UR[4] - UL[4];
  // wave strengths (Toro 2009, §11.2.2 form; alpha5 written mirror-symmetrically to alpha1, R21)
  const T al3 = du3 - v * du1;
  const T al4 = du4 - w * du1;
  const T du5b = du5 - al3 * v - al4 * w;
  const T al2 = (gamma - T(1.0)) / a2 * (du1 * (H - u * u) + u * du2 - du5b);
  const T al1 = (du1 * (u + a) - du2 - a * al2) / (T(2.0) * a);
  const T al5 = (du1 * (a - u) + du2 - a * al2) / (T(2.0) * a);
  R.alpha[0] = al1; R.alpha[1] = al2; R.alpha[2] = al3; R.alpha[3] = al4; R.alpha[4] = al5;
  R.lambda[0] = u - a; R.lambda[1] = u; R.lambda[2] = u; R.lambda[3] = u; R.lambda[4] = u + a;
  const T ua = u * a;
  const T zero(0.0), one(1.0);
  const T K1[5] = {one, u - a, v, w, H - ua};
  const T K2[5] = {one, u, v, w, T(0.5) * V2};
  const T K3[5] = {zero, zero, one, zero, v};
  const T K4[5] = {zero, zero, zero, one, w};
  const T K5[5] = {one, u + a, v, w, H + ua};
  for (int c = 0; c < 5; ++c) {
    R.K[0][c] = K1[c]; R.K[1][c] = K2[c]; R.K[2][c] = K3[c]; R.K[3][c] = K4[c]; R.K[4][c] = K5[c];
  }
}

// O5.  F = 1/2 [F(UL) + F(UR)] - 1/2 sum_i alpha_i |lambda_i| K_i, no entropy fix (R8); returned in
// the global component order (rho, mx, my, mz, E), flux density along +axis d.
// flags (default 0 = the plain solver above, readings R8b / R8c):
//   ENTROPY_FIX   Harten & Hyman's fix of the two acoustic waves: with lambda_L, lambda_R the wave's speed u -+ a in the
//                 states on its two sides (the outer state and the intermediate state U*_L = UL + alpha_1 K_1, resp.
//                 U*_R = UR - alpha_5 K_5) and delta = max(0, lambda~ - lambda_L, lambda_R - lambda~), |lambda~| is
//                 replaced by (lambda~^2 / delta + delta) / 2 wherever |lambda~| < delta, i.e. only inside a
//                 transonic expansion, where plain Roe admits an expansion shock.
//   HLLE_FALLBACK if either intermediate state of the linearisation, U*_L = UL + alpha_1 K_1 or U*_R = UR - alpha_5 K_5,
//                 is non-physical (rho* <= 0 or 2 rho* E* <= |m*|^2), the flux is Einfeldt's HLLE flux
//                 (b+ F_L - b- F_R + b+ b- (UR - UL)) / (b+ - b-), b- = min(u_L - a_L, u~ - a~, 0),
//                 b+ = max(u_R + a_R, u~ + a~, 0), which is positivity preserving.
template <class T>
inline void roe_flux(const T UL[5], const T UR[5], T gamma, int d, T F[5], int flags = 0, bool* used_hlle = nullptr) {
  const int n = d, t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  const int to_global[5] = {0, 1 + n, 1 + t1, 1 + t2, 4};
  RoeDecomp<T> R;
  roe_decompose(UL, UR, gamma, d, R);
  T FL[5], FR[5];
  phys_flux(UL, R.WL, d, FL);
  phys_flux(UR, R.WR, d, FR);
  if (used_hlle) *used_hlle = false;
  T absl1 = o_abs(R.lambda[0]), absl5 = o_abs(R.lambda[4]);
  if (flags != 0) {
    const T aL = o_sqrt(gamma * R.WL[4] / R.WL[0]), aR = o_sqrt(gamma * R.WR[4] / R.WR[0]);
    const T uL = R.WL[1 + n], uR = R.WR[1 + n];
    if (flags & HLLE_FALLBACK) {
      // intermediate states in the rotated order (rho, m_n, m_t1, m_t2, E)
      bool bad = false;
      for (int side = 0; side < 2; ++side) {
        const T* U = side == 0 ? UL : UR;
        const T al = side == 0 ? R.alpha[0] : -R.alpha[4];
        const T* K = side == 0 ? R.K[0] : R.K[4];
        const T rs = U[0] + al * K[0];
        const T mn = U[1 + n] + al * K[1], ma = U[1 + t1] + al * K[2], mb = U[1 + t2] + al * K[3];
        const T Es = U[4] + al * K[4];
        const T m2 = mn * mn + ma * ma + mb * mb;
        if (!(o_value(rs) > 0.0 && o_value(T(2.0) * rs * Es) > o_value(m2))) bad = true;
      }
      if (bad) {
        T bm = o_min(uL - aL, R.lambda[0]);
        bm = o_min(bm, T(0.0));
        T bp = -o_min(-(uR + aR), -R.lambda[4]);
        bp = -o_min(-bp, T(0.0));
        const T inv = T(1.0) / (bp - bm);
        for (int q = 0; q < 5; ++q) F[q] = ((bp * FL[q] - bm * FR[q]) + (bp * bm) * (UR[q] - UL[q])) * inv;
        if (used_hlle) *used_hlle = true;
        return;
      }
    }
    if (flags & ENTROPY_FIX) {
      // speed of the acoustic wave on its two sides: in the outer state and in the intermediate state next to it
      // (U*_L = UL + alpha_1 K_1 right of wave 1, U*_R = UR - alpha_5 K_5 left of wave 5); a non-physical
      // intermediate state leaves the wave unfixed
      for (int wave = 0; wave < 2; ++wave) {
        const T* U = wave == 0 ? UL : UR;
        const T al = wave == 0 ? R.alpha[0] : -R.alpha[4];
        const T* K = wave == 0 ? R.K[0] : R.K[4];
        const T sgn = wave == 0 ? T(-1.0) : T(1.0);
        const T rs = U[0] + al * K[0];
        const T mn = U[1 + n] + al * K[1], ma = U[1 + t1] + al * K[2], mb = U[1 + t2] + al * K[3];
        const T Es = U[4] + al * K[4];
        const T ps = (gamma - T(1.0)) * (Es - T(0.5) * (mn * mn + ma * ma + mb * mb) / rs);
        if (!(o_value(rs) > 0.0 && o_value(ps) > 0.0)) continue;
        const T lam_star = mn / rs + sgn * o_sqrt(gamma * ps / rs);
        const T lam_out = (wave == 0 ? uL : uR) + sgn * (wave == 0 ? aL : aR);
        const T lamL = wave == 0 ? lam_out : lam_star, lamR = wave == 0 ? lam_star : lam_out;
        const T lam = wave == 0 ? R.lambda[0] : R.lambda[4];
        T delta = -o_min(-(lam - lamL), -(lamR - lam));   // max of the two
        delta = -o_min(-delta, T(0.0));                   // max(0, .)
        T& absl = wave == 0 ? absl1 : absl5;
        if (o_value(absl) < o_value(delta)) absl = T(0.5) * (lam * lam / delta + delta);
      }
    }
  }
  // c_i = alpha_i |lambda_i|
  const T c1 = R.alpha[0] * absl1;
  const T c2 = R.alpha[1] * o_abs(R.lambda[1]);
  const T c3 = R.alpha[2] * o_abs(R.lambda[2]);
  const T c4 = R.alpha[3] * o_abs(R.lambda[3]);
  const T c5 = R.alpha[4] * absl5;
  // D = sum_i c_i K_i, component by component in the rotated order. Waves 1 and 5 are paired first so
  // that a mirror reflection reproduces the same bits (R21); structural 0/1 eigenvector entries
  // (K1[0]=K2[0]=K5[0]=1, K3[2]=K4[3]=1, the zeros of K3, K4) are written out, not multiplied.
  T D[5];
  D[0] = (c1 + c5) + c2;
  D[1] = (c1 * R.K[0][1] + c5 * R.K[4][1]) + c2 * R.K[1][1];
  D[2] = ((c1 * R.K[0][2] + c5 * R.K[4][2]) + c2 * R.K[1][2]) + c3;
  D[3] = ((c1 * R.K[0][3] + c5 * R.K[4][3]) + c2 * R.K[1][3]) + c4;
  D[4] = ((c1 * R.K[0][4] + c5 * R.K[4][4]) + c2 * R.K[1][4]) + (c3 * R.K[2][4] + c4 * R.K[3][4]);
  for (int q = 0; q < 5; ++q) {
    const int g = to_global[q];
    F[g] = T(0.5) * (FL[g] + FR[g]) - T(0.5) * D[q];
  }
}

// ---------------------------------------------------------------------------------------------------
// One step on a box of nx*ny*nz interior cells stored with a ghost shell of width g >= 2:
//   U_in [5][nz+2g][ny+2g][nx+2g]   (x fastest; interior cell (i,j,k) at (i+g, j+g, k+g))      [R13]
//   U_out[5][nz][ny][nx]
//   bflux: six arrays (nullable as a whole), flux density along +axis on the outer faces       [R12, O7]
//          face 0/1 = -x/+x : [5][nz][ny]   face 2/3 = -y/+y : [5][nz][nx]   face 4/5 = -z/+z : [5][ny][nx]
//          stored consecutively in that order; for a cubic group this is [6][5][N][N].
//   guard [(nz+2)][(ny+2)][(nx+2)] (nullable): 1 where the R7 fallback fired (cells of the set R only)
//   margin same shape (nullable): min over the six predicted face states of
//          (2 rho E - |m|^2) / (2 rho E), i.e. internal/total energy of the worst face state; it is a
//          diagnostic for the parity harness (cells with |margin| ~ eps can flip in fp32), not used here.
//   flags: RiemannFlags for O5 (default 0 = plain Roe).
//   midflux (nullable): the fluxes on the three MID-planes of the box (the faces at index n/2 - 1/2 along each axis,
//          between the two halves a group of 2 x 2 x 2 patches consists of; reading R12b): [3][5][.][.] in the
//          in-face layout of the outer faces of the same axis, x mid-plane first. Needs even nx, ny, nz.
//   hlle_faces (nullable): [3][nz+1][ny+1][nx+1] bytes, 1 where the face on the LOWER side of cell (i,j,k) along axis d
//          took the HLLE branch (flags & HLLE_FALLBACK): like `guard`, a diagnostic for the parity harness (a face whose
//          intermediate state is marginal can take the other branch in fp32), not used here. Entries of faces that do
//          not exist (index nx along y or z, ...) are left untouched.
// A patch group is the special case nx = ny = nz = N (O8: the per-group and global forms are the same text).
struct StepStats { unsigned long long guard_cells = 0, nonpositive_out = 0; };

template <class T>
StepStats step_box(const T* U_in, int nx, int ny, int nz, int g, T dt, T dx, T gamma, int limiter,
                   T* U_out, T* bflux, unsigned char* guard, double* margin, int flags = 0, T* midflux = nullptr,
                   unsigned char* hlle_faces = nullptr) {
  StepStats stats;
  const int sx = nx + 2 * g, sy = ny + 2 * g, sz = nz + 2 * g;
  const size_t plane = (size_t)sx * sy, vol = plane * sz;
  auto in_at = [&](int q, int i, int j, int k) -> const T& {  // interior-relative indices
    return U_in[q * vol + (size_t)(k + g) * plane + (size_t)(j + g) * sx + (i + g)];
  };
  // O0. lambda = dt/dx
  const T lam = dt / dx;

  // extended index space e = (i+2, j+2, k+2) over [-2, n+1]^3 for intermediates
  const int ex = nx + 4, ey = ny + 4, ez = nz + 4;
  auto eidx = [&](int i, int j, int k) -> size_t { return ((size_t)(k + 2) * ey + (j + 2)) * ex + (i + 2); };
  auto depth = [](int i, int n) { return i < 0 ? -i : (i >= n ? i - n + 1 : 0); };  // 0 interior, 1, 2
  const size_t evol = (size_t)ex * ey * ez;
  const double qnan = std::nan("");

  // O1. primitives on every cell whose value is ever read: depth triples (0,0,0),(1,0,0),(2,0,0),(1,1,0)
  // and permutations (7360 of the 8000 stored cells of a 16^3 group). Others stay NaN on purpose.
  std::vector<T> W(5 * evol, T(qnan));
  for (int k = -2; k < nz + 2; ++k)
    for (int j = -2; j < ny + 2; ++j)
      for (int i = -2; i < nx + 2; ++i) {
        const int a = depth(i, nx), b = depth(j, ny), c = depth(k, nz);
        // depth sums <= 2 are exactly the triples (0,0,0),(1,0,0),(2,0,0),(1,1,0) and permutations
        const bool needed = (a + b + c) <= 2;
        if (!needed) continue;
        T U[5], Wc[5];
        for (int q = 0; q < 5; ++q) U[q] = in_at(q, i, j, k);
        cons_to_prim(U, gamma, Wc);
        for (int q = 0; q < 5; ++q) W[q * evol + eidx(i, j, k)] = Wc[q];
      }

  // O2–O4. predicted face states Ubar[c][d][side][q] for c in R = interior + first-layer ghosts with
  // exactly one ghost index (5632 cells for a 16^3 group). side 0 = '-', 1 = '+'.
  std::vector<T> Ubar(30 * evol, T(qnan));
  auto ub = [&](int i, int j, int k, int d, int side, int q) -> T& {
    return Ubar[(((size_t)eidx(i, j, k) * 3 + d) * 2 + side) * 5 + q];
  };
  const int e[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
  for (int k = -1; k < nz + 1; ++k)
    for (int j = -1; j < ny + 1; ++j)
      for (int i = -1; i < nx + 1; ++i) {
        if (depth(i, nx) + depth(j, ny) + depth(k, nz) > 1) continue;
        T Wc[5], Wf[3][2][5], Uf[3][2][5];
        for (int q = 0; q < 5; ++q) Wc[q] = W[q * evol + eidx(i, j, k)];
        for (int d = 0; d < 3; ++d) {
          T* Wm = Wf[d][0];
          T* Wp = Wf[d][1];
          for (int q = 0; q < 5; ++q) {
            const T Wl = W[q * evol + eidx(i - e[d][0], j - e[d][1], k - e[d][2])];
            const T Wr = W[q * evol + eidx(i + e[d][0], j + e[d][1], k + e[d][2])];
            // O2 slopes
            const T dL = Wc[q] - Wl, dR = Wr - Wc[q];
            const T slope = limited_slope(dL, dR, limiter);
            // O3 face values W -+ 1/2 slope
            Wm[q] = Wc[q] - T(0.5) * slope;
            Wp[q] = Wc[q] + T(0.5) * slope;
          }
          prim_to_cons(Wm, gamma, Uf[d][0]);
          prim_to_cons(Wp, gamma, Uf[d][1]);
        }
        // O4 predictor: dU = -(lam/2) * sum_d [F_d(U_{d,+}) - F_d(U_{d,-})], differences first (R18)
        T dU[5];
        {
          T diff[3][5];
          for (int d = 0; d < 3; ++d) {
            T Fp[5], Fm[5];
            phys_flux(Uf[d][1], Wf[d][1], d, Fp);
            phys_flux(Uf[d][0], Wf[d][0], d, Fm);
            for (int q = 0; q < 5; ++q) diff[d][q] = Fp[q] - Fm[q];
          }
          for (int q = 0; q < 5; ++q) dU[q] = -(T(0.5) * lam) * ((diff[0][q] + diff[1][q]) + diff[2][q]);
        }
        bool ok = true;
        double worst = 1.0e300;
        T Up[3][2][5];
        for (int d = 0; d < 3; ++d)
          for (int s = 0; s < 2; ++s) {
            for (int q = 0; q < 5; ++q) Up[d][s][q] = Uf[d][s][q] + dU[q];
            // guard (R7): rho > 0 and 2 rho E > |m|^2, written so that NaN fails
            const T m2 = Up[d][s][1] * Up[d][s][1] + Up[d][s][2] * Up[d][s][2] + Up[d][s][3] * Up[d][s][3];
            const T twoRhoE = T(2.0) * Up[d][s][0] * Up[d][s][4];
            if (!(o_value(Up[d][s][0]) > 0.0 && o_value(twoRhoE) > o_value(m2))) ok = false;
            const double mg = (o_value(twoRhoE) - o_value(m2)) / o_value(twoRhoE);
            if (!(o_value(Up[d][s][0]) > 0.0)) worst = -1.0;
            else if (!(mg >= worst)) worst = (mg == mg) ? mg : -1.0;
          }
        if (!ok) {
          ++stats.guard_cells;
          for (int d = 0; d < 3; ++d)
            for (int s = 0; s < 2; ++s)
              for (int q = 0; q < 5; ++q) Up[d][s][q] = in_at(q, i, j, k);
        }
        for (int d = 0; d < 3; ++d)
          for (int s = 0; s < 2; ++s)
            for (int q = 0; q < 5; ++q) ub(i, j, k, d, s, q) = Up[d][s][q];
        const size_t gi = ((size_t)(k + 1) * (ny + 2) + (j + 1)) * (nx + 2) + (i + 1);
        if (guard) guard[gi] = ok ? 0 : 1;
        if (margin) margin[gi] = worst;
      }

  // O5. Roe flux at every face: index f in -1/2 .. n-1/2 along d, interior indices on the other axes.
  std::vector<T> F[3];
  size_t fstride[3][3];
  for (int d = 0; d < 3; ++d) {
    const int fx = nx + (d == 0), fy = ny + (d == 1), fz = nz + (d == 2);
    F[d].assign((size_t)5 * fx * fy * fz, T(qnan));
    fstride[d][0] = 1; fstride[d][1] = fx; fstride[d][2] = (size_t)fx * fy;
  }
  auto fl = [&](int d, int q, int i, int j, int k) -> T& {  // face on the LOWER side of cell (i,j,k) along d
    const int fx = nx + (d == 0), fy = ny + (d == 1), fz = nz + (d == 2);
    return F[d][(size_t)q * fx * fy * fz + (size_t)k * fstride[d][2] + (size_t)j * fstride[d][1] + i];
  };
  for (int d = 0; d < 3; ++d)
    for (int k = 0; k < nz + (d == 2); ++k)
      for (int j = 0; j < ny + (d == 1); ++j)
        for (int i = 0; i < nx + (d == 0); ++i) {
          T UL[5], UR[5], Ff[5];
          for (int q = 0; q < 5; ++q) {
            UL[q] = ub(i - e[d][0], j - e[d][1], k - e[d][2], d, 1, q);  // left cell's '+' state
            UR[q] = ub(i, j, k, d, 0, q);                                // right cell's '-' state
          }
          bool took_hlle = false;
          roe_flux(UL, UR, gamma, d, Ff, flags, &took_hlle);
          if (hlle_faces)   // diagnostic for the parity harness: which faces took the HLLE branch (R8c)
            hlle_faces[(((size_t)d * (nz + 1) + k) * (ny + 1) + j) * (nx + 1) + i] = took_hlle ? 1 : 0;
          for (int q = 0; q < 5; ++q) fl(d, q, i, j, k) = Ff[q];
        }

  // O6. conservative update from the INPUT conserved values, differences formed first (R18); no floor (R10).
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        T out[5];
        for (int q = 0; q < 5; ++q) {
          const T dFx = fl(0, q, i + 1, j, k) - fl(0, q, i, j, k);
          const T dFy = fl(1, q, i, j + 1, k) - fl(1, q, i, j, k);
          const T dFz = fl(2, q, i, j, k + 1) - fl(2, q, i, j, k);
          out[q] = in_at(q, i, j, k) - lam * ((dFx + dFy) + dFz);
          U_out[((size_t)q * nz + k) * ny * nx + (size_t)j * nx + i] = out[q];
        }
        const double m2 = o_value(out[1]) * o_value(out[1]) + o_value(out[2]) * o_value(out[2]) +
                          o_value(out[3]) * o_value(out[3]);
        if (!(o_value(out[0]) > 0.0 && 2.0 * o_value(out[0]) * o_value(out[4]) > m2)) ++stats.nonpositive_out;
      }

  // O7. boundary fluxes on the six outer faces (R12): lower in-face axis fastest.
  if (bflux) {
    T* p = bflux;
    for (int side = 0; side < 2; ++side)  // -x, +x : [5][nz][ny]
      for (int q = 0; q < 5; ++q)
        for (int k = 0; k < nz; ++k)
          for (int j = 0; j < ny; ++j) p[(((size_t)side * 5 + q) * nz + k) * ny + j] = fl(0, q, side ? nx : 0, j, k);
    p += (size_t)2 * 5 * nz * ny;
    for (int side = 0; side < 2; ++side)  // -y, +y : [5][nz][nx]
      for (int q = 0; q < 5; ++q)
        for (int k = 0; k < nz; ++k)
          for (int i = 0; i < nx; ++i) p[(((size_t)side * 5 + q) * nz + k) * nx + i] = fl(1, q, i, side ? ny : 0, k);
    p += (size_t)2 * 5 * nz * nx;
    for (int side = 0; side < 2; ++side)  // -z, +z : [5][ny][nx]
      for (int q = 0; q < 5; ++q)
        for (int j = 0; j < ny; ++j)
          for (int i = 0; i < nx; ++i) p[(((size_t)side * 5 + q) * ny + j) * nx + i] = fl(2, q, i, j, side ? nz : 0);
  }
  // O7b. mid-plane fluxes (R12b)
  if (midflux) {
    T* p = midflux;
    for (int q = 0; q < 5; ++q)
      for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j) p[((size_t)q * nz + k) * ny + j] = fl(0, q, nx / 2, j, k);
    p += (size_t)5 * nz * ny;
    for (int q = 0; q < 5; ++q)
      for (int k = 0; k < nz; ++k)
        for (int i = 0; i < nx; ++i) p[((size_t)q * nz + k) * nx + i] = fl(1, q, i, ny / 2, k);
    p += (size_t)5 * nz * nx;
    for (int q = 0; q < 5; ++q)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) p[((size_t)q * ny + j) * nx + i] = fl(2, q, i, j, nz / 2);
  }
  return stats;
}

}  // namespace mhm_oracle
