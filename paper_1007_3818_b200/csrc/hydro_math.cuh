// csrc/hydro_math.cuh — device arithmetic of the MUSCL-Hancock + Roe step, shared by the generic and the
// fused sm_100a kernels of this library (and by nothing else: the CPU oracle under oracle/ is a separate
// text). Follows PAPER.md:15 (the four steps) with the readings of DESIGN.md §3.
//
// Conventions: W = (rho, vx, vy, vz, P) primitives; U = (rho, mx, my, mz, E) conserved; axis n in {0,1,2}.
// `Fast` selects MUFU approximations (rcp/rsqrt, |rel err| ~ 1e-7) for float; double always uses IEEE ops.
#pragma once
#include <cuda_runtime.h>

namespace gh {

// Debug aid of the parity harness (gamer_hydro_set_guard_map, R7): when non-null, the kernels mark the cells
// whose predicted states fell back to first order in map[g][k+1][j+1][i+1] (unsigned char, (N+2)^3 per group). Read on
// the rare fallback path only.
__device__ unsigned char* gh_guard_map = nullptr;
__device__ __forceinline__ void mark_guard(long long g, int N, int i, int j, int k) {
  unsigned char* m = gh_guard_map;
  if (m) m[((g * (N + 2) + (k + 1)) * (N + 2) + (j + 1)) * (N + 2) + (i + 1)] = 1;
}

// The same for the HLLE fallback of the variant kernels (gamer_hydro_set_hlle_map): when non-null,
// a face that took the HLLE branch is marked in map[g][n][k][j][i], (N+1)^3 bytes per axis n, the face being the one on
// the lower side of cell (i, j, k) along n. Read on the fallback path only.
__device__ unsigned char* gh_hlle_map = nullptr;
__device__ __forceinline__ void mark_hlle(long long g, int N, int n, int i, int j, int k) {
  unsigned char* m = gh_hlle_map;
  if (m) m[(((g * 3 + n) * (N + 1) + k) * (N + 1) + j) * (N + 1) + i] = 1;
}

template <class R>
struct GasConst {
  R gamma;      // ratio of specific heats
  R g1;         // gamma - 1
  R ig1;        // 1 / (gamma - 1)
  R gg1;        // gamma / (gamma - 1)
  R lam;        // dt / dx
  R hlam;       // dt / (2 dx)
};

template <class R>
__host__ __device__ inline GasConst<R> make_consts(R dt, R dx, R gamma) {
  GasConst<R> c;
  c.gamma = gamma;
  c.g1 = gamma - R(1);
  c.ig1 = R(1) / (gamma - R(1));
  c.gg1 = gamma / (gamma - R(1));
  c.lam = dt / dx;
  c.hlam = R(0.5) * (dt / dx);
  return c;
}

// ---- scalar primitives -------------------------------------------------------------------------------
template <bool Fast>
__device__ __forceinline__ float rcp_(float x) {
  if (Fast) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
  }
  return 1.0f / x;
}
template <bool Fast>
__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }

template <bool Fast>
__device__ __forceinline__ float rsqrt_(float x) {
  if (Fast) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
  }
  return 1.0f / sqrtf(x);
}
template <bool Fast>
__device__ __forceinline__ double rsqrt_(double x) { return 1.0 / sqrt(x); }

__device__ __forceinline__ float min_(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double min_(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ double max_(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float abs_(float a) { return fabsf(a); }
__device__ __forceinline__ double abs_(double a) { return fabs(a); }

// ---- step 0: conserved -> primitive (ideal gas) -------------------------------------------------------
template <class R, bool Fast>
__device__ __forceinline__ void cons2prim(const R U[5], const GasConst<R>& c, R W[5]) {
  const R r = rcp_<Fast>(U[0]);
  W[0] = U[0];
  W[1] = U[1] * r;
  W[2] = U[2] * r;
  W[3] = U[3] * r;
  const R ke2 = U[1] * W[1] + U[2] * W[2] + U[3] * W[3];
  W[4] = c.g1 * (U[4] - R(0.5) * ke2);
}

// ---- step 1: limited slope ("spatial data reconstruction"; R3) --------------------
// MinMod written branch-free: max(0, min(dL,dR)) + min(0, max(dL,dR)) is sign(dL) min(|dL|,|dR|) when the
// signs agree and 0 otherwise (zero included).
template <class R, int LIM, bool Fast>
__device__ __forceinline__ R limited_slope(R dL, R dR) {
  if (LIM == 0) {
    return max_(R(0), min_(dL, dR)) + min_(R(0), max_(dL, dR));
  } else if (LIM == 2) {
    // MC (monotonized central, R3b): sign * min(2|dL|, 2|dR|, |dL + dR| / 2) when the signs agree
    const R m = min_(min_(R(2) * abs_(dL), R(2) * abs_(dR)), R(0.5) * abs_(dL + dR));
    return dL * dR > R(0) ? (dL > R(0) ? m : -m) : R(0);
  } else {
    const R p = dL * dR;
    const R s = dL + dR;
    const R q = (R(2) * p) * rcp_<Fast>(s);
    return p > R(0) ? q : R(0);
  }
}

// conserved state and own-direction flux of one face state given as primitives
template <class R, int n>
__device__ __forceinline__ void face_cons_flux(const R W[5], const GasConst<R>& c, R U[5], R F[5]) {
  U[0] = W[0];
  U[1] = W[0] * W[1];
  U[2] = W[0] * W[2];
  U[3] = W[0] * W[3];
  const R q = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  U[4] = (R(0.5) * W[0]) * q + W[4] * c.ig1;
  const R vn = W[1 + n];
  F[0] = U[1 + n];
  F[1] = U[1] * vn;
  F[2] = U[2] * vn;
  F[3] = U[3] * vn;
  F[1 + n] += W[4];
  F[4] = (U[4] + W[4]) * vn;
}

// ---- steps 1+2 for one cell: reconstruction and half-step prediction (R2-R7) -----
// In : Wc and its six neighbours' primitives.  Out: the six predicted face states as PRIMITIVES,
//      Wf[d][s] (d axis, s = 0 for the '-' face, 1 for '+').  Returns false when the positivity guard fired
//      (all six states were then replaced by the cell's own state, R7).
template <class R, int LIM, bool Fast>
__device__ __forceinline__ bool predict_cell(const R Wc[5], const R Wm[3][5], const R Wp[3][5],
                                             const GasConst<R>& c, R Wf[3][2][5]) {
  R Uf[3][2][5];
  R dF[5];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    R Wl[5], Wr[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      const R s = limited_slope<R, LIM, Fast>(Wc[q] - Wm[d][q], Wp[d][q] - Wc[q]);
      Wl[q] = Wc[q] - R(0.5) * s;
      Wr[q] = Wc[q] + R(0.5) * s;
    }
    R Fl[5], Fr[5];
    if (d == 0) { face_cons_flux<R, 0>(Wl, c, Uf[d][0], Fl); face_cons_flux<R, 0>(Wr, c, Uf[d][1], Fr); }
    if (d == 1) { face_cons_flux<R, 1>(Wl, c, Uf[d][0], Fl); face_cons_flux<R, 1>(Wr, c, Uf[d][1], Fr); }
    if (d == 2) { face_cons_flux<R, 2>(Wl, c, Uf[d][0], Fl); face_cons_flux<R, 2>(Wr, c, Uf[d][1], Fr); }
#pragma unroll
    for (int q = 0; q < 5; ++q) dF[q] = (d == 0) ? (Fr[q] - Fl[q]) : dF[q] + (Fr[q] - Fl[q]);
  }
  bool ok = true;
#pragma unroll
  for (int d = 0; d < 3; ++d)
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      R Ub[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) Ub[q] = Uf[d][s][q] - c.hlam * dF[q];
      cons2prim<R, Fast>(Ub, c, Wf[d][s]);
      // guard (R7): rho > 0 and P > 0 (for rho > 0, P > 0 <=> 2 rho E > |m|^2); NaN fails
      ok = ok && (Wf[d][s][0] > R(0)) && (Wf[d][s][4] > R(0));
    }
  if (!ok) {
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int q = 0; q < 5; ++q) Wf[d][s][q] = Wc[q];
  }
  return ok;
}

// ---- step 3: Roe's approximate Riemann solver (Roe 1981; R8, R9) -----------------
// Left/right states as primitives; returns the flux density along +axis n in global component order.
// Wave strengths in the primitive-jump (Roe–Pike) form, which is algebraically identical to the
// conserved-jump form the oracle uses:  a1,5 = (dp -+ rho~ a~ du)/(2 a~^2), a2 = drho - dp/a~^2,
// a3,4 = rho~ dv, rho~ dw with rho~ = sqrt(rhoL rhoR). flags = 0 (a literal in the default kernels, so the variant code
// folds away): plain Roe, no entropy fix. Bit 0: Harten-Hyman entropy fix; bit 1: HLLE fallback when an intermediate
// state of the linearisation is non-physical (readings R8b / R8c).
template <class R, int n, bool Fast>
__device__ __forceinline__ void roe_flux(const R L[5], const R Rt[5], const GasConst<R>& c, R F[5], int flags = 0,
                                         bool* took_hlle = nullptr) {
  constexpr int t1 = (n + 1) % 3, t2 = (n + 2) % 3;
  const R uL = L[1 + n], vL = L[1 + t1], wL = L[1 + t2];
  const R uR = Rt[1 + n], vR = Rt[1 + t1], wR = Rt[1 + t2];
  const R rsL = rsqrt_<Fast>(L[0]), rsR = rsqrt_<Fast>(Rt[0]);
  const R sL = L[0] * rsL, sR = Rt[0] * rsR;          // sqrt(rho)
  const R HL = (c.gg1 * L[4]) * (rsL * rsL) + R(0.5) * (uL * uL + vL * vL + wL * wL);
  const R HR = (c.gg1 * Rt[4]) * (rsR * rsR) + R(0.5) * (uR * uR + vR * vR + wR * wR);
  const R inv = rcp_<Fast>(sL + sR);
  const R fL = sL * inv, fR = sR * inv;
  const R u = fL * uL + fR * uR;
  const R v = fL * vL + fR * vR;
  const R w = fL * wL + fR * wR;
  const R H = fL * HL + fR * HR;
  const R hq = R(0.5) * (u * u + v * v + w * w);
  const R a2 = c.g1 * (H - hq);
  const R rsa = rsqrt_<Fast>(a2);
  const R a = a2 * rsa;
  const R rt = sL * sR;
  const R dr = Rt[0] - L[0], du = uR - uL, dv = vR - vL, dw = wR - wL, dp = Rt[4] - L[4];
  const R t = dp * (rsa * rsa);
  const R s = (rt * du) * rsa;
  const R um = u - a, up = u + a;
  const R mL = L[0] * uL, mR = Rt[0] * uR;
  R absl1 = abs_(um), absl5 = abs_(up);
  if (flags != 0) {
    // intermediate states U*_L = UL + alpha_1 K_1, U*_R = UR - alpha_5 K_5 (rotated conserved components)
    const R al1 = R(0.5) * (t - s), al5 = R(0.5) * (t + s), ua_ = u * a;
    const R EL = L[0] * HL - L[4], ER = Rt[0] * HR - Rt[4];
    const R r1 = L[0] + al1, n1 = mL + al1 * um, p1 = L[0] * vL + al1 * v, q1 = L[0] * wL + al1 * w, E1 = EL + al1 * (H - ua_);
    const R r5 = Rt[0] - al5, n5 = mR - al5 * up, p5 = Rt[0] * vR - al5 * v, q5 = Rt[0] * wR - al5 * w, E5 = ER - al5 * (H + ua_);
    const R k1 = n1 * n1 + p1 * p1 + q1 * q1, k5 = n5 * n5 + p5 * p5 + q5 * q5;
    const bool ok1 = r1 > R(0) && R(2) * r1 * E1 > k1, ok5 = r5 > R(0) && R(2) * r5 * E5 > k5;
    const R aL = sqrt(c.gamma * L[4] * (rsL * rsL)), aR = sqrt(c.gamma * Rt[4] * (rsR * rsR));
    if ((flags & 2) && !(ok1 && ok5)) {
      const R bm = min_(min_(uL - aL, um), R(0)), bp = max_(max_(uR + aR, up), R(0));
      const R inv_b = R(1) / (bp - bm), bb = bp * bm;
      F[0] = ((bp * mL - bm * mR) + bb * dr) * inv_b;
      F[1 + n] = ((bp * (mL * uL + L[4]) - bm * (mR * uR + Rt[4])) + bb * (mR - mL)) * inv_b;
      F[1 + t1] = ((bp * (mL * vL) - bm * (mR * vR)) + bb * (Rt[0] * vR - L[0] * vL)) * inv_b;
      F[1 + t2] = ((bp * (mL * wL) - bm * (mR * wR)) + bb * (Rt[0] * wR - L[0] * wL)) * inv_b;
      F[4] = ((bp * (mL * HL) - bm * (mR * HR)) + bb * (ER - EL)) * inv_b;
      if (took_hlle) *took_hlle = true;
      return;
    }
    if (flags & 1) {
      if (ok1) {
        const R ir = R(1) / r1;
        const R ls = n1 * ir - sqrt(c.gamma * (c.g1 * (E1 - R(0.5) * k1 * ir)) * ir);   // u* - a* right of wave 1
        const R delta = max_(R(0), max_(um - (uL - aL), ls - um));
        if (absl1 < delta) absl1 = R(0.5) * (um * um / delta + delta);
      }
      if (ok5) {
        const R ir = R(1) / r5;
        const R ls = n5 * ir + sqrt(c.gamma * (c.g1 * (E5 - R(0.5) * k5 * ir)) * ir);   // u* + a* left of wave 5
        const R delta = max_(R(0), max_(up - ls, (uR + aR) - up));
        if (absl5 < delta) absl5 = R(0.5) * (up * up / delta + delta);
      }
    }
  }
  // c_i = alpha_i |lambda_i|, with the overall factor 1/2 of the flux formula folded in
  const R c1 = (R(0.25) * (t - s)) * absl1;
  const R c5 = (R(0.25) * (t + s)) * absl5;
  const R au = R(0.5) * abs_(u);
  const R c2 = (dr - t) * au;
  const R c3 = (rt * dv) * au;
  const R c4 = (rt * dw) * au;
  const R D0 = (c1 + c5) + c2;
  const R Dn = (c1 * um + c5 * up) + c2 * u;
  const R Dt1 = D0 * v + c3;
  const R Dt2 = D0 * w + c4;
  const R ua = u * a;
  const R D4 = ((c1 * (H - ua) + c5 * (H + ua)) + c2 * hq) + (c3 * v + c4 * w);
  F[0] = R(0.5) * (mL + mR) - D0;
  F[1 + n] = R(0.5) * ((mL * uL + L[4]) + (mR * uR + Rt[4])) - Dn;
  F[1 + t1] = R(0.5) * (mL * vL + mR * vR) - Dt1;
  F[1 + t2] = R(0.5) * (mL * wL + mR * wR) - Dt2;
  F[4] = R(0.5) * (mL * HL + mR * HR) - D4;
}

}  // namespace gh
