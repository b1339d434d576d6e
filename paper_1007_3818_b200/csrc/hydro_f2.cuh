// csrc/hydro_f2.cuh — packed `*.f32x2` arithmetic helpers (SASS FADD2 / FMUL2 / FFMA2) and the pieces of the
// MUSCL-Hancock + Roe step (readings of DESIGN.md §3) written with them: limiters, cons -> prim,
// predicted face state, Roe's solver in the primitive-jump form. Shared by the fp32 kernels hydro_zpair.cuh and
// hydro_duo.cuh (and by nothing under oracle/).
#pragma once
#include <cuda.h>
#include <stdint.h>
#include <string.h>

#include "hydro_fused.cuh"  // mbarrier / TMA helpers, GasConst, FN / FS

namespace gh {
// ---- packed pair of floats in one 64-bit register ---------------------------------------------------------
struct f2 {
  unsigned long long v;
};
__device__ __forceinline__ f2 mk2(float a, float b) {
  f2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ float lo(f2 a) {
  float x;
  asm("mov.b64 {%0, _}, %1;" : "=f"(x) : "l"(a.v));
  return x;
}
__device__ __forceinline__ float hi(f2 a) {
  float y;
  asm("mov.b64 {_, %0}, %1;" : "=f"(y) : "l"(a.v));
  return y;
}
__device__ __forceinline__ f2 splat(float c) { return mk2(c, c); }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) {
  f2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
  return r;
}
__device__ __forceinline__ f2 operator-(f2 a, f2 b) {
  f2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
  return r;
}
__device__ __forceinline__ f2 operator*(f2 a, f2 b) {
  f2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
  return r;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {
  f2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
  return r;
}
__device__ __forceinline__ f2 abs2(f2 a) { return mk2(fabsf(lo(a)), fabsf(hi(a))); }

__device__ __forceinline__ float rcp1(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsq1(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float sqrt1(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ f2 rcp2(f2 a) { return mk2(rcp1(lo(a)), rcp1(hi(a))); }
__device__ __forceinline__ f2 rsq2(f2 a) { return mk2(rsq1(lo(a)), rsq1(hi(a))); }
__device__ __forceinline__ f2 sqrt2(f2 a) { return mk2(sqrt1(lo(a)), sqrt1(hi(a))); }

// MinMod of one pair of one-sided differences (reading R3): sign(a) min(|a|,|b|) when the signs agree, else 0.
// min.xorsign.abs gives min(|a|,|b|) carrying sign(a) xor sign(b): negative exactly when the signs differ.
__device__ __forceinline__ float minmod1(float a, float b) {
  float d;
  asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return copysignf(fmaxf(d, 0.0f), a);
}
// van Leer (harmonic mean) limiter, zero when a b <= 0
__device__ __forceinline__ float vanleer1(float a, float b, float p, float s) {
  const float q = (p + p) * rcp1(s);
  return p > 0.0f ? q : 0.0f;
}
// MC (monotonized central, R3b): sign(a) min(2|a|, 2|b|, |a + b| / 2) when the signs agree, else 0
__device__ __forceinline__ float mc1(float a, float b, float s) {
  float d;
  asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));    // min(|a|,|b|), negative when the signs differ
  const float m = fminf(d + d, 0.5f * fabsf(s));
  return copysignf(fmaxf(m, 0.0f), a);
}
template <int LIM>
__device__ __forceinline__ f2 limited_slope2(f2 a, f2 b) {
  if (LIM == 0) {
    return mk2(minmod1(lo(a), lo(b)), minmod1(hi(a), hi(b)));
  } else if (LIM == 2) {
    const f2 s = a + b;
    return mk2(mc1(lo(a), lo(b), lo(s)), mc1(hi(a), hi(b), hi(s)));
  } else {
    // 2 a b / (a + b) with the doubling and the product packed (the same roundings as the scalar form), the
    // reciprocal and the sign test per lane
    const f2 p = a * b, q = (p + p) * rcp2(a + b);
    return mk2(lo(p) > 0.0f ? lo(q) : 0.0f, hi(p) > 0.0f ? hi(q) : 0.0f);
  }
}

// constants of one launch, pre-packed
struct PairConst {
  f2 g1, hg1n, gg1, gg1n, ig1, ig1n, lamn, hlamn, half, halfn, quartn, one, onen;
  float lam;
};
__host__ inline unsigned long long pack_host(float a) {
  unsigned int u;
  memcpy(&u, &a, 4);
  return ((unsigned long long)u << 32) | u;
}
__host__ inline PairConst make_pair_consts(float dt, float dx, float gamma) {
  PairConst c;
  const float g1 = gamma - 1.0f, lam = dt / dx;
  c.g1.v = pack_host(g1);
  c.hg1n.v = pack_host(-0.5f * g1);
  c.gg1.v = pack_host(gamma / g1);
  c.gg1n.v = pack_host(-(gamma / g1));
  c.ig1.v = pack_host(1.0f / g1);
  c.ig1n.v = pack_host(-(1.0f / g1));
  c.lamn.v = pack_host(-lam);
  c.hlamn.v = pack_host(-0.5f * lam);
  c.half.v = pack_host(0.5f);
  c.halfn.v = pack_host(-0.5f);
  c.quartn.v = pack_host(-0.25f);
  c.one.v = pack_host(1.0f);
  c.onen.v = pack_host(-1.0f);
  c.lam = lam;
  return c;
}

// a predicted face state as the Roe solver wants it
struct St2 {
  f2 r, u, v, w, p, h;  // rho, vx, vy, vz, P, H = (E + P) / rho
};

// ---- cons -> prim (step a0) -----------------------------------------------------------------------------------
__device__ __forceinline__ void cons2prim2(const f2 U[5], const PairConst& c, f2 W[5]) {
  const f2 r = rcp2(U[0]);
  W[0] = U[0];
  W[1] = U[1] * r;
  W[2] = U[2] * r;
  W[3] = U[3] * r;
  const f2 ke2 = fma2(U[3], W[3], fma2(U[2], W[2], U[1] * W[1]));
  W[4] = fma2(c.hg1n, ke2, c.g1 * U[4]);
}

// 3-input minimum that propagates NaN (so that a NaN state fails the guard)
__device__ __forceinline__ float min3nan(float a, float b, float c) {
  float d;
  asm("min.NaN.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
  return d;
}

// ---- D: Roe's solver (step a3; readings R8, R9), primitive-jump wave strengths -------------------------------------
// Flux density along +axis n in global component order. Every dissipation term is built with its minus sign
// (the quarter / half factors are negative constants) so that F = 1/2 (FL + FR) + Dneg is one fma per component.
template <int n>
__device__ __forceinline__ void roe2(const St2& L, const St2& R, const PairConst& c, f2 F[5]) {
  constexpr int t1 = (n + 1) % 3, t2 = (n + 2) % 3;
  const f2 Lv[3] = {L.u, L.v, L.w}, Rv[3] = {R.u, R.v, R.w};
  const f2 uL = Lv[n], vL = Lv[t1], wL = Lv[t2], uR = Rv[n], vR = Rv[t1], wR = Rv[t2];
  const f2 z = R.r * rsq2(L.r * R.r);             // sqrt(rhoR / rhoL) = rhoR / sqrt(rhoL rhoR)
  const f2 fR = z * rcp2(z + c.one);              // weight of the right state
  const f2 rt = L.r * z;                          // sqrt(rhoL rhoR)
  const f2 du = uR - uL, dv = vR - vL, dw = wR - wL, dH = R.h - L.h, dp = R.p - L.p, dr = R.r - L.r;
  const f2 u = fma2(fR, du, uL), v = fma2(fR, dv, vL), w = fma2(fR, dw, wL), H = fma2(fR, dH, L.h);
  const f2 q2 = fma2(w, w, fma2(v, v, u * u));
  const f2 a2 = fma2(c.hg1n, q2, c.g1 * H);
  const f2 hq = c.half * q2;
  const f2 rsa = rsq2(a2);
  const f2 a = a2 * rsa;
  const f2 t = dp * (rsa * rsa);                  // dp / a^2
  const f2 sg = (rt * du) * rsa;                  // rho~ du / a
  const f2 l1 = u - a, l5 = u + a;
  const float al1 = fabsf(lo(l1)), al5 = fabsf(lo(l5)), bl1 = fabsf(hi(l1)), bl5 = fabsf(hi(l5));
  const f2 P4n = c.quartn * mk2(al5 + al1, bl5 + bl1);
  const f2 M4n = c.quartn * mk2(al5 - al1, bl5 - bl1);
  const f2 sN = fma2(M4n, sg, P4n * t);           // -(c1 + c5) / 2
  const f2 dN = fma2(P4n, sg, M4n * t);           // -(c5 - c1) / 2
  const f2 aun = mk2(-0.5f * fabsf(lo(u)), -0.5f * fabsf(hi(u)));
  const f2 c2N = (dr - t) * aun;
  const f2 raN = rt * aun;
  const f2 c3N = raN * dv, c4N = raN * dw;
  const f2 D0 = sN + c2N;
  const f2 ad = a * dN;
  const f2 Dn = fma2(u, D0, ad);
  const f2 Dt1 = fma2(v, D0, c3N), Dt2 = fma2(w, D0, c4N);
  const f2 D4 = fma2(w, c4N, fma2(v, c3N, fma2(hq, c2N, fma2(u, ad, H * sN))));
  const f2 mL = L.r * uL, mR = R.r * uR;
  F[0] = fma2(c.half, mL + mR, D0);
  F[1 + n] = fma2(c.half, fma2(mL, uL, L.p) + fma2(mR, uR, R.p), Dn);
  F[1 + t1] = fma2(c.half, fma2(mL, vL, mR * vR), Dt1);
  F[1 + t2] = fma2(c.half, fma2(mL, wL, mR * wR), Dt2);
  F[4] = fma2(c.half, fma2(mL, L.h, mR * R.h), D4);
}

__device__ __forceinline__ f2 lds2(const float* p) {   // one 64-bit shared load (p is 8-byte aligned)
  f2 r;
  r.v = *reinterpret_cast<const unsigned long long*>(p);
  return r;
}
__device__ __forceinline__ void sts2(float* p, f2 a) { *reinterpret_cast<unsigned long long*>(p) = a.v; }

template <int LIM>
__device__ __forceinline__ float limited_slope1(float a, float b) {
  if (LIM == 0) return minmod1(a, b);
  if (LIM == 2) return mc1(a, b, a + b);
  const float p = a * b, s = a + b;
  return vanleer1(a, b, p, s);
}

constexpr int PRAW = 5 * FS * FS; // floats per raw plane (TMA box 20 x 20 x 1 x 5)

}  // namespace gh
