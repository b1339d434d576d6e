// csrc/hydro_pair.cuh — the fp32 performance path for sm_100a: the fused MUSCL-Hancock + Roe step of
// PAPER.md:15 with TWO cells per thread, every add / mul / fma issued as a packed Blackwell `*.f32x2`
// instruction (SASS FADD2 / FMUL2 / FFMA2).
//
// Why (measured, profiles/r1a_README.md): the step is bound by instruction ISSUE, not by a pipe or by memory.
// FFMA2 & co. run at half the issue rate of their scalar forms, i.e. the same FLOP/s for half the issue slots,
// which leaves the other half to the shared-memory, MUFU and min/max instructions.
//
// Structure. N = 16. A CTA of 160 threads owns one patch group at a time and marches through
// its z planes k = -1 .. 16. The 320 cells of a plane whose predicted face states are needed (18 x 18 cross:
// interior + first ghost layer without the corners) are dealt out as 160 PAIRS (A, B) of cells of the same
// column i, 9 rows apart (8 in the two ghost columns): both halves of every packed register run the same
// instruction stream on two independent cells. Raw conserved planes arrive by TMA (5-D box loads) in a ring of
// shared-memory stages, one mbarrier per stage. Per plane:
//   A   cons -> prim of plane k+1 (own pair + the layer-2 / corner ghosts dealt to threads 0..33) -> primitive
//       plane in shared memory (float4 + float per cell, double-buffered)
//   B1  slopes, face values, own-direction face fluxes of plane k -> dU (half-step increment)
//   B2  the six predicted face states as (rho, u, v, w, P, H); guard (reading R7); x+ / y+ states published;
//       Roe flux at the lower z face (left state = previous plane's z+ state, kept in registers)
//   -- barrier --
//   D   Roe flux at the lower x and y faces; Fx, Fy published
//   -- barrier --
//   E   flux differences; conservative update of cell (i,j,k-1); U_out store; boundary-flux copy
// Two CTAs are resident per SM so that one CTA's barrier wait is covered by the other.
#pragma once
#include <cuda.h>
#include <stdint.h>

#include "hydro_fused.cuh"  // mbarrier / TMA helpers, GasConst

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
  float x, y;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a.v));
  return x;
}
__device__ __forceinline__ float hi(f2 a) {
  float x, y;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a.v));
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
template <int LIM>
__device__ __forceinline__ f2 limited_slope2(f2 a, f2 b) {
  if (LIM == 0) {
    return mk2(minmod1(lo(a), lo(b)), minmod1(hi(a), hi(b)));
  } else {
    const f2 p = a * b, s = a + b;
    return mk2(vanleer1(lo(a), lo(b), lo(p), lo(s)), vanleer1(hi(a), hi(b), hi(p), hi(s)));
  }
}

// constants of one launch, pre-packed
struct PairConst {
  f2 g1, hg1n, gg1, gg1n, ig1, lamn, hlamn, half, halfn, quartn, one, onen;
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

// ---- B1: one direction of the predictor: slopes, face values, flux difference accumulated into acc[] --------
// n = axis. s[q] receives the limited slope (not halved). acc[] (+)= F_n(W+) - F_n(W-) in global component order,
// with F_n = (m_n, m_n u + P e_n, (gg1 P + 1/2 rho q) u_n). nrho = -rho of the cell: the '-' face carries its
// minus sign on the density so that every term is one fma into the accumulator.
template <int n, int LIM, bool FIRST>
__device__ __forceinline__ void predict_dir(const f2 Wc[5], f2 nrho, const f2 dL[5], const f2 dR[5], const PairConst& c,
                                            f2 s[5], f2 acc[5]) {
  constexpr int t1 = (n + 1) % 3, t2 = (n + 2) % 3;
  f2 Wp[5], Wm[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    s[q] = limited_slope2<LIM>(dL[q], dR[q]);
    Wp[q] = fma2(c.half, s[q], Wc[q]);
    if (q > 0) Wm[q] = fma2(c.halfn, s[q], Wc[q]);
  }
  Wm[0] = fma2(c.half, s[0], nrho);  // -(rho - s/2)
  {
    const f2 mn = Wp[0] * Wp[1 + n];
    const f2 q = fma2(Wp[3], Wp[3], fma2(Wp[2], Wp[2], Wp[1] * Wp[1]));
    const f2 e = fma2(c.half * Wp[0], q, c.gg1 * Wp[4]);
    if (FIRST) {
      acc[0] = mn;
      acc[1 + n] = fma2(mn, Wp[1 + n], s[4]);  // P+ - P- = slope of P
      acc[1 + t1] = mn * Wp[1 + t1];
      acc[1 + t2] = mn * Wp[1 + t2];
      acc[4] = e * Wp[1 + n];
    } else {
      acc[0] = acc[0] + mn;
      acc[1 + n] = fma2(mn, Wp[1 + n], acc[1 + n] + s[4]);
      acc[1 + t1] = fma2(mn, Wp[1 + t1], acc[1 + t1]);
      acc[1 + t2] = fma2(mn, Wp[1 + t2], acc[1 + t2]);
      acc[4] = fma2(e, Wp[1 + n], acc[4]);
    }
  }
  {
    const f2 mn = Wm[0] * Wm[1 + n];  // -m_n
    const f2 q = fma2(Wm[3], Wm[3], fma2(Wm[2], Wm[2], Wm[1] * Wm[1]));
    const f2 e = fma2(c.half * Wm[0], q, c.gg1n * Wm[4]);  // -(gg1 P + 1/2 rho q)
    acc[0] = acc[0] + mn;
    acc[1 + n] = fma2(mn, Wm[1 + n], acc[1 + n]);
    acc[1 + t1] = fma2(mn, Wm[1 + t1], acc[1 + t1]);
    acc[1 + t2] = fma2(mn, Wm[1 + t2], acc[1 + t2]);
    acc[4] = fma2(e, Wm[1 + n], acc[4]);
  }
}

// 3-input minimum that propagates NaN (so that a NaN state fails the guard)
__device__ __forceinline__ float min3nan(float a, float b, float c) {
  float d;
  asm("min.NaN.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
  return d;
}

// ---- B2: one predicted face state (steps a1 tail + a2 of DESIGN.md §1) ------------------------------------------
// W = Wc +- s/2;  Ubar = U(W) + dU;  returned as (rho, v, P, H) of Ubar. gmin accumulates min(rho, P) over the
// states of the cell for the guard (reading R7). SIGN = +1 / -1.
template <int SIGN>
__device__ __forceinline__ St2 face_state(const f2 Wc[5], const f2 s[5], const f2 dU[5], const PairConst& c, f2& gmin) {
  const f2 hs = SIGN > 0 ? c.half : c.halfn;
  const f2 rho = fma2(hs, s[0], Wc[0]);
  const f2 u = fma2(hs, s[1], Wc[1]), v = fma2(hs, s[2], Wc[2]), w = fma2(hs, s[3], Wc[3]);
  const f2 P = fma2(hs, s[4], Wc[4]);
  const f2 rb = rho + dU[0];
  const f2 mx = fma2(rho, u, dU[1]), my = fma2(rho, v, dU[2]), mz = fma2(rho, w, dU[3]);
  const f2 q = fma2(w, w, fma2(v, v, u * u));
  const f2 Eb = fma2(c.half * rho, q, fma2(P, c.ig1, dU[4]));
  const f2 r = rcp2(rb);
  St2 o;
  o.r = rb;
  o.u = mx * r;
  o.v = my * r;
  o.w = mz * r;
  const f2 ke2 = fma2(mz, o.w, fma2(my, o.v, mx * o.u));
  o.p = fma2(c.hg1n, ke2, c.g1 * Eb);
  o.h = (Eb + o.p) * r;
  gmin = mk2(min3nan(lo(gmin), lo(rb), lo(o.p)), min3nan(hi(gmin), hi(rb), hi(o.p)));
  return o;
}

// ---- D: Roe's solver (step a3; readings R8, R9), primitive-jump wave strengths -------------------------------------
// Flux density along +axis n in global component order. Every dissipation term is built with its minus sign
// (the quarter / half factors are negative constants) so that F = 1/2 (FL + FR) + Dneg is one fma per component.
template <int n>
__device__ __forceinline__ void roe2(const St2& L, const St2& R, const PairConst& c, f2 F[5]) {
  constexpr int t1 = (n + 1) % 3, t2 = (n + 2) % 3;
  const f2 Lv[3] = {L.u, L.v, L.w}, Rv[3] = {R.u, R.v, R.w};
  const f2 uL = Lv[n], vL = Lv[t1], wL = Lv[t2], uR = Rv[n], vR = Rv[t1], wR = Rv[t2];
  const f2 z = sqrt2(R.r * rcp2(L.r));            // sqrt(rhoR / rhoL)
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

// ---- geometry of the pair kernel -----------------------------------------------------------------------------
constexpr int PNT = 160;          // threads per CTA = cell pairs per plane
#ifndef GH_PREGS
#define GH_PREGS 200
#endif
constexpr int PREGS = GH_PREGS;   // registers per thread: 2 CTAs x 5 warps x 32 x 200 = 64000 of the 65536 per SM
constexpr int PNSTAGE = 6;        // raw-plane ring depth
constexpr int PHALF = 162;        // slots per half: 9 thread rows x 18 columns
constexpr int PNSLOT = 392;       // 2 x 162 cross slots + 68 layer-2 / corner ghost slots
constexpr int PRAW = 5 * FS * FS; // floats per raw plane (TMA box 20 x 20 x 1 x 5)

struct PairSmem {
  static constexpr int raw_stage_bytes = ((PRAW * 4 + 127) / 128) * 128;
  static constexpr int raw_tx_bytes = PRAW * 4;
  static constexpr int arr = PNSLOT * 4;                     // one quantity of one plane
  static constexpr int off_raw = 0;
  static constexpr int off_w = off_raw + PNSTAGE * raw_stage_bytes;   // 2 primitive planes x 5
  static constexpr int off_xs = off_w + 2 * 5 * arr;                  // x+ states, 6 quantities
  static constexpr int off_ys = off_xs + 6 * arr;
  static constexpr int off_fx = off_ys + 6 * arr;                     // Fx, 5 components
  static constexpr int off_fy = off_fx + 5 * arr;
  static constexpr int off_bar = ((off_fy + 5 * arr + 15) / 16) * 16;
  static constexpr int total = off_bar + PNSTAGE * 8 + 16;
};

// Slot of cell (i, j) of a plane in the shared-memory arrays. The 320 cross cells are laid out in THREAD order
// (half, thread row, column) so that a warp's own-cell accesses are consecutive words; the 68 cells that are only
// ever neighbours (layer-2 ghosts, inner corners) follow. Cells that are never read map to slot 0.
__device__ __forceinline__ int pair_slot(int i, int j) {
  const bool in_x = (i >= 0 && i < FN), in_y = (j >= 0 && j < FN);
  if (in_x && j >= -1 && j <= FN) return j <= 7 ? (j + 1) * 18 + (i + 1) : PHALF + (j - 8) * 18 + (i + 1);
  if ((i == -1 || i == FN) && in_y) return j <= 7 ? (j + 1) * 18 + (i + 1) : PHALF + (j - 7) * 18 + (i + 1);
  if (i == -2 && in_y) return 324 + j;
  if (i == FN + 1 && in_y) return 340 + j;
  if (j == -2 && in_x) return 356 + i;
  if (j == FN + 1 && in_x) return 372 + i;
  if (i == -1 && j == -1) return 388;
  if (i == FN && j == -1) return 389;
  if (i == -1 && j == FN) return 390;
  if (i == FN && j == FN) return 391;
  return 0;
}

__device__ __forceinline__ void st_state(float* base, int slot_a, int slot_b, const St2& s) {
  const f2 q[6] = {s.r, s.u, s.v, s.w, s.p, s.h};
#pragma unroll
  for (int m = 0; m < 6; ++m) {
    base[m * PNSLOT + slot_a] = lo(q[m]);
    base[m * PNSLOT + slot_b] = hi(q[m]);
  }
}
__device__ __forceinline__ St2 ld_state(const float* base, int slot_a, int slot_b) {
  f2 q[6];
#pragma unroll
  for (int m = 0; m < 6; ++m) q[m] = mk2(base[m * PNSLOT + slot_a], base[m * PNSLOT + slot_b]);
  St2 s;
  s.r = q[0]; s.u = q[1]; s.v = q[2]; s.w = q[3]; s.p = q[4]; s.h = q[5];
  return s;
}
__device__ __forceinline__ f2 sel2(bool a, bool b, f2 x, f2 y) { return mk2(a ? lo(x) : lo(y), b ? hi(x) : hi(y)); }

template <int LIM>
__global__ void __maxnreg__(PREGS)
    pair_kernel(const __grid_constant__ CUtensorMap in_map, float* __restrict__ U_out, float* __restrict__ bflux,
                int n_groups, int goff, const __grid_constant__ PairConst c, unsigned long long* __restrict__ status) {
  using SM = PairSmem;
  extern __shared__ __align__(128) unsigned char smem[];
  float* const wring = reinterpret_cast<float*>(smem + SM::off_w);
  float* const xs = reinterpret_cast<float*>(smem + SM::off_xs);
  float* const ys = reinterpret_cast<float*>(smem + SM::off_ys);
  float* const fxs = reinterpret_cast<float*>(smem + SM::off_fx);
  float* const fys = reinterpret_cast<float*>(smem + SM::off_fy);
  const uint32_t raw_base = smem_u32(smem + SM::off_raw);
  const uint32_t bar_base = smem_u32(smem + SM::off_bar);

  // ---- thread -> pair of cells (A, B): same column i, rows jA and jB
  const int t = threadIdx.x;
  int r, col;
  if (t < 16) { r = 0; col = t + 1; }
  else { r = 1 + (t - 16) / 18; col = (t - 16) % 18; }
  const int i = col - 1;
  const bool in_x = (i >= 0 && i < FN);
  const int jA = r - 1, jB = in_x ? r + 8 : r + 7;
  const bool inA = in_x && jA >= 0, inB = in_x && jB < FN;               // interior cells
  const int oA = r * 18 + col, oB = oA + PHALF;                          // own slots
  const int nxmA = pair_slot(i - 1, jA), nxpA = pair_slot(i + 1, jA);    // neighbour slots
  const int nxmB = pair_slot(i - 1, jB), nxpB = pair_slot(i + 1, jB);
  const int nymA = pair_slot(i, jA - 1), nypA = pair_slot(i, jA + 1);
  const int nymB = pair_slot(i, jB - 1), nypB = pair_slot(i, jB + 1);
  const int rawA = (jA + 2) * FS + (i + 2), rawB = (jB + 2) * FS + (i + 2);
  const int outA = jA * FN + i, outB = jB * FN + i;
  // the layer-2 / corner ghosts this thread converts as well (threads 0..33 only)
  int eiA = 0, ejA = 0, eiB = 0, ejB = 0;
  if (t < 16) { eiA = -2; ejA = t; eiB = FN + 1; ejB = t; }
  else if (t < 32) { eiA = t - 16; ejA = -2; eiB = t - 16; ejB = FN + 1; }
  else if (t == 32) { eiA = -1; ejA = -1; eiB = FN; ejB = -1; }
  else if (t == 33) { eiA = -1; ejA = FN; eiB = FN; ejB = FN; }
  const bool has_extra = t < 34;
  const int rawEA = (ejA + 2) * FS + (eiA + 2), rawEB = (ejB + 2) * FS + (eiB + 2);
  const int oEA = pair_slot(eiA, ejA), oEB = pair_slot(eiB, ejB);
  // boundary-flux copy: thread -> (side, component, in-face index) of the x faces and of the y faces
  const int bf_side = t / 80, bf_q = (t % 80) / 16, bf_m = t % 16;
  const int bfx_slot = pair_slot(bf_side ? FN : 0, bf_m), bfy_slot = pair_slot(bf_m, bf_side ? FN : 0);

  const int n_local = (n_groups - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_planes = n_local * FPLANES;
  int issued = 0;
  auto issue_upto = [&](int limit) {  // thread 0 only
    if (limit > total_planes) limit = total_planes;
    while (issued < limit) {
      const int it = issued / FPLANES, p = issued % FPLANES;
      const int slot = issued % PNSTAGE;
      const int g = (int)blockIdx.x + it * (int)gridDim.x;
      const uint32_t bar = bar_base + 8 * slot;
      mbar_expect_tx(bar, SM::raw_tx_bytes);
      tma_load_plane(raw_base + slot * SM::raw_stage_bytes, &in_map, goff, goff, goff + p, g, bar);
      ++issued;
    }
  };
  if (t == 0) {
    for (int s = 0; s < PNSTAGE; ++s) mbar_init(bar_base + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (t == 0) issue_upto(PNSTAGE);

  auto raw_ptr = [&](int seq) -> const float* {
    return reinterpret_cast<const float*>(smem + SM::off_raw + (seq % PNSTAGE) * SM::raw_stage_bytes);
  };
  auto wait_plane = [&](int seq) { mbar_wait(bar_base + 8 * (seq % PNSTAGE), (seq / PNSTAGE) & 1); };
  // cons -> prim of this thread's pair of plane `seq`; optionally published in the primitive plane
  auto convert = [&](int seq, f2 W[5], bool publish, bool extras) {
    const float* raw = raw_ptr(seq);
    f2 U[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U[q] = mk2(raw[q * (FS * FS) + rawA], raw[q * (FS * FS) + rawB]);
    cons2prim2(U, c, W);
    if (publish) {
      float* wpl = wring + (seq & 1) * (5 * PNSLOT);
#pragma unroll
      for (int q = 0; q < 5; ++q) { wpl[q * PNSLOT + oA] = lo(W[q]); wpl[q * PNSLOT + oB] = hi(W[q]); }
      if (extras && has_extra) {
        f2 We[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) U[q] = mk2(raw[q * (FS * FS) + rawEA], raw[q * (FS * FS) + rawEB]);
        cons2prim2(U, c, We);
#pragma unroll
        for (int q = 0; q < 5; ++q) { wpl[q * PNSLOT + oEA] = lo(We[q]); wpl[q * PNSLOT + oEB] = hi(We[q]); }
      }
    }
  };

  unsigned int n_guard = 0, n_nonpos = 0;

  for (int it = 0; it < n_local; ++it) {
    const int g = (int)blockIdx.x + it * (int)gridDim.x;
    const int seq0 = it * FPLANES;  // sequence number of plane -2
    float* const outg = U_out + (size_t)g * (5 * FN * FN * FN);
    float* const bfg = bflux ? bflux + (size_t)g * (30 * FN * FN) : nullptr;

    f2 Wm[5], Wc[5], Wp[5], acc[5], Fzm[5];
    St2 zplus;
    wait_plane(seq0);
    convert(seq0, Wm, false, false);
    wait_plane(seq0 + 1);
    convert(seq0 + 1, Wc, true, false);
    zplus.r = zplus.u = zplus.v = zplus.w = zplus.p = zplus.h = c.one;
#pragma unroll
    for (int q = 0; q < 5; ++q) { acc[q] = c.one; Fzm[q] = c.one; }
    __syncthreads();

    for (int k = -1; k <= FN; ++k) {
      const int seq = seq0 + k + 2;  // sequence number of plane k
      const bool ghost_plane = (k < 0 || k >= FN);
      // ---- A: primitives of plane k+1
      wait_plane(seq + 1);
      convert(seq + 1, Wp, true, k + 1 < FN);

      // ---- B1: slopes, face values, own-direction fluxes -> dU
      const float* wpl = wring + (seq & 1) * (5 * PNSLOT);
      f2 sx[5], sy[5], sz[5], dU[5];
      {
        const f2 nrho = c.onen * Wc[0];
        f2 dL[5], dR[5], accF[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          dL[q] = Wc[q] - mk2(wpl[q * PNSLOT + nxmA], wpl[q * PNSLOT + nxmB]);
          dR[q] = mk2(wpl[q * PNSLOT + nxpA], wpl[q * PNSLOT + nxpB]) - Wc[q];
        }
        predict_dir<0, LIM, true>(Wc, nrho, dL, dR, c, sx, accF);
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          dL[q] = Wc[q] - mk2(wpl[q * PNSLOT + nymA], wpl[q * PNSLOT + nymB]);
          dR[q] = mk2(wpl[q * PNSLOT + nypA], wpl[q * PNSLOT + nypB]) - Wc[q];
        }
        predict_dir<1, LIM, false>(Wc, nrho, dL, dR, c, sy, accF);
#pragma unroll
        for (int q = 0; q < 5; ++q) { dL[q] = Wc[q] - Wm[q]; dR[q] = Wp[q] - Wc[q]; }
        predict_dir<2, LIM, false>(Wc, nrho, dL, dR, c, sz, accF);
#pragma unroll
        for (int q = 0; q < 5; ++q) dU[q] = c.hlamn * accF[q];
      }

      // ---- B2: the six predicted states; guard; publish x+ / y+; Roe at the lower z face
      f2 gmin = c.one;
      St2 xm = face_state<-1>(Wc, sx, dU, c, gmin);
      St2 ym = face_state<-1>(Wc, sy, dU, c, gmin);
      St2 zm = face_state<-1>(Wc, sz, dU, c, gmin);
      St2 zp = face_state<+1>(Wc, sz, dU, c, gmin);
      {
        St2 xp = face_state<+1>(Wc, sx, dU, c, gmin);
        St2 yp = face_state<+1>(Wc, sy, dU, c, gmin);
        if (!ghost_plane) { st_state(xs, oA, oB, xp); st_state(ys, oA, oB, yp); }
      }
      {
        // cells of the plane whose predicted states are used: the whole cross on interior planes, the interior on
        // the two ghost planes. Only those may count as guard failures.
        const bool useA = ghost_plane ? inA : true, useB = ghost_plane ? inB : true;
        const bool okA = lo(gmin) > 0.0f, okB = hi(gmin) > 0.0f;
        if (!(okA && okB)) {  // rare: first-order fallback for the failing cell(s) (reading R7)
          St2 fb;
          fb.r = Wc[0]; fb.u = Wc[1]; fb.v = Wc[2]; fb.w = Wc[3]; fb.p = Wc[4];
          const f2 q = fma2(Wc[3], Wc[3], fma2(Wc[2], Wc[2], Wc[1] * Wc[1]));
          fb.h = fma2(c.half, q, (c.gg1 * Wc[4]) * rcp2(Wc[0]));
          auto fix = [&](St2& s) {
            s.r = sel2(okA, okB, s.r, fb.r); s.u = sel2(okA, okB, s.u, fb.u); s.v = sel2(okA, okB, s.v, fb.v);
            s.w = sel2(okA, okB, s.w, fb.w); s.p = sel2(okA, okB, s.p, fb.p); s.h = sel2(okA, okB, s.h, fb.h);
          };
          fix(xm); fix(ym); fix(zm); fix(zp);
          if (!ghost_plane) {
            const float fbv[6][2] = {{lo(fb.r), hi(fb.r)}, {lo(fb.u), hi(fb.u)}, {lo(fb.v), hi(fb.v)},
                                     {lo(fb.w), hi(fb.w)}, {lo(fb.p), hi(fb.p)}, {lo(fb.h), hi(fb.h)}};
#pragma unroll
            for (int m = 0; m < 6; ++m) {
              if (!okA) { xs[m * PNSLOT + oA] = fbv[m][0]; ys[m * PNSLOT + oA] = fbv[m][0]; }
              if (!okB) { xs[m * PNSLOT + oB] = fbv[m][1]; ys[m * PNSLOT + oB] = fbv[m][1]; }
            }
          }
          n_guard += ((!okA && useA) ? 1u : 0u) + ((!okB && useB) ? 1u : 0u);
        }
      }
      f2 Fz[5];
      if (k >= 0) {
        roe2<2>(zplus, zm, c, Fz);
        if (bfg && (k == 0 || k == FN)) {
          float* p = bfg + (4 + (k == FN)) * (5 * FN * FN);
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            if (inA) p[q * (FN * FN) + outA] = lo(Fz[q]);
            if (inB) p[q * (FN * FN) + outB] = hi(Fz[q]);
          }
        }
      }
      zplus = zp;
      __syncthreads();  // S1: x+ / y+ states and primitive plane k+1 visible; raw planes <= k-2 retired
      if (t == 0) issue_upto(seq0 + k + 1 + PNSTAGE);

      if (!ghost_plane) {
        // ---- D: Roe fluxes at the lower x and y faces
        f2 Fx[5], Fy[5];
        {
          const St2 L = ld_state(xs, nxmA, nxmB);
          roe2<0>(L, xm, c, Fx);
        }
        {
          const St2 L = ld_state(ys, nymA, nymB);
          roe2<1>(L, ym, c, Fy);
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          fxs[q * PNSLOT + oA] = lo(Fx[q]); fxs[q * PNSLOT + oB] = hi(Fx[q]);
          fys[q * PNSLOT + oA] = lo(Fy[q]); fys[q * PNSLOT + oB] = hi(Fy[q]);
        }
        __syncthreads();  // S2: Fx, Fy visible
        // ---- E: finish cell (i,j,k-1) with its upper z flux, then start cell (i,j,k)
        if (k >= 1) {
          const float* rawp = raw_ptr(seq - 1);
          f2 out[5];
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            const f2 Uin = mk2(rawp[q * (FS * FS) + rawA], rawp[q * (FS * FS) + rawB]);
            out[q] = fma2(c.lamn, acc[q] + (Fz[q] - Fzm[q]), Uin);
            if (inA) outg[(size_t)q * (FN * FN * FN) + (k - 1) * (FN * FN) + outA] = lo(out[q]);
            if (inB) outg[(size_t)q * (FN * FN * FN) + (k - 1) * (FN * FN) + outB] = hi(out[q]);
          }
          const f2 m2 = fma2(out[3], out[3], fma2(out[2], out[2], out[1] * out[1]));
          const f2 tre = (out[0] + out[0]) * out[4];
          n_nonpos += (inA && !(lo(out[0]) > 0.0f && lo(tre) > lo(m2)) ? 1u : 0u) +
                      (inB && !(hi(out[0]) > 0.0f && hi(tre) > hi(m2)) ? 1u : 0u);
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const f2 fxr = mk2(fxs[q * PNSLOT + nxpA], fxs[q * PNSLOT + nxpB]);
          const f2 fyr = mk2(fys[q * PNSLOT + nypA], fys[q * PNSLOT + nypB]);
          acc[q] = (fxr - Fx[q]) + (fyr - Fy[q]);
          Fzm[q] = Fz[q];
        }
        if (bfg) {  // outer x and y faces of this plane: 2 sides x 5 components x 16 in-face cells each
          bfg[((bf_side * 5 + bf_q) * FN + k) * FN + bf_m] = fxs[bf_q * PNSLOT + bfx_slot];
          bfg[(((2 + bf_side) * 5 + bf_q) * FN + k) * FN + bf_m] = fys[bf_q * PNSLOT + bfy_slot];
        }
      } else if (k == FN) {
        const float* rawp = raw_ptr(seq - 1);
        f2 out[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const f2 Uin = mk2(rawp[q * (FS * FS) + rawA], rawp[q * (FS * FS) + rawB]);
          out[q] = fma2(c.lamn, acc[q] + (Fz[q] - Fzm[q]), Uin);
          if (inA) outg[(size_t)q * (FN * FN * FN) + (k - 1) * (FN * FN) + outA] = lo(out[q]);
          if (inB) outg[(size_t)q * (FN * FN * FN) + (k - 1) * (FN * FN) + outB] = hi(out[q]);
        }
        const f2 m2 = fma2(out[3], out[3], fma2(out[2], out[2], out[1] * out[1]));
        const f2 tre = (out[0] + out[0]) * out[4];
        n_nonpos += (inA && !(lo(out[0]) > 0.0f && lo(tre) > lo(m2)) ? 1u : 0u) +
                    (inB && !(hi(out[0]) > 0.0f && hi(tre) > hi(m2)) ? 1u : 0u);
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) { Wm[q] = Wc[q]; Wc[q] = Wp[q]; }
    }
    __syncthreads();  // all reads of this group's planes and exchange arrays done before the next group starts
  }

  for (int o = 16; o > 0; o >>= 1) {
    n_guard += __shfl_xor_sync(0xffffffffu, n_guard, o);
    n_nonpos += __shfl_xor_sync(0xffffffffu, n_nonpos, o);
  }
  if ((t & 31) == 0) {
    if (n_guard) atomicAdd(&status[0], (unsigned long long)n_guard);
    if (n_nonpos) atomicAdd(&status[1], (unsigned long long)n_nonpos);
  }
}

}  // namespace gh
