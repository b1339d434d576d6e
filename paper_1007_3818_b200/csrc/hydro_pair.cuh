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
// interior + first ghost layer without the corners) are dealt out as 160 PAIRS of cells: warps 0..3 own the
// 256 interior cells as x-adjacent pairs, warp 4 the 64 first-layer ghosts. Pairs are laid out in shared
// memory so that own and y-neighbour accesses are single 64-bit loads / stores into packed registers. Raw
// conserved planes arrive by TMA (5-D box loads) in a ring of shared-memory stages, one mbarrier per stage.
// ONE CTA barrier per plane: everything a neighbour publishes is double-buffered and consumed one phase later.
//   before the barrier of plane k:
//     A   cons -> prim of plane k+1 (own pair; warp 4 also the layer-2 / corner ghosts) -> primitive plane
//     B1  slopes, face values, own-direction face fluxes of plane k -> dU (half-step increment)
//     B2  the six predicted face states as (rho, u, v, w, P, H); guard (reading R7); x+ / y+ states published;
//         Roe flux at the lower z face (left state = previous plane's z+ state, kept in registers)
//   after it:
//     E   conservative update of cell (i,j,k-1) with the x / y fluxes of plane k-1 published one phase
//         earlier; U_out store; boundary-flux copy
//     D   Roe flux at the lower x and y faces of plane k; Fx, Fy published
// Two CTAs are resident per SM (168 registers, 3 warps per sub-partition).
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

// ---- geometry of the pair kernel -----------------------------------------------------------------------------
// 160 threads = 160 cell pairs (A, B) per plane = the 320 cells of the 18 x 18 cross whose predicted states are
// needed. Pairs are chosen so that both cells of a pair, and both cells of each of its neighbour pairs in y, sit
// in ADJACENT shared-memory slots: every own / y-neighbour access is one 64-bit LDS / STS straight into a packed
// register pair.
//   t <  128 : interior,   j = t / 8, A = (2p, j), B = (2p + 1, j), p = t % 8         (warps 0..3)
//   t <  144 : row ghosts, j = -1 (t < 136) or 16, A = (2p, j), B = (2p + 1, j)        (warp 4, lanes 0..15)
//   t <  160 : column ghosts, j = t - 144, A = (-1, j), B = (16, j)                    (warp 4, lanes 16..31)
// All five warps run the same instruction stream; only per-thread offsets differ.
constexpr int PNT = 160;          // threads per CTA = cell pairs per plane
#ifndef GH_PREGS
#define GH_PREGS 168
#endif
constexpr int PREGS = GH_PREGS;   // 168 registers x 32 lanes x 3 warps fill one SM sub-partition's 16384 registers
constexpr int PNSTAGE = 5;        // raw-plane ring depth
constexpr int PNSLOT = 388;       // slots of a primitive plane (320 cross cells + 68 layer-2 / corner ghosts)
constexpr int PNEX = 324;         // slots of an exchange array (interior + first ghost layer)
constexpr int PRAW = 5 * FS * FS; // floats per raw plane (TMA box 20 x 20 x 1 x 5)

struct PairSmem {
  static constexpr int raw_stage_bytes = ((PRAW * 4 + 127) / 128) * 128;
  static constexpr int raw_tx_bytes = PRAW * 4;
  static constexpr int off_raw = 0;
  static constexpr int off_w = off_raw + PNSTAGE * raw_stage_bytes;   // 2 buffers x 5 x PNSLOT primitives
  static constexpr int off_xs = off_w + 2 * 5 * PNSLOT * 4;           // 2 x 6 x PNEX   x+ states
  static constexpr int off_ys = off_xs + 2 * 6 * PNEX * 4;            // 2 x 6 x PNEX   y+ states
  static constexpr int off_fx = off_ys + 2 * 6 * PNEX * 4;            // 2 x 5 x PNEX   Roe fluxes at lower x faces
  static constexpr int off_fy = off_fx + 2 * 5 * PNEX * 4;            // 2 x 5 x PNEX   Roe fluxes at lower y faces
  static constexpr int off_bar = ((off_fy + 2 * 5 * PNEX * 4 + 15) / 16) * 16;
  static constexpr int off_sync = off_bar + PNSTAGE * 8;      // the CTA's split (arrive / wait) barrier
  static constexpr int total = off_sync + 16;
};

// Slot of cell (i, j) of a plane. Interior cells row-major; ghost columns as [j][side] and ghost rows as
// [side][i] so that the pairs named above are adjacent. Cells that are never read map to slot 0.
__device__ __forceinline__ int pair_slot(int i, int j) {
  const bool in_x = (i >= 0 && i < FN), in_y = (j >= 0 && j < FN);
  if (in_x && in_y) return FN * j + i;
  if ((i == -1 || i == FN) && j >= -1 && j <= FN) return 256 + 2 * (j + 1) + (i == FN ? 1 : 0);
  if ((j == -1 || j == FN) && in_x) return 292 + (j == FN ? FN : 0) + i;
  if ((j == -2 || j == FN + 1) && in_x) return 324 + (j == FN + 1 ? FN : 0) + i;
  if ((i == -2 || i == FN + 1) && in_y) return 356 + 2 * j + (i == FN + 1 ? 1 : 0);
  return 0;
}

__device__ __forceinline__ f2 lds2(const float* p) {   // one 64-bit shared load (p is 8-byte aligned)
  f2 r;
  r.v = *reinterpret_cast<const unsigned long long*>(p);
  return r;
}
__device__ __forceinline__ void sts2(float* p, f2 a) { *reinterpret_cast<unsigned long long*>(p) = a.v; }
__device__ __forceinline__ f2 sel2(bool a, bool b, f2 x, f2 y) { return mk2(a ? lo(x) : lo(y), b ? hi(x) : hi(y)); }
__device__ __forceinline__ void st_state2(float* base, int slot, const St2& s) {
  sts2(base + 0 * PNEX + slot, s.r); sts2(base + 1 * PNEX + slot, s.u); sts2(base + 2 * PNEX + slot, s.v);
  sts2(base + 3 * PNEX + slot, s.w); sts2(base + 4 * PNEX + slot, s.p); sts2(base + 5 * PNEX + slot, s.h);
}

#ifdef GH_PROBE
__device__ unsigned long long gh_probe[4 * 5 * 4];
#endif

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
  const uint32_t sync_bar = smem_u32(smem + SM::off_sync);

  // ---- thread -> pair of cells (A, B)
  const int t = threadIdx.x;
  const bool ghost_warp = t >= 128;  // warp-uniform: warp 4 owns the 64 first-layer ghost cells of a plane
  int iA, jA, iB, jB;
  if (t < 128) { jA = jB = t >> 3; iA = 2 * (t & 7); iB = iA + 1; }
  else if (t < 144) { jA = jB = (t < 136) ? -1 : FN; iA = 2 * (t & 7); iB = iA + 1; }
  else { jA = jB = t - 144; iA = -1; iB = FN; }
  const int own = pair_slot(iA, jA);                                     // B sits in slot own + 1
  const int xmA = pair_slot(iA - 1, jA), xpB = pair_slot(iB + 1, jB);    // outer x neighbours (scalar accesses)
  const int ym = pair_slot(iA, jA - 1), yp = pair_slot(iA, jA + 1);      // y neighbour pairs (64-bit accesses)
  const int rawA = (jA + 2) * FS + (iA + 2);
  // warp 4 only (recomputed where used so that they do not occupy registers in warps 0..3): the inner x
  // neighbours of a column-ghost pair are not the pair's own cells, and its raw cells are not adjacent
  auto xmB_of = [&]() { return pair_slot(iB - 1, jB); };
  auto xpA_of = [&]() { return pair_slot(iA + 1, jA); };
  auto rawB_of = [&]() { return (jB + 2) * FS + (iB + 2); };
  // Neighbours inside the exchange arrays (PNEX slots): where the thread's face is never used the offset falls
  // back to the thread's own slot, which always holds finite data.
  const int exA = xmA < PNEX ? xmA : own;   // used by warps 0..3 only

  const int n_local = (n_groups - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_planes = n_local * FPLANES;
  // TMA producer state (thread 0 only): next plane to request, kept incrementally (no div / mod on the hot path)
  int issued = 0, iss_p = 0, iss_g = (int)blockIdx.x;
  uint32_t iss_slot = 0;
  auto issue_upto = [&](int limit) {
    if (limit > total_planes) limit = total_planes;
#pragma unroll 1
    while (issued < limit) {
      const uint32_t bar = bar_base + 8 * iss_slot;
      mbar_expect_tx(bar, SM::raw_tx_bytes);
      tma_load_plane(raw_base + iss_slot * SM::raw_stage_bytes, &in_map, goff, goff, goff + iss_p, iss_g, bar);
      ++issued;
      if (++iss_p == FPLANES) { iss_p = 0; iss_g += (int)gridDim.x; }
      if (++iss_slot == PNSTAGE) iss_slot = 0;
    }
  };
  if (t == 0) {
    for (int s = 0; s < PNSTAGE; ++s) mbar_init(bar_base + 8 * s, 1);
    mbar_init(sync_bar, PNT);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (t == 0) issue_upto(PNSTAGE);
  // split barrier: arrive once this plane's data is published, wait before reading the neighbours' data
  uint32_t sync_phase = 0;
  auto cta_arrive = [&]() { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(sync_bar) : "memory"); };
#ifdef GH_PROBE
  unsigned long long probe_wait = 0, probe_t0 = clock64(), probe_A = 0, probe_conv = 0, probe_ta = 0;
  auto cta_wait = [&]() { const long long a = clock64(); mbar_wait(sync_bar, sync_phase); sync_phase ^= 1u; probe_wait += clock64() - a; };
#else
  auto cta_wait = [&]() { mbar_wait(sync_bar, sync_phase); sync_phase ^= 1u; };
#endif

  // raw-ring consumer state: slot and mbarrier phase of the next plane this thread converts
  uint32_t rs = 0, rph = 0;
  auto next_plane = [&]() -> const float* {
    mbar_wait(bar_base + 8 * rs, rph);
    const float* p = reinterpret_cast<const float*>(smem + SM::off_raw + rs * SM::raw_stage_bytes);
    if (++rs == PNSTAGE) { rs = 0; rph ^= 1u; }
    return p;
  };
  // conserved pair of a raw plane: one 64-bit load where the pair is adjacent in x (warps 0..3)
  auto load_pair = [&](const float* raw, int a, int b, f2 U[5]) {
    if (ghost_warp) {
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = mk2(raw[q * (FS * FS) + a], raw[q * (FS * FS) + b]);
    } else {
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = lds2(raw + q * (FS * FS) + a);
    }
  };
  auto publish_w = [&](float* wpl, int slot, const f2 W[5]) {
#pragma unroll
    for (int q = 0; q < 5; ++q) sts2(wpl + q * PNSLOT + slot, W[q]);
  };
  // warp 4 also converts the 68 cells of a plane that are only ever neighbours (layer-2 ghosts, inner corners)
  auto convert_extras = [&](const float* raw, float* wpl) {
    int a, b, slot;
    if (t < 144) { const int jj = (t < 136) ? -2 : FN + 1; a = (jj + 2) * FS + (iA + 2); b = a + 1; slot = (t < 136) ? ym : yp; }
    else { a = (jA + 2) * FS; b = a + FS - 1; slot = xmA; }  // (-2, j) and (17, j)
    f2 U[5], W[5];
    load_pair(raw, a, b, U);
    cons2prim2(U, c, W);
    publish_w(wpl, slot, W);
    if (t == 144 || t == 159) {  // inner corners (-1,-1),(16,-1) and (-1,16),(16,16)
      const int jj = (t == 144) ? -1 : FN;
      load_pair(raw, (jj + 2) * FS + 1, (jj + 2) * FS + FN + 2, U);
      cons2prim2(U, c, W);
      publish_w(wpl, t == 144 ? ym : yp, W);
    }
  };

  unsigned int n_guard = 0, n_nonpos = 0;

  for (int it = 0; it < n_local; ++it) {
    const int g = (int)blockIdx.x + it * (int)gridDim.x;
    const int seq0 = it * FPLANES;  // sequence number of plane -2 (even, so plane k lives in buffer k & 1)
    float* const outg = U_out + (size_t)g * (5 * FN * FN * FN);
    float* const bfg = bflux ? bflux + (size_t)g * (30 * FN * FN) : nullptr;

    f2 Wc[5], dLz[5], accd[5], Fz[5];
    St2 zplus;
    {  // prologue: planes -2 and -1 of the thread's own pair
      f2 U[5], Wm[5];
      load_pair(next_plane(), rawA, ghost_warp ? rawB_of() : 0, U);
      cons2prim2(U, c, Wm);
      load_pair(next_plane(), rawA, ghost_warp ? rawB_of() : 0, U);
      cons2prim2(U, c, Wc);
      publish_w(wring + 5 * PNSLOT, own, Wc);
#pragma unroll
      for (int q = 0; q < 5; ++q) { dLz[q] = Wc[q] - Wm[q]; accd[q] = c.one; Fz[q] = c.one; }
      zplus.r = zplus.u = zplus.v = zplus.w = zplus.p = zplus.h = c.one;
    }
    __syncthreads();
    if (t == 0) issue_upto(seq0 + 2 + PNSTAGE);

    for (int k = -1; k <= FN; ++k) {
      const int buf = k & 1;
      const bool ghost_plane = (k < 0 || k >= FN);
      const bool active = !(ghost_warp && ghost_plane);  // warp-uniform: ghost cells of ghost planes are never used

      // ---- A: primitives of plane k+1 (own pair; warp 4 also the cells that are only neighbours)
#ifdef GH_PROBE
      probe_ta = clock64();
#endif
      f2 Wp[5];
      {
        const float* raw = next_plane();  // plane k+1
        f2 U[5];
        load_pair(raw, rawA, ghost_warp ? rawB_of() : 0, U);
        cons2prim2(U, c, Wp);
        float* wpl = wring + (buf ^ 1) * (5 * PNSLOT);
        if (k + 1 <= FN) publish_w(wpl, own, Wp);
        if (ghost_warp && k + 1 >= 0 && k + 1 < FN) convert_extras(raw, wpl);
      }
#ifdef GH_PROBE
      probe_conv += clock64() - probe_ta;
#endif
      f2 dRz[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) dRz[q] = Wp[q] - Wc[q];

#pragma unroll
      for (int q = 0; q < 5; ++q) { const f2 d = dRz[q]; dRz[q] = dLz[q]; dLz[q] = d; }  // dRz: lower, dLz: upper difference

      St2 xm, ymS;
      if (active) {
        // ---- B1: slopes, face values, own-direction fluxes -> dU
        const float* wpl = wring + buf * (5 * PNSLOT);
        f2 sx[5], sy[5], sz[5], dU[5];
        {
          const f2 nrho = c.onen * Wc[0];
          f2 dL[5], dR[5], accF[5];
          if (ghost_warp) {
            const int xmB = xmB_of(), xpA = xpA_of();
#pragma unroll
            for (int q = 0; q < 5; ++q) {
              dL[q] = Wc[q] - mk2(wpl[q * PNSLOT + xmA], wpl[q * PNSLOT + xmB]);
              dR[q] = mk2(wpl[q * PNSLOT + xpA], wpl[q * PNSLOT + xpB]) - Wc[q];
            }
          } else {  // x-adjacent pair: the inner neighbours are the pair's own cells
#pragma unroll
            for (int q = 0; q < 5; ++q) {
              dL[q] = Wc[q] - mk2(wpl[q * PNSLOT + xmA], lo(Wc[q]));
              dR[q] = mk2(hi(Wc[q]), wpl[q * PNSLOT + xpB]) - Wc[q];
            }
          }
          predict_dir<0, LIM, true>(Wc, nrho, dL, dR, c, sx, accF);
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            dL[q] = Wc[q] - lds2(wpl + q * PNSLOT + ym);
            dR[q] = lds2(wpl + q * PNSLOT + yp) - Wc[q];
          }
          predict_dir<1, LIM, false>(Wc, nrho, dL, dR, c, sy, accF);
          predict_dir<2, LIM, false>(Wc, nrho, dRz, dLz, c, sz, accF);
#pragma unroll
          for (int q = 0; q < 5; ++q) dU[q] = c.hlamn * accF[q];
        }

        // ---- B2: the six predicted states; guard; publish x+ / y+; Roe at the lower z face
        // ---- B2: the six predicted states; guard; publish x+ / y+
        f2 gmin = c.one;
        {
          const St2 xpS = face_state<+1>(Wc, sx, dU, c, gmin);
          if (!ghost_plane) st_state2(xs + buf * (6 * PNEX), own, xpS);
        }
        {
          const St2 ypS = face_state<+1>(Wc, sy, dU, c, gmin);
          if (!ghost_plane) st_state2(ys + buf * (6 * PNEX), own, ypS);
        }
        xm = face_state<-1>(Wc, sx, dU, c, gmin);
        ymS = face_state<-1>(Wc, sy, dU, c, gmin);
        St2 zm = face_state<-1>(Wc, sz, dU, c, gmin);
        St2 zp = face_state<+1>(Wc, sz, dU, c, gmin);
        {
          const bool okA = lo(gmin) > 0.0f, okB = hi(gmin) > 0.0f;
          if (__builtin_expect(!(okA && okB), 0)) {  // rare: first-order fallback for the failing cell(s) (reading R7)
            St2 fb;
            fb.r = Wc[0]; fb.u = Wc[1]; fb.v = Wc[2]; fb.w = Wc[3]; fb.p = Wc[4];
            const f2 q = fma2(Wc[3], Wc[3], fma2(Wc[2], Wc[2], Wc[1] * Wc[1]));
            fb.h = fma2(c.half, q, (c.gg1 * Wc[4]) * rcp2(Wc[0]));
            auto fix = [&](St2& s) {
              s.r = sel2(okA, okB, s.r, fb.r); s.u = sel2(okA, okB, s.u, fb.u); s.v = sel2(okA, okB, s.v, fb.v);
              s.w = sel2(okA, okB, s.w, fb.w); s.p = sel2(okA, okB, s.p, fb.p); s.h = sel2(okA, okB, s.h, fb.h);
            };
            fix(xm); fix(ymS); fix(zm); fix(zp);
            if (!ghost_plane) {
              float* xsb = xs + buf * (6 * PNEX);
              float* ysb = ys + buf * (6 * PNEX);
              const float fbv[6][2] = {{lo(fb.r), hi(fb.r)}, {lo(fb.u), hi(fb.u)}, {lo(fb.v), hi(fb.v)},
                                       {lo(fb.w), hi(fb.w)}, {lo(fb.p), hi(fb.p)}, {lo(fb.h), hi(fb.h)}};
#pragma unroll
              for (int m = 0; m < 6; ++m) {
                if (!okA) { xsb[m * PNEX + own] = fbv[m][0]; ysb[m * PNEX + own] = fbv[m][0]; }
                if (!okB) { xsb[m * PNEX + own + 1] = fbv[m][1]; ysb[m * PNEX + own + 1] = fbv[m][1]; }
              }
            }
            n_guard += (okA ? 0u : 1u) + (okB ? 0u : 1u);   // every cell that gets here is one whose states are used
          }
        }
        // everything the neighbours need from this thread is published: arrive, then do the work that needs
        // no neighbour (the z face) while the other warps catch up
#ifdef GH_PROBE
        probe_A += clock64() - probe_ta;
#endif
        cta_arrive();
        if (!ghost_warp && k >= 0) {
          f2 Fn[5];
          roe2<2>(zplus, zm, c, Fn);
#pragma unroll
          for (int q = 0; q < 5; ++q) { accd[q] = Fn[q] - accd[q]; Fz[q] = Fn[q]; }  // upper z flux minus the lower-face sum
          if (bfg && (k == 0 || k == FN)) {
            float* p = bfg + (4 + (k == FN)) * (5 * FN * FN) + own;
#pragma unroll
            for (int q = 0; q < 5; ++q) sts2(p + q * (FN * FN), Fn[q]);
          }
        }
        zplus = zp;
      } else {
        cta_arrive();
      }
      cta_wait();  // x+ / y+ states of plane k, primitives of plane k+1, fluxes of plane k-1 visible
      if (t == 0) issue_upto(seq0 + k + 1 + PNSTAGE);

      // ---- E: conservative update of plane k-1 (its x / y fluxes were published before this barrier)
      if (!ghost_warp && k >= 1) {
        const float* fxb = fxs + (buf ^ 1) * (5 * PNEX);
        const float* fyb = fys + (buf ^ 1) * (5 * PNEX);
        const int us = (int)rs - 3 + ((int)rs < 3 ? PNSTAGE : 0);  // slot of plane k-1 (rs points at plane k+2)
        const float* rawp = reinterpret_cast<const float*>(smem + SM::off_raw + us * SM::raw_stage_bytes);
        float* op = outg + (k - 1) * (FN * FN) + own;
        f2 out[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const f2 Uin = lds2(rawp + q * (FS * FS) + rawA);
          const f2 ux = mk2(fxb[q * PNEX + own + 1], fxb[q * PNEX + xpB]);
          const f2 uy = lds2(fyb + q * PNEX + yp);
          out[q] = fma2(c.lamn, (ux + uy) + accd[q], Uin);
          sts2(op + (size_t)q * (FN * FN * FN), out[q]);
        }
        const f2 m2 = fma2(out[3], out[3], fma2(out[2], out[2], out[1] * out[1]));
        const f2 tre = (out[0] + out[0]) * out[4];
        n_nonpos += (!(lo(out[0]) > 0.0f && lo(tre) > lo(m2)) ? 1u : 0u) +
                    (!(hi(out[0]) > 0.0f && hi(tre) > hi(m2)) ? 1u : 0u);
      }
      // ---- D: Roe fluxes at the lower x and y faces of plane k
      if (!ghost_plane && !ghost_warp) {
        const float* xsb = xs + buf * (6 * PNEX);
        const float* ysb = ys + buf * (6 * PNEX);
        float* fxo = fxs + buf * (5 * PNEX) + own;
        float* fyo = fys + buf * (5 * PNEX) + own;
        f2 Fx[5], Fy[5];
        {  // faces (iA - 1/2) and (iA + 1/2): the second one lies between the pair's own cells
          St2 L;
          L.r = mk2(xsb[0 * PNEX + exA], xsb[0 * PNEX + own]); L.u = mk2(xsb[1 * PNEX + exA], xsb[1 * PNEX + own]);
          L.v = mk2(xsb[2 * PNEX + exA], xsb[2 * PNEX + own]); L.w = mk2(xsb[3 * PNEX + exA], xsb[3 * PNEX + own]);
          L.p = mk2(xsb[4 * PNEX + exA], xsb[4 * PNEX + own]); L.h = mk2(xsb[5 * PNEX + exA], xsb[5 * PNEX + own]);
          roe2<0>(L, xm, c, Fx);
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) sts2(fxo + q * PNEX, Fx[q]);
        {
          St2 L;
          L.r = lds2(ysb + 0 * PNEX + ym); L.u = lds2(ysb + 1 * PNEX + ym); L.v = lds2(ysb + 2 * PNEX + ym);
          L.w = lds2(ysb + 3 * PNEX + ym); L.p = lds2(ysb + 4 * PNEX + ym); L.h = lds2(ysb + 5 * PNEX + ym);
          roe2<1>(L, ymS, c, Fy);
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          sts2(fyo + q * PNEX, Fy[q]);
          accd[q] = (Fx[q] + Fy[q]) + Fz[q];  // sum of the lower-face fluxes of plane k
        }
        // a5: outer faces -x (cells i = 0) and -y (row 0) of this plane
        if (bfg) {
          if (iA == 0) {
#pragma unroll
            for (int q = 0; q < 5; ++q) bfg[(q * FN + k) * FN + jA] = lo(Fx[q]);
          }
          if (t < 8) {
#pragma unroll
            for (int q = 0; q < 5; ++q) sts2(bfg + ((10 + q) * FN + k) * FN + iA, Fy[q]);
          }
        }
      } else if (!ghost_plane && t >= 136) {
        // Warp 4: the only faces its cells own are x = 15.5 (B cells of the column ghosts) and y = 15.5 (row 16).
        // One solve does both: the row-16 lanes rotate their states so that y is the normal direction.
        const float* xsb = xs + buf * (6 * PNEX);
        const float* ysb = ys + buf * (6 * PNEX);
        const bool rowl = t < 144;
        St2 L, R;
        if (rowl) {
          R.r = ymS.r; R.u = ymS.v; R.v = ymS.w; R.w = ymS.u; R.p = ymS.p; R.h = ymS.h;
          L.r = lds2(ysb + 0 * PNEX + ym); L.u = lds2(ysb + 2 * PNEX + ym); L.v = lds2(ysb + 3 * PNEX + ym);
          L.w = lds2(ysb + 1 * PNEX + ym); L.p = lds2(ysb + 4 * PNEX + ym); L.h = lds2(ysb + 5 * PNEX + ym);
        } else {
          const int exB = xmB_of();  // cell (15, j)
          R = xm;
          L.r = mk2(lo(xm.r), xsb[0 * PNEX + exB]); L.u = mk2(lo(xm.u), xsb[1 * PNEX + exB]);
          L.v = mk2(lo(xm.v), xsb[2 * PNEX + exB]); L.w = mk2(lo(xm.w), xsb[3 * PNEX + exB]);
          L.p = mk2(lo(xm.p), xsb[4 * PNEX + exB]); L.h = mk2(lo(xm.h), xsb[5 * PNEX + exB]);
        }
        f2 F[5];
        roe2<0>(L, R, c, F);
        if (rowl) {  // rotated back: normal -> my, first transverse -> mz, second -> mx
          float* fyo = fys + buf * (5 * PNEX) + own;
          sts2(fyo + 0 * PNEX, F[0]); sts2(fyo + 1 * PNEX, F[3]); sts2(fyo + 2 * PNEX, F[1]);
          sts2(fyo + 3 * PNEX, F[2]); sts2(fyo + 4 * PNEX, F[4]);
          if (bfg) {
            float* p = bfg + (15 * FN + k) * FN + iA;
            sts2(p + 0 * (FN * FN), F[0]); sts2(p + 1 * (FN * FN), F[3]); sts2(p + 2 * (FN * FN), F[1]);
            sts2(p + 3 * (FN * FN), F[2]); sts2(p + 4 * (FN * FN), F[4]);
          }
        } else {
          float* fxo = fxs + buf * (5 * PNEX) + own;
#pragma unroll
          for (int q = 0; q < 5; ++q) sts2(fxo + q * PNEX, F[q]);
          if (bfg) {
#pragma unroll
            for (int q = 0; q < 5; ++q) bfg[((5 + q) * FN + k) * FN + jA] = hi(F[q]);
          }
        }
      }
      if (k < FN) {
        const float* wnx = wring + (buf ^ 1) * (5 * PNSLOT) + own;
#pragma unroll
        for (int q = 0; q < 5; ++q) Wc[q] = lds2(wnx + q * PNSLOT);
      }
    }
  }

#ifdef GH_PROBE
  if ((t & 31) == 0 && blockIdx.x < 4) {
    unsigned int wid, smid;
    asm volatile("mov.u32 %0, %%warpid;" : "=r"(wid));
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    unsigned long long* pr = gh_probe + (blockIdx.x * 5 + (t >> 5)) * 4;
    pr[0] = probe_wait; pr[1] = clock64() - probe_t0; pr[2] = probe_A; pr[3] = probe_conv;
  }
#endif
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
