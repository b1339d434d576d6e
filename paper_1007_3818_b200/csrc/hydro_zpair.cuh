// csrc/hydro_zpair.cuh — fp32 performance path, variant "z-pair": every thread owns ONE column (i, j) of the
// 18 x 18 cross of a patch group and marches it TWO z planes at a time; the two lanes of every Blackwell `*.f32x2`
// instruction (SASS FADD2 / FMUL2 / FFMA2) carry the planes (2p-1, 2p) of that column.
//
// Why (profiles/r1d_README.md): the step is bound by instruction issue and by the FMA pipe. With the
// planes of a pair in the two lanes ALL arithmetic of the step is packed — the predictor, the x, y AND z Roe solves,
// the update — every neighbour exchange is ONE 64-bit shared-memory access straight into a packed register (the
// exchange arrays hold plane pairs), and the per-plane bookkeeping (barriers, TMA waits, loop) is paid once per two
// planes (968 -> 645 thread-instructions per cell-update against the one-cell kernel; a packed instruction still costs
// the scheduler two clocks — profiles/r2b_README.md — so it is the non-FP half of the stream that shrinks). Lane
// crossing happens only along z and only through registers: the z slopes use the scalar differences
// W(2p-1) - W(2p-2), W(2p) - W(2p-1), W(2p+1) - W(2p); the z-face solve takes its left states as
// (z+ of plane 2p-2 kept from the previous pair, z+ of plane 2p-1) and its right states as the pair's z- states.
//
// Structure. N = 16, ghost = 2. One CTA of 320 threads (10 warps) per SM streams patch groups through a flat
// pipeline of SLOTS, 11 per group: slot gs handles the plane pair (2 gs - 3, 2 gs - 2), gs = 0 .. 10; gs = 1 .. 9 are
// the nine pairs (-1,0) .. (15,16) whose predicted states are needed, gs = 0 / 10 only convert / update.
//   warps 0..7  interior cells, j = t / 16, i = t % 16 (a half-warp = one row: 64-bit accesses are conflict-free)
//   warp  8     "upper" ghosts: column i = 16 (lanes 0..15) and row j = 16 (lanes 16..31): own '-' state along the
//               normal + the Roe solve of the face they own
//   warp  9     "lower" ghosts: column i = -1 and row j = -1: own '+' state along the normal; also the TMA producer
//               and the x / y boundary-flux stores (the 68 neighbour-only cells of the conversion go to warps 2, 3, 6, 7)
// All ten warps run ONE instruction stream with the same arithmetic (a ghost column is predicted exactly like an
// interior one, so data uniform along an axis stay bit-identically uniform); the roles differ in a few warp-uniform
// branches and in which states a lane publishes or keeps.
// Per slot s (plane pair s of the flat sequence; everything a neighbour publishes is double-buffered):
//   C  cons -> prim of pair s+1 (raw pairs arrive by TMA: box 20 x 20 x 2 x 5, ring of ZNS stages) -> W[(s+1)&1]
//   P  slopes, face values, own-direction fluxes -> dU, the six predicted states, guard (reading R7);
//      x+ / y+ states -> S[s&1];                                            arrive(S)
//   Z  (interior) packed Roe solve at the two lower z faces of the pair (own registers only)
//      wait(S)
//   R  packed Roe solves at the lower x and the lower y face of the pair -> F[s&1]
//   U  (interior) conservative update of pair s-1 from F[(s-1)&1], U_out stores; (warp 9) boundary fluxes of pair s-1
// ONE split barrier per slot (mbarrier, arrive by one elected lane per warp / try_wait): everything a warp publishes in
// slot s — W[(s+1)&1] in C, S[s&1] in P, F[(s-1)&1] in the R of slot s-1 — is ordered before its arrive(S) of slot s;
// a warp that has passed wait(S) of slot s therefore sees the states of pair s, the fluxes of pair s-1 and the
// primitives of pair s+1, and knows that every warp has finished slot s-1 (so S[s&1], F[s&1] and W[(s+1)&1], last read
// in slots s-2 / s-1, may be overwritten). Z sits between arrive and wait and absorbs the skew between warps. The TMA
// producer refills a raw stage after wait(S) of slot s: the pairs <= s-2 are retired (last reader: the U of slot s-1).
// (Tried and dropped, profiles/r2b_README.md: splitting the warps into two half-CTA sets that run half a slot apart —
// the extra cross-set waits cost more than the overlap of P with Z / R / U gains.)
// Follows PAPER.md:15 with the readings of DESIGN.md §3; shares no code with oracle/.
#pragma once
#include <cuda.h>
#include <stdint.h>

#include <type_traits>

#include "hydro_f2.cuh"

namespace gh {

constexpr int ZNT = 320;            // threads per CTA: 8 interior warps + 2 ghost warps
constexpr int ZNW = ZNT / 32;       // warps (arrival count of the slot barrier)
constexpr int ZNS = 6;              // raw ring depth in plane PAIRS (6 x 16 KB: the most that fits; 5 is 1.2 % slower)
constexpr int ZSLOTS = 11;          // pipeline slots (= TMA loads) per group
constexpr int ZWP = 21;             // row pitch of a primitive pair-plane in 8-byte elements (odd: the ghost columns read conflict-free)
constexpr int ZWQ = FS * ZWP;       // elements per component
constexpr int ZNX = 17 * FN;        // x-face arrays: index i + 17 j, i = 0..16 (face i - 1/2; x+ state of cell i - 1)
constexpr int ZNY = FN * 17;        // y-face arrays: index i + 16 j, j = 0..16

struct ZSmem {
  static constexpr int raw_tx_bytes = 2 * PRAW * 4;                       // 16000
  static constexpr int raw_stage_bytes = ((raw_tx_bytes + 127) / 128) * 128;
  static constexpr int w_bytes = 5 * ZWQ * 8;                             // one primitive pair-plane
  static constexpr int s_bytes = 6 * (ZNX + ZNY) * 8;                     // x+ and y+ states of one pair
  static constexpr int f_bytes = 5 * (ZNX + ZNY) * 8;                     // x and y fluxes of one pair
  static constexpr int off_raw = 0;
  static constexpr int off_w = off_raw + ZNS * raw_stage_bytes;
  static constexpr int off_s = off_w + 2 * w_bytes;
  static constexpr int off_f = off_s + 2 * s_bytes;
  static constexpr int off_bar = ((off_f + 2 * f_bytes + 15) / 16) * 16;  // ZNS full barriers, S (even slots), S (odd slots)
  static constexpr int total = off_bar + (ZNS + 2) * 8;
};
static_assert(ZSmem::total <= 232448, "z-pair kernel: shared memory over the 227 KB limit");

// wait with a suspend-time hint: the warp sleeps in hardware until the phase completes (or the hint expires) instead
// of polling — the polls of waiting warps take issue slots from the working warps of the same scheduler
__device__ __forceinline__ void mbar_wait_sleep(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity), "r"(20000u)
      : "memory");
}

__device__ __forceinline__ void tma_load_pair(uint32_t dst, const CUtensorMap* map, int x, int y, int z, int g, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(0), "r"(g), "r"(bar)
      : "memory");
}

// in-place replacement of the failing lanes of a packed value (rare guard path: no register copies on the hot path)
__device__ __forceinline__ void fix2(f2& d, bool ok_lo, bool ok_hi, f2 a) {
  asm volatile(
      "{\n.reg .f32 x, y, ax, ay;\n.reg .pred p, q;\n"
      "mov.b64 {x, y}, %0;\nmov.b64 {ax, ay}, %3;\n"
      "setp.ne.u32 p, %1, 0;\nsetp.ne.u32 q, %2, 0;\n"
      "@!p mov.f32 x, ax;\n@!q mov.f32 y, ay;\n"
      "mov.b64 %0, {x, y};\n}\n"
      : "+l"(d.v)
      : "r"((unsigned)ok_lo), "r"((unsigned)ok_hi), "l"(a.v));
}
__device__ __forceinline__ void fix_state(St2& s, bool ok_lo, bool ok_hi, const St2& a) {
  fix2(s.r, ok_lo, ok_hi, a.r); fix2(s.u, ok_lo, ok_hi, a.u); fix2(s.v, ok_lo, ok_hi, a.v);
  fix2(s.w, ok_lo, ok_hi, a.w); fix2(s.p, ok_lo, ok_hi, a.p); fix2(s.h, ok_lo, ok_hi, a.h);
}

// ---- steps a1 + a2, one direction n (slot index of the normal velocity is 1 + n): face values from the limited
// slopes s[], the conserved face states U+ and NEGATED U- (the '-' face carries its minus sign on the density, so
// that every flux term is one fma into the accumulator and Ubar- = dU - (-U-)), and acc (+)= F_n(W+) - F_n(W-).
template <int n, bool FIRST>
__device__ __forceinline__ void zp_dir(const f2 Wc[5], f2 nrho, const f2 s[5], const PairConst& c, f2 acc[5], f2 Up[5],
                                       f2 Um[5]) {
  constexpr int t1 = (n + 1) % 3, t2 = (n + 2) % 3;
  {
    const f2 rho = fma2(c.half, s[0], Wc[0]);
    const f2 v[3] = {fma2(c.half, s[1], Wc[1]), fma2(c.half, s[2], Wc[2]), fma2(c.half, s[3], Wc[3])};
    const f2 P = fma2(c.half, s[4], Wc[4]);
    const f2 q = fma2(v[2], v[2], fma2(v[1], v[1], v[0] * v[0]));
    const f2 E = fma2(c.half * rho, q, c.ig1 * P);
    Up[0] = rho; Up[1] = rho * v[0]; Up[2] = rho * v[1]; Up[3] = rho * v[2]; Up[4] = E;
    const f2 mn = Up[1 + n];
    if (FIRST) {
      acc[0] = mn;
      acc[1 + n] = fma2(mn, v[n], s[4]);            // P+ - P- = slope of P
      acc[1 + t1] = mn * v[t1];
      acc[1 + t2] = mn * v[t2];
      acc[4] = (E + P) * v[n];
    } else {
      acc[0] = acc[0] + mn;
      acc[1 + n] = fma2(mn, v[n], acc[1 + n] + s[4]);
      acc[1 + t1] = fma2(mn, v[t1], acc[1 + t1]);
      acc[1 + t2] = fma2(mn, v[t2], acc[1 + t2]);
      acc[4] = fma2(E + P, v[n], acc[4]);
    }
  }
  {
    const f2 nr = fma2(c.half, s[0], nrho);         // -(rho - s/2)
    const f2 v[3] = {fma2(c.halfn, s[1], Wc[1]), fma2(c.halfn, s[2], Wc[2]), fma2(c.halfn, s[3], Wc[3])};
    const f2 P = fma2(c.halfn, s[4], Wc[4]);
    const f2 q = fma2(v[2], v[2], fma2(v[1], v[1], v[0] * v[0]));
    const f2 nE = fma2(c.half * nr, q, c.ig1n * P);  // -E
    Um[0] = nr; Um[1] = nr * v[0]; Um[2] = nr * v[1]; Um[3] = nr * v[2]; Um[4] = nE;
    const f2 nmn = Um[1 + n];
    acc[0] = acc[0] + nmn;
    acc[1 + n] = fma2(nmn, v[n], acc[1 + n]);
    acc[1 + t1] = fma2(nmn, v[t1], acc[1 + t1]);
    acc[1 + t2] = fma2(nmn, v[t2], acc[1 + t2]);
    acc[4] = fma2(nE - P, v[n], acc[4]);
  }
}

// predicted state Ubar = U_face + dU as (rho, v, P, H); SIGN = -1 takes the negated face state of zp_dir.
// gmin accumulates min(rho, P) over the states of the cell for the guard (reading R7), NaN-propagating.
template <int SIGN>
__device__ __forceinline__ St2 zp_state(const f2 Uf[5], const f2 dU[5], const PairConst& c, f2& gmin) {
  f2 rb, m1, m2, m3, Eb;
  if (SIGN > 0) { rb = Uf[0] + dU[0]; m1 = Uf[1] + dU[1]; m2 = Uf[2] + dU[2]; m3 = Uf[3] + dU[3]; Eb = Uf[4] + dU[4]; }
  else { rb = dU[0] - Uf[0]; m1 = dU[1] - Uf[1]; m2 = dU[2] - Uf[2]; m3 = dU[3] - Uf[3]; Eb = dU[4] - Uf[4]; }
  const f2 r = rcp2(rb);
  St2 o;
  o.r = rb;
  o.u = m1 * r;
  o.v = m2 * r;
  o.w = m3 * r;
  const f2 ke2 = fma2(m3, o.w, fma2(m2, o.v, m1 * o.u));
  o.p = fma2(c.hg1n, ke2, c.g1 * Eb);
  o.h = (Eb + o.p) * r;
  gmin = mk2(min3nan(lo(gmin), lo(rb), lo(o.p)), min3nan(hi(gmin), hi(rb), hi(o.p)));
  return o;
}

// One instruction stream for all ten warps (the three roles differ in a few warp-uniform branches and in per-lane
// shared-memory offsets only): role 0 = interior warps; 1 = upper ghosts (warp 8); 2 = lower ghosts (warp 9)
template <int LIM>
__device__ __forceinline__ void zp_run(const CUtensorMap& in_map, float* __restrict__ U_out, float* __restrict__ bflux,
                                       int n_groups, int goff, const PairConst& c,
                                       unsigned long long* __restrict__ status, unsigned char* smem) {
  using SM = ZSmem;
  float* const wbase = reinterpret_cast<float*>(smem + SM::off_w);
  float* const sbase = reinterpret_cast<float*>(smem + SM::off_s);
  float* const fbase = reinterpret_cast<float*>(smem + SM::off_f);
  const uint32_t raw_base = smem_u32(smem + SM::off_raw);
  const uint32_t bar_base = smem_u32(smem + SM::off_bar);
  const uint32_t s_bar = bar_base + 8 * ZNS;   // the slot barrier, as an (even slot, odd slot) pair

  // ---- thread -> column (i, j); ghost lanes: rot = the normal is y
  const int t = (int)threadIdx.x, lane = t & 31;
  // warp-uniform, and read through a shuffle so that the compiler knows it (uniform branches need no reconvergence
  // bookkeeping): warps 0..7 interior (0), warp 8 upper ghosts (1), warp 9 lower ghosts (2)
  const int role = __shfl_sync(0xffffffffu, t < 256 ? 0 : 1 + ((t >> 5) & 1), 0);
  int i, j;
  bool rot = false;
  if (role == 0) { j = t >> 4; i = t & 15; }
  else {
    const int l = lane & 15;
    rot = lane >= 16;
    if (role == 1) { i = rot ? l : FN; j = rot ? FN : l; }
    else { i = rot ? l : -1; j = rot ? -1 : l; }
  }
  const int w_own = 2 * ((j + 2) * ZWP + (i + 2));          // float offsets (8-byte elements)
  const int raw_own = (j + 2) * FS + (i + 2);
  // exchange arrays of one pair: [SX: 6 x ZNX][SY: 6 x ZNY] and [FX: 5 x ZNX][FY: 5 x ZNY], 8-byte elements
  const int ix = 2 * (i + 17 * j), iy = 2 * (i + 16 * j);   // own lower x / y face (float offsets)
  // who publishes which '+' state: x+ of cell (i, j) -> SX[(i+1) + 17 j] (interior and the ghost column i = -1),
  // y+ -> SY[i + 16 (j+1)] (interior and the ghost row j = -1)
  const bool pub_x = role == 0 || (role == 2 && !rot), pub_y = role == 0 || (role == 2 && rot);

  const int n_local = (n_groups - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int n_slots = n_local * ZSLOTS;

  // ---- TMA producer (lane 0 of warp 9)
  int issued = 0, iss_m = 0, iss_g = (int)blockIdx.x;
  uint32_t iss_stage = 0;
  auto issue_upto = [&](int limit) {
    if (limit > n_slots + 1) limit = n_slots + 1;   // one pair past the end (zero-filled) keeps the conversion unconditional
#pragma unroll 1
    while (issued < limit) {
      const uint32_t bar = bar_base + 8 * iss_stage;
      mbar_expect_tx(bar, SM::raw_tx_bytes);
      tma_load_pair(raw_base + iss_stage * SM::raw_stage_bytes, &in_map, goff, goff, goff + 2 * iss_m - 1, iss_g, bar);
      ++issued;
      if (++iss_m == ZSLOTS) { iss_m = 0; iss_g += (int)gridDim.x; }
      if (++iss_stage == ZNS) iss_stage = 0;
    }
  };
  const bool producer = t == 288;
  if (producer) issue_upto(ZNS);

  auto warp_arrive = [&](uint32_t bar) {
    __syncwarp();
    if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
  };
  // raw ring: stage / parity of the pair converted next, stage of the pair updated next
  uint32_t c_stage = 0, c_par = 0, u_stage = ZNS - 1;   // slot s updates the raw pair s-1
  auto next_raw = [&]() -> const float* {
    mbar_wait(bar_base + 8 * c_stage, c_par);
    const float* p = reinterpret_cast<const float*>(smem + SM::off_raw + c_stage * SM::raw_stage_bytes);
    if (++c_stage == ZNS) { c_stage = 0; c_par ^= 1u; }
    return p;
  };
  auto skip_raw = [&]() { if (++c_stage == ZNS) { c_stage = 0; c_par ^= 1u; } };
  auto convert = [&](const float* raw, int off, f2 W[5]) {
    f2 U[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U[q] = mk2(raw[q * (2 * FS * FS) + off], raw[q * (2 * FS * FS) + FS * FS + off]);
    cons2prim2(U, c, W);
  };
  auto load_own = [&](const float* wpl, f2 W[5]) {   // own column of a primitive pair-plane, rotated frame
#pragma unroll
    for (int q = 0; q < 5; ++q) W[q] = lds2(wpl + w_own + 2 * q * ZWQ);
  };

  unsigned int n_guard = 0, n_nonpos = 0;
  f2 Wc[5];
  float az[5];                                       // W(lo plane of the pair) - W(plane below it)
  {  // pair 0 of the flat sequence (planes -3, -2 of the first group)
    f2 W[5];
    convert(next_raw(), raw_own, W);
#pragma unroll
    for (int q = 0; q < 5; ++q) Wc[q] = W[q];
#pragma unroll
    for (int q = 0; q < 5; ++q) az[q] = 0.0f;
  }
  // interior: z+ state of the pair's upper plane (left state of the next pair's first z face) and the z-flux
  // differences of the pair awaiting its update
  float Lz[6] = {1.0f, 1.0f, 1.0f, 1.0f, 1.0f, 1.0f};
  float dzlo[5], Fzh[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) { dzlo[q] = 0.0f; Fzh[q] = 0.0f; }

  // The slot body is written as straight-line PHASES (lambdas, inlined) so that each region between two barrier
  // operations is one basic block the scheduler can interleave: {C, P}, {Z, U}, {R, reload}. Slot-dependent special
  // cases (the two light slots of a group, the first / last update, boundary-flux stores) live in warp-uniform side
  // branches.
  int gs = 0, g = (int)blockIdx.x;

  // ---- C: primitives of pair s+1 -> W[(s+1)&1]
  // cz: W(lower plane of pair s+1) - W(upper plane of pair s)
  auto phaseC = [&](float* w_nxt, float cz[5]) {
    const float* raw = next_raw();
    f2 Wn[5];
    convert(raw, raw_own, Wn);
#pragma unroll
    for (int q = 0; q < 5; ++q) sts2(w_nxt + w_own + 2 * q * ZWQ, Wn[q]);
    if (role == 0 && (t & 64)) {
      // the 68 cells of a plane that are only ever neighbours (rows -2 / 17, columns -2 / 17, inner corners): 17 each for
      // the interior warps 2, 3, 6, 7 — the warps on the two schedulers that carry no ghost warp
      const int e = 17 * (((t >> 7) << 1) | ((t >> 5) & 1)) + lane;
      if (lane < 17) {
        int ei, ej;
        if (e < 32) { ei = e & 15; ej = (e < 16) ? -2 : FN + 1; }
        else if (e < 64) { ej = e & 15; ei = (e < 48) ? -2 : FN + 1; }
        else { ei = (e & 1) ? FN : -1; ej = (e & 2) ? FN : -1; }
        f2 We[5];
        convert(raw, (ej + 2) * FS + (ei + 2), We);
        float* we = w_nxt + 2 * ((ej + 2) * ZWP + (ei + 2));
#pragma unroll
        for (int q = 0; q < 5; ++q) sts2(we + 2 * q * ZWQ, We[q]);
      }
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) cz[q] = lo(Wn[q]) - hi(Wc[q]);
  };

  // ---- P: reconstruction + half-step prediction of the pair; publishes the x+ / y+ states into S[buf]
  // Sm1, Sm2: the '-' states along the two in-plane directions (interior: x-, y-; upper ghosts use Sm1); Szm, Szp: z-, z+
  auto phaseP = [&](const float* w_cur, float* sx, float* sy, const float cz[5], St2& Sm1, St2& Sm2, St2& Szm, St2& Szp) {
    f2 s1[5], s2[5], s3[5];
    {
      const float* wp = w_cur + w_own;
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const int o = 2 * q * ZWQ;
        const f2 a1 = Wc[q] - lds2(wp + o - 2), b1 = lds2(wp + o + 2) - Wc[q];
        const f2 a2 = Wc[q] - lds2(wp + o - 2 * ZWP), b2 = lds2(wp + o + 2 * ZWP) - Wc[q];
        s1[q] = limited_slope2<LIM>(a1, b1);
        s2[q] = limited_slope2<LIM>(a2, b2);
        const float bz = hi(Wc[q]) - lo(Wc[q]);
        s3[q] = mk2(limited_slope1<LIM>(az[q], bz), limited_slope1<LIM>(bz, cz[q]));
      }
    }
    f2 acc[5], U1p[5], U1m[5], U2p[5], U2m[5], U3p[5], U3m[5], dU[5];
    {
      const f2 nrho = c.onen * Wc[0];
      zp_dir<0, true>(Wc, nrho, s1, c, acc, U1p, U1m);
      zp_dir<1, false>(Wc, nrho, s2, c, acc, U2p, U2m);
      zp_dir<2, false>(Wc, nrho, s3, c, acc, U3p, U3m);
#pragma unroll
      for (int q = 0; q < 5; ++q) dU[q] = c.hlamn * acc[q];
    }
    f2 gmin = c.one;
    // x+ / y+ states: published where a neighbour needs them (the ghost columns run the very same arithmetic as the
    // interior ones — no rotated frame — so that data uniform along an axis give bit-identical states along it)
    {
      const St2 S = zp_state<+1>(U1p, dU, c, gmin);
      if (pub_x) {
        float* o = sx + ix + 2;
        sts2(o, S.r); sts2(o + 2 * ZNX, S.u); sts2(o + 4 * ZNX, S.v); sts2(o + 6 * ZNX, S.w);
        sts2(o + 8 * ZNX, S.p); sts2(o + 10 * ZNX, S.h);
      }
    }
    {
      const St2 S = zp_state<+1>(U2p, dU, c, gmin);
      if (pub_y) {
        float* o = sy + iy + 2 * FN;
        sts2(o, S.r); sts2(o + 2 * ZNY, S.u); sts2(o + 4 * ZNY, S.v); sts2(o + 6 * ZNY, S.w);
        sts2(o + 8 * ZNY, S.p); sts2(o + 10 * ZNY, S.h);
      }
    }
    Sm1 = zp_state<-1>(U1m, dU, c, gmin);
    Sm2 = zp_state<-1>(U2m, dU, c, gmin);
    Szm = zp_state<-1>(U3m, dU, c, gmin);
    Szp = zp_state<+1>(U3p, dU, c, gmin);
    // all six states enter the guard (as in the oracle), also in the ghost columns that use one of them; the ghost
    // columns of the two ghost planes (-1: lower lane of the first pair, 16: upper lane of the last) are never used
    const bool ok_lo = lo(gmin) > 0.0f || (role != 0 && gs == 1), ok_hi = hi(gmin) > 0.0f || (role != 0 && gs == 9);
    if (__builtin_expect(!(ok_lo && ok_hi), 0)) {
      // rare: first-order fallback (reading R7) — all six states of the failing cell become its own input state
      f2 W0[5];
      load_own(w_cur, W0);
      St2 fb;
      fb.r = W0[0]; fb.u = W0[1]; fb.v = W0[2]; fb.w = W0[3]; fb.p = W0[4];
      const f2 q = fma2(W0[3], W0[3], fma2(W0[2], W0[2], W0[1] * W0[1]));
      fb.h = fma2(c.half, q, (c.gg1 * W0[4]) * rcp2(W0[0]));
      fix_state(Sm1, ok_lo, ok_hi, fb); fix_state(Sm2, ok_lo, ok_hi, fb);
      fix_state(Szm, ok_lo, ok_hi, fb); fix_state(Szp, ok_lo, ok_hi, fb);
      const float fl[6] = {lo(fb.r), lo(fb.u), lo(fb.v), lo(fb.w), lo(fb.p), lo(fb.h)};
      const float fh[6] = {hi(fb.r), hi(fb.u), hi(fb.v), hi(fb.w), hi(fb.p), hi(fb.h)};
      float* ox = sx + ix + 2;
      float* oy = sy + iy + 2 * FN;
#pragma unroll
      for (int m = 0; m < 6; ++m) {
        if (pub_x) {
          if (!ok_lo) ox[2 * m * ZNX] = fl[m];
          if (!ok_hi) ox[2 * m * ZNX + 1] = fh[m];
        }
        if (pub_y) {
          if (!ok_lo) oy[2 * m * ZNY] = fl[m];
          if (!ok_hi) oy[2 * m * ZNY + 1] = fh[m];
        }
      }
      n_guard += (ok_lo ? 0u : 1u) + (ok_hi ? 0u : 1u);   // every cell that gets here is one whose states are used
      if (!ok_lo) mark_guard(g, FN, i, j, 2 * gs - 3);
      if (!ok_hi) mark_guard(g, FN, i, j, 2 * gs - 2);
    }
  };

  // ---- Z (interior): the two lower z faces of the pair; left states (z+ of the plane below, z+ of the pair's lower
  // plane). The pair awaiting its update (slot s-1) gets its last z difference; this pair starts its own.
  // dzz: (Fz_up - Fz_lo) of the pair awaiting its update
  auto phaseZ = [&](const St2& Szm, const St2& Szp, f2 dzz[5]) {
    St2 Lq;
    Lq.r = mk2(Lz[0], lo(Szp.r)); Lq.u = mk2(Lz[1], lo(Szp.u)); Lq.v = mk2(Lz[2], lo(Szp.v));
    Lq.w = mk2(Lz[3], lo(Szp.w)); Lq.p = mk2(Lz[4], lo(Szp.p)); Lq.h = mk2(Lz[5], lo(Szp.h));
    Lz[0] = hi(Szp.r); Lz[1] = hi(Szp.u); Lz[2] = hi(Szp.v); Lz[3] = hi(Szp.w); Lz[4] = hi(Szp.p); Lz[5] = hi(Szp.h);
    f2 Fz[5];
    roe2<2>(Lq, Szm, c, Fz);
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      dzz[q] = mk2(dzlo[q], lo(Fz[q]) - Fzh[q]);
      dzlo[q] = hi(Fz[q]) - lo(Fz[q]);
      Fzh[q] = hi(Fz[q]);
    }
  };

  // ---- U: conservative update of pair s-1 (planes k_lo = 2 gs - 5, k_hi = 2 gs - 4) from F[buf ^ 1]; VLO / VHI: which
  // of the two planes is an interior one (both, except in the first and the last update of a group)
  auto phaseU = [&](auto vlo_c, auto vhi_c, const float* fx, const float* fy, float* outg, float* bfg, const f2 dzz[5]) {
    constexpr bool VLO = decltype(vlo_c)::value, VHI = decltype(vhi_c)::value;
    const int k_lo = 2 * gs - 5;
    if (role == 0) {
      const float* rawp = reinterpret_cast<const float*>(smem + SM::off_raw + u_stage * SM::raw_stage_bytes) + raw_own;
      float* op = outg + k_lo * (FN * FN) + j * FN + i;
      f2 out[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const f2 Uin = mk2(rawp[q * (2 * FS * FS)], rawp[q * (2 * FS * FS) + FS * FS]);
        const f2 dx = lds2(fx + 2 * q * ZNX + ix + 2) - lds2(fx + 2 * q * ZNX + ix);
        const f2 dy = lds2(fy + 2 * q * ZNY + iy + 2 * FN) - lds2(fy + 2 * q * ZNY + iy);
        out[q] = fma2(c.lamn, (dx + dy) + dzz[q], Uin);
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        if (VLO) op[q * (FN * FN * FN)] = lo(out[q]);
        if (VHI) op[q * (FN * FN * FN) + FN * FN] = hi(out[q]);
      }
      const f2 m2 = fma2(out[3], out[3], fma2(out[2], out[2], out[1] * out[1]));
      const f2 tre = (out[0] + out[0]) * out[4];
      if (VLO) n_nonpos += ((lo(out[0]) > 0.0f) & (lo(tre) > lo(m2))) ? 0u : 1u;
      if (VHI) n_nonpos += ((hi(out[0]) > 0.0f) & (hi(tre) > hi(m2))) ? 0u : 1u;
    }
    if (role == 2 && bfg) {
      // a5: the x / y boundary fluxes of pair s-1, from the flux arrays: lanes 0..15 the lower face, 16..31 the upper
      const int l = lane & 15, side = lane >> 4;
      const float* px = fx + 2 * (side * FN + 17 * l);
      const float* py = fy + 2 * (l + FN * (side * FN));
      float* bx = bfg + (side * 5) * (FN * FN) + k_lo * FN + l;
      float* by = bfg + ((2 + side) * 5) * (FN * FN) + k_lo * FN + l;
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const f2 vx = lds2(px + 2 * q * ZNX), vy = lds2(py + 2 * q * ZNY);
        if (VLO) { bx[q * (FN * FN)] = lo(vx); by[q * (FN * FN)] = lo(vy); }
        if (VHI) { bx[q * (FN * FN) + FN] = hi(vx); by[q * (FN * FN) + FN] = hi(vy); }
      }
    }
  };
  using T_ = std::true_type;
  using F_ = std::false_type;

  // ---- R: Roe fluxes at the lower x and the lower y face of the pair -> F[buf]
  auto phaseR = [&](const float* sx, const float* sy, float* fx, float* fy, const St2& Sm1, const St2& Sm2) {
    if (role == 0) {
      // y solve and its stores first, then x: 0.8 % faster than both solves followed by both stores (register lifetimes)
      {
        f2 Fy[5];
        St2 Ly;
        const float* p = sy + iy;
        Ly.r = lds2(p); Ly.u = lds2(p + 2 * ZNY); Ly.v = lds2(p + 4 * ZNY); Ly.w = lds2(p + 6 * ZNY);
        Ly.p = lds2(p + 8 * ZNY); Ly.h = lds2(p + 10 * ZNY);
        roe2<1>(Ly, Sm2, c, Fy);
#pragma unroll
        for (int q = 0; q < 5; ++q) sts2(fy + 2 * q * ZNY + iy, Fy[q]);
      }
      {
        f2 Fx[5];
        St2 Lx;
        const float* p = sx + ix;
        Lx.r = lds2(p); Lx.u = lds2(p + 2 * ZNX); Lx.v = lds2(p + 4 * ZNX); Lx.w = lds2(p + 6 * ZNX);
        Lx.p = lds2(p + 8 * ZNX); Lx.h = lds2(p + 10 * ZNX);
        roe2<0>(Lx, Sm1, c, Fx);
#pragma unroll
        for (int q = 0; q < 5; ++q) sts2(fx + 2 * q * ZNX + ix, Fx[q]);
      }
    } else if (role == 1) {
      // the face this ghost owns: x = 15.5 (column i = 16: left state SX[16 + 17 j], right state its x- state) or
      // y = 15.5 (row j = 16: SY[i + 256], its y- state). The row lanes feed the solver their velocities in the cyclic
      // order (v, w, u) of the interior's y solve, so that both perform the same operations on the same operands
      const float* p = rot ? (sy + iy) : (sx + ix);
      const int st = rot ? 2 * ZNY : 2 * ZNX;
      const int o1 = rot ? 2 * st : st, o2 = rot ? 3 * st : 2 * st, o3 = rot ? st : 3 * st;   // slots of (normal, t1, t2)
      St2 Lq, Rq;
      Lq.r = lds2(p); Lq.u = lds2(p + o1); Lq.v = lds2(p + o2); Lq.w = lds2(p + o3);
      Lq.p = lds2(p + 4 * st); Lq.h = lds2(p + 5 * st);
      Rq.r.v = rot ? Sm2.r.v : Sm1.r.v; Rq.p.v = rot ? Sm2.p.v : Sm1.p.v; Rq.h.v = rot ? Sm2.h.v : Sm1.h.v;
      Rq.u.v = rot ? Sm2.v.v : Sm1.u.v; Rq.v.v = rot ? Sm2.w.v : Sm1.v.v; Rq.w.v = rot ? Sm2.u.v : Sm1.w.v;
      f2 F[5];
      roe2<0>(Lq, Rq, c, F);
      float* o = rot ? (fy + iy) : (fx + ix);
      sts2(o, F[0]); sts2(o + o1, F[1]); sts2(o + o2, F[2]); sts2(o + o3, F[3]); sts2(o + 4 * st, F[4]);
    }
  };

#pragma unroll 1
  for (int s = 0; s < n_slots; ++s) {
    const int buf = s & 1;
    float* const outg = U_out + (size_t)g * (5 * FN * FN * FN);
    float* const bfg = bflux ? bflux + (size_t)g * (30 * FN * FN) : nullptr;
    float* const w_cur = wbase + buf * (SM::w_bytes / 4);
    float* const w_nxt = wbase + (buf ^ 1) * (SM::w_bytes / 4);
    float* const sx = sbase + buf * (SM::s_bytes / 4);
    float* const sy = sx + 12 * ZNX;
    float* const fx = fbase + buf * (SM::f_bytes / 4);
    float* const fy = fx + 10 * ZNX;
    const float* const fxp = fbase + (buf ^ 1) * (SM::f_bytes / 4);   // fluxes of slot s-1
    const float* const fyp = fxp + 10 * ZNX;

    const uint32_t sbar = s_bar + 8u * (uint32_t)(s & 1), spar = (uint32_t)(s >> 1) & 1u;   // barrier / parity of slot s
    auto wait_s = [&]() {
      mbar_wait_sleep(sbar, spar);           // see the header: states of pair s, fluxes of pair s-1, primitives of pair s+1
      if (producer) issue_upto(s - 1 + ZNS); // pairs <= s-2 are retired (their last reader is the update in slot s-1)
    };
    float cz[5];
    phaseC(w_nxt, cz);
    if (gs >= 1 && gs <= 9) {
      // ================= a full slot: the pair (2 gs - 3, 2 gs - 2) =================
      St2 Sm1, Sm2, Szm, Szp;
      phaseP(w_cur, sx, sy, cz, Sm1, Sm2, Szm, Szp);
      warp_arrive(sbar);                    // everything the neighbours need from this warp is published
      f2 dzz[5];
      if (role == 0) phaseZ(Szm, Szp, dzz);
      if (role == 0 && bfg && (gs == 1 || gs == 9)) {   // a5: faces -z (the upper face of plane -1) and +z (of plane 15)
        float* p = bfg + (4 + (gs == 9)) * (5 * FN * FN) + j * FN + i;
#pragma unroll
        for (int q = 0; q < 5; ++q) p[q * (FN * FN)] = Fzh[q];
      }
      wait_s();
      phaseR(sx, sy, fx, fy, Sm1, Sm2);
      if (gs >= 3) phaseU(T_{}, T_{}, fxp, fyp, outg, bfg, dzz);
      else if (gs == 2) phaseU(F_{}, T_{}, fxp, fyp, outg, bfg, dzz);
    } else {
      // ================= a light slot: gs = 0 (planes -3, -2) converts the first pair, gs = 10 finishes the last =====
      warp_arrive(sbar);
      wait_s();
      if (gs == ZSLOTS - 1) {
        f2 dzz[5];   // plane 16 gets no update; plane 15 needs the z difference it already has
#pragma unroll
        for (int q = 0; q < 5; ++q) dzz[q] = mk2(dzlo[q], 0.0f);
        phaseU(T_{}, F_{}, fxp, fyp, outg, bfg, dzz);
      }
    }
    // ---- next pair: own column of W[(s+1)&1] (written by this thread in C), the z difference below it
    load_own(w_nxt, Wc);
#pragma unroll
    for (int q = 0; q < 5; ++q) az[q] = cz[q];
    if (++u_stage == ZNS) u_stage = 0;
    if (++gs == ZSLOTS) { gs = 0; g += (int)gridDim.x; }
  }

  for (int o = 16; o > 0; o >>= 1) {
    n_guard += __shfl_xor_sync(0xffffffffu, n_guard, o);
    n_nonpos += __shfl_xor_sync(0xffffffffu, n_nonpos, o);
  }
  if (lane == 0) {
    if (n_guard) atomicAdd(&status[0], (unsigned long long)n_guard);
    if (n_nonpos) atomicAdd(&status[1], (unsigned long long)n_nonpos);
  }
}

template <int LIM>
__global__ void __launch_bounds__(ZNT, 1)
    zpair_kernel(const __grid_constant__ CUtensorMap in_map, float* __restrict__ U_out, float* __restrict__ bflux,
                 int n_groups, int goff, const __grid_constant__ PairConst c, unsigned long long* __restrict__ status) {
  extern __shared__ __align__(128) unsigned char zsmem[];
  if (threadIdx.x == 0) {
    const uint32_t bar_base = smem_u32(zsmem + ZSmem::off_bar);
    for (int s = 0; s < ZNS; ++s) mbar_init(bar_base + 8 * s, 1);
    mbar_init(bar_base + 8 * ZNS, ZNW);
    mbar_init(bar_base + 8 * ZNS + 8, ZNW);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  zp_run<LIM>(in_map, U_out, bflux, n_groups, goff, c, status, zsmem);
}

}  // namespace gh
