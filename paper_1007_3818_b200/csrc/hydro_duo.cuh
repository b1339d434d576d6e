// csrc/hydro_duo.cuh — fp32 performance path, variant "duo": ONE cell per thread (the 320-thread cross of
// hydro_fused.cuh, 96 registers, 20 warps per SM) with the two LANES of every Blackwell `*.f32x2` instruction
// carrying two directions of the same cell instead of two cells:
//   lanes (x, y)  for the '+' face states, the '-' face states, their own-direction fluxes and the x / y Roe solves
//                 (the y lane holds its velocity components as (v, u, w) so that slot 1 is the normal one),
//   lanes (z-, z+) for the two z face states and their fluxes (same slot orders, slot 3 = w is normal in both).
// The packed forms (helpers in hydro_f2.cuh, shared with hydro_zpair.cuh) keep the issue-slot saving of packed math
// (half the slots per FLOP) without the register appetite of round 1's two-cells-per-thread kernel (since removed), so five warps per scheduler stay resident to hide the dependent-issue latency (profiles/r1c_README.md).
// Schedule per plane: TWO split (arrive / wait) mbarrier barriers — "states of plane k published" and "x / y fluxes of
// plane k published" — instead of __syncthreads; everything a neighbour publishes is double-buffered and consumed one
// phase later, and the work between an arrive and its wait absorbs the skew between warps.
// One CTA = two independent 320-thread halves (own shared-memory region, TMA ring and barriers), so that the 20 warps
// of an SM sit five on each scheduler (profiles/r1d_README.md). Follows PAPER.md:15 with the readings of DESIGN.md §3.
#pragma once
#include <cuda.h>
#include <stdint.h>

#include "hydro_f2.cuh"  // f2 helpers, PairConst, St2, roe2, limiters, mbarrier / TMA helpers

namespace gh {

constexpr int DNSTAGE = 5;   // raw-plane ring depth
constexpr int DHALVES = 2;   // independent 320-thread halves per CTA (see duo_kernel)

struct DuoSmem {
  static constexpr int raw_stage_bytes = ((PRAW * 4 + 127) / 128) * 128;
  static constexpr int raw_tx_bytes = PRAW * 4;
  static constexpr int w_plane = WPITCH * FS;                       // floats per primitive plane, rows [r][q][c]
  static constexpr int off_raw = 0;
  static constexpr int off_w = off_raw + DNSTAGE * raw_stage_bytes;
  static constexpr int off_st = off_w + 2 * w_plane * 4;            // 2 x 6 x FNT x (x+ state, y+ state in slot order)
  static constexpr int off_fl = off_st + 2 * 6 * FNT * 8;           // 2 x 5 x FNT x (Fx, Fy in slot order) at the lower faces
  static constexpr int off_bar = ((off_fl + 2 * 5 * FNT * 8 + 15) / 16) * 16;
  static constexpr int off_sync = off_bar + DNSTAGE * 8;
  static constexpr int off_nbr = off_sync + 16;                // HALO: 2 x 27 neighbour group ids (+ pad)
  static constexpr int total = off_nbr + 2 * 32 * 4;
  static constexpr int total_padded = ((total + 127) / 128) * 128;   // one half-CTA's region
};

// overwrite a packed register in place (the operand is read-write, so no new register is allocated)
__device__ __forceinline__ void set2(f2& d, float a, float b) {
  asm volatile("mov.b64 %0, {%1, %2};" : "+l"(d.v) : "f"(a), "f"(b));
}

// Exchange arrays hold, per quantity m, FNT (lo, hi) lane pairs with the two lanes in separate FNT-word planes: two
// 32-bit stores, conflict-free 32-bit reads (pair-packed 64-bit stores make the reads of one lane 2-way conflicted:
// 4.933 against 4.901 ms on the headline configuration).
__device__ __forceinline__ int ex_off(int slot, int lane) { return lane * FNT + slot; }
__device__ __forceinline__ void ex_put(float* base /* + ex_off(t, 0) */, int m, f2 v) {
  base[m * (2 * FNT)] = lo(v);
  base[m * (2 * FNT) + FNT] = hi(v);
}

// scalar state for the z-face solve
struct St1 {
  float r, u, v, w, p, h;
};
__device__ __forceinline__ St1 lane_lo(const St2& s) { return St1{lo(s.r), lo(s.u), lo(s.v), lo(s.w), lo(s.p), lo(s.h)}; }
__device__ __forceinline__ St1 lane_hi(const St2& s) { return St1{hi(s.r), hi(s.u), hi(s.v), hi(s.w), hi(s.p), hi(s.h)}; }

// own-direction physical flux of a packed face (step a2): slot N is the normal velocity of both lanes
template <int N>
__device__ __forceinline__ void flux_slot(const f2 W[5], const PairConst& c, f2 F[5]) {
  const f2 mn = W[0] * W[N];
  const f2 q = fma2(W[3], W[3], fma2(W[2], W[2], W[1] * W[1]));
  const f2 e = fma2(c.half * W[0], q, c.gg1 * W[4]);      // E + P = gg1 P + 1/2 rho q
  F[0] = mn;
  F[1] = (N == 1) ? fma2(mn, W[1], W[4]) : mn * W[1];
  F[2] = (N == 2) ? fma2(mn, W[2], W[4]) : mn * W[2];
  F[3] = (N == 3) ? fma2(mn, W[3], W[4]) : mn * W[3];
  F[4] = e * W[N];
}

// face values (primitives) + half-step increment -> predicted state (rho, velocities, P, H) of both lanes;
// gmin accumulates min(rho, P) for the guard (reading R7)
__device__ __forceinline__ St2 state_from_face(const f2 Wf[5], const f2 dU[5], const PairConst& c, f2& gmin) {
  const f2 rb = Wf[0] + dU[0];
  const f2 m1 = fma2(Wf[0], Wf[1], dU[1]), m2 = fma2(Wf[0], Wf[2], dU[2]), m3 = fma2(Wf[0], Wf[3], dU[3]);
  const f2 q = fma2(Wf[3], Wf[3], fma2(Wf[2], Wf[2], Wf[1] * Wf[1]));
  const f2 Eb = fma2(c.half * Wf[0], q, fma2(Wf[4], c.ig1, dU[4]));
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

// scalar Roe solve along z (same algebra as roe2<2>): flux density in global component order
__device__ __forceinline__ void roe1_z(const St1& L, const St1& R, float g1, float F[5]) {
  const float z = R.r * rsq1(L.r * R.r);
  const float fR = z * rcp1(z + 1.0f);
  const float rt = L.r * z;
  const float du = R.w - L.w, dv = R.u - L.u, dw = R.v - L.v, dH = R.h - L.h, dp = R.p - L.p, dr = R.r - L.r;
  const float u = fmaf(fR, du, L.w), v = fmaf(fR, dv, L.u), w = fmaf(fR, dw, L.v), H = fmaf(fR, dH, L.h);
  const float q2 = fmaf(w, w, fmaf(v, v, u * u));
  const float a2 = fmaf(-0.5f * g1, q2, g1 * H);
  const float hq = 0.5f * q2;
  const float rsa = rsq1(a2);
  const float a = a2 * rsa;
  const float t = dp * (rsa * rsa);
  const float sg = (rt * du) * rsa;
  const float l1 = u - a, l5 = u + a;
  const float P4n = -0.25f * (fabsf(l5) + fabsf(l1)), M4n = -0.25f * (fabsf(l5) - fabsf(l1));
  const float sN = fmaf(M4n, sg, P4n * t);
  const float dN = fmaf(P4n, sg, M4n * t);
  const float aun = -0.5f * fabsf(u);
  const float c2N = (dr - t) * aun;
  const float raN = rt * aun;
  const float c3N = raN * dv, c4N = raN * dw;
  const float D0 = sN + c2N;
  const float ad = a * dN;
  const float Dn = fmaf(u, D0, ad);
  const float Dt1 = fmaf(v, D0, c3N), Dt2 = fmaf(w, D0, c4N);
  const float D4 = fmaf(w, c4N, fmaf(v, c3N, fmaf(hq, c2N, fmaf(u, ad, H * sN))));
  const float mL = L.r * L.w, mR = R.r * R.w;
  F[0] = fmaf(0.5f, mL + mR, D0);
  F[3] = fmaf(0.5f, fmaf(mL, L.w, L.p) + fmaf(mR, R.w, R.p), Dn);
  F[1] = fmaf(0.5f, fmaf(mL, L.u, mR * R.u), Dt1);
  F[2] = fmaf(0.5f, fmaf(mL, L.v, mR * R.v), Dt2);
  F[4] = fmaf(0.5f, fmaf(mL, L.h, mR * R.h), D4);
}

// One half-CTA (320 threads). HALF is a template parameter so that every shared-memory address and the named
// barrier id stay compile-time constants: a run-time half offset costs registers this kernel does not have.
// Grid description of the fused-halo variant (HALO = true): the batch is ONE periodic uniform grid of gx x gy x gz
// groups (x-fastest index); besides U_out the kernel writes every updated cell straight into the ghosted array of the
// NEXT step — its own interior position and the ghost shells of up to seven neighbouring groups — and accumulates the
// signal-speed maximum of the new state, so that a multi-step run needs no separate ghost-refill pass.
struct HaloGrid {
  float* U_next;        // [G][5][20][20][20], must not alias the input
  unsigned int* vmax;   // bit pattern of the running maximum (zeroed by the caller)
  int gx, gy, gz;
};

template <int LIM, int HALF, bool HALO>
__device__ __forceinline__ void duo_half(const CUtensorMap& in_map, float* __restrict__ U_out, float* __restrict__ bflux,
                                         int n_groups, int goff, const PairConst& c,
                                         unsigned long long* __restrict__ status, unsigned char* smem_cta,
                                         const HaloGrid& hg) {
  using SM = DuoSmem;
  // The CTA is TWO independent halves of 320 threads (10 warps), each with its own shared-memory region, group
  // stream, TMA ring and barriers. Why one 20-warp CTA instead of two 10-warp CTAs: a 10-warp CTA puts 3, 3, 2, 2
  // warps on the four schedulers and the hardware places two such CTAs the same way (6, 6, 4, 4: measured with
  // clock probes, the warps of the two light schedulers idle 13 % at the barrier); warps 10..19 of one CTA land
  // on schedulers 2, 3, 0, 1, ... and make it 5, 5, 5, 5.
  constexpr int half_id = HALF;
  unsigned char* const smem = smem_cta + HALF * SM::total_padded;
  const int vblock = (int)blockIdx.x * DHALVES + HALF, vgrid = (int)gridDim.x * DHALVES;
  auto half_sync = [&]() { asm volatile("bar.sync %0, %1;" ::"n"(1 + HALF), "n"(FNT) : "memory"); };
  float* const wring = reinterpret_cast<float*>(smem + SM::off_w);
  float* const stx = reinterpret_cast<float*>(smem + SM::off_st);   // [buf][m][ex_off(t, lane)]
  float* const flx = reinterpret_cast<float*>(smem + SM::off_fl);
  const uint32_t raw_base = smem_u32(smem + SM::off_raw);
  const uint32_t bar_base = smem_u32(smem + SM::off_bar);
  const uint32_t sync_bar = smem_u32(smem + SM::off_sync);       // "states of plane k published"
  const uint32_t flux_bar = sync_bar + 8;                          // "x / y fluxes of plane k published"

  // ---- thread -> cell (i, j) of the cross-shaped footprint (as in hydro_fused.cuh)
  const int t = (int)threadIdx.x - half_id * FNT;
  int i, j;
  if (t < 288) { j = t / 18; i = t % 18 - 1; }
  else if (t < 304) { j = -1; i = t - 288; }
  else { j = FN; i = t - 304; }
  const bool in_x = (i >= 0 && i < FN), in_y = (j >= 0 && j < FN), interior = in_x && in_y;
  auto tid_of = [](int ii, int jj) { return jj < 0 ? 288 + ii : (jj >= FN ? 304 + ii : jj * 18 + ii + 1); };
  // the extra cell this thread also converts (layer-2 ghost behind a first-layer ghost; inner corners)
  // The 68 cells of a plane that are only ever neighbours (layer-2 ghosts, inner corners) are converted by warp 9
  // alone (the ghost rows: the lightest warp), three per lane, instead of by the lanes next to them in every warp.
  // Extra e = lane + 32 r, r = 0..2: rows -2 / 17 (e < 32), columns -2 / 17 (e < 64), corners (e < 68).
  auto extra_cell = [&](int e, int& ei, int& ej) {
    if (e < 32) { ei = e & 15; ej = (e < 16) ? -2 : FN + 1; }
    else if (e < 64) { ej = e & 15; ei = (e < 48) ? -2 : FN + 1; }
    else { ei = (e & 1) ? FN : -1; ej = (e & 2) ? FN : -1; }
  };
  const int raw_own = (j + 2) * FS + (i + 2);            // [q][r][c] dense, + q*400
  const int w_own = (j + 2) * WPITCH + (i + 2);          // [r][q][c], + q*20
  // x neighbours in the exchange arrays are threads t -+ 1 (same row): immediate offsets. For the lanes whose x face
  // is never used (i = -1; the ghost rows) these read an unrelated but valid shared-memory word.
  const int t_yl = in_x ? tid_of(i, j - 1 < -1 ? -1 : j - 1) : t;   // thread (i, j-1)
  const int t_yu = in_x ? tid_of(i, j + 1 > FN ? FN : j + 1) : t;   // thread (i, j+1)
  const bool do_x = in_y && i >= 0;                      // owns the face (i-1/2, j), i in [0,16]
  const bool do_y = in_x && j >= 0;                      // owns the face (i, j-1/2), j in [0,16]

  const int n_local = (n_groups - vblock + vgrid - 1) / vgrid;
  const int total_planes = n_local * FPLANES;
  // TMA producer state (thread 0 only), kept incrementally
  int issued = 0, iss_p = 0, iss_g = vblock;
  uint32_t iss_slot = 0;
  auto issue_upto = [&](int limit) {
    if (limit > total_planes) limit = total_planes;
#pragma unroll 1
    while (issued < limit) {
      const uint32_t bar = bar_base + 8 * iss_slot;
      mbar_expect_tx(bar, SM::raw_tx_bytes);
      tma_load_plane(raw_base + iss_slot * SM::raw_stage_bytes, &in_map, goff, goff, goff + iss_p, iss_g, bar);
      ++issued;
      if (++iss_p == FPLANES) { iss_p = 0; iss_g += vgrid; }
      if (++iss_slot == DNSTAGE) iss_slot = 0;
    }
  };
  if (t == 0) {
    for (int s = 0; s < DNSTAGE; ++s) mbar_init(bar_base + 8 * s, 1);
    mbar_init(sync_bar, FNT);
    mbar_init(flux_bar, FNT);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  half_sync();
  if (t == 0) issue_upto(DNSTAGE);
  uint32_t sync_phase = 0;
  auto cta_arrive = [&]() { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(sync_bar) : "memory"); };
  auto cta_wait = [&]() { mbar_wait(sync_bar, sync_phase); sync_phase ^= 1u; };
  // second split barrier for the fluxes: its wait (before the update of plane k-1) targets the arrive at the END of the
  // previous plane, so it is almost always already complete; the first wait passes on the fresh barrier (parity 1)
  uint32_t flux_phase = 1;
  auto flux_arrive = [&]() { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(flux_bar) : "memory"); };
  auto flux_wait = [&]() { mbar_wait(flux_bar, flux_phase); flux_phase ^= 1u; };
  uint32_t rs = 0, rph = 0;  // raw-ring consumer state
  auto next_plane = [&]() -> const float* {
    mbar_wait(bar_base + 8 * rs, rph);
    const float* p = reinterpret_cast<const float*>(smem + SM::off_raw + rs * SM::raw_stage_bytes);
    if (++rs == DNSTAGE) { rs = 0; rph ^= 1u; }
    return p;
  };
  const GasConst<float> gc = {lo(c.g1) + 1.0f, lo(c.g1), lo(c.ig1), lo(c.gg1), c.lam, 0.5f * c.lam};
  auto convert = [&](const float* raw, int off, float W[5]) {
    float U[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) U[q] = raw[q * (FS * FS) + off];
    cons2prim<float, true>(U, gc, W);
  };

  unsigned int n_guard = 0, n_nonpos = 0;
  float vmax_thread = 0.0f;                                   // HALO only
  int* const nbr_tab = reinterpret_cast<int*>(smem + SM::off_nbr);

  for (int it = 0; it < n_local; ++it) {
    const int g = vblock + it * vgrid;
    if (HALO && t < 27) {  // neighbour group ids of this group (periodic), double-buffered by group parity
      const int bx = g % hg.gx, by = (g / hg.gx) % hg.gy, bz = g / (hg.gx * hg.gy);
      const int ox = t % 3 - 1, oy = (t / 3) % 3 - 1, oz = t / 9 - 1;
      const int nx_ = (bx + ox + hg.gx) % hg.gx, ny_ = (by + oy + hg.gy) % hg.gy, nz_ = (bz + oz + hg.gz) % hg.gz;
      nbr_tab[(it & 1) * 32 + t] = (nz_ * hg.gy + ny_) * hg.gx + nx_;
    }
    const int seq0 = it * FPLANES;
    float* const outg = U_out + (size_t)g * (5 * FN * FN * FN);
    float* const bfg = bflux ? bflux + (size_t)g * (30 * FN * FN) : nullptr;

    float Wc[5], dLz[5], accd[5], Fz[5];
    St1 zplus;
    {  // prologue: planes -2 and -1 of the thread's own cell
      float Wm[5];
      convert(next_plane(), raw_own, Wm);
      convert(next_plane(), raw_own, Wc);
      float* wpl = wring + SM::w_plane;  // plane -1 lives in buffer 1
#pragma unroll
      for (int q = 0; q < 5; ++q) { wpl[w_own + q * FS] = Wc[q]; dLz[q] = Wc[q] - Wm[q]; accd[q] = 1.0f; Fz[q] = 1.0f; }
      zplus = St1{1.0f, 1.0f, 1.0f, 1.0f, 1.0f, 1.0f};
    }
    half_sync();
    if (t == 0) issue_upto(seq0 + 2 + DNSTAGE);

    for (int k = -1; k <= FN; ++k) {
      const int buf = k & 1;
      const bool ghost_plane = (k < 0 || k >= FN);
      // ---- A: primitives of plane k+1 (own cell + the layer-2 / corner ghost this thread is responsible for)
      float dRz[5];
      {
        float Wp[5];
        const float* raw = next_plane();
        convert(raw, raw_own, Wp);
        float* wnext = wring + (buf ^ 1) * SM::w_plane;
        if (k + 1 <= FN) {
#pragma unroll
          for (int q = 0; q < 5; ++q) wnext[w_own + q * FS] = Wp[q];
        }
        if (t >= 288 && k + 1 >= 0 && k + 1 < FN) {  // warp 9 (warp-uniform)
#pragma unroll
          for (int r = 0; r < 3; ++r) {
            const int e = (t - 288) + 32 * r;
            if (e < 68) {
              int ei, ej;
              extra_cell(e, ei, ej);
              float We[5];
              convert(raw, (ej + 2) * FS + (ei + 2), We);
              float* we = wnext + (ej + 2) * WPITCH + (ei + 2);
#pragma unroll
              for (int q = 0; q < 5; ++q) we[q * FS] = We[q];
            }
          }
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) dRz[q] = Wp[q] - Wc[q];
      }

      St2 SA;      // the x- and y- predicted states (lanes x, y)
      St1 zm, zp;  // the z- and z+ predicted states
      const bool do_pred = ghost_plane ? interior : true;
      if (do_pred) {
        // ---- B1: slopes, face values, own-direction fluxes -> dU
        const float* wpl = wring + buf * SM::w_plane + w_own;
        // lanes (x, y): the hi lane carries (rho, v, u, w, P) so that slot 1 is the normal velocity of both lanes;
        // the (z-, z+) pair uses the same two slot orders (slot 3 = w is the normal one in both)
        const f2 Wrot[5] = {mk2(Wc[0], Wc[0]), mk2(Wc[1], Wc[2]), mk2(Wc[2], Wc[1]), mk2(Wc[3], Wc[3]), mk2(Wc[4], Wc[4])};
        f2 sxy[5];
        float sz[5];
        {
          constexpr int QY[5] = {0, 2, 1, 3, 4};  // component held by the hi lane of slot q
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            const int qy = QY[q];
            const f2 dL = Wrot[q] - mk2(wpl[q * FS - 1], wpl[qy * FS - WPITCH]);   // one-sided differences, both lanes
            const f2 dR = mk2(wpl[q * FS + 1], wpl[qy * FS + WPITCH]) - Wrot[q];
            sxy[q] = mk2(limited_slope1<LIM>(lo(dL), lo(dR)), limited_slope1<LIM>(hi(dL), hi(dR)));
            sz[q] = limited_slope1<LIM>(dLz[q], dRz[q]);
          }
        }
        f2 WB[5], WA[5], WC[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          WB[q] = fma2(c.half, sxy[q], Wrot[q]);     // '+' faces
          WA[q] = fma2(c.halfn, sxy[q], Wrot[q]);    // '-' faces
        }
        WC[0] = mk2(fmaf(-0.5f, sz[0], Wc[0]), fmaf(0.5f, sz[0], Wc[0]));  // lanes (z-, z+)
        WC[1] = mk2(fmaf(-0.5f, sz[1], Wc[1]), fmaf(0.5f, sz[2], Wc[2]));
        WC[2] = mk2(fmaf(-0.5f, sz[2], Wc[2]), fmaf(0.5f, sz[1], Wc[1]));
        WC[3] = mk2(fmaf(-0.5f, sz[3], Wc[3]), fmaf(0.5f, sz[3], Wc[3]));
        WC[4] = mk2(fmaf(-0.5f, sz[4], Wc[4]), fmaf(0.5f, sz[4], Wc[4]));
        float d[5];
        {
          f2 FB[5], FA[5], FC[5], D[5];
          flux_slot<1>(WB, c, FB);
          flux_slot<1>(WA, c, FA);
          flux_slot<3>(WC, c, FC);
#pragma unroll
          for (int q = 0; q < 5; ++q) D[q] = FB[q] - FA[q];
          const float hl = lo(c.hlamn);
          d[0] = hl * ((lo(D[0]) + hi(D[0])) + (hi(FC[0]) - lo(FC[0])));
          d[1] = hl * ((lo(D[1]) + hi(D[2])) + (hi(FC[2]) - lo(FC[1])));
          d[2] = hl * ((lo(D[2]) + hi(D[1])) + (hi(FC[1]) - lo(FC[2])));
          d[3] = hl * ((lo(D[3]) + hi(D[3])) + (hi(FC[3]) - lo(FC[3])));
          d[4] = hl * ((lo(D[4]) + hi(D[4])) + (hi(FC[4]) - lo(FC[4])));
        }
        const f2 dUrot[5] = {mk2(d[0], d[0]), mk2(d[1], d[2]), mk2(d[2], d[1]), mk2(d[3], d[3]), mk2(d[4], d[4])};

        // ---- B2: the six predicted states; guard; publish x+ / y+
        f2 gmin = c.one;
        {
          const St2 SB = state_from_face(WB, dUrot, c, gmin);
          if (!ghost_plane) {
            float* so = stx + buf * (12 * FNT) + ex_off(t, 0);
            ex_put(so, 0, SB.r); ex_put(so, 1, SB.u); ex_put(so, 2, SB.v);
            ex_put(so, 3, SB.w); ex_put(so, 4, SB.p); ex_put(so, 5, SB.h);
          }
        }
        SA = state_from_face(WA, dUrot, c, gmin);
        St2 SC = state_from_face(WC, dUrot, c, gmin);
        if (__builtin_expect(!(lo(gmin) > 0.0f && hi(gmin) > 0.0f), 0)) {
          // rare: first-order fallback (reading R7) — all six states become the cell's own input state
          const float q = fmaf(Wc[3], Wc[3], fmaf(Wc[2], Wc[2], Wc[1] * Wc[1]));
          const float h = fmaf(0.5f, q, (lo(c.gg1) * Wc[4]) * rcp1(Wc[0]));
          // overwritten IN PLACE (read-write asm operands): otherwise the compiler resolves the merge of the two
          // definitions with two dozen register copies on the hot path
          set2(SA.r, Wc[0], Wc[0]); set2(SA.u, Wc[1], Wc[2]); set2(SA.v, Wc[2], Wc[1]); set2(SA.w, Wc[3], Wc[3]);
          set2(SA.p, Wc[4], Wc[4]); set2(SA.h, h, h);
          set2(SC.r, Wc[0], Wc[0]); set2(SC.u, Wc[1], Wc[2]); set2(SC.v, Wc[2], Wc[1]); set2(SC.w, Wc[3], Wc[3]);
          set2(SC.p, Wc[4], Wc[4]); set2(SC.h, h, h);
          if (!ghost_plane) {
            float* so = stx + buf * (12 * FNT) + ex_off(t, 0);
            ex_put(so, 0, SA.r); ex_put(so, 1, SA.u); ex_put(so, 2, SA.v);
            ex_put(so, 3, SA.w); ex_put(so, 4, SA.p); ex_put(so, 5, SA.h);
          }
          n_guard += 1u;  // every cell that gets here is one whose states are used
          mark_guard(g, FN, i, j, k);
        }
        zm = lane_lo(SC);
        zp = St1{hi(SC.r), hi(SC.v), hi(SC.u), hi(SC.w), hi(SC.p), hi(SC.h)};  // hi lane: slots (v, u, w)
      }
      // everything the neighbours need from this thread is published: arrive, then the z face (needs no neighbour)
      cta_arrive();
      if (interior && k >= 0) {
        float Fn[5];
        roe1_z(zplus, zm, lo(c.g1), Fn);
#pragma unroll
        for (int q = 0; q < 5; ++q) { accd[q] = Fn[q] - accd[q]; Fz[q] = Fn[q]; }  // upper z flux minus the lower-face sum
        if (bfg && (k == 0 || k == FN)) {
          float* p = bfg + (4 + (k == FN)) * (5 * FN * FN) + j * FN + i;
#pragma unroll
          for (int q = 0; q < 5; ++q) p[q * (FN * FN)] = Fn[q];
        }
      }
      zplus = zp;
      if (k < FN) {  // (own data, so still before the wait) next plane: W(k+1) was published above, so neither it nor the z difference stays in registers
        const float* wn = wring + (buf ^ 1) * SM::w_plane + w_own;
#pragma unroll
        for (int q = 0; q < 5; ++q) { const float wp = wn[q * FS]; dLz[q] = wp - Wc[q]; Wc[q] = wp; }
      }
      flux_wait();  // x / y fluxes of plane k-1 visible (published before the END of the previous plane)
      // ---- E: conservative update of plane k-1 (its x / y fluxes were published one phase earlier)
      if (interior && k >= 1) {
        const float* fxb = flx + (buf ^ 1) * (10 * FNT) + ex_off(t + 1, 0);  // lane lo: Fx of the upper x neighbour
        const float* fyb = flx + (buf ^ 1) * (10 * FNT) + ex_off(t_yu, 1);   // lane hi: Fy (slot order) of the upper y neighbour
        const int us = (int)rs - 3 + ((int)rs < 3 ? DNSTAGE : 0);  // slot of plane k-1 (rs points at plane k+2)
        const float* rawp = reinterpret_cast<const float*>(smem + SM::off_raw + us * SM::raw_stage_bytes) + raw_own;
        float* op = outg + (k - 1) * (FN * FN) + j * FN + i;
        float out[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const int qs = (q == 1) ? 2 : (q == 2 ? 1 : q);  // slot of global component q in the y lane
          out[q] = fmaf(-c.lam, (fxb[q * (2 * FNT)] + fyb[qs * (2 * FNT)]) + accd[q], rawp[q * (FS * FS)]);
          op[(size_t)q * (FN * FN * FN)] = out[q];
        }
        const float m2 = fmaf(out[3], out[3], fmaf(out[2], out[2], out[1] * out[1]));
        n_nonpos += (out[0] > 0.0f && (out[0] + out[0]) * out[4] > m2) ? 0u : 1u;
        if (HALO) {
          // signal speed of the new state (R15) for the next time step
          const float ir = rcp1(out[0]);
          const float P = fmaxf(lo(c.g1) * fmaf(-0.5f * m2, ir, out[4]), 0.0f);
          const float sp = (fabsf(out[1]) + fabsf(out[2]) + fabsf(out[3])) * ir + 3.0f * sqrt1((lo(c.g1) + 1.0f) * P * ir);
          vmax_thread = (sp > vmax_thread || sp != sp) ? sp : vmax_thread;
          // the cell in the next step's ghosted array: own interior position, and the ghost shells of the neighbours
          // it is within two cells of (per axis: none, or the one at -1 / +1)
          const int kk = k - 1;
          const int sx = i < 2 ? -1 : (i >= FN - 2 ? 1 : 0), sy = j < 2 ? -1 : (j >= FN - 2 ? 1 : 0);
          const int sz = kk < 2 ? -1 : (kk >= FN - 2 ? 1 : 0);
          const int* nt = nbr_tab + (it & 1) * 32;
#pragma unroll
          for (int oz = 0; oz < 2; ++oz) {
            if (oz && !sz) continue;
            const int zc = oz ? kk + 2 - FN * sz : kk + 2;
#pragma unroll
            for (int oy = 0; oy < 2; ++oy) {
              if (oy && !sy) continue;
              const int yc = oy ? j + 2 - FN * sy : j + 2;
#pragma unroll
              for (int ox = 0; ox < 2; ++ox) {
                if (ox && !sx) continue;
                const int xc = ox ? i + 2 - FN * sx : i + 2;
                const int gid = nt[(oz * sz + 1) * 9 + (oy * sy + 1) * 3 + (ox * sx + 1)];
                float* np_ = hg.U_next + (size_t)gid * (5 * FS * FS * FS) + (zc * FS + yc) * FS + xc;
#pragma unroll
                for (int q = 0; q < 5; ++q) np_[q * (FS * FS * FS)] = out[q];
              }
            }
          }
        }
      }
      cta_wait();  // x+ / y+ states of plane k and primitives of plane k+1 visible
      if (t == 0) issue_upto(seq0 + k + 1 + DNSTAGE);

      // ---- D: Roe fluxes at the lower x face (lane x) and the lower y face (lane y) of plane k, one packed solve
      if (!ghost_plane) {
        const float* xl = stx + buf * (12 * FNT) + ex_off(t - 1, 0);  // lane lo of the lower x neighbour's pair
        const float* yl = stx + buf * (12 * FNT) + ex_off(t_yl, 1);   // lane hi of the lower y neighbour's pair
        St2 L;
        L.r = mk2(xl[0 * (2 * FNT)], yl[0 * (2 * FNT)]); L.u = mk2(xl[1 * (2 * FNT)], yl[1 * (2 * FNT)]);
        L.v = mk2(xl[2 * (2 * FNT)], yl[2 * (2 * FNT)]); L.w = mk2(xl[3 * (2 * FNT)], yl[3 * (2 * FNT)]);
        L.p = mk2(xl[4 * (2 * FNT)], yl[4 * (2 * FNT)]); L.h = mk2(xl[5 * (2 * FNT)], yl[5 * (2 * FNT)]);
        f2 F[5];
        roe2<0>(L, SA, c, F);
        // lane x is in global component order; lane y comes back as (rho, my, mx, mz, E)
        const float Fy[5] = {hi(F[0]), hi(F[2]), hi(F[1]), hi(F[3]), hi(F[4])};
        float* fo = flx + buf * (10 * FNT) + ex_off(t, 0);
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          ex_put(fo, q, F[q]);
          accd[q] = (lo(F[q]) + Fy[q]) + Fz[q];  // sum of the lower-face fluxes of plane k
        }
        if (bfg) {  // a5: outer faces of this plane
          if (do_x && (i == 0 || i == FN)) {
#pragma unroll
            for (int q = 0; q < 5; ++q) bfg[(((i == FN ? 5 : 0) + q) * FN + k) * FN + j] = lo(F[q]);
          }
          if (do_y && (j == 0 || j == FN)) {
#pragma unroll
            for (int q = 0; q < 5; ++q) bfg[(((j == FN ? 15 : 10) + q) * FN + k) * FN + i] = Fy[q];
          }
        }
      }

      flux_arrive();
    }
  }

  for (int o = 16; o > 0; o >>= 1) {
    n_guard += __shfl_xor_sync(0xffffffffu, n_guard, o);
    n_nonpos += __shfl_xor_sync(0xffffffffu, n_nonpos, o);
  }
  if ((t & 31) == 0) {
    if (n_guard) atomicAdd(&status[0], (unsigned long long)n_guard);
    if (n_nonpos) atomicAdd(&status[1], (unsigned long long)n_nonpos);
  }
  if (HALO) {
    for (int o = 16; o > 0; o >>= 1) {
      const float other = __shfl_xor_sync(0xffffffffu, vmax_thread, o);
      vmax_thread = (other > vmax_thread || other != other) ? other : vmax_thread;
    }
    if ((t & 31) == 0) atomicMax(hg.vmax, __float_as_uint(vmax_thread));
  }
}

template <int LIM>
__global__ void __launch_bounds__(FNT * DHALVES, 1)
    duo_kernel(const __grid_constant__ CUtensorMap in_map, float* __restrict__ U_out, float* __restrict__ bflux,
               int n_groups, int goff, const __grid_constant__ PairConst c, unsigned long long* __restrict__ status) {
  extern __shared__ __align__(128) unsigned char smem_cta[];
  const HaloGrid none = {nullptr, nullptr, 1, 1, 1};
  if (threadIdx.x < FNT) duo_half<LIM, 0, false>(in_map, U_out, bflux, n_groups, goff, c, status, smem_cta, none);
  else duo_half<LIM, 1, false>(in_map, U_out, bflux, n_groups, goff, c, status, smem_cta, none);
}

// the fused-halo variant: same step, plus the next step's ghosted array and signal-speed maximum (HaloGrid)
template <int LIM>
__global__ void __launch_bounds__(FNT * DHALVES, 1)
    duo_halo_kernel(const __grid_constant__ CUtensorMap in_map, float* __restrict__ U_out, float* __restrict__ bflux,
                    int n_groups, int goff, const __grid_constant__ PairConst c, unsigned long long* __restrict__ status,
                    const __grid_constant__ HaloGrid hg) {
  extern __shared__ __align__(128) unsigned char smem_cta[];
  if (threadIdx.x < FNT) duo_half<LIM, 0, true>(in_map, U_out, bflux, n_groups, goff, c, status, smem_cta, hg);
  else duo_half<LIM, 1, true>(in_map, U_out, bflux, n_groups, goff, c, status, smem_cta, hg);
}

}  // namespace gh
