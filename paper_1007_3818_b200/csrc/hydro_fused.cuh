// csrc/hydro_fused.cuh — the sm_100a performance path: one persistent CTA per patch-group stream, all four
// steps of PAPER.md:15 fused in one kernel, intermediates never leave the SM.
//
// Design. N = 16, two ghost layers used. A CTA of 320 threads owns one 16^3 group at a time
// and marches through its z planes k = -1 .. 16. Thread t owns the column (i,j) of the 18x18 cross-shaped
// footprint (interior + first ghost layer, corners excluded) — exactly the cells whose predicted face states
// are needed (320 = 10 warps, no idle lanes in the predictor):
//     t <  288 : j = t / 18 in [0,16), i = t % 18 - 1 in [-1,16]
//     t >= 288 : the two ghost rows j = -1 (288..303) and j = 16 (304..319), i in [0,16)   (= warp 9)
// Per plane:  A  convert the thread's own cell of plane k+1 to primitives (raw planes arrive by TMA into a
//                ring of NSTAGE shared-memory stages, one 5x20x20 box per plane, mbarrier-signalled);
//             B  reconstruct + half-step predict plane k (z neighbours in registers, x/y neighbours from the
//                primitive plane in shared memory); publish the x+ / y+ states;            -- barrier --
//             D  Roe fluxes at the thread's lower x, y, z faces (z: previous plane's z+ state is in
//                registers); publish Fx, Fy; write boundary fluxes;                          -- barrier --
//             E  conservative update of cell (i,j,k-1) from flux differences; store U_out.
// The raw ring is refilled by thread 0 right after the barrier that retires a stage, so the loads of the
// next planes — and of the next group — overlap the arithmetic of the current ones.
#pragma once
#include <cuda.h>
#include <stdint.h>

#include "hydro_math.cuh"

namespace gh {

constexpr int FN = 16;              // interior cells per axis
constexpr int FS = FN + 4;          // stored cells per axis that are read (2 ghost layers)
constexpr int FNT = 320;            // threads per CTA
constexpr int FMINB = 2;            // resident CTAs per SM the fp32 instantiation is compiled for
constexpr int FPLANES = FN + 4;     // planes -2 .. 17 per group
constexpr int FNSTAGE = 6;          // raw ring depth
constexpr int WPITCH = 114;         // row pitch (reals) of the primitive plane: rows [r][q][c], 114 = 18 mod 32
                                    // so that address = t + const (mod 32) for a warp of consecutive t

template <class R>
struct FusedSmem {
  static constexpr int raw_stage_bytes = ((5 * FS * FS * (int)sizeof(R) + 127) / 128) * 128;
  static constexpr int raw_tx_bytes = 5 * FS * FS * (int)sizeof(R);
  static constexpr int w_plane = WPITCH * FS;                         // reals per primitive plane
  static constexpr int off_raw = 0;
  static constexpr int off_w = off_raw + FNSTAGE * raw_stage_bytes;
  static constexpr int off_xs = off_w + 2 * w_plane * (int)sizeof(R);
  static constexpr int exch = 5 * FNT * (int)sizeof(R);
  static constexpr int off_ys = off_xs + exch;
  static constexpr int off_fx = off_ys + exch;
  static constexpr int off_fy = off_fx + exch;
  static constexpr int off_zs = off_fy + exch;                        // the thread's own z+ state of the plane below (kept out of registers)
  static constexpr int off_wm = off_zs + exch;                        // the thread's own primitives of the plane below
  static constexpr int off_acc = off_wm + exch;                       // (xy flux differences - lower z flux) of the plane awaiting its update
  static constexpr int off_bar = ((off_acc + exch + 15) / 16) * 16;
  static constexpr int total = off_bar + FNSTAGE * 8 + 16;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_plane(uint32_t dst, const CUtensorMap* map, int x, int y, int z, int g,
                                               uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(0), "r"(g), "r"(bar)
      : "memory");
}

// VAR = true: the robustness variants — run-time Riemann flags and the mid-plane flux array;
// VAR = false is the plain kernel (flags fold to the literal 0, no extra argument is read).
template <class R, int LIM, bool Fast, bool VAR = false>
__global__ void __launch_bounds__(FNT, sizeof(R) == 4 ? FMINB : 1)
    fused_kernel(const __grid_constant__ CUtensorMap in_map, R* __restrict__ U_out, R* __restrict__ bflux,
                 int n_groups, int goff, GasConst<R> c, unsigned long long* __restrict__ status, int flags_rt = 0,
                 R* __restrict__ midflux = nullptr) {
  const int flags = VAR ? flags_rt : 0;
  using SM = FusedSmem<R>;
  extern __shared__ __align__(128) unsigned char smem[];
  R* const wring = reinterpret_cast<R*>(smem + SM::off_w);
  R* const xs = reinterpret_cast<R*>(smem + SM::off_xs);
  R* const ys = reinterpret_cast<R*>(smem + SM::off_ys);
  R* const fxs = reinterpret_cast<R*>(smem + SM::off_fx);
  R* const fys = reinterpret_cast<R*>(smem + SM::off_fy);
  R* const zs = reinterpret_cast<R*>(smem + SM::off_zs);
  R* const wms = reinterpret_cast<R*>(smem + SM::off_wm);
  R* const accs = reinterpret_cast<R*>(smem + SM::off_acc);
  const uint32_t raw_base = smem_u32(smem + SM::off_raw);
  const uint32_t bar_base = smem_u32(smem + SM::off_bar);

  const int t = threadIdx.x;
  int i, j;
  if (t < 288) { j = t / 18; i = t % 18 - 1; }
  else if (t < 304) { j = -1; i = t - 288; }
  else { j = FN; i = t - 304; }
  const bool in_x = (i >= 0 && i < FN), in_y = (j >= 0 && j < FN), interior = in_x && in_y;
  // thread owning (i',j') in the cross footprint
  auto tid_of = [](int ii, int jj) { return jj < 0 ? 288 + ii : (jj >= FN ? 304 + ii : jj * 18 + ii + 1); };
  // the extra cell this thread also converts: first-ghost-layer threads take the layer-2 ghost behind
  // them; the four interior corner threads take the inner corner ghosts (-1,-1), (16,-1), (-1,16), (16,16),
  // which are x/y neighbours of predicted ghost cells. 320 own + 68 extra = the 388 cells a plane needs.
  int ei = i, ej = j;
  bool has_extra = true;
  if (i == -1) ei = -2;
  else if (i == FN) ei = FN + 1;
  else if (j == -1) ej = -2;
  else if (j == FN) ej = FN + 1;
  else if ((i == 0 || i == FN - 1) && (j == 0 || j == FN - 1)) { ei = (i == 0) ? -1 : FN; ej = (j == 0) ? -1 : FN; }
  else has_extra = false;
  // offsets inside one plane
  const int raw_own = (j + 2) * FS + (i + 2);            // [q][r][c] dense, + q*400
  const int raw_ext = (ej + 2) * FS + (ei + 2);
  const int w_own = (j + 2) * WPITCH + (i + 2);          // [r][q][c], + q*20
  const int w_ext = (ej + 2) * WPITCH + (ei + 2);
  const int t_xl = t - 1;                                // thread (i-1, j): same row
  const int t_xr = t + 1;                                // thread (i+1, j)
  const int t_yl = in_x ? tid_of(i, j - 1) : t;          // thread (i, j-1)
  const int t_yu = in_x ? tid_of(i, j + 1 > FN ? FN : j + 1) : t;  // thread (i, j+1)

  const int n_local = (n_groups - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_planes = n_local * FPLANES;
  int issued = 0;
  auto issue_upto = [&](int limit) {  // thread 0 only
    if (limit > total_planes) limit = total_planes;
    while (issued < limit) {
      const int it = issued / FPLANES, p = issued % FPLANES;
      const int slot = issued % FNSTAGE;
      const int g = (int)blockIdx.x + it * (int)gridDim.x;
      const uint32_t bar = bar_base + 8 * slot;
      mbar_expect_tx(bar, SM::raw_tx_bytes);
      tma_load_plane(raw_base + slot * SM::raw_stage_bytes, &in_map, goff, goff, goff + p, g, bar);
      ++issued;
    }
  };
  if (t == 0) {
    for (int s = 0; s < FNSTAGE; ++s) mbar_init(bar_base + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (t == 0) issue_upto(FNSTAGE);

  auto raw_ptr = [&](int seq) -> const R* {
    return reinterpret_cast<const R*>(smem + SM::off_raw + (seq % FNSTAGE) * SM::raw_stage_bytes);
  };
  auto wait_plane = [&](int seq) { mbar_wait(bar_base + 8 * (seq % FNSTAGE), (seq / FNSTAGE) & 1); };

  unsigned int n_guard = 0, n_nonpos = 0;

  for (int it = 0; it < n_local; ++it) {
    const int g = (int)blockIdx.x + it * (int)gridDim.x;
    const int seq0 = it * FPLANES;  // sequence number of plane -2
    R* const outg = U_out + (size_t)g * (5 * FN * FN * FN);
    R* const bfg = bflux ? bflux + (size_t)g * (30 * FN * FN) : nullptr;
    R* const mfg = (VAR && midflux) ? midflux + (size_t)g * (15 * FN * FN) : nullptr;

    R Wc[5];
    // prologue: planes -2 (own cell only) and -1 (own + extra, published for the x/y neighbours)
    {
      wait_plane(seq0);
      const R* raw = raw_ptr(seq0);
      R U[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = raw[q * (FS * FS) + raw_own];
      {
        R Wm[5];
        cons2prim<R, Fast>(U, c, Wm);
#pragma unroll
        for (int q = 0; q < 5; ++q) wms[q * FNT + t] = Wm[q];
      }
      wait_plane(seq0 + 1);
      raw = raw_ptr(seq0 + 1);
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = raw[q * (FS * FS) + raw_own];
      cons2prim<R, Fast>(U, c, Wc);
      R* wpl = wring + ((seq0 + 1) & 1) * SM::w_plane;
#pragma unroll
      for (int q = 0; q < 5; ++q) wpl[w_own + q * FS] = Wc[q];
      if (has_extra) {
        R We[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) U[q] = raw[q * (FS * FS) + raw_ext];
        cons2prim<R, Fast>(U, c, We);
#pragma unroll
        for (int q = 0; q < 5; ++q) wpl[w_ext + q * FS] = We[q];
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) { zs[q * FNT + t] = Wc[q]; accs[q * FNT + t] = R(0); }
    }
    __syncthreads();

    for (int k = -1; k <= FN; ++k) {
      const int seq = seq0 + k + 2;  // sequence number of plane k
      const bool ghost_plane = (k < 0 || k >= FN);
      // ---- A: primitives of plane k+1 (own cell + extra), published for the next step's x/y neighbours
      {
        wait_plane(seq + 1);
        const R* raw = raw_ptr(seq + 1);
        R U[5], Wp[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) U[q] = raw[q * (FS * FS) + raw_own];
        cons2prim<R, Fast>(U, c, Wp);
        R* wpl = wring + ((seq + 1) & 1) * SM::w_plane;
#pragma unroll
        for (int q = 0; q < 5; ++q) wpl[w_own + q * FS] = Wp[q];   // read back from here where needed: not held in registers
        if (has_extra) {
          R We[5];
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = raw[q * (FS * FS) + raw_ext];
          cons2prim<R, Fast>(U, c, We);
#pragma unroll
          for (int q = 0; q < 5; ++q) wpl[w_ext + q * FS] = We[q];
        }
      }
      // ---- B: reconstruction + half-step prediction of plane k
      R Wf[3][2][5];
      const bool do_pred = ghost_plane ? interior : true;
      if (do_pred) {
        const R* wpl = wring + (seq & 1) * SM::w_plane;
        const volatile R* wnx = wring + ((seq + 1) & 1) * SM::w_plane;
        R Wn_m[3][5], Wn_p[3][5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          Wn_m[0][q] = wpl[w_own + q * FS - 1];
          Wn_p[0][q] = wpl[w_own + q * FS + 1];
          Wn_m[1][q] = wpl[w_own + q * FS - WPITCH];
          Wn_p[1][q] = wpl[w_own + q * FS + WPITCH];
          Wn_m[2][q] = wms[q * FNT + t];
          Wn_p[2][q] = wnx[w_own + q * FS];
        }
        const bool ok = predict_cell<R, LIM, Fast>(Wc, Wn_m, Wn_p, c, Wf);
        n_guard += ok ? 0u : 1u;
        if (!ok) mark_guard(g, FN, i, j, k);
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          xs[q * FNT + t] = Wf[0][1][q];
          ys[q * FNT + t] = Wf[1][1][q];
        }
      }
      __syncthreads();  // S1: x+/y+ states and primitive plane k+1 visible; raw planes <= k-2 retired
      if (t == 0) issue_upto(seq0 + k + 1 + FNSTAGE);  // planes with seq < seq0 + (k-2) + 2 + 1 are free

      // ---- D: Roe fluxes at the lower faces
      R Fx[5], Fy[5], Fz[5];
      const bool do_x = !ghost_plane && in_y && i >= 0;       // face (i-1/2, j, k), i in [0,16]
      const bool do_y = !ghost_plane && in_x && j >= 0;       // face (i, j-1/2, k), j in [0,16]
      const bool do_z = interior && k >= 0;                   // face (i, j, k-1/2), k in [0,16]
      if (do_x) {
        R L[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) L[q] = xs[q * FNT + t_xl];
        bool hl0 = false;
        roe_flux<R, 0, Fast>(L, Wf[0][0], c, Fx, flags, VAR ? &hl0 : nullptr);
        if (VAR && hl0) mark_hlle(g, FN, 0, i, j, k);
        if (VAR && mfg && i == FN / 2) {
#pragma unroll
          for (int q = 0; q < 5; ++q) mfg[(q * FN + k) * FN + j] = Fx[q];
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) fxs[q * FNT + t] = Fx[q];
        if (bfg && (i == 0 || i == FN)) {
          const int face = (i == FN);
#pragma unroll
          for (int q = 0; q < 5; ++q) bfg[((face * 5 + q) * FN + k) * FN + j] = Fx[q];
        }
      }
      if (do_y) {
        R L[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) L[q] = ys[q * FNT + t_yl];
        bool hl1 = false;
        roe_flux<R, 1, Fast>(L, Wf[1][0], c, Fy, flags, VAR ? &hl1 : nullptr);
        if (VAR && hl1) mark_hlle(g, FN, 1, i, j, k);
        if (VAR && mfg && j == FN / 2) {
#pragma unroll
          for (int q = 0; q < 5; ++q) mfg[((5 + q) * FN + k) * FN + i] = Fy[q];
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) fys[q * FNT + t] = Fy[q];
        if (bfg && (j == 0 || j == FN)) {
          const int face = 2 + (j == FN);
#pragma unroll
          for (int q = 0; q < 5; ++q) bfg[((face * 5 + q) * FN + k) * FN + i] = Fy[q];
        }
      }
      if (do_z) {
        R zplus[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) zplus[q] = zs[q * FNT + t];
        bool hl2 = false;
        roe_flux<R, 2, Fast>(zplus, Wf[2][0], c, Fz, flags, VAR ? &hl2 : nullptr);
        if (VAR && hl2) mark_hlle(g, FN, 2, i, j, k);
        if (VAR && mfg && k == FN / 2) {
#pragma unroll
          for (int q = 0; q < 5; ++q) mfg[((10 + q) * FN + j) * FN + i] = Fz[q];
        }
        if (bfg && (k == 0 || k == FN)) {
          const int face = 4 + (k == FN);
#pragma unroll
          for (int q = 0; q < 5; ++q) bfg[((face * 5 + q) * FN + j) * FN + i] = Fz[q];
        }
      }
      __syncthreads();  // S2: Fx, Fy visible

      // ---- E: finish cell (i,j,k-1) with its upper z flux; start cell (i,j,k)
      if (interior) {
        if (k >= 1) {
          const R* rawp = raw_ptr(seq - 1);  // plane k-1 is still resident (retired only after the next S1)
          R out[5];
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            const R Uin = rawp[q * (FS * FS) + raw_own];
            out[q] = Uin - c.lam * (accs[q * FNT + t] + Fz[q]);
            outg[(size_t)q * (FN * FN * FN) + ((k - 1) * FN + j) * FN + i] = out[q];
          }
          const R m2 = out[1] * out[1] + out[2] * out[2] + out[3] * out[3];
          n_nonpos += (out[0] > R(0) && R(2) * out[0] * out[4] > m2) ? 0u : 1u;
        }
        if (k >= 0 && k < FN) {
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            accs[q * FNT + t] = ((fxs[q * FNT + t_xr] - Fx[q]) + (fys[q * FNT + t_yu] - Fy[q])) - Fz[q];
          }
        }
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        wms[q * FNT + t] = Wc[q];
        Wc[q] = (wring + ((seq + 1) & 1) * SM::w_plane)[w_own + q * FS];
        zs[q * FNT + t] = Wf[2][1][q];
      }
    }
    __syncthreads();  // all reads of this group's planes done before its stages are reused
  }

  // diagnostics: one atomic per warp
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
