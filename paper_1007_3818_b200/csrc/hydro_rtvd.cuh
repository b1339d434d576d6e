// csrc/hydro_rtvd.cuh — the relaxing-TVD hydrodynamic solver ("second-order relaxing total variation
// diminishing (TVD) method (Trac & Pen 2003)", dimensionally split; "seven points" => 3 ghost cells) for
// sm_100a: SURVEY.md §8(f) rank 3, the second workload. Readings RT1–RT8 of DESIGN.md §13.
//
// One persistent CTA per SM streams 16^3 patch groups. A group with its 3-cell ghost shell is ONE contiguous block
// of 5 x 22^3 floats = 212 960 B, so it arrives in shared memory by 1-D bulk async copies (cp.async.bulk, SASS
// UBLKCP, one per variable, completion on one mbarrier) — a tiled tensor map cannot describe it (88-byte rows); the
// tile is single-buffered (it fills shared memory), so the next group's copy starts variable by variable behind the
// output copy of the current one, and is prefetched into L2 during the sweeps. The three sweeps
// run in place in that tile: a thread owns one LINE of 22 cells along the sweep axis and marches along it with the
// half-step state, the right- / left-moving fluxes of the last four cells and the last face flux in registers; a
// cell is overwritten three steps after it was last read, so no second tile is needed. Lines are independent: one
// CTA barrier between sweeps. Per group 484 + 352 + 256 lines (the valid range shrinks by 3 per side along a swept
// axis only). The updated 16^3 interior goes out with coalesced row stores.
#pragma once
#include <cuda.h>
#include <stdint.h>

#include <type_traits>

#include "hydro_fused.cuh"  // mbarrier helpers, smem_u32

namespace gh {

constexpr int RN = 16, RG = 3, RS = RN + 2 * RG;   // 22
constexpr int RNT = 512;                           // threads per CTA
constexpr int RVOL = RS * RS * RS;                 // 10648 cells per variable
constexpr int RTILE_BYTES = 5 * RVOL * 4;          // 212960
struct RtvdSmem {
  static constexpr int off_tile = 0;
  static constexpr int off_bar = ((RTILE_BYTES + 15) / 16) * 16;
  static constexpr int total = off_bar + 16;
};

struct RtvdConst {
  float lam, hlam, g1, gamma;
};

__device__ __forceinline__ float r_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float r_sqrt(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// right- / left-moving fluxes fr = (c u + F_d(u)) / 2, fl = (c u - F_d(u)) / 2 of one cell (RT1, RT6)
template <int d>
__device__ __forceinline__ void rtvd_split(const float u[5], const RtvdConst& c, float fr[5], float fl[5]) {
  const float ir = r_rcp(u[0]);
  const float v = u[1 + d] * ir;
  const float ke = 0.5f * (u[1] * u[1] + u[2] * u[2] + u[3] * u[3]) * ir;
  const float P = c.g1 * (u[4] - ke);
  const float cs = r_sqrt(c.gamma * fmaxf(P, 0.0f) * ir);
  const float hc = 0.5f * (fabsf(v) + cs), hv = 0.5f * v, hP = 0.5f * P;
  // F = u v + P e_d (momentum along d), (E + P) v (energy): halved on the fly
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const float hF = u[q] * hv + ((q == 1 + d) ? hP : 0.0f);
    fr[q] = fmaf(hc, u[q], hF);
    fl[q] = fmaf(hc, u[q], -hF);
  }
  const float hF4 = (u[4] + P) * hv;
  fr[4] = fmaf(hc, u[4], hF4);
  fl[4] = fmaf(hc, u[4], -hF4);
}

// van Leer limiter of the two one-sided HALF differences x / 2, y / 2 (RT3), given the whole differences:
// 2 (x/2)(y/2) / (x/2 + y/2) = x y / (x + y); the halvings are exact, so the result has the bits of the textbook form
__device__ __forceinline__ float rtvd_vanleer_half(float x, float y) {
  const float p = x * y;
  const float q = p * r_rcp(x + y);
  return p > 0.0f ? q : 0.0f;
}

// One line of 22 cells along axis d, in place (cells 3 .. 18 change). p: the line's first cell of variable 0;
// st: stride between cells of the line (floats); variables are RVOL floats apart.
// The march is unrolled by four so that the queues of the last four cells' split fluxes rotate by RENAMING (slot
// (m + k) & 3 is a compile-time constant inside the unrolled body) instead of by register moves — a quarter of the
// instructions of the rolled loop were MOVs.
template <int d>
__device__ __forceinline__ void rtvd_line(float* p, int st, const RtvdConst& c) {
  float up[5], h_prev[5], frp[5];          // previous cell, previous half-step face flux, its right-moving flux
  float A[4][5], B[4][5];                  // fr / fl of the half-step state of the cells m-4 .. m-1: cell n in slot n & 3
  float DA[4][5], DB[4][5];                // their differences to the cell before (only the live ones occupy registers)
  float fu_prev[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    up[q] = h_prev[q] = frp[q] = fu_prev[q] = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) A[k][q] = B[k][q] = DA[k][q] = DB[k][q] = 0.0f;
  }
  // one cell of the march; R = m & 3 (compile time: the queue slots), the three stages switched on at compile time so
  // that the first cells (which only fill the queues) and the steady part are each straight-line code without merges
  auto cell = [&](auto r_c, auto u1_c, auto tvd_c, auto store_c, int m) {
    constexpr int r = decltype(r_c)::value;
    constexpr bool DO_U1 = decltype(u1_c)::value, DO_TVD = decltype(tvd_c)::value, DO_STORE = decltype(store_c)::value;
    float uc[5], fr[5], fl[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) uc[q] = p[q * RVOL + m * st];
    rtvd_split<d>(uc, c, fr, fl);
    float h[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) h[q] = frp[q] - fl[q];                 // half-step face flux at m - 1/2
    if (DO_U1) {
      // half-step state of cell m-1 and its split fluxes (RT2) -> slot (m - 1) & 3 = (r + 3) & 3
      float u1[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) u1[q] = fmaf(-c.hlam, h[q] - h_prev[q], up[q]);
      rtvd_split<d>(u1, c, A[(r + 3) & 3], B[(r + 3) & 3]);
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        DA[(r + 3) & 3][q] = A[(r + 3) & 3][q] - A[(r + 2) & 3][q];
        DB[(r + 3) & 3][q] = B[(r + 3) & 3][q] - B[(r + 2) & 3][q];
      }
      if (DO_TVD) {
        // second-order TVD flux at the face j + 1/2, j = m - 3 (cell n lives in slot n & 3: j in r + 1):
        // FR = fr_j + vl((fr_j - fr_j-1) / 2, (fr_j+1 - fr_j) / 2), FL = fl_j+1 + vl((fl_j - fl_j+1) / 2, (fl_j+1 - fl_j+2) / 2)
        // and vl is odd
        float fu[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const float FR = A[(r + 1) & 3][q] + rtvd_vanleer_half(DA[(r + 1) & 3][q], DA[(r + 2) & 3][q]);
          const float FL = B[(r + 2) & 3][q] - rtvd_vanleer_half(DB[(r + 2) & 3][q], DB[(r + 3) & 3][q]);
          fu[q] = FR - FL;
        }
        if (DO_STORE) {
          float* o = p + (m - 3) * st;
#pragma unroll
          for (int q = 0; q < 5; ++q) o[q * RVOL] = fmaf(-c.lam, fu[q] - fu_prev[q], o[q * RVOL]);   // RT8
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) fu_prev[q] = fu[q];
      }
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) { up[q] = uc[q]; h_prev[q] = h[q]; frp[q] = fr[q]; }
  };
  using Y = std::true_type;
  using N = std::false_type;
  using R0 = std::integral_constant<int, 0>;
  using R1 = std::integral_constant<int, 1>;
  using R2 = std::integral_constant<int, 2>;
  using R3 = std::integral_constant<int, 3>;
  cell(R0{}, N{}, N{}, N{}, 0); cell(R1{}, N{}, N{}, N{}, 1);
  cell(R2{}, Y{}, N{}, N{}, 2); cell(R3{}, Y{}, N{}, N{}, 3);
  cell(R0{}, Y{}, N{}, N{}, 4); cell(R1{}, Y{}, Y{}, N{}, 5);
  cell(R2{}, Y{}, Y{}, Y{}, 6); cell(R3{}, Y{}, Y{}, Y{}, 7);
#pragma unroll 1
  for (int m0 = 8; m0 < 20; m0 += 4) {
    cell(R0{}, Y{}, Y{}, Y{}, m0); cell(R1{}, Y{}, Y{}, Y{}, m0 + 1);
    cell(R2{}, Y{}, Y{}, Y{}, m0 + 2); cell(R3{}, Y{}, Y{}, Y{}, m0 + 3);
  }
  cell(R0{}, Y{}, Y{}, Y{}, 20); cell(R1{}, Y{}, Y{}, Y{}, 21);
}

// all lines of one sweep: `na` x `nb` lines, line (ia, ib) starts at a0 * sa + b0 * sb + ia * sa + ib * sb
template <int d>
__device__ __forceinline__ void rtvd_sweep(float* tile, int na, int nb, int a_lo, int b_lo, int sa, int sb, int st,
                                           const RtvdConst& c) {
  for (int l = (int)threadIdx.x; l < na * nb; l += RNT) {
    const int ia = l % na, ib = l / na;
    rtvd_line<d>(tile + (a_lo + ia) * sa + (b_lo + ib) * sb, st, c);
  }
}

template <int SWEEP>
__global__ void __launch_bounds__(RNT, 1)
    rtvd_kernel(const float* __restrict__ U_in, float* __restrict__ U_out, int n_groups, const RtvdConst c) {
  extern __shared__ __align__(128) unsigned char rsmem[];
  float* const tile = reinterpret_cast<float*>(rsmem + RtvdSmem::off_tile);
  const uint32_t bar = smem_u32(rsmem + RtvdSmem::off_bar);
  const uint32_t tile_s = smem_u32(tile);
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  uint32_t phase = 0;
  // one variable of a group's tile: 22^3 floats = 42 592 B (a multiple of 16), its own bulk copy on the common barrier
  auto load_var = [&](int g, int q) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     tile_s + (uint32_t)(q * RVOL * 4)),
                 "l"(U_in + (size_t)g * (5 * RVOL) + (size_t)q * RVOL), "r"(RVOL * 4), "r"(bar)
                 : "memory");
  };
  if (threadIdx.x == 0 && (int)blockIdx.x < n_groups) {
    mbar_expect_tx(bar, RTILE_BYTES);
    for (int q = 0; q < 5; ++q) load_var((int)blockIdx.x, q);
  }
  for (int g = (int)blockIdx.x; g < n_groups; g += (int)gridDim.x) {
    mbar_wait(bar, phase);
    phase ^= 1u;
    const int g_next = g + (int)gridDim.x;
    // the tile is single-buffered (213 KB): the next group's copy starts variable by variable behind the output copy
    // below; pull it into L2 meanwhile
    if (threadIdx.x == 0 && g_next < n_groups)
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(U_in + (size_t)g_next * (5 * RVOL)), "r"(RTILE_BYTES)
                   : "memory");
    // x fastest: cell (x, y, z) of variable q at q RVOL + z 484 + y 22 + x (RT7)
    if (SWEEP == 0) {
      rtvd_sweep<0>(tile, RS, RS, 0, 0, RS, RS * RS, 1, c);              // x lines: all (y, z)
      __syncthreads();
      rtvd_sweep<1>(tile, RN, RS, RG, 0, 1, RS * RS, RS, c);             // y lines: x interior, all z
      __syncthreads();
      rtvd_sweep<2>(tile, RN, RN, RG, RG, 1, RS, RS * RS, c);            // z lines: x, y interior
    } else {
      rtvd_sweep<2>(tile, RS, RS, 0, 0, 1, RS, RS * RS, c);              // z lines: all (x, y)
      __syncthreads();
      rtvd_sweep<1>(tile, RS, RN, 0, RG, 1, RS * RS, RS, c);             // y lines: all x, z interior
      __syncthreads();
      rtvd_sweep<0>(tile, RN, RN, RG, RG, RS, RS * RS, 1, c);            // x lines: y, z interior
    }
    __syncthreads();
    float* const og = U_out + (size_t)g * (5 * RN * RN * RN);
    if (threadIdx.x == 0 && g_next < n_groups) mbar_expect_tx(bar, RTILE_BYTES);
    for (int q = 0; q < 5; ++q) {
      for (int e = (int)threadIdx.x; e < RN * RN * RN; e += RNT) {
        const int x = e & 15, y = (e >> 4) & 15, z = e >> 8;
        og[q * (RN * RN * RN) + e] = tile[q * RVOL + ((z + RG) * RS + (y + RG)) * RS + (x + RG)];
      }
      __syncthreads();   // every read of variable q's part of the tile is done: the next group's variable q may land
      if (threadIdx.x == 0 && g_next < n_groups) {
        // those reads went through the generic proxy: order them before the async write
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        load_var(g_next, q);
      }
    }
  }
}

}  // namespace gh
