// csrc/hydro_generic.cuh — shape-generic path (any N >= 1, ghost >= 2, float or double): three plain
// kernels with intermediates in a global scratch buffer. It exists for shapes the fused sm_100a kernel does
// not cover and as a second, structurally different GPU implementation for the parity tests; it is not
// the performance path (its HBM traffic is ~10x the algorithmic bytes).
//
//   predict_kernel : one thread per cell of the (N+2)^3 cube around the group; steps 1+2 of PAPER.md:15
//                    -> six predicted face states (primitives) in scratch FS[g][face][q][cell]
//   flux_kernel    : one thread per face; step 3 (Roe) -> scratch FL[g][axis][q][face]; boundary fluxes
//   update_kernel  : one thread per interior cell; step 4 -> U_out
#pragma once
#include "hydro_math.cuh"

namespace gh {

struct GenericShape {
  int N, ghost, S, E;               // E = N + 2
  long long in_stride, out_stride;  // reals per group
  long long fs_stride, fl_stride;   // scratch reals per group
};

__host__ __device__ inline GenericShape make_shape(int N, int ghost) {
  GenericShape s;
  s.N = N; s.ghost = ghost; s.S = N + 2 * ghost; s.E = N + 2;
  s.in_stride = 5LL * s.S * s.S * s.S;
  s.out_stride = 5LL * N * N * N;
  s.fs_stride = 30LL * s.E * s.E * s.E;
  s.fl_stride = 15LL * (N + 1) * N * N;
  return s;
}

template <class R>
__device__ __forceinline__ void load_prim(const R* __restrict__ Ug, const GenericShape& sh, int i, int j, int k,
                                          const GasConst<R>& c, R W[5]) {
  const long long vol = (long long)sh.S * sh.S * sh.S;
  const long long at = ((long long)(k + sh.ghost) * sh.S + (j + sh.ghost)) * sh.S + (i + sh.ghost);
  R U[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) U[q] = Ug[q * vol + at];
  cons2prim<R, false>(U, c, W);
}

template <class R, int LIM>
__global__ void __launch_bounds__(128) predict_kernel(const R* __restrict__ U_in, R* __restrict__ FS, GenericShape sh,
                                                      GasConst<R> c, unsigned long long* __restrict__ status,
                                                      long long g0) {
  const int E = sh.E, N = sh.N;
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (long long)E * E * E) return;
  const int i = (int)(e % E) - 1, j = (int)((e / E) % E) - 1, k = (int)(e / ((long long)E * E)) - 1;
  const int nghost = (i < 0 || i >= N) + (j < 0 || j >= N) + (k < 0 || k >= N);
  if (nghost > 1) return;  // only interior cells and first-layer ghosts with one ghost index are needed
  const R* Ug = U_in + (long long)blockIdx.y * sh.in_stride;
  R Wc[5], Wm[3][5], Wp[3][5];
  load_prim(Ug, sh, i, j, k, c, Wc);
  load_prim(Ug, sh, i - 1, j, k, c, Wm[0]); load_prim(Ug, sh, i + 1, j, k, c, Wp[0]);
  load_prim(Ug, sh, i, j - 1, k, c, Wm[1]); load_prim(Ug, sh, i, j + 1, k, c, Wp[1]);
  load_prim(Ug, sh, i, j, k - 1, c, Wm[2]); load_prim(Ug, sh, i, j, k + 1, c, Wp[2]);
  R Wf[3][2][5];
  const bool ok = predict_cell<R, LIM, false>(Wc, Wm, Wp, c, Wf);
  if (!ok) {
    atomicAdd(&status[0], 1ULL);
    mark_guard(g0 + blockIdx.y, N, i, j, k);
  }
  R* out = FS + (long long)blockIdx.y * sh.fs_stride + e;
  const long long ev = (long long)E * E * E;
#pragma unroll
  for (int d = 0; d < 3; ++d)
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int q = 0; q < 5; ++q) out[((d * 2 + s) * 5 + q) * ev] = Wf[d][s][q];
}

template <class R, int n>
__device__ __forceinline__ void flux_face(const R* __restrict__ FSg, R* __restrict__ FLg, R* __restrict__ bf,
                                          const GenericShape& sh, const GasConst<R>& c, int i, int j, int k, int flags,
                                          R* __restrict__ mf, long long g) {
  // face on the lower side of cell (i,j,k) along axis n; i in [0, N] along n
  const int E = sh.E, N = sh.N;
  const long long ev = (long long)E * E * E;
  const int di = (n == 0), dj = (n == 1), dk = (n == 2);
  const long long er = ((long long)(k + 1) * E + (j + 1)) * E + (i + 1);
  const long long el = ((long long)(k + 1 - dk) * E + (j + 1 - dj)) * E + (i + 1 - di);
  R L[5], Rt[5], F[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    L[q] = FSg[((n * 2 + 1) * 5 + q) * ev + el];
    Rt[q] = FSg[((n * 2 + 0) * 5 + q) * ev + er];
  }
  bool hl = false;
  roe_flux<R, n, false>(L, Rt, c, F, flags, flags ? &hl : nullptr);
  if (hl) mark_hlle(g, N, n, i, j, k);
  const int fx = N + di, fy = N + dj;
  const long long nf = (long long)(N + 1) * N * N;
  const long long f = ((long long)k * fy + j) * fx + i;
#pragma unroll
  for (int q = 0; q < 5; ++q) FLg[(n * 5 + q) * nf + f] = F[q];
  if (mf && (n == 0 ? i : (n == 1 ? j : k)) == N / 2) {   // mid-plane fluxes (R12b), in-face layout of the outer faces
    const int a = n == 2 ? j : k, b = n == 0 ? j : i;
#pragma unroll
    for (int q = 0; q < 5; ++q) mf[((n * 5 + q) * N + a) * N + b] = F[q];
  }
  if (bf) {
    const int along = n == 0 ? i : (n == 1 ? j : k);
    if (along == 0 || along == N) {
      const int side = along == N;
      // in-face index: x faces [k][j], y faces [k][i], z faces [j][i]
      const int a = n == 2 ? j : k, b = n == 0 ? j : i;
#pragma unroll
      for (int q = 0; q < 5; ++q) bf[(((2 * n + side) * 5 + q) * N + a) * N + b] = F[q];
    }
  }
}

template <class R>
__global__ void __launch_bounds__(128) flux_kernel(const R* __restrict__ FS, R* __restrict__ FL, R* __restrict__ bflux,
                                                   GenericShape sh, GasConst<R> c, int flags, R* __restrict__ midflux,
                                                   long long g0) {
  const int N = sh.N;
  const long long nf = (long long)(N + 1) * N * N;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 3 * nf) return;
  const int n = (int)(t / nf);
  const long long f = t % nf;
  const R* FSg = FS + (long long)blockIdx.y * sh.fs_stride;
  R* FLg = FL + (long long)blockIdx.y * sh.fl_stride;
  R* bf = bflux ? bflux + (long long)blockIdx.y * 30 * N * N : nullptr;
  R* mf = midflux ? midflux + (long long)blockIdx.y * 15 * N * N : nullptr;
  const int fx = N + (n == 0), fy = N + (n == 1);
  const int i = (int)(f % fx), j = (int)((f / fx) % fy), k = (int)(f / ((long long)fx * fy));
  const long long g = g0 + blockIdx.y;
  if (n == 0) flux_face<R, 0>(FSg, FLg, bf, sh, c, i, j, k, flags, mf, g);
  else if (n == 1) flux_face<R, 1>(FSg, FLg, bf, sh, c, i, j, k, flags, mf, g);
  else flux_face<R, 2>(FSg, FLg, bf, sh, c, i, j, k, flags, mf, g);
}

template <class R>
__global__ void __launch_bounds__(128) update_kernel(const R* __restrict__ U_in, const R* __restrict__ FL,
                                                     R* __restrict__ U_out, GenericShape sh, GasConst<R> c,
                                                     unsigned long long* __restrict__ status) {
  const int N = sh.N, S = sh.S;
  const long long nc = (long long)N * N * N;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nc) return;
  const int i = (int)(t % N), j = (int)((t / N) % N), k = (int)(t / ((long long)N * N));
  const R* Ug = U_in + (long long)blockIdx.y * sh.in_stride;
  const R* FLg = FL + (long long)blockIdx.y * sh.fl_stride;
  R* Og = U_out + (long long)blockIdx.y * sh.out_stride;
  const long long nf = (long long)(N + 1) * N * N;
  const long long vol = (long long)S * S * S;
  const long long at = ((long long)(k + sh.ghost) * S + (j + sh.ghost)) * S + (i + sh.ghost);
  const long long fxl = ((long long)k * N + j) * (N + 1) + i;   // x faces: [k][j][i'], i' in [0,N]
  const long long fyl = ((long long)k * (N + 1) + j) * N + i;   // y faces: [k][j'][i]
  const long long fzl = ((long long)k * N + j) * N + i;         // z faces: [k'][j][i]
  R out[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const R dFx = FLg[(0 * 5 + q) * nf + fxl + 1] - FLg[(0 * 5 + q) * nf + fxl];
    const R dFy = FLg[(1 * 5 + q) * nf + fyl + N] - FLg[(1 * 5 + q) * nf + fyl];
    const R dFz = FLg[(2 * 5 + q) * nf + fzl + (long long)N * N] - FLg[(2 * 5 + q) * nf + fzl];
    out[q] = Ug[q * vol + at] - c.lam * ((dFx + dFy) + dFz);
    Og[q * nc + t] = out[q];
  }
  const R m2 = out[1] * out[1] + out[2] * out[2] + out[3] * out[3];
  if (!(out[0] > R(0) && R(2) * out[0] * out[4] > m2)) atomicAdd(&status[1], 1ULL);
}

}  // namespace gh
