// csrc/hydro_aux.cuh — the two steps either side of the hot path that a device-resident multi-step run on one
// uniform grid needs (the paper does both on the CPU): the CFL signal-speed
// maximum of reading R15 and the same-level ghost-shell refill of reading R16. Plain streaming kernels: both are
// HBM-bound copies / reductions with no reuse worth staging.
#pragma once
#include <cuda_runtime.h>

namespace gh {

// max over the interior cells of all groups of |vx| + |vy| + |vz| + 3 c_s (R15). U: [G][5][S][S][S] with
// S = N + 2 ghost (ghost = 0 for U_out). The result is accumulated with an integer atomicMax on the bit pattern
// (non-negative IEEE values order like unsigned integers; a NaN orders above them all, so a state holding NaN gives
// a NaN maximum and the caller's dt check trips), so *out must be zeroed before the launch. A cell with rho <= 0 gives
// NaN only while its pressure expression is positive (root of a negative number); with the pressure clamped to 0 its
// speed is <= 0 and it drops out of the maximum — the check is for NaN states, not a positivity check (R10 counts those).
// NC, GC > 0: compile-time patch size and ghost width (the 16 / 2 of the configs: the index arithmetic becomes shifts).
template <class R, class Bits, int NC, int GC>
__global__ void max_speed_kernel(const R* __restrict__ U, long long n_cells, int N_rt, int ghost_rt, R gamma, Bits* out) {
  const int N = NC > 0 ? NC : N_rt, ghost = NC > 0 ? GC : ghost_rt;
  const int S = N + 2 * ghost;
  const long long S3 = (long long)S * S * S, N3 = (long long)N * N * N;
  R m = R(0);
  for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < n_cells; c += (long long)gridDim.x * blockDim.x) {
    const long long g = c / N3;
    const int r = (int)(c - g * N3);
    const int i = r % N, j = (r / N) % N, k = r / (N * N);
    const R* p = U + g * 5 * S3 + ((long long)(k + ghost) * S + (j + ghost)) * S + (i + ghost);
    const R rho = p[0], mx = p[S3], my = p[2 * S3], mz = p[3 * S3], E = p[4 * S3];
    const R ir = R(1) / rho;
    R P = (gamma - R(1)) * (E - R(0.5) * (mx * mx + my * my + mz * mz) * ir);
    P = P > R(0) ? P : R(0);
    const R v = (fabs(mx) + fabs(my) + fabs(mz)) * ir + R(3) * sqrt(gamma * P * ir);
    m = (v > m || v != v) ? v : m;   // a NaN cell makes the maximum NaN (its bit pattern also wins the atomicMax)
  }
  for (int o = 16; o > 0; o >>= 1) {
    const R other = __shfl_xor_sync(0xffffffffu, m, o);
    m = (other > m || other != other) ? other : m;
  }
  if ((threadIdx.x & 31) == 0) {
    Bits b;
    memcpy(&b, &m, sizeof(R));
    atomicMax(out, b);
  }
}

// Ghost-shell refill on one uniform grid of gx x gy x gz groups (group index x-fastest): every stored cell of
// U_in — interior and ghost — is gathered from the interior arrays U_out of the group that owns it, with periodic
// wrap (bc = 0) or outflow = nearest interior cell (bc = 1) per axis (R16). Pure data movement; one CTA per
// group, 32-bit index arithmetic. Since every cell passes through a thread with all five variables, the
// kernel also accumulates the signal-speed maximum of the NEW state (ghost cells are copies of interior cells, so
// they do not change it): vmax may be null.
template <class R> struct alignas(2 * sizeof(R)) Vec2 { R a, b; };

// VEC = 2 (N and ghost even): cells are moved as aligned pairs (x, x+1), which never straddle a group boundary.
// NC, GC > 0: compile-time patch size and ghost width (the 16 / 2 of the configs: constant divisors); 0 = run time.
template <class R, class Bits, int VEC, int NC, int GC>
__global__ void fill_ghosts_kernel(const R* __restrict__ U_out, R* __restrict__ U_in, int gx, int gy, int gz, int N_rt,
                                   int ghost_rt, int bcx, int bcy, int bcz, R gamma, Bits* vmax) {
  const int N = NC > 0 ? NC : N_rt, ghost = NC > 0 ? GC : ghost_rt;
  const int S = N + 2 * ghost;
  const int g = blockIdx.x;
  const int bx = g % gx, by = (g / gx) % gy, bz = g / (gx * gy);
  const int nx = gx * N, ny = gy * N, nz = gz * N;
  const size_t S3 = (size_t)S * S * S, N3 = (size_t)N * N * N;
  R* const dst_group = U_in + (size_t)g * 5 * S3;
  R m = R(0);
  const int SV = S / VEC;
  for (int rv = threadIdx.x; rv < S * S * SV; rv += blockDim.x) {
    const int z = rv / (S * SV), ry = rv - z * (S * SV);
    const int y = ry / SV, x = (ry - y * SV) * VEC, r = y * S + x;
    int Z = bz * N + z - ghost;
    Z = bcz ? (Z < 0 ? 0 : (Z >= nz ? nz - 1 : Z)) : (Z < 0 ? Z + nz : (Z >= nz ? Z - nz : Z));
    const int sgz = Z / N, cz = Z - sgz * N;
    R* const dst_plane = dst_group + (size_t)z * S * S;
    int X = bx * N + x - ghost, Y = by * N + y - ghost;
    X = bcx ? (X < 0 ? 0 : (X >= nx ? nx - 1 : X)) : (X < 0 ? X + nx : (X >= nx ? X - nx : X));
    Y = bcy ? (Y < 0 ? 0 : (Y >= ny ? ny - 1 : Y)) : (Y < 0 ? Y + ny : (Y >= ny ? Y - ny : Y));
    const int sgx = X / N, sgy = Y / N;
    const R* src = U_out + ((size_t)(sgz * gy + sgy) * gx + sgx) * 5 * N3 + (size_t)(cz * N + (Y - sgy * N)) * N + (X - sgx * N);
    R v[VEC][5];
    if (VEC == 2) {
      Vec2<R> t[5];
      // the pair's second cell: contiguous in the source except where an outflow boundary clamps both to one cell
      int X1 = bx * N + x + 1 - ghost;
      X1 = bcx ? (X1 < 0 ? 0 : (X1 >= nx ? nx - 1 : X1)) : (X1 < 0 ? X1 + nx : (X1 >= nx ? X1 - nx : X1));
      if (X1 == X + 1) {
#pragma unroll
        for (int q = 0; q < 5; ++q) t[q] = *reinterpret_cast<const Vec2<R>*>(src + q * N3);
      } else {
        const int d = X1 - X;   // 0 at a clamped boundary
#pragma unroll
        for (int q = 0; q < 5; ++q) { t[q].a = src[q * N3]; t[q].b = src[q * N3 + d]; }
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        *reinterpret_cast<Vec2<R>*>(dst_plane + q * S3 + r) = t[q];
        v[0][q] = t[q].a;
        v[VEC - 1][q] = t[q].b;
      }
    } else {
#pragma unroll
      for (int q = 0; q < 5; ++q) v[0][q] = src[q * N3];
#pragma unroll
      for (int q = 0; q < 5; ++q) dst_plane[q * S3 + r] = v[0][q];
    }
    if (vmax) {
#pragma unroll
      for (int e = 0; e < VEC; ++e) {
        const R ir = R(1) / v[e][0];
        R P = (gamma - R(1)) * (v[e][4] - R(0.5) * (v[e][1] * v[e][1] + v[e][2] * v[e][2] + v[e][3] * v[e][3]) * ir);
        P = P > R(0) ? P : R(0);
        const R sp = (fabs(v[e][1]) + fabs(v[e][2]) + fabs(v[e][3])) * ir + R(3) * sqrt(gamma * P * ir);
        m = (sp > m || sp != sp) ? sp : m;
      }
    }
  }
  if (vmax) {
    // one atomic per CTA (the slot is a single address: with one atomic per warp the 32 768 x 32 of them serialise in L2)
    __shared__ R red[32];
    for (int o = 16; o > 0; o >>= 1) {
      const R other = __shfl_xor_sync(0xffffffffu, m, o);
      m = (other > m || other != other) ? other : m;
    }
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
      m = threadIdx.x < ((blockDim.x + 31) >> 5) ? red[threadIdx.x] : R(0);
      for (int o = 16; o > 0; o >>= 1) {
        const R other = __shfl_xor_sync(0xffffffffu, m, o);
        m = (other > m || other != other) ? other : m;
      }
      if (threadIdx.x == 0) {
        Bits b;
        memcpy(&b, &m, sizeof(R));
        atomicMax(vmax, b);
      }
    }
  }
}

}  // namespace gh
