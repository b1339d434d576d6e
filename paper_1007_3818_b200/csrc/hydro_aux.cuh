// csrc/hydro_aux.cuh — the two steps either side of the hot path that a device-resident multi-step run on one
// uniform grid needs (the paper does both on the CPU): the CFL signal-speed
// maximum of reading R15 and the same-level ghost-shell refill of reading R16. Plain streaming kernels: both are
// HBM-bound copies / reductions with no reuse worth staging.
#pragma once
#include <cuda_runtime.h>

namespace gh {

// max over the interior cells of all groups of |vx| + |vy| + |vz| + 3 c_s (R15). U: [G][5][S][S][S] with
// S = N + 2 ghost (ghost = 0 for U_out). The result is accumulated with an integer atomicMax on the bit pattern
// (non-negative IEEE values order like unsigned integers), so *out must be zeroed before the launch.
template <class R, class Bits>
__global__ void max_speed_kernel(const R* __restrict__ U, long long n_cells, int N, int ghost, R gamma, Bits* out) {
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
    m = v > m ? v : m;   // NaN never wins
  }
  for (int o = 16; o > 0; o >>= 1) {
    const R other = __shfl_xor_sync(0xffffffffu, m, o);
    m = other > m ? other : m;
  }
  if ((threadIdx.x & 31) == 0) {
    Bits b;
    memcpy(&b, &m, sizeof(R));
    atomicMax(out, b);
  }
}

// Ghost-shell refill on one uniform grid of gx x gy x gz groups (group index x-fastest): every stored cell of
// U_in — interior and ghost — is gathered from the interior arrays U_out of the group that owns it, with periodic
// wrap (bc = 0) or outflow = nearest interior cell (bc = 1) per axis (R16). Pure data movement.
template <class R>
__global__ void fill_ghosts_kernel(const R* __restrict__ U_out, R* __restrict__ U_in, int gx, int gy, int gz, int N,
                                   int ghost, int bcx, int bcy, int bcz) {
  const int S = N + 2 * ghost;
  const long long S3 = (long long)S * S * S, N3 = (long long)N * N * N;
  const long long total = (long long)gx * gy * gz * S3;
  const int nx = gx * N, ny = gy * N, nz = gz * N;
  for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < total; c += (long long)gridDim.x * blockDim.x) {
    const long long g = c / S3;
    const int r = (int)(c - g * S3);
    const int x = r % S, y = (r / S) % S, z = r / (S * S);
    const int bx = (int)(g % gx), by = (int)((g / gx) % gy), bz = (int)(g / ((long long)gx * gy));
    int X = bx * N + x - ghost, Y = by * N + y - ghost, Z = bz * N + z - ghost;
    X = bcx ? (X < 0 ? 0 : (X >= nx ? nx - 1 : X)) : ((X % nx) + nx) % nx;
    Y = bcy ? (Y < 0 ? 0 : (Y >= ny ? ny - 1 : Y)) : ((Y % ny) + ny) % ny;
    Z = bcz ? (Z < 0 ? 0 : (Z >= nz ? nz - 1 : Z)) : ((Z % nz) + nz) % nz;
    const long long sg = ((long long)(Z / N) * gy + (Y / N)) * gx + (X / N);
    const R* src = U_out + sg * 5 * N3 + ((long long)(Z % N) * N + (Y % N)) * N + (X % N);
    R* dst = U_in + g * 5 * S3 + r;
#pragma unroll
    for (int q = 0; q < 5; ++q) dst[q * S3] = src[q * N3];
  }
}

}  // namespace gh
