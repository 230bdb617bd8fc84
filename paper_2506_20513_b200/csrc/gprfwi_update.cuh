// gprfwi_update.cuh -- iteration epilogue: TV term of Algorithm 3
// (Eq. (17); reading R20), gradient mask near the sources
// (reading R18), Adam step with one learning rate per parameter
// (Eqs. (14)-(15), reading R19) and the clamps of PAPER.md:258-260.
// All planes are [nz][pitch] fp32; every kernel is one thread per cell; ~1e-6 of an iteration's work.
//
// TV term of a parameter X (reading R20): s = max|X|, U0 = X/s, U = U0, Z = B = 0; n_it times
//   div = D^T (Z - B)                     circular backward differences
//   U  <- (U0 + rho div + rho sum of the 4 neighbours of U) / (1 + 4 rho)      one Jacobi sweep
//   G  = D U                              circular forward differences
//   Z  = shrink(G + B, lambda / rho)      isotropic: v max(1 - t/|v|, 0), Eq. (17)
//   B += G - Z
// tv_grad = alpha (X - s U).
#pragma once
#include "gprfwi_common.cuh"

namespace gprfwi {

#if defined(__CUDACC__)
__device__ __forceinline__ int wrap(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

// max |x| over the nz x nx cells -> *out (as the bit pattern of a non-negative float; *out zeroed before)
__global__ void absmax_kernel(const float* __restrict__ x, int nz, int nx, int pitch, unsigned* out)
{
  float m = 0.f;
  for (int j = blockIdx.x; j < nz; j += gridDim.x)
    for (int i = threadIdx.x; i < nx; i += blockDim.x) m = fmaxf(m, fabsf(x[(long long)j * pitch + i]));
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));
}

// U0 = U = X / s, Z = B = 0
__global__ void tv_init_kernel(const float* __restrict__ x, int nz, int nx, int pitch, const unsigned* smax,
                               float* u0, float* u, float* zx, float* zz, float* bx, float* bz)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx) return;
  const float s = __uint_as_float(*smax);
  const long long o = (long long)j * pitch + i;
  const float v = s > 0.f ? x[o] / s : 0.f;
  u0[o] = v; u[o] = v; zx[o] = 0.f; zz[o] = 0.f; bx[o] = 0.f; bz[o] = 0.f;
}

// one Jacobi sweep: un from u (old), Z, B
__global__ void tv_jacobi_kernel(int nz, int nx, int pitch, float rho, const float* __restrict__ u0,
                                 const float* __restrict__ u, const float* __restrict__ zx,
                                 const float* __restrict__ zz, const float* __restrict__ bx,
                                 const float* __restrict__ bz, float* __restrict__ un)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx) return;
  const int im = wrap(i - 1, nx), ip = wrap(i + 1, nx), jm = wrap(j - 1, nz), jp = wrap(j + 1, nz);
  const long long r = (long long)j * pitch, rm = (long long)jm * pitch, rp = (long long)jp * pitch;
  // D^T w = -(backward difference of w): (D^T w)[k] = w[k-1] - w[k]
  const float div = ((zx[r + im] - bx[r + im]) - (zx[r + i] - bx[r + i])) +
                    ((zz[rm + i] - bz[rm + i]) - (zz[r + i] - bz[r + i]));
  const float nb = u[r + im] + u[r + ip] + u[rm + i] + u[rp + i];
  un[r + i] = (u0[r + i] + rho * div + rho * nb) / (1.f + 4.f * rho);
}

// G = D u, Z = shrink(G + B, t), B += G - Z
__global__ void tv_shrink_kernel(int nz, int nx, int pitch, float t, const float* __restrict__ u,
                                 float* __restrict__ zx, float* __restrict__ zz, float* __restrict__ bx,
                                 float* __restrict__ bz)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx) return;
  const long long r = (long long)j * pitch, rp = (long long)wrap(j + 1, nz) * pitch;
  const float gx = u[r + wrap(i + 1, nx)] - u[r + i], gz = u[rp + i] - u[r + i];
  const float vx = gx + bx[r + i], vz = gz + bz[r + i];
  const float nrm = sqrtf(vx * vx + vz * vz);
  const float f = nrm > t ? 1.f - t / nrm : 0.f;
  const float nzx = f * vx, nzz = f * vz;
  zx[r + i] = nzx; zz[r + i] = nzz;
  bx[r + i] += gx - nzx; bz[r + i] += gz - nzz;
}

// grad += alpha (X - s U)
__global__ void tv_add_kernel(const float* __restrict__ x, int nz, int nx, int pitch, const unsigned* smax,
                              float alpha, const float* __restrict__ u, float* __restrict__ grad)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx) return;
  const long long o = (long long)j * pitch + i;
  grad[o] += alpha * (x[o] - __uint_as_float(*smax) * u[o]);
}

// mask rows j < mask_rows, Adam moments, bias-corrected step, clamp
__global__ void adam_kernel(int nz, int nx, int pitch, int mask_rows, float lr, float b1, float b2, float eps,
                            float c1, float c2, float xmin, const float* __restrict__ grad,
                            float* __restrict__ m, float* __restrict__ v, float* __restrict__ x)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx) return;
  const long long o = (long long)j * pitch + i;
  const float g = j < mask_rows ? 0.f : grad[o];
  const float mn = b1 * m[o] + (1.f - b1) * g, vn = b2 * v[o] + (1.f - b2) * g * g;
  m[o] = mn; v[o] = vn;
  const float xn = x[o] - lr * (mn * c1) / (sqrtf(vn * c2) + eps);        // c1 = 1/(1-b1^t), c2 = 1/(1-b2^t)
  x[o] = fmaxf(xn, xmin);
}

// Zero-phase FIR along time for the multiscale (frequency-staged) strategy, PAPER.md:529-531:
// out[s][n][r] = sum_k taps[k] * in[s][n + k - (ntaps-1)/2][r], samples outside [0, nt) taken as 0.
// Thread = one (n, r) of one shot; r fastest, so reads and writes are coalesced along receivers.
__global__ void lowpass_kernel(const float* __restrict__ in, float* __restrict__ out, int nt, int nrec,
                               const float* __restrict__ taps, int ntaps)
{
  const long long base = (long long)blockIdx.y * nt * nrec;
  const int half = (ntaps - 1) / 2;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < (long long)nt * nrec;
       k += (long long)gridDim.x * blockDim.x) {
    const int n = (int)(k / nrec), r = (int)(k % nrec);
    float acc = 0.f;
    for (int q = 0; q < ntaps; ++q) {
      const int m = n + q - half;
      if (m >= 0 && m < nt) acc = fmaf(taps[q], in[base + (long long)m * nrec + r], acc);
    }
    out[base + k] = acc;
  }
}

// ---- coarse grid of the early multiscale stages (reading R23): node-aligned 2:1
// coarsening, coarse node (J, I) = fine node (2J, 2I).
// Full-weighting restriction: tensor product of (1/4, 1/2, 1/4) around the fine node, a neighbour outside
// the grid folded onto the centre.
__global__ void restrict_kernel(const float* __restrict__ fine, int nz, int nx, int pitch, float* __restrict__ coarse,
                                int nzc, int nxc, int pitchc)
{
  const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y;
  if (I >= nxc || J >= nzc) return;
  const int jc = 2 * J, ic = 2 * I;
  float acc = 0.f;
#pragma unroll
  for (int dj = -1; dj <= 1; ++dj) {
    const int j = (jc + dj >= 0 && jc + dj < nz) ? jc + dj : jc;
    const float wj = dj == 0 ? 0.5f : 0.25f;
    float row = 0.f;
#pragma unroll
    for (int di = -1; di <= 1; ++di) {
      const int i = (ic + di >= 0 && ic + di < nx) ? ic + di : ic;
      row += (di == 0 ? 0.5f : 0.25f) * fine[(long long)j * pitch + i];
    }
    acc += wj * row;
  }
  coarse[(long long)J * pitchc + I] = acc;
}
// fine += scale * bilinear prolongation of coarse (even fine nodes copy, odd ones average their coarse neighbours)
__global__ void prolong_add_kernel(const float* __restrict__ coarse, int nzc, int nxc, int pitchc, float scale,
                                   float* __restrict__ fine, int nz, int nx, int pitch)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx || j >= nz) return;
  const int j0 = j >> 1, j1 = (j & 1) ? min(j0 + 1, nzc - 1) : j0;
  const int i0 = i >> 1, i1 = (i & 1) ? min(i0 + 1, nxc - 1) : i0;
  const float v = 0.25f * (coarse[(long long)j0 * pitchc + i0] + coarse[(long long)j0 * pitchc + i1] +
                           coarse[(long long)j1 * pitchc + i0] + coarse[(long long)j1 * pitchc + i1]);
  fine[(long long)j * pitch + i] += scale * v;
}
#endif

}  // namespace gprfwi
