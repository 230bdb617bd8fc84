// gprfwi_misc.cuh -- coefficient build (kernel a), gradient chain rule, residual/misfit.
#pragma once
#include "gprfwi_common.cuh"

namespace gprfwi {

constexpr float kEps0 = 8.8541878128e-12f;   // 1/(mu0 c0^2)
constexpr float kPecSigma = 100.0f;          // sigma above this is treated as PEC

// Ca = uE0 = EB/EA, Cb = uE4 = 1/EA with EA = e0*er/dt + sigma/2, EB = e0*er/dt - sigma/2
// (the paper's `ucget`; listing truncated after EA, reading R2).
GPR_HD void coef_cell(float er, float sg, float rdt, float& ca, float& cb)
{
  if (sg > kPecSigma) { ca = 0.f; cb = 0.f; return; }
  const float a = kEps0 * er * rdt;
  const float EA = a + 0.5f * sg, EB = a - 0.5f * sg;
  ca = EB / EA;
  cb = 1.0f / EA;
}

// chain rule Ca, Cb -> eps_r, sigma.  gcb_cb is the adjoint kernel's sum
// mu (E^{n+1} - Ca E^n), i.e. Cb * dJ/dCb; with Cb = 1/EA the division by Cb is a multiplication by EA.
GPR_HD void grad_cell(float er, float sg, float rdt, float gca, float gcb_cb, float& ge, float& gs)
{
  if (sg > kPecSigma) { ge = 0.f; gs = 0.f; return; }
  const float a = kEps0 * er * rdt;
  const float EA = a + 0.5f * sg;
  const float gcb = gcb_cb * EA;
  const float r2 = 1.0f / (EA * EA);
  ge = kEps0 * rdt * (gca * sg - gcb) * r2;
  gs = -(gca * a + 0.5f * gcb) * r2;
}

#if defined(__CUDACC__)
// mu_r (optional, [nz][upitch]): per-cell Db = (dt/mu0) / mu_r in the internal column order (the paper's uH4,
// PAPER.md:291-295; reading R22), 0 outside the grid; with mu_r = 1 it equals the scalar Db bit for bit
__global__ void coef_kernel(const float* __restrict__ eps_r, const float* __restrict__ sigma,
                            const float* __restrict__ mu_r, int upitch, int nz, int nx, int pitch, float rdt,
                            float Db, float* __restrict__ ca, float* __restrict__ cb, float* __restrict__ dbc)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= pitch || j >= nz) return;
  float a = 0.f, b = 0.f;
  // the PEC ring (never updated, reading R5) and the pitch padding carry Ca = Cb = 0: the update
  // kernels then keep those nodes at zero without any bounds test
  if (i >= 1 && i <= nx - 2 && j >= 1 && j <= nz - 2)
    coef_cell(eps_r[(long long)j * upitch + i], sigma[(long long)j * upitch + i], rdt, a, b);
  ca[(long long)j * pitch + col_pos(i)] = a;          // internal column order: gprfwi_common.cuh
  cb[(long long)j * pitch + col_pos(i)] = b;
  if (mu_r) dbc[(long long)j * pitch + col_pos(i)] = i < nx ? __fdiv_rn(Db, mu_r[(long long)j * upitch + i]) : 0.f;
}

__global__ void grad_finalize_kernel(const float* __restrict__ eps_r, const float* __restrict__ sigma, int upitch,
                                     int nz, int nx, int pitch, long long plane, int ngroups, float rdt,
                                     const float* __restrict__ gca, const float* __restrict__ gcb,
                                     float* __restrict__ grad_eps, float* __restrict__ grad_sig)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= nx || j >= nz) return;
  float sa = 0.f, sb = 0.f;
  for (int g = 0; g < ngroups; ++g) {
    sa += gca[g * plane + (long long)j * pitch + col_pos(i)];      // internal column order
    sb += gcb[g * plane + (long long)j * pitch + col_pos(i)];
  }
  float ge = 0.f, gs = 0.f;                                  // the PEC ring does not depend on the model
  if (i >= 1 && i <= nx - 2 && j >= 1 && j <= nz - 2)
    grad_cell(eps_r[(long long)j * upitch + i], sigma[(long long)j * upitch + i], rdt, sa, sb, ge, gs);
  grad_eps[(long long)j * upitch + i] = ge;
  grad_sig[(long long)j * upitch + i] = gs;
}

// residual = d_syn - d_obs; optional 0.5*sum(residual^2) in float64 (Eq. (6))
__global__ void residual_kernel(const float* __restrict__ d_syn, const float* __restrict__ d_obs,
                                float* __restrict__ res, size_t n, double* misfit)
{
  double acc = 0.0;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
    const float r = d_syn[k] - d_obs[k];
    res[k] = r;
    acc += 0.5 * (double)r * (double)r;
  }
  if (misfit) {
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    __shared__ double sm[32];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sm[w] = acc;
    __syncthreads();
    if (w == 0) {
      acc = l < (int)(blockDim.x >> 5) ? sm[l] : 0.0;
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
      if (l == 0) atomicAdd(misfit, acc);
    }
  }
}
#endif

}  // namespace gprfwi
