// gprfwi_adj.cuh -- one reverse time step of the exact discrete adjoint + gradient accumulation
// (kernel e of north_star; Algorithm 2).  Transposes gprfwi_fwd.cuh's step:
//
//   mu   = lamE (0 on the PEC ring)                      gCa += mu * E^n
//   q    = Cb * mu                                       gCb += mu * (E^{n+1} - Ca E^n) / Cb
//   tx   = q/kex + cex*(lpezx + q)      lpezx' = bex*(lpezx + q)          (transpose of E CPML)
//   tz   = -q/kez + cez*(lpezz - q)     lpezz' = bez*(lpezz - q)
//   lamHy' = lamHy + (tx[i] - tx[i+1])/dx     lamHx' = lamHx + (tz[j] - tz[j+1])/dx
//   sx   = Db*lamHy'/khx + chx*(lphyx + Db*lamHy')    lphyx' = bhx*(...)  (transpose of H CPML)
//   sz   = -Db*lamHx'/khz + chz*(lphxz - Db*lamHx')   lphxz' = bhz*(...)
//   lamE' = Ca*mu + (sz[j-1] - sz[j])/dx + (sx[i-1] - sx[i])/dx  [+ residual[n] at receivers]
//
// (derivation: DESIGN.md section 4).  Same structure as the forward step -- a 5-point gather on lamE
// through the intermediate lamH -- so the same ping-pong / recompute-the-edge scheme is used.
// Gradients are reduced over the shots of a group inside the thread (the thread owns its cells'
// accumulators for its group), so no atomics are needed and the result is deterministic.
#pragma once
#include "gprfwi_common.cuh"

namespace gprfwi {

struct AdjArgs {
  Geo g;
  State in, out;              // adjoint variables, ping-pong
  const float *ca, *cb;       // [nz][pitch]
  const float *en, *en1;      // forward Ez^n, Ez^{n+1}: [S][nz][pitch] (local shot 0)
  float *gca, *gcb;           // [ngroups][nz][pitch] accumulators
  const float* residual;      // sample n of local shot 0, receiver 0; shot s at + s*trace_stride
  long long trace_stride;     // nt * R
  const int* rec_off;         // [S][R] (local shot 0)
  const int* blk_start;       // [S][tiles_y*tiles_x + 1] CSR: receivers inside each block tile
  const int* blk_rec;         // [S][R] receiver indices sorted by block
  int R;
  int nshots;                 // shots in this pass
  int group;                  // shots per gradient group
  int tiles_x, tiles_y;
};

// lamE row j (columns i0-1..i0+4) times Cb -> q[0..5]; mu[0..5]; zero on/outside the PEC ring
GPR_HD void adj_load_q6(const AdjArgs& a, int s, int j, int i0, float* mu, float* q)
{
  const Geo& g = a.g;
  if (j < 1 || j > g.nz - 2) {
#pragma unroll
    for (int k = 0; k < 6; ++k) { mu[k] = 0.f; q[k] = 0.f; }
    return;
  }
  const float* row = a.in.ez + s * g.plane + (long long)j * g.pitch;
  const float* cbr = a.cb + (long long)j * g.pitch;
  float cb[6];
  unpack(ld4(row + i0), mu + 1);
  unpack(ld4(cbr + i0), cb + 1);
  mu[0] = i0 > 0 ? row[i0 - 1] : 0.f;
  cb[0] = i0 > 0 ? cbr[i0 - 1] : 0.f;
  mu[5] = i0 + 4 < g.nx ? row[i0 + 4] : 0.f;
  cb[5] = i0 + 4 < g.nx ? cbr[i0 + 4] : 0.f;
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    const int i = i0 - 1 + k;
    if (i < 1 || i > g.nx - 2) mu[k] = 0.f;
    q[k] = cb[k] * mu[k];
  }
}

// tz (row j, columns i0..i0+3) from q4 = q[j][i0..i0+3]; updates lpezz of row j if `store`
GPR_HD void adj_tz_row(const AdjArgs& a, int s, int j, int i0, const float* q4, float* tz, bool store)
{
  const Geo& g = a.g;
  const int zs = (j >= 1 && j <= g.nz - 2) ? strip_e(j, g.nz, g.P) : -1;
  if (zs < 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) tz[k] = -q4[k];        // q is 0 on the ring rows
    return;
  }
  const long long po = s * g.zstrip + (long long)zs * g.pitch + i0;
  float p[4];
  unpack(ld4(a.in.pezz + po), p);
  const float b = g.bez[j], c = g.cez[j], ik = g.kez[j];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int i = i0 + k;
    if (i < 1 || i > g.nx - 2) { tz[k] = 0.f; p[k] = 0.f; continue; }
    const float T = p[k] - q4[k];
    tz[k] = -q4[k] * ik + c * T;
    p[k] = b * T;
  }
  if (store) st4(a.out.pezz + po, mk4(p[0], p[1], p[2], p[3]));
}

// sz (row j) from the updated lamHx of row j = lamHx + (tz[j] - tz[j+1])/dx; stores if `store`
GPR_HD void adj_sz_row(const AdjArgs& a, int s, int j, int i0, const float* tz_j, const float* tz_j1,
                       float* sz, bool store)
{
  const Geo& g = a.g;
  if (j < 0 || j > g.nz - 2) {
    sz[0] = sz[1] = sz[2] = sz[3] = 0.f;
    if (store && j >= 0 && j < g.nz) st4(a.out.hx + s * g.plane + (long long)j * g.pitch + i0, mk4(0, 0, 0, 0));
    return;
  }
  const long long o = s * g.plane + (long long)j * g.pitch + i0;
  float h[4];
  unpack(ld4(a.in.hx + o), h);
#pragma unroll
  for (int k = 0; k < 4; ++k) h[k] += (tz_j[k] - tz_j1[k]) * g.rdx;
  if (store) st4(a.out.hx + o, mk4(h[0], h[1], h[2], h[3]));
  const int zs = strip_h(j, g.nz, g.P);
  if (zs >= 0) {
    const long long po = s * g.zstrip + (long long)zs * g.pitch + i0;
    float p[4];
    unpack(ld4(a.in.phxz + po), p);
    const float b = g.bhz[j], c = g.chz[j], ik = g.khz[j];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float px = -g.Db * h[k];
      const float T = p[k] + px;
      sz[k] = px * ik + c * T;
      p[k] = b * T;
    }
    if (store) st4(a.out.phxz + po, mk4(p[0], p[1], p[2], p[3]));
  } else {
#pragma unroll
    for (int k = 0; k < 4; ++k) sz[k] = -g.Db * h[k];
  }
}

GPR_HD void adj_thread_shot(const AdjArgs& a, int s, int grp, int i0, int j0)
{
  const Geo& g = a.g;
  const bool xpml_e = (i0 - 1 < g.P) || (i0 + 4 >= g.nx - g.P);
  const bool xpml_h = (i0 - 1 < g.P) || (i0 + 3 >= g.nx - 1 - g.P);
  float mu_c[6], q_c[6], mu_n[6], q_n[6], tz_c[4], tz_n[4], sz_p[4], sz_c[4];
  {
    float mu_m[6], q_m[6], tz_m[4];
    adj_load_q6(a, s, j0 - 1, i0, mu_m, q_m);
    adj_load_q6(a, s, j0, i0, mu_c, q_c);
    adj_tz_row(a, s, j0 - 1, i0, q_m + 1, tz_m, false);
    adj_tz_row(a, s, j0, i0, q_c + 1, tz_c, true);
    adj_sz_row(a, s, j0 - 1, i0, tz_m, tz_c, sz_p, false);       // halo row, recomputed
  }
  const int j1 = j0 + kRZ < g.nz ? j0 + kRZ : g.nz;
  for (int j = j0; j < j1; ++j) {
    adj_load_q6(a, s, j + 1, i0, mu_n, q_n);
    adj_tz_row(a, s, j + 1, i0, q_n + 1, tz_n, j + 1 < j1);
    adj_sz_row(a, s, j, i0, tz_c, tz_n, sz_c, true);
    const long long ro = (long long)j * g.pitch + i0;
    const long long o = s * g.plane + ro;
    // tx for columns i0-1..i0+4 (transpose of the E-side x CPML)
    float tx[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const int i = i0 - 1 + k;
      tx[k] = q_c[k];
      if (j < 1 || j > g.nz - 2 || i < 1 || i > g.nx - 2) { tx[k] = 0.f; continue; }
      const int xs = xpml_e ? strip_e(i, g.nx, g.P) : -1;
      if (xs >= 0) {
        const long long po = s * g.xstrip + (long long)j * g.xw + xs;
        const float T = a.in.pezx[po] + q_c[k];
        tx[k] = q_c[k] * g.kex[i] + g.cex[i] * T;
        if (k >= 1 && k <= 4) a.out.pezx[po] = g.bex[i] * T;
      }
    }
    // lamHy' and sx for columns i0-1..i0+3
    float hy[5], sx[5];
    unpack(ld4(a.in.hy + o), hy + 1);
    hy[0] = i0 > 0 ? a.in.hy[o - 1] : 0.f;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const int i = i0 - 1 + k;
      if (i < 0 || i > g.nx - 2) { hy[k] = 0.f; sx[k] = 0.f; continue; }
      hy[k] += (tx[k] - tx[k + 1]) * g.rdx;
      const float py = g.Db * hy[k];
      sx[k] = py;
      const int xs = xpml_h ? strip_h(i, g.nx, g.P) : -1;
      if (xs >= 0) {
        const long long po = s * g.xstrip + (long long)j * g.xw + xs;
        const float T = a.in.phyx[po] + py;
        sx[k] = py * g.khx[i] + g.chx[i] * T;
        if (k >= 1) a.out.phyx[po] = g.bhx[i] * T;
      }
    }
    st4(a.out.hy + o, mk4(hy[1], hy[2], hy[3], hy[4]));
    // lamE' and the gradient terms of step n
    float le[4] = {0.f, 0.f, 0.f, 0.f};
    if (j >= 1 && j <= g.nz - 2) {
      float ca[4], cb[4], e0[4], e1[4], ga[4], gb[4];
      unpack(ld4(a.ca + ro), ca);
      unpack(ld4(a.cb + ro), cb);
      unpack(ld4(a.en + o), e0);
      unpack(ld4(a.en1 + o), e1);
      float* gca = a.gca + grp * g.plane + ro;
      float* gcb = a.gcb + grp * g.plane + ro;
      unpack(ld4(gca), ga);
      unpack(ld4(gcb), gb);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int i = i0 + k;
        if (i < 1 || i > g.nx - 2) continue;
        const float m = mu_c[k + 1];
        ga[k] += m * e0[k];
        if (cb[k] != 0.f) gb[k] += m * ((e1[k] - ca[k] * e0[k]) / cb[k]);
        le[k] = ca[k] * m + (sz_p[k] - sz_c[k]) * g.rdx + (sx[k] - sx[k + 1]) * g.rdx;
      }
      st4(gca, mk4(ga[0], ga[1], ga[2], ga[3]));
      st4(gcb, mk4(gb[0], gb[1], gb[2], gb[3]));
    }
    st4(a.out.ez + o, mk4(le[0], le[1], le[2], le[3]));
#pragma unroll
    for (int k = 0; k < 6; ++k) { mu_c[k] = mu_n[k]; q_c[k] = q_n[k]; }
#pragma unroll
    for (int k = 0; k < 4; ++k) { tz_c[k] = tz_n[k]; sz_p[k] = sz_c[k]; }
  }
}

// transpose of recording: lamE'[rec] += residual[n][r] for the receivers inside this block's tile
// (after all threads of the block have stored their lamE'; coincident receivers sum)
GPR_HD void adj_inject(const AdjArgs& a, int s, int tile, int t, int nthreads)
{
  const int ntile = a.tiles_x * a.tiles_y;
  const int* st = a.blk_start + (long long)s * (ntile + 1);
  for (int k = st[tile] + t; k < st[tile + 1]; k += nthreads) {
    const int r = a.blk_rec[(long long)s * a.R + k];
    float* dst = a.out.ez + s * a.g.plane + a.rec_off[(long long)s * a.R + r];
    const float v = a.residual[s * a.trace_stride + r];
#if defined(__CUDA_ARCH__)
    atomicAdd(dst, v);
#else
    *dst += v;
#endif
  }
}

#if defined(__CUDACC__)
__global__ void __launch_bounds__(32 * kWarpsY) adj_step_kernel(const AdjArgs a)
{
  const int i0 = (blockIdx.x * 32 + threadIdx.x) * 4;
  const int j0 = (blockIdx.y * kWarpsY + threadIdx.y) * kRZ;
  const int grp = blockIdx.z;
  const bool active = i0 < a.g.nx && j0 < a.g.nz;
  const int s_end = min((grp + 1) * a.group, a.nshots);
  for (int s = grp * a.group; s < s_end; ++s) {
    if (active) adj_thread_shot(a, s, grp, i0, j0);
    __syncthreads();
    adj_inject(a, s, blockIdx.y * a.tiles_x + blockIdx.x, threadIdx.y * 32 + threadIdx.x, 32 * kWarpsY);
  }
}
#endif

}  // namespace gprfwi
