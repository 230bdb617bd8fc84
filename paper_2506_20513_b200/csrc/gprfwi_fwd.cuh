// gprfwi_fwd.cuh -- forward time step: H update + H CPML, E update + E CPML, source injection,
// receiver gather, history store, all in ONE pass over the data (kernels b, c, d of north_star).
//
// One launch advances state n -> n+1 for all shots of the batch (Algorithm 1 stages 1-7,
// PAPER.md:466-474; Eqs. (3)-(5)).  The state is ping-ponged: every thread reads
// state n from `in` and writes state n+1 to `out`, so threads are independent (a pure gather) and
// the H values a thread needs on its left / upper edge are recomputed, not exchanged.
// `out.ez` is the history plane n+1 when the history is stored, so "save wavefield" costs nothing.
//
// Thread = one float4 of x (4 cells) streamed down kRZ rows; Ez rows j-1, j, j+1 and the previous
// row's new Hx live in registers.
#pragma once
#include "gprfwi_common.cuh"

namespace gprfwi {

struct FwdArgs {
  Geo g;
  State in, out;
  const float *ca, *cb;       // [nz][pitch]
  const float* wavelet;       // sample n of local shot 0; shot s at + s * wav_stride
  long long wav_stride;       // nt or 0
  const int* src_off;         // [S] j*pitch + i of the source
  const int* rec_off;         // [S][R] j*pitch + i of each receiver
  float* traces;              // sample n of local shot 0, receiver 0; shot s at + s*nt*R; may be NULL
  long long trace_stride;     // nt * R
  int R;
  int nshots;
  int tiles_y;                // blockIdx.y >= tiles_y: receiver-gather blocks
};

// new Hx (row j, columns i0..i0+3) from Ez rows j (lo) and j+1 (hi).  Eq. (4).
GPR_HD void fwd_hx_row(const FwdArgs& a, int s, int j, int i0, const float* e_lo, const float* e_hi,
                       float* hxn, bool store)
{
  const Geo& g = a.g;
  if (j < 0 || j > g.nz - 2) {
    hxn[0] = hxn[1] = hxn[2] = hxn[3] = 0.f;
    if (store && j >= 0 && j < g.nz) st4(a.out.hx + s * g.plane + (long long)j * g.pitch + i0, mk4(0, 0, 0, 0));
    return;
  }
  const long long o = s * g.plane + (long long)j * g.pitch + i0;
  float h[4];
  unpack(ld4(a.in.hx + o), h);
  const int zs = strip_h(j, g.nz, g.P);
  if (zs >= 0) {
    const long long po = s * g.zstrip + (long long)zs * g.pitch + i0;
    float p[4];
    unpack(ld4(a.in.phxz + po), p);
    const float b = g.bhz[j], c = g.chz[j], ik = g.khz[j];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float d = (e_hi[k] - e_lo[k]) * g.rdx;
      p[k] = b * p[k] + c * d;
      hxn[k] = h[k] - g.Db * (d * ik + p[k]);
    }
    if (store) st4(a.out.phxz + po, mk4(p[0], p[1], p[2], p[3]));
  } else {
#pragma unroll
    for (int k = 0; k < 4; ++k) hxn[k] = h[k] - g.Db * ((e_hi[k] - e_lo[k]) * g.rdx);
  }
  if (store) st4(a.out.hx + o, mk4(hxn[0], hxn[1], hxn[2], hxn[3]));
}

// new Hy (row j, columns i0-1..i0+3 -> hyn[0..4]) from e[0..5] = Ez[j][i0-1..i0+4].
// Column i0-1 is the left neighbour's cell, recomputed here and not stored.  Eq. (5).
GPR_HD void fwd_hy_row(const FwdArgs& a, int s, int j, int i0, const float* e, float* hyn)
{
  const Geo& g = a.g;
  const long long o = s * g.plane + (long long)j * g.pitch + i0;
  float h[5];
  unpack(ld4(a.in.hy + o), h + 1);
  h[0] = i0 > 0 ? a.in.hy[o - 1] : 0.f;
  const bool xpml = (i0 - 1 < g.P) || (i0 + 3 >= g.nx - 1 - g.P);
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const int i = i0 - 1 + k;
    if (i < 0 || i > g.nx - 2) { hyn[k] = 0.f; continue; }
    const float d = (e[k + 1] - e[k]) * g.rdx;
    const int xs = xpml ? strip_h(i, g.nx, g.P) : -1;
    if (xs >= 0) {
      const long long po = s * g.xstrip + (long long)j * g.xw + xs;
      const float p = g.bhx[i] * a.in.phyx[po] + g.chx[i] * d;
      hyn[k] = h[k] + g.Db * (d * g.khx[i] + p);
      if (k > 0) a.out.phyx[po] = p;
    } else {
      hyn[k] = h[k] + g.Db * d;
    }
  }
  st4(a.out.hy + o, mk4(hyn[1], hyn[2], hyn[3], hyn[4]));
}

// Ez rows j (-> e[0..5] = columns i0-1..i0+4); zero outside the grid
GPR_HD void fwd_load_e6(const FwdArgs& a, int s, int j, int i0, float* e)
{
  const Geo& g = a.g;
  if (j < 0 || j >= g.nz) { e[0] = e[1] = e[2] = e[3] = e[4] = e[5] = 0.f; return; }
  const float* row = a.in.ez + s * g.plane + (long long)j * g.pitch;
  unpack(ld4(row + i0), e + 1);
  e[0] = i0 > 0 ? row[i0 - 1] : 0.f;
  e[5] = i0 + 4 < g.nx ? row[i0 + 4] : 0.f;
}

GPR_HD void fwd_thread(const FwdArgs& a, int s, int c4, int chunk)
{
  const Geo& g = a.g;
  const int i0 = c4 * 4, j0 = chunk * kRZ;
  if (i0 >= g.nx || j0 >= g.nz) return;
  const int src = a.src_off[s];
  const float wn = a.wavelet[s * a.wav_stride];
  const bool xpml = (i0 < g.P) || (i0 + 3 >= g.nx - g.P);

  float e_c[6], e_n[6], hx_p[4], hx_c[4], hy_c[5];
  float e_m[6];
  fwd_load_e6(a, s, j0 - 1, i0, e_m);
  fwd_load_e6(a, s, j0, i0, e_c);
  fwd_hx_row(a, s, j0 - 1, i0, e_m + 1, e_c + 1, hx_p, false);     // halo row, recomputed

  const int j1 = j0 + kRZ < g.nz ? j0 + kRZ : g.nz;
  for (int j = j0; j < j1; ++j) {
    fwd_load_e6(a, s, j + 1, i0, e_n);
    fwd_hx_row(a, s, j, i0, e_c + 1, e_n + 1, hx_c, true);
    fwd_hy_row(a, s, j, i0, e_c, hy_c);
    // E update + E CPML.  Eq. (3) in the Ca/Cb form of PAPER.md:415-424; PEC ring stays 0.
    const long long ro = (long long)j * g.pitch + i0;
    float en[4] = {0.f, 0.f, 0.f, 0.f};
    if (j >= 1 && j <= g.nz - 2) {
      float ca[4], cb[4];
      unpack(ld4(a.ca + ro), ca);
      unpack(ld4(a.cb + ro), cb);
      const int zs = strip_e(j, g.nz, g.P);
      float pz[4] = {0.f, 0.f, 0.f, 0.f};
      float bz = 0.f, cz = 0.f, kz = 1.f;
      const long long pzo = s * g.zstrip + (long long)(zs < 0 ? 0 : zs) * g.pitch + i0;
      if (zs >= 0) { unpack(ld4(a.in.pezz + pzo), pz); bz = g.bez[j]; cz = g.cez[j]; kz = g.kez[j]; }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int i = i0 + k;
        if (i < 1 || i > g.nx - 2) { pz[k] = 0.f; continue; }
        const float dxh = (hy_c[k + 1] - hy_c[k]) * g.rdx;
        const float dzh = (hx_c[k] - hx_p[k]) * g.rdx;
        float vx = dxh, vz = dzh;
        const int xs = xpml ? strip_e(i, g.nx, g.P) : -1;
        if (xs >= 0) {
          const long long po = s * g.xstrip + (long long)j * g.xw + xs;
          const float p = g.bex[i] * a.in.pezx[po] + g.cex[i] * dxh;
          a.out.pezx[po] = p;
          vx = dxh * g.kex[i] + p;
        }
        if (zs >= 0) {
          pz[k] = bz * pz[k] + cz * dzh;
          vz = dzh * kz + pz[k];
        }
        en[k] = ca[k] * e_c[k + 1] + cb[k] * (vx - vz);
        // stage 6: source:  Ez -= uE4 * w * dl/(dx dy dz), dl = dz
        if ((int)ro + k == src) en[k] -= cb[k] * wn * (g.rdx * g.rdx);
      }
      if (zs >= 0) st4(a.out.pezz + pzo, mk4(pz[0], pz[1], pz[2], pz[3]));
    }
    st4(a.out.ez + s * g.plane + ro, mk4(en[0], en[1], en[2], en[3]));
#pragma unroll
    for (int k = 0; k < 6; ++k) e_c[k] = e_n[k];
#pragma unroll
    for (int k = 0; k < 4; ++k) hx_p[k] = hx_c[k];
  }
}

// stage 1 of Algorithm 1: traces[s][n][r] = Ez^n at receiver r, read from the (immutable) input plane
GPR_HD void fwd_gather(const FwdArgs& a, int s, int t, int nthreads)
{
  if (!a.traces) return;
  for (int r = t; r < a.R; r += nthreads)
    a.traces[s * a.trace_stride + r] = a.in.ez[s * a.g.plane + a.rec_off[(long long)s * a.R + r]];
}

#if defined(__CUDACC__)
__global__ void __launch_bounds__(32 * kWarpsY) fwd_step_kernel(const FwdArgs a)
{
  const int s = blockIdx.z;
  if ((int)blockIdx.y >= a.tiles_y) {
    fwd_gather(a, s, blockIdx.x * (32 * kWarpsY) + threadIdx.y * 32 + threadIdx.x, gridDim.x * 32 * kWarpsY);
    return;
  }
  fwd_thread(a, s, blockIdx.x * 32 + threadIdx.x, blockIdx.y * kWarpsY + threadIdx.y);
}
#endif

}  // namespace gprfwi
