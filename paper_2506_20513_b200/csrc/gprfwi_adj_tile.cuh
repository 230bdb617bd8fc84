// gprfwi_adj_tile.cuh -- temporally blocked adjoint kernel (kernel e of north_star): ONE launch takes
// a group of shots back by up to T time steps (Algorithm 2 stages 1-6) and
// accumulates dJ/dCa, dJ/dCb in registers over those steps and over the shots of the group.
//
// Same tiling as gprfwi_fwd_tile.cuh (TZ x TX tile + halo staged in shared memory, halo recomputed).
// Reverse step n, with mu = lamE (0 on the PEC ring), q = Cb*mu:
//   [inject]  lamE[rec] += residual[n+1]                  (transpose of recording; region-wide)
//   [phase B] tx = q/kex + cex*(psiEx + q), tz = -q/kez + cez*(psiEz - q)   (plain q, -q off the CPML)
//             lamHy += (tx[i] - tx[i+1])/dx,  lamHx += (tz[j] - tz[j+1])/dx
//   [phase C] gCa += mu*E^n,  gCb += mu*(E^{n+1} - Ca*E^n)/Cb          (owned cells, registers)
//             psiEx <- bex*(psiEx + q),  psiEz <- bez*(psiEz - q)       (own cell)
//             sx = p/khx + chx*(psiHx + p), p = Db*lamHy;  sz likewise with p = -Db*lamHx
//             lamE <- Ca*mu + (sz[j-1] - sz[j])/dx + (sx[i-1] - sx[i])/dx
// tx, tz, sx, sz are never stored: neighbours recompute them from lamE / lamH and the OLD psi, and
// the psi recursions are applied by the owning thread one phase later ("lazy"), psiH at the start
// of the next phase B (or in the final store), so no reader ever sees a half-updated psi.
#pragma once
#include "gprfwi_common.cuh"
#include "gprfwi_fwd_tile.cuh"

namespace gprfwi {

struct AdjTileArgs {
  Geo g;
  State in, out;                      // adjoint variables, ping-pong (pointers of local shot 0)
  const float *ca, *cb;
  const float* ez_planes[kMaxT + 1];  // [t] = forward Ez^{n_hi - t} (local shot 0), t = 0..nsub
  float *gca, *gcb;                   // [ngroups][nz][pitch]
  const float* residual;              // sample n_hi of local shot 0 (sample n_hi - t at - t*R)
  long long trace_stride;             // nt * R
  const int* rec_off;                 // [S][R]
  const int* reg_start;               // [S*tiles + 1] CSR of receivers by REGION (tile + halo)
  const int* reg_rec;
  int R, nsub, n_hi, nt;
  int nshots, group;
  int tiles_x, tiles_y;
  int zcap, xcap;
  int shot_base;                      // global index of local shot 0 (for the CSR)
};

template <int TZ, int TX, int T>
struct AdjTile {
  using F = FwdTile<TZ, TX, T>;
  static constexpr int RH = F::RH, RW = F::RW, RW4 = F::RW4, NU = F::NU, KU = F::KU;
  struct Regs { float ca[KU][4], ga[KU][4], gb[KU][4], e1[KU][4]; };
  struct Smem { float *le, *hx, *hy, *cb, *pzh, *pze, *pxh, *pxe, *tz, *tx; };
  GPR_HD static size_t smem_floats(int zcap, int xcap)
  {
    return (size_t)4 * RH * RW + (size_t)2 * zcap * RW + (size_t)2 * RH * xcap + 6 * RH + 6 * RW;
  }
  struct Ctx {
    Smem m;
    int s, gj0, gi0, zmin_e, zmin_h, xmin_e, xmin_h;
  };
  GPR_HD static Ctx make_ctx(const AdjTileArgs& a, float* base, int ty, int tx)
  {
    Ctx c;
    Smem& m = c.m;
    m.le = base; m.hx = m.le + RH * RW; m.hy = m.hx + RH * RW; m.cb = m.hy + RH * RW;
    m.pzh = m.cb + RH * RW; m.pze = m.pzh + a.zcap * RW;
    m.pxh = m.pze + a.zcap * RW; m.pxe = m.pxh + RH * a.xcap;
    m.tz = m.pxe + RH * a.xcap; m.tx = m.tz + 6 * RH;
    c.s = 0; c.gj0 = ty * TZ - T; c.gi0 = tx * TX - 4;
    c.zmin_e = F::strip_min(c.gj0, a.g.nz, a.g.P, false);
    c.zmin_h = F::strip_min(c.gj0, a.g.nz, a.g.P, true);
    c.xmin_e = F::strip_min(c.gi0, a.g.nx, a.g.P, false);
    c.xmin_h = F::strip_min(c.gi0, a.g.nx, a.g.P, true);
    return c;
  }
  GPR_HD static bool owned(int r, int lc) { return r >= T && r < T + TZ && lc >= 4 && lc < 4 + TX; }

  // once per CTA: tables, Cb region, Ca registers, zeroed accumulators
  GPR_HD static void setup(const AdjTileArgs& a, const Ctx& c, int tid, Regs& rg)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
    for (int r = tid; r < RH; r += kTileThreads) {
      const int gj = c.gj0 + r;
      const bool in = gj >= 0 && gj < g.nz;
      m.tz[0 * RH + r] = in ? g.bhz[gj] : 0.f; m.tz[1 * RH + r] = in ? g.chz[gj] : 0.f;
      m.tz[2 * RH + r] = in ? g.khz[gj] : 1.f; m.tz[3 * RH + r] = in ? g.bez[gj] : 0.f;
      m.tz[4 * RH + r] = in ? g.cez[gj] : 0.f; m.tz[5 * RH + r] = in ? g.kez[gj] : 1.f;
    }
    for (int q = tid; q < RW; q += kTileThreads) {
      const int gi = c.gi0 + q;
      const bool in = gi >= 0 && gi < g.nx;
      m.tx[0 * RW + q] = in ? g.bhx[gi] : 0.f; m.tx[1 * RW + q] = in ? g.chx[gi] : 0.f;
      m.tx[2 * RW + q] = in ? g.khx[gi] : 1.f; m.tx[3 * RW + q] = in ? g.bex[gi] : 0.f;
      m.tx[4 * RW + q] = in ? g.cex[gi] : 0.f; m.tx[5 * RW + q] = in ? g.kex[gi] : 1.f;
    }
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      const int u = tid + k * kTileThreads;
#pragma unroll
      for (int q = 0; q < 4; ++q) rg.ca[k][q] = rg.ga[k][q] = rg.gb[k][q] = rg.e1[k][q] = 0.f;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      float4 cb = mk4(0, 0, 0, 0);
      if (gj >= 1 && gj <= g.nz - 2 && gi >= 0 && gi < g.nx) {      // Cb = 0 on ring rows: q = 0 there
        cb = ld4(a.cb + (long long)gj * g.pitch + gi);
        unpack(ld4(a.ca + (long long)gj * g.pitch + gi), rg.ca[k]);
        if (gi == 0) cb.x = 0.f;                                    // ring columns
        if (gi + 0 == g.nx - 1) cb.x = 0.f;
        if (gi + 1 >= g.nx - 1) cb.y = 0.f;
        if (gi + 2 >= g.nx - 1) cb.z = 0.f;
        if (gi + 3 >= g.nx - 1) cb.w = 0.f;
      }
      st4(m.cb + r * RW + lc, cb);
    }
  }

  // per shot: stage the adjoint state of the region; first history plane into registers
  GPR_HD static void load(const AdjTileArgs& a, const Ctx& c, int tid, Regs& rg)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      const int u = tid + k * kTileThreads;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      const bool in = gj >= 0 && gj < g.nz && gi >= 0 && gi < g.nx;
      float4 e = mk4(0, 0, 0, 0), hx = e, hy = e;
      if (in) {
        const long long o = c.s * g.plane + (long long)gj * g.pitch + gi;
        e = ld4(a.in.ez + o); hx = ld4(a.in.hx + o); hy = ld4(a.in.hy + o);
        const int zh = strip_h(gj, g.nz, g.P), ze = strip_e(gj, g.nz, g.P);
        if (zh >= 0) st4(m.pzh + (zh - c.zmin_h) * RW + lc, ld4(a.in.phxz + c.s * g.zstrip + (long long)zh * g.pitch + gi));
        if (ze >= 0) st4(m.pze + (ze - c.zmin_e) * RW + lc, ld4(a.in.pezz + c.s * g.zstrip + (long long)ze * g.pitch + gi));
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int xh = strip_h(gi + q, g.nx, g.P), xe = strip_e(gi + q, g.nx, g.P);
          const long long po = c.s * g.xstrip + (long long)gj * g.xw;
          if (xh >= 0) m.pxh[r * a.xcap + xh - c.xmin_h] = a.in.phyx[po + xh];
          if (xe >= 0) m.pxe[r * a.xcap + xe - c.xmin_e] = a.in.pezx[po + xe];
        }
        if (owned(r, lc)) unpack(ld4(a.ez_planes[0] + o), rg.e1[k]);
      }
      st4(m.le + r * RW + lc, e); st4(m.hx + r * RW + lc, hx); st4(m.hy + r * RW + lc, hy);
    }
  }

  // transpose of recording: residual sample n+1 enters lamE at every receiver of the REGION
  GPR_HD static void inject(const AdjTileArgs& a, const Ctx& c, int tile, int tid, int t)
  {
    const int n1 = a.n_hi - t;                     // = n + 1 for reverse step n = n_hi - 1 - t
    if (n1 >= a.nt) return;
    const long long row = (long long)(a.shot_base + c.s) * (a.tiles_x * a.tiles_y) + tile;
    for (int k = a.reg_start[row] + tid; k < a.reg_start[row + 1]; k += kTileThreads) {
      const int r = a.reg_rec[k];
      const int off = a.rec_off[(long long)c.s * a.R + r];
      const int lj = off / a.g.pitch - c.gj0, li = off % a.g.pitch - c.gi0;
      const float v = a.residual[c.s * a.trace_stride - (long long)t * a.R + r];
#if defined(__CUDA_ARCH__)
      atomicAdd(c.m.le + lj * RW + li, v);         // coincident receivers sum
#else
      c.m.le[lj * RW + li] += v;
#endif
    }
  }

  GPR_HD static float tz_of(const Ctx& c, const Geo& g, int r, int gj, int col, float q)
  {
    const int ze = strip_e(gj, g.nz, g.P);
    if (ze < 0) return -q;
    const float T_ = c.m.pze[(ze - c.zmin_e) * RW + col] - q;
    return -q * c.m.tz[5 * RH + r] + c.m.tz[4 * RH + r] * T_;
  }
  GPR_HD static float tx_of(const AdjTileArgs& a, const Ctx& c, int r, int gi, int col, float q)
  {
    const int xe = strip_e(gi, a.g.nx, a.g.P);
    if (xe < 0) return q;
    const float T_ = c.m.pxe[r * a.xcap + xe - c.xmin_e] + q;
    return q * c.m.tx[5 * RW + col] + c.m.tx[4 * RW + col] * T_;
  }
  GPR_HD static float sz_of(const Ctx& c, const Geo& g, int r, int gj, int col)
  {
    const float px = -g.Db * c.m.hx[r * RW + col];
    const int zh = strip_h(gj, g.nz, g.P);
    if (zh < 0) return px;
    return px * c.m.tz[2 * RH + r] + c.m.tz[1 * RH + r] * (c.m.pzh[(zh - c.zmin_h) * RW + col] + px);
  }
  GPR_HD static float sx_of(const AdjTileArgs& a, const Ctx& c, int r, int gi, int col)
  {
    const float py = a.g.Db * c.m.hy[r * RW + col];
    const int xh = strip_h(gi, a.g.nx, a.g.P);
    if (xh < 0) return py;
    return py * c.m.tx[2 * RW + col] + c.m.tx[1 * RW + col] * (c.m.pxh[r * a.xcap + xh - c.xmin_h] + py);
  }
  // the deferred psiH recursion of the previous step for this thread's own cells
  GPR_HD static void lazy_psih(const AdjTileArgs& a, const Ctx& c, int r, int lc, int gj, int gi)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
    const int zh = gj <= g.nz - 2 ? strip_h(gj, g.nz, g.P) : -1;
    if (zh >= 0) {
      float* pp = m.pzh + (zh - c.zmin_h) * RW + lc;
      const float b = m.tz[0 * RH + r];
#pragma unroll
      for (int q = 0; q < 4; ++q) pp[q] = b * (pp[q] - g.Db * m.hx[r * RW + lc + q]);
    }
    if (gi < g.P || gi + 3 >= g.nx - 1 - g.P) {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int xh = strip_h(gi + q, g.nx, g.P);
        if (xh < 0) continue;
        float* pp = m.pxh + r * a.xcap + xh - c.xmin_h;
        *pp = m.tx[0 * RW + lc + q] * (*pp + g.Db * m.hy[r * RW + lc + q]);
      }
    }
  }

  // transpose of the E update + E CPML, applied to lamH
  GPR_HD static void phase_b(const AdjTileArgs& a, const Ctx& c, int tid, int t)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      const int u = tid + k * kTileThreads;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      if (gj < 0 || gj >= g.nz || gi < 0 || gi >= g.nx) continue;
      if (t > 0) lazy_psih(a, c, r, lc, gj, gi);
      float q[5];
      {
        float le[5], cb[5];
        unpack(ld4(m.le + r * RW + lc), le);
        unpack(ld4(m.cb + r * RW + lc), cb);
        le[4] = lc + 4 < RW ? m.le[r * RW + lc + 4] : 0.f;
        cb[4] = lc + 4 < RW ? m.cb[r * RW + lc + 4] : 0.f;
#pragma unroll
        for (int x = 0; x < 5; ++x) q[x] = cb[x] * le[x];
      }
      if (r + 1 < RH && gj <= g.nz - 2) {
        float ln[4], cn[4], h[4];
        unpack(ld4(m.le + (r + 1) * RW + lc), ln);
        unpack(ld4(m.cb + (r + 1) * RW + lc), cn);
        unpack(ld4(m.hx + r * RW + lc), h);
#pragma unroll
        for (int x = 0; x < 4; ++x)
          h[x] += (tz_of(c, g, r, gj, lc + x, q[x]) - tz_of(c, g, r + 1, gj + 1, lc + x, cn[x] * ln[x])) * g.rdx;
        st4(m.hx + r * RW + lc, mk4(h[0], h[1], h[2], h[3]));
      }
      {
        float h[4];
        unpack(ld4(m.hy + r * RW + lc), h);
        const bool xpml = (gi < g.P) || (gi + 4 >= g.nx - g.P);
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          if (lc + x + 1 >= RW || gi + x > g.nx - 2) continue;
          const float t0 = xpml ? tx_of(a, c, r, gi + x, lc + x, q[x]) : q[x];
          const float t1 = xpml ? tx_of(a, c, r, gi + x + 1, lc + x + 1, q[x + 1]) : q[x + 1];
          h[x] += (t0 - t1) * g.rdx;
        }
        st4(m.hy + r * RW + lc, mk4(h[0], h[1], h[2], h[3]));
      }
    }
  }

  // gradient terms, psiE recursion, transpose of the H update + H CPML applied to lamE
  GPR_HD static void phase_c(const AdjTileArgs& a, const Ctx& c, int tid, Regs& rg, int t)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      const int u = tid + k * kTileThreads;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      if (gj < 0 || gj >= g.nz || gi < 0 || gi >= g.nx) continue;
      float mu[4], cb[4];
      unpack(ld4(m.le + r * RW + lc), mu);
      unpack(ld4(m.cb + r * RW + lc), cb);
      const bool own = owned(r, lc);
      if (own) {                                   // E^n of this step; E^{n+1} is carried in registers
        float e0[4];
        unpack(ld4(a.ez_planes[t + 1] + c.s * g.plane + (long long)gj * g.pitch + gi), e0);
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          if (cb[x] != 0.f) {
            rg.ga[k][x] += mu[x] * e0[x];
            rg.gb[k][x] += mu[x] * ((rg.e1[k][x] - rg.ca[k][x] * e0[x]) / cb[x]);
          }
          rg.e1[k][x] = e0[x];
        }
      }
      if (!(r >= 1 && r <= RH - 2 && gj >= 1 && gj <= g.nz - 2)) continue;
      const int ze = strip_e(gj, g.nz, g.P);
      if (ze >= 0) {
        float* pp = m.pze + (ze - c.zmin_e) * RW + lc;
        const float b = m.tz[3 * RH + r];
#pragma unroll
        for (int x = 0; x < 4; ++x) pp[x] = b * (pp[x] - cb[x] * mu[x]);
      }
      const bool xpml_e = (gi < g.P) || (gi + 3 >= g.nx - g.P);
      const bool xpml_h = (gi - 1 < g.P) || (gi + 3 >= g.nx - 1 - g.P);
      float le[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        const int lcol = lc + x, i = gi + x;
        le[x] = mu[x];
        if (lcol < 1 || lcol > RW - 2) continue;                 // region edge: stale, left as is
        if (i < 1 || i > g.nx - 2) { le[x] = 0.f; continue; }    // PEC ring column
        if (xpml_e) {
          const int xe = strip_e(i, g.nx, g.P);
          if (xe >= 0) {
            float* pp = m.pxe + r * a.xcap + xe - c.xmin_e;
            *pp = m.tx[3 * RW + lcol] * (*pp + cb[x] * mu[x]);
          }
        }
        const float szm = sz_of(c, g, r - 1, gj - 1, lcol), szc = gj <= g.nz - 2 ? sz_of(c, g, r, gj, lcol) : 0.f;
        float sxm, sxc;
        if (xpml_h) {
          sxm = sx_of(a, c, r, i - 1, lcol - 1);
          sxc = i <= g.nx - 2 ? sx_of(a, c, r, i, lcol) : 0.f;
        } else {
          sxm = g.Db * m.hy[r * RW + lcol - 1];
          sxc = g.Db * m.hy[r * RW + lcol];
        }
        le[x] = rg.ca[k][x] * mu[x] + (szm - szc) * g.rdx + (sxm - sxc) * g.rdx;
      }
      st4(m.le + r * RW + lc, mk4(le[0], le[1], le[2], le[3]));
    }
  }

  // per shot: write back the owned part of the adjoint state (psiH with its pending recursion)
  GPR_HD static void store(const AdjTileArgs& a, const Ctx& c, int tid)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      const int u = tid + k * kTileThreads;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      if (!owned(r, lc) || gj >= g.nz || gi >= g.nx) continue;
      if (a.nsub > 0) lazy_psih(a, c, r, lc, gj, gi);
      const long long o = c.s * g.plane + (long long)gj * g.pitch + gi;
      st4(a.out.ez + o, ld4(m.le + r * RW + lc));
      st4(a.out.hx + o, ld4(m.hx + r * RW + lc));
      st4(a.out.hy + o, ld4(m.hy + r * RW + lc));
      const int zh = strip_h(gj, g.nz, g.P), ze = strip_e(gj, g.nz, g.P);
      if (zh >= 0) st4(a.out.phxz + c.s * g.zstrip + (long long)zh * g.pitch + gi, ld4(m.pzh + (zh - c.zmin_h) * RW + lc));
      if (ze >= 0) st4(a.out.pezz + c.s * g.zstrip + (long long)ze * g.pitch + gi, ld4(m.pze + (ze - c.zmin_e) * RW + lc));
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int xh = strip_h(gi + q, g.nx, g.P), xe = strip_e(gi + q, g.nx, g.P);
        const long long po = c.s * g.xstrip + (long long)gj * g.xw;
        if (xh >= 0) a.out.phyx[po + xh] = m.pxh[r * a.xcap + xh - c.xmin_h];
        if (xe >= 0) a.out.pezx[po + xe] = m.pxe[r * a.xcap + xe - c.xmin_e];
      }
    }
  }

  // once per CTA: add the register accumulators to this group's gCa / gCb planes
  GPR_HD static void flush(const AdjTileArgs& a, const Ctx& c, int tid, int grp, const Regs& rg)
  {
    const Geo& g = a.g;
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      const int u = tid + k * kTileThreads;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      if (!owned(r, lc) || gj >= g.nz || gi >= g.nx) continue;
      float* pa = a.gca + grp * g.plane + (long long)gj * g.pitch + gi;
      float* pb = a.gcb + grp * g.plane + (long long)gj * g.pitch + gi;
      float4 va = ld4(pa), vb = ld4(pb);
      va.x += rg.ga[k][0]; va.y += rg.ga[k][1]; va.z += rg.ga[k][2]; va.w += rg.ga[k][3];
      vb.x += rg.gb[k][0]; vb.y += rg.gb[k][1]; vb.z += rg.gb[k][2]; vb.w += rg.gb[k][3];
      st4(pa, va); st4(pb, vb);
    }
  }
};

#if defined(__CUDACC__)
template <int TZ, int TX, int T>
__global__ void __launch_bounds__(kTileThreads) adj_tile_kernel(const AdjTileArgs a)
{
  using K = AdjTile<TZ, TX, T>;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, grp = blockIdx.z;
  typename K::Ctx c = K::make_ctx(a, reinterpret_cast<float*>(smem4), blockIdx.y, blockIdx.x);
  const int tile = blockIdx.y * a.tiles_x + blockIdx.x;
  typename K::Regs rg;
  K::setup(a, c, tid, rg);
  const int s_end = min((grp + 1) * a.group, a.nshots);
  for (int s = grp * a.group; s < s_end; ++s) {
    c.s = s;
    __syncthreads();                 // previous shot's store has finished with shared memory
    K::load(a, c, tid, rg);
    __syncthreads();
    for (int t = 0; t < a.nsub; ++t) {
      K::inject(a, c, tile, tid, t);
      __syncthreads();
      K::phase_b(a, c, tid, t);
      __syncthreads();
      K::phase_c(a, c, tid, rg, t);
      __syncthreads();
    }
    K::store(a, c, tid);
  }
  K::flush(a, c, tid, grp, rg);
}
#endif

}  // namespace gprfwi
