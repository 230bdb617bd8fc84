// gprfwi_fwd_tile.cuh -- temporally blocked forward kernel (kernels b, c, d of north_star fused):
// ONE launch advances all shots by up to T time steps (Algorithm 1 stages 1-7).
//
// A CTA owns a TZ x TX tile of one shot.  It stages the tile plus a halo of T rows / 4 columns of
// Ez, Hx, Hy and the CPML psi strips that cross it in shared memory, runs the T leap-frog steps
// there (H phase, barrier, E phase, barrier), and writes back only what it owns: each step's Ez
// plane (the stored history / recompute segment, if wanted), the traces of its receivers, and the
// final Hx, Hy, psi.  The halo is recomputed redundantly instead of exchanged; after t steps the
// outermost t halo rings are stale, which is why the halo is T deep.  State is ping-ponged
// between launches so CTAs never race.  Per cell-step HBM traffic drops from 24 B (one step per
// pass) to about 24*1.4/T B plus the 4 B history store.
//
// Thread = float4 "units" (4 cells of a row) of the staged region, the same units every step, so
// Ca/Cb of a thread's cells stay in registers for the whole launch.
#pragma once
#include "gprfwi_common.cuh"

namespace gprfwi {

constexpr int kTileThreads = 256;
constexpr int kMaxT = 8;

struct FwdTileArgs {
  Geo g;
  State in, out;              // out.ez: Ez plane after the last step of this launch
  const float *ca, *cb;
  float* ez_hist[kMaxT];      // [t]: plane for Ez after step t (1 <= t < nsub) or NULL; [0] unused
  const float* wavelet;       // sample n of local shot 0
  long long wav_stride;
  const int* src_off;         // [S] j*pitch + i
  const int* rec_off;         // [S][R]
  const int* blk_start;       // [S][tiles + 1] CSR of receivers by owning tile (this tiling)
  const int* blk_rec;         // [S][R]
  float* traces;              // sample n of local shot 0 (NULL: do not record)
  long long trace_stride;     // nt * R
  int R, nsub;                // receivers per shot; steps in this launch (<= T)
  int tiles_x, tiles_y;
  int zcap, xcap;             // rows / columns of psi strips staged per CTA
};

// Update expressions off the CPML, written once with explicit fma so that the fast path, the general
// path and every CTA that recomputes a halo cell round identically (results do not depend on the
// time blocking or on which tile computed a cell).
GPR_HD float fwd_h_minus(float h, float kap, float hi, float lo) { return fmaf(-kap, hi - lo, h); }
GPR_HD float fwd_h_plus(float h, float kap, float hi, float lo) { return fmaf(kap, hi - lo, h); }
GPR_HD float fwd_e_plain(float ca, float e, float cb, float hy1, float hy0, float hxc, float hxm, float rdx)
{
  return fmaf(cb, ((hy1 - hy0) - (hxc - hxm)) * rdx, ca * e);
}

template <int TZ, int TX, int T>
struct FwdTile {
  static constexpr int RH = TZ + 2 * T, RW = TX + 8, RW4 = RW / 4;
  static constexpr int NU = RH * RW4;
  static constexpr int KU = (NU + kTileThreads - 1) / kTileThreads;
  // per-thread state kept for the whole launch: Ca/Cb of the thread's cells and, per unit, the
  // shared-memory offset and a class mask (bit 0: in the grid; 1: H fast path; 2: E fast path;
  // 3: owned by this tile).  Fast path = no CPML, no grid or region edge, no source in the unit.
  struct Regs { float ca[KU][4], cb[KU][4]; int off[KU], goff[KU]; unsigned fl[KU]; };
  static constexpr unsigned kIn = 1u, kHFast = 2u, kEFast = 4u, kOwn = 8u;

  // shared-memory carve-up (floats)
  struct Smem {
    float *ez, *hx, *hy, *pzh, *pze, *pxh, *pxe, *tz, *tx;
  };
  GPR_HD static size_t smem_floats(int zcap, int xcap)
  {
    return (size_t)3 * RH * RW + (size_t)2 * zcap * RW + (size_t)2 * RH * xcap + 6 * RH + 6 * RW;
  }
  GPR_HD static Smem carve(float* base, int zcap, int xcap)
  {
    Smem m;
    m.ez = base; m.hx = m.ez + RH * RW; m.hy = m.hx + RH * RW;
    m.pzh = m.hy + RH * RW; m.pze = m.pzh + zcap * RW;
    m.pxh = m.pze + zcap * RW; m.pxe = m.pxh + RH * xcap;
    m.tz = m.pxe + RH * xcap; m.tx = m.tz + 6 * RH;
    return m;
  }
  // first strip index met by a region starting at global index lo (E- or H-located strips)
  GPR_HD static int strip_min(int lo, int n, int P, bool hloc)
  {
    if (lo < 0) lo = 0;
    if (lo < P) return lo;
    const int nb = hloc ? n - 1 - P : n - P;
    return P + (lo > nb ? lo - nb : 0);
  }

  struct Ctx {
    Smem m;
    int s, gj0, gi0;
    int zmin_e, zmin_h, xmin_e, xmin_h;
  };
  GPR_HD static Ctx make_ctx(const FwdTileArgs& a, float* smem, int s, int ty, int tx)
  {
    Ctx c;
    c.m = carve(smem, a.zcap, a.xcap);
    c.s = s; c.gj0 = ty * TZ - T; c.gi0 = tx * TX - 4;
    c.zmin_e = strip_min(c.gj0, a.g.nz, a.g.P, false);
    c.zmin_h = strip_min(c.gj0, a.g.nz, a.g.P, true);
    c.xmin_e = strip_min(c.gi0, a.g.nx, a.g.P, false);
    c.xmin_h = strip_min(c.gi0, a.g.nx, a.g.P, true);
    return c;
  }

  // ---- stage the region ------------------------------------------------------------------------
  GPR_HD static void load(const FwdTileArgs& a, const Ctx& c, int tid, Regs& rg)
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
      rg.ca[k][0] = rg.ca[k][1] = rg.ca[k][2] = rg.ca[k][3] = 0.f;
      rg.cb[k][0] = rg.cb[k][1] = rg.cb[k][2] = rg.cb[k][3] = 0.f;
      rg.off[k] = 0; rg.goff[k] = 0; rg.fl[k] = 0u;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      const bool in = gj >= 0 && gj < g.nz && gi >= 0 && gi < g.nx;
      rg.off[k] = r * RW + lc;
      rg.goff[k] = gj * g.pitch + gi;
      if (in) {
        const int src = a.src_off[c.s];
        const int sj = src / g.pitch, si = src % g.pitch;
        const bool nozh = strip_h(gj, g.nz, g.P) < 0, noze = strip_e(gj, g.nz, g.P) < 0;
        const bool noxh = gi >= g.P && gi + 3 < g.nx - 1 - g.P, noxe = gi >= g.P && gi + 3 < g.nx - g.P;
        unsigned f = kIn;
        if (r + 1 < RH && gj <= g.nz - 2 && lc + 4 < RW && gi + 3 <= g.nx - 2 && nozh && noxh) f |= kHFast;
        if (r >= 1 && r <= RH - 2 && gj >= 1 && gj <= g.nz - 2 && lc >= 4 && lc + 3 <= RW - 2 && gi >= 1 &&
            gi + 3 <= g.nx - 2 && noze && noxe && !(gj == sj && si >= gi && si <= gi + 3))
          f |= kEFast;
        if (r >= T && r < T + TZ && lc >= 4 && lc < 4 + TX) f |= kOwn;
        rg.fl[k] = f;
      }
      float4 e = mk4(0, 0, 0, 0), hx = e, hy = e;
      if (in) {
        const long long o = c.s * g.plane + (long long)gj * g.pitch + gi;
        e = ld4(a.in.ez + o); hx = ld4(a.in.hx + o); hy = ld4(a.in.hy + o);
        unpack(ld4(a.ca + (long long)gj * g.pitch + gi), rg.ca[k]);
        unpack(ld4(a.cb + (long long)gj * g.pitch + gi), rg.cb[k]);
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
      }
      st4(m.ez + r * RW + lc, e); st4(m.hx + r * RW + lc, hx); st4(m.hy + r * RW + lc, hy);
    }
  }

  // ---- stage 1: receivers owned by this tile, sample n + t --------------------------------------
  GPR_HD static void record(const FwdTileArgs& a, const Ctx& c, int tile, int tid, int t)
  {
    if (!a.traces) return;
    const int ntile = a.tiles_x * a.tiles_y;
    const int* st = a.blk_start + (long long)c.s * (ntile + 1);
    for (int k = st[tile] + tid; k < st[tile + 1]; k += kTileThreads) {
      const int r = a.blk_rec[(long long)c.s * a.R + k];
      const int off = a.rec_off[(long long)c.s * a.R + r];
      const int lj = off / a.g.pitch - c.gj0, li = off % a.g.pitch - c.gi0;
      a.traces[c.s * a.trace_stride + (long long)t * a.R + r] = c.m.ez[lj * RW + li];
    }
  }

  // ---- stages 2-3: H update + H CPML (Eqs. 4-5) ---------------------------------
  GPR_HD static void phase_h(const FwdTileArgs& a, const Ctx& c, int tid, const Regs& rg)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
    const float kap = g.Db * g.rdx;
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      if (!(rg.fl[k] & kIn)) continue;
      if (rg.fl[k] & kHFast) {
        const int o = rg.off[k];
        const float4 e4 = ld4(m.ez + o), en = ld4(m.ez + o + RW);
        const float e5 = m.ez[o + 4];
        float4 hx = ld4(m.hx + o), hy = ld4(m.hy + o);
        hx.x = fwd_h_minus(hx.x, kap, en.x, e4.x); hx.y = fwd_h_minus(hx.y, kap, en.y, e4.y);
        hx.z = fwd_h_minus(hx.z, kap, en.z, e4.z); hx.w = fwd_h_minus(hx.w, kap, en.w, e4.w);
        hy.x = fwd_h_plus(hy.x, kap, e4.y, e4.x); hy.y = fwd_h_plus(hy.y, kap, e4.z, e4.y);
        hy.z = fwd_h_plus(hy.z, kap, e4.w, e4.z); hy.w = fwd_h_plus(hy.w, kap, e5, e4.w);
        st4(m.hx + o, hx); st4(m.hy + o, hy);
        continue;
      }
      const int u = tid + k * kTileThreads;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      float e[5];
      unpack(ld4(m.ez + r * RW + lc), e);
      e[4] = lc + 4 < RW ? m.ez[r * RW + lc + 4] : 0.f;
      if (r + 1 < RH && gj <= g.nz - 2) {
        float en[4], h[4];
        unpack(ld4(m.ez + (r + 1) * RW + lc), en);
        unpack(ld4(m.hx + r * RW + lc), h);
        const int zh = strip_h(gj, g.nz, g.P);
        if (zh >= 0) {
          float* pp = m.pzh + (zh - c.zmin_h) * RW + lc;
          float p[4];
          unpack(ld4(pp), p);
          const float b = m.tz[0 * RH + r], cc = m.tz[1 * RH + r], ik = m.tz[2 * RH + r];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const float d = (en[q] - e[q]) * g.rdx;
            p[q] = b * p[q] + cc * d;
            h[q] -= g.Db * (d * ik + p[q]);
          }
          st4(pp, mk4(p[0], p[1], p[2], p[3]));
        } else {
#pragma unroll
          for (int q = 0; q < 4; ++q) h[q] = fwd_h_minus(h[q], kap, en[q], e[q]);
        }
        st4(m.hx + r * RW + lc, mk4(h[0], h[1], h[2], h[3]));
      }
      {
        float h[4];
        unpack(ld4(m.hy + r * RW + lc), h);
        const bool xpml = (gi < g.P) || (gi + 3 >= g.nx - 1 - g.P);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (lc + q + 1 >= RW || gi + q > g.nx - 2) continue;
          const float d = (e[q + 1] - e[q]) * g.rdx;
          const int xh = xpml ? strip_h(gi + q, g.nx, g.P) : -1;
          if (xh >= 0) {
            float* pp = m.pxh + r * a.xcap + xh - c.xmin_h;
            const float p = m.tx[0 * RW + lc + q] * (*pp) + m.tx[1 * RW + lc + q] * d;
            *pp = p;
            h[q] += g.Db * (d * m.tx[2 * RW + lc + q] + p);
          } else {
            h[q] = fwd_h_plus(h[q], kap, e[q + 1], e[q]);
          }
        }
        st4(m.hy + r * RW + lc, mk4(h[0], h[1], h[2], h[3]));
      }
    }
  }

  // ---- stages 4-7: E update + E CPML (Eq. 3 in Ca/Cb form), source, save wavefield --------------
  GPR_HD static void phase_e(const FwdTileArgs& a, const Ctx& c, int tid, const Regs& rg, int t, float* ez_out)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
    const int src = a.src_off[c.s];
    const int sj = src / g.pitch, si = src % g.pitch;
    const float wn = a.wavelet[c.s * a.wav_stride + t] * (g.rdx * g.rdx);
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      if (!(rg.fl[k] & kIn)) continue;
      if (rg.fl[k] & kEFast) {
        const int o = rg.off[k];
        float4 ev = ld4(m.ez + o);
        const float4 hy = ld4(m.hy + o), hxc = ld4(m.hx + o), hxm = ld4(m.hx + o - RW);
        const float hy0 = m.hy[o - 1];
        ev.x = fwd_e_plain(rg.ca[k][0], ev.x, rg.cb[k][0], hy.x, hy0, hxc.x, hxm.x, g.rdx);
        ev.y = fwd_e_plain(rg.ca[k][1], ev.y, rg.cb[k][1], hy.y, hy.x, hxc.y, hxm.y, g.rdx);
        ev.z = fwd_e_plain(rg.ca[k][2], ev.z, rg.cb[k][2], hy.z, hy.y, hxc.z, hxm.z, g.rdx);
        ev.w = fwd_e_plain(rg.ca[k][3], ev.w, rg.cb[k][3], hy.w, hy.z, hxc.w, hxm.w, g.rdx);
        st4(m.ez + o, ev);
        if (ez_out && (rg.fl[k] & kOwn)) st4(ez_out + c.s * g.plane + rg.goff[k], ev);
        continue;
      }
      const int u = tid + k * kTileThreads;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      float e[4];
      unpack(ld4(m.ez + r * RW + lc), e);
      if (r >= 1 && r <= RH - 2 && gj >= 1 && gj <= g.nz - 2) {
        float hy[5], hxc[4], hxm[4];
        unpack(ld4(m.hy + r * RW + lc), hy + 1);
        hy[0] = lc > 0 ? m.hy[r * RW + lc - 1] : 0.f;
        unpack(ld4(m.hx + r * RW + lc), hxc);
        unpack(ld4(m.hx + (r - 1) * RW + lc), hxm);
        const int ze = strip_e(gj, g.nz, g.P);
        float pz[4] = {0.f, 0.f, 0.f, 0.f};
        float* pzp = m.pze + (ze < 0 ? 0 : ze - c.zmin_e) * RW + lc;
        if (ze >= 0) unpack(ld4(pzp), pz);
        const float bz = m.tz[3 * RH + r], cz = m.tz[4 * RH + r], kz = m.tz[5 * RH + r];
        const bool xpml = (gi < g.P) || (gi + 3 >= g.nx - g.P);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int lcol = lc + q, i = gi + q;
          if (lcol < 1 || lcol > RW - 2 || i < 1 || i > g.nx - 2) continue;
          const float dxh = (hy[q + 1] - hy[q]) * g.rdx;
          const float dzh = (hxc[q] - hxm[q]) * g.rdx;
          float vx = dxh, vz = dzh;
          const int xe = xpml ? strip_e(i, g.nx, g.P) : -1;
          if (xe >= 0) {
            float* pp = m.pxe + r * a.xcap + xe - c.xmin_e;
            const float p = m.tx[3 * RW + lcol] * (*pp) + m.tx[4 * RW + lcol] * dxh;
            *pp = p;
            vx = dxh * m.tx[5 * RW + lcol] + p;
          }
          if (ze >= 0) {
            pz[q] = bz * pz[q] + cz * dzh;
            vz = dzh * kz + pz[q];
          }
          if (xe < 0 && ze < 0) e[q] = fwd_e_plain(rg.ca[k][q], e[q], rg.cb[k][q], hy[q + 1], hy[q], hxc[q], hxm[q], g.rdx);
          else e[q] = rg.ca[k][q] * e[q] + rg.cb[k][q] * (vx - vz);
          // stage 6: source; every CTA whose region holds the cell injects
          if (gj == sj && i == si) e[q] -= rg.cb[k][q] * wn;
        }
        if (ze >= 0) st4(pzp, mk4(pz[0], pz[1], pz[2], pz[3]));
        st4(m.ez + r * RW + lc, mk4(e[0], e[1], e[2], e[3]));
      }
      // stage 7: save wavefield (owned cells only)
      if (ez_out && r >= T && r < T + TZ && lc >= 4 && lc < 4 + TX)
        st4(ez_out + c.s * g.plane + (long long)gj * g.pitch + gi, mk4(e[0], e[1], e[2], e[3]));
    }
  }

  // ---- write back what this tile owns ----------------------------------------------------------
  GPR_HD static void store(const FwdTileArgs& a, const Ctx& c, int tid)
  {
    const Geo& g = a.g;
    const Smem& m = c.m;
#pragma unroll
    for (int k = 0; k < KU; ++k) {
      const int u = tid + k * kTileThreads;
      if (u >= NU) continue;
      const int r = u / RW4, lc = (u % RW4) * 4;
      const int gj = c.gj0 + r, gi = c.gi0 + lc;
      if (r < T || r >= T + TZ || lc < 4 || lc >= 4 + TX || gj >= g.nz || gi >= g.nx) continue;
      const long long o = c.s * g.plane + (long long)gj * g.pitch + gi;
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
};

#if defined(__CUDACC__)
template <int TZ, int TX, int T>
__global__ void __launch_bounds__(kTileThreads) fwd_tile_kernel(const FwdTileArgs a)
{
  using K = FwdTile<TZ, TX, T>;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x;
  const typename K::Ctx c = K::make_ctx(a, reinterpret_cast<float*>(smem4), blockIdx.z, blockIdx.y, blockIdx.x);
  const int tile = blockIdx.y * a.tiles_x + blockIdx.x;
  typename K::Regs rg;
  K::load(a, c, tid, rg);
  __syncthreads();
  for (int t = 0; t < a.nsub; ++t) {
    K::record(a, c, tile, tid, t);
    K::phase_h(a, c, tid, rg);
    __syncthreads();
    K::phase_e(a, c, tid, rg, t, t + 1 == a.nsub ? a.out.ez : a.ez_hist[t + 1]);
    __syncthreads();
  }
  K::store(a, c, tid);
}
#endif

}  // namespace gprfwi
