// gprfwi_adj_kernel.cuh -- adjoint kernel (kernel e of north_star): ONE launch takes a group of shots
// back by up to T = 4 time steps of Algorithm 2 -- the exact transpose of the
// forward step -- and accumulates dJ/dCa, dJ/dCb in registers over those steps
// and over the shots of the group.  Same register tile as the forward kernel (gprfwi_tile.cuh).
//
// Reverse step n, lamE written mu (masked: Ca = Cb = 0 on the PEC ring), q = Cb*mu:
//   [A]  mu[rec] += residual[n+1]                          transpose of recording (staged in rowbuf)
//        gCa += mu*E^n,  gCb += mu*(E^{n+1} - Ca*E^n)/Cb   owned cells; the /Cb is applied in grad_finalize
//   [B]  tx = q/kex + cex*(psiEx + q),  psiEx <- bex*(psiEx + q)       (tx = q off the CPML)
//        tz = -q/kez + cez*(psiEz - q), psiEz <- bez*(psiEz - q)       (tz = -q)
//        lamHy += (tx[i] - tx[i+1])/dx,  lamHx += (tz[j] - tz[j+1])/dx,  mu <- Ca*mu
//   [C]  sx = p/khx + chx*(psiHx + p), psiHx <- bhx*(psiHx + p), p = Db*lamHy    (sx = p off the CPML)
//        sz likewise with p = -Db*lamHx
//        mu += (sx[i-1] - sx[i])/dx;  mu += (sz[j-1] - sz[j])/dx
// tz of a warp's first row and sz of its last row cross warps through the exchange slots, with one
// barrier each; everything else is the thread's own registers or a lane shuffle.
#pragma once
#include "gprfwi_tile.cuh"

namespace gprfwi {

struct AdjArgs {
  Geo g;
  State in, out;                      // adjoint variables, ping-pong (pointers of local shot 0)
  const float *ca, *cb;               // masked as in the forward kernel
  const float* ez_planes[kMaxT + 1];  // [t] = forward Ez^{n_hi - t} (local shot 0), t = 0..nsub
  float *gca, *gcb;                   // [ngroups][nz][pitch]
  const float* residual;              // sample n_hi of local shot 0 (sample n_hi - t at - t*nrec)
  long long trace_stride;             // nt * nrec
  const int* reg_start;               // [S*tiles + 1] CSR of receivers by REGION (tile + halo)
  const int2* reg_ent;                // in CSR order: (row*128 + column inside the region, receiver index)
  int nrec, nsub, n_hi, nt;
  int nshots, group;
  int tiles_x, tiles_y;
  int hz, oz;
  int shot_base;                      // global index of local shot 0 (for the CSR)
};

#if defined(__CUDACC__)
// transpose of recording: residual sample n_hi - t enters lamE at the start of reverse step n_hi-1-t;
// it is staged in rowbuf (zero between uses) one barrier ahead of its use.  The receivers of the
// region are dealt out one per thread (entry + its residual samples in registers).
template <int R, int NW>
__device__ __forceinline__ void adj_stage(const AdjArgs& a, const TileCtx<R, NW, 3>& c, int s, int rk0, int rk1,
                                          int2 ent, const float (&rv)[kMaxT], int t)
{
  using L = RegTile<R, NW, 3>;
  if (a.n_hi - t >= a.nt) return;
  if (ent.x >= 0) {
    float v = rv[0];
#pragma unroll
    for (int k = 1; k < kMaxT; ++k) v = t == k ? rv[k] : v;
    atomicAdd(c.rowbuf_() + ent.x, v);                                 // coincident receivers sum
  }
  for (int k = rk0 + L::THREADS + threadIdx.x; k < rk1; k += L::THREADS) {   // more receivers than threads
    const int2 e2 = a.reg_ent[k];
    atomicAdd(c.rowbuf_() + e2.x, a.residual[s * a.trace_stride - (long long)t * a.nrec + e2.y]);
  }
}

// owned rows of forward plane Ez^{n_hi - t} -> slot t % 3 of the thread's history ring (one commit group)
template <int R, int NW>
__device__ __forceinline__ void adj_fetch(const AdjArgs& a, const TileCtx<R, NW, 3>& c, int s, int t)
{
  using L = RegTile<R, NW, 3>;
  if (t <= a.nsub) {
    const float* src = a.ez_planes[t] + s * a.g.plane + (long long)c.gj0 * a.g.pitch + c.gi;
    float* dst = c.hist_() + (t % 3) * (L::ROWS * kRegW);
#pragma unroll
    for (int r = 0; r < R; ++r)
      if ((c.own >> r) & 1u) cp_async16(dst + r * kRegW, src + (long long)r * a.g.pitch);
  }
  cp_async_commit();
}

// The T reverse steps of one warp for one shot; ZP / XP as in fwd_steps (the psi forms below give
// exactly tx = q, tz = -q, sx, sz = +-Db lamH with the trivial coefficients outside the CPML).
template <int R, int NW, bool ZP, bool XP>
__device__ __forceinline__ void adj_steps(const AdjArgs& a, const TileCtx<R, NW, 3>& c, int s, int rk0, int rk1,
                                          int2 ent, const float (&rv)[kMaxT], unsigned iflags, float (&le)[R][4], float (&lhx)[R][4], float (&lhy)[R][4],
                                          const float (&ca)[R][4], const float (&cb)[R][4],
                                          float (&ga)[R][4], float (&gb)[R][4])
{
  using L = RegTile<R, NW, 3>;
  const Geo& g = a.g;
  const unsigned full = 0xffffffffu;
  const float rdx = g.rdx, Db = g.Db;
  #pragma unroll 1
  for (int t = 0; t < a.nsub; ++t) {
    // ---- [A] adjoint source, gradient terms ------------------------------------------------------
    adj_fetch<R, NW>(a, c, s, t + 2);                   // two steps ahead; planes t and t+1 have landed after the wait
    cp_async_wait<1>();
    const float* h1 = c.hist_() + (t % 3) * (L::ROWS * kRegW);
    const float* h0 = c.hist_() + ((t + 1) % 3) * (L::ROWS * kRegW);
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if ((iflags >> r) & 1u) {
        float v[4];
        float* rb = c.rowbuf_() + (c.lr0 + r) * kRegW + c.l4;
        lds4a(rb, v);
        le[r][0] = FA(le[r][0], v[0]); le[r][1] = FA(le[r][1], v[1]);
        le[r][2] = FA(le[r][2], v[2]); le[r][3] = FA(le[r][3], v[3]);
        zero4(v);
        st4a(rb, v);
      }
      if ((c.own >> r) & 1u) {
        float e0[4], e1[4];
        lds4a(h0 + r * kRegW, e0);                     // E^n
        lds4a(h1 + r * kRegW, e1);                     // E^{n+1}
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          ga[r][q] = FF(le[r][q], e0[q], ga[r][q]);
          gb[r][q] = FF(le[r][q], FF(-ca[r][q], e0[q], e1[q]), gb[r][q]);
        }
      }
    }
    // ---- [B] transpose of the E update + E CPML ----------------------------------------------------
    float tzp[4], tz0[4];                             // tz of the previous row; of the warp's row R-1
#pragma unroll
    for (int r = 0; r < R; ++r) {
      float tx[4], tz[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float qv = FM(cb[r][q], le[r][q]);
        tx[q] = qv; tz[q] = -qv;
        le[r][q] = FM(ca[r][q], le[r][q]);
      }
      if (ZP) {
        float p[4];
        lds4a(c.pez_() + r * kRegW, p);
        const float b = c.tabz_()[3 * L::ROWS + c.lr0 + r], cc = c.tabz_()[4 * L::ROWS + c.lr0 + r],
                    ik = c.tabz_()[5 * L::ROWS + c.lr0 + r];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const float T_ = FA(p[q], tz[q]);           // psiEz - q
          tz[q] = FF(cc, T_, FM(tz[q], ik));
          p[q] = FM(b, T_);
        }
        st4a(c.pez_() + r * kRegW, p);
      }
      if (XP) {                          // (all lanes: trivial coefficients off the CPML give tx = q exactly)
        float p[4], b[4], cc[4], ik[4];
        lds4a(c.pex_() + r * kRegW, p);
        lds4a(c.tabx_() + 3 * kRegW + c.l4, b); lds4a(c.tabx_() + 4 * kRegW + c.l4, cc); lds4a(c.tabx_() + 5 * kRegW + c.l4, ik);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          {
            const float T_ = FA(p[q], tx[q]);         // psiEx + q
            tx[q] = FF(cc[q], T_, FM(tx[q], ik[q]));
            p[q] = FM(b[q], T_);
          }
        }
        st4a(c.pex_() + r * kRegW, p);
      }
      const float txn[4] = {tx[1], tx[2], tx[3], __shfl_down_sync(full, tx[0], 1)};     // tx to the right
#pragma unroll
      for (int q = 0; q < 4; ++q) lhy[r][q] = FF(rdx, FS(tx[q], txn[q]), lhy[r][q]);
      if (r == 0) st4a(c.xe_() + c.w * kRegW + c.l4, tz);
      else {
#pragma unroll
        for (int q = 0; q < 4; ++q) lhx[r - 1][q] = FF(rdx, FS(tzp[q], tz[q]), lhx[r - 1][q]);
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) tzp[q] = tz[q];
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) tz0[q] = tzp[q];
    __syncthreads();
    if (t + 1 < a.nsub) adj_stage<R, NW>(a, c, s, rk0, rk1, ent, rv, t + 1);
    {
      float tzb[4];                                   // tz of the row below the warp's last row
      lds4a(c.xe_() + (c.w + 1) * kRegW + c.l4, tzb);
#pragma unroll
      for (int q = 0; q < 4; ++q) lhx[R - 1][q] = FF(rdx, FS(tz0[q], tzb[q]), lhx[R - 1][q]);
    }
    // ---- [C] transpose of the H update + H CPML ----------------------------------------------------
    float szp[4], sz0[4];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      float sx[4], sz[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) { sz[q] = FM(-Db, lhx[r][q]); sx[q] = FM(Db, lhy[r][q]); }
      if (ZP) {
        float p[4];
        lds4a(c.phz_() + r * kRegW, p);
        const float b = c.tabz_()[0 * L::ROWS + c.lr0 + r], cc = c.tabz_()[1 * L::ROWS + c.lr0 + r],
                    ik = c.tabz_()[2 * L::ROWS + c.lr0 + r];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const float T_ = FA(p[q], sz[q]);
          sz[q] = FF(cc, T_, FM(sz[q], ik));
          p[q] = FM(b, T_);
        }
        st4a(c.phz_() + r * kRegW, p);
      }
      if (XP) {                          // (all lanes: trivial coefficients off the CPML give sx = Db lamHy)
        float p[4], b[4], cc[4], ik[4];
        lds4a(c.phx_() + r * kRegW, p);
        lds4a(c.tabx_() + 0 * kRegW + c.l4, b); lds4a(c.tabx_() + 1 * kRegW + c.l4, cc); lds4a(c.tabx_() + 2 * kRegW + c.l4, ik);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          {
            const float T_ = FA(p[q], sx[q]);
            sx[q] = FF(cc[q], T_, FM(sx[q], ik[q]));
            p[q] = FM(b[q], T_);
          }
        }
        st4a(c.phx_() + r * kRegW, p);
      }
      const float sxl[4] = {__shfl_up_sync(full, sx[3], 1), sx[0], sx[1], sx[2]};       // sx to the left
#pragma unroll
      for (int q = 0; q < 4; ++q) le[r][q] = FF(rdx, FS(sxl[q], sx[q]), le[r][q]);
      if (r == 0) {
#pragma unroll
        for (int q = 0; q < 4; ++q) sz0[q] = sz[q];
      } else {
#pragma unroll
        for (int q = 0; q < 4; ++q) le[r][q] = FF(rdx, FS(szp[q], sz[q]), le[r][q]);
      }
      if (r == R - 1) st4a(c.xh_() + (c.w + 1) * kRegW + c.l4, sz);
#pragma unroll
      for (int q = 0; q < 4; ++q) szp[q] = sz[q];
    }
    __syncthreads();
    {
      float sza[4];                                   // sz of the row above the warp's first row
      lds4a(c.xh_() + c.w * kRegW + c.l4, sza);
#pragma unroll
      for (int q = 0; q < 4; ++q) le[0][q] = FF(rdx, FS(sza[q], sz0[q]), le[0][q]);
    }
  }

}

template <int R, int NW, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB) adj_kernel(const AdjArgs a)
{
  using L = RegTile<R, NW, 3>;
  extern __shared__ float4 smem4[];
  const Geo& g = a.g;
  TileCtx<R, NW, 3> c;
  c.init(reinterpret_cast<float*>(smem4), g, blockIdx.x, blockIdx.y, a.oz, a.hz);
  const int grp = blockIdx.z, tile = blockIdx.y * a.tiles_x + blockIdx.x;
  pdl_launch_dependents();
  c.template stage_tables<false>(g);
  c.zero_psi(g);
  for (int k = threadIdx.x; k < L::ROWS * kRegW / 4; k += L::THREADS)
    reinterpret_cast<float4*>(c.rowbuf_())[k] = make_float4(0.f, 0.f, 0.f, 0.f);

  float ca[R][4], cb[R][4], ga[R][4], gb[R][4];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    zero4(ca[r]); zero4(cb[r]); zero4(ga[r]); zero4(gb[r]);
    if (c.colin && ((c.rin >> r) & 1u)) {
      const long long o = (long long)(c.gj0 + r) * g.pitch + c.gi;
      ldg4a(a.ca + o, ca[r]);
      ldg4a(a.cb + o, cb[r]);
    }
  }

  pdl_wait();                          // everything below reads what the previous launch wrote
  const int s_end = min((grp + 1) * a.group, a.nshots);
  for (int s = grp * a.group; s < s_end; ++s) {
    // ---- everything this shot needs from global memory, issued together ----------------------------
    const long long row = (long long)(a.shot_base + s) * (a.tiles_x * a.tiles_y) + tile;
    const int rk0 = a.reg_start[row], rk1 = a.reg_start[row + 1];
    float le[R][4], lhx[R][4], lhy[R][4];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      zero4(le[r]); zero4(lhx[r]); zero4(lhy[r]);
      if (c.colin && ((c.rin >> r) & 1u)) {
        const long long o = s * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
        ldg4a(a.in.ez + o, le[r]);
        ldg4a(a.in.hx + o, lhx[r]);
        ldg4a(a.in.hy + o, lhy[r]);
      }
    }
    adj_fetch<R, NW>(a, c, s, 0);
    adj_fetch<R, NW>(a, c, s, 1);
    if (threadIdx.x < 2) c.mask_()[threadIdx.x] = 0u;
    c.fetch_psi(g, a.in, s);           // lands with the history planes: step 0 waits for all but the newest group
    // the receiver this thread injects, with its residual samples of this launch
    int2 ent = make_int2(-1, 0);
    float rv[kMaxT];
#pragma unroll
    for (int t = 0; t < kMaxT; ++t) rv[t] = 0.f;
    if (rk0 + (int)threadIdx.x < rk1) {
      ent = a.reg_ent[rk0 + threadIdx.x];
#pragma unroll
      for (int t = 0; t < kMaxT; ++t)
        if (t < a.nsub && a.n_hi - t < a.nt) rv[t] = a.residual[s * a.trace_stride - (long long)t * a.nrec + ent.y];
    }
    __syncthreads();                   // mask zeroed; the previous shot left rowbuf all zero
    if (ent.x >= 0) atomicOr(c.mask_() + ((ent.x / kRegW) >> 5), 1u << ((ent.x / kRegW) & 31));
    for (int k = rk0 + L::THREADS + threadIdx.x; k < rk1; k += L::THREADS) {
      const int rw = a.reg_ent[k].x / kRegW;
      atomicOr(c.mask_() + (rw >> 5), 1u << (rw & 31));
    }
    adj_stage<R, NW>(a, c, s, rk0, rk1, ent, rv, 0);
    __syncthreads();
    const unsigned iflags = c.row_flags();

    if (c.zp && c.xp) adj_steps<R, NW, true, true>(a, c, s, rk0, rk1, ent, rv, iflags, le, lhx, lhy, ca, cb, ga, gb);
    else if (c.zp) adj_steps<R, NW, true, false>(a, c, s, rk0, rk1, ent, rv, iflags, le, lhx, lhy, ca, cb, ga, gb);
    else if (c.xp) adj_steps<R, NW, false, true>(a, c, s, rk0, rk1, ent, rv, iflags, le, lhx, lhy, ca, cb, ga, gb);
    else adj_steps<R, NW, false, false>(a, c, s, rk0, rk1, ent, rv, iflags, le, lhx, lhy, ca, cb, ga, gb);

    // ---- write back the owned part of the adjoint state ------------------------------------------------
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (!((c.own >> r) & 1u)) continue;
      const long long o = s * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
      st4a(a.out.ez + o, le[r]);
      st4a(a.out.hx + o, lhx[r]);
      st4a(a.out.hy + o, lhy[r]);
    }
    if (c.zp || c.xp) c.store_psi(g, a.out, s);
  }

  // ---- once per CTA: add the register partial sums to this group's gCa / gCb planes --------------------
  // Fire-and-forget vector reductions (no CTA ever shares a cell of a group plane, so they are
  // uncontended and the result does not depend on their order).  gb holds sum mu (E^{n+1} - Ca E^n);
  // its division by Cb is done once per cell in grad_finalize_kernel.
#pragma unroll
  for (int r = 0; r < R; ++r) {
    if (!((c.own >> r) & 1u)) continue;
    const long long o = grp * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
    atomicAdd(reinterpret_cast<float4*>(a.gca + o), make_float4(ga[r][0], ga[r][1], ga[r][2], ga[r][3]));
    atomicAdd(reinterpret_cast<float4*>(a.gcb + o), make_float4(gb[r][0], gb[r][1], gb[r][2], gb[r][3]));
  }
}
#endif

}  // namespace gprfwi
