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
  const uint2* reg_mask;              // [S*tiles]: bit j = row j of the region holds a receiver of the shot
  int nrec, nsub, n_hi, nt;
  int nshots, group;
  int tiles_x, tiles_y;
  int hz, oz;
  int shot_base;                      // global index of local shot 0 (for the CSR)
};

#if defined(__CUDACC__)
// transpose of recording: residual sample n_hi - t enters lamE at the start of reverse step n_hi-1-t;
// it is staged in rowbuf (zero between uses) one barrier ahead of its use.  The receivers of the
// region are dealt out one per thread (its residual samples of the launch sit in the thread's private
// shared-memory slot).
template <int R, int NW>
__device__ __forceinline__ void adj_stage(const AdjArgs& a, const TileCtx<R, NW, 3>& c, int s, int rk0, int rk1,
                                          int entx, int t)
{
  using L = RegTile<R, NW, 3>;
  if (a.n_hi - t >= a.nt) return;
  if (entx >= 0) atomicAdd(c.rowbuf_() + entx, c.priv_()[t]);          // coincident receivers sum
  if (rk1 - rk0 > L::THREADS)                                                // more receivers than threads
    for (int k = rk0 + L::THREADS + threadIdx.x; k < rk1; k += L::THREADS) {
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
}

// A warp that touches no CPML never uses its thread-private psi slots: they serve as the landing zone for
// the NEXT shot's adjoint state (field f: 0 lamE, 1 lamHx, 2 lamHy), fetched while this shot is stepped, so
// that the next shot does not start with the state loads exposed.
template <int R, int NW>
__device__ __forceinline__ float* adj_land(const TileCtx<R, NW, 3>& c, int f)
{
  return f == 0 ? c.phz_() : (f == 1 ? c.pez_() : c.phx_());
}
template <int R, int NW>
__device__ __forceinline__ void adj_prefetch_state(const AdjArgs& a, const TileCtx<R, NW, 3>& c, int s_next, int f)
{
  const float* src = (f == 0 ? a.in.ez : (f == 1 ? a.in.hx : a.in.hy)) + s_next * a.g.plane + (long long)c.gj0 * a.g.pitch + c.gi;
  float* dst = adj_land<R, NW>(c, f);
#pragma unroll
  for (int r = 0; r < R; ++r)
    if (c.colin && ((c.rin >> r) & 1u)) cp_async16(dst + r * kRegW, src + (long long)r * a.g.pitch);
}

// The T reverse steps of one warp for one shot; ZP / XP as in fwd_steps (the psi forms below give
// exactly tx = q, tz = -q, sx, sz = +-Db lamH with the trivial coefficients outside the CPML).
// Packed pairs as in the forward kernel: P = (c0, c2), Q = (c1, c3).
template <int R, int NW, bool ZP, bool XP>
__device__ __forceinline__ void adj_steps(const AdjArgs& a, const TileCtx<R, NW, 3>& c, int s, int rk0, int rk1,
                                          int entx, unsigned iflags, bool prefetch,
                                          P2 (&le)[R], P2 (&lhx)[R], P2 (&lhy)[R], const P2 (&ca)[R], const P2 (&cb)[R],
                                          P2 (&ga)[R], P2 (&gb)[R])
{
  using L = RegTile<R, NW, 3>;
  const unsigned full = 0xffffffffu;
  const u64 rdx2 = bc2(a.g.rdx), Db2 = bc2(a.g.Db), nDb2 = bc2(-a.g.Db);
#pragma unroll 1
  for (int t = 0; t < a.nsub; ++t) {
    // ---- [A] adjoint source, gradient terms ------------------------------------------------------
    adj_fetch<R, NW>(a, c, s, t + 2);                   // two steps ahead; planes t and t+1 have landed after the wait
    if (prefetch) {                                     // next shot's state, one field per step, in the same commit group
      if (t < 3) adj_prefetch_state<R, NW>(a, c, s + 1, t);
      if (t + 1 == a.nsub)
        for (int f = t + 1; f < 3; ++f) adj_prefetch_state<R, NW>(a, c, s + 1, f);
    }
    cp_async_commit();
    cp_async_wait<1>();
    const float* h1 = c.hist_() + (t % 3) * (L::ROWS * kRegW);
    const float* h0 = c.hist_() + ((t + 1) % 3) * (L::ROWS * kRegW);
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if ((iflags >> r) & 1u) {
        float* rb = c.rowbuf_() + (c.lr0 + r) * kRegW + c.l4;
        const P2 v = ld2(rb);
        le[r].p = add2(le[r].p, v.p); le[r].q = add2(le[r].q, v.q);
        st2(rb, zero2());
      }
      {                                                 // (every thread: the ring slots of cells the tile does not own
                                                        //  are never fetched into and stay zero, so they add nothing)
        const P2 e0 = ld2(h0 + r * kRegW), e1 = ld2(h1 + r * kRegW);      // E^n, E^{n+1}
        ga[r].p = fma2(le[r].p, e0.p, ga[r].p); ga[r].q = fma2(le[r].q, e0.q, ga[r].q);
        gb[r].p = fma2(le[r].p, fma2(neg2(ca[r].p), e0.p, e1.p), gb[r].p);
        gb[r].q = fma2(le[r].q, fma2(neg2(ca[r].q), e0.q, e1.q), gb[r].q);
      }
    }
    // ---- [B] transpose of the E update + E CPML ----------------------------------------------------
    P2 xb = zero2(), xc = zero2(), xk = zero2();
    if (XP) { xb = ld2(c.tabx_() + 3 * kRegW + c.l4); xc = ld2(c.tabx_() + 4 * kRegW + c.l4); xk = ld2(c.tabx_() + 5 * kRegW + c.l4); }
    P2 tzp = zero2();                                   // tz of the previous row; after the loop: of row R-1
#pragma unroll
    for (int r = 0; r < R; ++r) {
      P2 tx, tz;
      tx.p = mul2(cb[r].p, le[r].p); tx.q = mul2(cb[r].q, le[r].q);       // q = Cb mu
      tz.p = neg2(tx.p); tz.q = neg2(tx.q);
      le[r].p = mul2(ca[r].p, le[r].p); le[r].q = mul2(ca[r].q, le[r].q);
      if (ZP) {
        P2 p = ld2(c.pez_() + r * kRegW);
        const u64 b = bc2(c.tabz_()[3 * L::ROWS + c.lr0 + r]), cc = bc2(c.tabz_()[4 * L::ROWS + c.lr0 + r]),
                  ik = bc2(c.tabz_()[5 * L::ROWS + c.lr0 + r]);
        const u64 Tp = add2(p.p, tz.p), Tq = add2(p.q, tz.q);             // psiEz - q
        tz.p = fma2(cc, Tp, mul2(tz.p, ik)); tz.q = fma2(cc, Tq, mul2(tz.q, ik));
        p.p = mul2(b, Tp); p.q = mul2(b, Tq);
        st2(c.pez_() + r * kRegW, p);
      }
      if (XP) {                                         // (all lanes: trivial coefficients off the CPML give tx = q exactly)
        P2 p = ld2(c.pex_() + r * kRegW);
        const u64 Tp = add2(p.p, tx.p), Tq = add2(p.q, tx.q);             // psiEx + q
        tx.p = fma2(xc.p, Tp, mul2(tx.p, xk.p)); tx.q = fma2(xc.q, Tq, mul2(tx.q, xk.q));
        p.p = mul2(xb.p, Tp); p.q = mul2(xb.q, Tq);
        st2(c.pex_() + r * kRegW, p);
      }
      // tx to the right of (c0, c2) is Q; to the right of (c1, c3) it is (c2, c0 of the next lane)
      const u64 txnq = pk(hi2(tx.p), __shfl_down_sync(full, lo2(tx.p), 1));
      lhy[r].p = fma2(rdx2, sub2(tx.p, tx.q), lhy[r].p);
      lhy[r].q = fma2(rdx2, sub2(tx.q, txnq), lhy[r].q);
      if (r == 0) st2(c.xe_() + c.w * kRegW + c.l4, tz);
      else {
        lhx[r - 1].p = fma2(rdx2, sub2(tzp.p, tz.p), lhx[r - 1].p);
        lhx[r - 1].q = fma2(rdx2, sub2(tzp.q, tz.q), lhx[r - 1].q);
      }
      tzp = tz;
    }
    __syncthreads();
    if (t + 1 < a.nsub) adj_stage<R, NW>(a, c, s, rk0, rk1, entx, t + 1);
    {
      const P2 tzb = ld2(c.xe_() + (c.w + 1) * kRegW + c.l4);             // tz of the row below the warp's last row
      lhx[R - 1].p = fma2(rdx2, sub2(tzp.p, tzb.p), lhx[R - 1].p);
      lhx[R - 1].q = fma2(rdx2, sub2(tzp.q, tzb.q), lhx[R - 1].q);
    }
    // ---- [C] transpose of the H update + H CPML ----------------------------------------------------
    if (XP) { xb = ld2(c.tabx_() + 0 * kRegW + c.l4); xc = ld2(c.tabx_() + 1 * kRegW + c.l4); xk = ld2(c.tabx_() + 2 * kRegW + c.l4); }
    P2 szp = zero2(), sz0 = zero2();
#pragma unroll
    for (int r = 0; r < R; ++r) {
      P2 sx, sz;
      sz.p = mul2(nDb2, lhx[r].p); sz.q = mul2(nDb2, lhx[r].q);
      sx.p = mul2(Db2, lhy[r].p); sx.q = mul2(Db2, lhy[r].q);
      if (ZP) {
        P2 p = ld2(c.phz_() + r * kRegW);
        const u64 b = bc2(c.tabz_()[0 * L::ROWS + c.lr0 + r]), cc = bc2(c.tabz_()[1 * L::ROWS + c.lr0 + r]),
                  ik = bc2(c.tabz_()[2 * L::ROWS + c.lr0 + r]);
        const u64 Tp = add2(p.p, sz.p), Tq = add2(p.q, sz.q);
        sz.p = fma2(cc, Tp, mul2(sz.p, ik)); sz.q = fma2(cc, Tq, mul2(sz.q, ik));
        p.p = mul2(b, Tp); p.q = mul2(b, Tq);
        st2(c.phz_() + r * kRegW, p);
      }
      if (XP) {                                         // (all lanes: trivial coefficients off the CPML give sx = Db lamHy)
        P2 p = ld2(c.phx_() + r * kRegW);
        const u64 Tp = add2(p.p, sx.p), Tq = add2(p.q, sx.q);
        sx.p = fma2(xc.p, Tp, mul2(sx.p, xk.p)); sx.q = fma2(xc.q, Tq, mul2(sx.q, xk.q));
        p.p = mul2(xb.p, Tp); p.q = mul2(xb.q, Tq);
        st2(c.phx_() + r * kRegW, p);
      }
      // sx to the left of (c0, c2) is (c3 of the previous lane, c1); to the left of (c1, c3) it is P
      const u64 sxlp = pk(__shfl_up_sync(full, hi2(sx.q), 1), lo2(sx.q));
      le[r].p = fma2(rdx2, sub2(sxlp, sx.p), le[r].p);
      le[r].q = fma2(rdx2, sub2(sx.p, sx.q), le[r].q);
      if (r == 0) sz0 = sz;
      else {
        le[r].p = fma2(rdx2, sub2(szp.p, sz.p), le[r].p);
        le[r].q = fma2(rdx2, sub2(szp.q, sz.q), le[r].q);
      }
      if (r == R - 1) st2(c.xh_() + (c.w + 1) * kRegW + c.l4, sz);
      szp = sz;
    }
    __syncthreads();
    {
      const P2 sza = ld2(c.xh_() + c.w * kRegW + c.l4);                   // sz of the row above the warp's first row
      le[0].p = fma2(rdx2, sub2(sza.p, sz0.p), le[0].p);
      le[0].q = fma2(rdx2, sub2(sza.q, sz0.q), le[0].q);
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
  // per-shot scalars of the whole group (static input: nothing a previous launch writes), word k of 4:
  // receiver range [rk0, rk1) of the region, 64-bit mask of the region rows that hold a receiver
  const int s_beg = grp * a.group, s_end = min((grp + 1) * a.group, a.nshots);
  for (int k = threadIdx.x; k < 4 * (s_end - s_beg); k += L::THREADS) {
    const long long row = (long long)(a.shot_base + s_beg + (k >> 2)) * (a.tiles_x * a.tiles_y) + tile;
    const int q = k & 3;
    c.meta_()[k] = q < 2 ? a.reg_start[row + q] : (q == 2 ? (int)a.reg_mask[row].x : (int)a.reg_mask[row].y);
  }
  c.template stage_tables<false>(g);
  c.zero_psi(g);
  for (int k = threadIdx.x; k < L::ROWS * kRegW / 4; k += L::THREADS)
    reinterpret_cast<float4*>(c.rowbuf_())[k] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int k = 0; k < 3 * R; ++k)      // the thread's own slots of the Ez-history ring (see [A])
    st2(c.hist_() + (k / R) * (L::ROWS * kRegW) + (k % R) * kRegW, zero2());

  P2 ca[R], cb[R], ga[R], gb[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    ca[r] = zero2(); cb[r] = zero2(); ga[r] = zero2(); gb[r] = zero2();
    if (c.colin && ((c.rin >> r) & 1u)) {
      const long long o = (long long)(c.gj0 + r) * g.pitch + c.gi;
      ca[r] = ldg2(a.ca + o);
      cb[r] = ldg2(a.cb + o);
    }
  }
  __syncthreads();                     // the group's scalars are visible
  // the receiver this thread injects (receivers of the region are dealt out one per thread); fetched one
  // shot ahead into the thread's private slot so that no shot starts with a chain of dependent loads
  {
    int2 e0 = make_int2(-1, 0);
    if (c.meta_()[0] + (int)threadIdx.x < c.meta_()[1]) e0 = a.reg_ent[c.meta_()[0] + threadIdx.x];
    *reinterpret_cast<int2*>(c.priv_() + 4) = e0;
  }

  pdl_wait();                          // everything below reads what the previous launch wrote
  const bool can_land = g.P > 0 && !(c.zp || c.xp);     // (warp-uniform; the psi slots exist only when npml > 0)
  bool landed = false;
  for (int s = s_beg; s < s_end; ++s) {
    // ---- everything this shot needs from global memory, issued together ----------------------------
    const int* m = c.meta_() + (s - s_beg) * 4;
    const int rk0 = m[0], rk1 = m[1];
    const unsigned iflags = (unsigned)((((unsigned long long)(unsigned)m[3] << 32) | (unsigned)m[2]) >> c.lr0) & ((1u << R) - 1u);
    const int2 ent = *reinterpret_cast<const int2*>(c.priv_() + 4);
    P2 le[R], lhx[R], lhy[R];
    if (landed) cp_async_wait<0>();    // this shot's state was fetched into the warp's landing slots during the previous one
#pragma unroll
    for (int r = 0; r < R; ++r) {
      le[r] = zero2(); lhx[r] = zero2(); lhy[r] = zero2();
      if (c.colin && ((c.rin >> r) & 1u)) {
        if (landed) {
          le[r] = ld2(adj_land<R, NW>(c, 0) + r * kRegW);
          lhx[r] = ld2(adj_land<R, NW>(c, 1) + r * kRegW);
          lhy[r] = ld2(adj_land<R, NW>(c, 2) + r * kRegW);
        } else {
          const long long o = s * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
          le[r] = ldcg2(a.in.ez + o);  // (written by the previous launch: not through the read-only path)
          lhx[r] = ldcg2(a.in.hx + o);
          lhy[r] = ldcg2(a.in.hy + o);
        }
      }
    }
    const bool prefetch = can_land && s + 1 < s_end;
    adj_fetch<R, NW>(a, c, s, 0);
    cp_async_commit();
    adj_fetch<R, NW>(a, c, s, 1);
    cp_async_commit();
    c.fetch_psi(g, a.in, s);           // lands with the history planes: step 0 waits for all but the newest group
    // this thread's residual samples of this launch, and the receiver it injects for the next shot
    float rv[kMaxT];
#pragma unroll
    for (int t = 0; t < kMaxT; ++t) rv[t] = 0.f;
    if (ent.x >= 0) {
#pragma unroll
      for (int t = 0; t < kMaxT; ++t)
        if (t < a.nsub && a.n_hi - t < a.nt) rv[t] = a.residual[s * a.trace_stride - (long long)t * a.nrec + ent.y];
    }
    int2 ent_next = make_int2(-1, 0);
    if (s + 1 < s_end && m[4] + (int)threadIdx.x < m[5]) ent_next = a.reg_ent[m[4] + threadIdx.x];
    *reinterpret_cast<float4*>(c.priv_()) = make_float4(rv[0], rv[1], rv[2], rv[3]);
    *reinterpret_cast<int2*>(c.priv_() + 4) = ent_next;
    const int entx = ent.x;
    adj_stage<R, NW>(a, c, s, rk0, rk1, entx, 0);         // (the previous shot left rowbuf all zero, two barriers ago)
    __syncthreads();

    if (c.zp && c.xp) adj_steps<R, NW, true, true>(a, c, s, rk0, rk1, entx, iflags, prefetch, le, lhx, lhy, ca, cb, ga, gb);
    else if (c.zp) adj_steps<R, NW, true, false>(a, c, s, rk0, rk1, entx, iflags, prefetch, le, lhx, lhy, ca, cb, ga, gb);
    else if (c.xp) adj_steps<R, NW, false, true>(a, c, s, rk0, rk1, entx, iflags, prefetch, le, lhx, lhy, ca, cb, ga, gb);
    else adj_steps<R, NW, false, false>(a, c, s, rk0, rk1, entx, iflags, prefetch, le, lhx, lhy, ca, cb, ga, gb);

    // ---- write back the owned part of the adjoint state ------------------------------------------------
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (!((c.own >> r) & 1u)) continue;
      const long long o = s * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
      st2(a.out.ez + o, le[r]);
      st2(a.out.hx + o, lhx[r]);
      st2(a.out.hy + o, lhy[r]);
    }
    if (c.zp || c.xp) c.store_psi(g, a.out, s);
    landed = prefetch;
  }

  // ---- once per CTA: add the register partial sums to this group's gCa / gCb planes --------------------
  // Fire-and-forget vector reductions (no CTA ever shares a cell of a group plane, so they are
  // uncontended and the result does not depend on their order).  gb holds sum mu (E^{n+1} - Ca E^n);
  // its division by Cb is done once per cell in grad_finalize_kernel.
#pragma unroll
  for (int r = 0; r < R; ++r) {
    if (!((c.own >> r) & 1u)) continue;
    const long long o = grp * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
    // (memory order inside a unit is c0 c2 c1 c3 = P.lo P.hi Q.lo Q.hi, like every internal plane)
    atomicAdd(reinterpret_cast<float4*>(a.gca + o), make_float4(lo2(ga[r].p), hi2(ga[r].p), lo2(ga[r].q), hi2(ga[r].q)));
    atomicAdd(reinterpret_cast<float4*>(a.gcb + o), make_float4(lo2(gb[r].p), hi2(gb[r].p), lo2(gb[r].q), hi2(gb[r].q)));
  }
}
#endif

}  // namespace gprfwi
