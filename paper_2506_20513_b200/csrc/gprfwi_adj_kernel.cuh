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

#if defined(GPRFWI_PROBE) && GPRFWI_PROBE == 1
#define GPR_APROBE(shot, k) GPR_PROBE(shot, k)
#else
#define GPR_APROBE(shot, k) do { } while (0)
#endif

namespace gprfwi {

struct AdjArgs {
  // TMA views of the workspace as one 3-D array [plane][nz][roundup4(nx)] of fp32 (all field planes sit a
  // whole number of planes from its first byte): box = 128 columns x the tile's owned rows / x all the
  // region's rows
  alignas(64) CUtensorMap tm_own;
  alignas(64) CUtensorMap tm_reg;
  Geo g;
  State in, out;                      // adjoint variables, ping-pong (pointers of local shot 0)
  const float *ca, *cb;               // masked as in the forward kernel
  const float* dbc;                   // per-cell Db as in the forward kernel, or NULL: mu_r = 1
  int ez_pl[kMaxT + 1];               // [t] = workspace plane index of forward Ez^{n_hi - t} (local shot 0), t = 0..nsub
  int in_pl[3];                       // workspace plane indices of in.ez, in.hx, in.hy (local shot 0)
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
// Rare paths, kept out of line so that they do not sit in the step loop's instruction stream (the loops'
// code size matters: DESIGN.md section 9): receivers beyond the first THREADS of a region, and receivers
// that share their cell with another one of the region (the shared-memory float add is a CAS loop).
__device__ __noinline__ void adj_stage_overflow(const AdjArgs& a, float* rowbuf, int threads, int s, int rk0, int rk1, int t)
{
  for (int k = rk0 + threads + threadIdx.x; k < rk1; k += threads) {
    const int2 e2 = a.reg_ent[k];
    atomicAdd(rowbuf + (e2.x & kEntMask), a.residual[s * a.trace_stride - (long long)t * a.nrec + e2.y]);
  }
}
__device__ __noinline__ void adj_stage_shared_cell(float* cell, float v) { atomicAdd(cell, v); }

template <int R, int NW>
__device__ __forceinline__ void adj_stage(const AdjArgs& a, const TileCtx<R, NW, kAdjRing>& c, int s, int rk0, int rk1,
                                          int entx, int t)
{
  using L = RegTile<R, NW, kAdjRing>;
  if (a.n_hi - t >= a.nt) return;
  if (entx >= 0) {
    // a cell that holds one receiver of the region has one writer (rowbuf is zero between uses);
    // coincident receivers (entry flagged by the host) sum atomically
    if (entx & kEntShared) adj_stage_shared_cell(c.rowbuf_() + (entx & kEntMask), c.priv_()[t]);
    else c.rowbuf_()[entx] = c.priv_()[t];
  }
  if (rk1 - rk0 > L::THREADS) adj_stage_overflow(a, c.rowbuf_(), L::THREADS, s, rk0, rk1, t);   // more receivers than threads
}

// The forward Ez planes a CTA reads form one stream: planes 0 .. nsub of its first shot (plane t =
// Ez^{n_hi - t}), then those of its next shot, and so on.  Stream position `pos` lands in slot pos % kAdjRing
// of the history ring; the mbarrier of a slot completes once per fetch into it, so the fetch at position pos
// is awaited with parity (pos / kAdjRing) & 1.  Step t of the shot whose plane 0 sits at position q0 reads
// positions q0 + t and q0 + t + 1 and has position q0 + t + kAdjRing - 1 fetched (a shot has one plane more
// than it has steps: position q0 + kAdjRing - 2 is fetched when the shot begins), so the first plane(s) of
// the next shot are in flight during the last step(s) of this one.  ONE thread issues the copy (TMA: box = 128 columns x the owned rows, placed at the
// owned rows of the slot; cells outside the grid arrive as zeros); it does so right after a CTA barrier that
// follows every thread's last read of the slot's previous contents (position pos - kAdjRing).
template <int R, int NW>
__device__ __forceinline__ void adj_fetch(const AdjArgs& a, const TileCtx<R, NW, kAdjRing>& c, int s, int s_end, int q0, int pos)
{
  using L = RegTile<R, NW, kAdjRing>;
  int t = pos - q0;
  if (t > a.nsub) { t -= a.nsub + 1; ++s; }             // a plane of the next shot
  if (s >= s_end) return;
  const unsigned bar = smem_u32(c.sm + L::MBAR) + 8u * (unsigned)(pos % kAdjRing);
  mbar_expect_tx(bar, (unsigned)(a.oz * kRegW * sizeof(float)));
  tma_load_3d(smem_u32(c.sm + L::HIST + (pos % kAdjRing) * (L::ROWS * kRegW) + a.hz * kRegW), &a.tm_own, c.ri0,
              c.rj0 + a.hz, a.ez_pl[t] + s, bar);
}
template <int R, int NW>
__device__ __forceinline__ void adj_await(const TileCtx<R, NW, kAdjRing>& c, int pos)
{
  using L = RegTile<R, NW, kAdjRing>;
  mbar_wait(smem_u32(c.sm + L::MBAR) + 8u * (unsigned)(pos % kAdjRing), (unsigned)(pos / kAdjRing) & 1u);
}

// A CTA that touches no CPML never uses the psi region of its shared memory: it serves as the landing zone
// [3][ROWS][128] for the NEXT shot's adjoint state (lamE, lamHx, lamHy: three TMA boxes of the whole region
// on mbarrier kAdjRing), fetched while this shot is stepped, so that the next shot does not start with its state
// loads exposed.
template <int R, int NW>
__device__ __forceinline__ void adj_prefetch_state(const AdjArgs& a, const TileCtx<R, NW, kAdjRing>& c, int s_next)
{
  using L = RegTile<R, NW, kAdjRing>;
  const unsigned bar = smem_u32(c.sm + L::MBAR) + 8u * kAdjRing;
  mbar_expect_tx(bar, (unsigned)(3 * L::ROWS * kRegW * sizeof(float)));
#pragma unroll
  for (int f = 0; f < 3; ++f)
    tma_load_3d(smem_u32(c.sm + L::LAND + f * (L::ROWS * kRegW)), &a.tm_reg, c.ri0, c.rj0, a.in_pl[f] + s_next, bar);
}

// The T reverse steps of one warp for one shot; ZP / XP as in fwd_steps (the psi forms below give
// exactly tx = q, tz = -q, sx, sz = +-Db lamH with the trivial coefficients outside the CPML).
// Packed pairs as in the forward kernel: P = (c0, c2), Q = (c1, c3).
template <int R, int NW, bool ZP, bool XP, bool MU>
__device__ __forceinline__ void adj_steps(const AdjArgs& a, const TileCtx<R, NW, kAdjRing>& c, int s, int rk0, int rk1,
                                          int entx, unsigned iflags, bool prefetch, int q0, int s_end,
                                          P2 (&le)[R], P2 (&lhx)[R], P2 (&lhy)[R], const P2 (&ca)[R], const P2 (&cb)[R],
                                          P2 (&ga)[R], P2 (&gb)[R])
{
  using L = RegTile<R, NW, kAdjRing>;
  const unsigned full = 0xffffffffu;
  const u64 rdx2 = bc2(a.g.rdx), Db2 = bc2(a.g.Db), nDb2 = bc2(-a.g.Db);
#pragma unroll 1
  for (int t = 0; t < a.nsub; ++t) {
    // ---- [A] adjoint source, gradient terms ------------------------------------------------------
    if (threadIdx.x == 0) {                             // (every thread is past the previous step's barriers)
      adj_fetch<R, NW>(a, c, s, s_end, q0, q0 + t + kAdjRing - 1);           // kAdjRing - 1 positions ahead
      if (t == 0 && prefetch) adj_prefetch_state<R, NW>(a, c, s + 1);
    }
    if (t == 0) adj_await<R, NW>(c, q0);                // planes t and t + 1 (plane t was awaited a step ago)
    adj_await<R, NW>(c, q0 + t + 1);
    const float* h1 = c.hist_() + ((q0 + t) % kAdjRing) * (L::ROWS * kRegW);
    const float* h0 = c.hist_() + ((q0 + t + 1) % kAdjRing) * (L::ROWS * kRegW);
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if ((iflags >> r) & 1u) {
        float* rb = c.rowbuf_() + (c.lr0 + r) * kRegW + c.l4;
        const P2 v = ld2(rb);
        le[r].p = add2(le[r].p, v.p); le[r].q = add2(le[r].q, v.q);
        st2(rb, zero2());
      }
      {                                                 // (every thread: what the accumulators of cells the tile does not
                                                        //  own collect is never flushed)
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
      if (MU) {                                         // per-cell Db (mu_r model, reading R22)
        const P2 db = ld2(c.dbc_(a.g) + r * kRegW);
        sz.p = mul2(neg2(db.p), lhx[r].p); sz.q = mul2(neg2(db.q), lhx[r].q);
        sx.p = mul2(db.p, lhy[r].p); sx.q = mul2(db.q, lhy[r].q);
      } else {
        sz.p = mul2(nDb2, lhx[r].p); sz.q = mul2(nDb2, lhx[r].q);
        sx.p = mul2(Db2, lhy[r].p); sx.q = mul2(Db2, lhy[r].q);
      }
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
    GPR_APROBE(s % a.group, 4 + t);
  }
}

template <int R, int NW, int MINB, bool MU>
__global__ void __launch_bounds__(NW * 32, MINB) adj_kernel(const __grid_constant__ AdjArgs a)
{
  using L = RegTile<R, NW, kAdjRing>;
  extern __shared__ __align__(128) float4 smem4[];
  const Geo& g = a.g;
  TileCtx<R, NW, kAdjRing> c;
  c.init(reinterpret_cast<float*>(smem4), g, blockIdx.x, blockIdx.y, a.oz, a.hz);
  const int grp = blockIdx.z, tile = blockIdx.y * a.tiles_x + blockIdx.x;
  pdl_launch_dependents();
  if (threadIdx.x == 0) {              // mbarriers 0 .. kAdjRing-1: history ring slots, kAdjRing: state landing zone
#pragma unroll
    for (int k = 0; k <= kAdjRing; ++k) mbar_init(smem_u32(c.sm + L::MBAR) + 8u * k, 1u);
    mbar_init_fence();
  }
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
  if (MU) c.load_dbc(g, a.dbc);
  for (int k = threadIdx.x; k < L::ROWS * kRegW / 4; k += L::THREADS)
    reinterpret_cast<float4*>(c.rowbuf_())[k] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int k = 0; k < kAdjRing * R; ++k)      // the thread's own slots of the Ez-history ring (rows the copies never fill)
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
  // a CTA none of whose warps touches the CPML lands the next shot's state in the (unused) psi region
  const bool can_land = g.P > 0 && !__syncthreads_or((c.zp || c.xp) ? 1 : 0);      // (barrier: the group's scalars are visible)
  // the receiver this thread injects (receivers of the region are dealt out one per thread); fetched one
  // shot ahead into the thread's private slot so that no shot starts with a chain of dependent loads
  {
    int2 e0 = make_int2(-1, 0);
    if (c.meta_()[0] + (int)threadIdx.x < c.meta_()[1]) e0 = a.reg_ent[c.meta_()[0] + threadIdx.x];
    *reinterpret_cast<int2*>(c.priv_() + 4) = e0;
  }

  pdl_wait();                          // everything below reads what the previous launch wrote
  bool landed = false;
  int q0 = 0, nland = 0;               // stream position of this shot's plane 0; state landings so far
  for (int s = s_beg; s < s_end; ++s, q0 += a.nsub + 1) {
    // ---- everything this shot needs from global memory, issued together ----------------------------
    GPR_APROBE(s - s_beg, 0);
    const int* m = c.meta_() + (s - s_beg) * 4;
    const int rk0 = m[0], rk1 = m[1];
    const unsigned iflags = (unsigned)((((unsigned long long)(unsigned)m[3] << 32) | (unsigned)m[2]) >> c.lr0) & ((1u << R) - 1u);
    const int2 ent = *reinterpret_cast<const int2*>(c.priv_() + 4);
    P2 le[R], lhx[R], lhy[R];
    if (threadIdx.x == 0) {            // (every thread is past the last barrier of the previous shot; planes
                                       //  0 .. kAdjRing - 3 of a later shot came during the previous shot's last steps)
      for (int k = (s == s_beg ? 0 : kAdjRing - 2); k < kAdjRing - 1; ++k) adj_fetch<R, NW>(a, c, s, s_end, q0, q0 + k);
    }
    if (landed) {                      // this shot's state was fetched into the landing zone during the previous one
      mbar_wait(smem_u32(c.sm + L::MBAR) + 8u * kAdjRing, (unsigned)(nland - 1) & 1u);
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      le[r] = zero2(); lhx[r] = zero2(); lhy[r] = zero2();
      if (c.colin && ((c.rin >> r) & 1u)) {
        if (landed) {
          le[r] = ld2(c.sm + L::LAND + 0 * (L::ROWS * kRegW) + c.toff + r * kRegW);
          lhx[r] = ld2(c.sm + L::LAND + 1 * (L::ROWS * kRegW) + c.toff + r * kRegW);
          lhy[r] = ld2(c.sm + L::LAND + 2 * (L::ROWS * kRegW) + c.toff + r * kRegW);
        } else {
          const long long o = s * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
          le[r] = ldcg2(a.in.ez + o);  // (written by the previous launch: not through the read-only path)
          lhx[r] = ldcg2(a.in.hx + o);
          lhy[r] = ldcg2(a.in.hy + o);
        }
      }
    }
    GPR_APROBE(s - s_beg, 1);
    const bool prefetch = can_land && s + 1 < s_end;
    c.fetch_psi(g, a.in, s);           // (one cp.async group, awaited before the barrier below)
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
    GPR_APROBE(s - s_beg, 2);
    cp_async_wait<0>();
    __syncthreads();
    GPR_APROBE(s - s_beg, 3);

#define GPR_ADJ_STEPS(ZP_, XP_) \
  adj_steps<R, NW, ZP_, XP_, MU>(a, c, s, rk0, rk1, entx, iflags, prefetch, q0, s_end, le, lhx, lhy, ca, cb, ga, gb)
    if (c.zp && c.xp) GPR_ADJ_STEPS(true, true);
    else if (c.zp) GPR_ADJ_STEPS(true, false);
    else if (c.xp) GPR_ADJ_STEPS(false, true);
    else GPR_ADJ_STEPS(false, false);
#undef GPR_ADJ_STEPS

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
    nland += prefetch ? 1 : 0;
    GPR_APROBE(s - s_beg, 8);
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
