// gprfwi_fwd_kernel.cuh -- forward kernel (kernels b, c, d of north_star fused): ONE launch advances
// all shots by up to T = 4 time steps of Algorithm 1:
//   stage 1  record receivers (trace sample n = Ez BEFORE step n)
//   stage 2-3  H update + H-side CPML  (Eqs. (4)-(5))
//   stage 4-5  E update + E-side CPML  (Eq. (3) in the Ca/Cb form of the paper's kernel)
//   stage 6  source:  Ez[src] -= Cb[src] * w[n] / dx^2   (PAPER.md:364-384 with dl = dz)
//   stage 7  save wavefield: every step's Ez plane of the owned cells (history / recompute segment)
// on the register tile of gprfwi_tile.cuh.  Per step: H phase, barrier, E phase, barrier.
//
// CPML (reading R4): psi <- b psi + c d, derivative term d/kappa + psi with d the difference
// quotient, written with pre-multiplied tables so that with the trivial coefficients outside the CPML
// (b = c = 0, kappa = 1) every expression rounds EXACTLY like the plain one:
//   Hx -= Db psi + (Db/(dx kappa)) (E[j+1] - E[j]),   psi <- b psi + (c/dx) (E[j+1] - E[j])
//   Ez  = Ca Ez + Cb (((Hy - Hy[i-1])/kx - (Hx - Hx[j-1])/kz)/dx + (psix - psiz))
// A warp whose rows (ZP) / whose CTA's columns (XP) touch the CPML runs the psi form on all its
// cells, every other warp the plain form; a cell's value does not depend on which form computed it.
// All arithmetic is packed fp32 pairs (FFMA2 / FADD2 / FMUL2, gprfwi_tile.cuh): each component is
// rounded exactly like the scalar operation, at half the issue slots.
#pragma once
#include "gprfwi_tile.cuh"

#if defined(GPRFWI_PROBE) && GPRFWI_PROBE == 2
#define GPR_FPROBE(shot, k) GPR_PROBE(shot, k)
#else
#define GPR_FPROBE(shot, k) do { } while (0)
#endif

namespace gprfwi {

struct FwdArgs {
  // TMA view of the workspace as one 3-D array of planes (gprfwi_adj_kernel.cuh), box = 128 columns x the region's rows
  alignas(64) CUtensorMap tm_reg;
  int in_pl[3];               // workspace plane indices of in.ez, in.hx, in.hy (local shot 0)
  Geo g;
  State in, out;              // out.ez: Ez plane after the last step of this launch
  const float *ca, *cb;       // [nz][pitch], 0 on the PEC ring, in PEC cells and in the pitch padding
  const float* dbc;           // [nz][pitch] Db = dt / (mu0 mu_r) per cell, or NULL: mu_r = 1 (Geo::Db, Geo::kap)
  float* ez_mid;              // plane for Ez after step 1 of this launch (local shot 0) or NULL: not kept;
  long long ez_mid_stride;    //   the planes after steps 2 .. nsub-1 follow at this stride (floats)
  const float* wavelet;       // sample n of local shot 0
  long long wav_stride;       // nt or 0
  const int2* src_zx;         // [S] (row, column) of the source cell
  const int* blk_start;       // [S][tiles + 1] CSR of receivers by owning tile
  const int2* blk_ent;        // [S][nrec] in CSR order: (row*128 + column inside the tile's region, receiver index)
  const uint2* blk_mask;      // [S][tiles]: bit j = row j of the tile's region holds a receiver of the shot
  float* traces;              // sample n of local shot 0 (NULL: do not record)
  long long trace_stride;     // nt * nrec
  int nrec, nsub;             // receivers per shot; steps in this launch (<= hz)
  int nshots, group;          // shots in this launch; shots swept by one CTA, one after the other
  int tiles_x, tiles_y;
  int hz, oz;                 // halo rows; owned rows per tile (= NW*R - 2*hz)
};

#if defined(__CUDACC__)
// rare path, out of line (code size of the step loop): receivers of a tile beyond its first THREADS
__device__ __noinline__ void fwd_record_overflow(const FwdArgs& a, const float* rowbuf, int threads, int s, int rk0, int rk1, int t)
{
  for (int k = rk0 + threads + threadIdx.x; k < rk1; k += threads) {
    const int2 en2 = a.blk_ent[(long long)s * a.nrec + k];
    a.traces[s * a.trace_stride + (long long)t * a.nrec + en2.y] = rowbuf[en2.x];
  }
}

// The T-step loop of one warp.  All variants hit the same barriers, so the warps of one CTA may run
// different variants.  Every field row of the thread is two packed pairs P = (c0, c2), Q = (c1, c3):
// differences to the right / left neighbour are Q - P resp. P - Q for half the cells and need one
// repacked pair (with the lane shuffle) for the other half.
// MU: the problem has a mu_r model (reading R22) -- Db and Db/dx come per cell from the thread's shared-memory
// slot instead of the two scalars; with mu_r = 1 every product below rounds like the scalar form.
template <int R, int NW, bool ZP, bool XP, bool MU>
__device__ __forceinline__ void fwd_steps(const FwdArgs& a, const TileCtx<R, NW, 3>& c, int s, int rk0, int rk1,
                                          int2 ent, unsigned rflags, int src_r, int src_c, const float (&wv)[kMaxT],
                                          P2 (&e)[R], P2 (&hx)[R], P2 (&hy)[R], const P2 (&ca)[R], const P2 (&cb)[R])
{
  using L = RegTile<R, NW, 3>;
  const Geo& g = a.g;
  const unsigned full = 0xffffffffu;
  const u64 rdx2 = bc2(g.rdx), Db2 = bc2(g.Db), kap2 = bc2(g.kap);
  const long long hoff = s * g.plane + (long long)c.gj0 * g.pitch + c.gi;     // this thread's row 0 in a plane of shot s
  float* const trp = a.traces + (s * a.trace_stride + ent.y);                 // this thread's receiver, sample n
#pragma unroll 1
  for (int t = 0; t < a.nsub; ++t) {
    // ---- stage 1: trace sample n + t from the published receiver rows ----------------------------
    if (ent.x >= 0) trp[(long long)t * a.nrec] = c.rowbuf_()[ent.x];
    if (rk1 - rk0 > L::THREADS) fwd_record_overflow(a, c.rowbuf_(), L::THREADS, s, rk0, rk1, t);   // more receivers than threads

    // ---- stages 2-3: H update + H CPML -------------------------------------------------------------
    // x tables of this lane's columns (XP only; every lane of an XP warp runs the psi form -- lanes off
    // the CPML have the trivial coefficients and a psi of zero; predicating them off costs more in
    // divergent branches than the shared-memory traffic it saves: measured)
    P2 xb = zero2(), xc = zero2(), xk = zero2();
    if (XP) { xb = ld2(c.tabx_() + 0 * kRegW + c.l4); xc = ld2(c.tabx_() + 1 * kRegW + c.l4); xk = ld2(c.tabx_() + 2 * kRegW + c.l4); }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const P2 eb = (r + 1 < R) ? e[r + 1] : ld2(c.xe_() + (c.w + 1) * kRegW + c.l4);     // Ez of the row below
      // Ez to the right of (c1, c3) is (c2, c0 of the next lane); to the right of (c0, c2) it is Q itself
      const u64 enq = pk(hi2(e[r].p), __shfl_down_sync(full, lo2(e[r].p), 1));
      P2 db, kp;                                        // Db and Db/dx of the thread's cells
      if (MU) { db = ld2(c.dbc_(g) + r * kRegW); kp.p = mul2(db.p, rdx2); kp.q = mul2(db.q, rdx2); }
      else { db.p = db.q = Db2; kp.p = kp.q = kap2; }
      if (ZP) {
        P2 p = ld2(c.phz_() + r * kRegW);
        const u64 b = bc2(c.tabz_()[0 * L::ROWS + c.lr0 + r]), cr = bc2(c.tabz_()[1 * L::ROWS + c.lr0 + r]),
                  kk = bc2(c.tabz_()[2 * L::ROWS + c.lr0 + r]);          // Db/(dx kappa); with MU: 1/kappa
        const u64 kkp = MU ? mul2(kp.p, kk) : kk, kkq = MU ? mul2(kp.q, kk) : kk;
        const u64 dp = sub2(eb.p, e[r].p), dq = sub2(eb.q, e[r].q);
        p.p = fma2(b, p.p, mul2(cr, dp)); p.q = fma2(b, p.q, mul2(cr, dq));
        hx[r].p = fma2(neg2(db.p), p.p, fma2(neg2(kkp), dp, hx[r].p)); hx[r].q = fma2(neg2(db.q), p.q, fma2(neg2(kkq), dq, hx[r].q));
        st2(c.phz_() + r * kRegW, p);
      } else {
        hx[r].p = fma2(neg2(kp.p), sub2(eb.p, e[r].p), hx[r].p);
        hx[r].q = fma2(neg2(kp.q), sub2(eb.q, e[r].q), hx[r].q);
      }
      if (XP) {
        P2 p = ld2(c.phx_() + r * kRegW);
        const u64 dp = sub2(e[r].q, e[r].p), dq = sub2(enq, e[r].q);
        const u64 xkp = MU ? mul2(kp.p, xk.p) : xk.p, xkq = MU ? mul2(kp.q, xk.q) : xk.q;
        p.p = fma2(xb.p, p.p, mul2(xc.p, dp)); p.q = fma2(xb.q, p.q, mul2(xc.q, dq));
        hy[r].p = fma2(db.p, p.p, fma2(xkp, dp, hy[r].p)); hy[r].q = fma2(db.q, p.q, fma2(xkq, dq, hy[r].q));
        st2(c.phx_() + r * kRegW, p);
      } else {
        hy[r].p = fma2(kp.p, sub2(e[r].q, e[r].p), hy[r].p);
        hy[r].q = fma2(kp.q, sub2(enq, e[r].q), hy[r].q);
      }
    }
    st2(c.xh_() + (c.w + 1) * kRegW + c.l4, hx[R - 1]);
    __syncthreads();

    // ---- stages 4-7: E update + E CPML, source, save wavefield --------------------------------------
    if (XP) { xb = ld2(c.tabx_() + 3 * kRegW + c.l4); xc = ld2(c.tabx_() + 4 * kRegW + c.l4); xk = ld2(c.tabx_() + 5 * kRegW + c.l4); }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const P2 ha = (r > 0) ? hx[r - 1] : ld2(c.xh_() + c.w * kRegW + c.l4);              // Hx of the row above
      // Hy to the left of (c0, c2) is (c3 of the previous lane, c1); to the left of (c1, c3) it is P itself
      const u64 hlp = pk(__shfl_up_sync(full, hi2(hy[r].q), 1), lo2(hy[r].q));
      const u64 txp = sub2(hy[r].p, hlp), txq = sub2(hy[r].q, hy[r].p);
      const u64 tzp = sub2(hx[r].p, ha.p), tzq = sub2(hx[r].q, ha.q);
      if (ZP || XP) {
        P2 pz = zero2(), px = zero2();
        u64 bz = zf2(), cz = zf2(), kz = zf2();
        if (ZP) {
          pz = ld2(c.pez_() + r * kRegW);
          bz = bc2(c.tabz_()[3 * L::ROWS + c.lr0 + r]); cz = bc2(c.tabz_()[4 * L::ROWS + c.lr0 + r]); kz = bc2(c.tabz_()[5 * L::ROWS + c.lr0 + r]);
          pz.p = fma2(bz, pz.p, mul2(cz, tzp)); pz.q = fma2(bz, pz.q, mul2(cz, tzq));
        }
        if (XP) {
          px = ld2(c.pex_() + r * kRegW);
          px.p = fma2(xb.p, px.p, mul2(xc.p, txp)); px.q = fma2(xb.q, px.q, mul2(xc.q, txq));
        }
        u64 ddp, ddq, ppp, ppq;                         // (tx/kx - tz/kz) and (psix - psiz)
        if (ZP && XP) {
          ddp = sub2(mul2(txp, xk.p), mul2(tzp, kz)); ddq = sub2(mul2(txq, xk.q), mul2(tzq, kz));
          ppp = sub2(px.p, pz.p); ppq = sub2(px.q, pz.q);
        } else if (ZP) {
          ddp = sub2(txp, mul2(tzp, kz)); ddq = sub2(txq, mul2(tzq, kz));
          ppp = neg2(pz.p); ppq = neg2(pz.q);
        } else {
          ddp = sub2(mul2(txp, xk.p), tzp); ddq = sub2(mul2(txq, xk.q), tzq);
          ppp = px.p; ppq = px.q;
        }
        e[r].p = fma2(cb[r].p, fma2(ddp, rdx2, ppp), mul2(ca[r].p, e[r].p));
        e[r].q = fma2(cb[r].q, fma2(ddq, rdx2, ppq), mul2(ca[r].q, e[r].q));
        if (ZP) st2(c.pez_() + r * kRegW, pz);
        if (XP) st2(c.pex_() + r * kRegW, px);
      } else {
        e[r].p = fma2(cb[r].p, mul2(sub2(txp, tzp), rdx2), mul2(ca[r].p, e[r].p));
        e[r].q = fma2(cb[r].q, mul2(sub2(txq, tzq), rdx2), mul2(ca[r].q, e[r].q));
      }
    }
    if (src_r >= 0) {                                   // every CTA whose region holds the source injects
      float wn = wv[0];
#pragma unroll
      for (int k = 1; k < kMaxT; ++k) wn = t == k ? wv[k] : wn;
#pragma unroll
      for (int r = 0; r < R; ++r)
        if (r == src_r) {                               // src_c: 0 -> P.lo, 1 -> Q.lo, 2 -> P.hi, 3 -> Q.hi
          float v[4] = {lo2(e[r].p), lo2(e[r].q), hi2(e[r].p), hi2(e[r].q)};
          const float k4[4] = {lo2(cb[r].p), lo2(cb[r].q), hi2(cb[r].p), hi2(cb[r].q)};
#pragma unroll
          for (int q = 0; q < 4; ++q)
            if (q == src_c) v[q] = FF(-k4[q], wn, v[q]);
          e[r].p = pk(v[0], v[2]); e[r].q = pk(v[1], v[3]);
        }
    }
    const bool last = t + 1 == a.nsub;
    if (last || a.ez_mid) {
      float* dst = (last ? a.out.ez : a.ez_mid + t * a.ez_mid_stride) + hoff;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        if ((c.own >> r) & 1u) st2(dst, e[r]);
        dst += g.pitch;
      }
    }
    if (rflags) {
#pragma unroll
      for (int r = 0; r < R; ++r)
        if ((rflags >> r) & 1u) st2(c.rowbuf_() + (c.lr0 + r) * kRegW + c.l4, e[r]);
    }
    st2(c.xe_() + c.w * kRegW + c.l4, e[0]);
    __syncthreads();
    GPR_FPROBE(s % a.group, 4 + t);
  }
}

// per-shot scalars, word k of kMetaW: receiver range [rk0, rk1) of the tile, source row and column, 4 wavelet
// samples, the 64-bit mask of region rows that hold a receiver.  All of it is static input (nothing a
// previous launch writes), so the whole group's table is loaded once per CTA in the launch prologue.
__device__ __forceinline__ int fwd_meta_word(const FwdArgs& a, int s, int tile, int ntile, int k)
{
  if (k == 0) return a.traces ? a.blk_start[(long long)s * (ntile + 1) + tile] : 0;
  if (k == 1) return a.traces ? a.blk_start[(long long)s * (ntile + 1) + tile + 1] : 0;
  if (k == 2) return a.src_zx[s].x;
  if (k == 3) return a.src_zx[s].y;
  if (k < 8) return (k - 4 < a.nsub) ? __float_as_int(a.wavelet[s * a.wav_stride + (k - 4)]) : 0;
  if (k == 8) return a.traces ? (int)a.blk_mask[(long long)s * ntile + tile].x : 0;
  if (k == 9) return a.traces ? (int)a.blk_mask[(long long)s * ntile + tile].y : 0;
  return 0;
}

// Ez, Hx, Hy of shot s (the whole region) -> the CTA's landing zone [3][ROWS][128], three TMA boxes issued by
// ONE thread and completing on mbarrier 0; cells outside the grid arrive as zeros
template <int R, int NW>
__device__ __forceinline__ void fwd_fetch(const FwdArgs& a, const TileCtx<R, NW, 3>& c, int s)
{
  using L = RegTile<R, NW, 3>;
  const unsigned bar = smem_u32(c.sm + L::MBAR);
  mbar_expect_tx(bar, (unsigned)(3 * L::ROWS * kRegW * sizeof(float)));
#pragma unroll
  for (int f = 0; f < 3; ++f)
    tma_load_3d(smem_u32(c.sm + L::HIST + f * (L::ROWS * kRegW)), &a.tm_reg, c.ri0, c.rj0, a.in_pl[f] + s, bar);
}

template <int R, int NW, int MINB, bool MU>
__global__ void __launch_bounds__(NW * 32, MINB) fwd_kernel(const __grid_constant__ FwdArgs a)
{
  using L = RegTile<R, NW, 3>;
  extern __shared__ __align__(128) float4 smem4[];
  const Geo& g = a.g;
  TileCtx<R, NW, 3> c;
  c.init(reinterpret_cast<float*>(smem4), g, blockIdx.x, blockIdx.y, a.oz, a.hz);
  const int tile = blockIdx.y * a.tiles_x + blockIdx.x, ntile = a.tiles_x * a.tiles_y;
  const int s0 = blockIdx.z * a.group, s1 = min(s0 + a.group, a.nshots);
  const int tid = threadIdx.x;

  // once per CTA, overlapping the previous launch's tail: CPML tables -> shared memory, Ca / Cb of the
  // region -> registers; then, once the previous launch's state is complete, the first shot's fields
  pdl_launch_dependents();
  if (tid == 0) {
    mbar_init(smem_u32(c.sm + L::MBAR), 1u);
    mbar_init_fence();
  }
  for (int k = tid; k < kMetaW * (s1 - s0); k += L::THREADS)
    c.meta_()[k] = fwd_meta_word(a, s0 + k / kMetaW, tile, ntile, k % kMetaW);
  c.template stage_tables<true>(g, MU);
  c.zero_psi(g);
  if (MU) c.load_dbc(g, a.dbc);
  P2 ca[R], cb[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    ca[r] = zero2(); cb[r] = zero2();
    if (c.colin && ((c.rin >> r) & 1u)) {
      const long long o = (long long)(c.gj0 + r) * g.pitch + c.gi;
      ca[r] = ldg2(a.ca + o);
      cb[r] = ldg2(a.cb + o);
    }
  }
  __syncthreads();                     // mbarrier initialised, tables and the group's scalars visible
  pdl_wait();
  if (tid == 0) fwd_fetch<R, NW>(a, c, s0);
  // the receiver this thread records (receivers of the tile are dealt out one per thread)
  int2 ent_next = make_int2(-1, 0);
  if (c.meta_()[0] + tid < c.meta_()[1]) ent_next = a.blk_ent[(long long)s0 * a.nrec + c.meta_()[0] + tid];

#pragma unroll 1
  for (int s = s0; s < s1; ++s) {
    GPR_FPROBE(s - s0, 0);
    const int* m = c.meta_() + (s - s0) * kMetaW;
    const int rk0 = m[0], rk1 = m[1];
    float wv[kMaxT];
#pragma unroll
    for (int t = 0; t < kMaxT; ++t) wv[t] = __int_as_float(m[4 + t]) * (g.rdx * g.rdx);
    const int2 ent = ent_next;
    // the source cell, if this thread holds it
    int src_r = -1, src_c = 0;
    {
      const int dj = m[2] - c.gj0, di = m[3] - c.gi;
      if (dj >= 0 && dj < R && di >= 0 && di < 4) { src_r = dj; src_c = di; }
    }
    // ---- this shot's fields have landed in the thread's slots: move them to registers ---------------
    P2 e[R], hx[R], hy[R];
    c.fetch_psi(g, a.in, s);           // (one cp.async group; the previous shot's psi went out in its store_psi)
    mbar_wait(smem_u32(c.sm + L::MBAR), (unsigned)(s - s0) & 1u);      // this shot's fields have landed
#pragma unroll
    for (int r = 0; r < R; ++r) {      // (cells outside the grid arrived as zeros)
      e[r] = ld2(c.hist_() + 0 * L::ROWS * kRegW + r * kRegW);
      hx[r] = ld2(c.hist_() + 1 * L::ROWS * kRegW + r * kRegW);
      hy[r] = ld2(c.hist_() + 2 * L::ROWS * kRegW + r * kRegW);
    }
    GPR_FPROBE(s - s0, 1);
    // this warp's R bits of the mask of region rows that hold a receiver of this shot
    const unsigned rflags = (unsigned)((((unsigned long long)(unsigned)m[9] << 32) | (unsigned)m[8]) >> c.lr0) & ((1u << R) - 1u);
    // publish: row 0 for the warp above, the receiver rows for the first trace sample
    st2(c.xe_() + c.w * kRegW + c.l4, e[0]);
    if (rflags) {
#pragma unroll
      for (int r = 0; r < R; ++r)
        if ((rflags >> r) & 1u) st2(c.rowbuf_() + (c.lr0 + r) * kRegW + c.l4, e[r]);
    }
    // ---- next shot: the receiver this thread records; its fields into the landing zone once every thread
    // has taken this shot's out of it
    ent_next = make_int2(-1, 0);
    if (s + 1 < s1) {
      const int* mn = m + kMetaW;
      if (mn[0] + tid < mn[1]) ent_next = a.blk_ent[(long long)(s + 1) * a.nrec + mn[0] + tid];
    }
    cp_async_wait<0>();                // psi landed
    GPR_FPROBE(s - s0, 2);
    __syncthreads();                   // exchange row and receiver rows published; landing zone free
    GPR_FPROBE(s - s0, 3);
    if (tid == 0 && s + 1 < s1) fwd_fetch<R, NW>(a, c, s + 1);

#define GPR_FWD_STEPS(ZP_, XP_) \
  fwd_steps<R, NW, ZP_, XP_, MU>(a, c, s, rk0, rk1, ent, rflags, src_r, src_c, wv, e, hx, hy, ca, cb)
    if (c.zp && c.xp) GPR_FWD_STEPS(true, true);
    else if (c.zp) GPR_FWD_STEPS(true, false);
    else if (c.xp) GPR_FWD_STEPS(false, true);
    else GPR_FWD_STEPS(false, false);
#undef GPR_FWD_STEPS

    // ---- write back what this tile owns (out.ez was written by the last E phase) --------------------
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (!((c.own >> r) & 1u)) continue;
      const long long o = s * g.plane + (long long)(c.gj0 + r) * g.pitch + c.gi;
      st2(a.out.hx + o, hx[r]);
      st2(a.out.hy + o, hy[r]);
    }
    if (c.zp || c.xp) c.store_psi(g, a.out, s);
    GPR_FPROBE(s - s0, 8);
  }
}
#endif

}  // namespace gprfwi
