// gprfwi_tile.cuh -- the register tile shared by the forward and adjoint kernels of libgprfwi.
//
// A CTA of NW warps works on a REGION of NW*R rows x 128 columns of one shot: warp w holds rows
// [w*R, w*R + R), lane l holds columns [4l, 4l + 4) of each of them, as float4 REGISTERS for the
// whole launch (up to T = 4 leap-frog steps).  Nothing of the three fields lives in shared memory:
//   x neighbours   come from the adjacent lane by warp shuffle,
//   z neighbours   inside a warp's R rows are the thread's own registers; across warps ONE row per
//                  warp per phase goes through a 512-byte shared-memory exchange slot.
// The region is the owned tile (NW*R - 2*hz rows x 120 columns) plus a halo of hz rows / 4 columns
// that is recomputed redundantly instead of exchanged between CTAs: after t steps the outermost t
// rings of the region are stale (they have seen the garbage beyond the region edge), which is why
// the halo is as deep as the number of fused steps.  State is ping-ponged between launches, so CTAs
// never race.  Cells outside the grid are loaded as 0 and stay 0 by themselves (masked Ca = Cb = 0
// there and on the PEC ring), so no update needs a bounds test.
//
// Shared memory (floats), per CTA:
//   xe   [NW+1][128]  exchange slot A: row 0 of warp w (forward: Ez, adjoint: tz); slot NW stays 0
//   xh   [NW+1][128]  exchange slot B: row R-1 of warp w in slot w+1 (forward: Hx, adjoint: sz); slot 0 stays 0
//   rowbuf [NW*R][128] rows that hold receivers: forward publishes Ez there for the trace gather,
//                     the adjoint stages the residual there for injection
//   tabx [6][128]     CPML x tables of the region's columns: bhx chx khx bex cex kex
//   tabz [6][NW*R]    CPML z tables of the region's rows:    bhz chz khz bez cez kez
//   meta [kMaxGroup][kMetaW] per-shot scalars of the shots of the CTA's group (receiver range, source, wavelet,
//                     mask of the region rows that hold a receiver), loaded once per CTA
//   priv [THREADS][8]  thread-private scalars (adjoint: the thread's residual samples of this launch, its receiver
//                     entry for the next shot)
//   mbar [8]          mbarriers of the TMA copies
//   hist [NH][NW*R][128] landing zone, rows x 128 columns of the region like the registers: adjoint = ring of
//                     forward Ez planes (owned rows) fetched two steps ahead by TMA; forward = Ez, Hx, Hy of the
//                     NEXT shot fetched by cp.async while this one is stepped
//   psi  [4][NW*R][128]  CPML psi of the region, thread-private (only when npml > 0): hz ez hx ex
#pragma once
#include <cuda.h>          // CUtensorMap (type only; the encoder is fetched through the runtime)

#include "gprfwi_common.cuh"

namespace gprfwi {

// Offset (floats) of the thread-private landing / psi arrays from a 128-byte boundary.  Measured on
// config 2 (B200): odd multiples of 4 floats (16 B) give 256-257 Gcell-updates/s, multiples of 8 floats
// (32 B, including the "natural" 128-byte alignment) 248-250 -- the cp.async landing rows and the
// exchange rows then collide in the shared-memory pipe.  28 was the best of 0, 4, ..., 28.
#ifndef GPRFWI_SMEM_PAD
#define GPRFWI_SMEM_PAD 28
#endif
constexpr int kMaxT = 4;       // fused steps per launch <= x halo (4 columns = one float4)
constexpr int kRegW = 128;     // region width  = 32 lanes x float4
constexpr int kOwnW = 120;     // owned width   = lanes 1..30
constexpr int kMaxGroup = 32;  // shots one CTA sweeps at most (size of the per-shot scalar table in shared memory)
constexpr int kMetaW = 12;     // words per shot in that table
// adjoint receiver entries: row*128 + column inside the region, plus a flag when another receiver of the
// region sits on the same cell (then the residual samples are summed atomically)
constexpr int kEntShared = 1 << 30;
constexpr int kEntMask = kEntShared - 1;
#ifndef GPRFWI_ADJ_RING
#define GPRFWI_ADJ_RING 4
#endif
constexpr int kAdjRing = GPRFWI_ADJ_RING;   // slots of the adjoint's ring of forward Ez planes (3: 275.6, 4: 286.3 Gcell-updates/s on config 4)

template <int R, int NW, int NH = 0>
struct RegTile {
  static constexpr int ROWS = R * NW;
  static constexpr int THREADS = NW * 32;
  static constexpr int XE = 0;
  static constexpr int XH = XE + (NW + 1) * kRegW;
  static constexpr int ROWBUF = XH + (NW + 1) * kRegW;
  static constexpr int TABX = ROWBUF + ROWS * kRegW;
  static constexpr int TABZ = TABX + 6 * kRegW;
  static constexpr int META = TABZ + 6 * ROWS;                 // kMaxGroup x kMetaW words: per-shot scalars of the CTA's group
  static constexpr int PRIV = META + kMetaW * kMaxGroup;       // THREADS x 8 words, thread-private (adjoint: residual samples, next receiver)
  static constexpr int MBAR = (PRIV + 8 * THREADS + 1) / 2 * 2;  // 8 mbarriers (8 bytes each) for the TMA copies
  static constexpr int HIST = (MBAR + 16 + 31) / 32 * 32;      // 128-byte aligned: TMA destination
  static constexpr int LAND = HIST + NH * ROWS * kRegW + 32;   // 128-byte aligned: the psi region doubles as a TMA landing zone
  static constexpr int PSI = LAND + GPRFWI_SMEM_PAD;
  // (a problem with a mu_r model appends one more [ROWS][128] array: the per-cell Db of the region, thread-private)
  GPR_HD static size_t smem_bytes(bool pml, bool mu = false)
  {
    return sizeof(float) * (size_t)(PSI + (pml ? 4 * ROWS * kRegW : 0) + (mu ? ROWS * kRegW : 0));
  }
};

#if defined(__CUDACC__)
// exactly rounded, never contracted: every cell's arithmetic is the same whichever CTA computes it
__device__ __forceinline__ float FM(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float FS(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float FA(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float FF(float a, float b, float c) { return __fmaf_rn(a, b, c); }

// ---- packed pairs of fp32 (sm_100: one FFMA2 / FADD2 / FMUL2 does two IEEE-rounded operations in one
// issue slot).  A float4 unit of a row is held as P = (c0, c2), Q = (c1, c3): see gprfwi_common.cuh.
// The pairs are plain float2 values and the operations the sm_100 intrinsics of crt/sm_100_rt.h (explicit
// round-to-nearest per component, never contracted), so that ptxas sees the components: negations fold
// into operand modifiers and scalar operands into the broadcast form instead of costing LOP3 / MOV pairs.
typedef float2 u64;
struct P2 { u64 p, q; };
__device__ __forceinline__ u64 pk(float lo, float hi) { return make_float2(lo, hi); }
__device__ __forceinline__ float lo2(u64 v) { return v.x; }
__device__ __forceinline__ float hi2(u64 v) { return v.y; }
__device__ __forceinline__ u64 bc2(float v) { return make_float2(v, v); }
__device__ __forceinline__ u64 zf2() { return make_float2(0.f, 0.f); }
__device__ __forceinline__ u64 neg2(u64 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ P2 zero2() { P2 v; v.p = zf2(); v.q = zf2(); return v; }
__device__ __forceinline__ P2 mkP2(float4 v) { P2 r; r.p = make_float2(v.x, v.y); r.q = make_float2(v.z, v.w); return r; }
__device__ __forceinline__ float4 f4of(P2 v) { return make_float4(v.p.x, v.p.y, v.q.x, v.q.y); }
__device__ __forceinline__ P2 ldg2(const float* p) { return mkP2(__ldg(reinterpret_cast<const float4*>(p))); }     // read-only global, 128 bit
// global through L2 only (data a previous launch wrote), 128 bit
__device__ __forceinline__ P2 ldcg2(const float* p) { return mkP2(__ldcg(reinterpret_cast<const float4*>(p))); }
__device__ __forceinline__ P2 ld2(const float* p) { return mkP2(*reinterpret_cast<const float4*>(p)); }            // shared / generic, 128 bit
__device__ __forceinline__ void st2(float* p, P2 v) { *reinterpret_cast<float4*>(p) = f4of(v); }
__device__ __forceinline__ void stcs2(float* p, P2 v) { __stcs(reinterpret_cast<float4*>(p), f4of(v)); }

__device__ __forceinline__ void ldg4a(const float* p, float* o)
{
  const float4 v = __ldg(reinterpret_cast<const float4*>(p));
  o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void ldcs4a(const float* p, float* o)      // streaming (evict-first) load
{
  const float4 v = __ldcs(reinterpret_cast<const float4*>(p));
  o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void lds4a(const float* p, float* o)
{
  const float4 v = *reinterpret_cast<const float4*>(p);
  o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void st4a(float* p, const float* v)
{
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void stcs4a(float* p, const float* v)      // streaming (evict-first) store
{
  __stcs(reinterpret_cast<float4*>(p), make_float4(v[0], v[1], v[2], v[3]));
}
// 16-byte asynchronous copy global -> shared (bypasses L1 and the register file)
__device__ __forceinline__ void cp_async16(float* smem, const float* gmem)
{
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
// Programmatic dependent launch: the next launch on the stream may start its prologue (everything that
// does not read the previous launch's output) while this grid drains; pdl_wait() blocks until the
// previous grid has completed and its writes are visible.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void zero4(float* v) { v[0] = v[1] = v[2] = v[3] = 0.f; }

// ---- TMA (cp.async.bulk.tensor) + mbarrier: one elected thread copies a whole [rows][128] box of a field
// plane into shared memory; the copy engine does the addressing, the bounds handling (cells outside the
// grid arrive as zeros) and the transfer, and no thread spends load/store-pipe issue slots on it.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// box of the 3-D tensor (x = column, y = row, z = plane of the workspace) -> shared memory, completing on `bar`
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* map, int x, int y, int z, unsigned bar)
{
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(dst), "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar) : "memory");
}

// Per-thread view of the region: where this lane's 4 columns and this warp's R rows sit in the grid,
// which of them carry CPML psi, and the shared-memory carve-up.
template <int R, int NW, int NH = 0>
struct TileCtx {
  using L = RegTile<R, NW, NH>;
  float* sm;            // shared-memory base; every array is a compile-time offset from it
  int toff;             // lr0 * 128 + l4: this thread's row-0 slot inside a [ROWS][128] array
  int lane, w, l4, lr0;
  int gj0, gi;          // grid row of this warp's row 0, grid column of this lane's component 0
  int rj0, ri0;         // grid row / column of the region's origin
  bool colin;           // the lane's float4 holds at least one grid column: inside [0, roundup4(nx))
  int xslot;            // float offset of this lane's unit in an x-strip row, -1 if it holds no CPML column
  bool xp, zp;          // the CTA's columns / this warp's rows touch the x / z CPML (warp-uniform)
  unsigned zsH, zsE;    // bit r: row gj0 + r carries H- / E-located z psi (warp-uniform)
  unsigned rin;         // bit r: row inside the grid (warp-uniform)
  unsigned own;         // bit r: row owned by this tile (and inside the grid); 0 for lanes 0 and 31

  __device__ __forceinline__ float* xe_() const { return sm + L::XE; }
  __device__ __forceinline__ float* xh_() const { return sm + L::XH; }
  __device__ __forceinline__ float* rowbuf_() const { return sm + L::ROWBUF; }
  __device__ __forceinline__ float* tabx_() const { return sm + L::TABX; }
  __device__ __forceinline__ float* tabz_() const { return sm + L::TABZ; }
  __device__ __forceinline__ int* meta_() const { return reinterpret_cast<int*>(sm + L::META); }
  __device__ __forceinline__ float* priv_() const { return sm + L::PRIV + 8 * threadIdx.x; }
  __device__ __forceinline__ float* hist_() const { return sm + L::HIST + toff; }
  // the forward kernel's thread-private cp.async landing slots: the same region, shifted (see GPRFWI_SMEM_PAD)
  __device__ __forceinline__ float* fland_() const { return sm + L::HIST + GPRFWI_SMEM_PAD + toff; }
  __device__ __forceinline__ float* phz_() const { return sm + L::PSI + 0 * L::ROWS * kRegW + toff; }
  __device__ __forceinline__ float* pez_() const { return sm + L::PSI + 1 * L::ROWS * kRegW + toff; }
  __device__ __forceinline__ float* phx_() const { return sm + L::PSI + 2 * L::ROWS * kRegW + toff; }
  __device__ __forceinline__ float* pex_() const { return sm + L::PSI + 3 * L::ROWS * kRegW + toff; }
  // per-cell Db = dt / (mu0 mu_r) of the thread's cells (only when the problem has a mu_r model)
  __device__ __forceinline__ float* dbc_(const Geo& g) const { return sm + L::PSI + (g.P > 0 ? 4 : 0) * L::ROWS * kRegW + toff; }
  __device__ __forceinline__ void load_dbc(const Geo& g, const float* dbc) const
  {
#pragma unroll
    for (int r = 0; r < R; ++r) {
      P2 v = zero2();
      if (colin && ((rin >> r) & 1u)) v = ldg2(dbc + (long long)(gj0 + r) * g.pitch + gi);
      st2(dbc_(g) + r * kRegW, v);
    }
  }

  __device__ __forceinline__ void init(float* sm_, const Geo& g, int tile_x, int tile_y, int oz, int hz)
  {
    lane = threadIdx.x & 31; w = threadIdx.x >> 5; l4 = lane * 4; lr0 = w * R;
    rj0 = tile_y * oz - hz; ri0 = tile_x * kOwnW - 4;
    gj0 = rj0 + lr0; gi = ri0 + l4;
    sm = sm_; toff = lr0 * kRegW + l4;
    // columns at or beyond roundup4(nx) belong to no tile (lanes 1..30 own columns < 120 * tiles_x only up to
    // the grid edge's unit): nothing ever writes them, so they are never loaded either
    colin = gi >= 0 && gi < ((g.nx + 3) & ~3);
    xslot = (g.P > 0 && colin) ? xstrip_slot(gi >> 2, g.xnl, g.xur, g.pitch) : -1;
    zsH = zsE = rin = own = 0u;
    xp = g.P > 0 && (ri0 < g.P || ri0 + kRegW > g.nx - 1 - g.P);
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int gj = gj0 + r;
      if (gj >= 0 && gj < g.nz) {
        rin |= 1u << r;
        if (g.P > 0 && strip_h(gj, g.nz, g.P) >= 0) zsH |= 1u << r;
        if (g.P > 0 && strip_e(gj, g.nz, g.P) >= 0) zsE |= 1u << r;
        if (lr0 + r >= hz && lr0 + r < L::ROWS - hz && lane >= 1 && lane <= 30 && colin) own |= 1u << r;
      }
    }
    zp = (zsH | zsE) != 0u;
  }

  // CPML tables of the region's rows and columns -> shared memory (outside the grid: b = c = 0, 1/kappa = 1).
  // FWD: (b, c/dx, Db/(dx kappa)) at H nodes and (b, c/dx, 1/kappa) at E nodes; else (b, c, 1/kappa) at both.
  // (FWD with a mu_r model: Db is per cell, so the H sets keep the bare 1/kappa and the kernel multiplies)
  template <bool FWD>
  __device__ __forceinline__ void stage_tables(const Geo& g, bool mu = false) const
  {
    const int r1 = FWD ? 3 : 1, r2h = (FWD && !mu) ? 4 : 2;
    const float k0 = (FWD && !mu) ? g.kap : 1.f;
    if (w == 0) {
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int i = gi + c;
        const bool in = i >= 0 && i < g.nx;
        tabx_()[0 * kRegW + l4 + unit_perm(c)] = in ? g.thx[i] : 0.f;
        tabx_()[1 * kRegW + l4 + unit_perm(c)] = in ? g.thx[r1 * g.nx + i] : 0.f;
        tabx_()[2 * kRegW + l4 + unit_perm(c)] = in ? g.thx[r2h * g.nx + i] : k0;
        tabx_()[3 * kRegW + l4 + unit_perm(c)] = in ? g.tex[i] : 0.f;
        tabx_()[4 * kRegW + l4 + unit_perm(c)] = in ? g.tex[r1 * g.nx + i] : 0.f;
        tabx_()[5 * kRegW + l4 + unit_perm(c)] = in ? g.tex[2 * g.nx + i] : 1.f;
      }
    }
    for (int k = threadIdx.x; k < L::ROWS; k += L::THREADS) {
      const int gj = rj0 + k;
      const bool in = gj >= 0 && gj < g.nz;
      tabz_()[0 * L::ROWS + k] = in ? g.thz[gj] : 0.f;
      tabz_()[1 * L::ROWS + k] = in ? g.thz[r1 * g.nz + gj] : 0.f;
      tabz_()[2 * L::ROWS + k] = in ? g.thz[r2h * g.nz + gj] : k0;
      tabz_()[3 * L::ROWS + k] = in ? g.tez[gj] : 0.f;
      tabz_()[4 * L::ROWS + k] = in ? g.tez[r1 * g.nz + gj] : 0.f;
      tabz_()[5 * L::ROWS + k] = in ? g.tez[2 * g.nz + gj] : 1.f;
    }
    // the two exchange slots nobody publishes: below the last warp, above the first
    if (w == NW - 1) *reinterpret_cast<float4*>(xe_() + NW * kRegW + l4) = make_float4(0.f, 0.f, 0.f, 0.f);
    if (w == 0) *reinterpret_cast<float4*>(xh_() + l4) = make_float4(0.f, 0.f, 0.f, 0.f);
  }

  // once per CTA: all psi slots of this thread to zero (slots that hold no CPML psi stay zero for good:
  // the trivial coefficients keep them there)
  __device__ __forceinline__ void zero_psi(const Geo& g) const
  {
    if (g.P <= 0 || !(zp || xp)) return;
    const float z[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int r = 0; r < R; ++r) {
      st4a(phz_() + r * kRegW, z); st4a(pez_() + r * kRegW, z); st4a(phx_() + r * kRegW, z); st4a(pex_() + r * kRegW, z);
    }
  }

  // psi strips of shot s -> the thread's shared-memory slots, asynchronously (one commit group)
  __device__ __forceinline__ void fetch_psi(const Geo& g, const State& st, int s) const
  {
    if (g.P > 0 && (zp || xp)) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const int gj = gj0 + r;
        const bool in = colin && ((rin >> r) & 1u);
        if (in && ((zsH >> r) & 1u))
          cp_async16(phz_() + r * kRegW, st.phxz + s * g.zstrip + (long long)strip_h(gj, g.nz, g.P) * g.pitch + gi);
        if (in && ((zsE >> r) & 1u))
          cp_async16(pez_() + r * kRegW, st.pezz + s * g.zstrip + (long long)strip_e(gj, g.nz, g.P) * g.pitch + gi);
        if (in && xslot >= 0) {
          const long long po = s * g.xstrip + (long long)gj * g.xw + xslot;
          cp_async16(phx_() + r * kRegW, st.phyx + po);
          cp_async16(pex_() + r * kRegW, st.pezx + po);
        }
      }
    }
    cp_async_commit();
  }

  // owned psi -> the output state
  __device__ __forceinline__ void store_psi(const Geo& g, const State& st, int s) const
  {
    if (g.P <= 0) return;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (!((own >> r) & 1u)) continue;
      const int gj = gj0 + r;
      float v[4];
      if ((zsH >> r) & 1u) { lds4a(phz_() + r * kRegW, v); st4a(st.phxz + s * g.zstrip + (long long)strip_h(gj, g.nz, g.P) * g.pitch + gi, v); }
      if ((zsE >> r) & 1u) { lds4a(pez_() + r * kRegW, v); st4a(st.pezz + s * g.zstrip + (long long)strip_e(gj, g.nz, g.P) * g.pitch + gi, v); }
      if (xslot >= 0) {
        const long long po = s * g.xstrip + (long long)gj * g.xw + xslot;
        lds4a(phx_() + r * kRegW, v); st4a(st.phyx + po, v);
        lds4a(pex_() + r * kRegW, v); st4a(st.pezx + po, v);
      }
    }
  }
};
// Tuning aid (builds with -DGPRFWI_PROBE only): clock64 stamps of every warp of one interior CTA at fixed
// points of each shot, read back with gprfwi_probe_read (gprfwi.cu).  GPRFWI_PROBE=1: adjoint kernel, 2: forward.
#ifdef GPRFWI_PROBE
#ifndef GPRFWI_PROBE_BX
#define GPRFWI_PROBE_BX (gridDim.x / 2)
#define GPRFWI_PROBE_BY (gridDim.y / 2)
#endif
__device__ long long g_probe[kMaxGroup][16][12];
#define GPR_PROBE(shot, k)                                                                          \
  do {                                                                                              \
    if (blockIdx.x == GPRFWI_PROBE_BX && blockIdx.y == GPRFWI_PROBE_BY && blockIdx.z == 0 && (threadIdx.x & 31) == 0) \
      g_probe[(shot)][threadIdx.x >> 5][(k)] = clock64();                                           \
  } while (0)
#else
#define GPR_PROBE(shot, k) do { } while (0)
#endif

// transpose of recording: residual sample n_hi - t enters lamE at the start of reverse step n_hi-1-t;
// it is staged in rowbuf (zero between uses) one barrier ahead of its use.  The receivers of the
// region are dealt out one per thread (its residual samples of the launch sit in the thread's private
// shared-memory slot).
#endif

}  // namespace gprfwi
