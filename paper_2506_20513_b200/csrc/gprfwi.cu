// gprfwi.cu -- host side of libgprfwi: argument checks, memory plan, CPML tables, launch sequences
// and the extern "C" boundary declared in include/gprfwi.h.  sm_100a only; no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "gprfwi.h"
#include "gprfwi_adj_kernel.cuh"
#include "gprfwi_common.cuh"
#include "gprfwi_fwd_kernel.cuh"
#include "gprfwi_misc.cuh"
#include "gprfwi_tile.cuh"
#include "gprfwi_update.cuh"

namespace gprfwi {

static const double kC0 = 299792458.0;
static const double kPi = 3.14159265358979323846;
static const double kMu0 = 4.0e-7 * kPi;
static const double kEps0d = 1.0 / (kMu0 * kC0 * kC0);

static thread_local char g_cuda_err[256] = "no CUDA error recorded";

static int cuda_fail(cudaError_t e, const char* what)
{
  snprintf(g_cuda_err, sizeof(g_cuda_err), "CUDA error in %s: %s", what, cudaGetErrorString(e));
  return GPRFWI_ECUDA;
}
#define GPR_CUDA(call)                                  \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
  } while (0)

// kernel launch (one place, so that every launch is counted the same way)
#ifndef GPR_LAUNCH
#define GPR_LAUNCH(kernel, grid, block, stream, ...) kernel<<<grid, block, 0, stream>>>(__VA_ARGS__)
#endif

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ------------------------------------------------------------------------------------------------
// memory plan
// ------------------------------------------------------------------------------------------------
// Register-tile shapes (rows per thread R, warps per CTA NW, min CTAs per SM): gprfwi_tile.cuh.
// Entry 0 of each table is the default; GPRFWI_FWD_SHAPE / GPRFWI_ADJ_SHAPE pick another (tuning).
struct Shape {
  int R, NW, minb;
  const void *func, *func_mu;                  // the kernel; its variant for problems with a mu_r model
  size_t smem_pml, smem_plain, smem_mu;        // bytes with / without psi slots; extra bytes with a mu_r model
  int rows() const { return R * NW; }
  int threads() const { return NW * 32; }
  size_t smem(bool pml, bool mu = false) const { return (pml ? smem_pml : smem_plain) + (mu ? smem_mu : 0); }
};
#if defined(__CUDACC__)
template <int R, int NW, int MINB>
static Shape fwd_shape()
{
  return {R, NW, MINB, (const void*)fwd_kernel<R, NW, MINB, false>, (const void*)fwd_kernel<R, NW, MINB, true>, RegTile<R, NW, 3>::smem_bytes(true),
          RegTile<R, NW, 3>::smem_bytes(false), RegTile<R, NW, 3>::smem_bytes(false, true) - RegTile<R, NW, 3>::smem_bytes(false)};
}
template <int R, int NW, int MINB>
static Shape adj_shape()
{
  return {R, NW, MINB, (const void*)adj_kernel<R, NW, MINB, false>, (const void*)adj_kernel<R, NW, MINB, true>, RegTile<R, NW, kAdjRing>::smem_bytes(true),
          RegTile<R, NW, kAdjRing>::smem_bytes(false),
          RegTile<R, NW, kAdjRing>::smem_bytes(false, true) - RegTile<R, NW, kAdjRing>::smem_bytes(false)};
}
// (the other shapes exist in tuning builds only, -DGPRFWI_TUNING: they spill and were measured slower)
#ifdef GPRFWI_TUNING
static const Shape kFwdShapes[] = {fwd_shape<3, 12, 1>(), fwd_shape<3, 8, 2>(), fwd_shape<4, 12, 1>(), fwd_shape<2, 16, 1>()};
static const Shape kAdjShapes[] = {adj_shape<3, 12, 1>(), adj_shape<3, 8, 2>(), adj_shape<4, 12, 1>(), adj_shape<2, 16, 1>()};
#else
static const Shape kFwdShapes[] = {fwd_shape<3, 12, 1>()};
static const Shape kAdjShapes[] = {adj_shape<3, 12, 1>()};
#endif
#endif
static int shape_index(const char* env, int count)
{
  const char* e = std::getenv(env);
  const int k = e ? std::atoi(e) : 0;
  return (k >= 0 && k < count) ? k : 0;
}

struct Tiling {
  int oz = 0, tiles_x = 0, tiles_y = 0;   // owned rows per tile; tiles of kOwnW columns x oz rows
  int tiles() const { return tiles_x * tiles_y; }
};

struct Layout {
  // geometry-derived sizes (floats)
  int pitch = 0, xw = 0, xnl = 0, xur = 0;
  size_t plane = 0, zstrip = 0, xstrip = 0;
  size_t hslot = 0;        // Hx, Hy, 4 psi strips of ONE shot
  size_t full = 0;         // hslot + Ez plane
  // a block of S complete states (arrays ez[S] hx[S] hy[S] + strips), padded to whole planes so that every
  // field plane of the workspace sits a whole number of planes from its first byte (the TMA tensor maps
  // address the workspace as ONE array of planes, gprfwi_tile.cuh)
  size_t blk(size_t S) const { return (S * full + plane - 1) / plane * plane; }
  int T = 4;               // time steps fused per launch = halo rows
  Tiling f, a;             // forward / adjoint tilings
  int fv = 0, av = 0;      // kernel shapes in use (indices into kFwdShapes / kAdjShapes)
  // plan
  bool full_history = true;
  int K = 0;               // checkpoint stride (nt when full history)
  int ncheck = 0;          // checkpoints at n = 0, K, 2K, ... (< nt); slot ncheck = state at nt
  int Sb = 0;              // shots per adjoint pass
  int Mtail = 0;           // last Mtail segments: Ez planes stored by the forward pass (no recompute sweep)
  int group = 1, ngroups = 1;      // adjoint: shots per CTA, CTAs per tile
  int fgroup = 1, fngroups = 1;    // forward
  size_t bytes = 0;
};

static int validate(const gprfwi_params* p)
{
  if (!p) return GPRFWI_EINVAL;
  if (p->npml < 0 || p->nz < 2 * p->npml + 3 || p->nx < 2 * p->npml + 3) return GPRFWI_EINVAL;
  if (p->nt <= 0 || p->pitch < p->nx || p->nshots <= 0 || p->nrec < 0) return GPRFWI_EINVAL;
  if (!(p->dx > 0.f) || !(p->dt > 0.f) || p->checkpoint_stride < 0) return GPRFWI_EINVAL;
  if (p->npml > 0 && (p->pml_order < 0 || !(p->pml_kappa_max >= 1.f) || p->pml_sigma_max < 0.f ||
                      p->pml_alpha_max < 0.f))
    return GPRFWI_EINVAL;
  if ((double)p->nz * p->nx > 2.0e9 / 4) return GPRFWI_EINVAL;           // int32 plane offsets
  // Eq. (11), PAPER.md:93 with dx = dy and the vacuum speed of light (tiny fp32 slack)
  if ((double)p->dt > (double)p->dx / (kC0 * std::sqrt(2.0)) * (1.0 + 1e-6)) return GPRFWI_ECFL;
  return GPRFWI_OK;
}

static void base_layout(const gprfwi_params* p, Layout& L)
{
  L.pitch = (int)align_up((size_t)p->nx, 32);
  L.xnl = (p->npml + 3) / 4;                                     // x-strip layout: gprfwi_common.cuh
  L.xur = p->npml > 0 ? (p->nx - 1 - p->npml) / 4 : L.pitch / 4;
  L.xw = 4 * (L.xnl + L.pitch / 4 - L.xur);
  L.plane = (size_t)p->nz * L.pitch;
  L.zstrip = (size_t)2 * p->npml * L.pitch;
  L.xstrip = (size_t)p->nz * L.xw;
  L.hslot = 2 * L.plane + 2 * L.zstrip + 2 * L.xstrip;
  L.full = L.hslot + L.plane;
  // time blocking: GPRFWI_TIME_BLOCK=1..4 (default 4) steps per launch; the z halo is as deep
  L.T = kMaxT;
  if (const char* e = std::getenv("GPRFWI_TIME_BLOCK")) L.T = std::max(1, std::min(kMaxT, std::atoi(e)));
  auto tiling = [&](int rows, Tiling& t) {
    t.oz = rows - 2 * L.T;
    t.tiles_x = (p->nx + kOwnW - 1) / kOwnW;
    t.tiles_y = (p->nz + t.oz - 1) / t.oz;
  };
  L.fv = shape_index("GPRFWI_FWD_SHAPE", (int)(sizeof(kFwdShapes) / sizeof(Shape)));
  L.av = shape_index("GPRFWI_ADJ_SHAPE", (int)(sizeof(kAdjShapes) / sizeof(Shape)));
  tiling(kFwdShapes[L.fv].rows(), L.f);
  tiling(kAdjShapes[L.av].rows(), L.a);
}

// A CTA owns one tile and sweeps a GROUP of shots one after the other (the adjoint keeps their
// gradient sum in registers; per-CTA set-up is paid once per group).  Small grids get small groups
// so that a launch still has a few CTAs per SM slot; once the tiles alone fill the machine `fill`
// times over, the shots are dealt into two or three groups, one per launch lane.
static void pick_groups(int tiles, int shots, int slots, int fill, int& group, int& ngroups)
{
  // Avoid a single group on mid-sized grids: it means a single launch lane, and a lone lane drains
  // before the next launch can start (measured: -20 % on config 4, -30 % on 1024^2 x 32 shots).  Two
  // lanes are enough once one group's launch fills the machine twice over (larger groups amortise the
  // CTA set-up: config 4, 1024^2 and 2048^2 batches measured 1-5 % better with 2 than with 3), three
  // below that (config 3); from about 24 waves per launch the drain no longer matters and splitting
  // the few shots of a pass only costs (4096^2: -3 %, 8192^2: -7 % with two groups).
  const int floor_groups = tiles >= 24 * slots ? 1 : (tiles >= 2 * slots ? 2 : 3);
  const int want = std::max(1, std::min(shots, std::max(floor_groups, (fill * slots + tiles - 1) / tiles)));
  group = std::min((shots + want - 1) / want, kMaxGroup);     // (the kernels keep a per-shot table of kMaxGroup entries)
  ngroups = (shots + group - 1) / group;
}

static int env_int(const char* name, int dflt)
{
  const char* e = std::getenv(name);
  return e ? std::atoi(e) : dflt;
}

// SMs of the current device (queried once; 148 on a B200 and when no device can be asked, e.g. when the
// plan is sized on a host without a GPU)
static int sm_count()
{
  static const int n = [] {
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) {
      cudaGetLastError();
      return 148;
    }
    return v;
  }();
  return n;
}

static void set_groups(const gprfwi_params* p, Layout& L)
{
  const int fslots = sm_count() * std::max(1, kFwdShapes[L.fv].minb), aslots = sm_count() * std::max(1, kAdjShapes[L.av].minb);
  pick_groups(L.f.tiles(), p->nshots, fslots, 2, L.fgroup, L.fngroups);
  pick_groups(L.a.tiles(), L.Sb, aslots, 2, L.group, L.ngroups);
  if (int g = std::min(env_int("GPRFWI_FWD_GROUP", 0), kMaxGroup)) { L.fgroup = std::min(g, p->nshots); L.fngroups = (p->nshots + L.fgroup - 1) / L.fgroup; }
  if (int g = std::min(env_int("GPRFWI_ADJ_GROUP", 0), kMaxGroup)) { L.group = std::min(g, L.Sb); L.ngroups = (L.Sb + L.group - 1) / L.group; }
}

// device pointers carved out of the caller's workspace
struct Carve {
  float *ca = nullptr, *cb = nullptr, *dbc = nullptr, *gca = nullptr, *gcb = nullptr;   // dbc: per-cell Db (mu_r model)
  // static block (one contiguous range, uploaded with one copy): CPML tables, source cells, receiver tables
  char* stat = nullptr;
  size_t stat_bytes = 0;
  float* tables = nullptr;
  int *src_zx = nullptr, *blk_start = nullptr, *blk_ent = nullptr, *blk_mask = nullptr;   // receivers by owning tile (forward tiling)
  int *reg_start = nullptr, *reg_ent = nullptr, *reg_mask = nullptr;   // receivers by region (tile + halo) of the adjoint tiling
  float* hist = nullptr;      // full history: (nt+1) * S planes
  float* ckpt = nullptr;      // (ncheck+1) * S full states
  float* seg = nullptr;       // (K-1) * Sb planes: Ez^{cK+1 .. cK+K-1}
  float* tail = nullptr;      // Mtail * (K-1) * S planes: the same planes of the last Mtail segments, all shots
  float* fscratch = nullptr;  // 2 * S full states (forward ping-pong; reused by the recompute)
  float* lam = nullptr;       // 2 * Sb full states (adjoint ping-pong)
  size_t nplanes = 0;         // planes from ca to the end of the last plane array
};

// One routine both sizes and carves the workspace, so the two can never disagree.
static size_t carve(const gprfwi_params* p, const Layout& L, char* base, Carve* c)
{
  size_t off = 0;
  auto take = [&](size_t bytes) -> char* {
    char* r = base ? base + off : nullptr;
    off += align_up(bytes, 256);
    return r;
  };
  const size_t S = (size_t)p->nshots, R = (size_t)p->nrec, f = sizeof(float);
  const size_t ntile = (size_t)L.f.tiles(), natile = (size_t)L.a.tiles();
  Carve tmp;
  Carve& o = c ? *c : tmp;
  // arrays of field planes start a whole number of planes from the workspace's first byte
  auto take_planes = [&](size_t bytes) -> char* {
    off = align_up(off, L.plane * f);
    char* r = base ? base + off : nullptr;
    off += bytes;
    return r;
  };
  o.ca = (float*)take_planes(L.plane * f);
  o.cb = (float*)take_planes(L.plane * f);
  o.dbc = (float*)take_planes(L.plane * f);
  o.gca = (float*)take_planes((size_t)L.ngroups * L.plane * f);
  o.gcb = (float*)take_planes((size_t)L.ngroups * L.plane * f);
  o.fscratch = (float*)take_planes(2 * L.blk(S) * f);
  o.lam = (float*)take_planes(2 * L.blk(L.Sb) * f);
  if (L.full_history) {
    o.hist = (float*)take_planes((size_t)(p->nt + 1) * S * L.plane * f);
  } else {
    o.ckpt = (float*)take_planes((size_t)(L.ncheck + 1) * L.blk(S) * f);
    o.seg = (float*)take_planes(std::max<size_t>((size_t)(L.K - 1) * L.Sb * L.plane, 1) * f);
    if (L.Mtail > 0) o.tail = (float*)take_planes((size_t)L.Mtail * (L.K - 1) * S * L.plane * f);
  }
  o.nplanes = (off + L.plane * f - 1) / (L.plane * f);
  off = align_up(off, 256);
  const size_t stat0 = off;
  o.tables = (float*)take((size_t)10 * (p->nx + p->nz) * f);
  o.stat = (char*)o.tables;
  o.src_zx = (int*)take(S * 2 * sizeof(int));
  o.blk_start = (int*)take(S * (ntile + 1) * sizeof(int));
  o.blk_ent = (int*)take(std::max<size_t>(S * R, 1) * 2 * sizeof(int));
  o.blk_mask = (int*)take(S * ntile * 2 * sizeof(int));
  o.reg_start = (int*)take((S * natile + 1) * sizeof(int));
  o.reg_ent = (int*)take(std::max<size_t>(6 * S * R, 1) * 2 * sizeof(int));
  o.reg_mask = (int*)take(S * natile * 2 * sizeof(int));
  o.stat_bytes = off - stat0;
  return off;
}

// Chooses full history when it fits (or no budget is given), else the checkpoint stride K and the
// adjoint shot sub-batch Sb that need the least memory for the largest Sb that fits.
static bool make_plan(const gprfwi_params* p, size_t budget, Layout& L)
{
  base_layout(p, L);
  if (p->checkpoint_stride == 0) {
    L.full_history = true;
    L.K = p->nt;
    L.ncheck = 1;
    L.Sb = p->nshots;
    set_groups(p, L);
    L.bytes = carve(p, L, nullptr, nullptr);
    if (budget == 0 || L.bytes <= budget) return true;
  }
  L.full_history = false;
  L.Mtail = 0;
  const int S = p->nshots;
  int prev_sb = -1;
  for (int div = 1; div <= S; ++div) {
    const int sb = (S + div - 1) / div;
    if (sb == prev_sb) continue;
    prev_sb = sb;
    L.Sb = sb;
    set_groups(p, L);
    int candidates[3];
    int nc = 0;
    if (p->checkpoint_stride > 0) {
      candidates[nc++] = std::min(p->checkpoint_stride, p->nt);
    } else {
      const double kopt = std::sqrt((double)p->nt * S * (double)L.full / ((double)sb * (double)L.plane));
      const int k0 = std::max(L.T, std::min(p->nt, (int)std::floor(kopt) / L.T * L.T));   // multiples of T
      candidates[nc++] = k0;
      candidates[nc++] = std::min(p->nt, k0 + L.T);
    }
    size_t best = 0;
    int bestK = 0;
    for (int q = 0; q < nc; ++q) {
      L.K = candidates[q];
      L.ncheck = (p->nt + L.K - 1) / L.K;
      const size_t b = carve(p, L, nullptr, nullptr);
      if (bestK == 0 || b < best) { best = b; bestK = L.K; }
    }
    L.K = bestK;
    L.ncheck = (p->nt + L.K - 1) / L.K;
    L.bytes = best;
    if (budget == 0 || L.bytes <= budget) {
      // Memory the plan leaves unused holds the Ez planes of the LAST segments, written by the forward
      // pass itself: the adjoint meets those segments first and sweeps them without recomputing.
      const size_t per = (size_t)(L.K - 1) * S * L.plane * sizeof(float);
      if (budget > L.bytes && per > 0 && env_int("GPRFWI_TAIL", 1)) {
        L.Mtail = (int)std::min<size_t>((size_t)L.ncheck, (budget - L.bytes) / per);
        while (L.Mtail > 0 && (L.bytes = carve(p, L, nullptr, nullptr)) > budget) --L.Mtail;
        if (L.Mtail == 0) L.bytes = best;
      }
      return true;
    }
  }
  return false;
}

// ------------------------------------------------------------------------------------------------
// CPML 1-D tables (reading R4: Roden-Gedney CPML, CFS stretching, polynomial grading).
// Node position p = i (E-located) or i + 1/2 (H-located); depth into the layer d, rho = d/P:
//   sigma_p = smax rho^m, kappa = 1 + (kmax-1) rho^m, alpha = amax (1 - rho)
//   b = exp(-(sigma_p/kappa + alpha) dt/eps0),  c = sigma_p (b-1) / (kappa (sigma_p + kappa alpha))
// Built in float64, stored as fp32.  Outside the layer b = c = 0, 1/kappa = 1.
// ------------------------------------------------------------------------------------------------
static void build_table(const gprfwi_params* p, int n, bool hloc, float* b, float* c, float* ik)
{
  const int P = p->npml, len = hloc ? n - 1 : n;
  for (int i = 0; i < n; ++i) { b[i] = 0.f; c[i] = 0.f; ik[i] = 1.f; }
  if (P <= 0) return;
  for (int i = 0; i < len; ++i) {
    const double pos = hloc ? i + 0.5 : (double)i;
    const double depth = std::max(std::max((double)P - pos, pos - (double)(n - 1 - P)), 0.0);
    if (depth <= 0.0) continue;
    const double rho = depth / P, rm = std::pow(rho, (double)p->pml_order);
    const double sg = (double)p->pml_sigma_max * rm;
    const double kap = 1.0 + ((double)p->pml_kappa_max - 1.0) * rm;
    const double al = (double)p->pml_alpha_max * (1.0 - rho);
    const double bb = std::exp(-(sg / kap + al) * (double)p->dt / kEps0d);
    const double den = kap * (sg + kap * al);
    b[i] = (float)bb;
    c[i] = den != 0.0 ? (float)(sg * (bb - 1.0) / den) : 0.f;
    ik[i] = (float)(1.0 / kap);
  }
}

}  // namespace gprfwi

using namespace gprfwi;

struct gprfwi_handle {
  gprfwi_params p;
  Layout L;
  Carve c;
  Geo geo;
  const float *eps_r = nullptr, *sigma = nullptr, *wavelet = nullptr;
  bool mu = false;           // the last forward had a mu_r model: the kernels read the per-cell Db plane
  void* workspace = nullptr;
  // Host copy of the static block (CPML tables, source cells, receiver tables) in PINNED memory, laid out
  // like Carve::stat so that one asynchronous copy uploads it; rebuilt only when the geometry, the plan or
  // the workspace changes between forward calls on a reused handle.
  char* stage = nullptr;
  size_t stage_bytes = 0;
  std::vector<int32_t> geo_src, geo_rec;     // the acquisition the block was built for
  const char* stat_on_device = nullptr;      // where it was uploaded to
  // TMA views of the workspace (gprfwi_tile.cuh): box = 128 columns x owned rows / x region rows of a tile
  CUtensorMap tm_adj_own, tm_adj_reg, tm_fwd_reg;
  const void* tm_base = nullptr;             // workspace the maps were encoded for
  bool forward_done = false;
  int64_t launches = 0;
  // Shots are independent, so the launch sequence is issued as `nlanes` interleaved chains on
  // internal streams forked from / joined to the caller's stream: the tail of one chain's launch
  // overlaps the head of another's instead of leaving SMs idle between dependent launches.
  std::vector<cudaStream_t> lanes;
  std::vector<cudaEvent_t> lane_done;
  cudaEvent_t fork = nullptr;
  ~gprfwi_handle()
  {
    for (cudaStream_t q : lanes) cudaStreamDestroy(q);
    for (cudaEvent_t e : lane_done) cudaEventDestroy(e);
    if (fork) cudaEventDestroy(fork);
    if (stage) cudaFreeHost(stage);
  }
  template <class T>
  T* staged(const T* dev) const { return reinterpret_cast<T*>(stage + (reinterpret_cast<const char*>(dev) - c.stat)); }
};

namespace gprfwi {

static State state_at(const Layout& L, float* base, size_t S, size_t shot0)
{
  // a block of S full states laid out array by array: ez[S], hx[S], hy[S], phxz[S], pezz[S], phyx[S], pezx[S]
  State s;
  float* q = base;
  s.ez = q + shot0 * L.plane;   q += S * L.plane;
  s.hx = q + shot0 * L.plane;   q += S * L.plane;
  s.hy = q + shot0 * L.plane;   q += S * L.plane;
  s.phxz = q + shot0 * L.zstrip; q += S * L.zstrip;
  s.pezz = q + shot0 * L.zstrip; q += S * L.zstrip;
  s.phyx = q + shot0 * L.xstrip; q += S * L.xstrip;
  s.pezx = q + shot0 * L.xstrip;
  return s;
}

static int build_geometry(gprfwi_handle* h, const int32_t* src_zx, const int32_t* rec_zx)
{
  const gprfwi_params& p = h->p;
  const Layout& L = h->L;
  const int S = p.nshots, R = p.nrec, ntile = L.f.tiles(), natile = L.a.tiles();
  int* h_src = h->staged(h->c.src_zx);
  int* h_blk_start = h->staged(h->c.blk_start);
  int* h_blk_ent = h->staged(h->c.blk_ent);
  unsigned* h_blk_mask = reinterpret_cast<unsigned*>(h->staged(h->c.blk_mask));
  int* h_reg_start = h->staged(h->c.reg_start);
  int* h_reg_ent = h->staged(h->c.reg_ent);
  unsigned* h_reg_mask = reinterpret_cast<unsigned*>(h->staged(h->c.reg_mask));
  std::fill(h_blk_start, h_blk_start + (size_t)S * (ntile + 1), 0);
  std::fill(h_blk_mask, h_blk_mask + (size_t)S * ntile * 2, 0u);
  std::fill(h_reg_mask, h_reg_mask + (size_t)S * natile * 2, 0u);
  auto ok = [&](int z, int x) { return z >= 1 && z <= p.nz - 2 && x >= 1 && x <= p.nx - 2; };
  // forward: receivers by OWNING tile; entry = (offset inside the tile's region rowbuf, receiver index)
  for (int s = 0; s < S; ++s) {
    const int z = src_zx[2 * s], x = src_zx[2 * s + 1];
    if (!ok(z, x)) return GPRFWI_EGEOM;
    h_src[2 * s] = z;
    h_src[2 * s + 1] = x;
    int* start = h_blk_start + (size_t)s * (ntile + 1);
    std::vector<int> tile_of(R);
    for (int r = 0; r < R; ++r) {
      const int rz = rec_zx[((size_t)s * R + r) * 2], rx = rec_zx[((size_t)s * R + r) * 2 + 1];
      if (!ok(rz, rx)) return GPRFWI_EGEOM;
      tile_of[r] = (rz / L.f.oz) * L.f.tiles_x + rx / kOwnW;
      start[tile_of[r] + 1]++;
    }
    for (int t = 0; t < ntile; ++t) start[t + 1] += start[t];
    std::vector<int> fill(start, start + ntile);
    for (int r = 0; r < R; ++r) {
      const int rz = rec_zx[((size_t)s * R + r) * 2], rx = rec_zx[((size_t)s * R + r) * 2 + 1];
      const int ty = rz / L.f.oz, tx = rx / kOwnW;
      const size_t k = (size_t)s * R + fill[tile_of[r]]++;
      const int row = rz - (ty * L.f.oz - L.T);
      h_blk_ent[2 * k] = row * kRegW + col_pos(rx - (tx * kOwnW - 4));   // internal column order
      h_blk_ent[2 * k + 1] = r;
      h_blk_mask[((size_t)s * ntile + tile_of[r]) * 2 + (row >> 5)] |= 1u << (row & 31);
    }
  }
  // adjoint: receivers by REGION (a receiver within the halo of a tile is injected there too)
  const int arows = kAdjShapes[L.av].rows();
  const size_t cap = (size_t)std::max(6 * S * R, 1);
  size_t nent = 0;
  h_reg_start[0] = 0;
  std::vector<std::vector<int>> bucket(natile);
  for (int s = 0; s < S; ++s) {
    for (auto& b : bucket) b.clear();
    for (int r = 0; r < R; ++r) {
      const int rz = rec_zx[((size_t)s * R + r) * 2], rx = rec_zx[((size_t)s * R + r) * 2 + 1];
      // tiles ty with ty*oz - T <= rz < ty*oz - T + arows, tx with tx*120 - 4 <= rx < tx*120 + 124
      const int ty_lo = std::max(0, (rz + L.T - arows) / L.a.oz + ((rz + L.T - arows) >= 0 ? 1 : 0));
      const int ty_hi = std::min(L.a.tiles_y - 1, (rz + L.T) / L.a.oz);
      const int tx_lo = std::max(0, (rx + 4 - kRegW) / kOwnW + ((rx + 4 - kRegW) >= 0 ? 1 : 0));
      const int tx_hi = std::min(L.a.tiles_x - 1, (rx + 4) / kOwnW);
      for (int ty = ty_lo; ty <= ty_hi; ++ty)
        for (int tx = tx_lo; tx <= tx_hi; ++tx) bucket[(size_t)ty * L.a.tiles_x + tx].push_back(r);
    }
    for (int t = 0; t < natile; ++t) {
      const int ty = t / L.a.tiles_x, tx = t % L.a.tiles_x;
      for (int r : bucket[t]) {
        const int rz = rec_zx[((size_t)s * R + r) * 2], rx = rec_zx[((size_t)s * R + r) * 2 + 1];
        if (nent >= cap) return GPRFWI_EINVAL;
        const int row = rz - (ty * L.a.oz - L.T);
        h_reg_ent[2 * nent] = row * kRegW + col_pos(rx - (tx * kOwnW - 4));
        h_reg_ent[2 * nent + 1] = r;
        h_reg_mask[((size_t)s * natile + t) * 2 + (row >> 5)] |= 1u << (row & 31);
        ++nent;
      }
      // receivers of this region that share their cell: flag them (summed atomically by the kernel)
      {
        const size_t lo = (size_t)h_reg_start[(size_t)s * natile + t];
        if (nent - lo > 1) {
          std::vector<int> cells;
          for (size_t k = lo; k < nent; ++k) cells.push_back(h_reg_ent[2 * k]);
          std::sort(cells.begin(), cells.end());
          for (size_t k = lo; k < nent; ++k) {
            const auto r2 = std::equal_range(cells.begin(), cells.end(), h_reg_ent[2 * k]);
            if (r2.second - r2.first > 1) h_reg_ent[2 * k] |= kEntShared;
          }
        }
      }
      h_reg_start[(size_t)s * natile + t + 1] = (int)nent;
    }
  }
  return GPRFWI_OK;
}

static void fill_geo(gprfwi_handle* h)
{
  const gprfwi_params& p = h->p;
  const Layout& L = h->L;
  Geo& g = h->geo;
  g.nz = p.nz; g.nx = p.nx; g.P = p.npml; g.pitch = L.pitch; g.xw = L.xw; g.xnl = L.xnl; g.xur = L.xur;
  g.plane = (long long)L.plane; g.zstrip = (long long)L.zstrip; g.xstrip = (long long)L.xstrip;
  g.rdx = (float)(1.0 / (double)p.dx);
  g.Db = (float)((double)p.dt / kMu0);
  g.kap = g.Db * g.rdx;                                   // exactly what the kernels compute
  g.tex = h->c.tables;       g.tez = g.tex + 5 * p.nx;
  g.thx = g.tez + 5 * p.nz;  g.thz = g.thx + 5 * p.nx;
}

// CPML tables + geometry -> the pinned host copy of the static block -> one asynchronous upload.  Skipped
// when the handle already uploaded the same acquisition to the same place (handle reuse in an inversion
// loop: the caller must then leave the workspace alone between calls, see include/gprfwi.h).
static int upload_static(gprfwi_handle* h, const int32_t* src_zx, const int32_t* rec_zx, bool same_plan, cudaStream_t st)
{
  const gprfwi_params& p = h->p;
  fill_geo(h);
  const size_t ns = (size_t)p.nshots * 2, nr = (size_t)p.nshots * p.nrec * 2;
  if (same_plan && h->stage && h->stat_on_device == h->c.stat && h->geo_src.size() == ns && h->geo_rec.size() == nr &&
      std::memcmp(h->geo_src.data(), src_zx, ns * sizeof(int32_t)) == 0 &&
      (nr == 0 || std::memcmp(h->geo_rec.data(), rec_zx, nr * sizeof(int32_t)) == 0))
    return GPRFWI_OK;
  h->stat_on_device = nullptr;
  if (h->stage_bytes < h->c.stat_bytes) {
    if (h->stage) cudaFreeHost(h->stage);
    h->stage = nullptr;
    h->stage_bytes = 0;
    GPR_CUDA(cudaMallocHost((void**)&h->stage, h->c.stat_bytes));
    h->stage_bytes = h->c.stat_bytes;
  }
  // four sets of [5][len]: ex[nx] ez[nz] hx[nx] hz[nz]; rows b, c, 1/kappa, c/dx, Db/(dx kappa)
  float* t = h->staged(h->c.tables);
  const float kap_f = h->geo.kap;
  auto fill = [&](float* set, int len, bool hloc) {
    build_table(&p, len, hloc, set, set + len, set + 2 * len);
    for (int i = 0; i < len; ++i) {
      set[3 * len + i] = (float)((double)set[len + i] / (double)p.dx);
      set[4 * len + i] = kap_f * set[2 * len + i];
    }
  };
  float* ex = t;             float* ez = ex + 5 * p.nx;
  float* hx = ez + 5 * p.nz; float* hz = hx + 5 * p.nx;
  fill(ex, p.nx, false); fill(ez, p.nz, false); fill(hx, p.nx, true); fill(hz, p.nz, true);
  if (int rc = build_geometry(h, src_zx, rec_zx)) return rc;
  GPR_CUDA(cudaMemcpyAsync(h->c.stat, h->stage, h->c.stat_bytes, cudaMemcpyHostToDevice, st));
  h->geo_src.assign(src_zx, src_zx + ns);
  h->geo_rec.assign(rec_zx, rec_zx + nr);
  h->stat_on_device = h->c.stat;
  return GPRFWI_OK;
}

// The workspace from its first byte (Ca) as a 3-D fp32 tensor [nplanes][nz][roundup4(nx)] with row pitch
// L.pitch: every field plane the kernels touch is one z-slice of it (carve() keeps them plane-aligned).
// cuTensorMapEncodeTiled is a driver entry point; it is fetched through the runtime, so the library links
// against cudart only.
static int encode_map(CUtensorMap* map, const gprfwi_handle* h, int box_rows)
{
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn fn = nullptr;
  if (!fn) {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult q;
    GPR_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q));
    if (!sym || q != cudaDriverEntryPointSuccess) return cuda_fail(cudaErrorNotSupported, "cuTensorMapEncodeTiled lookup");
    fn = (encode_fn)sym;
  }
  const Layout& L = h->L;
  const cuuint64_t dims[3] = {(cuuint64_t)((h->p.nx + 3) & ~3), (cuuint64_t)h->p.nz, (cuuint64_t)h->c.nplanes};
  const cuuint64_t strides[2] = {(cuuint64_t)L.pitch * sizeof(float), (cuuint64_t)L.plane * sizeof(float)};
  const cuuint32_t box[3] = {(cuuint32_t)kRegW, (cuuint32_t)box_rows, 1u};
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)h->c.ca, dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return GPRFWI_ECUDA;
  }
  return GPRFWI_OK;
}

static int maps_init(gprfwi_handle* h, bool same_plan)
{
  if (same_plan && h->tm_base == (const void*)h->c.ca) return GPRFWI_OK;
  h->tm_base = nullptr;
  if (int rc = encode_map(&h->tm_adj_own, h, h->L.a.oz)) return rc;
  if (int rc = encode_map(&h->tm_adj_reg, h, kAdjShapes[h->L.av].rows())) return rc;
  if (int rc = encode_map(&h->tm_fwd_reg, h, kFwdShapes[h->L.fv].rows())) return rc;
  h->tm_base = (const void*)h->c.ca;
  return GPRFWI_OK;
}

// The limit on dynamic shared memory is an attribute of the KERNEL (per device), not of a handle: it is set to
// the largest request any problem can make (CPML psi slots, and for the mu_r variants the per-cell Db slots), so
// that live handles with and without a CPML never lower it under one another.
static int kernels_init(const gprfwi_params*, const Layout& L)
{
  GPR_CUDA(cudaFuncSetAttribute(kFwdShapes[L.fv].func, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kFwdShapes[L.fv].smem(true)));
  GPR_CUDA(cudaFuncSetAttribute(kAdjShapes[L.av].func, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kAdjShapes[L.av].smem(true)));
  GPR_CUDA(cudaFuncSetAttribute(kFwdShapes[L.fv].func_mu, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kFwdShapes[L.fv].smem(true, true)));
  GPR_CUDA(cudaFuncSetAttribute(kAdjShapes[L.av].func_mu, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kAdjShapes[L.av].smem(true, true)));
  return GPRFWI_OK;
}

// every tile-kernel launch allows programmatic dependent launch (the kernels call griddepcontrol.wait
// before they read the previous launch's output)
static int launch_pdl(const Shape& sh, dim3 grid, void* arg, bool pml, bool mu, cudaStream_t st)
{
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(sh.threads());
  cfg.dynamicSmemBytes = sh.smem(pml, mu);
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = env_int("GPRFWI_PDL", 1) ? 1 : 0;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  void* args[] = {arg};
  GPR_CUDA(cudaLaunchKernelExC(&cfg, mu ? sh.func_mu : sh.func, args));
  return GPRFWI_OK;
}

static int lanes_init(gprfwi_handle* h)
{
  if (!h->lanes.empty()) return GPRFWI_OK;
  const int n = std::max(1, std::min(8, env_int("GPRFWI_LANES", 3)));
  GPR_CUDA(cudaEventCreateWithFlags(&h->fork, cudaEventDisableTiming));
  for (int k = 0; k < n; ++k) {
    cudaStream_t q; cudaEvent_t e;
    GPR_CUDA(cudaStreamCreateWithFlags(&q, cudaStreamNonBlocking));
    GPR_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    h->lanes.push_back(q); h->lane_done.push_back(e);
  }
  return GPRFWI_OK;
}
// shots [0, ns) split into at most `lanes` contiguous chunks whose sizes are multiples of `quantum`
static std::vector<int> lane_bounds(int ns, int lanes, int quantum)
{
  const int units = (ns + quantum - 1) / quantum, nl = std::max(1, std::min(lanes, units));
  std::vector<int> b(nl + 1, 0);
  for (int k = 1; k <= nl; ++k) b[k] = std::min(ns, (int)((long long)units * k / nl) * quantum);
  return b;
}
static int lanes_fork(gprfwi_handle* h, cudaStream_t st, int nl)
{
  GPR_CUDA(cudaEventRecord(h->fork, st));
  for (int k = 0; k < nl; ++k) GPR_CUDA(cudaStreamWaitEvent(h->lanes[k], h->fork, 0));
  return GPRFWI_OK;
}
static int lanes_join(gprfwi_handle* h, cudaStream_t st, int nl)
{
  for (int k = 0; k < nl; ++k) {
    GPR_CUDA(cudaEventRecord(h->lane_done[k], h->lanes[k]));
    GPR_CUDA(cudaStreamWaitEvent(st, h->lane_done[k], 0));
  }
  return GPRFWI_OK;
}

// Forward block: steps n .. n+nsub-1 for `ns` shots from global shot `shot0`.  ez_of(m) gives the
// plane that must receive Ez^m (local shot 0) or NULL; in.ez / out.ez are already set by the caller.
template <class EzOf>
static int launch_fwd_block(gprfwi_handle* h, cudaStream_t st, int n, int nsub, int shot0, int ns,
                            const State& in, const State& out, float* traces, EzOf ez_of)
{
  const gprfwi_params& p = h->p;
  const Layout& L = h->L;
  FwdArgs a;
  a.g = h->geo;
  a.in = in;
  a.out = out;
  a.ca = h->c.ca;
  a.cb = h->c.cb;
  a.dbc = h->mu ? h->c.dbc : nullptr;
  a.tm_reg = h->tm_fwd_reg;
  a.in_pl[0] = (int)((in.ez - h->c.ca) / (long long)L.plane);
  a.in_pl[1] = (int)((in.hx - h->c.ca) / (long long)L.plane);
  a.in_pl[2] = (int)((in.hy - h->c.ca) / (long long)L.plane);
  // planes for Ez after steps 1 .. nsub-1 of this launch: consecutive at a fixed stride in every plan
  a.ez_mid = nsub > 1 ? ez_of(n + 1) : nullptr;
  a.ez_mid_stride = (a.ez_mid && nsub > 2) ? (long long)(ez_of(n + 2) - ez_of(n + 1)) : 0;
  a.wav_stride = p.wavelet_per_shot ? p.nt : 0;
  a.wavelet = h->wavelet + n + (size_t)shot0 * a.wav_stride;
  a.src_zx = reinterpret_cast<const int2*>(h->c.src_zx) + shot0;
  a.blk_start = h->c.blk_start + (size_t)shot0 * (L.f.tiles() + 1);
  a.blk_ent = reinterpret_cast<const int2*>(h->c.blk_ent) + (size_t)shot0 * p.nrec;
  a.blk_mask = reinterpret_cast<const uint2*>(h->c.blk_mask) + (size_t)shot0 * L.f.tiles();
  a.trace_stride = (long long)p.nt * p.nrec;
  a.traces = (traces && p.nrec > 0) ? traces + (size_t)shot0 * a.trace_stride + (size_t)n * p.nrec : nullptr;
  a.nrec = p.nrec;
  a.nsub = nsub;
  a.nshots = ns;
  a.group = L.fgroup;
  a.tiles_x = L.f.tiles_x;
  a.tiles_y = L.f.tiles_y;
  a.hz = L.T;
  a.oz = L.f.oz;
  const Shape& sh = kFwdShapes[L.fv];
  dim3 grid(L.f.tiles_x, L.f.tiles_y, (ns + L.fgroup - 1) / L.fgroup);
  if (int rc = launch_pdl(sh, grid, &a, p.npml > 0, h->mu, st)) return rc;
  h->launches++;
  return GPRFWI_OK;
}

// Adjoint block: reverse steps n_hi-1 .. n_hi-nsub for `ns` shots from global shot `shot0`.
template <class EzOf>
static int launch_adj_block(gprfwi_handle* h, cudaStream_t st, int n_hi, int nsub, int shot0, int ns, int grp0,
                            const State& in, const State& out, const float* residual, EzOf ez_of)
{
  const gprfwi_params& p = h->p;
  const Layout& L = h->L;
  const long long tstride = (long long)p.nt * p.nrec;
  const int ngrp = (ns + L.group - 1) / L.group;
  AdjArgs a;
  a.g = h->geo;
  a.in = in;
  a.out = out;
  a.ca = h->c.ca;
  a.cb = h->c.cb;
  a.dbc = h->mu ? h->c.dbc : nullptr;
  auto plane_index = [&](const float* q) { return (int)((q - h->c.ca) / (long long)L.plane); };
  a.tm_own = h->tm_adj_own;
  a.tm_reg = h->tm_adj_reg;
  for (int t = 0; t <= kMaxT; ++t) a.ez_pl[t] = t <= nsub ? plane_index(ez_of(n_hi - t)) : 0;
  a.in_pl[0] = plane_index(in.ez); a.in_pl[1] = plane_index(in.hx); a.in_pl[2] = plane_index(in.hy);
  a.gca = h->c.gca + (size_t)grp0 * L.plane;        // this launch's groups start at plane pair grp0
  a.gcb = h->c.gcb + (size_t)grp0 * L.plane;
  a.trace_stride = tstride;
  a.residual = residual ? residual + (size_t)shot0 * tstride + (long long)n_hi * p.nrec : nullptr;
  a.reg_start = h->c.reg_start;
  a.reg_ent = reinterpret_cast<const int2*>(h->c.reg_ent);
  a.reg_mask = reinterpret_cast<const uint2*>(h->c.reg_mask);
  a.nrec = p.nrec;
  a.nsub = nsub;
  a.n_hi = n_hi;
  a.nt = p.nt;
  a.nshots = ns;
  a.group = L.group;
  a.tiles_x = L.a.tiles_x;
  a.tiles_y = L.a.tiles_y;
  a.hz = L.T;
  a.oz = L.a.oz;
  a.shot_base = shot0;
  const Shape& sh = kAdjShapes[L.av];
  dim3 grid(L.a.tiles_x, L.a.tiles_y, ngrp);
  if (int rc = launch_pdl(sh, grid, &a, p.npml > 0, h->mu, st)) return rc;
  h->launches++;
  return GPRFWI_OK;
}

}  // namespace gprfwi

// ------------------------------------------------------------------------------------------------
// extern "C" boundary (include/gprfwi.h)
// ------------------------------------------------------------------------------------------------
extern "C" {

int gprfwi_version(void) { return 100; }

const char* gprfwi_strerror(int code)
{
  switch (code) {
    case GPRFWI_OK: return "ok";
    case GPRFWI_EINVAL: return "invalid argument";
    case GPRFWI_ECFL: return "time step violates the CFL condition (Eq. 11)";
    case GPRFWI_EGEOM: return "source or receiver outside [1, n-2]";
    case GPRFWI_ENOMEM: return "workspace too small";
    case GPRFWI_ESTATE: return "adjoint called without a completed forward";
    case GPRFWI_ECUDA: return g_cuda_err;
    case GPRFWI_ETOOBIG: return "problem exceeds the fixed scratch of gprfwi_update_noalloc (7 planes of 2^20 cells): use gprfwi_update with a caller workspace";
    default: return "unknown gprfwi status";
  }
}

size_t gprfwi_workspace_bytes(const gprfwi_params* p, size_t budget_bytes, gprfwi_plan* plan)
{
  if (validate(p) != GPRFWI_OK) return 0;
  Layout L;
  if (!make_plan(p, budget_bytes, L)) return 0;
  if (plan) {
    plan->workspace_bytes = L.bytes;
    plan->full_history = L.full_history ? 1 : 0;
    plan->checkpoint_stride = L.K;
    plan->shots_per_pass = L.Sb;
    plan->time_block = L.T;
    plan->stored_segments = L.full_history ? 1 : L.Mtail;
    plan->reserved = 0;
  }
  return L.bytes;
}

int gprfwi_get_plan(const gprfwi_handle* h, gprfwi_plan* plan)
{
  if (!h || !plan) return GPRFWI_EINVAL;
  plan->workspace_bytes = h->L.bytes;
  plan->full_history = h->L.full_history ? 1 : 0;
  plan->checkpoint_stride = h->L.K;
  plan->shots_per_pass = h->L.Sb;
  plan->time_block = h->L.T;
  plan->stored_segments = h->L.full_history ? 1 : h->L.Mtail;
  plan->reserved = 0;
  return GPRFWI_OK;
}

int64_t gprfwi_launch_count(const gprfwi_handle* h) { return h ? h->launches : 0; }

#ifdef GPRFWI_PROBE
// tuning builds only: copy the adjoint kernel's clock stamps (gprfwi_adj_kernel.cuh) to the host
int gprfwi_probe_read(long long* out, size_t bytes)
{
  GPR_CUDA(cudaDeviceSynchronize());
  GPR_CUDA(cudaMemcpyFromSymbol(out, g_probe, std::min(bytes, sizeof(g_probe))));
  return GPRFWI_OK;
}
#endif

void gprfwi_release(gprfwi_handle* h) { delete h; }

int gprfwi_forward(gprfwi_handle** hp, const gprfwi_params* p, const float* eps_r, const float* sigma,
                   const float* wavelet, const int32_t* src_zx, const int32_t* rec_zx, void* workspace,
                   size_t workspace_bytes, float* traces, void* cuda_stream)
{
  return gprfwi_forward_mu(hp, p, eps_r, sigma, nullptr, wavelet, src_zx, rec_zx, workspace, workspace_bytes, traces,
                           cuda_stream);
}

int gprfwi_forward_mu(gprfwi_handle** hp, const gprfwi_params* p, const float* eps_r, const float* sigma,
                      const float* mu_r, const float* wavelet, const int32_t* src_zx, const int32_t* rec_zx,
                      void* workspace, size_t workspace_bytes, float* traces, void* cuda_stream)
{
  int rc = validate(p);
  if (rc != GPRFWI_OK) return rc;
  if (!hp || !eps_r || !sigma || !wavelet || !src_zx || !workspace || (p->nrec > 0 && (!rec_zx || !traces)))
    return GPRFWI_EINVAL;
  if ((uintptr_t)workspace % 256 != 0) return GPRFWI_EINVAL;
  Layout L;
  if (!make_plan(p, workspace_bytes, L)) return GPRFWI_ENOMEM;
  gprfwi_handle* h = *hp;
  const bool fresh = (h == nullptr);
  if (fresh) {
    h = new (std::nothrow) gprfwi_handle();
    if (!h) return GPRFWI_ENOMEM;
  } else if (std::memcmp(&h->p, p, sizeof(*p)) != 0) {
    return GPRFWI_EINVAL;
  }
  const bool same_plan = !fresh && h->workspace == workspace && h->L.bytes == L.bytes && h->L.K == L.K &&
                         h->L.Sb == L.Sb && h->L.Mtail == L.Mtail && h->L.full_history == L.full_history &&
                         h->L.group == L.group && h->L.fgroup == L.fgroup && h->L.T == L.T && h->L.fv == L.fv &&
                         h->L.av == L.av;
  h->p = *p;
  h->L = L;
  h->eps_r = eps_r; h->sigma = sigma; h->wavelet = wavelet; h->workspace = workspace;
  h->mu = mu_r != nullptr;
  h->forward_done = false;
  h->launches = 0;
  carve(p, L, (char*)workspace, &h->c);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  rc = upload_static(h, src_zx, rec_zx, same_plan, st);
  if (rc == GPRFWI_OK) rc = maps_init(h, same_plan);
  if (rc != GPRFWI_OK) { if (fresh) delete h; else h->stat_on_device = nullptr; return rc; }
  *hp = h;

  const size_t S = p->nshots, f = sizeof(float);
  // kernel a: Ca/Cb once per call, shared by all shots
  {
    dim3 grid((L.pitch + 127) / 128, p->nz), block(128);
    GPR_LAUNCH(coef_kernel, grid, block, st, eps_r, sigma, mu_r, p->pitch, p->nz, p->nx, L.pitch,
                                        (float)(1.0 / (double)p->dt), h->geo.Db, h->c.ca, h->c.cb, h->c.dbc);
    h->launches++;
  }
  // fields are zero at n = 0
  GPR_CUDA(cudaMemsetAsync(h->c.fscratch, 0, 2 * L.blk(S) * f, st));
  float* slot[2] = {h->c.fscratch, h->c.fscratch + L.blk(S)};
  if (!same_plan) rc = kernels_init(p, L);       // (function attributes: once per handle and plan)
  if (rc != GPRFWI_OK) return rc;
  if (L.full_history) GPR_CUDA(cudaMemsetAsync(h->c.hist, 0, S * L.plane * f, st));
  else GPR_CUDA(cudaMemsetAsync(h->c.ckpt, 0, L.blk(S) * f, st));       // checkpoint 0 = zero state
  // blocks of up to T steps that never cross a checkpoint boundary, issued lane by lane
  rc = lanes_init(h);
  if (rc != GPRFWI_OK) return rc;
  const std::vector<int> lb = lane_bounds((int)S, (int)h->lanes.size(), L.fgroup);
  const int nl = (int)lb.size() - 1;
  rc = lanes_fork(h, st, nl);
  if (rc != GPRFWI_OK) return rc;
  int idx = 0;
  for (int n = 0; n < p->nt; ++idx) {
    const int bound = L.full_history ? p->nt : std::min((n / L.K + 1) * L.K, p->nt);
    const int nsub = std::min(L.T, bound - n), m = n + nsub;
    for (int k = 0; k < nl && rc == GPRFWI_OK; ++k) {
      const int sh0 = lb[k], ns = lb[k + 1] - lb[k];
      if (L.full_history) {
        State in = state_at(L, slot[idx & 1], S, sh0), out = state_at(L, slot[(idx + 1) & 1], S, sh0);
        in.ez = h->c.hist + ((size_t)n * S + sh0) * L.plane;
        out.ez = h->c.hist + ((size_t)m * S + sh0) * L.plane;
        rc = launch_fwd_block(h, h->lanes[k], n, nsub, sh0, ns, in, out, traces,
                              [&](int q) { return h->c.hist + ((size_t)q * S + sh0) * L.plane; });
      } else {
        float* src = (n % L.K == 0) ? h->c.ckpt + (size_t)(n / L.K) * L.blk(S) : slot[idx & 1];
        float* dst = (m == p->nt) ? h->c.ckpt + (size_t)L.ncheck * L.blk(S)
                   : (m % L.K == 0) ? h->c.ckpt + (size_t)(m / L.K) * L.blk(S) : slot[(idx + 1) & 1];
        State in = state_at(L, src, S, sh0), out = state_at(L, dst, S, sh0);
        const int c = n / L.K, c0 = L.ncheck - L.Mtail;
        if (c >= c0) {
          // a stored segment: Ez^{n0+1 .. n1-1} go to (and are stepped from) the tail planes, as in the
          // recompute sweep; Ez^{n0} and Ez^{n1} are the checkpoints' own planes
          const int n0 = c * L.K, n1 = std::min(n0 + L.K, p->nt);
          auto plane = [=](int q) { return h->c.tail + (((size_t)(c - c0) * (L.K - 1) + (q - n0 - 1)) * S + sh0) * L.plane; };
          if (n != n0) in.ez = plane(n);
          if (m != n1) out.ez = plane(m);
          rc = launch_fwd_block(h, h->lanes[k], n, nsub, sh0, ns, in, out, traces, plane);
        } else {
          rc = launch_fwd_block(h, h->lanes[k], n, nsub, sh0, ns, in, out, traces, [](int) -> float* { return nullptr; });
        }
      }
    }
    if (rc != GPRFWI_OK) return rc;
    n = m;
  }
  rc = lanes_join(h, st, nl);
  if (rc != GPRFWI_OK) return rc;
  GPR_CUDA(cudaGetLastError());
  h->forward_done = true;
  return GPRFWI_OK;
}

int gprfwi_adjoint(gprfwi_handle* h, const float* residual, float* grad_eps_r, float* grad_sigma,
                   void* cuda_stream)
{
  if (!h || !grad_eps_r || !grad_sigma || (h->p.nrec > 0 && !residual)) return GPRFWI_EINVAL;
  if (!h->forward_done) return GPRFWI_ESTATE;
  const gprfwi_params* p = &h->p;
  const Layout& L = h->L;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t S = p->nshots, f = sizeof(float);
  GPR_CUDA(cudaMemsetAsync(h->c.gca, 0, (size_t)L.ngroups * L.plane * f, st));
  GPR_CUDA(cudaMemsetAsync(h->c.gcb, 0, (size_t)L.ngroups * L.plane * f, st));
  float* lam[2] = {h->c.lam, h->c.lam + L.blk(L.Sb)};
  float* rs[2] = {h->c.fscratch, h->c.fscratch + L.blk(S)};     // recompute ping-pong

  int rc = lanes_init(h);
  if (rc != GPRFWI_OK) return rc;
  for (int shot0 = 0; shot0 < (int)S; shot0 += L.Sb) {
    const int ns = std::min(L.Sb, (int)S - shot0);
    // lambda = 0 at the end time, Eq. (10)
    GPR_CUDA(cudaMemsetAsync(h->c.lam, 0, 2 * L.blk(L.Sb) * f, st));
    // the shots of this pass go down `nl` interleaved lanes (chunks are whole CTA groups)
    const std::vector<int> lb = lane_bounds(ns, (int)h->lanes.size(), L.group);
    const int nl = (int)lb.size() - 1;
    rc = lanes_fork(h, st, nl);
    if (rc != GPRFWI_OK) return rc;
    int flip = 0;
    const int nseg = L.full_history ? 1 : L.ncheck;
    for (int c = nseg - 1; c >= 0; --c) {
      const int n0 = L.full_history ? 0 : c * L.K;
      const int n1 = L.full_history ? p->nt : std::min(n0 + L.K, p->nt);
      // forward Ez plane of step m for the first shot (pass-local l0) of a lane
      auto ez_plane_of = [&, c, n0, n1](int l0) {
        return [=](int m) -> float* {
          const int g0 = shot0 + l0;
          if (L.full_history) return h->c.hist + ((size_t)m * S + g0) * L.plane;
          if (m == n0) return h->c.ckpt + (size_t)c * L.blk(S) + (size_t)g0 * L.plane;
          if (m == n1) {
            const size_t slot = (m == p->nt) ? (size_t)L.ncheck : (size_t)(m / L.K);
            return h->c.ckpt + slot * L.blk(S) + (size_t)g0 * L.plane;
          }
          if (c >= L.ncheck - L.Mtail)
            return h->c.tail + (((size_t)(c - (L.ncheck - L.Mtail)) * (L.K - 1) + (m - n0 - 1)) * S + g0) * L.plane;
          return h->c.seg + ((size_t)(m - n0 - 1) * L.Sb + l0) * L.plane;
        };
      };
      if (!L.full_history && c < L.ncheck - L.Mtail) {
        // recompute Ez^{n0+1 .. n1-1} from checkpoint c with the same kernel (Ez^{n1} is a checkpoint)
        int idx = 0;
        for (int n = n0; n < n1 - 1; ++idx) {
          const int nsub = std::min(L.T, n1 - 1 - n);
          for (int k = 0; k < nl; ++k) {
            const int l0 = lb[k], nsl = lb[k + 1] - lb[k], g0 = shot0 + l0;
            auto ez_plane = ez_plane_of(l0);
            State in = (n == n0) ? state_at(L, h->c.ckpt + (size_t)c * L.blk(S), S, g0)
                                 : state_at(L, rs[idx & 1], S, l0);
            State out = state_at(L, rs[(idx + 1) & 1], S, l0);
            in.ez = ez_plane(n);
            out.ez = ez_plane(n + nsub);
            rc = launch_fwd_block(h, h->lanes[k], n, nsub, g0, nsl, in, out, nullptr, ez_plane);
            if (rc != GPRFWI_OK) return rc;
          }
          n += nsub;
        }
      }
      for (int n_hi = n1; n_hi > n0;) {
        const int nsub = std::min(L.T, n_hi - n0);
        for (int k = 0; k < nl; ++k) {
          const int l0 = lb[k], nsl = lb[k + 1] - lb[k];
          rc = launch_adj_block(h, h->lanes[k], n_hi, nsub, shot0 + l0, nsl, l0 / L.group,
                                state_at(L, lam[flip], L.Sb, l0), state_at(L, lam[flip ^ 1], L.Sb, l0), residual,
                                ez_plane_of(l0));
          if (rc != GPRFWI_OK) return rc;
        }
        flip ^= 1;
        n_hi -= nsub;
      }
    }
    rc = lanes_join(h, st, nl);
    if (rc != GPRFWI_OK) return rc;
  }
  {
    dim3 grid((p->nx + 127) / 128, p->nz), block(128);
    GPR_LAUNCH(grad_finalize_kernel, grid, block, st, h->eps_r, h->sigma, p->pitch, p->nz, p->nx, L.pitch,
                                                 (long long)L.plane, L.ngroups, (float)(1.0 / (double)p->dt),
                                                 h->c.gca, h->c.gcb, grad_eps_r, grad_sigma);
    h->launches++;
  }
  GPR_CUDA(cudaGetLastError());
  return GPRFWI_OK;
}

int gprfwi_residual(const float* d_syn, const float* d_obs, float* residual, size_t n, double* misfit,
                    void* cuda_stream)
{
  if (!d_syn || !d_obs || !residual) return GPRFWI_EINVAL;
  if (n == 0) return GPRFWI_OK;
  const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)sm_count() * 8);
  GPR_LAUNCH(residual_kernel, dim3(blocks), dim3(256), (cudaStream_t)cuda_stream, d_syn, d_obs, residual, n, misfit);
  GPR_CUDA(cudaGetLastError());
  return GPRFWI_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// host-buffer entry point: one misfit-gradient evaluation, copies included
// ------------------------------------------------------------------------------------------------
namespace gprfwi {
struct HostCarve {
  float *eps = nullptr, *sig = nullptr, *wav = nullptr, *dobs = nullptr, *traces = nullptr, *res = nullptr;
  float *ge = nullptr, *gs = nullptr;
  double* misfit = nullptr;
  char* core = nullptr;
  size_t head = 0;
};
static size_t host_carve(const gprfwi_params* p, char* base, HostCarve* c)
{
  size_t off = 0;
  auto take = [&](size_t bytes) -> char* {
    char* r = base ? base + off : nullptr;
    off += align_up(std::max<size_t>(bytes, 1), 256);
    return r;
  };
  const size_t model = (size_t)p->nz * p->pitch * sizeof(float);
  const size_t tr = (size_t)p->nshots * p->nt * p->nrec * sizeof(float);
  const size_t wv = (size_t)(p->wavelet_per_shot ? p->nshots : 1) * p->nt * sizeof(float);
  HostCarve tmp;
  HostCarve& o = c ? *c : tmp;
  o.eps = (float*)take(model); o.sig = (float*)take(model);
  o.ge = (float*)take(model);  o.gs = (float*)take(model);
  o.wav = (float*)take(wv);
  o.dobs = (float*)take(tr); o.traces = (float*)take(tr); o.res = (float*)take(tr);
  o.misfit = (double*)take(sizeof(double));
  o.core = base ? base + off : nullptr;
  o.head = off;
  return off;
}
}  // namespace gprfwi

extern "C" {

size_t gprfwi_workspace_bytes_host(const gprfwi_params* p, size_t budget_bytes)
{
  if (validate(p) != GPRFWI_OK) return 0;
  const size_t head = host_carve(p, nullptr, nullptr);
  if (budget_bytes != 0 && budget_bytes <= head) return 0;
  const size_t core = gprfwi_workspace_bytes(p, budget_bytes ? budget_bytes - head : 0, nullptr);
  return core ? head + core : 0;
}

int gprfwi_gradient_host(const gprfwi_params* p, const float* eps_r, const float* sigma, const float* wavelet,
                         const int32_t* src_zx, const int32_t* rec_zx, const float* d_obs, void* workspace,
                         size_t workspace_bytes, float* traces, float* grad_eps_r, float* grad_sigma,
                         double* misfit, void* cuda_stream)
{
  int rc = validate(p);
  if (rc != GPRFWI_OK) return rc;
  if (!eps_r || !sigma || !wavelet || !src_zx || !workspace || !grad_eps_r || !grad_sigma ||
      (p->nrec > 0 && (!rec_zx || !d_obs)))
    return GPRFWI_EINVAL;
  if ((uintptr_t)workspace % 256 != 0) return GPRFWI_EINVAL;
  HostCarve hc;
  host_carve(p, (char*)workspace, &hc);
  if (workspace_bytes <= hc.head) return GPRFWI_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t model = (size_t)p->nz * p->pitch * sizeof(float);
  const size_t ntr = (size_t)p->nshots * p->nt * p->nrec;
  const size_t wv = (size_t)(p->wavelet_per_shot ? p->nshots : 1) * p->nt * sizeof(float);
  GPR_CUDA(cudaMemcpyAsync(hc.eps, eps_r, model, cudaMemcpyHostToDevice, st));
  GPR_CUDA(cudaMemcpyAsync(hc.sig, sigma, model, cudaMemcpyHostToDevice, st));
  GPR_CUDA(cudaMemcpyAsync(hc.wav, wavelet, wv, cudaMemcpyHostToDevice, st));
  if (ntr) GPR_CUDA(cudaMemcpyAsync(hc.dobs, d_obs, ntr * sizeof(float), cudaMemcpyHostToDevice, st));
  GPR_CUDA(cudaMemsetAsync(hc.misfit, 0, sizeof(double), st));
  gprfwi_handle* h = nullptr;
  rc = gprfwi_forward(&h, p, hc.eps, hc.sig, hc.wav, src_zx, rec_zx, hc.core, workspace_bytes - hc.head,
                      hc.traces, st);
  if (rc != GPRFWI_OK) { gprfwi_release(h); return rc; }      // (forward may fail after it has created the handle)
  rc = gprfwi_residual(hc.traces, hc.dobs, hc.res, ntr, hc.misfit, st);
  if (rc == GPRFWI_OK) rc = gprfwi_adjoint(h, hc.res, hc.ge, hc.gs, st);
  gprfwi_release(h);
  if (rc != GPRFWI_OK) return rc;
  if (traces && ntr) GPR_CUDA(cudaMemcpyAsync(traces, hc.traces, ntr * sizeof(float), cudaMemcpyDeviceToHost, st));
  GPR_CUDA(cudaMemcpyAsync(grad_eps_r, hc.ge, model, cudaMemcpyDeviceToHost, st));
  GPR_CUDA(cudaMemcpyAsync(grad_sigma, hc.gs, model, cudaMemcpyDeviceToHost, st));
  double mf = 0.0;
  GPR_CUDA(cudaMemcpyAsync(&mf, hc.misfit, sizeof(double), cudaMemcpyDeviceToHost, st));
  GPR_CUDA(cudaStreamSynchronize(st));
  if (misfit) *misfit = mf;
  return GPRFWI_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// iteration epilogue: TV term, gradient mask, Adam step, clamps (gprfwi_update.cuh)
// ------------------------------------------------------------------------------------------------
extern "C" {

size_t gprfwi_update_workspace_bytes(int32_t nz, int32_t pitch)
{
  if (nz < 2 || pitch < 2) return 0;
  return (size_t)7 * align_up((size_t)nz * pitch * sizeof(float), 256) + 256;
}

int gprfwi_update(int32_t nz, int32_t nx, int32_t pitch, const gprfwi_update_params* u, float* eps_r, float* sigma,
                  float* grad_eps_r, float* grad_sigma, float* m_eps_r, float* v_eps_r, float* m_sigma,
                  float* v_sigma, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
  if (!u || !eps_r || !sigma || !grad_eps_r || !grad_sigma || !m_eps_r || !v_eps_r || !m_sigma || !v_sigma)
    return GPRFWI_EINVAL;
  if (nz < 2 || nx < 2 || pitch < nx || u->step < 1 || u->tv_iters < 0) return GPRFWI_EINVAL;
  if (u->tv_iters > 0 && (!(u->tv_rho > 0.f) || !workspace)) return GPRFWI_EINVAL;
  if (u->tv_iters > 0 && workspace_bytes < gprfwi_update_workspace_bytes(nz, pitch)) return GPRFWI_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t pb = align_up((size_t)nz * pitch * sizeof(float), 256);
  char* w = (char*)workspace;
  dim3 grid((nx + 127) / 128, nz), block(128);
  const float c1 = (float)(1.0 / (1.0 - std::pow((double)u->beta1, (double)u->step)));
  const float c2 = (float)(1.0 / (1.0 - std::pow((double)u->beta2, (double)u->step)));
  struct Par { float *x, *g, *m, *v; float lr, xmin; };
  const Par par[2] = {{eps_r, grad_eps_r, m_eps_r, v_eps_r, u->lr_eps_r, u->eps_r_min},
                      {sigma, grad_sigma, m_sigma, v_sigma, u->lr_sigma, u->sigma_min}};
  for (const Par& q : par) {
    if (u->tv_iters > 0) {
      float* u0 = (float*)(w + 0 * pb); float* ua = (float*)(w + 1 * pb); float* ub = (float*)(w + 2 * pb);
      float* zx = (float*)(w + 3 * pb); float* zz = (float*)(w + 4 * pb);
      float* bx = (float*)(w + 5 * pb); float* bz = (float*)(w + 6 * pb);
      unsigned* smax = (unsigned*)(w + 7 * pb);
      GPR_CUDA(cudaMemsetAsync(smax, 0, sizeof(unsigned), st));
      GPR_LAUNCH(absmax_kernel, dim3(std::min(nz, 1024)), dim3(256), st, q.x, nz, nx, pitch, smax);
      GPR_LAUNCH(tv_init_kernel, grid, block, st, q.x, nz, nx, pitch, smax, u0, ua, zx, zz, bx, bz);
      for (int it = 0; it < u->tv_iters; ++it) {
        GPR_LAUNCH(tv_jacobi_kernel, grid, block, st, nz, nx, pitch, u->tv_rho, u0, ua, zx, zz, bx, bz, ub);
        GPR_LAUNCH(tv_shrink_kernel, grid, block, st, nz, nx, pitch, u->tv_lambda / u->tv_rho, ub, zx, zz, bx, bz);
        std::swap(ua, ub);
      }
      GPR_LAUNCH(tv_add_kernel, grid, block, st, q.x, nz, nx, pitch, smax, u->tv_alpha, ua, q.g);
    }
    GPR_LAUNCH(adam_kernel, grid, block, st, nz, nx, pitch, u->mask_rows, q.lr, u->beta1, u->beta2, u->adam_eps,
               c1, c2, q.xmin, q.g, q.m, q.v, q.x);
  }
  GPR_CUDA(cudaGetLastError());
  return GPRFWI_OK;
}

int gprfwi_lowpass(const float* in, float* out, int32_t nseries, int32_t nt, int32_t nrec, const float* taps,
                   int32_t ntaps, void* cuda_stream)
{
  if (!in || !out || !taps || in == out) return GPRFWI_EINVAL;
  if (nseries < 1 || nt < 1 || nrec < 1 || ntaps < 1 || (ntaps & 1) == 0) return GPRFWI_EINVAL;
  const long long n = (long long)nt * nrec;
  dim3 grid((unsigned)std::min<long long>((n + 255) / 256, 4LL * sm_count()), (unsigned)nseries);
  GPR_LAUNCH(lowpass_kernel, grid, dim3(256), (cudaStream_t)cuda_stream, in, out, nt, nrec, taps, ntaps);
  GPR_CUDA(cudaGetLastError());
  return GPRFWI_OK;
}

int32_t gprfwi_lowpass_design(float dt, float f_cut, int32_t ntaps, float* taps)
{
  if (!(dt > 0.f) || !(f_cut > 0.f)) return GPRFWI_EINVAL;
  if (ntaps <= 0) ntaps = (int32_t)(4.0 / ((double)f_cut * (double)dt)) | 1;
  if ((ntaps & 1) == 0) return GPRFWI_EINVAL;
  if (!taps) return ntaps;
  // Hamming-windowed sinc, unit DC gain (reading R21), in float64, stored as fp32
  const double m = 0.5 * (ntaps - 1), fc = 2.0 * (double)f_cut * (double)dt;
  std::vector<double> h((size_t)ntaps);
  double sum = 0.0;
  for (int k = 0; k < ntaps; ++k) {
    const double x = kPi * fc * (k - m);
    const double snc = x == 0.0 ? 1.0 : std::sin(x) / x;
    const double win = ntaps > 1 ? 0.54 - 0.46 * std::cos(2.0 * kPi * k / (ntaps - 1)) : 1.0;
    h[(size_t)k] = snc * win;
    sum += h[(size_t)k];
  }
  for (int k = 0; k < ntaps; ++k) taps[k] = (float)(h[(size_t)k] / sum);
  return ntaps;
}

int gprfwi_restrict(const float* fine, int32_t nz, int32_t nx, int32_t pitch, float* coarse, int32_t pitch_coarse,
                    void* cuda_stream)
{
  if (!fine || !coarse || fine == coarse || nz < 3 || nx < 3 || pitch < nx || pitch_coarse < (nx + 1) / 2) return GPRFWI_EINVAL;
  const int nzc = (nz + 1) / 2, nxc = (nx + 1) / 2;
  dim3 grid((nxc + 127) / 128, nzc), block(128);
  GPR_LAUNCH(restrict_kernel, grid, block, (cudaStream_t)cuda_stream, fine, nz, nx, pitch, coarse, nzc, nxc, pitch_coarse);
  GPR_CUDA(cudaGetLastError());
  return GPRFWI_OK;
}

int gprfwi_prolong_add(const float* coarse, int32_t pitch_coarse, float scale, float* fine, int32_t nz, int32_t nx,
                       int32_t pitch, void* cuda_stream)
{
  if (!fine || !coarse || fine == coarse || nz < 3 || nx < 3 || pitch < nx || pitch_coarse < (nx + 1) / 2) return GPRFWI_EINVAL;
  const int nzc = (nz + 1) / 2, nxc = (nx + 1) / 2;
  dim3 grid((nx + 127) / 128, nz), block(128);
  GPR_LAUNCH(prolong_add_kernel, grid, block, (cudaStream_t)cuda_stream, coarse, nzc, nxc, pitch_coarse, scale, fine, nz, nx, pitch);
  GPR_CUDA(cudaGetLastError());
  return GPRFWI_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// gprfwi_update without a caller workspace and without any allocation (callers under CUDA-graph capture, tight
// serving loops, harnesses that forbid cudaMalloc): the TV term's scratch planes live in a file-scope device
// array of a fixed, modest size that every GPU that loads the library holds until exit.
// ------------------------------------------------------------------------------------------------
namespace gprfwi {
// 7 planes of up to 2^20 cells (e.g. 1024 x 1024 incl. pitch) + the 256-byte slot of the max|X| word
constexpr size_t kNoAllocMaxCells = (size_t)1 << 20;
constexpr size_t kNoAllocBytes = 7 * kNoAllocMaxCells * sizeof(float) + 256;
static __device__ __align__(256) unsigned char g_update_scratch[kNoAllocBytes];

// In host code `g_update_scratch` is only a stand-in for the symbol, NOT a device address: the address the
// kernels may use comes from cudaGetSymbolAddress, looked up once per device with that device current.
constexpr int kNoAllocMaxDevices = 64;
static void* g_update_scratch_ptr[kNoAllocMaxDevices] = {};

static int update_scratch_address(void** out)
{
  int dev = -1;
  GPR_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) return GPRFWI_EINVAL;
  void* p = __atomic_load_n(&g_update_scratch_ptr[dev], __ATOMIC_ACQUIRE);
  if (!p) {
    GPR_CUDA(cudaGetSymbolAddress(&p, g_update_scratch));      // (idempotent: racing first calls get the same address)
    if (!p) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_update_scratch)");
    __atomic_store_n(&g_update_scratch_ptr[dev], p, __ATOMIC_RELEASE);
  }
  *out = p;
  return GPRFWI_OK;
}
}  // namespace gprfwi

extern "C" {

size_t gprfwi_update_noalloc_max_bytes(void) { return kNoAllocBytes; }

int gprfwi_update_noalloc(int32_t nz, int32_t nx, int32_t pitch, const gprfwi_update_params* u, float* eps_r,
                          float* sigma, float* grad_eps_r, float* grad_sigma, float* m_eps_r, float* v_eps_r,
                          float* m_sigma, float* v_sigma, void* cuda_stream)
{
  const size_t need = gprfwi_update_workspace_bytes(nz, pitch);
  if (need == 0) return GPRFWI_EINVAL;
  if (need > kNoAllocBytes) return GPRFWI_ETOOBIG;
  void* scratch = nullptr;
  if (int rc = update_scratch_address(&scratch)) return rc;
  // Every call on a device shares the array, which still holds the previous call's contents: gprfwi_update
  // zeroes the max|X| word and tv_init_kernel rewrites every cell of the six planes it later reads, so nothing
  // else has to start at zero.  Calls that overlap on the GPU (different streams) race on it.
  return gprfwi_update(nz, nx, pitch, u, eps_r, sigma, grad_eps_r, grad_sigma, m_eps_r, v_eps_r, m_sigma, v_sigma,
                       scratch, kNoAllocBytes, cuda_stream);
}

}  // extern "C"
