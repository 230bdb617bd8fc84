// gprfwi_common.cuh -- device-side data layout shared by all kernels of libgprfwi.
//
// Layout in HBM, all fp32, shot index outermost:
//   field plane   [S][nz][pitch]     pitch = internal row pitch, multiple of 32 floats (128 B)
//                 Ez at (j,i); Hx at (j+1/2,i) (row nz-1 unused, kept 0); Hy at (j,i+1/2)
//                 (column nx-1 unused, kept 0); columns [nx, roundup4(nx)) are written as 0.
//   z-strips      [S][2P][pitch]     CPML psi of the z-derivative, only the 2P rows where it lives
//   x-strips      [S][nz][xw]        CPML psi of the x-derivative, only the float4 units of a row that
//                                    touch the left / right CPML: units [0, xnl) then [xur, pitch/4)
//   Ca, Cb        [nz][pitch]        shared by all shots
//   1-D CPML tables (b, c, 1/kappa, c/dx, Db/(dx kappa)) per axis and per E/H location, built on the
//   host in float64.
#pragma once
#include <stdint.h>
#include <vector_types.h>

#if defined(__CUDACC__)
#define GPR_HD __host__ __device__ __forceinline__
#else
#define GPR_HD inline
#endif

namespace gprfwi {

struct Geo {
  int nz, nx, P;        // full grid, CPML thickness
  int pitch;            // internal row pitch in floats
  int xw;               // x-strip row width in floats = 4 * (xnl + pitch/4 - xur)
  int xnl, xur;         // float4 units [0, xnl) hold the left CPML columns, units [xur, pitch/4) the right ones
  long long plane;      // nz * pitch
  long long zstrip;     // 2P * pitch   (per shot)
  long long xstrip;     // nz * xw      (per shot)
  float rdx, Db, kap;   // 1/dx ; dt/mu0 (the paper's uH4 with mu_r = 1) ; fp32 product Db*rdx
  // 1-D CPML tables, one set per axis and per E/H location, each [5][n]: b, c, 1/kappa, c/dx, and
  // (H sets) Db/(dx kappa).  The last two are the forward kernel's pre-multiplied forms.
  const float *tex, *tez;   // E nodes: x axis (n = nx), z axis (n = nz)
  const float *thx, *thz;   // H nodes (i + 1/2): x axis, z axis
};

// One complete state of the scheme for a batch of shots (pointers are for local shot 0).
// Forward: ez = Ez, hx/hy = H, p* = psi.  Adjoint: the same slots hold the adjoint variables.
struct State {
  float* ez;     // [S][nz][pitch]
  float* hx;     // [S][nz][pitch]
  float* hy;     // [S][nz][pitch]
  float* phxz;   // [S][2P][pitch]  psi of dEz/dz in the Hx update (H-z located rows)
  float* pezz;   // [S][2P][pitch]  psi of dHx/dz in the Ez update (E-z located rows)
  float* phyx;   // [S][nz][xw]     psi of dEz/dx in the Hy update (H-x located columns)
  float* pezx;   // [S][nz][xw]     psi of dHy/dx in the Ez update (E-x located columns)
};

// strip index of an E-located / H-located node along an axis of n Ez nodes, or -1 outside the CPML
GPR_HD int strip_e(int i, int n, int P) { return i < P ? i : ((i >= n - P && i < n) ? i - (n - P) + P : -1); }
GPR_HD int strip_h(int i, int n, int P)
{
  return i < P ? i : ((i >= n - 1 - P && i < n - 1) ? i - (n - 1 - P) + P : -1);
}

// float offset of float4 unit u (columns 4u..4u+3) inside an x-strip row, or -1 if the unit holds no CPML column
GPR_HD int xstrip_slot(int u, int xnl, int xur, int pitch)
{
  return u < 0 ? -1 : (u < xnl ? 4 * u : ((u >= xur && 4 * u < pitch) ? 4 * (xnl + u - xur) : -1));
}

// INTERNAL column order (every [..][pitch] array the library owns: fields, psi, Ca, Cb, history, gCa, gCb):
// inside each aligned group of four columns (c0 c1 c2 c3) the floats are stored as (c0 c2 c1 c3), so that a
// 128-bit load yields two packed pairs P = (c0, c2), Q = (c1, c3) for the sm_100 FFMA2 / FADD2 / FMUL2
// instructions with every x-neighbour difference (c1 - c0, c3 - c2) a plain pair operation.
GPR_HD int unit_perm(int c) { return c == 1 ? 2 : (c == 2 ? 1 : c); }
GPR_HD int col_pos(int i) { return (i & ~3) | unit_perm(i & 3); }

GPR_HD float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
GPR_HD void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
GPR_HD float4 mk4(float a, float b, float c, float d) { float4 v; v.x = a; v.y = b; v.z = c; v.w = d; return v; }
GPR_HD void unpack(float4 v, float* o) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }

}  // namespace gprfwi
