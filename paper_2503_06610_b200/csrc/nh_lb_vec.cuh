// nh_lb_vec.cuh -- the wide LB kernel: one thread updates V consecutive cells of an x row with
// 16-byte loads and stores (V = 4 in FP32, 2 in FP64).  Same arithmetic as nh_lb.cuh (it calls
// the same collide<>), Eqs. 14-23; bounce-back PAPER.md:141; periodic x, y
// PAPER.md:225.
//
// Pull scheme on the SoA layout f[i][z][y][x]:
//   - all 19 stores and the 9 gathers with e_x = 0 are aligned 16-byte vectors;
//   - the 10 gathers with e_x = +-1 read the aligned vector of the thread's own columns and take
//     the one missing element from the neighbouring lane (warp shuffle); only a lane at a warp
//     or row edge issues one extra 4/8-byte load (the periodic wrap lives there);
//   - at the plate-adjacent layers the gather of a direction that would come out of the plate
//     reads the opposite direction at the thread's own cells instead (half-way bounce-back), which
//     is an aligned vector again.
// Requires nx % V == 0 (otherwise the library uses the one-cell-per-thread kernel).
#pragma once
#include <cuda_runtime.h>
#include "nh_lb.cuh"

namespace nh {

template <typename T, int V> struct VecOf;
template <> struct VecOf<float, 4> { using type = float4; };
template <> struct VecOf<double, 2> { using type = double2; };

template <typename T, int V> struct alignas(16) Pack { T v[V]; };

// streaming 16-byte load through the read-only path; populations are read exactly once per step
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> ldv(const T* p) {
  using VT = typename VecOf<T, V>::type;
  const VT r = __ldcs(reinterpret_cast<const VT*>(p));
  Pack<T, V> o;
  *reinterpret_cast<VT*>(o.v) = r;
  return o;
}
// 16-byte load of a field that is re-read by later steps (F^LC): default caching
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> ldv_keep(const T* p) {
  using VT = typename VecOf<T, V>::type;
  const VT r = __ldg(reinterpret_cast<const VT*>(p));
  Pack<T, V> o;
  *reinterpret_cast<VT*>(o.v) = r;
  return o;
}
template <typename T, int V>
__device__ __forceinline__ void stv(T* p, const Pack<T, V>& a) {
  using VT = typename VecOf<T, V>::type;
  __stcs(reinterpret_cast<VT*>(p), *reinterpret_cast<const VT*>(a.v));
}

// Gathered populations of the V cells of one thread.
template <typename T, int V> struct PopV { Pack<T, V> f[Q]; };

// Where one thread's cells are, and what its warp neighbours can give it.
struct Where {
  unsigned c;       // index of the first cell (x0, y, z)
  unsigned r0;      // index of (0, y, z)
  unsigned rym, ryp;// index of (0, y-1, z), (0, y+1, z)  (periodic)
  int x0, nx;
  unsigned plane;
  bool lo, hi;      // z-1 / z+1 is a plate layer
  bool ledge, redge;// no usable left / right lane: warp edge or row edge
  unsigned xl, xr;  // wrapped columns x0-1 and x0+V
};

// e_x = 0: aligned vector from row `row` (index of its x = 0 cell)
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> take0(const T* __restrict__ fi, unsigned row, const Where& w) {
  return ldv<T, V>(fi + row + w.x0);
}
// e_x = +1: cells x0-1 .. x0+V-2 of row `row`
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> takeP(const T* __restrict__ fi, unsigned row, const Where& w) {
  const Pack<T, V> a = ldv<T, V>(fi + row + w.x0);
  T left = __shfl_up_sync(0xffffffffu, a.v[V - 1], 1);
  if (w.ledge) left = __ldg(fi + row + w.xl);
  Pack<T, V> o;
  o.v[0] = left;
#pragma unroll
  for (int j = 1; j < V; ++j) o.v[j] = a.v[j - 1];
  return o;
}
// e_x = -1: cells x0+1 .. x0+V of row `row`
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> takeM(const T* __restrict__ fi, unsigned row, const Where& w) {
  const Pack<T, V> a = ldv<T, V>(fi + row + w.x0);
  T right = __shfl_down_sync(0xffffffffu, a.v[0], 1);
  if (w.redge) right = __ldg(fi + row + w.xr);
  Pack<T, V> o;
#pragma unroll
  for (int j = 0; j < V - 1; ++j) o.v[j] = a.v[j + 1];
  o.v[V - 1] = right;
  return o;
}
// The same three with the plate test in front: `bounce` -> the opposite direction `fo` at the
// thread's own cells.  The shuffle inside takeP / takeM is executed by every lane either way.
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> take0_bb(const T* __restrict__ fi, const T* __restrict__ fo,
                                               unsigned row, bool bounce, const Where& w) {
  return ldv<T, V>(bounce ? fo + w.c : fi + row + w.x0);
}
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> takeP_bb(const T* __restrict__ fi, const T* __restrict__ fo,
                                               unsigned row, bool bounce, const Where& w) {
  const Pack<T, V> a = ldv<T, V>(bounce ? fo + w.c : fi + row + w.x0);
  T left = __shfl_up_sync(0xffffffffu, a.v[V - 1], 1);
  if (bounce) return a;
  if (w.ledge) left = __ldg(fi + row + w.xl);
  Pack<T, V> o;
  o.v[0] = left;
#pragma unroll
  for (int j = 1; j < V; ++j) o.v[j] = a.v[j - 1];
  return o;
}
template <typename T, int V>
__device__ __forceinline__ Pack<T, V> takeM_bb(const T* __restrict__ fi, const T* __restrict__ fo,
                                               unsigned row, bool bounce, const Where& w) {
  const Pack<T, V> a = ldv<T, V>(bounce ? fo + w.c : fi + row + w.x0);
  T right = __shfl_down_sync(0xffffffffu, a.v[0], 1);
  if (bounce) return a;
  if (w.redge) right = __ldg(fi + row + w.xr);
  Pack<T, V> o;
#pragma unroll
  for (int j = 0; j < V - 1; ++j) o.v[j] = a.v[j + 1];
  o.v[V - 1] = right;
  return o;
}

// f_i(x, t) = f*_i(x - e_i, t-1) for the V cells of this thread (direction table in nh_lb.cuh).
template <typename T, int V>
__device__ __forceinline__ void pull_vec(const T* __restrict__ fs, size_t N, const Where& w, PopV<T, V>& P) {
  const unsigned dn = w.plane;
  P.f[0] = take0<T, V>(fs, w.r0, w);
  P.f[1] = takeP<T, V>(fs + 1 * N, w.r0, w);
  P.f[2] = takeM<T, V>(fs + 2 * N, w.r0, w);
  P.f[3] = take0<T, V>(fs + 3 * N, w.rym, w);
  P.f[4] = take0<T, V>(fs + 4 * N, w.ryp, w);
  P.f[7] = takeP<T, V>(fs + 7 * N, w.rym, w);
  P.f[8] = takeM<T, V>(fs + 8 * N, w.ryp, w);
  P.f[9] = takeP<T, V>(fs + 9 * N, w.ryp, w);
  P.f[10] = takeM<T, V>(fs + 10 * N, w.rym, w);
  // e_z = +1 comes from z-1, or bounces off the bottom plate
  P.f[5] = take0_bb<T, V>(fs + 5 * N, fs + 6 * N, w.r0 - dn, w.lo, w);
  P.f[11] = takeP_bb<T, V>(fs + 11 * N, fs + 12 * N, w.r0 - dn, w.lo, w);
  P.f[14] = takeM_bb<T, V>(fs + 14 * N, fs + 13 * N, w.r0 - dn, w.lo, w);
  P.f[15] = take0_bb<T, V>(fs + 15 * N, fs + 16 * N, w.rym - dn, w.lo, w);
  P.f[18] = take0_bb<T, V>(fs + 18 * N, fs + 17 * N, w.ryp - dn, w.lo, w);
  // e_z = -1 comes from z+1, or bounces off the top plate
  P.f[6] = take0_bb<T, V>(fs + 6 * N, fs + 5 * N, w.r0 + dn, w.hi, w);
  P.f[12] = takeM_bb<T, V>(fs + 12 * N, fs + 11 * N, w.r0 + dn, w.hi, w);
  P.f[13] = takeP_bb<T, V>(fs + 13 * N, fs + 14 * N, w.r0 + dn, w.hi, w);
  P.f[16] = take0_bb<T, V>(fs + 16 * N, fs + 15 * N, w.ryp + dn, w.hi, w);
  P.f[17] = take0_bb<T, V>(fs + 17 * N, fs + 18 * N, w.rym + dn, w.hi, w);
}

// Group k = V consecutive fluid cells.  Every lane of the warp computes a (clamped) position so
// that all of them take part in the shuffles; `active` says whether the group exists.
template <int V>
__device__ __forceinline__ Where where_of(unsigned k, unsigned ngroups, const Geom& G, bool& active) {
  active = k < ngroups;
  if (!active) k = ngroups - 1;
  const unsigned cell = k * V;                  // fluid-cell index of the first cell
  const unsigned zz = cell / G.plane;
  const unsigned xy = cell - zz * G.plane;
  const unsigned yy = xy / (unsigned)G.nx;
  const int x0 = (int)(xy - yy * (unsigned)G.nx);
  const int z = (int)zz + 1;
  const unsigned zbase = (unsigned)z * G.plane;
  Where w;
  w.nx = G.nx;
  w.plane = G.plane;
  w.x0 = x0;
  w.r0 = zbase + yy * (unsigned)G.nx;
  w.c = w.r0 + (unsigned)x0;
  w.rym = zbase + (yy == 0 ? (unsigned)G.ny - 1 : yy - 1) * (unsigned)G.nx;
  w.ryp = zbase + (yy == (unsigned)G.ny - 1 ? 0u : yy + 1) * (unsigned)G.nx;
  w.lo = (z == 1);
  w.hi = (z == G.nz - 2);
  const unsigned lane = threadIdx.x & 31u;
  w.ledge = (lane == 0) || (x0 == 0);
  w.redge = (lane == 31) || (x0 + V == G.nx);
  w.xl = (x0 == 0) ? (unsigned)G.nx - 1 : (unsigned)x0 - 1;
  w.xr = (x0 + V == G.nx) ? 0u : (unsigned)(x0 + V);
  return w;
}

template <typename T, bool SHIFTED, int V>
__global__ void __launch_bounds__(256)
lb_step_vec_kernel(const T* __restrict__ fsrc, T* __restrict__ fdst, const T* __restrict__ Flc,
                   Geom G, LbConst<T> C, unsigned ngroups, int reverse) {
  const unsigned k = sweep_block(reverse) * blockDim.x + threadIdx.x;
  bool active;
  const Where w = where_of<V>(k, ngroups, G, active);
  PopV<T, V> P;
  pull_vec<T, V>(fsrc, G.N, w, P);
  if (!active) return;
  Pack<T, V> Fx, Fy, Fz;
  if (C.use_flc) {
    Fx = ldv_keep<T, V>(Flc + w.c);
    Fy = ldv_keep<T, V>(Flc + G.N + w.c);
    Fz = ldv_keep<T, V>(Flc + 2 * G.N + w.c);
  } else {
#pragma unroll
    for (int j = 0; j < V; ++j) Fx.v[j] = Fy.v[j] = Fz.v[j] = T(0);
  }
#pragma unroll
  for (int j = 0; j < V; ++j) {
    Pop<T> p;
#pragma unroll
    for (int i = 0; i < Q; ++i) p.f[i] = P.f[i].v[j];
    collide<T, SHIFTED>(p, Fx.v[j], Fy.v[j], Fz.v[j], C);
#pragma unroll
    for (int i = 0; i < Q; ++i) P.f[i].v[j] = p.f[i];
  }
#pragma unroll
  for (int i = 0; i < Q; ++i) stv<T, V>(fdst + (size_t)i * G.N + w.c, P.f[i]);
}

}  // namespace nh
