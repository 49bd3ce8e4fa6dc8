// nh_lb.cuh -- D3Q19 lattice-Boltzmann kernels for sm_100a (flow side of the hot path).
//
// PAPER.md:118-166 (Sec. II.C): SRT collision with Guo forcing (Eqs. 14, 18), equilibrium
// (Eq. 15), moments (Eqs. 16-17), and their shifted forms (Eqs. 19-23, evaluation order
// PAPER.md:187); half-way bounce-back at the plates; periodic x, y.
//
// Scheme: two-lattice PULL.  The stored state is the post-collision population f*_i(x, t-1).
// One launch gathers f_i(x, t) = f*_i(x - e_i, t-1) (or f*_ibar(x, t-1) when x - e_i is a plate
// layer), takes the moments, collides and writes f*_i(x, t) to the other buffer at the thread's
// own cell, so every store is aligned and fully coalesced; only 10 of the 19 gathers are shifted
// by one element along x.  Layout: SoA, f[i][z][y][x], x fastest.
#pragma once
#include <cuda_runtime.h>

namespace nh {

// D3Q19 directions (this file's own order; pairs (2k-1, 2k) are opposites):
//  0: rest
//  1:(+x) 2:(-x) 3:(+y) 4:(-y) 5:(+z) 6:(-z)
//  7:(+x+y) 8:(-x-y) 9:(+x-y) 10:(-x+y)
// 11:(+x+z) 12:(-x-z) 13:(+x-z) 14:(-x+z)
// 15:(+y+z) 16:(-y-z) 17:(+y-z) 18:(-y+z)
constexpr int Q = 19;

struct Geom {
  int nx, ny, nz;
  unsigned plane;   // nx*ny
  unsigned nfluid;  // nx*ny*(nz-2)
  size_t N;         // nx*ny*nz
};

template <typename T>
struct LbConst {
  T omega;      // 1/tau
  T somega;     // 1 - 1/(2 tau)
  T gx, gy, gz; // body acceleration
  int use_flc;  // coupling bit0
};

// 19 gathered populations of one cell
template <typename T>
struct Pop { T f[Q]; };

template <typename T>
__device__ __forceinline__ T ldg_stream(const T* p) { return __ldg(p); }

// Gather f_i(x, t) for the cell (x, y, z) from the post-collision buffer `fs`.
template <typename T>
__device__ __forceinline__ void pull(const T* __restrict__ fs, const Geom& G, int x, int y, int z,
                                     Pop<T>& P) {
  const size_t N = G.N;
  const int nx = G.nx;
  const int xm = (x == 0) ? nx - 1 : x - 1;        // source column for e_x = +1
  const int xp = (x == nx - 1) ? 0 : x + 1;        // source column for e_x = -1
  const int ym = (y == 0) ? G.ny - 1 : y - 1;
  const int yp = (y == G.ny - 1) ? 0 : y + 1;
  const unsigned r0 = (unsigned)z * G.plane + (unsigned)y * nx;    // own row
  const unsigned rym = (unsigned)z * G.plane + (unsigned)ym * nx;  // row y-1, same z
  const unsigned ryp = (unsigned)z * G.plane + (unsigned)yp * nx;
  const unsigned c = r0 + x;
  const bool lo = (z == 1);           // z-1 is the bottom plate
  const bool hi = (z == G.nz - 2);    // z+1 is the top plate

  P.f[0] = ldg_stream(fs + c);
  P.f[1] = ldg_stream(fs + 1 * N + r0 + xm);
  P.f[2] = ldg_stream(fs + 2 * N + r0 + xp);
  P.f[3] = ldg_stream(fs + 3 * N + rym + x);
  P.f[4] = ldg_stream(fs + 4 * N + ryp + x);
  P.f[7] = ldg_stream(fs + 7 * N + rym + xm);
  P.f[8] = ldg_stream(fs + 8 * N + ryp + xp);
  P.f[9] = ldg_stream(fs + 9 * N + ryp + xm);
  P.f[10] = ldg_stream(fs + 10 * N + rym + xp);
  // directions with e_z = +1 come from z-1; at z = 1 they bounce off the bottom plate:
  // f_i(x, t) = f*_ibar(x, t-1)
  {
    const unsigned dn = G.plane;  // one layer
    P.f[5] = lo ? ldg_stream(fs + 6 * N + c) : ldg_stream(fs + 5 * N + c - dn);
    P.f[11] = lo ? ldg_stream(fs + 12 * N + c) : ldg_stream(fs + 11 * N + r0 - dn + xm);
    P.f[14] = lo ? ldg_stream(fs + 13 * N + c) : ldg_stream(fs + 14 * N + r0 - dn + xp);
    P.f[15] = lo ? ldg_stream(fs + 16 * N + c) : ldg_stream(fs + 15 * N + rym - dn + x);
    P.f[18] = lo ? ldg_stream(fs + 17 * N + c) : ldg_stream(fs + 18 * N + ryp - dn + x);
    // directions with e_z = -1 come from z+1; at z = nz-2 they bounce off the top plate
    P.f[6] = hi ? ldg_stream(fs + 5 * N + c) : ldg_stream(fs + 6 * N + c + dn);
    P.f[12] = hi ? ldg_stream(fs + 11 * N + c) : ldg_stream(fs + 12 * N + r0 + dn + xp);
    P.f[13] = hi ? ldg_stream(fs + 14 * N + c) : ldg_stream(fs + 13 * N + r0 + dn + xm);
    P.f[16] = hi ? ldg_stream(fs + 15 * N + c) : ldg_stream(fs + 16 * N + ryp + dn + x);
    P.f[17] = hi ? ldg_stream(fs + 18 * N + c) : ldg_stream(fs + 17 * N + rym + dn + x);
  }
}

// Moments.  Shifted: drho = sum f (Eq. 20), rho = 1 + drho; unshifted: rho = sum f (Eq. 16).
// j = sum e_i f_i.  The sums are grouped in opposite pairs, smallest magnitudes first.
template <typename T, bool SHIFTED>
__device__ __forceinline__ void moments(const Pop<T>& P, T& drho, T& rho, T& jx, T& jy, T& jz) {
  const T* f = P.f;
  const T sxy = (f[7] + f[8]) + (f[9] + f[10]);
  const T sxz = (f[11] + f[12]) + (f[13] + f[14]);
  const T syz = (f[15] + f[16]) + (f[17] + f[18]);
  const T sax = ((f[1] + f[2]) + (f[3] + f[4])) + (f[5] + f[6]);
  const T s = ((sxy + sxz) + syz) + sax + f[0];
  if (SHIFTED) { drho = s; rho = T(1) + s; }
  else         { rho = s; drho = s - T(1); }
  jx = (f[1] - f[2]) + (((f[7] - f[8]) + (f[9] - f[10])) + ((f[11] - f[12]) + (f[13] - f[14])));
  jy = (f[3] - f[4]) + (((f[7] - f[8]) - (f[9] - f[10])) + ((f[15] - f[16]) + (f[17] - f[18])));
  jz = (f[5] - f[6]) + (((f[11] - f[12]) - (f[13] - f[14])) + ((f[15] - f[16]) - (f[17] - f[18])));
}

// Collide one opposite pair (a: direction e, b: direction -e).
//   f^eq,s = w [drho + rho (3 eu + 4.5 eu^2 - 1.5 u^2)]            Eq. 22 (never forms w + small)
//   f^eq   = w rho [1 + 3 eu + 4.5 eu^2 - 1.5 u^2]                 Eq. 15
//   S      = w [3 eF + 9 eu eF - 3 uF]                             Eq. 18 with c_s^2 = 1/3
//   f*     = f - (f - f^eq)/tau + (1 - 1/(2 tau)) S                Eqs. 14 / 23
template <typename T, bool SHIFTED>
__device__ __forceinline__ void collide_pair(T& fa, T& fb, T w, T eu, T eF, T base, T rho, T sbase,
                                             const LbConst<T>& C) {
  // base = SHIFTED ? drho - 1.5 rho u^2 : rho (1 - 1.5 u^2);  sbase = -3 uF
  const T even = base + T(4.5) * rho * eu * eu;
  const T odd = T(3) * rho * eu;
  const T seven = sbase + T(9) * eu * eF;
  const T sodd = T(3) * eF;
  const T feq_a = w * (even + odd), feq_b = w * (even - odd);
  const T S_a = w * (seven + sodd), S_b = w * (seven - sodd);
  fa = fa - C.omega * (fa - feq_a) + C.somega * S_a;
  fb = fb - C.omega * (fb - feq_b) + C.somega * S_b;
}

template <typename T, bool SHIFTED>
__device__ __forceinline__ void collide(Pop<T>& P, T Flx, T Fly, T Flz, const LbConst<T>& C) {
  T drho, rho, jx, jy, jz;
  moments<T, SHIFTED>(P, drho, rho, jx, jy, jz);
  // total force F = F^LC + rho g (reading G8); u = (j + F/2)/rho  (Eq. 21 / 17)
  const T Fx = Flx + rho * C.gx, Fy = Fly + rho * C.gy, Fz = Flz + rho * C.gz;
  const T inv = T(1) / rho;
  const T ux = (jx + T(0.5) * Fx) * inv, uy = (jy + T(0.5) * Fy) * inv, uz = (jz + T(0.5) * Fz) * inv;
  const T u2 = ux * ux + uy * uy + uz * uz;
  const T uF = ux * Fx + uy * Fy + uz * Fz;
  const T base = SHIFTED ? drho - T(1.5) * rho * u2 : rho - T(1.5) * rho * u2;
  const T sbase = T(-3) * uF;
  const T w0 = T(1) / T(3), w1 = T(1) / T(18), w2 = T(1) / T(36);
  T* f = P.f;
  f[0] = f[0] - C.omega * (f[0] - w0 * base) + C.somega * (w0 * sbase);
  collide_pair<T, SHIFTED>(f[1], f[2], w1, ux, Fx, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[3], f[4], w1, uy, Fy, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[5], f[6], w1, uz, Fz, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[7], f[8], w2, ux + uy, Fx + Fy, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[9], f[10], w2, ux - uy, Fx - Fy, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[11], f[12], w2, ux + uz, Fx + Fz, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[13], f[14], w2, ux - uz, Fx - Fz, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[15], f[16], w2, uy + uz, Fy + Fz, base, rho, sbase, C);
  collide_pair<T, SHIFTED>(f[17], f[18], w2, uy - uz, Fy - Fz, base, rho, sbase, C);
}

__device__ __forceinline__ void cell_of(unsigned fluid_index, const Geom& G, int& x, int& y, int& z) {
  const unsigned zz = fluid_index / G.plane;
  const unsigned xy = fluid_index - zz * G.plane;
  const unsigned yy = xy / (unsigned)G.nx;
  z = (int)zz + 1;
  y = (int)yy;
  x = (int)(xy - yy * (unsigned)G.nx);
}

// Sweep direction.  Consecutive launches traverse the lattice in opposite directions: a launch
// then starts on the cells whose populations the previous launch wrote last, which are still in
// the 126 MB L2, so part of every gather is served without touching HBM.
__device__ __forceinline__ unsigned sweep_block(int reverse) {
  return reverse ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
}

// One LB step, one thread per fluid cell (baseline variant; nh_lb_vec.cuh holds the wide one).
template <typename T, bool SHIFTED>
__global__ void __launch_bounds__(256)
lb_step_kernel(const T* __restrict__ fsrc, T* __restrict__ fdst, const T* __restrict__ Flc,
               Geom G, LbConst<T> C, int reverse) {
  const unsigned k = sweep_block(reverse) * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const size_t c = (size_t)k + G.plane;
  Pop<T> P;
  pull<T>(fsrc, G, x, y, z, P);
  T Fx = T(0), Fy = T(0), Fz = T(0);
  if (C.use_flc) { Fx = __ldg(Flc + c); Fy = __ldg(Flc + G.N + c); Fz = __ldg(Flc + 2 * G.N + c); }
  collide<T, SHIFTED>(P, Fx, Fy, Fz, C);
#pragma unroll
  for (int i = 0; i < Q; ++i) fdst[(size_t)i * G.N + c] = P.f[i];
}

// rho, u of the populations that the NEXT step will gather (i.e. at the current time t), with the
// current force: Eqs. 20-21 (16-17).  Writes u in the device precision for the FD kernels.
template <typename T, bool SHIFTED>
__global__ void __launch_bounds__(256)
velocity_kernel(const T* __restrict__ fsrc, const T* __restrict__ Flc, T* __restrict__ u,
                Geom G, LbConst<T> C, int reverse) {
  const unsigned k = sweep_block(reverse) * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const size_t c = (size_t)k + G.plane;
  Pop<T> P;
  pull<T>(fsrc, G, x, y, z, P);
  T drho, rho, jx, jy, jz;
  moments<T, SHIFTED>(P, drho, rho, jx, jy, jz);
  T Fx = T(0), Fy = T(0), Fz = T(0);
  if (C.use_flc) { Fx = __ldg(Flc + c); Fy = __ldg(Flc + G.N + c); Fz = __ldg(Flc + 2 * G.N + c); }
  Fx += rho * C.gx; Fy += rho * C.gy; Fz += rho * C.gz;
  const T inv = T(1) / rho;
  u[c] = (jx + T(0.5) * Fx) * inv;
  u[G.N + c] = (jy + T(0.5) * Fy) * inv;
  u[2 * G.N + c] = (jz + T(0.5) * Fz) * inv;
}

// Same moments, written as FP64 to the staging buffer for nh_get_fields: out = [rho | ux uy uz],
// each [N]; plate layers get rho = 1, u = 0.  One thread per cell of the WHOLE grid.
template <typename T, bool SHIFTED>
__global__ void __launch_bounds__(256)
fields_kernel(const T* __restrict__ fsrc, const T* __restrict__ Flc, double* __restrict__ rho_out,
              double* __restrict__ u_out, Geom G, LbConst<T> C) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= G.N) return;
  const unsigned zz = (unsigned)(c / G.plane);
  double r = 1.0, vx = 0.0, vy = 0.0, vz = 0.0;
  if (zz != 0 && zz != (unsigned)G.nz - 1) {
    int x, y, z;
    cell_of((unsigned)(c - G.plane), G, x, y, z);
    Pop<T> P;
    pull<T>(fsrc, G, x, y, z, P);
    T drho, rho, jx, jy, jz;
    moments<T, SHIFTED>(P, drho, rho, jx, jy, jz);
    T Fx = T(0), Fy = T(0), Fz = T(0);
    if (C.use_flc) { Fx = Flc[c]; Fy = Flc[G.N + c]; Fz = Flc[2 * G.N + c]; }
    Fx += rho * C.gx; Fy += rho * C.gy; Fz += rho * C.gz;
    const T inv = T(1) / rho;
    r = (double)rho;
    vx = (double)((jx + T(0.5) * Fx) * inv);
    vy = (double)((jy + T(0.5) * Fy) * inv);
    vz = (double)((jz + T(0.5) * Fz) * inv);
  }
  if (rho_out) rho_out[c] = r;
  if (u_out) { u_out[c] = vx; u_out[G.N + c] = vy; u_out[2 * G.N + c] = vz; }
}

// Rest state rho = 1, u = 0 on the fluid cells: shifted populations 0 (Eq. 19), unshifted w_i.
template <typename T, bool SHIFTED>
__global__ void __launch_bounds__(256) rest_kernel(T* __restrict__ f, Geom G) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= G.N) return;
  const unsigned zz = (unsigned)(c / G.plane);
  const bool fluid = (zz != 0 && zz != (unsigned)G.nz - 1);
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const T w = (i == 0) ? T(1) / T(3) : (i < 7 ? T(1) / T(18) : T(1) / T(36));
    f[(size_t)i * G.N + c] = (SHIFTED || !fluid) ? T(0) : w;
  }
}

}  // namespace nh
