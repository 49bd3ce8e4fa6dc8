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
#include <cooperative_groups.h>

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

// Programmatic dependent launch (PTX griddepcontrol; no-ops when the launch does not carry the attribute)
__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ float fmaf_t(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fmaf_t(double a, double b, double c) { return fma(a, b, c); }

// Load policies of the gathers: LD_NC read-only path (data not written during the launch),
// LD_CS the same with the streaming (evict-first) hint, LD_CG coherent at L2 (data that another CTA
// of the SAME launch has written: the ring of the two-step kernel, nh_lb2.cuh).
enum { LD_NC = 0, LD_CS = 1, LD_CG = 2 };
template <typename T, int LD>
__device__ __forceinline__ T ldp(const T* p) {
  if constexpr (LD == LD_NC) return __ldg(p);
  else if constexpr (LD == LD_CS) return __ldcs(p);
  else return __ldcg(p);
}

// Where the three z planes a gather touches live inside a population array: element offsets of
// the planes z-1, z, z+1 and the stride between directions.  The lattice arrays use
// (z-1, z, z+1)*plane and stride N; the plane ring of nh_lb2.cuh maps planes to ring slots.
struct PlaneMap {
  size_t stride;
  unsigned zm, z0, zp;
};
__device__ __forceinline__ PlaneMap lattice_map(const Geom& G, int z) {
  PlaneMap M;
  M.stride = G.N;
  M.z0 = (unsigned)z * G.plane;
  M.zm = M.z0 - G.plane;
  M.zp = M.z0 + G.plane;
  return M;
}

// Gather f_i(x, t) for the cell (x, y) of the plane M.z0 from the post-collision array `fs`.
// lo / hi: the plane below / above is a plate layer (half-way bounce-back).
template <typename T, int LD>
__device__ __forceinline__ void pull_map(const T* __restrict__ fs, const Geom& G, const PlaneMap& M,
                                         int x, int y, bool lo, bool hi, Pop<T>& P) {
  const size_t N = M.stride;
  const int nx = G.nx;
  const int xm = (x == 0) ? nx - 1 : x - 1;        // source column for e_x = +1
  const int xp = (x == nx - 1) ? 0 : x + 1;        // source column for e_x = -1
  const int ym = (y == 0) ? G.ny - 1 : y - 1;
  const int yp = (y == G.ny - 1) ? 0 : y + 1;
  const unsigned o0 = (unsigned)y * nx, om = (unsigned)ym * nx, op = (unsigned)yp * nx;
  const unsigned r0 = M.z0 + o0;                   // own row
  const unsigned rym = M.z0 + om;                  // row y-1, same z
  const unsigned ryp = M.z0 + op;
  const unsigned c = r0 + x;

  P.f[0] = ldp<T, LD>(fs + c);
  P.f[1] = ldp<T, LD>(fs + 1 * N + r0 + xm);
  P.f[2] = ldp<T, LD>(fs + 2 * N + r0 + xp);
  P.f[3] = ldp<T, LD>(fs + 3 * N + rym + x);
  P.f[4] = ldp<T, LD>(fs + 4 * N + ryp + x);
  P.f[7] = ldp<T, LD>(fs + 7 * N + rym + xm);
  P.f[8] = ldp<T, LD>(fs + 8 * N + ryp + xp);
  P.f[9] = ldp<T, LD>(fs + 9 * N + ryp + xm);
  P.f[10] = ldp<T, LD>(fs + 10 * N + rym + xp);
  // directions with e_z = +1 come from z-1; at z = 1 they bounce off the bottom plate:
  // f_i(x, t) = f*_ibar(x, t-1)
  P.f[5] = lo ? ldp<T, LD>(fs + 6 * N + c) : ldp<T, LD>(fs + 5 * N + M.zm + o0 + x);
  P.f[11] = lo ? ldp<T, LD>(fs + 12 * N + c) : ldp<T, LD>(fs + 11 * N + M.zm + o0 + xm);
  P.f[14] = lo ? ldp<T, LD>(fs + 13 * N + c) : ldp<T, LD>(fs + 14 * N + M.zm + o0 + xp);
  P.f[15] = lo ? ldp<T, LD>(fs + 16 * N + c) : ldp<T, LD>(fs + 15 * N + M.zm + om + x);
  P.f[18] = lo ? ldp<T, LD>(fs + 17 * N + c) : ldp<T, LD>(fs + 18 * N + M.zm + op + x);
  // directions with e_z = -1 come from z+1; at z = nz-2 they bounce off the top plate
  P.f[6] = hi ? ldp<T, LD>(fs + 5 * N + c) : ldp<T, LD>(fs + 6 * N + M.zp + o0 + x);
  P.f[12] = hi ? ldp<T, LD>(fs + 11 * N + c) : ldp<T, LD>(fs + 12 * N + M.zp + o0 + xp);
  P.f[13] = hi ? ldp<T, LD>(fs + 14 * N + c) : ldp<T, LD>(fs + 13 * N + M.zp + o0 + xm);
  P.f[16] = hi ? ldp<T, LD>(fs + 15 * N + c) : ldp<T, LD>(fs + 16 * N + M.zp + op + x);
  P.f[17] = hi ? ldp<T, LD>(fs + 18 * N + c) : ldp<T, LD>(fs + 17 * N + M.zp + om + x);
}

// The same for a cell (x, y, z) of a lattice array.
template <typename T>
__device__ __forceinline__ void pull(const T* __restrict__ fs, const Geom& G, int x, int y, int z,
                                     Pop<T>& P) {
  pull_map<T, LD_NC>(fs, G, lattice_map(G, z), x, y, z == 1, z == G.nz - 2, P);
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

// Collision of one cell, grouped so that every opposite pair shares its even and odd parts:
//   f^eq,s = w [drho + rho (3 eu + 4.5 eu^2 - 1.5 u^2)]            Eq. 22 (never forms w + small)
//   f^eq   = w rho [1 + 3 eu + 4.5 eu^2 - 1.5 u^2]                 Eq. 15
//   S      = w [3 eF + 9 eu eF - 3 uF]                             Eq. 18 with c_s^2 = 1/3
//   f*     = f - (f - f^eq)/tau + (1 - 1/(2 tau)) S                Eqs. 14 / 23
// With omega = 1/tau, s = 1 - omega/2, base = drho - 1.5 rho u^2 (shifted) or rho - 1.5 rho u^2:
//   f*_(+-e) = (1 - omega) f_(+-e) + E +- O
//   E = w [omega base - 3 s uF] + eu (4.5 w omega rho eu + 9 w s eF)     even in e
//   O = 3 w omega rho eu + 3 w s eF                                       odd in e
// (same terms as Eq. 23, summed in this fixed order.)
template <typename T>
struct PairConst { T k0, a, b3, c, d; };   // k0 = w(omega base - 3 s uF), a = 4.5 w omega rho, c = 3 w omega rho, d = 3 w s, b3 = 3 d

template <typename T>
__device__ __forceinline__ void collide_pair(T& fa, T& fb, T eu, T eF, const PairConst<T>& K, T keep) {
  const T m = K.d * eF;                       // 3 w s eF
  const T E = fmaf_t(eu, fmaf_t(K.a, eu, K.b3 * eF), K.k0);
  const T O = fmaf_t(K.c, eu, m);
  fa = fmaf_t(keep, fa, E + O);
  fb = fmaf_t(keep, fb, E - O);
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
  const T keep = T(1) - C.omega;
  const T t0 = C.omega * base - (T(3) * C.somega) * uF;   // omega base + s (-3 uF)
  const T orho = C.omega * rho;
  const T w0 = T(1) / T(3), w1 = T(1) / T(18), w2 = T(1) / T(36);
  PairConst<T> K1, K2;
  K1.k0 = w1 * t0; K1.a = (T(4.5) * w1) * orho; K1.c = (T(3) * w1) * orho; K1.d = (T(3) * w1) * C.somega; K1.b3 = (T(9) * w1) * C.somega;
  K2.k0 = w2 * t0; K2.a = (T(4.5) * w2) * orho; K2.c = (T(3) * w2) * orho; K2.d = (T(3) * w2) * C.somega; K2.b3 = (T(9) * w2) * C.somega;
  T* f = P.f;
  f[0] = fmaf_t(keep, f[0], w0 * t0);
  collide_pair<T>(f[1], f[2], ux, Fx, K1, keep);
  collide_pair<T>(f[3], f[4], uy, Fy, K1, keep);
  collide_pair<T>(f[5], f[6], uz, Fz, K1, keep);
  collide_pair<T>(f[7], f[8], ux + uy, Fx + Fy, K2, keep);
  collide_pair<T>(f[9], f[10], ux - uy, Fx - Fy, K2, keep);
  collide_pair<T>(f[11], f[12], ux + uz, Fx + Fz, K2, keep);
  collide_pair<T>(f[13], f[14], ux - uz, Fx - Fz, K2, keep);
  collide_pair<T>(f[15], f[16], uy + uz, Fy + Fz, K2, keep);
  collide_pair<T>(f[17], f[18], uy - uz, Fy - Fz, K2, keep);
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

// One LB step, one thread per fluid cell (the two-steps-per-launch form is nh_lb2.cuh).
template <typename T, bool SHIFTED>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? 6 : 3)
lb_step_kernel(const T* __restrict__ fsrc, T* __restrict__ fdst, const T* __restrict__ Flc,
               Geom G, LbConst<T> C, int reverse) {
  // Programmatic dependent launch between consecutive LB steps (launch_lb sets the attribute only then): the next
  // step's CTAs become resident as ours retire, and wait below before they read anything.  Every thread waits
  // (also the ones that then leave), so that this grid cannot complete before its predecessor has.
  grid_launch_dependents();
  const unsigned k = sweep_block(reverse) * blockDim.x + threadIdx.x;
  int x, y, z;
  cell_of(k < G.nfluid ? k : 0u, G, x, y, z);
  const size_t c = (size_t)k + G.plane;
  grid_dependency_wait();
  if (k >= G.nfluid) return;
  Pop<T> P;
  pull<T>(fsrc, G, x, y, z, P);
  T Fx = T(0), Fy = T(0), Fz = T(0);
  if (C.use_flc) { Fx = __ldg(Flc + c); Fy = __ldg(Flc + G.N + c); Fz = __ldg(Flc + 2 * G.N + c); }
  collide<T, SHIFTED>(P, Fx, Fy, Fz, C);
#pragma unroll
  for (int i = 0; i < Q; ++i) fdst[(size_t)i * G.N + c] = P.f[i];
}

// Small lattices (the whole grid resident on the SMs at once, the populations in the L2): `nsteps` LB steps in
// ONE cooperative launch, a grid-wide barrier between steps, one thread per fluid cell for the whole launch.
// Between two director updates the force is frozen, so it is read once.  Same gather and
// collision as lb_step_kernel (bit-identical); the gathers go to the L2 (written by other CTAs one barrier ago).
// Step s reads f[s & 1] and writes f[(s + 1) & 1].
template <typename T, bool SHIFTED>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? 4 : 2)
lb_resident_kernel(T* __restrict__ fa, T* __restrict__ fb, const T* __restrict__ Flc, Geom G, LbConst<T> C, int nsteps) {
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  const bool on = k < G.nfluid;
  int x, y, z;
  cell_of(on ? k : 0u, G, x, y, z);
  const size_t c = (size_t)(on ? k : 0u) + G.plane;
  const PlaneMap M = lattice_map(G, z);
  T Fx = T(0), Fy = T(0), Fz = T(0);
  if (C.use_flc && on) { Fx = __ldg(Flc + c); Fy = __ldg(Flc + G.N + c); Fz = __ldg(Flc + 2 * G.N + c); }
  T* src = fa;
  T* dst = fb;
  for (int s = 0; s < nsteps; ++s) {
    if (on) {
      Pop<T> P;
      pull_map<T, LD_CG>(src, G, M, x, y, z == 1, z == G.nz - 2, P);
      collide<T, SHIFTED>(P, Fx, Fy, Fz, C);
#pragma unroll
      for (int i = 0; i < Q; ++i) dst[(size_t)i * G.N + c] = P.f[i];
    }
    grid.sync();
    T* t = src; src = dst; dst = t;
  }
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
