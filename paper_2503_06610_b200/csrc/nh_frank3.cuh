// nh_frank3.cuh -- the three-constant Frank energy (row f2): splay K11, twist K22, bend K33.
//
// PAPER.md:70-73 (Eqs. 7-8): f = K11/2 (div n)^2 + K22/2 (n.curl n + q0)^2 + K33/2 |n x curl n|^2,
// molecular field Eq. 10, elastic stress Eq. 6.  Discrete form (DESIGN.md
// reading G24): every derivative is the central difference of Eq. 13, |n x curl n| = |(n.grad) n|, and
//   pi_{b c} = df/d(d_b n_c) = K11 delta_bc div n + K22 T eps_{a b c} n_a + K33 n_b b_c
//   df/dn_m  = K22 T (curl n)_m + K33 b_c d_m n_c            T = n.curl n + q0,  b = (n.grad) n
//   h_m      = -df/dn_m + d_b pi_{b m}  (+ W0 n_z z_hat)     sigma^e_{a b} = -d_a n_c pi_{b c}
// which makes h exactly minus the gradient of the discrete energy.  On the plate layers grad n = 0
// (uniform director inside the solid), so pi = K22 q0 eps_{a b c} n_a there.
//
// First, straightforward form: pi and df/dn go through global buffers, one thread per cell
//   pi3_kernel      m              -> pi [9][N] (row b = pi_{b .}), dfdn [3][N]
//   h3_kernel       m, pi, dfdn    -> h [3][N]
//   rhs3_kernel     m, u, h, (a)   -> predictor / corrector outputs (same staging as nh_fd_tile.cuh)
//   force3_kernel   n, u, pi, h    -> F^LC = d_b (sigma^e + sigma^v)_ab
#pragma once
#include <cuda_runtime.h>
#include "nh_fd.cuh"

namespace nh {

template <typename T>
struct Frank3 { T K11, K22, K33, q0; };

// rows of pi and df/dn at one cell from n and its central differences
template <typename T>
__device__ __forceinline__ void frank3_local(const Frank3<T>& K, V3<T> n, V3<T> dxn, V3<T> dyn, V3<T> dzn,
                                             V3<T>& pix, V3<T>& piy, V3<T>& piz, V3<T>& dfdn) {
  const T div = dxn.x + dyn.y + dzn.z;
  const V3<T> curl = {dyn.z - dzn.y, dzn.x - dxn.z, dxn.y - dyn.x};
  const T Tw = dot(n, curl) + K.q0;
  const V3<T> b = n.x * dxn + (n.y * dyn + n.z * dzn);        // b_c = n_a d_a n_c
  const T kt = K.K22 * Tw;
  const V3<T> zero = {T(0), T(0), T(0)};
  V3<T> ex = zero, ey = zero, ez = zero;
  ex.x = K.K11 * div; ey.y = K.K11 * div; ez.z = K.K11 * div;
  // sum_a eps_{a b c} n_a for b = x, y, z as vectors over c
  const V3<T> tx = {T(0), n.z, -n.y}, ty = {-n.z, T(0), n.x}, tz = {n.y, -n.x, T(0)};
  pix = ex + kt * tx + (K.K33 * n.x) * b;
  piy = ey + kt * ty + (K.K33 * n.y) * b;
  piz = ez + kt * tz + (K.K33 * n.z) * b;
  dfdn = kt * curl + K.K33 * V3<T>{dot(b, dxn), dot(b, dyn), dot(b, dzn)};
}

__device__ __forceinline__ bool cell_of_grid(size_t c, const Geom& G, int& x, int& y, int& z) {
  if (c >= G.N) return false;
  const unsigned zz = (unsigned)(c / G.plane);
  const unsigned xy = (unsigned)(c - (size_t)zz * G.plane);
  const unsigned yy = xy / (unsigned)G.nx;
  z = (int)zz; y = (int)yy; x = (int)(xy - yy * (unsigned)G.nx);
  return true;
}

template <typename T>
__device__ __forceinline__ void grad_global(const T* __restrict__ m, size_t N, const Nbr& b,
                                            V3<T>& dx, V3<T>& dy, V3<T>& dz) {
  const T h = T(0.5);
  dx = h * (ld3(m, N, b.xp) - ld3(m, N, b.xm));
  dy = h * (ld3(m, N, b.yp) - ld3(m, N, b.ym));
  dz = h * (ld3(m, N, b.zp) - ld3(m, N, b.zm));
}

// pi and df/dn on the WHOLE grid (plate layers: zero gradient)
template <typename T>
__global__ void __launch_bounds__(256)
pi3_kernel(const T* __restrict__ m, T* __restrict__ pi, T* __restrict__ dfdn, Geom G, Frank3<T> K) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  int x, y, z;
  if (!cell_of_grid(c, G, x, y, z)) return;
  const V3<T> zero = {T(0), T(0), T(0)};
  V3<T> dx = zero, dy = zero, dz = zero;
  if (z != 0 && z != G.nz - 1) grad_global(m, G.N, neighbours(G, x, y, z), dx, dy, dz);
  V3<T> px, py, pz, d;
  frank3_local(K, ld3(m, G.N, (unsigned)c), dx, dy, dz, px, py, pz, d);
  const size_t N = G.N;
  pi[c] = px.x; pi[N + c] = px.y; pi[2 * N + c] = px.z;
  pi[3 * N + c] = py.x; pi[4 * N + c] = py.y; pi[5 * N + c] = py.z;
  pi[6 * N + c] = pz.x; pi[7 * N + c] = pz.y; pi[8 * N + c] = pz.z;
  dfdn[c] = d.x; dfdn[N + c] = d.y; dfdn[2 * N + c] = d.z;
}

// h = -df/dn + d_b pi_b. + W0 n_z z_hat on the fluid cells
template <typename T>
__global__ void __launch_bounds__(256)
h3_kernel(const T* __restrict__ m, const T* __restrict__ pi, const T* __restrict__ dfdn, T* __restrict__ h,
          Geom G, T W0) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const Nbr b = neighbours(G, x, y, z);
  const size_t N = G.N;
  const T hf = T(0.5);
  V3<T> v = hf * (ld3(pi, N, b.xp) - ld3(pi, N, b.xm));
  v = v + hf * (ld3(pi + 3 * N, N, b.yp) - ld3(pi + 3 * N, N, b.ym));
  v = v + hf * (ld3(pi + 6 * N, N, b.zp) - ld3(pi + 6 * N, N, b.zm));
  v = v - ld3(dfdn, N, b.c);
  v.z += W0 * m[2 * N + b.c];
  h[b.c] = v.x; h[N + b.c] = v.y; h[2 * N + b.c] = v.z;
}

// Predictor (STAGE 0) / corrector (STAGE 1) with h from the buffer; same hand-over as the tiled
// kernels: STAGE 0: n^P = unit(n + dt k1), a = n + dt/2 k1;  STAGE 1: n' = unit(a + dt/2 k2).
template <typename T, int STAGE>
__global__ void __launch_bounds__(256)
rhs3_kernel(const T* __restrict__ m, const T* __restrict__ u, const T* __restrict__ h,
            const T* __restrict__ a_in, T* __restrict__ out_m, T* __restrict__ a_out, Geom G,
            FdConst<T> C, int with_flow) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const Nbr b = neighbours(G, x, y, z);
  const size_t N = G.N;
  const V3<T> mc = ld3(m, N, b.c);
  V3<T> dxm, dym, dzm;
  grad_global(m, N, b, dxm, dym, dzm);
  const V3<T> zero = {T(0), T(0), T(0)};
  V3<T> uc = zero, dxu = zero, dyu = zero, dzu = zero;
  if (with_flow) {
    uc = ld3(u, N, b.c);
    grad_global(u, N, b, dxu, dyu, dzu);
  }
  const V3<T> kk = director_rhs_tail(C, C.inv_gamma1 * ld3(h, N, b.c), mc, dxm, dym, dzm, uc, dxu, dyu, dzu);
  const T hdt = T(0.5) * C.dt;
  if (STAGE == 0) {
    const V3<T> v = unit(mc + C.dt * kk);
    const V3<T> a = mc + hdt * kk;
    out_m[b.c] = v.x; out_m[N + b.c] = v.y; out_m[2 * N + b.c] = v.z;
    a_out[b.c] = a.x; a_out[N + b.c] = a.y; a_out[2 * N + b.c] = a.z;
  } else {
    const V3<T> v = unit(ld3(a_in, N, b.c) + hdt * kk);
    out_m[b.c] = v.x; out_m[N + b.c] = v.y; out_m[2 * N + b.c] = v.z;
  }
}

// column b of sigma^e (+ sigma^v) at the cell (x, y, z): sigma_{a b} = -d_a n_c pi_{b c}; 0 on the plates
template <typename T>
__device__ __forceinline__ V3<T> stress3_column_at(const FdConst<T>& C, int bcol, const T* __restrict__ n,
                                                   const T* __restrict__ u, const T* __restrict__ pi,
                                                   const T* __restrict__ h, const Geom& G, int x, int y, int z) {
  if (z == 0 || z == G.nz - 1) return {T(0), T(0), T(0)};
  const Nbr q = neighbours(G, x, y, z);
  const size_t N = G.N;
  V3<T> dxn, dyn, dzn;
  grad_global(n, N, q, dxn, dyn, dzn);
  const V3<T> prow = ld3(pi + (size_t)3 * bcol * N, N, q.c);       // pi_{b .}
  V3<T> s = {-dot(dxn, prow), -dot(dyn, prow), -dot(dzn, prow)};
  if (C.visc) {
    V3<T> dxu, dyu, dzu;
    grad_global(u, N, q, dxu, dyu, dzu);
    const V3<T> zero = {T(0), T(0), T(0)};
    V3<T> vx = zero, vy = zero, vz = zero;
    viscous_add_h(C, ld3(n, N, q.c), C.inv_gamma1 * ld3(h, N, q.c), dxu, dyu, dzu, vx, vy, vz);
    s = s + (bcol == 0 ? vx : (bcol == 1 ? vy : vz));
  }
  return s;
}

template <typename T>
__global__ void __launch_bounds__(256)
force3_kernel(const T* __restrict__ n, const T* __restrict__ u, const T* __restrict__ pi,
              const T* __restrict__ h, T* __restrict__ F, Geom G, FdConst<T> C) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const int xm = (x == 0) ? G.nx - 1 : x - 1, xp = (x == G.nx - 1) ? 0 : x + 1;
  const int ym = (y == 0) ? G.ny - 1 : y - 1, yp = (y == G.ny - 1) ? 0 : y + 1;
  V3<T> f = stress3_column_at(C, 0, n, u, pi, h, G, xp, y, z) - stress3_column_at(C, 0, n, u, pi, h, G, xm, y, z);
  f = f + (stress3_column_at(C, 1, n, u, pi, h, G, x, yp, z) - stress3_column_at(C, 1, n, u, pi, h, G, x, ym, z));
  f = f + (stress3_column_at(C, 2, n, u, pi, h, G, x, y, z + 1) - stress3_column_at(C, 2, n, u, pi, h, G, x, y, z - 1));
  const size_t c = (size_t)k + G.plane;
  F[c] = T(0.5) * f.x; F[G.N + c] = T(0.5) * f.y; F[2 * G.N + c] = T(0.5) * f.z;
}

}  // namespace nh
