// nh_fd.cuh -- finite-difference kernels of the director side, baseline ("direct") variant:
// one thread per fluid cell, neighbours read straight from global memory through L1.
// nh_fd_tile.cuh holds the shared-memory tiled variant that the library uses by default; this
// one stays as the simple form the tiled one is checked against (option NH_OPT_FD_DIRECT).
//
// PAPER.md:101-112 (Sec. II.B): central differences Eq. 13, solid node values fixed, director
// equation Eq. 9 with D, W of Eq. 5, predictor-corrector;
// molecular field Eq. 10 for the one-constant energy with chiral term (
// DESIGN.md readings G1, G2); elastic stress Eq. 6 and force Eq. 12.
#pragma once
#include <cuda_runtime.h>
#include "nh_lb.cuh"

namespace nh {

template <typename T>
struct FdConst {
  T K;          // Frank modulus
  T Kq0;        // K * q0
  T inv_gamma1; // 1/gamma1
  T xi;         // flow alignment
  T dt;         // Delta t_FD = r
  T al[6];      // Leslie viscosities alpha1, alpha2, alpha3, alpha4', alpha5, alpha6 (Eqs. 3, 12)
  int visc;     // any of them non-zero: the force includes the viscous stress
  T W0;         // bulk anchoring along z: h_z += W0 n_z (reading G14)
};

template <typename T> struct V3 { T x, y, z; };

template <typename T>
__device__ __forceinline__ V3<T> ld3(const T* __restrict__ a, size_t N, unsigned c) {
  V3<T> v; v.x = __ldg(a + c); v.y = __ldg(a + N + c); v.z = __ldg(a + 2 * N + c); return v;
}
template <typename T> __device__ __forceinline__ V3<T> operator-(V3<T> a, V3<T> b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
template <typename T> __device__ __forceinline__ V3<T> operator+(V3<T> a, V3<T> b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
template <typename T> __device__ __forceinline__ V3<T> operator*(T s, V3<T> a) { return {s * a.x, s * a.y, s * a.z}; }
template <typename T> __device__ __forceinline__ T dot(V3<T> a, V3<T> b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <typename T> __device__ __forceinline__ V3<T> cross(V3<T> a, V3<T> b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
__device__ __forceinline__ float rsq(float s) { return 1.0f / sqrtf(s); }
__device__ __forceinline__ double rsq(double s) { return 1.0 / sqrt(s); }
template <typename T> __device__ __forceinline__ V3<T> unit(V3<T> v) { return rsq(dot(v, v)) * v; }

// Six neighbours of a cell (periodic x, y; z neighbours always exist for a fluid cell).
struct Nbr { unsigned xm, xp, ym, yp, zm, zp, c; };
__device__ __forceinline__ Nbr neighbours(const Geom& G, int x, int y, int z) {
  const int nx = G.nx;
  const unsigned row = (unsigned)z * G.plane + (unsigned)y * nx;
  const unsigned rz = (unsigned)z * G.plane;
  Nbr b;
  b.c = row + x;
  b.xm = row + (x == 0 ? nx - 1 : x - 1);
  b.xp = row + (x == nx - 1 ? 0 : x + 1);
  b.ym = rz + (unsigned)(y == 0 ? G.ny - 1 : y - 1) * nx + x;
  b.yp = rz + (unsigned)(y == G.ny - 1 ? 0 : y + 1) * nx + x;
  b.zm = b.c - G.plane;
  b.zp = b.c + G.plane;
  return b;
}

template <typename T>
__device__ __forceinline__ V3<T> director_rhs_tail(const FdConst<T>& C, V3<T> R, V3<T> m, V3<T> dxm, V3<T> dym,
                                                   V3<T> dzm, V3<T> u, V3<T> dxu, V3<T> dyu, V3<T> dzu);

// Right-hand side of Eq. 9 at one cell from the centre value and the six neighbours of m and u.
//   h   = K lap m - 2 K q0 curl m + W0 m_z z_hat   (7-point Laplacian, central curl; bulk anchoring)
//   R   = h/gamma1 + xi m.D - (u.grad) m + W.m,   D, W as printed in Eq. 5
//   R  <- R - (m.R) m                      (reading G3)
// d?m = central difference of m along ?, s?m = m(+) + m(-) along ?; same for u.
template <typename T>
__device__ __forceinline__ V3<T> director_rhs(const FdConst<T>& C, V3<T> m, V3<T> mxm, V3<T> mxp,
                                              V3<T> mym, V3<T> myp, V3<T> mzm, V3<T> mzp, V3<T> u,
                                              V3<T> dxu, V3<T> dyu, V3<T> dzu) {
  const T h = T(0.5);
  const V3<T> dxm = h * (mxp - mxm), dym = h * (myp - mym), dzm = h * (mzp - mzm);
  const V3<T> lap = ((mxp + mxm) + (myp + mym)) + (mzp + mzm) - T(6) * m;
  const V3<T> curl = {dym.z - dzm.y, dzm.x - dxm.z, dxm.y - dym.x};
  V3<T> R = C.inv_gamma1 * (C.K * lap - (T(2) * C.Kq0) * curl);
  R.z += C.inv_gamma1 * (C.W0 * m.z);
  return director_rhs_tail(C, R, m, dxm, dym, dzm, u, dxu, dyu, dzu);
}

// The same from a given h/gamma1 (three-constant energy, nh_frank3.cuh): flow terms and projection.
template <typename T>
__device__ __forceinline__ V3<T> director_rhs_tail(const FdConst<T>& C, V3<T> R, V3<T> m, V3<T> dxm, V3<T> dym,
                                                   V3<T> dzm, V3<T> u, V3<T> dxu, V3<T> dyu, V3<T> dzu) {
  const T h = T(0.5);
  // velocity gradient G[b][c] = d_b u_c: rows dxu, dyu, dzu
  // (m.D)_mu = m_a D_{a mu} = 1/2 m_a (d_a u_mu + d_mu u_a)
  // (W.m)_mu = W_{mu a} m_a = 1/2 (d_a u_mu - d_mu u_a) m_a
  // so  xi m.D + W.m = (xi+1)/2 (m.grad) u + (xi-1)/2 grad(u).m
  const V3<T> mgu = m.x * dxu + (m.y * dyu + m.z * dzu);            // m_a d_a u_mu
  const V3<T> gum = {dot(dxu, m), dot(dyu, m), dot(dzu, m)};       // d_mu u_a m_a
  const V3<T> adv = u.x * dxm + (u.y * dym + u.z * dzm);            // u_a d_a m_mu
  R = R + (h * (C.xi + T(1))) * mgu + (h * (C.xi - T(1))) * gum - adv;
  return R - dot(m, R) * m;
}

// RHS at cell (x, y, z) of field m with velocity u, everything from global memory.
template <typename T>
__device__ __forceinline__ V3<T> rhs_global(const FdConst<T>& C, const T* __restrict__ m,
                                            const T* __restrict__ u, size_t N, const Nbr& b,
                                            bool with_flow) {
  const V3<T> mc = ld3(m, N, b.c);
  V3<T> uc = {T(0), T(0), T(0)}, dxu = uc, dyu = uc, dzu = uc;
  if (with_flow) {
    uc = ld3(u, N, b.c);
    dxu = T(0.5) * (ld3(u, N, b.xp) - ld3(u, N, b.xm));
    dyu = T(0.5) * (ld3(u, N, b.yp) - ld3(u, N, b.ym));
    dzu = T(0.5) * (ld3(u, N, b.zp) - ld3(u, N, b.zm));
  }
  return director_rhs(C, mc, ld3(m, N, b.xm), ld3(m, N, b.xp), ld3(m, N, b.ym), ld3(m, N, b.yp),
                      ld3(m, N, b.zm), ld3(m, N, b.zp), uc, dxu, dyu, dzu);
}

// Predictor: n^P = normalise(n + dt R[n]) on fluid cells.
template <typename T>
__global__ void __launch_bounds__(256)
predictor_direct_kernel(const T* __restrict__ n, const T* __restrict__ u, T* __restrict__ nP,
                        Geom G, FdConst<T> C, int with_flow) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const Nbr b = neighbours(G, x, y, z);
  const V3<T> k1 = rhs_global(C, n, u, G.N, b, with_flow != 0);
  const V3<T> v = unit(ld3(n, G.N, b.c) + C.dt * k1);
  nP[b.c] = v.x; nP[G.N + b.c] = v.y; nP[2 * G.N + b.c] = v.z;
}

// Corrector: n' = normalise(n + dt/2 (R[n] + R[n^P])), same u.
template <typename T>
__global__ void __launch_bounds__(256)
corrector_direct_kernel(const T* __restrict__ n, const T* __restrict__ nP, const T* __restrict__ u,
                        T* __restrict__ nnew, Geom G, FdConst<T> C, int with_flow) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const Nbr b = neighbours(G, x, y, z);
  const V3<T> k1 = rhs_global(C, n, u, G.N, b, with_flow != 0);
  const V3<T> k2 = rhs_global(C, nP, u, G.N, b, with_flow != 0);
  const V3<T> v = unit(ld3(n, G.N, b.c) + (T(0.5) * C.dt) * (k1 + k2));
  nnew[b.c] = v.x; nnew[G.N + b.c] = v.y; nnew[2 * G.N + b.c] = v.z;
}

// Column b of the elastic stress at one cell: s_a = sigma_{a b},
//   sigma_ab = -K d_a n . d_b n  +  K q0 (n x d_a n)_b          (Eq. 6; the chiral part is
//   -K q0 eps_{mu b c} n_mu d_a n_c written as a cross product)
template <typename T>
__device__ __forceinline__ V3<T> stress_column(const FdConst<T>& C, int b, V3<T> n, V3<T> dxn,
                                               V3<T> dyn, V3<T> dzn) {
  const V3<T> db = (b == 0) ? dxn : (b == 1 ? dyn : dzn);
  const V3<T> cx = cross(n, dxn), cy = cross(n, dyn), cz = cross(n, dzn);
  const T qx = (b == 0) ? cx.x : (b == 1 ? cx.y : cx.z);
  const T qy = (b == 0) ? cy.x : (b == 1 ? cy.y : cy.z);
  const T qz = (b == 0) ? cz.x : (b == 1 ? cz.y : cz.z);
  return {C.Kq0 * qx - C.K * dot(dxn, db), C.Kq0 * qy - C.K * dot(dyn, db), C.Kq0 * qz - C.K * dot(dzn, db)};
}

template <typename T>
__device__ __forceinline__ void viscous_add_h(const FdConst<T>& C, V3<T> n, V3<T> hg, V3<T> dxu, V3<T> dyu,
                                              V3<T> dzu, V3<T>& sx, V3<T>& sy, V3<T>& sz);

// Leslie viscous stress, Eq. 3 with alpha4 -> alpha4' as in the force of Eq. 12
// (PAPER.md:97-99), added column by column: s?[a] += sigma^v_{a ?},
//   sigma^v_ab = a1 n_a n_b (n.D.n) + a2 n_b N_a + a3 n_a N_b + a4' D_ab + a5 n_b (n.D)_a + a6 n_a (n.D)_b
// D as printed in Eq. 5; N of Eq. 4 from Eq. 9: N = h/gamma1 + xi n.D, projected perpendicular
// to n (reading G22); h = K lap n - 2 K q0 curl n as in the director equation.
// d?n, d?u: central differences; lap: 7-point Laplacian of n.
template <typename T>
__device__ __forceinline__ void viscous_add(const FdConst<T>& C, V3<T> n, V3<T> dxn, V3<T> dyn, V3<T> dzn,
                                            V3<T> lap, V3<T> dxu, V3<T> dyu, V3<T> dzu,
                                            V3<T>& sx, V3<T>& sy, V3<T>& sz) {
  const V3<T> curl = {dyn.z - dzn.y, dzn.x - dxn.z, dxn.y - dyn.x};
  V3<T> hg = C.inv_gamma1 * (C.K * lap - (T(2) * C.Kq0) * curl);
  hg.z += C.inv_gamma1 * (C.W0 * n.z);
  viscous_add_h(C, n, hg, dxu, dyu, dzu, sx, sy, sz);
}

// The same from a given h/gamma1 (any energy).
template <typename T>
__device__ __forceinline__ void viscous_add_h(const FdConst<T>& C, V3<T> n, V3<T> hg, V3<T> dxu, V3<T> dyu,
                                              V3<T> dzu, V3<T>& sx, V3<T>& sy, V3<T>& sz) {
  const T h2 = T(0.5);
  const T Dxy = h2 * (dxu.y + dyu.x), Dxz = h2 * (dxu.z + dzu.x), Dyz = h2 * (dyu.z + dzu.y);
  const V3<T> Dx = {dxu.x, Dxy, Dxz}, Dy = {Dxy, dyu.y, Dyz}, Dz = {Dxz, Dyz, dzu.z};   // columns = rows
  const V3<T> nD = {dot(n, Dx), dot(n, Dy), dot(n, Dz)};
  const V3<T> A = hg + C.xi * nD;
  const V3<T> N = A - dot(n, A) * n;
  const T nnD = dot(n, nD);
  const V3<T> w = C.al[1] * N + C.al[4] * nD;                  // multiplies n_b
  sx = sx + (C.al[0] * n.x * nnD + C.al[2] * N.x + C.al[5] * nD.x) * n + n.x * w + C.al[3] * Dx;
  sy = sy + (C.al[0] * n.y * nnD + C.al[2] * N.y + C.al[5] * nD.y) * n + n.y * w + C.al[3] * Dy;
  sz = sz + (C.al[0] * n.z * nnD + C.al[2] * N.z + C.al[5] * nD.z) * n + n.z * w + C.al[3] * Dz;
}

// sigma_{. b} at the cell (x, y, z) read from global memory; zero on the plate layers (reading G6).
template <typename T>
__device__ __forceinline__ V3<T> stress_column_at(const FdConst<T>& C, int b, const T* __restrict__ n,
                                                  const T* __restrict__ u, const Geom& G, int x, int y, int z) {
  if (z == 0 || z == G.nz - 1) return {T(0), T(0), T(0)};
  const Nbr q = neighbours(G, x, y, z);
  const T h = T(0.5);
  const V3<T> nc = ld3(n, G.N, q.c);
  const V3<T> nxp = ld3(n, G.N, q.xp), nxm = ld3(n, G.N, q.xm), nyp = ld3(n, G.N, q.yp), nym = ld3(n, G.N, q.ym);
  const V3<T> nzp = ld3(n, G.N, q.zp), nzm = ld3(n, G.N, q.zm);
  const V3<T> dxn = h * (nxp - nxm), dyn = h * (nyp - nym), dzn = h * (nzp - nzm);
  V3<T> s = stress_column(C, b, nc, dxn, dyn, dzn);
  if (C.visc) {
    const V3<T> lap = ((nxp + nxm) + (nyp + nym)) + (nzp + nzm) - T(6) * nc;
    const V3<T> dxu = h * (ld3(u, G.N, q.xp) - ld3(u, G.N, q.xm)), dyu = h * (ld3(u, G.N, q.yp) - ld3(u, G.N, q.ym));
    const V3<T> dzu = h * (ld3(u, G.N, q.zp) - ld3(u, G.N, q.zm));
    V3<T> vx = {T(0), T(0), T(0)}, vy = vx, vz = vx;
    viscous_add(C, nc, dxn, dyn, dzn, lap, dxu, dyu, dzu, vx, vy, vz);
    s = s + (b == 0 ? vx : (b == 1 ? vy : vz));
  }
  return s;
}

// Force (Eq. 12): F_a = sum_b [sigma_ab(x + e_b) - sigma_ab(x - e_b)]/2, sigma = sigma^e (+ sigma^v).
template <typename T>
__global__ void __launch_bounds__(256)
force_direct_kernel(const T* __restrict__ n, const T* __restrict__ u, T* __restrict__ F, Geom G, FdConst<T> C) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nfluid) return;
  int x, y, z;
  cell_of(k, G, x, y, z);
  const int xm = (x == 0) ? G.nx - 1 : x - 1, xp = (x == G.nx - 1) ? 0 : x + 1;
  const int ym = (y == 0) ? G.ny - 1 : y - 1, yp = (y == G.ny - 1) ? 0 : y + 1;
  V3<T> f = stress_column_at(C, 0, n, u, G, xp, y, z) - stress_column_at(C, 0, n, u, G, xm, y, z);
  f = f + (stress_column_at(C, 1, n, u, G, x, yp, z) - stress_column_at(C, 1, n, u, G, x, ym, z));
  f = f + (stress_column_at(C, 2, n, u, G, x, y, z + 1) - stress_column_at(C, 2, n, u, G, x, y, z - 1));
  const size_t c = (size_t)k + G.plane;
  F[c] = T(0.5) * f.x; F[G.N + c] = T(0.5) * f.y; F[2 * G.N + c] = T(0.5) * f.z;
}

// ---- set_director helpers ---------------------------------------------------------------------
// flag |= 1 if any input vector has zero or non-finite length
__global__ void __launch_bounds__(256)
check_director_kernel(const double* __restrict__ in, size_t N, int* __restrict__ flag) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= N) return;
  const double a = in[c], b = in[N + c], d = in[2 * N + c];
  const double len = sqrt(a * a + b * b + d * d);
  if (!(len > 0.0) || !isfinite(len)) atomicOr(flag, 1);
}

// normalise in FP64, overwrite the plates with z_hat, store in the device precision
// into n, n^P and the corrector's output buffer (so its plates are set too)
// `bad` (may be null): the flag of check_director_kernel; if it is set nothing is stored (the lattice keeps its
// director and nh_set_director reports NH_EINVAL), so the host need not wait for the check before it enqueues this
template <typename T>
__global__ void __launch_bounds__(256)
store_director_kernel(const double* __restrict__ in, T* __restrict__ n, T* __restrict__ nP,
                      T* __restrict__ nnew, Geom G, const int* __restrict__ bad) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= G.N) return;
  if (bad && *bad) return;
  const unsigned zz = (unsigned)(c / G.plane);
  double a = 0.0, b = 0.0, d = 1.0;
  if (zz != 0 && zz != (unsigned)G.nz - 1) {
    a = in[c]; b = in[G.N + c]; d = in[2 * G.N + c];
    const double len = sqrt(a * a + b * b + d * d);
    a /= len; b /= len; d /= len;
  }
  n[c] = (T)a; n[G.N + c] = (T)b; n[2 * G.N + c] = (T)d;
  nP[c] = (T)a; nP[G.N + c] = (T)b; nP[2 * G.N + c] = (T)d;
  nnew[c] = (T)a; nnew[G.N + c] = (T)b; nnew[2 * G.N + c] = (T)d;
}

// Free plates (anchoring = 1; reading G23): the plate layers copy the adjacent
// fluid layer, so the stencils next to them see a zero normal derivative.  One thread per (c, y, x).
template <typename T>
__global__ void __launch_bounds__(256) mirror_plates_kernel(T* __restrict__ n, Geom G) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= 3u * G.plane) return;
  const unsigned comp = k / G.plane, xy = k - comp * G.plane;
  T* a = n + (size_t)comp * G.N + xy;
  a[0] = a[G.plane];
  a[(size_t)(G.nz - 1) * G.plane] = a[(size_t)(G.nz - 2) * G.plane];
}

__global__ void __launch_bounds__(256) fill_f64_kernel(double* __restrict__ p, double v, size_t n) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c < n) p[c] = v;
}

// device precision -> FP64 staging for nh_get_fields (whole grid, 3 components; `out` may sit in mapped host memory)
template <typename T>
__global__ void __launch_bounds__(256)
widen3_kernel(const T* __restrict__ a, double* __restrict__ out, size_t n3) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c < n3) out[c] = (double)a[c];
}

}  // namespace nh
