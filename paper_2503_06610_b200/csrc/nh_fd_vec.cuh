// nh_fd_vec.cuh -- director predictor / corrector with FOUR cells per thread along x (the default where rows
// are a multiple of 64 cells; nh_fd_tile.cuh keeps the one-cell-per-thread tiled form for every other width,
// nh_fd.cuh the plain form both are checked against).
//
// Same operation as director_tile_kernel: PAPER.md:101-112 (Sec. II.B) -- central differences Eq. 13, solid node
// values fixed, director equation Eq. 9 with D, W of Eq. 5, molecular field Eq. 10
// for the one-constant energy with chiral term (readings G1, G2), predictor
// and corrector with the same u, rate projected perpendicular to n and the result
// renormalised (reading G3).
//
// Why: the one-cell-per-thread kernels are bound by instruction issue (about 295 instructions per cell, 30 scalar
// shared-memory loads among them).  Here a thread owns 4 consecutive cells of a row: its stencil values arrive as
// 16-byte shared-memory loads (x neighbours come with the row), results leave as 16-byte stores, the loop, the
// staging and the address arithmetic are shared by four cells, and the halves of the central differences are
// folded into the coefficients.  The right-hand side is accumulated COMPONENT BY COMPONENT so that only one
// component's stencil (22 values for the 4 cells) is live at a time:
//   with raw differences  d_a f = f(x + e_a) - f(x - e_a)  (twice Eq. 13):
//   R_mu  = (K/gamma1) lap m_mu - (K q0/gamma1) (curl' m)_mu + (W0/gamma1) m_z delta_{mu z}     h/gamma1, Eq. 10
//         + (xi+1)/4 m_a d_a u_mu + (xi-1)/4 (d_mu u_a) m_a                    xi m.D + W.m, Eq. 5 as printed
//         - 1/2 u_a d_a m_mu                                                   advection
//   (curl' from raw differences; (xi+1)/4 = 1/2 (xi+1)/2 etc.: the same terms as director_rhs in nh_fd.cuh,
//   summed in a different order -- results agree to rounding, not bit for bit).
//
// Tile: 64 x 8 cells, 16 x 8 = 128 threads.  March along z with cp.async-staged planes (halo ring of one cell,
// periodic wrap applied when the plane is fetched, every copy 16 bytes), three plane slots per field: z and z+1 in
// use, z+2 in flight; the values of planes z-1 and z at the thread's own cells are carried in registers.  52 KB of
// shared memory per CTA: four CTAs = 16 warps per SM.  (Measured on the way: with six slots and three planes in
// flight only two CTAs fit an SM and the kernel got SLOWER, 0.062 against 0.056 ms: with four cells per thread
// the limit is warps per scheduler, not bytes in flight.)
#pragma once
#include <cuda_runtime.h>
#include "nh_fd.cuh"
#include "nh_fd_tile.cuh"

namespace nh {

constexpr int VX = 4;                    // cells per thread along x
constexpr int VTX = 16, VTY = 8;         // threads of a tile along x, y
constexpr int VW = VX * VTX;             // tile width in cells
constexpr int VTHREADS = VTX * VTY;
constexpr int VSLOTS = 3;                // staged planes per field: z, z+1 in use, z+2 in flight

template <int H>
struct VShape {
  static constexpr int CO = 4;                   // column of the tile's first cell (16-byte aligned for float and double)
  static constexpr int RS = CO + VW + 4;         // row stride in elements
  static constexpr int PY = VTY + 2 * H;
  static constexpr int CELLS = PY * RS;          // one component
  static constexpr int ELEMS = 3 * CELLS;
};

// What one thread copies of every plane: 16-byte chunks, fixed for the whole march.  A row is the chunk left of
// the tile (it holds the x halo; periodic), VW / EPV interior chunks and the chunk right of the tile.
template <typename T, int H>
struct VStager {
  using S = VShape<H>;
  static constexpr int EPV = 16 / (int)sizeof(T);
  static constexpr int CPR = VW / EPV + 2;
  static constexpr int NCH = 3 * S::PY * CPR;
  static constexpr int NOPS = (NCH + VTHREADS - 1) / VTHREADS;
  static_assert(H <= EPV, "the halo must fit one 16-byte chunk");
  unsigned g[NOPS];     // global element offset without the z term
  unsigned s[NOPS];     // shared byte offset, ~0u: nothing

  __device__ __forceinline__ void init(const Geom& G, int x0, int y0) {
#pragma unroll
    for (int k = 0; k < NOPS; ++k) {
      const int o = (int)threadIdx.x + k * VTHREADS;
      g[k] = 0u; s[k] = ~0u;
      if (o < NCH) {
        const int comp = o / (S::PY * CPR);
        const int rem = o - comp * (S::PY * CPR);
        const int row = rem / CPR, ch = rem - row * CPR;
        int gx = x0 + (ch - 1) * EPV;                       // nx is a multiple of VW, so a chunk never straddles the wrap
        if (gx < 0) gx += G.nx;
        if (gx >= G.nx) gx -= G.nx;
        int gy = (y0 + row - H) % G.ny; if (gy < 0) gy += G.ny;
        g[k] = (unsigned)comp * (unsigned)G.N + (unsigned)gy * (unsigned)G.nx + (unsigned)gx;
        s[k] = (unsigned)((comp * S::CELLS + row * S::RS + S::CO + (ch - 1) * EPV) * (int)sizeof(T));
      }
    }
  }
  __device__ __forceinline__ void fetch(const T* __restrict__ src, unsigned slot) const {
#pragma unroll
    for (int k = 0; k < NOPS; ++k)
      if (s[k] != ~0u) cp_async_bytes<16>(slot + s[k], src + g[k]);
  }
};

// four consecutive elements from shared or global memory (16-byte aligned)
__device__ __forceinline__ void ld4(const float* p, float (&v)[4]) {
  const float4 q = *reinterpret_cast<const float4*>(p);
  v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
}
__device__ __forceinline__ void ld4(const double* p, double (&v)[4]) {
  const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2);
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
__device__ __forceinline__ void st4(float* p, const float (&v)[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void st4(double* p, const double (&v)[4]) {
  *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
  *reinterpret_cast<double2*>(p + 2) = make_double2(v[2], v[3]);
}

// raw differences and (optionally) the 7-point Laplacian of ONE component for the 4 cells at staged offset `o`:
// zm, c = the cells' values one plane below and in this plane (registers), pc, pzp = staged planes z and z+1;
// zp returns the values one plane above
template <typename T, int H, bool LAP>
__device__ __forceinline__ void stencil4(const T (&zm)[4], const T* pc, const T* pzp, int o, const T (&c)[4],
                                         T (&zp)[4], T (&dx)[4], T (&dy)[4], T (&dz)[4], T (&lap)[4]) {
  using S = VShape<H>;
  T ym[4], yp[4];
  const T xl = pc[o - 1], xr = pc[o + VX];
  ld4(pc + o - S::RS, ym);
  ld4(pc + o + S::RS, yp);
  ld4(pzp + o, zp);
#pragma unroll
  for (int j = 0; j < VX; ++j) {
    const T xm = (j == 0) ? xl : c[j - 1];
    const T xp = (j == VX - 1) ? xr : c[j + 1];
    dx[j] = xp - xm; dy[j] = yp[j] - ym[j]; dz[j] = zp[j] - zm[j];
    if (LAP) lap[j] = fmaf_t(T(-6), c[j], ((xp + xm) + (yp[j] + ym[j])) + (zp[j] + zm[j]));
  }
}

template <typename T>
constexpr size_t director_vec_smem_bytes() { return (size_t)2 * VSLOTS * VShape<1>::ELEMS * sizeof(T); }

// STAGE 0: field = n;   k1 = R[n];   out_m = n^P = unit(n + dt k1), a_out = n + dt/2 k1
// STAGE 1: field = n^P; k2 = R[n^P]; out_m = n'  = unit(a_in + dt/2 k2)
template <typename T, int STAGE>
__global__ void __launch_bounds__(VTHREADS, sizeof(T) == 4 ? 4 : 1)
director_vec_kernel(const T* __restrict__ m, const T* __restrict__ u, const T* __restrict__ a_in,
                    T* __restrict__ out_m, T* __restrict__ a_out, Geom G, FdConst<T> C, int with_flow, int zchunk) {
  using S = VShape<1>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);          // [VSLOTS][ELEMS]  m
  T* su = sm + VSLOTS * S::ELEMS;                  // [VSLOTS][ELEMS]  u
  const int tx = threadIdx.x % VTX, ty = threadIdx.x / VTX;
  const int x0 = blockIdx.x * VW, y0 = blockIdx.y * VTY;
  const int z0 = 1 + blockIdx.z * zchunk;
  const int z1 = min(z0 + zchunk - 1, G.nz - 2);   // last plane this CTA updates
  const int x = x0 + VX * tx, y = y0 + ty;
  const bool active = y < G.ny;                    // (nx is a multiple of the tile width)
  const bool flow = with_flow != 0;
  const int oc = (ty + 1) * S::RS + S::CO + VX * tx;
  constexpr unsigned SLOT_BYTES = S::ELEMS * sizeof(T);
  const unsigned sm_addr = smem_u32(sm), su_addr = smem_u32(su);
  VStager<T, 1> st;
  st.init(G, x0, y0);

  // planes z0-1, z0, z0+1 -> slots 0, 1, 2
  const T* msrc = m + (size_t)(z0 - 1) * G.plane;
  const T* usrc = u + (size_t)(z0 - 1) * G.plane;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    st.fetch(msrc, sm_addr + k * SLOT_BYTES);
    if (flow) st.fetch(usrc, su_addr + k * SLOT_BYTES);
    msrc += G.plane; usrc += G.plane;
  }
  cp_async_commit();
  cp_async_wait_all();
  __syncthreads();
  // the own cells' values at planes z-1 and z, carried along the march
  T mzm[3][4], mc[3][4], uzm[3][4], uc[3][4];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    ld4(sm + k * S::CELLS + oc, mzm[k]);
    ld4(sm + S::ELEMS + k * S::CELLS + oc, mc[k]);
#pragma unroll
    for (int j = 0; j < VX; ++j) { uzm[k][j] = T(0); uc[k][j] = T(0); }
    if (flow) {
      ld4(su + k * S::CELLS + oc, uzm[k]);
      ld4(su + S::ELEMS + k * S::CELLS + oc, uc[k]);
    }
  }
  int sc = 1, sp = 2, sf = 0;                      // slots of plane z, z+1, and the one to refill (it held z-1)
  T an[3][4];                                      // corrector: a = n + dt/2 k1 of the own cells, one plane ahead
#pragma unroll
  for (int k = 0; k < 3; ++k) {
#pragma unroll
    for (int j = 0; j < VX; ++j) an[k][j] = T(0);
  }

  const unsigned N = (unsigned)G.N;
  unsigned c = (unsigned)z0 * G.plane + (unsigned)y * (unsigned)G.nx + (unsigned)x;
  const T hdt = T(0.5) * C.dt;
  const T kl = C.inv_gamma1 * C.K, kc = C.inv_gamma1 * C.Kq0, kw = C.inv_gamma1 * C.W0;
  const T c1 = T(0.25) * (C.xi + T(1)), c2 = T(0.25) * (C.xi - T(1));
  if (STAGE == 1 && active) {
#pragma unroll
    for (int k = 0; k < 3; ++k) ld4(a_in + c + k * N, an[k]);
  }

  for (int z = z0; z <= z1; ++z) {
    cp_async_wait_all();     // plane z+1 (enqueued one iteration ago)
    __syncthreads();         // ... is visible to everyone, and everyone is done with plane z-1
    if (z < z1) {            // plane z+2 goes where plane z-1 was
      st.fetch(msrc, sm_addr + sf * SLOT_BYTES);
      if (flow) st.fetch(usrc, su_addr + sf * SLOT_BYTES);
      msrc += G.plane; usrc += G.plane;
    }
    cp_async_commit();
    {
      T av[3][4];
      if (STAGE == 1) {      // a = n + dt/2 k1 of the own cells: this plane's was requested one iteration ago
#pragma unroll
        for (int k = 0; k < 3; ++k) {
#pragma unroll
          for (int j = 0; j < VX; ++j) av[k][j] = an[k][j];
          if (active && z < z1) ld4(a_in + c + G.plane + k * N, an[k]);
        }
      }
      const T* pc = sm + sc * S::ELEMS;
      const T* pzp = sm + sp * S::ELEMS;
      T R[3][4];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
#pragma unroll
        for (int j = 0; j < VX; ++j) R[k][j] = T(0);
      }
      if (flow) {
        const T* qc = su + sc * S::ELEMS;
        const T* qzp = su + sp * S::ELEMS;
#pragma unroll
        for (int k = 0; k < 3; ++k) {              // component k of u
          T zp[4], dx[4], dy[4], dz[4], unused[4];
          stencil4<T, 1, false>(uzm[k], qc + k * S::CELLS, qzp + k * S::CELLS, oc, uc[k], zp, dx, dy, dz, unused);
#pragma unroll
          for (int j = 0; j < VX; ++j) {
            // (xi+1)/4 m_a d_a u_k  into R_k;   (xi-1)/4 (d_mu u_k) m_k  into R_mu
            const T s = fmaf_t(mc[0][j], dx[j], fmaf_t(mc[1][j], dy[j], mc[2][j] * dz[j]));
            R[k][j] = fmaf_t(c1, s, R[k][j]);
            const T t = c2 * mc[k][j];
            R[0][j] = fmaf_t(t, dx[j], R[0][j]);
            R[1][j] = fmaf_t(t, dy[j], R[1][j]);
            R[2][j] = fmaf_t(t, dz[j], R[2][j]);
            uzm[k][j] = uc[k][j]; uc[k][j] = zp[j];          // one plane up: uzm now holds u of THIS plane
          }
        }
      }
      T mzp[3][4];
#pragma unroll
      for (int k = 0; k < 3; ++k) {                // component k of the director field
        T dx[4], dy[4], dz[4], lap[4];
        stencil4<T, 1, true>(mzm[k], pc + k * S::CELLS, pzp + k * S::CELLS, oc, mc[k], mzp[k], dx, dy, dz, lap);
#pragma unroll
        for (int j = 0; j < VX; ++j) {
          // (K/gamma1) lap m_k - 1/2 u . d m_k  into R_k   (u of this plane sits in uzm by now; 0 without flow)
          const T adv = fmaf_t(uzm[0][j], dx[j], fmaf_t(uzm[1][j], dy[j], uzm[2][j] * dz[j]));
          R[k][j] = fmaf_t(T(-0.5), adv, fmaf_t(kl, lap[j], R[k][j]));
          // -(K q0/gamma1) curl':  curl'_x = d_y m_z - d_z m_y,  curl'_y = d_z m_x - d_x m_z,  curl'_z = d_x m_y - d_y m_x
          if (k == 0) { R[1][j] = fmaf_t(-kc, dz[j], R[1][j]); R[2][j] = fmaf_t(kc, dy[j], R[2][j]); }
          if (k == 1) { R[2][j] = fmaf_t(-kc, dx[j], R[2][j]); R[0][j] = fmaf_t(kc, dz[j], R[0][j]); }
          if (k == 2) { R[0][j] = fmaf_t(-kc, dy[j], R[0][j]); R[1][j] = fmaf_t(kc, dx[j], R[1][j]); }
        }
      }
      T o0[4], o1[4], o2[4], b0[4], b1[4], b2[4];
#pragma unroll
      for (int j = 0; j < VX; ++j) {
        V3<T> r = {R[0][j], R[1][j], fmaf_t(kw, mc[2][j], R[2][j])};
        const V3<T> mm = {mc[0][j], mc[1][j], mc[2][j]};
        r = r - dot(mm, r) * mm;                   // reading G3
        V3<T> v;
        if (STAGE == 0) {
          v = unit_fast(mm + C.dt * r);
          const V3<T> a = mm + hdt * r;
          b0[j] = a.x; b1[j] = a.y; b2[j] = a.z;
        } else {
          const V3<T> a = {av[0][j], av[1][j], av[2][j]};
          v = unit_fast(a + hdt * r);
        }
        o0[j] = v.x; o1[j] = v.y; o2[j] = v.z;
      }
      if (active) {
        st4(out_m + c, o0); st4(out_m + c + N, o1); st4(out_m + c + 2 * N, o2);
        if (STAGE == 0) { st4(a_out + c, b0); st4(a_out + c + N, b1); st4(a_out + c + 2 * N, b2); }
      }
#pragma unroll
      for (int k = 0; k < 3; ++k) {
#pragma unroll
        for (int j = 0; j < VX; ++j) { mzm[k][j] = mc[k][j]; mc[k][j] = mzp[k][j]; }
      }
    }
    c += G.plane;
    const int t = sf; sf = sc; sc = sp; sp = t;
  }
  cp_async_wait_all();
}

}  // namespace nh
