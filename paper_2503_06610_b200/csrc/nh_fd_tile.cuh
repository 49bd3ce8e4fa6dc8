// nh_fd_tile.cuh -- the director side of the hot path as shared-memory tiled, z-marching kernels
// (the default; nh_fd.cuh keeps the one-thread-per-cell form they are checked against).
//
// PAPER.md:101-112 (Sec. II.B): central differences Eq. 13, solid node values fixed, director
// equation Eq. 9 with D, W of Eq. 5, predictor-corrector; molecular
// field Eq. 10 for the one-constant energy with chiral term;
// elastic stress Eq. 6 and force Eq. 12.
//
// Shape of every kernel here: a CTA owns a TX x TY column of cells and marches along z over
// `zchunk` planes.  Each xy plane of an input field (with its halo ring, periodic wrap applied
// when the plane is fetched) is staged in shared memory by cp.async (LDGSTS) into a small ring of
// plane slots, one plane ahead of the arithmetic, so every value is fetched from L2/HBM once per
// CTA and the stencil reads are shared-memory reads with constant offsets.  The centre column is
// carried in registers along z.  With VEC the 32 interior cells of a staged row travel as 16-byte
// copies (needs nx % 32 == 0) and only the halo columns as single elements; without it every
// element is its own copy (any nx, ny).
//
//   director_tile_kernel<T, 0>  predictor: k1 = R[n];   n^P = unit(n + dt k1);  a = n + dt/2 k1
//   director_tile_kernel<T, 1>  corrector: k2 = R[n^P]; n'  = unit(a + dt/2 k2)        (same u)
//   force_tile_kernel<T>        sigma once per cell (own cell + the tile's face halo), then
//                               F_a = sum_b [sigma_ab(x+e_b) - sigma_ab(x-e_b)]/2
#pragma once
#include <cuda_runtime.h>
#include "nh_fd.cuh"
#include "nh_frank3.cuh"

namespace nh {

constexpr int TX = 32;           // tile extent along x = one warp
constexpr int TY = 8;            // tile extent along y; TX*TY = 256 threads
constexpr int TILE_THREADS = TX * TY;

// ---- cp.async helpers ---------------------------------------------------------------------------
template <int BYTES>
__device__ __forceinline__ void cp_async_bytes(unsigned smem_addr, const void* gsrc) {
  if constexpr (BYTES == 16)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_addr), "l"(gsrc) : "memory");
  else if constexpr (BYTES == 8)
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(smem_addr), "l"(gsrc) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(smem_addr), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// One staged xy plane of a 3-vector field: [3][PY][RS]; the tile's first cell sits at column CO of
// row H, so that the 32 interior cells of every row start on a 16-byte boundary.
template <int H>
struct PlaneShape {
  static constexpr int CO = 4;                 // column of the tile's x0
  static constexpr int RS = 40;                // row stride (elements): CO + TX + H <= RS
  static constexpr int PX = TX + 2 * H;        // columns actually filled: CO-H .. CO+TX+H-1
  static constexpr int PY = TY + 2 * H;
  static constexpr int CELLS = PY * RS;        // elements of one component
  static constexpr int ELEMS = 3 * CELLS;
};

// What one thread copies of every plane: NOPS (global element offset without the z term, shared
// byte offset | kind) pairs, fixed for the whole march.  kind: 0 nothing, 1 one element, 2 16 bytes.
template <typename T, int H, bool VEC>
struct Stager {
  using S = PlaneShape<H>;
  static constexpr int EPV = 16 / (int)sizeof(T);
  static constexpr int CHUNKS_PER_ROW = TX / EPV;
  static constexpr int NCHUNK = VEC ? 3 * S::PY * CHUNKS_PER_ROW : 0;
  static constexpr int ELEM_PER_ROW = VEC ? 2 * H : S::PX;
  static constexpr int NELEM = 3 * S::PY * ELEM_PER_ROW;
  static constexpr int NOPS = (NCHUNK + NELEM + TILE_THREADS - 1) / TILE_THREADS;
  unsigned g[NOPS];
  unsigned s[NOPS];

  __device__ __forceinline__ void init(const Geom& G, int x0, int y0) {
#pragma unroll
    for (int k = 0; k < NOPS; ++k) {
      const int o = (int)threadIdx.x + k * TILE_THREADS;
      int comp = 0, row = 0, col = 0, kind = 0;      // col: staged column
      if (o < NCHUNK) {
        comp = o / (S::PY * CHUNKS_PER_ROW);
        const int rem = o - comp * (S::PY * CHUNKS_PER_ROW);
        row = rem / CHUNKS_PER_ROW;
        col = S::CO + (rem - row * CHUNKS_PER_ROW) * EPV;
        kind = 2;
      } else if (o - NCHUNK < NELEM) {
        const int e = o - NCHUNK;
        comp = e / (S::PY * ELEM_PER_ROW);
        const int rem = e - comp * (S::PY * ELEM_PER_ROW);
        row = rem / ELEM_PER_ROW;
        const int j = rem - row * ELEM_PER_ROW;
        col = VEC ? (j < H ? S::CO - H + j : S::CO + TX + (j - H)) : S::CO - H + j;
        kind = 1;
      }
      int gx = (x0 + col - S::CO) % G.nx; if (gx < 0) gx += G.nx;
      int gy = (y0 + row - H) % G.ny; if (gy < 0) gy += G.ny;
      g[k] = (unsigned)comp * (unsigned)G.N + (unsigned)gy * (unsigned)G.nx + (unsigned)gx;
      s[k] = (unsigned)((comp * S::CELLS + row * S::RS + col) * (int)sizeof(T)) | (unsigned)kind;
    }
  }
  // enqueue the copy of one plane: `src` = field + z*plane, `slot` = shared address of the slot
  __device__ __forceinline__ void fetch(const T* __restrict__ src, unsigned slot) const {
#pragma unroll
    for (int k = 0; k < NOPS; ++k) {
      const unsigned kind = s[k] & 3u, dst = slot + (s[k] & ~3u);
      if (VEC && kind == 2u) cp_async_bytes<16>(dst, src + g[k]);
      else if (kind == 1u) cp_async_bytes<(int)sizeof(T)>(dst, src + g[k]);
    }
  }
};

template <typename T, int H>
__device__ __forceinline__ V3<T> lds3(const T* plane, int off) {
  using S = PlaneShape<H>;
  return {plane[off], plane[S::CELLS + off], plane[2 * S::CELLS + off]};
}
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// v/|v|.  FP32: MUFU.RSQ plus one Newton step (<= 1 ulp); FP64: CUDA's rsqrt (<= 2 ulp).
__device__ __forceinline__ float rsq_fast(float s) {
  const float y = rsqrtf(s);
  return y * (1.5f - 0.5f * s * y * y);
}
__device__ __forceinline__ double rsq_fast(double s) { return rsqrt(s); }
template <typename T> __device__ __forceinline__ V3<T> unit_fast(V3<T> v) { return rsq_fast(dot(v, v)) * v; }

// ---- predictor / corrector ----------------------------------------------------------------------
// STAGE 0: m = n;   k1 = R[n];   out_m = n^P = unit(n + dt k1), a_out = n + dt/2 k1
// STAGE 1: m = n^P; k2 = R[n^P]; out_m = n'  = unit(a_in + dt/2 k2)
// The same u(t) serves both stages.  n + dt/2 (k1 + k2) is evaluated as
// (n + dt/2 k1) + dt/2 k2 so that k1 is not recomputed; the difference is one rounding.
// Dynamic shared memory: director_smem_bytes<T>().  Ring of 3 plane slots per field: while plane
// z is worked on, z+1 is resident and z+2 is in flight into the slot z-1 has left.
constexpr int DIR_SLOTS = 3;
template <typename T>
constexpr size_t director_smem_bytes() { return (size_t)2 * DIR_SLOTS * PlaneShape<1>::ELEMS * sizeof(T); }

template <typename T, int STAGE, bool VEC>
__global__ void __launch_bounds__(TILE_THREADS)
director_tile_kernel(const T* __restrict__ m, const T* __restrict__ u, const T* __restrict__ a_in,
                     T* __restrict__ out_m, T* __restrict__ a_out, Geom G, FdConst<T> C,
                     int with_flow, int zchunk) {
  using S = PlaneShape<1>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);          // [DIR_SLOTS][ELEMS]  m
  T* su = sm + DIR_SLOTS * S::ELEMS;               // [DIR_SLOTS][ELEMS]  u
  const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int z0 = 1 + blockIdx.z * zchunk;
  const int z1 = min(z0 + zchunk - 1, G.nz - 2);   // last plane this CTA updates
  const int x = x0 + tx, y = y0 + ty;
  const bool active = (x < G.nx) && (y < G.ny);
  const bool flow = with_flow != 0;
  const int oc = (ty + 1) * S::RS + S::CO + tx;    // own cell inside a staged plane
  constexpr unsigned SLOT_BYTES = S::ELEMS * sizeof(T);
  const unsigned sm_addr = smem_u32(sm), su_addr = smem_u32(su);
  Stager<T, 1, VEC> st;
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
  V3<T> mzm = lds3<T, 1>(sm, oc);
  V3<T> mc = lds3<T, 1>(sm + S::ELEMS, oc);
  const V3<T> zero = {T(0), T(0), T(0)};
  V3<T> uzm = zero, uc = zero;
  if (flow) {
    uzm = lds3<T, 1>(su, oc);
    uc = lds3<T, 1>(su + S::ELEMS, oc);
  }
  int sc = 1, sp = 2, sf = 0;                      // slots of plane z, z+1, and the one to refill
  unsigned c = (unsigned)z0 * G.plane + (unsigned)y * (unsigned)G.nx + (unsigned)x;
  const unsigned N = (unsigned)G.N;
  const T hdt = T(0.5) * C.dt;
  // corrector: a = n + dt/2 k1 of the own cell, read one plane ahead so that its latency hides behind the stencil
  V3<T> a_next = zero;
  if (STAGE == 1 && active) a_next = {a_in[c], a_in[c + N], a_in[c + 2 * N]};

  for (int z = z0; z <= z1; ++z) {
    cp_async_wait_all();     // plane z+1 (enqueued one iteration ago)
    __syncthreads();         // ... is visible to everyone, and everyone is done with plane z-1
    if (z < z1) {            // plane z+2 goes where plane z-1 was
      st.fetch(msrc, sm_addr + sf * SLOT_BYTES);
      if (flow) st.fetch(usrc, su_addr + sf * SLOT_BYTES);
      msrc += G.plane; usrc += G.plane;
    }
    cp_async_commit();
    const V3<T> a_own = a_next;
    if (STAGE == 1 && active && z < z1) {
      const unsigned cn = c + G.plane;
      a_next = {a_in[cn], a_in[cn + N], a_in[cn + 2 * N]};
    }
    const T* pm = sm + sc * S::ELEMS;
    const V3<T> mzp = lds3<T, 1>(sm + sp * S::ELEMS, oc);
    V3<T> uzp = zero, dxu = zero, dyu = zero, dzu = zero;
    if (flow) {
      const T* pu = su + sc * S::ELEMS;
      uzp = lds3<T, 1>(su + sp * S::ELEMS, oc);
      dxu = T(0.5) * (lds3<T, 1>(pu, oc + 1) - lds3<T, 1>(pu, oc - 1));
      dyu = T(0.5) * (lds3<T, 1>(pu, oc + S::RS) - lds3<T, 1>(pu, oc - S::RS));
      dzu = T(0.5) * (uzp - uzm);
    }
    const V3<T> k = director_rhs(C, mc, lds3<T, 1>(pm, oc - 1), lds3<T, 1>(pm, oc + 1),
                                 lds3<T, 1>(pm, oc - S::RS), lds3<T, 1>(pm, oc + S::RS), mzm, mzp,
                                 uc, dxu, dyu, dzu);
    if (active) {
      if (STAGE == 0) {
        const V3<T> v = unit_fast(mc + C.dt * k);
        const V3<T> a = mc + hdt * k;
        out_m[c] = v.x; out_m[c + N] = v.y; out_m[c + 2 * N] = v.z;
        a_out[c] = a.x; a_out[c + N] = a.y; a_out[c + 2 * N] = a.z;
      } else {
        const V3<T> v = unit_fast(a_own + hdt * k);
        out_m[c] = v.x; out_m[c + N] = v.y; out_m[c + 2 * N] = v.z;
      }
    }
    mzm = mc; mc = mzp;
    uzm = uc; uc = uzp;
    const int t = sf; sf = sc; sc = sp; sp = t;
    c += G.plane;
  }
  cp_async_wait_all();
}

// ---- elastic stress and force -------------------------------------------------------------------
// sigma_ab = -K d_a n . d_b n + K q0 (n x d_a n)_b   (Eq. 6; reading G1),
// zero on the plate layers (reading G6);  F_a = sum_b [sigma_ab(x+e_b) - sigma_ab(x-e_b)]/2
// (Eq. 12 last term).
//
// March over planes p = z0-1 .. z1+1.  At plane p every thread evaluates grad n and the full
// sigma ONCE at its own cell: the columns sigma_.x and sigma_.y go to a double-buffered shared
// plane, sigma_.z stays in registers (the z neighbours of a cell are the same thread one plane
// earlier and later).  The first 80 threads also evaluate the one column that the tile's face
// halo needs (sigma_.y on the two y faces, sigma_.x on the two x faces).  One plane later the
// force of plane p-1 is complete.  n is staged with a halo of 2 (ring of 4 planes: p-1, p, p+1
// in use, p+2 in flight).
constexpr int FORCE_SLOTS = 4;
struct SigShape {                       // sigma_.x / sigma_.y plane: [2 columns][3][TY+2][TX+2]
  static constexpr int PX = TX + 2, PY = TY + 2, CELLS = PX * PY, ELEMS = 6 * CELLS;
};
template <typename T, bool VISC = false>
constexpr size_t force_smem_bytes() {
  return ((size_t)(VISC ? 2 : 1) * FORCE_SLOTS * PlaneShape<2>::ELEMS + 2 * SigShape::ELEMS) * sizeof(T);
}

// grad n at the staged position `o` of plane slots (zm, c, zp)
template <typename T>
__device__ __forceinline__ void grad_staged(const T* pzm, const T* pc, const T* pzp, int o,
                                            V3<T>& n, V3<T>& dxn, V3<T>& dyn, V3<T>& dzn) {
  using S = PlaneShape<2>;
  const T h = T(0.5);
  n = lds3<T, 2>(pc, o);
  dxn = h * (lds3<T, 2>(pc, o + 1) - lds3<T, 2>(pc, o - 1));
  dyn = h * (lds3<T, 2>(pc, o + S::RS) - lds3<T, 2>(pc, o - S::RS));
  dzn = h * (lds3<T, 2>(pzp, o) - lds3<T, 2>(pzm, o));
}
// the same plus the 7-point Laplacian (the viscous stress needs the molecular field)
template <typename T>
__device__ __forceinline__ void grad_lap_staged(const T* pzm, const T* pc, const T* pzp, int o,
                                                V3<T>& n, V3<T>& dxn, V3<T>& dyn, V3<T>& dzn, V3<T>& lap) {
  using S = PlaneShape<2>;
  const T h = T(0.5);
  n = lds3<T, 2>(pc, o);
  const V3<T> xp = lds3<T, 2>(pc, o + 1), xm = lds3<T, 2>(pc, o - 1);
  const V3<T> yp = lds3<T, 2>(pc, o + S::RS), ym = lds3<T, 2>(pc, o - S::RS);
  const V3<T> zp = lds3<T, 2>(pzp, o), zm = lds3<T, 2>(pzm, o);
  dxn = h * (xp - xm); dyn = h * (yp - ym); dzn = h * (zp - zm);
  lap = ((xp + xm) + (yp + ym)) + (zp + zm) - T(6) * n;
}
// sigma^e + sigma^v at the staged position `o`: all three columns
template <typename T>
__device__ __forceinline__ void stress_visc_staged(const FdConst<T>& C, const T* nzm, const T* nc, const T* nzp,
                                                   const T* uzm, const T* uc, const T* uzp, int o,
                                                   V3<T>& sx, V3<T>& sy, V3<T>& sz) {
  V3<T> n, dxn, dyn, dzn, lap, u0, dxu, dyu, dzu;
  grad_lap_staged(nzm, nc, nzp, o, n, dxn, dyn, dzn, lap);
  grad_staged(uzm, uc, uzp, o, u0, dxu, dyu, dzu);
  stress_all(C, n, dxn, dyn, dzn, sx, sy, sz);
  viscous_add(C, n, dxn, dyn, dzn, lap, dxu, dyu, dzu, sx, sy, sz);
}

// All three columns of sigma at once: c_a = n x d_a n,  g_ab = d_a n . d_b n (symmetric),
// sigma_ab = K q0 (c_a)_b - K g_ab.  s[b] holds the column (sigma_xb, sigma_yb, sigma_zb).
template <typename T>
__device__ __forceinline__ void stress_all(const FdConst<T>& C, V3<T> n, V3<T> dx, V3<T> dy, V3<T> dz,
                                           V3<T>& sx, V3<T>& sy, V3<T>& sz) {
  const V3<T> cx = cross(n, dx), cy = cross(n, dy), cz = cross(n, dz);
  const T gxx = dot(dx, dx), gyy = dot(dy, dy), gzz = dot(dz, dz);
  const T gxy = dot(dx, dy), gxz = dot(dx, dz), gyz = dot(dy, dz);
  sx = {C.Kq0 * cx.x - C.K * gxx, C.Kq0 * cy.x - C.K * gxy, C.Kq0 * cz.x - C.K * gxz};
  sy = {C.Kq0 * cx.y - C.K * gxy, C.Kq0 * cy.y - C.K * gyy, C.Kq0 * cz.y - C.K * gyz};
  sz = {C.Kq0 * cx.z - C.K * gxz, C.Kq0 * cy.z - C.K * gyz, C.Kq0 * cz.z - C.K * gzz};
}

// three-constant energy (row f2): sigma^e_{a b} = -d_a n_c pi_{b c} with the LOCAL pi of nh_frank3.cuh;
// the viscous part takes h from the buffer that h3_kernel has filled (h needs pi at the neighbours)
template <typename T>
__device__ __forceinline__ void stress3_staged(const FdConst<T>& C, const Frank3<T>& K3, bool visc,
                                               const T* nzm, const T* nc, const T* nzp,
                                               const T* uzm, const T* uc, const T* uzp, int o,
                                               const T* __restrict__ hbuf, unsigned cell, unsigned N, bool cell_ok,
                                               V3<T>& sx, V3<T>& sy, V3<T>& sz) {
  V3<T> n, dxn, dyn, dzn, px, py, pz, dfdn;
  grad_staged(nzm, nc, nzp, o, n, dxn, dyn, dzn);
  frank3_local(K3, n, dxn, dyn, dzn, px, py, pz, dfdn);
  sx = {-dot(dxn, px), -dot(dyn, px), -dot(dzn, px)};
  sy = {-dot(dxn, py), -dot(dyn, py), -dot(dzn, py)};
  sz = {-dot(dxn, pz), -dot(dyn, pz), -dot(dzn, pz)};
  if (visc) {
    V3<T> u0, dxu, dyu, dzu;
    grad_staged(uzm, uc, uzp, o, u0, dxu, dyu, dzu);
    V3<T> h = {T(0), T(0), T(0)};
    if (cell_ok) h = {hbuf[cell], hbuf[cell + N], hbuf[cell + 2 * N]};
    viscous_add_h(C, n, C.inv_gamma1 * h, dxu, dyu, dzu, sx, sy, sz);
  }
}

// VISC: the Leslie viscous stress is added (Eq. 12 in full, row f1): u is staged like n.
// FR3: three-constant Frank energy (K3, hbuf).
template <typename T, bool VEC, bool VISC, bool FR3 = false>
__global__ void __launch_bounds__(TILE_THREADS)
force_tile_kernel(const T* __restrict__ n, const T* __restrict__ u, T* __restrict__ Fout, Geom G,
                  FdConst<T> C, int zchunk, Frank3<T> K3 = Frank3<T>(), const T* __restrict__ hbuf = nullptr) {
  using S = PlaneShape<2>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sn = reinterpret_cast<T*>(smem_raw);                 // [FORCE_SLOTS][S::ELEMS]
  T* ssig = sn + FORCE_SLOTS * S::ELEMS;                  // [2][SigShape::ELEMS]
  T* su = ssig + 2 * SigShape::ELEMS;                     // [FORCE_SLOTS][S::ELEMS] (VISC only)
  const unsigned su_addr = smem_u32(su);
  const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int z0 = 1 + blockIdx.z * zchunk;
  const int z1 = min(z0 + zchunk - 1, G.nz - 2);
  const int x = x0 + tx, y = y0 + ty;
  const bool active = (x < G.nx) && (y < G.ny);
  const int on = (ty + 2) * S::RS + S::CO + tx;           // own cell in a staged n plane
  const int os = (ty + 1) * SigShape::PX + (tx + 1);      // own cell in a sigma plane
  constexpr unsigned SLOT_BYTES = S::ELEMS * sizeof(T);
  const unsigned sn_addr = smem_u32(sn);
  Stager<T, 2, VEC> st;
  st.init(G, x0, y0);
  // face-halo duty of threads 0..79: which staged cell, which column (0: sigma_.x, 1: sigma_.y)
  int hn = -1, hs = 0, hcol = 0;
  unsigned hcell = 0;                                     // in-plane index of the halo cell (FR3 + VISC: h buffer)
  // in-plane index of the own cell, wrapped: threads hanging over the edge of the lattice still
  // compute sigma for their periodic image, which active neighbours read
  const unsigned ownw = (unsigned)(y % G.ny) * (unsigned)G.nx + (unsigned)(x % G.nx);
  {
    const int t = threadIdx.x;
    int hx = 0, hy = 0;                                    // tile-relative, -1 .. TX / TY
    if (t < 2 * TX) { hx = t % TX; hy = (t < TX) ? -1 : TY; hcol = 1; }
    else if (t < 2 * TX + 2 * TY) { const int q = t - 2 * TX; hy = q % TY; hx = (q < TY) ? -1 : TX; hcol = 0; }
    if (t < 2 * TX + 2 * TY) {
      hn = (hy + 2) * S::RS + S::CO + hx;
      hs = (hy + 1) * SigShape::PX + (hx + 1) + 3 * hcol * SigShape::CELLS;
      int gx = (x0 + hx) % G.nx; if (gx < 0) gx += G.nx;
      int gy = (y0 + hy) % G.ny; if (gy < 0) gy += G.ny;
      hcell = (unsigned)gy * (unsigned)G.nx + (unsigned)gx;
    }
  }
  const int pfirst = z0 - 1, plast = z1 + 1;
  // n planes needed at p: p-1, p, p+1 (none for a plate, sigma = 0 there); slot of plane z: z & 3
  const int zlo = max(pfirst - 1, 0), zhi = min(plast + 1, G.nz - 1);
  int zf = zlo;                                            // next plane to fetch
  const T* src = n + (size_t)zlo * G.plane;
  const T* usrc = u + (size_t)zlo * G.plane;
  for (; zf <= zlo + 2; ++zf) {
    st.fetch(src, sn_addr + (zf & 3) * SLOT_BYTES);
    if (VISC) { st.fetch(usrc, su_addr + (zf & 3) * SLOT_BYTES); usrc += G.plane; }
    src += G.plane;
  }
  cp_async_commit();
  const V3<T> zero = {T(0), T(0), T(0)};
  V3<T> szA = zero, szB = zero;                           // sigma_.z at planes p-2, p-1
  unsigned c = (unsigned)(z0 - 1) * G.plane + (unsigned)y * (unsigned)G.nx + (unsigned)x;   // cell (x, y, p)
  const unsigned N = (unsigned)G.N;

  for (int p = pfirst; p <= plast; ++p) {
    cp_async_wait_all();
    __syncthreads();
    if (zf <= zhi && zf <= p + 2) {                        // keep one plane ahead of p+1
      st.fetch(src, sn_addr + (zf & 3) * SLOT_BYTES);
      if (VISC) { st.fetch(usrc, su_addr + (zf & 3) * SLOT_BYTES); usrc += G.plane; }
      src += G.plane; ++zf;
    }
    cp_async_commit();
    T* sig = ssig + (p & 1) * SigShape::ELEMS;
    V3<T> szC = zero;
    if (p == 0 || p == G.nz - 1) {
#pragma unroll
      for (int q = 0; q < 6; ++q) sig[q * SigShape::CELLS + os] = T(0);
      if (hn >= 0) {
#pragma unroll
        for (int q = 0; q < 3; ++q) sig[q * SigShape::CELLS + hs] = T(0);
      }
    } else {
      const T* pzm = sn + ((p - 1) & 3) * S::ELEMS;
      const T* pc = sn + (p & 3) * S::ELEMS;
      const T* pzp = sn + ((p + 1) & 3) * S::ELEMS;
      V3<T> nn, dxn, dyn, dzn, sx, sy;
      const T* uzm = su + ((p - 1) & 3) * S::ELEMS;
      const T* uc = su + (p & 3) * S::ELEMS;
      const T* uzp = su + ((p + 1) & 3) * S::ELEMS;
      if (FR3) {
        stress3_staged(C, K3, VISC, pzm, pc, pzp, uzm, uc, uzp, on, hbuf, ownw + (unsigned)p * G.plane, N, true, sx, sy, szC);
      } else if (VISC) {
        stress_visc_staged(C, pzm, pc, pzp, uzm, uc, uzp, on, sx, sy, szC);
      } else {
        grad_staged(pzm, pc, pzp, on, nn, dxn, dyn, dzn);
        stress_all(C, nn, dxn, dyn, dzn, sx, sy, szC);
      }
      sig[0 * SigShape::CELLS + os] = sx.x; sig[1 * SigShape::CELLS + os] = sx.y; sig[2 * SigShape::CELLS + os] = sx.z;
      sig[3 * SigShape::CELLS + os] = sy.x; sig[4 * SigShape::CELLS + os] = sy.y; sig[5 * SigShape::CELLS + os] = sy.z;
      if (hn >= 0) {
        V3<T> sh;
        if (FR3) {
          // the halo cell's index: same plane, tile-relative (hx, hy) wrapped periodically
          V3<T> hx, hy, hz;
          stress3_staged(C, K3, VISC, pzm, pc, pzp, uzm, uc, uzp, hn, hbuf, hcell + (unsigned)p * G.plane, N, true, hx, hy, hz);
          sh = hcol == 0 ? hx : hy;
        } else if (VISC) {
          V3<T> hx, hy, hz;
          stress_visc_staged(C, pzm, pc, pzp, uzm, uc, uzp, hn, hx, hy, hz);
          sh = hcol == 0 ? hx : hy;
        } else {
          grad_staged(pzm, pc, pzp, hn, nn, dxn, dyn, dzn);
          sh = stress_column(C, hcol, nn, dxn, dyn, dzn);
        }
        sig[0 * SigShape::CELLS + hs] = sh.x;
        sig[1 * SigShape::CELLS + hs] = sh.y;
        sig[2 * SigShape::CELLS + hs] = sh.z;
      }
    }
    // force of plane p-1: its sigma_.x / sigma_.y plane was written one iteration ago
    if (p > z0 && active) {
      const T* sg = ssig + ((p - 1) & 1) * SigShape::ELEMS + os;
      constexpr int CS = SigShape::CELLS, PXs = SigShape::PX;
      const T fx = (sg[0 * CS + 1] - sg[0 * CS - 1]) + (sg[3 * CS + PXs] - sg[3 * CS - PXs]) + (szC.x - szA.x);
      const T fy = (sg[1 * CS + 1] - sg[1 * CS - 1]) + (sg[4 * CS + PXs] - sg[4 * CS - PXs]) + (szC.y - szA.y);
      const T fz = (sg[2 * CS + 1] - sg[2 * CS - 1]) + (sg[5 * CS + PXs] - sg[5 * CS - PXs]) + (szC.z - szA.z);
      const unsigned cm = c - G.plane;
      Fout[cm] = T(0.5) * fx; Fout[cm + N] = T(0.5) * fy; Fout[cm + 2 * N] = T(0.5) * fz;
    }
    szA = szB; szB = szC;
    c += G.plane;
  }
  cp_async_wait_all();
}

// ---- predictor / corrector with the three-constant energy (row f2) --------------------------------
// h_m = -df/dn_m + d_b pi_{b m} needs pi at the six neighbours, so the march is the force kernel's:
// at plane p every thread evaluates pi (rows pi_x., pi_y. to a double-buffered shared plane, pi_z. in
// registers) and df/dn at its own cell, the first 80 threads also the row the tile's face halo needs;
// one plane later h of plane p-1 is complete and the director's rate follows (flow terms and
// projection shared with the one-constant path).  The own cell's column of m and u is carried in
// registers (plane p-2 is being overwritten in the ring by then).
//   STAGE 0: out_m = n^P = unit(m + dt k1), a_out = m + dt/2 k1;  STAGE 1: out_m = unit(a_in + dt/2 k2)
//   STAGE 2: out_m = h itself (for N of the viscous stress in the force kernel)
template <typename T, int STAGE, bool VEC>
__global__ void __launch_bounds__(TILE_THREADS)
director3_tile_kernel(const T* __restrict__ m, const T* __restrict__ u, const T* __restrict__ a_in,
                      T* __restrict__ out_m, T* __restrict__ a_out, Geom G, FdConst<T> C, Frank3<T> K3,
                      int with_flow, int zchunk) {
  using S = PlaneShape<2>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sn = reinterpret_cast<T*>(smem_raw);                 // [FORCE_SLOTS][S::ELEMS]  m
  T* ssig = sn + FORCE_SLOTS * S::ELEMS;                  // [2][SigShape::ELEMS]     pi_x., pi_y.
  T* su = ssig + 2 * SigShape::ELEMS;                     // [FORCE_SLOTS][S::ELEMS]  u
  const unsigned su_addr = smem_u32(su);
  const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int z0 = 1 + blockIdx.z * zchunk;
  const int z1 = min(z0 + zchunk - 1, G.nz - 2);
  const int x = x0 + tx, y = y0 + ty;
  const bool active = (x < G.nx) && (y < G.ny);
  const bool flow = with_flow != 0;
  const int on = (ty + 2) * S::RS + S::CO + tx;
  const int os = (ty + 1) * SigShape::PX + (tx + 1);
  constexpr unsigned SLOT_BYTES = S::ELEMS * sizeof(T);
  const unsigned sn_addr = smem_u32(sn);
  Stager<T, 2, VEC> st;
  st.init(G, x0, y0);
  int hn = -1, hs = 0, hcol = 0;
  {
    const int t = threadIdx.x;
    int hx = 0, hy = 0;
    if (t < 2 * TX) { hx = t % TX; hy = (t < TX) ? -1 : TY; hcol = 1; }
    else if (t < 2 * TX + 2 * TY) { const int q = t - 2 * TX; hy = q % TY; hx = (q < TY) ? -1 : TX; hcol = 0; }
    if (t < 2 * TX + 2 * TY) {
      hn = (hy + 2) * S::RS + S::CO + hx;
      hs = (hy + 1) * SigShape::PX + (hx + 1) + 3 * hcol * SigShape::CELLS;
    }
  }
  const int pfirst = z0 - 1, plast = z1 + 1;
  const int zlo = max(pfirst - 1, 0), zhi = min(plast + 1, G.nz - 1);
  int zf = zlo;
  const T* src = m + (size_t)zlo * G.plane;
  const T* usrc = u + (size_t)zlo * G.plane;
  for (; zf <= zlo + 2; ++zf) {
    st.fetch(src, sn_addr + (zf & 3) * SLOT_BYTES);
    if (flow) st.fetch(usrc, su_addr + (zf & 3) * SLOT_BYTES);
    src += G.plane; usrc += G.plane;
  }
  cp_async_commit();
  const V3<T> zero = {T(0), T(0), T(0)};
  V3<T> pzA = zero, pzB = zero;                           // pi_z. at planes p-2, p-1
  V3<T> dfB = zero;                                       // df/dn at plane p-1
  V3<T> mA = zero, mB = zero, uA = zero, uB = zero;       // own cell of m, u at planes p-2, p-1
  unsigned c = (unsigned)(z0 - 1) * G.plane + (unsigned)y * (unsigned)G.nx + (unsigned)x;   // cell (x, y, p)
  const unsigned N = (unsigned)G.N;
  const T hdt = T(0.5) * C.dt;

  for (int p = pfirst; p <= plast; ++p) {
    cp_async_wait_all();
    __syncthreads();
    if (zf <= zhi && zf <= p + 2) {
      st.fetch(src, sn_addr + (zf & 3) * SLOT_BYTES);
      if (flow) st.fetch(usrc, su_addr + (zf & 3) * SLOT_BYTES);
      src += G.plane; usrc += G.plane; ++zf;
    }
    cp_async_commit();
    // corrector: a of the cell whose rate completes in this iteration, requested before the stencil work
    V3<T> a_own = zero;
    if (STAGE == 1 && active && p > z0) {
      const unsigned cm = c - G.plane;
      a_own = {a_in[cm], a_in[cm + N], a_in[cm + 2 * N]};
    }
    T* sig = ssig + (p & 1) * SigShape::ELEMS;
    const T* pc = sn + (p & 3) * S::ELEMS;
    const T* pzm = sn + ((p - 1) & 3) * S::ELEMS;
    const T* pzp = sn + ((p + 1) & 3) * S::ELEMS;
    const bool plate = (p == 0 || p == G.nz - 1);
    // pi and df/dn of plane p at the own cell (zero gradient inside the plates)
    V3<T> mC, dxm = zero, dym = zero, dzm = zero, px, py, pzC, dfC;
    if (plate) mC = lds3<T, 2>(pc, on);
    else grad_staged(pzm, pc, pzp, on, mC, dxm, dym, dzm);
    frank3_local(K3, mC, dxm, dym, dzm, px, py, pzC, dfC);
    sig[0 * SigShape::CELLS + os] = px.x; sig[1 * SigShape::CELLS + os] = px.y; sig[2 * SigShape::CELLS + os] = px.z;
    sig[3 * SigShape::CELLS + os] = py.x; sig[4 * SigShape::CELLS + os] = py.y; sig[5 * SigShape::CELLS + os] = py.z;
    if (hn >= 0) {
      V3<T> hm, hdx = zero, hdy = zero, hdz = zero, hx, hy, hz, hd;
      if (plate) hm = lds3<T, 2>(pc, hn);
      else grad_staged(pzm, pc, pzp, hn, hm, hdx, hdy, hdz);
      frank3_local(K3, hm, hdx, hdy, hdz, hx, hy, hz, hd);
      const V3<T> sh = hcol == 0 ? hx : hy;
      sig[0 * SigShape::CELLS + hs] = sh.x;
      sig[1 * SigShape::CELLS + hs] = sh.y;
      sig[2 * SigShape::CELLS + hs] = sh.z;
    }
    V3<T> uC = zero;
    if (flow) uC = lds3<T, 2>(su + (p & 3) * S::ELEMS, on);
    // the director's rate at plane p-1: its pi_x. / pi_y. plane was written one iteration ago
    if (p > z0) {
      const T* sg = ssig + ((p - 1) & 1) * SigShape::ELEMS + os;
      constexpr int CS = SigShape::CELLS, PXs = SigShape::PX;
      V3<T> h;
      h.x = T(0.5) * ((sg[0 * CS + 1] - sg[0 * CS - 1]) + (sg[3 * CS + PXs] - sg[3 * CS - PXs]) + (pzC.x - pzA.x)) - dfB.x;
      h.y = T(0.5) * ((sg[1 * CS + 1] - sg[1 * CS - 1]) + (sg[4 * CS + PXs] - sg[4 * CS - PXs]) + (pzC.y - pzA.y)) - dfB.y;
      h.z = T(0.5) * ((sg[2 * CS + 1] - sg[2 * CS - 1]) + (sg[5 * CS + PXs] - sg[5 * CS - PXs]) + (pzC.z - pzA.z)) - dfB.z;
      h.z += C.W0 * mB.z;
      const T* pm1 = sn + ((p - 1) & 3) * S::ELEMS;            // staged plane p-1 of m
      const V3<T> gxm = T(0.5) * (lds3<T, 2>(pm1, on + 1) - lds3<T, 2>(pm1, on - 1));
      const V3<T> gym = T(0.5) * (lds3<T, 2>(pm1, on + S::RS) - lds3<T, 2>(pm1, on - S::RS));
      const V3<T> gzm = T(0.5) * (mC - mA);
      V3<T> gxu = zero, gyu = zero, gzu = zero;
      if (flow) {
        const T* pu1 = su + ((p - 1) & 3) * S::ELEMS;
        gxu = T(0.5) * (lds3<T, 2>(pu1, on + 1) - lds3<T, 2>(pu1, on - 1));
        gyu = T(0.5) * (lds3<T, 2>(pu1, on + S::RS) - lds3<T, 2>(pu1, on - S::RS));
        gzu = T(0.5) * (uC - uA);
      }
      V3<T> kk = zero;
      if (STAGE != 2) kk = director_rhs_tail(C, C.inv_gamma1 * h, mB, gxm, gym, gzm, uB, gxu, gyu, gzu);
      if (active) {
        const unsigned cm = c - G.plane;
        if (STAGE == 2) {
          out_m[cm] = h.x; out_m[cm + N] = h.y; out_m[cm + 2 * N] = h.z;
        } else if (STAGE == 0) {
          const V3<T> v = unit_fast(mB + C.dt * kk);
          const V3<T> a = mB + hdt * kk;
          out_m[cm] = v.x; out_m[cm + N] = v.y; out_m[cm + 2 * N] = v.z;
          a_out[cm] = a.x; a_out[cm + N] = a.y; a_out[cm + 2 * N] = a.z;
        } else {
          const V3<T> v = unit_fast(a_own + hdt * kk);
          out_m[cm] = v.x; out_m[cm + N] = v.y; out_m[cm + 2 * N] = v.z;
        }
      }
    }
    pzA = pzB; pzB = pzC; dfB = dfC;
    mA = mB; mB = mC; uA = uB; uB = uC;
    c += G.plane;
  }
  cp_async_wait_all();
}

}  // namespace nh
