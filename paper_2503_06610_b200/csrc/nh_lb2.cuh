// nh_lb2.cuh -- TWO lattice-Boltzmann steps per pass over HBM (temporal blocking through the L2).
//
// Same arithmetic as nh_lb.cuh, cell by cell and bit by bit (the same moments<> and collide<>):
// PAPER.md:118-166, Eqs. 14-23; bounce-back PAPER.md:141; periodic x, y PAPER.md:225.
// Between two director updates the force is frozen, so consecutive LB steps
// depend on each other only through the populations, and two of them can share one sweep:
//
//   phase 1, plane k:  f*(t)   = collide(gather(A))      A  = lattice array in HBM (read once)
//                      -> ring slot k mod R              the ring holds R z-planes and stays in L2
//   phase 2, plane k:  f*(t+1) = collide(gather(ring))   needs ring planes k-1, k, k+1
//                      -> B                              B  = the other lattice array (written once)
//
// One launch runs both phases as a wavefront along z.
//   Unit of work: one PIECE (256*U consecutive cells: whole rows, or a whole fraction of a row) of
//   one plane of one phase, done by one CTA.  Units are ordered -- phase 1 of planes 0..D, then
//   phase 2 of plane k and phase 1 of plane k+D+1 alternating, piece by piece inside a plane -- and
//   a CTA takes the next unit from an atomic ticket counter when it starts to run.
//   Dependencies are per-piece flags in global memory holding a number that grows with every
//   launch and strip:
//     phase 2 of (k, piece)  needs phase 1 of planes k-1, k, k+1 at the neighbouring pieces
//     phase 1 of (k, piece)  needs phase 2 of planes k-R-1 .. k-R+1 at the pieces that read the
//                            ring slot it overwrites
//   Every unit depends only on units EARLIER in ticket order, and a ticket is drawn by a CTA that
//   is already running, so whatever a CTA waits for is running or done: no deadlock, no
//   cooperative launch.  A wait longer than ~4 s sets an error flag instead of hanging the device.
//
// Strips.  The lattice is cut along y into strips of YS rows so that one strip-plane (YS x nx cells) is
// what the resident CTAs can chew and R of them fit the L2 whatever the grid: the strips are done one
// after the other, each with its own wavefront along z.  Phase 1 of a strip also computes the two
// rows next to it (the ring plane has YS + 2 rows; ring row 0 / YS+1 are the lattice rows y0-1 /
// y0+YS, periodic), so phase 2 needs nothing from another strip; the first R planes of a strip's
// phase 1 wait until the previous strip has finished reading the ring.
//
// Each thread updates U cells 32 apart in x, so the address arithmetic is shared between them.
// DRAM traffic per cell and PAIR of steps: 19 words read + 19 written (+ F^LC), against 2 x that
// for two single launches; the ring traffic (19 written + 19 read) stays in the 126 MB L2.
#pragma once
#include <cuda_runtime.h>
#include "nh_lb.cuh"

namespace nh {


constexpr int WAVE_MAX_STRIPS = 32;

struct Wave {
  unsigned long long* ticket;     // device counter, never reset
  unsigned long long* flag1;      // [nzf][cps] strip number (epoch) of the last finished phase-1 unit
  unsigned long long* flag2;      // the same for phase 2
  unsigned long long* strip_done; // [nstrips] finished phase-2 units per strip, never reset
  volatile int* err;              // HOST-mapped word, set to 1 if a wait timed out (read by every API entry)
  long long timeout_cycles;       // bound of one wait, in SM clocks
  unsigned long long fault;       // test hook (nh_debug_tune): added to the epoch the waits ask for, so that they cannot be met
  unsigned long long ticket_base; // value of *ticket when this launch starts
  unsigned long long strip_target[WAVE_MAX_STRIPS];  // value of strip_done[s] when strip s of THIS launch is done
  unsigned long long epoch0;      // flags of strip s of this launch carry epoch0 + s (> 0, grows across launches; 64 bits: never wraps)
  int nzf;                        // fluid planes
  unsigned YS;                    // lattice rows per strip (ny = nstrips * YS)
  unsigned nstrips;
  unsigned cps;                   // pieces per strip-plane of phase 1 (YS + 2 rows); phase 2 uses fewer
  unsigned ppr;                   // pieces per row (1 when a piece holds whole rows)
  unsigned rows_per_piece;        // rows of one piece (1 when a row holds several pieces)
  unsigned units_per_strip;       // order_len * cps
  unsigned rplane;                // cells of one ring plane = (YS + 2) * nx
  int spr_shift;                  // log2(32*U-cell segments of one piece that lie in one row)
  int D;                          // lead of phase 1 over phase 2, in planes (>= 1)
  int R;                          // ring slots (planes), R >= D + 2
  int reverse;                    // sweep from the top plate down
  const unsigned* order;          // [order_len] logical plane, bit 31 set for phase 2, in launch order
};

// p[i] = start of direction i inside a population array
template <typename T> struct DirTab { T* p[Q]; };

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

// The flags a unit depends on: 3 planes x up to 3 piece rows x 3 pieces along x (periodic in x; no
// wrap along y: the ring has its own halo rows); lane l < 27 looks at one of them, lane 27 at the
// previous strip.  prow counts piece rows inside the strip-plane of the unit's own phase:
//   phase 2, piece row p: lattice rows p*rp .. = ring rows p*rp + 1 ..; it gathers ring rows
//            p*rp .. (p+1)*rp + 1, i.e. phase-1 piece rows p .. ((p+1)*rp + 1)/rp
//   phase 1, piece row p: ring rows p*rp .. (p+1)*rp - 1, read by the phase-2 piece rows
//            p - (rp == 1 ? 2 : 1) .. p of the planes that used the slot before
// Returns true when everything is in place.
__device__ __forceinline__ bool deps_ready(const Wave& W, int phase, int k, unsigned strip, unsigned prow,
                                           unsigned q, unsigned lane) {
  bool ok = true;
  const unsigned rp = W.rows_per_piece;
  if (lane < 27) {
    const int j = (phase == 2 ? k - 1 : k - W.R - 1) + (int)(lane / 9);
    if (j >= 0 && j < W.nzf) {
      const unsigned r9 = lane % 9, dr = r9 / 3, dq = r9 % 3;
      int p;
      bool valid;
      if (phase == 2) {
        const unsigned last1 = (W.YS + 1) / rp;                    // last phase-1 piece row
        unsigned hi = ((prow + 1) * rp + 1) / rp;
        if (hi > last1) hi = last1;
        p = (int)(prow + dr);
        valid = (unsigned)p <= hi;
      } else {
        const int last2 = (int)((W.YS - 1) / rp);                  // last phase-2 piece row
        p = (int)prow - (rp == 1 ? 2 : 1) + (int)dr;
        valid = p >= 0 && p <= (int)prow && p <= last2;
      }
      if (valid) {
        unsigned pq = q + dq;                                      // periodic along x, no division
        pq = (pq == 0) ? W.ppr - 1 : pq - 1;
        if (pq == W.ppr) pq = 0;
        const unsigned long long* f = (phase == 2 ? W.flag1 : W.flag2) + (size_t)j * W.cps + (unsigned)p * W.ppr + pq;
        ok = ld_acquire_u64(f) >= W.epoch0 + strip + W.fault;
      }
    }
  } else if (lane == 27 && phase == 1 && strip > 0 && k < W.R) {
    // the slot was last used by the previous strip: all of it must be done
    ok = ld_acquire_u64(W.strip_done + (strip - 1)) >= W.strip_target[strip - 1];
  }
  const bool all = __all_sync(0xffffffffu, ok);
  // The vote carries no memory ordering of its own, and the lanes that go on to read the ring are not only the ones
  // that did the acquire loads: the warp barrier orders every lane's later loads after all of those acquires.
  __syncwarp();
  return all;
}

// f_i(x, t) = f*_i(x - e_i, t-1) with half-way bounce-back for the U cells (xA + 32 j, y) of one
// thread.  zm, z0, zp: element offsets of the planes z-1, z, z+1 inside each direction's array;
// r0, rm, rp: offsets of the rows y, y-1, y+1 (periodic) inside a plane.  lo / hi: the plane
// below / above is a plate.  Directions as in nh_lb.cuh.
template <typename T, int LD, int U, typename Tab>
__device__ __forceinline__ void gather_cells(const Tab& S, unsigned zm, unsigned z0, unsigned zp,
                                             unsigned r0, unsigned rm, unsigned rp, unsigned xA,
                                             unsigned nx, bool lo, bool hi, Pop<T> (&P)[U]) {
  unsigned xm[U], xp[U];        // source columns for e_x = +1 / -1
#pragma unroll
  for (int j = 0; j < U; ++j) {
    const unsigned x = xA + 32u * j;
    xm[j] = (x == 0) ? nx - 1 : x - 1;
    xp[j] = (x == nx - 1) ? 0u : x + 1;
  }
  // e_x = 0: one address, the U cells are 32 elements apart
#define NH_SAME(i, src, off)                                            \
  {                                                                     \
    const T* q_ = S.p[src] + ((off) + xA);                              \
    _Pragma("unroll") for (int j = 0; j < U; ++j) P[j].f[i] = ldp<T, LD>(q_ + 32 * j); \
  }
#define NH_SHIFT(i, src, off, xs)                                       \
  {                                                                     \
    _Pragma("unroll") for (int j = 0; j < U; ++j) P[j].f[i] = ldp<T, LD>(S.p[src] + ((off) + xs[j])); \
  }
  const unsigned own = z0 + r0;
  NH_SAME(0, 0, own)
  NH_SHIFT(1, 1, own, xm)
  NH_SHIFT(2, 2, own, xp)
  NH_SAME(3, 3, z0 + rm)
  NH_SAME(4, 4, z0 + rp)
  NH_SHIFT(7, 7, z0 + rm, xm)
  NH_SHIFT(8, 8, z0 + rp, xp)
  NH_SHIFT(9, 9, z0 + rp, xm)
  NH_SHIFT(10, 10, z0 + rm, xp)
  if (lo) {   // e_z = +1 would come out of the bottom plate: the opposite direction at the own cell
    NH_SAME(5, 6, own)
    NH_SAME(11, 12, own)
    NH_SAME(14, 13, own)
    NH_SAME(15, 16, own)
    NH_SAME(18, 17, own)
  } else {
    NH_SAME(5, 5, zm + r0)
    NH_SHIFT(11, 11, zm + r0, xm)
    NH_SHIFT(14, 14, zm + r0, xp)
    NH_SAME(15, 15, zm + rm)
    NH_SAME(18, 18, zm + rp)
  }
  if (hi) {   // e_z = -1 would come out of the top plate
    NH_SAME(6, 5, own)
    NH_SAME(12, 11, own)
    NH_SAME(13, 14, own)
    NH_SAME(16, 15, own)
    NH_SAME(17, 18, own)
  } else {
    NH_SAME(6, 6, zp + r0)
    NH_SHIFT(12, 12, zp + r0, xp)
    NH_SHIFT(13, 13, zp + r0, xm)
    NH_SAME(16, 16, zp + rp)
    NH_SAME(17, 17, zp + rm)
  }
#undef NH_SAME
#undef NH_SHIFT
}

// One CTA per unit.  The CTA draws its ticket when it starts to run (W.ticket != nullptr); with
// NH_OPT_LB_BLOCKORDER the unit is blockIdx.x instead, which saves the atomic's round trip but relies
// on CTAs being dispatched in blockIdx order (the hardware does, CUDA does not promise it; the
// bounded waits turn a violation into an error flag, not a hang).  No loop-carried state; each warp
// checks the flags itself (28 lanes, one acquire load).  A phase-1 unit gathers first and checks
// its flags (the old readers of its ring slot) only before it stores; a phase-2 unit checks before
// it gathers.  One barrier at the end, then thread 0 publishes the unit (fence, flag, counter).
template <typename T, bool SHIFTED, int U, int NT>
__global__ void __launch_bounds__(NT, ((sizeof(T) == 4 ? (U == 4 ? 512 : (U == 1 ? 1536 : 1024)) : (U == 2 ? 256 : 512)) / NT) > 0
                                          ? (sizeof(T) == 4 ? (U == 4 ? 512 : (U == 1 ? 1536 : 1024)) : (U == 2 ? 256 : 512)) / NT : 1)
lb_wave_kernel(DirTab<const T> A, DirTab<T> ring, DirTab<T> B, const T* __restrict__ Flc,
               Geom G, LbConst<T> C, Wave W) {
  const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  // programmatic dependent launch after another lb_wave launch (launch_lb2_u): resident early, but no ticket, no
  // flag and no population is touched before the previous launch has completed
  grid_launch_dependents();
  grid_dependency_wait();
  // which unit: decoded once (by thread 0 from its ticket, or by everyone from blockIdx, which the
  // compiler keeps on the uniform datapath)
  int phase, k;
  unsigned strip, prow, q, slot;
  auto decode = [&](unsigned tk, int& ph, int& kk, unsigned& st, unsigned& pr, unsigned& qq) {
    st = tk / W.units_per_strip;
    const unsigned rem = tk - st * W.units_per_strip;
    const unsigned unit = rem / W.cps, piece = rem - unit * W.cps;
    const unsigned code = W.order[unit];
    ph = (code >> 31) ? 2 : 1; kk = (int)(code & 0x7fffffffu);
    pr = piece / W.ppr; qq = piece - pr * W.ppr;
  };
  if (W.ticket) {                       // safe order: a ticket drawn when the CTA starts to run
    __shared__ unsigned s_unit[6];
    if (threadIdx.x == 0) {
      int ph, kk;
      unsigned st, pr, qq;
      decode((unsigned)(atomicAdd(W.ticket, 1ull) - W.ticket_base), ph, kk, st, pr, qq);
      s_unit[0] = (unsigned)ph; s_unit[1] = (unsigned)kk; s_unit[2] = st; s_unit[3] = pr; s_unit[4] = qq;
      s_unit[5] = (unsigned)((W.reverse ? W.nzf - 1 - kk : kk) % W.R);     // ring slot of the plane
    }
    __syncthreads();
    phase = (int)s_unit[0]; k = (int)s_unit[1]; strip = s_unit[2]; prow = s_unit[3]; q = s_unit[4];
    slot = s_unit[5];
  } else {
    decode(blockIdx.x, phase, k, strip, prow, q);
    slot = (unsigned)((W.reverse ? W.nzf - 1 - k : k) % W.R);
  }
  const unsigned row_local = prow * W.rows_per_piece + (warp >> W.spr_shift);   // row inside the piece grid
  // phase 2 has two rows fewer than phase 1: its surplus pieces are empty
  if (phase == 2 && prow * W.rows_per_piece >= W.YS) return;
  auto wait_flags = [&]() {
    const long long t0 = clock64();
    unsigned ns = 32;
    while (!deps_ready(W, phase, k, strip, prow, q, lane)) {
      __nanosleep(ns);
      if (ns < 512) ns *= 2;
      // give up after the bound, or at once when another CTA already has: the launch then ends quickly and every
      // later API call on this lattice reports the error (nh_api.cu: wave_failed)
      const long long waited = clock64() - t0;
      if (waited > 2000000ll && *W.err) break;          // (the word lives in host memory: not looked at before ~1 ms)
      if (waited > W.timeout_cycles) { if (lane == 0) { *W.err = 1; __threadfence_system(); } break; }
    }
  };
  const unsigned nx = (unsigned)G.nx, ny = (unsigned)G.ny;
  const unsigned seg_x = (warp & ((1u << W.spr_shift) - 1u)) * (32u * U);
  const int z = (W.reverse ? W.nzf - 1 - k : k) + 1;
  const unsigned xA = q * (unsigned)(NT * U) + seg_x + lane;
  const unsigned y0 = strip * W.YS;
  // ring row and lattice row of this thread's cells
  const unsigned ry = (phase == 1) ? row_local : row_local + 1;
  const bool active = (phase == 1) ? (row_local < W.YS + 2) : (row_local < W.YS);
  unsigned y = y0 + ry;                               // = lattice row + 1
  y = (y == 0) ? ny - 1 : y - 1;
  if (y >= ny) y -= ny;
  const unsigned cell = (unsigned)z * G.plane + y * nx + xA;
  const unsigned rcell = slot * W.rplane + ry * nx + xA;
  if (phase == 2) wait_flags();
  Pop<T> P[U];
  T Fx[U], Fy[U], Fz[U];
  if (active) {
    const bool lo = (z == 1), hi = (z == G.nz - 2);
    if (phase == 1) {
      const unsigned z0 = (unsigned)z * G.plane;
      const unsigned rm = (y == 0 ? ny - 1 : y - 1) * nx, rp = (y == ny - 1 ? 0u : y + 1) * nx;
      gather_cells<T, LD_CS, U>(A, z0 - G.plane, z0, z0 + G.plane, y * nx, rm, rp, xA, nx, lo, hi, P);
    } else {
      const unsigned sm = (slot == 0 ? (unsigned)W.R - 1 : slot - 1), sp = (slot == (unsigned)W.R - 1 ? 0u : slot + 1);
      gather_cells<T, LD_CG, U>(ring, sm * W.rplane, slot * W.rplane, sp * W.rplane, ry * nx, (ry - 1) * nx,
                                (ry + 1) * nx, xA, nx, lo, hi, P);
    }
#pragma unroll
    for (int j = 0; j < U; ++j) {
      Fx[j] = Fy[j] = Fz[j] = T(0);
      if (C.use_flc) {
        const T* f = Flc + cell;
        Fx[j] = __ldg(f + 32 * j); Fy[j] = __ldg(f + G.N + 32 * j); Fz[j] = __ldg(f + 2 * G.N + 32 * j);
      }
    }
  }
  bool ready = true;
  if (phase == 1) ready = deps_ready(W, phase, k, strip, prow, q, lane);   // a look while the gathers fly
  if (active) {
#pragma unroll
    for (int j = 0; j < U; ++j) collide<T, SHIFTED>(P[j], Fx[j], Fy[j], Fz[j], C);
  }
  if (phase == 1 && !ready) wait_flags();
  if (active) {
    if (phase == 1) {
#pragma unroll
      for (int i = 0; i < Q; ++i) {
        T* d = ring.p[i] + rcell;
#pragma unroll
        for (int j = 0; j < U; ++j) d[32 * j] = P[j].f[i];
      }
    } else {
#pragma unroll
      for (int i = 0; i < Q; ++i) {
        T* d = B.p[i] + cell;
#pragma unroll
        for (int j = 0; j < U; ++j) __stcs(d + 32 * j, P[j].f[i]);
      }
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    // publish: everything this CTA read and wrote is ordered before the flag (and the strip counter)
    __threadfence();
    unsigned long long* f = (phase == 1 ? W.flag1 : W.flag2) + (size_t)k * W.cps + prow * W.ppr + q;
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(f), "l"(W.epoch0 + strip) : "memory");
    if (phase == 2) asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(W.strip_done + strip), "l"(1ull) : "memory");
  }
}

}  // namespace nh
