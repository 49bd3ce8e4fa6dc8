/* nh.h -- C ABI of the B200 (sm_100a) nematohydrodynamics hot path.
 *
 * One LB+FD time step of the hybrid solver of arXiv 2503.06610 ("Efficient single-precision
 * simulations of nematohydrodynamics"), in the reduced form BASELINE.json's north_star names:
 *
 *   flow     : D3Q19 single-relaxation-time lattice Boltzmann with Guo forcing on the SHIFTED
 *              populations f_i - w_i                      PAPER.md:118-166, Eqs. 14-23 (Sec. II.C)
 *              half-way bounce-back at the two plates     PAPER.md:141;  periodic x, y PAPER.md:225
 *   director : d_t n = h/gamma1 + xi n.D - (u.grad) n + W.n, projected perpendicular to n,
 *              predictor-corrector, renormalised           PAPER.md:77 (Eq. 9), 105-112 (Sec. II.B)
 *              h = K lap n - 2 K q0 curl n  (one-constant Frank energy with chiral term)
 *                                                          PAPER.md:70-73, 81 (Eqs. 7-8, 10)
 *   force    : F^LC_a = d_b sigma_ab,  sigma = elastic (Ericksen) stress
 *                                                          PAPER.md:66 (Eq. 6), 97 (Eq. 12, last term)
 *              optionally + the Leslie viscous stress      PAPER.md:50 (Eq. 3), 97-99 (Eq. 12)
 *   schedule : LB every step; director + force after every r-th step with Delta t_FD = r
 *                                                          PAPER.md:191-207 (Sec. II.D, Fig. 1)
 *
 * Every step of that path runs in hand-written CUDA kernels (paper_2503_06610_b200/csrc).  There
 * is no CPU fallback: without a CUDA device every compute entry returns NH_ECUDA.
 *
 * Conventions
 *   - Return value: 0 (NH_OK) or a negative code; the message is in nh_last_error() (per thread).
 *     No exception or abort crosses this boundary.
 *   - Fields are arrays [component][z][y][x], x fastest, N = nx*ny*nz cells.  Layers z = 0 and
 *     z = nz-1 are the solid plates (wall half-way between layers 0|1 and nz-2|nz-1); the fluid is
 *     z = 1..nz-2.  On the plates rho = 1, u = 0, F^LC = 0 and n = z_hat (anchoring 0) or the copy
 *     of the adjacent fluid layer (anchoring 1) are returned.
 *   - Every HOST array is FP64 whatever the device precision; conversion happens on the device.
 *   - Ownership: the caller owns all host arrays and the device workspace and keeps the workspace
 *     alive until nh_free.  The library owns only the handle.
 *   - All device work is enqueued on the stream given to nh_init_lattice.  nh_set_director and
 *     nh_get_fields synchronise that stream before returning; nh_step does not.
 *   - Errors that happen ON the device after an asynchronous call has returned (a wavefront dependency of the
 *     two-step LB kernel that is not met within its time bound, which would mean the launch order it relies on
 *     was violated) are sticky: the kernel records them in host-visible memory, the launch ends, and every later
 *     call that touches the lattice -- nh_step included -- returns NH_ECUDA; the lattice's state is then invalid.
 */
#ifndef NH_H
#define NH_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

#define NH_OK       0
#define NH_EINVAL  -1   /* null pointer, bad size or parameter                      */
#define NH_ENOMEM  -2   /* workspace smaller than nh_workspace_bytes()              */
#define NH_ECUDA   -3   /* a CUDA call failed (including: no device)                */
#define NH_ENUMERIC -4  /* a non-finite population or director was found (NH_OPT_CHECK_FINITE) */

/* precision */
#define NH_FP64_SHIFTED    0   /* Eqs. 19-23 in double                                */
#define NH_FP32_SHIFTED    1   /* Eqs. 19-23 in float: the paper's method            */
#define NH_FP32_UNSHIFTED  2   /* Eqs. 14-17 in float: the comparison PAPER.md:235   */
#define NH_FP64_UNSHIFTED  3   /* Eqs. 14-17 in double                                */

typedef struct nh_lattice nh_lattice;   /* opaque */

typedef struct {
  int    nx, ny, nz;   /* grid; nz counts the two plate layers; nx, ny >= 1, nz >= 3            */
  double tau;          /* SRT relaxation time, > 0.5; nu = (tau - 1/2)/3 */
  double K;            /* one-constant Frank modulus, >= 0 */
  double pitch;        /* cholesteric pitch P in cells, q0 = 2 pi/P; <= 0: q0 = 0 PAPER.md:73  */
  double xi;           /* flow-alignment parameter = -gamma2/gamma1  */
  double gamma1;       /* rotational viscosity, > 0  */
  double g[3];         /* body acceleration; the force on the fluid is rho g  */
  int    anchoring;    /* 0 = infinite homeotropic at both plates: n = z_hat there
                          1 = free plates: the plate layers copy the adjacent fluid layer (zero
                              normal derivative, no anchoring torque; G23) PAPER.md:229 */
  double W0;           /* bulk effective anchoring along z: h_z += W0 n_z, from the energy
                          -(W0/2) (n.z_hat)^2 per cell (G14) */
  int    fd_ratio;     /* default r = Delta t_FD / Delta t_LB, >= 0 */
  int    precision;    /* NH_FP64_SHIFTED .. NH_FP64_UNSHIFTED */
  int    coupling;     /* bit0: F^LC acts on the flow; bit1: the flow acts on n   (3 = paper)  */
  double alpha[6];     /* Leslie viscosities alpha1, alpha2, alpha3, alpha4', alpha5, alpha6 of the viscous
                          stress inside F^LC (Eq. 3 with alpha4 -> alpha4', Eq. 12); N of Eq. 4 is taken
                          from Eq. 9 as (h/gamma1 + xi n.D) perpendicular to n (reading G22).
                          All 0 (the north_star's reduced model): elastic stress only.  xi and gamma1 are
                          NOT derived from them (gamma1 = alpha3 - alpha2, gamma2 = alpha3 + alpha2 is
                          the caller's business) */
  double K3[3];        /* K11, K22, K33 (splay, twist, bend) of the Frank energy, Eqs. 7-8; all 0: the
                          one-constant energy with K (the north_star's model); otherwise K is ignored
                          and h, sigma^e follow from the three-constant energy (G24)
                                                                                  PAPER.md:70-73 */
} nh_params;

/* Bytes of device memory the lattice needs for these parameters (0 if they are invalid).
 * Layout: two population buffers [19][N], n, n^P, n', a, u, F^LC [3][N]
 * in the device precision, one FP64 staging buffer [3][N], the plane ring of the two-step LB
 * kernel (min(nz-2, 12) planes of 19 populations) and its flags, each 256-byte aligned. */
size_t nh_workspace_bytes(const nh_params* p);

/* Create a lattice in `dev_workspace` (DEVICE pointer, 256-byte aligned, >= nh_workspace_bytes).
 * `cuda_stream` is a cudaStream_t (NULL = legacy default stream).  State after the call: t = 0,
 * rho = 1, u = 0 (shifted populations 0, Eq. 19), n = z_hat, F^LC = 0.  PAPER.md:193-199. */
int nh_init_lattice(const nh_params* p, void* dev_workspace, size_t bytes, void* cuda_stream,
                    nh_lattice** out);

/* Set the director from a HOST array [3][nz][ny][nx] (FP64).  Each vector is normalised, the plate
 * layers are overwritten with z_hat (anchoring 0) or with the adjacent fluid layer (anchoring 1), n^P := n and F^LC is computed from it
 * (Eq. 12; reading G9).  Populations and t are untouched.  NH_EINVAL if a vector has
 * zero or non-finite length (checked on the device; the lattice is then unchanged). */
int nh_set_director(nh_lattice* L, const double* n_host);

/* Advance n_lb lattice-Boltzmann steps.  r = n_fd (n_fd < 0: params.fd_ratio; 0: director and
 * force frozen).  After each LB step t <- t+1 and, if r > 0 and t mod r == 0, the director
 * predictor-corrector and the force update run with Delta t_FD = r.
 * Asynchronous on the lattice's stream. */
int nh_step(nh_lattice* L, int n_lb, int n_fd);

/* Copy fields to HOST arrays (FP64); any pointer may be NULL.  rho [N] and u [3][N] are Eqs. 20-21
 * on the current (post-streaming) populations with the current force; n [3][N]; F_lc [3][N]. */
int nh_get_fields(nh_lattice* L, double* rho, double* u, double* n, double* F_lc);

/* Number of completed LB steps (-1 for a null handle). */
long nh_time(const nh_lattice* L);

/* Number of kernels this lattice has launched so far (bench.py's gpu_launches). */
long nh_launch_count(const nh_lattice* L);

/* Options (results agree within round-off whatever they are):
 *   NH_OPT_GRAPH         replay nh_step through CUDA graphs (launch-bound small grids): one executable graph per
 *                        distinct (n_lb, r, t mod r, buffer parity), captured on first use.  Needs a capturable
 *                        stream (not the legacy default stream), otherwise plain launches; the two-step LB kernel
 *                        and the small-lattice cooperative launch are not used under it.
 *   NH_OPT_TIMING        bracket every kernel launch with a CUDA-event pair on the lattice's stream (ignored while
 *                        graphs are on)
 *   NH_OPT_FD_DIRECT     use the one-thread-per-cell FD kernels instead of the tiled ones (cross-check form)
 *   NH_OPT_NO_SERPENTINE sweep the populations in the same direction on every launch
 *   NH_OPT_FD_NOVEC      stage the FD tiles element by element even where 16-byte copies fit
 *   NH_OPT_LB_TWOSTEP    two LB steps per launch through an L2-resident plane ring wherever no director update
 *                        falls between them and the grid tiles into pieces (nx a multiple of 64 that divides 512,
 *                        is a multiple of 512, or has a factor 3, 5, 6 or 7 in nx / 64; else one step per launch);
 *                        bit-identical results.  With neither this nor NH_OPT_LB_ONESTEP the library decides (FP32,
 *                        planes >= 256x256, ring <= 48 MB: DESIGN.md section 7).
 *   NH_OPT_LB_ONESTEP    one launch per LB step: neither the two-step kernel nor, on small lattices, the
 *                        cooperative launch that takes all the steps up to the next director update
 *   NH_OPT_CHECK_FINITE  after the steps of every nh_step call, one more kernel reads the populations and the director
 *                        (22 words per cell: about half an LB step) and records any NaN or Inf in host-visible memory.
 *                        Like the wavefront error above this is sticky and asynchronous: the nh_step that produced the
 *                        value returns NH_OK, every call on the lattice after the kernel has run returns NH_ENUMERIC.
 *                        For long unattended runs (the paper's are 5e8 steps): call nh_step in chunks.
 * Launch-shape tuning knobs are not part of this contract (include/nh_debug.h).  Bits not listed here are NH_EINVAL.
 * Setting options resets the timing accumulators. */
#define NH_OPT_GRAPH          1
#define NH_OPT_TIMING         2
#define NH_OPT_FD_DIRECT      4
#define NH_OPT_NO_SERPENTINE 16
#define NH_OPT_FD_NOVEC      32
#define NH_OPT_LB_TWOSTEP    64
#define NH_OPT_LB_ONESTEP   128
#define NH_OPT_CHECK_FINITE 256
int nh_set_options(nh_lattice* L, int options);

/* Accumulated CUDA-event time (ms) and number of launches of one kernel class since the last
 * nh_set_options; synchronises the stream.  Time is only accumulated while NH_OPT_TIMING is set.
 * which: 0 = LB collide+stream, 1 = velocity (moments, u store), 2 = predictor, 3 = corrector,
 *        4 = force, 5 = everything else (conversions, initialisation), 6 = two-step LB launches. */
int nh_kernel_time(nh_lattice* L, int which, double* ms_total, long* launches);

/* ---- Slab decomposition along y (the paper's own runs are single-GPU,
 * PAPER.md:284).  A rank's lattice holds its rows plus H halo rows on either side; its periodic wrap in y
 * then only feeds the outermost halo rows, and every operator eats into the valid halo by its stencil
 * radius, so the halos are refreshed from the neighbours between calls with the two
 * copies below.  Both are asynchronous on the lattice's stream and touch no other state.
 *
 * nh_get_rows: pack rows [y0, y0 + nrows) of one field -- all x, ALL z (plate layers included), all
 * components -- into the contiguous DEVICE buffer `dev_buf`, laid out [component][z][row][x] in the
 * lattice's storage type (4 or 8 bytes per word; nh_rows_bytes gives the size).  nh_set_rows is the inverse.
 * field: NH_FIELD_POPULATIONS  the 19 post-collision populations the next LB step gathers from
 *        NH_FIELD_DIRECTOR     the current director n (3 components)
 *        NH_FIELD_VELOCITY     u as stored by the last director update (3)
 *        NH_FIELD_FORCE        F^LC (3)
 * NH_EINVAL for a null handle or buffer, an unknown field, or rows outside [0, ny). */
#define NH_FIELD_POPULATIONS 0
#define NH_FIELD_DIRECTOR    1
#define NH_FIELD_VELOCITY    2
#define NH_FIELD_FORCE       3
size_t nh_rows_bytes(const nh_lattice* L, int field, int nrows);
int nh_get_rows(nh_lattice* L, int field, int y0, int nrows, void* dev_buf);
int nh_set_rows(nh_lattice* L, int field, int y0, int nrows, const void* dev_buf);

/* The same for TWO row ranges in one launch -- a slab's two edges, or its two halos: rows [y0_a, y0_a + nrows)
 * go to / come from the first half of `dev_buf`, rows [y0_b, y0_b + nrows) the second half; each half is laid out
 * like the buffer of nh_get_rows (2 x nh_rows_bytes(L, field, nrows) bytes in all). */
int nh_get_rows_pair(nh_lattice* L, int field, int y0_a, int y0_b, int nrows, void* dev_buf);
int nh_set_rows_pair(nh_lattice* L, int field, int y0_a, int y0_b, int nrows, const void* dev_buf);

/* Recompute F^LC (Eq. 12) from the director and the stored velocity now in the lattice -- the force
 * step of nh_step on its own, for use after the director's (and, with Leslie viscosities, the
 * velocity's) halo rows have been refreshed.  Asynchronous on the lattice's stream. */
int nh_update_force(nh_lattice* L);

/* on != 0: nh_step no longer recomputes F^LC after a director update; the caller owes an nh_update_force
 * before the next LB step (the slab driver refreshes the director's halo rows in between, so the force
 * computed inside nh_step would be thrown away).  Graph replay is bypassed while this is on.  Default 0. */
int nh_defer_force(nh_lattice* L, int on);

void nh_free(nh_lattice* L);
const char* nh_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
