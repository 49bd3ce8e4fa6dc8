/* nh_oracle.h -- CPU ORACLE for the hybrid nematohydrodynamics time step.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares no code,
 * header, table or helper with the CUDA path (paper_2503_06610_b200/csrc, include/).
 *
 * What it is: a plain, slow, FP64, loop-per-cell restatement of the method of
 * arXiv 2503.06610 in the reduced form BASELINE.json's north_star names
 * (one-constant Frank energy with chiral term, elastic stress only), following the
 * algorithm step by step in the paper's order:
 *   LB   : PAPER.md:118-166 (Sec. II.C, Eqs. 14-23), evaluation order PAPER.md:187
 *   walls: half-way bounce-back; periodic x,y PAPER.md:225
 *   FD   : central differences Eq. 13, solid values fixed,
 *          director equation Eq. 9 with D, W of Eq. 5,
 *          predictor-corrector PAPER.md:105-112
 *   force: Eq. 6 and the last term of Eq. 12; optionally the Leslie
 *          viscous stress of Eq. 3 in Eq. 12 (row f1, pins V1-V4)
 *   loop : Fig. 1 / Sec. II.D
 * Readings of gaps in the paper are SURVEY.md Sec. 8(c) G1-G21, listed in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_pins.py): P1 Poiseuille closed form, P2 mass, P3 shifted
 * vs unshifted, P4 uniform director fixed point, P5 brute-force energy derivative,
 * P6 energy descent, P7 Leslie angle, P8 helix, P9 zero net force, P10 stress identity,
 * P11 Heun order.  The coupled LC+flow step on a skyrmion has no worked example in the
 * paper: PARITY UNPINNED against the paper for that composite (each part is pinned).
 *
 * Layout of every field array: [component][z][y][x], x fastest, N = nx*ny*nz cells.
 * Layers z = 0 and z = nz-1 are solid plates (G7); fluid is z = 1..nz-2.
 * Population index i <-> lattice vector e_i (D3Q19):
 *   0:(0,0,0)  1:(+,0,0) 2:(-,0,0) 3:(0,+,0) 4:(0,-,0) 5:(0,0,+) 6:(0,0,-)
 *   7:(+,+,0) 8:(-,-,0) 9:(+,-,0) 10:(-,+,0) 11:(+,0,+) 12:(-,0,-) 13:(+,0,-) 14:(-,0,+)
 *   15:(0,+,+) 16:(0,-,-) 17:(0,+,-) 18:(0,-,+)
 */
#ifndef NH_ORACLE_H
#define NH_ORACLE_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct nh_oracle_lattice nh_oracle_lattice;

typedef struct {
  int    nx, ny, nz;   /* nz counts the two plate layers; nz >= 3                          */
  double tau;          /* SRT relaxation time > 0.5, nu = (tau-1/2)/3  */
  double K;            /* one-constant Frank modulus >= 0 */
  double pitch;        /* P in cells, q0 = 2 pi / P; pitch <= 0 -> q0 = 0   */
  double xi;           /* flow alignment = -gamma2/gamma1 (G4)   */
  double gamma1;       /* rotational viscosity > 0   */
  double g[3];         /* body acceleration */
  int    anchoring;    /* 0 = homeotropic, fixed at both plates
                          1 = free plates (no anchoring), reading G23  */
  double W0;           /* bulk effective anchoring along z: h_z += W0 n_z (reading G14)
                                                                            PAPER.md:229  */
  int    fd_ratio;     /* default Delta t_FD / Delta t_LB >= 0  */
  int    precision;    /* 0,1: shifted populations (Eqs. 19-23); 2,3: unshifted (Eqs. 14-17).
                          The oracle computes in FP64 whatever this says.                  */
  int    coupling;     /* bit0: F^LC acts on the flow; bit1: flow acts on n               */
  double alpha[6];     /* Leslie viscosities alpha1, alpha2, alpha3, alpha4', alpha5, alpha6 of the
                          viscous stress in the force, Eqs. 3, 12; all 0 = elastic stress only
                                                                         PAPER.md:50, 97-99 */
  double K3[3];        /* K11, K22, K33 of Eqs. 7-8 (splay, twist, bend); all 0 = the one-constant
                          energy with K; otherwise K is ignored (row f2, reading G24)
                                                                         PAPER.md:70-73   */
} nh_oracle_params;

int  nh_oracle_init_lattice(const nh_oracle_params*, nh_oracle_lattice** out);
int  nh_oracle_set_director(nh_oracle_lattice*, const double* n_host);
int  nh_oracle_step(nh_oracle_lattice*, int n_lb, int n_fd);
int  nh_oracle_get_fields(nh_oracle_lattice*, double* rho, double* u, double* n, double* F_lc);
int  nh_oracle_get_populations(nh_oracle_lattice*, double* f /* [19][nz][ny][nx] as stored */);
/* test-only: populations := equilibrium of (rho = 1, u_host) on fluid cells (pins P12, P13) */
int  nh_oracle_set_velocity(nh_oracle_lattice*, const double* u_host /* [3][nz][ny][nx] */);
long nh_oracle_time(const nh_oracle_lattice*);
void nh_oracle_free(nh_oracle_lattice*);
const char* nh_oracle_last_error(void);
int  nh_oracle_num_threads(void);

/* The FD building blocks on caller-owned arrays, so the pins can reach them directly.
 * periodic_z = 1: every layer is fluid and z wraps (used only by pins P5, P8, P9);
 * periodic_z = 0: values are produced on z = 1..nz-2 and are 0 on the two plate layers,
 *                 stencils read whatever the plate layers of the inputs hold.          */
int nh_oracle_molecular_field(int nx, int ny, int nz, int periodic_z, double K, double q0,
                              const double* n, double* h);
int nh_oracle_molecular_field_w0(int nx, int ny, int nz, int periodic_z, double K, double q0, double W0,
                                 const double* n, double* h);   /* + the bulk anchoring term */
int nh_oracle_director_rhs(int nx, int ny, int nz, int periodic_z, double K, double q0,
                           double xi, double gamma1, const double* n, const double* u, double* R);
int nh_oracle_elastic_stress(int nx, int ny, int nz, int periodic_z, double K, double q0,
                             const double* n, double* sigma /* [9][nz][ny][nx], index 3*alpha+beta */);
int nh_oracle_elastic_force(int nx, int ny, int nz, int periodic_z, double K, double q0,
                            const double* n, double* F);
/* Three-constant Frank energy (Eqs. 7-8), K3 = {K11, K22, K33}: molecular field h [3][N], elastic
 * stress sigma [9][N] and the total discrete energy; any output pointer may be NULL. */
int nh_oracle_frank3(int nx, int ny, int nz, int periodic_z, const double* K3, double q0, const double* n,
                     double* h, double* sigma, double* energy);
/* Leslie viscous stress of Eq. 3 with alpha4 -> alpha4' (Eq. 12), N from Eq. 9 (reading G22), and
 * the whole force F^LC = d_b (sigma^e + sigma^v)_ab.  alpha = {a1, a2, a3, a4', a5, a6}. */
int nh_oracle_viscous_stress(int nx, int ny, int nz, int periodic_z, double K, double q0, double xi,
                             double gamma1, const double* alpha, const double* n, const double* u,
                             double* sigma /* [9][nz][ny][nx] */);
int nh_oracle_lc_force(int nx, int ny, int nz, int periodic_z, double K, double q0, double xi,
                       double gamma1, const double* alpha, const double* n, const double* u, double* F);

#ifdef __cplusplus
}
#endif
#endif
