// nh_oracle.cpp -- CPU ORACLE (test infrastructure, not the product; see nh_oracle.h).
//
// Plain FP64 loops, one cell at a time, in the paper's order and notation.  No blocking,
// no fusion, no reordering beyond what the cited passage states.  Build with
//   g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC   (oracle/build.py)
// so that no FMA contraction changes the arithmetic.  The OpenMP pragmas
// only split independent cell loops over threads; every cell's arithmetic is unchanged.
#include "nh_oracle.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

thread_local std::string g_err;
int fail(int code, const std::string& msg) { g_err = msg; return code; }
constexpr int E_INVAL = -1;
constexpr int E_NOMEM = -2;

// ---- D3Q19: c_s^2 = 1/3, w = 1/3, 1/18, 1/36 -------------------------------
constexpr int Q = 19;
const int EX[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
const int EY[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
const int EZ[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
double weight_of(int i) {
  const int e2 = EX[i] * EX[i] + EY[i] * EY[i] + EZ[i] * EZ[i];
  return e2 == 0 ? 1.0 / 3.0 : (e2 == 1 ? 1.0 / 18.0 : 1.0 / 36.0);
}
int opposite_of(int i) {
  for (int j = 0; j < Q; ++j)
    if (EX[j] == -EX[i] && EY[j] == -EY[i] && EZ[j] == -EZ[i]) return j;
  return -1;
}
// looked up once per direction instead of once per cell; same values
struct Tables {
  double w[Q];
  int opp[Q];
  Tables() { for (int i = 0; i < Q; ++i) { w[i] = weight_of(i); opp[i] = opposite_of(i); } }
};
const Tables TAB;
double weight(int i) { return TAB.w[i]; }
int opposite(int i) { return TAB.opp[i]; }

// ---- grid helpers ------------------------------------------------------------------------
struct Grid {
  int nx, ny, nz;
  bool pz;  // periodic in z (pins only)
  double W0 = 0.0;  // bulk anchoring strength (row f3, reading G14): energy -(W0/2) (n.z_hat)^2 per cell
  size_t N() const { return (size_t)nx * ny * nz; }
  size_t at(int x, int y, int z) const { return ((size_t)z * ny + y) * nx + x; }
  int wx(int x) const { return (x + nx) % nx; }  // periodic x, y
  int wy(int y) const { return (y + ny) % ny; }
  int wz(int z) const { return pz ? (z + nz) % nz : z; }
  int z_lo() const { return pz ? 0 : 1; }       // first computed layer
  int z_hi() const { return pz ? nz : nz - 1; } // one past the last computed layer
  // neighbour of (x,y,z) displaced by +-1 along axis b
  size_t nb(int x, int y, int z, int b, int s) const {
    if (b == 0) return at(wx(x + s), y, z);
    if (b == 1) return at(x, wy(y + s), z);
    return at(x, y, wz(z + s));
  }
};

double levi_civita(int i, int j, int k) { return 0.5 * (i - j) * (j - k) * (k - i); }

// Central difference Eq. 13: d_b field_c at a cell, Delta x = 1.
double ddx(const Grid& G, const double* fld, int c, int x, int y, int z, int b) {
  const size_t N = G.N();
  return 0.5 * (fld[c * N + G.nb(x, y, z, b, +1)] - fld[c * N + G.nb(x, y, z, b, -1)]);
}

// Molecular field, Eq. 10 for the one-constant energy with chiral term
// f = (K/2) d_b n_c d_b n_c + K q0 n.curl n  (reading G1):  h = K lap n - 2 K q0 curl n,
// compact 7-point Laplacian (reading G2), central curl.
void molecular_field_cell(const Grid& G, double K, double q0, const double* m, int x, int y, int z,
                          double h[3]) {
  const size_t N = G.N();
  const size_t c0 = G.at(x, y, z);
  double dm[3][3];  // dm[b][c] = d_b m_c
  for (int b = 0; b < 3; ++b)
    for (int c = 0; c < 3; ++c) dm[b][c] = ddx(G, m, c, x, y, z, b);
  double curl[3];
  for (int mu = 0; mu < 3; ++mu) {
    curl[mu] = 0.0;
    for (int b = 0; b < 3; ++b)
      for (int c = 0; c < 3; ++c) curl[mu] += levi_civita(mu, b, c) * dm[b][c];
  }
  for (int c = 0; c < 3; ++c) {
    double lap = 0.0;
    for (int b = 0; b < 3; ++b)
      lap += m[c * N + G.nb(x, y, z, b, +1)] + m[c * N + G.nb(x, y, z, b, -1)] - 2.0 * m[c * N + c0];
    h[c] = K * lap - 2.0 * K * q0 * curl[c];
  }
  // bulk effective anchoring along z (its form is reading G14): h_z += W0 n_z
  h[2] += G.W0 * m[2 * N + c0];
}

// ---- three-constant Frank energy, Eqs. 7-8; row f2, reading G24 ----------
// Discrete energy density at a cell, every derivative the central difference of Eq. 13:
//   f = K11/2 (div n)^2 + K22/2 (n.curl n + q0)^2 + K33/2 |b|^2,   b = (n.grad) n
// (|n x curl n| = |(n.grad) n| for a unit vector).  Its derivatives
//   pi_{b c} = df/d(d_b n_c) = K11 delta_bc div n + K22 T eps_{a b c} n_a + K33 n_b b_c,  T = n.curl n + q0
//   df/dn_m  = K22 T (curl n)_m + K33 b_c d_m n_c
// give h_m = -df/dn_m + d_b pi_{b m} (Eq. 10) and sigma^e_{a b} = -d_a n_c pi_{b c} (Eq. 6).
bool any_K3(const double K3[3]) { return K3[0] != 0.0 || K3[1] != 0.0 || K3[2] != 0.0; }

void frank3_cell(const Grid& G, const double K3[3], double q0, const double* n, int x, int y, int z,
                 double pi[3][3], double dfdn[3], double* fdens) {
  const size_t N = G.N();
  const size_t c0 = G.at(x, y, z);
  double dn[3][3];  // dn[b][c] = d_b n_c
  for (int b = 0; b < 3; ++b)
    for (int c = 0; c < 3; ++c) dn[b][c] = ddx(G, n, c, x, y, z, b);
  const double nn[3] = {n[c0], n[N + c0], n[2 * N + c0]};
  const double div = dn[0][0] + dn[1][1] + dn[2][2];
  double curl[3], bb[3];
  for (int m = 0; m < 3; ++m) {
    curl[m] = 0.0;
    bb[m] = 0.0;
    for (int b = 0; b < 3; ++b) {
      bb[m] += nn[b] * dn[b][m];
      for (int c = 0; c < 3; ++c) curl[m] += levi_civita(m, b, c) * dn[b][c];
    }
  }
  const double T = nn[0] * curl[0] + nn[1] * curl[1] + nn[2] * curl[2] + q0;
  for (int b = 0; b < 3; ++b)
    for (int c = 0; c < 3; ++c) {
      double twist = 0.0;
      for (int a = 0; a < 3; ++a) twist += levi_civita(a, b, c) * nn[a];
      pi[b][c] = K3[0] * (b == c ? div : 0.0) + K3[1] * T * twist + K3[2] * nn[b] * bb[c];
    }
  for (int m = 0; m < 3; ++m) {
    double bend = 0.0;
    for (int c = 0; c < 3; ++c) bend += bb[c] * dn[m][c];
    dfdn[m] = K3[1] * T * curl[m] + K3[2] * bend;
  }
  if (fdens)
    *fdens = 0.5 * K3[0] * div * div + 0.5 * K3[1] * T * T +
             0.5 * K3[2] * (bb[0] * bb[0] + bb[1] * bb[1] + bb[2] * bb[2]);
}

// pi [9][N] (index 3 b + c) and df/dn [3][N] on the computed layers.  On the plate layers the director
// is uniform inside the solid (solid node values fixed), so grad n = 0 there:
// pi = K22 q0 eps_{a b c} n_a, df/dn unused.
void frank3_fields(const Grid& G, const double K3[3], double q0, const double* n, double* pi, double* dfdn) {
  const size_t N = G.N();
  std::memset(dfdn, 0, sizeof(double) * 3 * N);
  for (int z = 0; z < G.nz; ++z) {
    if (z >= G.z_lo() && z < G.z_hi()) continue;
    for (int y = 0; y < G.ny; ++y)
      for (int x = 0; x < G.nx; ++x) {
        const size_t c0 = G.at(x, y, z);
        for (int b = 0; b < 3; ++b)
          for (int c = 0; c < 3; ++c) {
            double twist = 0.0;
            for (int a = 0; a < 3; ++a) twist += levi_civita(a, b, c) * n[a * N + c0];
            pi[(3 * b + c) * N + c0] = K3[1] * q0 * twist;
          }
      }
  }
#pragma omp parallel for schedule(static)
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < G.ny; ++y)
      for (int x = 0; x < G.nx; ++x) {
        double p[3][3], d[3];
        frank3_cell(G, K3, q0, n, x, y, z, p, d, nullptr);
        const size_t c0 = G.at(x, y, z);
        for (int b = 0; b < 3; ++b)
          for (int c = 0; c < 3; ++c) pi[(3 * b + c) * N + c0] = p[b][c];
        for (int m = 0; m < 3; ++m) dfdn[m * N + c0] = d[m];
      }
}

// h_m = -df/dn_m + d_b pi_{b m} (+ the bulk anchoring term) at one cell, from the fields above.
void frank3_h_cell(const Grid& G, const double* n, const double* pi, const double* dfdn, int x, int y, int z,
                   double h[3]) {
  const size_t N = G.N();
  const size_t c0 = G.at(x, y, z);
  for (int m = 0; m < 3; ++m) {
    double s = -dfdn[m * N + c0];
    for (int b = 0; b < 3; ++b) s += ddx(G, pi, 3 * b + m, x, y, z, b);
    h[m] = s;
  }
  h[2] += G.W0 * n[2 * N + c0];
}

// Right-hand side of the director equation, Eq. 9, with xi = -gamma2/gamma1 (G4),
// D and W exactly as printed in Eq. 5 (G5), then projected perpendicular to m (G3).
// pi, dfdn: the three-constant fields of frank3_fields for this m, or null for the one-constant energy.
void director_rhs_cell(const Grid& G, double K, double q0, double xi, double gamma1,
                       const double* m, const double* u, int x, int y, int z, double R[3],
                       const double* pi = nullptr, const double* dfdn = nullptr) {
  const size_t N = G.N();
  const size_t c0 = G.at(x, y, z);
  double h[3];
  if (pi) frank3_h_cell(G, m, pi, dfdn, x, y, z, h);
  else molecular_field_cell(G, K, q0, m, x, y, z, h);
  double dm[3][3], du[3][3];  // d_b m_c, d_b u_c
  for (int b = 0; b < 3; ++b)
    for (int c = 0; c < 3; ++c) {
      dm[b][c] = ddx(G, m, c, x, y, z, b);
      du[b][c] = ddx(G, u, c, x, y, z, b);
    }
  double D[3][3], W[3][3];
  for (int a = 0; a < 3; ++a)
    for (int mu = 0; mu < 3; ++mu) {
      D[a][mu] = 0.5 * (du[a][mu] + du[mu][a]);  // D_{a mu} = (d_a u_mu + d_mu u_a)/2
      W[a][mu] = 0.5 * (du[mu][a] - du[a][mu]);  // W_{a mu} = (d_mu u_a - d_a u_mu)/2
    }
  double mm[3] = {m[c0], m[N + c0], m[2 * N + c0]};
  double uu[3] = {u[c0], u[N + c0], u[2 * N + c0]};
  for (int mu = 0; mu < 3; ++mu) {
    double align = 0.0, adv = 0.0, rot = 0.0;
    for (int a = 0; a < 3; ++a) {
      align += mm[a] * D[a][mu];
      adv += uu[a] * dm[a][mu];
      rot += W[mu][a] * mm[a];
    }
    R[mu] = h[mu] / gamma1 + xi * align - adv + rot;
  }
  const double mR = mm[0] * R[0] + mm[1] * R[1] + mm[2] * R[2];
  for (int mu = 0; mu < 3; ++mu) R[mu] -= mR * mm[mu];
}

// Elastic stress, Eq. 6 for the energy of G1:
// sigma_ab = -d_a n_c * dE/d(d_b n_c) = -K d_a n_c d_b n_c - K q0 eps_{mu b c} n_mu d_a n_c.
void elastic_stress_cell(const Grid& G, double K, double q0, const double* n, int x, int y, int z,
                         double sig[3][3], const double* pi = nullptr) {
  const size_t N = G.N();
  const size_t c0 = G.at(x, y, z);
  double dn[3][3];
  for (int b = 0; b < 3; ++b)
    for (int c = 0; c < 3; ++c) dn[b][c] = ddx(G, n, c, x, y, z, b);
  if (pi) {  // three constants: sigma_ab = -d_a n_c pi_{b c} (Eq. 6)
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        double s = 0.0;
        for (int c = 0; c < 3; ++c) s -= dn[a][c] * pi[(3 * b + c) * N + c0];
        sig[a][b] = s;
      }
    return;
  }
  const double nn[3] = {n[c0], n[N + c0], n[2 * N + c0]};
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      double s = 0.0;
      for (int c = 0; c < 3; ++c) {
        s += -K * dn[a][c] * dn[b][c];
        for (int mu = 0; mu < 3; ++mu) s += -K * q0 * levi_civita(mu, b, c) * nn[mu] * dn[a][c];
      }
      sig[a][b] = s;
    }
}

void elastic_stress_field(const Grid& G, double K, double q0, const double* n, double* sigma,
                          const double* pi = nullptr) {
  const size_t N = G.N();
  std::memset(sigma, 0, sizeof(double) * 9 * N);  // sigma = 0 on the plate layers (G6)
#pragma omp parallel for schedule(static)
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < G.ny; ++y)
      for (int x = 0; x < G.nx; ++x) {
        double s[3][3];
        elastic_stress_cell(G, K, q0, n, x, y, z, s, pi);
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) sigma[(3 * a + b) * N + G.at(x, y, z)] = s[a][b];
      }
}

// F^LC_a = d_b sigma_ab by central differences: the last term of Eq. 12.
void elastic_force_field(const Grid& G, double K, double q0, const double* n, double* F,
                         std::vector<double>& sigma) {
  const size_t N = G.N();
  sigma.resize(9 * N);
  elastic_stress_field(G, K, q0, n, sigma.data());
  std::memset(F, 0, sizeof(double) * 3 * N);
#pragma omp parallel for schedule(static)
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < G.ny; ++y)
      for (int x = 0; x < G.nx; ++x)
        for (int a = 0; a < 3; ++a) {
          double s = 0.0;
          for (int b = 0; b < 3; ++b) s += ddx(G, sigma.data(), 3 * a + b, x, y, z, b);
          F[a * N + G.at(x, y, z)] = s;
        }
}

// Leslie viscous stress, Eq. 3 as it enters the force of Eq. 12, with
// alpha_4 replaced by alpha_4':
//   sigma^v_ab = a1 n_a n_b n_m n_r D_mr + a2 n_b N_a + a3 n_a N_b + a4' D_ab + a5 n_b n_m D_ma + a6 n_a n_m D_mb
// al[] = {alpha1, alpha2, alpha3, alpha4', alpha5, alpha6}.  D as printed in Eq. 5.  The co-rotational
// rate N of Eq. 4 is taken from Eq. 9: N = d_t n + (u.grad) n - W.n = h/gamma1 + xi n.D, projected
// perpendicular to n like the director's rate itself (reading G22), so no time derivative
// is needed.
void viscous_stress_cell(const Grid& G, double K, double q0, double xi, double gamma1, const double al[6],
                         const double* n, const double* u, int x, int y, int z, double sig[3][3],
                         const double* pi = nullptr, const double* dfdn = nullptr) {
  const size_t N = G.N();
  const size_t c0 = G.at(x, y, z);
  double du[3][3];  // d_b u_c
  for (int b = 0; b < 3; ++b)
    for (int c = 0; c < 3; ++c) du[b][c] = ddx(G, u, c, x, y, z, b);
  double D[3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) D[a][b] = 0.5 * (du[a][b] + du[b][a]);
  const double nn[3] = {n[c0], n[N + c0], n[2 * N + c0]};
  double h[3];
  if (pi) frank3_h_cell(G, n, pi, dfdn, x, y, z, h);
  else molecular_field_cell(G, K, q0, n, x, y, z, h);
  double nD[3], A[3];  // nD_b = n_m D_mb
  for (int b = 0; b < 3; ++b) {
    nD[b] = 0.0;
    for (int m = 0; m < 3; ++m) nD[b] += nn[m] * D[m][b];
    A[b] = h[b] / gamma1 + xi * nD[b];
  }
  const double nA = nn[0] * A[0] + nn[1] * A[1] + nn[2] * A[2];
  double Nr[3];
  for (int b = 0; b < 3; ++b) Nr[b] = A[b] - nA * nn[b];
  double nnD = 0.0;  // n_m n_r D_mr
  for (int m = 0; m < 3; ++m) nnD += nn[m] * nD[m];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      sig[a][b] = al[0] * nn[a] * nn[b] * nnD + al[1] * nn[b] * Nr[a] + al[2] * nn[a] * Nr[b] +
                  al[3] * D[a][b] + al[4] * nn[b] * nD[a] + al[5] * nn[a] * nD[b];
}

bool any_alpha(const double al[6]) {
  for (int i = 0; i < 6; ++i)
    if (al[i] != 0.0) return true;
  return false;
}

// sigma (+)= sigma^v on the computed layers; the plate layers stay 0 (G6).
void viscous_stress_add(const Grid& G, double K, double q0, double xi, double gamma1, const double al[6],
                        const double* n, const double* u, double* sigma,
                        const double* pi = nullptr, const double* dfdn = nullptr) {
  const size_t N = G.N();
#pragma omp parallel for schedule(static)
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < G.ny; ++y)
      for (int x = 0; x < G.nx; ++x) {
        double s[3][3];
        viscous_stress_cell(G, K, q0, xi, gamma1, al, n, u, x, y, z, s, pi, dfdn);
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) sigma[(3 * a + b) * N + G.at(x, y, z)] += s[a][b];
      }
}

// F^LC_a = d_b (sigma^e_ab + sigma^v_ab) by central differences: Eq. 12.
void lc_force_field(const Grid& G, double K, double q0, double xi, double gamma1, const double al[6],
                    const double* n, const double* u, double* F, std::vector<double>& sigma,
                    const double* K3 = nullptr) {
  const size_t N = G.N();
  sigma.resize(9 * N);
  std::vector<double> pi, dfdn;
  const double* ppi = nullptr;
  const double* pdf = nullptr;
  if (K3 && any_K3(K3)) {
    pi.resize(9 * N);
    dfdn.resize(3 * N);
    frank3_fields(G, K3, q0, n, pi.data(), dfdn.data());
    ppi = pi.data();
    pdf = dfdn.data();
  }
  elastic_stress_field(G, K, q0, n, sigma.data(), ppi);
  if (any_alpha(al)) viscous_stress_add(G, K, q0, xi, gamma1, al, n, u, sigma.data(), ppi, pdf);
  std::memset(F, 0, sizeof(double) * 3 * N);
#pragma omp parallel for schedule(static)
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < G.ny; ++y)
      for (int x = 0; x < G.nx; ++x)
        for (int a = 0; a < 3; ++a) {
          double s = 0.0;
          for (int b = 0; b < 3; ++b) s += ddx(G, sigma.data(), 3 * a + b, x, y, z, b);
          F[a * N + G.at(x, y, z)] = s;
        }
}

void director_rhs_field(const Grid& G, double K, double q0, double xi, double gamma1,
                        const double* m, const double* u, double* R, const double* K3 = nullptr) {
  const size_t N = G.N();
  std::memset(R, 0, sizeof(double) * 3 * N);
  std::vector<double> pi, dfdn;
  const double* ppi = nullptr;
  const double* pdf = nullptr;
  if (K3 && any_K3(K3)) {
    pi.resize(9 * N);
    dfdn.resize(3 * N);
    frank3_fields(G, K3, q0, m, pi.data(), dfdn.data());
    ppi = pi.data();
    pdf = dfdn.data();
  }
#pragma omp parallel for schedule(static)
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < G.ny; ++y)
      for (int x = 0; x < G.nx; ++x) {
        double r[3];
        director_rhs_cell(G, K, q0, xi, gamma1, m, u, x, y, z, r, ppi, pdf);
        for (int c = 0; c < 3; ++c) R[c * N + G.at(x, y, z)] = r[c];
      }
}

bool bad_dims(int nx, int ny, int nz) { return nx < 1 || ny < 1 || nz < 3; }

}  // namespace

struct nh_oracle_lattice {
  nh_oracle_params p;
  Grid G;
  double q0;
  bool shifted;
  long t;
  std::vector<double> f, fnew;            // populations [i][cell]: f^shifted (Eq. 19) or f
  std::vector<double> n, nP, nnew, u, F;  // director, predictor, velocity scratch, F^LC
  std::vector<double> k1, k2, sigma, uv;  // uv: u(t) for the viscous stress (whatever coupling bit1 says)

  // Moments of one fluid cell.  Shifted: Eqs. 20-21; unshifted: Eqs. 16-17
  // (PAPER.md:131-135).  Ftot = [coupling bit0] F^LC + rho g (reading G8).
  void moments(size_t c, double& drho, double& rho, double uu[3], double Ftot[3]) const {
    const size_t N = G.N();
    double s = 0.0, j[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < Q; ++i) {
      const double fi = f[i * N + c];
      s += fi;
      j[0] += EX[i] * fi;
      j[1] += EY[i] * fi;
      j[2] += EZ[i] * fi;
    }
    if (shifted) { drho = s; rho = 1.0 + drho; }   // Eq. 20
    else         { rho = s;  drho = rho - 1.0; }   // Eq. 16
    for (int a = 0; a < 3; ++a) {
      const double flc = (p.coupling & 1) ? F[a * N + c] : 0.0;
      Ftot[a] = flc + rho * p.g[a];
      uu[a] = (j[a] + 0.5 * Ftot[a]) / rho;        // Eq. 21 / Eq. 17, Delta t = 1
    }
  }

  // One LB step: equilibrium, collision, streaming with half-way bounce-back (Fig. 1).
  void lb_step() {
    const size_t N = G.N();
    const double tau = p.tau;
#pragma omp parallel for schedule(static)
    for (int z = 1; z < G.nz - 1; ++z)
      for (int y = 0; y < G.ny; ++y)
        for (int x = 0; x < G.nx; ++x) {
          const size_t c = G.at(x, y, z);
          double drho, rho, uu[3], Ft[3];
          moments(c, drho, rho, uu, Ft);
          const double u2 = uu[0] * uu[0] + uu[1] * uu[1] + uu[2] * uu[2];
          const double uF = uu[0] * Ft[0] + uu[1] * Ft[1] + uu[2] * Ft[2];
          for (int i = 0; i < Q; ++i) {
            const double w = weight(i);
            const double eu = EX[i] * uu[0] + EY[i] * uu[1] + EZ[i] * uu[2];
            const double eF = EX[i] * Ft[0] + EY[i] * Ft[1] + EZ[i] * Ft[2];
            // Eq. 22 (shifted) or Eq. 15 (unshifted), c_s^2 = 1/3
            const double bracket = 3.0 * eu + 4.5 * eu * eu - 1.5 * u2;
            const double feq = shifted ? w * rho * bracket + drho * w : w * rho * (1.0 + bracket);
            // Eq. 18: (e.F)/c_s^2 + (e e - c_s^2 I):(uF + Fu)/(2 c_s^4) = 3 e.F + 9 (e.u)(e.F) - 3 u.F
            const double S = w * (3.0 * eF + 9.0 * eu * eF - 3.0 * uF);
            const double fi = f[i * N + c];
            // Eq. 23 / Eq. 14 with Delta t = 1 (G13)
            const double fstar = fi - (fi - feq) / tau + (1.0 - 1.0 / (2.0 * tau)) * S;
            // streaming: x + e_i, periodic in x and y; plates at z = 0 and nz-1
            const int zz = z + EZ[i];
            if (zz == 0 || zz == G.nz - 1) {
              fnew[opposite(i) * N + c] = fstar;  // half-way bounce-back: reflected, same node
            } else {
              fnew[i * N + G.at(G.wx(x + EX[i]), G.wy(y + EY[i]), zz)] = fstar;
            }
          }
        }
    f.swap(fnew);
    t += 1;
  }

  // rho, u on the whole grid from the current populations and the current F^LC (steps 5, a6).
  void velocity_field(double* rho_out, double* u_out) const {
    const size_t N = G.N();
    for (size_t c = 0; c < N; ++c) {
      if (rho_out) rho_out[c] = 1.0;
      if (u_out) u_out[c] = u_out[N + c] = u_out[2 * N + c] = 0.0;  // no-slip solid value (G6)
    }
#pragma omp parallel for schedule(static)
    for (int z = 1; z < G.nz - 1; ++z)
      for (int y = 0; y < G.ny; ++y)
        for (int x = 0; x < G.nx; ++x) {
          const size_t c = G.at(x, y, z);
          double drho, rho, uu[3], Ft[3];
          moments(c, drho, rho, uu, Ft);
          if (rho_out) rho_out[c] = rho;
          if (u_out)
            for (int a = 0; a < 3; ++a) u_out[a * N + c] = uu[a];
        }
  }

  void normalise_into(std::vector<double>& dst, const std::vector<double>& base,
                      const std::vector<double>& ka, const std::vector<double>* kb, double dt) {
    const size_t N = G.N();
    dst = n;  // plate layers keep their fixed values
#pragma omp parallel for schedule(static)
    for (int z = 1; z < G.nz - 1; ++z)
      for (int y = 0; y < G.ny; ++y)
        for (int x = 0; x < G.nx; ++x) {
          const size_t c = G.at(x, y, z);
          double v[3];
          for (int a = 0; a < 3; ++a) {
            const double rate = kb ? 0.5 * (ka[a * N + c] + (*kb)[a * N + c]) : ka[a * N + c];
            v[a] = base[a * N + c] + dt * rate;
          }
          const double len = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
          for (int a = 0; a < 3; ++a) dst[a * N + c] = v[a] / len;  // renormalise (G3)
        }
    mirror_plates(dst);
  }

  // Free plates (anchoring = 1, "no anchoring at the plates"; reading G23): the plate
  // layers carry no director of their own, they copy the adjacent fluid layer (zero normal
  // derivative), so the stencils at z = 1 and z = nz-2 see no anchoring torque.
  void mirror_plates(std::vector<double>& m) const {
    if (p.anchoring != 1) return;
    const size_t N = G.N();
    for (int a = 0; a < 3; ++a)
      for (int y = 0; y < G.ny; ++y)
        for (int x = 0; x < G.nx; ++x) {
          m[a * N + G.at(x, y, 0)] = m[a * N + G.at(x, y, 1)];
          m[a * N + G.at(x, y, G.nz - 1)] = m[a * N + G.at(x, y, G.nz - 2)];
        }
  }

  // F^LC from the current director (and, for the viscous part, the current velocity).
  void lc_force(bool have_u) {
    const double* uu = u.data();
    if (any_alpha(p.alpha)) {
      if (!have_u) { uv.resize(3 * G.N()); velocity_field(nullptr, uv.data()); uu = uv.data(); }
    }
    lc_force_field(G, p.K, q0, p.xi, p.gamma1, p.alpha, n.data(), uu, F.data(), sigma, p.K3);
  }

  // FD update with Delta t_FD = r, same u for both stages (G11).
  void fd_update(int r) {
    const size_t N = G.N();
    if (p.coupling & 2) velocity_field(nullptr, u.data());
    else std::fill(u.begin(), u.end(), 0.0);
    const double dt = (double)r;
    director_rhs_field(G, p.K, q0, p.xi, p.gamma1, n.data(), u.data(), k1.data(), p.K3);   // (d_t n)_old
    normalise_into(nP, n, k1, nullptr, dt);                                          // predictor
    director_rhs_field(G, p.K, q0, p.xi, p.gamma1, nP.data(), u.data(), k2.data(), p.K3);  // (d_t n)_P
    normalise_into(nnew, n, k1, &k2, dt);                                            // corrector
    n.swap(nnew);
    lc_force(/*have_u=*/(p.coupling & 2) != 0);                                     // Eq. 12
    (void)N;
  }
};

extern "C" {

const char* nh_oracle_last_error(void) { return g_err.c_str(); }

int nh_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int nh_oracle_init_lattice(const nh_oracle_params* p, nh_oracle_lattice** out) {
  if (!p || !out) return fail(E_INVAL, "null pointer");
  if (bad_dims(p->nx, p->ny, p->nz)) return fail(E_INVAL, "need nx, ny >= 1 and nz >= 3");
  if (!(p->tau > 0.5)) return fail(E_INVAL, "tau must be > 0.5");
  if (!(p->gamma1 > 0.0)) return fail(E_INVAL, "gamma1 must be > 0");
  if (p->K < 0.0) return fail(E_INVAL, "K must be >= 0");
  for (int i = 0; i < 3; ++i)
    if (!(p->K3[i] >= 0.0)) return fail(E_INVAL, "K11, K22, K33 must be >= 0");
  if (p->fd_ratio < 0) return fail(E_INVAL, "fd_ratio must be >= 0");
  if (p->precision < 0 || p->precision > 3) return fail(E_INVAL, "precision must be 0..3");
  if (p->anchoring != 0 && p->anchoring != 1) return fail(E_INVAL, "anchoring must be 0 (homeotropic plates) or 1 (free plates)");
  if (!std::isfinite(p->W0)) return fail(E_INVAL, "W0 must be finite");
  nh_oracle_lattice* L = new (std::nothrow) nh_oracle_lattice();
  if (!L) return fail(E_NOMEM, "out of memory");
  try {
    L->p = *p;
    L->G = Grid{p->nx, p->ny, p->nz, false};
    L->G.W0 = p->W0;
    L->q0 = p->pitch > 0.0 ? 2.0 * M_PI / p->pitch : 0.0;
    L->shifted = (p->precision == 0 || p->precision == 1);
    L->t = 0;
    const size_t N = L->G.N();
    // rho = 1, u = 0: f_i = w_i, i.e. f^shifted = 0 (Eq. 19); plate layers hold no populations
    L->f.assign(Q * N, 0.0);
    if (!L->shifted)
      for (int i = 0; i < Q; ++i)
        for (int z = 1; z < p->nz - 1; ++z)
          for (int y = 0; y < p->ny; ++y)
            for (int x = 0; x < p->nx; ++x) L->f[i * N + L->G.at(x, y, z)] = weight(i);
    L->fnew = L->f;
    L->n.assign(3 * N, 0.0);
    for (size_t c = 0; c < N; ++c) L->n[2 * N + c] = 1.0;  // n = z_hat
    L->nP = L->n;
    L->nnew = L->n;
    L->u.assign(3 * N, 0.0);
    L->F.assign(3 * N, 0.0);
    L->k1.assign(3 * N, 0.0);
    L->k2.assign(3 * N, 0.0);
  } catch (const std::bad_alloc&) {
    delete L;
    return fail(E_NOMEM, "out of memory");
  }
  *out = L;
  return 0;
}

int nh_oracle_set_director(nh_oracle_lattice* L, const double* n_host) {
  if (!L || !n_host) return fail(E_INVAL, "null pointer");
  const size_t N = L->G.N();
  for (size_t c = 0; c < N; ++c) {
    const double a = n_host[c], b = n_host[N + c], d = n_host[2 * N + c];
    const double len = std::sqrt(a * a + b * b + d * d);
    if (!(len > 0.0) || !std::isfinite(len)) return fail(E_INVAL, "zero-length or non-finite director");
  }
  for (size_t c = 0; c < N; ++c) {
    const double a = n_host[c], b = n_host[N + c], d = n_host[2 * N + c];
    const double len = std::sqrt(a * a + b * b + d * d);
    L->n[c] = a / len;
    L->n[N + c] = b / len;
    L->n[2 * N + c] = d / len;
  }
  // infinite homeotropic anchoring: plate layers hold z_hat and never change;
  // free plates (anchoring = 1): they copy the adjacent fluid layer instead
  L->mirror_plates(L->n);
  for (int zz = 0; zz < 2 && L->p.anchoring == 0; ++zz) {
    const int z = zz == 0 ? 0 : L->G.nz - 1;
    for (int y = 0; y < L->G.ny; ++y)
      for (int x = 0; x < L->G.nx; ++x) {
        const size_t c = L->G.at(x, y, z);
        L->n[c] = 0.0;
        L->n[N + c] = 0.0;
        L->n[2 * N + c] = 1.0;
      }
  }
  L->nP = L->n;
  L->lc_force(/*have_u=*/false);  // reading G9
  return 0;
}

int nh_oracle_step(nh_oracle_lattice* L, int n_lb, int n_fd) {
  if (!L) return fail(E_INVAL, "null pointer");
  if (n_lb < 0) return fail(E_INVAL, "n_lb must be >= 0");
  const int r = n_fd < 0 ? L->p.fd_ratio : n_fd;
  for (int s = 0; s < n_lb; ++s) {
    L->lb_step();
    if (r > 0 && L->t % r == 0) L->fd_update(r);  // PAPER.md:204, reading G10
  }
  return 0;
}

int nh_oracle_get_fields(nh_oracle_lattice* L, double* rho, double* u, double* n, double* F_lc) {
  if (!L) return fail(E_INVAL, "null pointer");
  const size_t N = L->G.N();
  if (rho || u) L->velocity_field(rho, u);
  if (n) std::memcpy(n, L->n.data(), sizeof(double) * 3 * N);
  if (F_lc) std::memcpy(F_lc, L->F.data(), sizeof(double) * 3 * N);
  return 0;
}

int nh_oracle_get_populations(nh_oracle_lattice* L, double* f) {
  if (!L || !f) return fail(E_INVAL, "null pointer");
  std::memcpy(f, L->f.data(), sizeof(double) * Q * L->G.N());
  return 0;
}

// Test-only entry (pins P12, P13): overwrite the populations of every fluid cell with the
// equilibrium of (rho = 1, u) -- Eq. 15, or Eq. 22 in shifted form.  Not part of the product ABI.
int nh_oracle_set_velocity(nh_oracle_lattice* L, const double* u_host) {
  if (!L || !u_host) return fail(E_INVAL, "null pointer");
  const size_t N = L->G.N();
  for (int z = 1; z < L->G.nz - 1; ++z)
    for (int y = 0; y < L->G.ny; ++y)
      for (int x = 0; x < L->G.nx; ++x) {
        const size_t c = L->G.at(x, y, z);
        const double uu[3] = {u_host[c], u_host[N + c], u_host[2 * N + c]};
        const double u2 = uu[0] * uu[0] + uu[1] * uu[1] + uu[2] * uu[2];
        for (int i = 0; i < Q; ++i) {
          const double eu = EX[i] * uu[0] + EY[i] * uu[1] + EZ[i] * uu[2];
          const double bracket = 3.0 * eu + 4.5 * eu * eu - 1.5 * u2;
          L->f[i * N + c] = L->shifted ? weight(i) * bracket : weight(i) * (1.0 + bracket);
        }
      }
  return 0;
}

long nh_oracle_time(const nh_oracle_lattice* L) { return L ? L->t : -1; }

void nh_oracle_free(nh_oracle_lattice* L) { delete L; }

int nh_oracle_molecular_field(int nx, int ny, int nz, int periodic_z, double K, double q0,
                              const double* n, double* h) {
  if (!n || !h || bad_dims(nx, ny, nz)) return fail(E_INVAL, "bad arguments");
  const Grid G{nx, ny, nz, periodic_z != 0};
  const size_t N = G.N();
  std::memset(h, 0, sizeof(double) * 3 * N);
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        double hh[3];
        molecular_field_cell(G, K, q0, n, x, y, z, hh);
        for (int c = 0; c < 3; ++c) h[c * N + G.at(x, y, z)] = hh[c];
      }
  return 0;
}

int nh_oracle_molecular_field_w0(int nx, int ny, int nz, int periodic_z, double K, double q0, double W0,
                                 const double* n, double* h) {
  if (!n || !h || bad_dims(nx, ny, nz)) return fail(E_INVAL, "bad arguments");
  Grid G{nx, ny, nz, periodic_z != 0};
  G.W0 = W0;
  const size_t N = G.N();
  std::memset(h, 0, sizeof(double) * 3 * N);
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        double hh[3];
        molecular_field_cell(G, K, q0, n, x, y, z, hh);
        for (int c = 0; c < 3; ++c) h[c * N + G.at(x, y, z)] = hh[c];
      }
  return 0;
}

int nh_oracle_director_rhs(int nx, int ny, int nz, int periodic_z, double K, double q0, double xi,
                           double gamma1, const double* n, const double* u, double* R) {
  if (!n || !u || !R || bad_dims(nx, ny, nz) || !(gamma1 > 0.0)) return fail(E_INVAL, "bad arguments");
  const Grid G{nx, ny, nz, periodic_z != 0};
  director_rhs_field(G, K, q0, xi, gamma1, n, u, R);
  return 0;
}

int nh_oracle_elastic_stress(int nx, int ny, int nz, int periodic_z, double K, double q0,
                             const double* n, double* sigma) {
  if (!n || !sigma || bad_dims(nx, ny, nz)) return fail(E_INVAL, "bad arguments");
  const Grid G{nx, ny, nz, periodic_z != 0};
  elastic_stress_field(G, K, q0, n, sigma);
  return 0;
}

int nh_oracle_elastic_force(int nx, int ny, int nz, int periodic_z, double K, double q0,
                            const double* n, double* F) {
  if (!n || !F || bad_dims(nx, ny, nz)) return fail(E_INVAL, "bad arguments");
  const Grid G{nx, ny, nz, periodic_z != 0};
  std::vector<double> sigma;
  elastic_force_field(G, K, q0, n, F, sigma);
  return 0;
}

/* three-constant energy (row f2): K3 = {K11, K22, K33}; E = sum of f over the computed layers */
int nh_oracle_frank3(int nx, int ny, int nz, int periodic_z, const double* K3, double q0, const double* n,
                     double* h, double* sigma, double* energy) {
  if (!n || !K3 || bad_dims(nx, ny, nz)) return fail(E_INVAL, "bad arguments");
  const Grid G{nx, ny, nz, periodic_z != 0};
  const size_t N = G.N();
  std::vector<double> pi(9 * N), dfdn(3 * N);
  frank3_fields(G, K3, q0, n, pi.data(), dfdn.data());
  if (h) std::memset(h, 0, sizeof(double) * 3 * N);
  if (sigma) std::memset(sigma, 0, sizeof(double) * 9 * N);
  double E = 0.0;
  for (int z = G.z_lo(); z < G.z_hi(); ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        const size_t c0 = G.at(x, y, z);
        if (h) {
          double hh[3];
          frank3_h_cell(G, n, pi.data(), dfdn.data(), x, y, z, hh);
          for (int c = 0; c < 3; ++c) h[c * N + c0] = hh[c];
        }
        if (sigma) {
          double s[3][3];
          elastic_stress_cell(G, 0.0, q0, n, x, y, z, s, pi.data());
          for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) sigma[(3 * a + b) * N + c0] = s[a][b];
        }
        double p[3][3], d[3], f;
        frank3_cell(G, K3, q0, n, x, y, z, p, d, &f);
        E += f;
      }
  if (energy) *energy = E;
  return 0;
}

int nh_oracle_viscous_stress(int nx, int ny, int nz, int periodic_z, double K, double q0, double xi,
                             double gamma1, const double* alpha, const double* n, const double* u,
                             double* sigma) {
  if (!n || !u || !sigma || !alpha || bad_dims(nx, ny, nz) || !(gamma1 > 0.0)) return fail(E_INVAL, "bad arguments");
  const Grid G{nx, ny, nz, periodic_z != 0};
  std::memset(sigma, 0, sizeof(double) * 9 * G.N());
  viscous_stress_add(G, K, q0, xi, gamma1, alpha, n, u, sigma);
  return 0;
}

int nh_oracle_lc_force(int nx, int ny, int nz, int periodic_z, double K, double q0, double xi,
                       double gamma1, const double* alpha, const double* n, const double* u, double* F) {
  if (!n || !u || !F || !alpha || bad_dims(nx, ny, nz) || !(gamma1 > 0.0)) return fail(E_INVAL, "bad arguments");
  const Grid G{nx, ny, nz, periodic_z != 0};
  std::vector<double> sigma;
  lc_force_field(G, K, q0, xi, gamma1, alpha, n, u, F, sigma);
  return 0;
}

}  // extern "C"
