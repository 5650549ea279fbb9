// =====================================================================================
// lbm_oracle.cpp -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, scalar fp64 implementation of one lattice Boltzmann time step of
// arxiv 2506.21804, in the BGK + Smagorinsky + HLBM reading that
// BASELINE.json names (reading G1).  It exists to check the CUDA path.  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call it.  It shares no code, header, table or constant with
// paper_2506_21804_b200/ (the product), and neither side includes the other.
//
// Kind of result: the method is an explicit time iteration, so the oracle is the algorithm
// itself, one loop nest per sub-step (O1..O5), two lattices, no fusion, no blocking, no
// algebraic rearrangement beyond what the cited passage states.
//
// Passages followed (PAPER.md line : equation):
//   O0 lattice tables      l.60 (D3Q19 named; table not printed -> DESIGN.md reading G13/R1)
//   O1 wall-model pre-pass l.117-131, Eq. 15-17 (Spalding law), coupling l.131 (reading G17/R8)
//   O2 collide             Eq. 6 (l.70) with f~(1) = f - f^eq (G1); Eq. 11 (l.94) up to H(2);
//                          Eq. 12 (l.99); Eq. 3-5 + Eq. 14 (l.50-56, l.110) closed form (G3-G8)
//   O3 stream              Eq. 6 left-hand side (l.70); halfway bounce-back (G14/R5);
//                          zero-gradient outlet (G16/R7)
//   O4 inlet fix-up        l.155 "regularized local velocity boundary condition" (G15/R6)
//   O6 moments             l.97 "fluid velocity moment u" (G19)
//
// Pins (tests/test_oracle_*.py, all run with -m "not gpu"): P1 isotropy identities, P2
// equilibrium fixed point, P3 conservation, P4 Cs=0 == separately written BGK, P5 porous
// decay closed form, P6 tau_eff self-consistency, P7 Taylor-Green decay vs exp(-4 nu k^2 t),
// P8 Poiseuille profile, P9 Spalding residual + viscous/log limits, P10 inlet moments /
// idempotence, P11a long-double brute force on 4^3, P12 bounce-back pulse + mass, P13 second
// order convergence, P14 lattice symmetry, P15 D3Q27.
// PARITY UNPINNED against the paper (no worked example printed): the wall-model coupling
// reading G17, the outlet rule G16 and the inlet variant G15.  They are pinned only as
// textbook definitions through P8, P9, P10.
//
// Layouts (all row-major, x fastest): f[Q][nz][ny][nx] double, d[nz][ny][nx] double,
// flag[nz][ny][nx] uint8.  Cell index = (z*ny + y)*nx + x.
// Flag byte: low nibble type {0 FLUID,1 SOLID,2 INLET,3 OUTLET,4 WALLMODEL}; for WALLMODEL the
// high nibble is the wall-normal code {0:+x,1:-x,2:+y,3:-y,4:+z,5:-z} (wall -> fluid).
// =====================================================================================
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int QMAX = 27;
enum CellType : int { FLUID = 0, SOLID = 1, INLET = 2, OUTLET = 3, WALLMODEL = 4 };

struct Lattice {
  int Q = 0;
  int c[QMAX][3];
  double w[QMAX];
  int opp[QMAX];
};

// O0 (reading R1). i = 0 is rest.  Directions 1..h (h = (Q-1)/2) are those whose first non-zero
// component is +1, sorted ascending by (|c|^2, -c_x, -c_y, -c_z); h+1..Q-1 are their negatives
// in the same order, hence opp(i) = i +- h.  D3Q19 keeps |c|^2 <= 2, D3Q27 keeps |c|^2 <= 3.
// Weights: D3Q19 1/3, 1/18, 1/36; D3Q27 8/27, 2/27, 1/54, 1/216 (by |c|^2 = 0,1,2,3).
bool make_lattice(int Q, Lattice& L) {
  if (Q != 19 && Q != 27) return false;
  const int max_c2 = (Q == 19) ? 2 : 3;
  L.Q = Q;
  struct Dir { int c2, x, y, z; };
  std::vector<Dir> half;
  for (int x = -1; x <= 1; ++x)
    for (int y = -1; y <= 1; ++y)
      for (int z = -1; z <= 1; ++z) {
        const int c2 = x * x + y * y + z * z;
        if (c2 == 0 || c2 > max_c2) continue;
        const int first = (x != 0) ? x : ((y != 0) ? y : z);
        if (first == 1) half.push_back({c2, x, y, z});
      }
  // insertion sort on the key (c2, -x, -y, -z)
  for (size_t a = 1; a < half.size(); ++a)
    for (size_t b = a; b > 0; --b) {
      const Dir& p = half[b - 1];
      const Dir& q = half[b];
      const int kp[4] = {p.c2, -p.x, -p.y, -p.z};
      const int kq[4] = {q.c2, -q.x, -q.y, -q.z};
      bool less = false;
      for (int k = 0; k < 4; ++k) {
        if (kq[k] < kp[k]) { less = true; break; }
        if (kq[k] > kp[k]) break;
      }
      if (!less) break;
      Dir t = half[b - 1]; half[b - 1] = half[b]; half[b] = t;
    }
  const int h = (Q - 1) / 2;
  if (static_cast<int>(half.size()) != h) return false;
  L.c[0][0] = L.c[0][1] = L.c[0][2] = 0;
  L.opp[0] = 0;
  for (int k = 0; k < h; ++k) {
    L.c[1 + k][0] = half[k].x;  L.c[1 + k][1] = half[k].y;  L.c[1 + k][2] = half[k].z;
    L.c[1 + h + k][0] = -half[k].x;  L.c[1 + h + k][1] = -half[k].y;  L.c[1 + h + k][2] = -half[k].z;
    L.opp[1 + k] = 1 + h + k;
    L.opp[1 + h + k] = 1 + k;
  }
  for (int i = 0; i < Q; ++i) {
    const int c2 = L.c[i][0] * L.c[i][0] + L.c[i][1] * L.c[i][1] + L.c[i][2] * L.c[i][2];
    if (Q == 19) L.w[i] = (c2 == 0) ? 1.0 / 3.0 : (c2 == 1) ? 1.0 / 18.0 : 1.0 / 36.0;
    else         L.w[i] = (c2 == 0) ? 8.0 / 27.0 : (c2 == 1) ? 2.0 / 27.0 : (c2 == 2) ? 1.0 / 54.0 : 1.0 / 216.0;
  }
  return true;
}

struct Params {           // the oracle's own copy of the step parameters (not shared with the product)
  double tau0;
  double cs_smago;
  int use_hlbm;
  double u_in[3];
  int wm_enable;
  double wm_kappa;
  double wm_E;
};

inline int cell_type(uint8_t flag) { return flag & 0x0F; }

// A4.  Eq. 11 (l.94) truncated after the H(2) term, c_s^2 = 1/3:
// f_i^eq = w_i rho (1 + 3 c.u + 4.5 (c.u)^2 - 1.5 u.u)
inline double feq_i(const Lattice& L, int i, double rho, const double u[3]) {
  const double cu = L.c[i][0] * u[0] + L.c[i][1] * u[1] + L.c[i][2] * u[2];
  const double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
  return L.w[i] * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
}

// A2.  rho = sum_i f_i,  u = sum_i c_i f_i / rho   (l.97, Listing 1 l.179-185)
inline void raw_moments(const Lattice& L, const double* fc, double& rho, double u[3]) {
  rho = 0.0;
  double j[3] = {0.0, 0.0, 0.0};
  for (int i = 0; i < L.Q; ++i) {
    rho += fc[i];
    j[0] += L.c[i][0] * fc[i];
    j[1] += L.c[i][1] * fc[i];
    j[2] += L.c[i][2] * fc[i];
  }
  u[0] = j[0] / rho;  u[1] = j[1] / rho;  u[2] = j[2] / rho;
}

// O2 for one cell.  fc[Q] in, fs[Q] out.  d = porosity (Eq. 12 convention: 0 fluid, 1 solid),
// ub = solid velocity u^B.  Returns tau_eff through *tau_out when non-null.
void collide_cell(const Lattice& L, const double* fc, double d, const double ub[3],
                  double tau0, double cs_smago, double* fs, double* tau_out) {
  double rho, u[3];
  raw_moments(L, fc, rho, u);                                            // A2
  double uh[3];
  for (int a = 0; a < 3; ++a) uh[a] = (1.0 - d) * u[a] + d * ub[a];      // A3, Eq. 12
  double feq[QMAX];
  for (int i = 0; i < L.Q; ++i) feq[i] = feq_i(L, i, rho, uh);           // A4, Eq. 11
  double tau = tau0;
  if (cs_smago > 0.0) {                                                  // A5, Eq. 3-5 + Eq. 14
    double Pi[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    for (int i = 0; i < L.Q; ++i)
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) Pi[a][b] += L.c[i][a] * L.c[i][b] * (fc[i] - feq[i]);
    const double nPi = std::sqrt(Pi[0][0] * Pi[0][0] + Pi[1][1] * Pi[1][1] + Pi[2][2] * Pi[2][2] +
                                 2.0 * (Pi[0][1] * Pi[0][1] + Pi[0][2] * Pi[0][2] + Pi[1][2] * Pi[1][2]));
    tau = 0.5 * (tau0 + std::sqrt(tau0 * tau0 + 18.0 * std::sqrt(2.0) * cs_smago * cs_smago * nPi / rho));
  }
  for (int i = 0; i < L.Q; ++i) fs[i] = fc[i] - (fc[i] - feq[i]) / tau;  // A6, Eq. 6
  if (tau_out) *tau_out = tau;
}

// Eq. 17 (l.127): y+ = Sp(u+), and its derivative.
inline double spalding(double up, double kappa, double E) {
  const double k = kappa * up;
  return up + (1.0 / E) * (std::exp(k) - 1.0 - k - k * k / 2.0 - k * k * k / 6.0);
}
inline double spalding_du(double up, double kappa, double E) {
  const double k = kappa * up;
  return 1.0 + (kappa / E) * (std::exp(k) - 1.0 - k - k * k / 2.0);
}

// O1 steps 4-7 for one wall-model cell: given the tangential speed U2 sampled at wall distance
// y2, return the modelled tangential speed U1 at wall distance y1.  Also returns u_tau and the
// Newton iteration counts.  (Eq. 15-17; reading R8: y2 = 1.5, y1 = 0.5.)
double wallmodel_speed(double U2, double nu, double kappa, double E, double y2, double y1,
                       double* utau_out, int* it1_out, int* it2_out) {
  // step 5: find u_tau > 0 with  R(u_tau) = Sp(U2/u_tau) - y2 u_tau / nu = 0   (strictly decreasing)
  double ut = std::sqrt(nu * U2 / y2);
  int it1 = 0;
  for (; it1 < 200; ++it1) {
    const double up = U2 / ut;
    const double R = spalding(up, kappa, E) - y2 * ut / nu;
    const double dR = spalding_du(up, kappa, E) * (-U2 / (ut * ut)) - y2 / nu;
    double un = ut - R / dR;
    if (!(un > 0.0)) un = 0.5 * ut;
    const double delta = std::fabs(un - ut);
    ut = un;
    if (delta <= 1e-13 * ut) { ++it1; break; }
  }
  // step 6: find u1+ >= 0 with Sp(u1+) = y1+   (strictly increasing)
  const double y1p = y1 * ut / nu;
  double lg = std::log(E * y1p) / kappa;
  if (!(lg > 0.0)) lg = 0.0;
  double up = (y1p < lg + 1.0) ? y1p : lg + 1.0;
  int it2 = 0;
  for (; it2 < 200; ++it2) {
    const double R = spalding(up, kappa, E) - y1p;
    const double dR = spalding_du(up, kappa, E);
    double un = up - R / dR;
    if (un < 0.0) un = 0.5 * up;
    const double delta = std::fabs(un - up);
    up = un;
    if (delta <= 1e-13 * std::fabs(up)) { ++it2; break; }
  }
  if (utau_out) *utau_out = ut;
  if (it1_out) *it1_out = it1;
  if (it2_out) *it2_out = it2;
  return up * ut;   // U1 = u1+ * u_tau   (Eq. 15)
}

inline void normal_of(uint8_t flag, int n[3]) {
  const int code = (flag >> 4) & 0x0F;
  n[0] = n[1] = n[2] = 0;
  n[code >> 1] = (code & 1) ? -1 : 1;
}

inline int wrap(int a, int n) { return (a < 0) ? a + n : ((a >= n) ? a - n : a); }

// O4 for one inlet cell (inward normal +x).  g[Q] is overwritten.
void inlet_fixup_cell(const Lattice& L, double* g, const double uw[3]) {
  double s0 = 0.0, sm = 0.0;
  for (int i = 0; i < L.Q; ++i) {
    if (L.c[i][0] == 0) s0 += g[i];
    else if (L.c[i][0] < 0) sm += g[i];
  }
  const double rho = (s0 + 2.0 * sm) / (1.0 - uw[0]);
  double feq[QMAX], n[QMAX];
  for (int i = 0; i < L.Q; ++i) feq[i] = feq_i(L, i, rho, uw);
  for (int i = 0; i < L.Q; ++i)
    if (L.c[i][0] <= 0) n[i] = g[i] - feq[i];
  for (int i = 0; i < L.Q; ++i)
    if (L.c[i][0] > 0) n[i] = n[L.opp[i]];                 // bounce-back of the non-equilibrium part
  double Pi[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
  for (int i = 0; i < L.Q; ++i)
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) Pi[a][b] += L.c[i][a] * L.c[i][b] * n[i];
  for (int i = 0; i < L.Q; ++i) {
    double s = 0.0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        s += (L.c[i][a] * L.c[i][b] - ((a == b) ? 1.0 / 3.0 : 0.0)) * Pi[a][b];
    g[i] = feq[i] + 4.5 * L.w[i] * s;                       // w_i / (2 c_s^4) = 4.5 w_i
  }
}

}  // namespace

extern "C" {

// ---- O0 -------------------------------------------------------------------------------------
int orc_lattice(int Q, int* c /*[Q*3]*/, double* w /*[Q]*/, int* opp /*[Q]*/) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  for (int i = 0; i < Q; ++i) {
    c[3 * i + 0] = L.c[i][0];  c[3 * i + 1] = L.c[i][1];  c[3 * i + 2] = L.c[i][2];
    w[i] = L.w[i];
    opp[i] = L.opp[i];
  }
  return 0;
}

// ---- per-cell entry points (used by the pins) ---------------------------------------------
int orc_feq(int Q, double rho, const double* u, double* out) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  for (int i = 0; i < Q; ++i) out[i] = feq_i(L, i, rho, u);
  return 0;
}

int orc_collide_cell(int Q, const double* fc, double d, const double* ub, double tau0, double cs_smago,
                     double* fs, double* tau_out) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  collide_cell(L, fc, d, ub, tau0, cs_smago, fs, tau_out);
  return 0;
}

int orc_inlet_fixup_cell(int Q, double* g, const double* uw) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  inlet_fixup_cell(L, g, uw);
  return 0;
}

double orc_spalding(double up, double kappa, double E) { return spalding(up, kappa, E); }

double orc_wallmodel_speed(double U2, double nu, double kappa, double E, double y2, double y1,
                           double* utau_out, int* it1_out, int* it2_out) {
  return wallmodel_speed(U2, nu, kappa, E, y2, y1, utau_out, it1_out, it2_out);
}

// ---- initial state: f = f^eq(rho, u) per cell (A4) --------------------------------------------
// rho[N], u[3][N] -> f[Q][N]
int orc_init_equilibrium(int Q, int64_t N, const double* rho, const double* u, double* f) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  for (int64_t x = 0; x < N; ++x) {
    const double uc[3] = {u[x], u[N + x], u[2 * N + x]};
    for (int i = 0; i < Q; ++i) f[i * N + x] = feq_i(L, i, rho[x], uc);
  }
  return 0;
}

// ---- the step: S_t -> S_{t+n}  (O1 -> O2 -> O3 -> O4 -> O5, n times) ------------------------------
// f is updated in place (the second lattice is internal).  d and flags may be NULL.
// nthreads <= 1: serial.  nthreads > 1: the same loop nests with "omp parallel for" over z.
// Returns 0, or -1 on bad arguments.
int orc_step(int Q, int nx, int ny, int nz, double* f, const double* d, const uint8_t* flags,
             const double* par /* tau0, cs, use_hlbm, uin0, uin1, uin2, wm_enable, kappa, E */,
             int nsteps, int nthreads) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  if (nx < 1 || ny < 1 || nz < 1 || nsteps < 0) return -1;
  Params p;
  p.tau0 = par[0];  p.cs_smago = par[1];  p.use_hlbm = (par[2] != 0.0);
  p.u_in[0] = par[3];  p.u_in[1] = par[4];  p.u_in[2] = par[5];
  p.wm_enable = (par[6] != 0.0);  p.wm_kappa = par[7];  p.wm_E = par[8];
  if (!(p.tau0 > 0.5) || p.cs_smago < 0.0) return -1;
#ifdef _OPENMP
  const int nth = (nthreads > 1) ? nthreads : 1;
#else
  (void)nthreads;
#endif
  const int64_t N = static_cast<int64_t>(nx) * ny * nz;
  std::vector<double> fstar(static_cast<size_t>(Q) * N);   // post-collision f*
  std::vector<double> g(static_cast<size_t>(Q) * N);       // second lattice
  // compact wall-model list
  std::vector<int64_t> wm_cells;
  std::vector<int32_t> wm_slot;
  if (flags && p.wm_enable) {
    for (int64_t x = 0; x < N; ++x)
      if (cell_type(flags[x]) == WALLMODEL) wm_cells.push_back(x);
    if (!wm_cells.empty()) {
      wm_slot.assign(N, -1);
      for (size_t k = 0; k < wm_cells.size(); ++k) wm_slot[wm_cells[k]] = static_cast<int32_t>(k);
    }
  }
  std::vector<double> uB(3 * wm_cells.size(), 0.0);
  double* cur = f;
  double* nxt = g.data();

  for (int step = 0; step < nsteps; ++step) {
    // ---- O1: wall-model pre-pass ----------------------------------------------------------
    const int64_t nwm = static_cast<int64_t>(wm_cells.size());
#pragma omp parallel for num_threads(nth) if (nth > 1)
    for (int64_t k = 0; k < nwm; ++k) {
      const int64_t x = wm_cells[k];
      const int xx = static_cast<int>(x % nx), yy = static_cast<int>((x / nx) % ny), zz = static_cast<int>(x / (static_cast<int64_t>(nx) * ny));
      int n[3];
      normal_of(flags[x], n);
      const int x2 = wrap(xx + n[0], nx), y2c = wrap(yy + n[1], ny), z2 = wrap(zz + n[2], nz);
      const int64_t s = (static_cast<int64_t>(z2) * ny + y2c) * nx + x2;
      double* ub = &uB[3 * k];
      ub[0] = ub[1] = ub[2] = 0.0;
      if (cell_type(flags[s]) == SOLID) continue;                          // step 1
      double fc[QMAX], rho2, u2[3];
      for (int i = 0; i < Q; ++i) fc[i] = cur[i * N + s];
      raw_moments(L, fc, rho2, u2);                                        // step 2
      const double un = u2[0] * n[0] + u2[1] * n[1] + u2[2] * n[2];
      const double ut[3] = {u2[0] - un * n[0], u2[1] - un * n[1], u2[2] - un * n[2]};   // step 3
      const double U2 = std::sqrt(ut[0] * ut[0] + ut[1] * ut[1] + ut[2] * ut[2]);
      if (U2 < 1e-14) continue;
      const double nu = (p.tau0 - 0.5) / 3.0;                              // step 4
      const double U1 = wallmodel_speed(U2, nu, p.wm_kappa, p.wm_E, 1.5, 0.5, nullptr, nullptr, nullptr);
      for (int a = 0; a < 3; ++a) ub[a] = (U1 / U2) * ut[a];               // step 7
    }

    // ---- O2: collide ------------------------------------------------------------------------
#pragma omp parallel for num_threads(nth) if (nth > 1)
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int xx = 0; xx < nx; ++xx) {
          const int64_t x = (static_cast<int64_t>(z) * ny + y) * nx + xx;
          const int type = flags ? cell_type(flags[x]) : FLUID;
          if (type == SOLID) {
            for (int i = 0; i < Q; ++i) fstar[i * N + x] = cur[i * N + x];
            continue;
          }
          double fc[QMAX], fs[QMAX];
          for (int i = 0; i < Q; ++i) fc[i] = cur[i * N + x];
          const double dd = (p.use_hlbm && d) ? d[x] : 0.0;
          double ub[3] = {0.0, 0.0, 0.0};
          if (type == WALLMODEL && p.wm_enable && !wm_slot.empty()) {
            const int32_t k = wm_slot[x];
            ub[0] = uB[3 * k];  ub[1] = uB[3 * k + 1];  ub[2] = uB[3 * k + 2];
          }
          collide_cell(L, fc, dd, ub, p.tau0, p.cs_smago, fs, nullptr);
          for (int i = 0; i < Q; ++i) fstar[i * N + x] = fs[i];
        }

    // ---- O3: stream (pull) with halfway bounce-back and outlet clamp -----------------------
#pragma omp parallel for num_threads(nth) if (nth > 1)
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int xx = 0; xx < nx; ++xx) {
          const int64_t x = (static_cast<int64_t>(z) * ny + y) * nx + xx;
          const int type = flags ? cell_type(flags[x]) : FLUID;
          if (type == SOLID) {
            for (int i = 0; i < Q; ++i) nxt[i * N + x] = cur[i * N + x];
            continue;
          }
          for (int i = 0; i < Q; ++i) {
            int sx = xx - L.c[i][0];
            if (type == OUTLET && sx > nx - 1) sx = nx - 1;      // ghost plane nx := plane nx-1
            sx = wrap(sx, nx);
            const int sy = wrap(y - L.c[i][1], ny);
            const int sz = wrap(z - L.c[i][2], nz);
            const int64_t s = (static_cast<int64_t>(sz) * ny + sy) * nx + sx;
            const bool solid = flags && cell_type(flags[s]) == SOLID;
            nxt[i * N + x] = solid ? fstar[L.opp[i] * N + x] : fstar[i * N + s];
          }
        }

    // ---- O4: inlet fix-up ----------------------------------------------------------------------
    if (flags) {
#pragma omp parallel for num_threads(nth) if (nth > 1)
      for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
          for (int xx = 0; xx < nx; ++xx) {
            const int64_t x = (static_cast<int64_t>(z) * ny + y) * nx + xx;
            if (cell_type(flags[x]) != INLET) continue;
            double gc[QMAX];
            for (int i = 0; i < Q; ++i) gc[i] = nxt[i * N + x];
            inlet_fixup_cell(L, gc, p.u_in);
            for (int i = 0; i < Q; ++i) nxt[i * N + x] = gc[i];
          }
    }

    // ---- O5: swap ------------------------------------------------------------------------------
    double* t = cur; cur = nxt; nxt = t;
  }
  if (cur != f) std::memcpy(f, cur, sizeof(double) * static_cast<size_t>(Q) * N);
  return 0;
}

// ---- O6: moments of the stored state, every cell (SOLID included) -----------------------------
int orc_moments(int Q, int64_t N, const double* f, double* rho, double* u /*[3][N]*/) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  for (int64_t x = 0; x < N; ++x) {
    double fc[QMAX], r, uc[3];
    for (int i = 0; i < Q; ++i) fc[i] = f[i * N + x];
    raw_moments(L, fc, r, uc);
    rho[x] = r;  u[x] = uc[0];  u[N + x] = uc[1];  u[2 * N + x] = uc[2];
  }
  return 0;
}

// ---- O7: totals over non-SOLID cells: mass, momentum xyz, kinetic energy ------------------
int orc_totals(int Q, int64_t N, const double* f, const uint8_t* flags, double* out /*[5]*/) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  for (int k = 0; k < 5; ++k) out[k] = 0.0;
  for (int64_t x = 0; x < N; ++x) {
    if (flags && cell_type(flags[x]) == SOLID) continue;
    double fc[QMAX], r, uc[3];
    for (int i = 0; i < Q; ++i) fc[i] = f[i * N + x];
    raw_moments(L, fc, r, uc);
    out[0] += r;
    out[1] += r * uc[0];  out[2] += r * uc[1];  out[3] += r * uc[2];
    out[4] += 0.5 * r * (uc[0] * uc[0] + uc[1] * uc[1] + uc[2] * uc[2]);
  }
  return 0;
}

int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
