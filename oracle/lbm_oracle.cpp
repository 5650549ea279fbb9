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
//   O4v Vortex Method inlet l.133-155, Eq. 18-21: per step the inflow velocity of every INLET cell from seeded
//                          vortices (readings G11, G34, G35); feeds O4.  Pinned by V1-V7 in tests/test_oracle_vm.py
//   O4p pressure outlet   l.255 "fixed local pressure condition" (reading G36): regularised local rule with rho
//                          imposed and the normal velocity taken from the known populations.  PARITY UNPINNED against the
//                          paper (not defined there); pinned as the mirror image of O4 + channel flow by B1-B4
//   O3s full-slip wall    l.255 "outer walls using full slip boundaries" (reading G37): specular reflection at halfway
//                          walls; wall-normal axes found from the single-axis neighbours.  Pinned by W1-W3 (a slip channel IS the mirror-extended
//                          periodic domain, bit for bit; tangential momentum conserved; uniform flow is a fixed point)
//   O2f fringe zone       l.255 "outlet using a fixed local pressure condition with fringe zone" (reading G38): a sponge,
//                          nu_mo(x) = nu_mo (1 + A xi^2) over the last L cells in x.  PARITY UNPINNED against the paper (neither
//                          the kind of fringe nor its profile is printed); pinned as stated by Z1-Z3
//   O3m moving wall       lid of the "established lid-driven cavity benchmark" (l.214): halfway bounce-back
//                          off a wall moving with u_w: + 2 w_i rho_w (c_i.u_w)/c_s^2 on the returned population, rho_w = 1
//                          (reading G33; the paper does not say how its lid is imposed -> PARITY UNPINNED against the
//                          paper, pinned as the textbook rule by M1-M4 in tests/test_oracle_cavity.py)
//   O2b solid velocity    Eq. 12 (l.99) with u^B(x,t) != 0 prescribed per cell (l.106 "non-zero solid velocities"; the moving
//                          bodies of Fig. 1) through orc_step_body; d(x,t) varies by stepping with a new d.  Pinned
//                          by U1-U4 in tests/test_oracle_body.py (closed-form relaxation towards u^B, Galilean image of P5,
//                          d = 1 drives u to u^B, u^B = 0 equals orc_step)
//   O6 moments             l.97 "fluid velocity moment u" (G19)
//   O2h collide, HRR form  (params.collision = 1; the paper's own collision)
//                          Eq. 6 (l.70) with f~(1) of Eq. 7 (l.74); Eq. 8-9 (l.81-86) regularised
//                          f(1), third-order coefficient by the recursion the method's name and
//                          refs [30,31] fix (G29); Eq. 10 (l.90) FD part with the sign and weight of
//                          reading G10; Eq. 11 (l.94) in full, third-order term = projection on the
//                          third-order Hermite polynomials the lattice supports (G9); sigma = 0 on
//                          wall-model cells (l.131); FD velocity = u^ of the same time level (G30-G32)
//   O2h', collision = 2    the same collision with the FD strain of Eq. 10 taken of u^(x, t - dt), the field of the previous
//                          level (reading G41: l.172 calls the collision a local cell model at 188 bytes); the first step
//                          of a call has no history and differences u^(x,t).  Pins L1-L5, tests/test_oracle_hrr_lag.py
//
// Pins (tests/test_oracle_*.py, all run with -m "not gpu"): P1 isotropy identities, P2
// equilibrium fixed point, P3 conservation, P4 Cs=0 == separately written BGK, P5 porous
// decay closed form, P6 tau_eff self-consistency, P7 Taylor-Green decay vs exp(-4 nu k^2 t),
// HRR pins (tests/test_oracle_hrr.py): H1 Hermite moments of the third-order equilibrium up to order
// 3, H2 fixed point, H3 conservation, H4 projection idempotence, H5 u = 0 reduction to the pinned
// BGK collide, H6 FD strain of a sine shear + closed-form post-collision stress at sigma = 0, H7
// Taylor-Green decay at sigma = 1, 0.5, 0 (fixes sign and factor of Eq. 10), H8 brute force via a
// numerically inverted Gram matrix, H9 lattice symmetry.
// P8 Poiseuille profile, P9 Spalding residual + viscous/log limits, P10 inlet moments /
// idempotence, P11a long-double brute force on 4^3, P12 bounce-back pulse + mass, P13 second
// order convergence, P14 lattice symmetry, P15 D3Q27.
// PARITY UNPINNED against the paper (no worked example printed): the wall-model coupling
// reading G17, the outlet rules G16 / G36, the inlet variant G15, the moving-wall rule G33 and the
// fringe zone G38.  They are pinned only as textbook definitions through P8, P9, P10, B1-B4,
// M1-M6, Z1-Z3.
//
// Layouts (all row-major, x fastest): f[Q][nz][ny][nx] double, d[nz][ny][nx] double,
// flag[nz][ny][nx] uint8.  Cell index = (z*ny + y)*nx + x.
// Flag byte: low nibble type {0 FLUID,1 SOLID,2 INLET,3 OUTLET,4 WALLMODEL,5 MOVINGWALL,6 POUTLET,7 SLIPWALL}; for WALLMODEL the
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
enum CellType : int { FLUID = 0, SOLID = 1, INLET = 2, OUTLET = 3, WALLMODEL = 4, MOVINGWALL = 5, POUTLET = 6, SLIPWALL = 7 };

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
  int collision;          // 0: BGK form of Eq. 6 (G1); 1: hybrid recursive-regularised (Eq. 6-11)
  double sigma;           // Eq. 7 hybridisation factor, in [0,1]
  double u_wall[3];       // velocity of the MOVINGWALL cells (lid of the lid-driven cavity, l.214; reading G33)
  double rho_out;         // density (pressure / c_s^2) imposed on POUTLET cells (l.255 "fixed local pressure"; reading G36)
  int fringe_len;         // fringe zone in front of the outlet plane (l.255; reading G38): the last fringe_len cells in x
  double fringe_factor;   // nu_mo(x) = nu_mo (1 + fringe_factor xi^2), xi = (x - (nx-1-fringe_len)) / fringe_len in [0,1]
};

inline int cell_type(uint8_t flag) { return flag & 0x0F; }
// a wall cell (resting SOLID or MOVINGWALL): inert, never collided, bounces populations back (R5, G33)
inline bool is_wall(int type) { return type == SOLID || type == MOVINGWALL || type == SLIPWALL; }

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

// ---- HRR form: Eq. 6-11 in full -----------------------------------------------------
// Third-order Hermite polynomial H(3)_abg of direction i:  c_a c_b c_g - c_s^2 (d_ab c_g + d_ag c_b + d_bg c_a).
inline double herm3(const Lattice& L, int i, int a, int b, int g) {
  const double ca = L.c[i][a], cb = L.c[i][b], cg = L.c[i][g];
  return ca * cb * cg - (1.0 / 3.0) * ((a == b ? cg : 0.0) + (a == g ? cb : 0.0) + (b == g ? ca : 0.0));
}

// Third-order coefficients carried by the lattices: index 0..6 = xxy, xxz, xyy, xzz, yyz, yzz, xyz.
constexpr int N3 = 7;
constexpr int IDX3[N3][3] = {{0, 0, 1}, {0, 0, 2}, {0, 1, 1}, {0, 2, 2}, {1, 1, 2}, {1, 2, 2}, {0, 1, 2}};

// The order-3 term of a Hermite series (Eq. 8 / Eq. 11) for direction i, WITHOUT the weight w_i: the
// orthogonal projection on the third-order polynomials the lattice supports (reading G9).
//  D3Q27: sum over the six aab-type components of H_aab a_aab / (2 c_s^6)  [1/3! times 3 index
//         permutations = the printed 1/(2 c_s^6)]  +  H_xyz a_xyz / c_s^6   [6 permutations].
//  D3Q19: H_xyz vanishes on the stencil and H_xxy, H_yzz (likewise H_xzz, H_xyy and H_yyz, H_xxz) are not
//         orthogonal; their sum and difference are (squared norms 2 c_s^6 and 6 c_s^6), which gives
//         [3 (H_xxy+H_yzz)(a_xxy+a_yzz) + (H_xxy-H_yzz)(a_xxy-a_yzz) + ...] / (6 c_s^6)   (refs [30,31]).
inline double order3_term(const Lattice& L, int i, const double a3[N3]) {
  double H[N3];
  for (int k = 0; k < N3; ++k) H[k] = herm3(L, i, IDX3[k][0], IDX3[k][1], IDX3[k][2]);
  const double cs6 = 1.0 / 27.0;
  if (L.Q == 27) {
    double s = 0.0;
    for (int k = 0; k < 6; ++k) s += H[k] * a3[k];
    return s / (2.0 * cs6) + H[6] * a3[6] / cs6;
  }
  // pairs (xxy, yzz) = (0,5), (xzz, xyy) = (3,2), (yyz, xxz) = (4,1)
  const int P[3][2] = {{0, 5}, {3, 2}, {4, 1}};
  double s = 0.0;
  for (int k = 0; k < 3; ++k) {
    const int p = P[k][0], q = P[k][1];
    s += 3.0 * (H[p] + H[q]) * (a3[p] + a3[q]) + (H[p] - H[q]) * (a3[p] - a3[q]);
  }
  return s / (6.0 * cs6);
}

// Eq. 11 (l.94) in full: a^_0^(0) = rho, a^_0^(n) = a^_0^(n-1) u^.
inline double feq3_i(const Lattice& L, int i, double rho, const double u[3]) {
  double a3[N3];
  for (int k = 0; k < N3; ++k) a3[k] = rho * u[IDX3[k][0]] * u[IDX3[k][1]] * u[IDX3[k][2]];
  return feq_i(L, i, rho, u) + L.w[i] * order3_term(L, i, a3);
}

// O2h for one cell.  S = S^FD(x,t) (symmetric 3x3), sigma = the cell's hybridisation factor.
void collide_cell_hrr(const Lattice& L, const double* fc, double d, const double ub[3], double tau0,
                      double cs_smago, double sigma, const double S[3][3], double* fs, double* tau_out) {
  double rho, u[3];
  raw_moments(L, fc, rho, u);                                            // A2
  double uh[3];
  for (int a = 0; a < 3; ++a) uh[a] = (1.0 - d) * u[a] + d * ub[a];      // A3, Eq. 12
  double feq[QMAX], f1[QMAX];
  for (int i = 0; i < L.Q; ++i) feq[i] = feq3_i(L, i, rho, uh);          // Eq. 11
  for (int i = 0; i < L.Q; ++i) f1[i] = fc[i] - feq[i];                  // raw non-equilibrium
  // Eq. 9: a_1^(n) = sum_i H_i^(n) f_i^(1), n = 0, 1, 2
  double a0 = 0.0, a1[3] = {0, 0, 0}, a2[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, Pi[3][3];
  for (int i = 0; i < L.Q; ++i) {
    a0 += f1[i];
    for (int a = 0; a < 3; ++a) {
      a1[a] += L.c[i][a] * f1[i];
      for (int b = 0; b < 3; ++b) a2[a][b] += (L.c[i][a] * L.c[i][b] - ((a == b) ? 1.0 / 3.0 : 0.0)) * f1[i];
    }
  }
  double tau = tau0;
  if (cs_smago > 0.0) {                                                  // A5 as in the BGK form: Pi = sum c c f1
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        Pi[a][b] = 0.0;
        for (int i = 0; i < L.Q; ++i) Pi[a][b] += L.c[i][a] * L.c[i][b] * f1[i];
      }
    const double nPi = std::sqrt(Pi[0][0] * Pi[0][0] + Pi[1][1] * Pi[1][1] + Pi[2][2] * Pi[2][2] +
                                 2.0 * (Pi[0][1] * Pi[0][1] + Pi[0][2] * Pi[0][2] + Pi[1][2] * Pi[1][2]));
    tau = 0.5 * (tau0 + std::sqrt(tau0 * tau0 + 18.0 * std::sqrt(2.0) * cs_smago * cs_smago * nPi / rho));
  }
  // recursion for the third-order coefficient (G29): a_1,abg = u^_a a_1,bg + u^_b a_1,ag + u^_g a_1,ab
  double a3[N3];
  for (int k = 0; k < N3; ++k) {
    const int a = IDX3[k][0], b = IDX3[k][1], g = IDX3[k][2];
    a3[k] = uh[a] * a2[b][g] + uh[b] * a2[a][g] + uh[g] * a2[a][b];
  }
  for (int i = 0; i < L.Q; ++i) {
    // Eq. 8: f(1)_i = w_i sum_n H^(n) : a_1^(n) / (c_s^2n n!)
    double h1 = 0.0, h2 = 0.0, hS = 0.0;
    for (int a = 0; a < 3; ++a) {
      h1 += L.c[i][a] * a1[a];
      for (int b = 0; b < 3; ++b) {
        const double H2 = L.c[i][a] * L.c[i][b] - ((a == b) ? 1.0 / 3.0 : 0.0);
        h2 += H2 * a2[a][b];
        hS += H2 * S[a][b];
      }
    }
    const double freg = L.w[i] * (a0 + 3.0 * h1 + 4.5 * h2 + order3_term(L, i, a3));
    // Eq. 10 with the sign and the weight of reading G10: -w_i rho tau / c_s^2  H(2) : S^FD  (tau = tau_eff, G31)
    const double ffd = -L.w[i] * rho * tau * 3.0 * hS;
    const double ft = sigma * freg + (1.0 - sigma) * ffd;                // Eq. 7 (G10)
    fs[i] = feq[i] + (1.0 - 1.0 / tau) * ft;                             // Eq. 6
  }
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

// O4p for one pressure-outlet cell on the plane x = nx-1 (outward normal +x, "fixed local
// pressure condition"; reading G36: the regularised local boundary rule of O4 with the roles of density and normal velocity
// exchanged).  Known after streaming: c_x >= 0; unknown: c_x < 0.  rho = rho_out is imposed, the normal velocity follows from
// the known populations, u_x = (sum_{c_x=0} g + 2 sum_{c_x>0} g)/rho_out - 1, the tangential velocity is 0; then all
// populations are replaced by f^eq + the second-order Hermite projection of the non-equilibrium stress, as in O4.
void pressure_fixup_cell(const Lattice& L, double* g, double rho_out) {
  double s0 = 0.0, sp = 0.0;
  for (int i = 0; i < L.Q; ++i) {
    if (L.c[i][0] == 0) s0 += g[i];
    else if (L.c[i][0] > 0) sp += g[i];
  }
  const double uw[3] = {(s0 + 2.0 * sp) / rho_out - 1.0, 0.0, 0.0};
  double feq[QMAX], n[QMAX];
  for (int i = 0; i < L.Q; ++i) feq[i] = feq_i(L, i, rho_out, uw);
  for (int i = 0; i < L.Q; ++i)
    if (L.c[i][0] >= 0) n[i] = g[i] - feq[i];
  for (int i = 0; i < L.Q; ++i)
    if (L.c[i][0] < 0) n[i] = n[L.opp[i]];                 // bounce-back of the non-equilibrium part
  double Pi[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
  for (int i = 0; i < L.Q; ++i)
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) Pi[a][b] += L.c[i][a] * L.c[i][b] * n[i];
  for (int i = 0; i < L.Q; ++i) {
    double s = 0.0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        s += (L.c[i][a] * L.c[i][b] - ((a == b) ? 1.0 / 3.0 : 0.0)) * Pi[a][b];
    g[i] = feq[i] + 4.5 * L.w[i] * s;
  }
}

// ---- Vortex Method inflow: Eq. 18-21 ------------------------------------------
// The inflow plane is x = 0 with d_inlet = (1,0,0); fields are [3][nz][ny] (component, z, y); mask[z][y] = 1 on INLET cells.
// Seeds p_i = (y_i, z_i) in cell coordinates and signs s_i are INPUTS (the random numbers the method draws).
//   k_i     = 3/2 (|u_mean(p_i)| I)^2                                                  (Eq. 18; u_mean at the nearest cell,
//                                                                                        0 if that cell is not an INLET cell)
//   Gamma_i = 4 s_i sqrt( pi A k_i / (3 N (2 ln 3 - 3 ln 2)) )                         (Eq. 19, reading G34: the printed
//             "sqrt(pi/(6 ln3 - 9 ln2)) k_i A/n" with the root over the whole quotient, as in ref. [12]; A = number of
//             INLET cells)
//   u_v(x)  = 1/(2 pi) sum_i Gamma_i ((p_i - x) x d) (1 - exp(-|x-p_i|^2 / (2 sigma^2))) / |x-p_i|^2   (Eq. 20, G11: exp(-..))
//   u(x)    = u_mean + u_v - (u_v . g^) d,  g^ = grad(u_prev . d)/|grad(u_prev . d)|   (Eq. 21, reading G35: in-plane
//             central differences, a neighbour that is not an INLET cell is replaced by the cell itself, y wraps; the
//             term is dropped where the gradient vanishes)
struct VortexInlet {
  const double* u_mean;   // [3][nz][ny]
  double* u_inflow;       // [3][nz][ny]: in = inflow of the previous step, out = inflow of the last step
  int nv;
  const double* pos;      // [nv][2] (y, z)
  const double* sign;     // [nv]
  double sigma_v, intensity;
};

void vm_inflow(int ny, int nz, const uint8_t* mask, const double* u_mean, const double* u_prev, int nv, const double* pos,
               const double* sign, double sigma_v, double intensity, double* out) {
  const int64_t P = static_cast<int64_t>(ny) * nz;
  const double PI = 3.14159265358979323846;
  int64_t A = 0;
  for (int64_t c = 0; c < P; ++c) A += mask[c] ? 1 : 0;
  std::vector<double> gamma(nv > 0 ? nv : 0);
  for (int i = 0; i < nv; ++i) {
    int yi = static_cast<int>(std::floor(pos[2 * i] + 0.5)), zi = static_cast<int>(std::floor(pos[2 * i + 1] + 0.5));
    yi = ((yi % ny) + ny) % ny;
    zi = (zi < 0) ? 0 : ((zi >= nz) ? nz - 1 : zi);
    const int64_t c = static_cast<int64_t>(zi) * ny + yi;
    double k = 0.0;
    if (mask[c]) {
      const double um = std::sqrt(u_mean[c] * u_mean[c] + u_mean[P + c] * u_mean[P + c] + u_mean[2 * P + c] * u_mean[2 * P + c]);
      k = 1.5 * (um * intensity) * (um * intensity);                                        // Eq. 18
    }
    gamma[i] = 4.0 * sign[i] * std::sqrt(PI * static_cast<double>(A) * k /
                                         (3.0 * nv * (2.0 * std::log(3.0) - 3.0 * std::log(2.0))));   // Eq. 19 (G34)
  }
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y) {
      const int64_t c = static_cast<int64_t>(z) * ny + y;
      if (!mask[c]) {
        for (int a = 0; a < 3; ++a) out[a * P + c] = u_mean[a * P + c];
        continue;
      }
      double uv[3] = {0.0, 0.0, 0.0};
      for (int i = 0; i < nv; ++i) {                                                         // Eq. 20
        const double ry = pos[2 * i] - y, rz = pos[2 * i + 1] - z;                           // p_i - x (in-plane)
        const double r2 = ry * ry + rz * rz;
        if (r2 == 0.0) continue;                                                             // limit of the summand is 0
        // (0, ry, rz) x (1, 0, 0) = (0, rz, -ry)
        const double fac = gamma[i] * (1.0 - std::exp(-r2 / (2.0 * sigma_v * sigma_v))) / r2 / (2.0 * PI);
        uv[1] += fac * rz;
        uv[2] += -fac * ry;
      }
      // Eq. 21 (G35): streamwise fluctuation along the gradient of the previous inflow's streamwise component
      const double* sp = u_prev;                                                             // component 0 = u_prev . d
      const int yp = (y + 1) % ny, ym = (y + ny - 1) % ny;
      const int64_t cyp = mask[static_cast<int64_t>(z) * ny + yp] ? static_cast<int64_t>(z) * ny + yp : c;
      const int64_t cym = mask[static_cast<int64_t>(z) * ny + ym] ? static_cast<int64_t>(z) * ny + ym : c;
      const int64_t czp = (z + 1 < nz && mask[c + ny]) ? c + ny : c;
      const int64_t czm = (z - 1 >= 0 && mask[c - ny]) ? c - ny : c;
      const double gy = 0.5 * (sp[cyp] - sp[cym]), gz = 0.5 * (sp[czp] - sp[czm]);
      const double gn = std::sqrt(gy * gy + gz * gz);
      double us = 0.0;
      if (gn > 0.0) us = -(uv[1] * gy + uv[2] * gz) / gn;
      out[c] = u_mean[c] + uv[0] + us;
      out[P + c] = u_mean[P + c] + uv[1];
      out[2 * P + c] = u_mean[2 * P + c] + uv[2];
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

// Eq. 11 in full (third-order equilibrium)
int orc_feq3(int Q, double rho, const double* u, double* out) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  for (int i = 0; i < Q; ++i) out[i] = feq3_i(L, i, rho, u);
  return 0;
}

// O2h on one cell; S = S^FD row-major [9]
int orc_collide_cell_hrr(int Q, const double* fc, double d, const double* ub, double tau0, double cs_smago,
                         double sigma, const double* S, double* fs, double* tau_out) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  double S33[3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) S33[a][b] = S[3 * a + b];
  collide_cell_hrr(L, fc, d, ub, tau0, cs_smago, sigma, S33, fs, tau_out);
  return 0;
}

int orc_pressure_fixup_cell(int Q, double* g, double rho_out) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  pressure_fixup_cell(L, g, rho_out);
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
}  // extern "C"
namespace {
int step_impl(int Q, int nx, int ny, int nz, double* f, const double* d, const uint8_t* flags,
             const double* par /* tau0, cs, use_hlbm, uin0, uin1, uin2, wm_enable, kappa, E, collision, sigma, uwall0, uwall1, uwall2, rho_out, fringe_len, fringe_factor */,
             int nsteps, int nthreads, VortexInlet* vm, const double* u_body = nullptr) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  if (nx < 1 || ny < 1 || nz < 1 || nsteps < 0) return -1;
  Params p;
  p.tau0 = par[0];  p.cs_smago = par[1];  p.use_hlbm = (par[2] != 0.0);
  p.u_in[0] = par[3];  p.u_in[1] = par[4];  p.u_in[2] = par[5];
  p.wm_enable = (par[6] != 0.0);  p.wm_kappa = par[7];  p.wm_E = par[8];
  p.collision = static_cast<int>(par[9]);  p.sigma = par[10];
  p.u_wall[0] = par[11];  p.u_wall[1] = par[12];  p.u_wall[2] = par[13];
  p.rho_out = par[14];
  p.fringe_len = static_cast<int>(par[15]);  p.fringe_factor = par[16];
  if (p.fringe_len < 0 || p.fringe_factor < 0.0) return -1;
  if (!(p.tau0 > 0.5) || p.cs_smago < 0.0) return -1;
  if (p.collision != 0 && p.collision != 1 && p.collision != 2) return -1;
  if (p.collision >= 1 && !(p.sigma >= 0.0 && p.sigma <= 1.0)) return -1;
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
  std::vector<double> uhat;                                // u^(x,t), [3][N], HRR form only
  if (p.collision >= 1) uhat.assign(3 * static_cast<size_t>(N), 0.0);
  // collision = 2 (reading G41): the HRR form with the FD strain of Eq. 10 taken of u^(x, t - dt), the field of the PREVIOUS
  // level (a collision that is local but for a stored field: l.172 quotes 188 bytes per collision for a "local cell model").
  // The state of this form is (S_t, u^_{t-1}); a call starts without history: its first step differences u^(x, t) like
  // collision = 1, every later step the field of the step before.
  std::vector<double> uhat_prev;
  if (p.collision == 2) uhat_prev.assign(3 * static_cast<size_t>(N), 0.0);
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
      if (is_wall(cell_type(flags[s]))) continue;                          // step 1
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

    // ---- O1b (HRR form): u^(x,t) of every cell, the field the FD strain is taken of (G30) ------
    // Wall cells at rest (SOLID, SLIPWALL): u^ = 0 whatever populations they hold (G30; G37: "the FD stencil sees u^ = 0 on
    // slip wall cells like on any resting wall").
    if (p.collision >= 1) {
#pragma omp parallel for num_threads(nth) if (nth > 1)
      for (int64_t x = 0; x < N; ++x) {
        const int type = flags ? cell_type(flags[x]) : FLUID;
        double uh[3] = {0.0, 0.0, 0.0};
        if (type == MOVINGWALL) {
          for (int a = 0; a < 3; ++a) uh[a] = p.u_wall[a];                 // the wall's own velocity (G33)
        } else if (!is_wall(type)) {
          double fc[QMAX], rho, u[3];
          for (int i = 0; i < Q; ++i) fc[i] = cur[i * N + x];
          raw_moments(L, fc, rho, u);
          const double dd = (p.use_hlbm && d) ? d[x] : 0.0;
          double ub[3] = {0.0, 0.0, 0.0};
          if (u_body)                                                      // O2b: prescribed solid velocity u^B(x,t), Eq. 12
            for (int a = 0; a < 3; ++a) ub[a] = u_body[a * N + x];
          if (type == WALLMODEL && p.wm_enable && !wm_slot.empty()) {
            const int32_t k = wm_slot[x];
            ub[0] = uB[3 * k];  ub[1] = uB[3 * k + 1];  ub[2] = uB[3 * k + 2];
          }
          for (int a = 0; a < 3; ++a) uh[a] = (1.0 - dd) * u[a] + dd * ub[a];
        }
        for (int a = 0; a < 3; ++a) uhat[a * N + x] = uh[a];
      }
    }

    // the field Eq. 10 differences: u^ of this level, or (collision = 2, from the second step of the call on) of the previous one
    const double* ufd = (p.collision == 2 && step > 0) ? uhat_prev.data() : uhat.data();
    // ---- O2: collide ------------------------------------------------------------------------
#pragma omp parallel for num_threads(nth) if (nth > 1)
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int xx = 0; xx < nx; ++xx) {
          const int64_t x = (static_cast<int64_t>(z) * ny + y) * nx + xx;
          const int type = flags ? cell_type(flags[x]) : FLUID;
          if (is_wall(type)) {
            for (int i = 0; i < Q; ++i) fstar[i * N + x] = cur[i * N + x];
            continue;
          }
          double fc[QMAX], fs[QMAX];
          for (int i = 0; i < Q; ++i) fc[i] = cur[i * N + x];
          const double dd = (p.use_hlbm && d) ? d[x] : 0.0;
          double ub[3] = {0.0, 0.0, 0.0};
          if (u_body)                                                      // O2b: prescribed solid velocity u^B(x,t), Eq. 12
            for (int a = 0; a < 3; ++a) ub[a] = u_body[a * N + x];
          if (type == WALLMODEL && p.wm_enable && !wm_slot.empty()) {      // the wall model prescribes u^B there (l.106)
            const int32_t k = wm_slot[x];
            ub[0] = uB[3 * k];  ub[1] = uB[3 * k + 1];  ub[2] = uB[3 * k + 2];
          }
          // fringe zone (G38): the molecular viscosity rises quadratically over the last fringe_len cells before the outlet
          double tau0x = p.tau0;
          if (p.fringe_len > 0 && xx > nx - 1 - p.fringe_len) {
            const double xi = static_cast<double>(xx - (nx - 1 - p.fringe_len)) / p.fringe_len;
            tau0x = 0.5 + (p.tau0 - 0.5) * (1.0 + p.fringe_factor * xi * xi);
          }
          if (p.collision >= 1) {
            // S^FD_ab = (D_a u^_b + D_b u^_a) / 2, D_a g = (g(x+e_a) - g(x-e_a)) / 2; periodic wrap, except
            // that the ghost planes beyond the INLET / OUTLET planes copy those planes (G32)
            const int pos[3] = {xx, y, z}, dim[3] = {nx, ny, nz};
            double D[3][3];   // D[a][b] = D_a u^_b
            for (int a = 0; a < 3; ++a) {
              int qp[3] = {xx, y, z}, qm[3] = {xx, y, z};
              qp[a] = wrap(pos[a] + 1, dim[a]);
              qm[a] = wrap(pos[a] - 1, dim[a]);
              if (a == 0 && (type == OUTLET || type == POUTLET)) qp[0] = xx;
              if (a == 0 && type == INLET) qm[0] = xx;
              const int64_t sp = (static_cast<int64_t>(qp[2]) * ny + qp[1]) * nx + qp[0];
              const int64_t sm = (static_cast<int64_t>(qm[2]) * ny + qm[1]) * nx + qm[0];
              for (int b = 0; b < 3; ++b) D[a][b] = 0.5 * (ufd[b * N + sp] - ufd[b * N + sm]);
            }
            double S[3][3];
            for (int a = 0; a < 3; ++a)
              for (int b = 0; b < 3; ++b) S[a][b] = 0.5 * (D[a][b] + D[b][a]);
            const double sig = (type == WALLMODEL && p.wm_enable) ? 0.0 : p.sigma;   // l.131
            collide_cell_hrr(L, fc, dd, ub, tau0x, p.cs_smago, sig, S, fs, nullptr);
          } else {
            collide_cell(L, fc, dd, ub, tau0x, p.cs_smago, fs, nullptr);
          }
          for (int i = 0; i < Q; ++i) fstar[i * N + x] = fs[i];
        }

    if (p.collision == 2) uhat_prev = uhat;                  // u^ of this level is the next step's history
    // ---- O3: stream (pull) with halfway bounce-back and outlet clamp -----------------------
#pragma omp parallel for num_threads(nth) if (nth > 1)
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int xx = 0; xx < nx; ++xx) {
          const int64_t x = (static_cast<int64_t>(z) * ny + y) * nx + xx;
          const int type = flags ? cell_type(flags[x]) : FLUID;
          if (is_wall(type)) {
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
            const int stype = flags ? cell_type(flags[s]) : FLUID;
            double v = is_wall(stype) ? fstar[L.opp[i] * N + x] : fstar[i * N + s];
            if (stype == SLIPWALL) {
              // full-slip wall (l.255 "outer walls using full slip boundaries", reading G37): specular reflection at
              // the halfway wall.  The wall-normal axes are those along which the cell's own single-axis neighbour
              // x - c_ia e_a is a slip wall cell: the population left the fluid cell x' = x - c_i + sum_a c_ia e_a with the
              // velocity c_i' = c_i with those components reversed.  No such axis (a convex edge met diagonally), or a wall
              // at x': plain bounce-back.
              int cr[3] = {L.c[i][0], L.c[i][1], L.c[i][2]};
              int pr[3] = {sx, sy, sz};
              const int pos[3] = {xx, y, z}, dim[3] = {nx, ny, nz};
              bool any = false;
              for (int a = 0; a < 3; ++a) {
                if (L.c[i][a] == 0) continue;
                int q[3] = {xx, y, z};
                q[a] = wrap(pos[a] - L.c[i][a], dim[a]);
                if (cell_type(flags[(static_cast<int64_t>(q[2]) * ny + q[1]) * nx + q[0]]) == SLIPWALL) {
                  cr[a] = -cr[a];
                  pr[a] = pos[a];
                  any = true;
                }
              }
              if (any) {
                const int64_t xr = (static_cast<int64_t>(pr[2]) * ny + pr[1]) * nx + pr[0];
                if (!is_wall(cell_type(flags[xr]))) {
                  int ir = -1;
                  for (int k = 0; k < Q; ++k)
                    if (L.c[k][0] == cr[0] && L.c[k][1] == cr[1] && L.c[k][2] == cr[2]) ir = k;
                  v = fstar[ir * N + xr];
                }
              }
            }
            if (stype == MOVINGWALL)   // moving-wall bounce-back (G33): + 2 w_i rho_w (c_i . u_w) / c_s^2, rho_w = 1, c_i = wall -> fluid
              v += 6.0 * L.w[i] * (L.c[i][0] * p.u_wall[0] + L.c[i][1] * p.u_wall[1] + L.c[i][2] * p.u_wall[2]);
            nxt[i * N + x] = v;
          }
        }

    // ---- O4v (Vortex Method inlet, Eq. 18-21): this step's inflow velocity field from the previous one ----------
    if (vm && flags) {
      const int64_t P = static_cast<int64_t>(ny) * nz;
      std::vector<uint8_t> mask(P);
      for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
          mask[static_cast<int64_t>(z) * ny + y] = cell_type(flags[(static_cast<int64_t>(z) * ny + y) * nx]) == INLET;
      std::vector<double> unew(3 * P);
      vm_inflow(ny, nz, mask.data(), vm->u_mean, vm->u_inflow, vm->nv, vm->pos, vm->sign, vm->sigma_v, vm->intensity, unew.data());
      std::memcpy(vm->u_inflow, unew.data(), sizeof(double) * 3 * P);
    }

    // ---- O4: inlet fix-up ----------------------------------------------------------------------
    if (flags) {
#pragma omp parallel for num_threads(nth) if (nth > 1)
      for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
          for (int xx = 0; xx < nx; ++xx) {
            const int64_t x = (static_cast<int64_t>(z) * ny + y) * nx + xx;
            if (cell_type(flags[x]) == POUTLET) {                        // O4p
              double gp[QMAX];
              for (int i = 0; i < Q; ++i) gp[i] = nxt[i * N + x];
              pressure_fixup_cell(L, gp, p.rho_out);
              for (int i = 0; i < Q; ++i) nxt[i * N + x] = gp[i];
              continue;
            }
            if (cell_type(flags[x]) != INLET) continue;
            double gc[QMAX];
            for (int i = 0; i < Q; ++i) gc[i] = nxt[i * N + x];
            double uw[3] = {p.u_in[0], p.u_in[1], p.u_in[2]};
            if (vm) {
              const int64_t P = static_cast<int64_t>(ny) * nz, c = static_cast<int64_t>(z) * ny + y;
              for (int a = 0; a < 3; ++a) uw[a] = vm->u_inflow[a * P + c];
            }
            inlet_fixup_cell(L, gc, uw);
            for (int i = 0; i < Q; ++i) nxt[i * N + x] = gc[i];
          }
    }

    // ---- O5: swap ------------------------------------------------------------------------------
    double* t = cur; cur = nxt; nxt = t;
  }
  if (cur != f) std::memcpy(f, cur, sizeof(double) * static_cast<size_t>(Q) * N);
  return 0;
}
}  // namespace

extern "C" {

int orc_step(int Q, int nx, int ny, int nz, double* f, const double* d, const uint8_t* flags, const double* par, int nsteps,
             int nthreads) {
  return step_impl(Q, nx, ny, nz, f, d, flags, par, nsteps, nthreads, nullptr);
}

// the step with a prescribed solid velocity field u^B(x,t) of Eq. 12 (l.99-106: "non-zero solid velocities"; the moving porous
// bodies of the FSI cases of Fig. 1): u_body [3][nz][ny][nx], constant over the nsteps steps (a body that moves
// is stepped one step at a time with new d and u_body).  WALLMODEL cells keep the wall model's u^B when wm_enable.
int orc_step_body(int Q, int nx, int ny, int nz, double* f, const double* d, const uint8_t* flags, const double* par, int nsteps,
                  int nthreads, const double* u_body) {
  return step_impl(Q, nx, ny, nz, f, d, flags, par, nsteps, nthreads, nullptr, u_body);
}

// the step with the Vortex Method inlet: u_inflow [3][nz][ny] holds the inflow of the previous step on entry (u_mean
// before the first step) and the inflow of the last step on return; seeds and signs stay fixed for the nsteps steps
int orc_step_vm(int Q, int nx, int ny, int nz, double* f, const double* d, const uint8_t* flags, const double* par, int nsteps,
                int nthreads, const double* u_mean, double* u_inflow, int nv, const double* pos, const double* sign,
                double sigma_v, double intensity) {
  if (!u_mean || !u_inflow || nv < 0 || (nv > 0 && (!pos || !sign)) || !(sigma_v > 0.0) || intensity < 0.0) return -1;
  VortexInlet vm{u_mean, u_inflow, nv, pos, sign, sigma_v, intensity};
  return step_impl(Q, nx, ny, nz, f, d, flags, par, nsteps, nthreads, &vm);
}

int orc_vm_inflow(int ny, int nz, const uint8_t* mask, const double* u_mean, const double* u_prev, int nv, const double* pos,
                  const double* sign, double sigma_v, double intensity, double* out) {
  if (ny < 1 || nz < 1 || !mask || !u_mean || !u_prev || !out || nv < 0 || !(sigma_v > 0.0)) return -1;
  vm_inflow(ny, nz, mask, u_mean, u_prev, nv, pos, sign, sigma_v, intensity, out);
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
    if (flags && is_wall(cell_type(flags[x]))) continue;
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
