// =====================================================================================
// lbm_kernels.cuh -- device code of the LBM hot path for sm_100a (B200).
//
// One fused kernel per time step: pull-propagation (A1) + moments (A2) + HLBM velocity (A3) +
// equilibrium (A4) + Smagorinsky tau_eff (A5) + relaxation (A6), with the masked boundary rules
// (A7: halfway bounce-back, velocity inlet, zero-gradient outlet) and the Spalding wall model (A8)
// on a warp-uniform slow path.  A9 (moments / totals) are separate kernels.
// Row and equation references are to SURVEY.md section 8(a) and /root/reference/PAPER.md.
//
// Storage: SoA f[i][z][y][x], x fastest, two lattices (ping-pong).  The stored array holds the
// POST-collision populations F_{t-1}; the state S_t of the ABI is stream(F_{t-1}) and is formed in
// registers by the pull.  This file shares nothing with oracle/.
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

namespace lbm {

enum : int { T_FLUID = 0, T_SOLID = 1, T_INLET = 2, T_OUTLET = 3, T_WM = 4, T_MOVING = 5, T_POUTLET = 6, T_SLIP = 7 };
// wall cells: resting SOLID (1), MOVINGWALL (5) and SLIPWALL (7): bits 1, 5, 7 of 0xA2
__host__ __device__ constexpr bool is_wall(int cls_or_type) { return ((0xA2 >> (cls_or_type & 7)) & 1) != 0; }
// internal class byte: bits 0-2 type, bits 3-5 wall-normal code,
//   bit 6 = ADJ:     the (non-SOLID) cell has at least one SOLID lattice neighbour (nbmask[] says which);
//   bit 7 = SPECIAL: the cell needs the per-cell path (list blocks): WALLMODEL cells (A8), OUTLET cells with a wall neighbour
//                    (their clamped pull needs a class lookup) and cells next to a SLIPWALL (specular pull, G37).
// Halfway bounce-back (A7, reading R5) on the READ side: the pull of direction i at a cell x whose source x - c_i is
// SOLID takes the cell's own F_opp(i)(x) instead.  Nobody ever consumes the lattice slots of a SOLID cell, so the
// step kernels write every 128-byte line they touch IN FULL (zeros on SOLID cells): a store stream with holes at
// the walls leaves partial sectors that the L2 has to fill from DRAM, which cost config 4 a third of its
// bandwidth (profiles/r1_k_step_vec_ncu.md).  SOLID cells' own values (inert, R5) are kept in a side buffer by
// the host side and patched back whenever the state is materialised.
constexpr uint8_t CLS_TYPE = 0x07;
constexpr uint8_t CLS_ADJ = 0x40;
constexpr uint8_t CLS_SPECIAL = 0x80;
constexpr int CLS_NORMAL_SHIFT = 3;

// kernel modes
enum : int { MODE_COLLIDE = 0,        // input holds S_t (fresh state): collide only           -> F_t
             MODE_STREAM_COLLIDE = 1, // input holds F_{t-1}: pull to S_t, collide             -> F_t
             MODE_STREAM = 2,         // input holds F_{t-1}: pull to S_t, store S_t (materialise)
             MODE_UHAT_PULL = 3,      // input holds F_{t-1}: pull to S_t, store u^(x,t) (HRR form, first pass)
             MODE_UHAT_PRE = 4,       // input holds S_t: store u^(x,t)
             MODE_MOMENTS_PULL = 5,   // A9: input holds F_{t-1}: pull to S_t, store rho, u of S_t into the caller's arrays
             MODE_MOMENTS_PRE = 6,    // A9: input holds S_t
             MODE_TOTALS_PULL = 7,    // A9: pull to S_t, reduce mass / momentum / kinetic energy over the non-wall cells
             MODE_TOTALS_PRE = 8 };
// collision forms (lbm_params.collision)
enum : int { COLL_BGK = 0, COLL_HRR = 1 };
__host__ __device__ constexpr bool mode_pulls(int mode) {
  return mode == MODE_STREAM_COLLIDE || mode == MODE_STREAM || mode == MODE_UHAT_PULL || mode == MODE_MOMENTS_PULL || mode == MODE_TOTALS_PULL;
}
__host__ __device__ constexpr bool mode_collides(int mode) { return mode == MODE_COLLIDE || mode == MODE_STREAM_COLLIDE; }
__host__ __device__ constexpr bool mode_uhat(int mode) { return mode == MODE_UHAT_PULL || mode == MODE_UHAT_PRE; }
__host__ __device__ constexpr bool mode_moments(int mode) { return mode == MODE_MOMENTS_PULL || mode == MODE_MOMENTS_PRE; }
__host__ __device__ constexpr bool mode_totals(int mode) { return mode == MODE_TOTALS_PULL || mode == MODE_TOTALS_PRE; }
__host__ __device__ constexpr bool mode_diag(int mode) { return mode_moments(mode) || mode_totals(mode); }
// modes that read the porosity / solid velocity (Eq. 12)
__host__ __device__ constexpr bool mode_hlbm(int mode) { return mode_collides(mode) || mode_uhat(mode); }

// Programmatic dependent launch (sm_90+): a kernel launched with the programmatic-serialization attribute may become resident
// while its predecessor in the stream drains; griddep_wait() returns once the predecessor has completed and its writes are
// visible.  Both are no-ops in a kernel launched the ordinary way.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- velocity set by rule R1 (G13), generated at compile time -------------------------
template <int Q>
struct Stencil {
  int c[Q][3];
  int opp[Q];
  int c2[Q];
  constexpr Stencil() : c{}, opp{}, c2{} {
    const int maxc2 = (Q == 19) ? 2 : 3;
    const int h = (Q - 1) / 2;
    int n = 1;
    // ascending (|c|^2, -cx, -cy, -cz): loop |c|^2 outermost, then cx, cy, cz descending
    for (int want = 1; want <= maxc2; ++want)
      for (int x = 1; x >= -1; --x)
        for (int y = 1; y >= -1; --y)
          for (int z = 1; z >= -1; --z) {
            const int s = x * x + y * y + z * z;
            if (s != want) continue;
            const int first = (x != 0) ? x : ((y != 0) ? y : z);
            if (first != 1) continue;
            c[n][0] = x;      c[n][1] = y;      c[n][2] = z;      c2[n] = s;      opp[n] = n + h;
            c[n + h][0] = -x; c[n + h][1] = -y; c[n + h][2] = -z; c2[n + h] = s;  opp[n + h] = n;
            ++n;
          }
  }
};

template <int Q, typename T>
__host__ __device__ constexpr T weight(int c2) {
  return (Q == 19) ? (c2 == 0 ? T(1.0 / 3.0) : (c2 == 1 ? T(1.0 / 18.0) : T(1.0 / 36.0)))
                   : (c2 == 0 ? T(8.0 / 27.0) : (c2 == 1 ? T(2.0 / 27.0) : (c2 == 2 ? T(1.0 / 54.0) : T(1.0 / 216.0))));
}

// Slip plane code of a cell (bits 3-5 of the class byte of a cell that is not a WALLMODEL cell; 0 = none): the cell lies next to ONE
// plane slip wall normal to y or z and nothing else complicates its specular pull (reading G37): 2 = wall at y-1 (normal +y),
// 3 = wall at y+1, 4 = wall at z-1, 5 = wall at z+1 -- the numbering of the wall-normal codes.  For such a cell the population i
// with c_i . n = +1 is pulled as the population with the n-component of c_i reversed from the cell x - c_i + n of its OWN plane:
// a different source row and slot, but the same aligned access pattern, so these cells run in the vector path (kernel variant
// WV bit 1) instead of the per-cell list path.  Everything less regular (edges, corners, wall-model cells at a slip wall, slip walls
// normal to x, a sector whose cells disagree) keeps the SPECIAL bit and the general rule slip_pull.
__host__ __device__ constexpr int slip_axis(int code) { return code >> 1; }                  // 1 = y, 2 = z
__host__ __device__ constexpr int slip_sign(int code) { return (code & 1) ? -1 : 1; }        // of the normal (wall -> fluid)
// population index of c_i with its y (my) or z (mz) component reversed
template <int Q>
struct Mirror {
  int my[Q], mz[Q];      // ... reversed
  int zy[Q], zz[Q];      // ... set to zero (0 = the rest population: the cell itself)
  constexpr Mirror() : my{}, mz{}, zy{}, zz{} {
    constexpr Stencil<Q> L{};
    for (int i = 0; i < Q; ++i)
      for (int k = 0; k < Q; ++k) {
        if (L.c[k][0] == L.c[i][0] && L.c[k][1] == -L.c[i][1] && L.c[k][2] == L.c[i][2]) my[i] = k;
        if (L.c[k][0] == L.c[i][0] && L.c[k][1] == L.c[i][1] && L.c[k][2] == -L.c[i][2]) mz[i] = k;
        if (L.c[k][0] == L.c[i][0] && L.c[k][1] == 0 && L.c[k][2] == L.c[i][2]) zy[i] = k;
        if (L.c[k][0] == L.c[i][0] && L.c[k][1] == L.c[i][1] && L.c[k][2] == 0) zz[i] = k;
      }
  }
};

// Moving-wall bounce-back (reading G33; lid of the lid-driven cavity): the population i that returns
// from a wall moving with u_w gains 2 w_i rho_w (c_i . u_w) / c_s^2 = 6 w_i (c_i . u_w), rho_w = 1, c_i = wall -> fluid.
template <int Q, typename T>
__device__ __forceinline__ T moving_wall_term(int i, const T (&uw)[3]) {
  constexpr Stencil<Q> L{};
  return T(6) * weight<Q, T>(L.c2[i]) * (T(L.c[i][0]) * uw[0] + T(L.c[i][1]) * uw[1] + T(L.c[i][2]) * uw[2]);
}

template <typename T>
struct StepArgs {
  const T* __restrict__ fin;      // [Q][N]
  T* __restrict__ fout;           // [Q][N]
  const T* __restrict__ d;        // [N] or nullptr (=> d = 0)
  const uint8_t* __restrict__ cls;  // [N]
  const uint32_t* __restrict__ nbmask;  // [N] bit j: neighbour x + c_j is SOLID (non-zero only on ADJ cells)
  int nx, ny, nz;
  long long N;                    // cells = population stride
  T tau0;
  T smago_k;                      // 18 sqrt(2) Cs^2 ; 0 => BGK
  T u_in[3];
  int wm_enable;
  double wm_kappa, wm_E, nu;
  // vector kernel only: cells of every vector that is not pure bulk, handled by the first list_z z-slices
  const int* __restrict__ list;
  int n_list;
  int list_z;
  int z_reverse;                  // vector kernel: walk the slab from its last slice down (serpentine sweep over consecutive launches)
  int z0;                         // first lattice z-slice of this launch (the launch covers the slab z0 .. z0 + nzs - 1)
  int zi0, zi1;                   // interior slices [zi0, zi1) of the lattice (all of it unless ghost slices are declared: lbm_set_halo);
                                  // list cells outside belong to ghost slices and are skipped
  int nzs;                        // z-slices of this launch (grid.z = list_z + nzs, except in the totals modes, whose blocks loop over z)
  // HRR form (Eq. 7-11): u^(x,t) of every cell [3][N] (written by the MODE_UHAT_* pass, SOLID cells 0), Eq. 7 factor
  T* __restrict__ uhat;
  // collision = 2 (reading G41: FD strain of the PREVIOUS level's u^): uhat holds u^(., t - dt), the fused step writes u^(., t) of its
  // cells into uhat_out (a second [3][N] buffer whose wall entries are already in place); nullptr: the two-pass form
  T* __restrict__ uhat_out;
  T sigma;
  const double* __restrict__ uin_field;  // [3][nz][ny] per-cell inlet velocity (Vortex Method inlet / mean profile) or nullptr => u_in;
                                         // fp64 for both dtypes: Eq. 21 normalises a gradient of this field (ill-conditioned in fp32)
  T rho_out;                      // density imposed on POUTLET cells (reading G36)
  T fringe_k;                     // fringe zone (reading G38): tau0(x) = tau0 + fringe_k max(0, x - fringe_x0)^2
  int fringe_x0;
  T u_wall[3];                    // velocity of the MOVINGWALL cells (only ever on the plane z = nz-1), reading G33
  const T* __restrict__ ub;       // [3][N] prescribed solid velocity u^B(x,t) of Eq. 12 (moving porous bodies, l.99-106) or nullptr => 0;
                                  // read only where d != 0 (it enters with weight d); WALLMODEL cells take the wall model's u^B (G39)
  // wall-model pre-pass (A8): u^B of the WALLMODEL cells [3][N] (only their entries are ever written or read), written by
  // k_wallmodel_prepass of the same time level, or nullptr => the per-cell paths solve Spalding's law in place
  T* __restrict__ wm_ub;
  const int* __restrict__ wm_list;   // WALLMODEL cells, ascending
  int n_wm;
  int pdl_wait_all;               // 1: every thread waits for the preceding kernel (it wrote this kernel's input);
                                  // 0: only the threads that read wm_ub wait (the predecessor is the wall-model pre-pass)
  // A9 outputs: caller arrays rho[N], u[3][N] (either may be nullptr); totals: slots[LBM slots][5] partial sums, a ticket, out[5]
  T* __restrict__ mom_rho;
  T* __restrict__ mom_u;
  double* __restrict__ tot_slots;
  unsigned* __restrict__ tot_ticket;
  double* __restrict__ tot_out;
  int tot_nslots;
};

// ---- math helpers ---------------------------------------------------------------------------------
// fp32: hardware approximations (MUFU) instead of the IEEE-rounded software sequences, which cost ~10
// instructions and a slow-path stub each.  rho is always a normal number near 1, so no denormal care is
// needed.  The reciprocal gets one Newton step (2 FMA) and is then within 1 ulp and unbiased, which keeps
// the momentum of the collision free of a systematic drift; sqrt only feeds tau_eff.
__device__ __forceinline__ float rcp_(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return fmaf(fmaf(-x, r, 1.0f), r, r);
}
__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }
__device__ __forceinline__ float sqrt_(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }

// A2..A6 on one cell held in registers.  f[] in: S_t, out: post-collision F_t.
// (ubx,uby,ubz) = u^B; d = porosity.  Eq. 6, 11 (to H2), 12, 14 with Eq. 3-5 in closed form:
//   tau_eff = (tau0 + sqrt(tau0^2 + 18 sqrt2 Cs^2 |Pi| / rho)) / 2,   Pi = sum_i c c (f_i - feq_i)
// Opposite directions are paired: sums s = f_i + f_opp and differences for the odd moments.
template <int Q, typename T>
__device__ __forceinline__ void collide_cell(T (&f)[Q], T d, T ubx, T uby, T ubz, T tau0, T smago_k) {
  constexpr Stencil<Q> L{};
  constexpr int H = (Q - 1) / 2;
  T rho = f[0], jx = T(0), jy = T(0), jz = T(0);
  T mxx = T(0), myy = T(0), mzz = T(0), mxy = T(0), mxz = T(0), myz = T(0);
#pragma unroll
  for (int i = 1; i <= H; ++i) {
    const T s = f[i] + f[i + H];
    const T a = f[i] - f[i + H];
    rho += s;
    if (L.c[i][0] == 1) jx += a; else if (L.c[i][0] == -1) jx -= a;
    if (L.c[i][1] == 1) jy += a; else if (L.c[i][1] == -1) jy -= a;
    if (L.c[i][2] == 1) jz += a; else if (L.c[i][2] == -1) jz -= a;
    if (L.c[i][0] != 0) mxx += s;
    if (L.c[i][1] != 0) myy += s;
    if (L.c[i][2] != 0) mzz += s;
    if (L.c[i][0] * L.c[i][1] == 1) mxy += s; else if (L.c[i][0] * L.c[i][1] == -1) mxy -= s;
    if (L.c[i][0] * L.c[i][2] == 1) mxz += s; else if (L.c[i][0] * L.c[i][2] == -1) mxz -= s;
    if (L.c[i][1] * L.c[i][2] == 1) myz += s; else if (L.c[i][1] * L.c[i][2] == -1) myz -= s;
  }
  const T inv_rho = rcp_(rho);
  const T keep = T(1) - d;                                  // Eq. 12
  const T ux = keep * (jx * inv_rho) + d * ubx;
  const T uy = keep * (jy * inv_rho) + d * uby;
  const T uz = keep * (jz * inv_rho) + d * ubz;
  T omega;
  if (smago_k > T(0)) {
    // second moment of f^eq(rho, u^) is rho (I/3 + u^ u^)
    const T qx = rho * ux, qy = rho * uy, qz = rho * uz;
    const T third = rho * T(1.0 / 3.0);
    const T pxx = (mxx - third) - qx * ux;
    const T pyy = (myy - third) - qy * uy;
    const T pzz = (mzz - third) - qz * uz;
    const T pxy = mxy - qx * uy;
    const T pxz = mxz - qx * uz;
    const T pyz = myz - qy * uz;
    const T off = pxy * pxy + pxz * pxz + pyz * pyz;
    const T npi = sqrt_(pxx * pxx + pyy * pyy + pzz * pzz + (off + off));
    const T tau = T(0.5) * (tau0 + sqrt_(tau0 * tau0 + smago_k * npi * inv_rho));
    omega = rcp_(tau);
  } else {
    omega = rcp_(tau0);
  }
  const T base = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
  const T keepf = T(1) - omega;
  const T ro = rho * omega;
  // per weight class (|c|^2 = 1, 2, 3): A = w rho omega base, B = 4.5 w rho omega, C = 3 w rho omega.
  // Conservation in fp32: the lattice weights are not exactly representable, so sum_i w_i != 1 and
  // sum_i 3 w_i c_ix^2 != 1 in floating point -- a systematic (not random) drift of mass and momentum of a few
  // 1e-8 per step.  Two remedies that cost (almost) nothing:
  //  * the odd-part constants c3[k] = 3 w_k are chosen so that 2 c3[1] + 8 c3[2] (+ 8 c3[3]) == 1 exactly
  //    (c3[1] takes the remainder), which makes sum_i c_i f^eq_i = rho u^ free of weight rounding;
  //  * the rest population takes what is left of the mass: f0' = (1-omega) f0 + (rho omega - 2 sum_pairs even),
  //    so sum_i f_i' = rho up to unbiased rounding of the individual operations.
  constexpr double c3_2 = static_cast<double>(static_cast<T>(3.0 * static_cast<double>(weight<Q, double>(2))));
  constexpr double c3_3 = (Q == 27) ? static_cast<double>(static_cast<T>(3.0 * static_cast<double>(weight<Q, double>(3)))) : 0.0;
  constexpr double c3_1 = (1.0 - 8.0 * c3_2 - 8.0 * c3_3) / 2.0;
  constexpr T c3[4] = {T(0), static_cast<T>(c3_1), static_cast<T>(c3_2), static_cast<T>(c3_3)};
  T A[4], B[4], C[4];
#pragma unroll
  for (int k = 1; k <= ((Q == 19) ? 2 : 3); ++k) {
    const T wr = weight<Q, T>(k) * ro;
    A[k] = wr * base;
    B[k] = wr * T(4.5);
    C[k] = c3[k] * ro;
  }
  T esum = T(0);
#pragma unroll
  for (int i = 1; i <= H; ++i) {
    T cu = T(0);
    if (L.c[i][0] == 1) cu += ux; else if (L.c[i][0] == -1) cu -= ux;
    if (L.c[i][1] == 1) cu += uy; else if (L.c[i][1] == -1) cu -= uy;
    if (L.c[i][2] == 1) cu += uz; else if (L.c[i][2] == -1) cu -= uz;
    const int k = L.c2[i];
    const T even = (B[k] * cu) * cu + A[k];
    const T odd = C[k] * cu;
    esum += even;
    f[i] = keepf * f[i] + (even + odd);
    f[i + H] = keepf * f[i + H] + (even - odd);
  }
  f[0] = keepf * f[0] + (ro - (esum + esum));
}

// ---- HRR form: the paper's own collision, Eq. 6-11 in full ------------------------------------
// Third-order Hermite coefficients carried by the lattices: k = 0..6 <-> xxy, xxz, xyy, xzz, yyz, yzz, xyz.
// h3<Q>(i, k) = the factor of coefficient A3[k] in the order-3 term of a Hermite series at direction i (without w_i):
//   D3Q27: H(3)_k(c_i) / (2 c_s^6) for the six aab components (Eq. 11 as printed), H(3)_xyz / c_s^6;
//   D3Q19: projection on the orthogonal combinations H_xxy +- H_yzz, H_xzz +- H_xyy, H_yyz +- H_xxz (reading G9):
//          [3 (Hp+Hq)(ap+aq) + (Hp-Hq)(ap-aq)] / (6 c_s^6)  =>  factor of ap: 18 Hp + 9 Hq, of aq: 9 Hp + 18 Hq.
__host__ __device__ constexpr double herm3_raw(int cx, int cy, int cz, int k) {
  // H(3)_abg = c_a c_b c_g - c_s^2 (d_ab c_g + d_ag c_b + d_bg c_a)
  return k == 0 ? cy * (cx * cx - 1.0 / 3.0)
       : k == 1 ? cz * (cx * cx - 1.0 / 3.0)
       : k == 2 ? cx * (cy * cy - 1.0 / 3.0)
       : k == 3 ? cx * (cz * cz - 1.0 / 3.0)
       : k == 4 ? cz * (cy * cy - 1.0 / 3.0)
       : k == 5 ? cy * (cz * cz - 1.0 / 3.0)
                : static_cast<double>(cx * cy * cz);
}
template <int Q>
__host__ __device__ constexpr double h3(int cx, int cy, int cz, int k) {
  if (Q == 27) return (k < 6 ? 13.5 : 27.0) * herm3_raw(cx, cy, cz, k);
  if (k == 6) return 0.0;
  // partner of k in the pairs (xxy,yzz) = (0,5), (xzz,xyy) = (3,2), (yyz,xxz) = (4,1)
  const int q = (k == 0) ? 5 : (k == 5) ? 0 : (k == 3) ? 2 : (k == 2) ? 3 : (k == 4) ? 1 : 4;
  return 18.0 * herm3_raw(cx, cy, cz, k) + 9.0 * herm3_raw(cx, cy, cz, q);
}

// A2..A6 in the HRR form on one cell held in registers.  f[] in: S_t, out: post-collision F_t.
//   f*_i = f^eq_i + (1 - 1/tau) [sigma f(1)_i + (1 - sigma) f(1,FD)_i]                          (Eq. 6, 7)
//   f^eq = w (rho + 3 c.rho u^ + 4.5 H2:rho u^u^ + order3(rho u^u^u^))                           (Eq. 11)
//   f(1) = w (a0 + 3 c.a1 + 4.5 H2:a2 + order3(a3)),  a_n = sum_i H(n)_i (f_i - f^eq_i),         (Eq. 8-9)
//          a3_abg = u^_a a2_bg + u^_b a2_ag + u^_g a2_ab                                          (G29)
//   f(1,FD) = -w rho tau / c_s^2 H2:S                                                            (Eq. 10, G10)
// Every part is a Hermite series with the same basis, so the coefficients are combined first (k = 1 - 1/tau):
//   A1 = rho u^ + k sigma a1,  A2 = rho u^u^ + k (sigma a2 - (1-sigma)(2/3) rho tau S),  A3 = rho u^u^u^ + k sigma a3
// and the series is evaluated once.  a0 = 0, a1 = rho (u - u^), a2 = M2 - rho (I/3 + u^u^) follow from the moments
// of Eq. 11 (its order-3 term has no moments below order 3).  tau = tau_eff from |a2| as in the BGK form (A5).
// S[6] = S^FD_xx, yy, zz, xy, xz, yz.
template <int Q, typename T>
__device__ __forceinline__ void collide_cell_hrr(T (&f)[Q], T d, T ubx, T uby, T ubz, T tau0, T smago_k, T sigma,
                                                 const T (&S)[6], T& uox, T& uoy, T& uoz) {   // uo: u^(x,t) of the cell (Eq. 12)
  constexpr Stencil<Q> L{};
  constexpr int H = (Q - 1) / 2;
  T rho = f[0], jx = T(0), jy = T(0), jz = T(0);
  T mxx = T(0), myy = T(0), mzz = T(0), mxy = T(0), mxz = T(0), myz = T(0);
#pragma unroll
  for (int i = 1; i <= H; ++i) {
    const T s = f[i] + f[i + H];
    const T a = f[i] - f[i + H];
    rho += s;
    if (L.c[i][0] == 1) jx += a; else if (L.c[i][0] == -1) jx -= a;
    if (L.c[i][1] == 1) jy += a; else if (L.c[i][1] == -1) jy -= a;
    if (L.c[i][2] == 1) jz += a; else if (L.c[i][2] == -1) jz -= a;
    if (L.c[i][0] != 0) mxx += s;
    if (L.c[i][1] != 0) myy += s;
    if (L.c[i][2] != 0) mzz += s;
    if (L.c[i][0] * L.c[i][1] == 1) mxy += s; else if (L.c[i][0] * L.c[i][1] == -1) mxy -= s;
    if (L.c[i][0] * L.c[i][2] == 1) mxz += s; else if (L.c[i][0] * L.c[i][2] == -1) mxz -= s;
    if (L.c[i][1] * L.c[i][2] == 1) myz += s; else if (L.c[i][1] * L.c[i][2] == -1) myz -= s;
  }
  const T inv_rho = rcp_(rho);
  const T keep = T(1) - d;                                  // Eq. 12
  const T ux = keep * (jx * inv_rho) + d * ubx;
  const T uy = keep * (jy * inv_rho) + d * uby;
  const T uz = keep * (jz * inv_rho) + d * ubz;
  uox = ux;  uoy = uy;  uoz = uz;
  const T qx = rho * ux, qy = rho * uy, qz = rho * uz;
  const T third = rho * T(1.0 / 3.0);
  // a2 (= Pi of the BGK form, now against the third-order equilibrium: same second moment)
  const T pxx = (mxx - third) - qx * ux;
  const T pyy = (myy - third) - qy * uy;
  const T pzz = (mzz - third) - qz * uz;
  const T pxy = mxy - qx * uy;
  const T pxz = mxz - qx * uz;
  const T pyz = myz - qy * uz;
  T tau = tau0, omega;
  if (smago_k > T(0)) {
    const T off = pxy * pxy + pxz * pxz + pyz * pyz;
    const T npi = sqrt_(pxx * pxx + pyy * pyy + pzz * pzz + (off + off));
    tau = T(0.5) * (tau0 + sqrt_(tau0 * tau0 + smago_k * npi * inv_rho));
  }
  omega = rcp_(tau);
  const T k = T(1) - omega;
  const T ks = k * sigma;
  const T kf = -(k - ks) * T(2.0 / 3.0) * rho * tau;        // k (1 - sigma) * (-(2/3) rho tau)
  const T A1x = qx + ks * (jx - qx), A1y = qy + ks * (jy - qy), A1z = qz + ks * (jz - qz);
  const T Axx = qx * ux + (ks * pxx + kf * S[0]);
  const T Ayy = qy * uy + (ks * pyy + kf * S[1]);
  const T Azz = qz * uz + (ks * pzz + kf * S[2]);
  const T Axy = qx * uy + (ks * pxy + kf * S[3]);
  const T Axz = qx * uz + (ks * pxz + kf * S[4]);
  const T Ayz = qy * uz + (ks * pyz + kf * S[5]);
  T A3[7];
  A3[0] = qx * ux * uy + ks * (T(2) * ux * pxy + uy * pxx);          // xxy
  A3[1] = qx * ux * uz + ks * (T(2) * ux * pxz + uz * pxx);          // xxz
  A3[2] = qx * uy * uy + ks * (ux * pyy + T(2) * uy * pxy);          // xyy
  A3[3] = qx * uz * uz + ks * (ux * pzz + T(2) * uz * pxz);          // xzz
  A3[4] = qy * uy * uz + ks * (T(2) * uy * pyz + uz * pyy);          // yyz
  A3[5] = qy * uz * uz + ks * (uy * pzz + T(2) * uz * pyz);          // yzz
  A3[6] = qx * uy * uz + ks * (ux * pyz + uy * pxz + uz * pxy);      // xyz
  // even part of direction i: w (rho - 1.5 tr A2 + 4.5 cc:A2); odd part: 3 w c.A1 + w sum_k h3 A3[k].
  // Conservation in fp32 as in collide_cell: c3[] sums to exactly 1 over the stencil, the rest population takes what
  // is left of rho.
  constexpr double c3_2 = static_cast<double>(static_cast<T>(3.0 * static_cast<double>(weight<Q, double>(2))));
  constexpr double c3_3 = (Q == 27) ? static_cast<double>(static_cast<T>(3.0 * static_cast<double>(weight<Q, double>(3)))) : 0.0;
  constexpr double c3_1 = (1.0 - 8.0 * c3_2 - 8.0 * c3_3) / 2.0;
  constexpr T c3[4] = {T(0), static_cast<T>(c3_1), static_cast<T>(c3_2), static_cast<T>(c3_3)};
  const T e0 = rho - T(1.5) * (Axx + Ayy + Azz);
  T esum = T(0);
#pragma unroll
  for (int i = 1; i <= H; ++i) {
    const int cx = L.c[i][0], cy = L.c[i][1], cz = L.c[i][2];
    const T w = weight<Q, T>(L.c2[i]);
    T cA = T(0), cc = T(0), o3 = T(0);
    if (cx == 1) cA += A1x; else if (cx == -1) cA -= A1x;
    if (cy == 1) cA += A1y; else if (cy == -1) cA -= A1y;
    if (cz == 1) cA += A1z; else if (cz == -1) cA -= A1z;
    if (cx != 0) cc += Axx;
    if (cy != 0) cc += Ayy;
    if (cz != 0) cc += Azz;
    T cross = T(0);
    if (cx * cy == 1) cross += Axy; else if (cx * cy == -1) cross -= Axy;
    if (cx * cz == 1) cross += Axz; else if (cx * cz == -1) cross -= Axz;
    if (cy * cz == 1) cross += Ayz; else if (cy * cz == -1) cross -= Ayz;
    cc += cross + cross;
#pragma unroll
    for (int kk = 0; kk < 7; ++kk) {
      const double hk = h3<Q>(cx, cy, cz, kk) * static_cast<double>(weight<Q, double>(L.c2[i]));
      if (hk != 0.0) o3 += static_cast<T>(hk) * A3[kk];
    }
    const T even = w * (e0 + T(4.5) * cc);
    const T odd = c3[L.c2[i]] * cA + o3;
    esum += even;
    f[i] = even + odd;
    f[i + H] = even - odd;
  }
  f[0] = rho - (esum + esum);
}

template <int Q, typename T>
__device__ __forceinline__ void collide_cell_hrr(T (&f)[Q], T d, T ubx, T uby, T ubz, T tau0, T smago_k, T sigma, const T (&S)[6]) {
  T a, b, c;
  collide_cell_hrr<Q, T>(f, d, ubx, uby, ubz, tau0, smago_k, sigma, S, a, b, c);
}

// O4 / reading R6: regularised velocity inlet on a cell of the plane x = 0 (inward normal +x).
template <int Q, typename T>
__device__ __forceinline__ void inlet_fixup(T (&g)[Q], T uwx, T uwy, T uwz) {
  constexpr Stencil<Q> L{};
  T s0 = T(0), sm = T(0);
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    if (L.c[i][0] == 0) s0 += g[i];
    else if (L.c[i][0] < 0) sm += g[i];
  }
  const T rho = (s0 + T(2) * sm) / (T(1) - uwx);
  const T base = T(1) - T(1.5) * (uwx * uwx + uwy * uwy + uwz * uwz);
  T feq[Q];
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const T cu = T(L.c[i][0]) * uwx + T(L.c[i][1]) * uwy + T(L.c[i][2]) * uwz;
    feq[i] = weight<Q, T>(L.c2[i]) * rho * (base + T(3) * cu + T(4.5) * cu * cu);
  }
  // non-equilibrium: known directions as they are, unknown (cx > 0) from the opposite one
  T pxx = T(0), pyy = T(0), pzz = T(0), pxy = T(0), pxz = T(0), pyz = T(0);
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const int k = (L.c[i][0] > 0) ? L.opp[i] : i;
    const T n = g[k] - feq[k];
    pxx += T(L.c[i][0] * L.c[i][0]) * n;
    pyy += T(L.c[i][1] * L.c[i][1]) * n;
    pzz += T(L.c[i][2] * L.c[i][2]) * n;
    pxy += T(L.c[i][0] * L.c[i][1]) * n;
    pxz += T(L.c[i][0] * L.c[i][2]) * n;
    pyz += T(L.c[i][1] * L.c[i][2]) * n;
  }
  const T tr3 = (pxx + pyy + pzz) * T(1.0 / 3.0);
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const T q = T(L.c[i][0] * L.c[i][0]) * pxx + T(L.c[i][1] * L.c[i][1]) * pyy + T(L.c[i][2] * L.c[i][2]) * pzz +
                T(2) * (T(L.c[i][0] * L.c[i][1]) * pxy + T(L.c[i][0] * L.c[i][2]) * pxz + T(L.c[i][1] * L.c[i][2]) * pyz) - tr3;
    g[i] = feq[i] + T(4.5) * weight<Q, T>(L.c2[i]) * q;
  }
}

// O4p / reading G36: regularised pressure outlet on a cell of the plane x = nx-1 (outward normal +x): rho_out is
// imposed, the normal velocity follows from the known populations (c_x >= 0), tangential velocity 0 -- the mirror image of
// inlet_fixup, which does the rest.
template <int Q, typename T>
__device__ __forceinline__ void pressure_fixup(T (&g)[Q], T rho_out) {
  constexpr Stencil<Q> L{};
  constexpr int H = (Q - 1) / 2;
  T s0 = T(0), sp = T(0);
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    if (L.c[i][0] == 0) s0 += g[i];
    else if (L.c[i][0] > 0) sp += g[i];
  }
  const T ux = (s0 + T(2) * sp) / rho_out - T(1);
  // reflect in x (directions with c_x != 0 swap with their x-mirror), impose -u_x as on an inlet, reflect back
  T m[Q];
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    int j = i;
    if (L.c[i][0] != 0) {
#pragma unroll
      for (int k = 1; k < Q; ++k)
        if (L.c[k][0] == -L.c[i][0] && L.c[k][1] == L.c[i][1] && L.c[k][2] == L.c[i][2]) j = k;
    }
    m[i] = g[j];
  }
  (void)H;
  inlet_fixup<Q, T>(m, -ux, T(0), T(0));
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    int j = i;
    if (L.c[i][0] != 0) {
#pragma unroll
      for (int k = 1; k < Q; ++k)
        if (L.c[k][0] == -L.c[i][0] && L.c[k][1] == L.c[i][1] && L.c[k][2] == L.c[i][2]) j = k;
    }
    g[i] = m[j];
  }
}

// Spalding's law (Eq. 17) and the two root solves of reading R8, in double for both dtypes (only the
// wall-model cells take this path).  Returns U1 / U2.
//   unknown p = u2+ = U2 / u_tau:   p Sp(p) = Re,  Re = U2 y2 / nu      (Eq. 15-16: y2+ u2+ = U2 y2 / nu)
//   then q = u1+:                   Sp(q) = y1+ = (y1 / y2) Re / p
// Both left sides are increasing and convex, so Newton converges monotonically once it is on the
// right of the root; the start values (viscous / log-law estimates) put it there or one step away.
// The roots are the unique ones the definition fixes, converged to 1e-14 relative.
__device__ __forceinline__ void spalding_eval(double up, double kappa, double invE, double& sp, double& dsp) {
  const double k = kappa * up;
  const double ek = exp(k);
  const double k2 = 0.5 * k * k;
  sp = up + invE * (ek - 1.0 - k - k2 - k2 * k * (1.0 / 3.0));
  dsp = 1.0 + kappa * invE * (ek - 1.0 - k - k2);
}

static __device__ __noinline__ double wallmodel_ratio(double U2, double nu, double kappa, double E) {
  const double y2 = 1.5, y1 = 0.5;
  const double invE = 1.0 / E;
  const double Re = U2 * y2 / nu;
  double p = sqrt(Re);                       // viscous sublayer: Sp(p) = p
  if (p > 8.0) {                             // log region estimate: p = ln(E Re / p) / kappa
    double q = 20.0;
#pragma unroll 1
    for (int it = 0; it < 3; ++it) q = log(E * Re / q) / kappa;
    if (q > 1.0 && q < p) p = q;
  }
#pragma unroll 1
  for (int it = 0; it < 100; ++it) {
    double sp, dsp;
    spalding_eval(p, kappa, invE, sp, dsp);
    const double G = p * sp - Re;
    const double dG = sp + p * dsp;
    double pn = p - G / dG;
    if (!(pn > 0.0)) pn = 0.5 * p;
    const double delta = fabs(pn - p);
    p = pn;
    if (delta <= 1e-14 * p) break;
  }
  const double y1p = (y1 / y2) * Re / p;
  double q = fmin(y1p, p);                   // Sp(q) >= y1+ at both candidates: right of the root
#pragma unroll 1
  for (int it = 0; it < 100; ++it) {
    double sp, dsp;
    spalding_eval(q, kappa, invE, sp, dsp);
    double qn = q - (sp - y1p) / dsp;
    if (qn < 0.0) qn = 0.5 * q;
    const double delta = fabs(qn - q);
    q = qn;
    if (delta <= 1e-14 * fabs(q)) break;
  }
  return q / p;                              // U1 / U2 = u1+ u_tau / (u2+ u_tau)
}

struct Coord {
  int x, y, z;
};

__device__ __forceinline__ long long cell_index(int x, int y, int z, int nx, int ny) {
  return (static_cast<long long>(z) * ny + y) * nx + x;
}

// Full-slip wall (reading G37): the population with velocity c = (cx,cy,cz) (wall -> fluid) that the cell (x,y,z)
// pulls from a SLIPWALL source is the specular image: it left the fluid cell x' = x - c + sum_a c_a e_a with the velocity c with the
// components a reversed, a = the axes along which the cell's single-axis neighbour x - c_a e_a is a slip wall.  No such axis, or a
// wall at x': `fallback` (plain bounce-back).  sx0 = the x coordinate of the source as pulled (OUTLET cells clamp it).
// Rare path (cells next to a slip wall only): kept out of line.
template <int Q, typename T>
__device__ __noinline__ T slip_pull(const StepArgs<T>& a, int x, int y, int z, int cx, int cy, int cz, int sx0, T fallback) {
  constexpr Stencil<Q> L{};
  const int pos[3] = {x, y, z}, dim[3] = {a.nx, a.ny, a.nz}, c[3] = {cx, cy, cz};
  int cr[3] = {cx, cy, cz};
  int pr[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const int t = pos[k] - c[k];
    pr[k] = (t < 0) ? t + dim[k] : ((t >= dim[k]) ? t - dim[k] : t);
  }
  const int wx = pr[0];
  pr[0] = sx0;
  bool any = false;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    if (c[k] == 0) continue;
    int q[3] = {x, y, z};
    q[k] = (k == 0) ? wx : pr[k];
    if ((a.cls[cell_index(q[0], q[1], q[2], a.nx, a.ny)] & CLS_TYPE) == T_SLIP) {
      cr[k] = -c[k];
      pr[k] = pos[k];
      any = true;
    }
  }
  if (!any) return fallback;
  const long long xr = cell_index(pr[0], pr[1], pr[2], a.nx, a.ny);
  if (is_wall(a.cls[xr])) return fallback;
  int ir = 0;
#pragma unroll
  for (int k = 1; k < Q; ++k)
    if (L.c[k][0] == cr[0] && L.c[k][1] == cr[1] && L.c[k][2] == cr[2]) ir = k;
  return __ldg(a.fin + static_cast<long long>(ir) * a.N + xr);
}

// molecular relaxation time of the plane x: tau0, raised quadratically inside the fringe zone in front of the outlet
// (l.255; reading G38: nu_mo(x) = nu_mo (1 + A xi^2), xi = (x - x0)/L; fringe_k = (tau0 - 1/2) A / L^2)
template <typename T>
__device__ __forceinline__ T tau0_at(const StepArgs<T>& a, int x) {
  const int xd = (x > a.fringe_x0) ? x - a.fringe_x0 : 0;
  return a.tau0 + a.fringe_k * static_cast<T>(xd * xd);
}

// velocity imposed on the INLET cell (0, y, z): the per-cell inflow field when one is set (Eq. 21 / mean profile), else u_in
template <typename T>
__device__ __forceinline__ void inlet_velocity(const StepArgs<T>& a, int y, int z, T& ux, T& uy, T& uz) {
  if (a.uin_field != nullptr) {
    const long long P = static_cast<long long>(a.ny) * a.nz, c = static_cast<long long>(z) * a.ny + y;
    ux = static_cast<T>(__ldg(a.uin_field + c));
    uy = static_cast<T>(__ldg(a.uin_field + P + c));
    uz = static_cast<T>(__ldg(a.uin_field + 2 * P + c));
  } else {
    ux = a.u_in[0];  uy = a.u_in[1];  uz = a.u_in[2];
  }
}

// Pull of one cell (A1 + A7): g_i(x) = A[i][x - c_i], periodic wrap; a SOLID source means halfway bounce-back:
// the cell's own opposite population (nbmask bit opp(i): the neighbour x + c_opp(i) = x - c_i is SOLID).  OUTLET
// cells clamp the source of the c_x < 0 populations to their own plane (R7: ghost plane nx := plane nx-1), so for
// those the class of the clamped source decides.  INLET cells get the fix-up R6.  `cls` is the cell's own class
// byte (not SOLID).
template <int Q, typename T>
__device__ __forceinline__ void pull_cell(const StepArgs<T>& a, int x, int y, int z, uint8_t cls, T (&f)[Q]) {
  constexpr Stencil<Q> L{};
  const int type = cls & CLS_TYPE;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const long long N = a.N;
  const long long self = cell_index(x, y, z, nx, ny);
  const uint32_t nbm = (cls & CLS_ADJ) ? a.nbmask[self] : 0u;
  const int xm = (x == 0) ? nx - 1 : x - 1;
  const int xp = (type == T_OUTLET) ? x : ((x == nx - 1) ? 0 : x + 1);
  const int ym = (y == 0) ? ny - 1 : y - 1, yp = (y == ny - 1) ? 0 : y + 1;
  const int zm = (z == 0) ? nz - 1 : z - 1, zp = (z == nz - 1) ? 0 : z + 1;
  const int sc = (type == T_WM) ? 0 : ((cls >> CLS_NORMAL_SHIFT) & 7);       // slip plane code (0 = none)
  constexpr Mirror<Q> MR{};
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const int sx = (L.c[i][0] == 0) ? x : ((L.c[i][0] == 1) ? xm : xp);
    int sy = (L.c[i][1] == 0) ? y : ((L.c[i][1] == 1) ? ym : yp);
    int sz = (L.c[i][2] == 0) ? z : ((L.c[i][2] == 1) ? zm : zp);
    if (sc != 0) {                                            // specular pull at a plane slip wall: own plane, mirrored slot
      if (L.c[i][1] != 0 && sc == ((L.c[i][1] == 1) ? 2 : 3)) {
        f[i] = __ldg(a.fin + MR.my[i] * N + cell_index(sx, y, sz, nx, ny));
        continue;
      }
      if (L.c[i][2] != 0 && sc == ((L.c[i][2] == 1) ? 4 : 5)) {
        f[i] = __ldg(a.fin + MR.mz[i] * N + cell_index(sx, sy, z, nx, ny));
        continue;
      }
    }
    const long long s = cell_index(sx, sy, sz, nx, ny);
    bool own = (i > 0) && ((nbm >> L.opp[i]) & 1u);
    if (L.c[i][0] == -1 && type == T_OUTLET) own = is_wall(a.cls[s]);
    f[i] = own ? __ldg(a.fin + L.opp[i] * N + self) : __ldg(a.fin + i * N + s);
    if (own) {
      const int st = a.cls[s] & CLS_TYPE;
      if (st == T_MOVING) f[i] += moving_wall_term<Q, T>(i, a.u_wall);
      else if (st == T_SLIP) f[i] = slip_pull<Q, T>(a, x, y, z, L.c[i][0], L.c[i][1], L.c[i][2], sx, f[i]);
    }
  }
  if (type == T_INLET) {
    T ux, uy, uz;
    inlet_velocity<T>(a, y, z, ux, uy, uz);
    inlet_fixup<Q, T>(f, ux, uy, uz);
  }
  if (type == T_POUTLET) pressure_fixup<Q, T>(f, a.rho_out);
}

// S_t of one non-SOLID cell, whatever the storage phase.  PULL = input holds F_{t-1}.
template <int Q, typename T, bool PULL>
__device__ __forceinline__ void load_state(const StepArgs<T>& a, int x, int y, int z, uint8_t cls, T (&f)[Q]) {
  if (!PULL) {
    const long long self = cell_index(x, y, z, a.nx, a.ny);
#pragma unroll
    for (int i = 0; i < Q; ++i) f[i] = __ldg(a.fin + i * a.N + self);
  } else {
    pull_cell<Q, T>(a, x, y, z, cls, f);
  }
}

// Store of one cell's Q values.
template <int Q, typename T>
__device__ __forceinline__ void store_cell(const StepArgs<T>& a, int x, int y, int z, const T (&f)[Q]) {
  const long long self = cell_index(x, y, z, a.nx, a.ny);
#pragma unroll
  for (int i = 0; i < Q; ++i) a.fout[i * a.N + self] = f[i];
}
// SOLID cells: nobody reads their slots; zeros keep every written sector whole.
template <int Q, typename T>
__device__ __forceinline__ void store_zero(const StepArgs<T>& a, long long self) {
#pragma unroll
  for (int i = 0; i < Q; ++i) a.fout[i * a.N + self] = T(0);
}

// A8 / reading R8: u^B of a wall-model cell from the tangential velocity at x + n.
template <int Q, typename T, bool PULL>
__device__ __forceinline__ void wallmodel_ub(const StepArgs<T>& a, int x, int y, int z, uint8_t cls, T& ubx, T& uby, T& ubz) {
  constexpr Stencil<Q> L{};
  ubx = uby = ubz = T(0);
  const int code = (cls >> CLS_NORMAL_SHIFT) & 7;
  int n[3] = {0, 0, 0};
  n[code >> 1] = (code & 1) ? -1 : 1;
  int x2 = x + n[0], y2 = y + n[1], z2 = z + n[2];
  x2 = (x2 < 0) ? x2 + a.nx : ((x2 >= a.nx) ? x2 - a.nx : x2);
  y2 = (y2 < 0) ? y2 + a.ny : ((y2 >= a.ny) ? y2 - a.ny : y2);
  z2 = (z2 < 0) ? z2 + a.nz : ((z2 >= a.nz) ? z2 - a.nz : z2);
  const uint8_t cls2 = a.cls[cell_index(x2, y2, z2, a.nx, a.ny)];
  if (is_wall(cls2)) return;
  T f2[Q];
  load_state<Q, T, PULL>(a, x2, y2, z2, cls2, f2);
  double rho = 0.0, j[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const double v = static_cast<double>(f2[i]);
    rho += v;
    j[0] += L.c[i][0] * v;
    j[1] += L.c[i][1] * v;
    j[2] += L.c[i][2] * v;
  }
  const double u2[3] = {j[0] / rho, j[1] / rho, j[2] / rho};
  const double un = u2[0] * n[0] + u2[1] * n[1] + u2[2] * n[2];
  const double t0 = u2[0] - un * n[0], t1 = u2[1] - un * n[1], t2 = u2[2] - un * n[2];
  const double U2 = sqrt(t0 * t0 + t1 * t1 + t2 * t2);
  if (U2 < 1e-14) return;
  const double r = wallmodel_ratio(U2, a.nu, a.wm_kappa, a.wm_E);
  ubx = static_cast<T>(r * t0);
  uby = static_cast<T>(r * t1);
  ubz = static_cast<T>(r * t2);
}

// S^FD(x,t) of one cell (Eq. 10): S_ab = (D_a u^_b + D_b u^_a)/2 with central differences of the stored u^ field,
// periodic wrap; the ghost planes beyond the INLET / OUTLET planes copy those planes (G32).  S = xx, yy, zz, xy, xz, yz.
template <typename T>
__device__ __forceinline__ void fd_strain_cell(const StepArgs<T>& a, int x, int y, int z, int type, T (&S)[6]) {
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const int xm = (type == T_INLET) ? x : ((x == 0) ? nx - 1 : x - 1);
  const int xp = (type == T_OUTLET || type == T_POUTLET) ? x : ((x == nx - 1) ? 0 : x + 1);
  const int ym = (y == 0) ? ny - 1 : y - 1, yp = (y == ny - 1) ? 0 : y + 1;
  const int zm = (z == 0) ? nz - 1 : z - 1, zp = (z == nz - 1) ? 0 : z + 1;
  T D[3][3];   // D[a][b] = u^_b(x + e_a) - u^_b(x - e_a)
#pragma unroll
  for (int b = 0; b < 3; ++b) {
    const T* u = a.uhat + b * a.N;
    D[0][b] = u[cell_index(xp, y, z, nx, ny)] - u[cell_index(xm, y, z, nx, ny)];
    D[1][b] = u[cell_index(x, yp, z, nx, ny)] - u[cell_index(x, ym, z, nx, ny)];
    D[2][b] = u[cell_index(x, y, zp, nx, ny)] - u[cell_index(x, y, zm, nx, ny)];
  }
  S[0] = T(0.5) * D[0][0];
  S[1] = T(0.5) * D[1][1];
  S[2] = T(0.5) * D[2][2];
  S[3] = T(0.25) * (D[0][1] + D[1][0]);
  S[4] = T(0.25) * (D[0][2] + D[2][0]);
  S[5] = T(0.25) * (D[1][2] + D[2][1]);
}

// u^ = (1-d) sum c f / sum f + d u^B of one cell (Eq. 12), the field the FD strain is taken of (G30).
template <int Q, typename T>
__device__ __forceinline__ void uhat_of(const T (&f)[Q], T d, T ubx, T uby, T ubz, T& ux, T& uy, T& uz) {
  constexpr Stencil<Q> L{};
  constexpr int H = (Q - 1) / 2;
  T rho = f[0], jx = T(0), jy = T(0), jz = T(0);
#pragma unroll
  for (int i = 1; i <= H; ++i) {
    rho += f[i] + f[i + H];
    const T df = f[i] - f[i + H];
    if (L.c[i][0] == 1) jx += df; else if (L.c[i][0] == -1) jx -= df;
    if (L.c[i][1] == 1) jy += df; else if (L.c[i][1] == -1) jy -= df;
    if (L.c[i][2] == 1) jz += df; else if (L.c[i][2] == -1) jz -= df;
  }
  const T inv_rho = rcp_(rho);
  const T keep = T(1) - d;
  ux = keep * (jx * inv_rho) + d * ubx;
  uy = keep * (jy * inv_rho) + d * uby;
  uz = keep * (jz * inv_rho) + d * ubz;
}

// prescribed solid velocity u^B of one cell (Eq. 12): three element loads, and only where the porosity gives it a weight
template <typename T>
__device__ __forceinline__ void body_velocity(const T* __restrict__ pub, long long N, T d, T& ubx, T& uby, T& ubz) {
  ubx = uby = ubz = T(0);
  if (pub != nullptr && d != T(0)) {
    ubx = __ldg(pub);
    uby = __ldg(pub + N);
    ubz = __ldg(pub + 2 * N);
  }
}

// raw moments of one cell held in registers (A2 / A9): rho = sum f, j = sum c f
template <int Q, typename T>
__device__ __forceinline__ void cell_moments(const T (&f)[Q], T& rho, T& jx, T& jy, T& jz) {
  constexpr Stencil<Q> L{};
  constexpr int H = (Q - 1) / 2;
  rho = f[0];
  jx = jy = jz = T(0);
#pragma unroll
  for (int i = 1; i <= H; ++i) {
    rho += f[i] + f[i + H];
    const T df = f[i] - f[i + H];
    if (L.c[i][0] == 1) jx += df; else if (L.c[i][0] == -1) jx -= df;
    if (L.c[i][1] == 1) jy += df; else if (L.c[i][1] == -1) jy -= df;
    if (L.c[i][2] == 1) jz += df; else if (L.c[i][2] == -1) jz -= df;
  }
}

// A9 totals: block partial sums -> slot (spreads the atomics over nslots x 5 addresses) -> the last block of the grid
// (ticket) adds the slots up in a fixed order, writes out[5] and leaves slots and ticket zeroed for the next launch.
// Every thread of the block must call it (warp shuffle tree -> shared memory -> one atomicAdd(double) per block and quantity).
__device__ __forceinline__ void reduce_totals(const double (&v)[5], double* __restrict__ slots, int nslots,
                                              unsigned* __restrict__ ticket, double* __restrict__ out) {
  __shared__ double part[5][8];
  __shared__ int s_last;
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double s = v[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (lane == 0) part[k][warp] = s;
  }
  __syncthreads();
  const int nwarps = (blockDim.x * blockDim.y + 31) >> 5;
  const unsigned nblocks = gridDim.x * gridDim.y * gridDim.z;
  const unsigned blk = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
  if (tid < 5) {
    double s = 0.0;
    for (int w = 0; w < nwarps; ++w) s += part[tid][w];
    if (s != 0.0) atomicAdd(slots + static_cast<size_t>(blk % nslots) * 5 + tid, s);
    __threadfence();
  }
  __syncthreads();
  if (tid == 0) s_last = (atomicInc(ticket, nblocks - 1u) == nblocks - 1u) ? 1 : 0;   // wraps to 0 on the last block
  __syncthreads();
  if (s_last) {
    // the last block: every warp takes quantities k = warp, warp + nwarps, ...; its lanes read the slots q = lane, lane + 32, ...
    // (independent loads, all in flight together -- one thread walking the 256 slots waited for 256 round trips to L2, 45 us),
    // then a shuffle tree in a fixed order; slots and ticket are left zeroed for the next launch
    __threadfence();
    for (int k = warp; k < 5; k += nwarps) {
      double s = 0.0;
      for (int q = lane; q < nslots; q += 32) {
        s += __ldcg(slots + static_cast<size_t>(q) * 5 + k);
        slots[static_cast<size_t>(q) * 5 + k] = 0.0;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
      if (lane == 0) out[k] = s;
    }
  }
}

// ---- the per-cell step (scalar kernel; list blocks of the vector kernel) ------------------------------
// One non-wall cell of any type: pull (modes that pull), wall model, then collide + store (collide modes), store S_t
// (MODE_STREAM), store u^ (MODE_UHAT_*), store rho, u (MODE_MOMENTS_*) or add to the totals acc[] (MODE_TOTALS_*).
template <int Q, typename T, int MODE, int COLL>
__device__ __forceinline__ void step_cell_any(const StepArgs<T>& a, int x, int y, int z, uint8_t cls, double (&acc)[5]) {
  constexpr bool PULL = mode_pulls(MODE);
  const long long self = cell_index(x, y, z, a.nx, a.ny);
  const int type = cls & CLS_TYPE;
  T d = T(0), ubx = T(0), uby = T(0), ubz = T(0);
  const bool wm = (type == T_WM) && a.wm_enable;
  if (mode_hlbm(MODE)) {
    if (a.d != nullptr) d = __ldg(a.d + self);
    if (wm) {
      if (a.wm_ub != nullptr) {                // written by the pre-pass of this time level (possibly still running: PDL)
        if (!a.pdl_wait_all) griddep_wait();
        ubx = __ldcg(a.wm_ub + self);
        uby = __ldcg(a.wm_ub + a.N + self);
        ubz = __ldcg(a.wm_ub + 2 * a.N + self);
      } else {
        wallmodel_ub<Q, T, PULL>(a, x, y, z, cls, ubx, uby, ubz);
      }
    } else if (a.ub != nullptr) {
      body_velocity<T>(a.ub + self, a.N, d, ubx, uby, ubz);
    }
  }
  T f[Q];
  load_state<Q, T, PULL>(a, x, y, z, cls, f);
  if (mode_diag(MODE)) {
    T rho, jx, jy, jz;
    cell_moments<Q, T>(f, rho, jx, jy, jz);
    if (mode_moments(MODE)) {
      const T ir = rcp_(rho);
      if (a.mom_rho != nullptr) a.mom_rho[self] = rho;
      if (a.mom_u != nullptr) {
        a.mom_u[self] = jx * ir;
        a.mom_u[a.N + self] = jy * ir;
        a.mom_u[2 * a.N + self] = jz * ir;
      }
    } else {
      const double r = static_cast<double>(rho), px = static_cast<double>(jx), py = static_cast<double>(jy), pz = static_cast<double>(jz);
      acc[0] += r;  acc[1] += px;  acc[2] += py;  acc[3] += pz;
      acc[4] += 0.5 * (px * px + py * py + pz * pz) / r;
    }
    return;
  }
  if (mode_uhat(MODE)) {
    T ux, uy, uz;
    uhat_of<Q, T>(f, d, ubx, uby, ubz, ux, uy, uz);
    a.uhat[self] = ux;
    a.uhat[a.N + self] = uy;
    a.uhat[2 * a.N + self] = uz;
    return;
  }
  if (mode_collides(MODE)) {
    if (COLL == COLL_HRR) {
      T S[6];
      fd_strain_cell<T>(a, x, y, z, type, S);
      T uox, uoy, uoz;
      collide_cell_hrr<Q, T>(f, d, ubx, uby, ubz, tau0_at<T>(a, x), a.smago_k, wm ? T(0) : a.sigma, S, uox, uoy, uoz);   // sigma = 0: l.131
      if (a.uhat_out != nullptr) {           // G41: this level's u^ is the next step's history
        a.uhat_out[self] = uox;
        a.uhat_out[a.N + self] = uoy;
        a.uhat_out[2 * a.N + self] = uoz;
      }
    } else {
      collide_cell<Q, T>(f, d, ubx, uby, ubz, tau0_at<T>(a, x), a.smago_k);
    }
  }
  store_cell<Q, T>(a, x, y, z, f);
}

// wall cell in the per-cell paths: zeros over its lattice slots (never read; keeps sectors whole) / u^ = the wall's velocity;
// the A9 modes leave it alone (moments: k_solid_moments reports the cell's own values; totals: walls do not count)
template <int Q, typename T, int MODE>
__device__ __forceinline__ void solid_cell_any(const StepArgs<T>& a, long long self) {
  if (mode_diag(MODE)) return;
  if (mode_uhat(MODE)) {
    const bool mv = (a.cls[self] & CLS_TYPE) == T_MOVING;     // u^ of a wall cell = the wall's velocity (G30, G33)
    a.uhat[self] = mv ? a.u_wall[0] : T(0);
    a.uhat[a.N + self] = mv ? a.u_wall[1] : T(0);
    a.uhat[2 * a.N + self] = mv ? a.u_wall[2] : T(0);
  } else {
    store_zero<Q, T>(a, self);
  }
}

// grid (ceil(nx/bx), ceil(ny/by), slab), block (bx, by): thread <-> cell, x fastest (coalesced rows).
// Fallback for row lengths the vector kernel does not take.
template <int Q, typename T, int MODE, int COLL>
__global__ void __launch_bounds__(256) k_step(const __grid_constant__ StepArgs<T> a) {
  if (a.pdl_wait_all) griddep_wait();
  griddep_launch();
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = a.z0 + blockIdx.z;
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (x < a.nx && y < a.ny) {
    const long long self = cell_index(x, y, z, a.nx, a.ny);
    const uint8_t cls = a.cls[self];
    if (is_wall(cls)) solid_cell_any<Q, T, MODE>(a, self);   // wall cells are inert (R5); their slots are never read
    else step_cell_any<Q, T, MODE, COLL>(a, x, y, z, cls, acc);
  }
  if constexpr (mode_totals(MODE)) reduce_totals(acc, a.tot_slots, a.tot_nslots, a.tot_ticket, a.tot_out);
}

// A8 as a pre-pass over the compact list of WALLMODEL cells (reading R8): u^B of every wall-model cell of this time level, so
// that the cells themselves run in the vector path like any other cell and only the two Newton solves stay per cell.
// PULL: the lattice holds F_{t-1} (the sample point's S_t is pulled).  Launched with programmatic serialization: the blocks
// wait for the step kernel that wrote the lattice, then let the next step kernel start beside them.
template <int Q, typename T, bool PULL>
__global__ void __launch_bounds__(128) k_wallmodel_prepass(const __grid_constant__ StepArgs<T> a) {
  griddep_wait();
  griddep_launch();
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= a.n_wm) return;
  const int cell = a.wm_list[k];
  const int plane = a.nx * a.ny;
  const int z = cell / plane, rem = cell - z * plane;
  const int y = rem / a.nx, x = rem - y * a.nx;
  T ubx, uby, ubz;
  wallmodel_ub<Q, T, PULL>(a, x, y, z, a.cls[cell], ubx, uby, ubz);
  a.wm_ub[cell] = ubx;
  a.wm_ub[a.N + cell] = uby;
  a.wm_ub[2 * a.N + cell] = ubz;
}

// ---- the vectorised step kernel (the hot one) ------------------------------------------------------
// One thread owns V = 16/sizeof(T) consecutive cells of a row (4 floats / 2 doubles): every population
// is moved with one aligned 128-bit load and one aligned 128-bit store per thread.  The populations
// with c_x = +-1 need the row shifted by one element: the thread loads its own aligned vector and takes
// the one missing element from the neighbouring lane with a warp shuffle (row ends: one scalar load).
// Vectors whose V cells are all plain bulk FLUID take this path; a vector that contains a SOLID,
// INLET, OUTLET, WALLMODEL or solid-adjacent cell is processed cell by cell out of line (A7/A8).
// cells per thread: 128-bit access for D3Q19 (4 floats / 2 doubles); D3Q27 takes half of that (64-bit access, still
// whole 32-byte sectors per warp instruction) because 27 x 4 live values leave room for only 8 warps per SM and the
// kernel then stalls on its own latency (ncu, profiles/: 12.5 % occupancy, 0.27 issue slots per cycle).
// The HRR form carries 15 more vectors (u^ of the six neighbours) and a longer collision: half the width again.
template <int Q, typename T, int COLL = COLL_BGK> struct VecOf;
template <> struct VecOf<19, float, COLL_BGK> { static constexpr int V = 4; };
template <> struct VecOf<19, double, COLL_BGK> { static constexpr int V = 2; };
template <> struct VecOf<27, float, COLL_BGK> { static constexpr int V = 2; };
template <> struct VecOf<27, double, COLL_BGK> { static constexpr int V = 1; };
template <> struct VecOf<19, float, COLL_HRR> { static constexpr int V = 2; };
template <> struct VecOf<19, double, COLL_HRR> { static constexpr int V = 1; };
template <> struct VecOf<27, float, COLL_HRR> { static constexpr int V = 2; };
template <> struct VecOf<27, double, COLL_HRR> { static constexpr int V = 1; };

template <bool STREAMING>
__device__ __forceinline__ void ld_vec_t(const float* p, float (&v)[4]) {
  const float4 t = STREAMING ? __ldcs(reinterpret_cast<const float4*>(p)) : __ldg(reinterpret_cast<const float4*>(p));
  v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
}
template <bool STREAMING>
__device__ __forceinline__ void ld_vec_t(const float* p, float (&v)[2]) {
  const float2 t = STREAMING ? __ldcs(reinterpret_cast<const float2*>(p)) : __ldg(reinterpret_cast<const float2*>(p));
  v[0] = t.x; v[1] = t.y;
}
template <bool STREAMING>
__device__ __forceinline__ void ld_vec_t(const float* p, float (&v)[1]) {
  v[0] = STREAMING ? __ldcs(p) : __ldg(p);
}
template <bool STREAMING>
__device__ __forceinline__ void ld_vec_t(const double* p, double (&v)[2]) {
  const double2 t = STREAMING ? __ldcs(reinterpret_cast<const double2*>(p)) : __ldg(reinterpret_cast<const double2*>(p));
  v[0] = t.x; v[1] = t.y;
}
template <bool STREAMING>
__device__ __forceinline__ void ld_vec_t(const double* p, double (&v)[1]) {
  v[0] = STREAMING ? __ldcs(p) : __ldg(p);
}
template <typename T, int V> __device__ __forceinline__ void ld_vec(const T* p, T (&v)[V]) { ld_vec_t<true>(p, v); }
template <typename T, int V> __device__ __forceinline__ void ld_vec_keep(const T* p, T (&v)[V]) { ld_vec_t<false>(p, v); }
__device__ __forceinline__ void st_vec(float* p, const float (&v)[4]) {
  __stcs(reinterpret_cast<float4*>(p), make_float4(v[0], v[1], v[2], v[3]));
}
__device__ __forceinline__ void st_vec(float* p, const float (&v)[2]) { __stcs(reinterpret_cast<float2*>(p), make_float2(v[0], v[1])); }
__device__ __forceinline__ void st_vec(float* p, const float (&v)[1]) { __stcs(p, v[0]); }
__device__ __forceinline__ void st_vec(double* p, const double (&v)[2]) {
  __stcs(reinterpret_cast<double2*>(p), make_double2(v[0], v[1]));
}
__device__ __forceinline__ void st_vec(double* p, const double (&v)[1]) { __stcs(p, v[0]); }
// class bytes of one 32-byte sector of a population row (8 floats / 4 doubles), one aligned load
__device__ __forceinline__ unsigned long long ld_cls_sector(const uint8_t* p, float) { return *reinterpret_cast<const unsigned long long*>(p); }
__device__ __forceinline__ unsigned long long ld_cls_sector(const uint8_t* p, double) { return *reinterpret_cast<const uint32_t*>(p); }
__device__ __forceinline__ void ld_nbmask(const uint32_t* p, uint32_t (&m)[4]) {
  const uint4 t = __ldg(reinterpret_cast<const uint4*>(p));
  m[0] = t.x; m[1] = t.y; m[2] = t.z; m[3] = t.w;
}
__device__ __forceinline__ void ld_nbmask(const uint32_t* p, uint32_t (&m)[2]) {
  const uint2 t = __ldg(reinterpret_cast<const uint2*>(p));
  m[0] = t.x; m[1] = t.y;
}
__device__ __forceinline__ void ld_nbmask(const uint32_t* p, uint32_t (&m)[1]) { m[0] = __ldg(p); }
__host__ __device__ constexpr uint32_t rep_byte(uint32_t b, int n) { return n <= 0 ? 0u : (b | (rep_byte(b, n - 1) << 8)); }

// HRR form, vector path: u^ of the six neighbours of the V cells of a vector.  gu[5 b + {0,1,2,3,4}] = component b at
// rows y+1, y-1, z+1, z-1 and the own row; gl / gr = the elements left / right of the vector (L1 hits: the
// neighbouring lanes load those lines).
template <typename T, int V>
__device__ __forceinline__ void ld_uhat_nb(const T* pu, long long N, int dyp, int dym, int dzp, int dzm, int exl, int exr,
                                           T (&gu)[15][V], T (&gl)[3], T (&gr)[3]) {
#pragma unroll
  for (int b = 0; b < 3; ++b) {
    ld_vec_keep(pu + dyp, gu[5 * b + 0]);
    ld_vec_keep(pu + dym, gu[5 * b + 1]);
    ld_vec_keep(pu + dzp, gu[5 * b + 2]);
    ld_vec_keep(pu + dzm, gu[5 * b + 3]);
    ld_vec_keep(pu, gu[5 * b + 4]);
    gl[b] = __ldg(pu + exl);
    gr[b] = __ldg(pu + exr);
    pu += N;
  }
}

// grid (ceil(nx/V/bx), ceil(ny/by), list_z + nz), block (bx, by), bx a power of two <= 32.
// The first list_z z-slices of the grid do not own a lattice slab: their threads walk the compact list
// of the cells of SPECIAL sectors (A8 wall model; OUTLET cells next to a wall), one cell per thread: the masked
// boundary kernel as a block role of the same launch (scheduled first, overlaps with the row blocks).
// Everything else -- bulk, solid-adjacent (read-side bounce-back), INLET and OUTLET cells -- runs in the vector path.
// WV: kernel variant for special walls, compiled out otherwise (they cost registers): bit 0 = the launch may meet MOVINGWALL cells,
// bit 1 = the lattice has cells with a slip plane code (specular pull in the vector path).
template <int Q, typename T, int MODE, int COLL, int WV>
__device__ __forceinline__ void step_vec_body(const StepArgs<T>& a, double (&acc)[5], const int bz) {   // bz: the block's z index in the (virtual) grid
  constexpr Stencil<Q> L{};
  constexpr int V = VecOf<Q, T, COLL>::V;
  constexpr bool MW = (WV & 1) != 0;       // the launch may meet MOVINGWALL cells
  constexpr bool SLIPV = (WV & 2) != 0;    // the lattice has cells with a slip plane code
  constexpr bool HRR = (COLL == COLL_HRR) && mode_collides(MODE);
  constexpr int SV = 32 / static_cast<int>(sizeof(T));      // cells per 32-byte sector
  constexpr int LG = 128 / (V * static_cast<int>(sizeof(T)));  // lanes per 128-byte line
  constexpr unsigned FULL = 0xffffffffu;
  constexpr bool PULL = mode_pulls(MODE);
  const int tx = threadIdx.x;
  if (bz < a.list_z) {
    const long long blk = (static_cast<long long>(bz) * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    const long long k = blk * (blockDim.x * blockDim.y) + threadIdx.y * blockDim.x + tx;
    if (k < a.n_list) {
      const int cell = a.list[k];
      const uint8_t c = a.cls[cell];
      const int plane = a.nx * a.ny;
      const int cz = cell / plane, rem = cell - cz * plane;
      if (cz < a.zi0 || cz >= a.zi1) return;   // a cell of a ghost slice: its values come from the neighbouring sub-domain
      if (is_wall(c)) {                    // wall sector-mate: zeros keep the sector whole
        solid_cell_any<Q, T, MODE>(a, cell);
      } else {
        const int cy = rem / a.nx, cx = rem - cy * a.nx;
        step_cell_any<Q, T, MODE, COLL>(a, cx, cy, cz, c, acc);
      }
    }
    return;
  }
  const int lane = (threadIdx.y * blockDim.x + tx) & 31;
  const int nvec = a.nx / V;
  const int qx = blockIdx.x * blockDim.x + tx;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  // serpentine sweep: a launch that runs against the direction of the previous one starts on the slices that launch wrote (or read)
  // last, which are still in the 126 MB L2
  const int kz = bz - a.list_z;
  const int z = a.z0 + (a.z_reverse ? (a.nzs - 1 - kz) : kz);
  const bool active = (qx < nvec) && (y < a.ny);
  const int x0 = qx * V;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const long long N = a.N;
  const long long row = active ? (static_cast<long long>(z) * ny + y) * nx : 0;
  const long long self = row + (active ? x0 : 0);
  // class bytes of the vector's 32-byte sector: a sector with a SPECIAL cell belongs to the list blocks
  unsigned long long secw = ~0ull;
  if (active) secw = ld_cls_sector(a.cls + row + (x0 & ~(SV - 1)), T(0));
  constexpr unsigned long long SPECIAL_ALL = (SV == 8) ? 0x8080808080808080ull : 0x80808080ull;
  constexpr uint32_t VMASK = rep_byte(0xffu, V);
  constexpr uint32_t ADJ_ALL = rep_byte(0x40u, V);
  const uint32_t clsw = static_cast<uint32_t>(secw >> (8 * (x0 & (SV - 1)))) & VMASK;
  unsigned wall_bits = 0;             // which cells of the vector are walls (bit v)
#pragma unroll
  for (int v = 0; v < V; ++v) wall_bits |= is_wall(static_cast<int>(clsw >> (8 * v))) ? (1u << v) : 0u;
  const bool all_solid = !active || (wall_bits == ((1u << V) - 1u));
  const bool special = (secw & SPECIAL_ALL) != 0;
  // an all-SOLID vector whose 128-byte line holds a non-SOLID vector stores zeros, so that the line is written whole
  const unsigned live_lanes = __ballot_sync(FULL, active && !all_solid);
  const unsigned group = (LG >= 32) ? FULL : (((1u << (LG & 31)) - 1u) << (lane & ~(LG - 1)));
  // (the u^ pass writes every wall vector: 12 bytes per cell, and the FD stencil may read any of them)
  const bool zero_fill = !mode_diag(MODE) && active && all_solid && !special && (mode_uhat(MODE) || ((live_lanes & group) != 0u));
  const bool mine = active && !all_solid && !special;       // this thread computes and stores the vector
  const bool doload = active && !all_solid;                 // neighbours may need its lanes' values
  // which cells of the vector are SOLID (bit v)
  const unsigned solid_bits = wall_bits;
  const bool adj = mine && PULL && ((clsw & ADJ_ALL) != 0);
  // INLET (only ever at x = 0) / OUTLET (only ever at x = nx-1; SPECIAL if next to a wall) cells
  const bool inlet0 = mine && (x0 == 0) && ((clsw & CLS_TYPE) == T_INLET);
  const bool outletN = mine && (qx == nvec - 1) && (((clsw >> (8 * (V - 1))) & CLS_TYPE) == T_OUTLET);
  const bool poutN = mine && (qx == nvec - 1) && (((clsw >> (8 * (V - 1))) & CLS_TYPE) == T_POUTLET);
  // WALLMODEL cells of the vector (bit v): their u^B comes from the pre-pass (A8); sigma = 0 there in the HRR form (l.131)
  unsigned wm_bits = 0;
  if (mode_hlbm(MODE) && a.wm_enable) {
#pragma unroll
    for (int v = 0; v < V; ++v) wm_bits |= (((clsw >> (8 * v)) & CLS_TYPE) == T_WM) ? (1u << v) : 0u;
  }
  if (!mine) wm_bits = 0;

  T f[Q][V];
  T d[V];
  uint32_t nbm[V];
#pragma unroll
  for (int v = 0; v < V; ++v) { d[v] = T(0); nbm[v] = 0u; }
  // porosity vector and the per-cell SOLID-neighbour masks of a solid-adjacent vector (one aligned 128 / 64-bit load each), issued
  // BEFORE the population loads (issued after them -- to take the wait for the class bytes out of the chain class bytes -> masks
  // -> populations -> own-cell loads that ncu shows on the ADJ warps of config 4 -- every workload ran 1 - 14 % slower: measured,
  // DESIGN.md 5.2)
  if (mode_hlbm(MODE) && mine && a.d != nullptr) {
    T dv[V];
    ld_vec_keep(a.d + self, dv);
#pragma unroll
    for (int v = 0; v < V; ++v) d[v] = dv[v];
  }
  if (adj) ld_nbmask(a.nbmask + self, nbm);
  // row offsets of the (dy, dz) neighbour rows; all deltas fit 32 bits because N < 2^31
  const int ym = (y == 0) ? ny - 1 : y - 1, yp = (y >= ny - 1) ? 0 : y + 1;
  const int zm = (z == 0) ? nz - 1 : z - 1, zp = (z == nz - 1) ? 0 : z + 1;
  const int dym = (ym - y) * nx, dyp = (yp - y) * nx;
  const int plane = nx * ny;
  const int dzm = (zm - z) * plane, dzp = (zp - z) * plane;
  const int xl = (x0 == 0) ? nx - 1 : x0 - 1;            // element left of the vector (periodic)
  const int xr = (x0 + V >= nx) ? 0 : x0 + V;            // element right of the vector
  const int exl = xl - x0, exr = xr - x0;                // relative to the vector start
  T gu[HRR ? 15 : 1][V], gl[3], gr[3];      // HRR form: u^ of the neighbours (FD strain, Eq. 10)
  if (!PULL) {
    if (mine) {
#pragma unroll
      for (int i = 0; i < Q; ++i) ld_vec(a.fin + i * N + self, f[i]);
    }
    if constexpr (HRR) {
      if (mine) ld_uhat_nb<T, V>(a.uhat + self, N, dyp, dym, dzp, dzm, exl, exr, gu, gl, gr);
    }
  } else {
    // phase 1: issue every load before anything consumes one (in-order issue: a shuffle placed right
    // after its load would serialise the loads).  One running pointer per population (+N each).
    T e[Q];   // the one element a shifted row needs from outside the warp / row (edge lanes only)
    // SLIPV variant: slip plane code of the vector (its non-wall cells agree: k_slip_uniform): the populations that would come out of
    // the slip plane are pulled from the vector's own plane and the mirrored slot instead (specular reflection, reading G37)
    int sc = 0;
    if (SLIPV) {
#pragma unroll
      for (int v = 0; v < V; ++v) {
        const int b = static_cast<int>(clsw >> (8 * v)) & 0xff;
        if (!is_wall(b) && (b & CLS_TYPE) != T_WM) sc |= (b >> CLS_NORMAL_SHIFT) & 7;
      }
      if (!active) sc = 0;
    }
    auto issue_loads = [&](auto slip_tag, const bool ld, const bool el, const bool er) {
      constexpr bool SL = decltype(slip_tag)::value;         // this warp pulls under a slip plane code
      const T* pself = a.fin + self;
      constexpr Mirror<Q> MR{};
#pragma unroll
      for (int i = 0; i < Q; ++i) {
        long long offy = static_cast<long long>((L.c[i][1] == 0) ? 0 : ((L.c[i][1] == 1) ? dym : dyp));
        long long offz = static_cast<long long>((L.c[i][2] == 0) ? 0 : ((L.c[i][2] == 1) ? dzm : dzp));
        long long slot = 0;
        if (SL && sc != 0) {
          if (L.c[i][1] != 0 && sc == ((L.c[i][1] == 1) ? 2 : 3)) { offy = 0; slot = static_cast<long long>(MR.my[i] - i) * N; }
          else if (L.c[i][2] != 0 && sc == ((L.c[i][2] == 1) ? 4 : 5)) { offz = 0; slot = static_cast<long long>(MR.mz[i] - i) * N; }
        }
        const T* src = pself + (offy + offz + slot);           // source row, at the vector's x
        pself += N;
#pragma unroll
        for (int v = 0; v < V; ++v) f[i][v] = T(0);
        e[i] = T(0);
        if (ld) ld_vec(src, f[i]);
        if (L.c[i][0] == 1 && el) e[i] = __ldg(src + exl);
        if (L.c[i][0] == -1 && er) e[i] = __ldg(src + exr);
      }
    };
    // a vector that is SOLID throughout loads nothing, but the rows its neighbour pulls from (y -+ 1, z -+ 1) may be
    // fluid at its end cells: that neighbour fetches the one element itself, like a lane at the edge of the warp
    // (SLIPV variant: the same where the neighbouring vector pulls under another slip plane code: its elements come from other rows)
    bool solid_l, solid_r;
    if constexpr (SLIPV) {
      const int nb_key = (all_solid ? 8 : 0) | sc;
      const int key_l = __shfl_up_sync(FULL, nb_key, 1), key_r = __shfl_down_sync(FULL, nb_key, 1);
      solid_l = (key_l & 8) != 0 || (key_l & 7) != sc;
      solid_r = (key_r & 8) != 0 || (key_r & 7) != sc;
    } else {
      solid_l = __shfl_up_sync(FULL, all_solid ? 1 : 0, 1) != 0;
      solid_r = __shfl_down_sync(FULL, all_solid ? 1 : 0, 1) != 0;
    }
    const bool edge_l = doload && ((lane == 0) || (tx == 0) || solid_l);
    const bool edge_r = doload && ((lane == 31) || (tx == static_cast<int>(blockDim.x) - 1) || (qx == nvec - 1) || solid_r);
    // (a warp-uniform branch: the warps of the bulk run the plain load sequence, without the slip arithmetic)
    if (SLIPV && __any_sync(FULL, sc != 0)) issue_loads(std::true_type{}, doload, edge_l, edge_r);
    else issue_loads(std::false_type{}, doload, edge_l, edge_r);
    if constexpr (HRR) {
      if (mine) ld_uhat_nb<T, V>(a.uhat + self, N, dyp, dym, dzp, dzm, exl, exr, gu, gl, gr);
    }
    // phase 2: realign the rows with c_x = +-1 by one element through the neighbouring lane
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      if (L.c[i][0] == 1) {                                  // source x - 1: shift right by one
        T nb = __shfl_up_sync(FULL, f[i][V - 1], 1);
        if (edge_l) nb = e[i];
#pragma unroll
        for (int v = V - 1; v > 0; --v) f[i][v] = f[i][v - 1];
        f[i][0] = nb;
      } else if (L.c[i][0] == -1) {                          // source x + 1: shift left by one
        T nb = __shfl_down_sync(FULL, f[i][0], 1);
        if (edge_r) nb = e[i];
        if (outletN) nb = f[i][V - 1];                       // R7: ghost plane nx := plane nx-1
#pragma unroll
        for (int v = 0; v < V - 1; ++v) f[i][v] = f[i][v + 1];
        f[i][V - 1] = nb;
      }
    }
  }
  T* pout = mode_uhat(MODE) ? a.uhat + self : a.fout + self;   // (unused by the A9 modes)
  if (zero_fill) {
    T zero[V];
#pragma unroll
    for (int v = 0; v < V; ++v) zero[v] = T(0);
    if constexpr (mode_uhat(MODE)) {                         // u^ of wall cells: 0, or u_w on MOVINGWALL cells
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        T uw[V];
#pragma unroll
        for (int v = 0; v < V; ++v) uw[v] = (((clsw >> (8 * v)) & CLS_TYPE) == T_MOVING) ? a.u_wall[b] : T(0);
        st_vec(pout, uw);
        pout += N;
      }
    } else {
#pragma unroll
      for (int i = 0; i < Q; ++i) {
        st_vec(pout, zero);
        pout += N;
      }
    }
    return;
  }
  if (!mine) return;   // SOLID throughout in an all-SOLID line, or a SPECIAL sector (list blocks)

  if (adj) {
    // R5, read side: where the source x - c_i of population i is SOLID (nbmask bit j = opp(i): x + c_j is SOLID), the
    // pulled value is replaced by the cell's own F_j(x).  Predicated element loads straight into the population
    // registers: no extra registers, and all of them are in flight together (one round trip).
    const T* pown = a.fin + self;
#pragma unroll
    for (int j = 1; j < Q; ++j) {
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (nbm[v] & (1u << j)) f[L.opp[j]][v] = __ldg(pown + static_cast<long long>(j) * N + v);
    }
    // moving wall (G33): MOVINGWALL cells exist only on the plane z = nz-1, so only directions towards that plane can meet one
    // (block-uniform test); the neighbour's class byte decides.  (Cells next to a SLIPWALL are SPECIAL: list blocks.)
    if (MW && (z >= nz - 2 || z == 0)) {
#pragma unroll
      for (int j = 1; j < Q; ++j) {
        const int zn = z + L.c[j][2];
        if (((zn < 0) ? zn + nz : ((zn >= nz) ? zn - nz : zn)) != nz - 1) continue;
        const long long off = static_cast<long long>((L.c[j][1] == 0) ? 0 : ((L.c[j][1] == 1) ? dyp : dym)) +
                              static_cast<long long>((L.c[j][2] == 0) ? 0 : ((L.c[j][2] == 1) ? dzp : dzm));
        const uint8_t* pc = a.cls + self + off;
#pragma unroll
        for (int v = 0; v < V; ++v) {
          if (nbm[v] & (1u << j)) {
            int ex = v + L.c[j][0];
            if (L.c[j][0] == -1 && v == 0) ex = exl;
            if (L.c[j][0] == 1 && v == V - 1) ex = exr;
            if ((pc[ex] & CLS_TYPE) == T_MOVING) f[L.opp[j]][v] += moving_wall_term<Q, T>(L.opp[j], a.u_wall);
          }
        }
      }
    }
  }
  if (PULL && inlet0) {                                      // R6 on the x = 0 cell of the row
    T fc[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) fc[i] = f[i][0];
    T uwx, uwy, uwz;
    inlet_velocity<T>(a, y, z, uwx, uwy, uwz);
    inlet_fixup<Q, T>(fc, uwx, uwy, uwz);
#pragma unroll
    for (int i = 0; i < Q; ++i) f[i][0] = fc[i];
  }
  if (PULL && poutN) {                                       // G36 on the x = nx-1 cell of the row
    T fc[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) fc[i] = f[i][V - 1];
    pressure_fixup<Q, T>(fc, a.rho_out);
#pragma unroll
    for (int i = 0; i < Q; ++i) f[i][V - 1] = fc[i];
  }
  if constexpr (mode_diag(MODE)) {                            // A9: raw moments of S_t (l.97, G19)
    T mr[V], mu[3][V], sr = T(0), sj[3] = {T(0), T(0), T(0)}, se = T(0);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      T fc[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) fc[i] = f[i][v];
      T rho, jx, jy, jz;
      cell_moments<Q, T>(fc, rho, jx, jy, jz);
      const bool wall = (solid_bits >> v) & 1u;
      if constexpr (mode_moments(MODE)) {
        const T ir = rcp_(wall ? T(1) : rho);
        mr[v] = wall ? T(0) : rho;              // wall cells of a mixed vector: k_solid_moments writes their own values afterwards
        mu[0][v] = wall ? T(0) : jx * ir;
        mu[1][v] = wall ? T(0) : jy * ir;
        mu[2][v] = wall ? T(0) : jz * ir;
      } else if (!wall) {
        sr += rho;  sj[0] += jx;  sj[1] += jy;  sj[2] += jz;
        se += T(0.5) * (jx * jx + jy * jy + jz * jz) * rcp_(rho);
      }
    }
    if constexpr (mode_moments(MODE)) {
      if (a.mom_rho != nullptr) st_vec(a.mom_rho + self, mr);
      if (a.mom_u != nullptr) {
#pragma unroll
        for (int b = 0; b < 3; ++b) st_vec(a.mom_u + b * N + self, mu[b]);
      }
    } else {
      acc[0] += static_cast<double>(sr);  acc[1] += static_cast<double>(sj[0]);  acc[2] += static_cast<double>(sj[1]);
      acc[3] += static_cast<double>(sj[2]);  acc[4] += static_cast<double>(se);
    }
    return;
  }
  if (wm_bits != 0u && a.wm_ub != nullptr && !a.pdl_wait_all) griddep_wait();   // u^B of this level: the pre-pass may still be running
  if constexpr (mode_uhat(MODE)) {                            // first pass of the HRR form: u^(x,t) (Eq. 12), SOLID cells 0
    T uo[3][V];
#pragma unroll
    for (int v = 0; v < V; ++v) {
      T fc[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) fc[i] = f[i][v];
      T ubx, uby, ubz;
      if ((wm_bits >> v) & 1u) {
        ubx = __ldcg(a.wm_ub + self + v);  uby = __ldcg(a.wm_ub + N + self + v);  ubz = __ldcg(a.wm_ub + 2 * N + self + v);
      } else {
        body_velocity<T>(a.ub == nullptr ? nullptr : a.ub + self + v, N, d[v], ubx, uby, ubz);
      }
      uhat_of<Q, T>(fc, d[v], ubx, uby, ubz, uo[0][v], uo[1][v], uo[2][v]);
      if (solid_bits & (1u << v)) {
        const bool mv = ((clsw >> (8 * v)) & CLS_TYPE) == T_MOVING;
        uo[0][v] = mv ? a.u_wall[0] : T(0);
        uo[1][v] = mv ? a.u_wall[1] : T(0);
        uo[2][v] = mv ? a.u_wall[2] : T(0);
      }
    }
#pragma unroll
    for (int b = 0; b < 3; ++b) {
      st_vec(pout, uo[b]);
      pout += N;
    }
    return;
  }
  if constexpr (mode_collides(MODE)) {
#pragma unroll
    for (int v = 0; v < V; ++v) {
      T fc[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) fc[i] = f[i][v];
      T ubx, uby, ubz;
      const bool wmc = (wm_bits >> v) & 1u;
      if (wmc) {
        ubx = __ldcg(a.wm_ub + self + v);  uby = __ldcg(a.wm_ub + N + self + v);  ubz = __ldcg(a.wm_ub + 2 * N + self + v);
      } else {
        body_velocity<T>(a.ub == nullptr ? nullptr : a.ub + self + v, N, d[v], ubx, uby, ubz);
      }
      if constexpr (HRR) {
        T D[3][3];   // D[a][b] = u^_b(x + e_a) - u^_b(x - e_a); G32: the planes beyond INLET / OUTLET copy those planes
#pragma unroll
        for (int b = 0; b < 3; ++b) {
          T left = (v > 0) ? gu[5 * b + 4][v > 0 ? v - 1 : 0] : gl[b];
          T right = (v < V - 1) ? gu[5 * b + 4][v < V - 1 ? v + 1 : 0] : gr[b];
          if (v == 0 && inlet0) left = gu[5 * b + 4][0];
          if (v == V - 1 && (outletN || poutN)) right = gu[5 * b + 4][V - 1];
          D[0][b] = right - left;
          D[1][b] = gu[5 * b + 0][v] - gu[5 * b + 1][v];
          D[2][b] = gu[5 * b + 2][v] - gu[5 * b + 3][v];
        }
        const T S[6] = {T(0.5) * D[0][0], T(0.5) * D[1][1], T(0.5) * D[2][2], T(0.25) * (D[0][1] + D[1][0]),
                        T(0.25) * (D[0][2] + D[2][0]), T(0.25) * (D[1][2] + D[2][1])};
        T uox, uoy, uoz;
        collide_cell_hrr<Q, T>(fc, d[v], ubx, uby, ubz, tau0_at<T>(a, x0 + v), a.smago_k, wmc ? T(0) : a.sigma, S, uox, uoy, uoz);   // sigma = 0: l.131
        if (a.uhat_out != nullptr) {         // G41: this level's u^ is the next step's history (wall cells of the vector: the wall's velocity)
          const bool wl = (solid_bits >> v) & 1u;
          const bool mv = ((clsw >> (8 * v)) & CLS_TYPE) == T_MOVING;
          T* po = a.uhat_out + self + v;
          po[0] = wl ? (mv ? a.u_wall[0] : T(0)) : uox;
          po[N] = wl ? (mv ? a.u_wall[1] : T(0)) : uoy;
          po[2 * N] = wl ? (mv ? a.u_wall[2] : T(0)) : uoz;
        }
      } else {
        collide_cell<Q, T>(fc, d[v], ubx, uby, ubz, tau0_at<T>(a, x0 + v), a.smago_k);
      }
#pragma unroll
      for (int i = 0; i < Q; ++i) f[i][v] = fc[i];
    }
  }
  if (solid_bits != 0) {   // SOLID cells inside the vector: their slots are never read; zeros, so that the store is whole
#pragma unroll
    for (int i = 0; i < Q; ++i)
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (solid_bits & (1u << v)) f[i][v] = T(0);
  }
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    st_vec(pout, f[i]);
    pout += N;
  }
}

template <int Q, typename T, int MODE, int COLL, int WV>
__global__ void __launch_bounds__(256, 2) k_step_vec(const __grid_constant__ StepArgs<T> a) {
  if (a.pdl_wait_all) griddep_wait();      // the preceding kernel wrote this kernel's input (see StepArgs)
  griddep_launch();
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if constexpr (mode_totals(MODE)) {
    // the blocks walk the z-slices with stride gridDim.z, so that one block-level reduction (shuffle trees, atomics, ticket)
    // serves many vectors per thread
    for (int bz = blockIdx.z; bz < a.list_z + a.nzs; bz += gridDim.z) step_vec_body<Q, T, MODE, COLL, WV>(a, acc, bz);
    reduce_totals(acc, a.tot_slots, a.tot_nslots, a.tot_ticket, a.tot_out);
  } else {
    step_vec_body<Q, T, MODE, COLL, WV>(a, acc, static_cast<int>(blockIdx.z));
  }
}

// ---- in-place propagation, AA pattern (one lattice) -- the propagation bake-off of DESIGN.md section 4 --------------------
// Lattices without a single wall / inlet / outlet / wall-model cell only (fully periodic bulk), BGK form.  Two alternating
// kernels on ONE array a[Q][N]:
//   even step (array holds S_t as a[i][x] = f_i(x,t)):           read a[i][x], collide, write F_i(x) to a[opp(i)][x]  -- all local;
//   odd step  (array holds F_t with swapped slots):               read S_{t+1,i}(x) = a[opp(i)][x - c_i], collide, write
//             F_{t+1,j}(x) to a[j][x + c_j], the slot and cell the value of direction opp(j) was read from: afterwards the
//             array holds S_{t+2} in the plain layout.
// Every location is read and written by the same cell, so one array suffices.  The vector form keeps all global accesses
// aligned: the thread that loads the aligned vector (slot, row, x0) is the one that stores it; the c_x = +-1 shift is a warp
// shuffle on the way in and on the way out, and at warp edges one scalar load on the way in and a shared-memory hand-over on
// the way out.  A block covers whole rows in x, so the one __syncthreads between the load phase and the store phase orders
// the edge loads of a thread before the stores of its x-neighbours.
template <typename T>
struct AAArgs {
  T* __restrict__ a;               // [Q][N], updated in place
  const T* __restrict__ d;         // porosity or nullptr
  const T* __restrict__ ub;        // solid velocity [3][N] or nullptr
  const uint8_t* __restrict__ cls;      // class bytes (WALLS variants)
  const uint32_t* __restrict__ nbmask;  // SOLID-neighbour masks (WALLS variants)
  int nx, ny, nz;
  long long N;
  T tau0, smago_k, fringe_k;
  int fringe_x0;
};

// collide the cells of a vector whose bit in `skip` is clear (wall cells keep what they hold)
template <int Q, typename T>
__device__ __forceinline__ void aa_collide_vec(const AAArgs<T>& a, long long self, int x0, T (&f)[Q][VecOf<Q, T, COLL_BGK>::V],
                                               unsigned skip = 0u) {
  constexpr int V = VecOf<Q, T, COLL_BGK>::V;
  T d[V];
#pragma unroll
  for (int v = 0; v < V; ++v) d[v] = T(0);
  if (a.d != nullptr) ld_vec_keep(a.d + self, d);
#pragma unroll
  for (int v = 0; v < V; ++v) {
    if ((skip >> v) & 1u) continue;
    T fc[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) fc[i] = f[i][v];
    T ubx, uby, ubz;
    body_velocity<T>(a.ub == nullptr ? nullptr : a.ub + self + v, a.N, d[v], ubx, uby, ubz);
    const int xd = (x0 + v > a.fringe_x0) ? x0 + v - a.fringe_x0 : 0;
    collide_cell<Q, T>(fc, d[v], ubx, uby, ubz, a.tau0 + a.fringe_k * static_cast<T>(xd * xd), a.smago_k);
#pragma unroll
    for (int i = 0; i < Q; ++i) f[i][v] = fc[i];
  }
}

// which cells of the vector at `self` are walls (bit v), from their class bytes
template <typename T, int V>
__device__ __forceinline__ unsigned aa_wall_bits(const uint8_t* __restrict__ cls, long long self) {
  unsigned w = 0;
#pragma unroll
  for (int v = 0; v < V; ++v) w |= is_wall(cls[self + v]) ? (1u << v) : 0u;
  return w;
}

// WALLS: the lattice has SOLID cells (halfway bounce-back, R5) and nothing else besides plain fluid.  In the AA pattern the
// bounce-back link of a cell needs the cell's OWN slots only: the even step is purely local anyway, and in the odd step the
// population i whose source x - c_i is a wall is read from a[i][x] (where the even step left F_opp(i)(x)) and the population j
// whose target x + c_j is a wall is written to a[opp(j)][x] -- the same location.  Wall cells' slots are never consumed, so whole
// vectors are stored whatever their wall lanes hold; their own (inert) values live in the side buffer like in the two-lattice scheme.
// grid (ceil(nvec / bx), ceil(ny / by), nz), block (bx, by)
template <int Q, typename T, bool WALLS>
__global__ void __launch_bounds__(256, 2) k_aa_even(const __grid_constant__ AAArgs<T> a) {
  constexpr Stencil<Q> L{};
  constexpr int V = VecOf<Q, T, COLL_BGK>::V;
  const int qx = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (qx >= a.nx / V || y >= a.ny) return;
  const int x0 = qx * V;
  const long long self = (static_cast<long long>(z) * a.ny + y) * a.nx + x0;
  unsigned walls = 0;
  if (WALLS) {
    walls = aa_wall_bits<T, V>(a.cls, self);
    if (walls == ((1u << V) - 1u)) return;               // walls throughout: nothing to do, nothing to move
  }
  T f[Q][V];
  T* p = a.a + self;
#pragma unroll
  for (int i = 0; i < Q; ++i) ld_vec(p + i * a.N, f[i]);
  aa_collide_vec<Q, T>(a, self, x0, f, walls);
#pragma unroll
  for (int i = 0; i < Q; ++i) st_vec(p + L.opp[i] * a.N, f[i]);
}

// grid (1, ceil(ny / by), nz), block (nvec, by): whole rows in x (nvec = nx / V a multiple of 32, nvec * by <= 256)
template <int Q, typename T, bool WALLS>
__global__ void __launch_bounds__(256, 2) k_aa_odd(const __grid_constant__ AAArgs<T> a) {
  constexpr Stencil<Q> L{};
  constexpr int V = VecOf<Q, T, COLL_BGK>::V;
  constexpr unsigned FULL = 0xffffffffu;
  constexpr unsigned VALL = (1u << V) - 1u;
  constexpr int NXP = (Q == 19) ? 5 : 9;                  // populations with c_x = +1 (and as many with c_x = -1)
  __shared__ T edge_r[NXP][8];                           // F_j of the LAST cell of every warp, j with c_x = +1 (goes to the next warp)
  __shared__ T edge_l[NXP][8];                           // F_j of the FIRST cell of every warp, j with c_x = -1 (goes to the previous warp)
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int lane = tx & 31;
  const int wrow = blockDim.x >> 5;                       // warps per row
  const int warp = ty * wrow + (tx >> 5);                 // warp of the block (rows are whole warps)
  const int y = blockIdx.y * blockDim.y + ty;
  const int z = blockIdx.z;
  const bool active = y < a.ny;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const long long N = a.N;
  const int x0 = tx * V;
  const int yy = active ? y : 0;
  const long long self = (static_cast<long long>(z) * ny + yy) * nx + x0;
  const int ym = (yy == 0) ? ny - 1 : yy - 1, yp = (yy >= ny - 1) ? 0 : yy + 1;
  const int zm = (z == 0) ? nz - 1 : z - 1, zp = (z == nz - 1) ? 0 : z + 1;
  const int dym = (ym - yy) * nx, dyp = (yp - yy) * nx;
  const int plane = nx * ny;
  const int dzm = (zm - z) * plane, dzp = (zp - z) * plane;
  const int exl = ((x0 == 0) ? nx - 1 : x0 - 1) - x0, exr = ((x0 + V >= nx) ? 0 : x0 + V) - x0;
  // WALLS: which own cells are walls / solid-adjacent, and whether the cells left and right of the vector are fluid (they are the
  // sources of the edge elements this thread stores)
  unsigned walls = 0, adjb = 0;
  bool fluid_l = true, fluid_r = true;
  if (WALLS) {
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const uint8_t c = a.cls[self + v];
      walls |= is_wall(c) ? (1u << v) : 0u;
      adjb |= (c & CLS_ADJ) ? (1u << v) : 0u;
    }
    fluid_l = !is_wall(a.cls[self + exl]);
    fluid_r = !is_wall(a.cls[self + exr]);
    if (!active) { walls = VALL; adjb = 0; fluid_l = fluid_r = false; }
  }
  const bool ld = active && walls != VALL;               // a vector of walls throughout loads nothing: nobody consumes its values
  // the element a shifted row needs from outside the warp -- or from a neighbouring lane that holds walls throughout and therefore
  // loads nothing (its ROWS of sources may well be fluid): fetched by the lane itself
  bool own_l = ld && lane == 0, own_r = ld && lane == 31;
  if (WALLS) {
    const bool wv_l = __shfl_up_sync(FULL, ld ? 0 : 1, 1) != 0, wv_r = __shfl_down_sync(FULL, ld ? 0 : 1, 1) != 0;
    own_l = ld && (lane == 0 || wv_l);
    own_r = ld && (lane == 31 || wv_r);
  }
  uint32_t nbm[V];
#pragma unroll
  for (int v = 0; v < V; ++v) nbm[v] = 0u;
  if (WALLS && adjb != 0u) ld_nbmask(a.nbmask + self, nbm);
  T f[Q][V], e[Q];
  // load phase: S_{t+1,i}(x) = a[opp(i)][x - c_i]: the aligned vector of the source row, realigned by one element for c_x = +-1
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const long long off = static_cast<long long>((L.c[i][1] == 0) ? 0 : ((L.c[i][1] == 1) ? dym : dyp)) +
                          static_cast<long long>((L.c[i][2] == 0) ? 0 : ((L.c[i][2] == 1) ? dzm : dzp));
    const T* src = a.a + L.opp[i] * N + self + off;
#pragma unroll
    for (int v = 0; v < V; ++v) f[i][v] = T(0);
    e[i] = T(0);
    if (ld) ld_vec(src, f[i]);
    if (L.c[i][0] == 1 && own_l) e[i] = __ldg(src + exl);
    if (L.c[i][0] == -1 && own_r) e[i] = __ldg(src + exr);
  }
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    if (L.c[i][0] == 1) {
      T nb = __shfl_up_sync(FULL, f[i][V - 1], 1);
      if (own_l) nb = e[i];
#pragma unroll
      for (int v = V - 1; v > 0; --v) f[i][v] = f[i][v - 1];
      f[i][0] = nb;
    } else if (L.c[i][0] == -1) {
      T nb = __shfl_down_sync(FULL, f[i][0], 1);
      if (own_r) nb = e[i];
#pragma unroll
      for (int v = 0; v < V - 1; ++v) f[i][v] = f[i][v + 1];
      f[i][V - 1] = nb;
    }
  }
  if (WALLS && adjb != 0u) {
    // R5 in the AA pattern: the population i = opp(j) whose source x + c_j is a wall is the cell's own a[i][x]
    T* pown = a.a + self;
#pragma unroll
    for (int j = 1; j < Q; ++j) {
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (nbm[v] & (1u << j)) f[L.opp[j]][v] = __ldg(pown + static_cast<long long>(L.opp[j]) * N + v);
    }
  }
  if (ld) aa_collide_vec<Q, T>(a, self, x0, f, walls);
  // store phase: F_j(x) goes to a[j][x + c_j]; the aligned vector (j, row + (c_y, c_z), x0) takes F_j(x - c_x)
  {
    int kp = 0, km = 0;
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      if (L.c[j][0] == 1) { if (lane == 31) edge_r[kp][warp] = f[j][V - 1]; ++kp; }
      else if (L.c[j][0] == -1) { if (lane == 0) edge_l[km][warp] = f[j][0]; ++km; }
    }
  }
  __syncthreads();                                       // every load of the block is done; the edge values are in place
  {
    const int wl = ty * wrow + (((tx >> 5) == 0) ? wrow - 1 : (tx >> 5) - 1);          // previous / next warp of the row (periodic)
    const int wr = ty * wrow + (((tx >> 5) == wrow - 1) ? 0 : (tx >> 5) + 1);
    // WALLS: an element is stored only if the cell it comes from (this row, shifted by c_x) is fluid: what would come out of a wall
    // cell must not overwrite the slot a fluid cell keeps its bounced population in
    const unsigned src0 = active ? (~walls & VALL) : 0u;
    const unsigned srcp = ((src0 << 1) | (fluid_l ? 1u : 0u)) & VALL;                  // c_x = +1: element e comes from cell e - 1
    const unsigned srcm = (src0 >> 1) | (fluid_r ? (1u << (V - 1)) : 0u);              // c_x = -1: element e comes from cell e + 1
    int kp = 0, km = 0;
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      const long long off = static_cast<long long>((L.c[j][1] == 0) ? 0 : ((L.c[j][1] == 1) ? dyp : dym)) +
                            static_cast<long long>((L.c[j][2] == 0) ? 0 : ((L.c[j][2] == 1) ? dzp : dzm));
      T* dst = a.a + j * N + self + off;
      T o[V];
      unsigned ok = src0;
      if (L.c[j][0] == 1) {
        T nb = __shfl_up_sync(FULL, f[j][V - 1], 1);
        if (lane == 0) nb = edge_r[kp][wl];
        ++kp;
#pragma unroll
        for (int v = V - 1; v > 0; --v) o[v] = f[j][v - 1];
        o[0] = nb;
        ok = srcp;
      } else if (L.c[j][0] == -1) {
        T nb = __shfl_down_sync(FULL, f[j][0], 1);
        if (lane == 31) nb = edge_l[km][wr];
        ++km;
#pragma unroll
        for (int v = 0; v < V - 1; ++v) o[v] = f[j][v + 1];
        o[V - 1] = nb;
        ok = srcm;
      } else {
#pragma unroll
        for (int v = 0; v < V; ++v) o[v] = f[j][v];
      }
      if (!WALLS) {
        if (active) st_vec(dst, o);
      } else if (ok == VALL) {
        st_vec(dst, o);
      } else if (ok != 0u) {
#pragma unroll
        for (int v = 0; v < V; ++v)
          if ((ok >> v) & 1u) dst[v] = o[v];
      }
    }
    if (WALLS && adjb != 0u) {
      // the population j whose target x + c_j is a wall stays in the cell: a[opp(j)][x] (where the next even step reads f_opp(j))
      T* pown = a.a + self;
#pragma unroll
      for (int j = 1; j < Q; ++j) {
#pragma unroll
        for (int v = 0; v < V; ++v)
          if (nbm[v] & (1u << j)) pown[static_cast<long long>(L.opp[j]) * N + v] = f[j][v];
      }
    }
  }
}

// the state S_{t+1} out of an array that holds F_t with swapped slots: out[i][x] = a[opp(i)][x - c_i], or the cell's own a[i][x]
// where x - c_i is a wall (materialisation; off the timed path: one thread per cell; wall cells are left to the side buffer)
template <int Q, typename T>
__global__ void __launch_bounds__(256) k_aa_unswap(const T* __restrict__ a, T* __restrict__ out, int nx, int ny, int nz, long long N,
                                                   const uint8_t* __restrict__ cls, const uint32_t* __restrict__ nbmask) {
  constexpr Stencil<Q> L{};
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= nx || y >= ny) return;
  const long long self = cell_index(x, y, z, nx, ny);
  const uint8_t c = cls[self];
  if (is_wall(c)) return;
  const uint32_t nbm = (c & CLS_ADJ) ? nbmask[self] : 0u;
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    int sx = x - L.c[i][0], sy = y - L.c[i][1], sz = z - L.c[i][2];
    sx = (sx < 0) ? sx + nx : ((sx >= nx) ? sx - nx : sx);
    sy = (sy < 0) ? sy + ny : ((sy >= ny) ? sy - ny : sy);
    sz = (sz < 0) ? sz + nz : ((sz >= nz) ? sz - nz : sz);
    const bool own = (i > 0) && ((nbm >> L.opp[i]) & 1u);
    out[i * N + self] = own ? a[i * N + self] : a[L.opp[i] * N + cell_index(sx, sy, sz, nx, ny)];
  }
}

// Slip plane codes are used by the vector kernel one VECTOR at a time: the non-wall cells of a 32-byte sector must agree on the
// code (a WALLMODEL / zero-gradient OUTLET cell counts as code 0).  Where they do not, the coded cells of the sector fall back
// to the per-cell path: SPECIAL, code cleared, ADJ set (the neighbour masks are built afterwards and then keep all their links).
template <int SV>
__global__ void __launch_bounds__(256) k_slip_uniform(uint8_t* __restrict__ cls, long long nsec_total, unsigned long long* __restrict__ counters) {
  const long long q = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (q >= nsec_total) return;
  int first = -1;
  bool mixed = false;
#pragma unroll
  for (int v = 0; v < SV; ++v) {
    const uint8_t c = cls[q * SV + v];
    if (is_wall(c)) continue;
    const int code = ((c & CLS_TYPE) == T_WM) ? 0 : ((c >> CLS_NORMAL_SHIFT) & 7);
    if (first < 0) first = code;
    else if (code != first) mixed = true;
  }
  if (!mixed) return;
#pragma unroll
  for (int v = 0; v < SV; ++v) {
    const uint8_t c = cls[q * SV + v];
    if (is_wall(c) || (c & CLS_TYPE) == T_WM || ((c >> CLS_NORMAL_SHIFT) & 7) == 0) continue;
    cls[q * SV + v] = static_cast<uint8_t>((c & CLS_TYPE) | CLS_ADJ | CLS_SPECIAL);
    atomicAdd(counters + 7, ~0ull);      // one coded cell less
  }
}

// marks the cells that the list blocks of k_step_vec must process: every cell of a 32-byte sector (SV = 8 floats /
// 4 doubles, aligned) that holds at least one SPECIAL cell.  mark[] feeds a stream compaction.
template <int SV>
__global__ void __launch_bounds__(256) k_mark_list(const uint8_t* __restrict__ cls, uint8_t* __restrict__ mark,
                                                   long long nsec_total, unsigned long long* __restrict__ counters) {
  const long long q = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (q >= nsec_total) return;
  bool m = false;
#pragma unroll
  for (int v = 0; v < SV; ++v) m = m || (cls[q * SV + v] & CLS_SPECIAL);
#pragma unroll
  for (int v = 0; v < SV; ++v) mark[q * SV + v] = m ? 1 : 0;
  if (m) atomicAdd(counters + 3, static_cast<unsigned long long>(SV));
}

// ---- A9 runs as modes of the step kernels (MODE_MOMENTS_*, MODE_TOTALS_*): the pull happens in registers, nothing is
// materialised.  Wall cells report their own (inert) populations, which live in the side buffer side[Q][n_solid]:
template <int Q, typename T>
__global__ void __launch_bounds__(256) k_solid_moments(const T* __restrict__ side, const int* __restrict__ solid_list, long long n_solid,
                                                       long long N, T* __restrict__ rho_out, T* __restrict__ u_out) {
  const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (k >= n_solid) return;
  T f[Q];
#pragma unroll
  for (int i = 0; i < Q; ++i) f[i] = side[i * n_solid + k];
  T rho, jx, jy, jz;
  cell_moments<Q, T>(f, rho, jx, jy, jz);
  const long long cell = solid_list[k];
  if (rho_out) rho_out[cell] = rho;
  if (u_out) {
    u_out[cell] = jx / rho;
    u_out[N + cell] = jy / rho;
    u_out[2 * N + cell] = jz / rho;
  }
}

// ---- A4 as an initialiser: f = f^eq(rho, u) ----------------------------------------------------------
template <int Q, typename T>
__global__ void __launch_bounds__(256) k_init_equilibrium(const T* __restrict__ rho_in, const T* __restrict__ u_in,
                                                          T* __restrict__ fa, long long N) {
  constexpr Stencil<Q> L{};
  const long long n = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (n >= N) return;
  const T rho = rho_in[n], ux = u_in[n], uy = u_in[N + n], uz = u_in[2 * N + n];
  const T base = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const T cu = T(L.c[i][0]) * ux + T(L.c[i][1]) * uy + T(L.c[i][2]) * uz;
    const T v = weight<Q, T>(L.c2[i]) * rho * (base + T(3) * cu + T(4.5) * cu * cu);
    fa[i * N + n] = v;
  }
}

// ---- flag validation + classification ------------------------------------------------------------
// cls = type | normal<<3 | ADJ | SPECIAL (see the top of this file).
// ---- Vortex Method inflow (Eq. 18-21; readings G11, G34, G35) --------------------
// Plane x = 0, d_inlet = (1,0,0); fields [3][nz][ny]; seeds (y_i, z_i) and signs are inputs.
// k_vm_gamma (one block): A = number of INLET cells of the plane; Gamma_i = 4 s_i sqrt(pi A k_i / (3 N (2 ln 3 - 3 ln 2))),
// k_i = 3/2 (|u_mean(p_i)| I)^2 with u_mean at the nearest cell (0 over a non-INLET cell).                    (Eq. 18-19)
template <typename T>
__global__ void __launch_bounds__(256) k_vm_gamma(const uint8_t* __restrict__ cls, int nx, int ny, int nz, const T* __restrict__ u_mean,
                                                  int nv, const double* __restrict__ pos, const double* __restrict__ sign,
                                                  double intensity, double* __restrict__ gamma) {
  __shared__ long long part[256];
  const long long P = static_cast<long long>(ny) * nz;
  long long cnt = 0;
  for (long long c = threadIdx.x; c < P; c += blockDim.x) cnt += ((cls[c * nx] & CLS_TYPE) == T_INLET) ? 1 : 0;
  part[threadIdx.x] = cnt;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (static_cast<int>(threadIdx.x) < s) part[threadIdx.x] += part[threadIdx.x + s];
    __syncthreads();
  }
  const double A = static_cast<double>(part[0]);
  const double PI = 3.14159265358979323846;
  for (int i = threadIdx.x; i < nv; i += blockDim.x) {
    int yi = static_cast<int>(floor(pos[2 * i] + 0.5)), zi = static_cast<int>(floor(pos[2 * i + 1] + 0.5));
    yi = ((yi % ny) + ny) % ny;
    zi = (zi < 0) ? 0 : ((zi >= nz) ? nz - 1 : zi);
    const long long c = static_cast<long long>(zi) * ny + yi;
    double k = 0.0;
    if ((cls[c * nx] & CLS_TYPE) == T_INLET) {
      const double a0 = static_cast<double>(u_mean[c]), a1 = static_cast<double>(u_mean[P + c]), a2 = static_cast<double>(u_mean[2 * P + c]);
      const double um = sqrt(a0 * a0 + a1 * a1 + a2 * a2);
      k = 1.5 * (um * intensity) * (um * intensity);
    }
    gamma[i] = 4.0 * sign[i] * sqrt(PI * A * k / (3.0 * nv * (2.0 * log(3.0) - 3.0 * log(2.0))));
  }
}

// dtype <-> fp64 copies of the inflow plane (the inflow fields are kept in fp64 whatever the lattice dtype)
template <typename A, typename B>
__global__ void __launch_bounds__(256) k_convert(const A* __restrict__ in, B* __restrict__ out, long long n) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i < n) out[i] = static_cast<B>(in[i]);
}

// k_vm_inflow: block = 64 cells of the inflow plane x 4 slices of the seeds (thread = one cell, every fourth seed); the seeds
// are staged through shared memory 256 at a time, the four partial sums of a cell are combined through shared memory.
//   u_v(x) = 1/(2 pi) sum_i Gamma_i ((p_i - x) x d)(1 - exp(-r^2 / 2 sigma^2)) / r^2                           (Eq. 20)
//   u(x)   = u_mean + u_v - (u_v . g^) d,  g^ = normalised in-plane central-difference gradient of u_prev . d   (Eq. 21)
// A path bound by plain ALU arithmetic (ny nz nv summands of ~12 flops + one exp), off the bandwidth path.
constexpr int VM_CELLS = 64, VM_SLICES = 4;
template <typename T>
__global__ void __launch_bounds__(VM_CELLS * VM_SLICES) k_vm_inflow(const uint8_t* __restrict__ cls, int nx, int ny, int nz,
                                                                    const T* __restrict__ u_mean, const T* __restrict__ u_prev, int nv,
                                                                    const double* __restrict__ pos, const double* __restrict__ gamma,
                                                                    T sigma_v, T* __restrict__ out) {
  constexpr int NT = VM_CELLS * VM_SLICES;
  __shared__ T sy[NT], sz[NT], sg[NT];
  __shared__ T py[VM_SLICES][VM_CELLS], pz[VM_SLICES][VM_CELLS];
  const long long P = static_cast<long long>(ny) * nz;
  const int lc = threadIdx.x % VM_CELLS, slice = threadIdx.x / VM_CELLS;
  const long long c = static_cast<long long>(blockIdx.x) * VM_CELLS + lc;
  const bool in_plane = c < P;
  const int z = in_plane ? static_cast<int>(c / ny) : 0, y = in_plane ? static_cast<int>(c - static_cast<long long>(z) * ny) : 0;
  const bool inlet = in_plane && ((cls[c * nx] & CLS_TYPE) == T_INLET);
  const T inv2s2 = T(1) / (T(2) * sigma_v * sigma_v);
  T uvy = T(0), uvz = T(0);
  for (int base = 0; base < nv; base += NT) {
    const int i = base + threadIdx.x;
    if (i < nv) {
      sy[threadIdx.x] = static_cast<T>(pos[2 * i]);
      sz[threadIdx.x] = static_cast<T>(pos[2 * i + 1]);
      sg[threadIdx.x] = static_cast<T>(gamma[i] * (0.5 / 3.14159265358979323846));
    }
    __syncthreads();
    const int m = (nv - base < NT) ? nv - base : NT;
    if (inlet) {
      for (int k = slice; k < m; k += VM_SLICES) {
        const T ry = sy[k] - T(y), rz = sz[k] - T(z);
        const T r2 = ry * ry + rz * rz;
        if (r2 == T(0)) continue;                        // the summand tends to 0 at the seed itself
        const T fac = sg[k] * (-expm1(-r2 * inv2s2)) / r2;
        uvy += fac * rz;
        uvz -= fac * ry;
      }
    }
    __syncthreads();
  }
  py[slice][lc] = uvy;
  pz[slice][lc] = uvz;
  __syncthreads();
  if (slice != 0 || !in_plane) return;
  uvy = (py[0][lc] + py[1][lc]) + (py[2][lc] + py[3][lc]);
  uvz = (pz[0][lc] + pz[1][lc]) + (pz[2][lc] + pz[3][lc]);
  T o0 = u_mean[c], o1 = u_mean[P + c], o2 = u_mean[2 * P + c];
  if (inlet) {
    const int yp = (y + 1 == ny) ? 0 : y + 1, ym = (y == 0) ? ny - 1 : y - 1;
    const long long row = static_cast<long long>(z) * ny;
    const long long cyp = ((cls[(row + yp) * nx] & CLS_TYPE) == T_INLET) ? row + yp : c;
    const long long cym = ((cls[(row + ym) * nx] & CLS_TYPE) == T_INLET) ? row + ym : c;
    const long long czp = (z + 1 < nz && (cls[(c + ny) * nx] & CLS_TYPE) == T_INLET) ? c + ny : c;
    const long long czm = (z >= 1 && (cls[(c - ny) * nx] & CLS_TYPE) == T_INLET) ? c - ny : c;
    const T gy = T(0.5) * (u_prev[cyp] - u_prev[cym]), gz = T(0.5) * (u_prev[czp] - u_prev[czm]);
    const T gn = sqrt(gy * gy + gz * gz);
    T us = T(0);
    if (gn > T(0)) us = -(uvy * gy + uvz * gz) / gn;
    o0 += us;
    o1 += uvy;
    o2 += uvz;
  }
  out[c] = o0;
  out[P + c] = o1;
  out[2 * P + c] = o2;
}

// counters[0] = invalid flag bytes, [1] = wall cells (SOLID + MOVINGWALL), [2] = masked cells (non-wall, not plain bulk FLUID),
// [4] = MOVINGWALL cells, [5] = SLIPWALL cells, [6] = WALLMODEL cells, [7] = cells with a slip plane code, [8] = non-wall cells of a type other than FLUID ([3] belongs to k_mark_list).
template <int Q>
__global__ void __launch_bounds__(256) k_classify(const uint8_t* __restrict__ flags, uint8_t* __restrict__ cls,
                                                  int nx, int ny, int nz, unsigned long long* __restrict__ counters, int wm_special, int slip_planes) {
  constexpr Stencil<Q> L{};
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= nx || y >= ny) return;
  const long long self = cell_index(x, y, z, nx, ny);
  const uint8_t fl = flags[self];
  const int type = fl & 0x0F, hi = fl >> 4;
  bool bad = type > T_SLIP;
  if (type == T_WM) bad = bad || hi > 5; else bad = bad || hi != 0;
  if (type == T_INLET && x != 0) bad = true;
  if ((type == T_OUTLET || type == T_POUTLET) && x != nx - 1) bad = true;
  if (type == T_MOVING && z != nz - 1) bad = true;
  if (bad) { atomicAdd(counters, 1ull); return; }
  uint32_t m = 0u;
  bool slipnb = false;
  int nt[Q];
  nt[0] = type;
  if (!is_wall(type)) {
#pragma unroll
    for (int j = 1; j < Q; ++j) {
      int sx = x + L.c[j][0], sy = y + L.c[j][1], sz = z + L.c[j][2];
      sx = (sx < 0) ? sx + nx : ((sx >= nx) ? sx - nx : sx);
      sy = (sy < 0) ? sy + ny : ((sy >= ny) ? sy - ny : sy);
      sz = (sz < 0) ? sz + nz : ((sz >= nz) ? sz - nz : sz);
      nt[j] = flags[cell_index(sx, sy, sz, nx, ny)] & 0x0F;
      if (is_wall(nt[j])) m |= (1u << j);
      if (nt[j] == T_SLIP) slipnb = true;
    }
  }
  // slip plane code (see slip_axis above): every neighbour on the wall side of ONE plane normal to y or z is a SLIPWALL cell, the
  // specular sources x + c_j + n (in the cell's own plane) are no walls, and no other neighbour is a slip wall (other walls are
  // fine: they stay in the neighbour mask and bounce back)
  int scode = 0;
  if (slipnb && slip_planes && type != T_WM && type != T_OUTLET) {
    constexpr Mirror<Q> MR{};
    for (int code = 2; code <= 5 && scode == 0; ++code) {
      const int ax = slip_axis(code), side = -slip_sign(code);
      bool ok = true;
      uint32_t handled = 0u;
#pragma unroll
      for (int j = 1; j < Q; ++j) {
        if (L.c[j][ax] == side) {
          handled |= (1u << j);
          const int back = (ax == 1) ? MR.zy[j] : MR.zz[j];       // x + c_j + n
          if (nt[j] != T_SLIP || (back != 0 && is_wall(nt[back]))) ok = false;
        } else if (nt[j] == T_SLIP) {
          ok = false;
        }
      }
      if (ok) {
        scode = code;
        m &= ~handled;
      }
    }
  }
  const bool adj_any = (m != 0u) || scode != 0;                // (statistics: the cell has a wall neighbour)
  const bool adj = (m != 0u);
  // cells next to a slip wall that have no slip plane code take the per-cell path (general specular pull slip_pull)
  // (wm_special: WALLMODEL cells solve Spalding's law in the list blocks instead of taking u^B from the pre-pass)
  const bool special = (type == T_WM && wm_special) || (type == T_OUTLET && adj) || (slipnb && scode == 0);
  cls[self] = static_cast<uint8_t>(type | ((type == T_WM ? hi : scode) << CLS_NORMAL_SHIFT) | (adj ? CLS_ADJ : 0) |
                                   (special ? CLS_SPECIAL : 0));
  if (is_wall(type)) atomicAdd(counters + 1, 1ull);
  if (type == T_MOVING) atomicAdd(counters + 4, 1ull);
  if (type == T_WM) atomicAdd(counters + 6, 1ull);
  if (type == T_SLIP) atomicAdd(counters + 5, 1ull);
  else if (adj_any || type != T_FLUID) atomicAdd(counters + 2, 1ull);
  if (scode != 0) atomicAdd(counters + 7, 1ull);
  if (!is_wall(type) && type != T_FLUID) atomicAdd(counters + 8, 1ull);
}

// nbmask of an accepted classification (a rejected flag array must leave the old geometry intact)
template <int Q>
__global__ void __launch_bounds__(256) k_nbmask(const uint8_t* __restrict__ cls, uint32_t* __restrict__ nbmask, int nx, int ny, int nz) {
  constexpr Stencil<Q> L{};
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= nx || y >= ny) return;
  const long long self = cell_index(x, y, z, nx, ny);
  uint32_t m = 0u;
  if (cls[self] & CLS_ADJ) {
#pragma unroll
    for (int j = 1; j < Q; ++j) {
      int sx = x + L.c[j][0], sy = y + L.c[j][1], sz = z + L.c[j][2];
      sx = (sx < 0) ? sx + nx : ((sx >= nx) ? sx - nx : sx);
      sy = (sy < 0) ? sy + ny : ((sy >= ny) ? sy - ny : sy);
      sz = (sz < 0) ? sz + nz : ((sz >= nz) ? sz - nz : sz);
      if (is_wall(cls[cell_index(sx, sy, sz, nx, ny)])) m |= (1u << j);
    }
  }
  const uint8_t c0 = cls[self];
  const int sc = ((c0 & CLS_TYPE) == T_WM || is_wall(c0)) ? 0 : ((c0 >> CLS_NORMAL_SHIFT) & 7);
  if (sc != 0) {                         // the links into the slip plane are served by the specular pull, not by bounce-back
#pragma unroll
    for (int j = 1; j < Q; ++j)
      if (L.c[j][slip_axis(sc)] == -slip_sign(sc)) m &= ~(1u << j);
  }
  nbmask[self] = m;
}

// mark[n] = 1 on SOLID cells (feeds the compaction of the SOLID-cell list)
static __global__ void __launch_bounds__(256) k_mark_solid(const uint8_t* __restrict__ cls, uint8_t* __restrict__ mark, long long N) {
  const long long n = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (n < N) mark[n] = is_wall(cls[n]) ? 1 : 0;
}

// populations of a box of cells out of a lattice that holds S_t: out[Q][bz][by][bx] (lbm_get_populations_box)
template <typename T>
__global__ void __launch_bounds__(256) k_gather_box(const T* __restrict__ f, long long N, int nx, int ny, int x0, int y0, int z0,
                                                    int bx, int by, int bz, int Q, T* __restrict__ out) {
  const long long n = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  const long long per = static_cast<long long>(bx) * by * bz;
  if (n >= per * Q) return;
  const int i = static_cast<int>(n / per);
  long long r = n - i * per;
  const int z = static_cast<int>(r / (static_cast<long long>(bx) * by));
  r -= static_cast<long long>(z) * bx * by;
  const int y = static_cast<int>(r / bx), x = static_cast<int>(r - static_cast<long long>(y) * bx);
  out[n] = f[i * N + cell_index(x0 + x, y0 + y, z0 + z, nx, ny)];
}

// the inverse: in[Q][bz][by][bx] -> the box's cells of a lattice that holds S_t (lbm_set_populations_box)
template <typename T>
__global__ void __launch_bounds__(256) k_scatter_box(T* __restrict__ f, long long N, int nx, int ny, int x0, int y0, int z0,
                                                     int bx, int by, int bz, int Q, const T* __restrict__ in) {
  const long long n = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  const long long per = static_cast<long long>(bx) * by * bz;
  if (n >= per * Q) return;
  const int i = static_cast<int>(n / per);
  long long r = n - i * per;
  const int z = static_cast<int>(r / (static_cast<long long>(bx) * by));
  r -= static_cast<long long>(z) * bx * by;
  const int y = static_cast<int>(r / bx), x = static_cast<int>(r - static_cast<long long>(y) * bx);
  f[i * N + cell_index(x0 + x, y0 + y, z0 + z, nx, ny)] = in[n];
}

// ---- halo exchange of a slab decomposition in z ----------------------------------------
// A face buffer holds n_planes planes of nx*ny values: the populations that cross the cut (c_z = -1 towards the lower, c_z = +1
// towards the upper neighbour: 5 of 19, 9 of 27) of one boundary slice, or the three components of u^ of that slice (HRR form).
// In the SoA layout every such plane is contiguous: base + idx[k] * N + z * plane.  PACK: lattice -> buffer, else buffer -> lattice.
struct HaloPlanes {
  int n;
  int idx[9];          // population (or component) index of plane k
};
template <typename T, bool PACK>
__global__ void __launch_bounds__(256) k_halo_planes(T* __restrict__ field, long long N, long long slice_off, long long plane,
                                                     HaloPlanes hp, T* __restrict__ buf) {
  const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
  for (int k = 0; k < hp.n; ++k) {
    T* __restrict__ row = field + hp.idx[k] * N + slice_off;
    T* __restrict__ b = buf + k * plane;
    for (long long n = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; n < plane; n += stride) {
      if (PACK) b[n] = row[n];
      else row[n] = b[n];
    }
  }
}

// wall-model cells whose sample point x + n lies in a ghost slice (their pre-pass would pull from beyond the halo): counted
// when a halo is set, the decomposition is refused if there are any
static __global__ void __launch_bounds__(256) k_count_wm_on_cut(const uint8_t* __restrict__ cls, long long plane, int nz, int ghost_lo,
                                                                int ghost_hi, unsigned long long* __restrict__ count) {
  const long long n = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (n >= plane) return;
  unsigned bad = 0;
  if (ghost_lo) {                       // first interior slice, normal -z (code 5)
    const uint8_t c = cls[static_cast<long long>(ghost_lo) * plane + n];
    if ((c & CLS_TYPE) == T_WM && ((c >> CLS_NORMAL_SHIFT) & 7) == 5) ++bad;
  }
  if (ghost_hi) {                       // last interior slice, normal +z (code 4)
    const uint8_t c = cls[static_cast<long long>(nz - 1 - ghost_hi) * plane + n];
    if ((c & CLS_TYPE) == T_WM && ((c >> CLS_NORMAL_SHIFT) & 7) == 4) ++bad;
  }
  if (bad) atomicAdd(count, static_cast<unsigned long long>(bad));
}

// mark[n] = 1 on WALLMODEL cells (feeds the compaction of the pre-pass list)
static __global__ void __launch_bounds__(256) k_mark_wm(const uint8_t* __restrict__ cls, uint8_t* __restrict__ mark, long long N) {
  const long long n = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (n < N) mark[n] = ((cls[n] & CLS_TYPE) == T_WM) ? 1 : 0;
}

// SOLID cells are inert (R5) but the step kernels write zeros over their slots: their own Q values live in a side buffer
// side[Q][n_solid].  SAVE: lattice -> side;  !SAVE: side -> lattice (after a materialisation).
template <typename T, bool SAVE>
__global__ void __launch_bounds__(256) k_solid_values(T* __restrict__ f, T* __restrict__ side, const int* __restrict__ solid_list,
                                                      long long n_solid, long long N, int Q) {
  const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (k >= n_solid) return;
  const long long cell = solid_list[k];
  for (int i = 0; i < Q; ++i) {
    if (SAVE) side[i * n_solid + k] = f[i * N + cell];
    else f[i * N + cell] = side[i * n_solid + k];
  }
}

}  // namespace lbm
