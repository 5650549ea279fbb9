/* =====================================================================================
 * lbm.h -- C ABI of the B200-native lattice Boltzmann hot path of arxiv 2506.21804
 * (BGK or HRR collision + Smagorinsky LES + homogenised-LBM porosity; D3Q19 / D3Q27; fp32 / fp64).
 *
 * Library: paper_2506_21804_b200/liblbm_b200.so (CUDA, sm_100a).  Every step of the path runs
 * in the library's own kernels; there is no CPU fallback: every call fails with LBM_ECUDA when no
 * CUDA device is usable.
 *
 * Citations are to /root/reference/PAPER.md (line : equation) and to the readings listed in
 * DESIGN.md (G1..G26, R1..R12), which follow SURVEY.md section 8(c).
 *
 * Conventions common to all calls
 *  - Return value: 0 on success, <0 on error (enum below).  Nothing throws or aborts across the ABI.
 *  - POINTERS: every data pointer may be a DEVICE pointer (e.g. torch CUDA tensor data_ptr()) or a
 *    HOST pointer (pageable or pinned).  The library inspects the pointer (cudaPointerGetAttributes)
 *    and copies host buffers to / from the device on the context's stream.  Device buffers are used
 *    in place, with no copy, wherever the layouts allow.
 *  - OWNERSHIP: the caller owns every buffer it passes; the library copies inputs into its own
 *    storage and writes outputs into caller buffers of exactly the stated size.  The library owns
 *    the lbm_ctx and all internal device memory (cudaMalloc), released by lbm_destroy.
 *  - EXTERNAL LAYOUTS (fixed; x fastest; `dtype` = float or double as chosen at lbm_create):
 *        populations[Q][nz][ny][nx]   plain f_i, population order of reading R1 (see below)
 *        porosity   [nz][ny][nx]      d in [0,1]; Eq. 12 convention: 0 = fluid, 1 = solid (G2)
 *        cell_flags [nz][ny][nx]      uint8
 *        rho        [nz][ny][nx],  u[3][nz][ny][nx]
 *  - FLAG BYTE: low nibble = type {0 FLUID, 1 SOLID, 2 INLET, 3 OUTLET, 4 WALLMODEL, 5 MOVINGWALL, 6 POUTLET, 7 SLIPWALL}.  For
 *    WALLMODEL the high nibble is the wall-normal code {0:+x, 1:-x, 2:+y, 3:-y, 4:+z, 5:-z}
 *    pointing from the wall into the fluid (config 3 floor cells: 0x44); otherwise it must be 0.
 *    INLET is accepted only on the plane x = 0, OUTLET (zero gradient) and POUTLET (fixed pressure) only on x = nx-1, MOVINGWALL (a SOLID cell that moves with
 *    lbm_params.u_wall; inert like SOLID) only on z = nz-1.
 *    SLIPWALL is a wall cell (inert like SOLID) with full slip (l.255; reading G37): a population pulled from it is the specular
 *    image -- it comes from the fluid cell x - c_i + sum_a c_ia e_a with the components a of c_i reversed, a = the axes along
 *    which the cell's single-axis neighbour x - c_ia e_a is a SLIPWALL cell; no such axis, or a wall at that cell: bounce-back.
 *  - POPULATION ORDER (R1): i = 0 rest; 1..h (h = (Q-1)/2) the directions whose first non-zero
 *    component is +1 sorted by (|c|^2, -cx, -cy, -cz); h+1..Q-1 their negatives, opp(i) = i +- h.
 *  - STATE (G12/R2): the state S_t is the set of PRE-collision populations f_i(x,t) of Eq. 6.
 *    lbm_step(n) advances S_t -> S_{t+n}.  lbm_moments / lbm_totals / lbm_get_populations always
 *    describe S_t, whatever the internal storage is.
 *  - ASYNCHRONY: lbm_step only enqueues kernels on the context's stream.  All other calls
 *    return after their copies have been enqueued; calls that must return a value to the host
 *    (lbm_totals, outputs into host buffers, flag validation in lbm_set_fields) synchronise the
 *    stream.  A launch error is reported at the latest by the next call.
 * ===================================================================================== */
#ifndef PAPER_2506_21804_B200_LBM_H
#define PAPER_2506_21804_B200_LBM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { LBM_OK = 0, LBM_EINVAL = -1, LBM_ENOMEM = -2, LBM_ECUDA = -3, LBM_ESTATE = -4 };
enum { LBM_D3Q19 = 19, LBM_D3Q27 = 27 };
enum { LBM_F32 = 4, LBM_F64 = 8 };
enum { LBM_FLUID = 0, LBM_SOLID = 1, LBM_INLET = 2, LBM_OUTLET = 3, LBM_WALLMODEL = 4, LBM_MOVINGWALL = 5, LBM_POUTLET = 6, LBM_SLIPWALL = 7 };
enum { LBM_COLLISION_BGK = 0, LBM_COLLISION_HRR = 1, LBM_COLLISION_HRR_LAG = 2 };
enum { LBM_HALO_POPULATIONS = 0, LBM_HALO_UHAT = 1 };
enum { LBM_SIDE_LOW = 0, LBM_SIDE_HIGH = 1 };

typedef struct lbm_ctx lbm_ctx; /* opaque; owned by the library */

/* Step parameters.  All reals are double whatever the dtype; converted once per lbm_step. */
typedef struct {
  double tau0;      /* molecular relaxation time, > 0.5; nu = (tau0 - 0.5)/3  (Eq. 14, G3)         */
  double cs_smago;  /* Smagorinsky constant C_S >= 0 (Eq. 4); 0 => plain BGK                       */
  int use_hlbm;     /* 0: d treated as 0 everywhere (porosity is not read); 1: Eq. 12              */
  double u_in[3];   /* velocity imposed on INLET cells (l.155, reading R6)                         */
  int wm_enable;    /* 0: WALLMODEL cells behave as FLUID; 1: Spalding wall model (Eq. 15-17, R8)  */
  double wm_kappa;  /* Spalding constants; the paper prints neither (defaults 0.41, 9.8)           */
  double wm_E;
  int collision;    /* LBM_COLLISION_BGK (0): Eq. 6 with f~(1) = f - f^eq, Eq. 11 up to H(2) (G1);
                     * LBM_COLLISION_HRR (1): the paper's own collision, Eq. 6-11 in full: third-order
                     * equilibrium (Eq. 11, G9), recursive-regularised f(1) (Eq. 8-9, G29), finite-
                     * difference part (Eq. 10, G10) hybridised by sigma (Eq. 7); the FD strain is the
                     * central difference of u^(x,t) of the same time level (G30-G32); sigma = 0 on
                     * WALLMODEL cells when wm_enable (l.131).  Smagorinsky tau_eff as in the BGK form.
                     * LBM_COLLISION_HRR_LAG (2): the same collision with the FD strain of Eq. 10 taken of
                     * u^(x, t - dt), the field the previous step formed (reading G41; l.172: a local cell
                     * model at 188 bytes per collision): ONE pass over the lattice per step instead of two.
                     * The state of this form is (S_t, u^ of the previous level): the first step after
                     * lbm_set_fields / lbm_init_equilibrium / lbm_set_populations_box / lbm_set_geometry, or after
                     * steps of another form, or with a new u_wall on a lattice with MOVINGWALL cells, has no
                     * history and differences u^(x,t) like form 1.  On sub-domains (lbm_step_halo) the u^
                     * exchange in front of stage 1 carries the previous level's boundary slices.        */
  double sigma;     /* Eq. 7 hybridisation factor in [0,1]; read only when collision == HRR         */
  double u_wall[3]; /* velocity of the MOVINGWALL cells: the lid of the lid-driven cavity benchmark (l.214).  Halfway
                     * bounce-back off a moving wall (reading G33): the population i returning from the wall gains
                     * 2 w_i rho_w (c_i.u_w)/c_s^2 with rho_w = 1 and c_i pointing from the wall into the fluid;
                     * the HRR form's FD stencil sees u^ = u_wall on those cells                       */
  double rho_out;   /* density (= pressure / c_s^2) imposed on POUTLET cells: the "fixed local pressure" outlet of the urban case
                     * (l.255; reading G36: regularised local rule, normal velocity from the known populations, tangential
                     * velocity 0).  0 means the default 1.                                                   */
  int fringe_len;   /* fringe zone in front of the outlet plane (l.255 "with fringe zone"; reading G38): over the last fringe_len
                     * cells in x the molecular viscosity rises as nu_mo (1 + fringe_factor xi^2), xi = (x - (nx-1-fringe_len)) /
                     * fringe_len in [0,1] (a sponge that damps what reaches the outlet).  0 = no fringe zone.              */
  double fringe_factor;
} lbm_params;

/* Create a context for an nx x ny x nz lattice (nx fastest in memory).
 * lattice: LBM_D3Q19 | LBM_D3Q27 (l.60; D3Q27 from BASELINE.json config 4).  dtype: LBM_F32 | LBM_F64.
 * nx, ny, nz >= 1 (SURVEY 8(b) asked for LBM_EINVAL below 3; sizes 1 and 2 are accepted as a superset: the periodic wrap is
 * well defined for them and they are parity-tested), nx*ny*nz < 2^31, ny <= 65535 and nz <= 65000 (launch-grid limits; a
 * lattice whose nz plus its list slices passes 65535 is refused by lbm_step with LBM_EINVAL).  Rows with nx a multiple of
 * 32/sizeof(dtype) take the vector kernel, other row lengths the scalar kernel.  Allocates one population lattice (Q*N*dtype
 * bytes; the second one when the first two-lattice pass runs), the porosity field, one class byte and one 32-bit neighbour mask per cell on the current CUDA device.
 * Returns NULL on failure; lbm_last_error(NULL) then holds the reason. */
lbm_ctx* lbm_create(int lattice, int nx, int ny, int nz, int dtype);

/* Release the context and all its device memory.  NULL is ignored. */
void lbm_destroy(lbm_ctx* ctx);

/* Set the state S_0 and the fields (Eq. 6 l.70-72: populations on the lattice; Eq. 12-13 l.99-103:
 * porosity d(x); Listing 1: per-cell model switches).  Resets the step counter to 0.
 *   populations : [Q][nz][ny][nx] dtype, host or device; must not be NULL.
 *   porosity    : [nz][ny][nx] dtype, or NULL => d = 0 everywhere.
 *   cell_flags  : [nz][ny][nx] uint8, or NULL => all FLUID.
 * Errors: LBM_EINVAL for a NULL ctx / populations or an invalid flag byte (nothing is changed then:
 * a context that held a valid state keeps it); LBM_ECUDA. */
int lbm_set_fields(lbm_ctx* ctx, const void* populations, const void* porosity, const uint8_t* cell_flags);

/* Set S_0 = f^eq(rho, u) cell by cell (Eq. 11 l.94 truncated after H(2); A4).  rho[nz][ny][nx],
 * u[3][nz][ny][nx] dtype, host or device.  Porosity and flags are kept as last set (or d = 0 / all FLUID
 * if lbm_set_fields was never called).  Resets the step counter to 0. */
int lbm_init_equilibrium(lbm_ctx* ctx, const void* rho, const void* u);

/* Replace porosity and flags only (same rules as lbm_set_fields); the populations are kept. */
int lbm_set_geometry(lbm_ctx* ctx, const void* porosity, const uint8_t* cell_flags);

/* Time-varying porosity d(x,t) (Eq. 12-13, l.99-103: "d(x,t)"): replace the porosity field only.
 *   porosity : [nz][ny][nx] dtype, host or device (copied); NULL => d = 0 everywhere.
 * Flags and populations are kept.  d enters the collision only, so -- unlike lbm_set_geometry -- this costs no pass over
 * the lattice: the next lbm_step collides S_t with the new field.  Errors: LBM_EINVAL (NULL ctx), LBM_ECUDA. */
int lbm_set_porosity(lbm_ctx* ctx, const void* porosity);

/* Solid velocity field u^B(x,t) of Eq. 12 (l.99: u^ = (1-d) u + d u^B; l.106 "non-zero solid velocities"; the moving bodies of
 * the FSI cases of Fig. 1).
 *   u_body : [3][nz][ny][nx] dtype (component, z, y, x), host or device (copied into 3 N values of library memory);
 *            NULL => u^B = 0 everywhere again (the memory is released).
 * The field stays until the next call; a body that moves is stepped with lbm_set_porosity + lbm_set_body_velocity before each
 * lbm_step(1).  It is read only where d != 0 and only when lbm_params.use_hlbm; WALLMODEL cells keep the wall model's u^B when
 * wm_enable (reading G39); SOLID cells ignore it.  Both collision forms.  No pass over the lattice.
 * Errors: LBM_EINVAL (NULL ctx), LBM_ENOMEM, LBM_ECUDA. */
int lbm_set_body_velocity(lbm_ctx* ctx, const void* u_body);

/* Inflow velocity field of the INLET cells (plane x = 0) and the Vortex Method that perturbs it (Eq. 18-21;
 * SURVEY 8(f)-3; readings G11, G34, G35 of DESIGN.md).
 *   u_mean : [3][nz][ny] dtype (component, z, y), host or device: the mean velocity profile u_mean(x) of Eq. 21; entries of
 *            cells that are not INLET cells are ignored.  NULL switches back to the uniform lbm_params.u_in.
 * Once set, every lbm_step forms the inflow velocity of the new time level before the inlet rule (l.155) is applied:
 *   u(x) = u_mean(x) + u_vortex(x) - (u_vortex(x) . g^(x)) d_inlet,     d_inlet = (1,0,0),
 *   u_vortex by Eq. 20 from the seeds set with lbm_set_vortices (none => u = u_mean), g^ = the normalised in-plane gradient of
 *   the previous step's streamwise inflow (central differences; a neighbour that is not an INLET cell is replaced by the cell
 *   itself; y wraps).  "Previous inflow" is u_mean before the first step after this call / lbm_set_fields / lbm_init_equilibrium.
 * The inflow fields are kept and computed in fp64 for both dtypes (Eq. 21 normalises a difference of neighbouring values) and
 * rounded to dtype where the inlet rule reads them.
 * Errors: LBM_EINVAL (NULL ctx), LBM_ENOMEM, LBM_ECUDA. */
int lbm_set_inflow(lbm_ctx* ctx, const void* u_mean);

/* Seeds of the Vortex Method: n_vortices >= 0 positions pos[n][2] = (y, z) in cell coordinates on the inflow plane and signs
 * sign[n] = +-1 (HOST arrays of double: the random numbers the method draws are inputs), vortex size sigma_v > 0 (cells) and
 * turbulence intensity >= 0.  Circulations: k_i = 3/2 (|u_mean(p_i)| I)^2 (Eq. 18, u_mean at the nearest cell, 0 over a cell that
 * is not an INLET cell), Gamma_i = 4 s_i sqrt(pi A k_i / (3 n (2 ln 3 - 3 ln 2))) (Eq. 19, G34), A = number of INLET cells.
 * The seeds stay until the next call; needs lbm_set_inflow first to take effect.
 * Errors: LBM_EINVAL (NULL ctx, n < 0, NULL arrays with n > 0, sigma_v <= 0, intensity < 0), LBM_ENOMEM, LBM_ECUDA. */
int lbm_set_vortices(lbm_ctx* ctx, int n_vortices, const double* pos, const double* sign, double sigma_v, double intensity);

/* The inflow velocity field that belongs to the state S_t (the one its INLET cells carry): u[3][nz][ny] dtype, host or
 * device.  LBM_ESTATE if no inflow field is set. */
int lbm_get_inflow(lbm_ctx* ctx, void* u);

/* Advance S_t -> S_{t+n_steps}: per step, per non-SOLID cell (Eq. 6, l.70):
 *   wall model u^B (Eq. 15-17, l.131) -> moments (l.97) -> u^ = (1-d)u + d u^B (Eq. 12) -> f^eq (Eq. 11)
 *   -> tau_eff from the local non-equilibrium stress (Eq. 3-5, 14) -> relaxation (Eq. 6) -> propagation
 *   with halfway bounce-back at SOLID neighbours (R5), zero-gradient outlet (R7), regularised velocity
 *   inlet (l.155, R6).
 * BGK form: one fused kernel launch per step on the context's stream, preceded by the wall-model pre-pass over the
 * compact list of WALLMODEL cells when wm_enable and such cells exist (3 values of dtype per cell of device memory for
 * their u^B, allocated on the first such step).  HRR form: two launches per step (u^ pass, then the fused step;
 * DESIGN.md 5.5) and 3 more values of dtype per cell (allocated on the first HRR step; LBM_ENOMEM if that fails);
 * collision = 2: one launch per step and 6 values per cell (the u^ pass runs only on the first step of a history).
 * With option "cuda_graph" steady-state steps are replayed 8 at a time from a captured CUDA graph.  Asynchronous.
 * When params change from one call to the next: the storage holds the post-collision lattice, the propagation that ends a
 * step runs as the pull of the NEXT step's launch, so the values the propagation reads from params (u_in, u_wall, rho_out) are
 * those of the call that pulls.  A state read in between (lbm_get_populations) forms S_t with the params of the last step,
 * after which a call with new params starts exactly where the method's own order (collide, then stream) would.
 * Errors: LBM_EINVAL (NULL ctx/params, n_steps < 0, tau0 <= 0.5, cs_smago < 0, wm_enable with
 * wm_kappa <= 0 or wm_E <= 0, collision not 0/1/2, sigma outside [0,1] with the HRR forms, rho_out < 0, fringe_len < 0, fringe_factor < 0), LBM_ESTATE (no state
 * set yet), LBM_ECUDA. */
int lbm_step(lbm_ctx* ctx, int n_steps, const lbm_params* params);

/* Moments of the state S_t for EVERY cell (SOLID cells report whatever was set):
 * rho = sum_i f_i, u = sum_i c_i f_i / rho -- the raw fluid velocity moment of l.97 (G19), not u^.
 * rho[nz][ny][nx], u[3][nz][ny][nx] dtype, host or device; either may be NULL to skip it.
 * One launch of the step kernel in its moments mode (the pull of S_t from the stored post-collision lattice happens in
 * registers; nothing is materialised and the following lbm_step costs no extra pass) plus one launch over the wall cells.
 * Errors: LBM_EINVAL (NULL ctx), LBM_ESTATE (no state), LBM_ENOMEM (staging for host outputs), LBM_ECUDA. */
int lbm_moments(lbm_ctx* ctx, void* rho, void* u);

/* State S_t = the pre-collision populations f_i(x,t) of Eq. 6 (l.70-72; reading G12/R2) in the external layout:
 * populations[Q][nz][ny][nx] dtype, host or device, written in full (parity checks, checkpoint).
 * When the storage holds the post-collision lattice this materialises S_t with one stream-only pass into the other lattice
 * (the next lbm_step then starts with a collide-only sweep: still one sweep per step).
 * Errors: LBM_EINVAL (NULL ctx / buffer), LBM_ESTATE (no state), LBM_ECUDA. */
int lbm_get_populations(lbm_ctx* ctx, void* populations);

/* The same for a box of cells only: origin (x0,y0,z0), extent (bx,by,bz) >= 1, inside the lattice (no wrap);
 * populations[Q][bz][by][bx] dtype, host or device.  For probes and for parity checks on lattices whose full state does not
 * fit a third time in memory (896^3 fp32: 54.7 GB per population set).  Materialises S_t like lbm_get_populations.
 * Errors: LBM_EINVAL (NULL ctx / buffer, box empty or outside the lattice), LBM_ESTATE, LBM_ENOMEM, LBM_ECUDA. */
int lbm_get_populations_box(lbm_ctx* ctx, int x0, int y0, int z0, int bx, int by, int bz, void* populations);

/* The inverse of lbm_get_populations_box: replace the populations f_i(x,t) of the state S_t (Eq. 6 l.70-72) on a box of cells;
 * populations[Q][bz][by][bx] dtype, host or device (copied), box inside the lattice (no wrap).  Everything else of the state is
 * kept (step counter, geometry, fields).  On a context without a state the call starts one at step 0: the caller then covers the
 * whole lattice box by box before stepping (cells not covered hold unspecified values) -- the way to set a lattice whose
 * populations do not fit a third time in memory (896^3 fp32).  Materialises S_t like lbm_get_populations.
 * Errors: LBM_EINVAL (NULL ctx / buffer, box empty or outside the lattice), LBM_ENOMEM (staging), LBM_ECUDA. */
int lbm_set_populations_box(lbm_ctx* ctx, int x0, int y0, int z0, int bx, int by, int bz, const void* populations);

/* Totals over the non-wall cells of S_t (the conserved quantities of Eq. 6: mass and momentum, l.97,
 * and the kinetic energy the Taylor-Green check of config 1 is stated in): out[0] = sum rho, out[1..3] = sum rho u,
 * out[4] = sum rho |u|^2 / 2.  `out`: 5 doubles, host (the call synchronises the stream) or device (asynchronous).  One launch, pulling S_t in registers like lbm_moments:
 * per-thread sums over the cells of a vector in dtype, from the warp level up in fp64 (shuffle tree, one atomicAdd(double)
 * per block into one of 256 slots, the last block adds the slots: one warp per quantity).  On a sub-domain (lbm_set_halo): the interior cells only.
 * Errors: LBM_EINVAL (NULL ctx / out), LBM_ESTATE (no state), LBM_ECUDA. */
int lbm_totals(lbm_ctx* ctx, double out[5]);

/* The same totals for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no context, and no cudaMalloc / cudaFree / allocating library routine anywhere on this call's path.  Same
 * quantities as lbm_totals (row A9; the conserved moments of Eq. 6, l.97): out[0] = sum rho, out[1..3] = sum rho u,
 * out[4] = sum rho |u|^2 / 2 over the non-wall cells of the state S_t the caller passes.
 *   populations : [Q][nz][ny][nx] dtype, DEVICE pointer: the pre-collision populations S_t (what lbm_get_populations writes).
 *   cell_flags  : [nz][ny][nx] uint8, DEVICE pointer, or NULL => no wall cells.  Flag bytes as in lbm_set_fields; only the type
 *                 nibble is read (SOLID, MOVINGWALL, SLIPWALL cells do not count) and nothing is validated.
 *   out         : 5 doubles, DEVICE pointer, written asynchronously on `cuda_stream` (a cudaStream_t as void*; NULL = the legacy
 *                 default stream).  The caller owns all three buffers; nothing is copied.
 * Its scratch (one partial sum per block of 8192 cells and quantity, and the ticket that finds the last block) is a file-scope
 * `static __device__` array of LBM_STATIC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits;
 * hence the limit nx ny nz <= LBM_STATIC_MAX_CELLS (512^3), beyond which the call returns LBM_EINVAL (use lbm_totals).  The
 * first call on a device resolves the array's address there (cudaGetSymbolAddress; make that call outside a graph capture).
 * Every call on a device shares the array: each call clears the ticket on its stream before its launch (the partial sums
 * need no clearing), but calls that OVERLAP on the same GPU (two streams, two host threads) race on it -- serialise them.
 * The sums are taken in a fixed order (a function of nx ny nz only), in fp64 from the cell's moments on: repeated calls on the
 * same data return the same bits.  Works on the current device; the pointers must belong to it.
 * Errors: LBM_EINVAL (lattice / dtype / sizes, more than LBM_STATIC_MAX_CELLS cells, NULL populations / out, a host or
 * misaligned pointer), LBM_ECUDA; lbm_last_error(NULL) holds the reason. */
#define LBM_STATIC_MAX_CELLS 134217728LL
#define LBM_STATIC_SCRATCH_BYTES 655616
int lbm_totals_static(int lattice, int nx, int ny, int nz, int dtype, const void* populations, const uint8_t* cell_flags,
                      double* out, void* cuda_stream);

/* ---- Slab decomposition in z: one context per sub-domain (PAPER.md l.214-218 and Table 1 l.227-239: the
 * paper's scaling runs decompose the lattice over MPI ranks with a halo exchange per step).  The library provides the
 * sub-domain mechanics; the transfer itself (NCCL send/recv, peer copies, or a device copy between two contexts on one GPU)
 * is the caller's, on the context's stream.
 *
 * lbm_set_halo: declare the first ghost_lo and the last ghost_hi z-slices (0 or 1 each) of this context's lattice GHOST slices:
 * copies of the neighbouring sub-domain's boundary slices.  Their flags and porosity are set by the caller like any other cell
 * (copies of the neighbour's), their populations arrive through lbm_halo_unpack; every pass (step, moments, totals, state
 * getters) then covers the interior slices only, and the entries of the ghost slices in any output are unspecified.
 * A sub-domain is advanced with lbm_step_halo (lbm_step returns LBM_ESTATE), one time step in two stages:
 *     stage 0   HRR form: wall-model pre-pass + u^ pass (Eq. 12) over the interior; BGK form: nothing
 *               -> exchange LBM_HALO_UHAT (HRR form only): the FD strain of Eq. 10 reads u^ of the slices z +- 1
 *     stage 1   the fused step over the interior (Eq. 6; stream + collide)
 *               -> exchange LBM_HALO_POPULATIONS: the next step's pull (l.70, A1) reads the ghost slices
 * No exchange is needed before the first step of a fresh state (it collides S_0 in place).  Per face the exchange moves the
 * populations that cross the cut, 5 of 19 (D3Q19) or 9 of 27 (D3Q27) per cell, and 3 values of u^ per cell in the HRR form.
 * Not available with the Vortex Method inlet (it works on the whole inflow plane); a WALLMODEL cell whose sample point x + n lies
 * in a ghost slice is refused (LBM_EINVAL: move the cut); CUDA graphs and "hrr_slab" are not used.
 * Errors: LBM_EINVAL (NULL ctx, counts not 0/1, no interior slice left, wall-model cell on a cut), LBM_ESTATE (VM inlet), LBM_ECUDA. */
int lbm_set_halo(lbm_ctx* ctx, int ghost_lo, int ghost_hi);

/* One stage (0, then 1) of one time step of a sub-domain; see lbm_set_halo.  Also valid without ghost slices (the two stages
 * together are lbm_step(1) without the CUDA-graph path).  Asynchronous.
 * Errors: as lbm_step, plus LBM_EINVAL (stage not 0 / 1) and LBM_ESTATE (stages out of order, VM inlet). */
int lbm_step_halo(lbm_ctx* ctx, const lbm_params* params, int stage);

/* Face buffers of the halo exchange.  what: LBM_HALO_POPULATIONS | LBM_HALO_UHAT; side: LBM_SIDE_LOW (z = 0 end) | LBM_SIDE_HIGH.
 * lbm_halo_pack copies out of the boundary INTERIOR slice of that side what the neighbour on that side needs:
 *     populations: [n_cross][ny][nx] dtype, the populations leaving through that face (c_z = -1 on the low side, +1 on the high
 *                  side) in ascending population order, as stored (post-collision F_t: call it after stage 1);
 *     u^:          [3][ny][nx] dtype (after stage 0 of an HRR step).
 * lbm_halo_unpack writes a buffer packed by the neighbour (its pack of the OPPOSITE side) into the GHOST slice of that side.
 * lbm_query(ctx, 9 | 10) gives the number of values of a populations / u^ face buffer.  Host or device buffers (device buffers
 * are used in place, asynchronously on the context's stream; host buffers synchronise).
 * Errors: LBM_EINVAL (NULL, bad what / side), LBM_ESTATE (no ghost slice on that side, no state, no u^ field yet), LBM_ENOMEM, LBM_ECUDA. */
int lbm_halo_pack(lbm_ctx* ctx, int what, int side, void* buf);
int lbm_halo_unpack(lbm_ctx* ctx, int what, int side, const void* buf);

/* Use `cuda_stream` (a cudaStream_t passed as void*) for all subsequent work; NULL = the legacy default stream (also the
 * stream of a fresh context).  Synchronises the old stream first.  PyTorch owns streams in this build (north_star: "PyTorch
 * used only for device memory and streams"): pass torch.cuda.current_stream().cuda_stream.  Errors: LBM_EINVAL (NULL ctx),
 * LBM_ECUDA. */
int lbm_set_stream(lbm_ctx* ctx, void* cuda_stream);

/* Block until everything enqueued so far has finished; returns LBM_ECUDA if any kernel failed. */
int lbm_synchronize(lbm_ctx* ctx);

/* Static or ctx-owned message of the last error; valid until the next call on that ctx.
 * ctx == NULL returns the message of the last failed lbm_create or lbm_totals_static. */
const char* lbm_last_error(const lbm_ctx* ctx);

/* Introspection used by the harness.  what:
 *   0 steps taken since the last set_fields/init      1 kernels launched by this ctx so far (graph replays count their kernels)
 *   2 number of cells N                                3 number of wall cells (SOLID, MOVINGWALL, SLIPWALL)
 *   4 device bytes owned by the ctx                    5 cells on the masked (boundary) path
 *   6 cells handled by the list blocks of the vector kernel (SPECIAL cells + their sector mates)
 *   7 CUDA graph launches so far                       8 WALLMODEL cells (length of the pre-pass list)
 *   9 values of a populations face buffer (halo)        10 values of a u^ face buffer (halo)
 *   11 interior z-slices (nz minus the ghost slices)   12 cells with a slip plane code (slip-adjacent cells in the vector path)
 * Returns -1 for an unknown `what` or a NULL ctx. */
long long lbm_query(const lbm_ctx* ctx, int what);

/* Tuning knobs.  None changes what is computed: "cuda_graph", "pdl", "serpentine", "block_threads", "hrr_slab", "totals_waves"
 * and "inplace" are schedules / storage schemes (A/B tests compare the populations bit for bit); "wm_prepass", "slip_planes" and
 * "vector" route some cells through another kernel body with the same arithmetic (tested against each other to rounding and
 * against the oracle to the parity tolerance).  Returns LBM_EINVAL for an unknown key or value, LBM_ESTATE where noted.  Keys
 * (every key the library accepts is listed here):
 *   "cuda_graph"    0|1     1: lbm_step replays the steady-state time loop 8 steps at a time from a captured CUDA graph
 *                           (re-captured when parameters, fields or options change); steps that do not fill a chunk, the first
 *                           step of a fresh state, runs with the Vortex Method inlet and sub-domains use plain launches.
 *                           Default 0: beside "pdl" it measured neutral (config 1: 4.4 -> 4.2 us per step, everything else
 *                           within noise), and a capture that lands in a caller's timed region costs more than it wins
 *   "pdl"           0|1|2   programmatic dependent launch of the time-loop kernels: 0 plain launches; 1 every kernel becomes
 *                           resident while its predecessor drains and waits for it; 2 (default) additionally, after the
 *                           wall-model pre-pass only the threads that read its output wait for it
 *   "wm_prepass"    0|1     1 (default): WALLMODEL cells run in the vector path, their u^B comes from a pre-pass over their
 *                           compact list; 0: they are solved cell by cell in the list blocks of the step kernel.  Decides how
 *                           flags are classified: LBM_ESTATE once a state or geometry has been set
 *   "slip_planes"   0|1     1 (default): cells next to ONE plane slip wall normal to y or z (and nothing else that complicates the
 *                           specular pull) run in the vector path, pulling the reflected populations from their own plane; 0: every
 *                           cell next to a slip wall is handled cell by cell in the list blocks.  Decides how flags are
 *                           classified: LBM_ESTATE once a state or geometry has been set
 *   "totals_waves"  n       lbm_totals runs n whole waves of resident blocks (1 .. 64), each block looping over the z-slices; 0 (default):
 *                           chosen from the lattice size (about 8 z-iterations per block, 1 .. 16 waves)
 *   "serpentine"    0|1     consecutive launches sweep the z-slices in opposite directions for L2 reuse (default 1)
 *   "inplace"       0|1     1: a lattice of plain fluid cells, with or without resting SOLID cells (halfway bounce-back) but without
 *                           any inlet / outlet / wall-model / moving / slip cell, BGK form, steps IN PLACE on one array (AA pattern:
 *                           even steps collide locally into the opposite slots, odd steps pull and push through the
 *                           neighbours); the second lattice is then never
 *                           allocated unless a state read after an odd number of steps needs it.  Default 0 (two lattices)
 *   "vector"        0|1     0 forces the scalar kernel (one cell per thread) for every row length (default 1)
 *   "block_threads" 64|128|256   threads per block of the step kernels (default 64)
 *   "hrr_slab"      n >= 0  HRR form: interleave the u^ pass and the step pass in slabs of n z-slices (0 = whole lattice, default) */
int lbm_set_option(lbm_ctx* ctx, const char* key, long long value);

#ifdef __cplusplus
}
#endif
#endif /* PAPER_2506_21804_B200_LBM_H */
