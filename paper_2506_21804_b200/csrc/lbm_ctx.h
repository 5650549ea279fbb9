// =====================================================================================
// lbm_ctx.h -- host-side state of one context and the launchers the API calls.
// The launchers are templates on (lattice Q, dtype T); they are defined in lbm_launch.cuh and instantiated in
// lbm_inst.cu, one object file per (Q, T, part), so that the step kernels compile in parallel.  No arithmetic
// of the method lives on the host side.
// =====================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lbm.h"

enum Phase { PHASE_NONE = 0,   // no state yet
             PHASE_PRE = 1,    // cur holds S_t (pre-collision), as handed in
             PHASE_POST = 2,   // cur holds F_{t-1} (post-collision, not yet streamed); S_t = stream(F_{t-1})
             PHASE_SWAPPED = 3 }; // in-place (AA) stepping after an odd number of steps: cur holds F_{t-1,i}(x) in slot opp(i)

constexpr int LBM_TOT_SLOTS = 256;      // partial-sum slots of the totals reduction (spreads the atomics)
constexpr int LBM_GRAPH_CHUNK = 8;      // time steps per captured CUDA graph (even: lattice roles and sweep direction return)
constexpr int LBM_GRAPH_CACHE = 4;      // one graph per (current lattice, sweep parity)

struct lbm_graph_entry {
  cudaGraphExec_t exec;
  lbm_params params;
  long long epoch;
  long long launches;    // kernels in the graph
  int cur, sweep_parity;
  bool valid;
};

struct lbm_ctx {
  int Q, nx, ny, nz, dtype;
  long long N;
  void* f[2];            // two population lattices, [Q][N] each
  void* d;               // porosity [N]
  bool has_d;
  uint8_t* cls;          // class byte per cell (see lbm_kernels.cuh)
  uint8_t* cls_alt;      // classification target before it is accepted
  uint8_t* flags_raw;    // device copy of the caller's flag bytes; afterwards the list marks
  uint32_t* nbmask;      // per cell: which lattice neighbours are SOLID (read-side bounce-back)
  int* solid_list;       // SOLID cells, ascending
  void* solid_vals;      // their own populations [Q][n_solid] (the step kernels write zeros over their lattice slots)
  long long n_solid_list;
  int* list;             // cells of the non-bulk vectors (vector kernel), ascending
  long long n_list;
  int* wm_list;          // WALLMODEL cells, ascending (wall-model pre-pass)
  long long n_wm;
  void* wm_ub;           // u^B of the wall-model cells [3][N] sparse: written by the pre-pass, read by the step kernel
  void* cub_tmp;
  size_t cub_tmp_bytes;
  int* list_count_dev;
  unsigned long long* counters;  // device [8]
  long long n_moving, n_slip;    // MOVINGWALL / SLIPWALL cells of the accepted geometry
  long long n_typed;             // non-wall cells of a type other than FLUID (inlet, outlet, wall model, ...)
  bool solid_dirty;              // in-place steps ran over wall cells' slots: their own values must be put back before the lattice is read
  long long n_slipcode;          // cells next to a plane slip wall that run in the vector path (slip plane code in their class byte)
  double* totals_dev;            // device [5] result + [LBM_TOT_SLOTS][5] partial sums + ticket counter
  void* staging;         // host<->device bounce buffer, grown on demand
  size_t staging_bytes;
  int cur;
  Phase phase;
  long long steps, launches, n_solid, n_masked;
  size_t device_bytes;
  cudaStream_t stream;
  int block_threads;
  int use_vector;        // 1: 128-bit vector kernel when nx % (32/dtype) == 0 (default); 0: scalar kernel
  int use_graph;         // 1: lbm_step replays captured CUDA graphs of LBM_GRAPH_CHUNK steps (default 0)
  cudaStream_t cap_stream;   // capture happens on a private stream (the caller's may be the legacy default stream)
  lbm_graph_entry graphs[LBM_GRAPH_CACHE];
  long long epoch;       // bumped whenever something baked into a captured graph changes (geometry, fields, options)
  long long graph_launches;
  // Vortex Method inlet / per-cell inflow field (lbm_set_inflow, lbm_set_vortices)
  double* uin_mean;      // [3][nz][ny] fp64 (whatever the dtype), nullptr = uniform params.u_in
  double* uin_field[2];  // inflow of the current / the previous time level, fp64
  float* uin_scratch;    // fp32 <-> fp64 conversion scratch of lbm_set_inflow / lbm_get_inflow (never touched by the side stream)
  int uin_cur;
  long long inflow_index;   // the time level t the current inflow field belongs to (S_t carries it)
  int nv;
  double* vpos;  double* vsign;  double* vgamma;     // device [nv][2], [nv], [nv]
  double vm_sigma, vm_intensity;
  bool gamma_dirty;
  // the inflow of level t+1 depends on the inflow of level t only, never on the lattice: it is formed on a side stream while
  // step t runs (events order the two streams; two field buffers)
  cudaStream_t vm_stream;
  cudaEvent_t ev_vm, ev_step[2];
  bool vm_pending;          // the newest field is still being written on vm_stream
  long long ev_step_level[2];   // time level of the step after which ev_step[k] was recorded (-1: never)
  void* ub;              // prescribed solid velocity u^B [3][N] (lbm_set_body_velocity), nullptr = 0 everywhere
  void* uhat;            // HRR form: u^(x,t) [3][N], allocated on the first HRR step
  // collision = 2 (G41): two u^ buffers (uhat, uhat2); buffer lag_cur holds u^ of the previous level while lag_valid; lag_active: the
  // launch being prepared is the fused step of that form (make_args hands the two buffers to the kernel)
  void* uhat2;
  bool lag_valid, lag_active;
  int lag_cur;
  double lag_u_wall[3];  // lid velocity the walls' u^ entries were written with
  int serpentine;        // 1: consecutive launches sweep z in opposite directions (L2 reuse)
  long long sweep_count; // BGK steps launched so far (parity = direction)
  int hrr_slab;          // HRR form: z-slices per slab of the two-pass step (0 = whole lattice)
  int inplace;           // 1: lattices without any boundary cell step in place (AA pattern), one lattice (option "inplace")
  int slip_planes;       // 1: cells next to a plane slip wall normal to y or z get a slip plane code and run in the vector path (default)
  int totals_waves;      // lbm_totals: waves of resident blocks in the grid (every block loops over z); 0 = auto
  int wm_prepass;        // 1: wall-model cells run in the vector path, u^B from a pre-pass over their compact list (default)
  int use_pdl;           // programmatic dependent launch of the time-loop kernels: 0 off, 1 every thread waits for the predecessor,
                         // 2 (default) after the wall-model pre-pass only the threads that read its output wait
  bool prev_launch_prepass;   // the last kernel enqueued on the stream was the wall-model pre-pass
  // slab decomposition in z (lbm_set_halo): the first ghost_lo / last ghost_hi slices (0 or 1 each) are ghost slices that hold
  // copies of the neighbouring sub-domain's boundary slices (lbm_halo_unpack); every pass covers the interior slices only
  int ghost_lo, ghost_hi;
  long long halo_wm_epoch;   // epoch at which the wall-model cells were last checked against the cuts
  int halo_stage;        // lbm_step_halo: 0 = a step may begin, 1 = stage 0 of the current step is done
  void* halo_buf;        // device staging of lbm_halo_pack / lbm_halo_unpack for host buffers
  size_t halo_buf_bytes;
  lbm_params last;       // parameters of the last lbm_step: the inlet rule is part of how S_t is formed from F_{t-1}
  char err[512];
};

namespace lbmhost {

// interior slices [zlo, zlo + zcount) of the local lattice (all of it without ghost slices)
inline int zlo(const lbm_ctx* c) { return c->ghost_lo; }
inline int zcount(const lbm_ctx* c) { return c->nz - c->ghost_lo - c->ghost_hi; }

int fail(lbm_ctx* c, int code, const char* fmt, ...);

#define LBM_CUDA(c, call)                                                                                       \
  do {                                                                                                          \
    cudaError_t e_ = (call);                                                                                    \
    if (e_ != cudaSuccess) return lbmhost::fail((c), LBM_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));       \
  } while (0)

// one time step (or one materialising pass) in the BGK / HRR form; `mode` is a lbm:: MODE_* value
template <int Q, typename T> int launch_step_bgk(lbm_ctx* c, const lbm_params* p, int mode);
template <int Q, typename T> int launch_step_hrr(lbm_ctx* c, const lbm_params* p, int mode, int stage);
// A9: rho, u of S_t into caller buffers (device pointers); totals into c->totals_dev[0..4]
template <int Q, typename T> int launch_moments(lbm_ctx* c, const lbm_params* p, void* rho, void* u);
template <int Q, typename T> int launch_totals(lbm_ctx* c, const lbm_params* p);
template <int Q, typename T> int launch_init(lbm_ctx* c, const void* rho, const void* u);
// in-place AA pattern: kind 0 even step, 1 odd step, 2 un-swap into the other lattice (which becomes current)
template <int Q, typename T> int launch_aa(lbm_ctx* c, const lbm_params* p, int kind);

}  // namespace lbmhost
