// =====================================================================================
// lbm_launch.cuh -- launch side of the step kernels: argument block, grid shapes, the sequence of launches that makes
// one time step in each collision form.  Included by lbm_inst.cu only (one object file per lattice, dtype and part).
// =====================================================================================
#pragma once
#include "lbm_ctx.h"
#include "lbm_kernels.cuh"

namespace lbmhost {

struct DiagOut {           // A9 outputs of a MODE_MOMENTS_* launch (device pointers; either may be null)
  void* rho;
  void* u;
};

inline void launch_dims(const lbm_ctx* c, dim3& grid, dim3& block) {
  int bx = 1;
  while (bx < c->nx && bx < c->block_threads) bx <<= 1;
  int by = c->block_threads / bx;
  int ny2 = 1;
  while (ny2 < c->ny) ny2 <<= 1;
  if (by > ny2) by = ny2;
  if (by < 1) by = 1;
  if (bx * by < 32) by = 32 / bx;   // whole warps only: the reductions use full-mask shuffles
  block = dim3(bx, by, 1);
  grid = dim3((c->nx + bx - 1) / bx, (c->ny + by - 1) / by, c->nz);
}

// does this step run the wall-model pre-pass (A8)?
inline bool wm_prepass_active(const lbm_ctx* c, const lbm_params* p) {
  return p && p->wm_enable && c->wm_prepass && c->n_wm > 0 && c->wm_ub != nullptr;
}

template <typename T>
lbm::StepArgs<T> make_args(const lbm_ctx* c, const lbm_params* p, int in, int out) {
  lbm::StepArgs<T> a;
  a.fin = static_cast<const T*>(c->f[in]);
  a.fout = static_cast<T*>(c->f[out]);
  a.d = (p && p->use_hlbm && c->has_d) ? static_cast<const T*>(c->d) : nullptr;
  a.ub = (a.d != nullptr && c->ub) ? static_cast<const T*>(c->ub) : nullptr;
  a.cls = c->cls;
  a.nbmask = c->nbmask;
  a.nx = c->nx;  a.ny = c->ny;  a.nz = c->nz;
  a.N = c->N;
  a.list = c->list;
  a.n_list = static_cast<int>(c->n_list);
  a.list_z = 0;
  a.z_reverse = 0;
  a.z0 = 0;
  a.nzs = c->nz;
  a.zi0 = zlo(c);
  a.zi1 = zlo(c) + zcount(c);
  a.uhat = static_cast<T*>(c->uhat);
  a.uhat_out = nullptr;
  if (c->lag_active) {                 // collision = 2: read the previous level's u^, write this level's
    a.uhat = static_cast<T*>(c->lag_cur == 0 ? c->uhat : c->uhat2);
    a.uhat_out = static_cast<T*>(c->lag_cur == 0 ? c->uhat2 : c->uhat);
  }
  a.sigma = p ? static_cast<T>(p->sigma) : T(1);
  for (int k = 0; k < 3; ++k) a.u_wall[k] = p ? static_cast<T>(p->u_wall[k]) : T(0);
  a.rho_out = (p && p->rho_out > 0.0) ? static_cast<T>(p->rho_out) : T(1);
  a.fringe_k = T(0);
  a.fringe_x0 = c->nx;
  if (p && p->fringe_len > 0 && p->fringe_factor > 0.0) {
    a.fringe_k = static_cast<T>((p->tau0 - 0.5) * p->fringe_factor / (static_cast<double>(p->fringe_len) * p->fringe_len));
    a.fringe_x0 = c->nx - 1 - p->fringe_len;
  }
  a.uin_field = c->uin_mean ? c->uin_field[c->uin_cur] : nullptr;
  if (p) {
    a.tau0 = static_cast<T>(p->tau0);
    a.smago_k = static_cast<T>(18.0 * 1.4142135623730951 * p->cs_smago * p->cs_smago);
    a.u_in[0] = static_cast<T>(p->u_in[0]);  a.u_in[1] = static_cast<T>(p->u_in[1]);  a.u_in[2] = static_cast<T>(p->u_in[2]);
    a.wm_enable = p->wm_enable;
    a.wm_kappa = p->wm_kappa;  a.wm_E = p->wm_E;
    a.nu = (p->tau0 - 0.5) / 3.0;
  } else {
    a.tau0 = T(1);  a.smago_k = T(0);
    a.u_in[0] = a.u_in[1] = a.u_in[2] = T(0);
    a.wm_enable = 0;  a.wm_kappa = 0.41;  a.wm_E = 9.8;  a.nu = 1.0 / 6.0;
  }
  a.wm_ub = wm_prepass_active(c, p) ? static_cast<T*>(c->wm_ub) : nullptr;
  a.wm_list = c->wm_list;
  a.n_wm = static_cast<int>(c->n_wm);
  a.pdl_wait_all = 1;
  a.mom_rho = nullptr;  a.mom_u = nullptr;
  a.tot_out = c->totals_dev;
  a.tot_slots = c->totals_dev + 8;
  a.tot_ticket = reinterpret_cast<unsigned*>(c->totals_dev + 8 + 5 * LBM_TOT_SLOTS);
  a.tot_nslots = LBM_TOT_SLOTS;
  return a;
}

// vector kernel: thread <-> V consecutive cells; block (bx quads, by rows)
template <int Q, typename T, int COLL>
void launch_dims_vec(const lbm_ctx* c, dim3& grid, dim3& block) {
  const int V = lbm::VecOf<Q, T, COLL>::V;
  const int nvec = c->nx / V;
  int bx = 1;
  while (bx < nvec && bx < 32) bx <<= 1;
  int by = c->block_threads / bx;
  int ny2 = 1;
  while (ny2 < c->ny) ny2 <<= 1;
  if (by > ny2) by = ny2;
  if (bx * by < 32) by = 32 / bx;
  block = dim3(bx, by, 1);
  grid = dim3((nvec + bx - 1) / bx, (c->ny + by - 1) / by, c->nz);
}

// kernel launch with (pdl) or without the programmatic-serialization attribute
template <typename Kern, typename Args>
cudaError_t launch_k(Kern kern, dim3 grid, dim3 block, cudaStream_t st, bool pdl, const Args& a) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = 0;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, a);
}

// One launch of a step kernel over the z-slices [z0, z0 + nzs) (+ the list blocks when with_list), lattice `in` -> `out`.
template <int Q, typename T, int MODE, int COLL>
int launch_one(lbm_ctx* c, const lbm_params* p, int in, int out, int z0, int nzs, bool with_list, bool may_meet_lid = true,
               const DiagOut* diag = nullptr) {
  dim3 grid, block;
  lbm::StepArgs<T> a = make_args<T>(c, p, in, out);
  a.z0 = z0;
  a.nzs = nzs;
  if (diag) {
    a.mom_rho = static_cast<T*>(diag->rho);
    a.mom_u = static_cast<T*>(diag->u);
  }
  // serpentine sweep (lbm_set_option "serpentine", default 1): BGK steps alternate their direction with the time level; in the
  // HRR form the u^ pass runs downwards and the step pass upwards; a diagnostic pass runs against the last step
  // (collision = 2 has no u^ pass: its fused steps alternate like the BGK steps)
  if (c->serpentine) a.z_reverse = lbm::mode_uhat(MODE) ? 1 : ((COLL == lbm::COLL_HRR && !c->lag_active) ? 0 : static_cast<int>(c->sweep_count & 1));
  // programmatic dependent launch for the kernels of the time loop: resident while the predecessor drains.  After the wall-model
  // pre-pass (which itself waited for the lattice) only the threads that read its output wait ("pdl" = 2).
  const bool timeloop = lbm::mode_collides(MODE) || lbm::mode_uhat(MODE);
  const bool pdl = timeloop && c->use_pdl > 0;
  a.pdl_wait_all = (pdl && c->use_pdl == 2 && c->prev_launch_prepass) ? 0 : 1;
  c->prev_launch_prepass = false;
  const bool vec = c->use_vector && (c->nx % (32 / static_cast<int>(sizeof(T))) == 0);   // whole 32-byte sectors per row
  cudaError_t e;
  if (vec) {
    launch_dims_vec<Q, T, COLL>(c, grid, block);
    a.list_z = 0;
    if (with_list) {
      const long long per_slice = static_cast<long long>(grid.x) * grid.y * block.x * block.y;
      a.list_z = static_cast<int>((c->n_list + per_slice - 1) / per_slice);
    }
    grid.z = nzs + a.list_z;
    if (grid.z == 0) return LBM_OK;
    if constexpr (lbm::mode_totals(MODE)) {
      // every block loops over the z-slices (one reduction per block); the grid is a whole number of waves of resident blocks (a
      // partly filled last wave of these long blocks would cost up to a wave: 2.19 waves measured 0.165 ms on config 3)
      int per_sm = 8, dev = 0, sms = 148;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lbm::k_step_vec<Q, T, MODE, COLL, 0>, block.x * block.y, 0) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 8;
      }
      const unsigned per_slice = grid.x * grid.y;
      int waves = c->totals_waves;          // 0 = auto: about 8 z-iterations per block, 1 .. 16 waves (measured: config 3 best at 1 - 4,
      if (waves <= 0) {                     // 256^3 at 4, 512^3 at 16)
        const long long all = static_cast<long long>(per_slice) * grid.z;
        waves = static_cast<int>(all / (8ll * per_sm * sms));
        waves = waves < 1 ? 1 : (waves > 16 ? 16 : waves);
      }
      unsigned want = static_cast<unsigned>(per_sm * sms * waves) / per_slice;
      if (want < 1) want = 1;
      if (grid.z > want) grid.z = want;
    }
    if (grid.z > 65535u || grid.y > 65535u)
      return fail(c, LBM_EINVAL, "lattice does not fit the launch grid (nz + list slices = %u, rows = %u; both must be <= 65535)", grid.z, grid.y);
    int wv = 0;      // kernel variant: bit 0 = the launch may meet the moving lid, bit 1 = cells with a slip plane code
    if constexpr (lbm::mode_pulls(MODE)) wv = ((c->n_moving > 0 && may_meet_lid) ? 1 : 0) | ((c->n_slipcode > 0) ? 2 : 0);
    if constexpr (lbm::mode_pulls(MODE)) {
      switch (wv) {
        case 1:  e = launch_k(lbm::k_step_vec<Q, T, MODE, COLL, 1>, grid, block, c->stream, pdl, a); break;
        case 2:  e = launch_k(lbm::k_step_vec<Q, T, MODE, COLL, 2>, grid, block, c->stream, pdl, a); break;
        case 3:  e = launch_k(lbm::k_step_vec<Q, T, MODE, COLL, 3>, grid, block, c->stream, pdl, a); break;
        default: e = launch_k(lbm::k_step_vec<Q, T, MODE, COLL, 0>, grid, block, c->stream, pdl, a); break;
      }
    } else {
      e = launch_k(lbm::k_step_vec<Q, T, MODE, COLL, 0>, grid, block, c->stream, pdl, a);
    }
  } else {
    if (nzs == 0) return LBM_OK;
    launch_dims(c, grid, block);
    grid.z = nzs;
    e = launch_k(lbm::k_step<Q, T, MODE, COLL>, grid, block, c->stream, pdl, a);
  }
  if (e != cudaSuccess) return fail(c, LBM_ECUDA, "kernel launch (mode %d): %s", MODE, cudaGetErrorString(e));
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  return LBM_OK;
}

// A8: u^B of the wall-model cells of this time level (no-op when the step does not use the pre-pass)
template <int Q, typename T, bool PULL>
int launch_prepass(lbm_ctx* c, const lbm_params* p, int in, int out) {
  if (!wm_prepass_active(c, p)) return LBM_OK;
  lbm::StepArgs<T> a = make_args<T>(c, p, in, out);
  const unsigned blocks = static_cast<unsigned>((c->n_wm + 127) / 128);
  cudaError_t e = launch_k(lbm::k_wallmodel_prepass<Q, T, PULL>, dim3(blocks), dim3(128), c->stream, c->use_pdl > 0, a);
  if (e != cudaSuccess) return fail(c, LBM_ECUDA, "wall-model pre-pass launch: %s", cudaGetErrorString(e));
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  c->prev_launch_prepass = true;
  return LBM_OK;
}

// HRR form (Eq. 7-11): the FD strain (Eq. 10) needs u^(x,t) of the six neighbours, i.e. their streamed populations, so
// a step is two passes: UHAT (pull, moments, Eq. 12 -> u^ field) and the fused step that reads it.  With "hrr_slab" the
// passes are interleaved slab by slab in z, the UHAT pass one slice ahead (measured slower, default off).
// The list cells go with the first UHAT launch and the last step launch.
template <int Q, typename T, int MODE_U, int MODE_S>
int launch_hrr_t(lbm_ctx* c, const lbm_params* p, int in, int out, int stage) {
  const int nz = c->nz;
  const bool halo = (c->ghost_lo + c->ghost_hi) > 0;
  int slab = (c->hrr_slab > 0 && !halo) ? c->hrr_slab : nz;
  int rc = LBM_OK;
  if (p->collision == LBM_COLLISION_HRR_LAG) {
    // G41: one pass per step.  Without history (fresh state) the u^ pass forms u^(., t) once, in buffer 0, whose copy gives buffer 1
    // its wall entries; from then on the fused step reads the buffer the previous step wrote and writes the other one.
    // On a sub-domain (stages): stage 0 = pre-pass (+ the u^ pass of a fresh history); the caller then exchanges the boundary slices
    // of the buffer the fused step is about to read (lbm_halo_pack / unpack with LBM_HALO_UHAT); stage 1 = the fused step.
    if (stage != 1) {
      rc = launch_prepass<Q, T, lbm::mode_pulls(MODE_U)>(c, p, in, out);
      if (rc != LBM_OK) return rc;
      if (!c->lag_valid) {
        rc = launch_one<Q, T, MODE_U, lbm::COLL_BGK>(c, p, in, out, zlo(c), zcount(c), true);
        if (rc != LBM_OK) return rc;
        LBM_CUDA(c, cudaMemcpyAsync(c->uhat2, c->uhat, 3 * static_cast<size_t>(c->N) * sizeof(T), cudaMemcpyDeviceToDevice, c->stream));
        c->lag_cur = 0;
        c->lag_valid = true;             // (the history of this step: u^ of its own level)
      }
      if (stage == 0) return LBM_OK;
    }
    c->lag_active = true;
    rc = launch_one<Q, T, MODE_S, lbm::COLL_HRR>(c, p, in, out, zlo(c), zcount(c), true);
    c->lag_active = false;
    if (rc != LBM_OK) return rc;
    c->lag_cur = 1 - c->lag_cur;
    c->lag_valid = true;
    return LBM_OK;
  }
  // stages of a step on a sub-domain (lbm_step_halo): 0 = pre-pass + u^ pass (the caller then exchanges the u^ boundary
  // slices), 1 = the fused step pass; stage < 0: the whole step
  if (stage != 1) rc = launch_prepass<Q, T, lbm::mode_pulls(MODE_U)>(c, p, in, out);
  if (rc != LBM_OK) return rc;
  if (slab >= nz - 1) {
    if (stage != 1) rc = launch_one<Q, T, MODE_U, lbm::COLL_BGK>(c, p, in, out, zlo(c), zcount(c), true);
    if (rc != LBM_OK || stage == 0) return rc;
    return launch_one<Q, T, MODE_S, lbm::COLL_HRR>(c, p, in, out, zlo(c), zcount(c), true);
  }
  // UHAT: slice nz-1 first (the periodic neighbour of slice 0), then [0, slab], [slab+1, 2 slab], ... up to nz-2
  rc = launch_one<Q, T, MODE_U, lbm::COLL_BGK>(c, p, in, out, nz - 1, 1, true);
  if (rc != LBM_OK) return rc;
  int udone = 0;                       // slices [0, udone) have their u^
  for (int z0 = 0; z0 < nz; z0 += slab) {
    const int zend = (z0 + slab < nz) ? z0 + slab : nz;          // step pass covers [z0, zend)
    int uneed = (zend + 1 < nz - 1) ? zend + 1 : nz - 1;         // needs u^ on [z0 - 1, zend]; nz-1 is done
    if (uneed > udone) {
      rc = launch_one<Q, T, MODE_U, lbm::COLL_BGK>(c, p, in, out, udone, uneed - udone, false);
      if (rc != LBM_OK) return rc;
      udone = uneed;
    }
    rc = launch_one<Q, T, MODE_S, lbm::COLL_HRR>(c, p, in, out, z0, zend - z0, zend == nz);
    if (rc != LBM_OK) return rc;
  }
  return LBM_OK;
}

// The timed BGK step.  With a moving lid (MOVINGWALL cells live on the plane z = nz-1 only) the slices that can meet it
// (z = nz-2, nz-1 and, through the periodic wrap, 0) take the kernel variant that looks the neighbour's class up; the bulk
// runs the plain variant: three launches instead of one.
template <int Q, typename T>
int launch_bgk_pull_t(lbm_ctx* c, const lbm_params* p, int in, int out) {
  const int nz = c->nz;
  int rc = launch_prepass<Q, T, true>(c, p, in, out);
  if (rc != LBM_OK) return rc;
  const int z0 = zlo(c), z1 = zlo(c) + zcount(c);            // interior slices [z0, z1)
  if (c->n_moving == 0 || nz < 8)
    return launch_one<Q, T, lbm::MODE_STREAM_COLLIDE, lbm::COLL_BGK>(c, p, in, out, z0, z1 - z0, true);
  // [1, nz-2) plain, [nz-2, nz) and [0, 1) on the variant that looks for the lid, each clipped to the interior
  auto piece = [&](int a, int b, bool with_list, bool lid) {
    a = a < z0 ? z0 : a;
    b = b > z1 ? z1 : b;
    if (b <= a && !with_list) return static_cast<int>(LBM_OK);
    return launch_one<Q, T, lbm::MODE_STREAM_COLLIDE, lbm::COLL_BGK>(c, p, in, out, a, b > a ? b - a : 0, with_list, lid);
  };
  rc = piece(1, nz - 2, true, false);
  if (rc == LBM_OK) rc = piece(nz - 2, nz, false, true);
  if (rc == LBM_OK) rc = piece(0, 1, false, true);
  return rc;
}

inline void step_done(lbm_ctx* c) {
  c->cur = 1 - c->cur;
  c->sweep_count++;
}

#if LBM_INST_PART == 0
template <int Q, typename T>
int launch_step_bgk(lbm_ctx* c, const lbm_params* p, int mode) {
  const int in = c->cur, out = 1 - c->cur;
  int rc;
  switch (mode) {
    case lbm::MODE_COLLIDE:
      rc = launch_prepass<Q, T, false>(c, p, in, out);
      if (rc == LBM_OK) rc = launch_one<Q, T, lbm::MODE_COLLIDE, lbm::COLL_BGK>(c, p, in, out, zlo(c), zcount(c), true);
      break;
    case lbm::MODE_STREAM_COLLIDE:
      rc = launch_bgk_pull_t<Q, T>(c, p, in, out);
      break;
    default:
      rc = launch_one<Q, T, lbm::MODE_STREAM, lbm::COLL_BGK>(c, p, in, out, zlo(c), zcount(c), true);
      break;
  }
  if (rc != LBM_OK) return rc;
  step_done(c);
  return LBM_OK;
}

template <int Q, typename T>
int launch_init(lbm_ctx* c, const void* rho, const void* u) {
  const int threads = 256;
  const long long blocks = (c->N + threads - 1) / threads;
  lbm::k_init_equilibrium<Q, T><<<static_cast<unsigned>(blocks), threads, 0, c->stream>>>(
      static_cast<const T*>(rho), static_cast<const T*>(u), static_cast<T*>(c->f[0]), c->N);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  return LBM_OK;
}
#endif

#if LBM_INST_PART == 1
template <int Q, typename T>
int launch_step_hrr(lbm_ctx* c, const lbm_params* p, int mode, int stage) {
  const int in = c->cur, out = 1 - c->cur;
  int rc = (mode == lbm::MODE_COLLIDE) ? launch_hrr_t<Q, T, lbm::MODE_UHAT_PRE, lbm::MODE_COLLIDE>(c, p, in, out, stage)
                                       : launch_hrr_t<Q, T, lbm::MODE_UHAT_PULL, lbm::MODE_STREAM_COLLIDE>(c, p, in, out, stage);
  if (rc != LBM_OK) return rc;
  if (stage != 0) step_done(c);
  return LBM_OK;
}
#endif

#if LBM_INST_PART == 3
// In-place AA pattern (propagation bake-off): one launch per step on the current lattice alone.
// odd = 0: even step (plain layout -> swapped slots), 1: odd step (swapped -> plain), 2: un-swap into the other lattice.
template <int Q, typename T>
int launch_aa(lbm_ctx* c, const lbm_params* p, int kind) {
  constexpr int V = lbm::VecOf<Q, T, lbm::COLL_BGK>::V;
  if (kind == 2) {
    dim3 grid, block;
    launch_dims(c, grid, block);
    lbm::k_aa_unswap<Q, T><<<grid, block, 0, c->stream>>>(static_cast<const T*>(c->f[c->cur]), static_cast<T*>(c->f[1 - c->cur]), c->nx, c->ny, c->nz, c->N,
                                                         c->cls, c->nbmask);
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
    c->cur = 1 - c->cur;
    return LBM_OK;
  }
  lbm::StepArgs<T> sa = make_args<T>(c, p, c->cur, c->cur);
  lbm::AAArgs<T> a;
  a.a = static_cast<T*>(c->f[c->cur]);
  a.d = sa.d;  a.ub = sa.ub;
  a.cls = c->cls;  a.nbmask = c->nbmask;
  const bool walls = c->n_solid > 0;     // SOLID cells with halfway bounce-back (nothing else: inplace_eligible)
  a.nx = c->nx;  a.ny = c->ny;  a.nz = c->nz;  a.N = c->N;
  a.tau0 = sa.tau0;  a.smago_k = sa.smago_k;  a.fringe_k = sa.fringe_k;  a.fringe_x0 = sa.fringe_x0;
  const int nvec = c->nx / V;
  if (kind == 0) {
    dim3 grid, block;
    launch_dims_vec<Q, T, lbm::COLL_BGK>(c, grid, block);
    if (walls) lbm::k_aa_even<Q, T, true><<<grid, block, 0, c->stream>>>(a);
    else       lbm::k_aa_even<Q, T, false><<<grid, block, 0, c->stream>>>(a);
  } else {
    int by = 64 / nvec;
    if (by < 1) by = 1;
    dim3 block(nvec, by, 1), grid(1, (c->ny + by - 1) / by, c->nz);
    if (walls) lbm::k_aa_odd<Q, T, true><<<grid, block, 0, c->stream>>>(a);
    else       lbm::k_aa_odd<Q, T, false><<<grid, block, 0, c->stream>>>(a);
  }
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  c->sweep_count++;
  return LBM_OK;
}
#endif

#if LBM_INST_PART == 2
// A9: rho, u of S_t for every cell: one launch of the step kernel in its moments mode (the pull happens in registers; the
// stored lattice and the phase stay as they are) + the wall cells' own values from their side buffer.
template <int Q, typename T>
int launch_moments(lbm_ctx* c, const lbm_params* p, void* rho, void* u) {
  const DiagOut out = {rho, u};
  int rc = (c->phase == PHASE_POST)
               ? launch_one<Q, T, lbm::MODE_MOMENTS_PULL, lbm::COLL_BGK>(c, p, c->cur, 1 - c->cur, zlo(c), zcount(c), true, true, &out)
               : launch_one<Q, T, lbm::MODE_MOMENTS_PRE, lbm::COLL_BGK>(c, p, c->cur, 1 - c->cur, zlo(c), zcount(c), true, true, &out);
  if (rc != LBM_OK) return rc;
  if (c->n_solid_list > 0) {
    const unsigned blocks = static_cast<unsigned>((c->n_solid_list + 255) / 256);
    lbm::k_solid_moments<Q, T><<<blocks, 256, 0, c->stream>>>(static_cast<const T*>(c->solid_vals), c->solid_list, c->n_solid_list, c->N,
                                                              static_cast<T*>(rho), static_cast<T*>(u));
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
  }
  return LBM_OK;
}

// A9: totals over the non-wall cells of S_t -> c->totals_dev[0..4]: one launch (block partials -> slots -> last block)
template <int Q, typename T>
int launch_totals(lbm_ctx* c, const lbm_params* p) {
  return (c->phase == PHASE_POST)
             ? launch_one<Q, T, lbm::MODE_TOTALS_PULL, lbm::COLL_BGK>(c, p, c->cur, 1 - c->cur, zlo(c), zcount(c), true)
             : launch_one<Q, T, lbm::MODE_TOTALS_PRE, lbm::COLL_BGK>(c, p, c->cur, 1 - c->cur, zlo(c), zcount(c), true);
}
#endif

}  // namespace lbmhost
