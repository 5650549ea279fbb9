// =====================================================================================
// lbm_api.cu -- host side of the C ABI declared in include/lbm.h.
// Argument checking, device storage, phase bookkeeping and kernel launches.  No arithmetic of
// the method lives here; it is all in lbm_kernels.cuh.
// =====================================================================================
#include "../../include/lbm.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include <cub/device/device_select.cuh>
#include <cub/iterator/counting_input_iterator.cuh>

#include "lbm_kernels.cuh"

namespace {

char g_create_error[512] = "no error";

enum Phase { PHASE_NONE = 0,   // no state yet
             PHASE_PRE = 1,    // cur holds S_t (pre-collision), as handed in
             PHASE_POST = 2 }; // cur holds F_{t-1} (post-collision, not yet streamed); S_t = stream(F_{t-1})

}  // namespace

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
  void* cub_tmp;
  size_t cub_tmp_bytes;
  int* list_count_dev;
  unsigned long long* counters;  // device [6]
  long long n_moving, n_slip;    // MOVINGWALL / SLIPWALL cells of the accepted geometry
  double* totals_dev;            // device [5]
  void* staging;         // host<->device bounce buffer, grown on demand
  size_t staging_bytes;
  int cur;
  Phase phase;
  long long steps, launches, n_solid, n_masked;
  size_t device_bytes;
  cudaStream_t stream;
  int block_threads;
  int use_vector;        // 1: 128-bit vector kernel when nx % (32/dtype) == 0 (default); 0: scalar kernel
  int use_graph;
  // Vortex Method inlet / per-cell inflow field (lbm_set_inflow, lbm_set_vortices)
  double* uin_mean;      // [3][nz][ny] fp64 (whatever the dtype), nullptr = uniform params.u_in
  double* uin_field[2];  // inflow of the current / the previous time level, fp64
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
  int serpentine;        // 1: consecutive launches sweep z in opposite directions (L2 reuse)
  long long sweep_count; // BGK steps launched so far (parity = direction)
  int hrr_slab;          // HRR form: z-slices per slab of the two-pass step (0 = whole lattice)
  lbm_params last;       // parameters of the last lbm_step: the inlet rule is part of how S_t is formed from F_{t-1}
  char err[512];
};

namespace {

int fail(lbm_ctx* c, int code, const char* fmt, ...) {
  char* dst = c ? c->err : g_create_error;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return code;
}

#define LBM_CUDA(c, call)                                                                             \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess) return fail((c), LBM_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));      \
  } while (0)

bool is_device_pointer(const void* p) {
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int dev_alloc(lbm_ctx* c, void** p, size_t bytes) {
  cudaError_t e = cudaMalloc(p, bytes ? bytes : 1);
  if (e != cudaSuccess) {
    *p = nullptr;
    cudaGetLastError();
    return fail(c, e == cudaErrorMemoryAllocation ? LBM_ENOMEM : LBM_ECUDA, "cudaMalloc(%zu bytes): %s", bytes,
                cudaGetErrorString(e));
  }
  c->device_bytes += bytes;
  return LBM_OK;
}

int ensure_staging(lbm_ctx* c, size_t bytes) {
  if (c->staging_bytes >= bytes) return LBM_OK;
  if (c->staging) {
    cudaStreamSynchronize(c->stream);
    cudaFree(c->staging);
    c->device_bytes -= c->staging_bytes;
    c->staging = nullptr;
    c->staging_bytes = 0;
  }
  int rc = dev_alloc(c, &c->staging, bytes);
  if (rc == LBM_OK) c->staging_bytes = bytes;
  return rc;
}

void launch_dims(const lbm_ctx* c, dim3& grid, dim3& block) {
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
  a.uhat = static_cast<T*>(c->uhat);
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

// One launch of a step kernel over the z-slices [z0, z0 + nzs) (+ the list blocks when with_list), lattice `in` -> `out`.
template <int Q, typename T, int MODE, int COLL>
int launch_one(lbm_ctx* c, const lbm_params* p, int in, int out, int z0, int nzs, bool with_list, bool may_meet_lid = true) {
  dim3 grid, block;
  lbm::StepArgs<T> a = make_args<T>(c, p, in, out);
  a.z0 = z0;
  // serpentine sweep (lbm_set_option "serpentine", default 1): BGK steps alternate their direction with the time level; in the
  // HRR form the u^ pass runs downwards and the step pass upwards
  if (c->serpentine) a.z_reverse = lbm::mode_uhat(MODE) ? 1 : ((COLL == lbm::COLL_HRR) ? 0 : static_cast<int>(c->sweep_count & 1));
  const bool vec = c->use_vector && (c->nx % (32 / static_cast<int>(sizeof(T))) == 0);   // whole 32-byte sectors per row
  if (vec) {
    launch_dims_vec<Q, T, COLL>(c, grid, block);
    a.list_z = 0;
    if (with_list) {
      const long long per_slice = static_cast<long long>(grid.x) * grid.y * block.x * block.y;
      a.list_z = static_cast<int>((c->n_list + per_slice - 1) / per_slice);
    }
    grid.z = nzs + a.list_z;
    if (grid.z == 0) return LBM_OK;
    if (c->n_moving > 0 && may_meet_lid && lbm::mode_pulls(MODE)) lbm::k_step_vec<Q, T, MODE, COLL, true><<<grid, block, 0, c->stream>>>(a);
    else                                          lbm::k_step_vec<Q, T, MODE, COLL, false><<<grid, block, 0, c->stream>>>(a);
  } else {
    if (nzs == 0) return LBM_OK;
    launch_dims(c, grid, block);
    grid.z = nzs;
    lbm::k_step<Q, T, MODE, COLL><<<grid, block, 0, c->stream>>>(a);
  }
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  return LBM_OK;
}

// HRR form (Eq. 7-11): the FD strain (Eq. 10) needs u^(x,t) of the six neighbours, i.e. their streamed populations, so
// a step is two passes: UHAT (pull, moments, Eq. 12 -> u^ field) and the fused step that reads it.  The passes are
// interleaved slab by slab in z, the UHAT pass one slice ahead, so that the populations the UHAT pass pulled are still
// in the 126 MB L2 when the step pass pulls them again.  The list cells (wall model, ...) go with the
// first UHAT launch and the last step launch.
template <int Q, typename T, int MODE_U, int MODE_S>
int launch_hrr_t(lbm_ctx* c, const lbm_params* p, int in, int out) {
  const int nz = c->nz;
  int slab = (c->hrr_slab > 0) ? c->hrr_slab : nz;
  if (slab >= nz - 1) {
    int rc = launch_one<Q, T, MODE_U, lbm::COLL_BGK>(c, p, in, out, 0, nz, true);
    if (rc != LBM_OK) return rc;
    return launch_one<Q, T, MODE_S, lbm::COLL_HRR>(c, p, in, out, 0, nz, true);
  }
  // UHAT: slice nz-1 first (the periodic neighbour of slice 0), then [0, slab], [slab+1, 2 slab], ... up to nz-2
  int rc = launch_one<Q, T, MODE_U, lbm::COLL_BGK>(c, p, in, out, nz - 1, 1, true);
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
  if (c->n_moving == 0 || nz < 8)
    return launch_one<Q, T, lbm::MODE_STREAM_COLLIDE, lbm::COLL_BGK>(c, p, in, out, 0, nz, true);
  int rc = launch_one<Q, T, lbm::MODE_STREAM_COLLIDE, lbm::COLL_BGK>(c, p, in, out, 1, nz - 3, true, false);
  if (rc == LBM_OK) rc = launch_one<Q, T, lbm::MODE_STREAM_COLLIDE, lbm::COLL_BGK>(c, p, in, out, nz - 2, 2, false);
  if (rc == LBM_OK) rc = launch_one<Q, T, lbm::MODE_STREAM_COLLIDE, lbm::COLL_BGK>(c, p, in, out, 0, 1, false);
  return rc;
}

template <int Q, typename T>
int launch_step_t(lbm_ctx* c, const lbm_params* p, int mode) {
  const int in = c->cur, out = 1 - c->cur;
  const bool hrr = p && p->collision == LBM_COLLISION_HRR;
  int rc;
  switch (mode) {
    case lbm::MODE_COLLIDE:
      rc = hrr ? launch_hrr_t<Q, T, lbm::MODE_UHAT_PRE, lbm::MODE_COLLIDE>(c, p, in, out)
               : launch_one<Q, T, lbm::MODE_COLLIDE, lbm::COLL_BGK>(c, p, in, out, 0, c->nz, true);
      break;
    case lbm::MODE_STREAM_COLLIDE:
      rc = hrr ? launch_hrr_t<Q, T, lbm::MODE_UHAT_PULL, lbm::MODE_STREAM_COLLIDE>(c, p, in, out)
               : launch_bgk_pull_t<Q, T>(c, p, in, out);
      break;
    default:
      rc = launch_one<Q, T, lbm::MODE_STREAM, lbm::COLL_BGK>(c, p, in, out, 0, c->nz, true);
      break;
  }
  if (rc != LBM_OK) return rc;
  c->cur = out;
  c->sweep_count++;
  return LBM_OK;
}

int launch_step(lbm_ctx* c, const lbm_params* p, int mode) {
  if (c->Q == 19) return c->dtype == LBM_F32 ? launch_step_t<19, float>(c, p, mode) : launch_step_t<19, double>(c, p, mode);
  return c->dtype == LBM_F32 ? launch_step_t<27, float>(c, p, mode) : launch_step_t<27, double>(c, p, mode);
}

template <int Q, typename T>
int launch_moments_t(lbm_ctx* c, const lbm_params* p, void* rho, void* u) {
  dim3 grid, block;
  launch_dims(c, grid, block);
  lbm::StepArgs<T> a = make_args<T>(c, p, c->cur, 1 - c->cur);
  lbm::k_moments<Q, T><<<grid, block, 0, c->stream>>>(a, static_cast<T*>(rho), static_cast<T*>(u));
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  return LBM_OK;
}

template <int Q, typename T>
int launch_totals_t(lbm_ctx* c, const lbm_params* p) {
  dim3 grid, block;
  launch_dims(c, grid, block);
  lbm::StepArgs<T> a = make_args<T>(c, p, c->cur, 1 - c->cur);
  lbm::k_totals<Q, T><<<grid, block, 0, c->stream>>>(a, c->totals_dev);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  return LBM_OK;
}

template <int Q, typename T>
int launch_init_t(lbm_ctx* c, const void* rho, const void* u) {
  const int threads = 256;
  const long long blocks = (c->N + threads - 1) / threads;
  lbm::k_init_equilibrium<Q, T><<<static_cast<unsigned>(blocks), threads, 0, c->stream>>>(
      static_cast<const T*>(rho), static_cast<const T*>(u), static_cast<T*>(c->f[0]), c->N);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  return LBM_OK;
}

#define LBM_DISPATCH(c, fn, ...)                                                                              \
  ((c)->Q == 19 ? ((c)->dtype == LBM_F32 ? fn<19, float>(__VA_ARGS__) : fn<19, double>(__VA_ARGS__))          \
                : ((c)->dtype == LBM_F32 ? fn<27, float>(__VA_ARGS__) : fn<27, double>(__VA_ARGS__)))

lbm_params default_params() {
  lbm_params p;
  std::memset(&p, 0, sizeof(p));
  p.tau0 = 1.0;
  p.wm_kappa = 0.41;
  p.wm_E = 9.8;
  return p;
}

int check_params(lbm_ctx* c, const lbm_params* p) {
  if (!p) return fail(c, LBM_EINVAL, "lbm_step: params is NULL");
  if (!(p->tau0 > 0.5)) return fail(c, LBM_EINVAL, "lbm_step: tau0 = %g must be > 0.5", p->tau0);
  if (!(p->cs_smago >= 0.0)) return fail(c, LBM_EINVAL, "lbm_step: cs_smago = %g must be >= 0", p->cs_smago);
  if (p->wm_enable && (!(p->wm_kappa > 0.0) || !(p->wm_E > 0.0)))
    return fail(c, LBM_EINVAL, "lbm_step: wm_enable needs wm_kappa > 0 and wm_E > 0");
  if (!(p->u_in[0] < 1.0)) return fail(c, LBM_EINVAL, "lbm_step: u_in[0] = %g must be < 1", p->u_in[0]);
  if (p->rho_out < 0.0) return fail(c, LBM_EINVAL, "lbm_step: rho_out = %g must be > 0 (0 = default 1)", p->rho_out);
  if (p->fringe_len < 0 || !(p->fringe_factor >= 0.0)) return fail(c, LBM_EINVAL, "lbm_step: fringe_len = %d, fringe_factor = %g must be >= 0", p->fringe_len, p->fringe_factor);
  if (p->collision != LBM_COLLISION_BGK && p->collision != LBM_COLLISION_HRR)
    return fail(c, LBM_EINVAL, "lbm_step: collision = %d must be 0 (BGK) or 1 (HRR)", p->collision);
  if (p->collision == LBM_COLLISION_HRR && !(p->sigma >= 0.0 && p->sigma <= 1.0))
    return fail(c, LBM_EINVAL, "lbm_step: sigma = %g must be in [0,1]", p->sigma);
  return LBM_OK;
}

// stream compaction of the cell indices n with flags_raw[n] != 0 (count known) into a new device array
int compact_marks(lbm_ctx* c, long long count, int** out) {
  *out = nullptr;
  if (count <= 0) return LBM_OK;
  int* arr = nullptr;
  int rc = dev_alloc(c, reinterpret_cast<void**>(&arr), static_cast<size_t>(count) * sizeof(int));
  if (rc != LBM_OK) return rc;
  cub::CountingInputIterator<int> it(0);
  size_t need = 0;
  LBM_CUDA(c, cub::DeviceSelect::Flagged(nullptr, need, it, c->flags_raw, arr, c->list_count_dev, static_cast<int>(c->N), c->stream));
  if (need > c->cub_tmp_bytes) {
    if (c->cub_tmp) { cudaFree(c->cub_tmp); c->device_bytes -= c->cub_tmp_bytes; c->cub_tmp = nullptr; c->cub_tmp_bytes = 0; }
    rc = dev_alloc(c, &c->cub_tmp, need);
    if (rc != LBM_OK) { cudaFree(arr); return rc; }
    c->cub_tmp_bytes = need;
  }
  LBM_CUDA(c, cub::DeviceSelect::Flagged(c->cub_tmp, need, it, c->flags_raw, arr, c->list_count_dev, static_cast<int>(c->N), c->stream));
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  *out = arr;
  return LBM_OK;
}

// SOLID cells' own values: lattice c->cur -> side buffer (save) or back (restore)
int solid_values(lbm_ctx* c, bool save) {
  if (c->n_solid_list <= 0) return LBM_OK;
  const unsigned blocks = static_cast<unsigned>((c->n_solid_list + 255) / 256);
  if (c->dtype == LBM_F32) {
    float* f = static_cast<float*>(c->f[c->cur]);
    float* sv = static_cast<float*>(c->solid_vals);
    if (save) lbm::k_solid_values<float, true><<<blocks, 256, 0, c->stream>>>(f, sv, c->solid_list, c->n_solid_list, c->N, c->Q);
    else      lbm::k_solid_values<float, false><<<blocks, 256, 0, c->stream>>>(f, sv, c->solid_list, c->n_solid_list, c->N, c->Q);
  } else {
    double* f = static_cast<double*>(c->f[c->cur]);
    double* sv = static_cast<double*>(c->solid_vals);
    if (save) lbm::k_solid_values<double, true><<<blocks, 256, 0, c->stream>>>(f, sv, c->solid_list, c->n_solid_list, c->N, c->Q);
    else      lbm::k_solid_values<double, false><<<blocks, 256, 0, c->stream>>>(f, sv, c->solid_list, c->n_solid_list, c->N, c->Q);
  }
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  return LBM_OK;
}

// copy flags to the device, validate + classify into cls_alt, accept on success
int classify(lbm_ctx* c, const uint8_t* cell_flags) {
  if (cell_flags) {
    LBM_CUDA(c, cudaMemcpyAsync(c->flags_raw, cell_flags, c->N, cudaMemcpyDefault, c->stream));
  } else {
    LBM_CUDA(c, cudaMemsetAsync(c->flags_raw, 0, c->N, c->stream));
  }
  LBM_CUDA(c, cudaMemsetAsync(c->counters, 0, 6 * sizeof(unsigned long long), c->stream));
  dim3 grid, block;
  launch_dims(c, grid, block);
  if (c->Q == 19) lbm::k_classify<19><<<grid, block, 0, c->stream>>>(c->flags_raw, c->cls_alt, c->nx, c->ny, c->nz, c->counters);
  else            lbm::k_classify<27><<<grid, block, 0, c->stream>>>(c->flags_raw, c->cls_alt, c->nx, c->ny, c->nz, c->counters);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  unsigned long long h[6];
  LBM_CUDA(c, cudaMemcpyAsync(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  if (h[0] != 0)
    return fail(c, LBM_EINVAL, "cell_flags: %llu invalid flag byte(s) (type > 7, bad high nibble, INLET off x=0, OUTLET / POUTLET off x=nx-1 or MOVINGWALL off z=nz-1)", h[0]);
  // compact list of the cells the vector kernel leaves to its list blocks
  const int SV = 32 / c->dtype;        // cells per 32-byte sector of a population row
  long long n_list = 0;
  if (c->nx % SV == 0) {
    const long long nsec = c->N / SV;
    const unsigned blocks = static_cast<unsigned>((nsec + 255) / 256);
    if (SV == 8) lbm::k_mark_list<8><<<blocks, 256, 0, c->stream>>>(c->cls_alt, c->flags_raw, nsec, c->counters);
    else         lbm::k_mark_list<4><<<blocks, 256, 0, c->stream>>>(c->cls_alt, c->flags_raw, nsec, c->counters);
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
    LBM_CUDA(c, cudaMemcpyAsync(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    LBM_CUDA(c, cudaStreamSynchronize(c->stream));
    n_list = static_cast<long long>(h[3]);
    int* new_list = nullptr;
    int rc = compact_marks(c, n_list, &new_list);
    if (rc != LBM_OK) return rc;
    if (c->list) { cudaFree(c->list); c->device_bytes -= static_cast<size_t>(c->n_list) * sizeof(int); }
    c->list = new_list;
  }
  // SOLID cells: list + side buffer for their own values
  {
    const long long n_solid = static_cast<long long>(h[1]);
    const unsigned blocks = static_cast<unsigned>((c->N + 255) / 256);
    lbm::k_mark_solid<<<blocks, 256, 0, c->stream>>>(c->cls_alt, c->flags_raw, c->N);
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
    int* new_list = nullptr;
    int rc = compact_marks(c, n_solid, &new_list);
    if (rc != LBM_OK) return rc;
    void* new_vals = nullptr;
    const size_t vbytes = static_cast<size_t>(n_solid) * c->Q * c->dtype;
    if (n_solid > 0) {
      rc = dev_alloc(c, &new_vals, vbytes);
      if (rc != LBM_OK) { cudaFree(new_list); return rc; }
    }
    if (c->solid_list) { cudaFree(c->solid_list); c->device_bytes -= static_cast<size_t>(c->n_solid_list) * sizeof(int); }
    if (c->solid_vals) { cudaFree(c->solid_vals); c->device_bytes -= static_cast<size_t>(c->n_solid_list) * c->Q * c->dtype; }
    c->solid_list = new_list;
    c->solid_vals = new_vals;
    c->n_solid_list = n_solid;
  }
  c->n_list = n_list;
  uint8_t* t = c->cls;  c->cls = c->cls_alt;  c->cls_alt = t;
  if (c->Q == 19) lbm::k_nbmask<19><<<grid, block, 0, c->stream>>>(c->cls, c->nbmask, c->nx, c->ny, c->nz);
  else            lbm::k_nbmask<27><<<grid, block, 0, c->stream>>>(c->cls, c->nbmask, c->nx, c->ny, c->nz);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  c->n_solid = static_cast<long long>(h[1]);
  c->n_masked = static_cast<long long>(h[2]);
  c->n_moving = static_cast<long long>(h[4]);
  c->n_slip = static_cast<long long>(h[5]);
  return LBM_OK;
}

// ---- Vortex Method inlet: host side (Eq. 18-21) ---------------------------------------------------------------------
// main stream waits for a field that is still being formed on the side stream
int vm_join(lbm_ctx* c) {
  if (c->vm_pending) {
    LBM_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_vm, 0));
    c->vm_pending = false;
  }
  return LBM_OK;
}

// form the inflow of the next level from the current one, on stream st
int vm_advance(lbm_ctx* c, cudaStream_t st) {
  const long long P = static_cast<long long>(c->ny) * c->nz;
  if (c->gamma_dirty && c->nv > 0) {
    lbm::k_vm_gamma<double><<<1, 256, 0, st>>>(c->cls, c->nx, c->ny, c->nz, c->uin_mean, c->nv, c->vpos, c->vsign,
                                               c->vm_intensity, c->vgamma);
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
  }
  c->gamma_dirty = false;
  const unsigned blocks = static_cast<unsigned>((P + lbm::VM_CELLS - 1) / lbm::VM_CELLS);
  lbm::k_vm_inflow<double><<<blocks, lbm::VM_CELLS * lbm::VM_SLICES, 0, st>>>(c->cls, c->nx, c->ny, c->nz, c->uin_mean, c->uin_field[c->uin_cur], c->nv,
                                                   c->vpos, c->vgamma, c->vm_sigma, c->uin_field[1 - c->uin_cur]);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  c->uin_cur = 1 - c->uin_cur;
  c->inflow_index++;
  return LBM_OK;
}

// the inflow field of time level t must be current before S_t is formed (pulled) for the first time
int ensure_inflow(lbm_ctx* c, long long t) {
  if (!c->uin_mean) return LBM_OK;
  int rc = vm_join(c);
  if (rc != LBM_OK) return rc;
  while (c->inflow_index < t) {
    rc = vm_advance(c, c->stream);
    if (rc != LBM_OK) return rc;
  }
  return LBM_OK;
}

// after the step of level t has been enqueued on the main stream: mark it, and form the inflow of level t+1 beside it
int vm_prefetch(lbm_ctx* c, long long t) {
  if (!c->uin_mean) return LBM_OK;
  if (!c->vm_stream) {
    int prio_lo = 0, prio_hi = 0;      // highest priority: its few blocks must not queue behind the step kernel's thousands
    LBM_CUDA(c, cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    LBM_CUDA(c, cudaStreamCreateWithPriority(&c->vm_stream, cudaStreamNonBlocking, prio_hi));
    LBM_CUDA(c, cudaEventCreateWithFlags(&c->ev_vm, cudaEventDisableTiming));
    LBM_CUDA(c, cudaEventCreateWithFlags(&c->ev_step[0], cudaEventDisableTiming));
    LBM_CUDA(c, cudaEventCreateWithFlags(&c->ev_step[1], cudaEventDisableTiming));
    c->ev_step_level[0] = c->ev_step_level[1] = -1;
  }
  const int k = static_cast<int>(t & 1);
  LBM_CUDA(c, cudaEventRecord(c->ev_step[k], c->stream));
  c->ev_step_level[k] = t;
  if (c->inflow_index != t) return LBM_OK;
  // the buffer about to be overwritten held level t-1: its last reader is the step of level t-1.  If that step's event is not
  // on record (first step of a run, inputs just changed) wait for the step just enqueued instead (no overlap, once).
  const int w = (c->ev_step_level[1 - k] == t - 1) ? 1 - k : k;
  LBM_CUDA(c, cudaStreamWaitEvent(c->vm_stream, c->ev_step[w], 0));
  int rc = vm_advance(c, c->vm_stream);
  if (rc != LBM_OK) return rc;
  LBM_CUDA(c, cudaEventRecord(c->ev_vm, c->vm_stream));
  c->vm_pending = true;
  return LBM_OK;
}

// "previous inflow" := u_mean; the current time level is c->steps
int reset_inflow(lbm_ctx* c) {
  if (!c->uin_mean) return LBM_OK;
  { int rcj = vm_join(c); if (rcj != LBM_OK) return rcj; }
  c->ev_step_level[0] = c->ev_step_level[1] = -1;      // inputs of the side stream change on the main stream: re-order once
  const size_t bytes = 3 * static_cast<size_t>(c->ny) * c->nz * sizeof(double);
  LBM_CUDA(c, cudaMemcpyAsync(c->uin_field[c->uin_cur], c->uin_mean, bytes, cudaMemcpyDeviceToDevice, c->stream));
  c->inflow_index = c->steps;
  return LBM_OK;
}

}  // namespace

extern "C" {

const char* lbm_last_error(const lbm_ctx* ctx) { return ctx ? ctx->err : g_create_error; }

lbm_ctx* lbm_create(int lattice, int nx, int ny, int nz, int dtype) {
  if (lattice != LBM_D3Q19 && lattice != LBM_D3Q27) { fail(nullptr, LBM_EINVAL, "lbm_create: lattice %d is not 19 or 27", lattice); return nullptr; }
  if (dtype != LBM_F32 && dtype != LBM_F64) { fail(nullptr, LBM_EINVAL, "lbm_create: dtype %d is not 4 (f32) or 8 (f64)", dtype); return nullptr; }
  if (nx < 1 || ny < 1 || nz < 1) { fail(nullptr, LBM_EINVAL, "lbm_create: nx, ny, nz must be >= 1 (got %d %d %d)", nx, ny, nz); return nullptr; }
  const long long N = static_cast<long long>(nx) * ny * nz;
  if (N >= (1ll << 31) || nz > 65535) { fail(nullptr, LBM_EINVAL, "lbm_create: lattice too large (N = %lld must be < 2^31, nz <= 65535)", N); return nullptr; }
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    fail(nullptr, LBM_ECUDA, "lbm_create: no usable CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
    return nullptr;
  }
  lbm_ctx* c = new (std::nothrow) lbm_ctx;
  if (!c) { fail(nullptr, LBM_ENOMEM, "lbm_create: host allocation failed"); return nullptr; }
  std::memset(c, 0, sizeof(*c));
  c->Q = lattice;  c->nx = nx;  c->ny = ny;  c->nz = nz;  c->dtype = dtype;  c->N = N;
  c->phase = PHASE_NONE;
  c->block_threads = 64;
  c->use_vector = 1;
  c->serpentine = 1;
  c->last = default_params();
  std::snprintf(c->err, sizeof(c->err), "no error");
  const size_t pop = static_cast<size_t>(lattice) * N * dtype;
  int rc = dev_alloc(c, &c->f[0], pop);
  if (rc == LBM_OK) rc = dev_alloc(c, &c->f[1], pop);
  if (rc == LBM_OK) rc = dev_alloc(c, &c->d, static_cast<size_t>(N) * dtype);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->cls), N);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->cls_alt), N);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->flags_raw), N);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->nbmask), static_cast<size_t>(N) * sizeof(uint32_t));
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->counters), 6 * sizeof(unsigned long long));
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->totals_dev), 5 * sizeof(double));
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->list_count_dev), sizeof(int));
  if (rc == LBM_OK && cudaMemset(c->cls, 0, N) != cudaSuccess) rc = fail(c, LBM_ECUDA, "cudaMemset failed");
  if (rc == LBM_OK && cudaMemset(c->nbmask, 0, static_cast<size_t>(N) * sizeof(uint32_t)) != cudaSuccess) rc = fail(c, LBM_ECUDA, "cudaMemset failed");
  if (rc != LBM_OK) {
    std::snprintf(g_create_error, sizeof(g_create_error), "lbm_create: %.480s", c->err);
    lbm_destroy(c);
    return nullptr;
  }
  return c;
}

void lbm_destroy(lbm_ctx* c) {
  if (!c) return;
  cudaStreamSynchronize(c->stream);
  if (c->vm_stream) {
    cudaStreamSynchronize(c->vm_stream);
    cudaStreamDestroy(c->vm_stream);
    cudaEventDestroy(c->ev_vm);  cudaEventDestroy(c->ev_step[0]);  cudaEventDestroy(c->ev_step[1]);
  }
  cudaFree(c->f[0]);  cudaFree(c->f[1]);  cudaFree(c->d);  cudaFree(c->uhat);  cudaFree(c->ub);
  cudaFree(c->uin_mean);  cudaFree(c->uin_field[0]);  cudaFree(c->uin_field[1]);  cudaFree(c->vpos);  cudaFree(c->vsign);  cudaFree(c->vgamma);
  cudaFree(c->cls);  cudaFree(c->cls_alt);  cudaFree(c->flags_raw);
  cudaFree(c->counters);  cudaFree(c->totals_dev);  cudaFree(c->staging);
  cudaFree(c->list);  cudaFree(c->cub_tmp);  cudaFree(c->list_count_dev);
  cudaFree(c->nbmask);  cudaFree(c->solid_list);  cudaFree(c->solid_vals);
  cudaGetLastError();
  delete c;
}

int lbm_set_stream(lbm_ctx* c, void* cuda_stream) {
  if (!c) return LBM_EINVAL;
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  return LBM_OK;
}

int lbm_synchronize(lbm_ctx* c) {
  if (!c) return LBM_EINVAL;
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  LBM_CUDA(c, cudaGetLastError());
  return LBM_OK;
}

static int set_geometry_fields(lbm_ctx* c, const void* porosity, const uint8_t* cell_flags) {
  int rc = classify(c, cell_flags);
  if (rc != LBM_OK) return rc;
  c->gamma_dirty = true;   // A and the seeds' cells depend on the flags
  if (c->uhat)   // cells that turned SOLID must read u^ = 0 (the UHAT pass does not visit all-SOLID lines)
    LBM_CUDA(c, cudaMemsetAsync(c->uhat, 0, 3 * static_cast<size_t>(c->N) * c->dtype, c->stream));
  if (porosity) {
    LBM_CUDA(c, cudaMemcpyAsync(c->d, porosity, static_cast<size_t>(c->N) * c->dtype, cudaMemcpyDefault, c->stream));
    c->has_d = true;
  } else {
    c->has_d = false;
  }
  return LBM_OK;
}

int lbm_set_fields(lbm_ctx* c, const void* populations, const void* porosity, const uint8_t* cell_flags) {
  if (!c) return LBM_EINVAL;
  if (!populations) return fail(c, LBM_EINVAL, "lbm_set_fields: populations is NULL");
  int rc = set_geometry_fields(c, porosity, cell_flags);
  if (rc != LBM_OK) return rc;
  const size_t pop = static_cast<size_t>(c->Q) * c->N * c->dtype;
  LBM_CUDA(c, cudaMemcpyAsync(c->f[0], populations, pop, cudaMemcpyDefault, c->stream));
  if (!is_device_pointer(populations)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  c->cur = 0;
  c->phase = PHASE_PRE;
  c->steps = 0;
  { int rci = reset_inflow(c); if (rci != LBM_OK) return rci; }
  return solid_values(c, true);      // SOLID cells' own values -> side buffer (the step kernels overwrite their slots)
}

int lbm_init_equilibrium(lbm_ctx* c, const void* rho, const void* u) {
  if (!c) return LBM_EINVAL;
  if (!rho || !u) return fail(c, LBM_EINVAL, "lbm_init_equilibrium: rho or u is NULL");
  const size_t cell_bytes = static_cast<size_t>(c->N) * c->dtype;
  const void* drho = rho;
  const void* du = u;
  const bool hr = !is_device_pointer(rho), hu = !is_device_pointer(u);
  if (hr || hu) {
    int rc = ensure_staging(c, 4 * cell_bytes);
    if (rc != LBM_OK) return rc;
    char* s = static_cast<char*>(c->staging);
    if (hr) { LBM_CUDA(c, cudaMemcpyAsync(s, rho, cell_bytes, cudaMemcpyDefault, c->stream)); drho = s; }
    if (hu) { LBM_CUDA(c, cudaMemcpyAsync(s + cell_bytes, u, 3 * cell_bytes, cudaMemcpyDefault, c->stream)); du = s + cell_bytes; }
  }
  int rc = LBM_DISPATCH(c, launch_init_t, c, drho, du);
  if (rc != LBM_OK) return rc;
  if (hr || hu) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  c->cur = 0;
  c->phase = PHASE_PRE;
  c->steps = 0;
  { int rci = reset_inflow(c); if (rci != LBM_OK) return rci; }
  return solid_values(c, true);
}

// POST -> PRE: write S_t = stream(F_{t-1}) into the other lattice and make it current
static int materialise(lbm_ctx* c) {
  if (c->phase != PHASE_POST) return LBM_OK;
  lbm_params p = c->last;
  int rci = ensure_inflow(c, c->steps);
  if (rci != LBM_OK) return rci;
  int rc = launch_step(c, &p, lbm::MODE_STREAM);
  if (rc != LBM_OK) return rc;
  c->phase = PHASE_PRE;
  return solid_values(c, false);     // the stream pass leaves zeros or stale data on SOLID cells: put their own values back
}

int lbm_set_geometry(lbm_ctx* c, const void* porosity, const uint8_t* cell_flags) {
  if (!c) return LBM_EINVAL;
  // S_t is defined with the geometry it was computed under: fix it before the geometry changes
  int rc = materialise(c);
  if (rc != LBM_OK) return rc;
  rc = set_geometry_fields(c, porosity, cell_flags);
  if (rc != LBM_OK) return rc;
  if (c->phase == PHASE_PRE) return solid_values(c, true);   // the SOLID set changed: save the new set's values
  return LBM_OK;
}

// Neither call touches the populations or the pull: d and u^B enter the collision only (Eq. 12), so the stored
// post-collision state F_{t-1} stays valid and no pass over the lattice is needed (unlike lbm_set_geometry).
int lbm_set_porosity(lbm_ctx* c, const void* porosity) {
  if (!c) return LBM_EINVAL;
  if (!porosity) {
    c->has_d = false;
    return LBM_OK;
  }
  LBM_CUDA(c, cudaMemcpyAsync(c->d, porosity, static_cast<size_t>(c->N) * c->dtype, cudaMemcpyDefault, c->stream));
  if (!is_device_pointer(porosity)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  c->has_d = true;
  return LBM_OK;
}

int lbm_set_body_velocity(lbm_ctx* c, const void* u_body) {
  if (!c) return LBM_EINVAL;
  const size_t bytes = 3 * static_cast<size_t>(c->N) * c->dtype;
  if (!u_body) {
    if (c->ub) {
      LBM_CUDA(c, cudaStreamSynchronize(c->stream));
      cudaFree(c->ub);
      c->ub = nullptr;
      c->device_bytes -= bytes;
    }
    return LBM_OK;
  }
  if (!c->ub) {
    int rc = dev_alloc(c, &c->ub, bytes);
    if (rc != LBM_OK) return rc;
  }
  LBM_CUDA(c, cudaMemcpyAsync(c->ub, u_body, bytes, cudaMemcpyDefault, c->stream));
  if (!is_device_pointer(u_body)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

int lbm_set_inflow(lbm_ctx* c, const void* u_mean) {
  if (!c) return LBM_EINVAL;
  const long long n = 3ll * c->ny * c->nz;
  const size_t bytes = static_cast<size_t>(n) * sizeof(double);       // kept in fp64 whatever the dtype
  // the state S_t keeps the inflow it was formed with
  int rc = materialise(c);
  if (rc != LBM_OK) return rc;
  if (!u_mean) {
    if (c->uin_mean) {
      LBM_CUDA(c, cudaStreamSynchronize(c->stream));
      cudaFree(c->uin_mean);  cudaFree(c->uin_field[0]);  cudaFree(c->uin_field[1]);
      c->uin_mean = c->uin_field[0] = c->uin_field[1] = nullptr;
      c->device_bytes -= 3 * bytes;
    }
    return LBM_OK;
  }
  if (!c->uin_mean) {
    rc = dev_alloc(c, reinterpret_cast<void**>(&c->uin_mean), bytes);
    if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->uin_field[0]), bytes);
    if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->uin_field[1]), bytes);
    if (rc != LBM_OK) return rc;
    c->uin_cur = 0;
  }
  if (c->dtype == LBM_F64) {
    LBM_CUDA(c, cudaMemcpyAsync(c->uin_mean, u_mean, bytes, cudaMemcpyDefault, c->stream));
  } else {                               // fp32 input -> staging (the other field buffer) -> fp64
    float* tmp = reinterpret_cast<float*>(c->uin_field[1 - c->uin_cur]);
    LBM_CUDA(c, cudaMemcpyAsync(tmp, u_mean, static_cast<size_t>(n) * sizeof(float), cudaMemcpyDefault, c->stream));
    lbm::k_convert<float, double><<<static_cast<unsigned>((n + 255) / 256), 256, 0, c->stream>>>(tmp, c->uin_mean, n);
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
  }
  if (!is_device_pointer(u_mean)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  c->gamma_dirty = true;
  return reset_inflow(c);
}

int lbm_set_vortices(lbm_ctx* c, int n, const double* pos, const double* sign, double sigma_v, double intensity) {
  if (!c) return LBM_EINVAL;
  if (n < 0 || (n > 0 && (!pos || !sign))) return fail(c, LBM_EINVAL, "lbm_set_vortices: n = %d, pos / sign must not be NULL", n);
  if (!(sigma_v > 0.0) || !(intensity >= 0.0)) return fail(c, LBM_EINVAL, "lbm_set_vortices: sigma_v = %g must be > 0, intensity = %g >= 0", sigma_v, intensity);
  int rc = materialise(c);             // S_t keeps the inflow it was formed with
  if (rc != LBM_OK) return rc;
  rc = vm_join(c);
  if (rc != LBM_OK) return rc;
  c->ev_step_level[0] = c->ev_step_level[1] = -1;
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  if (c->vpos) { cudaFree(c->vpos); cudaFree(c->vsign); cudaFree(c->vgamma); c->device_bytes -= 4 * sizeof(double) * static_cast<size_t>(c->nv); }
  c->vpos = c->vsign = c->vgamma = nullptr;
  c->nv = 0;
  if (n > 0) {
    rc = dev_alloc(c, reinterpret_cast<void**>(&c->vpos), 2 * sizeof(double) * n);
    if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->vsign), sizeof(double) * n);
    if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->vgamma), sizeof(double) * n);
    if (rc != LBM_OK) return rc;
    LBM_CUDA(c, cudaMemcpyAsync(c->vpos, pos, 2 * sizeof(double) * n, cudaMemcpyHostToDevice, c->stream));
    LBM_CUDA(c, cudaMemcpyAsync(c->vsign, sign, sizeof(double) * n, cudaMemcpyHostToDevice, c->stream));
    LBM_CUDA(c, cudaStreamSynchronize(c->stream));
    c->nv = n;
  }
  c->vm_sigma = sigma_v;
  c->vm_intensity = intensity;
  c->gamma_dirty = true;
  return LBM_OK;
}

int lbm_get_inflow(lbm_ctx* c, void* u) {
  if (!c) return LBM_EINVAL;
  if (!u) return fail(c, LBM_EINVAL, "lbm_get_inflow: u is NULL");
  if (!c->uin_mean) return fail(c, LBM_ESTATE, "lbm_get_inflow: no inflow field set (lbm_set_inflow)");
  int rc = ensure_inflow(c, c->steps);
  if (rc != LBM_OK) return rc;
  const long long n = 3ll * c->ny * c->nz;
  if (c->dtype == LBM_F64) {
    LBM_CUDA(c, cudaMemcpyAsync(u, c->uin_field[c->uin_cur], static_cast<size_t>(n) * sizeof(double), cudaMemcpyDefault, c->stream));
  } else {                               // fp64 -> fp32 through the idle field buffer
    float* tmp = reinterpret_cast<float*>(c->uin_field[1 - c->uin_cur]);
    lbm::k_convert<double, float><<<static_cast<unsigned>((n + 255) / 256), 256, 0, c->stream>>>(c->uin_field[c->uin_cur], tmp, n);
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
    LBM_CUDA(c, cudaMemcpyAsync(u, tmp, static_cast<size_t>(n) * sizeof(float), cudaMemcpyDefault, c->stream));
  }
  if (!is_device_pointer(u)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

int lbm_step(lbm_ctx* c, int n_steps, const lbm_params* params) {
  if (!c) return LBM_EINVAL;
  int rc = check_params(c, params);
  if (rc != LBM_OK) return rc;
  if (n_steps < 0) return fail(c, LBM_EINVAL, "lbm_step: n_steps = %d must be >= 0", n_steps);
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_step: no state; call lbm_set_fields or lbm_init_equilibrium first");
  c->last = *params;
  if (params->collision == LBM_COLLISION_HRR && !c->uhat && n_steps > 0) {
    const size_t bytes = 3 * static_cast<size_t>(c->N) * c->dtype;
    rc = dev_alloc(c, &c->uhat, bytes);
    if (rc != LBM_OK) return rc;
    // SOLID cells of all-SOLID lines are never written by the UHAT pass: u^ = 0 there (resting wall) from here on
    LBM_CUDA(c, cudaMemsetAsync(c->uhat, 0, bytes, c->stream));
  }
  for (int s = 0; s < n_steps; ++s) {
    if (c->phase == PHASE_PRE) {
      rc = launch_step(c, params, lbm::MODE_COLLIDE);          // S_t -> F_t
      c->phase = PHASE_POST;
    } else {
      rc = ensure_inflow(c, c->steps + s);                     // Vortex Method inlet: the inflow S_t carries (Eq. 21)
      if (rc != LBM_OK) return rc;
      rc = launch_step(c, params, lbm::MODE_STREAM_COLLIDE);   // F_{t-1} -> S_t -> F_t
    }
    if (rc != LBM_OK) return rc;
    rc = vm_prefetch(c, c->steps + s);                         // inflow of the next level, beside this step
    if (rc != LBM_OK) return rc;
  }
  c->steps += n_steps;
  return LBM_OK;
}

int lbm_moments(lbm_ctx* c, void* rho, void* u) {
  if (!c) return LBM_EINVAL;
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_moments: no state");
  if (!rho && !u) return LBM_OK;
  const size_t cell_bytes = static_cast<size_t>(c->N) * c->dtype;
  const bool hr = rho && !is_device_pointer(rho), hu = u && !is_device_pointer(u);
  void* drho = rho;
  void* du = u;
  if (hr || hu) {
    int rc = ensure_staging(c, 4 * cell_bytes);
    if (rc != LBM_OK) return rc;
    char* s = static_cast<char*>(c->staging);
    if (hr) drho = s;
    if (hu) du = s + cell_bytes;
  }
  lbm_params p = c->last;
  int rc = materialise(c);           // S_t in the cell's own storage (one extra pass when the storage held F_{t-1})
  if (rc != LBM_OK) return rc;
  rc = LBM_DISPATCH(c, launch_moments_t, c, &p, drho, du);
  if (rc != LBM_OK) return rc;
  if (hr) LBM_CUDA(c, cudaMemcpyAsync(rho, drho, cell_bytes, cudaMemcpyDefault, c->stream));
  if (hu) LBM_CUDA(c, cudaMemcpyAsync(u, du, 3 * cell_bytes, cudaMemcpyDefault, c->stream));
  if (hr || hu) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

int lbm_get_populations(lbm_ctx* c, void* populations) {
  if (!c) return LBM_EINVAL;
  if (!populations) return fail(c, LBM_EINVAL, "lbm_get_populations: populations is NULL");
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_get_populations: no state");
  int rc = materialise(c);
  if (rc != LBM_OK) return rc;
  const size_t pop = static_cast<size_t>(c->Q) * c->N * c->dtype;
  LBM_CUDA(c, cudaMemcpyAsync(populations, c->f[c->cur], pop, cudaMemcpyDefault, c->stream));
  if (!is_device_pointer(populations)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

int lbm_totals(lbm_ctx* c, double out[5]) {
  if (!c) return LBM_EINVAL;
  if (!out) return fail(c, LBM_EINVAL, "lbm_totals: out is NULL");
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_totals: no state");
  LBM_CUDA(c, cudaMemsetAsync(c->totals_dev, 0, 5 * sizeof(double), c->stream));
  lbm_params p = c->last;
  int rc = materialise(c);
  if (rc != LBM_OK) return rc;
  rc = LBM_DISPATCH(c, launch_totals_t, c, &p);
  if (rc != LBM_OK) return rc;
  LBM_CUDA(c, cudaMemcpyAsync(out, c->totals_dev, 5 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

long long lbm_query(const lbm_ctx* c, int what) {
  if (!c) return -1;
  switch (what) {
    case 0: return c->steps;
    case 1: return c->launches;
    case 2: return c->N;
    case 3: return c->n_solid;
    case 4: return static_cast<long long>(c->device_bytes);
    case 5: return c->n_masked;
    case 6: return c->n_list;
    default: return -1;
  }
}

int lbm_set_option(lbm_ctx* c, const char* key, long long value) {
  if (!c || !key) return LBM_EINVAL;
  if (std::strcmp(key, "cuda_graph") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "cuda_graph must be 0 or 1");
    c->use_graph = static_cast<int>(value);
    return LBM_OK;
  }
  if (std::strcmp(key, "block_threads") == 0) {
    if (value != 64 && value != 128 && value != 256) return fail(c, LBM_EINVAL, "block_threads must be 64, 128 or 256");
    c->block_threads = static_cast<int>(value);
    return LBM_OK;
  }
  if (std::strcmp(key, "serpentine") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "serpentine must be 0 or 1");
    c->serpentine = static_cast<int>(value);
    return LBM_OK;
  }
  if (std::strcmp(key, "hrr_slab") == 0) {
    if (value < 0) return fail(c, LBM_EINVAL, "hrr_slab must be >= 0");
    c->hrr_slab = static_cast<int>(value);
    return LBM_OK;
  }
  if (std::strcmp(key, "vector") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "vector must be 0 or 1");
    c->use_vector = static_cast<int>(value);
    return LBM_OK;
  }
  return fail(c, LBM_EINVAL, "unknown option '%s'", key);
}

}  // extern "C"
