// =====================================================================================
// lbm_api.cu -- host side of the C ABI declared in include/lbm.h.
// Argument checking, device storage, phase bookkeeping and kernel launches.  No arithmetic of
// the method lives here; it is all in lbm_kernels.cuh.
// =====================================================================================
#include "lbm_ctx.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include <cub/device/device_select.cuh>
#include <cub/iterator/counting_input_iterator.cuh>

#include "lbm_kernels.cuh"

namespace {
char g_create_error[512] = "no error";
}  // namespace

namespace lbmhost {
int fail(lbm_ctx* c, int code, const char* fmt, ...) {
  char* dst = c ? c->err : g_create_error;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return code;
}
}  // namespace lbmhost

namespace {

using lbmhost::fail;

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
  if (bx * by < 32) by = 32 / bx;
  block = dim3(bx, by, 1);
  grid = dim3((c->nx + bx - 1) / bx, (c->ny + by - 1) / by, c->nz);
}

// the launchers live in lbm_inst.cu (one object per lattice, dtype and part)
#define LBM_DISPATCH(c, fn, ...)                                                                                                \
  ((c)->Q == 19 ? ((c)->dtype == LBM_F32 ? lbmhost::fn<19, float>(__VA_ARGS__) : lbmhost::fn<19, double>(__VA_ARGS__))          \
                : ((c)->dtype == LBM_F32 ? lbmhost::fn<27, float>(__VA_ARGS__) : lbmhost::fn<27, double>(__VA_ARGS__)))

// stage: -1 = the whole step; 0 / 1 = the two stages of a step on a sub-domain (lbm_step_halo; the BGK form has no stage 0)
// the second lattice is allocated when a two-lattice pass first needs it (a lattice that only ever steps in place never does)
int ensure_lattice1(lbm_ctx* c) {
  if (c->f[1]) return LBM_OK;
  return dev_alloc(c, &c->f[1], static_cast<size_t>(c->Q) * c->N * c->dtype);
}

int launch_step(lbm_ctx* c, const lbm_params* p, int mode, int stage = -1) {
  { int rca = ensure_lattice1(c); if (rca != LBM_OK) return rca; }
  const bool hrr = p && p->collision != LBM_COLLISION_BGK && mode != lbm::MODE_STREAM;
  if (hrr) return LBM_DISPATCH(c, launch_step_hrr, c, p, mode, stage);
  if (stage == 0) return LBM_OK;
  return LBM_DISPATCH(c, launch_step_bgk, c, p, mode);
}

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
  if (p->collision != LBM_COLLISION_BGK && p->collision != LBM_COLLISION_HRR && p->collision != LBM_COLLISION_HRR_LAG)
    return fail(c, LBM_EINVAL, "lbm_step: collision = %d must be 0 (BGK), 1 (HRR) or 2 (HRR, FD strain of the previous level)", p->collision);
  if (p->collision != LBM_COLLISION_BGK && !(p->sigma >= 0.0 && p->sigma <= 1.0))
    return fail(c, LBM_EINVAL, "lbm_step: sigma = %g must be in [0,1]", p->sigma);
  return LBM_OK;
}

// stream compaction of the cell indices n with flags_raw[n] != 0 (count known) into a new device array
// (cub::DeviceSelect: a library primitive at set-up time only, never inside lbm_step)
int compact_marks(lbm_ctx* c, long long count, int** out) {
  *out = nullptr;
  if (count <= 0) return LBM_OK;
  int* arr = nullptr;
  int rc = dev_alloc(c, reinterpret_cast<void**>(&arr), static_cast<size_t>(count) * sizeof(int));
  if (rc != LBM_OK) return rc;
  cub::CountingInputIterator<int> it(0);
  size_t need = 0;
  cudaError_t e = cub::DeviceSelect::Flagged(nullptr, need, it, c->flags_raw, arr, c->list_count_dev, static_cast<int>(c->N), c->stream);
  if (e == cudaSuccess && need > c->cub_tmp_bytes) {
    if (c->cub_tmp) { cudaFree(c->cub_tmp); c->device_bytes -= c->cub_tmp_bytes; c->cub_tmp = nullptr; c->cub_tmp_bytes = 0; }
    rc = dev_alloc(c, &c->cub_tmp, need);
    if (rc == LBM_OK) c->cub_tmp_bytes = need;
  }
  if (rc == LBM_OK && e == cudaSuccess)
    e = cub::DeviceSelect::Flagged(c->cub_tmp, need, it, c->flags_raw, arr, c->list_count_dev, static_cast<int>(c->N), c->stream);
  if (rc == LBM_OK && e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (rc == LBM_OK && e != cudaSuccess) rc = fail(c, LBM_ECUDA, "list compaction: %s", cudaGetErrorString(e));
  if (rc != LBM_OK) {
    cudaFree(arr);
    c->device_bytes -= static_cast<size_t>(count) * sizeof(int);
    return rc;
  }
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

// copy flags to the device, validate + classify into cls_alt, build the new compact lists, accept everything together on
// success; on any failure the context keeps the geometry it had (lists, counts, class bytes, neighbour masks)
int classify(lbm_ctx* c, const uint8_t* cell_flags) {
  if (cell_flags) {
    LBM_CUDA(c, cudaMemcpyAsync(c->flags_raw, cell_flags, c->N, cudaMemcpyDefault, c->stream));
  } else {
    LBM_CUDA(c, cudaMemsetAsync(c->flags_raw, 0, c->N, c->stream));
  }
  LBM_CUDA(c, cudaMemsetAsync(c->counters, 0, 16 * sizeof(unsigned long long), c->stream));
  dim3 grid, block;
  launch_dims(c, grid, block);
  const int wm_special = c->wm_prepass ? 0 : 1;
  const int slip_planes = c->slip_planes;
  if (c->Q == 19) lbm::k_classify<19><<<grid, block, 0, c->stream>>>(c->flags_raw, c->cls_alt, c->nx, c->ny, c->nz, c->counters, wm_special, slip_planes);
  else            lbm::k_classify<27><<<grid, block, 0, c->stream>>>(c->flags_raw, c->cls_alt, c->nx, c->ny, c->nz, c->counters, wm_special, slip_planes);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  unsigned long long h[16];
  LBM_CUDA(c, cudaMemcpyAsync(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  if (h[0] != 0)
    return fail(c, LBM_EINVAL, "cell_flags: %llu invalid flag byte(s) (type > 7, bad high nibble, INLET off x=0, OUTLET / POUTLET off x=nx-1 or MOVINGWALL off z=nz-1)", h[0]);
  int* new_list = nullptr;
  int* new_solid = nullptr;
  int* new_wm = nullptr;
  void* new_vals = nullptr;
  const long long n_solid = static_cast<long long>(h[1]);
  const long long n_wm = static_cast<long long>(h[6]);
  const size_t vbytes = static_cast<size_t>(n_solid) * c->Q * c->dtype;
  long long n_list = 0;
  int rc = LBM_OK;
  // (1) cells the vector kernel leaves to its list blocks: every cell of a 32-byte sector that holds a SPECIAL cell
  const int SV = 32 / c->dtype;        // cells per 32-byte sector of a population row
  if (c->nx % SV == 0) {
    const long long nsec = c->N / SV;
    const unsigned blocks = static_cast<unsigned>((nsec + 255) / 256);
    if (h[7] != 0) {                   // cells with a slip plane code: the cells of a sector must agree (vector path)
      if (SV == 8) lbm::k_slip_uniform<8><<<blocks, 256, 0, c->stream>>>(c->cls_alt, nsec, c->counters);
      else         lbm::k_slip_uniform<4><<<blocks, 256, 0, c->stream>>>(c->cls_alt, nsec, c->counters);
      c->launches++;
    }
    if (SV == 8) lbm::k_mark_list<8><<<blocks, 256, 0, c->stream>>>(c->cls_alt, c->flags_raw, nsec, c->counters);
    else         lbm::k_mark_list<4><<<blocks, 256, 0, c->stream>>>(c->cls_alt, c->flags_raw, nsec, c->counters);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return fail(c, LBM_ECUDA, "classify (list marks): %s", cudaGetErrorString(e));
    c->launches++;
    n_list = static_cast<long long>(h[3]);
    rc = compact_marks(c, n_list, &new_list);
  }
  // (2) wall cells: list + side buffer for their own values
  if (rc == LBM_OK) {
    const unsigned blocks = static_cast<unsigned>((c->N + 255) / 256);
    lbm::k_mark_solid<<<blocks, 256, 0, c->stream>>>(c->cls_alt, c->flags_raw, c->N);
    if (cudaGetLastError() != cudaSuccess) rc = fail(c, LBM_ECUDA, "classify (wall marks): launch failed");
    else { c->launches++; rc = compact_marks(c, n_solid, &new_solid); }
    if (rc == LBM_OK && n_solid > 0) rc = dev_alloc(c, &new_vals, vbytes);
  }
  // (3) WALLMODEL cells: list of the pre-pass
  if (rc == LBM_OK) {
    const unsigned blocks = static_cast<unsigned>((c->N + 255) / 256);
    lbm::k_mark_wm<<<blocks, 256, 0, c->stream>>>(c->cls_alt, c->flags_raw, c->N);
    if (cudaGetLastError() != cudaSuccess) rc = fail(c, LBM_ECUDA, "classify (wall-model marks): launch failed");
    else { c->launches++; rc = compact_marks(c, n_wm, &new_wm); }
  }
  if (rc != LBM_OK) {                  // nothing of the old geometry has been touched
    if (new_list) { cudaFree(new_list); c->device_bytes -= static_cast<size_t>(n_list) * sizeof(int); }
    if (new_solid) { cudaFree(new_solid); c->device_bytes -= static_cast<size_t>(n_solid) * sizeof(int); }
    if (new_wm) { cudaFree(new_wm); c->device_bytes -= static_cast<size_t>(n_wm) * sizeof(int); }
    if (new_vals) { cudaFree(new_vals); c->device_bytes -= vbytes; }
    return rc;
  }
  // accept: swap lists, counts, class bytes together
  if (c->list) { cudaFree(c->list); c->device_bytes -= static_cast<size_t>(c->n_list) * sizeof(int); }
  if (c->solid_list) { cudaFree(c->solid_list); c->device_bytes -= static_cast<size_t>(c->n_solid_list) * sizeof(int); }
  if (c->solid_vals) { cudaFree(c->solid_vals); c->device_bytes -= static_cast<size_t>(c->n_solid_list) * c->Q * c->dtype; }
  if (c->wm_list) { cudaFree(c->wm_list); c->device_bytes -= static_cast<size_t>(c->n_wm) * sizeof(int); }
  c->list = new_list;          c->n_list = n_list;
  c->solid_list = new_solid;   c->solid_vals = new_vals;   c->n_solid_list = n_solid;
  c->wm_list = new_wm;         c->n_wm = n_wm;
  uint8_t* t = c->cls;  c->cls = c->cls_alt;  c->cls_alt = t;
  if (c->Q == 19) lbm::k_nbmask<19><<<grid, block, 0, c->stream>>>(c->cls, c->nbmask, c->nx, c->ny, c->nz);
  else            lbm::k_nbmask<27><<<grid, block, 0, c->stream>>>(c->cls, c->nbmask, c->nx, c->ny, c->nz);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  c->n_solid = n_solid;
  c->n_masked = static_cast<long long>(h[2]);
  c->n_moving = static_cast<long long>(h[4]);
  c->n_slip = static_cast<long long>(h[5]);
  c->n_slipcode = static_cast<long long>(h[7]);
  c->n_typed = static_cast<long long>(h[8]);
  c->epoch++;
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
  if (N >= (1ll << 31) || nz > 65000 || ny > 65535) {
    fail(nullptr, LBM_EINVAL, "lbm_create: lattice too large (N = %lld must be < 2^31, ny <= 65535, nz <= 65000: grid limits)", N);
    return nullptr;
  }
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
  c->wm_prepass = 1;
  c->slip_planes = 1;
  c->use_pdl = 2;
  c->use_graph = 0;
  c->totals_waves = 0;
  c->last = default_params();
  std::snprintf(c->err, sizeof(c->err), "no error");
  const size_t pop = static_cast<size_t>(lattice) * N * dtype;
  int rc = dev_alloc(c, &c->f[0], pop);          // (the second lattice: ensure_lattice1, on first use)
  if (rc == LBM_OK) rc = dev_alloc(c, &c->d, static_cast<size_t>(N) * dtype);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->cls), N);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->cls_alt), N);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->flags_raw), N);
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->nbmask), static_cast<size_t>(N) * sizeof(uint32_t));
  const size_t tot_bytes = (8 + 5 * LBM_TOT_SLOTS + 1) * sizeof(double);      // result, slots, ticket (see make_args)
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->counters), 16 * sizeof(unsigned long long));
  if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->totals_dev), tot_bytes);
  if (rc == LBM_OK && cudaMemset(c->totals_dev, 0, tot_bytes) != cudaSuccess) rc = fail(c, LBM_ECUDA, "cudaMemset failed");
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
  cudaFree(c->f[0]);  cudaFree(c->f[1]);  cudaFree(c->d);  cudaFree(c->uhat);  cudaFree(c->uhat2);  cudaFree(c->ub);
  cudaFree(c->uin_mean);  cudaFree(c->uin_field[0]);  cudaFree(c->uin_field[1]);  cudaFree(c->vpos);  cudaFree(c->vsign);  cudaFree(c->vgamma);
  cudaFree(c->cls);  cudaFree(c->cls_alt);  cudaFree(c->flags_raw);
  cudaFree(c->counters);  cudaFree(c->totals_dev);  cudaFree(c->staging);
  cudaFree(c->list);  cudaFree(c->cub_tmp);  cudaFree(c->list_count_dev);
  cudaFree(c->nbmask);  cudaFree(c->solid_list);  cudaFree(c->solid_vals);
  cudaFree(c->wm_list);  cudaFree(c->wm_ub);  cudaFree(c->uin_scratch);  cudaFree(c->halo_buf);
  for (int k = 0; k < LBM_GRAPH_CACHE; ++k)
    if (c->graphs[k].valid) cudaGraphExecDestroy(c->graphs[k].exec);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
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
  c->lag_valid = false;    // collision = 2: a new geometry or state has no u^ history (G41)
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
  c->solid_dirty = false;
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
  int rc = LBM_DISPATCH(c, launch_init, c, drho, du);
  if (rc != LBM_OK) return rc;
  if (hr || hu) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  c->cur = 0;
  c->phase = PHASE_PRE;
  c->solid_dirty = false;
  c->lag_valid = false;
  c->steps = 0;
  { int rci = reset_inflow(c); if (rci != LBM_OK) return rci; }
  return solid_values(c, true);
}

// POST -> PRE: write S_t = stream(F_{t-1}) into the other lattice and make it current
static int materialise(lbm_ctx* c) {
  if (c->phase == PHASE_SWAPPED) {       // in-place stepping, odd number of steps: un-swap and stream into the other lattice
    lbm_params p = c->last;
    int rc = ensure_lattice1(c);
    if (rc == LBM_OK) rc = LBM_DISPATCH(c, launch_aa, c, &p, 2);
    if (rc != LBM_OK) return rc;
    c->phase = PHASE_PRE;
    c->solid_dirty = false;
    return solid_values(c, false);       // the wall cells' own values into the lattice that now holds S_t
  }
  if (c->phase == PHASE_PRE && c->solid_dirty) {     // in-place steps left whatever in the wall cells' slots: put their own values back
    c->solid_dirty = false;
    return solid_values(c, false);
  }
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
    if (c->has_d) c->epoch++;
    c->has_d = false;
    return LBM_OK;
  }
  LBM_CUDA(c, cudaMemcpyAsync(c->d, porosity, static_cast<size_t>(c->N) * c->dtype, cudaMemcpyDefault, c->stream));
  if (!is_device_pointer(porosity)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  if (!c->has_d) c->epoch++;
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
      c->epoch++;
    }
    return LBM_OK;
  }
  if (!c->ub) {
    int rc = dev_alloc(c, &c->ub, bytes);
    if (rc != LBM_OK) return rc;
    c->epoch++;
  }
  LBM_CUDA(c, cudaMemcpyAsync(c->ub, u_body, bytes, cudaMemcpyDefault, c->stream));
  if (!is_device_pointer(u_body)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

int lbm_set_inflow(lbm_ctx* c, const void* u_mean) {
  if (!c) return LBM_EINVAL;
  const long long n = 3ll * c->ny * c->nz;
  const size_t bytes = static_cast<size_t>(n) * sizeof(double);       // kept in fp64 whatever the dtype
  if (u_mean && (c->ghost_lo || c->ghost_hi))
    return fail(c, LBM_ESTATE, "lbm_set_inflow: the Vortex Method inlet works on the whole inflow plane; not available on a sub-domain (lbm_set_halo)");
  // the state S_t keeps the inflow it was formed with
  int rc = materialise(c);
  if (rc != LBM_OK) return rc;
  if (!u_mean) {
    if (c->uin_mean) {
      LBM_CUDA(c, cudaStreamSynchronize(c->stream));
      cudaFree(c->uin_mean);  cudaFree(c->uin_field[0]);  cudaFree(c->uin_field[1]);  cudaFree(c->uin_scratch);
      c->uin_mean = c->uin_field[0] = c->uin_field[1] = nullptr;
      c->uin_scratch = nullptr;
      c->device_bytes -= 3 * bytes + static_cast<size_t>(n) * sizeof(float);
      c->epoch++;
    }
    return LBM_OK;
  }
  if (!c->uin_mean) {
    rc = dev_alloc(c, reinterpret_cast<void**>(&c->uin_mean), bytes);
    if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->uin_field[0]), bytes);
    if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->uin_field[1]), bytes);
    // fp32 <-> fp64 conversions go through a buffer of their own: the idle field buffer belongs to the side stream, which may
    // be writing the next level's inflow into it while a queued conversion still reads or writes it
    if (rc == LBM_OK) rc = dev_alloc(c, reinterpret_cast<void**>(&c->uin_scratch), static_cast<size_t>(n) * sizeof(float));
    if (rc != LBM_OK) return rc;
    c->uin_cur = 0;
    c->epoch++;
  }
  if (c->dtype == LBM_F64) {
    LBM_CUDA(c, cudaMemcpyAsync(c->uin_mean, u_mean, bytes, cudaMemcpyDefault, c->stream));
  } else {                               // fp32 input -> scratch -> fp64
    float* tmp = c->uin_scratch;
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
  } else {                               // fp64 -> fp32 through the conversion scratch (main stream only)
    float* tmp = c->uin_scratch;
    lbm::k_convert<double, float><<<static_cast<unsigned>((n + 255) / 256), 256, 0, c->stream>>>(c->uin_field[c->uin_cur], tmp, n);
    LBM_CUDA(c, cudaGetLastError());
    c->launches++;
    LBM_CUDA(c, cudaMemcpyAsync(u, tmp, static_cast<size_t>(n) * sizeof(float), cudaMemcpyDefault, c->stream));
  }
  if (!is_device_pointer(u)) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

// ---- CUDA graphs ("cuda_graph", default off: measured neutral beside programmatic dependent launch, and a capture inside a
// caller's timed region costs more than it can win): the steady-state time loop is replayed in chunks of LBM_GRAPH_CHUNK steps from a
// captured graph (one graph launch instead of 8 .. 24 kernel launches: matters where a step is shorter than its launches, i.e.
// small lattices and the three-launch steps of the lid-driven cavity).  A chunk is an even number of steps, so the lattice roles
// and the sweep direction are back where they started; one graph per (current lattice, sweep parity), re-captured when the
// parameters or anything else baked into the kernel arguments changed (epoch).  Not used with the Vortex Method inlet (its
// side stream and events are ordered on the host) and not for the first step of a fresh state.
static void graph_drop(lbm_graph_entry& g) {
  if (g.valid) cudaGraphExecDestroy(g.exec);
  g.valid = false;
}

static int graph_chunk(lbm_ctx* c, const lbm_params* params, bool* done) {
  *done = false;
  const int parity = static_cast<int>(c->sweep_count & 1);
  lbm_graph_entry& g = c->graphs[c->cur * 2 + parity];
  if (g.valid && (g.epoch != c->epoch || std::memcmp(&g.params, params, sizeof(lbm_params)) != 0)) graph_drop(g);
  if (!g.valid) {
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
      cudaGetLastError();
      c->use_graph = 0;
  c->totals_waves = 0;
      return LBM_OK;
    }
    // capture on the private stream; nothing executes, so the bookkeeping the launches advance is put back afterwards
    const cudaStream_t user = c->stream;
    const int cur0 = c->cur;
    const long long sweep0 = c->sweep_count, launches0 = c->launches;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
      cudaGetLastError();
      c->use_graph = 0;
  c->totals_waves = 0;
      return LBM_OK;
    }
    c->stream = c->cap_stream;
    c->prev_launch_prepass = false;
    int rc = LBM_OK;
    for (int k = 0; k < LBM_GRAPH_CHUNK && rc == LBM_OK; ++k) rc = launch_step(c, params, lbm::MODE_STREAM_COLLIDE);
    const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
    c->stream = user;
    c->cur = cur0;
    c->sweep_count = sweep0;
    g.launches = c->launches - launches0;
    c->launches = launches0;
    c->prev_launch_prepass = false;
    if (rc != LBM_OK || e != cudaSuccess || graph == nullptr) {
      if (graph) cudaGraphDestroy(graph);
      cudaGetLastError();
      c->use_graph = 0;                 // capture is not available here: the plain launch path does the same work
      return LBM_OK;
    }
    const cudaError_t ei = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess) {
      cudaGetLastError();
      c->use_graph = 0;
  c->totals_waves = 0;
      return LBM_OK;
    }
    g.valid = true;
    g.params = *params;
    g.epoch = c->epoch;
    g.cur = cur0;
    g.sweep_parity = parity;
  }
  LBM_CUDA(c, cudaGraphLaunch(g.exec, c->stream));
  c->sweep_count += LBM_GRAPH_CHUNK;        // cur is unchanged after an even number of steps
  c->launches += g.launches;
  c->graph_launches++;
  c->prev_launch_prepass = false;
  *done = true;
  return LBM_OK;
}

// In-place (AA pattern) stepping applies to lattices without a single boundary cell, BGK form, rows the vector kernels take
static bool inplace_eligible(const lbm_ctx* c, const lbm_params* p) {
  if (!c->inplace || !c->use_vector || c->uin_mean || c->ghost_lo || c->ghost_hi) return false;
  // plain fluid, or plain fluid + resting SOLID cells (halfway bounce-back): no inlet / outlet / wall-model / moving / slip cell
  if (c->n_typed != 0 || c->n_moving != 0 || c->n_slip != 0 || c->n_list != 0) return false;
  if (p->collision != LBM_COLLISION_BGK) return false;
  const int V = (c->Q == 19 ? 16 : 8) / c->dtype;             // cells per thread of the BGK vector kernels
  if (V < 1 || c->nx % V != 0) return false;
  const int nvec = c->nx / V;
  return nvec % 32 == 0 && nvec <= 256;
}

// buffers a step needs beyond the lattices: u^ field (HRR form), u^B of the wall-model cells (pre-pass)
static int step_buffers(lbm_ctx* c, const lbm_params* params, int n_steps) {
  int rc = LBM_OK;
  if (params->collision != LBM_COLLISION_BGK && !c->uhat && n_steps > 0) {
    const size_t bytes = 3 * static_cast<size_t>(c->N) * c->dtype;
    rc = dev_alloc(c, &c->uhat, bytes);
    if (rc != LBM_OK) return rc;
    // SOLID cells of all-SOLID lines are never written by the UHAT pass: u^ = 0 there (resting wall) from here on
    LBM_CUDA(c, cudaMemsetAsync(c->uhat, 0, bytes, c->stream));
    c->epoch++;
  }
  if (params->collision == LBM_COLLISION_HRR_LAG && !c->uhat2 && n_steps > 0) {     // G41: the second u^ buffer
    rc = dev_alloc(c, &c->uhat2, 3 * static_cast<size_t>(c->N) * c->dtype);
    if (rc != LBM_OK) return rc;
    c->lag_valid = false;
    c->epoch++;
  }
  if (params->wm_enable && c->wm_prepass && c->n_wm > 0 && !c->wm_ub && n_steps > 0) {
    // u^B of the wall-model cells, addressed by cell (only their entries are ever touched)
    rc = dev_alloc(c, &c->wm_ub, 3 * static_cast<size_t>(c->N) * c->dtype);
    if (rc != LBM_OK) return rc;
    c->epoch++;
  }
  return LBM_OK;
}

int lbm_step(lbm_ctx* c, int n_steps, const lbm_params* params) {
  if (!c) return LBM_EINVAL;
  int rc = check_params(c, params);
  if (rc != LBM_OK) return rc;
  if (n_steps < 0) return fail(c, LBM_EINVAL, "lbm_step: n_steps = %d must be >= 0", n_steps);
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_step: no state; call lbm_set_fields or lbm_init_equilibrium first");
  if (c->ghost_lo + c->ghost_hi > 0)
    return fail(c, LBM_ESTATE, "lbm_step: the context is a sub-domain with ghost slices (lbm_set_halo): advance it with lbm_step_halo and exchange the halos");
  c->last = *params;
  if (params->collision != LBM_COLLISION_HRR_LAG && n_steps > 0) c->lag_valid = false;   // G41: steps of another form drop the u^ history
  // ... and so does a new lid velocity: the u^ entries of MOVINGWALL cells in all-wall vectors are written by the u^ pass only
  if (c->n_moving > 0 && std::memcmp(c->lag_u_wall, params->u_wall, sizeof(c->lag_u_wall)) != 0) {
    c->lag_valid = false;
    std::memcpy(c->lag_u_wall, params->u_wall, sizeof(c->lag_u_wall));
  }
  rc = step_buffers(c, params, n_steps);
  if (rc != LBM_OK) return rc;
  int s = 0;
  const bool inplace = inplace_eligible(c, params);
  if (!inplace && c->phase == PHASE_SWAPPED && n_steps > 0) {
    rc = materialise(c);
    if (rc != LBM_OK) return rc;
  }
  while (s < n_steps) {
    if (inplace) {                                             // AA pattern on the current lattice alone (option "inplace")
      if (c->phase == PHASE_POST) {
        rc = materialise(c);
        if (rc != LBM_OK) return rc;
      }
      rc = LBM_DISPATCH(c, launch_aa, c, params, c->phase == PHASE_PRE ? 0 : 1);
      if (rc != LBM_OK) return rc;
      c->phase = (c->phase == PHASE_PRE) ? PHASE_SWAPPED : PHASE_PRE;
      if (c->n_solid > 0) c->solid_dirty = true;
      ++s;
      continue;
    }
    if (c->phase == PHASE_PRE) {
      rc = launch_step(c, params, lbm::MODE_COLLIDE);          // S_t -> F_t
      c->phase = PHASE_POST;
    } else if (c->use_graph && !c->uin_mean && params->collision != LBM_COLLISION_HRR_LAG && n_steps - s >= LBM_GRAPH_CHUNK) {
      bool done = false;
      rc = graph_chunk(c, params, &done);
      if (rc != LBM_OK) return rc;
      if (done) { s += LBM_GRAPH_CHUNK; continue; }
      continue;                                                // capture unavailable: use_graph is off now
    } else {
      rc = ensure_inflow(c, c->steps + s);                     // Vortex Method inlet: the inflow S_t carries (Eq. 21)
      if (rc != LBM_OK) return rc;
      rc = launch_step(c, params, lbm::MODE_STREAM_COLLIDE);   // F_{t-1} -> S_t -> F_t
    }
    if (rc != LBM_OK) return rc;
    rc = vm_prefetch(c, c->steps + s);                         // inflow of the next level, beside this step
    if (rc != LBM_OK) return rc;
    ++s;
  }
  c->steps += n_steps;
  return LBM_OK;
}

// A9.  Neither call changes the stored lattice or its phase: with the storage holding F_{t-1} the kernels pull S_t in
// registers (one launch over the lattice + one over the wall cells' side buffer for lbm_moments).
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
  int rc = (c->phase == PHASE_SWAPPED) ? materialise(c) : LBM_OK;
  if (rc != LBM_OK) return rc;
  rc = (c->phase == PHASE_POST) ? ensure_inflow(c, c->steps) : LBM_OK;     // the inlet rule is part of the pull
  if (rc != LBM_OK) return rc;
  rc = LBM_DISPATCH(c, launch_moments, c, &p, drho, du);
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

int lbm_get_populations_box(lbm_ctx* c, int x0, int y0, int z0, int bx, int by, int bz, void* populations) {
  if (!c) return LBM_EINVAL;
  if (!populations) return fail(c, LBM_EINVAL, "lbm_get_populations_box: populations is NULL");
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_get_populations_box: no state");
  if (bx < 1 || by < 1 || bz < 1 || x0 < 0 || y0 < 0 || z0 < 0 || x0 + bx > c->nx || y0 + by > c->ny || z0 + bz > c->nz)
    return fail(c, LBM_EINVAL, "lbm_get_populations_box: box (%d,%d,%d)+(%d,%d,%d) is empty or leaves the lattice", x0, y0, z0, bx, by, bz);
  const long long n = static_cast<long long>(c->Q) * bx * by * bz;
  const size_t bytes = static_cast<size_t>(n) * c->dtype;
  int rc = materialise(c);
  if (rc != LBM_OK) return rc;
  const bool host = !is_device_pointer(populations);
  void* dst = populations;
  if (host) {
    rc = ensure_staging(c, bytes);
    if (rc != LBM_OK) return rc;
    dst = c->staging;
  }
  const unsigned blocks = static_cast<unsigned>((n + 255) / 256);
  if (c->dtype == LBM_F32)
    lbm::k_gather_box<float><<<blocks, 256, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), c->N, c->nx, c->ny, x0, y0, z0, bx, by, bz, c->Q, static_cast<float*>(dst));
  else
    lbm::k_gather_box<double><<<blocks, 256, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), c->N, c->nx, c->ny, x0, y0, z0, bx, by, bz, c->Q, static_cast<double*>(dst));
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  if (host) {
    LBM_CUDA(c, cudaMemcpyAsync(populations, dst, bytes, cudaMemcpyDeviceToHost, c->stream));
    LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return LBM_OK;
}

int lbm_set_populations_box(lbm_ctx* c, int x0, int y0, int z0, int bx, int by, int bz, const void* populations) {
  if (!c) return LBM_EINVAL;
  if (!populations) return fail(c, LBM_EINVAL, "lbm_set_populations_box: populations is NULL");
  if (bx < 1 || by < 1 || bz < 1 || x0 < 0 || y0 < 0 || z0 < 0 || x0 + bx > c->nx || y0 + by > c->ny || z0 + bz > c->nz)
    return fail(c, LBM_EINVAL, "lbm_set_populations_box: box (%d,%d,%d)+(%d,%d,%d) is empty or leaves the lattice", x0, y0, z0, bx, by, bz);
  const long long n = static_cast<long long>(c->Q) * bx * by * bz;
  const size_t bytes = static_cast<size_t>(n) * c->dtype;
  int rc = LBM_OK;
  if (c->phase == PHASE_NONE) {          // no state yet: this call starts one (the caller covers the lattice box by box)
    c->cur = 0;
    c->phase = PHASE_PRE;
    c->steps = 0;
    rc = reset_inflow(c);
  } else {
    rc = materialise(c);                 // the lattice must hold S_t itself (wall cells' own values included)
  }
  c->lag_valid = false;                  // the state changes under the u^ history of collision = 2 (G41)
  if (rc != LBM_OK) return rc;
  const bool host = !is_device_pointer(populations);
  const void* src = populations;
  if (host) {
    rc = ensure_staging(c, bytes);
    if (rc != LBM_OK) return rc;
    LBM_CUDA(c, cudaMemcpyAsync(c->staging, populations, bytes, cudaMemcpyHostToDevice, c->stream));
    src = c->staging;
  }
  const unsigned blocks = static_cast<unsigned>((n + 255) / 256);
  if (c->dtype == LBM_F32)
    lbm::k_scatter_box<float><<<blocks, 256, 0, c->stream>>>(static_cast<float*>(c->f[c->cur]), c->N, c->nx, c->ny, x0, y0, z0, bx, by, bz, c->Q, static_cast<const float*>(src));
  else
    lbm::k_scatter_box<double><<<blocks, 256, 0, c->stream>>>(static_cast<double*>(c->f[c->cur]), c->N, c->nx, c->ny, x0, y0, z0, bx, by, bz, c->Q, static_cast<const double*>(src));
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  if (host) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return solid_values(c, true);          // wall cells inside the box: their own values live in the side buffer
}

int lbm_totals(lbm_ctx* c, double out[5]) {
  if (!c) return LBM_EINVAL;
  if (!out) return fail(c, LBM_EINVAL, "lbm_totals: out is NULL");
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_totals: no state");
  lbm_params p = c->last;
  int rc = (c->phase == PHASE_SWAPPED) ? materialise(c) : LBM_OK;
  if (rc != LBM_OK) return rc;
  rc = (c->phase == PHASE_POST) ? ensure_inflow(c, c->steps) : LBM_OK;
  if (rc != LBM_OK) return rc;
  rc = LBM_DISPATCH(c, launch_totals, c, &p);
  if (rc != LBM_OK) return rc;
  const bool dev = is_device_pointer(out);
  LBM_CUDA(c, cudaMemcpyAsync(out, c->totals_dev, 5 * sizeof(double), cudaMemcpyDefault, c->stream));
  if (!dev) LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  return LBM_OK;
}

// ---- slab decomposition in z: ghost slices, staged step, halo pack / unpack ------
// wall-model cells whose sample point lies in a ghost slice cannot be served (their pre-pass would pull from beyond the halo)
static int check_wm_cut(lbm_ctx* c, int ghost_lo, int ghost_hi) {
  c->halo_wm_epoch = c->epoch;
  if (!(ghost_lo || ghost_hi) || c->n_wm <= 0) return LBM_OK;
  LBM_CUDA(c, cudaMemsetAsync(c->counters, 0, sizeof(unsigned long long), c->stream));
  const long long plane = static_cast<long long>(c->nx) * c->ny;
  lbm::k_count_wm_on_cut<<<static_cast<unsigned>((plane + 255) / 256), 256, 0, c->stream>>>(c->cls, plane, c->nz, ghost_lo, ghost_hi, c->counters);
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  unsigned long long bad = 0;
  LBM_CUDA(c, cudaMemcpyAsync(&bad, c->counters, sizeof(bad), cudaMemcpyDeviceToHost, c->stream));
  LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  if (bad) {
    c->halo_wm_epoch = -1;
    return fail(c, LBM_EINVAL, "halo: %llu WALLMODEL cell(s) sample their velocity in a ghost slice (wall normal across the cut): move the cut", bad);
  }
  return LBM_OK;
}

int lbm_set_halo(lbm_ctx* c, int ghost_lo, int ghost_hi) {
  if (!c) return LBM_EINVAL;
  if ((ghost_lo != 0 && ghost_lo != 1) || (ghost_hi != 0 && ghost_hi != 1))
    return fail(c, LBM_EINVAL, "lbm_set_halo: ghost_lo = %d, ghost_hi = %d must be 0 or 1", ghost_lo, ghost_hi);
  if (c->nz - ghost_lo - ghost_hi < 1) return fail(c, LBM_EINVAL, "lbm_set_halo: no interior slice left (nz = %d)", c->nz);
  if ((ghost_lo || ghost_hi) && c->uin_mean)
    return fail(c, LBM_ESTATE, "lbm_set_halo: the Vortex Method inlet works on the whole inflow plane; not available on a sub-domain");
  { int rcw = check_wm_cut(c, ghost_lo, ghost_hi); if (rcw != LBM_OK) return rcw; }
  int rc = materialise(c);               // a pass over the old interior; the ghost slices start without valid contents
  if (rc != LBM_OK) return rc;
  c->ghost_lo = ghost_lo;
  c->ghost_hi = ghost_hi;
  c->halo_stage = 0;
  c->epoch++;
  c->halo_wm_epoch = c->epoch;
  return LBM_OK;
}

int lbm_step_halo(lbm_ctx* c, const lbm_params* params, int stage) {
  if (!c) return LBM_EINVAL;
  int rc = check_params(c, params);
  if (rc != LBM_OK) return rc;
  if (stage != 0 && stage != 1) return fail(c, LBM_EINVAL, "lbm_step_halo: stage = %d must be 0 or 1", stage);
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "lbm_step_halo: no state");
  if (c->uin_mean) return fail(c, LBM_ESTATE, "lbm_step_halo: not available with the Vortex Method inlet");
  if (stage != c->halo_stage) return fail(c, LBM_ESTATE, "lbm_step_halo: stage %d called where stage %d is due", stage, c->halo_stage);
  if (params->wm_enable && c->halo_wm_epoch != c->epoch) {       // the geometry changed since the cut was checked
    rc = check_wm_cut(c, c->ghost_lo, c->ghost_hi);
    if (rc != LBM_OK) return rc;
  }
  if (c->phase == PHASE_SWAPPED) {
    rc = materialise(c);
    if (rc != LBM_OK) return rc;
  }
  c->last = *params;
  if (params->collision != LBM_COLLISION_HRR_LAG && stage != 1) c->lag_valid = false;   // G41: steps of another form drop the u^ history
  if (c->n_moving > 0 && stage != 1 && std::memcmp(c->lag_u_wall, params->u_wall, sizeof(c->lag_u_wall)) != 0) {
    c->lag_valid = false;
    std::memcpy(c->lag_u_wall, params->u_wall, sizeof(c->lag_u_wall));
  }
  rc = step_buffers(c, params, 1);
  if (rc != LBM_OK) return rc;
  const int mode = (c->phase == PHASE_PRE) ? lbm::MODE_COLLIDE : lbm::MODE_STREAM_COLLIDE;
  rc = launch_step(c, params, mode, stage);
  if (rc != LBM_OK) return rc;
  if (stage == 0) {
    c->halo_stage = 1;
  } else {
    c->halo_stage = 0;
    c->phase = PHASE_POST;
    c->steps += 1;
  }
  return LBM_OK;
}

// planes of one face buffer and the slice they live in
static int halo_planes(lbm_ctx* c, const char* who, int what, int side, bool pack, lbm::HaloPlanes* hp, int* z, void** field) {
  if (what != LBM_HALO_POPULATIONS && what != LBM_HALO_UHAT) return fail(c, LBM_EINVAL, "%s: what = %d must be 0 (populations) or 1 (u^)", who, what);
  if (side != LBM_SIDE_LOW && side != LBM_SIDE_HIGH) return fail(c, LBM_EINVAL, "%s: side = %d must be 0 (low) or 1 (high)", who, side);
  if ((side == LBM_SIDE_LOW && !c->ghost_lo) || (side == LBM_SIDE_HIGH && !c->ghost_hi))
    return fail(c, LBM_ESTATE, "%s: no ghost slice on side %d (lbm_set_halo)", who, side);
  if (c->phase == PHASE_NONE) return fail(c, LBM_ESTATE, "%s: no state", who);
  // pack reads the boundary INTERIOR slice, unpack writes the GHOST slice
  if (side == LBM_SIDE_LOW) *z = pack ? c->ghost_lo : 0;
  else *z = pack ? c->nz - 1 - c->ghost_hi : c->nz - 1;
  if (what == LBM_HALO_UHAT) {
    if (!c->uhat) return fail(c, LBM_ESTATE, "%s: no u^ field (the HRR form has not run yet)", who);
    hp->n = 3;
    hp->idx[0] = 0;  hp->idx[1] = 1;  hp->idx[2] = 2;
    // collision = 2 (G41): the buffer the next fused step READS -- u^ of the previous level (or, on the first step of a history, the
    // u^ pass's output), whose ghost slices the exchange fills
    *field = (c->last.collision == LBM_COLLISION_HRR_LAG && c->uhat2 && c->lag_cur == 1) ? c->uhat2 : c->uhat;
    return LBM_OK;
  }
  // the populations that cross the cut: leaving downwards (c_z = -1) from the low boundary slice, upwards from the high one;
  // the ghost slice on the low side receives what travels upwards (c_z = +1), the one on the high side c_z = -1
  const int want = ((side == LBM_SIDE_LOW) == pack) ? -1 : +1;
  hp->n = 0;
  if (c->Q == 19) {
    constexpr lbm::Stencil<19> L{};
    for (int i = 0; i < 19; ++i) if (L.c[i][2] == want) hp->idx[hp->n++] = i;
  } else {
    constexpr lbm::Stencil<27> L{};
    for (int i = 0; i < 27; ++i) if (L.c[i][2] == want) hp->idx[hp->n++] = i;
  }
  *field = c->f[c->cur];
  return LBM_OK;
}

static int halo_copy(lbm_ctx* c, const char* who, int what, int side, void* buf, bool pack) {
  if (!c) return LBM_EINVAL;
  if (!buf) return fail(c, LBM_EINVAL, "%s: buffer is NULL", who);
  lbm::HaloPlanes hp;
  int z = 0;
  void* field = nullptr;
  int rc = halo_planes(c, who, what, side, pack, &hp, &z, &field);
  if (rc != LBM_OK) return rc;
  const long long plane = static_cast<long long>(c->nx) * c->ny;
  const size_t bytes = static_cast<size_t>(hp.n) * plane * c->dtype;
  const bool host = !is_device_pointer(buf);
  void* dbuf = buf;
  if (host) {
    if (c->halo_buf_bytes < bytes) {
      if (c->halo_buf) { cudaStreamSynchronize(c->stream); cudaFree(c->halo_buf); c->device_bytes -= c->halo_buf_bytes; c->halo_buf = nullptr; c->halo_buf_bytes = 0; }
      rc = dev_alloc(c, &c->halo_buf, bytes);
      if (rc != LBM_OK) return rc;
      c->halo_buf_bytes = bytes;
    }
    dbuf = c->halo_buf;
    if (!pack) LBM_CUDA(c, cudaMemcpyAsync(dbuf, buf, bytes, cudaMemcpyHostToDevice, c->stream));
  }
  unsigned blocks = static_cast<unsigned>((plane + 255) / 256);
  if (blocks > 148u * 8u) blocks = 148u * 8u;
  const long long off = static_cast<long long>(z) * plane;
  if (c->dtype == LBM_F32) {
    if (pack) lbm::k_halo_planes<float, true><<<blocks, 256, 0, c->stream>>>(static_cast<float*>(field), c->N, off, plane, hp, static_cast<float*>(dbuf));
    else      lbm::k_halo_planes<float, false><<<blocks, 256, 0, c->stream>>>(static_cast<float*>(field), c->N, off, plane, hp, static_cast<float*>(dbuf));
  } else {
    if (pack) lbm::k_halo_planes<double, true><<<blocks, 256, 0, c->stream>>>(static_cast<double*>(field), c->N, off, plane, hp, static_cast<double*>(dbuf));
    else      lbm::k_halo_planes<double, false><<<blocks, 256, 0, c->stream>>>(static_cast<double*>(field), c->N, off, plane, hp, static_cast<double*>(dbuf));
  }
  LBM_CUDA(c, cudaGetLastError());
  c->launches++;
  if (host) {
    if (pack) LBM_CUDA(c, cudaMemcpyAsync(buf, dbuf, bytes, cudaMemcpyDeviceToHost, c->stream));
    LBM_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return LBM_OK;
}

int lbm_halo_pack(lbm_ctx* c, int what, int side, void* buf) { return halo_copy(c, "lbm_halo_pack", what, side, buf, true); }
int lbm_halo_unpack(lbm_ctx* c, int what, int side, const void* buf) {
  return halo_copy(c, "lbm_halo_unpack", what, side, const_cast<void*>(buf), false);
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
    case 7: return c->graph_launches;
    case 8: return c->n_wm;
    case 9: return static_cast<long long>(c->Q == 19 ? 5 : 9) * c->nx * c->ny;
    case 10: return 3ll * c->nx * c->ny;
    case 11: return c->nz - c->ghost_lo - c->ghost_hi;
    case 12: return c->n_slipcode;
    default: return -1;
  }
}

// options that change how the geometry is classified or what the kernel arguments hold invalidate the captured graphs
int lbm_set_option(lbm_ctx* c, const char* key, long long value) {
  if (!c || !key) return LBM_EINVAL;
  if (std::strcmp(key, "cuda_graph") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "cuda_graph must be 0 or 1");
    c->use_graph = static_cast<int>(value);
    return LBM_OK;
  }
  if (std::strcmp(key, "pdl") == 0) {
    if (value < 0 || value > 2) return fail(c, LBM_EINVAL, "pdl must be 0, 1 or 2");
    c->use_pdl = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  if (std::strcmp(key, "wm_prepass") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "wm_prepass must be 0 or 1");
    if (c->phase != PHASE_NONE || c->n_wm > 0)
      return fail(c, LBM_ESTATE, "wm_prepass decides how the flags are classified: set it before lbm_set_fields / lbm_set_geometry");
    c->wm_prepass = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  if (std::strcmp(key, "slip_planes") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "slip_planes must be 0 or 1");
    if (c->phase != PHASE_NONE || c->n_slip > 0)
      return fail(c, LBM_ESTATE, "slip_planes decides how the flags are classified: set it before lbm_set_fields / lbm_set_geometry");
    c->slip_planes = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  if (std::strcmp(key, "totals_waves") == 0) {
    if (value < 0 || value > 64) return fail(c, LBM_EINVAL, "totals_waves must be in [0, 64]");
    c->totals_waves = static_cast<int>(value);
    return LBM_OK;
  }
  if (std::strcmp(key, "block_threads") == 0) {
    if (value != 64 && value != 128 && value != 256) return fail(c, LBM_EINVAL, "block_threads must be 64, 128 or 256");
    c->block_threads = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  if (std::strcmp(key, "serpentine") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "serpentine must be 0 or 1");
    c->serpentine = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  if (std::strcmp(key, "hrr_slab") == 0) {
    if (value < 0) return fail(c, LBM_EINVAL, "hrr_slab must be >= 0");
    c->hrr_slab = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  if (std::strcmp(key, "inplace") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "inplace must be 0 or 1");
    c->inplace = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  if (std::strcmp(key, "vector") == 0) {
    if (value != 0 && value != 1) return fail(c, LBM_EINVAL, "vector must be 0 or 1");
    c->use_vector = static_cast<int>(value);
    c->epoch++;
    return LBM_OK;
  }
  return fail(c, LBM_EINVAL, "unknown option '%s'", key);
}

}  // extern "C"
