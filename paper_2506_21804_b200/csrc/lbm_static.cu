// =====================================================================================
// lbm_static.cu -- lbm_totals_static: the A9 totals (the conserved moments of Eq. 6) for
// callers that cannot allocate: no lbm_ctx, no cudaMalloc / cudaFree / allocating library routine anywhere on its path.
//
// It is a variant of the totals kernel (lbm_kernels.cuh, reduce_totals): that one adds block partial sums into slots the
// context allocated with cudaMalloc; this one keeps its scratch -- one partial sum per block and quantity, and the ticket that
// finds the last block -- in the file-scope array `lbm_static_scratch` below, which every GPU that loads the library holds
// until the process exits (LBM_STATIC_SCRATCH_BYTES = 655 616 bytes).
//
// The array's NAME is a device symbol: in host code it is only a host-side stand-in, never a device address.  Its address on
// the CURRENT device is resolved once per device with cudaGetSymbolAddress (scratch_address below) and handed to the kernel
// as an ordinary pointer argument.
//
// Every call on a device shares the array.  A call clears what must start at zero (the ticket) on its stream before its
// launch; the partial sums need no clearing (every block overwrites its own entries, the last block reads only the entries of
// this launch).  Calls that overlap on the same GPU (two streams, two host threads) race on the array: serialise them.
// =====================================================================================
#include <mutex>

#include "../../include/lbm.h"
#include "lbm_ctx.h"
#include "lbm_kernels.cuh"

namespace {

constexpr int ST_THREADS = 256;                       // threads per block
constexpr int ST_CELLS_PER_BLOCK = 8192;              // consecutive cells per block: fixed, so the summation order is a function of N only
constexpr int ST_MAX_BLOCKS = 16384;                  // => LBM_STATIC_MAX_CELLS = 8192 x 16384 = 134 217 728 cells (512^3)
constexpr int ST_TAIL_DOUBLES = 32;                   // the ticket (an unsigned) lives in the first of them
constexpr size_t ST_SCRATCH_DOUBLES = 5 * static_cast<size_t>(ST_MAX_BLOCKS) + ST_TAIL_DOUBLES;
static_assert(static_cast<long long>(ST_CELLS_PER_BLOCK) * ST_MAX_BLOCKS == LBM_STATIC_MAX_CELLS, "lbm.h states the limit");
static_assert(ST_SCRATCH_DOUBLES * sizeof(double) == LBM_STATIC_SCRATCH_BYTES, "lbm.h states the size");

// part[k][block] (k = 0..4: sum rho, sum j_x, j_y, j_z, sum |j|^2 / (2 rho)), then the ticket
static __device__ __align__(256) double lbm_static_scratch[ST_SCRATCH_DOUBLES];

template <typename T, int V> struct FlagVec;
template <> struct FlagVec<float, 4> { using type = uint32_t; };
template <> struct FlagVec<double, 2> { using type = uint16_t; };
template <> struct FlagVec<float, 1> { using type = uint8_t; };
template <> struct FlagVec<double, 1> { using type = uint8_t; };

// One block = ST_CELLS_PER_BLOCK consecutive cells of S_t, thread = V consecutive cells per iteration (aligned vector loads of
// every population; the host picks V = 1 when N or a pointer does not allow whole vectors).  Per cell: rho = sum f, j = sum c f
// in dtype (cell_moments, as every kernel of the path), accumulated in fp64 from there on: thread -> warp shuffle tree ->
// shared memory -> part[k][block].  The last block (ticket) adds the partial sums of this launch in a fixed order.
template <int Q, typename T, int V>
__global__ void __launch_bounds__(ST_THREADS) k_totals_static(const T* __restrict__ f, const uint8_t* __restrict__ flags, long long N,
                                                              double* __restrict__ scratch, double* __restrict__ out) {
  using FV = typename FlagVec<T, V>::type;
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  const long long base = static_cast<long long>(blockIdx.x) * ST_CELLS_PER_BLOCK;
#pragma unroll 1
  for (int it = 0; it < ST_CELLS_PER_BLOCK / (ST_THREADS * V); ++it) {
    const long long cell = base + (static_cast<long long>(it) * ST_THREADS + threadIdx.x) * V;
    if (cell >= N) break;                               // (N is a multiple of V: a vector is inside or outside as a whole)
    FV fl = 0;
    if (flags != nullptr) fl = *reinterpret_cast<const FV*>(flags + cell);
    T fv[Q][V];
#pragma unroll
    for (int i = 0; i < Q; ++i) lbm::ld_vec(f + static_cast<long long>(i) * N + cell, fv[i]);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      if (lbm::is_wall(static_cast<int>(fl >> (8 * v)) & 15)) continue;      // SOLID, MOVINGWALL, SLIPWALL cells do not count
      T fc[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) fc[i] = fv[i][v];
      T rho, jx, jy, jz;
      lbm::cell_moments<Q, T>(fc, rho, jx, jy, jz);
      const double r = static_cast<double>(rho), x = static_cast<double>(jx), y = static_cast<double>(jy), z = static_cast<double>(jz);
      acc[0] += r;  acc[1] += x;  acc[2] += y;  acc[3] += z;
      acc[4] += 0.5 * (x * x + y * y + z * z) / r;
    }
  }
  __shared__ double part[5][ST_THREADS / 32];
  __shared__ int s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double s = acc[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (lane == 0) part[k][warp] = s;
  }
  __syncthreads();
  if (threadIdx.x < 5) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < ST_THREADS / 32; ++w) s += part[threadIdx.x][w];
    scratch[static_cast<size_t>(threadIdx.x) * ST_MAX_BLOCKS + blockIdx.x] = s;
    __threadfence();
  }
  __syncthreads();
  unsigned* ticket = reinterpret_cast<unsigned*>(scratch + 5 * static_cast<size_t>(ST_MAX_BLOCKS));
  if (threadIdx.x == 0) s_last = (atomicInc(ticket, gridDim.x - 1u) == gridDim.x - 1u) ? 1 : 0;     // wraps to 0 on the last block
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (warp < 5) {                                        // one warp per quantity; lanes take the blocks lane, lane + 32, ... in order
    double s = 0.0;
    for (unsigned b = lane; b < gridDim.x; b += 32) s += __ldcg(scratch + static_cast<size_t>(warp) * ST_MAX_BLOCKS + b);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (lane == 0) out[warp] = s;
  }
}

// ---- host side ----------------------------------------------------------------------------------
constexpr int ST_MAX_DEVICES = 64;
std::mutex g_mutex;
double* g_scratch_dev[ST_MAX_DEVICES];        // device address of lbm_static_scratch, per device (nullptr = not resolved yet)

// Address of the array on the CURRENT device, resolved once per device (the symbol itself is not a device address)
int scratch_address(double** p) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return lbmhost::fail(nullptr, LBM_ECUDA, "lbm_totals_static: no usable CUDA device (%s)", cudaGetErrorString(e));
  if (dev < 0 || dev >= ST_MAX_DEVICES) return lbmhost::fail(nullptr, LBM_EINVAL, "lbm_totals_static: device ordinal %d not supported (< %d)", dev, ST_MAX_DEVICES);
  std::lock_guard<std::mutex> lock(g_mutex);
  if (g_scratch_dev[dev] == nullptr) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), lbm_static_scratch);
    if (e != cudaSuccess || ptr == nullptr) {
      cudaGetLastError();
      return lbmhost::fail(nullptr, LBM_ECUDA, "lbm_totals_static: cudaGetSymbolAddress(lbm_static_scratch) on device %d: %s", dev, cudaGetErrorString(e));
    }
    g_scratch_dev[dev] = ptr;
  }
  *p = g_scratch_dev[dev];
  return LBM_OK;
}

bool on_device(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

template <int Q, typename T, int V>
cudaError_t launch(const void* f, const uint8_t* flags, long long N, double* scratch, double* out, cudaStream_t st) {
  const unsigned blocks = static_cast<unsigned>((N + ST_CELLS_PER_BLOCK - 1) / ST_CELLS_PER_BLOCK);
  k_totals_static<Q, T, V><<<blocks, ST_THREADS, 0, st>>>(static_cast<const T*>(f), flags, N, scratch, out);
  return cudaGetLastError();
}

template <int Q>
cudaError_t launch_q(int dtype, bool vec, const void* f, const uint8_t* flags, long long N, double* scratch, double* out, cudaStream_t st) {
  if (dtype == LBM_F32) return vec ? launch<Q, float, 4>(f, flags, N, scratch, out, st) : launch<Q, float, 1>(f, flags, N, scratch, out, st);
  return vec ? launch<Q, double, 2>(f, flags, N, scratch, out, st) : launch<Q, double, 1>(f, flags, N, scratch, out, st);
}

}  // namespace

extern "C" int lbm_totals_static(int lattice, int nx, int ny, int nz, int dtype, const void* populations, const uint8_t* cell_flags,
                                 double* out, void* cuda_stream) {
  using lbmhost::fail;
  if (lattice != LBM_D3Q19 && lattice != LBM_D3Q27) return fail(nullptr, LBM_EINVAL, "lbm_totals_static: lattice %d is not 19 or 27", lattice);
  if (dtype != LBM_F32 && dtype != LBM_F64) return fail(nullptr, LBM_EINVAL, "lbm_totals_static: dtype %d is not 4 (f32) or 8 (f64)", dtype);
  if (nx < 1 || ny < 1 || nz < 1) return fail(nullptr, LBM_EINVAL, "lbm_totals_static: nx, ny, nz must be >= 1 (got %d %d %d)", nx, ny, nz);
  const long long N = static_cast<long long>(nx) * ny * nz;
  if (N > LBM_STATIC_MAX_CELLS)
    return fail(nullptr, LBM_EINVAL, "lbm_totals_static: %lld cells exceed the limit of %lld (LBM_STATIC_MAX_CELLS: the static scratch array "
                "holds one partial sum per block of %d cells); use lbm_totals on a context", N, static_cast<long long>(LBM_STATIC_MAX_CELLS), ST_CELLS_PER_BLOCK);
  if (populations == nullptr || out == nullptr) return fail(nullptr, LBM_EINVAL, "lbm_totals_static: populations and out must not be NULL");
  if (!on_device(populations) || !on_device(out) || (cell_flags != nullptr && !on_device(cell_flags)))
    return fail(nullptr, LBM_EINVAL, "lbm_totals_static: populations, cell_flags and out must be DEVICE pointers (a host buffer would need staging memory)");
  if (reinterpret_cast<uintptr_t>(populations) % static_cast<unsigned>(dtype) != 0 || reinterpret_cast<uintptr_t>(out) % 8 != 0)
    return fail(nullptr, LBM_EINVAL, "lbm_totals_static: populations / out are not aligned to their element size");
  double* scratch = nullptr;
  int rc = scratch_address(&scratch);
  if (rc != LBM_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // whole 16-byte vectors of every population (and whole flag words) or one cell per thread
  const int V = 16 / dtype;
  const bool vec = (N % V == 0) && (reinterpret_cast<uintptr_t>(populations) % 16 == 0) &&
                   (cell_flags == nullptr || reinterpret_cast<uintptr_t>(cell_flags) % V == 0);
  // what must start at zero: the ticket (the last block of a completed launch leaves it at zero, a failed launch may not)
  cudaError_t e = cudaMemsetAsync(scratch + 5 * static_cast<size_t>(ST_MAX_BLOCKS), 0, sizeof(unsigned), st);
  if (e == cudaSuccess) e = (lattice == LBM_D3Q19) ? launch_q<19>(dtype, vec, populations, cell_flags, N, scratch, out, st)
                                                   : launch_q<27>(dtype, vec, populations, cell_flags, N, scratch, out, st);
  if (e != cudaSuccess) return fail(nullptr, LBM_ECUDA, "lbm_totals_static: %s", cudaGetErrorString(e));
  return LBM_OK;
}
