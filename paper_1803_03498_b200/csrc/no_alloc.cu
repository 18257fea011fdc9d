// no_alloc.cu -- heom_level_max_static: the growth monitor of heom_level_max (Eq. 38; R6/A7) for
// callers that may not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  A variant of level_max_kernel (kernels_generic.cu) whose scratch -- the per-level running maxima and
// the counter that elects the finishing block -- lives in a file-scope __device__ array of fixed size instead of
// the context's workspace.  The entry point calls no cudaMalloc / cudaFree and no allocating library routine; the
// caller passes the state, the level of every node and the output, all DEVICE pointers.
//
// Every GPU that loads the library holds the array (kStaticScratchBytes = 768 bytes) until the process exits.
// Every call on a device shares it: the call clears it first (stream-ordered), so the contents a previous call
// left behind never leak into a result, but two calls that OVERLAP on the GPU (different streams, no ordering
// between them) race on it.  Order them (same stream, or an event) or use heom_level_max.
#include "../../include/heom.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

namespace {

constexpr int kStaticMaxDepth = HEOM_STATIC_MAX_DEPTH;        // levels L = 0..63
constexpr int kStaticSlots = kStaticMaxDepth + 1;              // running maxima (bit patterns of doubles >= 0)
constexpr int kStaticWords = 96;                               // 64 maxima + finished-blocks counter, padded
constexpr size_t kStaticScratchBytes = kStaticWords * sizeof(unsigned long long);
constexpr int kMaxDevices = 64;
static_assert(kStaticSlots + 1 <= kStaticWords && kStaticScratchBytes % 256 == 0, "scratch layout");

// In host code this name is a host-side stand-in, NOT a device address: the address the kernel gets comes from
// cudaGetSymbolAddress (scratch_of below), once per device, with that device current.
static __device__ __align__(256) unsigned long long g_static_scratch[kStaticWords];

thread_local char t_error[256] = "";

heom_status fail(heom_status st, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) std::snprintf(t_error, sizeof t_error, "%s: %s", what, cudaGetErrorString(e));
  else std::snprintf(t_error, sizeof t_error, "%s", what);
  return st;
}

std::mutex g_mutex;
unsigned long long* g_scratch_ptr[kMaxDevices] = {};

// device address of g_static_scratch on `device` (which must be current)
cudaError_t scratch_of(int device, unsigned long long** out) {
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch_ptr[device]) {
    unsigned long long* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_ptr[device] = ptr;
  }
  *out = g_scratch_ptr[device];
  return cudaSuccess;
}

// max(|Re|, |Im|) over the nodes of every hierarchy level.  scratch[L], L <= depth: running maximum (cleared by
// the caller); scratch[kStaticSlots]: number of blocks that have finished.  The last block to finish converts the
// maxima to doubles in out[0..depth].  Levels above depth (a malformed level array) are ignored.
__global__ void __launch_bounds__(256) level_max_static_kernel(const double2* __restrict__ state,
                                                               const uint8_t* __restrict__ level, long long nodes,
                                                               int per, int depth, unsigned long long* scratch,
                                                               double* __restrict__ out) {
  __shared__ unsigned long long smax[kStaticSlots];
  __shared__ bool last;
  for (int e = threadIdx.x; e < kStaticSlots; e += blockDim.x) smax[e] = 0ULL;
  __syncthreads();
  const long long total = nodes * per;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const double2 v = state[t];
    const double a = fmax(fabs(v.x), fabs(v.y));          // max-norm of the element: |re|, |im|
    // NaN counts as +inf (fmax drops a NaN operand: test the parts themselves)
    const double m = (v.x == v.x && v.y == v.y) ? a : __longlong_as_double(0x7ff0000000000000LL);
    const int L = level[t / per];
    if (L <= depth) atomicMax(&smax[L], (unsigned long long)__double_as_longlong(m));
  }
  __syncthreads();
  for (int e = threadIdx.x; e <= depth; e += blockDim.x)
    if (smax[e]) atomicMax(&scratch[e], smax[e]);
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) last = atomicAdd(&scratch[kStaticSlots], 1ULL) == (unsigned long long)gridDim.x - 1ULL;
  __syncthreads();
  if (!last) return;
  __threadfence();
  for (int e = threadIdx.x; e <= depth; e += blockDim.x)
    out[e] = __longlong_as_double((long long)atomicMax(&scratch[e], 0ULL));   // atomic read of the final value
}

}  // namespace

extern "C" const char* heom_static_last_error(void) { return t_error; }

extern "C" heom_status heom_level_max_static(int device, const void* state_dev, const uint8_t* level_dev,
                                             int64_t nodes, int elems_per_node, int depth, double* max_abs_dev,
                                             void* cuda_stream) {
  t_error[0] = 0;
  if (!state_dev || !level_dev || !max_abs_dev) return fail(HEOM_EINVAL, "heom_level_max_static: NULL pointer");
  if (device < 0 || device >= kMaxDevices) return fail(HEOM_EINVAL, "heom_level_max_static: device ordinal out of range");
  if (depth < 0 || depth > kStaticMaxDepth) {
    std::snprintf(t_error, sizeof t_error,
                  "heom_level_max_static: depth %d is outside 0..%d, the levels the static scratch holds "
                  "(use heom_level_max)", depth, kStaticMaxDepth);
    return HEOM_EINVAL;
  }
  if (nodes < 0 || elems_per_node < 1 || elems_per_node > 65536 || nodes > (int64_t)1 << 40)
    return fail(HEOM_EINVAL, "heom_level_max_static: nodes or elems_per_node out of range");
  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e != cudaSuccess) return fail(HEOM_ECUDA, "cudaGetDevice", e);
  if (prev != device && (e = cudaSetDevice(device)) != cudaSuccess) return fail(HEOM_ECUDA, "cudaSetDevice", e);
  heom_status st = HEOM_OK;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  unsigned long long* scratch = nullptr;
  if ((e = scratch_of(device, &scratch)) != cudaSuccess) st = fail(HEOM_ECUDA, "cudaGetSymbolAddress", e);
  // the array keeps the last call's maxima (and, after an aborted call, a partial counter): clear all of it
  if (st == HEOM_OK && (e = cudaMemsetAsync(scratch, 0, kStaticScratchBytes, s)) != cudaSuccess)
    st = fail(HEOM_ECUDA, "cudaMemsetAsync(static scratch)", e);
  if (st == HEOM_OK) {
    long long blocks = (nodes * elems_per_node + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    level_max_static_kernel<<<(int)blocks, 256, 0, s>>>((const double2*)state_dev, level_dev, (long long)nodes,
                                                        elems_per_node, depth, scratch, max_abs_dev);
    if ((e = cudaGetLastError()) != cudaSuccess) st = fail(HEOM_ECUDA, "level_max_static_kernel launch", e);
  }
  if (prev != device) cudaSetDevice(prev);
  return st;
}
