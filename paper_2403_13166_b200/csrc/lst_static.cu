// lst_static.cu -- lst_sort_hits_static(): step a0 (hit ingest, SPEC.md 4.0) for callers that cannot allocate.
//
// Who this is for.  Every other entry point of include/lst.h works in a workspace the caller allocates.  Some callers
// have no way to do that: a reconstruction plugin loaded into a trigger / event-processing job whose framework handed
// out all device memory at start-up and gives a module pointers to its inputs and outputs and nothing else, or an event
// loop in which cudaMalloc / cudaFree are banned because they synchronise the whole device and take an unbounded time.
// Such a caller can still pass its input and output buffers, but it has no place for the temporaries of the sort (the
// per-sensor counters, each hit's arrival slot, the sensor-ordered index list).  Here those temporaries live in ONE
// file-scope `static __device__` array of a fixed, modest size (LST_STATIC_SCRATCH_BYTES below, about 1.3 MB) that the
// CUDA runtime places on every GPU that loads this library and keeps until the process exits.  The function itself
// calls no cudaMalloc, cudaFree, cudaMallocAsync or any library routine that allocates.
//
// What follows from one shared array:
//  * sizes are bounded: n_hits <= LST_STATIC_MAX_HITS and n_modules <= LST_STATIC_MAX_MODULES, else LST_ETOOBIG;
//  * the array keeps whatever the last call left in it, so each call clears the part that must start at zero
//    (counters, flags) on the caller's stream before using it; everything else is written before it is read;
//  * two calls whose work overlaps on one GPU (different streams, or two host threads) use the same counters at the same
//    time and corrupt each other: callers must serialise them (same stream, or an event between them).
//  * the first call on each device looks up the array's device address (cudaGetSymbolAddress, a set-up step that must
//    not fall inside a stream capture): make that first call on a device before any capture begins.
//
// The kernels are the a0 kernels of lst_kernels.cuh (k_hist / scan / k_scatter / k_rank) restated over plain pointers;
// the existing chain is untouched and shares no state with this file.
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include "../../include/lst.h"

namespace {

constexpr int MAX_HITS = LST_STATIC_MAX_HITS;
constexpr int MAX_SENSORS = 2 * LST_STATIC_MAX_MODULES;

// layout of the scratch array, in 32-bit words
constexpr size_t W_FLAGS = 0;                              // [64]  flags[0] = status bits, flags[1] = hits kept (zeroed per call)
constexpr size_t W_COUNT = 64;                             // [MAX_SENSORS + 64] hits per sensor (zeroed per call)
constexpr size_t W_ZERO_END = W_COUNT + MAX_SENSORS + 64;  // words [0, W_ZERO_END) are cleared at the start of every call
constexpr size_t W_ARRIVAL = W_ZERO_END;                   // [MAX_HITS] arrival slot of hit i within its sensor
constexpr size_t W_ORDER = W_ARRIVAL + MAX_HITS;           // [MAX_HITS] original hit index, sensor by sensor in arrival order
constexpr size_t W_TOTAL = W_ORDER + MAX_HITS;
static_assert(W_TOTAL * 4 == LST_STATIC_SCRATCH_BYTES, "include/lst.h states the size of the static scratch");

// The scratch itself.  In HOST code this name is only a handle for cudaGetSymbolAddress, never a device address:
// a kernel handed `g_scratch` directly would read host memory or fault.  scratch_ptr() below does the look-up.
static __device__ __align__(256) unsigned char g_scratch[LST_STATIC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
int* g_dev_ptr[MAX_DEVICES] = {};   // device address of g_scratch on each device, filled on first use

// Device address of the scratch array on the CURRENT device (the one the caller's stream and buffers belong to).
cudaError_t scratch_ptr(int** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_dev_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_scratch);      // once per device, with that device current
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_dev_ptr[dev] = static_cast<int*>(p);
  }
  *out = g_dev_ptr[dev];
  return cudaSuccess;
}

// hits per sensor; each in-range hit remembers the slot it took (its arrival order, not yet the stable order)
__global__ void k_static_hist(const uint32_t* __restrict__ key, int n, unsigned S, int* __restrict__ count,
                              int* __restrict__ arrival, int* __restrict__ flags) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const unsigned k = key[i];
    if (k < S) arrival[i] = atomicAdd(count + k, 1);
    else atomicOr(reinterpret_cast<unsigned*>(flags), LST_ST_BAD_KEY);
  }
}

// one block: exclusive scan of count[0..S) -> sensor_start[0..S], total -> out_count[0], status -> out_count[1]
constexpr int SCAN_T = 1024;
__global__ void __launch_bounds__(SCAN_T) k_static_scan(const int* __restrict__ count, int S, int* __restrict__ sensor_start,
                                                         const int* __restrict__ flags, int* __restrict__ out_count) {
  __shared__ int part[SCAN_T];
  const int t = threadIdx.x;
  const int per = (S + SCAN_T - 1) / SCAN_T;
  const int b = min(t * per, S), e = min(b + per, S);
  int sum = 0;
  for (int i = b; i < e; ++i) sum += count[i];
  part[t] = sum;
  __syncthreads();
  for (int d = 1; d < SCAN_T; d <<= 1) {          // inclusive scan of the per-thread sums
    const int v = (t >= d) ? part[t - d] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  int run = part[t] - sum;
  for (int i = b; i < e; ++i) { sensor_start[i] = run; run += count[i]; }
  if (t == SCAN_T - 1) {
    sensor_start[S] = part[t];
    out_count[0] = part[t];
    out_count[1] = flags[0];
  }
}

// original indices gathered sensor by sensor (arrival order inside a sensor)
__global__ void k_static_scatter(const uint32_t* __restrict__ key, int n, unsigned S, const int* __restrict__ sensor_start,
                                 const int* __restrict__ arrival, int* __restrict__ order) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const unsigned k = key[i];
    if (k < S) order[sensor_start[k] + arrival[i]] = i;
  }
}

// stable order inside a sensor: a hit's rank = number of hits of its sensor with a smaller original index
__global__ void k_static_rank(const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z,
                              const uint32_t* __restrict__ key, const int* __restrict__ sensor_start, int S,
                              const int* __restrict__ order, float4* __restrict__ hit, int* __restrict__ hit_orig) {
  const int n = sensor_start[S];
  for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < n; p += gridDim.x * blockDim.x) {
    const int o = order[p];
    const unsigned k = key[o];
    const int b = sensor_start[k], e = sensor_start[k + 1];
    int rank = 0;
    for (int q = b; q < e; ++q) rank += (order[q] < o);
    const float hx = x[o], hy = y[o];
    hit[b + rank] = make_float4(hx, hy, z[o], __fsqrt_rn(__fadd_rn(__fmul_rn(hx, hx), __fmul_rn(hy, hy))));   // r as SPEC.md 4.1
    hit_orig[b + rank] = o;
  }
}

}  // namespace

extern "C" int lst_sort_hits_static(int32_t n_hits, int32_t n_modules, const float* d_x, const float* d_y, const float* d_z,
                                    const uint32_t* d_key, float* d_hit_xyzr, int32_t* d_hit_orig, int32_t* d_sensor_start,
                                    int32_t* d_count, void* cuda_stream) {
  if (n_hits < 0 || n_modules <= 0) return LST_EINVAL;
  if (n_hits > MAX_HITS || n_modules > LST_STATIC_MAX_MODULES) return LST_ETOOBIG;      // the static scratch cannot hold more
  if (!d_sensor_start || !d_count) return LST_EINVAL;
  if (n_hits > 0 && (!d_x || !d_y || !d_z || !d_key || !d_hit_xyzr || !d_hit_orig)) return LST_EINVAL;
  if (reinterpret_cast<uintptr_t>(d_hit_xyzr) % 16) return LST_EINVAL;                   // rows are written as float4
  int* w = nullptr;
  if (scratch_ptr(&w) != cudaSuccess) return LST_ECUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int S = 2 * n_modules;
  int* flags = w + W_FLAGS; int* count = w + W_COUNT; int* arrival = w + W_ARRIVAL; int* order = w + W_ORDER;
  // the array still holds the previous call's counters: clear what this call accumulates into
  if (cudaMemsetAsync(w, 0, sizeof(int) * (W_COUNT + (size_t)S + 1), st) != cudaSuccess) return LST_ECUDA;
  const int tpb = 256;
  int blocks = (n_hits + tpb - 1) / tpb;
  if (blocks < 1) blocks = 1;
  if (blocks > 148 * 8) blocks = 148 * 8;
  k_static_hist<<<blocks, tpb, 0, st>>>(d_key, n_hits, (unsigned)S, count, arrival, flags);
  k_static_scan<<<1, SCAN_T, 0, st>>>(count, S, d_sensor_start, flags, d_count);
  k_static_scatter<<<blocks, tpb, 0, st>>>(d_key, n_hits, (unsigned)S, d_sensor_start, arrival, order);
  k_static_rank<<<blocks, tpb, 0, st>>>(d_x, d_y, d_z, d_key, d_sensor_start, S, order, reinterpret_cast<float4*>(d_hit_xyzr), d_hit_orig);
  return cudaGetLastError() == cudaSuccess ? LST_OK : LST_ECUDA;
}
