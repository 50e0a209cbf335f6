// soma_noalloc.cu -- soma_validate_noalloc: the validation report of soma_validate_state for a state the
// caller holds in device memory, computed without allocating anything (include/soma.h has the contract).
//
// Who this is for.  Everything else in this library either lives in a handle's workspace or calls
// cudaMalloc.  Some callers can do neither:
//   * a particle simulation that was started next to another GPU code (in the paper's coupled runs SOMA
//     is spawned beside the continuum solver; under PyTorch the caching allocator has
//     usually taken the free HBM already): its device footprint was fixed when it started, a late
//     cudaMalloc may simply fail, and if it succeeds it takes memory the neighbour was counting on;
//   * a time-critical loop: cudaMalloc and cudaFree are device-wide synchronisation points, so one call
//     stalls every other stream of the process, not only the caller's;
//   * a checkpoint checker that runs before any handle exists, so there is no workspace to borrow from.
// Such a caller still wants to know, before it loads a state or after it has received one, that no
// coordinate is NaN, that the density grids hold every bead, and how long the bonds are.
//
// How.  The per-tile partial results and the final report -- the only global memory the two passes need
// beyond the caller's inputs -- live in g_noalloc_scratch, a file-scope device array of fixed size
// (kScratchBytes, about 1.6 MB).  It is part of the library image: every GPU that loads libsoma_b200.so
// carries it until the process exits, whether or not this function is ever called.  Its size fixes the
// largest state that fits (kMaxBeads beads per call); a larger one is refused, never truncated.
//
// The array's name means two different things.  In device code it is the array.  In host code it is only a
// handle the runtime uses to look the array up; handing it to a kernel as if it were a pointer would make
// the kernel read host memory (or fault).  So the host side asks the runtime for the real device address
// with cudaGetSymbolAddress, once per device with that device current, and passes that address on.
//
// This file stands alone: it includes none of the library's other sources, so no existing kernel or host
// path changes by its presence.  The squared bond length is written out again below with the operation order
// of DESIGN.md section 2 step 5.4, so that max_bond_sq is the same fp32 number the existing path reports.
#include "../../include/soma.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>

#include <cuda_runtime.h>

namespace {

// squared bond length, DESIGN.md section 2 step 5.4: fma(sz,sz, fma(sy,sy, sx*sx)), nothing contracted or reordered
__device__ __forceinline__ float bond_sq(float ax, float ay, float az, float bx, float by, float bz) {
  const float sx = __fsub_rn(ax, bx), sy = __fsub_rn(ay, by), sz = __fsub_rn(az, bz);
  return __fmaf_rn(sz, sz, __fmaf_rn(sy, sy, __fmul_rn(sx, sx)));
}

constexpr uint32_t kThreads = 256;                       // threads of a tile block
constexpr uint32_t kPerThread = 16;                      // beads per thread
constexpr uint32_t kTileBeads = kThreads * kPerThread;   // 4096 beads per tile = one partial result
constexpr uint32_t kMaxTiles = 65536;
constexpr uint64_t kMaxBeads = (uint64_t)kTileBeads * kMaxTiles;   // 268 435 456 (cfg4 holds 134 217 728)
constexpr uint32_t kDensBlocks = 256;                    // partial sums per type of the density pass
constexpr uint32_t kMaxTypes = 8;                        // soma_validation.density_per_type has 8 entries
constexpr uint32_t kReportWords = 11;                    // [0] non-finite, [1..8] per type, [9] max bits, [10] bond sum
constexpr int kMaxDevices = 64;

// layout of the scratch array, in 8-byte words
constexpr uint32_t kTileOff = 0;                                   // [kMaxTiles][3]: non-finite, max bits, bond sum
constexpr uint32_t kDensOff = kTileOff + 3u * kMaxTiles;           // [kMaxTypes][kDensBlocks]
constexpr uint32_t kReportOff = kDensOff + kMaxTypes * kDensBlocks;
constexpr uint32_t kScratchWords = kReportOff + 16u;
constexpr size_t kScratchBytes = (size_t)kScratchWords * 8;
static_assert(kScratchBytes == 1589376, "include/soma.h and README.md state this size");
static_assert(kMaxBeads == (1ull << 28), "include/soma.h and README.md state this limit");

// The scratch itself.  Shared by every call on this device and never cleared between calls: see the
// comments at the kernels for why no slot needs to start at zero.
static __device__ __align__(256) unsigned long long g_noalloc_scratch[kScratchWords];

// Pass 1: one block per tile of 4096 beads.  Each block leaves exactly one partial result in its own slot;
// nothing is accumulated across blocks here, so no slot has to be zero beforehand and the result does not
// depend on the order in which blocks run.  (The existing path adds into one report with atomics instead.)
__global__ void __launch_bounds__(kThreads)
noalloc_tile_kernel(uint32_t B, uint32_t N, const float* __restrict__ x, const float* __restrict__ y,
                    const float* __restrict__ z, unsigned long long* __restrict__ scratch) {
  __shared__ unsigned s_bad[kThreads / 32];
  __shared__ float s_max[kThreads / 32];
  __shared__ double s_sum[kThreads / 32];
  const uint32_t base = blockIdx.x * kTileBeads;
  unsigned bad = 0;
  float qm = 0.0f;
  double qs = 0.0;
  for (uint32_t k = 0; k < kPerThread; ++k) {
    const uint32_t j = base + k * kThreads + threadIdx.x;
    if (j >= B) break;
    const float px = x[j], py = y[j], pz = z[j];
    bad += (isfinite(px) ? 0u : 1u) + (isfinite(py) ? 0u : 1u) + (isfinite(pz) ? 0u : 1u);
    if (j % N + 1u < N) {                                       // bond (i, i+1) of the same chain
      const float q = bond_sq(px, py, pz, x[j + 1], y[j + 1], z[j + 1]);
      if (q == q) { qm = fmaxf(qm, q); qs += (double)q; }       // a NaN bond is already counted in `bad`
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bad += __shfl_xor_sync(0xffffffffu, bad, o);
    qm = fmaxf(qm, __shfl_xor_sync(0xffffffffu, qm, o));
    qs += __shfl_xor_sync(0xffffffffu, qs, o);
  }
  const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
  if (lane == 0) { s_bad[w] = bad; s_max[w] = qm; s_sum[w] = qs; }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long b = 0;
    float m = 0.0f;
    double s = 0.0;
    for (uint32_t q = 0; q < kThreads / 32; ++q) { b += s_bad[q]; m = fmaxf(m, s_max[q]); s += s_sum[q]; }
    unsigned long long* slot = scratch + kTileOff + 3ull * blockIdx.x;
    slot[0] = b;
    slot[1] = (unsigned long long)__float_as_uint(m);
    slot[2] = (unsigned long long)__double_as_longlong(s);
  }
}

// Pass 1b: density grids, [T][cells] uint32 as soma_get_density returns them.  Block (bx, t) sums its stride of
// type t's grid into slot [t][bx]; again one plain store per slot.
__global__ void __launch_bounds__(kThreads)
noalloc_density_kernel(uint64_t cells, const uint32_t* __restrict__ counts, unsigned long long* __restrict__ scratch) {
  __shared__ unsigned long long s_part[kThreads / 32];
  const uint32_t t = blockIdx.y;
  const uint32_t* g = counts + (size_t)t * cells;
  unsigned long long sum = 0;
  for (uint64_t c = (uint64_t)blockIdx.x * kThreads + threadIdx.x; c < cells; c += (uint64_t)kDensBlocks * kThreads) sum += g[c];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if ((threadIdx.x & 31u) == 0) s_part[threadIdx.x >> 5] = sum;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long s = 0;
    for (uint32_t q = 0; q < kThreads / 32; ++q) s += s_part[q];
    scratch[kDensOff + t * kDensBlocks + blockIdx.x] = s;
  }
}

// Pass 2: one block folds the slots that THIS call wrote (n_tiles tile slots, n_types rows of density slots)
// into the 11-word report.  Slots beyond those still hold an earlier call's values and are never read.  The
// additions happen in a fixed order, so the same state gives the same mean_bond_sq bit for bit every time.
__global__ void __launch_bounds__(1024)
noalloc_finish_kernel(uint32_t n_tiles, uint32_t n_types, unsigned long long* __restrict__ scratch) {
  __shared__ unsigned long long s_bad[1024];
  __shared__ uint32_t s_max[1024];
  __shared__ double s_sum[1024];
  const uint32_t tid = threadIdx.x;
  unsigned long long bad = 0;
  uint32_t mx = 0;                                         // bit patterns of non-negative floats order like integers
  double sum = 0.0;
  for (uint32_t k = tid; k < n_tiles; k += 1024u) {
    const unsigned long long* slot = scratch + kTileOff + 3ull * k;
    bad += slot[0];
    mx = max(mx, (uint32_t)slot[1]);
    sum += __longlong_as_double((long long)slot[2]);
  }
  s_bad[tid] = bad; s_max[tid] = mx; s_sum[tid] = sum;
  __syncthreads();
  for (uint32_t half = 512; half > 0; half >>= 1) {
    if (tid < half) {
      s_bad[tid] += s_bad[tid + half];
      s_max[tid] = max(s_max[tid], s_max[tid + half]);
      s_sum[tid] += s_sum[tid + half];
    }
    __syncthreads();
  }
  unsigned long long* report = scratch + kReportOff;
  if (tid == 0) {
    report[0] = s_bad[0];
    report[9] = s_max[0];
    report[10] = (unsigned long long)__double_as_longlong(s_sum[0]);
  }
  if (tid < kMaxTypes) {                                  // integer sums: any order gives the same value
    unsigned long long d = 0;
    if (tid < n_types)
      for (uint32_t q = 0; q < kDensBlocks; ++q) d += scratch[kDensOff + tid * kDensBlocks + q];
    report[1 + tid] = d;
  }
}

// Device address of g_noalloc_scratch on every device this process has used the entry point on.
std::mutex g_setup_mutex;
unsigned long long* g_scratch_addr[kMaxDevices] = {};

int report_error(char* errbuf, size_t errbuf_len, int code, const char* fmt, ...) {
  if (errbuf && errbuf_len) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, errbuf_len, fmt, ap);
    va_end(ap);
  }
  return code;
}

}  // namespace

extern "C" int soma_validate_noalloc(const float* x, const float* y, const float* z, uint64_t n_chains,
                                     uint32_t beads_per_chain, const uint32_t* counts, uint32_t n_types, uint64_t cells,
                                     void* cuda_stream, soma_validation* out, char* errbuf, size_t errbuf_len) {
  if (errbuf && errbuf_len) errbuf[0] = '\0';
  if (!x || !y || !z || !out) return report_error(errbuf, errbuf_len, SOMA_EINVAL, "x, y, z and out must not be NULL");
  if (n_chains == 0 || beads_per_chain == 0) return report_error(errbuf, errbuf_len, SOMA_EINVAL, "n_chains and beads_per_chain must be >= 1");
  // the size check comes before anything touches the device: B beyond the scratch array's capacity is refused
  if (n_chains > kMaxBeads / beads_per_chain)
    return report_error(errbuf, errbuf_len, SOMA_EINVAL,
                        "soma_validate_noalloc: %llu chains x %u beads exceed the %llu beads the fixed scratch array holds "
                        "(one partial result per %u beads, %u slots); validate the state in pieces or use soma_validate_state",
                        (unsigned long long)n_chains, beads_per_chain, (unsigned long long)kMaxBeads, kTileBeads, kMaxTiles);
  if (counts) {
    if (n_types == 0 || n_types > kMaxTypes) return report_error(errbuf, errbuf_len, SOMA_EINVAL, "n_types must be in [1, 8] when counts is given");
    if (cells == 0 || cells * n_types >= (1ull << 32)) return report_error(errbuf, errbuf_len, SOMA_EINVAL, "cells must be >= 1 and n_types * cells < 2^32");
  }
  const uint32_t B = (uint32_t)(n_chains * beads_per_chain);
  const uint32_t n_tiles = (B + kTileBeads - 1) / kTileBeads;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);

#define NA_CU(call)                                                                                               \
  do {                                                                                                            \
    cudaError_t e_ = (call);                                                                                      \
    if (e_ != cudaSuccess) return report_error(errbuf, errbuf_len, SOMA_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

  // Set-up, once per device: look up where g_noalloc_scratch lives on the CURRENT device.  This may load the
  // library's device code, which is why the first call on a device should come before any stream capture.
  int dev = -1;
  NA_CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return report_error(errbuf, errbuf_len, SOMA_EINVAL, "device ordinal %d is outside [0, %d)", dev, kMaxDevices);
  unsigned long long* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
      void* p = nullptr;
      NA_CU(cudaGetSymbolAddress(&p, g_noalloc_scratch));
      g_scratch_addr[dev] = static_cast<unsigned long long*>(p);
    }
    scratch = g_scratch_addr[dev];
  }

  noalloc_tile_kernel<<<n_tiles, kThreads, 0, stream>>>(B, beads_per_chain, x, y, z, scratch);
  const uint32_t T = counts ? n_types : 0u;
  if (T) noalloc_density_kernel<<<dim3(kDensBlocks, T), kThreads, 0, stream>>>(cells, counts, scratch);
  noalloc_finish_kernel<<<1, 1024, 0, stream>>>(n_tiles, T, scratch);
  NA_CU(cudaGetLastError());
  unsigned long long host[kReportWords];
  NA_CU(cudaMemcpyAsync(host, scratch + kReportOff, sizeof host, cudaMemcpyDeviceToHost, stream));
  NA_CU(cudaStreamSynchronize(stream));
#undef NA_CU

  std::memset(out, 0, sizeof *out);
  out->n_nonfinite = host[0];
  for (uint32_t t = 0; t < T; ++t) { out->density_per_type[t] = host[1 + t]; out->density_total += host[1 + t]; }
  const uint32_t qbits = (uint32_t)host[9];
  std::memcpy(&out->max_bond_sq, &qbits, 4);
  double sum;
  std::memcpy(&sum, &host[10], 8);
  const uint64_t n_bonds = n_chains * (uint64_t)(beads_per_chain - 1);
  out->mean_bond_sq = n_bonds ? sum / (double)n_bonds : 0.0;
  out->ok = (out->n_nonfinite == 0 && (!counts || out->density_total == (uint64_t)B)) ? 1u : 0u;
  return SOMA_OK;
}
