// soma_init.cuh -- initial state that reproduces supplied concentration fields (SURVEY.md section 8(f) row
// f4; "generating particle positions that reproduce the supplied concentration fields.  Molecules
// are placed within half a mean end-to-end distance of their target positions"; reading R25).
//
//   quantise_target_kernel   Q_t(c) = (uint32) rint(phi*_t(c) 2^16); flags negative / NaN / >= 65536 values
//   cell_weight_kernel       W(c) = sum_t m_t Q_t(c) for one chain pattern (m_t = its beads of type t) or one
//                            single-bead species, as uint64
//   scan_* kernels           inclusive prefix sums of W in place (integer, so the order of the additions does
//                            not matter): chunk sums, scan of the chunk sums by one block, rescan with offsets
//   place_chains_kernel      one thread per chain: target cell by inverse CDF (64-bit draw times the total,
//                            high word; first prefix that exceeds it), target point uniform in that cell, the
//                            Gaussian random walk of DESIGN.md R22 shifted so that its centre of mass sits there
//   place_singles_kernel     single-bead molecules at their target points
#pragma once

#include "soma_kernels.cuh"

namespace soma {

constexpr uint32_t kScanChunk = 2048;        // elements per block of the prefix-sum passes (256 threads x 8)

__global__ void __launch_bounds__(256)
quantise_target_kernel(uint64_t n, const float* __restrict__ phi, uint32_t* __restrict__ Q, uint32_t* __restrict__ bad_flag) {
  const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const float v = phi[k];
  if (!(v >= 0.0f) || !(v < 65536.0f)) { *bad_flag = 1u; Q[k] = 0u; return; }
  Q[k] = __float2uint_rn(__fmul_rn(v, 65536.0f));            // round to nearest even, as rintf
}

struct TypeCounts { uint32_t m[kMaxTypes]; };

__global__ void __launch_bounds__(256)
cell_weight_kernel(uint32_t cells, uint32_t T, TypeCounts M, const uint32_t* __restrict__ Q, unsigned long long* __restrict__ W) {
  const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= cells) return;
  unsigned long long w = 0;
  for (uint32_t t = 0; t < T; ++t) w += (unsigned long long)M.m[t] * Q[(size_t)t * cells + c];
  W[c] = w;
}

// sum of every chunk of kScanChunk elements
__global__ void __launch_bounds__(256)
scan_chunk_sums_kernel(uint32_t n, const unsigned long long* __restrict__ v, unsigned long long* __restrict__ chunk_sum) {
  __shared__ unsigned long long part[8];
  const uint32_t base = blockIdx.x * kScanChunk + threadIdx.x * 8u;
  unsigned long long s = 0;
#pragma unroll
  for (uint32_t k = 0; k < 8; ++k) if (base + k < n) s += v[base + k];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31u) == 0) part[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    for (int w = 0; w < 8; ++w) t += part[w];
    chunk_sum[blockIdx.x] = t;
  }
}

// exclusive scan of the chunk sums in place, one block (a few thousand entries); entry n receives the total
__global__ void __launch_bounds__(1024)
scan_small_kernel(uint32_t n, unsigned long long* __restrict__ v) {
  __shared__ unsigned long long warp_sum[32];
  __shared__ unsigned long long carry_s;
  const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (uint32_t base = 0; base < n; base += 1024u) {
    const uint32_t k = base + threadIdx.x;
    const unsigned long long val = k < n ? v[k] : 0ull;
    unsigned long long inc = val;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= (uint32_t)o) inc += t;
    }
    if (lane == 31) warp_sum[w] = inc;
    __syncthreads();
    if (w == 0) {
      unsigned long long ws = warp_sum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, ws, o);
        if (lane >= (uint32_t)o) ws += t;
      }
      warp_sum[lane] = ws;
    }
    __syncthreads();
    const unsigned long long carry = carry_s;
    if (k < n) v[k] = carry + (w ? warp_sum[w - 1] : 0ull) + inc - val;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = carry + warp_sum[31];
    __syncthreads();
  }
  if (threadIdx.x == 0) v[n] = carry_s;
}

// inclusive prefix sums of v in place, given the exclusive offsets of the chunks
__global__ void __launch_bounds__(256)
scan_apply_kernel(uint32_t n, unsigned long long* __restrict__ v, const unsigned long long* __restrict__ chunk_offset) {
  __shared__ unsigned long long part[8];
  const uint32_t base = blockIdx.x * kScanChunk + threadIdx.x * 8u;
  const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
  unsigned long long e[8], s = 0;
#pragma unroll
  for (uint32_t k = 0; k < 8; ++k) { e[k] = base + k < n ? v[base + k] : 0ull; s += e[k]; }
  unsigned long long inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (uint32_t)o) inc += t;
  }
  if (lane == 31) part[w] = inc;
  __syncthreads();
  unsigned long long run = chunk_offset[blockIdx.x] + inc - s;
  for (uint32_t q = 0; q < w; ++q) run += part[q];
#pragma unroll
  for (uint32_t k = 0; k < 8; ++k) { run += e[k]; if (base + k < n) v[base + k] = run; }
}

struct PlaceArgs {
  uint32_t n_chains, N;             // chains of the species being placed, their length
  uint32_t chain0;                  // logical id of its first chain
  uint32_t pattern;                 // place the chains of this pattern
  uint32_t cells, ny, nz;
  uint32_t k0, k1;                  // generator seed
  double hx, hy, hz;                // cell edges, (double)box / (double)grid
  double sigma;                     // b / sqrt 3
  const uint8_t* __restrict__ chain_pattern;          // [n_chains] of this species
  const unsigned long long* __restrict__ prefix;      // [cells] inclusive prefix sums of the cell weights
  float* __restrict__ x; float* __restrict__ y; float* __restrict__ z;
};

// target point of molecule `id`: DESIGN.md R25
__device__ __forceinline__ void target_point(const PlaceArgs& A, uint32_t id, double& rx, double& ry, double& rz) {
  const Words4 w = philox4x32_10(0u, id, 0u, 3u << 8, A.k0, A.k1);
  const Words4 v = philox4x32_10(1u, id, 0u, 3u << 8, A.k0, A.k1);
  const unsigned long long u64 = ((unsigned long long)w.w0 << 32) | w.w1;
  const unsigned long long k = __umul64hi(u64, A.prefix[A.cells - 1u]);
  uint32_t lo = 0, hi = A.cells - 1u;                         // first cell whose prefix exceeds k
  while (lo < hi) {
    const uint32_t mid = lo + (hi - lo) / 2u;
    if (A.prefix[mid] > k) hi = mid; else lo = mid + 1u;
  }
  const uint32_t iz = lo % A.nz, iy = (lo / A.nz) % A.ny, ix = lo / (A.nz * A.ny);
  rx = __dmul_rn(__dadd_rn((double)ix, unit_open(w.w2)), A.hx);
  ry = __dmul_rn(__dadd_rn((double)iy, unit_open(w.w3)), A.hy);
  rz = __dmul_rn(__dadd_rn((double)iz, unit_open(v.w0)), A.hz);
}

// bond i -> i+1 of the random walk of DESIGN.md R22 (domain-1 draws of bead i)
__device__ __forceinline__ void walk_step(const PlaceArgs& A, uint32_t c /* logical id */, uint32_t i, double& r0, double& r1, double& r2) {
  const double two_pi = 6.283185307179586;
  const Words4 w = philox4x32_10(i, c, 0u, 1u << 8, A.k0, A.k1);
  const double ra = sqrt(-2.0 * log(unit_open(w.w0))), rb = sqrt(-2.0 * log(unit_open(w.w2)));
  const double t1 = two_pi * unit_open(w.w1), t3 = two_pi * unit_open(w.w3);
  r0 = __dadd_rn(r0, __dmul_rn(A.sigma, __dmul_rn(ra, cos(t1))));
  r1 = __dadd_rn(r1, __dmul_rn(A.sigma, __dmul_rn(ra, sin(t1))));
  r2 = __dadd_rn(r2, __dmul_rn(A.sigma, __dmul_rn(rb, cos(t3))));
}

__global__ void __launch_bounds__(128)
place_chains_kernel(PlaceArgs A) {
  const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= A.n_chains || A.chain_pattern[c] != A.pattern) return;
  const uint32_t id = A.chain0 + c;
  double tx, ty, tz;
  target_point(A, id, tx, ty, tz);
  // first pass: centre of mass of the walk that starts at the origin (sums in bead order)
  double r0 = 0.0, r1 = 0.0, r2 = 0.0, s0 = 0.0, s1 = 0.0, s2 = 0.0;
  for (uint32_t i = 1; i < A.N; ++i) {
    walk_step(A, id, i, r0, r1, r2);
    s0 = __dadd_rn(s0, r0); s1 = __dadd_rn(s1, r1); s2 = __dadd_rn(s2, r2);
  }
  const double b0 = __dsub_rn(tx, __ddiv_rn(s0, (double)A.N)), b1 = __dsub_rn(ty, __ddiv_rn(s1, (double)A.N)),
               b2 = __dsub_rn(tz, __ddiv_rn(s2, (double)A.N));
  // second pass: the same walk, shifted
  const uint64_t j0 = (uint64_t)c * A.N;
  r0 = r1 = r2 = 0.0;
  for (uint32_t i = 0; i < A.N; ++i) {
    if (i) walk_step(A, id, i, r0, r1, r2);
    A.x[j0 + i] = (float)__dadd_rn(b0, r0); A.y[j0 + i] = (float)__dadd_rn(b1, r1); A.z[j0 + i] = (float)__dadd_rn(b2, r2);
  }
}

// molecules [first, first + count) of the single-bead arrays; logical chain id = id0 + index
__global__ void __launch_bounds__(256)
place_singles_kernel(PlaceArgs A, uint32_t first, uint32_t count, uint32_t id0) {
  const uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= count) return;
  double tx, ty, tz;
  target_point(A, id0 + first + m, tx, ty, tz);
  A.x[first + m] = (float)tx; A.y[first + m] = (float)ty; A.z[first + m] = (float)tz;
}

}  // namespace soma
