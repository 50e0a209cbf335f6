// soma_lean.cuh -- the move + bin kernel of the SCMF Monte-Carlo step for the configs' geometry
// (rows a1+a2+a3+a5 of SURVEY.md section 8(a)).
//
// Same data flow and bit-for-bit the same arithmetic as fused_step_kernel<.., FAST = true>
// (soma_kernels.cuh): a chain lives in the registers of P = N/2 lanes, two consecutive beads per lane,
// both half-sweeps run there with warp shuffles for the cross-lane neighbours.  It exists for the case
// every BASELINE.json config is in -- power-of-two grid, cell size and move half-width powers of two --
// and differs in what the round-1 ncu captures showed to bound that kernel (profiles/):
//   * all four omega gathers of an iteration (old and trial cell of both beads) are issued before the
//     first Metropolis decision: the trial position of the odd bead does not depend on the even
//     bead's decision, only its bond energy does.  One exposed gather latency per iteration, not two;
//   * the instruction stream is cut from 389 to ~250 per iteration: 32-bit indices with the 64-bit
//     address formed by one IMAD.WIDE at the access, pointers advanced by a compile-time stride,
//     the bead type folded into the cell index by the LOP3 that masks it, no re-materialised
//     parameters;
//   * WIN: a block owns one tile of the box (the chains are kept sorted by the tile of their centre of
//     mass) and counts its beads with RED.shared in a window (tile + halo) of shared memory, which it
//     adds to the global density grid with one bulk reduce-add per z row when it is done
//     (cp.reduce.async.bulk ... .add.u32: one L2 request per 32-byte sector of the window instead of one
//     per bead).  A bead outside its block's window is counted with a global atomic as before, so the
//     result never depends on the tiling.
#pragma once

#include "soma_kernels.cuh"

namespace soma {

struct LeanArgs {
  float inv_hx, inv_hy, inv_hz;      // powers of two >= 1
  uint32_t mx, my, mz;               // nx - 1, ny - 1, nz - 1 (power-of-two grid)
  uint32_t ny, nz;
  uint32_t cells;                    // C
  uint32_t n_chains;
  uint32_t groups_per_block;         // !WIN: warp groups per block (a multiple of the warps per block)
  float a2, ac, kb;                  // 2a, a(2^-23 - 1), 1.5/b^2
  PhiloxKeys keys;
  uint32_t u0, u1;                   // hi(M1 step) ^ k0[0], lo(M1 step)
  uint32_t ctr3_base;
  float* __restrict__ x;
  float* __restrict__ y;
  float* __restrict__ z;
  const float* __restrict__ omega;           // [T][C]
  uint32_t* __restrict__ counts_next;        // [T][C], zeroed before the launch
  const uint32_t* __restrict__ slot_chain;
  const uint8_t* __restrict__ slot_pattern;
  const uint8_t* __restrict__ patterns;
  unsigned long long* __restrict__ accepted;
  // WIN
  const uint32_t* __restrict__ tile_start;   // [n_tiles + 1] first slot of every tile (tiles numbered z fastest)
  uint32_t tcx, tcy, tcz;                    // tile core in cells
  uint32_t hx, hy, hz;                       // halo
  uint32_t wx, wy, wz;                       // window = core + 2 halo; wz and hz multiples of 4
  uint32_t nty, ntz;                         // tiles along y and z
  uint32_t T;
};

__device__ __forceinline__ uint32_t lean_floor_bits(float r, float inv_h, float magic) {
  return __float_as_uint(__fmaf_rd(r, inv_h, magic));
}

// (type, cell) index into a [T][C] grid: floor of every axis by one FFMA.RD (exact: inv_h is a power of
// two), the y and z indices masked, the x index masked together with or-ing in type * C
__device__ __forceinline__ uint32_t lean_cell(const LeanArgs& A, float x, float y, float z, uint32_t type_off) {
  const uint32_t ix = lean_floor_bits(x, A.inv_hx, kFloorMagic);
  const uint32_t iy = lean_floor_bits(y, A.inv_hy, kFloorMagic) & A.my;
  const uint32_t iz = lean_floor_bits(z, A.inv_hz, kFloorMagic) & A.mz;
  return (((ix * A.ny + iy) * A.nz + iz) & (A.cells - 1u)) | type_off;
}

__device__ __forceinline__ float lean_trial(const LeanArgs& A, float r, uint32_t w) {
  const float h = __fadd_rn(__uint_as_float(0x3f800000u | (w >> 9)), -1.0f);
  return __fadd_rn(r, __fmaf_rn(A.a2, h, A.ac));
}

// accept iff fl(dE + lnu) <= 0 (DESIGN.md section 2 step 5.6): the arithmetic of
// metropolis_accept_fma with u 2^24 already converted.  `live` = false forces a rejection (lanes
// beyond the end of the block's range).
__device__ __forceinline__ bool lean_accept(float dE, float u24, bool live) {
  const float m = __fmaf_rn(lg2_approx(u24), kLn2, dE);
  bool acc = (m < kLnT - kLnBand) && live;
  if (!(m < kLnT - kLnBand) && m <= kLnT + kLnBand)            // ~6e-5 of the moves: exact logarithm
    acc = (__fadd_rn(dE, lnu_exact(__fmul_rn(u24, 0x1p-24f))) <= 0.0f) && live;
  return acc;
}
// selects spelled as selp so that the accepted state is taken by predicated moves, not by a branch
__device__ __forceinline__ float selp_f(bool p, float a, float b) {
  float r;
  asm("{ .reg .pred q; setp.ne.u32 q, %3, 0; selp.f32 %0, %1, %2, q; }" : "=f"(r) : "f"(a), "f"(b), "r"((uint32_t)p));
  return r;
}
__device__ __forceinline__ uint32_t selp_u(bool p, uint32_t a, uint32_t b) {
  uint32_t r;
  asm("{ .reg .pred q; setp.ne.u32 q, %3, 0; selp.u32 %0, %1, %2, q; }" : "=r"(r) : "r"(a), "r"(b), "r"((uint32_t)p));
  return r;
}

__device__ __forceinline__ void reds_inc(uint32_t saddr) {
  asm volatile("red.shared::cta.add.u32 [%0], 1;" ::"r"(saddr) : "memory");
}
__device__ __forceinline__ void bulk_reduce_add_u32(void* gdst, uint32_t ssrc, uint32_t bytes) {
  asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.u32 [%0], [%1], %2;" ::"l"(gdst), "r"(ssrc), "r"(bytes)
               : "memory");
}

#ifndef SOMA_LEAN_PREFETCH_L2
#define SOMA_LEAN_PREFETCH_L2 1
#endif
constexpr bool PREFETCH_L2 = SOMA_LEAN_PREFETCH_L2 != 0;

template <int P, bool MULTI_PAT, bool WIN, int NT>
__global__ void __launch_bounds__(NT, 1024 / NT)
lean_step_kernel(const __grid_constant__ LeanArgs A) {
  constexpr uint32_t G = 32 / P;                                // chains per warp
  constexpr uint32_t N = 2u * P;
  constexpr uint32_t WPB = NT / 32;                             // warps per block
  constexpr uint32_t STEP = WPB * G;                            // slots per block iteration
  extern __shared__ __align__(16) uint32_t win[];               // WIN: [T][wx][wy][wz] bead counts of this block's window
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  const uint32_t l = lane % P, sub = lane / P;

  // ---- the block's range of slots ----
  uint32_t s_begin, s_end;
  float mgx = 0.f, mgy = 0.f, mgz = 0.f;                        // WIN: floor magic minus the window origin, per axis
  if (WIN) {
    s_begin = __ldg(A.tile_start + blockIdx.x);
    s_end = __ldg(A.tile_start + blockIdx.x + 1u);
    if (s_begin == s_end) return;                               // uniform over the block
    const uint32_t tz = blockIdx.x % A.ntz, ty = (blockIdx.x / A.ntz) % A.nty, tx = blockIdx.x / (A.ntz * A.nty);
    mgx = kFloorMagic - (float)((int)(tx * A.tcx) - (int)A.hx);
    mgy = kFloorMagic - (float)((int)(ty * A.tcy) - (int)A.hy);
    mgz = kFloorMagic - (float)((int)(tz * A.tcz) - (int)A.hz);
    const uint32_t words = A.T * A.wx * A.wy * A.wz;
    for (uint32_t k = threadIdx.x; k < words / 4u; k += NT) reinterpret_cast<uint4*>(win)[k] = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
  } else {
    const uint64_t b = (uint64_t)blockIdx.x * A.groups_per_block * G;
    if (b >= A.n_chains) return;
    s_begin = (uint32_t)b;
    const uint64_t e = b + (uint64_t)A.groups_per_block * G;
    s_end = e < A.n_chains ? (uint32_t)e : A.n_chains;
  }
  const uint32_t win_base = (uint32_t)__cvta_generic_to_shared(win);
  const uint32_t win_type = A.wx * A.wy * A.wz;

  // ---- per-lane constants ----
  const bool has_l = l > 0, has_r = l + 1 < P;                  // does the left / right cross-lane neighbour exist
  const PhiloxLane L0 = philox_lane(A.keys, A.u1, 2u * l, A.ctr3_base);
  const PhiloxLane L1 = philox_lane(A.keys, A.u1, 2u * l + 1u, A.ctr3_base | 1u);
  uint32_t t0 = 0, t1 = 0;                                      // bead types of this lane
  if (!MULTI_PAT) {
    const uint16_t tt = *reinterpret_cast<const uint16_t*>(A.patterns + 2u * l);
    t0 = tt & 0xffu; t1 = tt >> 8;
  }
  unsigned n_acc = 0;
  const float2* __restrict__ x2 = reinterpret_cast<const float2*>(A.x);
  const float2* __restrict__ y2 = reinterpret_cast<const float2*>(A.y);
  const float2* __restrict__ z2 = reinterpret_cast<const float2*>(A.z);

  // One 32-bit index serves every array: bead pair `pair` = slot P + l, slot = pair / P.
  for (uint32_t slot = s_begin + warp * G + sub; slot - sub < s_end; slot += STEP) {      // slot - sub: warp-uniform
    const bool live = slot < s_end;
    const uint32_t pair = slot * P + l;
    // positions are streamed (read once, written once): keep them from evicting omega out of L1
    const float2 X = __ldcs(x2 + pair), Y = __ldcs(y2 + pair), Z = __ldcs(z2 + pair);
    const uint32_t chain = __ldg(A.slot_chain + slot);
    if (MULTI_PAT) {
      const uint16_t tt = __ldg(reinterpret_cast<const uint16_t*>(A.patterns + (uint32_t)__ldg(A.slot_pattern + slot) * N) + l);
      t0 = tt & 0xffu; t1 = tt >> 8;
    }
    if (PREFETCH_L2 && (l & 3u) == 0u && slot - sub + STEP < s_end) {     // one prefetch per 32-byte sector of the next group
      asm volatile("prefetch.global.L2 [%0];" ::"l"(x2 + pair + STEP * P));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(y2 + pair + STEP * P));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(z2 + pair + STEP * P));
    }
    const uint32_t toff0 = t0 * A.cells, toff1 = t1 * A.cells;
    float ex = X.x, ey = Y.x, ez = Z.x;                         // even bead 2l
    float ox = X.y, oy = Y.y, oz = Z.y;                         // odd bead 2l+1

    // ---- everything that does not depend on a decision: old cells, both trial positions, four gathers ----
    uint32_t cell_e = lean_cell(A, ex, ey, ez, toff0);
    uint32_t cell_o = lean_cell(A, ox, oy, oz, toff1);
    const float w_old_e = __ldg(A.omega + cell_e);
    const float w_old_o = __ldg(A.omega + cell_o);
    const uint32_t c0_1 = A.u0 ^ chain;
    const Words4 We = philox_tail(A.keys, L0, c0_1);
    const float tex = lean_trial(A, ex, We.w0), tey = lean_trial(A, ey, We.w1), tez = lean_trial(A, ez, We.w2);
    const uint32_t cell_te = lean_cell(A, tex, tey, tez, toff0);
    const float w_new_e = __ldg(A.omega + cell_te);
    const Words4 Wo = philox_tail(A.keys, L1, c0_1);
    const float tox = lean_trial(A, ox, Wo.w0), toy = lean_trial(A, oy, Wo.w1), toz = lean_trial(A, oz, Wo.w2);
    const uint32_t cell_to = lean_cell(A, tox, toy, toz, toff1);
    const float w_new_o = __ldg(A.omega + cell_to);
    const float u24_e = umap_int(We.w3), u24_o = umap_int(Wo.w3);

    // ---- half-sweep 0: even bead; left neighbour = odd bead of lane l-1, right neighbour = own odd bead ----
    const float lx = __shfl_up_sync(0xffffffffu, ox, 1, P);
    const float ly = __shfl_up_sync(0xffffffffu, oy, 1, P);
    const float lz = __shfl_up_sync(0xffffffffu, oz, 1, P);
    float qA = bond_sq(ex, ey, ez, ox, oy, oz);                 // |even - odd|^2
    float qB = bond_sq(ex, ey, ez, lx, ly, lz);                 // |even - odd of lane l-1|^2 (unused if there is none)
    {
      const float ql_new = bond_sq(tex, tey, tez, lx, ly, lz);
      const float qr_new = bond_sq(tex, tey, tez, ox, oy, oz);
      const float dql = __fsub_rn(ql_new, qB), dqr = __fsub_rn(qr_new, qA);
      const float dq = has_l ? __fadd_rn(dql, dqr) : dqr;       // DESIGN.md section 2 step 5.4: only the bonds that exist
      const float dE = __fmaf_rn(A.kb, dq, __fsub_rn(w_new_e, w_old_e));
      const bool acc = lean_accept(dE, u24_e, live);
      ex = selp_f(acc, tex, ex); ey = selp_f(acc, tey, ey); ez = selp_f(acc, tez, ez);
      cell_e = selp_u(acc, cell_te, cell_e);
      qB = selp_f(acc, ql_new, qB); qA = selp_f(acc, qr_new, qA);
      n_acc += acc ? 1u : 0u;
    }
    // ---- half-sweep 1: odd bead; left = own even bead (moved), right = even bead of lane l+1 (moved) ----
    {
      const float rx = __shfl_down_sync(0xffffffffu, ex, 1, P);
      const float ry = __shfl_down_sync(0xffffffffu, ey, 1, P);
      const float rz = __shfl_down_sync(0xffffffffu, ez, 1, P);
      const float qR = __shfl_down_sync(0xffffffffu, qB, 1, P);
      const float ql_new = bond_sq(tox, toy, toz, ex, ey, ez);
      const float qr_new = bond_sq(tox, toy, toz, rx, ry, rz);
      const float dql = __fsub_rn(ql_new, qA), dqr = __fsub_rn(qr_new, qR);
      const float dq = has_r ? __fadd_rn(dql, dqr) : dql;
      const float dE = __fmaf_rn(A.kb, dq, __fsub_rn(w_new_o, w_old_o));
      const bool acc = lean_accept(dE, u24_o, live);
      ox = selp_f(acc, tox, ox); oy = selp_f(acc, toy, oy); oz = selp_f(acc, toz, oz);
      cell_o = selp_u(acc, cell_to, cell_o);
      n_acc += acc ? 1u : 0u;
    }
    if (live) {
      __stcs(const_cast<float2*>(x2) + pair, make_float2(ex, ox));
      __stcs(const_cast<float2*>(y2) + pair, make_float2(ey, oy));
      __stcs(const_cast<float2*>(z2) + pair, make_float2(ez, oz));
      if (WIN) {
        // window-relative cell of the final positions; a bead outside the window goes to the global grid
        const uint32_t ax = (lean_floor_bits(ex, A.inv_hx, mgx) & A.mx), ay = (lean_floor_bits(ey, A.inv_hy, mgy) & A.my),
                       az = (lean_floor_bits(ez, A.inv_hz, mgz) & A.mz);
        const uint32_t bx = (lean_floor_bits(ox, A.inv_hx, mgx) & A.mx), by = (lean_floor_bits(oy, A.inv_hy, mgy) & A.my),
                       bz = (lean_floor_bits(oz, A.inv_hz, mgz) & A.mz);
        if (ax < A.wx && ay < A.wy && az < A.wz) reds_inc(win_base + 4u * (t0 * win_type + (ax * A.wy + ay) * A.wz + az));
        else atomicAdd(A.counts_next + cell_e, 1u);
        if (bx < A.wx && by < A.wy && bz < A.wz) reds_inc(win_base + 4u * (t1 * win_type + (bx * A.wy + by) * A.wz + bz));
        else atomicAdd(A.counts_next + cell_o, 1u);
      } else {
        atomicAdd(A.counts_next + cell_e, 1u);
        atomicAdd(A.counts_next + cell_o, 1u);
      }
    }
  }

  if (WIN) {
    // ---- the window goes to the global grid: one bulk reduce-add per z row (split where the row wraps) ----
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    const uint32_t tz = blockIdx.x % A.ntz, ty = (blockIdx.x / A.ntz) % A.nty, tx = blockIdx.x / (A.ntz * A.nty);
    const uint32_t oxc = (tx * A.tcx - A.hx) & A.mx, oyc = (ty * A.tcy - A.hy) & A.my, ozc = (tz * A.tcz - A.hz) & A.mz;
    const uint32_t rows = A.T * A.wx * A.wy;
    const uint32_t nz = A.mz + 1u;
    for (uint32_t r = threadIdx.x; r < rows; r += NT) {
      const uint32_t ry = r % A.wy, rx = (r / A.wy) % A.wx, t = r / (A.wy * A.wx);
      const uint4* row = reinterpret_cast<const uint4*>(win + (size_t)r * A.wz);
      uint32_t any = 0;
      for (uint32_t k = 0; k < A.wz / 4u; ++k) { const uint4 v = row[k]; any |= v.x | v.y | v.z | v.w; }
      if (!any) continue;
      const uint32_t gx = (oxc + rx) & A.mx, gy = (oyc + ry) & A.my;
      uint32_t* g = A.counts_next + (size_t)t * A.cells + ((size_t)gx * A.ny + gy) * nz;
      const uint32_t srow = win_base + 4u * r * A.wz;
      const uint32_t first = nz - ozc < A.wz ? nz - ozc : A.wz;        // cells before the row wraps around z
      bulk_reduce_add_u32(g + ozc, srow, 4u * first);
      if (first < A.wz) bulk_reduce_add_u32(g, srow + 4u * first, 4u * (A.wz - first));
    }
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
  // accepted-move count: warp reduce, one atomic per warp
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
  if (lane == 0 && n_acc) atomicAdd(A.accepted, (unsigned long long)n_acc);
}

}  // namespace soma
