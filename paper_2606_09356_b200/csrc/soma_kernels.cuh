// soma_kernels.cuh -- sm_100a kernels of the SCMF Monte-Carlo step (DESIGN.md sections 6-7).
//
//   fused_step_kernel<P>   rows a1+a2+a3+a5: a chain lives in the registers of P = N/2 lanes (two
//                          consecutive beads per lane), both half-sweeps run there with warp
//                          shuffles for the cross-lane neighbours, positions are read once and
//                          written once, and every bead is binned into the next density grid with
//                          one red.global.add.u32.
//   half_sweep_kernel      rows a1/a2 for any N (one thread per same-parity bead, neighbours from
//                          global memory); bin_kernel = row a3.  The generic path.
//   omega_kernel<T>        row a4: omega from the fresh counts; also zeroes the other count buffer.
//   chain_key / bin_scan / chain_permute   internal re-ordering of the chains in memory by the
//                          coarse cell of their middle bead (results do not depend on it: the
//                          random stream is keyed by the logical chain id).
#pragma once

#include "soma_device.cuh"

namespace soma {

constexpr int kMaxTypes = 8;

// Everything a move needs, passed by value as a kernel parameter.
struct StepArgs {
  Grid grid;
  uint32_t cells;             // C
  uint32_t n_chains;          // n
  uint32_t N;                 // beads per chain
  uint32_t pat_stride;        // row length of `patterns` (= N unless the system holds species of several lengths)
  uint32_t packed;            // layout of the density counters (soma_device.cuh)
  float a;                    // trial half-width
  float kb;                   // 1.5f/(b*b)
  float gA, sq2A, inv4A;      // bond-force-biased moves (R24): fl(A * 2 kb), (float)sqrt(2A), (float)(1/(4A)); gA = 0: uniform moves
  PhiloxKeys keys;            // round keys of (seed lo, seed hi)
  uint32_t ctr2;              // (uint32) step
  uint32_t ctr3_base;         // domain << 8 | (uint32)(step >> 32) << 16; parity is or-ed in
  float* __restrict__ x;      // positions in slot order: bead i of slot s at s*N + i
  float* __restrict__ y;
  float* __restrict__ z;
  const float* __restrict__ omega;          // [T][C], field of the previous step
  uint32_t* __restrict__ counts_next;       // [T][C], zeroed, receives this step's binning
  const uint32_t* __restrict__ slot_chain;  // [n] logical chain id held by each slot
  const uint8_t* __restrict__ slot_pattern; // [n] pattern id of that chain
  const uint8_t* __restrict__ patterns;     // [n_patterns][N]
  unsigned long long* __restrict__ accepted;
};

// One Metropolis trial move given the bead's position and its (up to two) bonded neighbours.
// Returns the accept decision; on accept (rx,ry,rz) and `cell` are replaced by the trial values.
template <bool POW2>
__device__ __forceinline__ bool move_bead(const StepArgs& A, uint32_t chain, uint32_t i, uint32_t parity,
                                          const float* __restrict__ omega_t,   // omega + type*C
                                          float& rx, float& ry, float& rz, uint32_t& cell,
                                          bool has_l, float lx, float ly, float lz,
                                          bool has_r, float qx, float qy, float qz) {
  const Words4 w = philox4x32_10(i, chain, A.ctr2, A.ctr3_base | parity, A.keys);
  const Trial t = trial_position(rx, ry, rz, A.a, w);
  float dq = 0.0f;
  if (has_l) dq = __fsub_rn(bond_sq(t.x, t.y, t.z, lx, ly, lz), bond_sq(rx, ry, rz, lx, ly, lz));
  if (has_r) {
    const float dqr = __fsub_rn(bond_sq(t.x, t.y, t.z, qx, qy, qz), bond_sq(rx, ry, rz, qx, qy, qz));
    dq = has_l ? __fadd_rn(dq, dqr) : dqr;
  }
  const uint32_t cell_new = cell_of<POW2>(A.grid, t.x, t.y, t.z);
  const float dw = __fsub_rn(__ldg(omega_t + cell_new), __ldg(omega_t + cell));
  const float dE = __fmaf_rn(A.kb, dq, dw);
  const bool acc = metropolis_accept(dE, w.w3);
  if (acc) { rx = t.x; ry = t.y; rz = t.z; cell = cell_new; }
  return acc;
}

// Bond-force-biased move (R24): proposal r' = r + A F + sqrt(2A) xi with the bonded force
// F = -2 kb S, S = sum over the bonded neighbours of (r - r_j); margin = dE + (qr - qf)/(4A) + ln u.
template <bool POW2>
__device__ __forceinline__ bool move_bead_smc(const StepArgs& A, uint32_t chain, uint32_t i, uint32_t parity,
                                              const float* __restrict__ omega_t,
                                              float& rx, float& ry, float& rz, uint32_t& cell,
                                              bool has_l, float lx, float ly, float lz,
                                              bool has_r, float qx, float qy, float qz) {
  const Words4 w = philox4x32_10(i, chain, A.ctr2, A.ctr3_base | parity, A.keys);
  const Words4 v = philox4x32_10(i, chain, A.ctr2, A.ctr3_base | parity | (2u << 8), A.keys);
  float x0, x1, x2;
  smc_deviates(w, v, x0, x1, x2);
  float Sx = 0.f, Sy = 0.f, Sz = 0.f;
  if (has_l) { Sx = __fsub_rn(rx, lx); Sy = __fsub_rn(ry, ly); Sz = __fsub_rn(rz, lz); }
  if (has_r) {
    const float ax = __fsub_rn(rx, qx), ay = __fsub_rn(ry, qy), az = __fsub_rn(rz, qz);
    Sx = has_l ? __fadd_rn(Sx, ax) : ax; Sy = has_l ? __fadd_rn(Sy, ay) : ay; Sz = has_l ? __fadd_rn(Sz, az) : az;
  }
  const float dx = __fmaf_rn(-A.gA, Sx, __fmul_rn(A.sq2A, x0));
  const float dy = __fmaf_rn(-A.gA, Sy, __fmul_rn(A.sq2A, x1));
  const float dz = __fmaf_rn(-A.gA, Sz, __fmul_rn(A.sq2A, x2));
  const float tx = __fadd_rn(rx, dx), ty = __fadd_rn(ry, dy), tz = __fadd_rn(rz, dz);
  float Tx = 0.f, Ty = 0.f, Tz = 0.f, dq = 0.0f;
  if (has_l) {
    Tx = __fsub_rn(tx, lx); Ty = __fsub_rn(ty, ly); Tz = __fsub_rn(tz, lz);
    dq = __fsub_rn(bond_sq(tx, ty, tz, lx, ly, lz), bond_sq(rx, ry, rz, lx, ly, lz));
  }
  if (has_r) {
    const float ax = __fsub_rn(tx, qx), ay = __fsub_rn(ty, qy), az = __fsub_rn(tz, qz);
    Tx = has_l ? __fadd_rn(Tx, ax) : ax; Ty = has_l ? __fadd_rn(Ty, ay) : ay; Tz = has_l ? __fadd_rn(Tz, az) : az;
    const float dqr = __fsub_rn(bond_sq(tx, ty, tz, qx, qy, qz), bond_sq(rx, ry, rz, qx, qy, qz));
    dq = has_l ? __fadd_rn(dq, dqr) : dqr;
  }
  const float ax_ = __fmaf_rn(A.gA, Sx, dx), ay_ = __fmaf_rn(A.gA, Sy, dy), az_ = __fmaf_rn(A.gA, Sz, dz);
  const float bx_ = __fmaf_rn(-A.gA, Tx, dx), by_ = __fmaf_rn(-A.gA, Ty, dy), bz_ = __fmaf_rn(-A.gA, Tz, dz);
  const float qf = __fmaf_rn(az_, az_, __fmaf_rn(ay_, ay_, __fmul_rn(ax_, ax_)));
  const float qr = __fmaf_rn(bz_, bz_, __fmaf_rn(by_, by_, __fmul_rn(bx_, bx_)));
  const uint32_t cell_new = cell_of<POW2>(A.grid, tx, ty, tz);
  const float dw = __fsub_rn(__ldg(omega_t + cell_new), __ldg(omega_t + cell));
  const float dE = __fmaf_rn(A.kb, dq, dw);
  const float meff = __fmaf_rn(A.inv4A, __fsub_rn(qr, qf), dE);
  // accept iff fl(meff + lnu) <= 0: the general decision routine without its dE <= 0 shortcut argument
  // (meff <= 0 still implies acceptance, since lnu <= 0)
  const bool acc = metropolis_accept(meff, w.w3);
  if (acc) { rx = tx; ry = ty; rz = tz; cell = cell_new; }
  return acc;
}

// The move of the fused kernel: the same arithmetic with the loop-invariant work taken out.
//  * Philox rounds 1-3 are partially folded per lane (PhiloxLane, soma_device.cuh);
//  * the squared lengths of the bead's two bonds are carried along (q_l, q_r; on return the lengths
//    after the move) instead of being recomputed, and a missing neighbour contributes
//    h * (finite) = 0 (h = 0 or 1) -- one fp32 add as in DESIGN.md section 2 step 5.4;
//  * FAST (a and all inv_h powers of two, inv_h >= 1, power-of-two grid): a tmap(w) = 2a h + a(2^-23 - 1)
//    is exact in one FFMA, and r inv_h is exact so the floor is one FFMA.RD;
//  * the decision comes from one FFMA on the hardware logarithm with a guard band (metropolis_accept_fma).
struct FusedConst { float a2, ac; uint32_t u0; };   // 2a, a(2^-23 - 1), hi(M1 step) ^ k0[0]

template <bool POW2, bool FAST>
__device__ __forceinline__ uint32_t cell_of_fused(const Grid& g, float x, float y, float z) {
  if (POW2 && FAST) {
    const uint32_t ix = __float_as_uint(__fmaf_rd(x, g.inv_hx, kFloorMagic)) & (g.nx - 1u);
    const uint32_t iy = __float_as_uint(__fmaf_rd(y, g.inv_hy, kFloorMagic)) & (g.ny - 1u);
    const uint32_t iz = __float_as_uint(__fmaf_rd(z, g.inv_hz, kFloorMagic)) & (g.nz - 1u);
    return (ix * g.ny + iy) * g.nz + iz;
  }
  return cell_of<POW2>(g, x, y, z);
}

template <bool FAST>
__device__ __forceinline__ float trial_axis_fused(const StepArgs& A, const FusedConst& F, float r, uint32_t w) {
  if (FAST) {
    const float h = __fadd_rn(__uint_as_float(0x3f800000u | (w >> 9)), -1.0f);
    return __fadd_rn(r, __fmaf_rn(F.a2, h, F.ac));
  }
  return __fadd_rn(r, __fmul_rn(A.a, tmap(w)));
}

template <bool POW2, bool FAST, bool EVEN>
__device__ __forceinline__ bool fused_move(const StepArgs& A, const FusedConst& F, const PhiloxLane& L, uint32_t c0_1,
                                           const float* __restrict__ omega_t,
                                           float& rx, float& ry, float& rz, uint32_t& cell,
                                           float lx, float ly, float lz, float& q_l,
                                           float qx, float qy, float qz, float& q_r, float h) {
  const Words4 w = philox_tail(A.keys, L, c0_1);
  const float tx = trial_axis_fused<FAST>(A, F, rx, w.w0);
  const float ty = trial_axis_fused<FAST>(A, F, ry, w.w1);
  const float tz = trial_axis_fused<FAST>(A, F, rz, w.w2);
  const float ql_new = bond_sq(tx, ty, tz, lx, ly, lz);
  const float qr_new = bond_sq(tx, ty, tz, qx, qy, qz);
  const float dql = __fsub_rn(ql_new, q_l), dqr = __fsub_rn(qr_new, q_r);
  const float dq = EVEN ? __fmaf_rn(h, dql, dqr) : __fmaf_rn(h, dqr, dql);
  const uint32_t cell_new = cell_of_fused<POW2, FAST>(A.grid, tx, ty, tz);
  const float dw = __fsub_rn(__ldg(omega_t + cell_new), __ldg(omega_t + cell));
  const float dE = __fmaf_rn(A.kb, dq, dw);
  const bool acc = metropolis_accept_fma(dE, w.w3);
  if (acc) { rx = tx; ry = ty; rz = tz; cell = cell_new; q_l = ql_new; q_r = qr_new; }
  return acc;
}

// ---------------------------------------------------------------------------------------------
// Generic path: one thread per bead of the given parity.
// ---------------------------------------------------------------------------------------------
template <bool POW2>
__global__ void __launch_bounds__(256)
half_sweep_kernel(StepArgs A, uint32_t parity, uint32_t n_par /* beads of this parity per chain */) {
  const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const uint64_t total = (uint64_t)A.n_chains * n_par;
  bool acc = false;
  if (k < total) {
    const uint32_t slot = (uint32_t)(k / n_par);
    const uint32_t i = parity + 2u * (uint32_t)(k % n_par);
    const uint64_t j = (uint64_t)slot * A.N + i;
    const uint32_t chain = A.slot_chain[slot];
    const uint32_t type = A.patterns[(uint32_t)A.slot_pattern[slot] * A.pat_stride + i];
    float rx = A.x[j], ry = A.y[j], rz = A.z[j];
    const bool has_l = i > 0, has_r = i + 1 < A.N;
    float lx = 0, ly = 0, lz = 0, qx = 0, qy = 0, qz = 0;
    if (has_l) { lx = A.x[j - 1]; ly = A.y[j - 1]; lz = A.z[j - 1]; }
    if (has_r) { qx = A.x[j + 1]; qy = A.y[j + 1]; qz = A.z[j + 1]; }
    uint32_t cell = cell_of<POW2>(A.grid, rx, ry, rz);
    acc = A.gA > 0.0f ? move_bead_smc<POW2>(A, chain, i, parity, A.omega + (size_t)type * A.cells, rx, ry, rz, cell,
                                            has_l, lx, ly, lz, has_r, qx, qy, qz)
                      : move_bead<POW2>(A, chain, i, parity, A.omega + (size_t)type * A.cells, rx, ry, rz, cell,
                                        has_l, lx, ly, lz, has_r, qx, qy, qz);
    if (acc) { A.x[j] = rx; A.y[j] = ry; A.z[j] = rz; }
  }
  const unsigned n_acc = __popc(__ballot_sync(0xffffffffu, acc));
  if ((threadIdx.x & 31u) == 0 && n_acc) atomicAdd(A.accepted, (unsigned long long)n_acc);
}

// Row a3 on its own.  `range_flag` (may be null) is set to 1 if any bead's cell coordinate leaves
// the range in which the conversion-free floor of soma_device.cuh is exact.
template <bool POW2>
__global__ void __launch_bounds__(256)
bin_kernel(Grid grid, uint32_t cells, uint32_t N, uint32_t pat_stride, uint32_t packed, uint64_t B, const float* __restrict__ x,
           const float* __restrict__ y, const float* __restrict__ z,
           const uint8_t* __restrict__ slot_pattern, const uint8_t* __restrict__ patterns,
           uint32_t* __restrict__ counts, uint32_t* __restrict__ range_flag) {
  const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= B) return;
  const uint32_t slot = (uint32_t)(j / N), i = (uint32_t)(j % N);
  const uint32_t type = patterns[(uint32_t)slot_pattern[slot] * pat_stride + i];
  const float px = x[j], py = y[j], pz = z[j];
  if (range_flag) {
    const float m = fmaxf(fabsf(__fmul_rn(px, grid.inv_hx)), fmaxf(fabsf(__fmul_rn(py, grid.inv_hy)), fabsf(__fmul_rn(pz, grid.inv_hz))));
    if (!(m < kCellCoordLimit)) *range_flag = 1u;            // also catches NaN
  }
  atomicAdd(counts + count_word(type, cells, packed) + cell_of<POW2>(grid, px, py, pz), count_inc(type, packed));
}

// ---------------------------------------------------------------------------------------------
// Fused path: N = 2P, P in {1,2,4,8,16,32}.  Lane l of a P-lane group holds beads 2l and 2l+1.
// A warp carries G = 32/P chains.  Every block owns a CONTIGUOUS run of `groups_per_block` warp
// groups of the slot list and its warps walk that run side by side, so that -- the chains being
// kept sorted by position -- the omega gathers of a block stay inside a small neighbourhood that
// the L1 keeps, and the atomics of concurrently running blocks fall into a bounded part of L2.
// ---------------------------------------------------------------------------------------------
#ifndef SOMA_FUSED_MIN_BLOCKS
#define SOMA_FUSED_MIN_BLOCKS 4      /* 62 registers: 4 blocks per SM; measured best on cfg4 (3: 1.61 ms, 4: 1.13, 5: 1.16, 6: 1.28) */
#endif
// SMC: bond-force-biased moves (R24) instead of uniform ones; their normal
// deviates need more registers: that variant runs 3 blocks per SM (80 registers; measured 3 / 4 blocks = 2.02 / 2.13 ms on cfg4).
template <int P, bool POW2, bool MULTI_PAT, bool FAST, bool SMC = false>
__global__ void __launch_bounds__(256, SMC ? 3 : SOMA_FUSED_MIN_BLOCKS)
fused_step_kernel(StepArgs A, uint32_t groups_per_block) {
  constexpr int G = 32 / P;                                   // chains per warp
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t l = lane % P;                                // position of the lane in its chain
  const uint32_t sub = lane / P;                              // which of the warp's chains
  const uint32_t wpb = blockDim.x >> 5;
  const uint64_t n_groups = ((uint64_t)A.n_chains + G - 1) / G;
  unsigned n_acc = 0;

  const float hl = l > 0 ? 1.0f : 0.0f, hr = l + 1 < P ? 1.0f : 0.0f;    // does the left / right cross-lane neighbour exist
  FusedConst F;
  F.a2 = __fmul_rn(2.0f, A.a);
  F.ac = __fmul_rn(A.a, -0.99999988079071044921875f);                    // a (2^-23 - 1): exact when a is a power of two
  const uint64_t m1 = (uint64_t)kPhiloxM1 * A.ctr2;
  F.u0 = (uint32_t)(m1 >> 32) ^ A.keys.k0[0];
  const PhiloxLane L0 = philox_lane(A.keys, (uint32_t)m1, 2u * l, A.ctr3_base);
  const PhiloxLane L1 = philox_lane(A.keys, (uint32_t)m1, 2u * l + 1u, A.ctr3_base | 1u);
  // bead types of this lane (loop-invariant when every chain has the same pattern)
  uint32_t type0 = 0, type1 = 0;
  if (!MULTI_PAT) {
    const uint16_t tt = *reinterpret_cast<const uint16_t*>(A.patterns + 2u * l);
    type0 = tt & 0xffu; type1 = tt >> 8;
  }

  // Every block takes one chunk of `groups_per_block` consecutive warp groups.  The hardware hands
  // the blocks out in launch order as earlier ones retire, so at any moment the whole grid works on
  // one contiguous stretch of the position-sorted chain list: the omega values and density counters
  // that stretch touches (a few MB) stay in L2, which one long run per block (every block in a
  // different part of the box) does not allow.
  const uint64_t g_begin = (uint64_t)blockIdx.x * groups_per_block;
  uint64_t g_end = g_begin + groups_per_block;
  if (g_end > n_groups) g_end = n_groups;
  // positions and chain id of the warp's next group are fetched one iteration ahead
  float2 Xn = make_float2(0.f, 0.f), Yn = Xn, Zn = Xn;
  uint32_t chain_n = 0;
  auto fetch = [&](uint64_t wg) {
    const uint64_t s64 = wg * G + sub;
    const uint32_t sl = s64 < A.n_chains ? (uint32_t)s64 : 0u;
    const uint64_t jj = (uint64_t)sl * A.N + 2u * l;
    // positions are streamed (read once, written once): keep them from evicting omega out of L1
    Xn = __ldcs(reinterpret_cast<const float2*>(A.x + jj));
    Yn = __ldcs(reinterpret_cast<const float2*>(A.y + jj));
    Zn = __ldcs(reinterpret_cast<const float2*>(A.z + jj));
    chain_n = A.slot_chain[sl];
  };
  if (g_begin + (threadIdx.x >> 5) < g_end) fetch(g_begin + (threadIdx.x >> 5));
  for (uint64_t wg = g_begin + (threadIdx.x >> 5); wg < g_end; wg += wpb) {
    const uint64_t slot64 = wg * G + sub;
    const bool live = slot64 < A.n_chains;
    const uint32_t slot = live ? (uint32_t)slot64 : 0u;       // dead lanes shadow slot 0, never store
    const uint64_t j = (uint64_t)slot * A.N + 2u * l;
    const float2 X = Xn, Y = Yn, Z = Zn;
    const uint32_t chain = chain_n;
    if (wg + wpb < g_end) fetch(wg + wpb);
    if (MULTI_PAT) {
      const uint16_t tt = *reinterpret_cast<const uint16_t*>(A.patterns + (uint32_t)A.slot_pattern[slot] * A.pat_stride + 2u * l);
      type0 = tt & 0xffu; type1 = tt >> 8;
    }
    const float* om0 = A.omega + (size_t)type0 * A.cells;
    const float* om1 = A.omega + (size_t)type1 * A.cells;

    float ex = X.x, ey = Y.x, ez = Z.x;                       // even bead 2l
    float ox = X.y, oy = Y.y, oz = Z.y;                       // odd bead 2l+1
    uint32_t cell_e = cell_of_fused<POW2, FAST>(A.grid, ex, ey, ez);
    uint32_t cell_o = cell_of_fused<POW2, FAST>(A.grid, ox, oy, oz);
    const uint32_t c0_1 = F.u0 ^ chain;

    // half-sweep 0: even bead; left neighbour = odd bead of lane l-1, right neighbour = own odd bead.
    // qA = |even - odd|^2, qB = |odd of lane l-1 - even|^2
    const float lx = __shfl_up_sync(0xffffffffu, ox, 1, P);
    const float ly = __shfl_up_sync(0xffffffffu, oy, 1, P);
    const float lz = __shfl_up_sync(0xffffffffu, oz, 1, P);
    float qA = bond_sq(ex, ey, ez, ox, oy, oz);
    float qB = bond_sq(ex, ey, ez, lx, ly, lz);
    if (SMC) {
      const bool acc = move_bead_smc<POW2>(A, chain, 2u * l, 0u, om0, ex, ey, ez, cell_e, l > 0, lx, ly, lz, true, ox, oy, oz);
      n_acc += (acc && live) ? 1u : 0u;
    } else {
      const bool acc = fused_move<POW2, FAST, true>(A, F, L0, c0_1, om0, ex, ey, ez, cell_e,
                                                    lx, ly, lz, qB, ox, oy, oz, qA, hl);
      n_acc += (acc && live) ? 1u : 0u;
    }
    // half-sweep 1: odd bead; left = own even bead (new), right = even bead of lane l+1 (new)
    {
      const float qx = __shfl_down_sync(0xffffffffu, ex, 1, P);
      const float qy = __shfl_down_sync(0xffffffffu, ey, 1, P);
      const float qz = __shfl_down_sync(0xffffffffu, ez, 1, P);
      float qR = __shfl_down_sync(0xffffffffu, qB, 1, P);
      const bool acc = SMC ? move_bead_smc<POW2>(A, chain, 2u * l + 1u, 1u, om1, ox, oy, oz, cell_o, true, ex, ey, ez, l + 1 < P, qx, qy, qz)
                           : fused_move<POW2, FAST, false>(A, F, L1, c0_1, om1, ox, oy, oz, cell_o,
                                                           ex, ey, ez, qA, qx, qy, qz, qR, hr);
      n_acc += (acc && live) ? 1u : 0u;
    }
    if (live) {
      __stcs(reinterpret_cast<float2*>(A.x + j), make_float2(ex, ox));
      __stcs(reinterpret_cast<float2*>(A.y + j), make_float2(ey, oy));
      __stcs(reinterpret_cast<float2*>(A.z + j), make_float2(ez, oz));
      {
        const uint32_t pk = SMC ? 0u : A.packed;                  // bond-force-biased moves never run on packed counters (soma_device.cuh)
        atomicAdd(A.counts_next + count_word(type0, A.cells, pk) + cell_e, count_inc(type0, pk));
        atomicAdd(A.counts_next + count_word(type1, A.cells, pk) + cell_o, count_inc(type1, pk));
      }
    }
  }
  // accepted-move count: warp reduce, one atomic per warp
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
  if (lane == 0 && n_acc) atomicAdd(A.accepted, (unsigned long long)n_acc);
}

// ---------------------------------------------------------------------------------------------
// Row a4: omega from the counts (DESIGN.md section 2 step 3).  One thread per cell; the same pass
// zeroes the count buffer the next step will bin into.
// ---------------------------------------------------------------------------------------------
struct OmegaArgs {
  uint32_t cells, T;
  float dens_scale, kappaN, invN;
  float chiN[kMaxTypes * kMaxTypes];         // [T][T]
  uint32_t packed;                           // layout of the counters (soma_device.cuh)
  uint32_t guard_mask;                       // packed: bits of a word that are set once a 16-bit field has reached the guard level
  uint32_t* __restrict__ guard_flag;         // packed: set to 1 if that happened
  const uint32_t* __restrict__ counts;       // fresh counts
  uint32_t* __restrict__ counts_to_zero;     // buffer for the next step (may be null)
  float* __restrict__ omega;                 // [T][C]
  const float* __restrict__ ext;             // [T][C] external field added to omega (R21), or null
  const float* __restrict__ phi_tgt;         // [T][C] target concentrations of the umbrella potential (R25), or null
  float umbrella_k;
};

template <int T_>
__global__ void __launch_bounds__(256)
omega_kernel(OmegaArgs A) {
  const uint32_t T = T_ > 0 ? (uint32_t)T_ : A.T;
  const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= A.cells) return;
  float phi[kMaxTypes];
  float tot = 0.0f;
#pragma unroll
  for (uint32_t s = 0; s < (T_ > 0 ? T_ : kMaxTypes); ++s) {
    if (s < T) {
      const uint32_t cnt = count_get(A.counts, s, A.cells, c, A.packed);
      if (A.packed && (cnt & A.guard_mask)) *A.guard_flag = 1u;
      phi[s] = __fmul_rn((float)cnt, A.dens_scale);
      tot = s == 0 ? phi[0] : __fadd_rn(tot, phi[s]);
      if (A.counts_to_zero && (!A.packed || s == 0)) A.counts_to_zero[(size_t)s * A.cells + c] = 0u;
    }
  }
  const float p = __fmul_rn(A.kappaN, __fsub_rn(tot, 1.0f));
#pragma unroll
  for (uint32_t t = 0; t < (T_ > 0 ? T_ : kMaxTypes); ++t) {
    if (t < T) {
      float acc = p;
#pragma unroll
      for (uint32_t s = 0; s < (T_ > 0 ? T_ : kMaxTypes); ++s)
        if (s < T && s != t) acc = __fmaf_rn(A.chiN[t * T + s], phi[s], acc);
      float w = __fmul_rn(A.invN, acc);
      if (A.ext) w = __fadd_rn(w, A.ext[(size_t)t * A.cells + c]);
      if (A.phi_tgt) w = __fadd_rn(w, __fmul_rn(A.umbrella_k, __fsub_rn(phi[t], A.phi_tgt[(size_t)t * A.cells + c])));
      A.omega[(size_t)t * A.cells + c] = w;
    }
  }
}

// The same pass, four consecutive cells per thread with 128-bit loads and stores (cells a multiple of 4;
// every cell goes through omega_cell's arithmetic, so the results are those of omega_kernel bit for bit).
template <int T_>
__global__ void __launch_bounds__(256)
omega_kernel_x4(OmegaArgs A) {
  static_assert(T_ > 0, "fixed number of types");
  const uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) * 4u;
  if (c >= A.cells) return;
  uint4 n[T_];
  if (A.packed) {                                               // T_ <= 2: both types in one word
    const uint4 p = *reinterpret_cast<const uint4*>(A.counts + c);
    if (A.counts_to_zero) *reinterpret_cast<uint4*>(A.counts_to_zero + c) = make_uint4(0u, 0u, 0u, 0u);
    n[0] = make_uint4(p.x & 0xffffu, p.y & 0xffffu, p.z & 0xffffu, p.w & 0xffffu);
    if (T_ > 1) n[T_ > 1 ? 1 : 0] = make_uint4(p.x >> 16, p.y >> 16, p.z >> 16, p.w >> 16);
    if ((p.x | p.y | p.z | p.w) & A.guard_mask) *A.guard_flag = 1u;
  } else {
#pragma unroll
    for (int s = 0; s < T_; ++s) {
      n[s] = *reinterpret_cast<const uint4*>(A.counts + (size_t)s * A.cells + c);
      if (A.counts_to_zero) *reinterpret_cast<uint4*>(A.counts_to_zero + (size_t)s * A.cells + c) = make_uint4(0u, 0u, 0u, 0u);
    }
  }
  float4 w[T_];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    float phi[T_], tot = 0.0f;
#pragma unroll
    for (int s = 0; s < T_; ++s) {
      const uint32_t cnt = k == 0 ? n[s].x : k == 1 ? n[s].y : k == 2 ? n[s].z : n[s].w;
      phi[s] = __fmul_rn((float)cnt, A.dens_scale);
      tot = s == 0 ? phi[0] : __fadd_rn(tot, phi[s]);
    }
    const float p = __fmul_rn(A.kappaN, __fsub_rn(tot, 1.0f));
#pragma unroll
    for (int t = 0; t < T_; ++t) {
      float acc = p;
#pragma unroll
      for (int s = 0; s < T_; ++s)
        if (s != t) acc = __fmaf_rn(A.chiN[t * T_ + s], phi[s], acc);
      float v = __fmul_rn(A.invN, acc);
      if (A.ext) v = __fadd_rn(v, A.ext[(size_t)t * A.cells + c + k]);
      if (A.phi_tgt) v = __fadd_rn(v, __fmul_rn(A.umbrella_k, __fsub_rn(phi[t], A.phi_tgt[(size_t)t * A.cells + c + k])));
      (k == 0 ? w[t].x : k == 1 ? w[t].y : k == 2 ? w[t].z : w[t].w) = v;
    }
  }
#pragma unroll
  for (int t = 0; t < T_; ++t) *reinterpret_cast<float4*>(A.omega + (size_t)t * A.cells + c) = w[t];
}

// ---------------------------------------------------------------------------------------------
// Chain re-ordering: a counting sort of the slots by the coarse bin (cb^3 cells, row-major) that
// holds the chain's middle bead.  key -> per-bin count and rank (one atomic with return per chain),
// exclusive scan of the bin counts, then every chain is copied to slot bin_start[bin] + rank.
// The rank order inside a bin depends on atomic arrival order; nothing observable depends on the
// slot a chain sits in.
// ---------------------------------------------------------------------------------------------
struct SortArgs {
  Grid grid;
  uint32_t n_chains, N;
  uint32_t cbx, cby, cbz;          // coarse bin edges in cells
  uint32_t ncy, ncz;               // coarse bins along y and z (x is implied)
};

// bin of a chain = coarse bin of the cell that holds its centre of mass (fp32 mean of the beads)
template <bool POW2>
__global__ void __launch_bounds__(256)
chain_key_kernel(SortArgs S, const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z,
                 uint32_t* __restrict__ bin_count, uint32_t* __restrict__ key, uint32_t* __restrict__ rank) {
  const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= S.n_chains) return;
  const uint64_t j0 = (uint64_t)s * S.N;
  float sx = 0.f, sy = 0.f, sz = 0.f;
  if ((S.N & 3u) == 0 && ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(y) | reinterpret_cast<uintptr_t>(z)) & 15u) == 0) {
    for (uint32_t i = 0; i < S.N; i += 4) {    // (a species may start at any bead offset: 128-bit loads only where they are aligned)
      const float4 a = *reinterpret_cast<const float4*>(x + j0 + i);
      const float4 b = *reinterpret_cast<const float4*>(y + j0 + i);
      const float4 c = *reinterpret_cast<const float4*>(z + j0 + i);
      sx += (a.x + a.y) + (a.z + a.w); sy += (b.x + b.y) + (b.z + b.w); sz += (c.x + c.y) + (c.z + c.w);
    }
  } else {
    for (uint32_t i = 0; i < S.N; ++i) { sx += x[j0 + i]; sy += y[j0 + i]; sz += z[j0 + i]; }
  }
  const float inv = 1.0f / (float)S.N;
  const uint32_t cell = cell_of<POW2>(S.grid, sx * inv, sy * inv, sz * inv);
  const uint32_t iz = cell % S.grid.nz, iy = (cell / S.grid.nz) % S.grid.ny, ix = cell / (S.grid.nz * S.grid.ny);
  const uint32_t bin = ((ix / S.cbx) * S.ncy + iy / S.cby) * S.ncz + iz / S.cbz;
  key[s] = bin;
  rank[s] = atomicAdd(bin_count + bin, 1u);
}

// exclusive scan of `n` counts in place, one block; n is at most a few million
__global__ void __launch_bounds__(1024)
bin_scan_kernel(uint32_t n, uint32_t* __restrict__ v) {
  __shared__ uint32_t warp_sum[32];
  __shared__ uint32_t carry_s;
  const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (uint32_t base = 0; base < n; base += 1024u) {
    const uint32_t k = base + threadIdx.x;
    const uint32_t val = k < n ? v[k] : 0u;
    uint32_t inc = val;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= (uint32_t)o) inc += t;
    }
    if (lane == 31) warp_sum[w] = inc;
    __syncthreads();
    if (w == 0) {
      uint32_t ws = warp_sum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, ws, o);
        if (lane >= (uint32_t)o) ws += t;
      }
      warp_sum[lane] = ws;                                   // inclusive over warps
    }
    __syncthreads();
    const uint32_t carry = carry_s;
    const uint32_t before = carry + (w ? warp_sum[w - 1] : 0u) + inc - val;
    if (k < n) v[k] = before;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = carry + warp_sum[31];
    __syncthreads();
  }
}

// The same scan over many blocks for grids with many coarse bins (cfg4: 131 073 entries, where one block took 0.12 ms of
// a 1.1 ms re-ordering): sums of chunks of kBinScanChunk entries, bin_scan_kernel over the chunk sums, then every block
// scans its own chunk and adds its offset.  Integer sums: the result is the single-block kernel's.
constexpr uint32_t kBinScanChunk = 1024;      // 256 threads x 4 entries

__global__ void __launch_bounds__(256)
bin_chunk_sums_kernel(uint32_t n, const uint32_t* __restrict__ v, uint32_t* __restrict__ chunk_sum) {
  __shared__ uint32_t part[8];
  const uint32_t base = blockIdx.x * kBinScanChunk + threadIdx.x * 4u;
  uint32_t s = 0;
#pragma unroll
  for (uint32_t k = 0; k < 4; ++k) if (base + k < n) s += v[base + k];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31u) == 0) part[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
    for (int w = 0; w < 8; ++w) t += part[w];
    chunk_sum[blockIdx.x] = t;
  }
}

__global__ void __launch_bounds__(256)
bin_scan_apply_kernel(uint32_t n, uint32_t* __restrict__ v, const uint32_t* __restrict__ chunk_offset) {
  __shared__ uint32_t part[8];
  const uint32_t base = blockIdx.x * kBinScanChunk + threadIdx.x * 4u;
  const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
  uint32_t e[4], s = 0;
#pragma unroll
  for (uint32_t k = 0; k < 4; ++k) { e[k] = base + k < n ? v[base + k] : 0u; s += e[k]; }
  uint32_t inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (uint32_t)o) inc += t;
  }
  if (lane == 31) part[w] = inc;
  __syncthreads();
  uint32_t run = chunk_offset[blockIdx.x] + inc - s;            // entries before this thread's four
  for (uint32_t q = 0; q < w; ++q) run += part[q];
#pragma unroll
  for (uint32_t k = 0; k < 4; ++k) { if (base + k < n) v[base + k] = run; run += e[k]; }
}

// one thread per bead: slot s -> slot bin_start[key[s]] + rank[s]
__global__ void __launch_bounds__(256)
chain_permute_kernel(uint64_t B, uint32_t N, const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ key,
                     const uint32_t* __restrict__ rank,
                     const float* __restrict__ sx, const float* __restrict__ sy, const float* __restrict__ sz,
                     float* __restrict__ dx, float* __restrict__ dy, float* __restrict__ dz,
                     const uint32_t* __restrict__ s_chain, const uint8_t* __restrict__ s_pat,
                     uint32_t* __restrict__ d_chain, uint8_t* __restrict__ d_pat) {
  const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= B) return;
  const uint32_t s = (uint32_t)(j / N), i = (uint32_t)(j % N);
  const uint32_t d = bin_start[key[s]] + rank[s];
  const uint64_t k = (uint64_t)d * N + i;
  dx[k] = sx[j]; dy[k] = sy[j]; dz[k] = sz[j];
  if (i == 0) { d_chain[d] = s_chain[s]; d_pat[d] = s_pat[s]; }
}

// the same for chain lengths that are multiples of four (and 16-byte aligned arrays): one thread per four beads,
// 128-bit loads and stores, no division by the chain length (quads per chain passed in)
__global__ void __launch_bounds__(256)
chain_permute4_kernel(uint64_t n_quads, uint32_t quads_per_chain, const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ key,
                      const uint32_t* __restrict__ rank,
                      const float4* __restrict__ sx, const float4* __restrict__ sy, const float4* __restrict__ sz,
                      float4* __restrict__ dx, float4* __restrict__ dy, float4* __restrict__ dz,
                      const uint32_t* __restrict__ s_chain, const uint8_t* __restrict__ s_pat,
                      uint32_t* __restrict__ d_chain, uint8_t* __restrict__ d_pat) {
  const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_quads) return;
  const uint32_t s = (uint32_t)(j / quads_per_chain), q = (uint32_t)(j - (uint64_t)s * quads_per_chain);
  const uint32_t d = __ldg(bin_start + __ldg(key + s)) + __ldg(rank + s);
  const uint64_t k = (uint64_t)d * quads_per_chain + q;
  dx[k] = __ldcs(sx + j); dy[k] = __ldcs(sy + j); dz[k] = __ldcs(sz + j);
  if (q == 0) { d_chain[d] = s_chain[s]; d_pat[d] = s_pat[s]; }
}

// sets *range_flag if a bead's cell coordinate is NaN or beyond kCellCoordLimit (see floor_bits)
__global__ void __launch_bounds__(256)
range_check_kernel(Grid grid, uint64_t B, const float* __restrict__ x, const float* __restrict__ y,
                   const float* __restrict__ z, uint32_t* __restrict__ range_flag) {
  const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= B) return;
  const float m = fmaxf(fabsf(__fmul_rn(x[j], grid.inv_hx)), fmaxf(fabsf(__fmul_rn(y[j], grid.inv_hy)), fabsf(__fmul_rn(z[j], grid.inv_hz))));
  if (!(m < kCellCoordLimit)) *range_flag = 1u;
}

// ---------------------------------------------------------------------------------------------
// Single-bead molecules next to the chains (solvent species, R23):
// molecule m = bead 0 of logical chain n_chains + m, moved in half-sweep 0, no bonds, so
// dE = fma(kb, 0, dw) = omega_t(new cell) - omega_t(old cell).  One thread per molecule; positions in
// their own arrays (never re-ordered), type by the per-type start table.
// ---------------------------------------------------------------------------------------------
struct SingleArgs {
  StepArgs S;                       // grid, cells, a, kb, keys, ctr2, ctr3_base, omega, accepted; n_chains = first logical id
  uint32_t n_total, T;
  uint32_t start[kMaxTypes + 1];    // molecules of type t are [start[t], start[t+1])
  float* __restrict__ x; float* __restrict__ y; float* __restrict__ z;
  uint32_t* __restrict__ counts;    // grid to bin into: [T][C]
  uint32_t* __restrict__ range_flag;  // may be null
  int do_move, do_bin;
};

template <bool POW2>
__global__ void __launch_bounds__(256)
singles_kernel(SingleArgs A) {
  const uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
  bool acc = false;
  if (m < A.n_total) {
    uint32_t type = 0;
    while (m >= A.start[type + 1]) ++type;
    float rx = A.x[m], ry = A.y[m], rz = A.z[m];
    const Grid& G = A.S.grid;
    if (A.range_flag) {
      const float mm = fmaxf(fabsf(__fmul_rn(rx, G.inv_hx)), fmaxf(fabsf(__fmul_rn(ry, G.inv_hy)), fabsf(__fmul_rn(rz, G.inv_hz))));
      if (!(mm < kCellCoordLimit)) *A.range_flag = 1u;
    }
    if (A.do_move) {
      const Words4 w = philox4x32_10(0u, A.S.n_chains + m, A.S.ctr2, A.S.ctr3_base, A.S.keys);
      const Trial t = trial_position(rx, ry, rz, A.S.a, w);
      const float* om = A.S.omega + (size_t)type * A.S.cells;
      const float dw = __fsub_rn(__ldg(om + cell_of<POW2>(G, t.x, t.y, t.z)), __ldg(om + cell_of<POW2>(G, rx, ry, rz)));
      acc = metropolis_accept(__fmaf_rn(A.S.kb, 0.0f, dw), w.w3);
      if (acc) { rx = t.x; ry = t.y; rz = t.z; A.x[m] = rx; A.y[m] = ry; A.z[m] = rz; }
    }
    if (A.do_bin) atomicAdd(A.counts + count_word(type, A.S.cells, A.S.packed) + cell_of<POW2>(G, rx, ry, rz), count_inc(type, A.S.packed));
  }
  const unsigned n_acc = __popc(__ballot_sync(0xffffffffu, acc));
  if ((threadIdx.x & 31u) == 0 && n_acc) atomicAdd(A.S.accepted, (unsigned long long)n_acc);
}

// single-bead molecules of the generated initial state: the bead-0 rule with chain id n_chains + m
__global__ void __launch_bounds__(256)
generate_singles_kernel(uint32_t n_total, uint32_t first_id, uint32_t k0, uint32_t k1, double bx, double by, double bz,
                        float* __restrict__ x, float* __restrict__ y, float* __restrict__ z) {
  const uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n_total) return;
  const Words4 w = philox4x32_10(0u, first_id + m, 0u, 1u << 8, k0, k1);
  x[m] = (float)(bx * (((double)w.w0 + 0.5) * 0x1p-32));
  y[m] = (float)(by * (((double)w.w1 + 0.5) * 0x1p-32));
  z[m] = (float)(bz * (((double)w.w2 + 0.5) * 0x1p-32));
}

// ---------------------------------------------------------------------------------------------
// Initial state on the device (R22): Gaussian random-walk
// chains, first bead uniform in the box.  One thread per chain; draws keyed by (bead, chain) in
// Philox domain 1; double-precision Box-Muller and accumulation, one rounding to fp32 per coordinate.
// ---------------------------------------------------------------------------------------------
struct GenArgs {
  uint32_t n_chains, N;            // chains of this species and their length
  uint32_t chain0;                 // logical id of its first chain
  uint32_t k0, k1;                 // generator seed, low and high word
  double box[3];
  double sigma;                    // b / sqrt(3)
  float* __restrict__ x; float* __restrict__ y; float* __restrict__ z;
};

__device__ __forceinline__ double unit_open(uint32_t w) { return ((double)w + 0.5) * 0x1p-32; }

// One thread per chain (the walk is sequential along the chain); the coordinates go through a per-warp tile of
// shared memory so that the stores are 128-byte rows of one chain instead of 32 rows strided by the chain length.
__global__ void __launch_bounds__(64)
generate_state_kernel(GenArgs G) {
  __shared__ float tile[2][3][32][33];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  const uint32_t c0 = blockIdx.x * blockDim.x + warp * 32u;      // first chain of this warp
  if (c0 >= G.n_chains) return;
  const uint32_t c = c0 + lane;
  const bool live = c < G.n_chains;
  const uint32_t n_here = G.n_chains - c0 < 32u ? G.n_chains - c0 : 32u;
  const double two_pi = 6.283185307179586;
  double r0 = 0.0, r1 = 0.0, r2 = 0.0;
  for (uint32_t i0 = 0; i0 < G.N; i0 += 32u) {
    const uint32_t cnt = G.N - i0 < 32u ? G.N - i0 : 32u;
    for (uint32_t k = 0; k < cnt; ++k) {
      const uint32_t i = i0 + k;
      if (live) {
        const Words4 w = philox4x32_10(i, G.chain0 + c, 0u, 1u << 8, G.k0, G.k1);
        if (i == 0) {
          r0 = G.box[0] * unit_open(w.w0); r1 = G.box[1] * unit_open(w.w1); r2 = G.box[2] * unit_open(w.w2);
        } else {
          const double ra = sqrt(-2.0 * log(unit_open(w.w0))), rb = sqrt(-2.0 * log(unit_open(w.w2)));
          const double t1 = two_pi * unit_open(w.w1), t3 = two_pi * unit_open(w.w3);
          r0 = __dadd_rn(r0, __dmul_rn(G.sigma, __dmul_rn(ra, cos(t1))));
          r1 = __dadd_rn(r1, __dmul_rn(G.sigma, __dmul_rn(ra, sin(t1))));
          r2 = __dadd_rn(r2, __dmul_rn(G.sigma, __dmul_rn(rb, cos(t3))));
        }
      }
      tile[warp][0][lane][k] = (float)r0; tile[warp][1][lane][k] = (float)r1; tile[warp][2][lane][k] = (float)r2;
    }
    __syncwarp();
    for (uint32_t r = 0; r < n_here; ++r) {                      // row r of the tile = beads i0 .. i0 + cnt - 1 of chain c0 + r
      const uint64_t j = (uint64_t)(c0 + r) * G.N + i0 + lane;
      if (lane < cnt) { G.x[j] = tile[warp][0][r][lane]; G.y[j] = tile[warp][1][r][lane]; G.z[j] = tile[warp][2][r][lane]; }
    }
    __syncwarp();
  }
}

// ---------------------------------------------------------------------------------------------
// Validation of the current state (the paper's "validation functions").
// report[0] = non-finite coordinates, report[1 + t] = beads of type t in the density grids,
// report[9] = bit pattern of the largest squared bond length, bond_sum = sum of squared bond lengths.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
validate_positions_kernel(uint64_t B, uint32_t N, const float* __restrict__ x, const float* __restrict__ y,
                          const float* __restrict__ z, unsigned long long* __restrict__ report, double* __restrict__ bond_sum) {
  const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned bad = 0;
  float q = 0.0f;
  if (j < B) {
    const float px = x[j], py = y[j], pz = z[j];
    bad = (isfinite(px) ? 0u : 1u) + (isfinite(py) ? 0u : 1u) + (isfinite(pz) ? 0u : 1u);
    if ((uint32_t)(j % N) + 1u < N) q = bond_sq(px, py, pz, x[j + 1], y[j + 1], z[j + 1]);   // bond (i, i+1) of the same chain
  }
  // NaN never wins a maximum taken on bit patterns of non-negative floats; it is counted in `bad`
  float qm = q == q ? q : 0.0f;
  double qs = q == q ? (double)q : 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bad += __shfl_xor_sync(0xffffffffu, bad, o);
    qm = fmaxf(qm, __shfl_xor_sync(0xffffffffu, qm, o));
    qs += __shfl_xor_sync(0xffffffffu, qs, o);
  }
  if ((threadIdx.x & 31u) == 0) {
    if (bad) atomicAdd(report, (unsigned long long)bad);
    atomicMax(report + 9, (unsigned long long)__float_as_uint(qm));
    atomicAdd(bond_sum, qs);
  }
}

__global__ void __launch_bounds__(256)
validate_density_kernel(uint32_t cells, uint32_t T, uint32_t packed, const uint32_t* __restrict__ counts, unsigned long long* __restrict__ report) {
  const uint32_t t = blockIdx.y;
  unsigned long long sum = 0;
  for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < cells; c += gridDim.x * blockDim.x) sum += count_get(counts, t, cells, c, packed);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if ((threadIdx.x & 31u) == 0 && sum) atomicAdd(report + 1 + t, sum);
}

// packed counters -> [T][C] uint32 (soma_get_density)
__global__ void __launch_bounds__(256)
unpack_counts_kernel(uint32_t cells, uint32_t T, const uint32_t* __restrict__ packed_counts, uint32_t* __restrict__ out) {
  const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= cells) return;
  const uint32_t w = packed_counts[c];
  out[c] = w & 0xffffu;
  if (T > 1) out[(size_t)cells + c] = w >> 16;
}

// ---- data movement helpers ----
// dst[slot_chain[s]*N + i] = src[s*N + i]  (slot order -> caller's chain order), one thread per bead
__global__ void __launch_bounds__(256)
unpermute_kernel(uint64_t B, uint32_t N, uint32_t first_chain, const uint32_t* __restrict__ slot_chain,
                 const float* __restrict__ sx, const float* __restrict__ sy, const float* __restrict__ sz,
                 float* __restrict__ dx, float* __restrict__ dy, float* __restrict__ dz) {
  const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= B) return;
  const uint32_t slot = (uint32_t)(j / N), i = (uint32_t)(j % N);
  const uint64_t d = (uint64_t)(slot_chain[slot] - first_chain) * N + i;
  dx[d] = sx[j]; dy[d] = sy[j]; dz[d] = sz[j];
}

__global__ void __launch_bounds__(256)
iota_kernel(uint32_t n, uint32_t* __restrict__ out) {
  const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) out[k] = k;
}

// ---- test hooks ----
__global__ void debug_philox_kernel(uint64_t n, const uint32_t* ctr, PhiloxKeys K, uint32_t* out) {
  const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const Words4 w = philox4x32_10(ctr[4 * k], ctr[4 * k + 1], ctr[4 * k + 2], ctr[4 * k + 3], K);
  out[4 * k] = w.w0; out[4 * k + 1] = w.w1; out[4 * k + 2] = w.w2; out[4 * k + 3] = w.w3;
}
__global__ void debug_maps_kernel(uint64_t n, const uint32_t* words, float* t, float* u, float* lnu, float* lnu_f) {
  const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  t[k] = tmap(words[k]);
  u[k] = umap(words[k]);
  lnu[k] = lnu_exact(umap(words[k]));
  if (lnu_f) lnu_f[k] = lnu_fast(words[k]);
}
__global__ void debug_accept_kernel(uint64_t n, const float* dE, const uint32_t* words, uint8_t* out) {
  const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  out[k] = metropolis_accept(dE[k], words[k]) ? 1 : 0;
}
// the decision routine of the fused kernels (one FFMA on the hardware logarithm + guard band)
__global__ void debug_accept_fma_kernel(uint64_t n, const float* dE, const uint32_t* words, uint8_t* out) {
  const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  out[k] = metropolis_accept_fma(dE[k], words[k]) ? 1 : 0;
}
template <bool POW2>
__global__ void debug_cell_kernel(Grid g, uint64_t n, const float* x, const float* y, const float* z, uint32_t* out) {
  const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) out[k] = cell_of<POW2>(g, x[k], y[k], z[k]);
}

// Throughput of the density increments on their own (soma_debug_red_throughput): every thread issues `per_thread`
// increments.  mode 0: red.global at uniformly random counters; mode 1: red.global with the locality of the sorted
// melt (a warp's 32 lanes fall into a window of 2048 counters that moves along with the warp index); mode 2:
// red.shared at random counters of a 32 KB window.
__global__ void __launch_bounds__(256)
debug_red_kernel(uint32_t* __restrict__ counters, uint32_t n_counters, uint32_t per_thread, int mode) {
  __shared__ uint32_t win[8192];
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (mode == 2) {
    for (uint32_t k = threadIdx.x; k < 8192u; k += blockDim.x) win[k] = 0u;
    __syncthreads();
  }
  uint32_t h = tid * 2654435761u + 12345u;
  const uint32_t base = (uint32_t)(((uint64_t)(tid >> 5) * 613u) % n_counters);
  for (uint32_t k = 0; k < per_thread; ++k) {
    h = h * 1664525u + 1013904223u;
    const uint32_t r = h >> 8;
    if (mode == 0) atomicAdd(counters + r % n_counters, 1u);
    else if (mode == 1) atomicAdd(counters + (base + (r & 2047u)) % n_counters, 1u);
    else atomicAdd(win + (r & 8191u), 1u);
  }
  if (mode == 2) {
    __syncthreads();
    if (threadIdx.x == 0 && win[h & 8191u] == 0xffffffffu) counters[0] = 1u;     // keeps the window alive
  }
}

// The same probe for a window that is spread over the shared memories of a thread-block cluster (distributed shared
// memory): every CTA of the cluster holds 8192 words (32 KB), the window is cluster-size x 8192 words, and a thread
// reaches word w of CTA r through mapa + red.shared::cluster / ld.shared::cluster.  gather = 0: increments at uniformly
// random words of the cluster's window ((size-1)/size of them land in another SM's memory); gather = 1: loads with the
// locality of the sorted melt (the 32 lanes of a warp fall into 2048 consecutive words, i.e. into one or two CTAs'
// memories).  This is the data flow a cluster-windowed step kernel would have; the probe says what it could cost at best.
__global__ void __launch_bounds__(256)
debug_cluster_kernel(uint32_t* __restrict__ sink, uint32_t per_thread, int gather) {
  __shared__ uint32_t win[8192];
  uint32_t csize;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(csize));
  for (uint32_t k = threadIdx.x; k < 8192u; k += blockDim.x) win[k] = gather ? k : 0u;
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
  const uint32_t local = (uint32_t)__cvta_generic_to_shared(win);
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t total = csize * 8192u;                       // cluster sizes are powers of two
  uint32_t h = tid * 2654435761u + 12345u;
  const uint32_t base = ((tid >> 5) * 613u) & (total - 1u);
  uint32_t acc = 0;
  for (uint32_t k = 0; k < per_thread; ++k) {
    h = h * 1664525u + 1013904223u;
    const uint32_t r = h >> 8;
    const uint32_t idx = gather ? (base + (r & 2047u)) & (total - 1u) : r & (total - 1u);
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local + ((idx & 8191u) << 2)), "r"(idx >> 13));
    if (gather) {
      uint32_t v;
      asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(remote));
      acc += v;
    } else {
      asm volatile("red.relaxed.cluster.shared::cluster.add.u32 [%0], %1;" ::"r"(remote), "r"(1u) : "memory");
    }
  }
  // no CTA may leave while another one still reaches into its shared memory
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
  if (threadIdx.x == 0 && (acc == 0xdeadbeefu || win[h & 8191u] == 0xffffffffu)) sink[0] = 1u;   // keeps loads and window alive
}

}  // namespace soma
