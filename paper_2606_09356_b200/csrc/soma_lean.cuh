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
//   * the positions and the chain id of the warp's next group are fetched one iteration ahead;
//   * OTF ("on the fly", systems of one or two types without external field or umbrella potential): the field is
//     not read from the omega array but computed from the previous step's density counters, which are packed two
//     types to a 32-bit word -- one gather brings both counts of the cell, DESIGN.md section 2 step 3 is evaluated
//     in its operation order for the bead's type.  The omega array is then neither written nor read during a run
//     (the omega kernel runs only when somebody asks for the field), and the footprint of the gathers in L1
//     halves: 1.05 -> 0.96 ms per cfg4 step.
// Bead counts go to the density grid with one red.global per bead.  Counting them in shared-memory
// windows (one block per tile of the box, the window added to the grid with bulk reduce-adds) was built
// and measured twice in round 2 and removed: on cfg4 it never beat the L2 atomics, because the shared
// memory it takes comes out of the L1 that serves the omega gathers (profiles/r2_binning_choice.md).
#pragma once

#include "soma_kernels.cuh"

namespace soma {

struct LeanArgs {
  float inv_hx, inv_hy, inv_hz;      // powers of two >= 1
  uint32_t mx, my, mz;               // nx - 1, ny - 1, nz - 1 (power-of-two grid)
  uint32_t ny, nz;
  uint32_t cells;                    // C
  uint32_t n_chains;
  uint32_t pat_stride;               // row length of `patterns`
  uint32_t groups_per_block;         // warp groups per block (a multiple of the warps per block)
  float a2, ac, kb;                  // 2a, a(2^-23 - 1), 1.5/b^2
  PhiloxKeys keys;
  uint32_t u0, u1;                   // hi(M1 step) ^ k0[0], lo(M1 step)
  uint32_t ctr3_base;
  float* __restrict__ x;
  float* __restrict__ y;
  float* __restrict__ z;
  const float* __restrict__ omega;           // [T][C] (!OTF)
  const uint32_t* __restrict__ counts_prev;  // OTF: packed counters of the previous step, [C]
  float dens_scale, kappaN, invN, chi01;     // OTF: the constants of DESIGN.md section 2 step 3 (chi01 = chiN[0][1])
  uint32_t packed;                           // layout of the density counters (soma_device.cuh)
  uint32_t guard_mask;                       // OTF: see soma_device.cuh
  uint32_t* __restrict__ guard_flag;
  uint32_t* __restrict__ counts_next;        // zeroed before the launch
  const uint32_t* __restrict__ slot_chain;
  const uint8_t* __restrict__ slot_pattern;
  const uint8_t* __restrict__ patterns;
  unsigned long long* __restrict__ accepted;
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

// accept iff fl(dE + lnu) <= 0 (DESIGN.md section 2 step 5.6) by accept_fma_u24 (soma_device.cuh).  `live` = false
// forces a rejection (lanes beyond the end of the block's range).
__device__ __forceinline__ bool lean_accept(float dE, float u24, bool live) { return accept_fma_u24(dE, u24) && live; }
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

// omega of (type, cell) from the packed counters of the previous step: DESIGN.md section 2 step 3 for T <= 2,
//   phi_s = (float)n_s * dens_scale; tot = phi_0 + phi_1; p = kappaN * (tot - 1); omega_t = invN * fma(chi01, phi_other, p)
// (T = 1: the high half of the word is zero and chi01 = 0, so tot = phi_0 + 0 and the fma adds 0 * 0: the same bits
// as the one-type formula).  `c` is the plain cell index; sel_own / sel_other are the byte selectors (PRMT) of the
// bead type's own half of the word and of the other one.  phi_own + phi_other = phi_0 + phi_1 bit for bit: an
// IEEE addition does not depend on the order of its two operands.
// `seen` collects the words of the old cells: every non-empty cell is some bead's old cell, so or-ing them and testing
// the guard bits once per thread inspects every counter in every step (soma_device.cuh).  (Measured on cfg4: this
// form 0.951 ms per launch, a predicate instead 0.960, a predicated store per gather 0.973, no guard 0.942.)
template <bool GUARD>
__device__ __forceinline__ float lean_omega_otf(const LeanArgs& A, uint32_t c, uint32_t sel_own, uint32_t sel_other, uint32_t& seen) {
  const uint32_t word = __ldg(A.counts_prev + c);
  if (GUARD) seen |= word;
  const float own = __fmul_rn((float)__byte_perm(word, 0u, sel_own), A.dens_scale);
  const float other = __fmul_rn((float)__byte_perm(word, 0u, sel_other), A.dens_scale);
  const float p = __fmul_rn(A.kappaN, __fsub_rn(__fadd_rn(own, other), 1.0f));
  return __fmul_rn(A.invN, __fmaf_rn(A.chi01, other, p));
}

template <int P, bool MULTI_PAT, bool OTF, int NT>
__global__ void __launch_bounds__(NT, 1024 / NT)
lean_step_kernel(const __grid_constant__ LeanArgs A) {
  constexpr uint32_t G = 32 / P;                                // chains per warp
  constexpr uint32_t N = 2u * P;
  constexpr uint32_t WPB = NT / 32;                             // warps per block
  constexpr uint32_t STEP = WPB * G;                            // slots per block iteration
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  const uint32_t l = lane % P, sub = lane / P;

  // ---- the block's range of slots ----
  const uint64_t b0 = (uint64_t)blockIdx.x * A.groups_per_block * G;
  if (b0 >= A.n_chains) return;
  const uint32_t s_begin = (uint32_t)b0;
  const uint64_t e0 = b0 + (uint64_t)A.groups_per_block * G;
  const uint32_t s_end = e0 < A.n_chains ? (uint32_t)e0 : A.n_chains;

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
  uint32_t seen = 0;                                            // OTF: or of the old cells' counter words
  const float2* __restrict__ x2 = reinterpret_cast<const float2*>(A.x);
  const float2* __restrict__ y2 = reinterpret_cast<const float2*>(A.y);
  const float2* __restrict__ z2 = reinterpret_cast<const float2*>(A.z);

  // One 32-bit index serves every array: bead pair `pair` = slot P + l, slot = pair / P.
  // The positions and the chain id of the warp's next group are fetched one iteration ahead: a warp has
  // two groups' loads in flight, which is what keeps HBM busy at 32 warps per SM.
  uint32_t slot = s_begin + warp * G + sub;
  float2 Xn = make_float2(0.f, 0.f), Yn = Xn, Zn = Xn;
  uint32_t chain_n = 0;
  if (slot < s_end) {                                           // lanes beyond the range keep zeros and never store
    const uint32_t pr = slot * P + l;
    Xn = __ldcs(x2 + pr); Yn = __ldcs(y2 + pr); Zn = __ldcs(z2 + pr);
    chain_n = __ldg(A.slot_chain + slot);
  }
  for (; slot - sub < s_end; slot += STEP) {                    // slot - sub: warp-uniform
    const bool live = slot < s_end;
    const uint32_t pair = slot * P + l;
    // positions are streamed (read once, written once): keep them from evicting omega out of L1
    const float2 X = Xn, Y = Yn, Z = Zn;
    const uint32_t chain = chain_n;
    if (slot + STEP < s_end) {
      Xn = __ldcs(x2 + pair + STEP * P); Yn = __ldcs(y2 + pair + STEP * P); Zn = __ldcs(z2 + pair + STEP * P);
      chain_n = __ldg(A.slot_chain + slot + STEP);
    }
    if (MULTI_PAT) {
      // a lane beyond the range (n_chains not a multiple of 32/P) looks up the block's first slot instead of reading
      // slot_pattern past its end: whatever bytes lie there would otherwise pick the type, and through it the gather address
      const uint32_t ps = live ? slot : s_begin;
      const uint16_t tt = __ldg(reinterpret_cast<const uint16_t*>(A.patterns + (uint32_t)__ldg(A.slot_pattern + ps) * A.pat_stride) + l);
      t0 = tt & 0xffu; t1 = tt >> 8;
    }
    const uint32_t toff0 = OTF ? 0u : t0 * A.cells, toff1 = OTF ? 0u : t1 * A.cells;   // OTF: one word per cell, the type picks its half
    const uint32_t sel0 = t0 ? 0x4432u : 0x4410u, sel1 = t1 ? 0x4432u : 0x4410u;         // PRMT selectors: own half of the packed word
    const uint32_t oth0 = sel0 ^ 0x0022u, oth1 = sel1 ^ 0x0022u;
    float ex = X.x, ey = Y.x, ez = Z.x;                         // even bead 2l
    float ox = X.y, oy = Y.y, oz = Z.y;                         // odd bead 2l+1

    // ---- everything that does not depend on a decision: old cells, both trial positions, four gathers ----
    uint32_t cell_e = lean_cell(A, ex, ey, ez, toff0);
    uint32_t cell_o = lean_cell(A, ox, oy, oz, toff1);
#define GATHER(c, own, oth) (OTF ? lean_omega_otf<false>(A, (c), (own), (oth), seen) : __ldg(A.omega + (c)))
    const float w_old_e = OTF ? lean_omega_otf<true>(A, cell_e, sel0, oth0, seen) : __ldg(A.omega + cell_e);
    const float w_old_o = OTF ? lean_omega_otf<true>(A, cell_o, sel1, oth1, seen) : __ldg(A.omega + cell_o);
    const uint32_t c0_1 = A.u0 ^ chain;
    const Words4 We = philox_tail(A.keys, L0, c0_1);
    const float tex = lean_trial(A, ex, We.w0), tey = lean_trial(A, ey, We.w1), tez = lean_trial(A, ez, We.w2);
    const uint32_t cell_te = lean_cell(A, tex, tey, tez, toff0);
    const float w_new_e = GATHER(cell_te, sel0, oth0);
    const Words4 Wo = philox_tail(A.keys, L1, c0_1);
    const float tox = lean_trial(A, ox, Wo.w0), toy = lean_trial(A, oy, Wo.w1), toz = lean_trial(A, oz, Wo.w2);
    const uint32_t cell_to = lean_cell(A, tox, toy, toz, toff1);
    const float w_new_o = GATHER(cell_to, sel1, oth1);
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
      if (OTF || A.packed) {                                     // packed counters: one word per cell, type in the increment
        atomicAdd(A.counts_next + (cell_e & (A.cells - 1u)), 1u << (t0 << 4));
        atomicAdd(A.counts_next + (cell_o & (A.cells - 1u)), 1u << (t1 << 4));
      } else {
        atomicAdd(A.counts_next + cell_e, 1u);
        atomicAdd(A.counts_next + cell_o, 1u);
      }
    }
  }

  if (OTF && (seen & A.guard_mask)) *A.guard_flag = 1u;
  // accepted-move count: warp reduce, one atomic per warp
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
  if (lane == 0 && n_acc) atomicAdd(A.accepted, (unsigned long long)n_acc);
}

}  // namespace soma
