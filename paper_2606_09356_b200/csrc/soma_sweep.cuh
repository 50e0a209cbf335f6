// soma_sweep.cuh -- the swept-window kernel of the SCMF Monte-Carlo step (rows a1+a2+a3+a5), sm_100a.
//
// Same data flow as the column sweep of soma_tile.cuh (omega slabs TMA-loaded into a shared-memory
// ring ahead of the sweep, densities counted with RED.shared and TMA-reduce-added into the
// ghost-padded global grid behind it) with the bookkeeping taken off the consumer warps' issue
// slots (ncu, profiles/r1_ncu_cfg4_tile_v3.txt: 40 % of the old kernel's instructions were
// bookkeeping, and the kernel is issue-bound):
//   * chains of a unit are taken in slot order, G per warp iteration, regardless of slice
//     boundaries; each chain carries its slice index (slot_k), so there is no slice cursor;
//   * every consumer warp publishes `prog` = the first slice it may still touch, as one plain
//     shared-memory word; the producer retires (TMA-reduce-adds, zeroes, reloads) every slab below
//     the minimum of `prog`, recycling one batch behind the flush so that the wait for the
//     reduce-add's reads of shared memory does not stall the ring.  Consumers take the omega slabs
//     in order from the `full` mbarriers, with slot and phase kept in registers;
//   * an iteration whose beads all lie at least one cell inside their window runs a branch-free body
//     with no range tests (a bead moves by less than one cell per step, so neither the trial nor the
//     final position can leave the window); the near-threshold Metropolis decisions (|margin| <=
//     kLnBand, ~6e-5 of the moves) are only flagged there.  Iterations with a bead near a window
//     face, or with a flagged decision, are (re)done by the checked body -- the per-move tests and
//     global-memory fallbacks of soma_tile.cuh -- from the unchanged input registers.
// The results are those of DESIGN.md section 2 bit for bit on either body.
#pragma once

#include "soma_tile.cuh"

namespace soma {

// The consumers' progress words.  They are read and written with plain (volatile) shared-memory
// accesses: all shared-memory instructions of an SM go through one in-order pipe, so a store issued
// after a warp's RED.shared is seen after them; a release
// store would cost a MEMBAR.ALL.CTA, which also waits for the warp's outstanding global prefetches.
__device__ __forceinline__ uint32_t ld_acquire_shared(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.volatile.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_shared(uint32_t addr, uint32_t v) {
  asm volatile("st.volatile.shared::cta.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
// layout of the auxiliary shared-memory block (kSweepAuxBytes)
constexpr uint32_t kAuxProg = 320;      // u32[32]: per consumer warp, first slice it may still touch
constexpr uint32_t kAuxPtab = 512;      // float2[kMaxSlices]: ring slot of a slice's first slab, and that - R + 1

// shared address of omega at the cell of (x, y, z); the position is known to lie inside the window
template <bool FASTH>
__device__ __forceinline__ uint32_t win_addr_inside(const WinGeo& g, float x, float y, float z, float offx, float offy,
                                                    float offz, float p_f, float seam_f, float base_t_d) {
  float fx, fy, fz;
  if (FASTH) {
    fx = __fmaf_rd(x, g.inv_hx, offx); fy = __fmaf_rd(y, g.inv_hy, offy); fz = __fmaf_rd(z, g.inv_hz, offz);
  } else {
    fx = __fadd_rd(__fmul_rn(x, g.inv_hx), offx); fy = __fadd_rd(__fmul_rn(y, g.inv_hy), offy); fz = __fadd_rd(__fmul_rn(z, g.inv_hz), offz);
  }
  const float rx = __fadd_rn(fx, -kFloorMagic), ry = __fadd_rn(fy, -kFloorMagic), rz = __fadd_rn(fz, -kFloorMagic);
  const float slot = __fmaf_rn(fadd_sat(rx, seam_f), g.neg_R, __fadd_rn(rx, p_f));
  return __float_as_uint(__fmaf_rn(slot, g.slab_stride_d, __fmaf_rn(ry, g.sy_d, __fmaf_rn(rz, g.four_d, base_t_d))));
}

// the same for a bead's starting position, with the test "at least one cell inside the window"
template <bool FASTH>
__device__ __forceinline__ bool win_addr_margin(const WinGeo& g, float x, float y, float z, float offx, float offy,
                                                float offz, float p_f, float seam_f, float base_t_d,
                                                float wxm_f, float eym_f, float ezm_f, uint32_t& addr) {
  float fx, fy, fz;
  if (FASTH) {
    fx = __fmaf_rd(x, g.inv_hx, offx); fy = __fmaf_rd(y, g.inv_hy, offy); fz = __fmaf_rd(z, g.inv_hz, offz);
  } else {
    fx = __fadd_rd(__fmul_rn(x, g.inv_hx), offx); fy = __fadd_rd(__fmul_rn(y, g.inv_hy), offy); fz = __fadd_rd(__fmul_rn(z, g.inv_hz), offz);
  }
  const float rx = __fadd_rn(fx, -kFloorMagic), ry = __fadd_rn(fy, -kFloorMagic), rz = __fadd_rn(fz, -kFloorMagic);
  const float mx = __fadd_rn(fx, -(kFloorMagic + 1.0f)), my = __fadd_rn(fy, -(kFloorMagic + 1.0f)), mz = __fadd_rn(fz, -(kFloorMagic + 1.0f));
  const float slot = __fmaf_rn(fadd_sat(rx, seam_f), g.neg_R, __fadd_rn(rx, p_f));
  addr = __float_as_uint(__fmaf_rn(slot, g.slab_stride_d, __fmaf_rn(ry, g.sy_d, __fmaf_rn(rz, g.four_d, base_t_d))));
  // r - 1 in [0, extent - 2): one unsigned compare of bit patterns per axis (negative floats have the sign bit set)
  return (__float_as_uint(mx) < __float_as_uint(wxm_f)) & (__float_as_uint(my) < __float_as_uint(eym_f)) &
         (__float_as_uint(mz) < __float_as_uint(ezm_f));
}

// One trial move of the branch-free body.  `unc` collects "decision too close to call here".
template <bool FAST, bool EVEN>
__device__ __forceinline__ bool sweep_move(const PhiloxKeys& K, const LaneCtx& C, const PhiloxLane& L, uint32_t c0_1,
                                           float offx, float offy, float offz, float p_f, float seam_f, float base_t_d,
                                           float& rx, float& ry, float& rz, uint32_t& addr,
                                           float lx, float ly, float lz, float& q_l,
                                           float qx, float qy, float qz, float& q_r, float h, bool& unc) {
  const Words4 w = philox_tail(K, L, c0_1);
  const float tx = trial_axis<FAST>(C, rx, w.w0);
  const float ty = trial_axis<FAST>(C, ry, w.w1);
  const float tz = trial_axis<FAST>(C, rz, w.w2);
  const float ql_new = bond_sq(tx, ty, tz, lx, ly, lz);
  const float qr_new = bond_sq(tx, ty, tz, qx, qy, qz);
  const float dql = __fsub_rn(ql_new, q_l), dqr = __fsub_rn(qr_new, q_r);
  const float dq = EVEN ? __fmaf_rn(h, dql, dqr) : __fmaf_rn(h, dqr, dql);
  const uint32_t addr_new = win_addr_inside<FAST>(C.g, tx, ty, tz, offx, offy, offz, p_f, seam_f, base_t_d);
  const float dE = __fmaf_rn(C.kb, dq, __fsub_rn(lds_f32(addr_new), lds_f32(addr)));
  const float m = __fmaf_rn(lg2_approx(umap_int(w.w3)), kLn2, dE);
  const bool acc = m < kLnT - kLnBand;
  unc |= (!acc) & (m <= kLnT + kLnBand);
  if (acc) { rx = tx; ry = ty; rz = tz; addr = addr_new; q_l = ql_new; q_r = qr_new; }
  return acc;
}

// ---------------------------------------------------------------------------------------------
// The kernel.  Work unit, column, segment, slab, slice, window and ring as in soma_tile.cuh.
// Warp 0 is the producer, the other NT/32 - 1 warps are consumers; see the file header.
// ---------------------------------------------------------------------------------------------
template <int P, bool MULTI_PAT, int NT, bool FAST>
__global__ void __launch_bounds__(NT, 1)
sweep_step_kernel(const __grid_constant__ TileArgs A, const __grid_constant__ CUtensorMap tm_omega,
                  const __grid_constant__ CUtensorMap tm_counts) {
  constexpr int G = 32 / P;
  constexpr uint32_t NWC = NT / 32 - 1;                                       // consumer warps
  constexpr uint32_t N = 2u * P;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* omega_ring = smem_raw;
  unsigned char* counts_ring = smem_raw + A.counts_offset;
  unsigned char* aux = smem_raw + A.aux_offset;
  uint64_t* full = reinterpret_cast<uint64_t*>(aux);                          // [kMaxRing]
  const uint32_t prog_addr = smem_u32(aux + kAuxProg);
  float2* ptab = reinterpret_cast<float2*>(aux + kAuxPtab);
  const StepArgs& S = A.S;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t l = lane % P, sub = lane / P;
  const uint32_t R = A.R, K = A.K, stride = A.slab_stride;
  const uint32_t A_tot = A.Lseg + 2u * A.hx;                                  // slabs of a unit
  unsigned n_acc = 0;

  for (uint32_t k = tid; k < K; k += NT) {
    const uint32_t p = (k * A.slice) % R;
    ptab[k] = make_float2((float)p, (float)((int)p - (int)R + 1));
  }

  for (uint32_t unit = blockIdx.x; unit < A.n_units; unit += gridDim.x) {
    const uint32_t u_begin = __ldg(A.bin_start + 2u * K * unit), u_end = __ldg(A.bin_start + 2u * K * (unit + 1u));
    const uint32_t n_u = u_end - u_begin;
    if (n_u == 0) continue;                             // uniform over the CTA; nothing to bin
    const uint32_t F = (n_u + G - 1) / G;               // warp iterations of the unit
    const uint32_t sg = unit % A.nseg, col = unit / A.nseg;
    const int x0 = (int)(sg * A.Lseg), y0 = (int)((col / A.mtz) * A.cy), z0 = (int)((col % A.mtz) * A.cz);   // padded coordinates of slab 0
    __syncthreads();                                    // the previous unit is finished, its flushes have read the ring
    for (uint32_t k = tid; k < R * stride / 16u; k += NT) reinterpret_cast<uint4*>(counts_ring)[k] = make_uint4(0u, 0u, 0u, 0u);
    if (tid == 0)
      for (uint32_t r = 0; r < R; ++r) { mbar_inval(&full[r]); mbar_init(&full[r], 1); }
    if (tid >= 64 && tid < 96) reinterpret_cast<volatile uint32_t*>(aux + kAuxProg)[tid - 64] = (tid - 64 < NWC && tid - 64 < F) ? 0u : K;
    __syncthreads();

    if (warp == 0) {
      // ---------------- producer ----------------
      const uint32_t loaded = R < A_tot ? R : A_tot;    // the ring starts with the unit's first slabs
      if (lane == 0)
        for (uint32_t a = 0; a < loaded; ++a) {
          mbar_expect_tx(&full[a], A.slab_bytes);
          tma_load_4d(omega_ring + a * stride, &tm_omega, &full[a], z0, y0, x0 + (int)a, 0);
        }
      // Slabs below `fl` have been handed to the TMA reduce-add (one bulk group per batch); slabs
      // below `rc` have also been recycled (counters zeroed, omega of slab + R loading into the
      // slot).  Recycling runs one batch behind flushing, so the wait for the reduce-add's reads of
      // shared memory overlaps the next batch instead of stalling the ring.
      uint32_t fl = 0, fl_slot = 0, rc = 0, rc_slot = 0;
      auto recycle = [&](uint32_t upto) {               // uniform over the warp
        uint32_t s = rc_slot;
        for (uint32_t a = rc; a < upto; ++a) {
          if (a + R < A_tot) {
            uint4* c = reinterpret_cast<uint4*>(counts_ring + s * stride);
            for (uint32_t k = lane; k < A.slab_bytes / 16u; k += 32u) c[k] = make_uint4(0u, 0u, 0u, 0u);
          }
          if (++s == R) s = 0;
        }
        __syncwarp();
        if (lane == 0) {
          s = rc_slot;
          for (uint32_t a = rc; a < upto; ++a) {
            if (a + R < A_tot) {
              mbar_expect_tx(&full[s], A.slab_bytes);   // the zeroes above are visible to whoever sees this phase complete
              tma_load_4d(omega_ring + s * stride, &tm_omega, &full[s], z0, y0, x0 + (int)(a + R), 0);
            }
            if (++s == R) s = 0;
          }
        }
        rc_slot = (rc_slot + (upto - rc)) % R;
        rc = upto;
      };
      while (fl < A_tot) {
        const uint32_t pv = lane < NWC ? ld_acquire_shared(prog_addr + 4u * lane) : K;
        const uint32_t m = __reduce_min_sync(0xffffffffu, pv);
        __syncwarp();
        const uint32_t target = m >= K ? A_tot : m * A.slice;       // slabs below it are touched by no one any more
        if (fl < target) {
          if (lane == 0) {
            fence_proxy_async();
            uint32_t s = fl_slot;
            for (uint32_t a = fl; a < target; ++a) {
              tma_reduce_add_4d(&tm_counts, counts_ring + s * stride, z0, y0, x0 + (int)a, 0);
              if (++s == R) s = 0;
            }
            bulk_commit();
            asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");      // every batch but the one just committed
          }
          __syncwarp();
          recycle(fl);
          fl_slot = (fl_slot + (target - fl)) % R;
          fl = target;
        } else if (rc < fl) {
          if (lane == 0) bulk_wait_read0();
          __syncwarp();
          recycle(fl);
        } else {
          __nanosleep(64);
        }
      }
      if (lane == 0) bulk_wait_read0();
    } else {
      // ---------------- consumers ----------------
      LaneCtx C;
      C.g.inv_hx = S.grid.inv_hx; C.g.inv_hy = S.grid.inv_hy; C.g.inv_hz = S.grid.inv_hz;
      C.g.wx_f = (float)A.wx; C.g.ey_f = (float)A.ey; C.g.ez_f = (float)A.ez;
      C.g.neg_R = -(float)R;
      C.g.slab_stride_d = __uint_as_float(stride); C.g.sy_d = __uint_as_float(A.ez * 4u); C.g.four_d = __uint_as_float(4u);
      C.a = S.a; C.a2 = A.a2; C.ac = A.ac; C.kb = S.kb;
      const float wxm_f = (float)(A.wx - 2u), eym_f = (float)(A.ey - 2u), ezm_f = (float)(A.ez - 2u);
      const float hl = l > 0 ? 1.0f : 0.0f, hr = l + 1 < P ? 1.0f : 0.0f;
      const PhiloxLane L0 = philox_lane(S.keys, A.philox_u1, 2u * l, S.ctr3_base);
      const PhiloxLane L1 = philox_lane(S.keys, A.philox_u1, 2u * l + 1u, S.ctr3_base | 1u);
      const uint32_t omega_base = smem_u32(omega_ring);
      const uint32_t type_stride = A.ey * A.ez * 4u;
      uint32_t type0 = 0, type1 = 0;
      if (!MULTI_PAT) {
        const uint16_t tt = *reinterpret_cast<const uint16_t*>(S.patterns + 2u * l);
        type0 = tt & 0xffu; type1 = tt >> 8;
      }
      const uint32_t wc = warp - 1u;
      uint32_t ready_c = 0, rslot = 0, rpar = 0, k_cur = 0;    // slabs [0, ready_c) have landed; slot and phase of slab ready_c
      // The chain's window offsets and slice index are fetched one iteration ahead (5 registers); its
      // positions are loaded at the top of the iteration, behind an L2 prefetch issued one iteration
      // earlier, and are first needed after the ring synchronisation.
      float4 Mn;
      uint32_t slot_n = 0, k_n = 0;
      bool live_n = false;
      auto fetch = [&](uint32_t f) {
        const uint32_t rel = f * G + sub;
        live_n = rel < n_u;
        slot_n = u_begin + (live_n ? rel : n_u - 1u);                         // dead lanes shadow the unit's last chain
        Mn = __ldg(A.slot_meta + slot_n);
        k_n = __ldg(A.slot_k + slot_n);
        if (l % 4u == 0) {                                                     // one prefetch per 32-byte sector
          const uint64_t j = (uint64_t)slot_n * N + 2u * l;
          asm volatile("prefetch.global.L2 [%0];" ::"l"(S.x + j));
          asm volatile("prefetch.global.L2 [%0];" ::"l"(S.y + j));
          asm volatile("prefetch.global.L2 [%0];" ::"l"(S.z + j));
        }
      };
      if (wc < F) fetch(wc);
      for (uint32_t f = wc; f < F; f += NWC) {
        const float4 M = Mn;
        const uint32_t slot = slot_n, kk = k_n;
        const bool live = live_n;
        const uint64_t j = (uint64_t)slot * N + 2u * l;
        const float2 X = *reinterpret_cast<const float2*>(S.x + j);
        const float2 Y = *reinterpret_cast<const float2*>(S.y + j);
        const float2 Z = *reinterpret_cast<const float2*>(S.z + j);
        if (f + NWC < F) fetch(f + NWC);
        // ring synchronisation: slots are sorted by slice, so lane 0 holds the smallest and lane 31 the largest
        const uint32_t k_lo = __shfl_sync(0xffffffffu, kk, 0), k_hi = __shfl_sync(0xffffffffu, kk, 31);
        if (k_lo != k_cur) {
          __syncwarp();                                 // this warp's RED.shared of the slices it leaves come first
          if (lane == 0) st_release_shared(prog_addr + 4u * wc, k_lo);
          k_cur = k_lo;
        }
        // The warp's chains span slices k_lo..k_hi; their windows are all resident only if that span
        // fits in the ring.  If not (sparse units, rings of one window), the chains above k_lo go
        // through the global-memory fallbacks of the checked body and touch no shared memory.
        const bool span_fits = (k_hi - k_lo) * A.slice + A.wx <= R;
        const bool force_out = !span_fits && kk != k_lo;
        uint32_t need = (span_fits ? k_hi : k_lo) * A.slice + A.wx;
        if (need > A_tot) need = A_tot;
        while (ready_c < need) {                        // slabs land in any order; take them in order
          mbar_wait(&full[rslot], rpar);
          ++ready_c;
          if (++rslot == R) { rslot = 0; rpar ^= 1u; }
        }
        const float2 pt = ptab[kk];
        const float p_f = pt.x, seam_f = pt.y;

        const uint32_t c0_1 = A.philox_u0 ^ __float_as_uint(M.w);
        if (MULTI_PAT) {
          const uint16_t tt = *reinterpret_cast<const uint16_t*>(S.patterns + (uint32_t)S.slot_pattern[slot] * N + 2u * l);
          type0 = tt & 0xffu; type1 = tt >> 8;
        }
        const float base0 = __uint_as_float(omega_base + type0 * type_stride), base1 = __uint_as_float(omega_base + type1 * type_stride);
        float ex, ey, ez, ox, oy, oz;                   // even bead 2l, odd bead 2l+1
        uint32_t addr_e, addr_o;
        bool in_e = true, in_o = true;
        unsigned na = 0;
        // ---- branch-free body ----
        ex = X.x; ey = Y.x; ez = Z.x; ox = X.y; oy = Y.y; oz = Z.y;
        const bool ok_e = win_addr_margin<FAST>(C.g, ex, ey, ez, M.x, M.y, M.z, p_f, seam_f, base0, wxm_f, eym_f, ezm_f, addr_e);
        const bool ok_o = win_addr_margin<FAST>(C.g, ox, oy, oz, M.x, M.y, M.z, p_f, seam_f, base1, wxm_f, eym_f, ezm_f, addr_o);
        bool redo = !__all_sync(0xffffffffu, ok_e && ok_o) || !span_fits;
        if (!redo) {
          const float lx = __shfl_up_sync(0xffffffffu, ox, 1, P);
          const float ly = __shfl_up_sync(0xffffffffu, oy, 1, P);
          const float lz = __shfl_up_sync(0xffffffffu, oz, 1, P);
          float qA = bond_sq(ex, ey, ez, ox, oy, oz);   // bond (even, odd) of this lane
          float qB = bond_sq(ex, ey, ez, lx, ly, lz);   // bond (odd of lane l-1, even)
          bool unc = false;
          const bool acc0 = sweep_move<FAST, true>(S.keys, C, L0, c0_1, M.x, M.y, M.z, p_f, seam_f, base0,
                                                   ex, ey, ez, addr_e, lx, ly, lz, qB, ox, oy, oz, qA, hl, unc);
          const float rx = __shfl_down_sync(0xffffffffu, ex, 1, P);
          const float ry = __shfl_down_sync(0xffffffffu, ey, 1, P);
          const float rz = __shfl_down_sync(0xffffffffu, ez, 1, P);
          float qR = __shfl_down_sync(0xffffffffu, qB, 1, P);
          const bool acc1 = sweep_move<FAST, false>(S.keys, C, L1, c0_1, M.x, M.y, M.z, p_f, seam_f, base1,
                                                    ox, oy, oz, addr_o, ex, ey, ez, qA, rx, ry, rz, qR, hr, unc);
          na = (acc0 ? 1u : 0u) + (acc1 ? 1u : 0u);
          redo = __any_sync(0xffffffffu, unc);
        }
        if (redo) {
          // ---- checked body: per-move window tests, global-memory fallbacks, exact logarithm near the threshold ----
          ex = X.x; ey = Y.x; ez = Z.x; ox = X.y; oy = Y.y; oz = Z.y;
          in_e = win_addr<FAST>(C.g, ex, ey, ez, M.x, M.y, M.z, p_f, seam_f, base0, addr_e) && !force_out;
          in_o = win_addr<FAST>(C.g, ox, oy, oz, M.x, M.y, M.z, p_f, seam_f, base1, addr_o) && !force_out;
          const float lx = __shfl_up_sync(0xffffffffu, ox, 1, P);
          const float ly = __shfl_up_sync(0xffffffffu, oy, 1, P);
          const float lz = __shfl_up_sync(0xffffffffu, oz, 1, P);
          float qA = bond_sq(ex, ey, ez, ox, oy, oz);
          float qB = bond_sq(ex, ey, ez, lx, ly, lz);
          const bool acc0 = tile_move<FAST, true>(A, C, L0, c0_1, M.x, M.y, M.z, p_f, seam_f, base0, S.omega + (size_t)type0 * S.cells,
                                                  ex, ey, ez, addr_e, in_e, lx, ly, lz, qB, ox, oy, oz, qA, hl, force_out);
          const float rx = __shfl_down_sync(0xffffffffu, ex, 1, P);
          const float ry = __shfl_down_sync(0xffffffffu, ey, 1, P);
          const float rz = __shfl_down_sync(0xffffffffu, ez, 1, P);
          float qR = __shfl_down_sync(0xffffffffu, qB, 1, P);
          const bool acc1 = tile_move<FAST, false>(A, C, L1, c0_1, M.x, M.y, M.z, p_f, seam_f, base1, S.omega + (size_t)type1 * S.cells,
                                                   ox, oy, oz, addr_o, in_o, ex, ey, ez, qA, rx, ry, rz, qR, hr, force_out);
          na = (acc0 ? 1u : 0u) + (acc1 ? 1u : 0u);
        }
        if (live) {
          n_acc += na;
          *reinterpret_cast<float2*>(S.x + j) = make_float2(ex, ox);
          *reinterpret_cast<float2*>(S.y + j) = make_float2(ey, oy);
          *reinterpret_cast<float2*>(S.z + j) = make_float2(ez, oz);
          if (in_e) reds_inc(addr_e + A.counts_offset); else count_outside(A, type0, ex, ey, ez);
          if (in_o) reds_inc(addr_o + A.counts_offset); else count_outside(A, type1, ox, oy, oz);
        }
      }
      __syncwarp();
      if (lane == 0) st_release_shared(prog_addr + 4u * wc, K);
    }
  }
  if (tid == 0) bulk_wait0();
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
  if (lane == 0 && n_acc) atomicAdd(S.accepted, (unsigned long long)n_acc);
}

}  // namespace soma
