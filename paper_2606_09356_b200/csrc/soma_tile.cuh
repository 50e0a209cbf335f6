// soma_tile.cuh -- the tiled kernel of the SCMF Monte-Carlo step (rows a1+a2+a3+a5), sm_100a.
//
// The scattered part of a move -- two omega gathers and one density increment per bead -- costs
// about one L1/L2 transaction per lane when it goes to global memory (measured on B200: 185 G
// red.global/s, 280 G random L2 gathers/s chip-wide, i.e. ~1 ms per step at 134 M beads), but only
// ~0.23 cycles per lane in shared memory (1.2 T LDS or ATOMS per second).  So the kernel works on
// SPATIAL TILES: the chains are kept sorted by the tile that holds their centre of mass, one CTA
// per SM walks over tiles, and for each tile
//   1. TMA-loads the omega sub-box (tile core + halo, all types) from a ghost-padded copy of
//      omega into shared memory (one cp.async.bulk.tensor.4d, completion on an mbarrier),
//   2. runs both half-sweeps for every chain of the tile with the chain in registers (two beads
//      per lane, warp shuffles for the neighbours), reading omega with LDS and counting beads
//      with ATOMS into a shared-memory density tile,
//   3. adds the density tile into a ghost-padded global density grid with ONE TMA reduce-add
//      (cp.reduce.async.bulk.tensor.4d ... .add on u32).  Measured on B200: the reduce faults on
//      negative coordinates and on an innermost coordinate that is not a multiple of 16 bytes, so
//      the periodic wrap is not done by the TMA: every tile box lies inside the padded grid
//      (coordinate = tile index * core, the core's z edge a multiple of 4 cells) and the omega
//      pass folds the ghost layers back onto the periodic grid.
// A bead that has left the tile (chain longer than the halo, or drift since the last sort) falls
// back to the global-memory gather / atomic, so the result never depends on the tiling.
#pragma once

#include <cuda.h>

#include "soma_kernels.cuh"

namespace soma {

// ---- PTX wrappers -----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
__device__ __forceinline__ void tma_reduce_add_4d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
      ::"l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// ---- shared-memory access by 32-bit shared address ---------------------------------------------
__device__ __forceinline__ float lds_f32(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void reds_inc(uint32_t addr) {
  asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}

// ---- window-local cell ---------------------------------------------------------------------------
// A chain group works inside a WINDOW of the grid: wx x ey x ez cells whose omega values and
// density counters sit in shared memory, slab by slab along x (a slab = one x layer, [T][ey][ez]),
// the slabs forming a ring of R slots (slab a of the sweep lives in slot a mod R).
// `off` = kFloorMagic - window origin + the chain's periodic image shift (whole cells, set when the
// chains are sorted), so RD(r inv_h + off) - kFloorMagic is the bead's cell coordinate RELATIVE to
// the window origin as an exact small float, with no periodic wrap left to do.  FAST: inv_h is a
// power of two >= 1, so r inv_h is exact and one FFMA.RD gives the same value as FMUL + FADD.RD.
//
// Everything stays on the FMA pipe: the range test compares float bit patterns (a negative float
// has the sign bit set, so one unsigned compare per axis covers both ends); the ring slot of a bead
// at window-relative x is u - R [u >= R] with u = x + p, p = (slab of the window origin) mod R --
// the window is at most R slabs wide, so it crosses the ring seam at most once, and the indicator
// is a saturating add, sat(x + p - R + 1); and the shared address is assembled by FFMAs on
// DENORMALS: a float with bit pattern n is n 2^-149, so fma(idx, as_float(stride), as_float(base))
// has the bit pattern base + idx*stride as long as that stays below 2^23.
struct WinGeo {
  float inv_hx, inv_hy, inv_hz;
  float wx_f, ey_f, ez_f;       // window extent in cells (as floats: compared as bit patterns)
  float neg_R;                  // -R
  float slab_stride_d, sy_d, four_d;   // denormals whose bit patterns are the byte strides (slot, y, z)
};

__device__ __forceinline__ float fadd_sat(float a, float b) {
  float r;
  asm("add.sat.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
  return r;
}

template <bool FASTH>
__device__ __forceinline__ bool win_addr(const WinGeo& g, float x, float y, float z, float offx, float offy, float offz,
                                         float p_f /* slab of the window origin mod R */, float seam_f /* p - R + 1 */,
                                         float base_t_d, uint32_t& addr) {
  float fx, fy, fz;
  if (FASTH) {
    fx = __fmaf_rd(x, g.inv_hx, offx); fy = __fmaf_rd(y, g.inv_hy, offy); fz = __fmaf_rd(z, g.inv_hz, offz);
  } else {
    fx = __fadd_rd(__fmul_rn(x, g.inv_hx), offx); fy = __fadd_rd(__fmul_rn(y, g.inv_hy), offy); fz = __fadd_rd(__fmul_rn(z, g.inv_hz), offz);
  }
  const float rx = __fadd_rn(fx, -kFloorMagic), ry = __fadd_rn(fy, -kFloorMagic), rz = __fadd_rn(fz, -kFloorMagic);
  const float slot = __fmaf_rn(fadd_sat(rx, seam_f), g.neg_R, __fadd_rn(rx, p_f));
  addr = __float_as_uint(__fmaf_rn(slot, g.slab_stride_d, __fmaf_rn(ry, g.sy_d, __fmaf_rn(rz, g.four_d, base_t_d))));
  return (__float_as_uint(rx) < __float_as_uint(g.wx_f)) & (__float_as_uint(ry) < __float_as_uint(g.ey_f)) &
         (__float_as_uint(rz) < __float_as_uint(g.ez_f));
}

constexpr uint32_t kMaxRing = 32;      // ring slots
constexpr uint32_t kMaxSlices = 128;   // slices per unit
constexpr uint32_t kSweepAuxBytes = 4096;

struct TileArgs {
  StepArgs S;                 // omega = linear field (slow path); counts_next is not used by this kernel
  const float4* __restrict__ slot_meta;     // [n] per slot: floor offsets x, y, z and the chain id (bits)
  const uint16_t* __restrict__ slot_k;      // [n] per slot: slice index of the chain inside its unit (soma_sweep.cuh)
  uint32_t* __restrict__ counts_pad;        // [T][px][py][pz] ghost-padded density grid this step bins into
  const uint32_t* __restrict__ bin_start;   // [2 K n_units + 1]: per unit and slice, compact chains then extended ones
  uint32_t px, py, pz;        // padded dims: padded coordinate q holds cell (q - halo) mod n
  uint32_t T;
  uint32_t ey, ez, wx;        // window extent in cells: wx = slice + 2 hx
  uint32_t cy, cz;            // column core
  uint32_t hx, hy, hz;        // halo
  uint32_t slice, R, K, Lseg; // slice width (cells), ring slots, slices per unit, segment length = K * slice
  uint32_t mtz, nseg, n_units;// columns along z, segments along x, units = columns * segments
  uint32_t slab_bytes;        // T*ey*ez*4: bytes one TMA slab box writes
  uint32_t slab_stride;       // slab_bytes rounded up to 128
  uint32_t counts_offset;     // byte offset of the density ring in dynamic shared memory
  uint32_t aux_offset;        // byte offset of the barriers and slice tables
  uint32_t philox_u0, philox_u1;   // hi(M1 step) ^ k0[0], lo(M1 step)
  float a2, ac;               // FAST: 2a and a (2^-23 - 1)
};

// omega at a bead's cell on the slow path (some lane of the warp has a bead outside the window)
__device__ __noinline__ float omega_outside(const float* __restrict__ omega_t, Grid grid, float x, float y, float z) {
  return __ldg(omega_t + cell_of<true>(grid, x, y, z));
}

// density increment of a bead outside the window: straight into the padded grid, at the image that
// lies `halo` inside it
__device__ __noinline__ void count_outside(const TileArgs& A, uint32_t type, float x, float y, float z) {
  const Grid& G = A.S.grid;
  const uint32_t gx = floor_bits(__fmul_rn(x, G.inv_hx)) & (G.nx - 1u);
  const uint32_t gy = floor_bits(__fmul_rn(y, G.inv_hy)) & (G.ny - 1u);
  const uint32_t gz = floor_bits(__fmul_rn(z, G.inv_hz)) & (G.nz - 1u);
  atomicAdd(A.counts_pad + ((size_t)(type * A.px + gx + A.hx) * A.py + gy + A.hy) * A.pz + gz + A.hz, 1u);
}

// Kernel-constant scalars a move needs.
struct LaneCtx {
  WinGeo g;
  float a, a2, ac, kb;
};

// trial displacement along one axis (DESIGN.md section 2 steps 5.2-5.3): r' = r + a tmap(w)
template <bool FAST>
__device__ __forceinline__ float trial_axis(const LaneCtx& C, float r, uint32_t w) {
  if (FAST) {   // a is a power of two: a tmap(w) = 2a h + a(2^-23 - 1) is exact, one FFMA
    const float h = __fadd_rn(__uint_as_float(0x3f800000u | (w >> 9)), -1.0f);
    return __fadd_rn(r, __fmaf_rn(C.a2, h, C.ac));
  }
  return __fadd_rn(r, __fmul_rn(C.a, tmap(w)));
}

// One Metropolis trial move inside a window.  (rx,ry,rz), addr (shared address of omega at the
// bead's cell), in (bead inside the window) follow the bead.  q_l / q_r: current squared lengths of
// the bonds to the left / right neighbour; on return they hold the lengths after the move.
template <bool FAST, bool EVEN>
__device__ __forceinline__ bool tile_move(const TileArgs& A, const LaneCtx& C, const PhiloxLane& L, uint32_t c0_1,
                                          float offx, float offy, float offz, float p_f, float seam_f, float base_t_d,
                                          const float* __restrict__ omega_t,
                                          float& rx, float& ry, float& rz, uint32_t& addr, bool& in,
                                          float lx, float ly, float lz, float& q_l,
                                          float qx, float qy, float qz, float& q_r, float h, bool force_out = false) {
  const Words4 w = philox_tail(A.S.keys, L, c0_1);
  const float tx = trial_axis<FAST>(C, rx, w.w0);
  const float ty = trial_axis<FAST>(C, ry, w.w1);
  const float tz = trial_axis<FAST>(C, rz, w.w2);
  const float ql_new = bond_sq(tx, ty, tz, lx, ly, lz);
  const float qr_new = bond_sq(tx, ty, tz, qx, qy, qz);
  // dq = dq_left + dq_right (one fp32 add).  An even bead always has its right neighbour and an odd
  // bead its left one; the other may be missing, and then contributes h * (finite) = 0.
  const float dql = __fsub_rn(ql_new, q_l), dqr = __fsub_rn(qr_new, q_r);
  const float dq = EVEN ? __fmaf_rn(h, dql, dqr) : __fmaf_rn(h, dqr, dql);
  uint32_t addr_new;
  const bool in_new = win_addr<FAST>(C.g, tx, ty, tz, offx, offy, offz, p_f, seam_f, base_t_d, addr_new) && !force_out;
  float w_new, w_old;
  if (__any_sync(0xffffffffu, !(in_new && in))) {                  // rare, warp-uniform
    w_new = in_new ? lds_f32(addr_new) : omega_outside(omega_t, A.S.grid, tx, ty, tz);
    w_old = in ? lds_f32(addr) : omega_outside(omega_t, A.S.grid, rx, ry, rz);
  } else {
    w_new = lds_f32(addr_new);
    w_old = lds_f32(addr);
  }
  const float dE = __fmaf_rn(C.kb, dq, __fsub_rn(w_new, w_old));
  const bool acc = metropolis_accept_fma(dE, w.w3);
  if (acc) { rx = tx; ry = ty; rz = tz; addr = addr_new; in = in_new; q_l = ql_new; q_r = qr_new; }
  return acc;
}

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_inval(uint64_t* bar) {
  asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------------------------------------
// The kernel.  Work unit = (column, segment): a column is a cy x cz patch of the (y, z) plane with
// its halo, a segment is Lseg cells of x.  One CTA per SM takes units round-robin and SWEEPS each
// along x: the unit's chains are sorted by the x slice (`slice` cells) that holds their centre of
// mass; a chain of slice k works in the window of slabs [k slice, k slice + wx) of the unit
// (slab a = x layer a - hx of the segment).  Warp 0 is the producer: it TMA-loads omega slabs into
// the ring ahead of the sweep and, once every consumer warp has left slice j, TMA-reduce-adds the
// slabs that slice finished into the ghost-padded global density grid, zeroes them and loads the
// omega of the slabs R further on into their slots.  The other warps are consumers: chain in
// registers (two beads per lane, P = N/2 lanes per chain, next chain group prefetched), both
// half-sweeps, LDS for omega, RED.shared for the densities.  mbarriers: full[slot] (TMA bytes
// landed, counters zeroed), done[slice] (all consumer warps are past it).
// FAST: inv_h is a power of two >= 1 on every axis and a is a power of two (see win_addr,
// trial_axis); the results are identical either way.
// ---------------------------------------------------------------------------------------------
template <int P, bool MULTI_PAT, int NT, bool FAST>
__global__ void __launch_bounds__(NT, 1)
tile_step_kernel(const __grid_constant__ TileArgs A, const __grid_constant__ CUtensorMap tm_omega,
                 const __grid_constant__ CUtensorMap tm_counts) {
  constexpr int G = 32 / P;
  constexpr uint32_t NWC = NT / 32 - 1;                                       // consumer warps
  constexpr uint32_t N = 2u * P;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* omega_ring = smem_raw;
  unsigned char* counts_ring = smem_raw + A.counts_offset;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + A.aux_offset);     // [kMaxRing]
  uint64_t* done = full + kMaxRing;                                           // [kMaxSlices]
  uint32_t* cum = reinterpret_cast<uint32_t*>(done + kMaxSlices);             // [K + 1] chain groups before slice k
  uint32_t* sstart = cum + kMaxSlices + 1;                                    // [K + 1] first slot of slice k
  const StepArgs& S = A.S;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t l = lane % P, sub = lane / P;
  const uint32_t R = A.R, K = A.K, stride = A.slab_stride;
  const uint32_t A_tot = A.Lseg + 2u * A.hx;                                  // slabs of a unit
  unsigned n_acc = 0;

  LaneCtx C;
  C.g.inv_hx = S.grid.inv_hx; C.g.inv_hy = S.grid.inv_hy; C.g.inv_hz = S.grid.inv_hz;
  C.g.wx_f = (float)A.wx; C.g.ey_f = (float)A.ey; C.g.ez_f = (float)A.ez;
  C.g.neg_R = -(float)R;
  C.g.slab_stride_d = __uint_as_float(stride); C.g.sy_d = __uint_as_float(A.ez * 4u); C.g.four_d = __uint_as_float(4u);
  C.a = S.a; C.a2 = A.a2; C.ac = A.ac; C.kb = S.kb;
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

  for (uint32_t unit = blockIdx.x; unit < A.n_units; unit += gridDim.x) {
    const uint32_t sg = unit % A.nseg, col = unit / A.nseg;
    const int x0 = (int)(sg * A.Lseg), y0 = (int)((col / A.mtz) * A.cy), z0 = (int)((col % A.mtz) * A.cz);   // padded coordinates of slab 0
    __syncthreads();                                    // the previous unit is finished, its flushes have read the ring
    for (uint32_t k = tid; k <= K; k += NT) sstart[k] = A.bin_start[2u * (unit * K + k)];
    for (uint32_t k = tid; k < R * stride / 16u; k += NT) reinterpret_cast<uint4*>(counts_ring)[k] = make_uint4(0u, 0u, 0u, 0u);
    if (tid == 0) {
      for (uint32_t r = 0; r < R; ++r) { mbar_inval(&full[r]); mbar_init(&full[r], 1); }
      for (uint32_t k = 0; k < K; ++k) { mbar_inval(&done[k]); mbar_init(&done[k], NWC); }
    }
    __syncthreads();
    if (warp == 0) {                                    // chain groups per slice, exclusive scan (K <= 128: four slices per lane)
      uint32_t g[4], sum = 0;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t k = 4u * lane + q;
        g[q] = k < K ? (sstart[k + 1] - sstart[k] + G - 1) / G : 0u;
        sum += g[q];
      }
      uint32_t inc = sum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (uint32_t)o) inc += t;
      }
      uint32_t run = inc - sum;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t k = 4u * lane + q;
        if (k <= K) cum[k] = run;
        run += g[q];
      }
    }
    __syncthreads();
    const uint32_t F = cum[K];                          // chain groups of the unit
    if (F == 0) continue;                               // uniform over the CTA; nothing was binned

    if (warp == 0) {
      // ---------------- producer ----------------
      if (lane == 0) {
        const uint32_t first = R < A_tot ? R : A_tot;
        for (uint32_t a = 0; a < first; ++a) {
          mbar_expect_tx(&full[a], A.slab_bytes);
          tma_load_4d(omega_ring + a * stride, &tm_omega, &full[a], z0, y0, x0 + (int)a, 0);
        }
      }
      for (uint32_t j = 0; j < K; ++j) {
        if (lane == 0) mbar_wait(&done[j], 0);
        __syncwarp();
        const uint32_t lo = j * A.slice, hi = (j + 1 == K) ? A_tot : lo + A.slice;   // slabs no later slice touches
        if (lane == 0) {
          fence_proxy_async();
          for (uint32_t a = lo; a < hi; ++a)
            tma_reduce_add_4d(&tm_counts, counts_ring + (a % R) * stride, z0, y0, x0 + (int)a, 0);
          bulk_commit();
        }
        if (j + 1 == K) break;
        if (lo + R < A_tot) {                           // their slots take the slabs R further on
          if (lane == 0) bulk_wait_read0();
          __syncwarp();
          for (uint32_t a = lo; a < hi && a + R < A_tot; ++a) {
            uint4* c = reinterpret_cast<uint4*>(counts_ring + (a % R) * stride);
            for (uint32_t k = lane; k < A.slab_bytes / 16u; k += 32u) c[k] = make_uint4(0u, 0u, 0u, 0u);
          }
          __syncwarp();
          if (lane == 0)
            for (uint32_t a = lo; a < hi && a + R < A_tot; ++a) {
              mbar_expect_tx(&full[a % R], A.slab_bytes);      // release: the zeroes are visible to whoever sees the phase complete
              tma_load_4d(omega_ring + (a % R) * stride, &tm_omega, &full[a % R], z0, y0, x0 + (int)(a + R), 0);
            }
        }
      }
      if (lane == 0) bulk_wait_read0();
    } else {
      // ---------------- consumers ----------------
      const uint32_t wc = warp - 1u;
      uint32_t kf = 0;                                  // slice cursor of the prefetch
      float2 Xn, Yn, Zn;
      float4 Mn;
      uint32_t slot_n = 0, k_n = 0;
      bool live_n = false;
      auto fetch = [&](uint32_t f) {
        while (f >= cum[kf + 1]) ++kf;
        const uint32_t s0 = sstart[kf], n = sstart[kf + 1] - s0;
        const uint32_t rel = (f - cum[kf]) * G + sub;
        live_n = rel < n;
        slot_n = s0 + (live_n ? rel : 0u);                                    // dead lanes shadow the slice's first slot
        k_n = kf;
        const uint64_t j = (uint64_t)slot_n * N + 2u * l;
        Xn = *reinterpret_cast<const float2*>(S.x + j);
        Yn = *reinterpret_cast<const float2*>(S.y + j);
        Zn = *reinterpret_cast<const float2*>(S.z + j);
        Mn = __ldg(A.slot_meta + slot_n);
      };
      int kc = -1;                                      // slice being computed
      float p_f = 0.0f, seam_f = 0.0f;
      if (wc < F) fetch(wc);
      for (uint32_t f = wc; f < F; f += NWC) {
        const float2 X = Xn, Y = Yn, Z = Zn;
        const float4 M = Mn;
        const uint32_t slot = slot_n, k_this = k_n;
        const bool live = live_n;
        if (f + NWC < F) fetch(f + NWC);
        if ((int)k_this != kc) {                        // entering a new slice (uniform over the warp)
          __syncwarp();
          if (lane == 0)
            for (uint32_t j = kc < 0 ? 0u : (uint32_t)kc; j < k_this; ++j) mbar_arrive(&done[j]);
          uint32_t a_lo = kc < 0 ? 0u : (uint32_t)kc * A.slice + A.wx;
          uint32_t a_hi = k_this * A.slice + A.wx;
          if (a_hi > A_tot) a_hi = A_tot;
          for (uint32_t a = a_lo; a < a_hi; ++a) mbar_wait(&full[a % R], (a / R) & 1u);
          kc = (int)k_this;
          const uint32_t p = (k_this * A.slice) % R;
          p_f = (float)p;
          seam_f = (float)((int)p - (int)R + 1);
        }
        const uint32_t c0_1 = A.philox_u0 ^ __float_as_uint(M.w);
        if (MULTI_PAT) {
          const uint16_t tt = *reinterpret_cast<const uint16_t*>(S.patterns + (uint32_t)S.slot_pattern[slot] * N + 2u * l);
          type0 = tt & 0xffu; type1 = tt >> 8;
        }
        const float base0 = __uint_as_float(omega_base + type0 * type_stride), base1 = __uint_as_float(omega_base + type1 * type_stride);
        float ex = X.x, ey = Y.x, ez = Z.x;                                   // even bead 2l
        float ox = X.y, oy = Y.y, oz = Z.y;                                   // odd bead 2l+1
        uint32_t addr_e, addr_o;
        bool in_e = win_addr<FAST>(C.g, ex, ey, ez, M.x, M.y, M.z, p_f, seam_f, base0, addr_e);
        bool in_o = win_addr<FAST>(C.g, ox, oy, oz, M.x, M.y, M.z, p_f, seam_f, base1, addr_o);
        // squared lengths of this lane's two bonds: A = (even, odd), B = (odd of lane l-1, even)
        const float lx = __shfl_up_sync(0xffffffffu, ox, 1, P);
        const float ly = __shfl_up_sync(0xffffffffu, oy, 1, P);
        const float lz = __shfl_up_sync(0xffffffffu, oz, 1, P);
        float qA = bond_sq(ex, ey, ez, ox, oy, oz);
        float qB = bond_sq(ex, ey, ez, lx, ly, lz);
        // half-sweep 0: even bead; left neighbour = odd bead of lane l-1, right neighbour = own odd bead
        {
          const bool acc = tile_move<FAST, true>(A, C, L0, c0_1, M.x, M.y, M.z, p_f, seam_f, base0, S.omega + (size_t)type0 * S.cells,
                                                 ex, ey, ez, addr_e, in_e, lx, ly, lz, qB, ox, oy, oz, qA, hl);
          n_acc += (acc && live) ? 1u : 0u;
        }
        // half-sweep 1: odd bead; left = own even bead (new), right = even bead of lane l+1 (new)
        {
          const float rx = __shfl_down_sync(0xffffffffu, ex, 1, P);
          const float ry = __shfl_down_sync(0xffffffffu, ey, 1, P);
          const float rz = __shfl_down_sync(0xffffffffu, ez, 1, P);
          float qR = __shfl_down_sync(0xffffffffu, qB, 1, P);
          const bool acc = tile_move<FAST, false>(A, C, L1, c0_1, M.x, M.y, M.z, p_f, seam_f, base1, S.omega + (size_t)type1 * S.cells,
                                                  ox, oy, oz, addr_o, in_o, ex, ey, ez, qA, rx, ry, rz, qR, hr);
          n_acc += (acc && live) ? 1u : 0u;
        }
        if (live) {
          const uint64_t j = (uint64_t)slot * N + 2u * l;
          *reinterpret_cast<float2*>(S.x + j) = make_float2(ex, ox);
          *reinterpret_cast<float2*>(S.y + j) = make_float2(ey, oy);
          *reinterpret_cast<float2*>(S.z + j) = make_float2(ez, oz);
          if (in_e) reds_inc(addr_e + A.counts_offset); else count_outside(A, type0, ex, ey, ez);
          if (in_o) reds_inc(addr_o + A.counts_offset); else count_outside(A, type1, ox, oy, oz);
        }
      }
      __syncwarp();
      if (lane == 0)
        for (uint32_t j = kc < 0 ? 0u : (uint32_t)kc; j < K; ++j) mbar_arrive(&done[j]);
    }
  }
  if (tid == 0) bulk_wait0();
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
  if (lane == 0 && n_acc) atomicAdd(S.accepted, (unsigned long long)n_acc);
}

// ---------------------------------------------------------------------------------------------
// Sorting the chains for the kernel above.  Key of a chain = 2 (unit K + slice) + e: the unit and
// slice whose core holds the cell of its centre of mass, and e = 1 if a bead lies within `margin`
// cells of the window's faces or beyond (extended chains come last in their slice, so they share
// warps among themselves and the other warps never take the slow path).  The same pass writes the
// chain's floor offsets (see win_addr): off = kFloorMagic + (g - G) - window origin per axis, G the
// unwrapped and g the wrapped cell coordinate of the centre of mass.
// ---------------------------------------------------------------------------------------------
struct TileSortArgs {
  Grid grid;
  uint32_t n_chains, N;
  uint32_t cy, cz, hx, hy, hz, wx, ey, ez;
  uint32_t slice, K, Lseg, mtz, nseg;
  uint32_t margin;
};

__global__ void __launch_bounds__(256)
tile_key_kernel(TileSortArgs S, const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z,
                const uint32_t* __restrict__ slot_chain, uint32_t* __restrict__ bin_count, uint32_t* __restrict__ key,
                uint32_t* __restrict__ rank, float4* __restrict__ meta) {
  const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= S.n_chains) return;
  const uint64_t j0 = (uint64_t)s * S.N;
  float sx = 0.f, sy = 0.f, sz = 0.f;
  for (uint32_t i = 0; i < S.N; ++i) { sx += x[j0 + i]; sy += y[j0 + i]; sz += z[j0 + i]; }
  const float inv = 1.0f / (float)S.N;
  const int Gx = __float2int_rd(__fmul_rn(sx * inv, S.grid.inv_hx));
  const int Gy = __float2int_rd(__fmul_rn(sy * inv, S.grid.inv_hy));
  const int Gz = __float2int_rd(__fmul_rn(sz * inv, S.grid.inv_hz));
  const int gx = Gx & (int)(S.grid.nx - 1u), gy = Gy & (int)(S.grid.ny - 1u), gz = Gz & (int)(S.grid.nz - 1u);
  const uint32_t sg = (uint32_t)gx / S.Lseg, k = ((uint32_t)gx % S.Lseg) / S.slice;
  const uint32_t ty = (uint32_t)gy / S.cy, tz = (uint32_t)gz / S.cz;
  // window-relative cell of a bead = floor(r inv_h) + d, d = (g - G) - window origin
  const int dx = gx - Gx - ((int)(sg * S.Lseg + k * S.slice) - (int)S.hx);
  const int dy = gy - Gy - ((int)(ty * S.cy) - (int)S.hy);
  const int dz = gz - Gz - ((int)(tz * S.cz) - (int)S.hz);
  bool ext = false;
  const int m = (int)S.margin;
  for (uint32_t i = 0; i < S.N; ++i) {
    const int rx = __float2int_rd(__fmul_rn(x[j0 + i], S.grid.inv_hx)) + dx;
    const int ry = __float2int_rd(__fmul_rn(y[j0 + i], S.grid.inv_hy)) + dy;
    const int rz = __float2int_rd(__fmul_rn(z[j0 + i], S.grid.inv_hz)) + dz;
    ext |= rx < m || rx >= (int)S.wx - m || ry < m || ry >= (int)S.ey - m || rz < m || rz >= (int)S.ez - m;
  }
  const uint32_t unit = (ty * S.mtz + tz) * S.nseg + sg;
  const uint32_t kk = 2u * (unit * S.K + k) + (ext ? 1u : 0u);
  key[s] = kk;
  rank[s] = atomicAdd(bin_count + kk, 1u);
  meta[s] = make_float4(kFloorMagic + (float)dx, kFloorMagic + (float)dy, kFloorMagic + (float)dz,
                        __uint_as_float(slot_chain[s]));
}

// ---------------------------------------------------------------------------------------------
// Row a4 for the tiled path: omega from the counts, written both to the linear field and to the
// ghost-padded copy the tiles are loaded from.  One thread per PADDED cell.
// ---------------------------------------------------------------------------------------------
struct PadGeom {
  uint32_t px, py, pz;        // padded dims; padded coordinate q holds cell (q - halo) mod n
  uint32_t hx, hy, hz;
};

// Sum of the padded density grid over all periodic images of cell (gx, gy, gz).
__device__ __forceinline__ uint32_t fold_images(const uint32_t* __restrict__ cp, const Grid& grid, const PadGeom& pg,
                                                uint32_t gx, uint32_t gy, uint32_t gz) {
  uint32_t sum = 0;
  for (int kx = -1; kx <= 1; ++kx) {
    const int qx = (int)(gx + pg.hx) + kx * (int)grid.nx;
    if (qx < 0 || qx >= (int)pg.px) continue;
    for (int ky = -1; ky <= 1; ++ky) {
      const int qy = (int)(gy + pg.hy) + ky * (int)grid.ny;
      if (qy < 0 || qy >= (int)pg.py) continue;
      for (int kz = -1; kz <= 1; ++kz) {
        const int qz = (int)(gz + pg.hz) + kz * (int)grid.nz;
        if (qz < 0 || qz >= (int)pg.pz) continue;
        sum += cp[((size_t)qx * pg.py + qy) * pg.pz + qz];
      }
    }
  }
  return sum;
}

// counts_pad_in != nullptr: this step was binned by the tiled kernel into the padded grid; the
// densities are folded from it and written to the linear grid A.counts_out.  Otherwise they are
// read from the linear grid.  counts_pad_zero is the padded grid the NEXT tiled step bins into.
template <int T_>
__global__ void __launch_bounds__(256)
omega_pad_kernel(OmegaArgs A, Grid grid, PadGeom pg, float* __restrict__ omega_pad,
                 const uint32_t* __restrict__ counts_pad_in, uint32_t* __restrict__ counts_out,
                 uint32_t* __restrict__ counts_pad_zero) {
  const uint32_t T = T_ > 0 ? (uint32_t)T_ : A.T;
  const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t pcells = pg.px * pg.py * pg.pz;
  if (p >= pcells) return;
  const uint32_t qz = p % pg.pz, qy = (p / pg.pz) % pg.py, qx = p / (pg.pz * pg.py);
  const int gx0 = (int)qx - (int)pg.hx, gy0 = (int)qy - (int)pg.hy, gz0 = (int)qz - (int)pg.hz;
  const bool interior = gx0 >= 0 && gx0 < (int)grid.nx && gy0 >= 0 && gy0 < (int)grid.ny && gz0 >= 0 && gz0 < (int)grid.nz;
  const uint32_t gx = (uint32_t)(gx0 & (int)(grid.nx - 1u)), gy = (uint32_t)(gy0 & (int)(grid.ny - 1u)), gz = (uint32_t)(gz0 & (int)(grid.nz - 1u));
  const uint32_t c = (gx * grid.ny + gy) * grid.nz + gz;
  float phi[kMaxTypes];
  float tot = 0.0f;
#pragma unroll
  for (uint32_t s = 0; s < (T_ > 0 ? T_ : kMaxTypes); ++s) {
    if (s < T) {
      uint32_t n_s;
      if (counts_pad_in) {
        n_s = fold_images(counts_pad_in + (size_t)s * pcells, grid, pg, gx, gy, gz);
        if (interior) counts_out[(size_t)s * A.cells + c] = n_s;
      } else {
        n_s = A.counts[(size_t)s * A.cells + c];
      }
      counts_pad_zero[(size_t)s * pcells + p] = 0u;
      phi[s] = __fmul_rn((float)n_s, A.dens_scale);
      tot = s == 0 ? phi[0] : __fadd_rn(tot, phi[s]);
      if (interior && A.counts_to_zero) A.counts_to_zero[(size_t)s * A.cells + c] = 0u;
    }
  }
  const float pr = __fmul_rn(A.kappaN, __fsub_rn(tot, 1.0f));
#pragma unroll
  for (uint32_t t = 0; t < (T_ > 0 ? T_ : kMaxTypes); ++t) {
    if (t < T) {
      float acc = pr;
#pragma unroll
      for (uint32_t s = 0; s < (T_ > 0 ? T_ : kMaxTypes); ++s)
        if (s < T && s != t) acc = __fmaf_rn(A.chiN[t * T + s], phi[s], acc);
      float w = __fmul_rn(A.invN, acc);
      if (A.ext) w = __fadd_rn(w, A.ext[(size_t)t * A.cells + c]);
      omega_pad[(size_t)t * pcells + p] = w;
      if (interior) A.omega[(size_t)t * A.cells + c] = w;
    }
  }
}

}  // namespace soma
