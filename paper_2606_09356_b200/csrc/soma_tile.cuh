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

constexpr uint32_t kOutside = 0xffffffffu;

struct TileArgs {
  StepArgs S;                 // omega = linear field (fallback); counts_next is not used by this kernel
  uint32_t* __restrict__ counts_pad;   // [T][px][py][pz] ghost-padded density grid this step bins into
  uint32_t px, py, pz;        // padded dims: padded coordinate q holds cell (q - halo) mod n
  uint32_t T;
  uint32_t ex, ey, ez, E;     // tile extent in cells (core + 2*halo), E = ex*ey*ez
  uint32_t cx, cy, cz;        // core
  uint32_t hx, hy, hz;        // halo
  uint32_t mty, mtz, n_tiles; // tiles along y and z, total
  uint32_t counts_offset;     // byte offset of the density tile in dynamic shared memory
  const uint32_t* __restrict__ tile_start;   // [n_tiles + 1] first slot of every tile
};

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

// Per-tile geometry held in registers: floor magic minus the tile origin, so that the masked bit
// pattern of fadd_rd(r*inv_h, m) is directly the coordinate RELATIVE to the tile origin (mod grid).
struct TileGeom {
  float mx, my, mz;
};

__device__ __forceinline__ uint32_t local_cell(const TileArgs& A, const TileGeom& g, float x, float y, float z) {
  const Grid& G = A.S.grid;
  const uint32_t bx = __float_as_uint(__fadd_rd(__fmul_rn(x, G.inv_hx), g.mx)) & (G.nx - 1u);
  const uint32_t by = __float_as_uint(__fadd_rd(__fmul_rn(y, G.inv_hy), g.my)) & (G.ny - 1u);
  const uint32_t bz = __float_as_uint(__fadd_rd(__fmul_rn(z, G.inv_hz), g.mz)) & (G.nz - 1u);
  const bool inside = (bx < A.ex) & (by < A.ey) & (bz < A.ez);
  return inside ? (bx * A.ey + by) * A.ez + bz : kOutside;
}

__device__ __forceinline__ float omega_lookup(const TileArgs& A, const float* __restrict__ omega_s_t, uint32_t type_cells,
                                              uint32_t idx, float x, float y, float z) {
  if (idx != kOutside) return omega_s_t[idx];
  return __ldg(A.S.omega + type_cells + cell_of<true>(A.S.grid, x, y, z));
}

// One Metropolis trial move inside a tile.  Same arithmetic as move_bead; only where omega is read
// from differs.  `idx` is the bead's tile-local cell (or kOutside) and follows the bead.
__device__ __forceinline__ bool move_bead_tile(const TileArgs& A, const TileGeom& g, uint32_t chain, uint32_t i, uint32_t parity,
                                               const float* __restrict__ omega_s_t, uint32_t type_cells,
                                               float& rx, float& ry, float& rz, uint32_t& idx,
                                               bool has_l, float lx, float ly, float lz,
                                               bool has_r, float qx, float qy, float qz) {
  const StepArgs& S = A.S;
  const Words4 w = philox4x32_10(i, chain, S.ctr2, S.ctr3_base | parity, S.keys);
  const Trial t = trial_position(rx, ry, rz, S.a, w);
  float dq = 0.0f;
  if (has_l) dq = __fsub_rn(bond_sq(t.x, t.y, t.z, lx, ly, lz), bond_sq(rx, ry, rz, lx, ly, lz));
  if (has_r) {
    const float dqr = __fsub_rn(bond_sq(t.x, t.y, t.z, qx, qy, qz), bond_sq(rx, ry, rz, qx, qy, qz));
    dq = has_l ? __fadd_rn(dq, dqr) : dqr;
  }
  const uint32_t idx_new = local_cell(A, g, t.x, t.y, t.z);
  const float w_new = omega_lookup(A, omega_s_t, type_cells, idx_new, t.x, t.y, t.z);
  const float w_old = omega_lookup(A, omega_s_t, type_cells, idx, rx, ry, rz);
  const float dE = __fmaf_rn(S.kb, dq, __fsub_rn(w_new, w_old));
  const bool acc = metropolis_accept(dE, w.w3);
  if (acc) { rx = t.x; ry = t.y; rz = t.z; idx = idx_new; }
  return acc;
}

__device__ __forceinline__ void count_bead(const TileArgs& A, uint32_t* __restrict__ counts_s, uint32_t type,
                                           uint32_t idx, float x, float y, float z) {
  if (idx != kOutside) { atomicAdd(counts_s + type * A.E + idx, 1u); return; }
  // outside the tile: straight into the padded grid, at the image that lies `halo` inside it
  const Grid& G = A.S.grid;
  const uint32_t gx = floor_bits(__fmul_rn(x, G.inv_hx)) & (G.nx - 1u);
  const uint32_t gy = floor_bits(__fmul_rn(y, G.inv_hy)) & (G.ny - 1u);
  const uint32_t gz = floor_bits(__fmul_rn(z, G.inv_hz)) & (G.nz - 1u);
  atomicAdd(A.counts_pad + ((size_t)(type * A.px + gx + A.hx) * A.py + gy + A.hy) * A.pz + gz + A.hz, 1u);
}

template <int P, bool MULTI_PAT, int NT>
__global__ void __launch_bounds__(NT, 1)
tile_step_kernel(const __grid_constant__ TileArgs A, const __grid_constant__ CUtensorMap tm_omega,
                 const __grid_constant__ CUtensorMap tm_counts) {
  constexpr int G = 32 / P;
  constexpr uint32_t NW = NT / 32;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t mbar;
  float* omega_s = reinterpret_cast<float*>(smem_raw);                        // [T][E]
  uint32_t* counts_s = reinterpret_cast<uint32_t*>(smem_raw + A.counts_offset);   // [T][E]
  const StepArgs& S = A.S;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t l = lane % P, sub = lane / P;
  const uint32_t tile_words = A.T * A.E;
  unsigned n_acc = 0;
  uint32_t phase = 0;

  if (tid == 0) mbar_init(&mbar, 1);
  __syncthreads();

  uint32_t type0 = 0, type1 = 0;
  if (!MULTI_PAT) {
    const uint16_t tt = *reinterpret_cast<const uint16_t*>(S.patterns + 2u * l);
    type0 = tt & 0xffu; type1 = tt >> 8;
  }

  for (uint32_t tile = blockIdx.x; tile < A.n_tiles; tile += gridDim.x) {
    const uint32_t start = A.tile_start[tile], end = A.tile_start[tile + 1];
    if (start == end) continue;                                               // uniform over the CTA
    const uint32_t tz = tile % A.mtz, ty = (tile / A.mtz) % A.mty, tx = tile / (A.mtz * A.mty);
    const int ox = (int)(tx * A.cx) - (int)A.hx, oy = (int)(ty * A.cy) - (int)A.hy, oz = (int)(tz * A.cz) - (int)A.hz;
    TileGeom g;
    g.mx = kFloorMagic - (float)ox; g.my = kFloorMagic - (float)oy; g.mz = kFloorMagic - (float)oz;

    // omega tile in (the padded copy is indexed from -halo, so the coordinates are never negative);
    // the previous tile's density flush must have finished READING shared memory before it is zeroed
    if (tid == 0) {
      mbar_expect_tx(&mbar, tile_words * 4u);
      tma_load_4d(omega_s, &tm_omega, &mbar, oz + (int)A.hz, oy + (int)A.hy, ox + (int)A.hx, 0);
      bulk_wait_read0();
    }
    __syncthreads();
    for (uint32_t k = tid; k < tile_words / 4u; k += NT) reinterpret_cast<uint4*>(counts_s)[k] = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
    mbar_wait(&mbar, phase);
    phase ^= 1u;

    const uint32_t n_slots = end - start;
    const uint32_t n_groups = (n_slots + G - 1) / G;
    for (uint32_t wg = warp; wg < n_groups; wg += NW) {
      const uint32_t rel = wg * G + sub;
      const bool live = rel < n_slots;
      const uint32_t slot = start + (live ? rel : 0u);                        // dead lanes shadow the first slot
      const uint64_t j = (uint64_t)slot * S.N + 2u * l;
      const float2 X = *reinterpret_cast<const float2*>(S.x + j);
      const float2 Y = *reinterpret_cast<const float2*>(S.y + j);
      const float2 Z = *reinterpret_cast<const float2*>(S.z + j);
      const uint32_t chain = S.slot_chain[slot];
      if (MULTI_PAT) {
        const uint16_t tt = *reinterpret_cast<const uint16_t*>(S.patterns + (uint32_t)S.slot_pattern[slot] * S.N + 2u * l);
        type0 = tt & 0xffu; type1 = tt >> 8;
      }
      float ex = X.x, ey = Y.x, ez = Z.x;                                     // even bead 2l
      float ox_ = X.y, oy_ = Y.y, oz_ = Z.y;                                  // odd bead 2l+1
      uint32_t idx_e = local_cell(A, g, ex, ey, ez);
      uint32_t idx_o = local_cell(A, g, ox_, oy_, oz_);
      {
        const float lx = __shfl_up_sync(0xffffffffu, ox_, 1, P);
        const float ly = __shfl_up_sync(0xffffffffu, oy_, 1, P);
        const float lz = __shfl_up_sync(0xffffffffu, oz_, 1, P);
        const bool acc = move_bead_tile(A, g, chain, 2u * l, 0u, omega_s + type0 * A.E, type0 * S.cells, ex, ey, ez, idx_e,
                                        l > 0, lx, ly, lz, true, ox_, oy_, oz_);
        n_acc += (acc && live) ? 1u : 0u;
      }
      {
        const float qx = __shfl_down_sync(0xffffffffu, ex, 1, P);
        const float qy = __shfl_down_sync(0xffffffffu, ey, 1, P);
        const float qz = __shfl_down_sync(0xffffffffu, ez, 1, P);
        const bool acc = move_bead_tile(A, g, chain, 2u * l + 1u, 1u, omega_s + type1 * A.E, type1 * S.cells, ox_, oy_, oz_, idx_o,
                                        true, ex, ey, ez, l + 1 < P, qx, qy, qz);
        n_acc += (acc && live) ? 1u : 0u;
      }
      if (live) {
        *reinterpret_cast<float2*>(S.x + j) = make_float2(ex, ox_);
        *reinterpret_cast<float2*>(S.y + j) = make_float2(ey, oy_);
        *reinterpret_cast<float2*>(S.z + j) = make_float2(ez, oz_);
        count_bead(A, counts_s, type0, idx_e, ex, ey, ez);
        count_bead(A, counts_s, type1, idx_o, ox_, oy_, oz_);
      }
    }
    // density tile out
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {                                                           // padded coordinates: origin + halo = tile * core
      tma_reduce_add_4d(&tm_counts, counts_s, oz + (int)A.hz, oy + (int)A.hy, ox + (int)A.hx, 0);
      bulk_commit();
    }
  }
  if (tid == 0) bulk_wait0();
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
  if (lane == 0 && n_acc) atomicAdd(S.accepted, (unsigned long long)n_acc);
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
      const float w = __fmul_rn(A.invN, acc);
      omega_pad[(size_t)t * pcells + p] = w;
      if (interior) A.omega[(size_t)t * A.cells + c] = w;
    }
  }
}

}  // namespace soma
