// soma_device.cuh -- per-move device arithmetic of the SCMF Monte-Carlo step.
//
// Everything here is fp32 with the operation order of DESIGN.md section 2 spelled out through
// __f*_rn intrinsics (never contracted by the compiler), so that the result of every move is
// bit-identical to the definition regardless of optimisation level.  No code is shared with oracle/.
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

namespace soma {

// ---- Philox4x32-10 (R13; `north_star`: keyed by (seed, step, half-sweep, chain, bead)) ----
constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

struct Words4 { uint32_t w0, w1, w2, w3; };

__device__ __forceinline__ Words4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(kPhiloxM0, c0), lo0 = kPhiloxM0 * c0;
    const uint32_t hi1 = __umulhi(kPhiloxM1, c2), lo1 = kPhiloxM1 * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += kPhiloxW0;
    k1 += kPhiloxW1;
  }
  return Words4{c0, c1, c2, c3};
}

// The same generator with the ten round keys (k + r*W) precomputed on the host and read from the
// kernel's constant bank: every round is 2 IMAD.WIDE.U32 + 2 LOP3, no key arithmetic.
struct PhiloxKeys { uint32_t k0[10], k1[10]; };

__device__ __forceinline__ Words4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                const PhiloxKeys& K) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
    const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];
    c1 = (uint32_t)p1;
    c2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
    c3 = (uint32_t)p0;
  }
  return Words4{c0, c1, c2, c3};
}

// ---- uniform maps (R14) ----
// tmap(w) = (2k+1) 2^-23 - 1 with k = w >> 9.  Built from the bit pattern instead of an int->float
// conversion: as_float(0x3f800000 | k) - 1 = k 2^-23 exactly, then fma(2, ., 2^-23 - 1) is exact
// because the result (an odd multiple of 2^-23 below 1 in magnitude) is representable.
__device__ __forceinline__ float tmap(uint32_t w) {
  const float h = __fadd_rn(__uint_as_float(0x3f800000u | (w >> 9)), -1.0f);
  return __fmaf_rn(2.0f, h, -0.99999988079071044921875f);   // 2^-23 - 1
}
// u * 2^24 = (w >> 8) + 1 in [1, 2^24]: the integer converts exactly (I2FP.F32.U32, one instruction).
__device__ __forceinline__ float umap_int(uint32_t w) { return (float)((w >> 8) + 1u); }
__device__ __forceinline__ float umap(uint32_t w) { return __fmul_rn(umap_int(w), 0x1p-24f); }

// lnu = ln(u) correctly rounded to fp32 (R6b), slow path: double log, one rounding.
__device__ __noinline__ float lnu_exact(float u) { return (float)log((double)u); }

// hardware base-2 logarithm, one MUFU.LG2 (the argument is a normal number in [1, 2^24])
__device__ __forceinline__ float lg2_approx(float v) {
  float r;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}

// ln(u) by the fast route, |error| < kLnBand/16 over all 2^24 values of u (checked exhaustively by
// tests/test_gpu_units.py through soma_debug_maps).
__device__ __forceinline__ float lnu_fast(uint32_t w3) {
  return __fmul_rn(__fadd_rn(lg2_approx(umap_int(w3)), -24.0f), 0.693147182464599609375f);
}
constexpr float kLnBand = 1.0e-4f;

// ---- Metropolis decision (DESIGN.md section 2 step 5.6): accept iff fl32(dE + lnu) <= 0 ----
// Result-equivalent shortcuts:
//  * dE <= 0: lnu <= 0, so the fp32 sum is <= 0 -> accept without looking at u.
//  * otherwise m~ = dE + lnu_fast; if |m~| > kLnBand the sign of the exact margin is the sign of m~
//    (the fp32 rounding of dE + lnu moves it by < 1e-6).  Only the ~6e-5 of moves inside that band
//    take the double-precision path.
__device__ __forceinline__ bool metropolis_accept(float dE, uint32_t w3) {
  const float m_fast = __fadd_rn(dE, lnu_fast(w3));
  bool acc = (dE <= 0.0f) | (m_fast < -kLnBand);
  if (dE > 0.0f && fabsf(m_fast) <= kLnBand) {
    const float m = __fadd_rn(dE, lnu_exact(umap(w3)));
    acc = m <= 0.0f;
  }
  return acc;
}

// ---- Philox4x32-10 with the loop-invariant part of the first three rounds folded ---------------
// Counter of a move = (bead i, chain c, step, parity | domain<<8 | step_hi<<16).  Only c differs
// between the moves a lane makes, and it enters through round 1 as c0' = u0 ^ c, so for every lane
// and parity the values below are fixed for the whole kernel (derivation in DESIGN.md section 7):
//   LC = lo(M0 i) ^ k1[1]                       (xor-ed onto hi(M0 c0') in round 2)
//   LD = lo(M1 c2') ^ k0[2],  c2' = hi(M0 i) ^ ctr3 ^ k1[0]
//   LE = hi(M0 c0'') ^ k1[2], c0'' = hi(M1 c2') ^ u1 ^ k0[1]
//   LF = lo(M0 c0'')
// which leaves 16 wide multiplies and 18 xors per move instead of 20 + 20.
struct PhiloxLane { uint32_t LC, LD, LE, LF; };

__device__ __forceinline__ PhiloxLane philox_lane(const PhiloxKeys& K, uint32_t u1, uint32_t i, uint32_t ctr3) {
  const uint64_t p0 = (uint64_t)kPhiloxM0 * i;
  const uint32_t c2_1 = (uint32_t)(p0 >> 32) ^ ctr3 ^ K.k1[0];
  const uint64_t p1 = (uint64_t)kPhiloxM1 * c2_1;
  const uint32_t c0_2 = (uint32_t)(p1 >> 32) ^ u1 ^ K.k0[1];
  const uint64_t q0 = (uint64_t)kPhiloxM0 * c0_2;
  PhiloxLane L;
  L.LC = (uint32_t)p0 ^ K.k1[1];
  L.LD = (uint32_t)p1 ^ K.k0[2];
  L.LE = (uint32_t)(q0 >> 32) ^ K.k1[2];
  L.LF = (uint32_t)q0;
  return L;
}

// c0_1 = u0 ^ chain, u0 = hi(M1 step) ^ k0[0]
__device__ __forceinline__ Words4 philox_tail(const PhiloxKeys& K, const PhiloxLane& L, uint32_t c0_1) {
  const uint64_t r2 = (uint64_t)kPhiloxM0 * c0_1;                       // round 2
  const uint32_t c2_2 = (uint32_t)(r2 >> 32) ^ L.LC;
  const uint64_t r3 = (uint64_t)kPhiloxM1 * c2_2;                       // round 3
  uint32_t c0 = (uint32_t)(r3 >> 32) ^ L.LD;
  uint32_t c1 = (uint32_t)r3;
  uint32_t c2 = L.LE ^ (uint32_t)r2;
  uint32_t c3 = L.LF;
#pragma unroll
  for (int r = 3; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
    const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];
    c1 = (uint32_t)p1;
    c2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
    c3 = (uint32_t)p0;
  }
  return Words4{c0, c1, c2, c3};
}

// ---- Metropolis decision, one fused multiply-add from the hardware logarithm --------------------
// m = lg2(u 2^24) ln2 + dE = dE + ln u + 24 ln2 up to ~1e-5.  accept iff fl(dE + lnu) <= 0
// (DESIGN.md section 2 step 5.6); m outside [T - band, T + band] decides that exactly (this
// includes dE <= 0: then the exact rule accepts, and either m < T - band or the slow path runs).
constexpr float kLn2 = 0.693147182464599609375f;
constexpr float kLnT = 16.6355323791503906250f;            // 24 ln 2
// u24 = u 2^24 as a float (umap_int); this is the routine both fused kernels call and soma_debug_accept_fma tests
__device__ __forceinline__ bool accept_fma_u24(float dE, float u24) {
  const float m = __fmaf_rn(lg2_approx(u24), kLn2, dE);
  bool acc = m < kLnT - kLnBand;
  if (!acc && m <= kLnT + kLnBand)                              // ~6e-5 of the moves: exact logarithm
    acc = __fadd_rn(dE, lnu_exact(__fmul_rn(u24, 0x1p-24f))) <= 0.0f;
  return acc;
}
__device__ __forceinline__ bool metropolis_accept_fma(float dE, uint32_t w3) { return accept_fma_u24(dE, umap_int(w3)); }

// ---- standard normal deviates for the bond-force-biased move (R24) -------------------
// fp32 Box-Muller from U = ((w >> 9) + 0.5) 2^-23 with the logarithm and sine / cosine spelled out
// in IEEE fp32 operations only (add, mul, div, fma, sqrt -- each correctly rounded on any conforming
// implementation), so the deviates do not depend on a math library.  Written from DESIGN.md R24.
__device__ __forceinline__ float ln_ieee(float x) {                  // x in (0, 1]
  const uint32_t bits = __float_as_uint(x);
  int e = (int)((bits >> 23) & 0xffu) - 127;
  float m = __uint_as_float((bits & 0x007fffffu) | 0x3f800000u);   // [1, 2)
  if (m > 1.41421354f) { m = __fmul_rn(m, 0.5f); e += 1; }
  const float q = __fdiv_rn(__fadd_rn(m, -1.0f), __fadd_rn(m, 1.0f)), z = __fmul_rn(q, q);
  float p = 1.0f / 11.0f;
  p = __fmaf_rn(p, z, 1.0f / 9.0f); p = __fmaf_rn(p, z, 1.0f / 7.0f); p = __fmaf_rn(p, z, 1.0f / 5.0f); p = __fmaf_rn(p, z, 1.0f / 3.0f);
  const float q2 = __fmul_rn(2.0f, q);
  const float lm = __fmaf_rn(q2, __fmul_rn(z, p), q2);
  return __fmaf_rn((float)e, 0.693147182f, lm);
}
__device__ __forceinline__ void sincos_2pi_ieee(float u, float& sn, float& cs) {   // u in (0, 1)
  const float t = __fmul_rn(u, 4.0f);
  const float k = floorf(__fadd_rn(t, 0.5f));
  const float r = __fmul_rn(__fadd_rn(t, -k), 1.57079637f), z = __fmul_rn(r, r);
  float ps = 1.0f / 362880.0f;
  ps = __fmaf_rn(ps, z, -1.0f / 5040.0f); ps = __fmaf_rn(ps, z, 1.0f / 120.0f); ps = __fmaf_rn(ps, z, -1.0f / 6.0f);
  const float s0 = __fmaf_rn(__fmul_rn(r, z), ps, r);
  float pc = -1.0f / 3628800.0f;
  pc = __fmaf_rn(pc, z, 1.0f / 40320.0f); pc = __fmaf_rn(pc, z, -1.0f / 720.0f); pc = __fmaf_rn(pc, z, 1.0f / 24.0f); pc = __fmaf_rn(pc, z, -0.5f);
  const float c0 = __fmaf_rn(pc, z, 1.0f);
  const int qd = (int)k & 3;
  sn = qd == 0 ? s0 : qd == 1 ? c0 : qd == 2 ? -s0 : -c0;
  cs = qd == 0 ? c0 : qd == 1 ? -s0 : qd == 2 ? -c0 : s0;
}
__device__ __forceinline__ float unit23(uint32_t w) { return __fmul_rn(__fadd_rn((float)(w >> 9), 0.5f), 0x1p-23f); }

// xi[0..2]: deviates of a move from the words of its two Philox calls (domain 0: w, domain 2: v)
__device__ __forceinline__ void smc_deviates(const Words4& w, const Words4& v, float& x0, float& x1, float& x2) {
  float sn, cs, sn2, cs2;
  const float ra = __fsqrt_rn(__fmul_rn(-2.0f, ln_ieee(unit23(w.w0))));
  sincos_2pi_ieee(unit23(w.w1), sn, cs);
  const float rb = __fsqrt_rn(__fmul_rn(-2.0f, ln_ieee(unit23(v.w0))));
  sincos_2pi_ieee(unit23(v.w1), sn2, cs2);
  x0 = __fmul_rn(ra, cs); x1 = __fmul_rn(ra, sn); x2 = __fmul_rn(rb, cs2);
}

// ---- density counters ----------------------------------------------------
// Either one uint32 per cell and type, [T][C], or -- "packed", systems of at most two types -- one uint32 per
// cell that holds type 0 in its low and type 1 in its high 16 bits, [C].  An increment is one atomic add of
// 1 or 65536; a field never carries into its neighbour as long as a cell holds fewer than 65536 beads of a type.
// That is guaranteed, not assumed: with a move reach of r cells per step and axis a cell can receive, in one
// step, at most the beads of the (2r+1)^3 cells around it.  The guard level G is the largest power of two with
// ((2r+1)^3 + 1) G <= 65536 (r = 1: 2048 beads of one type in a cell -- two orders of magnitude above the
// configs' densities); the word of every non-empty cell is inspected in every step (by the omega pass, or by the
// old-cell gathers of the lean kernel when it computes omega itself), and a field that has reached G raises a
// flag that fails the next synchronising call.  While no flag is up every field is < G, so after one more
// step every field is < (2r+1)^3 G <= 65536 - G: it cannot have wrapped before it is seen.
// guard_mask = ~(G - 1) on both halves of a word, e.g. 0xF800F800.
__device__ __forceinline__ uint32_t count_word(uint32_t type, uint32_t cells, uint32_t packed) { return packed ? 0u : type * cells; }
__device__ __forceinline__ uint32_t count_inc(uint32_t type, uint32_t packed) { return packed ? 1u << (type << 4) : 1u; }
__device__ __forceinline__ uint32_t count_get(const uint32_t* __restrict__ counts, uint32_t type, uint32_t cells, uint32_t c, uint32_t packed) {
  return packed ? (counts[c] >> (type << 4)) & 0xffffu : counts[(size_t)type * cells + c];
}

// ---- geometry ----
struct Grid {
  uint32_t nx, ny, nz;          // cells per axis
  float inv_hx, inv_hy, inv_hz; // (float)grid[d]/box[d]
};

template <bool POW2>
__device__ __forceinline__ uint32_t wrap(int g, uint32_t n) {
  if (POW2) return (uint32_t)g & (n - 1u);          // two's complement: the non-negative residue
  if ((uint32_t)g >= n) {                           // rare: bead outside the primary box
    g %= (int)n;
    if (g < 0) g += (int)n;
  }
  return (uint32_t)g;
}

// floor(s) mod n for n a power of two without a conversion: s + 1.5*2^23 rounded DOWN has ulp 1, so
// its bit pattern is 0x4b400000 + floor(s) for |s| < 2^22, and the low bits under the mask n-1 are
// the non-negative residue (two's complement borrow for negative floors).  The library checks
// |s| < 2^21 when positions are loaded and re-checks before a bead could have drifted out of range.
constexpr float kFloorMagic = 12582912.0f;       // 1.5 * 2^23
constexpr float kCellCoordLimit = 2097152.0f;    // 2^21
__device__ __forceinline__ uint32_t floor_bits(float s) { return __float_as_uint(__fadd_rd(s, kFloorMagic)); }

// DESIGN.md section 2 step 1 (R8, R12).  Generic grids: cvt.rmi.s32.f32 = floor then convert.
template <bool POW2>
__device__ __forceinline__ uint32_t cell_of(const Grid& g, float x, float y, float z) {
  if (POW2) {
    const uint32_t ix = floor_bits(__fmul_rn(x, g.inv_hx)) & (g.nx - 1u);
    const uint32_t iy = floor_bits(__fmul_rn(y, g.inv_hy)) & (g.ny - 1u);
    const uint32_t iz = floor_bits(__fmul_rn(z, g.inv_hz)) & (g.nz - 1u);
    return (ix * g.ny + iy) * g.nz + iz;
  }
  const uint32_t ix = wrap<false>(__float2int_rd(__fmul_rn(x, g.inv_hx)), g.nx);
  const uint32_t iy = wrap<false>(__float2int_rd(__fmul_rn(y, g.inv_hy)), g.ny);
  const uint32_t iz = wrap<false>(__float2int_rd(__fmul_rn(z, g.inv_hz)), g.nz);
  return (ix * g.ny + iy) * g.nz + iz;
}

// squared bond length, DESIGN.md section 2 step 5.4: fma(sz,sz, fma(sy,sy, sx*sx))
__device__ __forceinline__ float bond_sq(float ax, float ay, float az, float bx, float by, float bz) {
  const float sx = __fsub_rn(ax, bx), sy = __fsub_rn(ay, by), sz = __fsub_rn(az, bz);
  return __fmaf_rn(sz, sz, __fmaf_rn(sy, sy, __fmul_rn(sx, sx)));
}

struct Trial { float x, y, z; };

// DESIGN.md section 2 steps 5.1-5.3: the trial position of bead (chain c, index i).
__device__ __forceinline__ Trial trial_position(float rx, float ry, float rz, float a, const Words4& w) {
  Trial t;
  t.x = __fadd_rn(rx, __fmul_rn(a, tmap(w.w0)));
  t.y = __fadd_rn(ry, __fmul_rn(a, tmap(w.w1)));
  t.z = __fadd_rn(rz, __fmul_rn(a, tmap(w.w2)));
  return t;
}

}  // namespace soma
