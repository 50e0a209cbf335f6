// scmf_oracle.cpp -- ORACLE (test infrastructure, not the product).
//
// Plain, slow, single-threaded CPU statement of the single-chain-in-mean-field (SCMF) Monte-Carlo
// step of the SOMA particle model (section 2: "Single-Chain-in-Mean-Field (SCMF)
// algorithm using a soft, coarse-grained polymer model", "quasi-instantaneous-field approximation
// for non-bonded interactions"; section 2.2: kernels mc_polymer_iteration -- "trial
// moves and energy evaluations" -- and update_density_fields -- "updates particle density
// fields").  The paper prints no equation for the step; every concrete choice below is either
// fixed by BASELINE.json `north_star` / `configs` (marked NS) or is the reading of SURVEY.md
// section 8(c) listed in DESIGN.md section 3 (marked R<k>).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// load this file.  It shares no code, header, table or constant generator with the CUDA path
// under paper_2606_09356_b200/; neither side includes or imports the other.
//
// The method is a stochastic iteration, so the oracle is the algorithm step by step, in the
// order of DESIGN.md section 2: no blocking, no fusion, no reordering.  Arithmetic is fp32 with
// the operation order written out (NS: "fp32" in every config; R17), compiled with
// -ffp-contract=off so that an FMA appears only where fmaf() is written.  ln u is the correctly
// rounded fp32 logarithm, obtained as (float)log((double)u) (R6b; the double rounding
// is checked exhaustively over all 2^24 values of u in tests/test_oracle_rng.py).
//
// Pins (tests/, -m "not gpu"): Philox known-answer vectors; exact uniform maps; bin counts by
// hand; omega against a finite difference of the grid Hamiltonian evaluated in Python; delta-E
// against E(x') - E(x) evaluated in Python; brute-force detailed balance; ideal-chain closed
// forms (<R_ee^2> = (N-1) b^2, Gaussian bond statistics, acceptance rate by quadrature).
// Unpinned (no number in the paper): the ordered morphologies at chiN > 0 -- "parity unpinned"
// for physics beyond the closed forms above; only GPU-vs-oracle agreement is claimed there.

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

namespace {

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (NS: "counter-based Philox4x32-10 random numbers keyed by (seed, step,
// half-sweep, chain, bead)"; constants and round function: DESIGN.md R13 -- the published
// Philox4x32 parameters; pinned by three known-answer vectors in tests/golden/philox_kat.txt).
// ---------------------------------------------------------------------------------------------
const uint32_t PHILOX_M0 = 0xD2511F53u;   // multiplies counter word 0
const uint32_t PHILOX_M1 = 0xCD9E8D57u;   // multiplies counter word 2
const uint32_t PHILOX_W0 = 0x9E3779B9u;   // key word 0 increment per round
const uint32_t PHILOX_W1 = 0xBB67AE85u;   // key word 1 increment per round

void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += PHILOX_W0;
    k1 += PHILOX_W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// DESIGN.md R14: symmetric 23-bit uniform in (-1, 1), never 0; every step is exact in fp32.
float tmap(uint32_t w) {
  const uint32_t k = w >> 9;                                 // 23 bits
  return (float)(2u * k + 1u) * 0x1p-23f - 1.0f;
}
// DESIGN.md R14: 24-bit uniform in (0, 1]; exact in fp32.
float umap(uint32_t w) {
  return (float)((w >> 8) + 1u) * 0x1p-24f;
}
// DESIGN.md R6b: correctly rounded fp32 natural logarithm of u.
float lnu32(float u) {
  return (float)std::log((double)u);
}

const uint32_t RNG_DOMAIN_MOVE = 0;   // DESIGN.md R13: counter word 3 = parity | domain<<8 | (t>>32)<<16

struct Oracle {
  // problem statement (NS: "chains, bead types, bond length b, chiN, kappaN, grid, box")
  uint64_t n_chains;
  uint32_t N, T, n_patterns;
  std::vector<uint8_t> type_patterns;   // [n_patterns][N]
  std::vector<uint8_t> chain_pattern;   // [n_chains]
  float b, kappaN, a;
  std::vector<float> chiN;              // [T][T]
  uint32_t grid[3];
  float box[3];
  uint64_t seed;
  // derived constants ("derived constants")
  float kb;                             // 1.5f/(b*b): harmonic bond, H_b/kT = kb*sum |r_i - r_{i+1}|^2 (R1)
  float inv_h[3];                       // (float)grid[d]/box[d]
  float dens_scale;                     // (float)((double)C/(double)B) = 1/nbar (R10)
  float invN;                           // 1.0f/(float)N (R3)
  uint64_t B, C;
  // state
  std::vector<float> x, y, z;           // [B], index c*N+i, unwrapped (R7)
  std::vector<uint32_t> counts;         // [T][C], cell = (ix*ny+iy)*nz+iz (R12)
  std::vector<float> omega;             // [T][C]
  std::vector<float> ext;               // [T][C] external field (empty = none), R21
  std::vector<float> phi_target;        // [T][C] target concentrations of the umbrella potential (empty = none), R25
  float umbrella_k = 0.0f;              // its strength in kT per bead and unit concentration
  // single-bead molecules (R23): n_single[t] of type t, stored after the chains in x, y, z,
  // type 0 first; molecule m has the logical chain id n_chains + m and bead index 0
  float smcA = 0.0f;                    // > 0: bond-force-biased moves with mobility A (R24), 0: uniform moves
  float gA = 0.0f, sq2A = 0.0f, inv4A = 0.0f;   // fl(A * 2 kb), (float)sqrt(2 A), (float)(1 / (4 A))
  std::vector<uint64_t> n_single;       // [T] (empty = none)
  uint64_t S = 0;                       // their total
  // polymer species of different chain lengths (R26): chains are stored species by species; N above is
  // then only the reference chain length of 1/N (R3) and Nstride the row length of type_patterns
  struct Species { uint64_t n, first_chain, bead_off; uint32_t N; };
  std::vector<Species> species;         // at least one entry
  uint32_t Nstride;
  uint64_t NB;                          // beads in chains (the single-bead molecules follow them)
  uint64_t t;                           // absolute step index
  bool loaded;
};

inline const Oracle::Species& species_of_chain(const Oracle& o, uint64_t c) {
  size_t k = 0;
  while (k + 1 < o.species.size() && c >= o.species[k + 1].first_chain) ++k;
  return o.species[k];
}
inline uint32_t chain_len(const Oracle& o, uint64_t c) { return species_of_chain(o, c).N; }
inline uint64_t chain_bead0(const Oracle& o, uint64_t c) {
  const Oracle::Species& sp = species_of_chain(o, c);
  return sp.bead_off + (c - sp.first_chain) * sp.N;
}
inline void bead_to_chain(const Oracle& o, uint64_t j, uint64_t* c, uint32_t* i) {
  size_t k = 0;
  while (k + 1 < o.species.size() && j >= o.species[k + 1].bead_off) ++k;
  const Oracle::Species& sp = o.species[k];
  *c = sp.first_chain + (j - sp.bead_off) / sp.N;
  *i = (uint32_t)((j - sp.bead_off) % sp.N);
}

inline uint8_t bead_type(const Oracle& o, uint64_t c, uint32_t i) {
  return o.type_patterns[(size_t)o.chain_pattern[c] * o.Nstride + i];
}

// DESIGN.md section 2 step 1 (R8): floorf, then a proper non-negative modulo per axis.
inline uint64_t cell_index(const Oracle& o, float rx, float ry, float rz) {
  const float r[3] = {rx, ry, rz};
  int32_t g[3];
  for (int d = 0; d < 3; ++d) {
    const float scaled = r[d] * o.inv_h[d];              // requires |scaled| < 2^31
    int32_t gi = (int32_t)floorf(scaled);
    const int32_t nd = (int32_t)o.grid[d];
    gi %= nd;                                            // C remainder: sign of the dividend
    if (gi < 0) gi += nd;                                // -> representative in [0, nd)
    g[d] = gi;
  }
  return ((uint64_t)g[0] * o.grid[1] + (uint64_t)g[1]) * o.grid[2] + (uint64_t)g[2];
}

inline uint32_t single_type(const Oracle& o, uint64_t m) {
  uint32_t t = 0;
  while (m >= o.n_single[t]) { m -= o.n_single[t]; ++t; }
  return t;
}

// DESIGN.md section 2 step 2 (NS part 2; R9 nearest-grid-point assignment): integer counts.
void bin(Oracle& o) {
  std::fill(o.counts.begin(), o.counts.end(), 0u);
  for (uint64_t m = 0; m < o.S; ++m) {
    const uint64_t j = o.NB + m;
    o.counts[(size_t)single_type(o, m) * o.C + cell_index(o, o.x[j], o.y[j], o.z[j])] += 1u;
  }
  for (uint64_t c = 0; c < o.n_chains; ++c)
    for (uint32_t i = 0; i < chain_len(o, c); ++i) {
      const uint64_t j = chain_bead0(o, c) + i;
      const uint64_t cell = cell_index(o, o.x[j], o.y[j], o.z[j]);
      o.counts[(size_t)bead_type(o, c, i) * o.C + cell] += 1u;
    }
}

// DESIGN.md section 2 step 3 (NS part 3; R2 formula):
//   phi_s(c) = n_s(c) * C/B;  omega_t(c) = (1/N) * ( kappaN*(sum_s phi_s - 1) + sum_{s != t} chiN_ts * phi_s ).
// With an external field ("umbrella potential"; R21):
//   omega_t(c) = fl32( fl32(invN * acc) + ext_t(c) ),  ext in kT per bead.
// With the umbrella potential toward target concentrations phi*_t(c) ("equilibrated using an
// umbrella potential"; R25: H_umb/kT = (k/2)(B/C) sum_{t,c} (phi_t(c) - phi*_t(c))^2, whose
// derivative with respect to n_t(c) is k (phi_t(c) - phi*_t(c))), added last:
//   omega_t(c) = fl32( omega_t(c) + fl32( k * fl32(phi_t(c) - phi*_t(c)) ) ).
void compute_omega(Oracle& o) {
  std::vector<float> phi(o.T);
  for (uint64_t c = 0; c < o.C; ++c) {
    float tot = 0.0f;
    for (uint32_t s = 0; s < o.T; ++s) {
      phi[s] = (float)o.counts[(size_t)s * o.C + c] * o.dens_scale;
      tot = (s == 0) ? phi[0] : (tot + phi[s]);
    }
    const float p = o.kappaN * (tot - 1.0f);
    for (uint32_t t = 0; t < o.T; ++t) {
      float acc = p;
      for (uint32_t s = 0; s < o.T; ++s)
        if (s != t) acc = fmaf(o.chiN[(size_t)t * o.T + s], phi[s], acc);
      float w = o.invN * acc;
      if (!o.ext.empty()) w = w + o.ext[(size_t)t * o.C + c];
      if (!o.phi_target.empty()) w = w + o.umbrella_k * (phi[t] - o.phi_target[(size_t)t * o.C + c]);
      o.omega[(size_t)t * o.C + c] = w;
    }
  }
}

// Squared bond length with the pinned operation order (DESIGN.md section 2 step 5.4).
inline float bond_sq(float ax, float ay, float az, float bx, float by, float bz) {
  const float sx = ax - bx, sy = ay - by, sz = az - bz;
  return fmaf(sz, sz, fmaf(sy, sy, sx * sx));
}

// Delta E (in kT) of moving bead (c, i) from its current position to (nx, ny, nz):
// DESIGN.md section 2 steps 5.4-5.5 (NS: "harmonic bond energy plus the bead type's
// quasi-instantaneous field omega at its grid cell").
inline float delta_energy(const Oracle& o, uint64_t c, uint32_t i, float nx, float ny, float nz) {
  const uint64_t j = chain_bead0(o, c) + i;
  const float rx = o.x[j], ry = o.y[j], rz = o.z[j];
  float dq = 0.0f;
  bool have = false;
  if (i > 0) {                                          // neighbour i-1 first
    const uint64_t k = j - 1;
    const float q_old = bond_sq(rx, ry, rz, o.x[k], o.y[k], o.z[k]);
    const float q_new = bond_sq(nx, ny, nz, o.x[k], o.y[k], o.z[k]);
    dq = q_new - q_old;
    have = true;
  }
  if (i + 1 < chain_len(o, c)) {                                    // then neighbour i+1
    const uint64_t k = j + 1;
    const float q_old = bond_sq(rx, ry, rz, o.x[k], o.y[k], o.z[k]);
    const float q_new = bond_sq(nx, ny, nz, o.x[k], o.y[k], o.z[k]);
    const float dqk = q_new - q_old;
    dq = have ? (dq + dqk) : dqk;
  }
  const size_t tb = (size_t)bead_type(o, c, i) * o.C;
  const float dw = o.omega[tb + cell_index(o, nx, ny, nz)] - o.omega[tb + cell_index(o, rx, ry, rz)];
  return fmaf(o.kb, dq, dw);
}

// The same Delta E in double from the same fp32 inputs: used only to classify near-threshold
// moves for the GPU-vs-oracle mismatch rule (NS: "|dE + ln u| < 1e-4 kT").
inline double delta_energy_f64(const Oracle& o, uint64_t c, uint32_t i, float nx, float ny, float nz) {
  const uint64_t j = chain_bead0(o, c) + i;
  const double r[3] = {o.x[j], o.y[j], o.z[j]}, n[3] = {nx, ny, nz};
  double dq = 0.0;
  for (int side = 0; side < 2; ++side) {
    if (side == 0 && i == 0) continue;
    if (side == 1 && i + 1 >= chain_len(o, c)) continue;
    const uint64_t k = side == 0 ? j - 1 : j + 1;
    const double nb[3] = {o.x[k], o.y[k], o.z[k]};
    double qo = 0.0, qn = 0.0;
    for (int d = 0; d < 3; ++d) {
      qo += (r[d] - nb[d]) * (r[d] - nb[d]);
      qn += (n[d] - nb[d]) * (n[d] - nb[d]);
    }
    dq += qn - qo;
  }
  const size_t tb = (size_t)bead_type(o, c, i) * o.C;
  const double dw = (double)o.omega[tb + cell_index(o, nx, ny, nz)] -
                    (double)o.omega[tb + cell_index(o, (float)r[0], (float)r[1], (float)r[2])];
  return (double)o.kb * dq + dw;
}

// ---- standard normal deviates with no library function in them (R24) -------------------
// Box-Muller in fp32 from U = ((w >> 9) + 0.5) 2^-23 (exact in fp32), with the logarithm and the
// sine / cosine written out as fixed sequences of IEEE fp32 operations (+, *, /, fma, sqrt), so that
// any conforming implementation produces the same bits.  Accuracy ~2e-7, the resolution of the fp32
// positions the deviates are added to.
inline float det_log(float x) {                         // x in (0, 1]
  uint32_t bits; std::memcpy(&bits, &x, 4);
  int e = (int)((bits >> 23) & 0xff) - 127;
  bits = (bits & 0x007fffffu) | 0x3f800000u;
  float m; std::memcpy(&m, &bits, 4);                   // m in [1, 2)
  if (m > 1.41421354f) { m = m * 0.5f; e += 1; }        // m in (sqrt 1/2, sqrt 2]
  const float sq = (m - 1.0f) / (m + 1.0f), z = sq * sq; // log m = 2 atanh(sq) = 2 sq (1 + z/3 + z^2/5 + ...)
  float p = 1.0f / 11.0f;
  p = fmaf(p, z, 1.0f / 9.0f); p = fmaf(p, z, 1.0f / 7.0f); p = fmaf(p, z, 1.0f / 5.0f); p = fmaf(p, z, 1.0f / 3.0f);
  const float lm = fmaf(2.0f * sq, z * p, 2.0f * sq);
  return fmaf((float)e, 0.693147182f, lm);
}
inline void det_sincos_2pi(float u, float* sn, float* cs) {   // sin, cos of 2 pi u, u in (0, 1)
  const float t = u * 4.0f;                              // quarter turns
  const float k = floorf(t + 0.5f);
  const float r = (t - k) * 1.57079637f, z = r * r;      // r in [-pi/4, pi/4]
  float ps = 1.0f / 362880.0f;                           // sin r = r (1 - z/3! + z^2/5! - z^3/7! + z^4/9!)
  ps = fmaf(ps, z, -1.0f / 5040.0f); ps = fmaf(ps, z, 1.0f / 120.0f); ps = fmaf(ps, z, -1.0f / 6.0f);
  const float s0 = fmaf(r * z, ps, r);
  float pc = -1.0f / 3628800.0f;                         // cos r = 1 - z/2! + z^2/4! - z^3/6! + z^4/8! - z^5/10!
  pc = fmaf(pc, z, 1.0f / 40320.0f); pc = fmaf(pc, z, -1.0f / 720.0f); pc = fmaf(pc, z, 1.0f / 24.0f); pc = fmaf(pc, z, -0.5f);
  const float c0 = fmaf(pc, z, 1.0f);
  const int q = (int)k & 3;                              // rotate by k quarter turns
  *sn = q == 0 ? s0 : q == 1 ? c0 : q == 2 ? -s0 : -c0;
  *cs = q == 0 ? c0 : q == 1 ? -s0 : q == 2 ? -c0 : s0;
}
inline float unit23(uint32_t w) { return ((float)(w >> 9) + 0.5f) * 0x1p-23f; }
// xi[0..2] of a move from the words of its two Philox calls (domain 0: w, domain 2: v)
inline void smc_deviates(const uint32_t* w, const uint32_t* v, float* xi) {
  float sn, cs, sn2, cs2;
  const float ra = sqrtf(-2.0f * det_log(unit23(w[0])));
  det_sincos_2pi(unit23(w[1]), &sn, &cs);
  const float rb = sqrtf(-2.0f * det_log(unit23(v[0])));
  det_sincos_2pi(unit23(v[1]), &sn2, &cs2);
  xi[0] = ra * cs; xi[1] = ra * sn; xi[2] = rb * cs2;
}

// Bond-force-biased ("smart Monte Carlo") trial move of bead (c, i), R24 (PAPER.md:41, :77:
// "bond-force-biased Monte-Carlo", "biased trial moves").  S = sum over the bonded neighbours of
// (r - r_j) (i-1 first), so the bonded force is F = -2 kb S.  Proposal r' = r + A F + sqrt(2A) xi:
//   dr_d = fma(-gA, S_d, sq2A * xi_d),  r'_d = r_d + dr_d,  gA = fl(A * fl(2 kb)).
// With S' the same sum at r', qf = |dr + gA S|^2 (forward), qr = |dr - gA S'|^2 (reverse), each
// fma(z,z, fma(y,y, x*x)); margin m = fma(inv4A, qr - qf, dE) + lnu, dE as for uniform moves; accept iff m <= 0.
// xi_0, xi_1 = fp32 Box-Muller pair of words (w0, w1) of the move's Philox call (domain 0); xi_2 = cosine
// member of the pair of words (v0, v1) of a second call with domain 2; u from w3 as before.
inline int trial_move_smc(Oracle& o, uint64_t c, uint32_t i, uint32_t parity, double* margin64) {
  const uint32_t hi = (uint32_t)(o.t >> 32) << 16;
  const uint32_t ctr[4] = {i, (uint32_t)c, (uint32_t)o.t, parity | (RNG_DOMAIN_MOVE << 8) | hi};
  const uint32_t ctr2[4] = {i, (uint32_t)c, (uint32_t)o.t, parity | (2u << 8) | hi};
  const uint32_t key[2] = {(uint32_t)o.seed, (uint32_t)(o.seed >> 32)};
  uint32_t w[4], v[4];
  philox4x32_10(ctr, key, w);
  philox4x32_10(ctr2, key, v);
  float xi[3];
  smc_deviates(w, v, xi);
  const float u = umap(w[3]);
  const uint64_t j = chain_bead0(o, c) + i;
  const float r[3] = {o.x[j], o.y[j], o.z[j]};
  float S[3] = {0.0f, 0.0f, 0.0f};
  bool have = false;
  for (int side = 0; side < 2; ++side) {
    if (side == 0 && i == 0) continue;
    if (side == 1 && i + 1 >= chain_len(o, c)) continue;
    const uint64_t k = side == 0 ? j - 1 : j + 1;
    const float s3[3] = {r[0] - o.x[k], r[1] - o.y[k], r[2] - o.z[k]};
    for (int d = 0; d < 3; ++d) S[d] = have ? S[d] + s3[d] : s3[d];
    have = true;
  }
  float dr[3], n[3];
  for (int d = 0; d < 3; ++d) { dr[d] = fmaf(-o.gA, S[d], o.sq2A * xi[d]); n[d] = r[d] + dr[d]; }
  float S2[3] = {0.0f, 0.0f, 0.0f};
  have = false;
  for (int side = 0; side < 2; ++side) {
    if (side == 0 && i == 0) continue;
    if (side == 1 && i + 1 >= chain_len(o, c)) continue;
    const uint64_t k = side == 0 ? j - 1 : j + 1;
    const float s3[3] = {n[0] - o.x[k], n[1] - o.y[k], n[2] - o.z[k]};
    for (int d = 0; d < 3; ++d) S2[d] = have ? S2[d] + s3[d] : s3[d];
    have = true;
  }
  float a[3], b_[3];
  for (int d = 0; d < 3; ++d) { a[d] = fmaf(o.gA, S[d], dr[d]); b_[d] = fmaf(-o.gA, S2[d], dr[d]); }
  const float qf = fmaf(a[2], a[2], fmaf(a[1], a[1], a[0] * a[0]));
  const float qr = fmaf(b_[2], b_[2], fmaf(b_[1], b_[1], b_[0] * b_[0]));
  const float dE = delta_energy(o, c, i, n[0], n[1], n[2]);
  const float meff = fmaf(o.inv4A, qr - qf, dE);
  const float m = meff + lnu32(u);
  if (margin64)
    *margin64 = delta_energy_f64(o, c, i, n[0], n[1], n[2]) + ((double)qr - (double)qf) * (double)o.inv4A + std::log((double)u);
  if (m <= 0.0f) { o.x[j] = n[0]; o.y[j] = n[1]; o.z[j] = n[2]; return 1; }
  return 0;
}

// One Metropolis trial move of bead (c, i) (DESIGN.md section 2 step 5).  Returns 1 if accepted.
inline int trial_move(Oracle& o, uint64_t c, uint32_t i, uint32_t parity, double* margin64) {
  if (o.smcA > 0.0f) return trial_move_smc(o, c, i, parity, margin64);
  const uint32_t ctr[4] = {i, (uint32_t)c, (uint32_t)o.t,
                           parity | (RNG_DOMAIN_MOVE << 8) | ((uint32_t)(o.t >> 32) << 16)};
  const uint32_t key[2] = {(uint32_t)o.seed, (uint32_t)(o.seed >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  const float dx = o.a * tmap(w[0]);
  const float dy = o.a * tmap(w[1]);
  const float dz = o.a * tmap(w[2]);
  const float u = umap(w[3]);
  const uint64_t j = chain_bead0(o, c) + i;
  const float nx = o.x[j] + dx, ny = o.y[j] + dy, nz = o.z[j] + dz;
  const float dE = delta_energy(o, c, i, nx, ny, nz);
  const float m = dE + lnu32(u);
  if (margin64) *margin64 = delta_energy_f64(o, c, i, nx, ny, nz) + std::log((double)u);
  if (m <= 0.0f) {                                      // R6: accept iff dE + ln u <= 0
    o.x[j] = nx; o.y[j] = ny; o.z[j] = nz;
    return 1;
  }
  return 0;
}

// The move of single-bead molecule m (R23): bead index 0 of logical chain n_chains + m, in
// half-sweep 0; no bonds, so dE = fma(kb, 0, dw) = dw = omega_t(new cell) - omega_t(old cell).
inline int trial_move_single(Oracle& o, uint64_t m, double* margin64) {
  const uint32_t ctr[4] = {0u, (uint32_t)(o.n_chains + m), (uint32_t)o.t,
                           0u | (RNG_DOMAIN_MOVE << 8) | ((uint32_t)(o.t >> 32) << 16)};
  const uint32_t key[2] = {(uint32_t)o.seed, (uint32_t)(o.seed >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  const uint64_t j = o.NB + m;
  const float nx = o.x[j] + o.a * tmap(w[0]), ny = o.y[j] + o.a * tmap(w[1]), nz = o.z[j] + o.a * tmap(w[2]);
  const float u = umap(w[3]);
  const size_t tb = (size_t)single_type(o, m) * o.C;
  const float w_new = o.omega[tb + cell_index(o, nx, ny, nz)], w_old = o.omega[tb + cell_index(o, o.x[j], o.y[j], o.z[j])];
  const float dE = fmaf(o.kb, 0.0f, w_new - w_old);
  const float mg = dE + lnu32(u);
  if (margin64) *margin64 = ((double)w_new - (double)w_old) + std::log((double)u);
  if (mg <= 0.0f) { o.x[j] = nx; o.y[j] = ny; o.z[j] = nz; return 1; }
  return 0;
}

// order: 0 ascending, 1 descending, 2 = caller-supplied permutation of the same-parity bead list
// (R5: same-parity beads of a linear chain share no bond and omega is frozen, so the
// visiting order within a half-sweep is immaterial; tests check that bit for bit).
uint64_t half_sweep(Oracle& o, uint32_t parity, int order, const uint64_t* perm, uint64_t n_perm,
                    uint8_t* accept_mask, double* margins) {
  uint64_t accepted = 0;
  if (order == 2) {
    for (uint64_t k = 0; k < n_perm; ++k) {
      const uint64_t j = perm[k];
      if (j >= o.NB) {                       // a single-bead molecule: half-sweep 0 only
        if (parity != 0) continue;
        const int acc = trial_move_single(o, j - o.NB, margins ? &margins[j] : nullptr);
        if (accept_mask) accept_mask[j] = (uint8_t)acc;
        accepted += (uint64_t)acc;
        continue;
      }
      uint64_t c;
      uint32_t i;
      bead_to_chain(o, j, &c, &i);
      if ((i & 1u) != parity) continue;
      const int acc = trial_move(o, c, i, parity, margins ? &margins[j] : nullptr);
      if (accept_mask) accept_mask[j] = (uint8_t)acc;
      accepted += (uint64_t)acc;
    }
    return accepted;
  }
  for (uint64_t cc = 0; cc < o.n_chains; ++cc) {
    const uint64_t c = order == 0 ? cc : o.n_chains - 1 - cc;
    const uint32_t n_par = (chain_len(o, c) + 1u - parity) / 2u;    // beads i = parity, parity+2, ... < N
    for (uint32_t kk = 0; kk < n_par; ++kk) {
      const uint32_t k = order == 0 ? kk : n_par - 1 - kk;
      const uint32_t i = parity + 2u * k;
      const uint64_t j = chain_bead0(o, c) + i;
      const int acc = trial_move(o, c, i, parity, margins ? &margins[j] : nullptr);
      if (accept_mask) accept_mask[j] = (uint8_t)acc;
      accepted += (uint64_t)acc;
    }
  }
  if (parity == 0)
    for (uint64_t mm = 0; mm < o.S; ++mm) {
      const uint64_t m = order == 0 ? mm : o.S - 1 - mm;
      const uint64_t j = o.NB + m;
      const int acc = trial_move_single(o, m, margins ? &margins[j] : nullptr);
      if (accept_mask) accept_mask[j] = (uint8_t)acc;
      accepted += (uint64_t)acc;
    }
  return accepted;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C ABI of the oracle (its own; unrelated to include/soma.h).
// ---------------------------------------------------------------------------------------------
extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  philox4x32_10(ctr, key, out);
}
float oracle_tmap(uint32_t w) { return tmap(w); }
float oracle_umap(uint32_t w) { return umap(w); }
float oracle_lnu(float u) { return lnu32(u); }
void oracle_lnu_array(const float* u, float* out, uint64_t n) {
  for (uint64_t k = 0; k < n; ++k) out[k] = lnu32(u[k]);
}

void* oracle_create(uint64_t n_chains, uint32_t N, uint32_t T, uint32_t n_patterns,
                    const uint8_t* type_patterns, const uint8_t* chain_pattern, float b,
                    const float* chiN, float kappaN, const uint32_t* grid, const float* box,
                    float move_halfwidth, uint64_t seed) {
  if (!n_chains || !N || !T || !n_patterns || !type_patterns || !chiN || !grid || !box) return nullptr;
  Oracle* o = new (std::nothrow) Oracle();
  if (!o) return nullptr;
  o->n_chains = n_chains; o->N = N; o->T = T; o->n_patterns = n_patterns;
  o->type_patterns.assign(type_patterns, type_patterns + (size_t)n_patterns * N);
  if (chain_pattern) o->chain_pattern.assign(chain_pattern, chain_pattern + n_chains);
  else o->chain_pattern.assign(n_chains, 0);
  o->b = b; o->kappaN = kappaN; o->a = move_halfwidth; o->seed = seed;
  o->chiN.assign(chiN, chiN + (size_t)T * T);
  for (int d = 0; d < 3; ++d) { o->grid[d] = grid[d]; o->box[d] = box[d]; }
  o->B = n_chains * N;
  o->NB = o->B;
  o->Nstride = N;
  o->species.assign(1, Oracle::Species{n_chains, 0, 0, N});
  o->C = (uint64_t)grid[0] * grid[1] * grid[2];
  o->kb = 1.5f / (b * b);
  for (int d = 0; d < 3; ++d) o->inv_h[d] = (float)grid[d] / box[d];
  o->dens_scale = (float)((double)o->C / (double)o->B);
  o->invN = 1.0f / (float)N;
  o->x.assign(o->B, 0.0f); o->y.assign(o->B, 0.0f); o->z.assign(o->B, 0.0f);
  o->counts.assign((size_t)T * o->C, 0u);
  o->omega.assign((size_t)T * o->C, 0.0f);
  o->t = 0; o->loaded = false;
  return o;
}

void oracle_destroy(void* h) { delete static_cast<Oracle*>(h); }

// DESIGN.md section 2 step 4: copy positions; t = step0; bin(); omega().
int oracle_load_state(void* h, const float* x, const float* y, const float* z, uint64_t step0) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(o.x.data(), x, o.B * sizeof(float));
  std::memcpy(o.y.data(), y, o.B * sizeof(float));
  std::memcpy(o.z.data(), z, o.B * sizeof(float));
  o.t = step0;
  bin(o);
  compute_omega(o);
  o.loaded = true;
  return 0;
}

// DESIGN.md section 2 step 6 (NS): half_sweep(0); half_sweep(1); bin(); omega(); t += 1.
uint64_t oracle_mc_steps(void* h, uint32_t n_steps) {
  Oracle& o = *static_cast<Oracle*>(h);
  uint64_t accepted = 0;
  for (uint32_t s = 0; s < n_steps; ++s) {
    accepted += half_sweep(o, 0, 0, nullptr, 0, nullptr, nullptr);
    accepted += half_sweep(o, 1, 0, nullptr, 0, nullptr, nullptr);
    bin(o);
    compute_omega(o);
    o.t += 1;
  }
  return accepted;
}

// Pieces of a step, for lock-step comparison and for frozen-field tests.
uint64_t oracle_half_sweep(void* h, uint32_t parity, int order, const uint64_t* perm, uint64_t n_perm,
                           uint8_t* accept_mask, double* margins) {
  return half_sweep(*static_cast<Oracle*>(h), parity, order, perm, n_perm, accept_mask, margins);
}
void oracle_bin(void* h) { bin(*static_cast<Oracle*>(h)); }
void oracle_compute_omega(void* h) { compute_omega(*static_cast<Oracle*>(h)); }
void oracle_finish_step(void* h) {
  Oracle& o = *static_cast<Oracle*>(h);
  bin(o); compute_omega(o); o.t += 1;
}

void oracle_get_positions(void* h, float* x, float* y, float* z) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(x, o.x.data(), o.B * sizeof(float));
  std::memcpy(y, o.y.data(), o.B * sizeof(float));
  std::memcpy(z, o.z.data(), o.B * sizeof(float));
}
// Overwrite the positions of selected beads (lock-step resynchronisation after a legal flip).
void oracle_set_beads(void* h, const uint64_t* idx, uint64_t n, const float* x, const float* y, const float* z) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (uint64_t k = 0; k < n; ++k) { o.x[idx[k]] = x[k]; o.y[idx[k]] = y[k]; o.z[idx[k]] = z[k]; }
}
void oracle_get_density(void* h, uint32_t* counts) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(counts, o.counts.data(), o.counts.size() * sizeof(uint32_t));
}
void oracle_set_density(void* h, const uint32_t* counts) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(o.counts.data(), counts, o.counts.size() * sizeof(uint32_t));
}
void oracle_get_omega(void* h, float* omega) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(omega, o.omega.data(), o.omega.size() * sizeof(float));
}
void oracle_set_omega(void* h, const float* omega) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(o.omega.data(), omega, o.omega.size() * sizeof(float));
}
uint64_t oracle_get_step(void* h) { return static_cast<Oracle*>(h)->t; }
// move type: A > 0 = bond-force-biased moves with mobility A (R24), 0 = uniform moves
void oracle_set_smc(void* h, float A) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.smcA = A;
  o.gA = A * (2.0f * o.kb);
  o.sq2A = (float)std::sqrt(2.0 * (double)A);
  o.inv4A = A > 0.0f ? (float)(1.0 / (4.0 * (double)A)) : 0.0f;
}
// the normal deviates of a move, for the tests: out[0..2] = xi, out[3] = u
void oracle_smc_draws(void* h, uint64_t c, uint32_t i, uint32_t parity, double* out) {
  Oracle& o = *static_cast<Oracle*>(h);
  const uint32_t hi = (uint32_t)(o.t >> 32) << 16;
  const uint32_t ctr[4] = {i, (uint32_t)c, (uint32_t)o.t, parity | hi}, ctr2[4] = {i, (uint32_t)c, (uint32_t)o.t, parity | (2u << 8) | hi};
  const uint32_t key[2] = {(uint32_t)o.seed, (uint32_t)(o.seed >> 32)};
  uint32_t w[4], v[4];
  philox4x32_10(ctr, key, w); philox4x32_10(ctr2, key, v);
  float xi[3];
  smc_deviates(w, v, xi);
  out[0] = xi[0]; out[1] = xi[1]; out[2] = xi[2]; out[3] = (double)umap(w[3]);
}
// fma(inv4A, qr - qf, dE) of moving bead `bead` to (nx, ny, nz): the bond-force-biased margin without ln u
float oracle_smc_margin(void* h, uint64_t bead, float nx, float ny, float nz) {
  Oracle& o = *static_cast<Oracle*>(h);
  const uint64_t j = bead;
  uint64_t c;
  uint32_t i;
  bead_to_chain(o, bead, &c, &i);
  const float r[3] = {o.x[j], o.y[j], o.z[j]}, n[3] = {nx, ny, nz};
  float S[3] = {0, 0, 0}, S2[3] = {0, 0, 0};
  bool have = false;
  for (int side = 0; side < 2; ++side) {
    if (side == 0 && i == 0) continue;
    if (side == 1 && i + 1 >= chain_len(o, c)) continue;
    const uint64_t k = side == 0 ? j - 1 : j + 1;
    const float nb[3] = {o.x[k], o.y[k], o.z[k]};
    for (int d = 0; d < 3; ++d) {
      S[d] = have ? S[d] + (r[d] - nb[d]) : r[d] - nb[d];
      S2[d] = have ? S2[d] + (n[d] - nb[d]) : n[d] - nb[d];
    }
    have = true;
  }
  float a[3], b_[3];
  for (int d = 0; d < 3; ++d) { const float dr = n[d] - r[d]; a[d] = fmaf(o.gA, S[d], dr); b_[d] = fmaf(-o.gA, S2[d], dr); }
  const float qf = fmaf(a[2], a[2], fmaf(a[1], a[1], a[0] * a[0]));
  const float qr = fmaf(b_[2], b_[2], fmaf(b_[1], b_[1], b_[0] * b_[0]));
  return fmaf(o.inv4A, qr - qf, delta_energy(o, c, i, nx, ny, nz));
}
void oracle_det_functions(double x, double* out) {       // out = {det_log(x), sin(2 pi x), cos(2 pi x)}, fp32 routines
  float sn, cs;
  out[0] = det_log((float)x);
  det_sincos_2pi((float)x, &sn, &cs);
  out[1] = sn; out[2] = cs;
}
// the same for n arguments at once (test plumbing: lets the pin visit every argument the deviates can take)
void oracle_det_functions_n(const float* x, uint64_t n, float* lg, float* sn, float* cs) {
  for (uint64_t k = 0; k < n; ++k) {
    lg[k] = det_log(x[k]);
    det_sincos_2pi(x[k], &sn[k], &cs[k]);
  }
}

// single-bead molecules: n_single[T] (call right after oracle_create, before any state is loaded)
int oracle_set_singles(void* h, const uint64_t* n_single) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.n_single.assign(n_single, n_single + o.T);
  o.S = 0;
  for (uint32_t t = 0; t < o.T; ++t) o.S += o.n_single[t];
  if (o.n_chains + o.S >= (1ull << 32)) return -1;
  o.B = o.NB + o.S;
  o.dens_scale = (float)((double)o.C / (double)o.B);
  o.x.assign(o.B, 0.0f); o.y.assign(o.B, 0.0f); o.z.assign(o.B, 0.0f);
  o.loaded = false;
  return 0;
}

// Polymer species of different chain lengths (SURVEY section 8(f) row f2 "mixed chain lengths"; PAPER.md:39, :133:
// polymer, solvent and non-solvent in one system; R26): species s has n[s] chains of N[s] beads; the
// chains are numbered and stored species by species (species 0 first), bead i of chain c at
// bead_off(species) + (c - first_chain(species)) N[s] + i; a chain of N[s] beads takes the first N[s] entries of
// its pattern row (rows have the length given at oracle_create, >= max N[s]); 1/N in omega and the N of chiN,
// kappaN stay the reference length N_ref (R3).  Call right after oracle_create (before oracle_set_singles).
int oracle_set_species(void* h, uint32_t n_species, const uint64_t* n, const uint32_t* N, uint32_t N_ref) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!n_species || !N_ref) return -1;
  o.species.clear();
  uint64_t chains = 0, beads = 0;
  for (uint32_t s = 0; s < n_species; ++s) {
    if (!n[s] || !N[s] || N[s] > o.Nstride) return -1;
    o.species.push_back(Oracle::Species{n[s], chains, beads, N[s]});
    chains += n[s];
    beads += n[s] * N[s];
  }
  if (chains != o.n_chains) return -1;
  o.N = N_ref;
  o.invN = 1.0f / (float)N_ref;
  o.NB = beads;
  o.B = beads + o.S;
  o.dens_scale = (float)((double)o.C / (double)o.B);
  o.x.assign(o.B, 0.0f); o.y.assign(o.B, 0.0f); o.z.assign(o.B, 0.0f);
  o.loaded = false;
  return 0;
}

// external field [T][C] (nullptr = none); omega is recomputed from the current densities
void oracle_set_external_field(void* h, const float* ext) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (ext) o.ext.assign(ext, ext + (size_t)o.T * o.C); else o.ext.clear();
  if (o.loaded) compute_omega(o);
}
// Initial state on the device's recipe ("generating bead
// coordinates"; R22, the configs' "Gaussian random-walk chains, bond components ~N(0, b^2/3),
// first bead uniform in the box"): for chain c, bead i draw (w0..w3) = Philox4x32-10(counter =
// (i, c, 0, 1 << 8), key = gen_seed)  -- domain 1, so no draw collides with a Monte-Carlo move's --
// and U(w) = (w + 0.5) 2^-32 in double.  Bead 0: r_d = box_d * U(w_d).  Bead i >= 1: Box-Muller,
// g0 = sqrt(-2 ln U(w0)) cos(2 pi U(w1)), g1 = the same with sin, g2 = sqrt(-2 ln U(w2)) cos(2 pi U(w3));
// r_d(i) = r_d(i-1) + (b / sqrt 3) g_d, accumulated in double; every stored coordinate is the double
// rounded once to fp32.  Then DESIGN.md section 2 step 4 with these positions.
int oracle_generate_state(void* h, uint64_t gen_seed, uint64_t step0) {
  Oracle& o = *static_cast<Oracle*>(h);
  const uint32_t key[2] = {(uint32_t)gen_seed, (uint32_t)(gen_seed >> 32)};
  const double sigma = (double)o.b / std::sqrt(3.0), two_pi = 6.283185307179586;
  auto U = [](uint32_t w) { return ((double)w + 0.5) * 0x1p-32; };
  for (uint64_t c = 0; c < o.n_chains; ++c) {
    double r[3] = {0.0, 0.0, 0.0};
    for (uint32_t i = 0; i < chain_len(o, c); ++i) {
      const uint32_t ctr[4] = {i, (uint32_t)c, 0u, 1u << 8};
      uint32_t w[4];
      philox4x32_10(ctr, key, w);
      if (i == 0) {
        for (int d = 0; d < 3; ++d) r[d] = (double)o.box[d] * U(w[d]);
      } else {
        const double ra = std::sqrt(-2.0 * std::log(U(w[0]))), rb = std::sqrt(-2.0 * std::log(U(w[2])));
        r[0] += sigma * (ra * std::cos(two_pi * U(w[1])));
        r[1] += sigma * (ra * std::sin(two_pi * U(w[1])));
        r[2] += sigma * (rb * std::cos(two_pi * U(w[3])));
      }
      const uint64_t j = chain_bead0(o, c) + i;
      o.x[j] = (float)r[0]; o.y[j] = (float)r[1]; o.z[j] = (float)r[2];
    }
  }
  for (uint64_t m = 0; m < o.S; ++m) {                 // single-bead molecules: the bead-0 rule with chain id n_chains + m
    const uint32_t ctr[4] = {0u, (uint32_t)(o.n_chains + m), 0u, 1u << 8};
    uint32_t w[4];
    philox4x32_10(ctr, key, w);
    const uint64_t j = o.NB + m;
    o.x[j] = (float)((double)o.box[0] * U(w[0]));
    o.y[j] = (float)((double)o.box[1] * U(w[1]));
    o.z[j] = (float)((double)o.box[2] * U(w[2]));
  }
  o.t = step0;
  bin(o);
  compute_omega(o);
  o.loaded = true;
  return 0;
}

// Umbrella potential toward target concentrations (R25): phi_target [T][C] (nullptr = off).
// omega of the current densities is recomputed at once.
void oracle_set_umbrella(void* h, const float* phi_target, float k) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (phi_target) o.phi_target.assign(phi_target, phi_target + (size_t)o.T * o.C); else o.phi_target.clear();
  o.umbrella_k = phi_target ? k : 0.0f;
  if (o.loaded) compute_omega(o);
}

// Initial state that reproduces supplied concentration fields (PAPER.md:119:
// "Each SOMA simulation begins by generating particle positions that reproduce the supplied concentration
// fields.  Molecules are placed within half a mean end-to-end distance of their target positions").  The
// paper gives no rule; R25 is the reading:
//   Q_t(c) = (uint32) rintf(phi*_t(c) * 65536)                       target concentration on a 2^-16 lattice
//   W_p(c) = sum_i Q_{type_p(i)}(c)                                  weight of cell c for a chain of pattern p (uint64)
//   chain c (pattern p): (w0..w3) = Philox(counter (0, c, 0, 3<<8), key = gen_seed),  (v0..) = Philox((1, c, 0, 3<<8));
//     k = floor( (w0 2^32 + w1) S_p / 2^64 ), S_p = sum_c W_p(c);  target cell = the first cell whose inclusive
//     prefix sum of W_p exceeds k, i.e. cell c with probability W_p(c)/S_p;  target point r* = (cell
//     coordinate + (U(w2), U(w3), U(v0))) * (box/grid) in double, U(w) = (w + 0.5) 2^-32;
//     shape = the Gaussian random walk of DESIGN.md R22 (same domain-1 draws: s_0 = 0, s_i = s_{i-1} + (b/sqrt 3) g(i));
//     m = (s_0 + s_1 + ... in bead order)/N;  bead i = (float)((r* - m) + s_i): the chain's centre of mass sits at
//     its target point, so every bead is within about R_e/2 of it.
//   single-bead molecule m of type t: the same with W = Q_t, chain id n_chains + m, placed at r*.
// Then DESIGN.md section 2 step 4 with these positions (t = step0).  Returns -1 if a target value is negative,
// NaN or >= 65536, -2 if a pattern (or single species) that has molecules has zero total weight.
int oracle_init_from_density(void* h, const float* phi_target, uint64_t gen_seed, uint64_t step0) {
  Oracle& o = *static_cast<Oracle*>(h);
  const uint32_t key[2] = {(uint32_t)gen_seed, (uint32_t)(gen_seed >> 32)};
  const double sigma = (double)o.b / std::sqrt(3.0), two_pi = 6.283185307179586;
  auto U = [](uint32_t w) { return ((double)w + 0.5) * 0x1p-32; };
  std::vector<uint32_t> Q((size_t)o.T * o.C);
  for (size_t k = 0; k < Q.size(); ++k) {
    const float v = phi_target[k];
    if (!(v >= 0.0f) || !(v < 65536.0f)) return -1;
    Q[k] = (uint32_t)rintf(v * 65536.0f);
  }
  const double hcell[3] = {(double)o.box[0] / (double)o.grid[0], (double)o.box[1] / (double)o.grid[1], (double)o.box[2] / (double)o.grid[2]};
  std::vector<uint64_t> prefix(o.C);
  // target point of molecule `id` drawn from the cell weights whose inclusive prefix sums are in `prefix`
  auto target_point = [&](uint64_t id, double* rstar) {
    const uint32_t ca[4] = {0u, (uint32_t)id, 0u, 3u << 8}, cb[4] = {1u, (uint32_t)id, 0u, 3u << 8};
    uint32_t w[4], v[4];
    philox4x32_10(ca, key, w); philox4x32_10(cb, key, v);
    const uint64_t u64 = ((uint64_t)w[0] << 32) | w[1];
    const uint64_t k = (uint64_t)(((unsigned __int128)u64 * prefix[o.C - 1]) >> 64);
    uint64_t lo = 0, hi = o.C - 1;                        // first cell with prefix > k
    while (lo < hi) { const uint64_t mid = (lo + hi) / 2; if (prefix[mid] > k) hi = mid; else lo = mid + 1; }
    const uint64_t iz = lo % o.grid[2], iy = (lo / o.grid[2]) % o.grid[1], ix = lo / ((uint64_t)o.grid[2] * o.grid[1]);
    rstar[0] = ((double)ix + U(w[2])) * hcell[0];
    rstar[1] = ((double)iy + U(w[3])) * hcell[1];
    rstar[2] = ((double)iz + U(v[0])) * hcell[2];
  };
  std::vector<double> sx(o.Nstride), sy(o.Nstride), sz(o.Nstride);
  for (const Oracle::Species& sp : o.species)            // a chain's cell weights depend on its pattern and its length
  for (uint32_t p = 0; p < o.n_patterns; ++p) {
    bool used = false;
    for (uint64_t c = sp.first_chain; c < sp.first_chain + sp.n && !used; ++c) used = o.chain_pattern[c] == p;
    if (!used) continue;
    uint64_t run = 0;
    for (uint64_t c = 0; c < o.C; ++c) {
      uint64_t wgt = 0;
      for (uint32_t i = 0; i < sp.N; ++i) wgt += Q[(size_t)o.type_patterns[(size_t)p * o.Nstride + i] * o.C + c];
      run += wgt;
      prefix[c] = run;
    }
    if (run == 0) return -2;
    for (uint64_t c = sp.first_chain; c < sp.first_chain + sp.n; ++c) {
      if (o.chain_pattern[c] != p) continue;
      double rstar[3];
      target_point(c, rstar);
      double r[3] = {0.0, 0.0, 0.0}, sum[3] = {0.0, 0.0, 0.0};
      for (uint32_t i = 0; i < sp.N; ++i) {
        if (i > 0) {
          const uint32_t ctr[4] = {i, (uint32_t)c, 0u, 1u << 8};
          uint32_t w[4];
          philox4x32_10(ctr, key, w);
          const double ra = std::sqrt(-2.0 * std::log(U(w[0]))), rb = std::sqrt(-2.0 * std::log(U(w[2])));
          r[0] += sigma * (ra * std::cos(two_pi * U(w[1])));
          r[1] += sigma * (ra * std::sin(two_pi * U(w[1])));
          r[2] += sigma * (rb * std::cos(two_pi * U(w[3])));
        }
        sx[i] = r[0]; sy[i] = r[1]; sz[i] = r[2];
        sum[0] += r[0]; sum[1] += r[1]; sum[2] += r[2];
      }
      const double base[3] = {rstar[0] - sum[0] / (double)sp.N, rstar[1] - sum[1] / (double)sp.N, rstar[2] - sum[2] / (double)sp.N};
      for (uint32_t i = 0; i < sp.N; ++i) {
        const uint64_t j = chain_bead0(o, c) + i;
        o.x[j] = (float)(base[0] + sx[i]); o.y[j] = (float)(base[1] + sy[i]); o.z[j] = (float)(base[2] + sz[i]);
      }
    }
  }
  uint64_t m0 = 0;
  for (uint32_t t = 0; t < o.T && o.S; ++t) {
    if (o.n_single[t] == 0) continue;
    uint64_t run = 0;
    for (uint64_t c = 0; c < o.C; ++c) { run += Q[(size_t)t * o.C + c]; prefix[c] = run; }
    if (run == 0) return -2;
    for (uint64_t m = m0; m < m0 + o.n_single[t]; ++m) {
      double rstar[3];
      target_point(o.n_chains + m, rstar);
      const uint64_t j = o.NB + m;
      o.x[j] = (float)rstar[0]; o.y[j] = (float)rstar[1]; o.z[j] = (float)rstar[2];
    }
    m0 += o.n_single[t];
  }
  o.t = step0;
  bin(o);
  compute_omega(o);
  o.loaded = true;
  return 0;
}

// Validation of a state (the paper's "validation functions"):
// out[0] = coordinates that are NaN or infinite; out[1] = total of the density grids;
// out[2 + t] = beads of type t in the grids (t < 8); bond[0] = largest squared bond length (fp32, the
// pinned operation order of step 5.4), bond[1] = mean squared bond length (accumulated in double).
void oracle_validate(void* h, uint64_t* out, double* bond) {
  Oracle& o = *static_cast<Oracle*>(h);
  uint64_t bad = 0;
  for (uint64_t j = 0; j < o.B; ++j)
    bad += (std::isfinite(o.x[j]) ? 0 : 1) + (std::isfinite(o.y[j]) ? 0 : 1) + (std::isfinite(o.z[j]) ? 0 : 1);
  out[0] = bad;
  out[1] = 0;
  for (uint32_t t = 0; t < 8; ++t) out[2 + t] = 0;
  for (uint32_t t = 0; t < o.T; ++t)
    for (uint64_t c = 0; c < o.C; ++c) { out[2 + t] += o.counts[(size_t)t * o.C + c]; out[1] += o.counts[(size_t)t * o.C + c]; }
  float qmax = 0.0f;
  double qsum = 0.0;
  uint64_t nb = 0;
  for (uint64_t c = 0; c < o.n_chains; ++c)
    for (uint32_t i = 0; i + 1 < chain_len(o, c); ++i) {
      const uint64_t j = chain_bead0(o, c) + i;
      const float q = bond_sq(o.x[j], o.y[j], o.z[j], o.x[j + 1], o.y[j + 1], o.z[j + 1]);
      if (q > qmax) qmax = q;
      qsum += (double)q;
      ++nb;
    }
  bond[0] = (double)qmax;
  bond[1] = nb ? qsum / (double)nb : 0.0;
}

void oracle_set_step(void* h, uint64_t t) { static_cast<Oracle*>(h)->t = t; }

uint64_t oracle_cell_index(void* h, float x, float y, float z) {
  return cell_index(*static_cast<Oracle*>(h), x, y, z);
}
float oracle_delta_energy(void* h, uint64_t bead, float nx, float ny, float nz) {
  Oracle& o = *static_cast<Oracle*>(h);
  uint64_t c;
  uint32_t i;
  bead_to_chain(o, bead, &c, &i);
  return delta_energy(o, c, i, nx, ny, nz);
}
// The trial position and u that the move stream gives bead `bead` at the current step (no move made).
void oracle_trial(void* h, uint64_t bead, uint32_t parity, float* trial_xyz, float* u) {
  Oracle& o = *static_cast<Oracle*>(h);
  uint64_t c;
  uint32_t i;
  bead_to_chain(o, bead, &c, &i);
  const uint32_t ctr[4] = {i, (uint32_t)c, (uint32_t)o.t,
                           parity | (RNG_DOMAIN_MOVE << 8) | ((uint32_t)(o.t >> 32) << 16)};
  const uint32_t key[2] = {(uint32_t)o.seed, (uint32_t)(o.seed >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  trial_xyz[0] = o.x[bead] + o.a * tmap(w[0]);
  trial_xyz[1] = o.y[bead] + o.a * tmap(w[1]);
  trial_xyz[2] = o.z[bead] + o.a * tmap(w[2]);
  *u = umap(w[3]);
}
void oracle_get_constants(void* h, float* out5) {     // kb, inv_h[3], dens_scale  (+ invN in out5[5])
  Oracle& o = *static_cast<Oracle*>(h);
  out5[0] = o.kb; out5[1] = o.inv_h[0]; out5[2] = o.inv_h[1]; out5[3] = o.inv_h[2];
  out5[4] = o.dens_scale; out5[5] = o.invN;
}

}  // extern "C"
