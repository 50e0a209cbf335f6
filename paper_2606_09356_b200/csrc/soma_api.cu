// soma_api.cu -- host side of libsoma_b200.so: the C ABI of include/soma.h.
// Argument checking, device memory layout, launch sequencing.  All arithmetic of the Monte-Carlo
// step runs in the kernels of soma_kernels.cuh.
#include "../../include/soma.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "soma_lean.cuh"
#include "soma_init.cuh"

using namespace soma;

namespace {

thread_local char g_last_error[256] = "";

constexpr uint64_t kAlign = 256;
constexpr uint32_t kMaxSpecies = 16;
inline uint64_t align_up(uint64_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {            // byte offsets into the workspace
  uint64_t pos[2][3];      // two position sets (x,y,z): the live one and a staging / re-order target
  uint64_t counts[2];      // [T][C] uint32, double-buffered
  uint64_t omega;          // [T][C] fp32
  uint64_t ext;            // [T][C] fp32 external field (used once soma_set_external_field has set one)
  uint64_t phi_tgt;        // [T][C] fp32 target concentrations of soma_init_from_density (umbrella potential)
  uint64_t stage;          // [T][C] uint32 staging area: unpacked counters on their way to the caller
  uint64_t cdf;            // [C] uint64 prefix sums of the cell weights, then [C / kScanChunk + 2] chunk sums
  uint64_t single[3];      // [S] fp32 each: positions of the single-bead molecules (never re-ordered)
  uint64_t slot_chain[2];  // [n] uint32: logical chain id of every slot (second copy: re-order target)
  uint64_t slot_pattern[2];// [n] uint8
  uint64_t patterns;       // [n_patterns][N] uint8
  uint64_t pattern0;       // [n] uint8: pattern id of every chain in the caller's order
  uint64_t accepted;       // uint64
  uint64_t range_flag;     // uint32
  uint64_t validate;       // 11 x 8 bytes: report of soma_validate_state
  uint64_t sort_key;       // [n] uint32
  uint64_t sort_rank;      // [n] uint32
  uint64_t sort_bins;      // [n_bins + 1] uint32: bin counts, then (scanned) bin starts
  uint64_t total;
};

// coarse bins of the chain re-ordering: cubes of kSortBinEdge cells
constexpr uint32_t kSortBinEdge = 4;
uint64_t sort_bin_count(const uint32_t grid[3]) {
  uint64_t n = 1;
  for (int d = 0; d < 3; ++d) n *= (grid[d] + kSortBinEdge - 1) / kSortBinEdge;
  return n;
}

// n_bins: entries of the sort_bins array
Layout make_layout(uint64_t B, uint64_t n, uint64_t TC, uint64_t pat_bytes, uint64_t n_bins, uint64_t S, uint64_t cells) {
  Layout L{};
  uint64_t off = 0;
  for (int s = 0; s < 2; ++s)
    for (int d = 0; d < 3; ++d) { L.pos[s][d] = off; off += align_up(B * 4); }
  for (int s = 0; s < 2; ++s) { L.counts[s] = off; off += align_up(TC * 4); }
  L.omega = off; off += align_up(TC * 4);
  L.ext = off; off += align_up(TC * 4);
  L.phi_tgt = off; off += align_up(TC * 4);
  L.stage = off; off += align_up(TC * 4);
  L.cdf = off; off += align_up((cells + cells / 2048 + 4) * 8);
  for (int d = 0; d < 3; ++d) { L.single[d] = off; off += align_up(S * 4); }
  for (int s = 0; s < 2; ++s) { L.slot_chain[s] = off; off += align_up(n * 4); }
  for (int s = 0; s < 2; ++s) { L.slot_pattern[s] = off; off += align_up(n); }
  L.patterns = off; off += align_up(pat_bytes);
  L.pattern0 = off; off += align_up(n);
  L.accepted = off; off += align_up(8);
  L.range_flag = off; off += align_up(8);      // [0] position out of range, [1] a 16-bit density counter at its guard level
  L.validate = off; off += align_up(88);
  L.sort_key = off; off += align_up(n * 4);
  L.sort_rank = off; off += align_up(n * 4);
  L.sort_bins = off; off += align_up(n_bins * 4);
  L.total = off;
  return L;
}

bool is_pow2(uint32_t v) { return v && !(v & (v - 1)); }

// row length of type_patterns: the chain length, or the longest species' (R26)
uint32_t pattern_stride(const soma_params* p) {
  if (p->n_species <= 1) return p->beads_per_chain;
  uint32_t m = 0;
  for (uint32_t k = 0; k < p->n_species; ++k) m = p->species_beads[k] > m ? p->species_beads[k] : m;
  return m;
}
uint64_t chain_beads(const soma_params* p) {
  if (p->n_species <= 1) return p->n_chains * p->beads_per_chain;
  uint64_t b = 0;
  for (uint32_t k = 0; k < p->n_species; ++k) b += p->species_n_chains[k] * p->species_beads[k];
  return b;
}

const char* validate(const soma_params* p) {
  if (!p) return "params is NULL";
  if (p->n_chains == 0 || p->n_chains >= (1ull << 32)) return "n_chains must be in [1, 2^32)";
  if (p->beads_per_chain == 0 || p->beads_per_chain > 65535) return "beads_per_chain must be in [1, 65535]";
  if (p->n_types == 0 || p->n_types > (uint32_t)kMaxTypes) return "n_types must be in [1, 8]";
  if (p->n_patterns == 0 || p->n_patterns > 256) return "n_patterns must be in [1, 256]";
  if (p->reserved2 || p->reserved3 != 0.0f) return "reserved fields must be 0";
  if (p->n_species > 1) {
    if (p->n_species > kMaxSpecies) return "n_species must be <= 16";
    if (!p->species_n_chains || !p->species_beads) return "species_n_chains / species_beads is NULL but n_species > 1";
    uint64_t tot = 0;
    for (uint32_t k = 0; k < p->n_species; ++k) {
      if (p->species_n_chains[k] == 0 || p->species_n_chains[k] >= (1ull << 32)) return "species_n_chains[s] must be in [1, 2^32)";
      if (p->species_beads[k] == 0 || p->species_beads[k] > 65535) return "species_beads[s] must be in [1, 65535]";
      tot += p->species_n_chains[k];
    }
    if (tot != p->n_chains) return "species_n_chains must sum to n_chains";
  }
  if (!(p->smc_mobility >= 0.0f) || p->smc_mobility > 1e6f) return "smc_mobility must be in [0, 1e6]";
  if (!p->type_patterns) return "type_patterns is NULL";
  if (!p->chiN) return "chiN is NULL";
  if (!(p->b > 0.0f)) return "b must be > 0";
  if (!(p->move_halfwidth >= 0.0f)) return "move_halfwidth must be >= 0";
  if (!(p->kappaN == p->kappaN)) return "kappaN is NaN";
  uint64_t cells = 1;
  for (int d = 0; d < 3; ++d) {
    if (p->grid[d] == 0 || p->grid[d] > (1u << 20)) return "grid[d] must be in [1, 2^20]";
    if (!(p->box[d] > 0.0f)) return "box[d] must be > 0";
    cells *= p->grid[d];
    if (cells >= (1ull << 32)) return "too many cells";
  }
  if (cells * p->n_types >= (1ull << 32)) return "n_types * cells must be < 2^32";
  if (p->n_single) {
    uint64_t S = 0;
    for (uint32_t t = 0; t < p->n_types; ++t) {
      if (p->n_single[t] >= (1ull << 32)) return "n_single[t] must be < 2^32";
      S += p->n_single[t];
    }
    if (p->n_chains + S >= (1ull << 32)) return "n_chains + single-bead molecules must be < 2^32";
  }
  const uint64_t npat = (uint64_t)p->n_patterns * pattern_stride(p);
  for (uint64_t k = 0; k < npat; ++k)
    if (p->type_patterns[k] >= p->n_types) return "type_patterns holds a type >= n_types";
  if (p->chain_pattern)
    for (uint64_t c = 0; c < p->n_chains; ++c)
      if (p->chain_pattern[c] >= p->n_patterns) return "chain_pattern holds an id >= n_patterns";
  if (p->n_patterns > 1 && !p->chain_pattern) return "chain_pattern is NULL but n_patterns > 1";
  const uint32_t T = p->n_types;
  for (uint32_t s = 0; s < T; ++s)
    for (uint32_t t = 0; t < T; ++t) {
      const float v = p->chiN[s * T + t];
      if (!(v == v)) return "chiN holds a NaN";
      if (s == t && v != 0.0f) return "chiN diagonal must be 0";
      if (v != p->chiN[t * T + s]) return "chiN must be symmetric";
    }
  return nullptr;
}

int fused_lanes(uint32_t N) {   // P = N/2 if the fused kernel supports N, else 0
  if (N < 2 || (N & 1u)) return 0;
  const uint32_t P = N / 2;
  return (P <= 32 && is_pow2(P)) ? (int)P : 0;
}

}  // namespace

struct soma_handle {
  // problem
  uint64_t n_chains, B;          // all chains; B = beads in chains
  // Polymer species of different chain lengths (R26): chains, slots and beads of species s are the
  // ranges [first_chain, first_chain + n) and [bead_off, bead_off + B) of every per-chain / per-bead array.
  // `v` is the species the per-species launchers below work on; N (below) is the reference chain length of 1/N.
  struct View { uint64_t n, first_chain, bead_off, B; uint32_t N; };
  View views[kMaxSpecies];
  uint32_t n_views;
  View v;
  uint32_t Nstride;              // row length of the type patterns
  uint64_t S, Btot;              // single-bead molecules (R23) and all beads
  uint32_t single_start[kMaxTypes + 1];
  uint32_t N, T, n_patterns, cells;
  Grid grid;
  bool pow2;
  float a, kb, dens_scale, invN, kappaN, b, box[3];
  float smcA, gA, sq2A, inv4A;   // bond-force-biased moves (R24); smcA = 0: uniform moves
  float chiN[kMaxTypes * kMaxTypes];
  uint64_t seed;
  // device
  int device;
  cudaStream_t stream;
  char* ws;
  bool owns_ws;
  Layout L;
  int live;              // which position set (and slot table) is current
  int cur;               // which count buffer holds the current densities
  uint32_t n_bins;       // coarse bins of the chain re-ordering
  PhiloxKeys keys;
  uint64_t steps_since_check;   // MC steps since the cell-coordinate range was last verified
  uint64_t steps_since_sort;
  uint64_t range_check_interval;
  // state
  bool loaded;
  bool has_ext;          // an external field is set (soma_set_external_field)
  // density counters packed two types to a word (soma_device.cuh) and omega computed on the fly by the lean kernel
  bool packed;           // layout of both count buffers for the state that is loaded
  int packed_opt, otf_opt;      // options "packed_counts", "omega_otf" (default -1 = by grid size)
  bool omega_valid;      // the omega array holds the field of the current densities
  bool guard_seen;       // the guard flag as verify_range last read it
  bool omega_custom;     // soma_debug_set_omega has replaced the field: the next step reads the array
  uint32_t guard_mask;   // bits of a packed word that are set once a 16-bit field has reached the guard level (soma_device.cuh); 0: never pack
  bool umbrella;         // the umbrella potential toward phi_tgt is on (inside soma_init_from_density)
  float umbrella_k;
  std::vector<uint8_t>* host_patterns;     // [n_patterns][N] copy of the type patterns
  std::vector<uint64_t>* pattern_chains;   // [n_patterns] chains of every pattern
  bool identity_order;   // slot_chain is the identity
  uint64_t step;
  int sm_count;
  // options
  int path;              // 0 auto, 1 generic, 2 fused
  int64_t resort_interval;      // re-order the chains every k steps (0 = never)
  int fused_chunk;              // warp groups per block of the fused kernel
  int fused_carveout;           // preferred shared-memory carve-out of the fused kernel in percent (-1: driver default)
  bool fast_arith;              // inv_h a power of two >= 1 on every axis and a a power of two: the one-FFMA shortcuts are exact
  bool sorted;                  // the slots are sorted by the cube of 4 cells that holds the chain's centre of mass
  // lean kernel (soma_lean.cuh)
  int fused_lean;               // use lean_step_kernel where it applies (option, default 1)
  int omega_x4;                 // use omega_kernel_x4 where it applies (option, default 1)
  int lean_threads;             // threads per block of the lean kernel: 256, 512 or 1024
  // counters
  uint64_t launches, steps_done, resorts;
  // per-kernel timing ("kernel_timing" option): event triples (before moves, after moves+bin, after omega)
  bool timing;
  std::vector<cudaEvent_t>* ev;      // 3 per recorded step
  size_t ev_used;                    // events recorded since the last soma_get_kernel_times
  bool sticky;
  char err[256];

  float* pos(int set, int d) const { return reinterpret_cast<float*>(ws + L.pos[set][d]); }
  float* vpos(int set, int d) const { return pos(set, d) + v.bead_off; }                       // ... of the current species
  uint32_t* counts(int s) const { return reinterpret_cast<uint32_t*>(ws + L.counts[s]); }
  float* omega() const { return reinterpret_cast<float*>(ws + L.omega); }
  float* ext() const { return reinterpret_cast<float*>(ws + L.ext); }
  float* phi_tgt() const { return reinterpret_cast<float*>(ws + L.phi_tgt); }
  unsigned long long* cdf() const { return reinterpret_cast<unsigned long long*>(ws + L.cdf); }
  float* single(int d) const { return reinterpret_cast<float*>(ws + L.single[d]); }
  uint32_t* slot_chain(int s) const { return reinterpret_cast<uint32_t*>(ws + L.slot_chain[s]); }
  uint8_t* slot_pattern(int s) const { return reinterpret_cast<uint8_t*>(ws + L.slot_pattern[s]); }
  uint32_t* slot_chain() const { return slot_chain(live); }
  uint8_t* slot_pattern() const { return slot_pattern(live); }
  uint32_t* vslot_chain(int s) const { return slot_chain(s) + v.first_chain; }
  uint8_t* vslot_pattern(int s) const { return slot_pattern(s) + v.first_chain; }
  uint32_t* range_flag() const { return reinterpret_cast<uint32_t*>(ws + L.range_flag); }
  uint32_t* sort_key() const { return reinterpret_cast<uint32_t*>(ws + L.sort_key); }
  uint32_t* sort_rank() const { return reinterpret_cast<uint32_t*>(ws + L.sort_rank); }
  uint32_t* sort_bins() const { return reinterpret_cast<uint32_t*>(ws + L.sort_bins); }
  uint8_t* patterns() const { return reinterpret_cast<uint8_t*>(ws + L.patterns); }
  uint8_t* pattern0() const { return reinterpret_cast<uint8_t*>(ws + L.pattern0); }
  unsigned long long* accepted() const { return reinterpret_cast<unsigned long long*>(ws + L.accepted); }
};

namespace {

void free_handle(soma_handle* h) {
  if (h->ev) {
    for (cudaEvent_t e : *h->ev) cudaEventDestroy(e);
    delete h->ev;
  }
  delete h->host_patterns;
  delete h->pattern_chains;
  delete h;
}

int fail(soma_handle* h, int code, const char* msg) {
  snprintf(h ? h->err : g_last_error, 256, "%s", msg);
  return code;
}
int cuda_fail(soma_handle* h, cudaError_t e, const char* where) {
  char buf[256];
  snprintf(buf, sizeof buf, "%s: %s", where, cudaGetErrorString(e));
  if (h) h->sticky = true;
  return fail(h, SOMA_ECUDA, buf);
}
#define CU(h, call)                                            \
  do {                                                         \
    cudaError_t e_ = (call);                                   \
    if (e_ != cudaSuccess) return cuda_fail((h), e_, #call);   \
  } while (0)

inline unsigned blocks_for(uint64_t n, unsigned bs) { return (unsigned)((n + bs - 1) / bs); }

StepArgs step_args(const soma_handle* h) {
  StepArgs A{};
  A.grid = h->grid;
  A.cells = h->cells;
  A.n_chains = (uint32_t)h->v.n;
  A.N = h->v.N;
  A.pat_stride = h->Nstride;
  A.packed = h->packed ? 1u : 0u;
  A.a = h->a;
  A.kb = h->kb;
  A.gA = h->gA; A.sq2A = h->sq2A; A.inv4A = h->inv4A;
  A.keys = h->keys;
  A.ctr2 = (uint32_t)h->step;
  A.ctr3_base = (0u << 8) | ((uint32_t)(h->step >> 32) << 16);   // domain 0 = MC move
  A.x = h->vpos(h->live, 0);
  A.y = h->vpos(h->live, 1);
  A.z = h->vpos(h->live, 2);
  A.omega = h->omega();
  A.counts_next = h->counts(h->cur ^ 1);
  A.slot_chain = h->vslot_chain(h->live);
  A.slot_pattern = h->vslot_pattern(h->live);
  A.patterns = h->patterns();
  A.accepted = h->accepted();
  return A;
}

int launch_half_sweep(soma_handle* h, uint32_t parity) {
  const uint32_t n_par = (h->v.N + 1u - parity) / 2u;
  if (n_par == 0) return SOMA_OK;                               // N == 1 has no odd beads
  const uint64_t total = h->v.n * n_par;
  const StepArgs A = step_args(h);
  if (h->pow2) half_sweep_kernel<true><<<blocks_for(total, 256), 256, 0, h->stream>>>(A, parity, n_par);
  else half_sweep_kernel<false><<<blocks_for(total, 256), 256, 0, h->stream>>>(A, parity, n_par);
  h->launches++;
  CU(h, cudaGetLastError());
  return SOMA_OK;
}

// Single-bead molecules: trial moves (half-sweep 0) and / or binning into `counts`.
int launch_singles(soma_handle* h, bool do_move, bool do_bin, uint32_t* counts, bool check_range = false) {
  if (h->S == 0) return SOMA_OK;
  SingleArgs A{};
  A.S = step_args(h);
  A.S.n_chains = (uint32_t)h->n_chains;                          // first logical id of the molecules
  A.n_total = (uint32_t)h->S; A.T = h->T;
  for (int t = 0; t <= kMaxTypes; ++t) A.start[t] = h->single_start[t];
  A.x = h->single(0); A.y = h->single(1); A.z = h->single(2);
  A.counts = counts;
  A.range_flag = check_range ? h->range_flag() : nullptr;
  A.do_move = do_move; A.do_bin = do_bin;
  if (h->pow2) singles_kernel<true><<<blocks_for(h->S, 256), 256, 0, h->stream>>>(A);
  else singles_kernel<false><<<blocks_for(h->S, 256), 256, 0, h->stream>>>(A);
  h->launches++;
  CU(h, cudaGetLastError());
  return SOMA_OK;
}

// bins the chains of the current species
int launch_bin_chains(soma_handle* h, uint32_t* counts, uint32_t* flag) {
  {
    if (h->pow2)
      bin_kernel<true><<<blocks_for(h->v.B, 256), 256, 0, h->stream>>>(
          h->grid, h->cells, h->v.N, h->Nstride, h->packed ? 1u : 0u, h->v.B, h->vpos(h->live, 0), h->vpos(h->live, 1), h->vpos(h->live, 2),
          h->vslot_pattern(h->live), h->patterns(), counts, flag);
    else
      bin_kernel<false><<<blocks_for(h->v.B, 256), 256, 0, h->stream>>>(
          h->grid, h->cells, h->v.N, h->Nstride, h->packed ? 1u : 0u, h->v.B, h->vpos(h->live, 0), h->vpos(h->live, 1), h->vpos(h->live, 2),
          h->vslot_pattern(h->live), h->patterns(), counts, flag);
    h->launches++;
    CU(h, cudaGetLastError());
  }
  return SOMA_OK;
}
// row a3 on its own: every species and the single-bead molecules
int launch_bin(soma_handle* h, uint32_t* counts, bool check_range = false) {
  int rc;
  for (uint32_t k = 0; k < h->n_views; ++k) {
    h->v = h->views[k];
    if ((rc = launch_bin_chains(h, counts, check_range ? h->range_flag() : nullptr)) != SOMA_OK) return rc;
  }
  return launch_singles(h, false, true, counts, check_range);
}

// omega from counts(cur); zero counts(cur^1) for the next step's binning.
int launch_omega(soma_handle* h) {
  OmegaArgs A{};
  A.cells = h->cells; A.T = h->T;
  A.dens_scale = h->dens_scale; A.kappaN = h->kappaN; A.invN = h->invN;
  std::memcpy(A.chiN, h->chiN, sizeof A.chiN);
  A.packed = h->packed ? 1u : 0u;
  A.guard_mask = h->guard_mask;
  A.guard_flag = h->range_flag() + 1;
  A.counts = h->counts(h->cur);
  A.counts_to_zero = h->counts(h->cur ^ 1);
  A.omega = h->omega();
  A.ext = h->has_ext ? h->ext() : nullptr;
  A.phi_tgt = h->umbrella ? h->phi_tgt() : nullptr;
  A.umbrella_k = h->umbrella_k;
  const unsigned g = blocks_for(h->cells, 256);
  if (h->cells % 4u == 0 && h->T <= 3 && h->omega_x4) {            // four cells per thread, 128-bit accesses
    const unsigned g4 = blocks_for(h->cells / 4u, 256);
    switch (h->T) {
      case 1: omega_kernel_x4<1><<<g4, 256, 0, h->stream>>>(A); break;
      case 2: omega_kernel_x4<2><<<g4, 256, 0, h->stream>>>(A); break;
      default: omega_kernel_x4<3><<<g4, 256, 0, h->stream>>>(A); break;
    }
    h->launches++;
    CU(h, cudaGetLastError());
    h->omega_valid = true;
    h->omega_custom = false;
    return SOMA_OK;
  }
  switch (h->T) {
    case 1: omega_kernel<1><<<g, 256, 0, h->stream>>>(A); break;
    case 2: omega_kernel<2><<<g, 256, 0, h->stream>>>(A); break;
    case 3: omega_kernel<3><<<g, 256, 0, h->stream>>>(A); break;
    default: omega_kernel<0><<<g, 256, 0, h->stream>>>(A); break;
  }
  h->launches++;
  CU(h, cudaGetLastError());
  h->omega_valid = true;
  h->omega_custom = false;
  return SOMA_OK;
}

// Does the lean kernel compute omega from the packed counters itself (soma_lean.cuh, OTF)?
// By default where the grids are too large to stay in the caches (>= 2^20 cells: cfg3 -3.6 %, cfg4 -8.9 % per
// step; on cfg1 / cfg2, whose grids are L2-resident, the extra arithmetic costs 2-4 %).
bool use_otf(const soma_handle* h) {
  const bool want = h->otf_opt < 0 ? h->cells >= (1u << 20) : h->otf_opt != 0;
  return h->packed && want && !h->has_ext && !h->umbrella && !h->omega_custom;
}

// The omega array is computed lazily while every mover computes the field itself: make it current.
int ensure_omega(soma_handle* h) {
  if (h->omega_valid) return SOMA_OK;
  OmegaArgs A{};
  A.cells = h->cells; A.T = h->T;
  A.dens_scale = h->dens_scale; A.kappaN = h->kappaN; A.invN = h->invN;
  std::memcpy(A.chiN, h->chiN, sizeof A.chiN);
  A.packed = h->packed ? 1u : 0u;
  A.guard_mask = h->guard_mask;
  A.guard_flag = h->range_flag() + 1;
  A.counts = h->counts(h->cur);
  A.counts_to_zero = nullptr;                                  // the next buffer was zeroed when the step ended
  A.omega = h->omega();
  A.ext = h->has_ext ? h->ext() : nullptr;
  A.phi_tgt = h->umbrella ? h->phi_tgt() : nullptr;
  A.umbrella_k = h->umbrella_k;
  const unsigned g = blocks_for(h->cells, 256);
  switch (h->T) {
    case 1: omega_kernel<1><<<g, 256, 0, h->stream>>>(A); break;
    case 2: omega_kernel<2><<<g, 256, 0, h->stream>>>(A); break;
    case 3: omega_kernel<3><<<g, 256, 0, h->stream>>>(A); break;
    default: omega_kernel<0><<<g, 256, 0, h->stream>>>(A); break;
  }
  h->launches++;
  CU(h, cudaGetLastError());
  h->omega_valid = true;
  return SOMA_OK;
}

bool lean_ok(const soma_handle* h) {
  return h->fused_lean && h->fast_arith && h->pow2 && h->smcA == 0.0f && fused_lanes(h->v.N) != 0;
}
template <int P, bool MULTI, bool OTF, int NT>
void launch_lean_k(soma_handle* h, LeanArgs& A) {
  constexpr int G = 32 / P;
  auto* k = lean_step_kernel<P, MULTI, OTF, NT>;
  const uint64_t n_groups = (h->v.n + G - 1) / G;
  const uint64_t wpb = NT / 32;
  const uint64_t gpb = ((uint64_t)h->fused_chunk * (NT / 256) + wpb - 1) / wpb * wpb;   // fused_chunk is per 256 threads
  A.groups_per_block = (uint32_t)gpb;
  if (h->fused_carveout >= 0) cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, h->fused_carveout);
  k<<<(unsigned)((n_groups + gpb - 1) / gpb), NT, 0, h->stream>>>(A);
}
template <int P, int NT>
int launch_lean_pn(soma_handle* h, LeanArgs& A) {
  if (use_otf(h)) { if (h->n_patterns > 1) launch_lean_k<P, true, true, NT>(h, A); else launch_lean_k<P, false, true, NT>(h, A); }
  else            { if (h->n_patterns > 1) launch_lean_k<P, true, false, NT>(h, A); else launch_lean_k<P, false, false, NT>(h, A); }
  h->launches++;
  CU(h, cudaGetLastError());
  return SOMA_OK;
}

template <int P>
int launch_lean_p(soma_handle* h) {
  LeanArgs A{};
  A.inv_hx = h->grid.inv_hx; A.inv_hy = h->grid.inv_hy; A.inv_hz = h->grid.inv_hz;
  A.mx = h->grid.nx - 1; A.my = h->grid.ny - 1; A.mz = h->grid.nz - 1;
  A.ny = h->grid.ny; A.nz = h->grid.nz;
  A.cells = h->cells;
  A.n_chains = (uint32_t)h->v.n;
  A.pat_stride = h->Nstride;
  A.a2 = 2.0f * h->a;
  A.ac = h->a * -0.99999988079071044921875f;       // a (2^-23 - 1), exact: a is a power of two
  A.kb = h->kb;
  A.keys = h->keys;
  const uint64_t m1 = (uint64_t)kPhiloxM1 * (uint32_t)h->step;
  A.u0 = (uint32_t)(m1 >> 32) ^ h->keys.k0[0];
  A.u1 = (uint32_t)m1;
  A.ctr3_base = (0u << 8) | ((uint32_t)(h->step >> 32) << 16);   // domain 0 = MC move
  A.x = h->vpos(h->live, 0); A.y = h->vpos(h->live, 1); A.z = h->vpos(h->live, 2);
  A.omega = h->omega();
  A.counts_prev = h->counts(h->cur);
  A.dens_scale = h->dens_scale; A.kappaN = h->kappaN; A.invN = h->invN;
  A.chi01 = h->T > 1 ? h->chiN[1] : 0.0f;
  A.packed = h->packed ? 1u : 0u;
  A.guard_mask = h->guard_mask;
  A.guard_flag = h->range_flag() + 1;
  A.counts_next = h->counts(h->cur ^ 1);
  A.slot_chain = h->vslot_chain(h->live);
  A.slot_pattern = h->vslot_pattern(h->live);
  A.patterns = h->patterns();
  A.accepted = h->accepted();
  switch (h->lean_threads) {
    case 256: return launch_lean_pn<P, 256>(h, A);
    case 512: return launch_lean_pn<P, 512>(h, A);
    default: return launch_lean_pn<P, 1024>(h, A);
  }
}

template <int P>
int launch_fused_p(soma_handle* h) {
  if (lean_ok(h)) return launch_lean_p<P>(h);
  const StepArgs A = step_args(h);
  constexpr int G = 32 / P;
  const uint64_t n_groups = (h->v.n + G - 1) / G;                // warps of work
  const unsigned bs = 256, wpb = bs / 32;
  // chunks of fused_chunk warp groups (a multiple of the warps per block)
  uint64_t gpb = ((uint64_t)h->fused_chunk + wpb - 1) / wpb * wpb;
  const uint64_t n_chunks = (n_groups + gpb - 1) / gpb;
  const uint64_t blocks = n_chunks;                // one block per chunk, in chain-list order
  const bool multi = h->n_patterns > 1;
  const bool fast = h->fast_arith && h->pow2;      // exact one-FFMA shortcuts apply (see fused_move)
#define SOMA_LAUNCH_FUSED(POW2, MULTI)                                                                          \
  do {                                                                                                          \
    if (h->fused_carveout >= 0 && fast && POW2)                                                                 \
      cudaFuncSetAttribute(fused_step_kernel<P, POW2, MULTI, POW2>, cudaFuncAttributePreferredSharedMemoryCarveout, h->fused_carveout); \
    if (h->smcA > 0.0f) fused_step_kernel<P, POW2, MULTI, false, true><<<(unsigned)blocks, bs, 0, h->stream>>>(A, (uint32_t)gpb); \
    else if (fast && POW2) fused_step_kernel<P, POW2, MULTI, POW2><<<(unsigned)blocks, bs, 0, h->stream>>>(A, (uint32_t)gpb); \
    else fused_step_kernel<P, POW2, MULTI, false><<<(unsigned)blocks, bs, 0, h->stream>>>(A, (uint32_t)gpb);    \
  } while (0)
  if (h->pow2) { if (multi) SOMA_LAUNCH_FUSED(true, true); else SOMA_LAUNCH_FUSED(true, false); }
  else         { if (multi) SOMA_LAUNCH_FUSED(false, true); else SOMA_LAUNCH_FUSED(false, false); }
#undef SOMA_LAUNCH_FUSED
  h->launches++;
  CU(h, cudaGetLastError());
  return SOMA_OK;
}

int launch_fused(soma_handle* h) {
  switch (fused_lanes(h->v.N)) {
    case 1: return launch_fused_p<1>(h);
    case 2: return launch_fused_p<2>(h);
    case 4: return launch_fused_p<4>(h);
    case 8: return launch_fused_p<8>(h);
    case 16: return launch_fused_p<16>(h);
    case 32: return launch_fused_p<32>(h);
  }
  return fail(h, SOMA_EINVAL, "fused path does not support this beads_per_chain");
}

bool use_fused(const soma_handle* h) {
  if (h->path == 1) return false;
  if ((h->Nstride & 1u) && h->n_patterns > 1) return false;     // the fused kernels read a lane's two types as one aligned 16-bit word
  if (h->v.bead_off & 1u) return false;                          // ... and a lane's two beads as one aligned 64-bit word
  return fused_lanes(h->v.N) != 0;
}
// Re-order the chains in memory by the coarse bin (cube of kSortBinEdge cells) of their centre of
// mass: a counting sort on the device.
int resort(soma_handle* h) {
  const int src = h->live, dst = h->live ^ 1;
  for (uint32_t k = 0; k < h->n_views; ++k) {                     // every species inside its own range of slots
    h->v = h->views[k];
    SortArgs S{};
    S.grid = h->grid; S.n_chains = (uint32_t)h->v.n; S.N = h->v.N;
    S.cbx = S.cby = S.cbz = kSortBinEdge;
    S.ncy = (h->grid.ny + kSortBinEdge - 1) / kSortBinEdge;
    S.ncz = (h->grid.nz + kSortBinEdge - 1) / kSortBinEdge;
    const uint32_t n_bins = h->n_bins;
    uint32_t* key = h->sort_key() + h->v.first_chain;
    uint32_t* rank = h->sort_rank() + h->v.first_chain;
    CU(h, cudaMemsetAsync(h->sort_bins(), 0, ((size_t)n_bins + 1) * 4, h->stream));
    if (h->pow2)
      chain_key_kernel<true><<<blocks_for(h->v.n, 256), 256, 0, h->stream>>>(
          S, h->vpos(src, 0), h->vpos(src, 1), h->vpos(src, 2), h->sort_bins(), key, rank);
    else
      chain_key_kernel<false><<<blocks_for(h->v.n, 256), 256, 0, h->stream>>>(
          S, h->vpos(src, 0), h->vpos(src, 1), h->vpos(src, 2), h->sort_bins(), key, rank);
    if (n_bins + 1 > 8u * kBinScanChunk) {                         // many bins: three short passes over many blocks
      const uint32_t chunks = (n_bins + 1 + kBinScanChunk - 1) / kBinScanChunk;
      uint32_t* chunk = reinterpret_cast<uint32_t*>(h->cdf());     // scratch of soma_init_from_density, idle here (same stream)
      bin_chunk_sums_kernel<<<chunks, 256, 0, h->stream>>>(n_bins + 1, h->sort_bins(), chunk);
      bin_scan_kernel<<<1, 1024, 0, h->stream>>>(chunks, chunk);
      bin_scan_apply_kernel<<<chunks, 256, 0, h->stream>>>(n_bins + 1, h->sort_bins(), chunk);
      h->launches += 2;
    } else {
      bin_scan_kernel<<<1, 1024, 0, h->stream>>>(n_bins + 1, h->sort_bins());    // entry n_bins becomes the total
    }
    if (h->v.N % 4u == 0 && h->v.bead_off % 4u == 0)               // whole 16-byte quads of a chain per thread
      chain_permute4_kernel<<<blocks_for(h->v.B / 4, 256), 256, 0, h->stream>>>(
          h->v.B / 4, h->v.N / 4, h->sort_bins(), key, rank,
          reinterpret_cast<const float4*>(h->vpos(src, 0)), reinterpret_cast<const float4*>(h->vpos(src, 1)), reinterpret_cast<const float4*>(h->vpos(src, 2)),
          reinterpret_cast<float4*>(h->vpos(dst, 0)), reinterpret_cast<float4*>(h->vpos(dst, 1)), reinterpret_cast<float4*>(h->vpos(dst, 2)),
          h->vslot_chain(src), h->vslot_pattern(src), h->vslot_chain(dst), h->vslot_pattern(dst));
    else
    chain_permute_kernel<<<blocks_for(h->v.B, 256), 256, 0, h->stream>>>(
        h->v.B, h->v.N, h->sort_bins(), key, rank,
        h->vpos(src, 0), h->vpos(src, 1), h->vpos(src, 2), h->vpos(dst, 0), h->vpos(dst, 1), h->vpos(dst, 2),
        h->vslot_chain(src), h->vslot_pattern(src), h->vslot_chain(dst), h->vslot_pattern(dst));
    h->launches += 3;
    CU(h, cudaGetLastError());
  }
  h->live = dst;
  h->identity_order = false;
  h->resorts++;
  h->steps_since_sort = 0;
  h->sorted = true;
  return SOMA_OK;
}

// The conversion-free floor needs |r * inv_h| < 2^22; positions are verified to be below 2^21 and a
// bead drifts by at most a * inv_h cells per step and axis, so the check is repeated before 2^21
// cells of drift could have accumulated.
int verify_range(soma_handle* h) {
  uint32_t flag[2] = {0, 0};
  CU(h, cudaMemcpyAsync(flag, h->range_flag(), 8, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  h->guard_seen = flag[1] != 0;
  if (flag[0]) {
    h->loaded = false;
    return fail(h, SOMA_EINVAL, "a position is NaN or beyond 2^21 cells from the origin");
  }
  if (flag[1] && h->packed && h->loaded) {                       // (at load time finish_load looks at the flag itself)
    h->loaded = false;
    return fail(h, SOMA_EINVAL, "a cell holds more beads of one type than the guard level of the 16-bit density counters "
                                "allows (2048 for moves of at most one cell): set option packed_counts = 0 and load the state again");
  }
  h->steps_since_check = 0;
  return SOMA_OK;
}

// After a call that has synchronised anyway: has a 16-bit density counter reached its guard level?
int guard_check(soma_handle* h) {
  if (!h->packed) return SOMA_OK;
  uint32_t flag = 0;
  CU(h, cudaMemcpyAsync(&flag, h->range_flag() + 1, 4, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  if (flag) {
    h->loaded = false;
    return fail(h, SOMA_EINVAL, "a cell holds more beads of one type than the guard level of the 16-bit density counters "
                                "allows (2048 for moves of at most one cell): set option packed_counts = 0 and load the state again");
  }
  return SOMA_OK;
}

constexpr size_t kMaxTimedSteps = 16384;

// next event of the timing pool, recorded on the handle's stream (nullptr: pool exhausted / error)
cudaEvent_t timing_mark(soma_handle* h) {
  if (h->ev_used >= 3 * kMaxTimedSteps) return nullptr;
  if (h->ev_used == h->ev->size()) {
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    h->ev->push_back(e);
  }
  cudaEvent_t e = (*h->ev)[h->ev_used++];
  cudaEventRecord(e, h->stream);
  return e;
}

int one_step(soma_handle* h) {
  int rc;
  if (h->resort_interval > 0 && (h->steps_since_sort >= (uint64_t)h->resort_interval || !h->sorted))
    if ((rc = resort(h)) != SOMA_OK) return rc;
  // Does anything read the omega array in this step?  The lean kernel in OTF mode computes the field itself.
  bool needs_omega = !use_otf(h) || h->S > 0;
  for (uint32_t k = 0; k < h->n_views && !needs_omega; ++k) {
    h->v = h->views[k];
    needs_omega = !(use_fused(h) && lean_ok(h));
  }
  if (needs_omega && (rc = ensure_omega(h)) != SOMA_OK) return rc;
  const bool timed = h->timing && h->ev_used + 3 <= 3 * kMaxTimedSteps;
  if (timed) timing_mark(h);
  // Chains interact only through omega, which is frozen during a step, so the species (and the single-bead
  // molecules) can take their half-sweeps one after the other, each on the kernels its chain length allows.
  for (uint32_t k = 0; k < h->n_views; ++k) {
    h->v = h->views[k];
    if (use_fused(h)) {
      if ((rc = launch_fused(h)) != SOMA_OK) return rc;            // a1 + a2 + a3 (+a5)
    } else {
      if ((rc = launch_half_sweep(h, 0)) != SOMA_OK) return rc;    // a1
      if ((rc = launch_half_sweep(h, 1)) != SOMA_OK) return rc;    // a2
      if ((rc = launch_bin_chains(h, h->counts(h->cur ^ 1), nullptr)) != SOMA_OK) return rc;   // a3
    }
  }
  if ((rc = launch_singles(h, true, true, h->counts(h->cur ^ 1))) != SOMA_OK) return rc;      // a1 + a3, single-bead molecules
  h->cur ^= 1;
  if (timed) timing_mark(h);
  if (needs_omega) {
    if ((rc = launch_omega(h)) != SOMA_OK) return rc;            // a4 (also zeroes the next count buffer)
  } else {                                                       // a4 happens inside the next step's moves
    CU(h, cudaMemsetAsync(h->counts(h->cur ^ 1), 0, (size_t)h->cells * 4, h->stream));
    h->omega_valid = false;                                      // (the lean kernel's old-cell gathers look at the 16-bit fields)
  }
  if (timed) timing_mark(h);
  h->step += 1;
  h->steps_done += 1;
  h->steps_since_sort += 1;
  h->steps_since_check += 1;
  return SOMA_OK;
}

int check(soma_handle* h) {
  if (!h) return fail(nullptr, SOMA_EINVAL, "handle is NULL");
  if (h->sticky) return SOMA_ECUDA;
  CU(h, cudaSetDevice(h->device));
  return SOMA_OK;
}

// copy [count] elements to the caller, host or device
template <typename Tp>
int copy_out(soma_handle* h, Tp* dst, const Tp* src, uint64_t count, int dst_is_device) {
  CU(h, cudaMemcpyAsync(dst, src, count * sizeof(Tp),
                        dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
  if (!dst_is_device) CU(h, cudaStreamSynchronize(h->stream));
  return SOMA_OK;
}

}  // namespace

extern "C" {

uint64_t soma_workspace_bytes(const soma_params* p) {
  const char* bad = validate(p);
  if (bad) { fail(nullptr, SOMA_EINVAL, bad); return 0; }
  const uint64_t B = chain_beads(p);
  const uint64_t TC = (uint64_t)p->grid[0] * p->grid[1] * p->grid[2] * p->n_types;
  uint64_t S = 0;
  if (p->n_single) for (uint32_t t = 0; t < p->n_types; ++t) S += p->n_single[t];
  return make_layout(B, p->n_chains, TC, (uint64_t)p->n_patterns * pattern_stride(p), sort_bin_count(p->grid) + 2, S, TC / p->n_types).total;
}

int soma_create(const soma_params* p, void* cuda_stream, soma_t** out) {
  if (!out) return fail(nullptr, SOMA_EINVAL, "out is NULL");
  *out = nullptr;
  const char* bad = validate(p);
  if (bad) return fail(nullptr, SOMA_EINVAL, bad);
  soma_handle* h = new (std::nothrow) soma_handle();
  if (!h) return fail(nullptr, SOMA_ENOMEM, "host allocation failed");
  std::memset(static_cast<void*>(h), 0, sizeof *h);
  h->ev = new (std::nothrow) std::vector<cudaEvent_t>();
  h->host_patterns = new (std::nothrow) std::vector<uint8_t>(p->type_patterns, p->type_patterns + (size_t)p->n_patterns * pattern_stride(p));
  const uint32_t n_views = p->n_species > 1 ? p->n_species : 1u;
  h->pattern_chains = new (std::nothrow) std::vector<uint64_t>((size_t)n_views * p->n_patterns, 0);      // [species][pattern]
  if (!h->ev || !h->host_patterns || !h->pattern_chains) { free_handle(h); return fail(nullptr, SOMA_ENOMEM, "host allocation failed"); }
  h->n_views = n_views;
  h->Nstride = pattern_stride(p);
  {
    uint64_t c0 = 0, b0 = 0;
    for (uint32_t k = 0; k < n_views; ++k) {
      soma_handle::View& V = h->views[k];
      V.n = n_views > 1 ? p->species_n_chains[k] : p->n_chains;
      V.N = n_views > 1 ? p->species_beads[k] : p->beads_per_chain;
      V.first_chain = c0; V.bead_off = b0; V.B = V.n * V.N;
      for (uint64_t c = c0; c < c0 + V.n; ++c) (*h->pattern_chains)[(size_t)k * p->n_patterns + (p->chain_pattern ? p->chain_pattern[c] : 0)]++;
      c0 += V.n; b0 += V.B;
    }
    h->v = h->views[0];
  }
  cudaError_t e = cudaGetDevice(&h->device);
  cudaDeviceProp prop{};
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, h->device);
  if (e != cudaSuccess) {
    snprintf(g_last_error, 256, "no usable CUDA device: %s", cudaGetErrorString(e));
    free_handle(h);
    return SOMA_ECUDA;
  }
  if (prop.major != 10) {
    snprintf(g_last_error, 256, "device is sm_%d%d; this library holds sm_100a code only", prop.major, prop.minor);
    free_handle(h);
    return SOMA_ECUDA;
  }
  h->sm_count = prop.multiProcessorCount;
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  h->n_chains = p->n_chains; h->N = p->beads_per_chain; h->T = p->n_types; h->n_patterns = p->n_patterns;
  h->B = chain_beads(p);
  h->S = 0;
  for (uint32_t t = 0; t < h->T; ++t) {
    h->single_start[t] = (uint32_t)h->S;
    if (p->n_single) h->S += p->n_single[t];
  }
  for (uint32_t t = h->T; t <= (uint32_t)kMaxTypes; ++t) h->single_start[t] = (uint32_t)h->S;
  h->Btot = h->B + h->S;
  h->cells = p->grid[0] * p->grid[1] * p->grid[2];
  h->grid.nx = p->grid[0]; h->grid.ny = p->grid[1]; h->grid.nz = p->grid[2];
  h->grid.inv_hx = (float)p->grid[0] / p->box[0];
  h->grid.inv_hy = (float)p->grid[1] / p->box[1];
  h->grid.inv_hz = (float)p->grid[2] / p->box[2];
  h->pow2 = is_pow2(p->grid[0]) && is_pow2(p->grid[1]) && is_pow2(p->grid[2]);
  h->a = p->move_halfwidth;
  h->b = p->b;
  for (int d = 0; d < 3; ++d) h->box[d] = p->box[d];
  h->kb = 1.5f / (p->b * p->b);
  h->smcA = p->smc_mobility;
  h->gA = h->smcA * (2.0f * h->kb);
  h->sq2A = (float)std::sqrt(2.0 * (double)h->smcA);
  h->inv4A = h->smcA > 0.0f ? (float)(1.0 / (4.0 * (double)h->smcA)) : 0.0f;
  h->dens_scale = (float)((double)h->cells / (double)h->Btot);
  h->invN = 1.0f / (float)h->N;
  h->kappaN = p->kappaN;
  for (uint32_t k = 0; k < h->T * h->T; ++k) h->chiN[k] = p->chiN[k];
  h->seed = p->seed;
  h->n_bins = (uint32_t)sort_bin_count(p->grid);
  h->L = make_layout(h->B, h->n_chains, (uint64_t)h->cells * h->T, (uint64_t)h->n_patterns * h->Nstride, sort_bin_count(p->grid) + 2, h->S, h->cells);
  if (p->workspace) {
    if (p->workspace_bytes < h->L.total || (reinterpret_cast<uintptr_t>(p->workspace) % kAlign)) {
      free_handle(h);
      return fail(nullptr, SOMA_ENOMEM, "lent workspace is too small or not 256-byte aligned");
    }
    h->ws = static_cast<char*>(p->workspace);
    h->owns_ws = false;
  } else {
    void* ptr = nullptr;
    e = cudaMalloc(&ptr, h->L.total);
    if (e != cudaSuccess) {
      snprintf(g_last_error, 256, "cudaMalloc(%llu bytes): %s", (unsigned long long)h->L.total, cudaGetErrorString(e));
      cudaGetLastError();
      free_handle(h);
      return SOMA_ENOMEM;
    }
    h->ws = static_cast<char*>(ptr);
    h->owns_ws = true;
  }
  // chain tables: identity slot order; pattern id per slot; pattern table
  auto bail = [&](cudaError_t err, const char* where) {
    snprintf(g_last_error, 256, "%s: %s", where, cudaGetErrorString(err));
    if (h->owns_ws) cudaFree(h->ws);
    free_handle(h);
    return SOMA_ECUDA;
  };
  if (p->chain_pattern) e = cudaMemcpyAsync(h->pattern0(), p->chain_pattern, h->n_chains, cudaMemcpyHostToDevice, h->stream);
  else e = cudaMemsetAsync(h->pattern0(), 0, h->n_chains, h->stream);
  if (e != cudaSuccess) return bail(e, "chain_pattern upload");
  e = cudaMemcpyAsync(h->patterns(), p->type_patterns, (size_t)h->n_patterns * h->Nstride, cudaMemcpyHostToDevice, h->stream);
  if (e != cudaSuccess) return bail(e, "type_patterns upload");
  if ((e = cudaStreamSynchronize(h->stream)) != cudaSuccess) return bail(e, "create sync");   // host buffers may go away
  for (int r = 0; r < 10; ++r) {
    h->keys.k0[r] = (uint32_t)p->seed + (uint32_t)r * kPhiloxW0;
    h->keys.k1[r] = (uint32_t)(p->seed >> 32) + (uint32_t)r * kPhiloxW1;
  }
  h->identity_order = true;
  h->path = 0;
  // chains are kept sorted by position when the system is large enough for it to matter
  h->resort_interval = h->n_chains >= 4096 ? 64 : 0;
  h->fused_chunk = 224;
  h->fused_carveout = -1;
  h->fused_lean = 1;
  h->omega_x4 = 1;
  h->packed_opt = -1;
  h->otf_opt = -1;
  h->lean_threads = 256;
  {
    auto pow2f = [](float v) { int e; return v > 0.0f && std::frexp(v, &e) == 0.5f && e > -100 && e < 100; };
    h->fast_arith = pow2f(h->a) && pow2f(h->grid.inv_hx) && pow2f(h->grid.inv_hy) && pow2f(h->grid.inv_hz) &&
                   h->grid.inv_hx >= 1.0f && h->grid.inv_hy >= 1.0f && h->grid.inv_hz >= 1.0f;
  }
  const double cells_per_step = (double)h->a * (double)fmaxf(h->grid.inv_hx, fmaxf(h->grid.inv_hy, h->grid.inv_hz));
  {
    // guard level of the packed 16-bit counters (soma_device.cuh): largest power of two G with ((2r+1)^3 + 1) G <= 65536
    h->guard_mask = 0;
    const double r = std::ceil(cells_per_step > 1.0 ? cells_per_step : 1.0);
    const double span = (2.0 * r + 1.0) * (2.0 * r + 1.0) * (2.0 * r + 1.0) + 1.0;
    if (h->smcA == 0.0f && span <= 1024.0) {                     // G >= 64
      uint32_t G = 32768u;
      while ((double)G * span > 65536.0) G >>= 1;
      h->guard_mask = (~(G - 1u) & 0xffffu) * 0x00010001u;
    }
  }
  const double k = cells_per_step > 0.0 ? 2097152.0 / cells_per_step : 1e18;
  h->range_check_interval = k >= 1e18 ? (1ull << 60) : (k < 1.0 ? 1ull : (uint64_t)k);
  // Bond-force-biased moves are Gaussian, not bounded by a: a step beyond 8 standard deviations (sqrt(2A) per
  // axis) plus the largest conceivable drift does not occur, but no bound is proven, so the range is simply
  // re-verified every 256 steps (2^21 cells of head-room against ~1 cell per step).
  if (h->smcA > 0.0f && h->range_check_interval > 256) h->range_check_interval = 256;
  *out = h;
  return SOMA_OK;
}

namespace {
// DESIGN.md section 2 step 4 for positions already in set 0: slot tables, bin(), omega(), range check, re-ordering
int finish_load(soma_handle* h, uint64_t step0) {
  int rc;
  // slot s holds chain s again
  iota_kernel<<<blocks_for(h->n_chains, 256), 256, 0, h->stream>>>((uint32_t)h->n_chains, h->slot_chain(0));
  h->launches++;
  CU(h, cudaGetLastError());
  CU(h, cudaMemcpyAsync(h->slot_pattern(0), h->pattern0(), h->n_chains, cudaMemcpyDeviceToDevice, h->stream));
  h->identity_order = true;
  h->step = step0;
  h->cur = 0;
  // 16-bit counters, two types to a word (soma_device.cuh), by default where the lean kernel then computes omega
  // from them (grids of >= 2^20 cells); on small dense grids two types in one word only add contention (cfg2: +5 %) ...
  // (never under bond-force-biased moves: their reach per step is unbounded, and they read the omega array anyway)
  h->packed = (h->packed_opt < 0 ? h->cells >= (1u << 20) : h->packed_opt != 0) && h->T <= 2 && h->guard_mask != 0;
  for (int attempt = 0; attempt < 2; ++attempt) {
    CU(h, cudaMemsetAsync(h->counts(0), 0, (size_t)h->cells * h->T * 4, h->stream));
    CU(h, cudaMemsetAsync(h->range_flag(), 0, 8, h->stream));
    if ((rc = launch_bin(h, h->counts(0), true)) != SOMA_OK) return rc;
    if ((rc = launch_omega(h)) != SOMA_OK) return rc;   // also zeroes counts(1) and raises the guard flag
    if ((rc = verify_range(h)) != SOMA_OK) return rc;   // synchronises: the caller may reuse its buffers
    if (!(h->packed && h->guard_seen)) break;
    h->packed = false;                                  // ... unless this state is too dense for them: 32-bit counters
  }
  h->steps_since_sort = 0;
  h->sorted = false;
  if (h->resort_interval > 0)
    if ((rc = resort(h)) != SOMA_OK) return rc;
  h->loaded = true;
  return SOMA_OK;
}
}  // namespace

int soma_load_state(soma_t* h, const float* x, const float* y, const float* z, uint64_t step0, int dev) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!x || !y || !z) return fail(h, SOMA_EINVAL, "position pointer is NULL");
  if (step0 >= (1ull << 48)) return fail(h, SOMA_EINVAL, "step0 must be < 2^48");
  const cudaMemcpyKind kind = dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  h->live = 0;
  h->loaded = false;
  const float* src[3] = {x, y, z};
  for (int d = 0; d < 3; ++d) CU(h, cudaMemcpyAsync(h->pos(0, d), src[d], h->B * 4, kind, h->stream));
  if (h->S)
    for (int d = 0; d < 3; ++d) CU(h, cudaMemcpyAsync(h->single(d), src[d] + h->B, h->S * 4, kind, h->stream));
  return finish_load(h, step0);
}

int soma_generate_state(soma_t* h, uint64_t gen_seed, uint64_t step0) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (step0 >= (1ull << 48)) return fail(h, SOMA_EINVAL, "step0 must be < 2^48");
  h->live = 0;
  h->loaded = false;
  GenArgs G{};
  G.k0 = (uint32_t)gen_seed; G.k1 = (uint32_t)(gen_seed >> 32);
  for (int d = 0; d < 3; ++d) G.box[d] = (double)h->box[d];
  G.sigma = (double)h->b / std::sqrt(3.0);
  for (uint32_t k = 0; k < h->n_views; ++k) {
    h->v = h->views[k];
    G.n_chains = (uint32_t)h->v.n; G.N = h->v.N; G.chain0 = (uint32_t)h->v.first_chain;
    G.x = h->vpos(0, 0); G.y = h->vpos(0, 1); G.z = h->vpos(0, 2);
    generate_state_kernel<<<blocks_for(h->v.n, 64), 64, 0, h->stream>>>(G);
    h->launches++;
    CU(h, cudaGetLastError());
  }
  if (h->S) {
    generate_singles_kernel<<<blocks_for(h->S, 256), 256, 0, h->stream>>>(
        (uint32_t)h->S, (uint32_t)h->n_chains, G.k0, G.k1, G.box[0], G.box[1], G.box[2], h->single(0), h->single(1), h->single(2));
    h->launches++;
    CU(h, cudaGetLastError());
  }
  return finish_load(h, step0);
}

namespace {
// inclusive prefix sums of the [cells] weights in h->cdf(), in place; *total receives their sum (synchronises)
int scan_weights(soma_handle* h, unsigned long long* total) {
  const uint32_t n = h->cells, chunks = (n + kScanChunk - 1) / kScanChunk;
  unsigned long long* chunk = h->cdf() + n;
  scan_chunk_sums_kernel<<<chunks, 256, 0, h->stream>>>(n, h->cdf(), chunk);
  scan_small_kernel<<<1, 1024, 0, h->stream>>>(chunks, chunk);
  scan_apply_kernel<<<chunks, 256, 0, h->stream>>>(n, h->cdf(), chunk);
  h->launches += 3;
  CU(h, cudaGetLastError());
  CU(h, cudaMemcpyAsync(total, chunk + chunks, 8, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  return SOMA_OK;
}
}  // namespace

int soma_init_from_density(soma_t* h, const float* phi_target, int dev, uint64_t gen_seed, uint64_t step0,
                           uint32_t n_equil_steps, float umbrella_k) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!phi_target) return fail(h, SOMA_EINVAL, "phi_target is NULL");
  if (step0 + n_equil_steps >= (1ull << 48)) return fail(h, SOMA_EINVAL, "step index would reach 2^48");
  if (!(umbrella_k == umbrella_k)) return fail(h, SOMA_EINVAL, "umbrella_k is NaN");
  h->live = 0;
  h->loaded = false;
  h->umbrella = false;
  const size_t TC = (size_t)h->cells * h->T;
  CU(h, cudaMemcpyAsync(h->phi_tgt(), phi_target, TC * 4, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
  // Q_t(c) in the first count buffer (re-initialised by the binning below)
  uint32_t* Q = h->counts(0);
  CU(h, cudaMemsetAsync(h->range_flag(), 0, 4, h->stream));
  quantise_target_kernel<<<blocks_for(TC, 256), 256, 0, h->stream>>>(TC, h->phi_tgt(), Q, h->range_flag());
  h->launches++;
  CU(h, cudaGetLastError());
  uint32_t bad = 0;
  CU(h, cudaMemcpyAsync(&bad, h->range_flag(), 4, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));                       // the caller's host array has been read
  if (bad) return fail(h, SOMA_EINVAL, "phi_target holds a negative, NaN or >= 65536 value");
  PlaceArgs P{};
  P.cells = h->cells; P.ny = h->grid.ny; P.nz = h->grid.nz;
  P.k0 = (uint32_t)gen_seed; P.k1 = (uint32_t)(gen_seed >> 32);
  P.hx = (double)h->box[0] / (double)h->grid.nx; P.hy = (double)h->box[1] / (double)h->grid.ny; P.hz = (double)h->box[2] / (double)h->grid.nz;
  P.sigma = (double)h->b / std::sqrt(3.0);
  P.prefix = h->cdf();
  for (uint32_t k = 0; k < h->n_views; ++k)                      // a chain's cell weights depend on its pattern and its length
  for (uint32_t pat = 0; pat < h->n_patterns; ++pat) {
    if ((*h->pattern_chains)[(size_t)k * h->n_patterns + pat] == 0) continue;
    h->v = h->views[k];
    P.n_chains = (uint32_t)h->v.n; P.N = h->v.N; P.chain0 = (uint32_t)h->v.first_chain;
    P.chain_pattern = h->pattern0() + h->v.first_chain;
    TypeCounts M{};
    for (uint32_t i = 0; i < h->v.N; ++i) M.m[(*h->host_patterns)[(size_t)pat * h->Nstride + i]]++;
    cell_weight_kernel<<<blocks_for(h->cells, 256), 256, 0, h->stream>>>(h->cells, h->T, M, Q, h->cdf());
    h->launches++;
    unsigned long long total = 0;
    if ((rc = scan_weights(h, &total)) != SOMA_OK) return rc;
    if (total == 0) return fail(h, SOMA_EINVAL, "phi_target gives a chain pattern zero total weight");
    P.pattern = pat;
    P.x = h->vpos(0, 0); P.y = h->vpos(0, 1); P.z = h->vpos(0, 2);
    place_chains_kernel<<<blocks_for(h->v.n, 128), 128, 0, h->stream>>>(P);
    h->launches++;
    CU(h, cudaGetLastError());
  }
  for (uint32_t t = 0; t < h->T && h->S; ++t) {
    const uint32_t count = h->single_start[t + 1] - h->single_start[t];
    if (count == 0) continue;
    TypeCounts M{};
    M.m[t] = 1;
    cell_weight_kernel<<<blocks_for(h->cells, 256), 256, 0, h->stream>>>(h->cells, h->T, M, Q, h->cdf());
    h->launches++;
    unsigned long long total = 0;
    if ((rc = scan_weights(h, &total)) != SOMA_OK) return rc;
    if (total == 0) return fail(h, SOMA_EINVAL, "phi_target gives a single-bead species zero total weight");
    P.x = h->single(0); P.y = h->single(1); P.z = h->single(2);
    place_singles_kernel<<<blocks_for(count, 256), 256, 0, h->stream>>>(P, h->single_start[t], count, (uint32_t)h->n_chains);
    h->launches++;
    CU(h, cudaGetLastError());
  }
  if ((rc = finish_load(h, step0)) != SOMA_OK) return rc;
  if (n_equil_steps) {                                           // equilibration under the umbrella potential, which is removed again
    h->umbrella = true;
    h->umbrella_k = umbrella_k;
    rc = launch_omega(h);
    if (rc == SOMA_OK) rc = soma_mc_steps(h, n_equil_steps, nullptr);
    h->umbrella = false;                                         // whatever happened: no later step may see the umbrella term
    if (rc == SOMA_OK) rc = launch_omega(h);
    if (rc == SOMA_OK) rc = guard_check(h);                      // the equilibration ran without a synchronising call of its own
    if (rc != SOMA_OK) {                                         // the omega array may still hold the umbrella field: the state has to be loaded again
      h->loaded = false;
      return rc;
    }
  }
  return SOMA_OK;
}

int soma_mc_steps(soma_t* h, uint32_t n_steps, uint64_t* accepted) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!h->loaded) return fail(h, SOMA_ESTATE, "soma_mc_steps before soma_load_state");
  if (h->step + n_steps >= (1ull << 48)) return fail(h, SOMA_EINVAL, "step index would reach 2^48");
  CU(h, cudaMemsetAsync(h->accepted(), 0, 8, h->stream));
  for (uint32_t s = 0; s < n_steps; ++s) {
    if (h->steps_since_check >= h->range_check_interval) {
      range_check_kernel<<<blocks_for(h->B, 256), 256, 0, h->stream>>>(
          h->grid, h->B, h->pos(h->live, 0), h->pos(h->live, 1), h->pos(h->live, 2), h->range_flag());
      h->launches++;
      CU(h, cudaGetLastError());
      if (h->S) {
        range_check_kernel<<<blocks_for(h->S, 256), 256, 0, h->stream>>>(h->grid, h->S, h->single(0), h->single(1), h->single(2), h->range_flag());
        h->launches++;
        CU(h, cudaGetLastError());
      }
      if ((rc = verify_range(h)) != SOMA_OK) return rc;
    }
    if ((rc = one_step(h)) != SOMA_OK) return rc;
  }
  if (accepted) {
    unsigned long long v = 0;
    CU(h, cudaMemcpyAsync(&v, h->accepted(), 8, cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    *accepted = v;
    return guard_check(h);
  }
  return SOMA_OK;
}

int soma_get_density(soma_t* h, uint32_t* counts, int dev) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!counts) return fail(h, SOMA_EINVAL, "counts is NULL");
  if (!h->loaded) return fail(h, SOMA_ESTATE, "no state loaded");
  if (h->packed) {                                       // unpack into the omega-sized staging area of the next count buffer's tail
    uint32_t* stage = reinterpret_cast<uint32_t*>(h->ws + h->L.stage);
    unpack_counts_kernel<<<blocks_for(h->cells, 256), 256, 0, h->stream>>>(h->cells, h->T, h->counts(h->cur), stage);
    h->launches++;
    CU(h, cudaGetLastError());
    rc = copy_out(h, counts, stage, (uint64_t)h->cells * h->T, dev);
    if (rc == SOMA_OK && !dev) rc = guard_check(h);
    return rc;
  }
  return copy_out(h, counts, h->counts(h->cur), (uint64_t)h->cells * h->T, dev);
}

int soma_get_omega(soma_t* h, float* omega, int dev) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!omega) return fail(h, SOMA_EINVAL, "omega is NULL");
  if (!h->loaded) return fail(h, SOMA_ESTATE, "no state loaded");
  if ((rc = ensure_omega(h)) != SOMA_OK) return rc;
  rc = copy_out(h, omega, h->omega(), (uint64_t)h->cells * h->T, dev);
  if (rc == SOMA_OK && !dev) rc = guard_check(h);
  return rc;
}

int soma_get_positions(soma_t* h, float* x, float* y, float* z, int dev) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!x || !y || !z) return fail(h, SOMA_EINVAL, "position pointer is NULL");
  if (!h->loaded) return fail(h, SOMA_ESTATE, "no state loaded");
  float* dst[3] = {x, y, z};
  int set = h->live;
  if (!h->identity_order) {      // back to the caller's chain order through the staging set
    set = h->live ^ 1;
    for (uint32_t k = 0; k < h->n_views; ++k) {
      h->v = h->views[k];
      unpermute_kernel<<<blocks_for(h->v.B, 256), 256, 0, h->stream>>>(
          h->v.B, h->v.N, (uint32_t)h->v.first_chain, h->vslot_chain(h->live), h->vpos(h->live, 0), h->vpos(h->live, 1), h->vpos(h->live, 2),
          h->vpos(set, 0), h->vpos(set, 1), h->vpos(set, 2));
      h->launches++;
      CU(h, cudaGetLastError());
    }
  }
  for (int d = 0; d < 3; ++d)
    CU(h, cudaMemcpyAsync(dst[d], h->pos(set, d), h->B * 4,
                          dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
  if (h->S)
    for (int d = 0; d < 3; ++d)
      CU(h, cudaMemcpyAsync(dst[d] + h->B, h->single(d), h->S * 4,
                            dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
  if (!dev) {
    CU(h, cudaStreamSynchronize(h->stream));
    return guard_check(h);                                       // positions + step index are a checkpoint: never hand one out past the guard
  }
  return SOMA_OK;
}

int soma_set_external_field(soma_t* h, const float* ext, int dev) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (ext) {
    CU(h, cudaMemcpyAsync(h->ext(), ext, (size_t)h->cells * h->T * 4,
                          dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
    if (!dev) CU(h, cudaStreamSynchronize(h->stream));           // the caller may reuse its buffer
  }
  h->has_ext = ext != nullptr;
  if (h->loaded) {                                               // omega of the current densities, with the new field
    if ((rc = launch_omega(h)) != SOMA_OK) return rc;
  }
  return SOMA_OK;
}

int soma_validate_state(soma_t* h, soma_validation* out) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!out) return fail(h, SOMA_EINVAL, "out is NULL");
  if (!h->loaded) return fail(h, SOMA_ESTATE, "no state loaded");
  unsigned long long* report = reinterpret_cast<unsigned long long*>(h->ws + h->L.validate);
  double* bond_sum = reinterpret_cast<double*>(report + 10);
  CU(h, cudaMemsetAsync(report, 0, 11 * 8, h->stream));
  uint64_t n_bonds = 0;
  for (uint32_t k = 0; k < h->n_views; ++k) {
    h->v = h->views[k];
    validate_positions_kernel<<<blocks_for(h->v.B, 256), 256, 0, h->stream>>>(
        h->v.B, h->v.N, h->vpos(h->live, 0), h->vpos(h->live, 1), h->vpos(h->live, 2), report, bond_sum);
    n_bonds += h->v.n * (uint64_t)(h->v.N - 1);
    if (k) h->launches++;
  }
  if (h->S) {      // N = 1 in the kernel: no bonds, only the finiteness test
    validate_positions_kernel<<<blocks_for(h->S, 256), 256, 0, h->stream>>>(h->S, 1u, h->single(0), h->single(1), h->single(2), report, bond_sum);
    h->launches++;
  }
  const unsigned gx = blocks_for(h->cells, 256) < 1024u ? blocks_for(h->cells, 256) : 1024u;
  validate_density_kernel<<<dim3(gx, h->T), 256, 0, h->stream>>>(h->cells, h->T, h->packed ? 1u : 0u, h->counts(h->cur), report);
  h->launches += 2;
  CU(h, cudaGetLastError());
  unsigned long long host[11];
  CU(h, cudaMemcpyAsync(host, report, sizeof host, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  std::memset(out, 0, sizeof *out);
  out->n_nonfinite = host[0];
  for (uint32_t t = 0; t < h->T; ++t) { out->density_per_type[t] = host[1 + t]; out->density_total += host[1 + t]; }
  const uint32_t qbits = (uint32_t)host[9];
  std::memcpy(&out->max_bond_sq, &qbits, 4);
  double sum;
  std::memcpy(&sum, &host[10], 8);
  out->mean_bond_sq = n_bonds ? sum / (double)n_bonds : 0.0;
  out->ok = (out->n_nonfinite == 0 && out->density_total == h->Btot) ? 1u : 0u;
  return guard_check(h);
}

int soma_get_step(soma_t* h, uint64_t* step) {
  if (!h || !step) return fail(h, SOMA_EINVAL, "NULL argument");
  *step = h->step;
  return SOMA_OK;
}

int soma_destroy(soma_t* h) {
  if (!h) return SOMA_OK;
  cudaSetDevice(h->device);
  cudaStreamSynchronize(h->stream);
  if (h->owns_ws) cudaFree(h->ws);
  free_handle(h);
  return SOMA_OK;
}

const char* soma_last_error(const soma_t* h) { return h ? h->err : g_last_error; }

int soma_set_option(soma_t* h, const char* name, int64_t value) {
  if (!h || !name) return fail(h, SOMA_EINVAL, "NULL argument");
  if (!std::strcmp(name, "path")) {
    if (value < 0 || value > 2) return fail(h, SOMA_EINVAL, "path must be 0, 1 or 2");
    if (value == 2) {
      bool any = false;
      for (uint32_t k = 0; k < h->n_views; ++k) any = any || fused_lanes(h->views[k].N) != 0;
      if (!any) return fail(h, SOMA_EINVAL, "fused path needs beads_per_chain = 2P, P a power of two <= 32");
    }
    h->path = (int)value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "kernel_timing")) {
    if (value != 0 && value != 1) return fail(h, SOMA_EINVAL, "kernel_timing must be 0 or 1");
    h->timing = value != 0;
    h->ev_used = 0;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "resort_interval")) {
    if (value < 0) return fail(h, SOMA_EINVAL, "resort_interval must be >= 0");
    h->resort_interval = value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "resort_now")) {
    int rc = check(h);
    if (rc != SOMA_OK) return rc;
    if (!h->loaded) return fail(h, SOMA_ESTATE, "no state loaded");
    return resort(h);
  }
  if (!std::strcmp(name, "fused_lean")) {              // 0: the general fused kernel even where the lean one applies
    if (value != 0 && value != 1) return fail(h, SOMA_EINVAL, "fused_lean must be 0 or 1");
    h->fused_lean = (int)value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "packed_counts")) {           // takes effect at the next soma_load_state / generate / init
    if (value < -1 || value > 1) return fail(h, SOMA_EINVAL, "packed_counts must be -1, 0 or 1");
    h->packed_opt = (int)value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "omega_otf")) {
    if (value < -1 || value > 1) return fail(h, SOMA_EINVAL, "omega_otf must be -1, 0 or 1");
    h->otf_opt = (int)value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "omega_x4")) {                // 0: the one-cell-per-thread omega kernel everywhere
    if (value != 0 && value != 1) return fail(h, SOMA_EINVAL, "omega_x4 must be 0 or 1");
    h->omega_x4 = (int)value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "lean_threads")) {
    if (value != 256 && value != 512 && value != 1024) return fail(h, SOMA_EINVAL, "lean_threads must be 256, 512 or 1024");
    h->lean_threads = (int)value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "fused_chunk")) {
    if (value < 1 || value > (1 << 20)) return fail(h, SOMA_EINVAL, "fused_chunk must be in [1, 2^20]");
    h->fused_chunk = (int)value;
    return SOMA_OK;
  }
  if (!std::strcmp(name, "fused_carveout")) {
    if (value < -1 || value > 100) return fail(h, SOMA_EINVAL, "fused_carveout must be in [-1, 100]");
    h->fused_carveout = (int)value;
    return SOMA_OK;
  }
  return fail(h, SOMA_EINVAL, "unknown option name");
}

int soma_get_counters(const soma_t* h, uint64_t* out) {
  if (!h || !out) return SOMA_EINVAL;
  out[0] = h->launches; out[1] = h->steps_done; out[2] = h->resorts;
  out[3] = 1;
  if (h->path != 1)
    for (uint32_t k = 0; k < h->n_views; ++k)
      if (fused_lanes(h->views[k].N) && !((h->Nstride & 1u) && h->n_patterns > 1) && !(h->views[k].bead_off & 1u)) out[3] = 2;    // a species of another length takes the generic kernels
  out[4] = h->packed ? 1 : 0;
  out[5] = (out[3] == 2 && use_otf(h)) ? 1 : 0;
  return SOMA_OK;
}

int soma_get_kernel_times(soma_t* h, double* ms, uint64_t* steps) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!ms || !steps) return fail(h, SOMA_EINVAL, "NULL argument");
  CU(h, cudaStreamSynchronize(h->stream));
  ms[0] = ms[1] = 0.0;
  const size_t n = h->ev_used / 3;
  for (size_t k = 0; k < n; ++k) {
    float a = 0.f, b = 0.f;
    CU(h, cudaEventElapsedTime(&a, (*h->ev)[3 * k], (*h->ev)[3 * k + 1]));
    CU(h, cudaEventElapsedTime(&b, (*h->ev)[3 * k + 1], (*h->ev)[3 * k + 2]));
    ms[0] += a; ms[1] += b;
  }
  *steps = n;
  h->ev_used = 0;
  return SOMA_OK;
}

// ---- test hooks ----------------------------------------------------------------------------------

int soma_debug_half_sweep(soma_t* h, uint32_t parity, uint64_t* accepted) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!h->loaded) return fail(h, SOMA_ESTATE, "no state loaded");
  if (parity > 1) return fail(h, SOMA_EINVAL, "parity must be 0 or 1");
  if ((rc = ensure_omega(h)) != SOMA_OK) return rc;
  CU(h, cudaMemsetAsync(h->accepted(), 0, 8, h->stream));
  for (uint32_t k = 0; k < h->n_views; ++k) {
    h->v = h->views[k];
    if ((rc = launch_half_sweep(h, parity)) != SOMA_OK) return rc;
  }
  if (parity == 0 && (rc = launch_singles(h, true, false, nullptr)) != SOMA_OK) return rc;
  if (accepted) {
    unsigned long long v = 0;
    CU(h, cudaMemcpyAsync(&v, h->accepted(), 8, cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    *accepted = v;
  }
  return SOMA_OK;
}

int soma_debug_finish_step(soma_t* h) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!h->loaded) return fail(h, SOMA_ESTATE, "no state loaded");
  if ((rc = launch_bin(h, h->counts(h->cur ^ 1))) != SOMA_OK) return rc;
  h->cur ^= 1;
  if ((rc = launch_omega(h)) != SOMA_OK) return rc;
  h->step += 1;
  return SOMA_OK;
}

int soma_debug_set_omega(soma_t* h, const float* omega) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!omega) return fail(h, SOMA_EINVAL, "omega is NULL");
  CU(h, cudaMemcpyAsync(h->omega(), omega, (size_t)h->cells * h->T * 4, cudaMemcpyHostToDevice, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  h->omega_valid = true;                                       // ... in the sense that nobody may overwrite it before the next step has used it
  h->omega_custom = true;
  return SOMA_OK;
}

namespace {
struct DevBuf {                       // tiny RAII device buffer for the debug entry points
  void* p = nullptr;
  cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 1); }
  ~DevBuf() { if (p) cudaFree(p); }
};
#define CUG(call)                                                                   \
  do {                                                                              \
    cudaError_t e_ = (call);                                                        \
    if (e_ != cudaSuccess) {                                                        \
      snprintf(g_last_error, 256, "%s: %s", #call, cudaGetErrorString(e_));         \
      return SOMA_ECUDA;                                                            \
    }                                                                               \
  } while (0)
}  // namespace

int soma_debug_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, uint64_t n) {
  if (!ctr || !key || !out) return fail(nullptr, SOMA_EINVAL, "NULL argument");
  if (n == 0) return SOMA_OK;
  DevBuf c, o;
  CUG(c.alloc(n * 16)); CUG(o.alloc(n * 16));
  CUG(cudaMemcpy(c.p, ctr, n * 16, cudaMemcpyHostToDevice));
  PhiloxKeys K;
  for (int r = 0; r < 10; ++r) { K.k0[r] = key[0] + (uint32_t)r * kPhiloxW0; K.k1[r] = key[1] + (uint32_t)r * kPhiloxW1; }
  debug_philox_kernel<<<blocks_for(n, 256), 256>>>(n, (const uint32_t*)c.p, K, (uint32_t*)o.p);
  CUG(cudaGetLastError());
  CUG(cudaMemcpy(out, o.p, n * 16, cudaMemcpyDeviceToHost));
  return SOMA_OK;
}

int soma_debug_maps(const uint32_t* words, float* t, float* u, float* lnu, float* lnu_fast, uint64_t n) {
  if (!words || !t || !u || !lnu) return fail(nullptr, SOMA_EINVAL, "NULL argument");
  if (n == 0) return SOMA_OK;
  DevBuf w, a, b, c, d;
  CUG(w.alloc(n * 4)); CUG(a.alloc(n * 4)); CUG(b.alloc(n * 4)); CUG(c.alloc(n * 4)); CUG(d.alloc(n * 4));
  CUG(cudaMemcpy(w.p, words, n * 4, cudaMemcpyHostToDevice));
  debug_maps_kernel<<<blocks_for(n, 256), 256>>>(n, (const uint32_t*)w.p, (float*)a.p, (float*)b.p, (float*)c.p, (float*)d.p);
  CUG(cudaGetLastError());
  if (lnu_fast) CUG(cudaMemcpy(lnu_fast, d.p, n * 4, cudaMemcpyDeviceToHost));
  CUG(cudaMemcpy(t, a.p, n * 4, cudaMemcpyDeviceToHost));
  CUG(cudaMemcpy(u, b.p, n * 4, cudaMemcpyDeviceToHost));
  CUG(cudaMemcpy(lnu, c.p, n * 4, cudaMemcpyDeviceToHost));
  return SOMA_OK;
}

int soma_debug_accept(const float* dE, const uint32_t* words, uint8_t* decision, uint64_t n) {
  if (!dE || !words || !decision) return fail(nullptr, SOMA_EINVAL, "NULL argument");
  if (n == 0) return SOMA_OK;
  DevBuf e, w, d;
  CUG(e.alloc(n * 4)); CUG(w.alloc(n * 4)); CUG(d.alloc(n));
  CUG(cudaMemcpy(e.p, dE, n * 4, cudaMemcpyHostToDevice));
  CUG(cudaMemcpy(w.p, words, n * 4, cudaMemcpyHostToDevice));
  debug_accept_kernel<<<blocks_for(n, 256), 256>>>(n, (const float*)e.p, (const uint32_t*)w.p, (uint8_t*)d.p);
  CUG(cudaGetLastError());
  CUG(cudaMemcpy(decision, d.p, n, cudaMemcpyDeviceToHost));
  return SOMA_OK;
}

int soma_debug_accept_fma(const float* dE, const uint32_t* words, uint8_t* decision, uint64_t n) {
  if (!dE || !words || !decision) return fail(nullptr, SOMA_EINVAL, "NULL argument");
  if (n == 0) return SOMA_OK;
  DevBuf e, w, d;
  CUG(e.alloc(n * 4)); CUG(w.alloc(n * 4)); CUG(d.alloc(n));
  CUG(cudaMemcpy(e.p, dE, n * 4, cudaMemcpyHostToDevice));
  CUG(cudaMemcpy(w.p, words, n * 4, cudaMemcpyHostToDevice));
  debug_accept_fma_kernel<<<blocks_for(n, 256), 256>>>(n, (const float*)e.p, (const uint32_t*)w.p, (uint8_t*)d.p);
  CUG(cudaGetLastError());
  CUG(cudaMemcpy(decision, d.p, n, cudaMemcpyDeviceToHost));
  return SOMA_OK;
}

int soma_debug_red_throughput(uint64_t n_counters, uint64_t n_ops, int mode, double* ms) {
  if (!ms || n_counters == 0 || n_counters >= (1ull << 32) || n_ops == 0 || mode < 0 || mode > 6) return fail(nullptr, SOMA_EINVAL, "bad argument");
  const unsigned cluster = mode == 3 || mode == 5 ? 8u : 16u;         // modes 3-6: a window in distributed shared memory
  if (mode >= 3 && cluster > 8)
    CUG(cudaFuncSetAttribute(debug_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  DevBuf c;
  CUG(c.alloc(n_counters * 4));
  CUG(cudaMemset(c.p, 0, n_counters * 4));
  const uint32_t per_thread = 64;
  const uint64_t threads = (n_ops + per_thread - 1) / per_thread;
  cudaEvent_t e0, e1;
  CUG(cudaEventCreate(&e0)); CUG(cudaEventCreate(&e1));
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {                                 // first pass warms up; best of the rest
    cudaEventRecord(e0);
    if (mode <= 2) {
      debug_red_kernel<<<blocks_for(threads, 256), 256>>>((uint32_t*)c.p, (uint32_t)n_counters, per_thread, mode);
    } else {
      cudaLaunchConfig_t cfg{};
      cfg.gridDim = dim3((blocks_for(threads, 256) + cluster - 1) / cluster * cluster);
      cfg.blockDim = dim3(256);
      cudaLaunchAttribute attr{};
      attr.id = cudaLaunchAttributeClusterDimension;
      attr.val.clusterDim.x = cluster; attr.val.clusterDim.y = 1; attr.val.clusterDim.z = 1;
      cfg.attrs = &attr; cfg.numAttrs = 1;
      cudaError_t le = cudaLaunchKernelEx(&cfg, debug_cluster_kernel, (uint32_t*)c.p, per_thread, mode >= 5 ? 1 : 0);
      if (le != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); snprintf(g_last_error, 256, "cluster launch: %s", cudaGetErrorString(le)); return SOMA_ECUDA; }
    }
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    float t = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); snprintf(g_last_error, 256, "%s", cudaGetErrorString(e)); return SOMA_ECUDA; }
    if (rep > 0 && t < best) best = t;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *ms = (double)best;
  return SOMA_OK;
}

int soma_debug_cell_index(soma_t* h, const float* x, const float* y, const float* z, uint32_t* cell, uint64_t n) {
  int rc = check(h);
  if (rc != SOMA_OK) return rc;
  if (!x || !y || !z || !cell) return fail(h, SOMA_EINVAL, "NULL argument");
  if (n == 0) return SOMA_OK;
  DevBuf a, b, c, o;
  CUG(a.alloc(n * 4)); CUG(b.alloc(n * 4)); CUG(c.alloc(n * 4)); CUG(o.alloc(n * 4));
  CUG(cudaMemcpy(a.p, x, n * 4, cudaMemcpyHostToDevice));
  CUG(cudaMemcpy(b.p, y, n * 4, cudaMemcpyHostToDevice));
  CUG(cudaMemcpy(c.p, z, n * 4, cudaMemcpyHostToDevice));
  if (h->pow2) debug_cell_kernel<true><<<blocks_for(n, 256), 256>>>(h->grid, n, (float*)a.p, (float*)b.p, (float*)c.p, (uint32_t*)o.p);
  else debug_cell_kernel<false><<<blocks_for(n, 256), 256>>>(h->grid, n, (float*)a.p, (float*)b.p, (float*)c.p, (uint32_t*)o.p);
  CUG(cudaGetLastError());
  CUG(cudaMemcpy(cell, o.p, n * 4, cudaMemcpyDeviceToHost));
  return SOMA_OK;
}

}  // extern "C"
