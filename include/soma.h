/* soma.h -- C ABI of libsoma_b200.so: the SCMF Monte-Carlo step of the SOMA particle model on one
 * NVIDIA B200 (sm_100a).
 *
 * What it computes: DESIGN.md section 2, i.e. BASELINE.json `north_star` parts (1)-(3) -- Metropolis
 * trial moves of every bead in two half-sweeps (even beads, then odd beads) scored by harmonic bond
 * energy plus the bead type's field omega at its grid cell; re-binning of all beads into per-type
 * integer density grids; omega recomputed from the densities -- the two kernels the paper reports as
 * 65 % + 25 % of SOMA's run time (section 2.2) plus the quasi-instantaneous field
 * update (section 2).  Entry-point names are the ones `north_star` lists.
 *
 * Conventions
 *   - Every function returns SOMA_OK (0) or a negative error code; nothing throws or aborts.
 *     soma_last_error(h) gives a text for the last failure on that handle.
 *   - One handle = one CUDA device (the current device at soma_create) + one CUDA stream.  All work
 *     is enqueued on that stream.  Calls that hand data back to the HOST synchronise the stream
 *     before returning; everything else is asynchronous with respect to the host.  Calls on one
 *     handle are not thread-safe.  There is no global state.
 *   - Ownership: the library copies everything it is given (parameters at create, positions at
 *     load_state).  The caller owns every buffer it passes in or receives results in.  The library
 *     owns its device memory, unless the caller lends a workspace (see soma_params.workspace).
 *   - Positions must stay within 2^21 cells of the origin (|r_d| * grid[d] / box[d] < 2^21);
 *     soma_load_state rejects others with SOMA_EINVAL and soma_mc_steps re-verifies before drift
 *     could exceed it.
 *   - Layouts: positions are structure-of-arrays fp32, x[B], y[B], z[B], B = n_chains *
 *     beads_per_chain, bead i of chain c at index c*beads_per_chain + i, UNWRAPPED (periodic images
 *     are applied only when a bead is assigned to a cell).  Grids are [type][ix][iy][iz] with iz
 *     fastest, cell = (ix*grid[1] + iy)*grid[2] + iz; densities are uint32 bead counts, omega fp32
 *     in units of kT.
 *   - "device pointer" = memory of the handle's device (e.g. a torch CUDA tensor's data_ptr);
 *     "host pointer" = ordinary or pinned host memory.  A flag argument says which.
 *   - There is no CPU fallback: without a usable sm_100 device every call fails with SOMA_ECUDA.
 */
#ifndef SOMA_B200_H
#define SOMA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SOMA_OK       0
#define SOMA_EINVAL  -1   /* NULL / out-of-range / inconsistent argument                      */
#define SOMA_ENOMEM  -2   /* device or host allocation failed, or the lent workspace is small  */
#define SOMA_ECUDA   -3   /* CUDA runtime error (sticky: later calls on the handle fail too)   */
#define SOMA_ESTATE  -4   /* call out of order (e.g. soma_mc_steps before soma_load_state)     */

typedef struct soma_handle soma_t;   /* opaque */

/* Problem statement (`north_star`: "chains, bead types, bond length b, chiN, kappaN, grid, box").
 * All chains are linear.  They have the same number of beads unless n_species > 1 (below).  Limits:
 * n_chains < 2^32, 1 <= n_types <= 8, n_types * cells < 2^32, beads_per_chain <= 65535. */
typedef struct soma_params {
  uint64_t n_chains;            /* n                                                            */
  uint32_t beads_per_chain;     /* N >= 1                                                       */
  uint32_t n_types;             /* T                                                            */
  uint32_t n_patterns;          /* >= 1                                                         */
  uint32_t n_species;           /* 0 or 1: every chain has beads_per_chain beads.  >= 2 (at most 16): polymer species
                                   of different chain lengths, see species_n_chains below                       */
  const uint8_t *type_patterns; /* host [n_patterns][N]: bead type at each position along a chain */
  const uint8_t *chain_pattern; /* host [n_chains]: pattern id of each chain, or NULL = all 0     */
  const float *chiN;            /* host [T][T]: chi*N, symmetric, zero diagonal                   */
  float b;                      /* bond length; harmonic bonds with k = 3/(2 b^2) kT (DESIGN R1)  */
  float kappaN;                 /* kappa*N, incompressibility                                     */
  float move_halfwidth;         /* a: trial displacement uniform in the cube (-a, a)^3           */
  float smc_mobility;           /* A >= 0.  0: unbiased uniform trial moves (the configs' move).  A > 0:
                                   bond-force-biased ("smart Monte Carlo") moves, the move the paper's
                                   mc_polymer_iteration performs (SURVEY.md section 8(f) row
                                   f1; R24): r' = r + A F_bonded(r) + sqrt(2A) xi, xi standard normal,
                                   accepted with min(1, e^-dE T(r'->r)/T(r->r')); move_halfwidth is then
                                   used only by the single-bead molecules (n_single), which have no bonded force
                                   and keep the uniform move.  Runs on the general fused or the generic kernels;
                                   the position range is re-verified every 256 steps.  Units: length^2/kT  */
  uint32_t grid[3];             /* cells per axis                                               */
  uint32_t reserved2;           /* must be 0                                                    */
  float box[3];                 /* periodic box lengths; cell size = box/grid                   */
  float reserved3;              /* must be 0                                                    */
  uint64_t seed;                /* Philox key                                                   */
  void *workspace;              /* device pointer lent by the caller (>= soma_workspace_bytes,
                                   256-byte aligned, must outlive the handle), or NULL = the
                                   library allocates with cudaMalloc                            */
  uint64_t workspace_bytes;     /* size of `workspace` (ignored when workspace == NULL)         */
  const uint64_t *n_single;     /* host [T] or NULL: single-bead molecules of each type next to the
                                   chains (solvent species, DESIGN.md
                                   R23).  They are stored AFTER the chains in every position array
                                   (type 0 first), so B = n_chains*N + sum(n_single); molecule m is
                                   bead 0 of logical chain n_chains + m for the random stream, moves
                                   in half-sweep 0 and has no bonds.  n_chains + sum < 2^32.     */
  const uint64_t *species_n_chains; /* host [n_species] (read only if n_species >= 2): chains of every species;   */
  const uint32_t *species_beads;    /* host [n_species]: beads per chain of every species.  Mixed chain lengths
                                   (the paper's systems hold polymer, solvent and
                                   non-solvent; R26): chains are numbered and stored
                                   species by species (species 0 first), bead i of chain c of species s at
                                   bead_off(s) + (c - first_chain(s)) * species_beads[s] + i in every position
                                   array; sum(species_n_chains) = n_chains; type_patterns rows are
                                   max(species_beads) long and a chain uses the first species_beads[s] entries of
                                   its row; beads_per_chain is then only the reference chain length N of chiN,
                                   kappaN and of the 1/N in omega.  A species whose length is not 2P (P a power of
                                   two <= 32), or whose first bead lies at an odd offset in the position arrays
                                   (an odd number of beads before it), runs on the generic kernels, the others
                                   on the fused one.                                                             */
} soma_params;

/* Device bytes a handle for `p` needs (positions x2, grids, chain tables).  0 on invalid `p`. */
uint64_t soma_workspace_bytes(const soma_params *p);

/* The problem statement becomes a handle (`north_star`: "soma_create ... whose arguments follow the paper's
 * problem statement: chains, bead types, bond length b, chiN, kappaN, grid, box"; the model itself is PAPER.md:41,
 * section 2: "soft, coarse-grained polymer model", harmonic bonds, non-bonded interactions through the
 * quasi-instantaneous field; readings R1-R3, R18).  Create a handle on the current CUDA device.  `cuda_stream` is a cudaStream_t (e.g.
 * torch.cuda.current_stream().cuda_stream), NULL = the default stream.  Copies all parameters.
 * Errors: SOMA_EINVAL (bad parameter, see limits), SOMA_ENOMEM, SOMA_ECUDA.  *out is NULL on error. */
int soma_create(const soma_params *p, void *cuda_stream, soma_t **out);

/* The state enters the library (`north_star`: "soma_load_state"; parts (2) and (3) of its step run here once: "re-binning
 * all beads into per-type integer density grids" -- the paper's update_density_fields kernel, section 2.2 --
 * and "recomputing omega from the densities", the quasi-instantaneous field of PAPER.md:41, section 2; the paper's SOMA
 * receives its start the same way, as positions reproducing a supplied image).  DESIGN.md section 2 step 4:
 * copy the positions in, set the absolute step index to `step0`, bin
 * all beads and compute omega, so that the next step sees the field of the loaded state.
 * x, y, z: [B] fp32, host or device according to `ptrs_are_device`.  (positions, step index) is a
 * complete checkpoint: the random stream is a pure function of (seed, step, half-sweep, chain,
 * bead).  Synchronises the stream before returning (also for device pointers).
 * Errors: SOMA_EINVAL (NULL pointer, NaN or out-of-range position), SOMA_ECUDA. */
int soma_load_state(soma_t *h, const float *x, const float *y, const float *z, uint64_t step0,
                    int ptrs_are_device);

/* Generate the initial state on the device instead of loading one (
 * the paper moved "generating bead coordinates" to the GPU; reading R22):
 * Gaussian random-walk chains as BASELINE.json `configs` describe them -- first bead uniform in the
 * box, bond components N(0, b^2/3), unwrapped.  Draws: Philox4x32-10, key = gen_seed, counter =
 * (bead, chain, 0, 1 << 8) (domain 1: disjoint from the Monte-Carlo stream whatever the seeds);
 * U(w) = (w + 0.5) 2^-32; bead 0 at box_d * U(w_d); bead i >= 1 at the previous bead plus
 * (b / sqrt 3) * (Box-Muller pair of (w0, w1), first of the pair of (w2, w3)), accumulated in double,
 * each coordinate rounded once to fp32.  Then exactly what soma_load_state does with those positions
 * (absolute step = step0, densities, omega).  Double-precision log/sin/cos differ in the last bit
 * between math libraries, so two implementations agree to 1 fp32 ulp on a ~1e-8 fraction of the
 * coordinates and bit for bit on the rest.  Errors: SOMA_EINVAL (step0 >= 2^48), SOMA_ECUDA. */
int soma_generate_state(soma_t *h, uint64_t gen_seed, uint64_t step0);

/* Initial state that reproduces supplied concentration fields, then equilibration under an umbrella
 * potential (section 3.2: "Each SOMA simulation begins by
 * generating particle positions that reproduce the supplied concentration fields.  Molecules are placed
 * within half a mean end-to-end distance of their target positions and equilibrated using an umbrella
 * potential").  The paper gives no rule; reading R25:
 *   phi_target [T][cells] fp32 (host or device by `ptr_is_device`), layout of omega, 0 <= value < 65536.
 *   Q_t(c) = (uint32) rint(phi_target_t(c) 2^16); a chain of pattern p draws its target cell with
 *   probability W_p(c) / sum W_p, W_p(c) = sum over its beads i of Q_type(i)(c), by inverse CDF on the
 *   integer prefix sums: k = floor((w0 2^32 + w1) sum W_p / 2^64) for (w0..w3) = Philox4x32-10(counter
 *   (0, chain, 0, 3 << 8), key = gen_seed); the target point is uniform in that cell (offsets U(w2), U(w3),
 *   U(v0), (v0..) = Philox((1, chain, 0, 3 << 8)), U(w) = (w + 0.5) 2^-32, in double); the chain is the
 *   Gaussian random walk of soma_generate_state (same domain-1 draws) translated so that its centre of
 *   mass sits at the target point, every coordinate rounded once to fp32.  Single-bead molecules of type t:
 *   weights Q_t, chain id n_chains + m, placed at the target point.  Then soma_load_state's binning and
 *   omega with step index step0.
 *   Equilibration: n_equil_steps MC steps (soma_mc_steps) during which
 *   omega_t(c) = fl32(omega_t(c) + fl32(umbrella_k * fl32(phi_t(c) - phi_target_t(c)))) -- the derivative of
 *   (umbrella_k / 2)(B / cells) sum (phi - phi_target)^2, added after any external field; afterwards the
 *   umbrella is removed and omega recomputed.  The step index ends at step0 + n_equil_steps.
 * Double log/sin/cos as in soma_generate_state: two implementations agree to 1 fp32 ulp on a tiny fraction
 * of the coordinates.  Errors: SOMA_EINVAL (NULL, bad target value, a molecule species whose target weight
 * is zero everywhere, step index >= 2^48), SOMA_ECUDA. */
int soma_init_from_density(soma_t *h, const float *phi_target, int ptr_is_device, uint64_t gen_seed,
                           uint64_t step0, uint32_t n_equil_steps, float umbrella_k);

/* Validation report of the current state (the paper's "validation functions", moved to the GPU
 * together with the generation of the coordinates): computed on the device in one
 * pass over the positions and one over the density grids; synchronises the stream. */
typedef struct soma_validation {
  uint64_t n_nonfinite;           /* coordinates that are NaN or infinite                          */
  uint64_t density_total;         /* sum of all density grids; must equal B                        */
  uint64_t density_per_type[8];   /* beads of each type in the grids                               */
  float    max_bond_sq;           /* largest squared bond length (fp32, operation order of step 5.4) */
  uint32_t ok;                    /* 1 iff n_nonfinite == 0 and density_total == B                 */
  double   mean_bond_sq;          /* mean squared bond length, accumulated in double (0 if N == 1); b^2 at equilibrium */
} soma_validation;
int soma_validate_state(soma_t *h, soma_validation *out);

/* The same report for a state the CALLER holds in device memory, without a handle and without allocating
 * anything: no cudaMalloc, no cudaFree, no library routine that allocates.  It is the one entry point of this
 * library that can be used by
 *   - a process whose device memory was handed out before it started and must not grow (the paper spawns the
 *     particle simulation next to a running continuum solver; a PyTorch host has usually given
 *     the free HBM to its caching allocator): there a late cudaMalloc can fail, or take what the neighbour needs;
 *   - a time-critical loop, where the device-wide synchronisation inside cudaMalloc / cudaFree would stall
 *     every other stream of the process;
 *   - a check of a checkpoint or of a received state before any handle (and so any workspace) exists.
 * What it computes is what soma_validate_state computes (the paper's "validation functions"):
 *   x, y, z   device [B] fp32, B = n_chains * beads_per_chain, bead i of chain c at c*beads_per_chain + i (one
 *             species per call: all chains of equal length; beads_per_chain = 1 for single-bead molecules);
 *   counts    device [n_types][cells] uint32 as soma_get_density returns them, or NULL: then the density fields of
 *             the report stay 0 and `ok` means only "no non-finite coordinate"; n_types <= 8, n_types*cells < 2^32;
 *   out       host; n_nonfinite, density_*, max_bond_sq are equal to soma_validate_state's, mean_bond_sq agrees to
 *             rounding (the sums run in another, fixed order: the same state gives the same bits on every call).
 * Scratch: the partial results live in one fixed array of 1 589 376 bytes (about 1.6 MB) that is part of the
 * library's device code, so every GPU that loads the library holds it until the process exits.  It has room for
 * 65 536 partial results of 4096 beads each: a state of more than 268 435 456 beads (2^28; the largest config has
 * 2^27) is refused with SOMA_EINVAL and a message that says so -- split it, or use soma_validate_state.
 * Sharing: all calls on one device use that one array and it keeps the last call's contents.  Every slot a call
 * reads it has written before, so nothing needs clearing and calls may follow each other freely on one stream;
 * two calls that can run on the GPU at the same time (different streams, different threads) overwrite each
 * other's partial results and both reports are then garbage.  Serialise them.
 * First call: the first call on each device looks up the array's device address (which may load the library's
 * device code).  Make that call with the device current and before any stream capture is begun; later calls on
 * that device only launch three kernels on `cuda_stream` (a cudaStream_t, NULL = default stream), copy 88 bytes
 * back and synchronise the stream.  The current device must be the one the pointers belong to.
 * errbuf (may be NULL): receives the text of the error, at most errbuf_len bytes with the terminator.
 * Errors: SOMA_EINVAL (NULL pointer, size 0, state too large for the scratch array, bad n_types / cells),
 * SOMA_ECUDA. */
int soma_validate_noalloc(const float *x, const float *y, const float *z, uint64_t n_chains, uint32_t beads_per_chain,
                          const uint32_t *counts, uint32_t n_types, uint64_t cells, void *cuda_stream,
                          soma_validation *out, char *errbuf, size_t errbuf_len);

/* The SCMF Monte-Carlo step itself, `n_steps` times (`north_star` parts (1)-(3): "Metropolis trial moves of every bead in two
 * half-sweeps (even beads, then odd beads), scored by harmonic bond energy plus the bead type's field omega at its grid
 * cell", "re-binning all beads into per-type integer density grids", "recomputing omega from the densities"; in the paper:
 * mc_polymer_iteration "performs biased trial moves and energy evaluations" (65 % of SOMA's run time) and
 * update_density_fields "updates particle density fields" (25 %), section 2.2, with the non-bonded interactions
 * in the quasi-instantaneous-field approximation, section 2).  DESIGN.md section 2 step 6: half-sweep(even),
 * half-sweep(odd), bin, omega, step += 1.  With packed 16-bit counters the guard flag is looked at whenever this call
 * synchronises by itself (every range-check interval, and at the end if `accepted` is given), so a guard hit surfaces after a
 * bounded number of steps and at the latest at the next synchronising call of any kind.  `accepted` (host pointer, may be NULL) receives the number of accepted moves of this
 * call; passing it synchronises the stream, passing NULL keeps the call asynchronous.
 * n_steps == 0 is a no-op.  Errors: SOMA_ESTATE (no state loaded), SOMA_ECUDA. */
int soma_mc_steps(soma_t *h, uint32_t n_steps, uint64_t *accepted);

/* Integer bead counts of the current configuration, [T][cells] uint32, host or device: the per-type density
 * grids of DESIGN.md section 2 step 2 (`north_star` part (2), "re-binning all beads into per-type density
 * grids"; the paper's update_density_fields kernel; nearest-grid-point assignment, R9), as the last
 * soma_load_state / soma_mc_steps left them.  Host destination: synchronises.  Errors: SOMA_EINVAL (NULL),
 * SOMA_ESTATE (no state loaded), SOMA_ECUDA. */
int soma_get_density(soma_t *h, uint32_t *counts, int ptr_is_device);

/* Current positions in the caller's (chain, bead) order, unwrapped, [B] each, host or device: the state the
 * half-sweeps of DESIGN.md section 2 step 5 (`north_star` part (1); the paper's mc_polymer_iteration kernel,
 * PAPER.md:77) have produced.  The library keeps the chains in an order of its own in memory (sorted by
 * position); this call undoes it.  Together with soma_get_step this is a complete checkpoint.  Host
 * destination: synchronises.  Errors: SOMA_EINVAL (NULL), SOMA_ESTATE (no state loaded), SOMA_ECUDA. */
int soma_get_positions(soma_t *h, float *x, float *y, float *z, int ptrs_are_device);

/* Current field omega, [T][cells] fp32 (helper; not in north_star's list). */
int soma_get_omega(soma_t *h, float *omega, int ptr_is_device);

/* External field (the SOMA side of the paper's "umbrella potential"
 * equilibration; reading R21): ext [T][cells] fp32, in kT per bead, same
 * layout as omega.  From now on omega_t(c) = fl32(fl32(invN * acc) + ext_t(c)) -- DESIGN.md section 2
 * step 3 plus one fp32 add.  The array is copied (host arrays: before the call returns); omega of
 * the current configuration is recomputed at once if a state is loaded, so the next step sees the
 * field.  ext == NULL removes it.  It survives soma_load_state.  Errors: SOMA_ECUDA. */
int soma_set_external_field(soma_t *h, const float *ext, int ptr_is_device);

/* Absolute step index (step0 + steps done). */
int soma_get_step(soma_t *h, uint64_t *step);

/* Free everything the library allocated (the last of `north_star`'s six calls): waits for the handle's
 * stream, frees the workspace unless the caller lent it, and the handle.  soma_destroy(NULL) is a no-op
 * returning SOMA_OK. */
int soma_destroy(soma_t *h);

/* Text of the last error on `h` ("" if none).  h == NULL: text of the last failed soma_create /
 * debug call of this thread. */
const char *soma_last_error(const soma_t *h);

/* Tuning / test switches.  Names:
 *   "path"            0 = automatic (the fused kernel where N allows it, else the generic ones),
 *                     1 = generic kernels (4 launches/step, any N),
 *                     2 = fused chain-in-registers kernel (N = 2P, P a power of two <= 32; else EINVAL).
 *                         Where the geometry allows it -- power-of-two grid, cell size a power of two
 *                         <= 1, move half-width a power of two, uniform moves -- this is the lean kernel
 *                         of soma_lean.cuh, else the general one of soma_kernels.cuh
 *   "fused_lean"      0 = path 2 always runs the general fused kernel (default 1)
 *   "fused_carveout"  preferred shared-memory carve-out of the fused kernel in percent (-1 = driver default; tuning)
 *   "kernel_timing"   1 = record CUDA events on the handle's stream around the kernels of every step
 *                     (read them with soma_get_kernel_times), 0 = off (default)
 *   "resort_interval" re-order the chains in memory by position at soma_load_state and then every k
 *                     steps (0 = never; default 64 for >= 4096 chains, else 0); results are
 *                     independent of it (the random stream is keyed by the logical chain id)
 *   "resort_now"      re-order once, now (value ignored)
 *   "fused_chunk"     warp groups (32 bead pairs each) per block of the fused kernel (default 224; tuning)
 *   "lean_threads"    threads per block of the lean kernel: 256 (default), 512 or 1024 (tuning)
 *   "packed_counts"   1 = in systems of one or two types (uniform moves) the density counters are kept as 16-bit fields,
 *                     two types to a 32-bit word, whenever no cell of the loaded state holds G or more beads of a type,
 *                     G = the guard level: the largest power of two with ((2r+1)^3 + 1) G <= 65536, r = the move reach
 *                     in cells (r = 1: G = 2048, a hundred times the configs' densities).  Decided at soma_load_state /
 *                     soma_generate_state / soma_init_from_density, which fall back to 32-bit counters by themselves.
 *                     Every non-empty cell is looked at in every step; should a field reach G during a run, the next
 *                     call that synchronises fails with SOMA_EINVAL (before any field can have wrapped: one step adds
 *                     at most the beads of the (2r+1)^3 cells around) and the state has to be loaded again with this
 *                     option 0.  0 = 32-bit counters.  -1 (default) = 1 for
 *                     grids of 2^20 cells or more, else 0.  soma_get_density returns uint32 [T][cells] either way.
 *                     Takes effect at the next load
 *   "omega_otf"       1 = with packed counters and neither an external field nor an umbrella potential the lean
 *                     kernel computes omega from the previous step's counters itself (DESIGN.md section 2 step 3 in
 *                     its operation order) and the omega array is only filled when it is asked for (soma_get_omega,
 *                     the generic kernels, single-bead molecules); 0 = omega array every step; -1 (default) = 1 for
 *                     grids of 2^20 cells or more (where it is faster), else 0.  Same results either way
 *   "omega_x4"        0 = the one-cell-per-thread omega kernel also where the four-cells-per-thread one applies
 *                     (cells a multiple of 4, at most 3 types; default 1; same results)
 * Errors: SOMA_EINVAL (unknown name / unsupported value). */
int soma_set_option(soma_t *h, const char *name, int64_t value);

/* Counters since soma_create: [0] kernels launched by this library, [1] MC steps done,
 * [2] chain re-orderings done; [3] the kernel path the next step will take (1 or 2); [4] 1 if the density
 * counters of the loaded state are packed 16-bit fields; [5] 1 if the next step computes omega on the fly
 * (options "packed_counts", "omega_otf").  `out` is a host pointer to 6 uint64. */
int soma_get_counters(const soma_t *h, uint64_t *out);

/* Device time spent since the last call (or since "kernel_timing" was switched on), summed over the
 * recorded steps (at most 16384 between two reads): ms[0] = rows a1+a2+a3 (the move and binning
 * kernels), ms[1] = row a4 (the omega kernel); *steps = number of steps recorded.  Synchronises the
 * stream.  `ms` is a host pointer to 2 doubles. */
int soma_get_kernel_times(soma_t *h, double *ms, uint64_t *steps);

/* ---- test hooks (used by tests/ only; each runs on the device) --------------------------------- */

/* One half-sweep only (DESIGN.md section 2 step 5); omega, densities and the step index are left
 * untouched.  `accepted` as in soma_mc_steps. */
int soma_debug_half_sweep(soma_t *h, uint32_t parity, uint64_t *accepted);
/* bin + omega + step += 1 (the rest of step 6 after two soma_debug_half_sweep calls). */
int soma_debug_finish_step(soma_t *h);
/* Overwrite omega with caller-supplied values ([T][cells], host pointer): frozen-field tests. */
int soma_debug_set_omega(soma_t *h, const float *omega);
/* Device evaluation of the pieces of DESIGN.md section 2 step 5.1-5.2 on host arrays:
 * philox: ctr [n][4], key [2] -> out [n][4];  maps: words [n] -> tmap [n], u [n], lnu [n] (lnu by the
 * kernel's slow path, i.e. the value it uses when a move is near the threshold), lnu_fast [n] (may
 * be NULL; the hardware-logarithm value that decides every move outside the +-1e-4 band);
 * accept: dE [n], words [n] -> decision [n] (0/1) by the kernel's full fast+slow accept routine
 * (generic kernels); accept_fma: the same rule by the routine of the fused kernels (one FFMA on the
 * hardware logarithm, guard band, exact logarithm inside the band). */
int soma_debug_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n);
int soma_debug_maps(const uint32_t *words, float *tmap, float *u, float *lnu, float *lnu_fast, uint64_t n);
int soma_debug_accept(const float *dE, const uint32_t *words, uint8_t *decision, uint64_t n);
int soma_debug_accept_fma(const float *dE, const uint32_t *words, uint8_t *decision, uint64_t n);
/* Throughput of the density increments on their own (`north_star`: "the atomic throughput of the histogram"):
 * ceil(n_ops / 64) * 64 increments by threads of 64 each into n_counters uint32 counters of a scratch buffer.
 * mode 0: red.global at uniformly random counters; 1: red.global with the locality of the sorted melt (the 32 lanes
 * of a warp fall into a moving window of 2048 counters); 2: red.shared at random counters of a 32 KB window per
 * block.  Modes 3-6 probe a window spread over the shared memories of a thread-block cluster (8192 words per CTA;
 * n_counters is not used): 3 / 4: red.shared::cluster at uniformly random words of an 8- / 16-CTA cluster's window;
 * 5 / 6: ld.shared::cluster gathers with the sorted-melt locality over an 8- / 16-CTA cluster.
 * *ms (host) = best of three timed launches, CUDA events.  Errors: SOMA_EINVAL, SOMA_ECUDA. */
int soma_debug_red_throughput(uint64_t n_counters, uint64_t n_ops, int mode, double *ms);
/* Cell index of host positions under the handle's grid/box. */
int soma_debug_cell_index(soma_t *h, const float *x, const float *y, const float *z, uint32_t *cell,
                          uint64_t n);

#ifdef __cplusplus
}
#endif
#endif /* SOMA_B200_H */
