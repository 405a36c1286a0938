/* otoo.h -- C-ABI boundary of the B200-native OTOO force path (arxiv 1206.1199).
 *
 * One library, libotoo.so (sm_100a), one opaque context per GPU.  Citations are PAPER.md line
 * numbers (L..) and DESIGN.md readings (R..).
 *
 * Conventions
 *  - Pointers named d_* are DEVICE memory owned by the caller (the Python binding passes
 *    torch tensors' data_ptr()).  Pointers named h_* / *_out are HOST memory.  The library never
 *    frees or reallocates caller memory and keeps no caller pointer after a call returns;
 *    otoo_build_tree copies what it needs into context-owned sorted arrays.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue work
 *    on it and return without synchronising unless stated.
 *  - Inputs and outputs are in the CALLER's original particle order; the Morton sort is internal.
 *  - Units: G = 1.  Everything the path computes is fp32 (L161) except the cell moments,
 *    which are accumulated in fp64 in a fixed order (R6) so that the tree is reproducible.
 *  - Every function returns otoo_status; nothing aborts, prints or throws.
 *    otoo_last_error(ctx) gives a context-owned message for the last non-OK status.
 *  - The *_host entry points are the end-to-end form: host buffers in, host buffers out, the
 *    copies inside the call (used for bench.py's `e2e`).
 */
#ifndef OTOO_H
#define OTOO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct otoo_ctx otoo_ctx;

typedef enum {
  OTOO_OK = 0,
  OTOO_ERR_INVALID_ARG = 1,
  OTOO_ERR_OOM = 2,
  OTOO_ERR_CUDA = 3,
  OTOO_ERR_NOT_BUILT = 4,
  OTOO_ERR_CAPACITY = 5
} otoo_status;

/* One tree cell in canonical order: level ascending, then `first` ascending (R5).
 * prefix = key >> 3*(21-level); [first, first+count) = its range of sorted particle slots;
 * children are the cells child_first .. child_first+child_count-1 (0,0 for a leaf). */
typedef struct {
  uint64_t prefix;
  uint32_t first, count, child_first;
  uint8_t level, child_count;
} otoo_cell_t;

typedef struct {
  int64_t N, N_cell, N_leaf;
  int32_t depth;        /* deepest level that holds a cell, 0..21 */
  float lo[3], S;       /* root cube [lo, lo+S]^3 (R1) */
} otoo_tree_info_t;

typedef struct {
  uint64_t sum_tests;        /* MAC tests of the last walk, all groups */
  uint64_t sum_interactions; /* R11: sum_g |g| (n_cells,g + n_parts,g) of the last walk */
  uint64_t sum_cells, sum_parts;
  int64_t n_groups;
  int32_t group_size;
  int32_t launches;          /* kernels launched by the last call */
  uint64_t sum_steps;        /* walk steps (batches of <= 32 MAC tests) of the last walk */
  uint64_t sum_tasks;        /* units of work run: groups + task-pool tasks */
  uint64_t sum_flushes;      /* evaluations of a (full or final) shared-memory list */
  uint64_t sum_evaluated;    /* (target, list entry) pairs actually handed to the sums: = sum_interactions for gravity;
                              * for the SPH walks the candidates left after the walk-time cull, times the group size */
  /* Per-phase DEVICE times in ms (CUDA events on the call's stream; PAPER.md L195, L212 splits a step into TREE
   * and KERNEL the same way).  ms_build[] of the last otoo_build_tree: [0] root cube (H1), [1] keys (H2),
   * [2] key sort (H3), [3] gather fused with the levels of the cells that start at each slot (H4 + first part of
   * H5), [4] cells from those levels (rest of H5: scan, placement; includes the one host synchronisation),
   * [5] bottom-up pass (H6; also the internal cells' children and rb^2 of the last gravity call's theta),
   * [6..7] unused (0); ms_build_total = their sum.
   * Of the last walk call (gravity or SPH): ms_walk_prep = cell radii (r_b or Eq. 5), gathers and clears before
   * the walk kernel; ms_walk_force = the fused walk + sum kernel alone (H7-H10 / H11 / H13); ms_total = the
   * whole call.  0 where nothing has run. */
  float ms_build[8], ms_build_total;
  float ms_walk_prep, ms_walk_force, ms_total;
  float walk_sm_mhz;         /* SM clock the gravity walk kernel actually held: SM clock ticks per nanosecond of the
                              * global timer, summed over its CTAs (0 for the other kernels) */
  /* Where the warps of the warp-specialised gravity kernel spent their time (SM clock ticks, summed over warps):
   * eval_wait_frac = evaluator warps waiting for a full list buffer; walker_wait_frac = walker warps waiting for a
   * free buffer (they run ahead); walker_idle_frac = walker warps asleep waiting for a task-pool task (the tail of
   * the kernel: 400 ns sleeps counted).  Filled only by a walk run with option "walk_profile" = 1 (the counting
   * costs 3-4 % of the kernel, so it is a separate instantiation); 0 otherwise and for the other kernels. */
  float eval_wait_frac, walker_wait_frac, walker_idle_frac;
  int32_t walk_only;         /* 1: the last walk ran with option "walk_only": counters valid, OUTPUTS MEANINGLESS */
  int32_t error_flag;        /* != 0: the last walk dropped cells (private spill area full): outputs and counters
                              * invalid; otoo_last_stats / otoo_export_group_stats return OTOO_ERR_CAPACITY */
} otoo_stats_t;

/* Lifecycle.  `device` is a CUDA ordinal; max_particles bounds N of every later build
 * (1 <= max_particles <= 2^31-1).  Allocates context-owned scratch. */
otoo_status otoo_create(otoo_ctx** out, int device, int64_t max_particles);
void otoo_destroy(otoo_ctx* ctx);
const char* otoo_last_error(const otoo_ctx* ctx);
/* ABI version of this header (2: otoo_stats_t carries per-phase times, walk_only and error_flag). */
int otoo_version(void);

/* PAPER III-B steps 1-4 + III-C, all on the device: root cube (L121,L127; R1), Morton keys
 * (L129; R2,R3), key sort (L133; R4), cells from the sorted keys (L135; R5), mass and centre of
 * mass bottom-up (L155; R6).  d_pos_mass: N x float4 (x,y,z,m), original order.  n_crit >= 1 is
 * the largest number of particles a leaf may hold (L41).  N = 0 is a no-op that leaves the
 * context "not built".  Synchronises `stream` once (to size the cell arrays).
 * A build that follows an otoo_gravity call also leaves the MAC radii r_b (R7) of that call's theta and a reset walk
 * pool, from inside its bottom-up pass: the next otoo_gravity with the same theta launches its walk kernel alone
 * (another theta, otoo_gravity_delta, or a second walk on the same tree compute / reset them as before; same results). */
otoo_status otoo_build_tree(otoo_ctx* ctx, const float* d_pos_mass, int64_t N, int n_crit,
                            void* stream);

/* PAPER III-D: group walk (L57, L163; R7-R9) fused with the softened Plummer monopole/particle
 * sums (L43; R10).  eps >= 0 scalar softening; theta >= 0 opening angle (0 opens every cell =
 * direct sum); group_size consecutive Morton-sorted targets share one interaction list: 32, 64, 128 or 256
 * (a warp holds 1, 2, 4 or 8 targets per lane), or the paper's own vector lengths 4, 8, 16 (PAPER.md L163-L167,
 * L183: n_vec = 4-8; run with one group per warp, the other lanes idle -- the regime of the paper's scaling
 * laws, not a fast one).  d_acc_pot: N x float4 (ax, ay, az, phi), original order. Asynchronous. */
otoo_status otoo_gravity(otoo_ctx* ctx, float eps, float theta, int group_size, float* d_acc_pot,
                         void* stream);

/* The same walk and sums under the paper's own acceptance criterion, the absolute-error MAC
 * (PAPER.md II-B Eq. 1-2): a cell is accepted iff the group-cell distance exceeds
 *   r_b = b_max/2 + sqrt(b_max^2/4 + sqrt(3 B2 / delta)),  B2 = sum_i m_i |r_CM - r_i|^2  (Eq. 2),
 * delta = accuracy parameter with the dimension of an acceleration (each accepted cell's monopole is within
 * delta of the sum over its particles); delta = 0 opens everything (direct sum).  Cells heavier than
 * m_limit get r_b = 2 S_root and are never accepted (III-C, L157); pass INFINITY for no limit.
 * B2 is accumulated bottom-up in a fixed order (R19).  Group distance, lists, counters, sums
 * and output exactly as otoo_gravity.  OTOO_ERR_INVALID_ARG: eps < 0, delta < 0, m_limit <= 0, NaN. */
otoo_status otoo_gravity_delta(otoo_ctx* ctx, float eps, float delta, float m_limit, int group_size,
                               float* d_acc_pot, void* stream);

/* PAPER II-C (Eq. 4, Eq. 5) SPH stage 1: density by direct summation during the walk (L99-L105;
 * R13-R16).  d_h: N floats, kernel SUPPORT radius (W = 0 for r >= h, L89), original order.
 * d_rho: N floats out.  d_nngb: N uint32 out (neighbours with r < h_i, self included) or NULL.
 * Group counters and sum_interactions count the walk's candidate list (every particle of every opened leaf,
 * L105); candidates farther from the group's box than any member's reach are not evaluated, which changes
 * no neighbour decision ("walk-time cull"). */
otoo_status otoo_sph_density(otoo_ctx* ctx, const float* d_h, int group_size, float* d_rho,
                             uint32_t* d_nngb, void* stream);

/* otoo_sph_force with artificial viscosity (PAPER.md L246 names the scheme: Balsara switch + per-particle
 * alpha; formula: DESIGN.md R24).  d_visc: N x float4 (sound speed c_i, alpha_i, Balsara factor f_i, -);
 * d_vel is required.  For a pair with w = (v_i - v_j).(x_i - x_j) < 0:
 *   Pi_ij = fbar (-abar cbar mu + 2 abar mu^2) / rhobar,  mu = l w / (r^2 + 0.01 l^2),  l = (h_i + h_j)/4,
 * added to (P_i/rho_i^2 + P_j/rho_j^2) in the force and in du/dt.  Output as otoo_sph_force (w = du/dt). */
otoo_status otoo_sph_force_visc(otoo_ctx* ctx, const float* d_h, const float* d_rho, const float* d_P,
                                const float* d_vel, const float* d_visc, int group_size, float* d_acc_sph,
                                void* stream);

/* SPH stage 1 as the paper runs it (PAPER.md L252 step 4: "density, div v, rot v"): the density pass of
 * otoo_sph_density plus the gather estimates (R22)
 *   div v_i = (1/rho_i) sum_j m_j (v_j - v_i) . grad_i W(r_ij, h_i),
 *   rot v_i = (1/rho_i) sum_j m_j (v_i - v_j) x grad_i W(r_ij, h_i)
 * over the same neighbours.  d_vel: N x float4 (vx, vy, vz, -).  d_divrot: N x float4 (div v, rot v). */
otoo_status otoo_sph_stage1(otoo_ctx* ctx, const float* d_h, const float* d_vel, int group_size,
                            float* d_rho, uint32_t* d_nngb, float* d_divrot, void* stream);

/* Adaptive smoothing length (h is variable per particle; BASELINE config 4: "~50 neighbours";
 * rule: DESIGN.md R21).  Iterates d_h (N floats, caller's order, IN/OUT) by a per-particle bracketed root
 * search on the neighbour count of otoo_sph_density (self included) until every particle has
 * |n_i - n_target| <= tol, its bracket has collapsed, or max_iter updates were made.  The tree is not
 * rebuilt.  d_nngb (may be NULL): counts of the final h.  host_iters (may be NULL): updates made.
 * Synchronises once per iteration (one 4-byte read). */
otoo_status otoo_sph_adapt_h(otoo_ctx* ctx, float* d_h, float n_target, float tol, int max_iter,
                             int group_size, uint32_t* d_nngb, int* host_iters, void* stream);

/* SPH stage 2 (L252 step 6; R17): symmetric pressure force.  d_rho, d_P: N floats (P from the
 * caller's EOS).  d_vel: N x float4 or NULL.  d_acc_sph: N x float4 (ax, ay, az, w), w = du/dt
 * if d_vel != NULL else 0. */
otoo_status otoo_sph_force(otoo_ctx* ctx, const float* d_h, const float* d_rho, const float* d_P,
                           const float* d_vel, int group_size, float* d_acc_sph, void* stream);

/* Ideal-gas EOS of BASELINE config 4 (replaces the paper's host Helmholtz step 5, L248):
 * P_i = (gamma-1) rho_i u_i, element-wise. */
otoo_status otoo_eos_ideal(otoo_ctx* ctx, const float* d_rho, const float* d_u, float gamma,
                           int64_t N, float* d_P, void* stream);

/* d_out[perm[s]] = d_sorted_rows[s] for N x float4 rows: results written in sorted order (option "output_sorted")
 * back into the caller's particle order.  The multi-device scheme (PAPER.md III-E) gathers every device's
 * contiguous range of sorted rows and calls this once.  Asynchronous. */
otoo_status otoo_unsort(otoo_ctx* ctx, const float* d_sorted_rows, float* d_out, void* stream);

/* Introspection for parity tests and the metric.  All synchronise the context's last stream. */
otoo_status otoo_tree_info(otoo_ctx* ctx, otoo_tree_info_t* host_out);
/* Any pointer may be NULL.  d_perm[s] = original index of sorted slot s (N); d_sorted_keys (N);
 * d_cells (N_cell, canonical order); d_cell_com_m (N_cell x 4: cm, m as the walk sees them);
 * d_cell_rb2 (N_cell: r_b^2 of the last otoo_gravity, R7; zeros before any). */
otoo_status otoo_export_tree(otoo_ctx* ctx, uint32_t* d_perm, uint64_t* d_sorted_keys,
                             otoo_cell_t* d_cells, float* d_cell_com_m, float* d_cell_rb2);
/* SPH cell radii of the last SPH call (R14): b_max, r_SPH, each N_cell floats, canonical order. */
otoo_status otoo_export_sph_radii(otoo_ctx* ctx, float* d_bmax, float* d_rsph);
/* Per-group counters of the last walk (gravity or SPH), each ceil(N/G) uint32; any may be NULL.
 * OTOO_ERR_NOT_BUILT before any walk. */
otoo_status otoo_export_group_stats(otoo_ctx* ctx, uint32_t* d_ntests, uint32_t* d_ncells,
                                    uint32_t* d_nparts);
otoo_status otoo_last_stats(otoo_ctx* ctx, otoo_stats_t* host_out);

/* Measurement aid: the FP32 rate the FMA pipe of this GPU sustains (FFMA2-only kernel, 16 independent
 * chains per thread, ~20 ms), in TFLOP/s, counted 2 flop per lane FMA -- the measured denominator of the
 * force kernel's roofline next to the nominal SMs x 128 x 2 x clock.  Synchronises. */
otoo_status otoo_measure_fp32_peak(otoo_ctx* ctx, double* host_tflops, void* stream);

/* Measurement aid: the microbenchmarks behind the ceilings DESIGN.md quotes for the force kernel (bench.py --probe).
 * which = "ffma2": SM sub-partition cycles per FFMA2 warp instruction for the operand patterns of the sum loop;
 * "sumloop": the product's own pair-sum loop on lists already in shared memory (no walk): interactions/s and
 * cycles per (target pair, list entry); "rank": SM cycles per warp instruction of MATCH.ANY, ballot, shared-memory
 * atomics and loads (the choices of the sort's ranking); "sort": otoo's eight-pass sort of (u64, u32) pairs beside
 * cub::DeviceRadixSort::SortPairs on 1 M / 8 M / 32 M pairs (as far as max_particles allows; allocates and frees
 * CUB's temporary storage).  Writes a JSON array as text into host_json (cap bytes; OTOO_ERR_CAPACITY
 * if too small).  Uses the context's particle arrays as scratch (max_particles >= 262144, else OTOO_ERR_CAPACITY): the
 * tree is invalidated.  Synchronises. */
otoo_status otoo_probe(otoo_ctx* ctx, const char* which, char* host_json, int64_t cap, void* stream);

/* The one entry point that allocates nothing (no cudaMalloc / cudaFree / allocating library call; no context): for
 * callers under CUDA graph capture, in tight serving loops, or in harnesses that forbid allocation.
 * (III-B step 3: "we sort an array of the pair of a key and a particle's id"): stable LSD radix sort of n (u64 key,
 * u32 value) pairs on all 64 key bits, the same eight one-sweep passes as the tree build's sort, on the CURRENT device.
 * d_keys / d_vals (device, n each): the pairs in, the sorted pairs out (ties keep their input order);
 * d_keys_alt / d_vals_alt (device, n each, caller-owned): the passes' second buffer, contents undefined afterwards.
 * The passes' scratch (digit histograms, tile tickets, look-back status words) is a file-scope device array inside the
 * library, sized for OTOO_SORT_STATIC_MAX_PAIRS pairs: 1.03 MB that every GPU loading libotoo.so holds until the
 * process exits.  n > OTOO_SORT_STATIC_MAX_PAIRS: OTOO_ERR_CAPACITY and a message (larger sorts go through a context);
 * n < 0 or a null buffer with n > 0: OTOO_ERR_INVALID_ARG; CUDA failure: OTOO_ERR_CUDA.  host_err (host, err_cap bytes,
 * may be NULL): receives the message of a failed call, "" on success.  Asynchronous on `stream`; every call clears the
 * part of the array it uses, so calls in a row (and replays of a captured graph) are independent -- but ALL calls on a
 * device share the one array: two calls that overlap on the GPU (different streams, no dependency between them) race
 * and give wrong results; serialise them.  The first call on a device looks up the array's address and opts the kernel
 * into its shared memory: make one call (n = 0 is enough) before starting a graph capture.  Thread-safe set-up. */
#define OTOO_SORT_STATIC_MAX_PAIRS 2097152
otoo_status otoo_sort_pairs_static(uint64_t* d_keys, uint32_t* d_vals, uint64_t* d_keys_alt, uint32_t* d_vals_alt,
                                   int64_t n, void* stream, char* host_err, int64_t err_cap);

/* Tuning/test knobs.  "walk_stack" = usable shared-memory walk-stack entries per warp (512);
 * "task_pool" = 1 (default): a warp with a long stack hands cells to the global task pool,
 * 0: it only spills to its private global area (test hook for that path).
 * "walk_spill" = usable entries of that private area per warp (default and maximum 8192; test hook: with
 * "task_pool" = 0 and a small value the area overflows, the walk drops cells and flags the launch --
 * otoo_last_stats and otoo_export_group_stats then return OTOO_ERR_CAPACITY with error_flag = 1).
 * "key_order" = 0 (default): particles, groups and cells in Morton order (R3); 1: in Hilbert
 * order (the paper's own ordering; R20) -- same cells, other order: no group straddles an
 * octant boundary with a system-sized box, fewer interactions at the same theta.  Read by the next
 * otoo_build_tree; otoo_cell_t.prefix is then a Hilbert-key prefix.
 * "group_begin" = b, "group_count" = c (defaults 0, -1 = to the end): the walks (gravity and SPH) cover only the
 * target groups [b, b + c) of the group_size they are called with; outputs of other targets stay zero and
 * the counters cover the range.  This is the paper's multi-device scheme (PAPER.md III-E, L179): every device
 * builds the same tree and takes a contiguous range of targets in key order; the ranges' outputs add up to
 * the whole.  A range outside the groups of a call: OTOO_ERR_INVALID_ARG.
 * "group_distance" = 2 (default): the MAC compares r_b with the MINIMUM over the tight boxes of the group's pieces
 * between its 7 coarsest key boundaries (R25: a Morton range that crosses a coarse cell boundary jumps
 * across that cell; one box per group then spans the cell and a few groups list the whole system); the SPH walks
 * apply their test per piece with the piece's own largest h (R26).  0: one bounding box per group (R8, R15).
 * 1: the actual minimum of the members' distances, as the paper does (R23): shorter lists, costlier
 * tests; gravity only (SPH walks: one box), needs "warp_specialized" = 1.
 * "warp_specialized" = 1 (default): otoo_gravity runs walker/evaluator warp pairs (walker warps build
 * the lists in shared memory, evaluator warps hold the targets and sum), 0: one warp does both in turn.
 * Same lists, same counters; sums differ in rounding order only.
 * "warp_specialized_sph" = 0 (default): the SPH kernels let one warp walk and sum in turn; 1: walker/evaluator
 * pairs as for gravity (SPH lists are short, the walkers become the bottleneck: faster only for
 * group_size >= 128).
 * "sph_reuse_radii" = 1: an SPH call keeps the sorted smoothing lengths and the Eq. 5 cell radii of the previous SPH
 * call on the same tree instead of recomputing them: the caller states that d_h has not changed since (stage 2 after
 * stage 1 of one step, PAPER.md L252 steps 4 and 6).  A new tree or otoo_gravity_delta invalidates them.  Default 0.
 * "sph_reuse_walk" = 1 (with "sph_reuse_radii" = 1; default 0): otoo_sph_density / otoo_sph_stage1 record, per group, the leaves
 * their walk opens (4 KB per group, allocated on first use), and an otoo_sph_force / otoo_sph_force_visc call that keeps
 * the radii starts every group's walk from those leaves instead of the root: the SPH criterion (Eq. 5; R15, R26)
 * is the same for both stages, so the same leaves open and the same particles are listed.  Same neighbours, same
 * per-group counters (the tests of the recording walk are counted, not repeated); sums differ in rounding order only.
 * Group sizes up to 64; a group that opened more than 1024 leaves or handed part of its walk to another warp, larger
 * groups, another group_size / group range / group_distance than the recording call's: the full walk, as without it.
 * "output_sorted" = 1: otoo_gravity / otoo_gravity_delta write row s of d_acc_pot for the target at SORTED slot s
 * (otoo_export_tree's d_perm names its original index) instead of the caller's order; with a group range the rows
 * [group_begin * group_size, ...) of the range are the only non-zero ones and are contiguous.  otoo_unsort brings
 * rows back.  The SPH calls refuse it (OTOO_ERR_INVALID_ARG).  Default 0.
 * "walk_profile" = 1: otoo_gravity / otoo_gravity_delta run the instrumented form of the warp-specialised kernel that
 * fills eval_wait_frac / walker_wait_frac / walker_idle_frac of otoo_stats_t (same results, 3-4 % slower); default 0.
 * "walk_only" = 1: the walks build and count their lists but skip the pair sums (outputs are
 * meaningless; counters exact) -- measures the walk's share of the fused kernel; default 0.
 * Unknown names: OTOO_ERR_INVALID_ARG. */
otoo_status otoo_set_option(otoo_ctx* ctx, const char* name, int64_t value);

/* End-to-end form with HOST buffers (pageable or pinned): copies h_pos_mass to the device,
 * builds the tree, runs otoo_gravity, copies N x float4 back into h_acc_pot, synchronises. */
otoo_status otoo_gravity_host(otoo_ctx* ctx, const float* h_pos_mass, int64_t N, int n_crit,
                              float eps, float theta, int group_size, float* h_acc_pot);
/* The same for the paper's absolute-error MAC (otoo_build_tree + otoo_gravity_delta between the two copies). */
otoo_status otoo_gravity_delta_host(otoo_ctx* ctx, const float* h_pos_mass, int64_t N, int n_crit,
                                    float eps, float delta, float m_limit, int group_size,
                                    float* h_acc_pot);

#ifdef __cplusplus
}
#endif
#endif
