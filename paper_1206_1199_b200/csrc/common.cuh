// common.cuh -- context layout and helpers shared by the kernels of libotoo.so (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include "../../include/otoo.h"

#define OTOO_MAXLEV 21
#define OTOO_NLEV 22                 // levels 0..21
#define OTOO_REC_CAP 1024             // recorded leaf ids per group (option sph_reuse_walk); a group that opens more walks again
#define OTOO_REC_MAX_BYTES ((size_t)8 << 30)   // no records beyond this size (4 KB per group): the walks then run in full
#define OTOO_POOL_SLOTS 16384         // task slots of the walk's pool (walk.cuh)
#define OTOO_WALK_STACK_MAX 512      // smem walk-stack entries per warp
#define OTOO_WALK_SPILL 8192         // global spill entries per warp (bound 8*32*21 = 5376)
#define OTOO_LIST_CAP 256            // smem interaction-list float4 per warp (small: leaves the SM's L1 for the tree)
#define OTOO_LIST_STRIDE (OTOO_LIST_CAP + 4)  // per-warp list buffer (+4: consecutive warps start on different banks)
#ifndef OTOO_SORT_TILE
#define OTOO_SORT_TILE 4096            // pairs per CTA of a radix pass (256 threads x 16; 1024 and 2048 measured slower)
#endif
// u32 words of sort scratch for n pairs: digit histograms + tickets (4096) + one u64 status word per tile and digit
#define OTOO_SORT_SCRATCH(n) ((size_t)(((n) + OTOO_SORT_TILE - 1) / OTOO_SORT_TILE) * 512 + 4096)
#define OTOO_WALK_WARPS 4            // warps per CTA of the walk kernels
#define OTOO_NSUMS 16
#define OTOO_BUILD_PHASES 6          // root cube, keys, sort, gather, cells (topology), moments

// Per-cell walk record, 16 B: the paper's 7-word node (L161) minus the 4 words of (cm, m).
//   x = rb^2 bits (gravity MAC, R7), y = first child id (internal) or first sorted slot (leaf),
//   z = child count (internal) or particle count (leaf), w = bit0 leaf flag | level << 8.
typedef uint4 cellb_t;

struct otoo_ctx {
  int device;
  int sm_count;
  int64_t maxN;
  char err[256];
  cudaStream_t last_stream;

  // ---- per-particle arrays, capacity maxN
  uint64_t* key[2];      // key double buffer for the LSD sort; key[0] holds the sorted keys after build
  uint32_t* val[2];      // id double buffer; val[0] = perm after build
  float4* spos;          // positions+mass in sorted order
  uint32_t* slot_nc;     // cells per level starting in each block of 256 slots (level-major), then its exclusive scan
  uint32_t* scan_tmp;    // scan scratch: tile ticket, then one 64-bit look-back status word per tile of 4096 elements
  size_t scan_cap;       // its size in words
  uint32_t scan_epoch;   // one epoch per scan tags the status words: stale ones never match
  uint32_t* hist;        // sort scratch: digit histograms, tile tickets, look-back status words
  uint32_t sort_epoch;   // one epoch per radix pass: stale status words never match
  bool sort_attr_set;
  size_t hist_cap;
  float* sorted_h;       // SPH: h in sorted order
  float4* sorted_aux;    // SPH force: (rho-independent) per-particle packed inputs in sorted order
  float4* sorted_vel;
  float4* sorted_vis;    // SPH viscosity: (alpha, Balsara f, -, -) in sorted order

  // ---- per-cell arrays, capacity cellCap (grow-only)
  int64_t cellCap;
  float4* cell_cm;       // (cm.xyz, m) fp32 -- what the walk reads
  cellb_t* cell_b;
  uint32_t* c_first;
  uint32_t* c_count;
  uint32_t* c_child_first;
  uint8_t* c_level;      // level in bits 0..4; bit 7: the cell is the first child of its parent (build.cu, H5c)
  uint8_t* c_child_count;
  double* c_MP;          // 4 per cell: M, Px, Py, Pz (R6)
  double* c_cm64;        // 3 per cell: fp64 centre of mass (needed for Eq. 5)
  double* c_s;           // |CM - geometric centre| (R7)
  double* c_B2;          // trace of the quadrupole tensor about the CM (PAPER Eq. 2; R19)
  float2* c_sph;         // (b_max, r_SPH) (R14)
  unsigned long long* sph_acc;  // 2 per cell: fp64 maxima as ordered bits
  uint64_t* tmp_key[2];  // (unused since the cells are placed at their canonical index directly)
  uint32_t* tmp_val[2];  // (unused since place_cells_kernel writes c_first directly)

  // ---- small device scalars
  float* d_bbox;         // 6 floats lo/hi as ordered ints, then lo[3], S, scale
  uint32_t* d_counters;  // [0..21] cells per level, [32] n_leaf, [33] work-queue counter, [34] error flag
  // pinned host mirror
  uint32_t* h_counters;
  float* h_root;         // lo[3], S

  // ---- walk outputs
  int64_t groupCap;
  uint32_t* g_ntests;
  uint32_t* g_ncells;
  uint32_t* g_nparts;
  uint32_t* walk_spill;  // OTOO_WALK_SPILL entries per resident warp
  int64_t spill_warps;
  unsigned long long* d_sums; // OTOO_NSUMS words: [0] tests [1] interactions [2] cells [3] parts [4] steps [5] tasks [6] flushes
                              // [7] error flag [8] SM clock ticks and [9] ns spent by the CTAs of the walk kernel [10..14] waiting
                              // times of the profiled kernel [15] (target, entry) pairs handed to the sums
  void* pool_slots;      // task pool (walk.cuh): TaskSlot[OTOO_POOL_SLOTS]
  void* pool_seq;        // uint32 sequence numbers
  void* walk_shared;     // WalkShared control block

  // ---- otoo_gravity_host staging (grow-only)
  float4* stage_in; float4* stage_out; int64_t stage_cap;

  // ---- state
  bool built;
  bool walked;
  bool sph_radii_valid;
  bool b2_valid;         // c_B2 computed for the current tree (on demand, by otoo_gravity_delta)
  // theta of the last otoo_gravity call: the next build leaves rb^2 (R7) of it in cell_b.x from inside its bottom-up
  // pass (l, s are in registers there), and resets the walk's control block and pool; a gravity call with the same
  // theta then launches the walk kernel alone.  Another theta, the Delta-MAC or a second walk on the same tree run the
  // r_b / reset kernels as before.
  bool spec_theta_set, rb2_valid, walk_reset_valid;
  float spec_theta, rb2_theta;
  int key_order_built;   // key order of the current tree
  int64_t N, N_cell, N_leaf;
  int n_crit, depth;
  float lo[3], S;
  uint32_t level_off[OTOO_NLEV + 1];
  int walk_stack;        // option "walk_stack"
  int walk_spill_cap;    // option "walk_spill" (test hook): usable private spill entries per warp
  int use_pool;          // option "task_pool"
  int64_t group_begin, group_count;   // options: the walks cover groups [begin, begin + count) only (count < 0: to the end)
  int key_order;         // option "key_order": 0 Morton (R3), 1 Hilbert (R20); read by the next build
  int out_sorted;        // option "output_sorted": otoo_gravity / otoo_gravity_delta write row s of the output for sorted slot s
  int sph_reuse;         // option "sph_reuse_radii": SPH calls keep sorted h and the Eq. 5 radii of the previous SPH call on this tree
  int sph_reuse_walk;    // option "sph_reuse_walk": the density / stage-1 walk records the leaves every group opens, and a force
                         // walk that keeps the radii (sph_reuse_radii) starts from them instead of the root (walk.cuh, REC)
  uint32_t* rec_cells; uint32_t* rec_count; uint32_t* rec_ntests;   // OTOO_REC_CAP leaf ids per group; leaves and MAC tests per group
  int64_t rec_groups_cap;
  bool rec_valid; int rec_G, rec_pieces; int64_t rec_gb, rec_gc;     // what the record was taken with
  int walk_only;         // option "walk_only" (diagnostic)
  int walk_profile;      // option "walk_profile": the gravity walk kernel counts its warps' waiting time (slower)
  int dist_kind;         // option "group_distance": 0 AABB (R8), 1 exact minimum over the group's members (R23)
  int use_ws;            // option "warp_specialized": gravity walk with walker/evaluator warp pairs
  int use_ws_sph;        // option "warp_specialized_sph": the same split for the SPH kernels (default off)
  int last_group_size;
  int64_t last_ngroups;
  int launches;          // kernels launched by the current/last API call
  int last_walk_only;    // the last walk ran with option "walk_only" (its outputs are meaningless)

  // ---- per-phase device times (the paper's TREE / KERNEL split): CUDA events
  // recorded on the call's stream, read by otoo_last_stats (which synchronises)
  cudaEvent_t ev_build[OTOO_BUILD_PHASES + 1];   // phase p = ev_build[p] .. ev_build[p + 1]
  cudaEvent_t ev_walk[3];                        // call start, walk kernel start, walk kernel end
  bool ev_build_valid, ev_walk_valid;
};
#define OTOO_EV(ctx, ev, st) OTOO_CUDA(ctx, cudaEventRecord((ev), (st)))

#define OTOO_CUDA(ctx, call)                                                                   \
  do {                                                                                         \
    cudaError_t e_ = (call);                                                                   \
    if (e_ != cudaSuccess) {                                                                   \
      snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call,     \
               cudaGetErrorString(e_));                                                        \
      return (e_ == cudaErrorMemoryAllocation) ? OTOO_ERR_OOM : OTOO_ERR_CUDA;                 \
    }                                                                                          \
  } while (0)

#define OTOO_TRY(call)                    \
  do {                                    \
    otoo_status s_ = (call);              \
    if (s_ != OTOO_OK) return s_;         \
  } while (0)

static inline otoo_status otoo_fail(otoo_ctx* ctx, otoo_status s, const char* msg) {
  if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s", msg);
  return s;
}
static inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ---- internal entry points (one per .cu file)
otoo_status otoo_sort_pairs(otoo_ctx* ctx, uint64_t* key[2], uint32_t* val[2], int64_t n,
                            int first_bit, int end_bit, cudaStream_t st, int* result_buf, bool hist_done = false);
otoo_status otoo_keys_and_hist(otoo_ctx* ctx, const float* d_pos_mass, int64_t n, cudaStream_t st);
otoo_status otoo_exclusive_scan_u32(otoo_ctx* ctx, uint32_t* data, int64_t n, uint32_t* total_out_dev,
                                    cudaStream_t st);
otoo_status otoo_build_impl(otoo_ctx* ctx, const float* d_pos_mass, int64_t N, int n_crit, cudaStream_t st);
// mac 0: theta criterion (p0 = theta); mac 1: the paper's absolute-error criterion (p0 = Delta, p1 = m_limit)
otoo_status otoo_gravity_impl(otoo_ctx* ctx, float eps, int mac, float p0, float p1, int G, float* d_acc_pot, cudaStream_t st);
otoo_status otoo_b2_impl(otoo_ctx* ctx, cudaStream_t st);     // B2 of every cell into c_B2 (build.cu), once per build
otoo_status otoo_bmax_impl(otoo_ctx* ctx, cudaStream_t st);   // fp64 b_max of every cell into sph_acc[2c] (sph.cu)
otoo_status otoo_sph_density_impl(otoo_ctx* ctx, const float* d_h, int G, float* d_rho, uint32_t* d_nngb,
                                  cudaStream_t st);
otoo_status otoo_sph_force_impl(otoo_ctx* ctx, const float* d_h, const float* d_rho, const float* d_P,
                                const float* d_vel, const float* d_visc, int G, float* d_acc, cudaStream_t st);
otoo_status otoo_sph_stage1_impl(otoo_ctx* ctx, const float* d_h, const float* d_vel, int G, float* d_rho, uint32_t* d_nngb,
                                 float* d_divrot, cudaStream_t st);
otoo_status otoo_sph_adapt_h_impl(otoo_ctx* ctx, float* d_h, float n_target, float tol, int max_iter, int G, uint32_t* d_nngb,
                                  int* host_iters, cudaStream_t st);
otoo_status otoo_ensure_groups(otoo_ctx* ctx, int64_t ngroups);
otoo_status otoo_ensure_spill(otoo_ctx* ctx, int64_t warps);
size_t otoo_walk_smem_bytes();
__host__ __device__ constexpr size_t otoo_walk_smem_bytes_dev() {   // lists + stacks of the one-warp-does-both walk kernels
  return (size_t)OTOO_WALK_WARPS * (OTOO_LIST_STRIDE * 16 + OTOO_WALK_STACK_MAX * 4);
}
otoo_status otoo_measure_fp32_peak_impl(otoo_ctx* ctx, double* tflops, cudaStream_t st);
