// walk.cuh -- the warp-level group walk shared by the gravity and SPH kernels.
//
// One warp owns one group of G = 32*T Morton-consecutive targets (n_vec targets
// share one traversal).  The traversal is the paper's rule set (L57: not accepted -> descend,
// accepted -> interact, particle -> interact) run 32 cells at a time from a LIFO stack in shared
// memory; accepted cells and opened leaves' particles are appended to an interaction list in
// shared memory that is consumed (all targets x all entries) whenever it fills.  The list never
// touches HBM.
//
// Load balance: a few groups straddle octant boundaries, have system-sized AABBs and lists up to
// N entries.  A warp whose stack is long hands its shallowest
// stack entries (largest subtrees) to a global task pool when other warps are idle or when its
// shared stack overflows; any warp can run such a task for the same group.  Results are therefore
// accumulated with atomicAdd into zero-initialised outputs; per-group counters likewise.
#pragma once
#include "common.cuh"

__device__ __forceinline__ unsigned lanemask_lt_() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// packed fp32x2 arithmetic (sm_100: FFMA2 / FADD2 / FMUL2 -- two lanes per issue slot)
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float& a, float& b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ float rsqrt_approx(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// R8: squared distance from the group's AABB to a point, the exact fp32 expression both sides use.
__device__ __forceinline__ float aabb_d2(const float glo[3], const float ghi[3], float cx, float cy, float cz) {
  float ex = fmaxf(0.0f, fmaxf(__fsub_rn(glo[0], cx), __fsub_rn(cx, ghi[0])));
  float ey = fmaxf(0.0f, fmaxf(__fsub_rn(glo[1], cy), __fsub_rn(cy, ghi[1])));
  float ez = fmaxf(0.0f, fmaxf(__fsub_rn(glo[2], cz), __fsub_rn(cz, ghi[2])));
  return __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex)));
}

// ---- reading R25: the group's pieces between its OTOO_PIECES - 1 coarsest key boundaries, each with its tight box.
// A Morton range that crosses the boundary of a coarse cell jumps across that cell, so the box of the whole group
// can be as large as the cell (a few groups list the whole system) while the pieces are compact; the group-cell
// distance is then the minimum over the pieces' box distances (same fp32 expression as R8 per piece).
#define OTOO_PIECES 8
__device__ __forceinline__ int key_cplev(uint64_t a, uint64_t b) {   // leading octree levels two keys share, 0..21
  const uint64_t x = a ^ b;
  return x == 0 ? OTOO_MAXLEV : 20 - (63 - __clzll((long long)x)) / 3;
}
__device__ __forceinline__ unsigned f2ord_(float f) { const unsigned u = __float_as_uint(f); return (u & 0x80000000u) ? ~u : (u | 0x80000000u); }
__device__ __forceinline__ float ord2f_(unsigned u) { return __uint_as_float((u & 0x80000000u) ? (u & 0x7FFFFFFFu) : ~u); }
// mem: the group's members in shared memory (slot g0 + i at mem[i], i < gcount); pbox[2p], pbox[2p+1] = (lo, hi) of
// piece p; an unused piece gets (+inf, -inf): its distance is +inf and never the minimum.  Boundary i (between
// members i-1 and i) has the key v = (shared levels << 16) | i; the OTOO_PIECES - 1 smallest keys are the cuts
// (ties: the lowest slot), a member's piece is the number of cuts at or before it.
template <int T>
__device__ __forceinline__ void group_pieces(const uint64_t* __restrict__ keys, int64_t g0, int gcount, int lane,
                                             const float4* mem, float4* pbox) {
  uint32_t v[T];
#pragma unroll
  for (int t = 0; t < T; t++) {
    const int i = t * 32 + lane;
    v[t] = (i >= 1 && i < gcount) ? (((uint32_t)key_cplev(keys[g0 + i - 1], keys[g0 + i]) << 16) | (uint32_t)i) : 0xFFFFFFFFu;
  }
  uint32_t piece[T];
#pragma unroll
  for (int t = 0; t < T; t++) piece[t] = 0u;
#pragma unroll 1
  for (int k = 0; k < OTOO_PIECES - 1; k++) {
    uint32_t m = v[0];
#pragma unroll
    for (int t = 1; t < T; t++) m = min(m, v[t]);
    const uint32_t w = __reduce_min_sync(0xFFFFFFFFu, m);
    if (w == 0xFFFFFFFFu) break;                      // fewer boundaries than cuts
    const int ci = (int)(w & 0xFFFFu);
#pragma unroll
    for (int t = 0; t < T; t++) {
      if (v[t] == w) v[t] = 0xFFFFFFFFu;
      piece[t] += (t * 32 + lane >= ci) ? 1u : 0u;
    }
  }
#pragma unroll 1
  for (int p = 0; p < OTOO_PIECES; p++) {
    unsigned lo[3] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu}, hi[3] = {0u, 0u, 0u}, wmax = 0u;
#pragma unroll
    for (int t = 0; t < T; t++) {
      const int i = t * 32 + lane;
      if (i < gcount && piece[t] == (uint32_t)p) {
        const float4 q = mem[i];
        lo[0] = min(lo[0], f2ord_(q.x)); hi[0] = max(hi[0], f2ord_(q.x));
        lo[1] = min(lo[1], f2ord_(q.y)); hi[1] = max(hi[1], f2ord_(q.y));
        lo[2] = min(lo[2], f2ord_(q.z)); hi[2] = max(hi[2], f2ord_(q.z));
        wmax = max(wmax, f2ord_(q.w));
      }
    }
#pragma unroll
    for (int k = 0; k < 3; k++) { lo[k] = __reduce_min_sync(0xFFFFFFFFu, lo[k]); hi[k] = __reduce_max_sync(0xFFFFFFFFu, hi[k]); }
    wmax = __reduce_max_sync(0xFFFFFFFFu, wmax);
    if (lane == 0) {
      const bool any = lo[0] != 0xFFFFFFFFu || hi[0] != 0u;     // (a member at the ordered value 0xFFFFFFFF is a NaN: not a position)
      // .w of the lo corner: the largest mem[].w of the piece (SPH walks stage h there: the piece's h_max, R26)
      pbox[2 * p] = any ? make_float4(ord2f_(lo[0]), ord2f_(lo[1]), ord2f_(lo[2]), ord2f_(wmax)) : make_float4(INFINITY, INFINITY, INFINITY, 0.f);
      pbox[2 * p + 1] = any ? make_float4(ord2f_(hi[0]), ord2f_(hi[1]), ord2f_(hi[2]), 0.f) : make_float4(-INFINITY, -INFINITY, -INFINITY, 0.f);
    }
  }
  __syncwarp();
}
// R8 box distance of one piece
__device__ __forceinline__ float piece_d2(const float4 lo, const float4 hi, float cx, float cy, float cz) {
  const float ex = fmaxf(0.0f, fmaxf(__fsub_rn(lo.x, cx), __fsub_rn(cx, hi.x)));
  const float ey = fmaxf(0.0f, fmaxf(__fsub_rn(lo.y, cy), __fsub_rn(cy, hi.y)));
  const float ez = fmaxf(0.0f, fmaxf(__fsub_rn(lo.z, cz), __fsub_rn(cz, hi.z)));
  return __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex)));
}
// minimum over the pieces of the R8 box distance
__device__ __forceinline__ float pieces_d2(const float4* pbox, float cx, float cy, float cz) {
  float m = INFINITY;
#pragma unroll
  for (int p = 0; p < OTOO_PIECES; p++) {
    const float4 lo = pbox[2 * p], hi = pbox[2 * p + 1];
    const float ex = fmaxf(0.0f, fmaxf(__fsub_rn(lo.x, cx), __fsub_rn(cx, hi.x)));
    const float ey = fmaxf(0.0f, fmaxf(__fsub_rn(lo.y, cy), __fsub_rn(cy, hi.y)));
    const float ez = fmaxf(0.0f, fmaxf(__fsub_rn(lo.z, cz), __fsub_rn(cz, hi.z)));
    m = fminf(m, __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex))));
  }
  return m;
}

__device__ __forceinline__ int warp_inclusive_scan(int x, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xFFFFFFFFu, x, o); if (lane >= o) x += y; }
  return x;
}

// ---- global task pool (multi-producer multi-consumer ring of fixed-size tasks)
#define OTOO_TASK_CELLS 256
#ifndef OTOO_MULTI_DONATE
#define OTOO_MULTI_DONATE 4
#endif
#define OTOO_POOL_MARGIN 4096        // > number of resident warps: concurrent producers cannot overrun
struct TaskSlot { uint32_t group, count, pad[2]; uint32_t cells[OTOO_TASK_CELLS]; };
struct WalkShared {                   // device-global control block, reset before every launch
  uint32_t queue;  uint32_t pad0[31]; // next group of the main queue
  uint32_t head;   uint32_t pad1[31]; // consumer tickets: idle warps take one and wait on their slot
  uint32_t tail;   uint32_t pad2[31]; // producer tickets
  int outstanding; uint32_t pad3[31]; // tasks created - (groups + tasks finished): starts at 0, all done at -ngroups
};
struct WalkCommon {
  const float4* spos; const float4* cell_cm; const cellb_t* cell_b; const uint32_t* perm;
  const uint64_t* keys;                                         // sorted keys (piece boundaries of R25)
  int64_t N, ngroups;                                           // ngroups: groups of THIS launch, starting at g_begin
  uint32_t g_begin;                                             // (target sharding over devices)
  uint32_t* g_ntests; uint32_t* g_ncells; uint32_t* g_nparts;   // zeroed before the launch
  unsigned long long* sums;                                    // tests, interactions, cells, parts
  WalkShared* ws; TaskSlot* slots; uint32_t* seq;               // seq[i] initialised to i
  uint32_t* spill;                                              // OTOO_WALK_SPILL per warp
  int out_sorted;                                               // 1: results are written at the SORTED slot of a target instead of its original index
  int gs;                                                       // group size: 32 * T of the kernel, or 4 / 8 / 16 with T = 1 (the paper's n_vec, L163)
  int stack_cap;
  int spill_cap;                                                // usable entries of a warp's private spill area (<= OTOO_WALK_SPILL)
  int use_pool;                                                 // 0: never donate (test hook: private spill only)
  int walk_only;                                                // 1: lists are built and counted but not evaluated (measures the walk)
  int dist_kind;                                                // gravity: 0 one box per group (R8), 1 exact minimum over the members (R23),
                                                                // 2 minimum over the boxes of the group's pieces (R25)
  // visitors with REC (the SPH walks): the leaves a group opens, recorded by one walk and replayed by the next one with
  // the same MAC (option "sph_reuse_walk": stage 2 of an SPH step opens exactly the leaves of stage 1, R15 / R26)
  int rec_mode;                                                 // 0 off, 1 record, 2 replay (host side: picks the kernel instantiation, V::REC)
  int rec_cap;                                                  // leaf ids per group
  uint32_t* rec_cells; uint32_t* rec_count; uint32_t* rec_ntests;   // [group][rec_cap]; per group: leaves (0xFFFFFFFF: none recorded), MAC tests of its walk
};

// member idx (0 .. 32 T - 1) of the group starting at slot g0 exists
__device__ __forceinline__ bool member_ok(const WalkCommon& c, int64_t g0, int idx) { return idx < c.gs && g0 + idx < c.N; }
// row of the caller's output that belongs to sorted slot s
__device__ __forceinline__ int64_t out_row(const WalkCommon& c, int64_t s) { return c.out_sorted ? s : (int64_t)c.perm[s]; }
__device__ __forceinline__ int group_count(const WalkCommon& c, int64_t g0) { const int64_t left = c.N - g0; return (int)(left < c.gs ? left : c.gs); }

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }

// Visitor contract (all members __forceinline__):
//   static constexpr int T;            targets per lane
//   static constexpr int E;            float4 per list entry
//   static constexpr int LCAP;         float4 per list buffer
//   void load_group(int64_t g0, int lane, float4* scratch)   targets into registers, AABB, zero accumulators
//   int  classify(uint32_t cell, float4& A, cellb_t& B)   0 = drop, 1 = accept (A goes to the list), 2 = open
//   struct Entry; Entry get(uint32_t slot); void put(float4* dst, const Entry&)   one particle entry (E float4)
//   static constexpr bool CULL;  true: keep(entry) decides per particle of an opened leaf whether it enters the
//                                list at all (the counters still count the paper's list: every particle)
//   static constexpr bool SUBMIT_LAST;  true: the last list of a unit of work is submitted even if empty
//   float4* submit(float4* list, int n, bool last)   consume n entries (fused visitors: all targets x n
//                                                  entries, same buffer back; the warp-specialised walker:
//                                                  hand the buffer to its evaluator warp, next buffer back)
//   void pad(float4* dst)                          a null entry
//   void mark_self(uint32_t first, uint32_t count, int64_t g0, int lane)
//   void store(int64_t g0, int lane)               atomicAdd results to the outputs
//   static constexpr int REC;   1: the walk records the leaves each whole group opens; 2: it starts from recorded leaves; 0: neither
//                               (compile time: the bookkeeping costs the SPH kernels 5-7 % when it is only switched off at run time)
template <class V>
__device__ __forceinline__ void walk_driver(const WalkCommon& c, V& v, float4* list0, uint32_t* stk, int lane, int64_t gwarp) {
  const int G = c.gs;                                // targets per group (<= 32 * V::T; below 32: the other lanes idle)
  constexpr int CAP = (V::LCAP / V::E) & ~3;         // list entries per buffer (multiple of the padding unit)
  constexpr int PADTO = 4;
  uint32_t* gspill = c.spill + gwarp * OTOO_WALK_SPILL;
  unsigned long long tot_tests = 0, tot_inter = 0, tot_cells = 0, tot_parts = 0;
  unsigned long long tot_steps = 0, tot_tasks = 0, tot_flushes = 0, tot_eval = 0;
  uint32_t idle_polls = 0;          // 400 ns sleeps of this warp while it waited for a pool task
  bool main_done = false, have_ticket = false;
  uint32_t my_ticket = 0;
  float4* list = list0;

  for (;;) {
    // ---------------- acquire a unit of work
    uint32_t g = 0; int sp = 0;
    bool got = false, whole = false;                   // whole: the unit is a group from the main queue, not a pool task
    auto take = [&](uint32_t ticket) {   // copy task `ticket` (already published) to the shared stack
      const uint32_t slot = ticket % OTOO_POOL_SLOTS;
      __threadfence();
      const TaskSlot* ts = c.slots + slot;
      g = __ldcg(&ts->group); sp = (int)__ldcg(&ts->count);
      for (int i = lane; i < sp; i += 32) stk[i] = __ldcg(&ts->cells[i]);
      __syncwarp();
      if (lane == 0) { __threadfence(); *reinterpret_cast<volatile uint32_t*>(&c.seq[slot]) = ticket + OTOO_POOL_SLOTS; }
    };
    // (taking pending pool tasks before new groups was tried twice -- CAS claims: every warp retrying on
    // one word; unconditional claims: overshooting warps wait -- and lost 3-5 %: the pool is drained at the end)
    if (!got && !main_done) {
      if (lane == 0) g = atomicAdd(&c.ws->queue, 1u);
      g = __shfl_sync(0xFFFFFFFFu, g, 0);
      if ((int64_t)g < c.ngroups) { got = true; whole = true; g += c.g_begin; if (lane == 0) stk[0] = 0u; sp = 1; }
      else main_done = true;
    }
    if (!got) {
      // idle: take a consumer ticket once, then wait on that slot (no contended atomics while waiting)
      if (!have_ticket) {
        if (lane == 0) my_ticket = atomicAdd(&c.ws->head, 1u);
        my_ticket = __shfl_sync(0xFFFFFFFFu, my_ticket, 0);
        have_ticket = true;
      }
      int ok = 0;
      if (lane == 0) {
        if (ld_volatile(&c.seq[my_ticket % OTOO_POOL_SLOTS]) == my_ticket + 1u) ok = 1;
        else if (*reinterpret_cast<volatile int*>(&c.ws->outstanding) + (int)c.ngroups <= 0) ok = -1;
      }
      ok = __shfl_sync(0xFFFFFFFFu, ok, 0);
      if (ok < 0) break;
      if (ok == 0) { __nanosleep(400); idle_polls++; continue; }
      take(my_ticket);
      have_ticket = false;
      got = true;
    }
    __syncwarp();

    const int64_t g0 = (int64_t)g * G;
    const int gcount = (int)((c.N - g0) < G ? (c.N - g0) : G);
    v.load_group(g0, lane, list);   // the list is empty here: usable as scratch
    int gsp = 0, nlist = 0;
    uint32_t ntests = 0, ncells = 0, nparts = 0, iter = 0, nflush = 0, nkept = 0;   // nkept: list entries handed to the sums (after a cull)
    // recorded leaves (REC): a whole group records the leaves it opens unless part of its walk goes to the pool; a whole
    // group with a record starts from those leaves (through the private spill area) instead of the root: the same MAC
    // opens every one of them again, the tests of the internal cells are not repeated but counted (rec_ntests)
    bool rec_on = false, rec_bad = false, replaying = false;
    uint32_t nrec = 0, rec_extra = 0;
    if constexpr (V::REC == 1) rec_on = whole;
    if constexpr (V::REC == 2) {
      if (whole) {
        const uint32_t cnt = c.rec_count[g];
        if (cnt != 0xFFFFFFFFu && (int)cnt <= c.spill_cap) {
          const uint32_t* src = c.rec_cells + (size_t)g * c.rec_cap;
          for (uint32_t i = lane; i < cnt; i += 32) gspill[i] = src[i];
          __syncwarp();
          gsp = (int)cnt; sp = 0;
          rec_extra = c.rec_ntests[g] - cnt;
          replaying = true;
        }
      }
    }

    auto flush = [&](bool last = false) {
      nkept += (uint32_t)nlist;
      const int np = (nlist + PADTO - 1) & ~(PADTO - 1);
      if (lane < np - nlist) v.pad(list + V::E * (nlist + lane));
      __syncwarp();
      list = v.submit(list, np, last);
      __syncwarp();
      nlist = 0; nflush++;
    };
    // task pool, producer side: pool_begin reserves a slot (NULL if the pool is full), the caller writes
    // `d` cell ids into it, pool_end publishes it
    uint32_t pticket = 0;
    auto pool_begin = [&]() -> TaskSlot* {
      int ok = 0;
      if (!c.use_pool) return nullptr;
      if (lane == 0) {
        uint32_t h = ld_volatile(&c.ws->head), t = ld_volatile(&c.ws->tail);
        if ((int)(t - h) < OTOO_POOL_SLOTS - OTOO_POOL_MARGIN) {
          ok = 1;
          atomicAdd(&c.ws->outstanding, 1);
          pticket = atomicAdd(&c.ws->tail, 1u);
          while (ld_volatile(&c.seq[pticket % OTOO_POOL_SLOTS]) != pticket) __nanosleep(64);
        }
      }
      ok = __shfl_sync(0xFFFFFFFFu, ok, 0);
      if (!ok) return nullptr;
      pticket = __shfl_sync(0xFFFFFFFFu, pticket, 0);
      return c.slots + (pticket % OTOO_POOL_SLOTS);
    };
    auto pool_end = [&](TaskSlot* ts, int d) {
      if (lane == 0) { __stcg(&ts->group, g); __stcg(&ts->count, (uint32_t)d); }
      __threadfence();
      __syncwarp();
      if (lane == 0) *reinterpret_cast<volatile uint32_t*>(&c.seq[pticket % OTOO_POOL_SLOTS]) = pticket + 1u;
    };
    // hand the `d` shallowest stack entries to the pool (returns false if the pool is full)
    auto donate = [&](int d) -> bool {
      TaskSlot* ts = pool_begin();
      if (!ts) return false;
      for (int i = lane; i < d; i += 32) __stcg(&ts->cells[i], stk[i]);
      pool_end(ts, d);
      if constexpr (V::REC == 1) rec_bad = true;     // part of this group's walk is someone else's now
      return true;
    };
    // drop the d bottom entries of the shared stack (after they were donated or spilled)
    auto shift_down = [&](int d) {
      for (int k = 0; k < sp - d; k += 32) {
        uint32_t x = (k + lane < sp - d) ? stk[d + k + lane] : 0u;
        __syncwarp();
        if (k + lane < sp - d) stk[k + lane] = x;
        __syncwarp();
      }
      sp -= d;
    };

    while (sp > 0 || gsp > 0) {
      if (sp == 0) {  // refill from the private spill
        const int k = gsp < OTOO_TASK_CELLS ? gsp : OTOO_TASK_CELLS;
        for (int i = lane; i < k; i += 32) stk[i] = gspill[gsp - k + i];
        __syncwarp();
        gsp -= k; sp = k;
      }
      const int k = sp < 32 ? sp : 32;
      const bool have = lane < k;
      uint32_t cell = 0;
      if (have) cell = stk[sp - k + lane];
      // waiting consumers = head - tail (when positive); loads issued early, used below
      const int idle_now = sp >= 16 ? (int)(ld_volatile(&c.ws->head) - ld_volatile(&c.ws->tail)) : 0;
      iter++;
      __syncwarp();
      sp -= k;
      float4 A = make_float4(0.f, 0.f, 0.f, 0.f);
      cellb_t B = make_uint4(0u, 0u, 0u, 0u);
      int cls = 0;
      if constexpr (V::REC == 2) {
        // a recorded leaf passed this very test in the recording walk (same group geometry, same radii): it is opened
        // without its centre of mass, its radii and the nine box tests; the test is counted all the same
        if (replaying) { if (have) { B = __ldg(c.cell_b + cell); cls = 2; } }
        else if (have) cls = v.classify(cell, A, B);
      } else {
        if (have) cls = v.classify(cell, A, B);
      }
      ntests += (uint32_t)k;
      const bool leaf = (B.w & 1u) != 0u;
      const bool accept = cls == 1, open_leaf = cls == 2 && leaf, open_int = cls == 2 && !leaf;

      // accepted cells -> list (the cell is a virtual particle at its centre of mass, L43)
      const unsigned am = __ballot_sync(0xFFFFFFFFu, accept);
      const int na = __popc(am);
      if (na) {
        if (nlist + na > CAP) flush();
        if (accept) list[V::E * (nlist + __popc(am & lanemask_lt_()))] = A;
        nlist += na; ncells += (uint32_t)na;
      }
      // opened internal cells -> push children (L57 rule 1: follow `more`)
      {
        const int nch = open_int ? (int)B.z : 0;
        const int inc = warp_inclusive_scan(nch, lane);
        const int total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        if (total) {
          bool pushed = false;
          if (sp + total > c.stack_cap) {
            // overflow (a group with a system-sized box): the new children become a pool task of their own
            // -- deep cells, small subtrees: the task is finished by whoever takes it and nothing circulates;
            // this warp keeps generating such tasks from its shallow backlog.  Pool full: spill privately.
            TaskSlot* ts = pool_begin();
            if (ts) {
              const int o = inc - nch;
              for (int i = 0; i < nch; i++) __stcg(&ts->cells[o + i], B.y + (uint32_t)i);
              pool_end(ts, total);
              pushed = true;
              if constexpr (V::REC == 1) rec_bad = true;
            } else {
              const int d = OTOO_TASK_CELLS;      // stack_cap >= 512, total <= 256
              if (gsp + d <= c.spill_cap) {
                for (int i = lane; i < d; i += 32) gspill[gsp + i] = stk[i];
                gsp += d;
              } else if (lane == 0) {
                // the private area is full too (cannot happen with the level-sorted stack bound of common.cuh;
                // reachable only through the test hooks): the cells are dropped and the launch is flagged --
                // otoo_last_stats / otoo_export_group_stats then return OTOO_ERR_CAPACITY
                atomicExch(c.sums + 7, 1ull);
              }
              __syncwarp();
              shift_down(d);
            }
          }
          if (!pushed) {
          const int o = sp + inc - nch;
          for (int i = 0; i < nch; i++) stk[o + i] = B.y + (uint32_t)i;
          __syncwarp();
          sp += total;
          }
        }
      }
      // load balance: feed idle warps with the shallowest entries
      if (sp >= 16 && idle_now > 0) {
        // several idle warps and a long stack: several smaller tasks at once (the shallowest entries first)
        int nt = idle_now < OTOO_MULTI_DONATE ? idle_now : OTOO_MULTI_DONATE;
        if (nt > (sp >> 4)) nt = sp >> 4;
        int d = (sp >> 1) / nt; if (d > OTOO_TASK_CELLS) d = OTOO_TASK_CELLS;
        for (int k = 0; k < nt; k++) {
          if (!donate(d)) break;
          shift_down(d);
        }
      }
      // opened leaves -> their particles (L57 rule 3)
      const unsigned lm = __ballot_sync(0xFFFFFFFFu, open_leaf);
      if constexpr (V::REC == 1) {
        if (rec_on && lm) {
          const uint32_t nl = (uint32_t)__popc(lm);
          if (nrec + nl <= (uint32_t)c.rec_cap) { if (open_leaf) c.rec_cells[(size_t)g * c.rec_cap + nrec + (uint32_t)__popc(lm & lanemask_lt_())] = cell; }
          else rec_bad = true;
          nrec += nl;
        }
      }
      if (lm) {
        const int cnt = open_leaf ? (int)B.z : 0;
        const int inc = warp_inclusive_scan(cnt, lane);
        const int total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        // only the few leaves that overlap the group's own slots can hold a target (one ballot instead of a
        // shuffle round per opened leaf: ~450 leaves are opened per group, ~10 of them overlap it)
        unsigned m = __ballot_sync(0xFFFFFFFFu, open_leaf && (int64_t)B.y < g0 + G && (int64_t)B.y + (int64_t)B.z > g0);
        while (m) {  // which targets sit in an opened leaf: their self term is in the list
          const int src = __ffs(m) - 1; m &= m - 1;
          v.mark_self(__shfl_sync(0xFFFFFFFFu, B.y, src), __shfl_sync(0xFFFFFFFFu, B.z, src), g0, lane);
        }
        // cooperative expansion: output position j -> (leaf, offset) by a shuffle binary search over the
        // inclusive counts; every lane loads one particle per chunk, loads of two chunks are in flight.
        const int startv = inc - cnt;
        auto locate = [&](int j) -> uint32_t {
          int L = 0;
#pragma unroll
          for (int st = 16; st; st >>= 1) { const int x = __shfl_sync(0xFFFFFFFFu, inc, L + st - 1); if (x <= j) L += st; }
          const uint32_t f = __shfl_sync(0xFFFFFFFFu, B.y, L);
          const int s0 = __shfl_sync(0xFFFFFFFFu, startv, L);
          return f + (uint32_t)(j - s0);
        };
        for (int j0 = 0; j0 < total;) {
          if (nlist + 32 > CAP) flush();
          const int room = (CAP - nlist) >> 5, need = (total - j0 + 31) >> 5;
          int nb = room < need ? room : need;
          for (; nb >= 2; nb -= 2, j0 += 64) {
            const int ja = j0 + lane, jb = j0 + 32 + lane;
            const uint32_t sa = locate(ja < total ? ja : total - 1), sb = locate(jb < total ? jb : total - 1);
            typename V::Entry ea = v.get(sa), eb = v.get(sb);
            if (V::CULL) {   // entries that cannot interact with any member of the group stay out of the list
              const bool ka = ja < total && v.keep(ea), kb = jb < total && v.keep(eb);
              const unsigned ma = __ballot_sync(0xFFFFFFFFu, ka), mb = __ballot_sync(0xFFFFFFFFu, kb);
              const int na = __popc(ma);
              if (ka) v.put(list + V::E * (nlist + __popc(ma & lanemask_lt_())), ea);
              if (kb) v.put(list + V::E * (nlist + na + __popc(mb & lanemask_lt_())), eb);
              nlist += na + __popc(mb);
            } else {
              if (ja < total) v.put(list + V::E * (nlist + lane), ea);
              if (jb < total) v.put(list + V::E * (nlist + 32 + lane), eb);
              nlist += (total - j0) < 64 ? (total - j0) : 64;
            }
          }
          if (nb == 1) {
            const int ja = j0 + lane;
            const uint32_t sa = locate(ja < total ? ja : total - 1);
            typename V::Entry ea = v.get(sa);
            if (V::CULL) {
              const bool ka = ja < total && v.keep(ea);
              const unsigned ma = __ballot_sync(0xFFFFFFFFu, ka);
              if (ka) v.put(list + V::E * (nlist + __popc(ma & lanemask_lt_())), ea);
              nlist += __popc(ma);
            } else {
              if (ja < total) v.put(list + V::E * (nlist + lane), ea);
              nlist += (total - j0) < 32 ? (total - j0) : 32;
            }
            j0 += 32;
          }
        }
        nparts += (uint32_t)total;
        __syncwarp();
      }
    }
    if (nlist || V::SUBMIT_LAST) flush(true);
    v.store(g0, lane);
    if constexpr (V::REC == 2) ntests += rec_extra;
    if constexpr (V::REC == 1) {
      if (rec_on && lane == 0) { c.rec_count[g] = rec_bad ? 0xFFFFFFFFu : nrec; c.rec_ntests[g] = ntests; }
    }
    if (lane == 0) {
      atomicAdd(c.g_ntests + g, ntests); atomicAdd(c.g_ncells + g, ncells); atomicAdd(c.g_nparts + g, nparts);
      __threadfence();
      atomicSub(&c.ws->outstanding, 1);
    }
    tot_tests += ntests; tot_cells += ncells; tot_parts += nparts;
    tot_steps += iter; tot_tasks += 1; tot_flushes += nflush;
    tot_inter += (unsigned long long)gcount * (ncells + nparts);
    tot_eval += (unsigned long long)gcount * nkept;
  }
  if (lane == 0 && tot_tests) {
    atomicAdd(c.sums + 0, tot_tests); atomicAdd(c.sums + 1, tot_inter);
    atomicAdd(c.sums + 2, tot_cells);
    atomicAdd(c.sums + 3, tot_parts);
    atomicAdd(c.sums + 4, tot_steps); atomicAdd(c.sums + 5, tot_tasks);
    atomicAdd(c.sums + 6, tot_flushes);
    atomicAdd(c.sums + 15, tot_eval);
  }
  if (lane == 0 && idle_polls) atomicAdd(c.sums + 14, (unsigned long long)idle_polls);
}

// host side (gravity.cu)
otoo_status otoo_walk_prepare(otoo_ctx* ctx, int G, WalkCommon* c, int* grid, size_t* smem, cudaStream_t st, bool reset = true);
