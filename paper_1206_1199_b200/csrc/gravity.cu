// gravity.cu -- theta-MAC radii (R7) and the fused group walk + softened Plummer sums
// (PAPER.md III-D L159-L167, L43, L57; readings R7-R11).
#include "grav_eval.cuh"

#ifndef OTOO_WALKER_BACKOFF
#define OTOO_WALKER_BACKOFF 500     // ns of __nanosleep between two polls of a walker waiting for a free list buffer
#endif
#ifndef OTOO_WS_MINB
#define OTOO_WS_MINB 3
#define OTOO_WS_EVAL_REGS 112
#define OTOO_WS_WALK_REGS 48
#endif

namespace {

// R7: r_b = l/theta + s in fp64, rb^2 rounded once to fp32.  theta = 0 -> +inf (open everything).
// the first OTOO_POOL_SLOTS threads of the r_b kernels also reset the walk's control block and the pool's sequence
// numbers (tickets restart from 0 every launch): was a kernel of its own
struct WalkReset { WalkShared* ws; uint32_t* seq; };
__device__ __forceinline__ void walk_reset(const WalkReset& r, int64_t i) {
  if (i < OTOO_POOL_SLOTS) r.seq[i] = (uint32_t)i;
  if (i == 0) { r.ws->queue = 0; r.ws->head = 0; r.ws->tail = 0; r.ws->outstanding = 0; }
}
__global__ void __launch_bounds__(256) rb2_kernel(const uint8_t* __restrict__ c_level, const double* __restrict__ c_s,
                                                  int64_t ncell, float S, float theta, cellb_t* __restrict__ cell_b, const WalkReset wr) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  walk_reset(wr, c);
  if (c >= ncell) return;
  float rb2;
  if (!(theta > 0.0f)) rb2 = INFINITY;
  else {
    double l = ldexp((double)S, -(int)(c_level[c] & 0x1F));   // (bit 7 of c_level: first-sibling flag of the build)
    double rb = __dadd_rn(__ddiv_rn(l, (double)theta), c_s[c]);
    rb2 = __double2float_rn(__dmul_rn(rb, rb));
  }
  reinterpret_cast<uint32_t*>(cell_b + c)[0] = __float_as_uint(rb2);
}

// PAPER Eq. 1: r_b = b/2 + sqrt(b^2/4 + sqrt(3 B2 / Delta)), b = b_max (fp64, from the radii pass); cells heavier
// than m_limit: r_b = 2 S_root (L157); Delta = 0: open everything.  Same fp64 operation order as the oracle.
__global__ void __launch_bounds__(256) rb2_delta_kernel(const double* __restrict__ c_B2, const double* __restrict__ c_MP,
                                                        const unsigned long long* __restrict__ bmax_bits, int64_t ncell,
                                                        float S, float delta, float m_limit, cellb_t* __restrict__ cell_b, const WalkReset wr) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  walk_reset(wr, c);
  if (c >= ncell) return;
  float rb2;
  if (!(delta > 0.0f)) rb2 = INFINITY;
  else {
    double rb;
    if (c_MP[4 * c] > (double)m_limit) rb = __dmul_rn(2.0, (double)S);
    else {
      const double h = __dmul_rn(0.5, __dsqrt_rn(__longlong_as_double((long long)bmax_bits[2 * c])));   // bmax_bits: max |x - CM|^2
      const double q = __dsqrt_rn(__ddiv_rn(__dmul_rn(3.0, c_B2[c]), (double)delta));
      rb = __dadd_rn(h, __dsqrt_rn(__dadd_rn(__dmul_rn(h, h), q)));
    }
    rb2 = __double2float_rn(__dmul_rn(rb, rb));
  }
  reinterpret_cast<uint32_t*>(cell_b + c)[0] = __float_as_uint(rb2);
}

template <int T, bool EPS0>
__global__ void __launch_bounds__(OTOO_WALK_WARPS * 32) walk_gravity_kernel(const GravParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float4* list = reinterpret_cast<float4*>(smem_raw) + warp * OTOO_LIST_STRIDE;
  uint32_t* stk = reinterpret_cast<uint32_t*>(smem_raw + OTOO_WALK_WARPS * OTOO_LIST_STRIDE * sizeof(float4)) +
                  warp * OTOO_WALK_STACK_MAX;
  GravVisitor<T, EPS0> v(p);
  v.pbox = reinterpret_cast<float4*>(smem_raw + otoo_walk_smem_bytes_dev()) + warp * (2 * OTOO_PIECES);
  walk_driver(p.c, v, list, stk, lane, (int64_t)blockIdx.x * OTOO_WALK_WARPS + warp);
}


// ---------------------------------------------------------------- warp-specialised form (walk_ws.cuh)
// Walker-side visitor: the MAC, the list entries and the self marks of GravVisitor without targets or
// sums; submit() publishes the filled buffer to the pair's evaluator warp and returns the next one.
// PROF: count the SM clock ticks spent waiting (option "walk_profile"; costs 3-4 % of the kernel, so it is a
// separate instantiation and never the timed one)
template <int T_, bool PROF = false>
struct GravWalker {
  static constexpr int T = T_, E = 1, LCAP = OTOO_WS_LCAP, NP = (T_ + 1) / 2;
  static constexpr bool SUBMIT_LAST = true;     // the evaluator needs the end-of-unit mark to store
  static constexpr bool CULL = false;
  static constexpr int REC = 0;
  template <class En> __device__ __forceinline__ bool keep(const En&) const { return true; }
  typedef WsPair<32 * NP * 3, 32 * T_> Pair;
  const GravParams& p;
  Pair& sm;
  float glo[3], ghi[3];
  unsigned selfmask;
  uint32_t group, buf, eparity, first;
  int lane_, nmem;
  __device__ __forceinline__ GravWalker(const GravParams& p_, Pair& sm_, int lane) : p(p_), sm(sm_), buf(0), eparity(~0u), first(0), lane_(lane) {}

  long long wait_ticks = 0;                          // SM clock ticks spent waiting for a free buffer (otoo_stats_t.walker_wait_frac)
  __device__ __forceinline__ float4* acquire() {     // wait until the evaluator has released buffer `buf`
    long long w0 = 0;
    if (PROF) w0 = clock64();
    mbar_wait<OTOO_WALKER_BACKOFF>(&sm.empty[buf], (eparity >> buf) & 1u);   // walkers run ahead: wait without stealing issue slots
    if (PROF) wait_ticks += clock64() - w0;
    eparity ^= 1u << buf;
    return sm.list[buf];
  }
  __device__ __forceinline__ void load_group(int64_t g0, int lane, float4*) {
#pragma unroll
    for (int t = 0; t < T; t++) {   // H7: the group's tight AABB
      int64_t s = g0 + t * 32 + lane;
      float4 v = p.c.spos[member_ok(p.c, g0, t * 32 + lane) ? s : g0];
      if (p.c.dist_kind) sm.mem[t * 32 + lane] = v;      // out-of-range slots mirror slot g0: harmless duplicates
      if (t == 0) { glo[0] = ghi[0] = v.x; glo[1] = ghi[1] = v.y; glo[2] = ghi[2] = v.z; }
      else {
        glo[0] = fminf(glo[0], v.x); ghi[0] = fmaxf(ghi[0], v.x);
        glo[1] = fminf(glo[1], v.y); ghi[1] = fmaxf(ghi[1], v.y);
        glo[2] = fminf(glo[2], v.z); ghi[2] = fmaxf(ghi[2], v.z);
      }
    }
#pragma unroll
    for (int k = 0; k < 3; k++)
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        glo[k] = fminf(glo[k], __shfl_xor_sync(0xFFFFFFFFu, glo[k], o));
        ghi[k] = fmaxf(ghi[k], __shfl_xor_sync(0xFFFFFFFFu, ghi[k], o));
      }
    selfmask = 0; first = WS_FIRST; group = (uint32_t)(g0 / p.c.gs);
    nmem = 32 * T;
    __syncwarp();
    if (p.c.dist_kind == 2) {
      group_pieces<T>(p.c.keys, g0, group_count(p.c, g0), lane, sm.mem, sm.pbox);
    }
    if (p.c.dist_kind == 1) {
      // tight boxes of 8 consecutive members (neighbours on the key curve): a box farther than r_b settles its
      // 8 members at once -- in fp32 too: rounding is monotone, so the box distance never exceeds a member's
      for (int b = lane; b < 4 * T; b += 32) {
        float4 lo = sm.mem[8 * b], hi = lo;
#pragma unroll
        for (int i = 1; i < 8; i++) {
          const float4 m = sm.mem[8 * b + i];
          lo.x = fminf(lo.x, m.x); lo.y = fminf(lo.y, m.y); lo.z = fminf(lo.z, m.z);
          hi.x = fmaxf(hi.x, m.x); hi.y = fmaxf(hi.y, m.y); hi.z = fmaxf(hi.z, m.z);
        }
        sm.sub[2 * b] = lo; sm.sub[2 * b + 1] = hi;
      }
      __syncwarp();
    }
  }
  __device__ __forceinline__ int classify(uint32_t cell, float4& A, cellb_t& B) {
    A = __ldg(p.c.cell_cm + cell);
    B = __ldg(p.c.cell_b + cell);
    const float rb2 = __uint_as_float(B.x);
    float d2 = aabb_d2(glo, ghi, A.x, A.y, A.z);
    if (d2 > rb2) return 1;                      // strict: equality opens (R8); the box distance bounds every member's from below
    if (!p.c.dist_kind) return 2;
    if (p.c.dist_kind == 2) return pieces_d2(sm.pbox, A.x, A.y, A.z) > rb2 ? 1 : 2;   // R25 (>= the whole box's distance, in fp32 too)
    // PAPER L163 (R23): the actual minimum of the members' distances decides: accept iff every member is
    // farther than r_b.  d_i^2 = fma(dz,dz, fma(dy,dy, dx*dx)), d = fl32(x_i - cm), as the oracle computes it.
    for (int b = 0; b < 4 * T; b++) {
      const float4 lo = sm.sub[2 * b], hi = sm.sub[2 * b + 1];
      const float blo[3] = {lo.x, lo.y, lo.z}, bhi[3] = {hi.x, hi.y, hi.z};
      if (aabb_d2(blo, bhi, A.x, A.y, A.z) > rb2) continue;
#pragma unroll
      for (int i = 0; i < 8; i++) {
        const float4 m = sm.mem[8 * b + i];
        const float dx = __fsub_rn(m.x, A.x), dy = __fsub_rn(m.y, A.y), dz = __fsub_rn(m.z, A.z);
        if (!(__fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx))) > rb2)) return 2;
      }
    }
    return 1;
  }
  struct Entry { float4 a; };
  __device__ __forceinline__ Entry get(uint32_t slot) const { Entry e; e.a = p.c.spos[slot]; return e; }
  __device__ __forceinline__ void put(float4* dst, const Entry& e) const { *dst = e.a; }
  __device__ __forceinline__ void pad(float4* dst) { *dst = make_float4(PAD_POS, PAD_POS, PAD_POS, 0.0f); }
  __device__ __forceinline__ void mark_self(uint32_t f, uint32_t n, int64_t g0, int lane) {
#pragma unroll
    for (int t = 0; t < T; t++) if (member_ok(p.c, g0, t * 32 + lane) && (uint32_t)(g0 + t * 32 + lane) - f < n) selfmask |= 1u << t;
  }
  __device__ __forceinline__ float4* submit(float4*, int n, bool last) {
    if (lane_ == 0) sm.meta[buf] = WsMeta{(uint32_t)n, first | (last ? WS_LAST : 0u), group, 0u};
    if (last) sm.self[buf][lane_] = selfmask;
    first = 0;
    mbar_arrive(&sm.full[buf]);
    buf = (buf + 1) % OTOO_WS_NBUF;
    return acquire();
  }
  __device__ __forceinline__ void store(int64_t, int) {}
  __device__ __forceinline__ void finish() {          // tell the evaluator to exit
    if (lane_ == 0) sm.meta[buf] = WsMeta{0u, WS_EXIT, 0u, 0u};
    mbar_arrive(&sm.full[buf]);
  }
};

#ifndef OTOO_EVAL_PB_T8
#define OTOO_EVAL_PB_T8 0      // target pairs per pass over a list buffer for G = 256 (0: 2)
#define OTOO_EVAL_UNR_T8 OTOO_EVAL_UNR
#endif
#ifndef OTOO_EVAL_UNR_T4
#define OTOO_EVAL_UNR_T4 OTOO_EVAL_UNR
#endif
template <int T> struct WsRegs { static constexpr int MINB = OTOO_WS_MINB, EVAL = OTOO_WS_EVAL_REGS, WALK = OTOO_WS_WALK_REGS, PB = 0, UNR = T == 4 ? OTOO_EVAL_UNR_T4 : OTOO_EVAL_UNR; };
template <> struct WsRegs<8> { static constexpr int MINB = 2, EVAL = 176, WALK = 80, PB = OTOO_EVAL_PB_T8, UNR = OTOO_EVAL_UNR_T8; };

template <int T, bool EPS0, bool PROF>
__global__ void __launch_bounds__(OTOO_WS_PAIRS * 64, WsRegs<T>::MINB) walk_gravity_ws_kernel(const GravParams p) {
  typedef typename GravWalker<T>::Pair Pair;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  Pair* pairs = reinterpret_cast<Pair*>(smem_raw);
  if (threadIdx.x < OTOO_WS_PAIRS) {
    Pair& s = pairs[threadIdx.x];
#pragma unroll
    for (int b = 0; b < OTOO_WS_NBUF; b++) { mbar_init(&s.full[b], 32); mbar_init(&s.empty[b], 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // SM clock held by this CTA (otoo_stats_t.walk_sm_mhz): clock64 ticks per globaltimer ns, evaluator warp 0
  long long ck0 = 0; unsigned long long ns0 = 0;
  if (threadIdx.x == 0) { ck0 = clock64(); asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns0)); }
  __syncthreads();
  if (warp >= OTOO_WS_PAIRS) {
    // ---- walker: L57 rules through walk_driver, lists into the pair's buffers
    if (WsRegs<T>::WALK) setmaxnreg_dec<WsRegs<T>::WALK>();
    Pair& sm = pairs[warp - OTOO_WS_PAIRS];
    GravWalker<T, PROF> w(p, sm, lane);
    long long wk0 = 0;
    if (PROF) wk0 = clock64();
    float4* list = w.acquire();
    walk_driver(p.c, w, list, sm.stk, lane, (int64_t)blockIdx.x * OTOO_WS_PAIRS + (warp - OTOO_WS_PAIRS));
    w.finish();
    if (PROF && lane == 0) { atomicAdd(p.c.sums + 11, (unsigned long long)w.wait_ticks); atomicAdd(p.c.sums + 13, (unsigned long long)(clock64() - wk0)); }
  } else {
    // ---- evaluator: targets and sums in registers, consumes the buffers in order
    if (WsRegs<T>::EVAL) setmaxnreg_inc<WsRegs<T>::EVAL>();
    Pair& sm = pairs[warp];
    GravVisitor<T, EPS0, WsRegs<T>::PB, WsRegs<T>::UNR> v(p);
    uint32_t buf = 0, fparity = 0;
    long long ewait = 0;
    long long ev0 = 0;
    if (PROF) ev0 = clock64();
    for (;;) {
      long long w0 = 0;
      if (PROF) w0 = clock64();
      mbar_wait(&sm.full[buf], (fparity >> buf) & 1u);
      if (PROF) ewait += clock64() - w0;
      fparity ^= 1u << buf;
      const WsMeta m = sm.meta[buf];
      if (m.flags & WS_EXIT) break;
      const int64_t g0 = (int64_t)m.group * p.c.gs;
      if (m.flags & WS_FIRST) { v.load_group(g0, lane, reinterpret_cast<float4*>(sm.tgt)); __syncwarp(); }
      if (!p.c.walk_only && m.count) v.eval(sm.list[buf], (int)m.count);
      if (m.flags & WS_LAST) { v.selfmask = sm.self[buf][lane]; v.store(g0, lane); }
      mbar_arrive(&sm.empty[buf]);
      buf = (buf + 1) % OTOO_WS_NBUF;
    }
    if (PROF && lane == 0) { atomicAdd(p.c.sums + 10, (unsigned long long)ewait); atomicAdd(p.c.sums + 12, (unsigned long long)(clock64() - ev0)); }
    if (threadIdx.x == 0) {
      unsigned long long ns1;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns1));
      atomicAdd(p.c.sums + 8, (unsigned long long)(clock64() - ck0));
      atomicAdd(p.c.sums + 9, ns1 - ns0);
    }
  }
}

template <int T, bool EPS0, bool PROF>
otoo_status launch_walk_ws3(otoo_ctx* ctx, const GravParams& p, cudaStream_t st) {
  const size_t smem = OTOO_WS_PAIRS * sizeof(typename GravWalker<T>::Pair);
  OTOO_CUDA(ctx, cudaFuncSetAttribute(walk_gravity_ws_kernel<T, EPS0, PROF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int occ = 1;
  OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, walk_gravity_ws_kernel<T, EPS0, PROF>, OTOO_WS_PAIRS * 64, smem));
  if (occ < 1) occ = 1;
  int64_t grid = (int64_t)ctx->sm_count * occ;                       // persistent: every CTA resident
  if (grid * OTOO_WS_PAIRS > p.c.ngroups) grid = cdiv(p.c.ngroups > 0 ? p.c.ngroups : 1, OTOO_WS_PAIRS);
  walk_gravity_ws_kernel<T, EPS0, PROF><<<(unsigned)grid, OTOO_WS_PAIRS * 64, smem, st>>>(p);
  return OTOO_OK;
}
template <int T, bool EPS0>
otoo_status launch_walk_ws2(otoo_ctx* ctx, const GravParams& p, cudaStream_t st) {
  return ctx->walk_profile ? launch_walk_ws3<T, EPS0, true>(ctx, p, st) : launch_walk_ws3<T, EPS0, false>(ctx, p, st);
}
template <int T>
otoo_status launch_walk_ws(otoo_ctx* ctx, const GravParams& p, bool eps0, cudaStream_t st) {
  return eps0 ? launch_walk_ws2<T, true>(ctx, p, st) : launch_walk_ws2<T, false>(ctx, p, st);
}

// reset the control block and the pool's sequence numbers (tickets restart from 0 every launch)
__global__ void __launch_bounds__(256) walk_init_kernel(WalkShared* ws, uint32_t* seq) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < OTOO_POOL_SLOTS) seq[i] = (uint32_t)i;
  if (i == 0) { ws->queue = 0; ws->head = 0; ws->tail = 0; ws->outstanding = 0; }
}

template <int T, bool EPS0>
otoo_status launch_walk2(otoo_ctx* ctx, const GravParams& p, int grid, size_t smem, cudaStream_t st) {
  OTOO_CUDA(ctx, cudaFuncSetAttribute(walk_gravity_kernel<T, EPS0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int occ = 1;
  OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, walk_gravity_kernel<T, EPS0>, OTOO_WALK_WARPS * 32, smem));
  if (occ < 1) occ = 1;
  if (grid > ctx->sm_count * occ) grid = ctx->sm_count * occ;   // persistent: every CTA resident
  walk_gravity_kernel<T, EPS0><<<grid, OTOO_WALK_WARPS * 32, smem, st>>>(p);
  return OTOO_OK;
}
template <int T>
otoo_status launch_walk(otoo_ctx* ctx, const GravParams& p, bool eps0, int grid, size_t smem, cudaStream_t st) {
  return eps0 ? launch_walk2<T, true>(ctx, p, grid, smem, st) : launch_walk2<T, false>(ctx, p, grid, smem, st);
}

}  // namespace

size_t otoo_walk_smem_bytes() {
  return (size_t)OTOO_WALK_WARPS * (OTOO_LIST_STRIDE * sizeof(float4) + OTOO_WALK_STACK_MAX * sizeof(uint32_t));
}
static size_t grav_fused_smem_bytes() { return otoo_walk_smem_bytes() + (size_t)OTOO_WALK_WARPS * 2 * OTOO_PIECES * sizeof(float4); }

// Common launch preparation of the walk kernels: persistent grid, task pool, zeroed counters.
otoo_status otoo_walk_prepare(otoo_ctx* ctx, int G, WalkCommon* c, int* grid, size_t* smem, cudaStream_t st, bool reset) {
  const int64_t total_groups = cdiv(ctx->N, G);
  // target sharding (PAPER III-E, L179: every device holds the whole tree and walks a contiguous range of targets)
  const int64_t g_begin = ctx->group_begin;
  const int64_t ngroups = ctx->group_count < 0 ? total_groups - g_begin : ctx->group_count;
  if (g_begin < 0 || ngroups < 0 || g_begin + ngroups > total_groups)
    return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_begin / group_count outside the groups of this group_size");
  OTOO_TRY(otoo_ensure_groups(ctx, total_groups));
  ctx->ev_walk_valid = false;
  OTOO_EV(ctx, ctx->ev_walk[0], st);
  *smem = otoo_walk_smem_bytes();
  int per_sm = (int)((227 * 1024) / (*smem + 1024));
  if (per_sm < 1) per_sm = 1;
  if (per_sm > 6) per_sm = 6;   // 24 warps per SM at most (registers allow 4-6 CTAs)
  const int64_t warps = (int64_t)ctx->sm_count * per_sm * OTOO_WALK_WARPS;
  if (warps >= OTOO_POOL_MARGIN) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "internal: task pool margin below resident warps");
  *grid = ctx->sm_count * per_sm;
  if ((int64_t)*grid * OTOO_WALK_WARPS > ngroups) *grid = (int)cdiv(ngroups > 0 ? ngroups : 1, OTOO_WALK_WARPS);
  OTOO_TRY(otoo_ensure_spill(ctx, warps));
  if (!ctx->pool_slots) {
    OTOO_CUDA(ctx, cudaMalloc((void**)&ctx->pool_slots, sizeof(TaskSlot) * (size_t)OTOO_POOL_SLOTS));
    OTOO_CUDA(ctx, cudaMalloc((void**)&ctx->pool_seq, sizeof(uint32_t) * (size_t)OTOO_POOL_SLOTS));
    OTOO_CUDA(ctx, cudaMalloc((void**)&ctx->walk_shared, sizeof(WalkShared)));
  }
  if (reset) {   // (the gravity calls do this inside their r_b kernel, or find it done by the build)
    if (!ctx->walk_reset_valid) {
      walk_init_kernel<<<OTOO_POOL_SLOTS / 256, 256, 0, st>>>((WalkShared*)ctx->walk_shared, (uint32_t*)ctx->pool_seq);
      ctx->launches += 1;
    }
    ctx->walk_reset_valid = false;                 // the walk that follows uses it up
  }
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->g_ntests, 0, 4 * (size_t)total_groups, st));
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->g_ncells, 0, 4 * (size_t)total_groups, st));
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->g_nparts, 0, 4 * (size_t)total_groups, st));
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->d_sums, 0, OTOO_NSUMS * sizeof(unsigned long long), st));
  c->spos = ctx->spos; c->keys = ctx->key[0]; c->cell_cm = ctx->cell_cm; c->cell_b = ctx->cell_b; c->perm = ctx->val[0];
  c->N = ctx->N; c->ngroups = ngroups; c->g_begin = (uint32_t)g_begin; c->gs = G; c->out_sorted = 0;
  c->g_ntests = ctx->g_ntests; c->g_ncells = ctx->g_ncells; c->g_nparts = ctx->g_nparts;
  c->sums = ctx->d_sums; c->ws = (WalkShared*)ctx->walk_shared; c->slots = (TaskSlot*)ctx->pool_slots;
  c->seq = (uint32_t*)ctx->pool_seq; c->spill = ctx->walk_spill; c->stack_cap = ctx->walk_stack; c->spill_cap = ctx->walk_spill_cap;
  c->use_pool = ctx->use_pool;
  c->walk_only = ctx->walk_only;
  c->dist_kind = 0;
  c->rec_mode = 0; c->rec_cap = 0; c->rec_cells = nullptr; c->rec_count = nullptr; c->rec_ntests = nullptr;
  ctx->last_group_size = G; ctx->last_ngroups = total_groups; ctx->last_walk_only = ctx->walk_only;
  return OTOO_OK;
}

otoo_status otoo_gravity_impl(otoo_ctx* ctx, float eps, int mac, float p0, float p1, int G, float* d_acc_pot, cudaStream_t st) {
  GravParams p;
  int grid; size_t smem;
  OTOO_TRY(otoo_walk_prepare(ctx, G, &p.c, &grid, &smem, st, false));
  smem = grav_fused_smem_bytes();                 // (the one-warp-does-both kernel: + the pieces' boxes)
  const WalkReset wr{p.c.ws, p.c.seq};
  const unsigned nbR = (unsigned)(cdiv(ctx->N_cell, 256) > OTOO_POOL_SLOTS / 256 ? cdiv(ctx->N_cell, 256) : OTOO_POOL_SLOTS / 256);
  int prep_launches = 1;
  if (mac == 0) {
    // the build has left rb^2 of the previous call's theta and a reset pool (build.cu): nothing to launch then
    const bool have_rb2 = ctx->rb2_valid && memcmp(&ctx->rb2_theta, &p0, sizeof(float)) == 0;
    if (!have_rb2) rb2_kernel<<<nbR, 256, 0, st>>>(ctx->c_level, ctx->c_s, ctx->N_cell, ctx->S, p0, ctx->cell_b, wr);
    else if (!ctx->walk_reset_valid) walk_init_kernel<<<OTOO_POOL_SLOTS / 256, 256, 0, st>>>(p.c.ws, p.c.seq);
    else prep_launches = 0;
    ctx->rb2_valid = true; ctx->rb2_theta = p0; ctx->spec_theta = p0; ctx->spec_theta_set = true;
  } else {
    OTOO_TRY(otoo_b2_impl(ctx, st));
    OTOO_TRY(otoo_bmax_impl(ctx, st));
    rb2_delta_kernel<<<nbR, 256, 0, st>>>(ctx->c_B2, ctx->c_MP, ctx->sph_acc, ctx->N_cell, ctx->S, p0, p1, ctx->cell_b, wr);
    ctx->rb2_valid = false;
  }
  ctx->walk_reset_valid = false;                   // the walk below uses the reset up
  OTOO_CUDA(ctx, cudaMemsetAsync(d_acc_pot, 0, 16 * (size_t)ctx->N, st));
  p.eps2 = eps * eps;
  p.acc_pot = reinterpret_cast<float4*>(d_acc_pot);
  const bool eps0 = !(eps > 0.0f);
  if (ctx->dist_kind == 1 && !ctx->use_ws)
    return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_distance = 1 needs warp_specialized = 1");
  p.c.dist_kind = ctx->dist_kind;
  p.c.out_sorted = ctx->out_sorted;
  OTOO_EV(ctx, ctx->ev_walk[1], st);
  if (ctx->use_ws) {
    switch (G) {
      case 4: case 8: case 16: case 32: OTOO_TRY(launch_walk_ws<1>(ctx, p, eps0, st)); break;
      case 64: OTOO_TRY(launch_walk_ws<2>(ctx, p, eps0, st)); break;
      case 128: OTOO_TRY(launch_walk_ws<4>(ctx, p, eps0, st)); break;
      case 256: OTOO_TRY(launch_walk_ws<8>(ctx, p, eps0, st)); break;
      default: return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
    }
  } else
  switch (G) {
    case 4: case 8: case 16: case 32: OTOO_TRY(launch_walk<1>(ctx, p, eps0, grid, smem, st)); break;
    case 64: OTOO_TRY(launch_walk<2>(ctx, p, eps0, grid, smem, st)); break;
    case 128: OTOO_TRY(launch_walk<4>(ctx, p, eps0, grid, smem, st)); break;
    case 256: OTOO_TRY(launch_walk<8>(ctx, p, eps0, grid, smem, st)); break;
    default: return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  }
  OTOO_EV(ctx, ctx->ev_walk[2], st);
  ctx->ev_walk_valid = true;
  ctx->launches += prep_launches + 1;
  OTOO_CUDA(ctx, cudaGetLastError());
  ctx->walked = true;
  return OTOO_OK;
}

// ---------------------------------------------------------------- the FP32 roofline denominator, measured
// 16 independent FFMA2 chains per thread, 8 warps per scheduler: what the FMA pipe of this GPU sustains at
// the clock it holds (bench.py reports the kernel against the nominal peak AND against this number).
namespace {
__global__ void __launch_bounds__(256) fp32_peak_kernel(float2* out, int iters, float2 a) {
  float2 acc[16];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = make_float2((float)(threadIdx.x + i), (float)i);
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = __ffma2_rn(acc[i], a, acc[i]);   // one register pair + one uniform operand:
                                                                          // three distinct pairs lose 15-25 % to the register banks
  }
  float2 s = make_float2(0.0f, 0.0f);
#pragma unroll
  for (int i = 0; i < 16; i++) { s.x += acc[i].x; s.y += acc[i].y; }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace

otoo_status otoo_measure_fp32_peak_impl(otoo_ctx* ctx, double* tflops, cudaStream_t st) {
  const int grid = ctx->sm_count * 8, iters = 20000;
  float2* out = reinterpret_cast<float2*>(ctx->key[1]);          // scratch: 8 B x grid x 256 <= capacity of key[1]?
  float2* tmp = nullptr;
  if ((int64_t)grid * 256 > ctx->maxN) { OTOO_CUDA(ctx, cudaMalloc((void**)&tmp, sizeof(float2) * (size_t)grid * 256)); out = tmp; }
  cudaEvent_t e0, e1;
  OTOO_CUDA(ctx, cudaEventCreate(&e0)); OTOO_CUDA(ctx, cudaEventCreate(&e1));
  fp32_peak_kernel<<<grid, 256, 0, st>>>(out, 200, make_float2(-1e-6f, -1e-6f));
  float best = 1e30f;
  for (int r = 0; r < 3; r++) {
    cudaEventRecord(e0, st);
    fp32_peak_kernel<<<grid, 256, 0, st>>>(out, iters, make_float2(-1e-6f, -1e-6f));
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0.0f; cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (tmp) cudaFree(tmp);
  OTOO_CUDA(ctx, cudaGetLastError());
  *tflops = (double)grid * 256.0 * 16.0 * 2.0 * 2.0 * (double)iters / ((double)best * 1e-3) / 1e12;
  return OTOO_OK;
}
