// walk_ws.cuh -- warp-specialised hand-off between walker warps and evaluator warps.
//
// The fused one-warp-does-both kernel leaves the FP32 pipe idle while a warp is in its walk phase
// (a chain of dependent L2/DRAM round trips, ~400 instructions per 32 MAC tests): ncu shows the walk
// alone at 40 % of the fused time and only a quarter of it hidden.  Here a CTA holds OTOO_WS_PAIRS
// (walker, evaluator) warp pairs.  The walker runs walk_driver (walk.cuh: same rules, same task pool)
// and fills a ring of OTOO_WS_NBUF interaction-list buffers in shared memory; its evaluator keeps the
// group's targets and accumulators in registers and consumes the buffers.  Hand-off by mbarriers
// (full/empty per buffer, 32 arrivals each).  Registers are moved from the walkers to the evaluators
// with setmaxnreg (the two roles are separate warpgroups).  The lists still never touch HBM.
#pragma once
#include "walk.cuh"

#define OTOO_WS_PAIRS 4     // (walker, evaluator) pairs per CTA: warps 0..3 evaluate, warps 4..7 walk
#ifndef OTOO_WS_NBUF
#define OTOO_WS_NBUF 2      // list buffers per pair
#endif
#ifndef OTOO_WS_LCAP
#define OTOO_WS_LCAP 256    // float4 entries per buffer
#endif

enum : uint32_t { WS_FIRST = 1u, WS_LAST = 2u, WS_EXIT = 4u };
struct WsMeta { uint32_t count, flags, group, pad; };

// shared memory of one pair; NT = float2 words of target staging (32 lanes x NP x 3)
// NM = float4 slots for the group's members (exact-minimum group distance of the gravity walker)
template <int NT, int NM = 1>
struct __align__(16) WsPair {
  float4 list[OTOO_WS_NBUF][OTOO_WS_LCAP + 4];   // +4 entries: consecutive buffers start on different banks
  float4 mem[NM];
  float4 sub[(NM + 7) / 8 * 2];                  // tight boxes of 8 consecutive members: (lo.xyz, -), (hi.xyz, -)
  float4 pbox[2 * OTOO_PIECES];                  // tight boxes of the group's pieces (R25)
  float2 tgt[NT];
  uint32_t stk[OTOO_WALK_STACK_MAX];
  uint32_t self[OTOO_WS_NBUF][32];
  WsMeta meta[OTOO_WS_NBUF];
  unsigned long long full[OTOO_WS_NBUF], empty[OTOO_WS_NBUF];
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void* bar) {   // release at CTA scope
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
template <int BACKOFF_NS = 0>
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) {   // acquire at CTA scope
  const uint32_t a = smem_u32(bar);
  uint32_t ok;
  for (;;) {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    if (ok) break;
    if (BACKOFF_NS) __nanosleep(BACKOFF_NS);
  }
}
template <int R> __device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R)); }
template <int R> __device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R)); }
