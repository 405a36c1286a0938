// walk.cuh -- warp-level machinery shared by the gravity and SPH walk kernels.
// One warp owns one group of G = 32*T Morton-consecutive targets (n_vec targets
// share one traversal).  The traversal is the paper's "open -> descend, accept -> interact, leaf ->
// its particles" rule set (L57) run 32 cells at a time from a LIFO stack in shared memory;
// accepted cells and opened leaves' particles are appended to an interaction list in shared
// memory, which is consumed (all targets x all entries) whenever it fills.  The list never
// touches HBM.
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

// R8: squared distance from the group's AABB to a point, the exact fp32 expression both sides use.
__device__ __forceinline__ float aabb_d2(const float glo[3], const float ghi[3], float cx, float cy, float cz) {
  float ex = fmaxf(0.0f, fmaxf(__fsub_rn(glo[0], cx), __fsub_rn(cx, ghi[0])));
  float ey = fmaxf(0.0f, fmaxf(__fsub_rn(glo[1], cy), __fsub_rn(cy, ghi[1])));
  float ez = fmaxf(0.0f, fmaxf(__fsub_rn(glo[2], cz), __fsub_rn(cz, ghi[2])));
  return __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex)));
}

// Per-warp LIFO of cell ids: shared memory on top, global-memory spill below it.
// With 32 cells popped per step the stack stays sorted by level and holds at most 8*32 entries per
// level, so OTOO_WALK_SPILL entries per warp can never overflow.
struct WarpStack {
  uint32_t* s;      // shared, cap entries
  uint32_t* g;      // global spill area of this warp
  int cap;          // usable shared entries (>= 512)
  int sp, gsp;      // warp-uniform

  __device__ __forceinline__ void init(uint32_t* smem, uint32_t* spill, int cap_) { s = smem; g = spill; cap = cap_; sp = 0; gsp = 0; }
  __device__ __forceinline__ bool empty() const { return sp == 0 && gsp == 0; }
  // make room for `total` (<= 256) pushes
  __device__ __forceinline__ void reserve(int total, int lane) {
    if (sp + total <= cap) return;
    const int H = cap >> 1;  // spill the bottom (shallowest) half
    for (int i = lane; i < H; i += 32) g[gsp + i] = s[i];
    __syncwarp();
    for (int c = 0; c < sp - H; c += 32) {
      uint32_t v = (c + lane < sp - H) ? s[H + c + lane] : 0u;
      __syncwarp();
      if (c + lane < sp - H) s[c + lane] = v;
      __syncwarp();
    }
    gsp += H; sp -= H;
  }
  __device__ __forceinline__ void refill(int lane) {  // sp == 0, gsp > 0
    const int H = cap >> 1;
    int k = gsp < H ? gsp : H;
    for (int i = lane; i < k; i += 32) s[i] = g[gsp - k + i];
    __syncwarp();
    gsp -= k; sp = k;
  }
};

// inclusive warp scan of small ints
__device__ __forceinline__ int warp_inclusive_scan(int x, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xFFFFFFFFu, x, o); if (lane >= o) x += y; }
  return x;
}
