// grav_eval.cuh -- the gravity visitor: targets and sums in registers, the R10 pair sum over a shared-memory list.
// Shared by the walk kernels (gravity.cu) and by the sum-loop probe (probe.cu), so that the probe times the very
// loop the product runs.
#pragma once
#include "walk_ws.cuh"

#ifndef OTOO_EVAL_UNR
#define OTOO_EVAL_UNR 4
#endif
#ifndef OTOO_EVAL_ACC
#define OTOO_EVAL_ACC 0
#endif

namespace {

struct GravParams {
  WalkCommon c;
  float eps2;
  float4* acc_pot;          // zeroed before the launch
};

constexpr float PAD_POS = 1.0e18f;  // zero-mass padding entries sit far away: contribute exactly 0

// Gravity visitor: R10 sums.  13 FP32 lane-ops + 1 MUFU per interaction, issued two targets at a
// time as FFMA2/FADD2/FMUL2; two-level summation (64-entry fp32 partial sums, then totals).
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 as2(f32x2 v) { float2 r; upk2(v, r.x, r.y); return r; }

// PB_ = target pairs per pass over the list (0: the default, min(NP, 2)); UNR_ = unroll factor of the entry loop
// ACC_ = form of the three accumulations c += (m/r^3) d: 0 packed FFMA2 (three distinct register pairs each), 1 six scalar FFMA
template <int T_, bool EPS0, int PB_ = 0, int UNR_ = OTOO_EVAL_UNR, int ACC_ = OTOO_EVAL_ACC>
struct GravVisitor {
  static constexpr int T = T_, E = 1, LCAP = OTOO_LIST_CAP, NP = (T_ + 1) / 2, PB = PB_ ? (PB_ < NP ? PB_ : NP) : (NP < 2 ? NP : 2), BLK = 64, UNR = UNR_;
  const GravParams& p;
  float pm[T];
  float glo[3], ghi[3];
  f32x2 PX[NP], PY[NP], PZ[NP];                       // two targets per aligned register pair (kept as b64)
  float2 AX[NP], AY[NP], AZ[NP], PH[NP];
  unsigned selfmask;
  float4* pbox;                                        // the pieces' boxes in shared memory (one-warp-does-both kernel, R25)
  __device__ __forceinline__ GravVisitor(const GravParams& p_) : p(p_), pbox(nullptr) {}

  __device__ __forceinline__ void load_group(int64_t g0, int lane, float4* scratch) {
    float px[T], py[T], pz[T];
#pragma unroll
    for (int t = 0; t < T; t++) {   // H7: lane holds slots g0 + t*32 + lane; out-of-range lanes mirror slot g0
      int64_t s = g0 + t * 32 + lane;
      float4 v = p.c.spos[member_ok(p.c, g0, t * 32 + lane) ? s : g0];
      px[t] = v.x; py[t] = v.y; pz[t] = v.z; pm[t] = v.w;
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
#pragma unroll
    for (int q = 0; q < NP; q++) {
      const int t1 = (2 * q + 1 < T) ? 2 * q + 1 : 2 * q;
      // Round trip through (idle) list memory: the pairs are born as 64-bit values in aligned register
      // pairs.  Without it ptxas keeps the LDG.128 quads and re-pairs x/y/z with 6 MOVs per target pair
      // and list entry inside the hot loop (measured: 25 % of all issued instructions).
      const unsigned sa = (unsigned)__cvta_generic_to_shared(scratch) + (unsigned)(lane * NP * 3 + q * 3) * 8u;
      asm volatile("st.shared.v2.f32 [%0], {%1,%2};" ::"r"(sa), "f"(px[2 * q]), "f"(px[t1]) : "memory");
      asm volatile("st.shared.v2.f32 [%0+8], {%1,%2};" ::"r"(sa), "f"(py[2 * q]), "f"(py[t1]) : "memory");
      asm volatile("st.shared.v2.f32 [%0+16], {%1,%2};" ::"r"(sa), "f"(pz[2 * q]), "f"(pz[t1]) : "memory");
      asm volatile("ld.shared.b64 %0, [%1];" : "=l"(PX[q]) : "r"(sa) : "memory");
      asm volatile("ld.shared.b64 %0, [%1+8];" : "=l"(PY[q]) : "r"(sa) : "memory");
      asm volatile("ld.shared.b64 %0, [%1+16];" : "=l"(PZ[q]) : "r"(sa) : "memory");
      AX[q] = AY[q] = AZ[q] = PH[q] = make_float2(0.0f, 0.0f);
    }
    selfmask = 0;
    if (pbox && p.c.dist_kind == 2) {
      // R25: members through the (idle) list memory, then the pieces' boxes
      __syncwarp();
#pragma unroll
      for (int t = 0; t < T; t++) scratch[t * 32 + lane] = make_float4(px[t], py[t], pz[t], 0.0f);
      __syncwarp();
      group_pieces<T>(p.c.keys, g0, group_count(p.c, g0), lane, scratch, pbox);
    }
  }
  __device__ __forceinline__ int classify(uint32_t cell, float4& A, cellb_t& B) {
    A = __ldg(p.c.cell_cm + cell);
    B = __ldg(p.c.cell_b + cell);
    float d2 = aabb_d2(glo, ghi, A.x, A.y, A.z);
    if (d2 > __uint_as_float(B.x)) return 1;    // strict: equality opens (R8)
    if (p.c.dist_kind != 2) return 2;
    return pieces_d2(pbox, A.x, A.y, A.z) > __uint_as_float(B.x) ? 1 : 2;   // R25
  }
  struct Entry { float4 a; };
  __device__ __forceinline__ Entry get(uint32_t slot) const { Entry e; e.a = p.c.spos[slot]; return e; }
  __device__ __forceinline__ void put(float4* dst, const Entry& e) const { *dst = e.a; }
  __device__ __forceinline__ void pad(float4* dst) { *dst = make_float4(PAD_POS, PAD_POS, PAD_POS, 0.0f); }
  __device__ __forceinline__ void mark_self(uint32_t f, uint32_t n, int64_t g0, int lane) {
#pragma unroll
    for (int t = 0; t < T; t++) if (member_ok(p.c, g0, t * 32 + lane) && (uint32_t)(g0 + t * 32 + lane) - f < n) selfmask |= 1u << t;
  }
  static constexpr bool SUBMIT_LAST = false, CULL = false;
  static constexpr int REC = 0;
  template <class En> __device__ __forceinline__ bool keep(const En&) const { return true; }
  __device__ __forceinline__ float4* submit(float4* list, int n, bool) {
    if (!p.c.walk_only) eval(list, n);
    return list;
  }
  // 13 FP32 lane-ops + 1 MUFU per interaction, as 13 packed FFMA2/FADD2/FMUL2 + 2 MUFU per target pair
  // (the list entry is a scalar broadcast operand); two-level summation: 64-entry partial sums, then totals.
  __device__ __forceinline__ void eval(const float4* __restrict__ list, int n) {
    const float2 e2 = bc2(p.eps2);
#pragma unroll
    for (int pb = 0; pb < NP; pb += PB) {
      for (int j0 = 0; j0 < n; j0 += BLK) {
        const int je = j0 + BLK < n ? j0 + BLK : n;
        float2 cx[PB], cy[PB], cz[PB], cp[PB];
#pragma unroll
        for (int q = 0; q < PB; q++) cx[q] = cy[q] = cz[q] = cp[q] = make_float2(0.0f, 0.0f);
#pragma unroll UNR
        for (int j = j0; j < je; j++) {
          const float4 s = list[j];
#pragma unroll
          for (int q = 0; q < PB; q++) {
            const float2 dx = __fadd2_rn(bc2(s.x), neg2(as2(PX[pb + q])));
            const float2 dy = __fadd2_rn(bc2(s.y), neg2(as2(PY[pb + q])));
            const float2 dz = __fadd2_rn(bc2(s.z), neg2(as2(PZ[pb + q])));
            const float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy, dy, __ffma2_rn(dz, dz, e2)));
            float2 ri = make_float2(rsqrt_approx(r2.x), rsqrt_approx(r2.y));
            if (EPS0) { ri.x = r2.x > 0.0f ? ri.x : 0.0f; ri.y = r2.y > 0.0f ? ri.y : 0.0f; }  // r = 0 pairs contribute 0
            const float2 mri = __fmul2_rn(bc2(s.w), ri);
            const float2 mr3 = __fmul2_rn(mri, __fmul2_rn(ri, ri));
            cp[q] = __fadd2_rn(cp[q], neg2(mri));
            if (ACC_ == 0) {
              cx[q] = __ffma2_rn(mr3, dx, cx[q]);
              cy[q] = __ffma2_rn(mr3, dy, cy[q]);
              cz[q] = __ffma2_rn(mr3, dz, cz[q]);
            } else {
              cx[q].x = __fmaf_rn(mr3.x, dx.x, cx[q].x); cy[q].x = __fmaf_rn(mr3.x, dy.x, cy[q].x); cz[q].x = __fmaf_rn(mr3.x, dz.x, cz[q].x);
              cx[q].y = __fmaf_rn(mr3.y, dx.y, cx[q].y); cy[q].y = __fmaf_rn(mr3.y, dy.y, cy[q].y); cz[q].y = __fmaf_rn(mr3.y, dz.y, cz[q].y);
            }
          }
        }
#pragma unroll
        for (int q = 0; q < PB; q++) {
          AX[pb + q] = __fadd2_rn(AX[pb + q], cx[q]); AY[pb + q] = __fadd2_rn(AY[pb + q], cy[q]);
          AZ[pb + q] = __fadd2_rn(AZ[pb + q], cz[q]); PH[pb + q] = __fadd2_rn(PH[pb + q], cp[q]);
        }
      }
    }
  }
  // H10: original order; the self term is removed from phi by whichever task saw it (R10)
  __device__ __forceinline__ void store(int64_t g0, int lane) {
    const float rie = EPS0 ? 0.0f : rsqrt_approx(p.eps2);
#pragma unroll
    for (int t = 0; t < T; t++) {
      const int64_t s = g0 + t * 32 + lane;
      const int q = t >> 1;
      float4 o = (t & 1) ? make_float4(AX[q].y, AY[q].y, AZ[q].y, PH[q].y) : make_float4(AX[q].x, AY[q].x, AZ[q].x, PH[q].x);
      if ((selfmask >> t) & 1u) o.w = __fmaf_rn(pm[t], rie, o.w);
      if (member_ok(p.c, g0, t * 32 + lane)) {
        float* dst = reinterpret_cast<float*>(p.acc_pot + out_row(p.c, s));
        atomicAdd(dst + 0, o.x); atomicAdd(dst + 1, o.y); atomicAdd(dst + 2, o.z); atomicAdd(dst + 3, o.w);
      }
    }
  }
};

}  // namespace
