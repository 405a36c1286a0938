// gravity.cu -- theta-MAC radii (R7) and the fused group walk + softened Plummer sums
// (PAPER.md III-D L159-L167, L43, L57; readings R7-R11).
#include "walk.cuh"

namespace {

// R7: r_b = l/theta + s in fp64, rb^2 rounded once to fp32.  theta = 0 -> +inf (open everything).
__global__ void __launch_bounds__(256) rb2_kernel(const uint8_t* __restrict__ c_level, const double* __restrict__ c_s,
                                                  int64_t ncell, float S, float theta, cellb_t* __restrict__ cell_b) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  float rb2;
  if (!(theta > 0.0f)) rb2 = INFINITY;
  else {
    double l = ldexp((double)S, -(int)c_level[c]);
    double rb = __dadd_rn(__ddiv_rn(l, (double)theta), c_s[c]);
    rb2 = __double2float_rn(__dmul_rn(rb, rb));
  }
  reinterpret_cast<uint32_t*>(cell_b + c)[0] = __float_as_uint(rb2);
}

struct GravParams {
  const float4* spos;
  const float4* cell_cm;
  const cellb_t* cell_b;
  const uint32_t* perm;
  int64_t N;
  int64_t ngroups;
  float eps2;
  float4* acc_pot;
  uint32_t* g_ntests; uint32_t* g_ncells; uint32_t* g_nparts;
  uint32_t* queue;          // work counter
  uint32_t* spill;          // OTOO_WALK_SPILL per warp
  unsigned long long* sums; // tests, interactions, cells, parts
  int stack_cap;
};

constexpr float PAD_POS = 1.0e18f;  // zero-mass padding entries sit far away: contribute exactly 0

// All targets of the lane x list[0..n) (n a multiple of 4).  R10.  13 FP32 lane-ops + 1 MUFU per
// interaction, issued two targets at a time as FFMA2/FADD2/FMUL2.
template <int T, bool EPS0>
__device__ __forceinline__ void eval_list(const float4* __restrict__ list, int n, f32x2 eps2p,
                                          const f32x2 (&PX)[(T + 1) / 2], const f32x2 (&PY)[(T + 1) / 2],
                                          const f32x2 (&PZ)[(T + 1) / 2], f32x2 (&AX)[(T + 1) / 2],
                                          f32x2 (&AY)[(T + 1) / 2], f32x2 (&AZ)[(T + 1) / 2], f32x2 (&PH)[(T + 1) / 2]) {
  constexpr int NP = (T + 1) / 2;
  constexpr int PB = NP < 2 ? NP : 2;  // pairs per pass over the list (4 targets)
#pragma unroll
  for (int pb = 0; pb < NP; pb += PB) {
#pragma unroll 4
    for (int j = 0; j < n; j++) {
      const float4 s = list[j];
      const f32x2 sx = pk2(s.x, s.x), sy = pk2(s.y, s.y), sz = pk2(s.z, s.z), sw = pk2(s.w, s.w);
#pragma unroll
      for (int q = pb; q < pb + PB; q++) {
        f32x2 dx = sub2(sx, PX[q]), dy = sub2(sy, PY[q]), dz = sub2(sz, PZ[q]);
        f32x2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, eps2p)));
        float r2a, r2b;
        upk2(r2, r2a, r2b);
        float ia = rsqrt_approx(r2a), ib = rsqrt_approx(r2b);
        if (EPS0) { ia = r2a > 0.0f ? ia : 0.0f; ib = r2b > 0.0f ? ib : 0.0f; }  // r = 0 pairs contribute 0
        f32x2 ri = pk2(ia, ib);
        f32x2 mri = mul2(sw, ri);
        f32x2 mr3 = mul2(mri, mul2(ri, ri));
        PH[q] = sub2(PH[q], mri);
        AX[q] = fma2(mr3, dx, AX[q]);
        AY[q] = fma2(mr3, dy, AY[q]);
        AZ[q] = fma2(mr3, dz, AZ[q]);
      }
    }
  }
}

template <int T, bool EPS0>
__global__ void __launch_bounds__(OTOO_WALK_WARPS * 32) walk_gravity_kernel(GravParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int NP = (T + 1) / 2;
  constexpr int G = 32 * T;
  float4* list = reinterpret_cast<float4*>(smem_raw) + warp * OTOO_LIST_CAP;
  uint32_t* stk = reinterpret_cast<uint32_t*>(smem_raw + OTOO_WALK_WARPS * OTOO_LIST_CAP * sizeof(float4)) +
                  warp * OTOO_WALK_STACK_MAX;
  const int64_t gwarp = (int64_t)blockIdx.x * OTOO_WALK_WARPS + warp;
  WarpStack st;
  const f32x2 eps2p = pk2(p.eps2, p.eps2);
  unsigned long long tot_tests = 0, tot_inter = 0, tot_cells = 0, tot_parts = 0;

  for (;;) {
    uint32_t g = 0;
    if (lane == 0) g = atomicAdd(p.queue, 1u);
    g = __shfl_sync(0xFFFFFFFFu, g, 0);
    if ((int64_t)g >= p.ngroups) break;
    const int64_t g0 = (int64_t)g * G;
    const int gcount = (int)((p.N - g0) < G ? (p.N - g0) : G);

    // ---- targets (H7): lane holds slots g0 + t*32 + lane; out-of-range lanes mirror slot g0
    float px[T], py[T], pz[T], pm[T];
    float glo[3], ghi[3];
#pragma unroll
    for (int t = 0; t < T; t++) {
      int64_t s = g0 + t * 32 + lane;
      float4 v = p.spos[s < p.N ? s : g0];
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
    f32x2 PX[NP], PY[NP], PZ[NP], AX[NP], AY[NP], AZ[NP], PH[NP];
#pragma unroll
    for (int q = 0; q < NP; q++) {
      const int t1 = (2 * q + 1 < T) ? 2 * q + 1 : 2 * q;
      PX[q] = pk2(px[2 * q], px[t1]); PY[q] = pk2(py[2 * q], py[t1]); PZ[q] = pk2(pz[2 * q], pz[t1]);
      AX[q] = AY[q] = AZ[q] = PH[q] = pk2(0.0f, 0.0f);
    }

    // ---- walk
    st.init(stk, p.spill + gwarp * OTOO_WALK_SPILL, p.stack_cap);
    if (lane == 0) stk[0] = 0u;  // root
    __syncwarp();
    st.sp = 1;
    int nlist = 0;
    uint32_t ntests = 0, ncells = 0, nparts = 0;
    unsigned selfmask = 0;

    auto flush = [&]() {
      int n4 = (nlist + 3) & ~3;
      if (lane < n4 - nlist) list[nlist + lane] = make_float4(PAD_POS, PAD_POS, PAD_POS, 0.0f);
      __syncwarp();
      eval_list<T, EPS0>(list, n4, eps2p, PX, PY, PZ, AX, AY, AZ, PH);
      __syncwarp();
      nlist = 0;
    };

    while (!st.empty()) {
      if (st.sp == 0) st.refill(lane);
      const int k = st.sp < 32 ? st.sp : 32;
      const bool have = lane < k;
      uint32_t cell = 0;
      if (have) cell = stk[st.sp - k + lane];
      __syncwarp();
      st.sp -= k;
      float4 A = make_float4(0.f, 0.f, 0.f, 0.f);
      cellb_t B = make_uint4(0u, 0u, 0u, 0u);
      bool accept = false;
      if (have) {
        A = __ldg(p.cell_cm + cell);
        B = __ldg(p.cell_b + cell);
        float d2 = aabb_d2(glo, ghi, A.x, A.y, A.z);
        accept = d2 > __uint_as_float(B.x);  // strict: equality opens (R8)
      }
      ntests += (uint32_t)k;
      const bool leaf = (B.w & 1u) != 0u;
      const bool open_leaf = have && !accept && leaf;
      const bool open_int = have && !accept && !leaf;

      // accepted cells -> list (the cell is a virtual particle at its centre of mass, L43)
      const unsigned am = __ballot_sync(0xFFFFFFFFu, accept);
      const int na = __popc(am);
      if (na) {
        if (nlist + na > OTOO_LIST_CAP) flush();
        if (accept) list[nlist + __popc(am & lanemask_lt_())] = A;
        nlist += na; ncells += (uint32_t)na;
      }
      // opened internal cells -> push children (L57 rule 1: follow `more`)
      {
        const int nch = open_int ? (int)B.z : 0;
        const int inc = warp_inclusive_scan(nch, lane);
        const int total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        if (total) {
          st.reserve(total, lane);
          const int o = st.sp + inc - nch;
          for (int i = 0; i < nch; i++) stk[o + i] = B.y + (uint32_t)i;
          __syncwarp();
          st.sp += total;
        }
      }
      // opened leaves -> their particles (L57 rule 3)
      const unsigned lm = __ballot_sync(0xFFFFFFFFu, open_leaf);
      if (lm) {
        const int cnt = open_leaf ? (int)B.z : 0;
        const int inc = warp_inclusive_scan(cnt, lane);
        const int total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        // which of my targets sit in an opened leaf (their self term is in the list)
        unsigned m = lm;
        while (m) {
          const int src = __ffs(m) - 1; m &= m - 1;
          const uint32_t f = __shfl_sync(0xFFFFFFFFu, B.y, src), c = __shfl_sync(0xFFFFFFFFu, B.z, src);
#pragma unroll
          for (int t = 0; t < T; t++) if ((uint32_t)(g0 + t * 32 + lane) - f < c) selfmask |= 1u << t;
        }
        if (total <= OTOO_LIST_CAP) {
          if (nlist + total > OTOO_LIST_CAP) flush();
          const int o = nlist + inc - cnt;
          for (int i = 0; i < cnt; i++) list[o + i] = p.spos[B.y + i];
          nlist += total;
        } else {  // huge leaves (coincident points at level 21): one leaf at a time, 32 particles a chunk
          m = lm;
          while (m) {
            const int src = __ffs(m) - 1; m &= m - 1;
            const uint32_t f = __shfl_sync(0xFFFFFFFFu, B.y, src), c = __shfl_sync(0xFFFFFFFFu, B.z, src);
            for (uint32_t i = 0; i < c; i += 32) {
              if (nlist + 32 > OTOO_LIST_CAP) flush();
              if (i + lane < c) list[nlist + lane] = p.spos[f + i + lane];
              nlist += (int)((c - i) < 32u ? (c - i) : 32u);
            }
          }
        }
        nparts += (uint32_t)total;
        __syncwarp();
      }
    }
    if (nlist) flush();

    // ---- results (H10): original order; remove the self term from phi (R10)
    const float rie = EPS0 ? 0.0f : rsqrt_approx(p.eps2);
#pragma unroll
    for (int t = 0; t < T; t++) {
      const int64_t s = g0 + t * 32 + lane;
      float ax0, ax1, ay0, ay1, az0, az1, ph0, ph1;
      upk2(AX[t >> 1], ax0, ax1); upk2(AY[t >> 1], ay0, ay1); upk2(AZ[t >> 1], az0, az1); upk2(PH[t >> 1], ph0, ph1);
      float4 o = (t & 1) ? make_float4(ax1, ay1, az1, ph1) : make_float4(ax0, ay0, az0, ph0);
      if ((selfmask >> t) & 1u) o.w = __fmaf_rn(pm[t], rie, o.w);
      if (s < p.N) p.acc_pot[p.perm[s]] = o;
    }
    const uint32_t nt = ntests;  // warp-uniform by construction
    if (lane == 0) { p.g_ntests[g] = nt; p.g_ncells[g] = ncells; p.g_nparts[g] = nparts; }
    tot_tests += nt; tot_cells += ncells; tot_parts += nparts;
    tot_inter += (unsigned long long)gcount * (ncells + nparts);
  }
  if (lane == 0 && tot_tests) {
    atomicAdd(p.sums + 0, tot_tests); atomicAdd(p.sums + 1, tot_inter);
    atomicAdd(p.sums + 2, tot_cells); atomicAdd(p.sums + 3, tot_parts);
  }
}

template <int T>
otoo_status launch_walk(otoo_ctx* ctx, const GravParams& p, bool eps0, int grid, size_t smem, cudaStream_t st) {
  if (eps0) {
    OTOO_CUDA(ctx, cudaFuncSetAttribute(walk_gravity_kernel<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    walk_gravity_kernel<T, true><<<grid, OTOO_WALK_WARPS * 32, smem, st>>>(p);
  } else {
    OTOO_CUDA(ctx, cudaFuncSetAttribute(walk_gravity_kernel<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    walk_gravity_kernel<T, false><<<grid, OTOO_WALK_WARPS * 32, smem, st>>>(p);
  }
  return OTOO_OK;
}

}  // namespace

size_t otoo_walk_smem_bytes() {
  return (size_t)OTOO_WALK_WARPS * (OTOO_LIST_CAP * sizeof(float4) + OTOO_WALK_STACK_MAX * sizeof(uint32_t));
}

otoo_status otoo_gravity_impl(otoo_ctx* ctx, float eps, float theta, int G, float* d_acc_pot, cudaStream_t st) {
  const int64_t ngroups = cdiv(ctx->N, G);
  OTOO_TRY(otoo_ensure_groups(ctx, ngroups));
  const size_t smem = otoo_walk_smem_bytes();
  int per_sm = (int)((227 * 1024) / (smem + 1024));
  if (per_sm > 16 / OTOO_WALK_WARPS * 4) per_sm = 16 / OTOO_WALK_WARPS * 4;
  if (per_sm < 1) per_sm = 1;
  int grid = ctx->sm_count * per_sm;
  if ((int64_t)grid * OTOO_WALK_WARPS > ngroups) grid = (int)cdiv(ngroups, OTOO_WALK_WARPS);
  OTOO_TRY(otoo_ensure_spill(ctx, (int64_t)ctx->sm_count * per_sm * OTOO_WALK_WARPS));
  rb2_kernel<<<(unsigned)cdiv(ctx->N_cell, 256), 256, 0, st>>>(ctx->c_level, ctx->c_s, ctx->N_cell, ctx->S, theta, ctx->cell_b);
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->d_counters + 33, 0, sizeof(uint32_t), st));
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->d_sums, 0, 4 * sizeof(unsigned long long), st));
  GravParams p;
  p.spos = ctx->spos; p.cell_cm = ctx->cell_cm; p.cell_b = ctx->cell_b; p.perm = ctx->val[0];
  p.N = ctx->N; p.ngroups = ngroups; p.eps2 = eps * eps;
  p.acc_pot = reinterpret_cast<float4*>(d_acc_pot);
  p.g_ntests = ctx->g_ntests; p.g_ncells = ctx->g_ncells; p.g_nparts = ctx->g_nparts;
  p.queue = ctx->d_counters + 33; p.spill = ctx->walk_spill; p.sums = ctx->d_sums; p.stack_cap = ctx->walk_stack;
  const bool eps0 = !(eps > 0.0f);
  switch (G) {
    case 32: OTOO_TRY(launch_walk<1>(ctx, p, eps0, grid, smem, st)); break;
    case 64: OTOO_TRY(launch_walk<2>(ctx, p, eps0, grid, smem, st)); break;
    case 128: OTOO_TRY(launch_walk<4>(ctx, p, eps0, grid, smem, st)); break;
    case 256: OTOO_TRY(launch_walk<8>(ctx, p, eps0, grid, smem, st)); break;
    default: return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 32, 64, 128 or 256");
  }
  ctx->launches += 2;
  OTOO_CUDA(ctx, cudaGetLastError());
  ctx->walked = true; ctx->last_group_size = G; ctx->last_ngroups = ngroups;
  return OTOO_OK;
}
