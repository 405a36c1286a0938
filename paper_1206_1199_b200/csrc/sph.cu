// sph.cu -- SPH cell radii (Eq. 5; R14), SPH group walk (R15) fused with the
// density sum (Eq. 4; R13, R16) and the symmetric pressure force (L252 step 6; R17).
// "There is no particle-cell interaction in SPH" (L105): the walk only produces a particle list.
#include "walk_ws.cuh"

namespace {

__global__ void __launch_bounds__(256) gather_h_kernel(const float* __restrict__ h, const uint32_t* __restrict__ perm,
                                                       int64_t n, float* __restrict__ hs) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) hs[s] = h[perm[s]];
}
// per sorted slot: (h, P/rho^2) and velocity
__global__ void __launch_bounds__(256) gather_force_inputs_kernel(const float* __restrict__ h, const float* __restrict__ rho,
                                                                  const float* __restrict__ P, const float4* __restrict__ vel,
                                                                  const float4* __restrict__ visc,
                                                                  const uint32_t* __restrict__ perm, int64_t n,
                                                                  float4* __restrict__ aux, float4* __restrict__ svel,
                                                                  float4* __restrict__ svis) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  uint32_t i = perm[s];
  float r = rho[i];
  aux[s] = make_float4(h[i], __fdiv_rn(P[i], __fmul_rn(r, r)), __fmul_rn(h[i], h[i]), r);   // (h, P/rho^2, h^2, rho)
  if (vel) { float4 v = vel[i]; if (visc) v.w = visc[i].x; svel[s] = v; }                        // (v, c)
  if (visc) svis[s] = make_float4(visc[i].y, visc[i].z, 0.0f, 0.0f);                            // (alpha, f)
}

__global__ void __launch_bounds__(256) gather_vel_kernel(const float4* __restrict__ vel, const uint32_t* __restrict__ perm, int64_t n,
                                                         float4* __restrict__ svel) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) svel[s] = vel[perm[s]];
}
// (div v, rot v) sums -> estimates: divide by the particle's density (R22)
// over the sorted slots [s0, s1) of the walked target groups only: with a group range (options group_begin /
// group_count) the other targets keep their zeros (0/0 would poison the sum over the ranges)
__global__ void __launch_bounds__(256) divrot_finish_kernel(const float* __restrict__ rho, const uint32_t* __restrict__ perm,
                                                            int64_t s0, int64_t s1, float4* __restrict__ dr) {
  const int64_t s = s0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= s1) return;
  const uint32_t i = perm[s];
  const float r = rho[i];
  float4 v = dr[i];
  dr[i] = make_float4(__fdiv_rn(v.x, r), __fdiv_rn(v.y, r), __fdiv_rn(v.z, r), __fdiv_rn(v.w, r));
}
// ---- R14: b_max and r_SPH over ALL particles of every cell, from the fp64 centre of mass.
// A particle at sorted slot s lies in one cell of every level 0 .. LL(s) (LL of the build's per-slot record `info`: the
// level of the slot's leaf), and that cell is the last level-l cell that starts at or before s.  Canonical cell indices
// count exactly those starts (build.cu, place_cells_kernel), so the index comes from the build's scanned per-block level
// counts (blk_off) plus a ballot -- no descent through the tree (the first form walked every particle from the root to its
// leaf: five or more dependent loads per level, 0.30 ms for 2 M particles).  Consecutive slots share cells, so a warp first
// reduces runs of equal cell id with shuffles and only run heads touch memory.
// F32: the maxima are kept as fp32 rounded up (what the SPH walks read: rounding up is monotone, so the maximum of the
// rounded values is the rounded maximum) in out32, by 32-bit atomics; else as fp64 bit patterns in acc (the Delta-MAC
// needs b_max in fp64).
template <bool F32>
__global__ void __launch_bounds__(256) sph_radii_kernel(const float4* __restrict__ spos, const float* __restrict__ hs, int64_t n,
                                                        const uint32_t* __restrict__ info, const uint32_t* __restrict__ blk_off,
                                                        const double* __restrict__ cm64,
                                                        unsigned long long* acc /* 2 per cell */, uint32_t* out32 /* 2 per cell */) {
  __shared__ uint32_t wc[8][OTOO_NLEV];          // level-l cells the warp starts, then the canonical index of its first one
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane < OTOO_NLEV) wc[warp][lane] = 0;      // (each warp its own row: no block barrier before the ballots)
  __syncwarp();
  const uint32_t my_off = threadIdx.x < OTOO_NLEV ? blk_off[(size_t)threadIdx.x * gridDim.x + blockIdx.x] : 0u;   // (used after the next barrier)
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = s < n;
  int lo = OTOO_NLEV, LL = -1;
  if (valid) { const uint32_t inf = info[s]; lo = (int)(inf & 0xFF); LL = (int)(inf >> 8); }
  const float4 p = valid ? spos[s] : make_float4(0, 0, 0, 0);
  const double h = (valid && hs) ? (double)hs[s] : 0.0;     // hs == NULL: b_max only (the Delta-MAC of gravity)
  const bool has = lo <= LL;
  const int wlo = __reduce_min_sync(0xFFFFFFFFu, has ? lo : OTOO_NLEV), whi = __reduce_max_sync(0xFFFFFFFFu, has ? LL : -1);
  for (int l = wlo; l <= whi; l++) {
    const unsigned st = __ballot_sync(0xFFFFFFFFu, lo <= l && l <= LL);
    if (lane == 0) wc[warp][l] = (uint32_t)__popc(st);
  }
  __syncthreads();
  if (threadIdx.x < OTOO_NLEV) {
    uint32_t run = my_off;
#pragma unroll
    for (int w = 0; w < 8; w++) { const uint32_t c = wc[w][threadIdx.x]; wc[w][threadIdx.x] = run; run += c; }
  }
  __syncthreads();
  unsigned le;
  asm("mov.u32 %0, %%lanemask_le;" : "=r"(le));
  const int amax = __reduce_max_sync(0xFFFFFFFFu, LL);        // deepest leaf among the warp's slots
  constexpr int LB = 4;                                       // levels per batch: their centres of mass are fetched together
  for (int l0 = 0; l0 <= amax; l0 += LB) {
    uint32_t cells[LB];
    double cx[LB], cy[LB], cz[LB];
#pragma unroll
    for (int j = 0; j < LB; j++) {
      const int l = l0 + j;
      const unsigned st = __ballot_sync(0xFFFFFFFFu, lo <= l && l <= LL);
      cells[j] = l <= LL ? wc[warp][l < OTOO_NLEV ? l : OTOO_NLEV - 1] + (uint32_t)__popc(st & le) - 1u : 0xFFFFFFFFu;
    }
#pragma unroll
    for (int j = 0; j < LB; j++) if (cells[j] != 0xFFFFFFFFu) {
      cx[j] = cm64[3 * (size_t)cells[j]]; cy[j] = cm64[3 * (size_t)cells[j] + 1]; cz[j] = cm64[3 * (size_t)cells[j] + 2];
    }
#pragma unroll
    for (int j = 0; j < LB; j++) {
      if (l0 + j > amax) break;
      const uint32_t cell = cells[j];
      double b = 0.0, r = 0.0;
      if (cell != 0xFFFFFFFFu) {
        double dx = __dsub_rn((double)p.x, cx[j]), dy = __dsub_rn((double)p.y, cy[j]), dz = __dsub_rn((double)p.z, cz[j]);
        b = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        // fp64 form: the maximum of the SQUARED distances (the correctly rounded square root is monotone: the root of
        // the maximum, taken once per cell by rb2_delta_kernel, is the maximum of the roots)
        if (F32) { b = __dsqrt_rn(b); r = __dadd_rn(b, h); }
      }
      // segmented max over runs of equal cell id (runs are contiguous in slot order); head = first lane of a run
      const uint32_t pc = __shfl_up_sync(0xFFFFFFFFu, cell, 1);
      const bool head = (lane == 0) || (pc != cell);
      if (F32) {
        // in the rounded-up fp32 domain from here (non-negative floats order as their bit patterns): one shuffle and
        // an integer max per value and step instead of two shuffles and an fp64 compare-select
        uint32_t bb = __float_as_uint(__double2float_ru(b)), rr = __float_as_uint(__double2float_ru(r));
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const uint32_t oc = __shfl_down_sync(0xFFFFFFFFu, cell, o);
          const uint32_t ob = __shfl_down_sync(0xFFFFFFFFu, bb, o), orr = __shfl_down_sync(0xFFFFFFFFu, rr, o);
          if (lane + o < 32 && oc == cell) { bb = bb > ob ? bb : ob; rr = rr > orr ? rr : orr; }
        }
        if (head && cell != 0xFFFFFFFFu) {
          // a maximum only grows: a value not above what the cell already holds needs no atomic (the cells of the top
          // levels take one atomic per warp otherwise: 65 000 on the root's two words for 2 M particles, and atomics on
          // one address run one after the other -- the kernel took 0.30 ms whatever else it did)
          const uint2 cur = __ldcg(reinterpret_cast<const uint2*>(out32 + 2 * (size_t)cell));
          if (bb > cur.x) atomicMax(out32 + 2 * (size_t)cell, bb);
          if (rr > cur.y) atomicMax(out32 + 2 * (size_t)cell + 1, rr);
        }
      } else {          // the Delta-MAC's b_max^2 alone, in fp64 (acc[2c]; acc[2c + 1] is not written)
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const uint32_t oc = __shfl_down_sync(0xFFFFFFFFu, cell, o);
          const double ob = __shfl_down_sync(0xFFFFFFFFu, b, o);
          if (lane + o < 32 && oc == cell) b = fmax(b, ob);
        }
        if (head && cell != 0xFFFFFFFFu) {
          const unsigned long long bb = (unsigned long long)__double_as_longlong(b);
          if (bb > __ldcg(acc + 2 * (size_t)cell)) atomicMax(acc + 2 * (size_t)cell, bb);
        }
      }
    }
  }
}
struct SphParams {
  WalkCommon c;
  const float* hs;      // h, sorted
  const float4* aux;    // (h, P/rho^2, -, -) sorted
  const float4* svel;   // sorted velocities (w: sound speed for the viscosity) or NULL
  const float4* svis;   // sorted (alpha, Balsara f, -, -) or NULL
  const float2* c_sph;  // (b_max, r_SPH) per cell
  int pieces;                   // 1: MAC and cull per piece of the group (R26); 0: one box per group (R15)
  float* rho; uint32_t* nngb;   // density outputs (zeroed before the launch)
  float4* acc;                  // force output (zeroed before the launch)
};

// MODE 0: density (R16).  MODE 1: pressure force (R17).  MODE 2: pressure force + du/dt.
// MODE 3: density + div v + rot v (SPH stage 1 of PAPER L252; R22).  MODE 4: MODE 2 + artificial viscosity (R24).
#ifndef OTOO_SPH_NZ
#define OTOO_SPH_NZ 1
#endif
#ifndef OTOO_SPH_PAIRS
#define OTOO_SPH_PAIRS 1    // pass-1 targets as 64-bit register pairs (2: in every mode)
#endif
#ifndef OTOO_SPH_CULL
#define OTOO_SPH_CULL 1    // walk-time cull of particles out of reach of the group's box (keep())
#endif
// volatile: the pair is built once per group, not rematerialised from its halves inside the pass-1 loop
__device__ __forceinline__ f32x2 pk2v(float a, float b) { f32x2 r; asm volatile("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 as2(f32x2 v) { float2 r; upk2(v, r.x, r.y); return r; }
// REC_: 1 the walk records the leaves every whole group opens, 2 it starts from recorded leaves (walk.cuh; option sph_reuse_walk)
template <int T_, int MODE, int REC_ = 0>
struct SphVisitor {
  static constexpr int T = T_, E = MODE == 0 ? 1 : (MODE == 1 || MODE == 3 ? 2 : (MODE == 4 ? 4 : 3));
  static constexpr int LCAP = OTOO_LIST_CAP;
  // measured at C4, G = 64: density 3.02 -> 2.83 ms, force + du/dt 4.33 -> 4.21 ms, plain force 3.78 -> 3.84 ms (kept scalar)
  static constexpr bool PAIRS = OTOO_SPH_PAIRS == 2 || (OTOO_SPH_PAIRS == 1 && MODE != 1);
  static constexpr bool GATHER = MODE == 0 || MODE == 3;     // neighbours by the target's own h only (R16)
  const SphParams& p;
  float px[T], py[T], pz[T], ph[T], ppr[T], vx[T], vy[T], vz[T];
  float prho[MODE == 4 ? T : 1], pc[MODE == 4 ? T : 1], pal[MODE == 4 ? T : 1], pf[MODE == 4 ? T : 1];   // viscosity inputs of the targets
  float h2[T], hinv[T], o0[T], o1[T], o2[T], o3[T], o4[T];
  f32x2 PX[(T + 1) / 2], PY[(T + 1) / 2], PZ[(T + 1) / 2], H2[(T + 1) / 2];   // pass 1: two targets per aligned register pair
  uint32_t cnt_ngb[T];
  float glo[3], ghi[3], hmax;
  float4* pbox;        // boxes (lo.xyz, h_max), (hi.xyz, -) of the group's pieces in shared memory (R26); set by the kernel
  __device__ __forceinline__ SphVisitor(const SphParams& p_) : p(p_), pbox(nullptr) {}

  __device__ __forceinline__ void load_group(int64_t g0, int lane, float4* scratch) {
    hmax = 0.0f;
#pragma unroll
    for (int t = 0; t < T; t++) {
      int64_t s = g0 + t * 32 + lane;
      s = member_ok(p.c, g0, t * 32 + lane) ? s : g0;
      float4 v = p.c.spos[s];
      px[t] = v.x; py[t] = v.y; pz[t] = v.z;
      if (GATHER) { ph[t] = p.hs[s]; ppr[t] = 0.0f; }
      else { float4 a = p.aux[s]; ph[t] = a.x; ppr[t] = a.y; if (MODE == 4) prho[t] = a.w; }
      if (MODE >= 2) { float4 w = p.svel[s]; vx[t] = w.x; vy[t] = w.y; vz[t] = w.z; if (MODE == 4) pc[t] = w.w; } else { vx[t] = vy[t] = vz[t] = 0.0f; }
      if (MODE == 4) { float4 q = p.svis[s]; pal[t] = q.x; pf[t] = q.y; }
      hmax = fmaxf(hmax, ph[t]);
      if (t == 0) { glo[0] = ghi[0] = v.x; glo[1] = ghi[1] = v.y; glo[2] = ghi[2] = v.z; }
      else {
        glo[0] = fminf(glo[0], v.x); ghi[0] = fmaxf(ghi[0], v.x);
        glo[1] = fminf(glo[1], v.y); ghi[1] = fmaxf(ghi[1], v.y);
        glo[2] = fminf(glo[2], v.z); ghi[2] = fmaxf(ghi[2], v.z);
      }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
#pragma unroll
      for (int k = 0; k < 3; k++) {
        glo[k] = fminf(glo[k], __shfl_xor_sync(0xFFFFFFFFu, glo[k], o));
        ghi[k] = fmaxf(ghi[k], __shfl_xor_sync(0xFFFFFFFFu, ghi[k], o));
      }
      hmax = fmaxf(hmax, __shfl_xor_sync(0xFFFFFFFFu, hmax, o));
    }
#pragma unroll
    for (int t = 0; t < T; t++) {
      h2[t] = __fmul_rn(ph[t], ph[t]); hinv[t] = 1.0f / ph[t];
      o0[t] = o1[t] = o2[t] = o3[t] = o4[t] = 0.0f; cnt_ngb[t] = 0;
    }
    // Pairs for pass 1.  Built from their halves, ptxas keeps the halves and re-pairs them with two MOVs per
    // operand inside the loop (6 of 16 instructions per entry); read back from shared memory as 64-bit words
    // they are register pairs from the start (the empty list buffer is the scratch: 4 float2 x T/2 per lane).
#pragma unroll
    for (int q = 0; q < (PAIRS ? T / 2 : 0); q++) {
      if (scratch) {
        volatile unsigned long long* sc = reinterpret_cast<volatile unsigned long long*>(scratch) + (q * 4) * 32 + lane;
        sc[0] = pk2(px[2 * q], px[2 * q + 1]); sc[32] = pk2(py[2 * q], py[2 * q + 1]);
        sc[64] = pk2(pz[2 * q], pz[2 * q + 1]); sc[96] = pk2(h2[2 * q], h2[2 * q + 1]);
        PX[q] = sc[0]; PY[q] = sc[32]; PZ[q] = sc[64]; H2[q] = sc[96];
      } else {
        PX[q] = pk2v(px[2 * q], px[2 * q + 1]); PY[q] = pk2v(py[2 * q], py[2 * q + 1]); PZ[q] = pk2v(pz[2 * q], pz[2 * q + 1]);
        H2[q] = pk2v(h2[2 * q], h2[2 * q + 1]);
      }
    }
    if (scratch) __syncwarp();
    if (scratch && pbox && p.pieces) {     // R26: members (x, y, z, h) through the idle list memory, then the pieces
#pragma unroll
      for (int t = 0; t < T; t++) scratch[t * 32 + lane] = make_float4(px[t], py[t], pz[t], ph[t]);
      __syncwarp();
      group_pieces<T>(p.c.keys, g0, group_count(p.c, g0), lane, scratch, pbox);
    }
  }
  // R15: open iff d^2 <= R^2, R = max(r_SPH, b_max + h_max,g); never "accept" (no p-c term, L105).
  // R26: the same test per piece of the group (its box, its own h_max); the whole-group test first: its distance
  // is not above any piece's and its R not below (in fp32 too: every step is monotone), so it only rejects what
  // every piece rejects.
  __device__ __forceinline__ int classify(uint32_t cell, float4& A, cellb_t& B) {
    A = __ldg(p.c.cell_cm + cell);
    B = __ldg(p.c.cell_b + cell);
    float2 rr = __ldg(p.c_sph + cell);
    float d2 = aabb_d2(glo, ghi, A.x, A.y, A.z);
    float R = fmaxf(rr.y, __fadd_rn(rr.x, hmax));
    if (!(d2 <= __fmul_rn(R, R))) return 0;
    if (!p.pieces) return 2;
    bool open = false;
#pragma unroll
    for (int q = 0; q < OTOO_PIECES; q++) {
      const float4 lo = pbox[2 * q], hi = pbox[2 * q + 1];
      const float Rq = fmaxf(rr.y, __fadd_rn(rr.x, lo.w));
      open = open || piece_d2(lo, hi, A.x, A.y, A.z) <= __fmul_rn(Rq, Rq);
    }
    return open ? 2 : 0;
  }
  struct Entry { float4 v[E]; };
  __device__ __forceinline__ Entry get(uint32_t s) const {
    Entry e;
    e.v[0] = p.c.spos[s];
    if (E >= 2) e.v[1] = MODE == 3 ? p.svel[s] : p.aux[s];
    if (E >= 3) e.v[2] = p.svel[s];
    if (E >= 4) e.v[3] = p.svis[s];
    return e;
  }
  __device__ __forceinline__ void put(float4* dst, const Entry& e) const {
#pragma unroll
    for (int k = 0; k < E; k++) dst[k] = e.v[k];
  }
  // Walk-time cull: a particle of an opened leaf enters the list only if it can be a neighbour of some member.
  // Its distance to the group's box, taken with the operations and the order of pass 1's r^2 chain, is never
  // above the fp32 r^2 to any member (every step is monotone in |component|), and the limit is the largest
  // one a member can have, so "box d^2 >= limit" implies that every pair test of this entry fails.
  static constexpr bool CULL = OTOO_SPH_CULL != 0;
  __device__ __forceinline__ bool keep(const Entry& e) const {
    const float4 a = e.v[0];
    const float bx = fmaxf(fmaxf(__fsub_rn(glo[0], a.x), __fsub_rn(a.x, ghi[0])), 0.0f);
    const float by = fmaxf(fmaxf(__fsub_rn(glo[1], a.y), __fsub_rn(a.y, ghi[1])), 0.0f);
    const float bz = fmaxf(fmaxf(__fsub_rn(glo[2], a.z), __fsub_rn(a.z, ghi[2])), 0.0f);
    const float d2 = __fmaf_rn(bz, bz, __fmaf_rn(by, by, __fmul_rn(bx, bx)));
    const float hm2 = __fmul_rn(hmax, hmax);
    const float hj2 = GATHER ? 0.0f : e.v[E >= 2 ? 1 : 0].z;
    if (!(d2 < fmaxf(hm2, hj2))) return false;
    if (!p.pieces) return true;
    // the same argument per piece: a member of piece q has r^2 >= the piece's box distance and a limit <= the
    // piece's largest one
    bool k = false;
#pragma unroll
    for (int q = 0; q < OTOO_PIECES; q++) {
      const float4 lo = pbox[2 * q], hi = pbox[2 * q + 1];
      const float ex = fmaxf(fmaxf(__fsub_rn(lo.x, a.x), __fsub_rn(a.x, hi.x)), 0.0f);
      const float ey = fmaxf(fmaxf(__fsub_rn(lo.y, a.y), __fsub_rn(a.y, hi.y)), 0.0f);
      const float ez = fmaxf(fmaxf(__fsub_rn(lo.z, a.z), __fsub_rn(a.z, hi.z)), 0.0f);
      k = k || __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex))) < fmaxf(__fmul_rn(lo.w, lo.w), hj2);
    }
    return k;
  }
  __device__ __forceinline__ void pad(float4* dst) {
    dst[0] = make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.0f);   // far away, zero mass
    if (E >= 2) dst[1] = make_float4(1.0f, 0.0f, 1.0f, 0.0f);
    if (E >= 3) dst[2] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (E >= 4) dst[3] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  }
  __device__ __forceinline__ void mark_self(uint32_t, uint32_t, int64_t, int) {}
  static constexpr bool SUBMIT_LAST = false;
  static constexpr int REC = REC_;
  __device__ __forceinline__ float4* submit(float4* list, int n, bool) {
    if (!p.c.walk_only) eval(list, n);
    return list;
  }
  // Only ~2 % of the (target, candidate) pairs are neighbours (C4: 5.6e9 candidates, 1.1e8 true pairs), so the
  // list is consumed in two passes.  Pass 1: the fp32 neighbour decision of R16/R17 alone (6 FP32 operations
  // + compare per pair), one result bit per pair, 32 candidates per mask word and target, words parked in
  // shared memory.  Pass 2: every lane walks the set bits of its own targets and evaluates the kernel for
  // those pairs only; the warp runs as many rounds as its busiest lane has hits.
  static constexpr int CAPE = (OTOO_LIST_CAP / E) & ~3, W = (CAPE + 31) / 32;
  uint32_t* msk;      // this warp's mask words in shared memory: [W][T][32 lanes]
  int lane_;
  __device__ __forceinline__ void eval(const float4* __restrict__ list, int n) {
    int w = 0;
    uint32_t nz[T];
#pragma unroll
    for (int t = 0; t < T; t++) nz[t] = 0u;
    for (int jb = 0; jb < n; jb += 32, w++) {
      uint32_t mk[T];
#pragma unroll
      for (int t = 0; t < T; t++) mk[t] = 0u;
      const int nb = n - jb < 32 ? n - jb : 32;
#pragma unroll 4
      for (int k = 0; k < nb; k++) {
        const float4 a = list[E * (jb + k)];
        float hj2 = 0.0f;
        if (!GATHER) hj2 = list[E * (jb + k) + 1].z;
        // exactly this chain on (x_j - x_i): both sides take the neighbour decision in fp32 (R16, R17);
        // two targets per packed instruction (FADD2 / FMUL2 / FFMA2 round each half like the scalar forms)
#pragma unroll
        for (int q = 0; q < T / 2; q++) {
          const float2 ex = __fadd2_rn(make_float2(a.x, a.x), PAIRS ? neg2(as2(PX[q])) : make_float2(-px[2 * q], -px[2 * q + 1]));
          const float2 ey = __fadd2_rn(make_float2(a.y, a.y), PAIRS ? neg2(as2(PY[q])) : make_float2(-py[2 * q], -py[2 * q + 1]));
          const float2 ez = __fadd2_rn(make_float2(a.z, a.z), PAIRS ? neg2(as2(PZ[q])) : make_float2(-pz[2 * q], -pz[2 * q + 1]));
          const float2 r2 = __ffma2_rn(ez, ez, __ffma2_rn(ey, ey, __fmul2_rn(ex, ex)));
          // r2 < lim  <=>  the sign bit of fl32(r2 - lim) (exact: the difference of two floats is negative iff
          // the first is smaller); one funnel shift appends it to the mask word
          const float2 hq = PAIRS ? as2(H2[q]) : make_float2(h2[2 * q], h2[2 * q + 1]);
          const float2 d = __fadd2_rn(r2, GATHER ? neg2(hq) : make_float2(-fmaxf(hq.x, hj2), -fmaxf(hq.y, hj2)));
          mk[2 * q] = __funnelshift_l(__float_as_uint(d.x), mk[2 * q], 1);
          mk[2 * q + 1] = __funnelshift_l(__float_as_uint(d.y), mk[2 * q + 1], 1);
        }
        if (T & 1) {
          const int t = T - 1;
          const float ex = __fsub_rn(a.x, px[t]), ey = __fsub_rn(a.y, py[t]), ez = __fsub_rn(a.z, pz[t]);
          const float r2 = __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex)));
          const float lim = GATHER ? h2[t] : fmaxf(h2[t], hj2);
          mk[t] = __funnelshift_l(__float_as_uint(__fsub_rn(r2, lim)), mk[t], 1);
        }
      }
#pragma unroll
      for (int t = 0; t < T; t++) {
        mk[t] <<= 32 - nb;                       // candidate k of the word sits at bit 31 - k
        if (GATHER) cnt_ngb[t] += (uint32_t)__popc(mk[t]);
        msk[(w * T + t) * 32 + lane_] = mk[t];
        nz[t] |= (mk[t] != 0u ? 1u : 0u) << w;   // most words are empty: pass 2 visits the others only
      }
    }
#pragma unroll
    for (int t = 0; t < T; t++) {
      int ww = 0;
#if OTOO_SPH_NZ
      uint32_t m = 0u, z = nz[t];
      for (;;) {
        if (m == 0u) {
          if (z == 0u) break;
          ww = __ffs(z) - 1; z &= z - 1u;
          m = msk[(ww * T + t) * 32 + lane_];
        }
#else
      uint32_t m = msk[t * 32 + lane_];
      for (;;) {
        while (m == 0u && ++ww < w) m = msk[(ww * T + t) * 32 + lane_];
        if (m == 0u) break;
#endif
        const int k = __clz(m);
        m &= ~(0x80000000u >> k);
        hit(list, (ww << 5) + k, t);
      }
    }
  }
  // one neighbour pair: cubic spline (R13), density term (R16) or symmetric pressure term (R17)
  __device__ __forceinline__ void hit(const float4* __restrict__ list, int j, int t) {
    const float PI_F = 3.14159265358979323846f;
    const float4 a = list[E * j];
    const float ex = __fsub_rn(a.x, px[t]), ey = __fsub_rn(a.y, py[t]), ez = __fsub_rn(a.z, pz[t]);
    const float r2 = __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex)));
    if (MODE == 3) {
      // R22: density term + the gather estimates of div v and rot v with the target's own h
      const float4 c = list[E * j + 1];                      // v_j
      const float rinv = r2 > 0.0f ? rsqrt_approx(r2) : 0.0f;
      const float q = fminf(r2 * rinv * hinv[t], 2.0f);
      const float u = 1.0f - q;
      o0[t] = fmaf(a.w, q <= 0.5f ? fmaf(-6.0f * q * q, u, 1.0f) : 2.0f * u * u * u, o0[t]);
      const float dq = q <= 0.5f ? fmaf(18.0f * q, q, -12.0f * q) : -6.0f * u * u;       // dW/dr in units of 8/(pi h^4)
      const float g = a.w * dq * rinv;                       // m_j (dW/dr)/r; e = x_j - x_i, grad_i W = -(..) e
      const float ux = c.x - vx[t], uy = c.y - vy[t], uz = c.z - vz[t];                  // v_j - v_i
      o1[t] = fmaf(-g, fmaf(ux, ex, fmaf(uy, ey, uz * ez)), o1[t]);                      // div:  m gw u.(x_i - x_j)
      o2[t] = fmaf(-g, ey * uz - ez * uy, o2[t]);                                        // rot:  m gw (x_i - x_j) x u = -g (e x u)
      o3[t] = fmaf(-g, ez * ux - ex * uz, o3[t]);
      o4[t] = fmaf(-g, ex * uy - ey * ux, o4[t]);
    } else if (MODE == 0) {
      float q = fminf(sqrt_approx(r2) * hinv[t], 2.0f);
      float u = 1.0f - q;
      float w1 = fmaf(-6.0f * q * q, u, 1.0f);   // 1 - 6q^2 + 6q^3
      float w2 = 2.0f * u * u * u;
      o0[t] = fmaf(a.w, q <= 0.5f ? w1 : w2, o0[t]);
    } else {
      const float4 b = list[E * j + 1];
      if (!(r2 > 0.0f)) return;                  // the target itself / coincident points: no force (R17)
      float hj = b.x;
      float rinv = rsqrt_approx(r2);
      float r = r2 * rinv;
      float hjinv = __fdividef(1.0f, hj);
      float qi = r * hinv[t], qj = r * hjinv;
      float ui = 1.0f - qi, uj = 1.0f - qj;
      float di = qi <= 0.5f ? fmaf(18.0f * qi, qi, -12.0f * qi) : (qi < 1.0f ? -6.0f * ui * ui : 0.0f);
      float dj = qj <= 0.5f ? fmaf(18.0f * qj, qj, -12.0f * qj) : (qj < 1.0f ? -6.0f * uj * uj : 0.0f);
      float hi2 = hinv[t] * hinv[t], hj2i = hjinv * hjinv;
      float gw = (8.0f / PI_F) * 0.5f * fmaf(di, hi2 * hi2, dj * hj2i * hj2i) * rinv;   // (dW_i + dW_j)/(2r)
      float vd = 0.0f, Pi = 0.0f;
      if (MODE == 2 || MODE == 4) {
        const float4 c = list[E * j + 2];
        // (v_i - v_j).(x_i - x_j) = -(v_i - v_j).e
        vd = -fmaf(vx[t] - c.x, ex, fmaf(vy[t] - c.y, ey, (vz[t] - c.z) * ez));
        if (MODE == 4 && vd < 0.0f) {
          // R24: approaching pair: Pi = fbar (-abar cbar mu + 2 abar mu^2) / rhobar, mu = l w / (r^2 + 0.01 l^2), l = (h_i + h_j)/4
          const float4 q = list[E * j + 3];
          const float l = 0.25f * (ph[t] + hj);
          const float mu = l * vd * __fdividef(1.0f, fmaf(0.01f * l, l, r2));
          const float ab = 0.5f * (pal[t] + q.x), cb = 0.5f * (pc[t] + c.w), fb = 0.5f * (pf[t] + q.y), rb = 0.5f * (prho[t] + b.w);
          Pi = fb * ab * mu * fmaf(2.0f, mu, -cb) * __fdividef(1.0f, rb);
        }
      }
      float f = a.w * (ppr[t] + b.y + Pi) * gw;
      // a_i -= f (x_i - x_j)  =  += f e
      o0[t] = fmaf(f, ex, o0[t]); o1[t] = fmaf(f, ey, o1[t]); o2[t] = fmaf(f, ez, o2[t]);
      if (MODE == 2 || MODE == 4) o3[t] = fmaf(0.5f * f, vd, o3[t]);
    }
  }
  __device__ __forceinline__ void store(int64_t g0, int lane) {
    const float PI_F = 3.14159265358979323846f;
#pragma unroll
    for (int t = 0; t < T; t++) {
      const int64_t s = g0 + t * 32 + lane;
      if (member_ok(p.c, g0, t * 32 + lane)) {
        const uint32_t i = p.c.perm[s];
        if (GATHER) {
          float hi3 = hinv[t] * hinv[t] * hinv[t];
          atomicAdd(p.rho + i, o0[t] * (8.0f / PI_F) * hi3);
          if (p.nngb) atomicAdd(p.nngb + i, cnt_ngb[t]);
          if (MODE == 3) {                                   // unnormalised: divided by rho after the walk
            const float k4 = (8.0f / PI_F) * hi3 * hinv[t];
            float* dst = reinterpret_cast<float*>(p.acc + i);
            atomicAdd(dst + 0, o1[t] * k4); atomicAdd(dst + 1, o2[t] * k4); atomicAdd(dst + 2, o3[t] * k4); atomicAdd(dst + 3, o4[t] * k4);
          }
        } else {
          float* dst = reinterpret_cast<float*>(p.acc + i);
          atomicAdd(dst + 0, o0[t]); atomicAdd(dst + 1, o1[t]); atomicAdd(dst + 2, o2[t]);
          if (MODE == 2 || MODE == 4) atomicAdd(dst + 3, o3[t]);
        }
      }
    }
  }
};

template <int T, int MODE, int REC>
__device__ __forceinline__ void walk_sph_body(const SphParams& p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float4* list = reinterpret_cast<float4*>(smem_raw) + warp * OTOO_LIST_STRIDE;
  uint32_t* stk = reinterpret_cast<uint32_t*>(smem_raw + OTOO_WALK_WARPS * OTOO_LIST_STRIDE * sizeof(float4)) +
                  warp * OTOO_WALK_STACK_MAX;
  SphVisitor<T, MODE, REC> v(p);
  v.msk = reinterpret_cast<uint32_t*>(smem_raw + otoo_walk_smem_bytes_dev()) + warp * (SphVisitor<T, MODE, REC>::W * T * 32);
  v.pbox = reinterpret_cast<float4*>(smem_raw + otoo_walk_smem_bytes_dev() + (size_t)OTOO_WALK_WARPS * SphVisitor<T, MODE, REC>::W * T * 32 * sizeof(uint32_t)) +
           warp * (2 * OTOO_PIECES);
  v.lane_ = lane;
  walk_driver(p.c, v, list, stk, lane, (int64_t)blockIdx.x * OTOO_WALK_WARPS + warp);
}
template <int T, int MODE, int REC>
__global__ void __launch_bounds__(OTOO_WALK_WARPS * 32) walk_sph_kernel(const SphParams p) { walk_sph_body<T, MODE, REC>(p); }
// The density walk of groups up to 64 with 5 CTAs per SM (96 registers instead of 122-126): A/B at C4, G = 64: 2.13 -> 2.03 ms
// (6 CTAs: 2.02).  The force kernels lose with 5 or 6 (force + du/dt 2.98 -> 3.22 / 3.32 ms) and keep ptxas' own choice.
template <int T, int MODE, int REC>
__global__ void __launch_bounds__(OTOO_WALK_WARPS * 32, 5) walk_sph_kernel_occ5(const SphParams p) { walk_sph_body<T, MODE, REC>(p); }
// rec = WalkCommon::rec_mode: the recording / replaying instantiations exist for groups up to 64 (T <= 2), recording for the
// gather stages (density, stage 1), replaying for the force stages; anything else runs the plain walk (a group without a
// record walks from the root in any case)
template <int T, int MODE>
void (*sph_kernel_ptr(int rec))(const SphParams) {
  constexpr bool GATHER = MODE == 0 || MODE == 3;
  if constexpr (T <= 2) {
    if (GATHER && rec == 1) { if constexpr (GATHER) { if constexpr (MODE == 0) return walk_sph_kernel_occ5<T, MODE, 1>; else return walk_sph_kernel<T, MODE, 1>; } }
    if (!GATHER && rec == 2) { if constexpr (!GATHER) return walk_sph_kernel<T, MODE, 2>; }
  }
  if constexpr (MODE == 0 && T <= 2) return walk_sph_kernel_occ5<T, MODE, 0>;
  else return walk_sph_kernel<T, MODE, 0>;
}


// ---------------------------------------------------------------- warp-specialised form (walk_ws.cuh)
// Walker-side visitor: the SPH MAC (R15) and the list entries of SphVisitor without targets or sums;
// submit() publishes the filled buffer to the pair's evaluator warp and returns the next one.
template <int T_, int MODE>
struct SphWalker {
  static constexpr int T = T_, E = MODE == 0 ? 1 : (MODE == 1 ? 2 : 3);
  static constexpr int LCAP = OTOO_WS_LCAP;
  static constexpr bool SUBMIT_LAST = true;
  static constexpr int REC = 0;
  typedef WsPair<2, 32 * T_> Pair;
  const SphParams& p;
  Pair& sm;
  float glo[3], ghi[3], hmax;
  uint32_t group, buf, eparity, first;
  int lane_;
  __device__ __forceinline__ SphWalker(const SphParams& p_, Pair& sm_, int lane) : p(p_), sm(sm_), buf(0), eparity(~0u), first(0), lane_(lane) {}
  __device__ __forceinline__ float4* acquire() {
    mbar_wait<500>(&sm.empty[buf], (eparity >> buf) & 1u);
    eparity ^= 1u << buf;
    return sm.list[buf];
  }
  __device__ __forceinline__ void load_group(int64_t g0, int lane, float4*) {
    hmax = 0.0f;
#pragma unroll
    for (int t = 0; t < T; t++) {
      int64_t s = g0 + t * 32 + lane;
      s = member_ok(p.c, g0, t * 32 + lane) ? s : g0;
      float4 v = p.c.spos[s];
      const float hh = MODE == 0 ? p.hs[s] : p.aux[s].x;
      hmax = fmaxf(hmax, hh);
      if (p.pieces) sm.mem[t * 32 + lane] = make_float4(v.x, v.y, v.z, hh);
      if (t == 0) { glo[0] = ghi[0] = v.x; glo[1] = ghi[1] = v.y; glo[2] = ghi[2] = v.z; }
      else {
        glo[0] = fminf(glo[0], v.x); ghi[0] = fmaxf(ghi[0], v.x);
        glo[1] = fminf(glo[1], v.y); ghi[1] = fmaxf(ghi[1], v.y);
        glo[2] = fminf(glo[2], v.z); ghi[2] = fmaxf(ghi[2], v.z);
      }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
#pragma unroll
      for (int k = 0; k < 3; k++) {
        glo[k] = fminf(glo[k], __shfl_xor_sync(0xFFFFFFFFu, glo[k], o));
        ghi[k] = fmaxf(ghi[k], __shfl_xor_sync(0xFFFFFFFFu, ghi[k], o));
      }
      hmax = fmaxf(hmax, __shfl_xor_sync(0xFFFFFFFFu, hmax, o));
    }
    first = WS_FIRST; group = (uint32_t)(g0 / p.c.gs);
    if (p.pieces) {
      __syncwarp();
      group_pieces<T>(p.c.keys, g0, group_count(p.c, g0), lane, sm.mem, sm.pbox);
    }
  }
  __device__ __forceinline__ int classify(uint32_t cell, float4& A, cellb_t& B) {
    A = __ldg(p.c.cell_cm + cell);
    B = __ldg(p.c.cell_b + cell);
    float2 rr = __ldg(p.c_sph + cell);
    float d2 = aabb_d2(glo, ghi, A.x, A.y, A.z);
    float R = fmaxf(rr.y, __fadd_rn(rr.x, hmax));
    if (!(d2 <= __fmul_rn(R, R))) return 0;
    if (!p.pieces) return 2;
    bool open = false;                            // R26, as SphVisitor::classify
#pragma unroll
    for (int q = 0; q < OTOO_PIECES; q++) {
      const float4 lo = sm.pbox[2 * q], hi = sm.pbox[2 * q + 1];
      const float Rq = fmaxf(rr.y, __fadd_rn(rr.x, lo.w));
      open = open || piece_d2(lo, hi, A.x, A.y, A.z) <= __fmul_rn(Rq, Rq);
    }
    return open ? 2 : 0;
  }
  struct Entry { float4 v[E]; };
  __device__ __forceinline__ Entry get(uint32_t s) const {
    Entry e;
    e.v[0] = p.c.spos[s];
    if (E >= 2) e.v[1] = p.aux[s];
    if (E >= 3) e.v[2] = p.svel[s];
    return e;
  }
  __device__ __forceinline__ void put(float4* dst, const Entry& e) const {
#pragma unroll
    for (int k = 0; k < E; k++) dst[k] = e.v[k];
  }
  // Walk-time cull: a particle of an opened leaf enters the list only if it can be a neighbour of some member.
  // Its distance to the group's box, taken with the operations and the order of pass 1's r^2 chain, is never
  // above the fp32 r^2 to any member (every step is monotone in |component|), and the limit is the largest
  // one a member can have, so "box d^2 >= limit" implies that every pair test of this entry fails.
  static constexpr bool CULL = OTOO_SPH_CULL != 0;
  __device__ __forceinline__ bool keep(const Entry& e) const {
    const float4 a = e.v[0];
    const float bx = fmaxf(fmaxf(__fsub_rn(glo[0], a.x), __fsub_rn(a.x, ghi[0])), 0.0f);
    const float by = fmaxf(fmaxf(__fsub_rn(glo[1], a.y), __fsub_rn(a.y, ghi[1])), 0.0f);
    const float bz = fmaxf(fmaxf(__fsub_rn(glo[2], a.z), __fsub_rn(a.z, ghi[2])), 0.0f);
    const float d2 = __fmaf_rn(bz, bz, __fmaf_rn(by, by, __fmul_rn(bx, bx)));
    const float hm2 = __fmul_rn(hmax, hmax);
    const float hj2 = MODE == 0 ? 0.0f : e.v[E >= 2 ? 1 : 0].z;
    if (!(d2 < fmaxf(hm2, hj2))) return false;
    if (!p.pieces) return true;
    bool k = false;                               // per piece, as SphVisitor::keep
#pragma unroll
    for (int q = 0; q < OTOO_PIECES; q++) {
      const float4 lo = sm.pbox[2 * q], hi = sm.pbox[2 * q + 1];
      k = k || piece_d2(lo, hi, a.x, a.y, a.z) < fmaxf(__fmul_rn(lo.w, lo.w), hj2);
    }
    return k;
  }
  __device__ __forceinline__ void pad(float4* dst) {
    dst[0] = make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.0f);
    if (E >= 2) dst[1] = make_float4(1.0f, 0.0f, 1.0f, 0.0f);
    if (E >= 3) dst[2] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  }
  __device__ __forceinline__ void mark_self(uint32_t, uint32_t, int64_t, int) {}
  __device__ __forceinline__ float4* submit(float4*, int n, bool last) {
    if (lane_ == 0) sm.meta[buf] = WsMeta{(uint32_t)n, first | (last ? WS_LAST : 0u), group, 0u};
    first = 0;
    mbar_arrive(&sm.full[buf]);
    buf = (buf + 1) % OTOO_WS_NBUF;
    return acquire();
  }
  __device__ __forceinline__ void store(int64_t, int) {}
  __device__ __forceinline__ void finish() {
    if (lane_ == 0) sm.meta[buf] = WsMeta{0u, WS_EXIT, 0u, 0u};
    mbar_arrive(&sm.full[buf]);
  }
};

#ifndef OTOO_SPH_WS_WREG
#define OTOO_SPH_WS_WREG 72     // registers of a walker thread (T <= 4; at 48 the SPH walker spilled 190-300 B); the evaluators get 160 - this
#endif
template <int T, int MODE>
__global__ void __launch_bounds__(OTOO_WS_PAIRS * 64, T >= 8 ? 2 : 3) walk_sph_ws_kernel(const SphParams p) {
  typedef typename SphWalker<T, MODE>::Pair Pair;
  typedef SphVisitor<T, MODE> Eval;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  Pair* pairs = reinterpret_cast<Pair*>(smem_raw);
  uint32_t* masks = reinterpret_cast<uint32_t*>(smem_raw + OTOO_WS_PAIRS * sizeof(Pair));
  if (threadIdx.x < OTOO_WS_PAIRS) {
    Pair& s = pairs[threadIdx.x];
#pragma unroll
    for (int b = 0; b < OTOO_WS_NBUF; b++) { mbar_init(&s.full[b], 32); mbar_init(&s.empty[b], 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (warp >= OTOO_WS_PAIRS) {
    if (T >= 8) setmaxnreg_dec<80>(); else setmaxnreg_dec<OTOO_SPH_WS_WREG>();
    Pair& sm = pairs[warp - OTOO_WS_PAIRS];
    SphWalker<T, MODE> w(p, sm, lane);
    float4* list = w.acquire();
    walk_driver(p.c, w, list, sm.stk, lane, (int64_t)blockIdx.x * OTOO_WS_PAIRS + (warp - OTOO_WS_PAIRS));
    w.finish();
  } else {
    if (T >= 8) setmaxnreg_inc<176>(); else setmaxnreg_inc<160 - OTOO_SPH_WS_WREG>();
    Pair& sm = pairs[warp];
    Eval v(p);
    v.msk = masks + warp * (Eval::W * T * 32);
    v.lane_ = lane;
    uint32_t buf = 0, fparity = 0;
    for (;;) {
      mbar_wait(&sm.full[buf], (fparity >> buf) & 1u);
      fparity ^= 1u << buf;
      const WsMeta m = sm.meta[buf];
      if (m.flags & WS_EXIT) break;
      const int64_t g0 = (int64_t)m.group * p.c.gs;
      if (m.flags & WS_FIRST) v.load_group(g0, lane, nullptr);
      if (!p.c.walk_only && m.count) v.eval(sm.list[buf], (int)m.count);
      __syncwarp();
      if (m.flags & WS_LAST) v.store(g0, lane);
      mbar_arrive(&sm.empty[buf]);
      buf = (buf + 1) % OTOO_WS_NBUF;
    }
  }
}

template <int T, int MODE>
otoo_status launch_sph_ws2(otoo_ctx* ctx, const SphParams& p, cudaStream_t st) {
  const size_t smem = OTOO_WS_PAIRS * (sizeof(typename SphWalker<T, MODE>::Pair) + (size_t)SphVisitor<T, MODE>::W * T * 32 * sizeof(uint32_t));
  OTOO_CUDA(ctx, cudaFuncSetAttribute(walk_sph_ws_kernel<T, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int occ = 1;
  OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, walk_sph_ws_kernel<T, MODE>, OTOO_WS_PAIRS * 64, smem));
  if (occ < 1) occ = 1;
  int64_t grid = (int64_t)ctx->sm_count * occ;
  if (grid * OTOO_WS_PAIRS > p.c.ngroups) grid = cdiv(p.c.ngroups > 0 ? p.c.ngroups : 1, OTOO_WS_PAIRS);
  OTOO_EV(ctx, ctx->ev_walk[1], st);
  walk_sph_ws_kernel<T, MODE><<<(unsigned)grid, OTOO_WS_PAIRS * 64, smem, st>>>(p);
  OTOO_EV(ctx, ctx->ev_walk[2], st);
  ctx->ev_walk_valid = true;
  return OTOO_OK;
}
template <int MODE>
otoo_status launch_sph_ws(otoo_ctx* ctx, const SphParams& p, int G, cudaStream_t st) {
  switch (G) {
    case 4: case 8: case 16: case 32: return launch_sph_ws2<1, MODE>(ctx, p, st);
    case 64: return launch_sph_ws2<2, MODE>(ctx, p, st);
    case 128: return launch_sph_ws2<4, MODE>(ctx, p, st);
    case 256: return launch_sph_ws2<8, MODE>(ctx, p, st);
    default: return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  }
}

template <int MODE>
otoo_status launch_sph(otoo_ctx* ctx, const SphParams& p, int G, int grid, size_t smem, cudaStream_t st) {
  int occ = 1;
  const size_t smem0 = smem;
  void (*kern)(const SphParams) = nullptr;
#define OTOO_SPH_CASE(TT)                                                                                              \
  smem = smem0 + (size_t)OTOO_WALK_WARPS * (SphVisitor<TT, MODE>::W * TT * 32 * sizeof(uint32_t) + 2 * OTOO_PIECES * sizeof(float4));   /* + the mask words + the pieces' boxes */   \
  kern = sph_kernel_ptr<TT, MODE>(p.c.rec_mode);                                                                      \
  OTOO_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                   \
  OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, OTOO_WALK_WARPS * 32, smem));                \
  if (occ < 1) occ = 1;                                                                                                 \
  if (grid > ctx->sm_count * occ) grid = ctx->sm_count * occ;                                                          \
  OTOO_EV(ctx, ctx->ev_walk[1], st);                                                                                    \
  kern<<<grid, OTOO_WALK_WARPS * 32, smem, st>>>(p);                                                                    \
  OTOO_EV(ctx, ctx->ev_walk[2], st);                                                                                    \
  ctx->ev_walk_valid = true;
  switch (G) {
    case 4: case 8: case 16: case 32: OTOO_SPH_CASE(1) break;
    case 64: OTOO_SPH_CASE(2) break;
    case 128: OTOO_SPH_CASE(4) break;
    case 256: OTOO_SPH_CASE(8) break;
    default: return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  }
#undef OTOO_SPH_CASE
  return OTOO_OK;
}

// gather_stage: the density / stage-1 walks (they may record the opened leaves); the force walks may replay them
otoo_status sph_prepare(otoo_ctx* ctx, const float* d_h, int G, SphParams* p, int* grid, size_t* smem, cudaStream_t st, bool gather_stage) {
  if (G != 4 && G != 8 && G != 16 && G != 32 && G != 64 && G != 128 && G != 256)
    return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  OTOO_TRY(otoo_walk_prepare(ctx, G, &p->c, grid, smem, st));
  const unsigned nbN = (unsigned)cdiv(ctx->N, 256);
  // Eq. 5 radii depend on h: recomputed per call ("update the cell properties for SPH", L248 step 3) unless the
  // caller says h has not changed since the previous SPH call on this tree (option "sph_reuse_radii": stage 2 of a
  // step after stage 1, L252 steps 4 and 6)
  const bool radii_kept = ctx->sph_reuse && ctx->sph_radii_valid;
  if (!radii_kept) {
    ctx->rec_valid = false;                          // other h: other radii, other opened leaves
    gather_h_kernel<<<nbN, 256, 0, st>>>(d_h, ctx->val[0], ctx->N, ctx->sorted_h);
    OTOO_CUDA(ctx, cudaMemsetAsync(ctx->c_sph, 0, sizeof(float2) * ctx->N_cell, st));
    sph_radii_kernel<true><<<nbN, 256, 0, st>>>(ctx->spos, ctx->sorted_h, ctx->N, ctx->val[1], ctx->slot_nc, ctx->c_cm64, nullptr,   // (val[1], slot_nc: the build's
                                                reinterpret_cast<uint32_t*>(ctx->c_sph));                                        // per-slot levels and scanned level counts)
    ctx->launches += 2;
  }
  p->hs = ctx->sorted_h; p->aux = ctx->sorted_aux; p->svel = nullptr; p->svis = nullptr; p->c_sph = ctx->c_sph;
  p->rho = nullptr; p->nngb = nullptr; p->acc = nullptr;
  p->pieces = ctx->dist_kind == 2;
  ctx->sph_radii_valid = true;
  // option sph_reuse_walk: stage 2 of a step opens exactly the leaves stage 1 opened (same MAC, R15 / R26, same radii)
  if (ctx->sph_reuse_walk && !ctx->use_ws_sph) {
    const int64_t total_groups = cdiv(ctx->N, G);
    if (gather_stage) {
      bool have = total_groups <= ctx->rec_groups_cap;
      // (the records are an optimisation: beyond OTOO_REC_MAX_BYTES -- tens of millions of small groups -- or if the
      // allocation fails, the walks simply run in full)
      if (!have && (size_t)total_groups * OTOO_REC_CAP * sizeof(uint32_t) <= OTOO_REC_MAX_BYTES) {
        ctx->rec_valid = false;
        for (uint32_t** q : {&ctx->rec_cells, &ctx->rec_count, &ctx->rec_ntests}) { if (*q) cudaFree(*q); *q = nullptr; }
        ctx->rec_groups_cap = 0;
        if (cudaMalloc((void**)&ctx->rec_cells, sizeof(uint32_t) * (size_t)total_groups * OTOO_REC_CAP) == cudaSuccess &&
            cudaMalloc((void**)&ctx->rec_count, sizeof(uint32_t) * (size_t)total_groups) == cudaSuccess &&
            cudaMalloc((void**)&ctx->rec_ntests, sizeof(uint32_t) * (size_t)total_groups) == cudaSuccess) {
          ctx->rec_groups_cap = total_groups;
          have = true;
        } else {
          cudaGetLastError();
          for (uint32_t** q : {&ctx->rec_cells, &ctx->rec_count, &ctx->rec_ntests}) { if (*q) cudaFree(*q); *q = nullptr; }
        }
      }
      if (have) {
        OTOO_CUDA(ctx, cudaMemsetAsync(ctx->rec_count, 0xFF, sizeof(uint32_t) * (size_t)total_groups, st));   // nothing recorded yet
        p->c.rec_mode = 1;
        ctx->rec_valid = true; ctx->rec_G = G; ctx->rec_pieces = p->pieces; ctx->rec_gb = ctx->group_begin; ctx->rec_gc = ctx->group_count;
      } else ctx->rec_valid = false;
    } else if (radii_kept && ctx->rec_valid && ctx->rec_G == G && ctx->rec_pieces == p->pieces && ctx->rec_gb == ctx->group_begin &&
               ctx->rec_gc == ctx->group_count) {
      p->c.rec_mode = 2;
    }
    p->c.rec_cap = OTOO_REC_CAP; p->c.rec_cells = ctx->rec_cells; p->c.rec_count = ctx->rec_count; p->c.rec_ntests = ctx->rec_ntests;
  }
  return OTOO_OK;
}

}  // namespace

// fp64 b_max (L63) of every cell for the absolute-error MAC: the Eq. 5 pass with h = 0; leaves the maxima of the SQUARED
// distances as ordered bits in sph_acc[2c] (b_max = their square root: rb2_delta_kernel).  The fp32 SPH radii are recomputed by every SPH call anyway.
otoo_status otoo_bmax_impl(otoo_ctx* ctx, cudaStream_t st) {
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->sph_acc, 0, 2 * sizeof(unsigned long long) * ctx->N_cell, st));
  sph_radii_kernel<false><<<(unsigned)cdiv(ctx->N, 256), 256, 0, st>>>(ctx->spos, nullptr, ctx->N, ctx->val[1], ctx->slot_nc, ctx->c_cm64, ctx->sph_acc, nullptr);
  ctx->launches += 1;
  ctx->sph_radii_valid = false;
  return OTOO_OK;
}

otoo_status otoo_sph_density_impl(otoo_ctx* ctx, const float* d_h, int G, float* d_rho, uint32_t* d_nngb, cudaStream_t st) {
  SphParams p; int grid; size_t smem;
  OTOO_TRY(sph_prepare(ctx, d_h, G, &p, &grid, &smem, st, true));
  p.rho = d_rho; p.nngb = d_nngb;
  OTOO_CUDA(ctx, cudaMemsetAsync(d_rho, 0, 4 * (size_t)ctx->N, st));
  if (d_nngb) OTOO_CUDA(ctx, cudaMemsetAsync(d_nngb, 0, 4 * (size_t)ctx->N, st));
  if (ctx->use_ws_sph) OTOO_TRY(launch_sph_ws<0>(ctx, p, G, st)); else OTOO_TRY(launch_sph<0>(ctx, p, G, grid, smem, st));
  ctx->launches += 1;
  OTOO_CUDA(ctx, cudaGetLastError());
  ctx->walked = true;
  return OTOO_OK;
}

otoo_status otoo_sph_stage1_impl(otoo_ctx* ctx, const float* d_h, const float* d_vel, int G, float* d_rho, uint32_t* d_nngb,
                                 float* d_divrot, cudaStream_t st) {
  SphParams p; int grid; size_t smem;
  OTOO_TRY(sph_prepare(ctx, d_h, G, &p, &grid, &smem, st, true));
  gather_vel_kernel<<<(unsigned)cdiv(ctx->N, 256), 256, 0, st>>>(reinterpret_cast<const float4*>(d_vel), ctx->val[0], ctx->N, ctx->sorted_vel);
  p.svel = ctx->sorted_vel; p.rho = d_rho; p.nngb = d_nngb; p.acc = reinterpret_cast<float4*>(d_divrot);
  OTOO_CUDA(ctx, cudaMemsetAsync(d_rho, 0, 4 * (size_t)ctx->N, st));
  if (d_nngb) OTOO_CUDA(ctx, cudaMemsetAsync(d_nngb, 0, 4 * (size_t)ctx->N, st));
  OTOO_CUDA(ctx, cudaMemsetAsync(d_divrot, 0, 16 * (size_t)ctx->N, st));
  OTOO_TRY(launch_sph<3>(ctx, p, G, grid, smem, st));
  {
    const int64_t s0 = (int64_t)p.c.g_begin * G, s1 = s0 + p.c.ngroups * G < ctx->N ? s0 + p.c.ngroups * G : ctx->N;
    if (s1 > s0)
      divrot_finish_kernel<<<(unsigned)cdiv(s1 - s0, 256), 256, 0, st>>>(d_rho, ctx->val[0], s0, s1, reinterpret_cast<float4*>(d_divrot));
  }
  ctx->launches += 3;
  OTOO_CUDA(ctx, cudaGetLastError());
  ctx->walked = true;
  return OTOO_OK;
}

otoo_status otoo_sph_force_impl(otoo_ctx* ctx, const float* d_h, const float* d_rho, const float* d_P, const float* d_vel,
                                const float* d_visc, int G, float* d_acc, cudaStream_t st) {
  SphParams p; int grid; size_t smem;
  OTOO_TRY(sph_prepare(ctx, d_h, G, &p, &grid, &smem, st, false));
  gather_force_inputs_kernel<<<(unsigned)cdiv(ctx->N, 256), 256, 0, st>>>(d_h, d_rho, d_P, reinterpret_cast<const float4*>(d_vel),
                                                                          reinterpret_cast<const float4*>(d_visc), ctx->val[0],
                                                                          ctx->N, ctx->sorted_aux, ctx->sorted_vel, ctx->sorted_vis);
  if (d_visc) {
    p.svel = ctx->sorted_vel; p.svis = ctx->sorted_vis;
    OTOO_CUDA(ctx, cudaMemsetAsync(d_acc, 0, 16 * (size_t)ctx->N, st));
    p.acc = reinterpret_cast<float4*>(d_acc);
    OTOO_TRY(launch_sph<4>(ctx, p, G, grid, smem, st));
    ctx->launches += 2;
    OTOO_CUDA(ctx, cudaGetLastError());
    ctx->walked = true;
    return OTOO_OK;
  }
  OTOO_CUDA(ctx, cudaMemsetAsync(d_acc, 0, 16 * (size_t)ctx->N, st));
  p.acc = reinterpret_cast<float4*>(d_acc);
  if (d_vel) p.svel = ctx->sorted_vel;
  if (ctx->use_ws_sph) { if (d_vel) OTOO_TRY(launch_sph_ws<2>(ctx, p, G, st)); else OTOO_TRY(launch_sph_ws<1>(ctx, p, G, st)); }
  else { if (d_vel) OTOO_TRY(launch_sph<2>(ctx, p, G, grid, smem, st)); else OTOO_TRY(launch_sph<1>(ctx, p, G, grid, smem, st)); }
  ctx->launches += 2;
  OTOO_CUDA(ctx, cudaGetLastError());
  ctx->walked = true;
  return OTOO_OK;
}

// ---------------------------------------------------------------- adaptive smoothing length (reading R21)
namespace {
// settle the particles whose count is within the tolerance, count the others
// (both kernels run over the sorted slots [s0, s1) of the walked target groups: with a group range the other
// particles' h is left alone)
__global__ void __launch_bounds__(256) adapt_check_kernel(const uint32_t* __restrict__ nngb, const uint32_t* __restrict__ perm,
                                                          int64_t s0, int64_t s1, double n_target, double tol,
                                                          const float* __restrict__ h, float* __restrict__ lo, float* __restrict__ hi,
                                                          uint32_t* __restrict__ bad) {
  const int64_t s = s0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool unsettled = false;
  if (s < s1) {
    const uint32_t i = perm[s];
    if (lo[i] != hi[i]) {                                           // lo == hi marks a settled particle
      if (!(fabs((double)nngb[i] - n_target) > tol)) lo[i] = hi[i] = h[i];
      else unsettled = true;
    }
  }
  const unsigned m = __ballot_sync(0xFFFFFFFFu, unsettled);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(bad, (uint32_t)__popc(m));
}
// one update of the bracketed root search, same operations as the oracle
__global__ void __launch_bounds__(256) adapt_update_kernel(const uint32_t* __restrict__ nngb, const uint32_t* __restrict__ perm,
                                                           int64_t s0, int64_t s1, double n_target,
                                                           float* __restrict__ h, float* __restrict__ lo, float* __restrict__ hi) {
  const int64_t s = s0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= s1) return;
  const uint32_t i = perm[s];
  if (lo[i] == hi[i]) return;
  const double ni = (double)nngb[i];
  float l = lo[i], u = hi[i];
  const float hc = h[i];
  if (ni < n_target) l = hc; else u = hc;
  if (l > 0.0f && u < INFINITY) {
    const float mid = __fmul_rn(0.5f, __fadd_rn(l, u));
    if (mid == l || mid == u) l = u = hc;                            // the count steps over the band: settled
    else h[i] = mid;
  } else {
    double f = __dadd_rn(1.0, __ddiv_rn(__dsub_rn(n_target, ni), __dmul_rn(3.0, ni)));
    if (f < 0.7) f = 0.7;
    if (f > 1.3) f = 1.3;
    h[i] = __double2float_rn(__dmul_rn((double)hc, f));
  }
  lo[i] = l; hi[i] = u;
}
__global__ void __launch_bounds__(256) adapt_init_kernel(int64_t n, float* __restrict__ lo, float* __restrict__ hi) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { lo[i] = 0.0f; hi[i] = INFINITY; }
}
}  // namespace

otoo_status otoo_sph_adapt_h_impl(otoo_ctx* ctx, float* d_h, float n_target, float tol, int max_iter, int G, uint32_t* d_nngb,
                                  int* host_iters, cudaStream_t st) {
  const int64_t N = ctx->N;
  // scratch inside sorted_aux (4 floats per particle, unused by the density pass): lo, hi, rho, counts
  float* lo = reinterpret_cast<float*>(ctx->sorted_aux);
  float* hi = lo + N;
  float* rho = lo + 2 * N;
  uint32_t* cnt = reinterpret_cast<uint32_t*>(lo + 3 * N);
  uint32_t* bad = ctx->d_counters + 48;
  const unsigned nb = (unsigned)cdiv(N, 256);
  const int64_t total_groups = cdiv(N, G);
  const int64_t gb = ctx->group_begin, gc = ctx->group_count < 0 ? total_groups - gb : ctx->group_count;
  if (gb < 0 || gc < 0 || gb + gc > total_groups)
    return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_begin / group_count outside the groups of this group_size");
  const int64_t s0 = gb * G, s1 = (gb + gc) * G < N ? (gb + gc) * G : N;
  const unsigned nbr = (unsigned)cdiv(s1 > s0 ? s1 - s0 : 1, 256);
  adapt_init_kernel<<<nb, 256, 0, st>>>(N, lo, hi);
  int it = 0, launches = 1;
  for (;;) {
    OTOO_TRY(otoo_sph_density_impl(ctx, d_h, G, rho, cnt, st));
    launches += ctx->launches; ctx->launches = 0;
    OTOO_CUDA(ctx, cudaMemsetAsync(bad, 0, sizeof(uint32_t), st));
    adapt_check_kernel<<<nbr, 256, 0, st>>>(cnt, ctx->val[0], s0, s1, (double)n_target, (double)tol, d_h, lo, hi, bad);
    OTOO_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters + 48, bad, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    OTOO_CUDA(ctx, cudaStreamSynchronize(st));
    launches += 1;
    if (ctx->h_counters[48] == 0 || it >= max_iter) break;
    adapt_update_kernel<<<nbr, 256, 0, st>>>(cnt, ctx->val[0], s0, s1, (double)n_target, d_h, lo, hi);
    launches += 1;
    it++;
  }
  if (d_nngb) OTOO_CUDA(ctx, cudaMemcpyAsync(d_nngb, cnt, 4 * (size_t)N, cudaMemcpyDeviceToDevice, st));
  OTOO_CUDA(ctx, cudaGetLastError());
  ctx->launches = launches;
  if (host_iters) *host_iters = it;
  return OTOO_OK;
}
