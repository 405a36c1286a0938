// build.cu -- device-side tree construction (PAPER.md III-B steps 1-4, III-C), readings R1-R7.
// The paper builds the tree on the host and calls the pointer set-up "difficult to parallelize"
// (L135, L151); here every step is a data-parallel kernel over the sorted keys:
//   a cell (level l, first slot s) exists  <=>  s starts a level-l prefix range AND the level-(l-1)
//   range holding s has more than n_crit particles  <=>  cpl(s) < l <= min(D(s)+1, 21), where
//   cpl(s) = common prefix levels of key[s-1], key[s] and D(s) = max over windows of n_crit+1
//   consecutive slots containing s of their common prefix levels.
#include "common.cuh"
#include "keys.cuh"
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

namespace {

__device__ __forceinline__ unsigned f2ord(float f) {
  unsigned u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(unsigned u) {
  return __uint_as_float((u & 0x80000000u) ? (u & 0x7FFFFFFFu) : ~u);
}

// H1 (L121, L127; R1): per-axis min/max.  d_bbox[0..2] = min (ordered uint), [3..5] = max.
__global__ void __launch_bounds__(256) bbox_kernel(const float4* __restrict__ pos, int64_t n, unsigned* bbox) {
  float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    float4 p = pos[i];
    lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
    lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
    lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
  }
#pragma unroll
  for (int k = 0; k < 3; k++)
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      lo[k] = fminf(lo[k], __shfl_xor_sync(0xFFFFFFFFu, lo[k], o));
      hi[k] = fmaxf(hi[k], __shfl_xor_sync(0xFFFFFFFFu, hi[k], o));
    }
  __shared__ float sh[8][6];                          // one partial per warp, then 6 atomics per CTA
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { for (int k = 0; k < 3; k++) { sh[warp][k] = lo[k]; sh[warp][3 + k] = hi[k]; } }
  __syncthreads();
  if (threadIdx.x < 6) {
    float v = sh[0][threadIdx.x];
    for (int w = 1; w < 8; w++) v = threadIdx.x < 3 ? fminf(v, sh[w][threadIdx.x]) : fmaxf(v, sh[w][threadIdx.x]);
    if (threadIdx.x < 3) atomicMin(&bbox[threadIdx.x], f2ord(v)); else atomicMax(&bbox[threadIdx.x], f2ord(v));
  }
  // the last block to arrive derives the root cube: floats at bbox[8..12] = lo.xyz, S, scale (bbox[6] counts arrivals)
  __shared__ bool last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) last = atomicAdd(&bbox[6], 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last || threadIdx.x != 0) return;
  __threadfence();
  float* out = reinterpret_cast<float*>(bbox) + 8;
  float S = 0.0f;
  for (int k = 0; k < 3; k++) {
    float lo = ord2f(__ldcg(&bbox[k])), hi = ord2f(__ldcg(&bbox[3 + k]));
    float d = __fsub_rn(hi, lo);
    if (d > S) S = d;
    out[k] = lo;
  }
  if (!(S > 0.0f)) S = 1.0f;
  out[3] = S;
  out[4] = __fdiv_rn(2097152.0f, S);  // R2: IEEE division
  // ready for the next build (was three memsets per build): min = 0xFFFFFFFF, max = 0, arrival counter = 0
  for (int k = 0; k < 3; k++) { bbox[k] = 0xFFFFFFFFu; bbox[3 + k] = 0u; }
  bbox[6] = 0u;
}

// H4: positions into sorted order
__global__ void __launch_bounds__(256) gather4_kernel(const float4* __restrict__ src, const uint32_t* __restrict__ perm,
                                                      int64_t n, float4* __restrict__ dst) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) dst[s] = src[perm[s]];
}

__device__ __forceinline__ int cplev(uint64_t a, uint64_t b) {  // common leading levels, 0..21
  uint64_t x = a ^ b;
  if (x == 0) return OTOO_MAXLEV;
  return 20 - (63 - __clzll((long long)x)) / 3;
}
// H5a: the levels of the cells that start at each sorted slot, and the cell counts per level -- of the whole system
// (level_count) and of every block of 256 slots (blk_lc[l * gridDim.x + block], level-major: one exclusive scan of
// that array gives every block the canonical index of its first cell of each level, see place_cells_kernel).
//   info[s] = (cpl+1) | LL << 8
// A level-l range starting at s is a cell iff some window of n_crit+1 slots containing s shares l-1 levels:
// c[t] = cplev(key[t], key[t + n_crit]) is computed once per t into shared memory (every thread of the
// plain form recomputed its n_crit+1 windows from global memory: 480 GB/s at 32 M particles), the per-level
// counts are warp-aggregated (one ballot per level instead of contended shared-memory atomics).
#define OTOO_SLOT_NCRIT_MAX 256
#ifndef OTOO_GATHER_L2HINT
#define OTOO_GATHER_L2HINT ".L2::64B"        // a miss fetches 64 B instead of the default 128 B (gather + levels 0.86 -> 0.81 ms at 32 M)
#endif
// H4 rides along: the block's 256 random 16-byte reads of the gather (HBM-latency-bound, 3.7 x its algorithmic bytes
// for an unordered input) are issued first and stored last, so they are in flight while the block does its
// issue-bound level arithmetic (as kernels of their own: 0.72 + 0.46 ms at 32 M particles).
__global__ void __launch_bounds__(256) slot_cells_kernel(const uint64_t* __restrict__ key, int64_t n, int n_crit,
                                                         uint32_t* __restrict__ blk_lc, uint32_t* __restrict__ info,
                                                         const float4* __restrict__ pos,
                                                         const uint32_t* __restrict__ perm, float4* __restrict__ spos) {
  __shared__ uint32_t lc[OTOO_NLEV + 1];
  __shared__ signed char cwa[256 + OTOO_SLOT_NCRIT_MAX], cwb[256 + OTOO_SLOT_NCRIT_MAX];
  const int64_t s0 = (int64_t)blockIdx.x * 256;
  float4 pv = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  if (s0 + threadIdx.x < n) {
    const float4* src = pos + perm[s0 + threadIdx.x];
    asm volatile("ld.global.nc.L1::no_allocate" OTOO_GATHER_L2HINT ".v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(pv.x), "=f"(pv.y), "=f"(pv.z), "=f"(pv.w) : "l"(src));
  }
  const int m = 256 + n_crit;                       // window starts t = s0 - n_crit + i, i < m
  if (threadIdx.x <= OTOO_NLEV) lc[threadIdx.x] = 0;
  for (int i = threadIdx.x; i < m; i += 256) {
    const int64_t t = s0 - n_crit + i;
    cwa[i] = (t >= 0 && t <= n - n_crit - 1) ? (signed char)cplev(key[t], key[t + n_crit]) : (signed char)-1;
  }
  __syncthreads();
  // D(s) = max of the n_crit + 1 consecutive values cw[tid .. tid + n_crit]: doubling (m_k[i] = max of 2^k values from
  // i) up to the largest power of two <= n_crit + 1, then two overlapping spans cover the window
  const int w = n_crit + 1;
  signed char *src = cwa, *dst = cwb;
  int span = 1;
  while (2 * span <= w) {
    for (int i = threadIdx.x; i < m; i += 256) {
      const signed char a = src[i], b = i + span < m ? src[i + span] : (signed char)-1;
      dst[i] = a > b ? a : b;
    }
    __syncthreads();
    signed char* tmp = src; src = dst; dst = tmp;
    span *= 2;
  }
  const int64_t s = s0 + threadIdx.x;
  int lo = OTOO_NLEV, LL = -1;   // empty level range for threads past the end
  if (s < n) {
    const int cpl = (s == 0) ? -1 : cplev(key[s - 1], key[s]);
    const signed char a = src[threadIdx.x], b = src[threadIdx.x + w - span];
    const int D = a > b ? a : b;
    LL = D + 1 > OTOO_MAXLEV ? OTOO_MAXLEV : D + 1;
    lo = cpl + 1;
    info[s] = (uint32_t)lo | ((uint32_t)LL << 8);
  }
  // per-level counts, warp-aggregated: only the levels some lane of the warp starts a cell at (a few around the
  // local leaf level, not all 22)
  const bool has = lo <= LL;
  const int wlo = __reduce_min_sync(0xFFFFFFFFu, has ? lo : OTOO_NLEV), whi = __reduce_max_sync(0xFFFFFFFFu, has ? LL : -1);
  for (int l = wlo; l <= whi; l++) {
    const unsigned b = __ballot_sync(0xFFFFFFFFu, lo <= l && l <= LL);
    if (b && (threadIdx.x & 31) == 0) atomicAdd(&lc[l], (uint32_t)__popc(b));
  }
  const unsigned hb = __ballot_sync(0xFFFFFFFFu, has);  // row OTOO_NLEV: slots that start cells = leaves (one per such slot)
  if (hb && (threadIdx.x & 31) == 0) atomicAdd(&lc[OTOO_NLEV], (uint32_t)__popc(hb));
  __syncthreads();
  // (no system-wide counters: the level totals and the leaf count are read off the scan of these rows; one global atomic
  // per block and level on 22 addresses cost more than the rest of the kernel)
  if (threadIdx.x <= OTOO_NLEV) blk_lc[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = lc[threadIdx.x];
  if (s < n) spos[s] = pv;                            // H4: the position in sorted order
}
// the same for n_crit > OTOO_SLOT_NCRIT_MAX (every thread scans its own windows)
__global__ void __launch_bounds__(256) slot_cells_wide_kernel(const uint64_t* __restrict__ key, int64_t n, int n_crit,
                                                              uint32_t* __restrict__ blk_lc, uint32_t* __restrict__ info) {
  __shared__ uint32_t lc[OTOO_NLEV + 1];
  if (threadIdx.x <= OTOO_NLEV) lc[threadIdx.x] = 0;
  __syncthreads();
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) {
    int cpl = (s == 0) ? -1 : cplev(key[s - 1], key[s]);
    int D = -1;
    int64_t tlo = s - n_crit; if (tlo < 0) tlo = 0;
    int64_t thi = n - n_crit - 1; if (thi > s) thi = s;
    for (int64_t t = tlo; t <= thi; t++) { int c = cplev(key[t], key[t + n_crit]); if (c > D) D = c; }
    int LL = D + 1 > OTOO_MAXLEV ? OTOO_MAXLEV : D + 1;
    info[s] = (uint32_t)(cpl + 1) | ((uint32_t)LL << 8);
    for (int l = cpl + 1; l <= LL; l++) atomicAdd(&lc[l], 1u);
    if (cpl + 1 <= LL) atomicAdd(&lc[OTOO_NLEV], 1u);
  }
  __syncthreads();
  if (threadIdx.x <= OTOO_NLEV) blk_lc[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = lc[threadIdx.x];
}
// H5b: every cell written straight at its canonical index, leaves complete.  Canonical order = (level, first slot):
// the index of a level-l cell starting at slot s is (cells of lower levels) + (level-l cells starting before s) -- the
// exclusive scan of the level-major per-block counts gives the first part plus the blocks before this one (blk_off), a
// ballot per level the rank inside the block.  Of the cells that start at slot s (levels lo .. LL) the one at LL is a
// leaf, the others are internal and their first child is the cell one level down at the same slot (L135: "slicing the
// keys"; R5).  A leaf ends at the next slot that starts a range of its level or a coarser one (lo <= LL): found in the
// block's shared-memory window of lo values (a leaf holds <= n_crit slots unless it sits at level 21), by a search on
// the key prefix beyond it.  Counts and child counts of the internal cells come bottom-up (moments_all_kernel).
// (Before: a kernel of its own found every cell's count and children by binary searches on the keys and the first slots.)
#define OTOO_PLACE_WIN 64
struct CellOut {
  uint32_t* c_first; uint32_t* c_count; uint32_t* c_child_first; uint8_t* c_level; uint8_t* c_child_count; cellb_t* cell_b;
};
__global__ void __launch_bounds__(256) place_cells_kernel(const uint32_t* __restrict__ info, const uint64_t* __restrict__ key, int64_t n,
                                                          const uint32_t* __restrict__ blk_off, const CellOut o) {
  __shared__ uint32_t wc[8][OTOO_NLEV];          // level-l cells the warp starts, then the canonical index of its first one
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane < OTOO_NLEV) wc[warp][lane] = 0;      // (each warp its own row: no block barrier before the ballots)
  __syncwarp();
  // (fetched now, used after two block barriers: the load's latency was a fifth of the kernel's stall samples)
  const uint32_t my_off = threadIdx.x < OTOO_NLEV ? blk_off[(size_t)threadIdx.x * gridDim.x + blockIdx.x] : 0u;
  const int64_t s0 = (int64_t)blockIdx.x * 256, s = s0 + threadIdx.x;
  int lo = OTOO_NLEV, LL = -1;
  if (s < n) { const uint32_t inf = info[s]; lo = (int)(inf & 0xFF); LL = (int)(inf >> 8); }
  const int lo_next = s + 32 < n ? (int)(info[s + 32] & 0xFF) : 0;      // lo of the slot 32 further on (0 past the end: ends every range)
  const bool has = lo <= LL;
  const int wlo = __reduce_min_sync(0xFFFFFFFFu, has ? lo : OTOO_NLEV), whi = __reduce_max_sync(0xFFFFFFFFu, has ? LL : -1);
  // the leaf's particle count = distance to the next slot that starts a range of the leaf's level or a coarser one:
  // per level a ballot over the warp's 32 slots and one over the 32 slots after them
  const int lo_term = s < n ? lo : 0;                                             // (slots past the end end every range)
  uint32_t count = 0;
  for (int l = wlo; l <= whi; l++) {
    const unsigned b = __ballot_sync(0xFFFFFFFFu, lo <= l && l <= LL);
    const unsigned m = __ballot_sync(0xFFFFFFFFu, lo_term <= l), m2 = __ballot_sync(0xFFFFFFFFu, lo_next <= l);
    if (lane == 0) wc[warp][l] = (uint32_t)__popc(b);
    if (l == LL) {
      const unsigned long long mm = (((unsigned long long)m2 << 32) | m) >> (lane + 1);
      count = mm ? (uint32_t)__ffsll((long long)mm) : 0u;           // 0: not within the next 63 - lane slots
    }
  }
  __syncthreads();
  if (threadIdx.x < OTOO_NLEV) {
    uint32_t run = my_off;
#pragma unroll
    for (int w = 0; w < 8; w++) { const uint32_t c = wc[w][threadIdx.x]; wc[w][threadIdx.x] = run; run += c; }
  }
  __syncthreads();
  if (has && (count == 0u || LL == 0)) {
    if (LL == 0) count = (uint32_t)n;
    else {
      // not within the 63 - lane slots the ballots cover (a leaf of more than 32 particles: n_crit > 32 or level 21):
      // the next OTOO_PLACE_WIN slots one by one, then a search on the key prefix
      int64_t j = s + 1;
      const int64_t jend = s + OTOO_PLACE_WIN < n ? s + OTOO_PLACE_WIN : n;
      while (j < jend && (int)(info[j] & 0xFF) > LL) j++;
      if (j < jend || j == n) count = (uint32_t)(j - s);
      else {                                       // beyond the window: gallop, then bisect for the end of the prefix range
        const int sh = 3 * (OTOO_MAXLEV - LL);
        const uint64_t prefix = key[s] >> sh;
        uint64_t step = 1, a = (uint64_t)s;        // key[a] has the prefix
        while (s + step < (uint64_t)n && (key[s + step] >> sh) == prefix) { a = s + step; step <<= 1; }
        uint64_t hi = s + step < (uint64_t)n ? s + step : (uint64_t)n;  // key[hi] lacks it (or hi == n)
        while (a + 1 < hi) { const uint64_t mid = (a + hi) >> 1; if ((key[mid] >> sh) == prefix) a = mid; else hi = mid; }
        count = (uint32_t)(hi - s);
      }
    }
  }
  unsigned lt;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(lt));
  uint32_t below = 0;                              // canonical index of this slot's cell one level down
  for (int l = whi; l >= wlo; l--) {
    const bool mine = lo <= l && l <= LL;
    const unsigned b = __ballot_sync(0xFFFFFFFFu, mine);
    if (mine) {
      const uint32_t c = wc[warp][l] + (uint32_t)__popc(b & lt);
      o.c_first[c] = (uint32_t)s;
      o.c_level[c] = (uint8_t)(l | (l > lo ? 0x80 : 0));   // bit 7: the parent starts at this slot too = first of its siblings
      if (l == LL) {
        o.c_count[c] = count; o.c_child_first[c] = 0u; o.c_child_count[c] = 0;
        o.cell_b[c] = make_uint4(0u, (uint32_t)s, count, 1u | ((uint32_t)l << 8));
      } else {
        o.c_child_first[c] = below;                                    // internal (>= 1): count and children bottom-up
      }
      below = c;
    }
  }
}

struct LevelOff { uint32_t v[OTOO_NLEV + 1]; };
#ifndef OTOO_MOMENTS_WIDE
#define OTOO_MOMENTS_WIDE (4u << 20)      // cells in the widest level from which the bottom-up pass runs 4 CTAs per SM
#endif

// H6 (L155; R6, R7): one level of the bottom-up pass; fp64, fixed summation order.
struct MomentArgs {
  const float4* spos; const uint64_t* key; const uint32_t* c_first; uint32_t* c_count;
  const uint32_t* c_child_first; uint8_t* c_child_count; const unsigned* bbox;
  double* MP; double* cm64; float4* cell_cm; double* c_s; double* c_B2;
  int hilbert;
  const uint8_t* c_level; cellb_t* cell_b;        // H5c for the internal cells (moments_all_kernel only)
  int do_rb2; float theta;                         // R7 for the theta of the last gravity call (moments_all_kernel only)
  uint32_t* walk_ws; uint32_t* walk_seq;           // the walk's control block and pool sequence numbers to reset (or null)
};
// level_end = canonical index one past the last cell of level + 1 (the children's level)
__device__ __forceinline__ void moments_cell(uint32_t c, int level, uint32_t level_end, const MomentArgs& a) {
  const float4* __restrict__ spos = a.spos; const uint64_t* __restrict__ key = a.key;
  const uint32_t* __restrict__ c_first = a.c_first; uint32_t* c_count = a.c_count;
  const uint32_t* __restrict__ c_child_first = a.c_child_first; uint8_t* c_child_count = a.c_child_count;
  const unsigned* __restrict__ bbox = a.bbox;
  double* MP = a.MP; double* cm64 = a.cm64; float4* cell_cm = a.cell_cm; double* c_s = a.c_s;
  const uint32_t first = c_first[c], ch = c_child_first[c];   // ch == 0: a leaf (the root's first child is cell 1)
  uint32_t count = c_count[c];                                 // (of a leaf; an internal cell's is found below)
  int nch = 0;
  double M = 0.0, Px = 0.0, Py = 0.0, Pz = 0.0;
  const float* r = reinterpret_cast<const float*>(bbox) + 8;
  // integer cell coordinates = top `level` bits of the quantised coordinates (R2) of any particle of the cell
  uint32_t qx = 0, qy = 0, qz = 0;
  if (ch == 0u) {
    for (uint32_t s0 = first; s0 < first + count; s0 += 8) {   // 8 loads in flight, sums in slot order (R6)
      float4 p[8];
      const uint32_t nv = first + count - s0 < 8u ? first + count - s0 : 8u;
#pragma unroll
      for (int j = 0; j < 8; j++) if ((uint32_t)j < nv) p[j] = spos[s0 + j];
      if (s0 == first && level > 0) {                          // from the first particle itself (no read of its key)
        const float scale = r[4];
        qx = quant(p[0].x, r[0], scale) >> (OTOO_MAXLEV - level); qy = quant(p[0].y, r[1], scale) >> (OTOO_MAXLEV - level);
        qz = quant(p[0].z, r[2], scale) >> (OTOO_MAXLEV - level);
      }
#pragma unroll
      for (int j = 0; j < 8; j++) if ((uint32_t)j < nv) {
        double m = (double)p[j].w;
        M = __dadd_rn(M, m);
        Px = __dadd_rn(Px, __dmul_rn(m, (double)p[j].x));
        Py = __dadd_rn(Py, __dmul_rn(m, (double)p[j].y));
        Pz = __dadd_rn(Pz, __dmul_rn(m, (double)p[j].z));
      }
    }
  } else {
    // H5c for an internal cell: its children are the cell one level down at its own first slot and the cells after
    // that one (canonical order = octant order) whose first slot starts a range of the children's level but not of
    // this cell's (bit 7 of c_level clear: not the first child of another parent); its particles are theirs
    unsigned sib = 1u;                                 // bit k: cell ch + k exists and is not the first child of the next parent
#pragma unroll
    for (int k = 1; k < 8; k++) if (ch + k < level_end && !(a.c_level[ch + k] & 0x80)) sib |= 1u << k;
    nch = __ffs(~sib) - 1;                             // the run of siblings from ch
    count = 0;
    for (int k = 0; k < nch; k++) {
      const double* q = MP + 4 * (size_t)(ch + k);
      M = __dadd_rn(M, q[0]); Px = __dadd_rn(Px, q[1]); Py = __dadd_rn(Py, q[2]); Pz = __dadd_rn(Pz, q[3]);
      count += __ldcg(&c_count[ch + k]);
    }
    c_count[c] = count; c_child_count[c] = (uint8_t)nch;
    a.cell_b[c] = make_uint4(0u, ch, (uint32_t)nch, (uint32_t)level << 8);
    if (level > 0) {                                   // (internal cells are few: from the key of the first particle)
      const uint64_t k0 = key[first];
      qx = compact3(k0 >> 2); qy = compact3(k0 >> 1); qz = compact3(k0);
      if (a.hilbert) hilbert_transpose_to_axes(qx, qy, qz);
      qx >>= OTOO_MAXLEV - level; qy >>= OTOO_MAXLEV - level; qz >>= OTOO_MAXLEV - level;
    }
  }
  double* o = MP + 4 * (size_t)c;
  o[0] = M; o[1] = Px; o[2] = Py; o[3] = Pz;
  double l = ldexp((double)r[3], -level);
  double g[3];
  g[0] = __dadd_rn((double)r[0], __dmul_rn((double)qx + 0.5, l));
  g[1] = __dadd_rn((double)r[1], __dmul_rn((double)qy + 0.5, l));
  g[2] = __dadd_rn((double)r[2], __dmul_rn((double)qz + 0.5, l));
  double cx, cy, cz;
  if (M != 0.0) { cx = __ddiv_rn(Px, M); cy = __ddiv_rn(Py, M); cz = __ddiv_rn(Pz, M); }
  else { cx = g[0]; cy = g[1]; cz = g[2]; }
  cm64[3 * (size_t)c] = cx; cm64[3 * (size_t)c + 1] = cy; cm64[3 * (size_t)c + 2] = cz;
  cell_cm[c] = make_float4(__double2float_rn(cx), __double2float_rn(cy), __double2float_rn(cz), __double2float_rn(M));
  double dx = __dsub_rn(cx, g[0]), dy = __dsub_rn(cy, g[1]), dz = __dsub_rn(cz, g[2]);
  const double sd = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
  c_s[c] = sd;
  if (a.do_rb2) {
    // R7, the operations of rb2_kernel (gravity.cu): r_b = l/theta + s in fp64, rb^2 rounded once to fp32
    float rb2 = INFINITY;
    if (a.theta > 0.0f) { const double rb = __dadd_rn(__ddiv_rn(l, (double)a.theta), sd); rb2 = __double2float_rn(__dmul_rn(rb, rb)); }
    reinterpret_cast<uint32_t*>(a.cell_b + c)[0] = __float_as_uint(rb2);
  }
}
// the whole bottom-up pass in ONE cooperative launch: every level deepest first, a grid-wide barrier
// between levels (per-level launches of the sparse top and bottom levels were pure launch latency)
// Levels 0 .. top are narrow (the top of the tree: 1, 8, 64, ... cells): one CTA finishes them with block barriers
// instead of grid barriers.
// MINB = CTAs per SM the register count must allow: 2 (128 registers) up to a few million cells per level, 4 (64 registers)
// beyond -- twice the loads in flight for the wide leaf levels (0.75 -> 0.69 ms at 32 M particles), but twice the blocks in
// every grid barrier (10-30 % slower at 1-8 M particles)
template <int MINB>
__global__ void __launch_bounds__(256, MINB) moments_all_kernel(const LevelOff off, const int depth, const int top, const MomentArgs a) {
  cg::grid_group grid = cg::this_grid();
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
  if (a.walk_seq) {                                  // the next walk finds its control block and pool reset (was part of the r_b kernel)
    for (uint32_t i = tid; i < OTOO_POOL_SLOTS; i += nthr) a.walk_seq[i] = i;
    if (tid < 128) a.walk_ws[tid] = 0u;              // WalkShared: queue, head, tail, outstanding, one 128-byte line each
  }
  for (int l = depth; l > top; l--) {
    for (uint32_t c = off.v[l] + tid; c < off.v[l + 1]; c += nthr) moments_cell(c, l, l < OTOO_MAXLEV ? off.v[l + 2] : off.v[l + 1], a);
    grid.sync();
  }
  if (blockIdx.x != 0) return;
  for (int l = top < depth ? top : depth; l >= 0; l--) {
    for (uint32_t c = off.v[l] + threadIdx.x; c < off.v[l + 1]; c += blockDim.x) moments_cell(c, l, l < OTOO_MAXLEV ? off.v[l + 2] : off.v[l + 1], a);
    __syncthreads();
  }
}

template <typename T>
otoo_status grow(otoo_ctx* ctx, T** p, size_t count) {
  if (*p) cudaFree(*p);
  *p = nullptr;
  OTOO_CUDA(ctx, cudaMalloc((void**)p, count * sizeof(T)));
  return OTOO_OK;
}

otoo_status ensure_cells(otoo_ctx* ctx, int64_t ncell) {
  if (ncell <= ctx->cellCap) return OTOO_OK;
  int64_t cap = ncell + ncell / 8 + 1024;
  ctx->cellCap = 0;
  OTOO_TRY(grow(ctx, &ctx->cell_cm, cap));
  OTOO_TRY(grow(ctx, &ctx->cell_b, cap));
  OTOO_TRY(grow(ctx, &ctx->c_first, cap));
  OTOO_TRY(grow(ctx, &ctx->c_count, cap));
  OTOO_TRY(grow(ctx, &ctx->c_child_first, cap));
  OTOO_TRY(grow(ctx, &ctx->c_level, cap));
  OTOO_TRY(grow(ctx, &ctx->c_child_count, cap));
  OTOO_TRY(grow(ctx, &ctx->c_MP, 4 * cap));
  OTOO_TRY(grow(ctx, &ctx->c_cm64, 3 * cap));
  OTOO_TRY(grow(ctx, &ctx->c_s, cap));
  OTOO_TRY(grow(ctx, &ctx->c_B2, cap));
  OTOO_TRY(grow(ctx, &ctx->c_sph, cap));
  OTOO_TRY(grow(ctx, &ctx->sph_acc, 2 * cap));
  ctx->cellCap = cap;
  return OTOO_OK;
}


// PAPER Eq. 2 for the absolute-error MAC, computed on demand (otoo_gravity_delta) after the moments pass
__device__ __forceinline__ void b2_cell(uint32_t c, const MomentArgs& a) {
  const float4* __restrict__ spos = a.spos;
  const uint32_t first = a.c_first[c], count = a.c_count[c];
  const int nch = a.c_child_count[c];
  const uint32_t* __restrict__ c_child_first = a.c_child_first;
  const double* cm64 = a.cm64; const double* MP = a.MP;
  const double cx = cm64[3 * (size_t)c], cy = cm64[3 * (size_t)c + 1], cz = cm64[3 * (size_t)c + 2];
  // PAPER Eq. 2, B2 = sum m |r_CM - r|^2, accumulated bottom-up in a fixed order (R19): leaf: its particles in
  // slot order; internal: children in octant order, B2 += B2_child, then B2 += M_child |CM_child - CM|^2
  double b2 = 0.0;
  if (nch == 0) {
    for (uint32_t s0 = first; s0 < first + count; s0 += 8) {
      float4 p[8];
      const uint32_t nv = first + count - s0 < 8u ? first + count - s0 : 8u;
#pragma unroll
      for (int j = 0; j < 8; j++) if ((uint32_t)j < nv) p[j] = spos[s0 + j];
#pragma unroll
      for (int j = 0; j < 8; j++) if ((uint32_t)j < nv) {
        const double ex = __dsub_rn((double)p[j].x, cx), ey = __dsub_rn((double)p[j].y, cy), ez = __dsub_rn((double)p[j].z, cz);
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
        b2 = __dadd_rn(b2, __dmul_rn((double)p[j].w, r2));
      }
    }
  } else {
    const uint32_t ch = c_child_first[c];
    for (int k = 0; k < nch; k++) {
      const double* q = cm64 + 3 * (size_t)(ch + k);
      const double ex = __dsub_rn(q[0], cx), ey = __dsub_rn(q[1], cy), ez = __dsub_rn(q[2], cz);
      const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
      b2 = __dadd_rn(b2, a.c_B2[ch + k]);
      b2 = __dadd_rn(b2, __dmul_rn(MP[4 * (size_t)(ch + k)], r2));
    }
  }
  a.c_B2[c] = b2;
}
__global__ void __launch_bounds__(256) b2_all_kernel(const LevelOff off, const int depth, const MomentArgs a) {
  cg::grid_group grid = cg::this_grid();
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
  for (int l = depth; l >= 0; l--) {
    for (uint32_t c = off.v[l] + tid; c < off.v[l + 1]; c += nthr) b2_cell(c, a);
    if (l > 0) grid.sync();
  }
}
}  // namespace

otoo_status otoo_build_impl(otoo_ctx* ctx, const float* d_pos_mass, int64_t N, int n_crit, cudaStream_t st) {
  ctx->built = false; ctx->walked = false; ctx->sph_radii_valid = false; ctx->b2_valid = false;
  ctx->rb2_valid = false; ctx->walk_reset_valid = false; ctx->rec_valid = false;
  const float4* pos = reinterpret_cast<const float4*>(d_pos_mass);
  unsigned* bbox = reinterpret_cast<unsigned*>(ctx->d_bbox);
  const unsigned nbN = (unsigned)cdiv(N, 256);
  ctx->ev_build_valid = false;
  OTOO_EV(ctx, ctx->ev_build[0], st);
  // H1
  // (the extrema and the arrival counter in d_bbox start from their initial values: set at otoo_create and put back by
  // the last block of every bbox_kernel)
  int gb = ctx->sm_count * 4; if ((int64_t)gb > (int64_t)nbN) gb = (int)nbN;
  bbox_kernel<<<gb, 256, 0, st>>>(pos, N, bbox);
  ctx->launches += 1;
  OTOO_EV(ctx, ctx->ev_build[1], st);
  // H2, H3, H4
  // keys and ids, and in the same read the eight digit histograms of the sort (otoo_keys_and_hist, sort.cu)
  OTOO_TRY(otoo_keys_and_hist(ctx, d_pos_mass, N, st));
  ctx->launches += 1;
  OTOO_EV(ctx, ctx->ev_build[2], st);
  int res = 0;
  OTOO_TRY(otoo_sort_pairs(ctx, ctx->key, ctx->val, N, 0, 64, st, &res, true));
  if (res != 0) return otoo_fail(ctx, OTOO_ERR_CUDA, "internal: sort result buffer");
  OTOO_EV(ctx, ctx->ev_build[3], st);
  // H4 + H5a: positions into sorted order and, in the same kernel, the levels of the cells that start at each slot
  uint32_t* info = ctx->val[1];
  uint32_t* blk_lc = ctx->slot_nc;                 // OTOO_NLEV x nbN per-block level counts, then their exclusive scan
  if (n_crit <= OTOO_SLOT_NCRIT_MAX)
    slot_cells_kernel<<<nbN, 256, 0, st>>>(ctx->key[0], N, n_crit, blk_lc, info, pos, ctx->val[0], ctx->spos);
  else {
    gather4_kernel<<<nbN, 256, 0, st>>>(pos, ctx->val[0], N, ctx->spos);
    slot_cells_wide_kernel<<<nbN, 256, 0, st>>>(ctx->key[0], N, n_crit, blk_lc, info);
    ctx->launches += 1;
  }
  ctx->launches += 1;
  OTOO_EV(ctx, ctx->ev_build[4], st);
  // one exclusive scan of the OTOO_NLEV + 1 rows: the canonical index of every block's first cell of each level, and at
  // the start of row l the number of cells of the levels below l (row OTOO_NLEV starts at N_cell; the rest is the leaves)
  OTOO_TRY(otoo_exclusive_scan_u32(ctx, blk_lc, (int64_t)(OTOO_NLEV + 1) * nbN, ctx->d_counters + 40, st));
  OTOO_CUDA(ctx, cudaMemcpy2DAsync(ctx->h_counters, sizeof(uint32_t), blk_lc, (size_t)nbN * sizeof(uint32_t), sizeof(uint32_t), OTOO_NLEV + 1,
                                   cudaMemcpyDeviceToHost, st));
  OTOO_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters + 40, ctx->d_counters + 40, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
  OTOO_CUDA(ctx, cudaMemcpyAsync(ctx->h_root, ctx->d_bbox + 8, 5 * sizeof(float), cudaMemcpyDeviceToHost, st));
  OTOO_CUDA(ctx, cudaStreamSynchronize(st));
  LevelOff off;
  int depth = 0;
  for (int l = 0; l <= OTOO_NLEV; l++) off.v[l] = ctx->h_counters[l];
  for (int l = 0; l < OTOO_NLEV; l++) if (off.v[l + 1] > off.v[l]) depth = l;
  const int64_t ncell = off.v[OTOO_NLEV];
  if (ncell < 1 || (int64_t)ctx->h_counters[40] < ncell || off.v[0] != 0u)
    return otoo_fail(ctx, OTOO_ERR_CUDA, "internal: level offsets disagree with the cell count");
  ctx->h_counters[32] = ctx->h_counters[40] - (uint32_t)ncell;          // N_leaf (otoo_tree_info)
  OTOO_TRY(ensure_cells(ctx, ncell));
  // H5b: cells in canonical order (level, first slot), leaves complete
  const CellOut co{ctx->c_first, ctx->c_count, ctx->c_child_first, ctx->c_level, ctx->c_child_count, ctx->cell_b};
  place_cells_kernel<<<nbN, 256, 0, st>>>(info, ctx->key[0], N, blk_lc, co);
  ctx->launches += 1;
  OTOO_EV(ctx, ctx->ev_build[5], st);
  // H5c of the internal cells + H6, deepest level first
  const MomentArgs ma{ctx->spos, ctx->key[0], ctx->c_first, ctx->c_count, ctx->c_child_first, ctx->c_child_count,
                      bbox, ctx->c_MP, ctx->c_cm64, ctx->cell_cm, ctx->c_s, ctx->c_B2, ctx->key_order, ctx->c_level, ctx->cell_b,
                      ctx->spec_theta_set ? 1 : 0, ctx->spec_theta, (uint32_t*)ctx->walk_shared, (uint32_t*)ctx->pool_seq};
  {
    uint32_t widest = 1;
    for (int l = 0; l <= depth; l++) if (off.v[l + 1] - off.v[l] > widest) widest = off.v[l + 1] - off.v[l];
    const void* kern = widest >= OTOO_MOMENTS_WIDE ? (const void*)moments_all_kernel<4> : (const void*)moments_all_kernel<2>;
    int occ = 1;
    OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 256, 0));
    if (occ > 4) occ = 4;
    int64_t grid = (int64_t)ctx->sm_count * (occ < 1 ? 1 : occ);
    if (grid > cdiv(widest, 256)) grid = cdiv(widest, 256);
    int depth_arg = depth, top = -1;
    while (top + 1 <= depth && off.v[top + 2] - off.v[top + 1] <= 256u) top++;       // levels 0 .. top hold <= 256 cells each (one per thread)
    void* args[] = {(void*)&off, (void*)&depth_arg, (void*)&top, (void*)&ma};
    OTOO_CUDA(ctx, cudaLaunchCooperativeKernel(kern, dim3((unsigned)grid), dim3(256), args, 0, st));
    ctx->launches += 1;
  }
  OTOO_EV(ctx, ctx->ev_build[6], st);
  ctx->ev_build_valid = true;
  if (ctx->spec_theta_set) { ctx->rb2_valid = true; ctx->rb2_theta = ctx->spec_theta; }
  ctx->walk_reset_valid = ctx->pool_seq != nullptr;
  OTOO_CUDA(ctx, cudaGetLastError());
  ctx->N = N; ctx->N_cell = ncell; ctx->n_crit = n_crit; ctx->depth = depth;
  for (int k = 0; k < 3; k++) ctx->lo[k] = ctx->h_root[k];
  ctx->S = ctx->h_root[3];
  for (int l = 0; l <= OTOO_NLEV; l++) ctx->level_off[l] = off.v[l];
  ctx->key_order_built = ctx->key_order;
  ctx->built = true;
  return OTOO_OK;
}

// B2 of every cell (PAPER Eq. 2; R19) for the absolute-error MAC: one cooperative bottom-up pass, once per build
otoo_status otoo_b2_impl(otoo_ctx* ctx, cudaStream_t st) {
  if (ctx->b2_valid) return OTOO_OK;
  LevelOff off;
  for (int l = 0; l <= OTOO_NLEV; l++) off.v[l] = ctx->level_off[l];
  const MomentArgs ma{ctx->spos, ctx->key[0], ctx->c_first, ctx->c_count, ctx->c_child_first, ctx->c_child_count,
                      reinterpret_cast<const unsigned*>(ctx->d_bbox), ctx->c_MP, ctx->c_cm64, ctx->cell_cm, ctx->c_s, ctx->c_B2, ctx->key_order_built,
                      nullptr, ctx->cell_b, 0, 0.0f, nullptr, nullptr};
  int occ = 1;
  OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, b2_all_kernel, 256, 0));
  if (occ > 4) occ = 4;
  int64_t grid = (int64_t)ctx->sm_count * (occ < 1 ? 1 : occ);
  uint32_t widest = 1;
  for (int l = 0; l <= ctx->depth; l++) if (off.v[l + 1] - off.v[l] > widest) widest = off.v[l + 1] - off.v[l];
  if (grid > cdiv(widest, 256)) grid = cdiv(widest, 256);
  int depth_arg = ctx->depth;
  void* args[] = {(void*)&off, (void*)&depth_arg, (void*)&ma};
  OTOO_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)b2_all_kernel, dim3((unsigned)grid), dim3(256), args, 0, st));
  ctx->launches += 1;
  ctx->b2_valid = true;
  return OTOO_OK;
}
