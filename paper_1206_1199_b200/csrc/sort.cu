// sort.cu -- device LSD radix sort of (u64 key, u32 value) pairs and a u32 exclusive scan.
// PAPER.md L133 (III-B step 3): "we sort an array of the pair of a key and a particle's id".
// The paper used a host parallel quicksort; here it is an 8-bit-digit stable LSD radix sort in the
// one-sweep form (stable + ids initially ascending = ties broken by original index, reading R4).
#include <cstdarg>
#include <mutex>
#include "common.cuh"
#include "keys.cuh"

namespace {

constexpr int SORT_THREADS = 256;
constexpr int SORT_TILE = OTOO_SORT_TILE;             // pairs per CTA

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// ---------------- one-sweep passes: global digit histograms up front, then one kernel per digit whose
// tiles find their global offsets by decoupled look-back (no per-pass histogram/scan kernels, 12 B read
// + 12 B written per pair and pass), keys ranked in the tile and staged through shared memory so that the
// global writes are runs of consecutive addresses.
constexpr int OS_MAXPASS = 8;
#ifndef OTOO_OS_LOOKBACK
#define OTOO_OS_LOOKBACK 8
#endif
constexpr int OS_LOOKBACK = OTOO_OS_LOOKBACK;      // status words of preceding tiles a thread has in flight
constexpr uint32_t OS_GHIST = 0;                       // u32 offsets into ctx->hist
constexpr uint32_t OS_TICKET = OS_MAXPASS * 256;       // one tile ticket counter per pass; [OS_TICKET + 255] counts the histogram blocks
constexpr uint32_t OS_STATUS = OS_TICKET + 256;        // u64 status words [tile][digit] from here (8 B aligned)
constexpr int OS_NMASK = 2;                            // peer-mask tables per warp: a lane's items alternate between them
constexpr int64_t OS_SMALL_N = 4 << 20;                // up to here: CTAs of 512 threads (2 per SM); above: 256 threads (3 per SM)
constexpr size_t os_smem(int threads) { return SORT_TILE * 12 + (size_t)(1 + OS_NMASK) * (threads / 32) * 256 * 4 + 256 * 4 + 16; }

// all digit histograms of the key bits [first_bit, first_bit + 8 * npass) in one read of the keys
__global__ void __launch_bounds__(SORT_THREADS) radix_hist_all_kernel(const uint64_t* __restrict__ keys, int64_t n,
                                                                      int first_bit, int npass,
                                                                      uint32_t* __restrict__ ghist, uint32_t* __restrict__ done) {
  __shared__ uint32_t sh[OS_MAXPASS][256];
  const int tid = threadIdx.x;
  for (int p = 0; p < npass; p++) sh[p][tid] = 0;
  __syncthreads();
  for (int64_t i = (int64_t)blockIdx.x * SORT_THREADS + tid; i < n; i += (int64_t)gridDim.x * SORT_THREADS) {
    const uint64_t k = keys[i] >> first_bit;
    for (int p = 0; p < npass; p++) atomicAdd(&sh[p][(unsigned)(k >> (8 * p)) & 0xFF], 1u);
  }
  __syncthreads();
  for (int p = 0; p < npass; p++) if (sh[p][tid]) atomicAdd(&ghist[p * 256 + tid], sh[p][tid]);
  // the last block to arrive turns the counts into exclusive digit offsets (was a kernel of its own)
  __shared__ bool last;
  __threadfence();
  __syncthreads();
  if (tid == 0) last = atomicAdd(done, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  for (int p = 0; p < npass; p++) {
    const uint32_t c = __ldcg(&ghist[p * 256 + tid]);
    sh[0][tid] = c;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {
      uint32_t y = tid >= o ? sh[0][tid - o] : 0;
      __syncthreads();
      sh[0][tid] += y;
      __syncthreads();
    }
    ghist[p * 256 + tid] = sh[0][tid] - c;
    __syncthreads();
  }
}

// H2 fused with the histograms: keys and ids of all particles and, in the same pass over them, the eight digit
// histograms of the 64-bit sort (one read of the positions instead of a key kernel plus a read of the keys)
__global__ void __launch_bounds__(SORT_THREADS) key_hist_kernel(const float4* __restrict__ pos, int64_t n, const unsigned* __restrict__ bbox,
                                                                uint64_t* __restrict__ key, int hilbert,
                                                                uint32_t* __restrict__ ghist, uint32_t* __restrict__ done) {
  __shared__ uint32_t sh[OS_MAXPASS][256];
  const int tid = threadIdx.x;
  for (int p = 0; p < OS_MAXPASS; p++) sh[p][tid] = 0;
  __syncthreads();
  const float* root = reinterpret_cast<const float*>(bbox) + 8;
  constexpr int KH = 4;                                // positions in flight per thread (one: 0.26 ms at 32 M particles, latency-bound)
  const int64_t stride = (int64_t)gridDim.x * SORT_THREADS;
  for (int64_t i0 = (int64_t)blockIdx.x * SORT_THREADS + tid; i0 < n; i0 += KH * stride) {
    float4 pv[KH];
#pragma unroll
    for (int j = 0; j < KH; j++) if (i0 + j * stride < n) pv[j] = pos[i0 + j * stride];
#pragma unroll
    for (int j = 0; j < KH; j++) if (i0 + j * stride < n) {
      const uint64_t k = particle_key(pv[j], root, hilbert);
      key[i0 + j * stride] = k;                        // (the ids 0, 1, 2, ... are not written: the first sort pass makes them up)
#pragma unroll
      for (int p = 0; p < OS_MAXPASS; p++) atomicAdd(&sh[p][(unsigned)(k >> (8 * p)) & 0xFF], 1u);
    }
  }
  __syncthreads();
  for (int p = 0; p < OS_MAXPASS; p++) if (sh[p][tid]) atomicAdd(&ghist[p * 256 + tid], sh[p][tid]);
  __shared__ bool last;
  __threadfence();
  __syncthreads();
  if (tid == 0) last = atomicAdd(done, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  for (int p = 0; p < OS_MAXPASS; p++) {           // counts -> exclusive digit offsets
    const uint32_t c = __ldcg(&ghist[p * 256 + tid]);
    sh[0][tid] = c;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {
      uint32_t y = tid >= o ? sh[0][tid - o] : 0;
      __syncthreads();
      sh[0][tid] += y;
      __syncthreads();
    }
    ghist[p * 256 + tid] = sh[0][tid] - c;
    __syncthreads();
  }
}

// status word: [63:34] epoch of the pass, [33:32] 1 = tile aggregate, 2 = inclusive prefix, [31:0] count
__device__ __forceinline__ unsigned long long os_pack(uint32_t epoch, uint32_t state, uint32_t v) {
  return ((unsigned long long)((epoch << 2) | state) << 32) | v;
}

// One pass: a CTA takes one tile of SORT_TILE pairs.  Ranking: the lanes that hold a lane's digit are found by ORing
// lane bits into the digit's word of a per-warp mask table in shared memory -- MATCH.ANY on 8-bit digits costs
// 60 SM cycles per warp instruction on this part, a shared-memory atomic 3.6 (otoo_probe "rank"; profiles/r2_probes.md),
// and with MATCH the ADU pipe (66 % busy at two CTAs per SM) kept a third CTA per SM from helping.
template <int OS_THREADS, int MINB>
__global__ void __launch_bounds__(OS_THREADS, MINB) onesweep_pass_kernel(const uint64_t* __restrict__ kin,
                                                                         const uint32_t* __restrict__ vin,
                                                                         uint64_t* __restrict__ kout,
                                                                         uint32_t* __restrict__ vout, int64_t n, int shift,
                                                                         const uint32_t* __restrict__ gbase,
                                                                         unsigned long long* status, uint32_t* ticket,
                                                                         uint32_t epoch) {
  constexpr int OS_WARPS = OS_THREADS / 32, OS_ITEMS = SORT_TILE / OS_THREADS;
  extern __shared__ __align__(16) unsigned char os_raw[];
  uint64_t* skey = reinterpret_cast<uint64_t*>(os_raw);
  uint32_t* sval = reinterpret_cast<uint32_t*>(os_raw + SORT_TILE * 8);
  uint32_t(*whist)[256] = reinterpret_cast<uint32_t(*)[256]>(os_raw + SORT_TILE * 12);
  uint32_t(*wmask)[256] = whist + OS_WARPS;            // [OS_NMASK * OS_WARPS][256]
  uint32_t* goff = reinterpret_cast<uint32_t*>(wmask + OS_NMASK * OS_WARPS);
  uint32_t* stile = goff + 256;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) *stile = atomicAdd(ticket, 1u);      // tiles are numbered in starting order: look-back cannot hang
  for (int i = tid; i < (1 + OS_NMASK) * OS_WARPS * 256; i += OS_THREADS) (&whist[0][0])[i] = 0;
  __syncthreads();
  const uint32_t tile = *stile;
  const int64_t tbase = (int64_t)tile * SORT_TILE;
  const int64_t base = tbase + warp * (32 * OS_ITEMS);
  uint64_t k[OS_ITEMS];
  uint32_t v[OS_ITEMS];
  uint32_t rk2[(OS_ITEMS + 1) / 2];  // rank among equal digits within the warp's chunk, in index order (stable); two 16-bit ranks per word
#pragma unroll
  for (int i = 0; i < (OS_ITEMS + 1) / 2; i++) rk2[i] = 0;
#pragma unroll
  for (int i = 0; i < OS_ITEMS; i++) {
    int64_t idx = base + i * 32 + lane;
    if (idx < n) { k[i] = kin[idx]; v[i] = vin ? vin[idx] : (uint32_t)idx; }   // vin == nullptr: the ids are still 0, 1, 2, ... (first pass of the build)
                                                                               // (values loaded after the ranking instead: 2.46 -> 3.53 ms at 32 M pairs)
    else { k[i] = ~0ull; v[i] = 0; }
  }
  const unsigned lt = lanemask_lt();
#pragma unroll
  for (int i = 0; i < OS_ITEMS; i++) {
    const bool valid = base + i * 32 + lane < n;
    const unsigned d = (unsigned)((k[i] >> shift) & 0xFF);
    uint32_t* mask = &wmask[(i & 1) * OS_WARPS + warp][d];
    if (valid) atomicOr(mask, 1u << lane);
    __syncwarp();
    const unsigned peers = valid ? *mask : 0u;
    const uint32_t b = valid ? whist[warp][d] : 0u;
    __syncwarp();
    // the lowest peer counts the digit and clears the mask word (two tables: the clear cannot meet the next item's
    // OR, and the count is ordered before the next item's read by that item's first __syncwarp; one table and a
    // third __syncwarp: 2 % slower)
    if (valid && (peers & lt) == 0u) { whist[warp][d] = b + __popc(peers); *mask = 0u; }
    rk2[i >> 1] |= (b + __popc(peers & lt)) << (16 * (i & 1));
  }
  __syncthreads();
  // digit `tid`: tile count, look-back over the preceding tiles, start of the digit in the sorted tile
  uint32_t cnt = 0, inc = 0;
  const volatile unsigned long long* status_v = status;
  volatile unsigned long long* st = status + (size_t)tile * 256 + tid;
  if (tid < 256) {
#pragma unroll
    for (int w = 0; w < OS_WARPS; w++) cnt += whist[w][tid];
    *st = os_pack(epoch, tile == 0 ? 2u : 1u, cnt);
    inc = cnt;                                         // exclusive scan of the tile's digit counts: warp shuffles + the warps' totals
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += y; }
    if (lane == 31) goff[warp] = inc;
  }
  __syncthreads();
  uint32_t my_start = inc - cnt, excl = 0;
  if (tid < 256) {
#pragma unroll
    for (int w = 0; w < 7; w++) if (w < warp) my_start += goff[w];
    uint32_t run = my_start;                          // whist[w][d] := position in the sorted tile of warp w's first key with digit d
#pragma unroll
    for (int w = 0; w < OS_WARPS; w++) { const uint32_t c = whist[w][tid]; whist[w][tid] = run; run += c; }
#ifdef OTOO_OS_NOLOOKBACK          /* timing experiment only: wrong offsets, no chain over the tiles */
    if (false) {
#else
    if (tile > 0) {
#endif
      // look back over the preceding tiles, 8 status words in flight at a time (when all tiles of a small
      // sort run in one wave the walk is long, and one L2 round trip per tile would dominate the pass)
      int64_t t = (int64_t)tile - 1;
      bool done = false;
      while (!done) {
        unsigned long long w[OS_LOOKBACK];
#pragma unroll
        for (int j = 0; j < OS_LOOKBACK; j++)
          w[j] = t - j >= 0 ? *(status_v + (size_t)(t - j) * 256 + tid) : os_pack(epoch, 2u, 0u);
        int used = 0;
#pragma unroll
        for (int j = 0; j < OS_LOOKBACK; j++) {
          if (!done && used == j) {
            const uint32_t state = (uint32_t)(w[j] >> 32) & 3u;
            if ((uint32_t)(w[j] >> 34) == epoch && state != 0u) {
              excl += (uint32_t)w[j];
              used = j + 1;
              done = state == 2u;
            }
          }
        }
        t -= used;
      }
      *st = os_pack(epoch, 2u, excl + cnt);
    }
  }
  __syncthreads();
  if (tid < 256) goff[tid] = gbase[tid] + excl - my_start;   // global slot = goff[digit] + position in the sorted tile
  __syncthreads();
#pragma unroll
  for (int i = 0; i < OS_ITEMS; i++) {
    if (base + i * 32 + lane < n) {
      const unsigned d = (unsigned)((k[i] >> shift) & 0xFF);
      const uint32_t pos = whist[warp][d] + ((rk2[i >> 1] >> (16 * (i & 1))) & 0xFFFFu);
      skey[pos] = k[i];
      sval[pos] = v[i];
    }
  }
  __syncthreads();
  const int cnt_tile = (int)((n - tbase) < SORT_TILE ? (n - tbase) : SORT_TILE);
  for (int j = tid; j < cnt_tile; j += OS_THREADS) {
    const uint64_t key = skey[j];
    const uint32_t dst = goff[(unsigned)((key >> shift) & 0xFF)] + (uint32_t)j;
    kout[dst] = key;
    vout[dst] = sval[j];
  }
}

// ---------------- exclusive scan (u32), reduce-then-scan, in place ----------------
constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t x, uint32_t* total) {
  __shared__ uint32_t wsum[SCAN_THREADS / 32];
  __shared__ uint32_t tot;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = x;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += y; }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < SCAN_THREADS / 32 ? wsum[lane] : 0;
    uint32_t winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xFFFFFFFFu, winc, o); if (lane >= o) winc += y; }
    if (lane < SCAN_THREADS / 32) wsum[lane] = winc - w;
    if (lane == 31) tot = winc;
  }
  __syncthreads();
  uint32_t r = inc - x + wsum[warp];
  *total = tot;
  __syncthreads();
  return r;
}

// One kernel, one pass over the data: a tile of SCAN_TILE elements per block, the tile's exclusive offset by decoupled
// look-back over the preceding tiles' status words (the sort's format: epoch | state | value; tiles numbered by a ticket
// so that the wait cannot hang; nothing is cleared between scans).  Was a reduce kernel + an apply kernel.
__global__ void __launch_bounds__(SCAN_THREADS) scan_onepass_kernel(uint32_t* __restrict__ data, int64_t n, unsigned long long* status,
                                                                    uint32_t* ticket, uint32_t epoch, uint32_t* total_out) {
  __shared__ uint32_t s_tile, s_excl;
  if (threadIdx.x == 0) {
    s_tile = atomicAdd(ticket, 1u);
    if (s_tile == gridDim.x - 1) *ticket = 0u;            // the last ticket: ready for the next scan
  }
  __syncthreads();
  const uint32_t tile = s_tile;
  const int64_t base = (int64_t)tile * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t x[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) { x[i] = base + i < n ? data[base + i] : 0; s += x[i]; }
  uint32_t tot;
  uint32_t run = block_exclusive_scan(s, &tot);
  volatile unsigned long long* st = status;
  if (threadIdx.x == 0) st[tile] = os_pack(epoch, tile == 0 ? 2u : 1u, tot);
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    uint32_t excl = 0;
    int64_t t = (int64_t)tile - 1;
    while (t >= 0) {                                      // 32 preceding tiles per round
      const int64_t idx = t - lane;
      const unsigned long long w = idx >= 0 ? st[idx] : os_pack(epoch, 2u, 0u);
      const uint32_t state = (uint32_t)(w >> 32) & 3u;
      const bool valid = (uint32_t)(w >> 34) == epoch && state != 0u;
      const unsigned incl = __ballot_sync(0xFFFFFFFFu, valid && state == 2u), bad = __ballot_sync(0xFFFFFFFFu, !valid);
      const int first_incl = incl ? __ffs(incl) - 1 : 32, first_bad = bad ? __ffs(bad) - 1 : 32;
      if (first_bad < (first_incl < 32 ? first_incl + 1 : 32)) continue;          // a word of this range is not there yet
      uint32_t c = lane <= first_incl ? (uint32_t)w : 0u;
#pragma unroll
      for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
      excl += c;
      if (first_incl < 32) break;
      t -= 32;
    }
    if (lane == 0) {
      s_excl = excl;
      if (tile > 0) st[tile] = os_pack(epoch, 2u, excl + tot);
      if (tile == gridDim.x - 1 && total_out) *total_out = excl + tot;
    }
  }
  __syncthreads();
  run += s_excl;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) { if (base + i < n) data[base + i] = run; run += x[i]; }
}

}  // namespace

otoo_status otoo_exclusive_scan_u32(otoo_ctx* ctx, uint32_t* data, int64_t n, uint32_t* total_out_dev,
                                    cudaStream_t st) {
  if (n <= 0) {
    if (total_out_dev) OTOO_CUDA(ctx, cudaMemsetAsync(total_out_dev, 0, 4, st));
    return OTOO_OK;
  }
  const int64_t nb = cdiv(n, SCAN_TILE);
  if (2 + 2 * nb > ctx->scan_cap) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "scan scratch too small");
  if (ctx->scan_epoch + 1u >= (1u << 30)) {          // the epochs ran out: clear the status words and restart
    OTOO_CUDA(ctx, cudaMemsetAsync(ctx->scan_tmp, 0, ctx->scan_cap * sizeof(uint32_t), st));
    ctx->scan_epoch = 0;
  }
  // scan_tmp: [0] tile ticket (left at 0 by every scan), [2..] one 64-bit status word per tile
  scan_onepass_kernel<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(data, n, reinterpret_cast<unsigned long long*>(ctx->scan_tmp + 2), ctx->scan_tmp,
                                                            ++ctx->scan_epoch, total_out_dev);
  ctx->launches += 1;
  OTOO_CUDA(ctx, cudaGetLastError());
  return OTOO_OK;
}

// one epoch per radix pass tags the look-back status words; when they run out the words are cleared and the count restarts
static otoo_status sort_epoch_check(otoo_ctx* ctx, int npass, cudaStream_t st) {
  if (ctx->sort_epoch + (uint32_t)npass >= (1u << 30)) {
    OTOO_CUDA(ctx, cudaMemsetAsync(ctx->hist, 0, ctx->hist_cap * sizeof(uint32_t), st));
    ctx->sort_epoch = 0;
  }
  return OTOO_OK;
}

// keys (R2, R3, R20) of the particles into key[0] (ids: see otoo_sort_pairs), and the digit offsets of the 8-pass sort that follows
otoo_status otoo_keys_and_hist(otoo_ctx* ctx, const float* d_pos_mass, int64_t n, cudaStream_t st) {
  OTOO_TRY(sort_epoch_check(ctx, OS_MAXPASS, st));
  OTOO_CUDA(ctx, cudaMemsetAsync(ctx->hist, 0, OS_STATUS * sizeof(uint32_t), st));   // histograms + tickets
  int gh = ctx->sm_count * 4; if (gh > (int)cdiv(n, SORT_THREADS)) gh = (int)cdiv(n, SORT_THREADS);
  key_hist_kernel<<<gh, SORT_THREADS, 0, st>>>(reinterpret_cast<const float4*>(d_pos_mass), n, reinterpret_cast<const unsigned*>(ctx->d_bbox),
                                               ctx->key[0], ctx->key_order, ctx->hist + OS_GHIST, ctx->hist + OS_TICKET + 255);
  OTOO_CUDA(ctx, cudaGetLastError());
  return OTOO_OK;
}

// Sort n pairs on bits [first_bit, end_bit) in 8-bit digits (stable).  Input in buffer 0; *result_buf
// tells which buffer holds the result.  Uses ctx->hist (digit histograms, tile tickets, look-back status).
// hist_done: otoo_keys_and_hist has left the digit offsets of all passes (no histogram kernel here).
otoo_status otoo_sort_pairs(otoo_ctx* ctx, uint64_t* key[2], uint32_t* val[2], int64_t n, int first_bit,
                            int end_bit, cudaStream_t st, int* result_buf, bool hist_done) {
  int cur = 0;
  if (n > 0) {
    const int nb = (int)cdiv(n, SORT_TILE);
    const int npass = (end_bit - first_bit + 7) / 8;
    if (npass > OS_MAXPASS || OTOO_SORT_SCRATCH(n) > ctx->hist_cap)
      return otoo_fail(ctx, OTOO_ERR_CAPACITY, "sort scratch too small");
    if (!ctx->sort_attr_set) {
      OTOO_CUDA(ctx, cudaFuncSetAttribute(onesweep_pass_kernel<256, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)os_smem(256)));
      OTOO_CUDA(ctx, cudaFuncSetAttribute(onesweep_pass_kernel<512, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)os_smem(512)));
      ctx->sort_attr_set = true;
    }
    if (!hist_done) OTOO_TRY(sort_epoch_check(ctx, npass, st));
    if (hist_done) {       // otoo_keys_and_hist has cleared the scratch and left the digit offsets of all passes
    } else {
      OTOO_CUDA(ctx, cudaMemsetAsync(ctx->hist, 0, OS_STATUS * sizeof(uint32_t), st));   // histograms + tickets
      int gh = ctx->sm_count * 4; if (gh > (int)cdiv(n, SORT_THREADS)) gh = (int)cdiv(n, SORT_THREADS);
      radix_hist_all_kernel<<<gh, SORT_THREADS, 0, st>>>(key[0], n, first_bit, npass, ctx->hist + OS_GHIST, ctx->hist + OS_TICKET + 255);
      ctx->launches += 1;
    }
    unsigned long long* status = reinterpret_cast<unsigned long long*>(ctx->hist + OS_STATUS);
    for (int p = 0; p < npass; p++) {
      const uint32_t* vin = (p == 0 && hist_done) ? nullptr : val[cur];   // after otoo_keys_and_hist the ids are 0, 1, 2, ... and not stored
      // few tiles per SM: 2 CTAs of 16 warps hide more latency; many: 3 CTAs of 8 warps keep the shared-memory pipe busier
      if (n <= OS_SMALL_N)
        onesweep_pass_kernel<512, 2><<<nb, 512, os_smem(512), st>>>(key[cur], vin, key[cur ^ 1], val[cur ^ 1], n, first_bit + 8 * p,
                                                                      ctx->hist + OS_GHIST + p * 256, status, ctx->hist + OS_TICKET + p, ++ctx->sort_epoch);
      else
        onesweep_pass_kernel<256, 3><<<nb, 256, os_smem(256), st>>>(key[cur], vin, key[cur ^ 1], val[cur ^ 1], n, first_bit + 8 * p,
                                                                      ctx->hist + OS_GHIST + p * 256, status, ctx->hist + OS_TICKET + p, ++ctx->sort_epoch);
      ctx->launches += 1;
      cur ^= 1;
    }
    OTOO_CUDA(ctx, cudaGetLastError());
  }
  *result_buf = cur;
  return OTOO_OK;
}

// ---------------------------------------------------------------- the no-allocation entry point (include/otoo.h)
// otoo_sort_pairs_static: the same radix passes as otoo_sort_pairs, for callers that may not allocate (CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc).  The passes' scratch -- digit histograms, tile tickets and the
// look-back status words -- is NOT a context's `hist` buffer but this file-scope device array, sized for
// OTOO_SORT_STATIC_MAX_PAIRS pairs; every GPU that loads libotoo.so holds it (1.03 MB) until the process exits.
// In host code `g_sort_static` is only a stand-in for the symbol: its device address comes from cudaGetSymbolAddress,
// once per device with that device current (sort_static_setup), and that pointer is what the kernels are given.
namespace {
static_assert(OTOO_SORT_STATIC_MAX_PAIRS <= OS_SMALL_N, "the static entry point launches the 512-thread pass only");
constexpr int64_t SORT_STATIC_TILES = (OTOO_SORT_STATIC_MAX_PAIRS + SORT_TILE - 1) / SORT_TILE;
constexpr size_t SORT_STATIC_WORDS = OS_STATUS + (size_t)SORT_STATIC_TILES * 256 * 2;      // u32 words: histograms, tickets, u64 status
static __device__ __align__(256) uint32_t g_sort_static[SORT_STATIC_WORDS];

constexpr int SORT_STATIC_MAXDEV = 64;
struct SortStaticDev { std::once_flag once; cudaError_t err = cudaSuccess; uint32_t* scratch = nullptr; int sm_count = 0; };
SortStaticDev g_sort_static_dev[SORT_STATIC_MAXDEV];

// once per device, that device current: the array's device address, the SM count, the kernels' shared-memory opt-in
cudaError_t sort_static_setup(int dev, SortStaticDev** out) {
  SortStaticDev& d = g_sort_static_dev[dev];
  std::call_once(d.once, [&]() {
    void* p = nullptr;
    d.err = cudaGetSymbolAddress(&p, g_sort_static);
    if (d.err == cudaSuccess) d.err = cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (d.err == cudaSuccess) d.err = cudaFuncSetAttribute(onesweep_pass_kernel<512, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)os_smem(512));
    if (d.err == cudaSuccess) d.scratch = static_cast<uint32_t*>(p);
  });
  *out = &d;
  return d.err;
}

otoo_status sort_static_fail(otoo_status code, char* host_err, int64_t err_cap, const char* fmt, ...) {
  if (host_err && err_cap > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(host_err, (size_t)err_cap, fmt, ap);
    va_end(ap);
  }
  return code;
}
}  // namespace

extern "C" otoo_status otoo_sort_pairs_static(uint64_t* d_keys, uint32_t* d_vals, uint64_t* d_keys_alt, uint32_t* d_vals_alt,
                                              int64_t n, void* stream, char* host_err, int64_t err_cap) {
  if (host_err && err_cap > 0) host_err[0] = 0;
  if (n < 0) return sort_static_fail(OTOO_ERR_INVALID_ARG, host_err, err_cap, "otoo_sort_pairs_static: n = %lld is negative", (long long)n);
  if (n > OTOO_SORT_STATIC_MAX_PAIRS)
    return sort_static_fail(OTOO_ERR_CAPACITY, host_err, err_cap,
                            "otoo_sort_pairs_static: n = %lld exceeds OTOO_SORT_STATIC_MAX_PAIRS = %lld (the static scratch is sized for that; "
                            "larger sorts go through a context: otoo_build_tree)", (long long)n, (long long)OTOO_SORT_STATIC_MAX_PAIRS);
  if (n > 0 && (!d_keys || !d_vals || !d_keys_alt || !d_vals_alt))
    return sort_static_fail(OTOO_ERR_INVALID_ARG, host_err, err_cap, "otoo_sort_pairs_static: null buffer");
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess && (dev < 0 || dev >= SORT_STATIC_MAXDEV))
    return sort_static_fail(OTOO_ERR_INVALID_ARG, host_err, err_cap, "otoo_sort_pairs_static: device index %d not supported (< %d)", dev, SORT_STATIC_MAXDEV);
  SortStaticDev* d = nullptr;
  if (e == cudaSuccess) e = sort_static_setup(dev, &d);
  if (e != cudaSuccess)
    return sort_static_fail(OTOO_ERR_CUDA, host_err, err_cap, "otoo_sort_pairs_static: set-up on device %d failed: %s", dev, cudaGetErrorString(e));
  if (n == 0) return OTOO_OK;                       // (a call with n = 0 does the set-up and nothing else)
  cudaStream_t st = (cudaStream_t)stream;
  uint32_t* hist = d->scratch;                      // the DEVICE address of g_sort_static, never the host-side symbol
  const int nb = (int)cdiv(n, SORT_TILE);
  // the array keeps the last call's contents: histograms, tickets and this call's status words start at zero (the
  // passes are tagged with epochs 1..8 of THIS call, so nothing is carried from call to call and a captured graph replays)
  e = cudaMemsetAsync(hist, 0, (OS_STATUS + (size_t)nb * 256 * 2) * sizeof(uint32_t), st);
  if (e != cudaSuccess) return sort_static_fail(OTOO_ERR_CUDA, host_err, err_cap, "otoo_sort_pairs_static: %s", cudaGetErrorString(e));
  int gh = d->sm_count * 4; if (gh > (int)cdiv(n, SORT_THREADS)) gh = (int)cdiv(n, SORT_THREADS);
  radix_hist_all_kernel<<<gh, SORT_THREADS, 0, st>>>(d_keys, n, 0, OS_MAXPASS, hist + OS_GHIST, hist + OS_TICKET + 255);
  unsigned long long* status = reinterpret_cast<unsigned long long*>(hist + OS_STATUS);
  uint64_t* key[2] = {d_keys, d_keys_alt};
  uint32_t* val[2] = {d_vals, d_vals_alt};
  int cur = 0;
  for (int p = 0; p < OS_MAXPASS; p++) {            // n <= 2 Mi pairs: the 512-thread form (as otoo_sort_pairs chooses below OS_SMALL_N)
    onesweep_pass_kernel<512, 2><<<nb, 512, os_smem(512), st>>>(key[cur], val[cur], key[cur ^ 1], val[cur ^ 1], n, 8 * p,
                                                                  hist + OS_GHIST + p * 256, status, hist + OS_TICKET + p, (uint32_t)(p + 1));
    cur ^= 1;
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return sort_static_fail(OTOO_ERR_CUDA, host_err, err_cap, "otoo_sort_pairs_static: launch failed: %s", cudaGetErrorString(e));
  return OTOO_OK;                                   // eight passes: the result is back in d_keys / d_vals
}
