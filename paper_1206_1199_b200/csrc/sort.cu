// sort.cu -- device LSD radix sort of (u64 key, u32 value) pairs and a u32 exclusive scan.
// PAPER.md L133 (III-B step 3): "we sort an array of the pair of a key and a particle's id".
// The paper used a host parallel quicksort; here it is an 8-bit-digit stable LSD radix sort
// (stable + ids initially ascending = ties broken by original index, reading R4).
#include "common.cuh"

namespace {

constexpr int SORT_THREADS = 256;
constexpr int SORT_ITEMS = 16;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;  // 4096 keys per CTA
constexpr int SORT_WARPS = SORT_THREADS / 32;

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// per-CTA digit histogram -> hist[d * nb + b]
__global__ void __launch_bounds__(SORT_THREADS) radix_hist_kernel(const uint64_t* __restrict__ keys, int64_t n,
                                                                  int shift, uint32_t* __restrict__ hist, int nb) {
  __shared__ uint32_t sh[256];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  sh[tid] = 0;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * SORT_TILE + warp * (32 * SORT_ITEMS);
#pragma unroll 4
  for (int i = 0; i < SORT_ITEMS; i++) {
    int64_t idx = base + i * 32 + lane;
    unsigned d = 0xFFFFFFFFu;
    if (idx < n) d = (unsigned)((keys[idx] >> shift) & 0xFF);
    unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
    if (d != 0xFFFFFFFFu && (peers & lanemask_lt()) == 0) atomicAdd(&sh[d], __popc(peers));
  }
  __syncthreads();
  hist[(size_t)tid * nb + blockIdx.x] = sh[tid];
}

// stable scatter of one digit
__global__ void __launch_bounds__(SORT_THREADS) radix_scatter_kernel(const uint64_t* __restrict__ kin,
                                                                     const uint32_t* __restrict__ vin,
                                                                     uint64_t* __restrict__ kout,
                                                                     uint32_t* __restrict__ vout, int64_t n, int shift,
                                                                     const uint32_t* __restrict__ offs, int nb) {
  __shared__ uint32_t whist[SORT_WARPS][256];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#pragma unroll
  for (int w = 0; w < SORT_WARPS; w++) whist[w][tid] = 0;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * SORT_TILE + warp * (32 * SORT_ITEMS);
  uint64_t k[SORT_ITEMS];
  uint32_t v[SORT_ITEMS];
  uint32_t rk[SORT_ITEMS];  // rank within the warp's chunk among equal digits
#pragma unroll
  for (int i = 0; i < SORT_ITEMS; i++) {
    int64_t idx = base + i * 32 + lane;
    if (idx < n) { k[i] = kin[idx]; v[i] = vin[idx]; }
    else { k[i] = ~0ull; v[i] = 0; }
  }
#pragma unroll
  for (int i = 0; i < SORT_ITEMS; i++) {
    int64_t idx = base + i * 32 + lane;
    bool valid = idx < n;
    unsigned d = valid ? (unsigned)((k[i] >> shift) & 0xFF) : 0xFFFFFFFFu;
    unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
    int leader = __ffs(peers) - 1;
    uint32_t b = 0;
    if (valid && lane == leader) { b = whist[warp][d]; whist[warp][d] = b + __popc(peers); }
    b = __shfl_sync(0xFFFFFFFFu, b, leader);
    rk[i] = b + __popc(peers & lanemask_lt());
    __syncwarp();
  }
  __syncthreads();
  {  // digit `tid`: global offset of this CTA, then exclusive prefix over the warps
    uint32_t run = offs[(size_t)tid * nb + blockIdx.x];
#pragma unroll
    for (int w = 0; w < SORT_WARPS; w++) { uint32_t c = whist[w][tid]; whist[w][tid] = run; run += c; }
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < SORT_ITEMS; i++) {
    int64_t idx = base + i * 32 + lane;
    if (idx < n) {
      unsigned d = (unsigned)((k[i] >> shift) & 0xFF);
      uint32_t dst = whist[warp][d] + rk[i];
      kout[dst] = k[i];
      vout[dst] = v[i];
    }
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

__global__ void __launch_bounds__(SCAN_THREADS) scan_reduce_kernel(const uint32_t* __restrict__ data, int64_t n,
                                                                   uint32_t* __restrict__ sums) {
  int64_t base = (int64_t)blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) if (base + i < n) s += data[base + i];
  uint32_t tot;
  block_exclusive_scan(s, &tot);
  if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(SCAN_THREADS) scan_sums_kernel(uint32_t* sums, int64_t nb, uint32_t* total_out) {
  uint32_t carry = 0;
  for (int64_t c = 0; c < nb; c += SCAN_THREADS) {
    int64_t i = c + threadIdx.x;
    uint32_t x = i < nb ? sums[i] : 0, tot;
    uint32_t e = block_exclusive_scan(x, &tot);
    if (i < nb) sums[i] = e + carry;
    carry += tot;
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}
__global__ void __launch_bounds__(SCAN_THREADS) scan_apply_kernel(uint32_t* __restrict__ data, int64_t n,
                                                                  const uint32_t* __restrict__ sums) {
  int64_t base = (int64_t)blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t x[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) { x[i] = base + i < n ? data[base + i] : 0; s += x[i]; }
  uint32_t tot;
  uint32_t run = block_exclusive_scan(s, &tot) + sums[blockIdx.x];
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
  int64_t nb = cdiv(n, SCAN_TILE);
  scan_reduce_kernel<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(data, n, ctx->scan_tmp);
  scan_sums_kernel<<<1, SCAN_THREADS, 0, st>>>(ctx->scan_tmp, nb, total_out_dev);
  scan_apply_kernel<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(data, n, ctx->scan_tmp);
  ctx->launches += 3;
  OTOO_CUDA(ctx, cudaGetLastError());
  return OTOO_OK;
}

// Sort n pairs on bits [first_bit, end_bit) in 8-bit digits. Input in buffer 0; *result_buf tells
// which buffer holds the result.  Uses ctx->hist and ctx->scan_tmp.
otoo_status otoo_sort_pairs(otoo_ctx* ctx, uint64_t* key[2], uint32_t* val[2], int64_t n, int first_bit,
                            int end_bit, cudaStream_t st, int* result_buf) {
  int cur = 0;
  if (n > 0) {
    int nb = (int)cdiv(n, SORT_TILE);
    if ((size_t)nb * 256 > ctx->hist_cap) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "sort histogram scratch too small");
    for (int shift = first_bit; shift < end_bit; shift += 8) {
      radix_hist_kernel<<<nb, SORT_THREADS, 0, st>>>(key[cur], n, shift, ctx->hist, nb);
      ctx->launches += 1;
      OTOO_TRY(otoo_exclusive_scan_u32(ctx, ctx->hist, (int64_t)nb * 256, nullptr, st));
      radix_scatter_kernel<<<nb, SORT_THREADS, 0, st>>>(key[cur], val[cur], key[cur ^ 1], val[cur ^ 1], n, shift,
                                                        ctx->hist, nb);
      ctx->launches += 1;
      cur ^= 1;
    }
    OTOO_CUDA(ctx, cudaGetLastError());
  }
  *result_buf = cur;
  return OTOO_OK;
}
