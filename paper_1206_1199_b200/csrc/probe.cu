// probe.cu -- microbenchmarks behind the ceilings quoted in DESIGN.md section 6 (otoo_probe; bench.py --probe).
//   "ffma2":   cycles per FFMA2 warp instruction and SM sub-partition for the operand patterns the sum loop uses
//              (one register pair + uniform; two pairs; three pairs; three pairs with one shared by three
//              consecutive instructions; pair + 32-bit broadcast register), by clock64() inside the kernel.
//   "sumloop": the product's own pair-sum loop (GravVisitor::eval of grav_eval.cuh) on lists already resident in
//              shared memory -- no walk, no hand-off: the evaluator's ceiling in interactions/s.
//   "rank":    SM cycles per warp instruction of the primitives a radix ranking can be built from (MATCH.ANY on 8- and
//              4-bit digits, ballot, shared-memory atomics, a random shared-memory load): why the sort's ranking ORs
//              lane bits into shared memory instead of using match.any.
//   "sort":    the product's eight-pass sort of (u64 key, u32 id) pairs (otoo_sort_pairs) beside the library's
//              cub::DeviceRadixSort::SortPairs on the same pairs -- a reference point, CUB is not on the force path.
// Measurement aids only: nothing here is on the force path.
#include <string>
#include <cub/device/device_radix_sort.cuh>
#include "grav_eval.cuh"

namespace {

// ---------------------------------------------------------------- FFMA2 operand patterns
constexpr int FP_ACC = 12;       // independent accumulators per thread
template <int MODE>
__global__ void __launch_bounds__(512, 1) ffma2_probe_kernel(const f32x2* __restrict__ in, f32x2* __restrict__ out, int iters,
                                                             f32x2 uni, unsigned long long* __restrict__ cycles) {
  f32x2 a[FP_ACC], b[FP_ACC], c[FP_ACC];
  const f32x2* src = in + (size_t)threadIdx.x * 3 * FP_ACC;     // 64-bit loads: the operands are born as register pairs
#pragma unroll
  for (int i = 0; i < FP_ACC; i++) { a[i] = src[i]; b[i] = src[FP_ACC + i]; c[i] = src[2 * FP_ACC + i]; }
  float s0, s1;
  upk2(src[0], s0, s1);
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < FP_ACC; i++) {
      if (MODE == 0) a[i] = fma2(a[i], uni, a[i]);                       // one register pair + a uniform (constant-bank) operand
      else if (MODE == 1) a[i] = fma2(a[i], b[i], a[i]);                 // two register pairs
      else if (MODE == 2) a[i] = fma2(b[i], c[i], a[i]);                 // three register pairs
      else if (MODE == 3) a[i] = fma2(b[i / 3], c[i], a[i]);             // three pairs, the first shared by three consecutive instructions
      else {                                                             // a pair + a 32-bit register broadcast to both halves
        float2 x = __ffma2_rn(make_float2(s0, s0), as2(b[i]), as2(a[i]));
        a[i] = pk2(x.x, x.y);
      }
    }
  }
  __syncthreads();                       // the slowest warp of the CTA ends the interval
  const long long t1 = clock64();
  f32x2 r = a[0];
#pragma unroll
  for (int i = 1; i < FP_ACC; i++) r = add2(r, a[i]);
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = r;
  if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
}

// ---------------------------------------------------------------- the sum loop alone
template <int T, int PB, int UNR, int ACC>
__global__ void __launch_bounds__(128, T >= 8 ? 2 : 3) sumloop_probe_kernel(const GravParams p, int reps, float4* __restrict__ sink,
                                                                             unsigned long long* __restrict__ cycles) {
  __shared__ __align__(16) float4 lists[4][OTOO_LIST_CAP + 4];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float4* list = lists[warp];
  // synthetic list: points of the unit cube by a counter hash, equal masses (values do not change the timing)
  for (int j = lane; j < OTOO_LIST_CAP; j += 32) {
    uint32_t h = (uint32_t)(j * 2654435761u) ^ (blockIdx.x * 40503u + warp * 97u);
    const float x = (float)(h & 1023u) * (1.0f / 1024.0f), y = (float)((h >> 10) & 1023u) * (1.0f / 1024.0f),
                z = (float)((h >> 20) & 1023u) * (1.0f / 1024.0f);
    list[j] = make_float4(x, y, z, 1.0f / OTOO_LIST_CAP);
  }
  __syncwarp();
  GravVisitor<T, false, PB, UNR, ACC> v(p);
  const int64_t g0 = ((int64_t)(blockIdx.x * 4 + warp) * (32 * T)) % (p.c.N - 32 * T);
  __shared__ __align__(16) float2 scratch[4][32 * ((T + 1) / 2) * 3];
  v.load_group(g0, lane, reinterpret_cast<float4*>(scratch[warp]));
  __syncthreads();
  const long long t0 = clock64();
  unsigned long long g0ns, g1ns;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0ns));
  for (int r = 0; r < reps; r++) v.eval(list, OTOO_LIST_CAP);
  __syncthreads();                       // the slowest warp of the CTA ends the interval
  const long long t1 = clock64();
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1ns));
  float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int q = 0; q < (T + 1) / 2; q++) { o.x += v.AX[q].x + v.AX[q].y; o.y += v.AY[q].x + v.AY[q].y; o.z += v.AZ[q].x + v.AZ[q].y; o.w += v.PH[q].x + v.PH[q].y; }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = o;
  if (threadIdx.x == 0) { cycles[blockIdx.x] = (unsigned long long)(t1 - t0); cycles[gridDim.x + blockIdx.x] = g1ns - g0ns; }
}

__global__ void __launch_bounds__(256) probe_fill_kernel(float4* pos, f32x2* pairs, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t h = (uint32_t)i * 2654435761u;
  pos[i] = make_float4((float)(h & 1023u) * (1.0f / 1024.0f), (float)((h >> 10) & 1023u) * (1.0f / 1024.0f),
                       (float)((h >> 20) & 1023u) * (1.0f / 1024.0f), 1.0f);
  if (pairs) pairs[i] = pk2(1.0f + 1e-7f * (float)(h & 255u), 1.0f - 1e-7f * (float)((h >> 8) & 255u));
}

// ---------------------------------------------------------------- ranking primitives
template <int MODE>
__global__ void __launch_bounds__(512, 1) rank_probe_kernel(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, int iters,
                                                            unsigned long long* __restrict__ cycles) {
  __shared__ uint32_t sm[16][256];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int i = tid; i < 16 * 256; i += blockDim.x) (&sm[0][0])[i] = 0;
  uint32_t d[8];
  for (int i = 0; i < 8; i++) d[i] = in[(size_t)tid * 8 + i] & 0xFFu;     // "random" 8-bit digits
  uint32_t acc = 0;
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 8; i++) {
      const uint32_t x = d[i];
      if (MODE == 0) acc += __match_any_sync(0xFFFFFFFFu, x);
      else if (MODE == 1) acc += __match_any_sync(0xFFFFFFFFu, x & 15u);
      else if (MODE == 2) acc += __ballot_sync(0xFFFFFFFFu, x & 1u);
      else if (MODE == 3) acc += atomicAdd(&sm[warp][x], 1u);
      else if (MODE == 4) atomicOr(&sm[warp][x], 1u << lane);
      else acc += sm[warp][x];
      d[i] = (x * 5u + 1u) & 0xFFu;
    }
  }
  __syncthreads();
  const long long t1 = clock64();
  out[(size_t)blockIdx.x * blockDim.x + tid] = acc + d[0] + sm[warp][lane];
  if (tid == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
}

__global__ void __launch_bounds__(256) sort_fill_kernel(uint64_t* k, uint32_t* v, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint64_t x = (uint64_t)i * 0x9E3779B97F4A7C15ull;      // SplitMix64 finaliser: 63 random key bits, ids ascending
  x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull; x ^= x >> 27; x *= 0x94D049BB133111EBull; x ^= x >> 31;
  k[i] = x >> 1; v[i] = (uint32_t)i;
}

struct Timer {
  cudaEvent_t e0, e1;
  Timer() { cudaEventCreate(&e0); cudaEventCreate(&e1); }
  ~Timer() { cudaEventDestroy(e0); cudaEventDestroy(e1); }
  void start(cudaStream_t st) { cudaEventRecord(e0, st); }
  float stop(cudaStream_t st) { cudaEventRecord(e1, st); cudaEventSynchronize(e1); float ms = 0; cudaEventElapsedTime(&ms, e0, e1); return ms; }
};

template <int MODE>
double run_ffma2(otoo_ctx* ctx, const f32x2* in, f32x2* out, unsigned long long* d_cyc, int warps_per_smsp, cudaStream_t st) {
  const int threads = 128 * warps_per_smsp, iters = 4096, grid = ctx->sm_count;
  const f32x2 uni = 0x3F8000003F800000ull;     // (1.0f, 1.0f)
  ffma2_probe_kernel<MODE><<<grid, threads, 0, st>>>(in, out, 64, uni, d_cyc);
  ffma2_probe_kernel<MODE><<<grid, threads, 0, st>>>(in, out, iters, uni, d_cyc);
  std::string dummy;
  unsigned long long h[256];
  cudaMemcpyAsync(h, d_cyc, sizeof(unsigned long long) * (grid < 256 ? grid : 256), cudaMemcpyDeviceToHost, st);
  cudaStreamSynchronize(st);
  double sum = 0;
  const int n = grid < 256 ? grid : 256;
  for (int i = 0; i < n; i++) sum += (double)h[i];
  // cycles per warp instruction and sub-partition: every SMSP issued warps_per_smsp x iters x FP_ACC FFMA2
  return sum / n / ((double)warps_per_smsp * iters * FP_ACC);
}

template <int MODE>
double run_rank(otoo_ctx* ctx, const uint32_t* in, uint32_t* out, unsigned long long* d_cyc, int warps, cudaStream_t st) {
  const int iters = 512, grid = ctx->sm_count;
  rank_probe_kernel<MODE><<<grid, 32 * warps, 0, st>>>(in, out, 8, d_cyc);
  rank_probe_kernel<MODE><<<grid, 32 * warps, 0, st>>>(in, out, iters, d_cyc);
  unsigned long long h[256];
  const int n = grid < 256 ? grid : 256;
  cudaMemcpyAsync(h, d_cyc, sizeof(unsigned long long) * n, cudaMemcpyDeviceToHost, st);
  cudaStreamSynchronize(st);
  double sum = 0;
  for (int i = 0; i < n; i++) sum += (double)h[i];
  return sum / n / ((double)iters * 8 * warps);          // SM cycles per warp instruction (all warps of the SM share the unit)
}

template <int T, int PB, int UNR, int ACC = OTOO_EVAL_ACC>
otoo_status run_sumloop(otoo_ctx* ctx, GravParams p, float4* sink, unsigned long long* d_cyc, cudaStream_t st, std::string& js,
                        int per_sm_arg = 0) {
  const int reps = 256;
  int occ = 0;
  OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sumloop_probe_kernel<T, PB, UNR, ACC>, 128, 0));
  cudaFuncAttributes fa;
  OTOO_CUDA(ctx, cudaFuncGetAttributes(&fa, sumloop_probe_kernel<T, PB, UNR, ACC>));
  const int per_sm = per_sm_arg ? per_sm_arg : (T >= 8 ? 2 : 3);   // CTAs of 4 evaluator warps per SM (default: the product kernel's)
  const int grid = ctx->sm_count * per_sm;
  // dynamic shared memory sized so that EXACTLY per_sm CTAs fit an SM: every SM then runs per_sm CTAs of the
  // grid at once (left to the occupancy of the kernel alone the block scheduler packs 4 on some SMs and 2 on others)
  const size_t dyn = (size_t)(227 * 1024) / per_sm - fa.sharedSizeBytes - 2048;
  OTOO_CUDA(ctx, cudaFuncSetAttribute(sumloop_probe_kernel<T, PB, UNR, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
  OTOO_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sumloop_probe_kernel<T, PB, UNR, ACC>, 128, dyn));
  if (occ != per_sm) return otoo_fail(ctx, OTOO_ERR_CUDA, "probe: occupancy is not the evaluator's");
  Timer tm;
  sumloop_probe_kernel<T, PB, UNR, ACC><<<grid, 128, dyn, st>>>(p, 4, sink, d_cyc);
  float best = 1e30f;
  for (int r = 0; r < 3; r++) {
    tm.start(st);
    sumloop_probe_kernel<T, PB, UNR, ACC><<<grid, 128, dyn, st>>>(p, reps, sink, d_cyc);
    const float ms = tm.stop(st);
    if (ms < best) best = ms;
  }
  OTOO_CUDA(ctx, cudaGetLastError());
  unsigned long long h[1024];
  const int n = grid < 512 ? grid : 512;
  OTOO_CUDA(ctx, cudaMemcpy(h, d_cyc, sizeof(unsigned long long) * n, cudaMemcpyDeviceToHost));
  OTOO_CUDA(ctx, cudaMemcpy(h + 512, d_cyc + grid, sizeof(unsigned long long) * n, cudaMemcpyDeviceToHost));
  double cyc = 0, ns = 0;
  for (int i = 0; i < n; i++) { cyc += (double)h[i]; ns += (double)h[512 + i]; }
  cyc /= n; ns /= n;
  const double sm_mhz = 1e3 * cyc / ns;                  // SM clock held during the loop: clock64 ticks per globaltimer ns
  const double inter = (double)grid * 4 * 32 * T * OTOO_LIST_CAP * reps;
  // SMSP cycles per (target pair, list entry) from the kernel's duration at the clock it held: every SMSP ran per_sm
  // warps x NP pairs x entries x reps (the CTAs' own tick counts are not used for this: the scheduler favours some
  // warps, so a CTA's mean is below the kernel's)
  (void)cyc;
  const double per_pair = (double)best * 1e-3 * sm_mhz * 1e6 / ((double)per_sm * ((T + 1) / 2) * OTOO_LIST_CAP * reps);
  char buf[512];
  snprintf(buf, sizeof buf,
           "{\"name\": \"sumloop G=%d\", \"accumulate\": \"%s\", \"pairs_per_pass\": %d, \"unroll\": %d, \"eval_warps_per_sm\": %d, \"registers\": %d, \"occupancy_ctas\": %d, \"ms\": %.4f, "
           "\"interactions_per_s\": %.6e, \"tflops_20flop\": %.3f, \"smsp_cycles_per_pair_entry\": %.3f, \"sm_mhz_during_loop\": %.0f}",
           32 * T, ACC ? "scalar FFMA" : "FFMA2", GravVisitor<T, false, PB, UNR>::PB, UNR, 4 * per_sm, fa.numRegs, occ, best, inter / (best * 1e-3), 20.0 * inter / (best * 1e-3) / 1e12, per_pair, sm_mhz);
  if (!js.empty()) js += ", ";
  js += buf;
  return OTOO_OK;
}

}  // namespace

extern "C" otoo_status otoo_probe(otoo_ctx* ctx, const char* which, char* host_json, int64_t cap, void* stream) {
  if (!ctx || !which || !host_json || cap < 64) return OTOO_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  // scratch inside the context's particle arrays: 64 Ki positions, and in key[1] (8 B per particle) the cycle counters
  // followed by one float4 per probe thread (<= 5 CTAs x 128 threads per SM): 2 MB
  if (ctx->maxN < (1 << 18)) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "otoo_probe needs max_particles >= 262144 of scratch");
  ctx->built = false; ctx->walked = false;               // the probes use the context's particle arrays as scratch
  const int64_t n = 1 << 16;
  f32x2* pairs = reinterpret_cast<f32x2*>(ctx->key[0]);
  probe_fill_kernel<<<(unsigned)cdiv(n, 256), 256, 0, st>>>(ctx->spos, pairs, n);
  unsigned long long* d_cyc = reinterpret_cast<unsigned long long*>(ctx->key[1]);
  std::string js;
  if (strcmp(which, "ffma2") == 0) {
    f32x2* out = reinterpret_cast<f32x2*>(ctx->key[1]) + 4096;
    const char* names[5] = {"one pair + uniform operand", "two pairs", "three pairs", "three pairs, one shared by 3 consecutive",
                            "pair + 32-bit broadcast register + pair"};
    for (int w = 2; w <= 4; w += 2) {
      const double c[5] = {run_ffma2<0>(ctx, pairs, out, d_cyc, w, st), run_ffma2<1>(ctx, pairs, out, d_cyc, w, st),
                           run_ffma2<2>(ctx, pairs, out, d_cyc, w, st), run_ffma2<3>(ctx, pairs, out, d_cyc, w, st),
                           run_ffma2<4>(ctx, pairs, out, d_cyc, w, st)};
      for (int m = 0; m < 5; m++) {
        char buf[256];
        snprintf(buf, sizeof buf, "%s{\"name\": \"FFMA2 %s\", \"warps_per_smsp\": %d, \"smsp_cycles_per_instruction\": %.3f}",
                 js.empty() ? "" : ", ", names[m], w, c[m]);
        js += buf;
      }
    }
    OTOO_CUDA(ctx, cudaGetLastError());
  } else if (strcmp(which, "sumloop") == 0) {
    GravParams p;
    memset(&p, 0, sizeof p);
    p.c.spos = ctx->spos; p.c.N = n; p.c.gs = 256; p.eps2 = 1e-6f;
    float4* sink = reinterpret_cast<float4*>(ctx->key[1]) + 4096;
    // the product's three configurations (pairs per pass = min(NP, 2), unroll OTOO_EVAL_UNR, 12 / 12 / 8 evaluator
    // warps per SM), then what was tried: other unroll factors and pairs per pass, more or fewer warps per SM
    OTOO_TRY((run_sumloop<2, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<8, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 2, 1>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 2, 2>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 2, 8>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 1, 4>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<8, 4, 2>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<8, 1, 4>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js, 1)));
    OTOO_TRY((run_sumloop<4, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js, 2)));
    OTOO_TRY((run_sumloop<4, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js, 4)));
    OTOO_TRY((run_sumloop<2, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js, 4)));
    OTOO_TRY((run_sumloop<2, 0, OTOO_EVAL_UNR>(ctx, p, sink, d_cyc, st, js, 5)));
    // the other form of the accumulations (scalar FFMA <-> FFMA2) at the product's three configurations
    OTOO_TRY((run_sumloop<2, 0, OTOO_EVAL_UNR, 1 - OTOO_EVAL_ACC>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 0, OTOO_EVAL_UNR, 1 - OTOO_EVAL_ACC>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<8, 0, OTOO_EVAL_UNR, 1 - OTOO_EVAL_ACC>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<4, 2, 8, 1 - OTOO_EVAL_ACC>(ctx, p, sink, d_cyc, st, js)));
    OTOO_TRY((run_sumloop<8, 4, 2, 1 - OTOO_EVAL_ACC>(ctx, p, sink, d_cyc, st, js)));
  } else if (strcmp(which, "rank") == 0) {
    sort_fill_kernel<<<64, 256, 0, st>>>(ctx->key[0], ctx->val[0], 64 * 256);
    const uint32_t* digits = reinterpret_cast<const uint32_t*>(ctx->key[0]);
    uint32_t* out = reinterpret_cast<uint32_t*>(ctx->key[1]) + 4096;
    const char* names[6] = {"MATCH.ANY, 8-bit digits", "MATCH.ANY, 4-bit digits", "VOTE (ballot)", "ATOMS.ADD with return, random digit",
                            "ATOMS.OR without return, random digit", "LDS, random word"};
    for (int w = 4; w <= 16; w += 12) {
      const double c[6] = {run_rank<0>(ctx, digits, out, d_cyc, w, st), run_rank<1>(ctx, digits, out, d_cyc, w, st),
                           run_rank<2>(ctx, digits, out, d_cyc, w, st), run_rank<3>(ctx, digits, out, d_cyc, w, st),
                           run_rank<4>(ctx, digits, out, d_cyc, w, st), run_rank<5>(ctx, digits, out, d_cyc, w, st)};
      for (int m = 0; m < 6; m++) {
        char buf[256];
        snprintf(buf, sizeof buf, "%s{\"name\": \"%s\", \"warps_per_sm\": %d, \"sm_cycles_per_warp_instruction\": %.2f}",
                 js.empty() ? "" : ", ", names[m], w, c[m]);
        js += buf;
      }
    }
    OTOO_CUDA(ctx, cudaGetLastError());
  } else if (strcmp(which, "sort") == 0) {
    Timer tm;
    for (int64_t ns = 1 << 20; ns <= ctx->maxN && ns <= (int64_t)1 << 25; ns <<= (ns == 1 << 20 ? 3 : 2)) {
      size_t tb = 0;
      OTOO_CUDA(ctx, cub::DeviceRadixSort::SortPairs(nullptr, tb, ctx->key[0], ctx->key[1], ctx->val[0], ctx->val[1], ns, 0, 63, st));
      void* tmp = nullptr;
      OTOO_CUDA(ctx, cudaMalloc(&tmp, tb));
      float ours = 1e30f, lib = 1e30f;
      for (int r = 0; r < 6; r++) {
        sort_fill_kernel<<<(unsigned)cdiv(ns, 256), 256, 0, st>>>(ctx->key[0], ctx->val[0], ns);
        int rb = 0;
        tm.start(st);
        const otoo_status s1 = otoo_sort_pairs(ctx, ctx->key, ctx->val, ns, 0, 63, st, &rb, false);
        const float a = tm.stop(st);
        if (s1 != OTOO_OK) { cudaFree(tmp); return s1; }
        sort_fill_kernel<<<(unsigned)cdiv(ns, 256), 256, 0, st>>>(ctx->key[0], ctx->val[0], ns);
        tm.start(st);
        cub::DeviceRadixSort::SortPairs(tmp, tb, ctx->key[0], ctx->key[1], ctx->val[0], ctx->val[1], ns, 0, 63, st);
        const float b = tm.stop(st);
        if (r >= 1) { if (a < ours) ours = a; if (b < lib) lib = b; }
      }
      cudaFree(tmp);
      OTOO_CUDA(ctx, cudaGetLastError());
      char buf[320];
      snprintf(buf, sizeof buf, "%s{\"name\": \"sort of (u64 key, u32 id) pairs, key bits 0..62\", \"pairs\": %lld, \"otoo_sort_pairs_ms\": %.4f, "
               "\"cub_DeviceRadixSort_SortPairs_ms\": %.4f, \"cub_temp_bytes\": %zu}", js.empty() ? "" : ", ", (long long)ns, ours, lib, tb);
      js += buf;
    }
  } else return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "unknown probe (ffma2, sumloop, rank, sort)");
  js = "[" + js + "]";
  if ((int64_t)js.size() + 1 > cap) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "probe output buffer too small");
  memcpy(host_json, js.c_str(), js.size() + 1);
  return OTOO_OK;
}
