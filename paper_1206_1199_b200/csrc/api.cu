// api.cu -- the C-ABI of include/otoo.h: argument checks, context lifecycle, exports.
#include <string.h>
#include <new>
#include "common.cuh"

namespace {

template <typename T>
otoo_status dalloc(otoo_ctx* ctx, T** p, size_t count) {
  *p = nullptr;
  OTOO_CUDA(ctx, cudaMalloc((void**)p, (count ? count : 1) * sizeof(T)));
  return OTOO_OK;
}

__global__ void __launch_bounds__(256) export_cells_kernel(int64_t ncell, const uint32_t* __restrict__ c_first,
                                                           const uint32_t* __restrict__ c_count,
                                                           const uint32_t* __restrict__ c_child_first,
                                                           const uint8_t* __restrict__ c_level,
                                                           const uint8_t* __restrict__ c_child_count,
                                                           const uint64_t* __restrict__ key, otoo_cell_t* __restrict__ out) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  otoo_cell_t o;
  memset(&o, 0, sizeof o);
  o.level = c_level[c] & 0x1F; o.first = c_first[c]; o.count = c_count[c];
  o.child_first = c_child_first[c]; o.child_count = c_child_count[c];
  o.prefix = (o.level > 0 && o.count > 0) ? key[o.first] >> (3 * (OTOO_MAXLEV - o.level)) : 0ull;
  out[c] = o;
}
__global__ void __launch_bounds__(256) export_rb2_kernel(int64_t ncell, const cellb_t* __restrict__ cell_b, float* __restrict__ out) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c < ncell) out[c] = __uint_as_float(cell_b[c].x);
}
__global__ void __launch_bounds__(256) export_sph_kernel(int64_t ncell, const float2* __restrict__ in, float* __restrict__ b, float* __restrict__ r) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c < ncell) { float2 v = in[c]; if (b) b[c] = v.x; if (r) r[c] = v.y; }
}
// out[perm[s]] = in[s]: rows in sorted order back into the caller's order (the inverse of the build's gather)
__global__ void __launch_bounds__(256) unsort4_kernel(const float4* __restrict__ in, const uint32_t* __restrict__ perm, int64_t n,
                                                      float4* __restrict__ out) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) out[perm[s]] = in[s];
}
__global__ void __launch_bounds__(256) eos_ideal_kernel(const float* __restrict__ rho, const float* __restrict__ u, float gm1,
                                                        int64_t n, float* __restrict__ P) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) P[i] = __fmul_rn(__fmul_rn(gm1, rho[i]), u[i]);
}

bool valid_group(int G) { return G == 4 || G == 8 || G == 16 || G == 32 || G == 64 || G == 128 || G == 256; }

}  // namespace

otoo_status otoo_ensure_groups(otoo_ctx* ctx, int64_t ngroups) {
  if (ngroups <= ctx->groupCap) return OTOO_OK;
  if (ctx->g_ntests) cudaFree(ctx->g_ntests);
  if (ctx->g_ncells) cudaFree(ctx->g_ncells);
  if (ctx->g_nparts) cudaFree(ctx->g_nparts);
  ctx->g_ntests = ctx->g_ncells = ctx->g_nparts = nullptr;   // a failed allocation below must not leave freed pointers
  ctx->groupCap = 0;
  OTOO_TRY(dalloc(ctx, &ctx->g_ntests, ngroups));
  OTOO_TRY(dalloc(ctx, &ctx->g_ncells, ngroups));
  OTOO_TRY(dalloc(ctx, &ctx->g_nparts, ngroups));
  ctx->groupCap = ngroups;
  return OTOO_OK;
}
otoo_status otoo_ensure_spill(otoo_ctx* ctx, int64_t warps) {
  if (warps <= ctx->spill_warps) return OTOO_OK;
  if (ctx->walk_spill) cudaFree(ctx->walk_spill);
  ctx->walk_spill = nullptr;
  ctx->spill_warps = 0;
  OTOO_TRY(dalloc(ctx, &ctx->walk_spill, (size_t)warps * OTOO_WALK_SPILL));
  ctx->spill_warps = warps;
  return OTOO_OK;
}

extern "C" {

int otoo_version(void) { return 2; }

otoo_status otoo_create(otoo_ctx** out, int device, int64_t max_particles) {
  if (!out) return OTOO_ERR_INVALID_ARG;
  *out = nullptr;
  if (max_particles < 1 || max_particles > 2147483647LL) return OTOO_ERR_INVALID_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return OTOO_ERR_CUDA;
  otoo_ctx* ctx = new (std::nothrow) otoo_ctx;
  if (!ctx) return OTOO_ERR_OOM;
  memset(ctx, 0, sizeof *ctx);
  ctx->device = device; ctx->maxN = max_particles; ctx->walk_stack = OTOO_WALK_STACK_MAX; ctx->walk_spill_cap = OTOO_WALK_SPILL; ctx->use_pool = 1; ctx->use_ws = 1; ctx->dist_kind = 2; ctx->group_begin = 0; ctx->group_count = -1;
  otoo_status s = OTOO_OK;
  auto body = [&]() -> otoo_status {
    OTOO_CUDA(ctx, cudaSetDevice(device));
    cudaDeviceProp prop;
    OTOO_CUDA(ctx, cudaGetDeviceProperties(&prop, device));
    ctx->sm_count = prop.multiProcessorCount;
    const size_t n = (size_t)max_particles;
    for (int b = 0; b < 2; b++) { OTOO_TRY(dalloc(ctx, &ctx->key[b], n)); OTOO_TRY(dalloc(ctx, &ctx->val[b], n)); }
    OTOO_TRY(dalloc(ctx, &ctx->spos, n));
    OTOO_TRY(dalloc(ctx, &ctx->slot_nc, (size_t)(OTOO_NLEV + 1) * (size_t)cdiv(max_particles, 256) + 64));   // per-block level counts and leaf counts (H5a)
    ctx->hist_cap = OTOO_SORT_SCRATCH(max_particles);   // look-back status (u64 per tile and digit) + histograms
    OTOO_TRY(dalloc(ctx, &ctx->hist, ctx->hist_cap));
    OTOO_CUDA(ctx, cudaMemset(ctx->hist, 0, ctx->hist_cap * sizeof(uint32_t)));
    ctx->scan_cap = (size_t)cdiv(max_particles, 4096) + 1024;
    OTOO_TRY(dalloc(ctx, &ctx->scan_tmp, ctx->scan_cap));
    OTOO_TRY(dalloc(ctx, &ctx->d_bbox, 16));
    OTOO_TRY(dalloc(ctx, &ctx->d_counters, 64));
    OTOO_TRY(dalloc(ctx, &ctx->d_sums, OTOO_NSUMS));
    OTOO_CUDA(ctx, cudaMemset(ctx->d_sums, 0, OTOO_NSUMS * sizeof(unsigned long long)));
    OTOO_CUDA(ctx, cudaMallocHost((void**)&ctx->h_counters, 64 * sizeof(uint32_t)));
    OTOO_CUDA(ctx, cudaMallocHost((void**)&ctx->h_root, 8 * sizeof(float)));
    OTOO_CUDA(ctx, cudaMemset(ctx->d_bbox, 0xFF, 12));                      // bbox_kernel: minima as ordered uints ...
    OTOO_CUDA(ctx, cudaMemset(reinterpret_cast<unsigned*>(ctx->d_bbox) + 3, 0, 16));   // ... maxima, arrival counter (kept so by the kernel)
    OTOO_CUDA(ctx, cudaMemset(ctx->d_counters, 0, 64 * sizeof(uint32_t)));
    OTOO_CUDA(ctx, cudaMemset(ctx->scan_tmp, 0, ctx->scan_cap * sizeof(uint32_t)));   // tile ticket and status words of the scan
    for (auto& e : ctx->ev_build) OTOO_CUDA(ctx, cudaEventCreate(&e));
    for (auto& e : ctx->ev_walk) OTOO_CUDA(ctx, cudaEventCreate(&e));
    return OTOO_OK;
  };
  s = body();
  if (s != OTOO_OK) { otoo_destroy(ctx); return s; }
  *out = ctx;
  return OTOO_OK;
}

void otoo_destroy(otoo_ctx* ctx) {
  if (!ctx) return;
  cudaSetDevice(ctx->device);
  void* ptrs[] = {ctx->key[0], ctx->key[1], ctx->val[0], ctx->val[1], ctx->spos, ctx->slot_nc, ctx->scan_tmp, ctx->hist,
                  ctx->sorted_h, ctx->sorted_aux, ctx->sorted_vel, ctx->sorted_vis, ctx->cell_cm, ctx->cell_b, ctx->c_first, ctx->c_count,
                  ctx->c_child_first, ctx->c_level, ctx->c_child_count, ctx->c_MP, ctx->c_cm64, ctx->c_s, ctx->c_B2, ctx->c_sph,
                  ctx->sph_acc, ctx->tmp_key[0], ctx->tmp_key[1], ctx->tmp_val[0], ctx->tmp_val[1], ctx->d_bbox,
                  ctx->d_counters, ctx->g_ntests, ctx->g_ncells, ctx->g_nparts, ctx->walk_spill, ctx->d_sums,
                  ctx->pool_slots, ctx->pool_seq, ctx->walk_shared, ctx->stage_in, ctx->stage_out,
                  ctx->rec_cells, ctx->rec_count, ctx->rec_ntests};
  for (void* p : ptrs) if (p) cudaFree(p);
  if (ctx->h_counters) cudaFreeHost(ctx->h_counters);
  if (ctx->h_root) cudaFreeHost(ctx->h_root);
  for (auto& e : ctx->ev_build) if (e) cudaEventDestroy(e);
  for (auto& e : ctx->ev_walk) if (e) cudaEventDestroy(e);
  delete ctx;
}

const char* otoo_last_error(const otoo_ctx* ctx) { return ctx ? ctx->err : "null context"; }

otoo_status otoo_build_tree(otoo_ctx* ctx, const float* d_pos_mass, int64_t N, int n_crit, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (N < 0 || n_crit < 1) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "N >= 0 and n_crit >= 1 required");
  if (N > ctx->maxN) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "N exceeds max_particles of otoo_create");
  ctx->launches = 0;
  ctx->last_stream = (cudaStream_t)stream;
  if (N == 0) { ctx->built = false; ctx->walked = false; ctx->N = 0; return OTOO_OK; }
  if (!d_pos_mass) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "d_pos_mass is NULL");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  return otoo_build_impl(ctx, d_pos_mass, N, n_crit, (cudaStream_t)stream);
}

otoo_status otoo_gravity(otoo_ctx* ctx, float eps, float theta, int group_size, float* d_acc_pot, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!(eps >= 0.0f) || !(theta >= 0.0f)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "eps >= 0 and theta >= 0 required");
  if (!valid_group(group_size)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_acc_pot) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "d_acc_pot is NULL");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  ctx->launches = 0; ctx->last_stream = (cudaStream_t)stream;
  return otoo_gravity_impl(ctx, eps, 0, theta, 0.0f, group_size, d_acc_pot, (cudaStream_t)stream);
}

otoo_status otoo_gravity_delta(otoo_ctx* ctx, float eps, float delta, float m_limit, int group_size, float* d_acc_pot,
                               void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!(eps >= 0.0f) || !(delta >= 0.0f) || !(m_limit > 0.0f))
    return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "eps >= 0, delta >= 0 and m_limit > 0 required");
  if (!valid_group(group_size)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_acc_pot) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "d_acc_pot is NULL");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  ctx->launches = 0; ctx->last_stream = (cudaStream_t)stream;
  return otoo_gravity_impl(ctx, eps, 1, delta, m_limit, group_size, d_acc_pot, (cudaStream_t)stream);
}

static otoo_status sph_scratch(otoo_ctx* ctx) {
  if (ctx->out_sorted) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "option output_sorted applies to the gravity calls only");
  if (!ctx->sorted_h) {
    OTOO_TRY(dalloc(ctx, &ctx->sorted_h, (size_t)ctx->maxN));
    OTOO_TRY(dalloc(ctx, &ctx->sorted_aux, (size_t)ctx->maxN));
    OTOO_TRY(dalloc(ctx, &ctx->sorted_vel, (size_t)ctx->maxN));
    OTOO_TRY(dalloc(ctx, &ctx->sorted_vis, (size_t)ctx->maxN));
  }
  return OTOO_OK;
}

otoo_status otoo_sph_density(otoo_ctx* ctx, const float* d_h, int group_size, float* d_rho, uint32_t* d_nngb, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!valid_group(group_size)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_h || !d_rho) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "d_h and d_rho must not be NULL");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  OTOO_TRY(sph_scratch(ctx));
  ctx->launches = 0; ctx->last_stream = (cudaStream_t)stream;
  return otoo_sph_density_impl(ctx, d_h, group_size, d_rho, d_nngb, (cudaStream_t)stream);
}

otoo_status otoo_sph_stage1(otoo_ctx* ctx, const float* d_h, const float* d_vel, int group_size, float* d_rho, uint32_t* d_nngb,
                            float* d_divrot, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!valid_group(group_size)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_h || !d_vel || !d_rho || !d_divrot) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "d_h, d_vel, d_rho, d_divrot must not be NULL");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  OTOO_TRY(sph_scratch(ctx));
  ctx->launches = 0; ctx->last_stream = (cudaStream_t)stream;
  return otoo_sph_stage1_impl(ctx, d_h, d_vel, group_size, d_rho, d_nngb, d_divrot, (cudaStream_t)stream);
}

otoo_status otoo_sph_adapt_h(otoo_ctx* ctx, float* d_h, float n_target, float tol, int max_iter, int group_size,
                             uint32_t* d_nngb, int* host_iters, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!valid_group(group_size)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_h) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "d_h must not be NULL");
  if (!(n_target >= 1.0f) || !(tol >= 0.0f) || max_iter < 0)
    return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "n_target >= 1, tol >= 0, max_iter >= 0 required");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  OTOO_TRY(sph_scratch(ctx));
  ctx->launches = 0; ctx->last_stream = (cudaStream_t)stream;
  return otoo_sph_adapt_h_impl(ctx, d_h, n_target, tol, max_iter, group_size, d_nngb, host_iters, (cudaStream_t)stream);
}

otoo_status otoo_sph_force(otoo_ctx* ctx, const float* d_h, const float* d_rho, const float* d_P, const float* d_vel,
                           int group_size, float* d_acc_sph, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!valid_group(group_size)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_h || !d_rho || !d_P || !d_acc_sph) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "NULL argument");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  OTOO_TRY(sph_scratch(ctx));
  ctx->launches = 0; ctx->last_stream = (cudaStream_t)stream;
  return otoo_sph_force_impl(ctx, d_h, d_rho, d_P, d_vel, nullptr, group_size, d_acc_sph, (cudaStream_t)stream);
}

otoo_status otoo_sph_force_visc(otoo_ctx* ctx, const float* d_h, const float* d_rho, const float* d_P, const float* d_vel,
                                const float* d_visc, int group_size, float* d_acc_sph, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!valid_group(group_size)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_size must be 4, 8, 16, 32, 64, 128 or 256");
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_h || !d_rho || !d_P || !d_vel || !d_visc || !d_acc_sph) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "NULL argument");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  OTOO_TRY(sph_scratch(ctx));
  ctx->launches = 0; ctx->last_stream = (cudaStream_t)stream;
  return otoo_sph_force_impl(ctx, d_h, d_rho, d_P, d_vel, d_visc, group_size, d_acc_sph, (cudaStream_t)stream);
}

otoo_status otoo_eos_ideal(otoo_ctx* ctx, const float* d_rho, const float* d_u, float gamma, int64_t N, float* d_P, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (N < 0 || !(gamma > 1.0f)) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "N >= 0 and gamma > 1 required");
  if (N == 0) return OTOO_OK;
  if (!d_rho || !d_u || !d_P) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "NULL argument");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  eos_ideal_kernel<<<(unsigned)cdiv(N, 256), 256, 0, (cudaStream_t)stream>>>(d_rho, d_u, gamma - 1.0f, N, d_P);
  ctx->launches = 1;
  OTOO_CUDA(ctx, cudaGetLastError());
  return OTOO_OK;
}

otoo_status otoo_unsort(otoo_ctx* ctx, const float* d_sorted_rows, float* d_out, void* stream) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  if (!d_sorted_rows || !d_out || d_sorted_rows == d_out) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "two distinct non-NULL buffers required");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  unsort4_kernel<<<(unsigned)cdiv(ctx->N, 256), 256, 0, (cudaStream_t)stream>>>(reinterpret_cast<const float4*>(d_sorted_rows), ctx->val[0],
                                                                               ctx->N, reinterpret_cast<float4*>(d_out));
  ctx->launches = 1; ctx->last_stream = (cudaStream_t)stream;
  OTOO_CUDA(ctx, cudaGetLastError());
  return OTOO_OK;
}

otoo_status otoo_tree_info(otoo_ctx* ctx, otoo_tree_info_t* o) {
  if (!ctx || !o) return OTOO_ERR_INVALID_ARG;
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  OTOO_CUDA(ctx, cudaStreamSynchronize(ctx->last_stream));
  ctx->N_leaf = ctx->h_counters[32];
  o->N = ctx->N; o->N_cell = ctx->N_cell; o->N_leaf = ctx->N_leaf; o->depth = ctx->depth;
  for (int k = 0; k < 3; k++) o->lo[k] = ctx->lo[k];
  o->S = ctx->S;
  return OTOO_OK;
}

otoo_status otoo_export_tree(otoo_ctx* ctx, uint32_t* d_perm, uint64_t* d_keys, otoo_cell_t* d_cells, float* d_com_m, float* d_rb2) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!ctx->built) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "otoo_build_tree has not succeeded");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->last_stream;
  const unsigned nbC = (unsigned)cdiv(ctx->N_cell, 256);
  if (d_perm) OTOO_CUDA(ctx, cudaMemcpyAsync(d_perm, ctx->val[0], 4 * (size_t)ctx->N, cudaMemcpyDeviceToDevice, st));
  if (d_keys) OTOO_CUDA(ctx, cudaMemcpyAsync(d_keys, ctx->key[0], 8 * (size_t)ctx->N, cudaMemcpyDeviceToDevice, st));
  if (d_cells)
    export_cells_kernel<<<nbC, 256, 0, st>>>(ctx->N_cell, ctx->c_first, ctx->c_count, ctx->c_child_first, ctx->c_level,
                                             ctx->c_child_count, ctx->key[0], d_cells);
  if (d_com_m) OTOO_CUDA(ctx, cudaMemcpyAsync(d_com_m, ctx->cell_cm, 16 * (size_t)ctx->N_cell, cudaMemcpyDeviceToDevice, st));
  if (d_rb2) export_rb2_kernel<<<nbC, 256, 0, st>>>(ctx->N_cell, ctx->cell_b, d_rb2);
  OTOO_CUDA(ctx, cudaGetLastError());
  OTOO_CUDA(ctx, cudaStreamSynchronize(st));
  return OTOO_OK;
}

otoo_status otoo_export_sph_radii(otoo_ctx* ctx, float* d_bmax, float* d_rsph) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!ctx->built || !ctx->sph_radii_valid) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "no SPH call since the last build");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  export_sph_kernel<<<(unsigned)cdiv(ctx->N_cell, 256), 256, 0, ctx->last_stream>>>(ctx->N_cell, ctx->c_sph, d_bmax, d_rsph);
  OTOO_CUDA(ctx, cudaGetLastError());
  OTOO_CUDA(ctx, cudaStreamSynchronize(ctx->last_stream));
  return OTOO_OK;
}

otoo_status otoo_export_group_stats(otoo_ctx* ctx, uint32_t* d_ntests, uint32_t* d_ncells, uint32_t* d_nparts) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (!ctx->built || !ctx->walked) return otoo_fail(ctx, OTOO_ERR_NOT_BUILT, "no walk since the last build");
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->last_stream;
  size_t b = 4 * (size_t)ctx->last_ngroups;
  if (d_ntests) OTOO_CUDA(ctx, cudaMemcpyAsync(d_ntests, ctx->g_ntests, b, cudaMemcpyDeviceToDevice, st));
  if (d_ncells) OTOO_CUDA(ctx, cudaMemcpyAsync(d_ncells, ctx->g_ncells, b, cudaMemcpyDeviceToDevice, st));
  if (d_nparts) OTOO_CUDA(ctx, cudaMemcpyAsync(d_nparts, ctx->g_nparts, b, cudaMemcpyDeviceToDevice, st));
  unsigned long long flag = 0;
  OTOO_CUDA(ctx, cudaMemcpyAsync(&flag, ctx->d_sums + 7, sizeof flag, cudaMemcpyDeviceToHost, st));
  OTOO_CUDA(ctx, cudaStreamSynchronize(st));
  if (flag) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "the last walk overflowed its private spill area: results invalid");
  return OTOO_OK;
}

otoo_status otoo_last_stats(otoo_ctx* ctx, otoo_stats_t* o) {
  if (!ctx || !o) return OTOO_ERR_INVALID_ARG;
  memset(o, 0, sizeof *o);
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  OTOO_CUDA(ctx, cudaStreamSynchronize(ctx->last_stream));
  if (ctx->walked) {
    unsigned long long h[OTOO_NSUMS];
    OTOO_CUDA(ctx, cudaMemcpy(h, ctx->d_sums, sizeof h, cudaMemcpyDeviceToHost));
    if (h[9]) o->walk_sm_mhz = (float)(1e3 * (double)h[8] / (double)h[9]);
    if (h[12]) o->eval_wait_frac = (float)((double)h[10] / (double)h[12]);
    if (h[13]) { o->walker_wait_frac = (float)((double)h[11] / (double)h[13]); o->walker_idle_frac = (float)((double)h[14] * 0.4e-6 * 1e9 * (h[9] ? (double)h[8] / (double)h[9] : 1.965) / (double)h[13]); }
    o->sum_tests = h[0]; o->sum_interactions = h[1]; o->sum_cells = h[2]; o->sum_parts = h[3];
    o->sum_steps = h[4]; o->sum_tasks = h[5]; o->sum_flushes = h[6]; o->sum_evaluated = h[15];
    o->error_flag = (int32_t)h[7];
    o->n_groups = ctx->last_ngroups; o->group_size = ctx->last_group_size;
    o->walk_only = ctx->last_walk_only;
  }
  o->launches = ctx->launches;
  // per-phase device times; events of other streams than last_stream have completed too if the caller kept to
  // one stream per context (the convention of otoo.h)
  if (ctx->ev_build_valid) {
    for (int p = 0; p < OTOO_BUILD_PHASES; p++)
      if (cudaEventElapsedTime(&o->ms_build[p], ctx->ev_build[p], ctx->ev_build[p + 1]) != cudaSuccess) { o->ms_build[p] = 0.0f; cudaGetLastError(); }
    for (int p = 0; p < OTOO_BUILD_PHASES; p++) o->ms_build_total += o->ms_build[p];
  }
  if (ctx->ev_walk_valid) {
    float a = 0.0f, b = 0.0f;
    if (cudaEventElapsedTime(&a, ctx->ev_walk[0], ctx->ev_walk[1]) == cudaSuccess &&
        cudaEventElapsedTime(&b, ctx->ev_walk[1], ctx->ev_walk[2]) == cudaSuccess) {
      o->ms_walk_prep = a; o->ms_walk_force = b; o->ms_total = a + b;
    } else cudaGetLastError();
  }
  if (o->error_flag) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "the last walk overflowed its private spill area: results invalid");
  return OTOO_OK;
}

otoo_status otoo_measure_fp32_peak(otoo_ctx* ctx, double* host_tflops, void* stream) {
  if (!ctx || !host_tflops) return OTOO_ERR_INVALID_ARG;
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  return otoo_measure_fp32_peak_impl(ctx, host_tflops, (cudaStream_t)stream);
}

otoo_status otoo_set_option(otoo_ctx* ctx, const char* name, int64_t value) {
  if (!ctx || !name) return OTOO_ERR_INVALID_ARG;
  if (strcmp(name, "walk_stack") == 0) {
    if (value < 512 || value > OTOO_WALK_STACK_MAX) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "walk_stack out of range");
    ctx->walk_stack = (int)value;
    return OTOO_OK;
  }
  if (strcmp(name, "walk_spill") == 0) {
    if (value < 0 || value > OTOO_WALK_SPILL) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "walk_spill out of range");
    ctx->walk_spill_cap = (int)value;
    return OTOO_OK;
  }
  if (strcmp(name, "task_pool") == 0) { ctx->use_pool = value != 0; return OTOO_OK; }
  if (strcmp(name, "key_order") == 0) {
    if (value != 0 && value != 1) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "key_order must be 0 (Morton) or 1 (Hilbert)");
    ctx->key_order = (int)value;
    return OTOO_OK;
  }
  if (strcmp(name, "group_begin") == 0) {
    if (value < 0) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_begin must be >= 0");
    ctx->group_begin = value;
    return OTOO_OK;
  }
  if (strcmp(name, "group_count") == 0) { ctx->group_count = value < 0 ? -1 : value; return OTOO_OK; }
  if (strcmp(name, "group_distance") == 0) {
    if (value < 0 || value > 2) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "group_distance must be 0 (one box), 1 (exact minimum) or 2 (pieces' boxes)");
    ctx->dist_kind = (int)value;
    return OTOO_OK;
  }
  if (strcmp(name, "sph_reuse_radii") == 0) { ctx->sph_reuse = value != 0; return OTOO_OK; }
  if (strcmp(name, "sph_reuse_walk") == 0) { ctx->sph_reuse_walk = value != 0; return OTOO_OK; }
  if (strcmp(name, "output_sorted") == 0) { ctx->out_sorted = value != 0; return OTOO_OK; }
  if (strcmp(name, "walk_only") == 0) { ctx->walk_only = value != 0; return OTOO_OK; }
  if (strcmp(name, "walk_profile") == 0) { ctx->walk_profile = value != 0; return OTOO_OK; }
  if (strcmp(name, "warp_specialized") == 0) { ctx->use_ws = value != 0; return OTOO_OK; }
  if (strcmp(name, "warp_specialized_sph") == 0) { ctx->use_ws_sph = value != 0; return OTOO_OK; }
  return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "unknown option");
}

static otoo_status gravity_host_impl(otoo_ctx* ctx, const float* h_pos_mass, int64_t N, int n_crit, float eps, int mac, float p0,
                                     float p1, int group_size, float* h_acc_pot) {
  if (!ctx) return OTOO_ERR_INVALID_ARG;
  if (N < 0 || !h_pos_mass || !h_acc_pot) return otoo_fail(ctx, OTOO_ERR_INVALID_ARG, "NULL host buffer or N < 0");
  if (N > ctx->maxN) return otoo_fail(ctx, OTOO_ERR_CAPACITY, "N exceeds max_particles of otoo_create");
  if (N == 0) return OTOO_OK;
  OTOO_CUDA(ctx, cudaSetDevice(ctx->device));
  // context-owned staging buffers (grow-only: no allocation on the repeated call of a time-step loop)
  if (N > ctx->stage_cap) {
    if (ctx->stage_in) cudaFree(ctx->stage_in);
    if (ctx->stage_out) cudaFree(ctx->stage_out);
    ctx->stage_in = ctx->stage_out = nullptr; ctx->stage_cap = 0;
    if (cudaMalloc((void**)&ctx->stage_in, 16 * (size_t)N) != cudaSuccess ||
        cudaMalloc((void**)&ctx->stage_out, 16 * (size_t)N) != cudaSuccess) {
      if (ctx->stage_in) cudaFree(ctx->stage_in);
      ctx->stage_in = nullptr;
      cudaGetLastError();
      return otoo_fail(ctx, OTOO_ERR_OOM, "staging allocation failed");
    }
    ctx->stage_cap = N;
  }
  float4 *d_in = ctx->stage_in, *d_out = ctx->stage_out;
  otoo_status s = OTOO_OK;
  cudaStream_t st = 0;
  if (cudaMemcpyAsync(d_in, h_pos_mass, 16 * (size_t)N, cudaMemcpyHostToDevice, st) != cudaSuccess) s = otoo_fail(ctx, OTOO_ERR_CUDA, "H2D copy failed");
  if (s == OTOO_OK) s = otoo_build_tree(ctx, reinterpret_cast<const float*>(d_in), N, n_crit, st);
  int l1 = ctx->launches;
  if (s == OTOO_OK)
    s = mac == 0 ? otoo_gravity(ctx, eps, p0, group_size, reinterpret_cast<float*>(d_out), st)
                 : otoo_gravity_delta(ctx, eps, p0, p1, group_size, reinterpret_cast<float*>(d_out), st);
  ctx->launches += l1;
  if (s == OTOO_OK && cudaMemcpyAsync(h_acc_pot, d_out, 16 * (size_t)N, cudaMemcpyDeviceToHost, st) != cudaSuccess) s = otoo_fail(ctx, OTOO_ERR_CUDA, "D2H copy failed");
  if (s == OTOO_OK && cudaStreamSynchronize(st) != cudaSuccess) s = otoo_fail(ctx, OTOO_ERR_CUDA, "synchronize failed");
  return s;
}

otoo_status otoo_gravity_host(otoo_ctx* ctx, const float* h_pos_mass, int64_t N, int n_crit, float eps, float theta,
                              int group_size, float* h_acc_pot) {
  return gravity_host_impl(ctx, h_pos_mass, N, n_crit, eps, 0, theta, 0.0f, group_size, h_acc_pot);
}
otoo_status otoo_gravity_delta_host(otoo_ctx* ctx, const float* h_pos_mass, int64_t N, int n_crit, float eps, float delta,
                                    float m_limit, int group_size, float* h_acc_pot) {
  return gravity_host_impl(ctx, h_pos_mass, N, n_crit, eps, 1, delta, m_limit, group_size, h_acc_pot);
}

}  // extern "C"
