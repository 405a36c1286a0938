// keys.cuh -- quantisation and key construction (PAPER.md III-B step 2, L129-L131; readings R2, R3, R20), shared by the
// key + histogram kernel (sort.cu) and the cell geometry of the bottom-up pass (build.cu).
#pragma once
#include "common.cuh"

namespace {

__device__ __forceinline__ uint64_t dilate3(uint32_t v) {
  uint64_t x = v & 0x1FFFFFu;
  x = (x | x << 32) & 0x001F00000000FFFFull;
  x = (x | x << 16) & 0x001F0000FF0000FFull;
  x = (x | x << 8) & 0x100F00F00F00F00Full;
  x = (x | x << 4) & 0x10C30C30C30C30C3ull;
  x = (x | x << 2) & 0x1249249249249249ull;
  return x;
}
__device__ __forceinline__ uint32_t compact3(uint64_t x) {
  x &= 0x1249249249249249ull;
  x = (x | x >> 2) & 0x10C30C30C30C30C3ull;
  x = (x | x >> 4) & 0x100F00F00F00F00Full;
  x = (x | x >> 8) & 0x001F0000FF0000FFull;
  x = (x | x >> 16) & 0x001F00000000FFFFull;
  x = (x | x >> 32) & 0x1FFFFFull;
  return (uint32_t)x;
}
// Hilbert order (reading R20): Skilling's transpose form of the 3-D Hilbert curve on the 21-bit
// quantised coordinates, x the most significant axis.  The key is the interleave of the transformed
// coordinates, so its top 3l bits still name the level-l octree cell.
__device__ __forceinline__ void hilbert_axes_to_transpose(uint32_t& x, uint32_t& y, uint32_t& z) {
  uint32_t X[3] = {x, y, z};
  for (uint32_t Q = 1u << (OTOO_MAXLEV - 1); Q > 1; Q >>= 1) {
    const uint32_t P = Q - 1;
#pragma unroll
    for (int i = 0; i < 3; i++) {
      if (X[i] & Q) X[0] ^= P;
      else { const uint32_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
    }
  }
  X[1] ^= X[0]; X[2] ^= X[1];
  uint32_t t = 0;
  for (uint32_t Q = 1u << (OTOO_MAXLEV - 1); Q > 1; Q >>= 1) if (X[2] & Q) t ^= Q - 1;
  x = X[0] ^ t; y = X[1] ^ t; z = X[2] ^ t;
}
__device__ __forceinline__ void hilbert_transpose_to_axes(uint32_t& x, uint32_t& y, uint32_t& z) {
  uint32_t X[3] = {x, y, z};
  uint32_t t = X[2] >> 1;
  X[2] ^= X[1]; X[1] ^= X[0]; X[0] ^= t;
  for (uint32_t Q = 2; Q != (2u << (OTOO_MAXLEV - 1)); Q <<= 1) {
    const uint32_t P = Q - 1;
#pragma unroll
    for (int i = 2; i >= 0; i--) {
      if (X[i] & Q) X[0] ^= P;
      else { t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
    }
  }
  x = X[0]; y = X[1]; z = X[2];
}
__device__ __forceinline__ uint32_t quant(float x, float lo, float scale) {
  float t = __fmul_rn(__fsub_rn(x, lo), scale);
  return (t >= 2097151.0f) ? 2097151u : (t > 0.0f ? __float2uint_rz(t) : 0u);
}
// H2 (L129; R2, R3): the 63-bit key of one particle: Morton by bit dilation, x most significant in each octant, or the
// Hilbert transform of the quantised coordinates first (R20).  root = lo.xyz, S, scale as the bbox kernel left them.
__device__ __forceinline__ uint64_t particle_key(const float4 p, const float* __restrict__ root, int hilbert) {
  const float scale = root[4];
  uint32_t qx = quant(p.x, root[0], scale), qy = quant(p.y, root[1], scale), qz = quant(p.z, root[2], scale);
  if (hilbert) hilbert_axes_to_transpose(qx, qy, qz);
  return (dilate3(qx) << 2) | (dilate3(qy) << 1) | dilate3(qz);
}

}  // namespace
