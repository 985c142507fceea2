// emm_device.cuh -- device helpers shared by the update kernels (emm_kernels.cu, emm_tile.cu): 128-bit accesses, the
// 4-node x derivative from a 12-wide window, the CPML recursion on a quad.
#pragma once
#include "emm_kernels.cuh"

namespace emm {

__device__ __forceinline__ float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void st4(float *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }
__device__ __forceinline__ float4 ldcs4(const float *p) { return __ldcs(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ void stcs4(float *p, float4 v) { __stcs(reinterpret_cast<float4 *>(p), v); }
__device__ __forceinline__ float4 zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ float4 fma4(float a, float4 b, float4 c) {
  return make_float4(fmaf(a, b.x, c.x), fmaf(a, b.y, c.y), fmaf(a, b.z, c.z), fmaf(a, b.w, c.w));
}
__device__ __forceinline__ float4 sub4(float4 a, float4 b) { return make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w); }
__device__ __forceinline__ float4 add4(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }

// slab index along an axis of length N (L317-333): low slab i < nb -> i, high slab -> nb + (N-1-i)
__device__ __forceinline__ int slab_of(int i, int N, int nb, int has_lo) {
  if (i < nb) return has_lo ? i : -1;
  if (i > N - 1 - nb) return nb + (N - 1 - i);
  return -1;
}

// x derivative of 4 nodes from a 12-wide window w[] holding nodes i0-4 .. i0+7; tap m of node n sits at
// i0+n-R+XO+m, i.e. window slot 4+n-R+XO+m.
template <int R, int XO>
__device__ __forceinline__ float4 ddx(const float (&w)[12], const float (&cx)[4][2 * R]) {
  float d[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) {
    float acc = 0.f;
#pragma unroll
    for (int m = 0; m < 2 * R; ++m) acc = fmaf(cx[n][m], w[4 + n - R + XO + m], acc);
    d[n] = acc;
  }
  return make_float4(d[0], d[1], d[2], d[3]);
}

__device__ __forceinline__ void window(float (&w)[12], float4 l, float4 c, float4 r) {
  w[0] = l.x; w[1] = l.y; w[2] = l.z; w[3] = l.w;
  w[4] = c.x; w[5] = c.y; w[6] = c.z; w[7] = c.w;
  w[8] = r.x; w[9] = r.y; w[10] = r.z; w[11] = r.w;
}

// CPML recursion on a quad: psi <- b psi + a D ; D <- D + psi  (Eq. 22-23 with kappa = 1, L317-333)
__device__ __forceinline__ void cpml4(float *psi, float a, float b, float4 &D) {
  float4 p = ld4(psi);
  p = make_float4(fmaf(b, p.x, a * D.x), fmaf(b, p.y, a * D.y), fmaf(b, p.z, a * D.z), fmaf(b, p.w, a * D.w));
  st4(psi, p);
  D = add4(D, p);
}

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

}  // namespace emm
