// emm_air_cluster.cu -- the air-water boundary (Eq. 17-21; [R10]) of a uniform x-y grid as ONE launch
// per pass: a thread-block cluster holds the whole FFT plane in its distributed shared memory and runs pack, forward 2-D
// transform, the spectral filters of every ghost level, the inverse transforms and the write-back without leaving the
// chip (hand-written batched FFT with fused spectral scaling, one launch per boundary condition).
//
// The library route (emm_air.cu) is pack -> 2-D cuFFT -> filter -> batched inverse 2-D cuFFT -> unpack: eight dependent
// launches of a few microseconds each per pass on the planes this route is for (cfg2: 168 x 168), i.e. a chain bound by
// launch latency, not by bytes or flops.  Here:
//
//   CTA c of the C-CTA cluster owns rows [c*rpc, (c+1)*rpc) of the plane: loads them from the surface plane (Ex + i Ey, or
//   Hz), transforms them along x in shared memory;
//   sends every element to the CTA that owns its column [c*cpc, (c+1)*cpc) with stores into that CTA's shared memory (the
//   transpose through distributed shared memory);                                              cluster barrier
//   transforms its columns along y: the 2-D spectrum, one column block per CTA, kept for all levels;
//   per ghost level: multiplies by the filter of that level (Eq. 21 for E; Eq. 17-20 with the half-cell phase factors for
//   H), inverse transform along y, sends every element back to the CTA that owns its row;       cluster barrier
//   inverse transform along x, real part -> component 1, imaginary part -> component 2 of the ghost plane.
//
// Transforms: Stockham autosort passes of radix 8, 4, 2, 3, 5, 7 (every plane size is 7-smooth, [R1]) between two
// shared-memory buffers, one butterfly per thread and pass, twiddles e^{-2 pi i k/M} from a table computed in fp64 on
// the host.  Only forward transforms exist: the inverse 2-D transform of X is the conjugate of the forward transform of
// conj(X), so the filter stores conjugates and the write-back takes -Im (half the code: the kernel is bound by latency
// and instruction fetch, not by flops).  The ghost levels are filtered and transformed together, as many at a time as
// the shared memory holds (more lines per pass: more threads busy).  Same arithmetic type (fp32) and the same filters
// as the library route; results agree with it to rounding.  One cluster per source; sources are independent.
#include <cooperative_groups.h>

#include "emm_kernels.cuh"

namespace cg = cooperative_groups;

namespace emm {
namespace {

constexpr int kClThreads = 512;
constexpr int kMaxPass = 20;

// n / d for n * d < 2^32 as one multiply-high (the index decodes of the butterfly and transpose loops)
struct FastDiv { unsigned d, m; };
__host__ inline FastDiv make_fastdiv(int d) { return FastDiv{(unsigned)d, d > 1 ? (unsigned)(0x100000000ull / (unsigned)d + 1ull) : 0u}; }
__device__ __forceinline__ unsigned fdiv(unsigned n, const FastDiv f) { return f.d == 1 ? n : __umulhi(n, f.m); }

struct ClusterArgs {
  int M1, M2, P1, k0, nlev, is_h, LG;   // LG: ghost levels filtered and transformed together
  int C, rpc, cpc, ld1, ld2;            // cluster size, rows / columns per CTA, line pitches (odd: bank spread of the transposes)
  long long PS, VS;
  float h[kMaxR];
  float dx, dy, scale;
  int np1, np2;
  unsigned char rad1[kMaxPass], rad2[kMaxPass];
  FastDiv nb1[kMaxPass], st1[kMaxPass], nb2[kMaxPass], st2[kMaxPass];   // per pass: butterflies per line, sub-transform stride
  FastDiv dM1, dM2, drpc, dcpc;
  const float2 *tw1, *tw2;
  const float *kx, *ky;
  const float *f_in1, *f_in2;
  float *f_o1, *f_o2;
};

__device__ __forceinline__ float2 cadd(const float2 a, const float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(const float2 a, const float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(const float2 a, const float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 mulmi(const float2 a) { return make_float2(a.y, -a.x); }   // -i a

// cos / sin of 2 pi m / P for the odd radices
__host__ __device__ constexpr float kCos(int P, int m) {
  m = m % P;
  if (m > P - m) m = P - m;
  if (P == 3) return m == 0 ? 1.f : -0.5f;
  if (P == 5) return m == 0 ? 1.f : m == 1 ? 0.30901699437494745f : -0.80901699437494734f;
  if (P == 7) return m == 0 ? 1.f : m == 1 ? 0.62348980185873348f : m == 2 ? -0.22252093395631439f : -0.90096886790241915f;
  return 0.f;
}
__host__ __device__ constexpr float kSin(int P, int m) {
  m = m % P;
  float sg = 1.f;
  if (m > P - m) { m = P - m; sg = -1.f; }
  if (P == 3) return sg * (m == 0 ? 0.f : 0.86602540378443860f);
  if (P == 5) return sg * (m == 0 ? 0.f : m == 1 ? 0.95105651629515353f : 0.58778525229247314f);
  if (P == 7) return sg * (m == 0 ? 0.f : m == 1 ? 0.78183148246802980f : m == 2 ? 0.97492791218182362f : 0.43388373911755812f);
  return 0.f;
}

__device__ __forceinline__ void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
  const float2 s0 = cadd(a0, a2), d0 = csub(a0, a2), s1 = cadd(a1, a3), jd = mulmi(csub(a1, a3));
  a0 = cadd(s0, s1);
  a2 = csub(s0, s1);
  a1 = cadd(d0, jd);
  a3 = csub(d0, jd);
}

// in-place forward DFT of P points, kernel e^{-2 pi i jk/P}
template <int P>
__device__ __forceinline__ void dft(float2 (&a)[P]) {
  if constexpr (P == 2) {
    const float2 t = a[0];
    a[0] = cadd(t, a[1]);
    a[1] = csub(t, a[1]);
  } else if constexpr (P == 4) {
    dft4(a[0], a[1], a[2], a[3]);
  } else if constexpr (P == 8) {
    dft4(a[0], a[2], a[4], a[6]);
    dft4(a[1], a[3], a[5], a[7]);
    constexpr float h = 0.70710678118654752f;
    const float2 o1 = make_float2(h * (a[3].x + a[3].y), h * (a[3].y - a[3].x));     // w8   a3, w8 = (1 - i)/sqrt 2
    const float2 o2 = mulmi(a[5]);                                                   // w8^2 a5
    const float2 o3 = make_float2(h * (a[7].y - a[7].x), -h * (a[7].x + a[7].y));    // w8^3 a7 = (-1 - i)/sqrt 2 a7
    const float2 e0 = a[0], e1 = a[2], e2 = a[4], e3 = a[6], o0 = a[1];
    a[0] = cadd(e0, o0); a[4] = csub(e0, o0);
    a[1] = cadd(e1, o1); a[5] = csub(e1, o1);
    a[2] = cadd(e2, o2); a[6] = csub(e2, o2);
    a[3] = cadd(e3, o3); a[7] = csub(e3, o3);
  } else {
    constexpr int H = (P - 1) / 2;
    float2 s[H + 1], d[H + 1];
#pragma unroll
    for (int k = 1; k <= H; ++k) { s[k] = cadd(a[k], a[P - k]); d[k] = csub(a[k], a[P - k]); }
    float2 o[P];
    o[0] = a[0];
#pragma unroll
    for (int k = 1; k <= H; ++k) o[0] = cadd(o[0], s[k]);
#pragma unroll
    for (int j = 1; j <= H; ++j) {
      float2 A = a[0], B = make_float2(0.f, 0.f);
#pragma unroll
      for (int k = 1; k <= H; ++k) {
        const float c = kCos(P, j * k), sn = kSin(P, j * k);
        A.x = fmaf(c, s[k].x, A.x); A.y = fmaf(c, s[k].y, A.y);
        B.x = fmaf(sn, d[k].x, B.x); B.y = fmaf(sn, d[k].y, B.y);
      }
      const float2 iB = mulmi(B);            // a_k w^{jk} + a_{P-k} w^{-jk} = s_k cos - i d_k sin
      o[j] = cadd(A, iB);
      o[P - j] = csub(A, iB);
    }
#pragma unroll
    for (int j = 0; j < P; ++j) a[j] = o[j];
  }
}

// The dynamic shared memory of the CTA as complex numbers.  The transform routines address it by offsets from this symbol,
// not through pointers handed across the call: the compiler then emits shared-memory loads and stores (LDS / STS)
// instead of generic ones.
extern __shared__ __align__(16) float2 g_sm[];

// one Stockham pass of radix P over `nlines` lines of length N = P * nb (pitch ld): sub-transform stride s, x -> y
// (xo, yo, two: offsets into g_sm)
template <int P>
__device__ __forceinline__ void fft_pass(unsigned xo, unsigned yo_, const FastDiv nb, const FastDiv s, int nlines, int ld, unsigned two) {
  const float2 *__restrict__ x = g_sm + xo;
  float2 *__restrict__ y = g_sm + yo_;
  const float2 *__restrict__ tw = g_sm + two;
  const unsigned ntask = (unsigned)nlines * nb.d;
  for (unsigned t = threadIdx.x; t < ntask; t += kClThreads) {
    const unsigned line = fdiv(t, nb), b = t - line * nb.d;
    const unsigned base = fdiv(b, s) * s.d, q = b - base;
    const float2 *xi = x + line * ld + b;
    float2 a[P];
#pragma unroll
    for (int k = 0; k < P; ++k) a[k] = xi[k * nb.d];
    dft<P>(a);
    float2 *yo = y + line * ld + q + P * base;
    yo[0] = a[0];
#pragma unroll
    for (int j = 1; j < P; ++j) yo[s.d * j] = cmul(a[j], tw[j * base]);
  }
}

// one pass of a transform: radix, butterflies per line, sub-transform stride (a copy in shared memory: read by every
// thread in every pass)
struct PassTab { unsigned rad; FastDiv nb, st; };

// all passes of a forward 1-D transform over the lines of a block, ping-pong between the buffers at offsets a and b of
// g_sm (the last pass into `last` unless kNone); returns the offset of the buffer that holds the result
constexpr unsigned kNone = 0xffffffffu;
__device__ __noinline__ unsigned fft_lines(unsigned a, unsigned b, unsigned last, int np, unsigned pt_off, int nlines, int ld, unsigned tw) {
  const PassTab *pt = reinterpret_cast<const PassTab *>(g_sm + pt_off);
  unsigned src = a;
  for (int i = 0; i < np; ++i) {
    const unsigned dst = (i == np - 1 && last != kNone) ? last : (src == a ? b : a);
    const PassTab p = pt[i];
    switch (p.rad) {
      case 2: fft_pass<2>(src, dst, p.nb, p.st, nlines, ld, tw); break;
      case 3: fft_pass<3>(src, dst, p.nb, p.st, nlines, ld, tw); break;
      case 4: fft_pass<4>(src, dst, p.nb, p.st, nlines, ld, tw); break;
      case 5: fft_pass<5>(src, dst, p.nb, p.st, nlines, ld, tw); break;
      case 7: fft_pass<7>(src, dst, p.nb, p.st, nlines, ld, tw); break;
      default: fft_pass<8>(src, dst, p.nb, p.st, nlines, ld, tw); break;
    }
    __syncthreads();
    src = dst;
  }
  return src;
}

__global__ void __launch_bounds__(kClThreads, 1) k_air_cluster(const __grid_constant__ ClusterArgs A) {
  cg::cluster_group cluster = cg::this_cluster();
  const int c = (int)cluster.block_rank();
  const int src = blockIdx.x / A.C;
  const unsigned tid = threadIdx.x;
  const int M1 = A.M1, M2 = A.M2, ld1 = A.ld1, ld2 = A.ld2, rpc = A.rpc, cpc = A.cpc;
  // offsets into g_sm (complex numbers)
  const unsigned oTw1 = 0, oTw2 = oTw1 + M1, oS = oTw2 + M2;
  const unsigned oR0 = oS + cpc * ld2, oR1 = oR0 + A.LG * rpc * ld1;
  const unsigned oT0 = oR1 + A.LG * rpc * ld1, oT1 = oT0 + A.LG * cpc * ld2;
  const unsigned oPhx = oT1 + A.LG * cpc * ld2, oPhy = oPhx + cpc;
  const unsigned oPt1 = oPhy + M2, oPt2 = oPt1 + kMaxPass * sizeof(PassTab) / sizeof(float2);
  float2 *tw1 = g_sm + oTw1, *tw2 = g_sm + oTw2, *S = g_sm + oS, *R0 = g_sm + oR0, *T0 = g_sm + oT0;
  float2 *phx = g_sm + oPhx;                               // per column of mine: i kx e^{-i kx dx/2} (H filter, Nyquist bin zeroed)
  float2 *phy = g_sm + oPhy;                               // per row: the same with ky
  PassTab *pt1 = reinterpret_cast<PassTab *>(g_sm + oPt1), *pt2 = reinterpret_cast<PassTab *>(g_sm + oPt2);
  float *kxs = reinterpret_cast<float *>(g_sm + oPt2 + kMaxPass * sizeof(PassTab) / sizeof(float2));
  float *kys = kxs + cpc;
  const int j0 = c * rpc, nrow = max(0, min(rpc, M2 - j0));
  const int i0 = c * cpc, ncol = max(0, min(cpc, M1 - i0));

  // every CTA of the cluster must be running before its shared memory is written from outside: arrive now, wait just
  // before the first remote store (the row transforms in between hide the barrier)
  cluster.barrier_arrive();
  for (unsigned t = tid; t < (unsigned)M1; t += kClThreads) tw1[t] = A.tw1[t];
  for (unsigned t = tid; t < (unsigned)M2; t += kClThreads) {
    tw2[t] = A.tw2[t];
    const float q = A.ky[t];
    kys[t] = q;
    float sn, cs;
    sincosf(-0.5f * q * A.dy, &sn, &cs);
    phy[t] = (((M2 & 1) == 0) && (int)t == M2 / 2) ? make_float2(0.f, 0.f) : make_float2(-sn * q, cs * q);
  }
  for (unsigned t = tid; t < (unsigned)ncol; t += kClThreads) {
    const float q = A.kx[i0 + t];
    kxs[t] = q;
    float sn, cs;
    sincosf(-0.5f * q * A.dx, &sn, &cs);
    phx[t] = (((M1 & 1) == 0) && (int)(i0 + t) == M1 / 2) ? make_float2(0.f, 0.f) : make_float2(-sn * q, cs * q);
  }
  if (tid < (unsigned)A.np1) pt1[tid] = PassTab{A.rad1[tid], A.nb1[tid], A.st1[tid]};
  if (tid >= 32 && tid < 32u + A.np2) pt2[tid - 32] = PassTab{A.rad2[tid - 32], A.nb2[tid - 32], A.st2[tid - 32]};
  {   // the surface plane: Ex + i Ey (E pass) or Hz (H pass)
    const float *f1 = A.f_in1 + (size_t)src * A.VS + (size_t)A.k0 * A.PS;
    const float *f2 = A.f_in2 ? A.f_in2 + (size_t)src * A.VS + (size_t)A.k0 * A.PS : nullptr;
#pragma unroll 4
    for (unsigned t = tid; t < (unsigned)(nrow * M1); t += kClThreads) {
      const unsigned jj = fdiv(t, A.dM1), i = t - jj * M1;
      const size_t o = (size_t)(j0 + jj) * A.P1 + i;
      R0[jj * ld1 + i] = make_float2(f1[o], f2 ? f2[o] : 0.f);
    }
  }
  __syncthreads();
  const float2 *Rres = g_sm + fft_lines(oR0, oR1, kNone, A.np1, oPt1, nrow, ld1, oTw1);
  cluster.barrier_wait();
  // transpose through distributed shared memory: every element of my rows goes to the CTA that owns its column (stores to
  // remote shared memory are not waited for; the cluster barrier publishes them).  T0 is idle everywhere at this point.
#pragma unroll 4
  for (unsigned t = tid; t < (unsigned)(nrow * M1); t += kClThreads) {
    const unsigned jj = fdiv(t, A.dM1), n1 = t - jj * M1;
    const unsigned owner = fdiv(n1, A.dcpc), ii = n1 - owner * cpc;
    float2 *rem = cluster.map_shared_rank(T0, owner);
    rem[ii * ld2 + j0 + jj] = Rres[jj * ld1 + n1];
  }
  cluster.sync();
  fft_lines(oT0, oT1, oS, A.np2, oPt2, ncol, ld2, oTw2);                    // the 2-D spectrum of my columns, kept in S

  for (int g0 = 0; g0 < A.nlev; g0 += A.LG) {
    const int L = min(A.LG, A.nlev - g0);
    // filters of levels g0 .. g0+L-1; conjugates are stored: forward transforms from here on give the conjugate of the inverse
    for (unsigned t = tid; t < (unsigned)(ncol * M2); t += kClThreads) {
      const unsigned ii = fdiv(t, A.dM2), n2 = t - ii * M2;
      float2 v = S[ii * ld2 + n2];
      const float qx = kxs[ii], qy = kys[n2];
      const float kh = sqrtf(qx * qx + qy * qy);
      if (A.is_h) {              // Eq. 17-20: Hx^ = i kx/k_h e^{-k_h h} Hz^ (Hy: ky) with the half-cell phases [R10]; k_h = 0 bin -> 0
        const float2 gx = phx[ii], gy = phy[n2];
        const float rk = kh > 0.f ? 1.f / kh : 0.f;
        v = cmul(v, make_float2((gx.x - gy.y) * rk, (gx.y + gy.x) * rk));    // (gx + i gy)/k_h: spectrum of Hx + i Hy
      }
      for (int l = 0; l < L; ++l) {                                         // Eq. 21: level m = e^{-k_h h_m} x surface spectrum
        const float e = expf(-kh * A.h[g0 + l]) * A.scale;
        T0[(l * ncol + ii) * ld2 + n2] = make_float2(v.x * e, -v.y * e);
      }
    }
    __syncthreads();
    const float2 *Tres = g_sm + fft_lines(oT0, oT1, kNone, A.np2, oPt2, L * ncol, ld2, oTw2);
    // transpose back: every element of my columns goes to the CTA that owns its row; the level blocks of a CTA are packed
    // by its own row count (the last CTA with rows may hold fewer).  R0 is idle everywhere: the forward transpose has been
    // read before the first barrier, and a further group waits for the barrier at the end of this loop.
    for (int l = 0; l < L; ++l) {
#pragma unroll 4
      for (unsigned t = tid; t < (unsigned)(ncol * M2); t += kClThreads) {
        const unsigned ii = fdiv(t, A.dM2), j = t - ii * M2;
        const unsigned owner = fdiv(j, A.drpc), jj = j - owner * rpc;
        const int nrow_owner = min(rpc, M2 - (int)owner * rpc);
        float2 *rem = cluster.map_shared_rank(R0, owner);
        rem[(l * nrow_owner + jj) * ld1 + i0 + ii] = Tres[(l * ncol + ii) * ld2 + j];
      }
    }
    cluster.sync();
    const float2 *Rr = g_sm + fft_lines(oR0, oR1, kNone, A.np1, oPt1, L * nrow, ld1, oTw1);
    for (int l = 0; l < L; ++l) {
      float *o1 = A.f_o1 + (size_t)src * A.VS + (size_t)(A.k0 - 1 - (g0 + l)) * A.PS;
      float *o2 = A.f_o2 + (size_t)src * A.VS + (size_t)(A.k0 - 1 - (g0 + l)) * A.PS;
      for (unsigned t = tid; t < (unsigned)(nrow * M1); t += kClThreads) {
        const unsigned jj = fdiv(t, A.dM1), i = t - jj * M1;
        const float2 v = Rr[(l * nrow + jj) * ld1 + i];
        const size_t o = (size_t)(j0 + jj) * A.P1 + i;
        o1[o] = v.x;                                                         // conjugate of the forward transform of the conjugate
        o2[o] = -v.y;
      }
    }
    if (g0 + A.LG < A.nlev) cluster.sync();                                  // the row blocks are refilled by the next group's transpose
  }
}

// Radices of the passes, odd ones first: a pass with sub-transform stride s stores runs of s consecutive numbers, the first
// pass (s = 1) stores with a stride of its radix: 3, 5 or 7 complex numbers spread over the banks, 8 would hit two of them.
int factor7(int n, unsigned char *rad) {
  int np = 0;
  const int odd[3] = {3, 5, 7};
  for (int p : odd) while (n % p == 0 && np < kMaxPass) { rad[np++] = (unsigned char)p; n /= p; }
  while (n % 8 == 0 && np < kMaxPass) { rad[np++] = 8; n /= 8; }
  const int even[2] = {4, 2};
  for (int p : even) while (n % p == 0 && np < kMaxPass) { rad[np++] = (unsigned char)p; n /= p; }
  return n == 1 ? np : -1;
}

size_t cluster_smem(const emm_grid *g, int C, int LG) {
  const size_t rpc = (g->M2 + C - 1) / C, cpc = (g->M1 + C - 1) / C;
  return sizeof(float2) * ((size_t)g->M1 + g->M2 + cpc * (g->M2 | 1) + 2 * LG * rpc * (g->M1 | 1) + 2 * LG * cpc * (g->M2 | 1) + cpc + g->M2) +
         sizeof(float) * (cpc + g->M2 + 1) + 2 * kMaxPass * sizeof(PassTab) + 16;
}

void cluster_config(const emm_grid *g, int C, int LG, cudaLaunchConfig_t *cfg, cudaLaunchAttribute *at, int nsrc, cudaStream_t st) {
  *cfg = cudaLaunchConfig_t{};
  cfg->gridDim = dim3((unsigned)(C * nsrc), 1, 1);
  cfg->blockDim = dim3(kClThreads, 1, 1);
  cfg->dynamicSmemBytes = cluster_smem(g, C, LG);
  cfg->stream = st;
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)C;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg->attrs = at;
  cfg->numAttrs = 1;
}

}  // namespace

// Cluster size for this grid's plane on the current device, 0 = the plane does not fit (the library route is used).
// Called by emm_bind_device (needs the device).  16 CTAs (non-portable size) when the device schedules such a cluster,
// else 8; per CTA: the twiddle tables, its block of the spectrum, and two row blocks and two column blocks for each of
// the LG ghost levels in flight (LG = all r levels if they fit, else fewer).
int air_cluster_plan(emm_grid *g) {
  g->air_cluster = 0;
  g->air_cluster_lg = 0;
  if (g->top != EMM_TOP_AIR || !g->uniform_xy || g->air_route == 1) return 0;
  if (g->M1 != g->N[0] || g->M2 != g->N[1]) return 0;
  unsigned char rad[kMaxPass];
  if (g->M1 > 4096 || g->M2 > 4096 || factor7(g->M1, rad) < 0 || factor7(g->M2, rad) < 0) return 0;
  int dev = 0, smem_max = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) {
    cudaGetLastError();
    return 0;
  }
  const int sizes[2] = {16, 8};
  for (int C : sizes)
    for (int LG = g->r; LG >= 1; --LG) {
      const size_t bytes = cluster_smem(g, C, LG);
      if (bytes > (size_t)smem_max) continue;
      if (cudaFuncSetAttribute(k_air_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) { cudaGetLastError(); continue; }
      if (C > 8 && cudaFuncSetAttribute(k_air_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) { cudaGetLastError(); continue; }
      cudaLaunchConfig_t cfg;
      cudaLaunchAttribute at[1];
      cluster_config(g, C, LG, &cfg, at, 1, nullptr);
      int n = 0;
      if (cudaOccupancyMaxActiveClusters(&n, k_air_cluster, &cfg) != cudaSuccess) { cudaGetLastError(); continue; }
      if (n >= 1) { g->air_cluster = C; g->air_cluster_lg = LG; return C; }
    }
  return 0;
}

int launch_air_cluster(emm_grid *g, const DevState &s, const DevRun &r, int is_h, cudaStream_t st) {
  (void)r;
  const int R = g->r, C = g->air_cluster;
  const int nlev = is_h ? R : R - 1;
  if (nlev <= 0) return 0;
  ClusterArgs a{};
  a.M1 = g->M1; a.M2 = g->M2; a.P1 = g->P1; a.k0 = g->k0; a.nlev = nlev; a.is_h = is_h;
  a.LG = std::min(nlev, g->air_cluster_lg);
  a.C = C;
  a.rpc = (g->M2 + C - 1) / C;
  a.cpc = (g->M1 + C - 1) / C;
  a.ld1 = g->M1 | 1;
  a.ld2 = g->M2 | 1;
  a.PS = g->dg.PS; a.VS = g->dg.VS;
  for (int m = 1; m <= nlev; ++m)
    a.h[m - 1] = (float)(is_h ? g->xn[2][g->k0] - g->xh[2][g->k0 - m] : g->xn[2][g->k0] - g->xn[2][g->k0 - m]);
  a.dx = (float)g->dxa; a.dy = (float)g->dya;
  a.scale = (float)(1.0 / ((double)g->M1 * (double)g->M2));
  a.np1 = factor7(g->M1, a.rad1);
  a.np2 = factor7(g->M2, a.rad2);
  for (int q = 0, st_ = 1; q < a.np1; st_ *= a.rad1[q], ++q) { a.nb1[q] = make_fastdiv(g->M1 / a.rad1[q]); a.st1[q] = make_fastdiv(st_); }
  for (int q = 0, st_ = 1; q < a.np2; st_ *= a.rad2[q], ++q) { a.nb2[q] = make_fastdiv(g->M2 / a.rad2[q]); a.st2[q] = make_fastdiv(st_); }
  a.dM1 = make_fastdiv(g->M1); a.dM2 = make_fastdiv(g->M2); a.drpc = make_fastdiv(a.rpc); a.dcpc = make_fastdiv(a.cpc);
  a.tw1 = g->T.tw1; a.tw2 = g->T.tw2;
  a.kx = g->T.kx; a.ky = g->T.ky;
  a.f_in1 = is_h ? s.H[2] : s.E[0];
  a.f_in2 = is_h ? nullptr : s.E[1];
  a.f_o1 = is_h ? s.H[0] : s.E[0];
  a.f_o2 = is_h ? s.H[1] : s.E[1];
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute at[1];
  cluster_config(g, C, g->air_cluster_lg, &cfg, at, s.nsrc, st);
  // per device attributes: set at every launch (cheap; a second device in the process has its own copy of the function)
  cudaError_t e = cudaFuncSetAttribute(k_air_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.dynamicSmemBytes);
  if (e == cudaSuccess && C > 8) e = cudaFuncSetAttribute(k_air_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e == cudaSuccess) e = cudaLaunchKernelEx(&cfg, k_air_cluster, a);
  if (e != cudaSuccess) return fail(EMM_ECUDA, "k_air_cluster launch: %s", cudaGetErrorString(e));
  g->launches++;
  return 0;
}

}  // namespace emm
