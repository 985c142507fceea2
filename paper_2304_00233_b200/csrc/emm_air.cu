// emm_air.cu -- plane kernels of the air-water boundary (Eq. 17-21) and the
// device-side effective-medium pass of emm_model_set (Eq. 26).
//
// Air boundary.  The paper runs 9 FFTs and 15 small kernels per step (Fig. 10).  Here the two
// tangential components are packed into ONE complex plane (Ex + i Ey, and Hx + i Hy on the way back):
// every spectral filter used is the transform of a real kernel (the Nyquist bins of the odd filters are
// zeroed, [R10]), so real and imaginary parts never mix.  Per step: E = 1 forward + (r-1) inverse
// transforms, H = 1 forward + r inverse, each side wrapped by one pack, one filter and one unpack kernel.
// On non-uniform x-y grids pack/unpack interpolate to/from the auxiliary uniform plane (L288).
#include "emm_kernels.cuh"

namespace emm {

struct AirArgs {
  int N1, N2, P1, M1, M2, k0, r, nlev;    // nlev ghost levels written
  long long PS;
  float h[kMaxR];                          // heights of the ghost levels above the surface
  float dx, dy;                            // FFT plane spacings
  float scale;                             // 1/(M1*M2): cuFFT transforms are unnormalised
  int uniform;
};

// ---- uniform x-y: the FFT plane is the padded plane itself ----
__global__ void k_air_pack(const AirArgs a, const float *__restrict__ f1, const float *__restrict__ f2, float2 *__restrict__ A) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= a.M1) return;
  const size_t o = (size_t)a.k0 * a.PS + (size_t)j * a.P1 + i;
  A[(size_t)j * a.M1 + i] = make_float2(f1[o], f2 ? f2[o] : 0.f);
}

__global__ void k_air_unpack(const AirArgs a, float *__restrict__ f1, float *__restrict__ f2, const float2 *__restrict__ B) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, m = blockIdx.z;   // level k0-1-m
  if (i >= a.N1) return;
  const float2 v = B[(size_t)m * a.M1 * a.M2 + (size_t)j * a.M1 + i];
  const size_t o = (size_t)(a.k0 - 1 - m) * a.PS + (size_t)j * a.P1 + i;
  f1[o] = v.x;
  f2[o] = v.y;
}

// ---- non-uniform x-y: 4x4-point Lagrange interpolation to / from the auxiliary plane ----
struct AuxTabs { const int *sx1, *sy1, *sx2, *sy2; const float *wx1, *wy1, *wx2, *wy2; };

// lattice -> auxiliary plane in two separable passes (4 taps each instead of 16 per point): x pass on the few
// lattice rows (T[j][m], both packed components), then y pass over the whole plane, coalesced along m.
__global__ void k_air_toaux_x(const AirArgs a, const AuxTabs t, const float *__restrict__ f1, const float *__restrict__ f2,
                              float2 *__restrict__ T) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (m >= a.M1) return;
  const float *p1 = f1 + (size_t)a.k0 * a.PS + (size_t)j * a.P1;
  const float4 w1 = *reinterpret_cast<const float4 *>(t.wx1 + 4 * m);
  const int i1 = t.sx1[m];
  float v1 = fmaf(w1.x, p1[i1], fmaf(w1.y, p1[i1 + 1], fmaf(w1.z, p1[i1 + 2], w1.w * p1[i1 + 3]))), v2 = 0.f;
  if (f2) {
    const float *p2 = f2 + (size_t)a.k0 * a.PS + (size_t)j * a.P1;
    const float4 w2 = *reinterpret_cast<const float4 *>(t.wx2 + 4 * m);
    const int i2 = t.sx2[m];
    v2 = fmaf(w2.x, p2[i2], fmaf(w2.y, p2[i2 + 1], fmaf(w2.z, p2[i2 + 2], w2.w * p2[i2 + 3])));
  }
  T[(size_t)j * a.M1 + m] = make_float2(v1, v2);
}

__global__ void k_air_toaux_y(const AirArgs a, const AuxTabs t, const float2 *__restrict__ T, float2 *__restrict__ A) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  if (m >= a.M1) return;
  const float4 w1 = *reinterpret_cast<const float4 *>(t.wy1 + 4 * n), w2 = *reinterpret_cast<const float4 *>(t.wy2 + 4 * n);
  const int j1 = t.sy1[n], j2 = t.sy2[n];
  const float v1 = fmaf(w1.x, T[(size_t)j1 * a.M1 + m].x, fmaf(w1.y, T[(size_t)(j1 + 1) * a.M1 + m].x,
                   fmaf(w1.z, T[(size_t)(j1 + 2) * a.M1 + m].x, w1.w * T[(size_t)(j1 + 3) * a.M1 + m].x)));
  const float v2 = fmaf(w2.x, T[(size_t)j2 * a.M1 + m].y, fmaf(w2.y, T[(size_t)(j2 + 1) * a.M1 + m].y,
                   fmaf(w2.z, T[(size_t)(j2 + 2) * a.M1 + m].y, w2.w * T[(size_t)(j2 + 3) * a.M1 + m].y)));
  A[(size_t)n * a.M1 + m] = make_float2(v1, v2);
}

__global__ void k_air_fromaux(const AirArgs a, const AuxTabs t, float *__restrict__ f1, float *__restrict__ f2,
                              const float2 *__restrict__ B) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, m = blockIdx.z;
  if (i >= a.N1) return;
  const float2 *P = B + (size_t)m * a.M1 * a.M2;
  float v1 = 0.f, v2 = 0.f;
  {
    const int ix = t.sx1[i], iy = t.sy1[j];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      float acc = 0.f;
#pragma unroll
      for (int c = 0; c < 4; ++c) acc = fmaf(t.wx1[4 * i + c], P[(size_t)(iy + b) * a.M1 + ix + c].x, acc);
      v1 = fmaf(t.wy1[4 * j + b], acc, v1);
    }
  }
  {
    const int ix = t.sx2[i], iy = t.sy2[j];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      float acc = 0.f;
#pragma unroll
      for (int c = 0; c < 4; ++c) acc = fmaf(t.wx2[4 * i + c], P[(size_t)(iy + b) * a.M1 + ix + c].y, acc);
      v2 = fmaf(t.wy2[4 * j + b], acc, v2);
    }
  }
  const size_t o = (size_t)(a.k0 - 1 - m) * a.PS + (size_t)j * a.P1 + i;
  f1[o] = v1;
  f2[o] = v2;
}

// ---- spectral filters ----
// One thread filters 4 bins (independent loads in flight), bins are numbered row-major over the whole plane.
// E: Laplace E = 0 above the surface (Eq. 21): level m is e^{-k_h h_m} times the surface spectrum.
__global__ void k_air_filter_E(const AirArgs a, const float *__restrict__ kx, const float *__restrict__ ky,
                               const float2 *__restrict__ A, float2 *__restrict__ B) {
  const size_t MM = (size_t)a.M1 * a.M2, T = (size_t)gridDim.x * blockDim.x;
  const size_t n0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  float2 v[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) v[q] = n0 + q * T < MM ? A[n0 + q * T] : make_float2(0.f, 0.f);
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const size_t n = n0 + q * T;
    if (n >= MM) break;
    const int n2 = (int)(n / a.M1), n1 = (int)(n - (size_t)n2 * a.M1);
    const float kh = sqrtf(kx[n1] * kx[n1] + ky[n2] * ky[n2]);
    for (int m = 0; m < a.nlev; ++m) {
      const float e = expf(-kh * a.h[m]) * a.scale;
      B[(size_t)m * MM + n] = make_float2(v[q].x * e, v[q].y * e);
    }
  }
}

// H: curl H = 0 and Laplace H = 0 in the air (Eq. 17-20): Hx^ = i kx/k_h e^{-k_h h} Hz^, Hy^ likewise with
// ky; on the uniform grid the half-cell offset between the Hz and Hx/Hy lattices is a phase factor [R10].
// Output plane = spectrum of Hx + i Hy.
__global__ void k_air_filter_H(const AirArgs a, const float *__restrict__ kx, const float *__restrict__ ky,
                               const float2 *__restrict__ A, float2 *__restrict__ B) {
  const size_t MM = (size_t)a.M1 * a.M2, T = (size_t)gridDim.x * blockDim.x;
  const size_t n0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  float2 v[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) v[q] = n0 + q * T < MM ? A[n0 + q * T] : make_float2(0.f, 0.f);
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const size_t n = n0 + q * T;
    if (n >= MM) break;
    const int n2 = (int)(n / a.M1), n1 = (int)(n - (size_t)n2 * a.M1);
    const float qx = kx[n1], qy = ky[n2];
    const float kh = sqrtf(qx * qx + qy * qy);
    const bool nyx = ((a.M1 & 1) == 0) && n1 == a.M1 / 2, nyy = ((a.M2 & 1) == 0) && n2 == a.M2 / 2;
    float2 gx = make_float2(0.f, 0.f), gy = make_float2(0.f, 0.f);   // i k/k_h [* e^{-i k d/2}]
    if (kh > 0.f) {
      if (!nyx) {
        float sn = 0.f, cs = 1.f;
        if (a.uniform) sincosf(-0.5f * qx * a.dx, &sn, &cs);
        gx = make_float2(-sn * qx / kh, cs * qx / kh);
      }
      if (!nyy) {
        float sn = 0.f, cs = 1.f;
        if (a.uniform) sincosf(-0.5f * qy * a.dy, &sn, &cs);
        gy = make_float2(-sn * qy / kh, cs * qy / kh);
      }
    }
    const float2 G = make_float2(gx.x - gy.y, gx.y + gy.x);             // gx + i gy
    const float2 vg = make_float2(v[q].x * G.x - v[q].y * G.y, v[q].x * G.y + v[q].y * G.x);
    for (int m = 0; m < a.nlev; ++m) {
      const float e = expf(-kh * a.h[m]) * a.scale;
      B[(size_t)m * MM + n] = make_float2(vg.x * e, vg.y * e);
    }
  }
}

#define EMM_LAUNCH_CHECK(g, what)                                                      \
  do {                                                                                 \
    cudaError_t e_ = cudaGetLastError();                                               \
    if (e_ != cudaSuccess) return fail(EMM_ECUDA, "%s: %s", what, cudaGetErrorString(e_)); \
    (g)->launches++;                                                                   \
  } while (0)

int launch_air(emm_grid *g, const DevState &s, const DevRun &r, int is_h, cudaStream_t st) {
  if (g->sep_air) return launch_air_sep(g, s, r, is_h, st);
  if (g->air_cluster) return launch_air_cluster(g, s, r, is_h, st);
  const int R = g->r;
  const int nlev = is_h ? R : R - 1;
  if (nlev <= 0) return 0;
  AirArgs a{};
  a.N1 = g->N[0]; a.N2 = g->N[1]; a.P1 = g->P1; a.M1 = g->M1; a.M2 = g->M2; a.k0 = g->k0; a.r = R; a.nlev = nlev;
  a.PS = g->dg.PS;
  for (int m = 1; m <= nlev; ++m)
    a.h[m - 1] = (float)(is_h ? g->xn[2][g->k0] - g->xh[2][g->k0 - m] : g->xn[2][g->k0] - g->xn[2][g->k0 - m]);
  a.dx = (float)g->dxa; a.dy = (float)g->dya;
  a.scale = (float)(1.0 / ((double)g->M1 * (double)g->M2));
  a.uniform = g->uniform_xy;
  AuxTabs t{};
  // component lattices: E pass packs Ex (half,node) + Ey (node,half); H pass reads Hz (half,half) and
  // writes Hx (node,half) + Hy (half,node)
  const int lat_in1[2] = {is_h ? 1 : 1, is_h ? 1 : 0}, lat_in2[2] = {0, 1};
  const int lat_out1[2] = {is_h ? 0 : 1, is_h ? 1 : 0}, lat_out2[2] = {is_h ? 1 : 0, is_h ? 0 : 1};
  float2 *A = r.air, *B = r.air + (size_t)g->M1 * g->M2;
  const dim3 blk(128, 1, 1);
  const dim3 gM((g->M1 + 127) / 128, g->M2, 1), gN((g->N[0] + 127) / 128, g->N[1], nlev);
  for (int src = 0; src < s.nsrc; ++src) {
    // sources finished earlier keep their ghost planes: harmless, nothing reads them any more
    float *f_in1 = (is_h ? s.H[2] : s.E[0]) + (size_t)src * g->dg.VS;
    float *f_in2 = is_h ? nullptr : s.E[1] + (size_t)src * g->dg.VS;
    float *f_o1 = (is_h ? s.H[0] : s.E[0]) + (size_t)src * g->dg.VS;
    float *f_o2 = (is_h ? s.H[1] : s.E[1]) + (size_t)src * g->dg.VS;
    if (g->uniform_xy) {
      k_air_pack<<<gM, blk, 0, st>>>(a, f_in1, f_in2, A);
    } else {
      t.sx1 = g->T.ta_start[0][lat_in1[0]]; t.wx1 = g->T.ta_w[0][lat_in1[0]];
      t.sy1 = g->T.ta_start[1][lat_in1[1]]; t.wy1 = g->T.ta_w[1][lat_in1[1]];
      t.sx2 = g->T.ta_start[0][lat_in2[0]]; t.wx2 = g->T.ta_w[0][lat_in2[0]];
      t.sy2 = g->T.ta_start[1][lat_in2[1]]; t.wy2 = g->T.ta_w[1][lat_in2[1]];
      float2 *Tx = r.air + (size_t)(1 + R) * g->M1 * g->M2;        // [N2][M1] x-interpolated lattice rows
      k_air_toaux_x<<<dim3((g->M1 + 127) / 128, g->N[1], 1), blk, 0, st>>>(a, t, f_in1, f_in2, Tx);
      EMM_LAUNCH_CHECK(g, "k_air_toaux_x");
      k_air_toaux_y<<<gM, blk, 0, st>>>(a, t, Tx, A);
    }
    EMM_LAUNCH_CHECK(g, "k_air_pack");
    if (cufftExecC2C(g->plan_fwd, A, A, CUFFT_FORWARD) != CUFFT_SUCCESS) return fail(EMM_ECUDA, "cufftExecC2C forward failed");
    const unsigned gF = (unsigned)(((size_t)g->M1 * g->M2 + 4 * 256 - 1) / (4 * 256));
    if (is_h) k_air_filter_H<<<gF, 256, 0, st>>>(a, g->T.kx, g->T.ky, A, B);
    else k_air_filter_E<<<gF, 256, 0, st>>>(a, g->T.kx, g->T.ky, A, B);
    EMM_LAUNCH_CHECK(g, "k_air_filter");
    if (cufftExecC2C(is_h ? g->plan_inv_h : g->plan_inv_e, B, B, CUFFT_INVERSE) != CUFFT_SUCCESS)
      return fail(EMM_ECUDA, "cufftExecC2C inverse failed");
    if (g->uniform_xy) {
      k_air_unpack<<<gN, blk, 0, st>>>(a, f_o1, f_o2, B);
    } else {
      t.sx1 = g->T.fa_start[0][lat_out1[0]]; t.wx1 = g->T.fa_w[0][lat_out1[0]];
      t.sy1 = g->T.fa_start[1][lat_out1[1]]; t.wy1 = g->T.fa_w[1][lat_out1[1]];
      t.sx2 = g->T.fa_start[0][lat_out2[0]]; t.wx2 = g->T.fa_w[0][lat_out2[0]];
      t.sy2 = g->T.fa_start[1][lat_out2[1]]; t.wy2 = g->T.fa_w[1][lat_out2[1]];
      k_air_fromaux<<<gN, blk, 0, st>>>(a, t, f_o1, f_o2, B);
    }
    EMM_LAUNCH_CHECK(g, "k_air_unpack");
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// Effective medium on the device (fp64): each E component sees the area-weighted arithmetic mean of the
// four cells sharing its edge (Eq. 26, [R3]); cells of the padding replicate the edge cell, cells
// above the air-water plane are air.  Pass 1 finds min sigma (v_max of Eq. 15), pass 2 writes dt/eps.
struct ModelArgs {
  int N1, N2, N3, P1, r, klo, air;
  int lo[3], nc[3];
  const double *xn[3];
  const float *sh, *sv;
};

__device__ __forceinline__ double cell_sigma(const ModelArgs &a, const float *s, int i, int j, int k) {
  int ci = i - a.lo[0], cj = j - a.lo[1], ck = k - a.lo[2];
  if (a.air && ck < 0) return 0.0;
  ci = min(max(ci, 0), a.nc[0] - 1);
  cj = min(max(cj, 0), a.nc[1] - 1);
  ck = min(max(ck, 0), a.nc[2] - 1);
  return (double)s[(size_t)ci + (size_t)a.nc[0] * ((size_t)cj + (size_t)a.nc[1] * (size_t)ck)];
}

__device__ __forceinline__ void sigma_bar(const ModelArgs &a, int i, int j, int k, double &s11, double &s22, double &s33) {
  const int im = max(i - 1, 0), jm = max(j - 1, 0), km = max(k - 1, 0);
  const double dx0 = a.xn[0][im + 1] - a.xn[0][im], dx1 = a.xn[0][i + 1] - a.xn[0][i];
  const double dy0 = a.xn[1][jm + 1] - a.xn[1][jm], dy1 = a.xn[1][j + 1] - a.xn[1][j];
  const double dz0 = a.xn[2][km + 1] - a.xn[2][km], dz1 = a.xn[2][k + 1] - a.xn[2][k];
  s11 = (cell_sigma(a, a.sh, i, jm, km) * dy0 * dz0 + cell_sigma(a, a.sh, i, j, km) * dy1 * dz0 +
         cell_sigma(a, a.sh, i, jm, k) * dy0 * dz1 + cell_sigma(a, a.sh, i, j, k) * dy1 * dz1) / ((dy0 + dy1) * (dz0 + dz1));
  s22 = (cell_sigma(a, a.sh, im, j, km) * dx0 * dz0 + cell_sigma(a, a.sh, i, j, km) * dx1 * dz0 +
         cell_sigma(a, a.sh, im, j, k) * dx0 * dz1 + cell_sigma(a, a.sh, i, j, k) * dx1 * dz1) / ((dx0 + dx1) * (dz0 + dz1));
  s33 = (cell_sigma(a, a.sv, im, jm, k) * dx0 * dy0 + cell_sigma(a, a.sv, i, jm, k) * dx1 * dy0 +
         cell_sigma(a, a.sv, im, j, k) * dx0 * dy1 + cell_sigma(a, a.sv, i, j, k) * dx1 * dy1) / ((dx0 + dx1) * (dy0 + dy1));
}

__device__ __forceinline__ bool node_updated(const ModelArgs &a, int i, int j, int k) {
  return i >= a.r && i <= a.N1 - 1 - a.r && j >= a.r && j <= a.N2 - 1 - a.r && k >= a.klo && k <= a.N3 - 1 - a.r;
}

__global__ void k_sigma_min(const ModelArgs a, unsigned long long *__restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  double m = __longlong_as_double(0x7ff0000000000000LL);
  if (i < a.N1 && node_updated(a, i, j, k)) {
    double s11, s22, s33;
    sigma_bar(a, i, j, k, s11, s22, s33);
    m = fmin(s11, fmin(s22, s33));
    if (!(m > 0.0)) m = 0.0;          // flags a non-positive effective conductivity
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMin(out, (unsigned long long)__double_as_longlong(m));   // positive doubles order as integers
}

__global__ void k_make_ce(const ModelArgs a, float *__restrict__ ce1, float *__restrict__ ce2, float *__restrict__ ce3, const double scale) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= a.P1) return;
  float v1 = 0.f, v2 = 0.f, v3 = 0.f;
  if (i < a.N1 && node_updated(a, i, j, k)) {
    double s11, s22, s33;
    sigma_bar(a, i, j, k, s11, s22, s33);
    v1 = (float)(scale / s11); v2 = (float)(scale / s22); v3 = (float)(scale / s33);   // dt/eps = dt*2*omega0/sigma (L47)
  }
  const size_t o = ((size_t)k * a.N2 + j) * a.P1 + i;
  ce1[o] = v1; ce2[o] = v2; ce3[o] = v3;
}

// Raw model scan: validity (every cell finite and > 0) and the smallest conductivity inside each of the six CPML slabs
// (reference speed of the profiles, [R5]).  out[0..5] = slab minima as ordered bit patterns of positive doubles
// (axis-major, low side first), out[6] = number of invalid cells.
struct ScanArgs { int nc[3]; int c0[3][2], c1[3][2]; const float *sh, *sv; };

__global__ void k_model_scan(const ScanArgs a, unsigned long long *__restrict__ out) {
  const size_t n = (size_t)a.nc[0] * a.nc[1] * a.nc[2];
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  double m[6] = {inf, inf, inf, inf, inf, inf};
  unsigned long long bad = 0;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
    const float h = a.sh[t], v = a.sv ? a.sv[t] : h;
    if (!(h > 0.f) || !(v > 0.f) || isinf(h) || isinf(v)) { ++bad; continue; }
    const int i = (int)(t % a.nc[0]), j = (int)((t / a.nc[0]) % a.nc[1]), k = (int)(t / ((size_t)a.nc[0] * a.nc[1]));
    const int idx[3] = {i, j, k};
    const double s = fmin((double)h, (double)v);
#pragma unroll
    for (int ax = 0; ax < 3; ++ax)
#pragma unroll
      for (int side = 0; side < 2; ++side)
        if (idx[ax] >= a.c0[ax][side] && idx[ax] <= a.c1[ax][side]) m[2 * ax + side] = fmin(m[2 * ax + side], s);
  }
#pragma unroll
  for (int q = 0; q < 6; ++q) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m[q] = fmin(m[q], __shfl_xor_sync(0xffffffffu, m[q], o));
    if ((threadIdx.x & 31) == 0) atomicMin(out + q, (unsigned long long)__double_as_longlong(m[q]));
  }
  if (bad) atomicAdd(out + 6, bad);
}

// values of selected raw cells (idx < 0: air, 0); which[n] = 1 reads sigma_v
__global__ void k_gather_cells(const float *__restrict__ sh, const float *__restrict__ sv, const long long *__restrict__ idx,
                               const int *__restrict__ which, const int n, float *__restrict__ out) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const long long t = idx[p];
  out[p] = t < 0 ? 0.f : (which[p] ? sv : sh)[t];
}

int launch_model_scan(emm_grid *g, const float *d_sh, const float *d_sv, unsigned long long *d_out) {
  ScanArgs a{};
  for (int ax = 0; ax < 3; ++ax) {
    a.nc[ax] = g->nc[ax];
    for (int side = 0; side < 2; ++side) {
      const int lo = side == 0 ? 0 : g->N[ax] - g->nb, hi = side == 0 ? g->nb - 1 : g->N[ax] - 1;   // padded cell range of the slab
      a.c0[ax][side] = std::min(std::max(lo - g->lo[ax], 0), g->nc[ax] - 1);
      a.c1[ax][side] = std::min(std::max(hi - g->lo[ax], 0), g->nc[ax] - 1);
    }
  }
  a.sh = d_sh; a.sv = d_sv;
  k_model_scan<<<148 * 8, 256, 0, g->stream>>>(a, d_out);
  EMM_LAUNCH_CHECK(g, "k_model_scan");
  return 0;
}

int launch_gather_cells(emm_grid *g, const float *d_sh, const float *d_sv, const long long *d_idx, const int *d_which, int n, float *d_out) {
  if (n <= 0) return 0;
  k_gather_cells<<<(n + 127) / 128, 128, 0, g->stream>>>(d_sh, d_sv, d_idx, d_which, n, d_out);
  EMM_LAUNCH_CHECK(g, "k_gather_cells");
  return 0;
}

static ModelArgs model_args(const emm_grid *g, const float *d_sh, const float *d_sv) {
  ModelArgs a{};
  a.N1 = g->N[0]; a.N2 = g->N[1]; a.N3 = g->N[2]; a.P1 = g->P1; a.r = g->r; a.klo = g->klo; a.air = g->top == EMM_TOP_AIR;
  for (int q = 0; q < 3; ++q) { a.lo[q] = g->lo[q]; a.nc[q] = g->nc[q]; a.xn[q] = g->T.xn[q]; }
  a.sh = d_sh; a.sv = d_sv;
  return a;
}

int launch_sigma_min(emm_grid *g, const float *d_sh, const float *d_sv, double *d_min) {
  const ModelArgs a = model_args(g, d_sh, d_sv);
  dim3 grid((g->N[0] + 127) / 128, g->N[1], g->N[2]);
  k_sigma_min<<<grid, 128, 0, g->stream>>>(a, reinterpret_cast<unsigned long long *>(d_min));
  EMM_LAUNCH_CHECK(g, "k_sigma_min");
  return 0;
}

int launch_make_ce(emm_grid *g, const float *d_sh, const float *d_sv, double scale) {
  const ModelArgs a = model_args(g, d_sh, d_sv);
  dim3 grid((g->P1 + 127) / 128, g->N[1], g->N[2]);
  k_make_ce<<<grid, 128, 0, g->stream>>>(a, g->T.ce[0], g->T.ce[1], g->T.ce[2], scale);
  EMM_LAUNCH_CHECK(g, "k_make_ce");
  return 0;
}

}  // namespace emm
