// emm_air_sep.cu -- air-water boundary on non-uniform x-y grids, separable route.
//
// PAPER.md Eq. 17-21 (L264-288) extrapolate the surface fields into the air through a 2-D Fourier transform;
// with non-uniform x-y spacing the transform runs on an auxiliary uniform plane reached by interpolation (L288,
// DESIGN.md [R9]).  That plane is large (cfg4: 3125 x 3125 complex = 78 MB against a 440 x 440 lattice).  The
// plane-sized route (emm_air.cu) interpolates to the plane, runs 2-D cuFFTs on it and interpolates back.
//
// Interpolation (tensor product of 1-D Lagrange stencils) and DFT are both separable and the surface fields are
// real, so the same numbers come out of transforms that never touch the full plane in x:
//
//   k_sep_xup    x-interpolate the N2 lattice rows to the M1 aux nodes; two real rows per complex row
//   cuFFT        batched 1-D transforms along x of those few rows, output written transposed: XT[k][row]
//   k_sep_yup    split the two real rows (Hermitian parts), keep k1 = 0..M1/2, y-interpolate each column to the
//                M2 aux nodes: V[c][k1][n]
//   cuFFT        batched 1-D transforms along y (contiguous)
//   k_sep_filter spectral filters of Eq. 17-21 per ghost level and output component: W[o][lev][k1][n]
//   cuFFT        batched inverse 1-D transforms along y
//   k_sep_ydown  y-interpolate back to the N2 lattice rows, Hermitian-extend in k1, pack the two real outputs into
//                one complex value and transpose through shared memory: ZR[lev*N2 + j][k]
//   cuFFT        batched inverse 1-D transforms along x (contiguous rows, in place)
//   k_sep_xdown  x-interpolate back to the lattice and write the ghost rows of the two field components
//
// Against the plane-sized route this halves the number of length-M transforms (no x transforms of the M2 - N2
// interpolated rows, only k1 >= 0) and more than halves the bytes moved.
#include <cmath>

#include "emm_kernels.cuh"

namespace emm {

namespace {

struct SepArgs {
  int N1, N2, P1, M1, M2, K1, k0, nlev, nrows_f, is_h, nsrc;
  long long PS, VS;
  float h[kMaxR];
  int hmul[kMaxR];      // h[m] = hmul[m] * h[0] (ghost planes continue the first water cell: 1, 2 for E, 1, 3, 5 for H); 0 = not a multiple
  float scale;
};

// e^{-k_h h_m} for every ghost level: one exponential and products when the heights are multiples of the first one
__device__ __forceinline__ void level_decay(const SepArgs &A, float kh, float (&e)[kMaxR]) {
  const float q = expf(-kh * A.h[0]);
  const float q2 = q * q;
  e[0] = q * A.scale;
#pragma unroll
  for (int m = 1; m < kMaxR; ++m) {
    if (m >= A.nlev) break;
    const int k = A.hmul[m];
    e[m] = k == 2 ? q2 * A.scale : k == 3 ? q2 * q * A.scale : k == 5 ? q2 * q2 * q * A.scale : expf(-kh * A.h[m]) * A.scale;
  }
}

struct Tab { const int *s; const float *w; };       // 4-point stencil table: start index and weights per target

__device__ __forceinline__ float lag4(const float *__restrict__ p, int s, const float *__restrict__ w) {
  const float4 c = *reinterpret_cast<const float4 *>(w);
  return fmaf(c.x, p[s], fmaf(c.y, p[s + 1], fmaf(c.z, p[s + 2], c.w * p[s + 3])));
}

// E pass: complex row j = (Ex row j, Ey row j).  H pass: complex row jj = (Hz row 2jj, Hz row 2jj+1).
__global__ void k_sep_xup(const SepArgs A, const float *__restrict__ fa, const float *__restrict__ fb, const Tab ta, const Tab tb,
                          float2 *__restrict__ XR) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x, row = blockIdx.y, src = blockIdx.z;
  if (m >= A.M1) return;
  const int ja = A.is_h ? 2 * row : row, jb = A.is_h ? 2 * row + 1 : row;
  const size_t so = (size_t)src * A.VS;
  const float va = lag4(fa + so + (size_t)ja * A.P1, ta.s[m], ta.w + 4 * m);
  const float vb = jb < A.N2 ? lag4(fb + so + (size_t)jb * A.P1, tb.s[m], tb.w + 4 * m) : 0.f;
  XR[((size_t)src * A.nrows_f + row) * A.M1 + m] = make_float2(va, vb);
}

// XT[k][row] holds the transform of (a + i b); the transform of the real row a is (U(k) + conj U(-k)) / 2, of b
// (U(k) - conj U(-k)) / (2i).  Lattice row j of component c: E pass (row j, part c), H pass (row j/2, part j%2).
__device__ __forceinline__ float2 real_part_spectrum(const float2 *__restrict__ XT, int nrows, int M1, int k1, int row, int part) {
  const float2 u = XT[(size_t)k1 * nrows + row], c = XT[(size_t)(k1 ? M1 - k1 : 0) * nrows + row];
  return part == 0 ? make_float2(0.5f * (u.x + c.x), 0.5f * (u.y - c.y)) : make_float2(0.5f * (u.y + c.y), 0.5f * (c.x - u.x));
}

// One block per (group of kYupCols wavenumbers k1, source, component): the real-part spectra of every lattice row at these
// k1 are formed once in shared memory, then the block sweeps the M2 aux nodes of its columns with coalesced writes; a thread
// loads the stencil of an aux node once and applies it to all columns of the group (the sweep is bound by the latency of
// those table loads, not by bytes: V stays in L2).
constexpr int kYupCols = 4;
__global__ void __launch_bounds__(256) k_sep_yup(const SepArgs A, const float2 *__restrict__ XT, const Tab t0, const Tab t1, float2 *__restrict__ V) {
  extern __shared__ float2 spec[];                     // [kYupCols][N2]
  const int ncomp = A.is_h ? 1 : 2;
  const int kb = blockIdx.x * kYupCols, src = blockIdx.y / ncomp, c = blockIdx.y - src * ncomp;
  const int nk = min(kYupCols, A.K1 - kb);
  const int nrows = A.nsrc * A.nrows_f, r0 = src * A.nrows_f;
  for (int t = threadIdx.x; t < nk * A.N2; t += blockDim.x) {
    const int q = t / A.N2, j = t - q * A.N2;
    spec[t] = A.is_h ? real_part_spectrum(XT, nrows, A.M1, kb + q, r0 + (j >> 1), j & 1) : real_part_spectrum(XT, nrows, A.M1, kb + q, r0 + j, c);
  }
  __syncthreads();
  const Tab t = c ? t1 : t0;
  float2 *out = V + (((size_t)src * 2 + c) * A.K1 + kb) * A.M2;
  for (int n = threadIdx.x; n < A.M2; n += blockDim.x) {
    const int s = t.s[n];
    const float4 w = *reinterpret_cast<const float4 *>(t.w + 4 * n);
#pragma unroll
    for (int q = 0; q < kYupCols; ++q) {
      if (q >= nk) break;
      const float2 *sp = spec + q * A.N2 + s;
      float2 acc = make_float2(0.f, 0.f);
      acc.x = fmaf(w.x, sp[0].x, acc.x); acc.y = fmaf(w.x, sp[0].y, acc.y);
      acc.x = fmaf(w.y, sp[1].x, acc.x); acc.y = fmaf(w.y, sp[1].y, acc.y);
      acc.x = fmaf(w.z, sp[2].x, acc.x); acc.y = fmaf(w.z, sp[2].y, acc.y);
      acc.x = fmaf(w.w, sp[3].x, acc.x); acc.y = fmaf(w.w, sp[3].y, acc.y);
      out[(size_t)q * A.M2 + n] = acc;
    }
  }
}

// E (Eq. 21): level m of component c is e^{-k_h h_m} times its surface spectrum.  H (Eq. 17-20): Hx^ = i kx/k_h
// e^{-k_h h} Hz^, Hy^ likewise with ky; odd filters vanish at their Nyquist bin [R10].  W[o][lev][k1][n].
__global__ void k_sep_filter(const SepArgs A, const float *__restrict__ kx, const float *__restrict__ ky, const float2 *__restrict__ V,
                             float2 *__restrict__ W) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x, k1 = blockIdx.y, src = blockIdx.z;
  if (n >= A.M2) return;
  const float qx = kx[k1], qy = ky[n];
  const float kh = sqrtf(qx * qx + qy * qy);
  const size_t plane = (size_t)A.K1 * A.M2, o0 = (size_t)k1 * A.M2 + n;
  V += (size_t)src * 2 * plane;
  W += (size_t)src * 2 * A.nlev * plane;
  float e[kMaxR];
  level_decay(A, kh, e);
  if (!A.is_h) {
    const float2 v0 = V[o0], v1 = V[plane + o0];
#pragma unroll
    for (int m = 0; m < kMaxR; ++m) {
      if (m >= A.nlev) break;
      W[(size_t)m * plane + o0] = make_float2(v0.x * e[m], v0.y * e[m]);
      W[(size_t)(A.nlev + m) * plane + o0] = make_float2(v1.x * e[m], v1.y * e[m]);
    }
  } else {
    const float2 v = V[o0];
    const bool nyx = ((A.M1 & 1) == 0) && k1 == A.M1 / 2, nyy = ((A.M2 & 1) == 0) && n == A.M2 / 2;
    const float rk = kh > 0.f ? 1.f / kh : 0.f;
    const float gx = nyx ? 0.f : qx * rk, gy = nyy ? 0.f : qy * rk;
#pragma unroll
    for (int m = 0; m < kMaxR; ++m) {
      if (m >= A.nlev) break;
      W[(size_t)m * plane + o0] = make_float2(-v.y * gx * e[m], v.x * gx * e[m]);            // i gx e v
      W[(size_t)(A.nlev + m) * plane + o0] = make_float2(-v.y * gy * e[m], v.x * gy * e[m]);
    }
  }
}

// ZR[row][k] (row = (src*nlev + lev)*N2 + j) = Za + i Zb for k = k1 and conj(Za) + i conj(Zb) for k = M1 - k1, with Za, Zb
// the columns of the two output components interpolated back to their own y lattices.  A block works on a tile of
// 32 lattice rows x 32 wavenumbers: the column reads run along j (one W row per warp), the row writes along k1, with
// a shared-memory transpose in between, so that the x transform that follows reads contiguous rows.
__global__ void __launch_bounds__(256) k_sep_ydown(const SepArgs A, const float2 *__restrict__ W, const Tab t0, const Tab t1,
                                                   float2 *__restrict__ ZR) {
  __shared__ float2 tp[32][33], tm[32][33];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int j0 = blockIdx.x * 32, k0 = blockIdx.y * 32, src = blockIdx.z / A.nlev, lev = blockIdx.z - src * A.nlev;
  const size_t plane = (size_t)A.K1 * A.M2;
  W += (size_t)src * 2 * A.nlev * plane;
  const int j = j0 + tx;
  if (j < A.N2) {
    const int sa = t0.s[j], sb = t1.s[j];
    const float4 wa = *reinterpret_cast<const float4 *>(t0.w + 4 * j), wb = *reinterpret_cast<const float4 *>(t1.w + 4 * j);
#pragma unroll
    for (int kk = ty; kk < 32; kk += 8) {
      const int k1 = k0 + kk;
      if (k1 >= A.K1) break;
      const float2 *ra = W + (size_t)lev * plane + (size_t)k1 * A.M2, *rb = W + (size_t)(A.nlev + lev) * plane + (size_t)k1 * A.M2;
      const float2 a0 = ra[sa], a1 = ra[sa + 1], a2 = ra[sa + 2], a3 = ra[sa + 3];
      const float2 b0 = rb[sb], b1 = rb[sb + 1], b2 = rb[sb + 2], b3 = rb[sb + 3];
      const float2 za = make_float2(fmaf(wa.x, a0.x, fmaf(wa.y, a1.x, fmaf(wa.z, a2.x, wa.w * a3.x))),
                                    fmaf(wa.x, a0.y, fmaf(wa.y, a1.y, fmaf(wa.z, a2.y, wa.w * a3.y))));
      const float2 zb = make_float2(fmaf(wb.x, b0.x, fmaf(wb.y, b1.x, fmaf(wb.z, b2.x, wb.w * b3.x))),
                                    fmaf(wb.x, b0.y, fmaf(wb.y, b1.y, fmaf(wb.z, b2.y, wb.w * b3.y))));
      tp[kk][tx] = make_float2(za.x - zb.y, za.y + zb.x);
      tm[kk][tx] = make_float2(za.x + zb.y, zb.x - za.y);
    }
  }
  __syncthreads();
  const int k1 = k0 + tx;
  if (k1 >= A.K1) return;
  const bool mirror = k1 > 0 && A.M1 - k1 != k1;
#pragma unroll
  for (int jj = ty; jj < 32; jj += 8) {
    if (j0 + jj >= A.N2) break;
    float2 *row = ZR + (((size_t)src * A.nlev + lev) * A.N2 + j0 + jj) * A.M1;
    row[k1] = tp[tx][jj];
    if (mirror) row[A.M1 - k1] = tm[tx][jj];
  }
}

__global__ void k_sep_xdown(const SepArgs A, const float2 *__restrict__ XR, const Tab ta, const Tab tb, float *__restrict__ fa,
                            float *__restrict__ fb) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, src = blockIdx.z / A.nlev, lev = blockIdx.z - src * A.nlev;
  if (i >= A.N1) return;
  const float2 *p = XR + (((size_t)src * A.nlev + lev) * A.N2 + j) * A.M1;
  const int ia = ta.s[i], ib = tb.s[i];
  const float4 wa = *reinterpret_cast<const float4 *>(ta.w + 4 * i), wb = *reinterpret_cast<const float4 *>(tb.w + 4 * i);
  const size_t o = (size_t)src * A.VS + (size_t)(A.k0 - 1 - lev) * A.PS + (size_t)j * A.P1 + i;
  fa[o] = fmaf(wa.x, p[ia].x, fmaf(wa.y, p[ia + 1].x, fmaf(wa.z, p[ia + 2].x, wa.w * p[ia + 3].x)));
  fb[o] = fmaf(wb.x, p[ib].y, fmaf(wb.y, p[ib + 1].y, fmaf(wb.z, p[ib + 2].y, wb.w * p[ib + 3].y)));
}

}  // namespace

// scratch (float2 elements) per source: XR rows [r*N2][M1] | XT / ZT [M1][r*N2] | V [2][K1][M2] | W [2r][K1][M2];
// every array carries a leading source dimension (all unfinished and finished sources go through one launch)
size_t sep_air_scratch(const emm_grid *g, int nsrc) {
  const size_t K1 = (size_t)g->M1 / 2 + 1, rows = (size_t)g->r * g->N[1];
  return (size_t)nsrc * (2 * rows * g->M1 + (size_t)(2 + 2 * g->r) * K1 * g->M2);
}

// 1-D batched plans for nsrc sources: 0/1 x forward (E/H), 2/3 y forward, 4/5 y inverse, 6/7 x inverse.  The forward x
// plans write the transposed layout [k][row] through cuFFT's strided data layout (k_sep_yup reads it along the rows).
int sep_air_make_plans(emm_grid *g, int nsrc) {
  if (g->sp_nsrc == nsrc) return 0;
  for (cufftHandle &h : g->sp) { if (h) cufftDestroy(h); h = 0; }
  g->sp_nsrc = 0;
  const int M1 = g->M1, M2 = g->M2, N2 = g->N[1], K1 = M1 / 2 + 1, R = g->r;
  for (int q = 0; q < 8; ++q) {
    const int is_h = q & 1, nlev = is_h ? R : R - 1;
    g->sp_ws[q] = 0;
    int n[1], batch, istride = 1, idist, ostride = 1, odist;
    if (q < 2) {                       // x forward: rows [row][M1] -> XT[k][row]
      batch = nsrc * (is_h ? (N2 + 1) / 2 : N2);
      n[0] = M1; idist = M1; ostride = batch; odist = 1;
    } else if (q < 4) {                // y forward, in place on V (two planes per source; the H pass fills one)
      batch = nsrc * 2 * K1;
      n[0] = M2; idist = odist = M2;
    } else if (q < 6) {                // y inverse, in place on W
      batch = nsrc * 2 * nlev * K1;
      n[0] = M2; idist = odist = M2;
    } else {                           // x inverse, in place on the rows [row][M1]
      batch = nsrc * nlev * N2;
      n[0] = M1; idist = odist = M1;
    }
    if (batch < 1) continue;
    if (q == 3 && nsrc == 1) batch = K1;                                  // single source, H pass: only the first plane is live
    if (cufftCreate(&g->sp[q]) != CUFFT_SUCCESS) return fail(EMM_ECUDA, "cufftCreate failed (no CUDA device?)");
    cufftSetAutoAllocation(g->sp[q], 0);
    if (cufftMakePlanMany(g->sp[q], 1, n, n, istride, idist, n, ostride, odist, CUFFT_C2C, batch, &g->sp_ws[q]) != CUFFT_SUCCESS)
      return fail(EMM_ECUDA, "cufftMakePlanMany failed for %d transforms of length %d", batch, n[0]);
  }
  g->sp_nsrc = nsrc;
  return 0;
}

#define EMM_SEP_CHECK(g, what)                                                         \
  do {                                                                                 \
    cudaError_t e_ = cudaGetLastError();                                               \
    if (e_ != cudaSuccess) return fail(EMM_ECUDA, "%s: %s", what, cudaGetErrorString(e_)); \
    (g)->launches++;                                                                   \
  } while (0)

int launch_air_sep(emm_grid *g, const DevState &s, const DevRun &r, int is_h, cudaStream_t st) {
  const int R = g->r;
  const int nlev = is_h ? R : R - 1;
  if (nlev <= 0) return 0;
  SepArgs a{};
  a.N1 = g->N[0]; a.N2 = g->N[1]; a.P1 = g->P1; a.M1 = g->M1; a.M2 = g->M2; a.K1 = g->M1 / 2 + 1; a.k0 = g->k0; a.nlev = nlev;
  a.is_h = is_h;
  a.nrows_f = is_h ? (a.N2 + 1) / 2 : a.N2;
  a.PS = g->dg.PS;
  for (int m = 1; m <= nlev; ++m)
    a.h[m - 1] = (float)(is_h ? g->xn[2][g->k0] - g->xh[2][g->k0 - m] : g->xn[2][g->k0] - g->xn[2][g->k0 - m]);
  a.scale = (float)(1.0 / ((double)g->M1 * (double)g->M2));
  for (int m = 0; m < nlev; ++m) {
    const double h0 = is_h ? g->xn[2][g->k0] - g->xh[2][g->k0 - 1] : g->xn[2][g->k0] - g->xn[2][g->k0 - 1];
    const double hm = is_h ? g->xn[2][g->k0] - g->xh[2][g->k0 - 1 - m] : g->xn[2][g->k0] - g->xn[2][g->k0 - 1 - m];
    const double k = hm / h0;
    const int ki = (int)std::lround(k);
    a.hmul[m] = (std::fabs(k - ki) < 1e-9 * k && (ki == 1 || ki == 2 || ki == 3 || ki == 5)) ? ki : 0;
  }
  // lattices (0 = node, 1 = half) per axis: Ex (1,0), Ey (0,1), Hz (1,1), Hx (0,1), Hy (1,0)
  const int in_x[2] = {1, is_h ? 1 : 0}, in_y[2] = {is_h ? 1 : 0, 1};
  const int out_x[2] = {is_h ? 0 : 1, is_h ? 1 : 0}, out_y[2] = {is_h ? 1 : 0, is_h ? 0 : 1};
  auto ta = [&](int axis, int lat) { return Tab{g->T.ta_start[axis][lat], g->T.ta_w[axis][lat]}; };
  auto fa = [&](int axis, int lat) { return Tab{g->T.fa_start[axis][lat], g->T.fa_w[axis][lat]}; };
  a.nsrc = s.nsrc;
  a.VS = g->dg.VS;
  if (g->sp_nsrc != s.nsrc) return fail(EMM_EINVAL, "air boundary: plans were made for %d sources, the run has %d", g->sp_nsrc, s.nsrc);
  const size_t rows = (size_t)s.nsrc * R * a.N2, plane = (size_t)a.K1 * a.M2;
  float2 *XR = r.air, *XT = XR + rows * a.M1, *V = XT + rows * a.M1, *W = V + (size_t)s.nsrc * 2 * plane;
  const int ncomp = is_h ? 1 : 2, ns = s.nsrc;
  const dim3 blk(128, 1, 1);
  // sources finished earlier keep their ghost planes: harmless, nothing reads them any more
  const size_t so = (size_t)g->k0 * a.PS;
  const float *f_a = (is_h ? s.H[2] : s.E[0]) + so, *f_b = (is_h ? s.H[2] : s.E[1]) + so;
  k_sep_xup<<<dim3((a.M1 + 127) / 128, a.nrows_f, ns), blk, 0, st>>>(a, f_a, f_b, ta(0, in_x[0]), ta(0, in_x[1]), XR);
  EMM_SEP_CHECK(g, "k_sep_xup");
  if (cufftExecC2C(g->sp[0 + is_h], XR, XT, CUFFT_FORWARD) != CUFFT_SUCCESS) return fail(EMM_ECUDA, "cufftExecC2C (x forward) failed");
  k_sep_yup<<<dim3((a.K1 + kYupCols - 1) / kYupCols, ns * ncomp, 1), dim3(256, 1, 1), (size_t)kYupCols * a.N2 * sizeof(float2), st>>>(a, XT, ta(1, in_y[0]), ta(1, in_y[1]), V);
  EMM_SEP_CHECK(g, "k_sep_yup");
  if (cufftExecC2C(g->sp[2 + is_h], V, V, CUFFT_FORWARD) != CUFFT_SUCCESS) return fail(EMM_ECUDA, "cufftExecC2C (y forward) failed");
  k_sep_filter<<<dim3((a.M2 + 127) / 128, a.K1, ns), blk, 0, st>>>(a, g->T.kx, g->T.ky, V, W);
  EMM_SEP_CHECK(g, "k_sep_filter");
  if (cufftExecC2C(g->sp[4 + is_h], W, W, CUFFT_INVERSE) != CUFFT_SUCCESS) return fail(EMM_ECUDA, "cufftExecC2C (y inverse) failed");
  k_sep_ydown<<<dim3((a.N2 + 31) / 32, (a.K1 + 31) / 32, nlev * ns), dim3(32, 8, 1), 0, st>>>(a, W, fa(1, out_y[0]), fa(1, out_y[1]), XR);
  EMM_SEP_CHECK(g, "k_sep_ydown");
  if (cufftExecC2C(g->sp[6 + is_h], XR, XR, CUFFT_INVERSE) != CUFFT_SUCCESS) return fail(EMM_ECUDA, "cufftExecC2C (x inverse) failed");
  k_sep_xdown<<<dim3((a.N1 + 127) / 128, a.N2, nlev * ns), blk, 0, st>>>(a, XR, fa(0, out_x[0]), fa(0, out_x[1]), is_h ? s.H[0] : s.E[0],
                                                                          is_h ? s.H[1] : s.E[1]);
  EMM_SEP_CHECK(g, "k_sep_xdown");
  return 0;
}

}  // namespace emm
