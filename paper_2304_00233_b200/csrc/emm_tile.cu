// emm_tile.cu -- the accumulator-free E / H update as a block-cooperative TMA tile pipeline (sm_100a).
//
// Same arithmetic, in the same order, as k_update<R, 0, IS_H> of emm_kernels.cu (Eq. 8, 13, 14, 22-24; Algorithm 1
// L476-479 / L486-489): the fields come out bit-identical.  What differs is how the operands reach the SM.  k_update
// loads every neighbour row through L1/L2 with per-thread LDG.128 and has as many bytes in flight as its registers
// hold; here one elected thread of a producer warp issues `cp.async.bulk.tensor` (TMA) copies of whole tiles -- the
// stencil fields with their x / y halo, the fields being updated, dt/eps -- into shared-memory rings guarded by
// mbarriers, several planes ahead of the 128 consumer threads, which read every operand with conflict-free LDS.128.
// Out-of-range halo elements are zero-filled by the TMA unit (the Dirichlet wall of [R2]).
//
//   tile       64 x 8 nodes (16 quads x 8 rows, one quad per consumer thread), marching over a chunk of z planes
//   ring A     A1 (tile + y halo) and A2 (tile + x halo) of plane p.  The 2R planes of the z stencil of plane k are all
//              resident (no register queue: the z taps are LDS.128 reads of the thread's own column), the one in the
//              middle also serves the y / x derivatives: depth 2R + P
//   ring B     A3 (tile + x and y halo), the three updated fields and (E kernel) the three dt/eps tiles of plane k:
//              depth P + 1
//   P          planes in flight beyond the ones in use
// CPML memory variables stay direct global accesses of the 5-14 % of threads inside a slab, prefetched into L2.
#include <cuda.h>

#include "emm_device.cuh"

namespace emm {

namespace {

constexpr int TX = 64, TY = 8;          // tile (nodes)
constexpr int WX = TX + 8;              // row length of a tile with one halo quad on either side
constexpr int NCONS = 128;              // consumer threads: 16 quads x 8 rows
constexpr int NTHREADS = NCONS + 32;    // + the producer warp

constexpr int kMaxKC = 32;              // most planes a block marches over

constexpr int align128(int bytes) { return (bytes + 127) / 128 * 128; }

template <int R, bool IS_H, int P>
struct TileLayout {
  static constexpr int O = IS_H ? 1 : 0;
  static constexpr int HY = TY + 2 * R - 1;                 // rows of a tile with y halo
  static constexpr int DA = 2 * R + P, DB = P + 1;
  static constexpr int A1_B = align128(TX * HY * 4), A2_B = align128(WX * TY * 4), A3_B = align128(WX * HY * 4), U_B = TX * TY * 4;
  static constexpr int NU = IS_H ? 3 : 6;                   // updated fields (+ dt/eps for E)
  static constexpr int STA_B = A1_B + A2_B, STB_B = A3_B + NU * U_B;
  static constexpr int TXA = TX * HY * 4 + WX * TY * 4;     // bytes the TMA unit delivers per stage (boxes, unpadded)
  static constexpr int TXB = WX * HY * 4 + NU * U_B;
  static constexpr int BAR_OFF = DA * STA_B + DB * STB_B;
  static constexpr int CZ_OFF = BAR_OFF + (2 * DA + 2 * DB) * 8;        // z coefficients of the chunk: kMaxKC planes x 2R
  static constexpr int SMEM = CZ_OFF + kMaxKC * 2 * R * 4 + 128;        // + slack to align the base to 128 bytes
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *b, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
// try_wait suspends the thread in hardware until the phase completes or the time hint (ns) runs out, so a waiting
// thread -- above all the producer, which mostly waits for a slot to come free -- leaves the issue slots alone
__device__ __forceinline__ void mbar_wait(unsigned long long *b, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(b)), "r"(parity), "r"(200000u) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, unsigned long long *bar, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
               ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, unsigned long long *bar, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
               ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ float4 lds4(const unsigned char *p) { return *reinterpret_cast<const float4 *>(p); }

// bufA / bufU: ring buffer x source index base of the stencil fields / the updated fields in
// the 4-D tensor maps (x, y, z, buffer * nsrc + source); the updated fields are written through plain pointers.
template <int R, bool IS_H, int P>
__global__ void __launch_bounds__(NTHREADS, 2)
k_tile(const __grid_constant__ TileMaps tm, const DevGrid g, const DevState s, const int kc, const int nchunks, const int chunk0,
       const int sel, const int bufA, const int bufU) {
  using L = TileLayout<R, IS_H, P>;
  constexpr int O = L::O, DA = L::DA, DB = L::DB;
  const int src = blockIdx.z / nchunks, chunk = chunk0 + blockIdx.z - src * nchunks;
  // the two flags that can end the block early are requested together; their latency is covered by the barrier set-up
  const int done = s.done[src], it = *s.it;
  const int kbeg = g.klo + chunk * kc;
  const int kend = min(kbeg + kc, g.N3 - R);

  extern __shared__ __align__(128) unsigned char smem_raw[];
  // 128-byte aligned base, by pointer arithmetic on the shared array itself (an integer round trip would turn every
  // later access into a generic load)
  unsigned char *sm = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  unsigned char *ringA = sm, *ringB = sm + DA * L::STA_B;
  unsigned long long *fullA = reinterpret_cast<unsigned long long *>(sm + L::BAR_OFF), *emptyA = fullA + DA, *fullB = emptyA + DA, *emptyB = fullB + DB;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int q = 0; q < DA; ++q) { mbar_init(fullA + q, 1); mbar_init(emptyA + q, NCONS / 32); }
    for (int q = 0; q < DB; ++q) { mbar_init(fullB + q, 1); mbar_init(emptyB + q, NCONS / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // every early exit is uniform over the block and comes before the first copy is issued
  if (done || kbeg >= kend) return;
  if ((sel == 1 || sel == 2) && ((sel == 2) != (it % s.dft_every == 0))) return;     // DTFT decimation, see k_update

  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int pA0 = kbeg - R + O;                      // first plane through ring A
  const int nA = (kend - kbeg) + 2 * R - 1;          // planes through ring A: the chunk + the rest of its z stencils

  if (warp == NCONS / 32) {
    // ---- producer: one thread feeds both rings in the order the consumers use them ----
    if (lane == 0) {
      const int wA = bufA * s.nsrc + src, wU = bufU * s.nsrc + src;
      int qa = 0, fa = 0, qb = 0, fb = 0;                  // slot and fill count of each ring
      for (int t = 0; t < nA; ++t) {
        {
          const int q = qa, fill = fa;
          if (++qa == DA) { qa = 0; ++fa; }
          if (fill > 0) mbar_wait(emptyA + q, (fill - 1) & 1);
          unsigned char *st = ringA + q * L::STA_B;
          mbar_expect_tx(fullA + q, L::TXA);
          tma_load_4d(st, &tm.A1, fullA + q, x0, y0 - R + O, pA0 + t, wA);
          tma_load_4d(st + L::A1_B, &tm.A2, fullA + q, x0 - 4, y0, pA0 + t, wA);
        }
        const int b = t - (2 * R - 1);
        if (b >= 0) {
          const int q = qb, fill = fb, k = kbeg + b;
          if (++qb == DB) { qb = 0; ++fb; }
          if (fill > 0) mbar_wait(emptyB + q, (fill - 1) & 1);
          unsigned char *st = ringB + q * L::STB_B;
          mbar_expect_tx(fullB + q, L::TXB);
          tma_load_4d(st, &tm.A3, fullB + q, x0 - 4, y0 - R + O, k, wA);
          tma_load_4d(st + L::A3_B, &tm.U1, fullB + q, x0, y0, k, wU);
          tma_load_4d(st + L::A3_B + L::U_B, &tm.U2, fullB + q, x0, y0, k, wU);
          tma_load_4d(st + L::A3_B + 2 * L::U_B, &tm.U3, fullB + q, x0, y0, k, wU);
          if (!IS_H) {
            tma_load_3d(st + L::A3_B + 3 * L::U_B, &tm.C1, fullB + q, x0, y0, k);
            tma_load_3d(st + L::A3_B + 4 * L::U_B, &tm.C2, fullB + q, x0, y0, k);
            tma_load_3d(st + L::A3_B + 5 * L::U_B, &tm.C3, fullB + q, x0, y0, k);
          }
        }
      }
    }
    return;
  }

  // ---- consumers ----
  const int tx = tid & 15, ty = tid >> 4;
  const int i0 = x0 + 4 * tx, j = y0 + ty;
  const bool valid = i0 < g.N1 && j >= R && j <= g.N2 - 1 - R;
  const int jc = valid ? j : R, ic = valid ? i0 : 0;        // table reads of idle threads stay in range

  float *const *Uo = IS_H ? s.Ho : s.Eo;
  const size_t node0 = (size_t)src * g.VS + (size_t)kbeg * g.PS + (size_t)jc * g.P1 + ic;     // the thread's quad in plane kbeg
  float *W1 = (Uo[0] ? Uo[0] : (IS_H ? s.H[0] : s.E[0])) + node0;
  float *W2 = (Uo[1] ? Uo[1] : (IS_H ? s.H[1] : s.E[1])) + node0;
  float *W3 = (Uo[2] ? Uo[2] : (IS_H ? s.H[2] : s.E[2])) + node0;
  const float *txc = IS_H ? g.cp[0] : g.cm[0];
  const float *tyc = IS_H ? g.cp[1] : g.cm[1];
  // z coefficients of the chunk's planes into shared memory (one uniform LDS per tap and plane instead of a global load)
  float *czs = reinterpret_cast<float *>(sm + L::CZ_OFF);
  {
    const float *tzc = (IS_H ? g.cp[2] : g.cm[2]) + (size_t)kbeg * 2 * R;
    for (int q = tid; q < (kend - kbeg) * 2 * R; q += NCONS) czs[q] = __ldg(tzc + q);
    asm volatile("bar.sync 1, %0;" ::"n"(NCONS) : "memory");      // consumer warps only
  }

  float cx[4][2 * R], cy[2 * R];
#pragma unroll
  for (int n = 0; n < 4; ++n)
#pragma unroll
    for (int m = 0; m < 2 * R; ++m) cx[n][m] = __ldg(txc + (size_t)(ic + n) * 2 * R + m);
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) cy[m] = __ldg(tyc + (size_t)jc * 2 * R + m);

  // update mask of the thread's four nodes (the outermost R layers are never updated, L563), folded into dt/mu for H
  float msk[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) msk[n] = ((i0 + n >= R) && (i0 + n <= g.N1 - 1 - R)) ? g.dtmu : 0.f;

  // CPML bookkeeping that does not depend on k: slab membership in x (per node) and y, Eq. 24 coefficients
  const float *ta[3] = {IS_H ? g.ap[0] : g.am[0], IS_H ? g.ap[1] : g.am[1], IS_H ? g.ap[2] : g.am[2]};
  const float *tb[3] = {IS_H ? g.bp[0] : g.bm[0], IS_H ? g.bp[1] : g.bm[1], IS_H ? g.bp[2] : g.bm[2]};
  const int sj = valid ? slab_of(j, g.N2, g.nb, 1) : -1;
  const bool xq = valid && ((i0 < g.nb) || (i0 + 3 > g.N1 - 1 - g.nb));
  float ay = 0.f, by = 0.f;
  if (sj >= 0) { ay = __ldg(ta[1] + sj); by = __ldg(tb[1] + sj); }
  int si[4];
  float axs[4], bxs[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) {
    si[n] = (xq && i0 + n < g.N1) ? slab_of(i0 + n, g.N1, g.nb, 1) : -1;
    axs[n] = si[n] >= 0 ? __ldg(ta[0] + si[n]) : 0.f;
    bxs[n] = si[n] >= 0 ? __ldg(tb[0] + si[n]) : 0.f;
  }
  constexpr int KI = IS_H ? 1 : 0;
  // memory variables of the thread's quad in plane kbeg; advanced by one plane per iteration
  float *psx0 = s.psx[KI][0] + ((size_t)src * g.N3 + kbeg) * g.N2 * g.XS + (size_t)jc * g.XS;
  float *psx1 = s.psx[KI][1] + ((size_t)src * g.N3 + kbeg) * g.N2 * g.XS + (size_t)jc * g.XS;
  float *psy0 = s.psy[KI][0] + (((size_t)src * g.N3 + kbeg) * 2 * g.nb + (sj >= 0 ? sj : 0)) * g.P1 + ic;
  float *psy1 = s.psy[KI][1] + (((size_t)src * g.N3 + kbeg) * 2 * g.nb + (sj >= 0 ? sj : 0)) * g.P1 + ic;
  float *const psz0 = s.psz[KI][0] + (size_t)src * 2 * g.nb * g.PS + (size_t)jc * g.P1 + ic;
  float *const psz1 = s.psz[KI][1] + (size_t)src * 2 * g.nb * g.PS + (size_t)jc * g.P1 + ic;
  const size_t psx_step = (size_t)g.N2 * g.XS, psy_step = (size_t)2 * g.nb * g.P1;

  const int oA1 = ((ty + R - O) * TX + 4 * tx) * 4;      // own quad in an A1 tile (byte offset)
  const int oA2 = L::A1_B + (ty * WX + 4 + 4 * tx) * 4;  // own quad in the A2 tile of a ring A stage
  const int oA3 = ((ty + R - O) * WX + 4 + 4 * tx) * 4;  // own quad in an A3 tile
  const int oU = L::A3_B + (ty * TX + 4 * tx) * 4;       // own quad in the first updated-field tile of a ring B stage
  const int oY1 = (ty * TX + 4 * tx) * 4, oY3 = (ty * WX + 4 + 4 * tx) * 4;   // first row of the y stencil in an A1 / A3 tile

  // ring A stages of the 2R planes of the z stencil (k-R+O .. k+R-1+O), as byte offsets; rotated once per plane
  int so[2 * R];
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) so[m] = m * L::STA_B;
#pragma unroll
  for (int m = 0; m < 2 * R - 1; ++m) mbar_wait(fullA + m, 0);        // the planes above the leading one of plane kbeg
  int qlead = 2 * R - 1, phlead = 0;     // slot / phase of the leading plane (DA >= 2R: its first fill)
  int qfirst = 0;                        // slot of the oldest plane
  int qb = 0, phb = 0;

  for (int k = kbeg; k < kend; ++k) {
    // operands that do not come through the rings are requested before the waits: the z coefficients of the plane and
    // the CPML memory variables of the slab threads (one L2 round trip, all at once)
    float cz[2 * R];
#pragma unroll
    for (int m = 0; m < 2 * R; ++m) cz[m] = czs[m];
    czs += 2 * R;
    float px0[4] = {0.f, 0.f, 0.f, 0.f}, px1[4] = {0.f, 0.f, 0.f, 0.f};
    float4 py0 = zero4(), py1 = zero4(), pz0 = zero4(), pz1 = zero4();
    const int sk = valid ? slab_of(k, g.N3, g.nb, g.zslab_lo) : -1;
    float az = 0.f, bz = 0.f;
    if (xq) {
#pragma unroll
      for (int n = 0; n < 4; ++n)
        if (si[n] >= 0) { px0[n] = psx0[si[n]]; px1[n] = psx1[si[n]]; }
      if (k + 1 < kend) { prefetch_l2(psx0 + psx_step); prefetch_l2(psx1 + psx_step); }
    }
    if (sj >= 0) {
      py0 = ld4(psy0); py1 = ld4(psy1);
      if (k + 1 < kend) { prefetch_l2(psy0 + psy_step); prefetch_l2(psy1 + psy_step); }
    }
    if (sk >= 0) {
      pz0 = ld4(psz0 + (size_t)sk * g.PS); pz1 = ld4(psz1 + (size_t)sk * g.PS); az = __ldg(ta[2] + sk); bz = __ldg(tb[2] + sk);
      const int skn = slab_of(k + 1, g.N3, g.nb, g.zslab_lo);
      if (skn >= 0 && k + 1 < kend) { prefetch_l2(psz0 + (size_t)skn * g.PS); prefetch_l2(psz1 + (size_t)skn * g.PS); }
    }

    mbar_wait(fullA + qlead, phlead);
    mbar_wait(fullB + qb, phb);
    const unsigned char *stB = ringB + qb * L::STB_B;

    if (valid) {
      // z derivatives (listing L212-236): the thread's own column of the 2R resident planes
      float4 D3A1 = zero4(), D3A2 = zero4(), a1c = zero4(), a2c = zero4();
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        const float4 v1 = lds4(ringA + so[m] + oA1), v2 = lds4(ringA + so[m] + oA2);
        if (m == R - O) { a1c = v1; a2c = v2; }                       // plane k itself
        D3A1 = fma4(cz[m], v1, D3A1);
        D3A2 = fma4(cz[m], v2, D3A2);
      }
      const unsigned char *stK = ringA + so[R - O];
      const float4 a3c = lds4(stB + oA3);
      // y derivatives: rows j-R+O+m of plane k = tile rows ty+m
      float4 D2A3 = zero4(), D2A1 = zero4();
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) {
        const float4 v3 = (m == R - O) ? a3c : lds4(stB + oY3 + m * WX * 4);
        const float4 v1 = (m == R - O) ? a1c : lds4(stK + oY1 + m * TX * 4);
        D2A3 = fma4(cy[m], v3, D2A3);
        D2A1 = fma4(cy[m], v1, D2A1);
      }
      // x derivatives from 12-wide windows (the halo quads of the tile; zero-filled outside the array)
      float4 D1A3, D1A2;
      {
        float w[12];
        window(w, lds4(stB + oA3 - 16), a3c, lds4(stB + oA3 + 16));
        D1A3 = ddx<R, O>(w, cx);
        window(w, lds4(stK + oA2 - 16), a2c, lds4(stK + oA2 + 16));
        D1A2 = ddx<R, O>(w, cx);
      }

      // CPML memory variables (only inside the slabs): psi <- b psi + a D ; D <- D + psi (Eq. 22-23, kappa = 1)
      if (xq) {
        float d3[4] = {D1A3.x, D1A3.y, D1A3.z, D1A3.w}, d2[4] = {D1A2.x, D1A2.y, D1A2.z, D1A2.w};
#pragma unroll
        for (int n = 0; n < 4; ++n)
          if (si[n] >= 0) {
            float p = fmaf(bxs[n], px0[n], axs[n] * d3[n]); psx0[si[n]] = p; d3[n] += p;
            p = fmaf(bxs[n], px1[n], axs[n] * d2[n]); psx1[si[n]] = p; d2[n] += p;
          }
        D1A3 = make_float4(d3[0], d3[1], d3[2], d3[3]);
        D1A2 = make_float4(d2[0], d2[1], d2[2], d2[3]);
      }
      if (sj >= 0) {
        py0 = make_float4(fmaf(by, py0.x, ay * D2A3.x), fmaf(by, py0.y, ay * D2A3.y), fmaf(by, py0.z, ay * D2A3.z), fmaf(by, py0.w, ay * D2A3.w));
        py1 = make_float4(fmaf(by, py1.x, ay * D2A1.x), fmaf(by, py1.y, ay * D2A1.y), fmaf(by, py1.z, ay * D2A1.z), fmaf(by, py1.w, ay * D2A1.w));
        st4(psy0, py0); st4(psy1, py1);
        D2A3 = add4(D2A3, py0); D2A1 = add4(D2A1, py1);
      }
      if (sk >= 0) {
        pz0 = make_float4(fmaf(bz, pz0.x, az * D3A2.x), fmaf(bz, pz0.y, az * D3A2.y), fmaf(bz, pz0.z, az * D3A2.z), fmaf(bz, pz0.w, az * D3A2.w));
        pz1 = make_float4(fmaf(bz, pz1.x, az * D3A1.x), fmaf(bz, pz1.y, az * D3A1.y), fmaf(bz, pz1.z, az * D3A1.z), fmaf(bz, pz1.w, az * D3A1.w));
        st4(psz0 + (size_t)sk * g.PS, pz0); st4(psz1 + (size_t)sk * g.PS, pz1);
        D3A2 = add4(D3A2, pz0); D3A1 = add4(D3A1, pz1);
      }

      // curl (L338-346) and update (Eq. 8)
      const float4 c1 = sub4(D2A3, D3A2), c2 = sub4(D3A1, D1A3), c3 = sub4(D1A2, D2A1);
      float4 u1 = lds4(stB + oU), u2 = lds4(stB + oU + L::U_B), u3 = lds4(stB + oU + 2 * L::U_B);
      if (IS_H) {
        u1 = make_float4(fmaf(-msk[0], c1.x, u1.x), fmaf(-msk[1], c1.y, u1.y), fmaf(-msk[2], c1.z, u1.z), fmaf(-msk[3], c1.w, u1.w));
        u2 = make_float4(fmaf(-msk[0], c2.x, u2.x), fmaf(-msk[1], c2.y, u2.y), fmaf(-msk[2], c2.z, u2.z), fmaf(-msk[3], c2.w, u2.w));
        u3 = make_float4(fmaf(-msk[0], c3.x, u3.x), fmaf(-msk[1], c3.y, u3.y), fmaf(-msk[2], c3.z, u3.z), fmaf(-msk[3], c3.w, u3.w));
      } else {
        const float4 e1 = lds4(stB + oU + 3 * L::U_B), e2 = lds4(stB + oU + 4 * L::U_B), e3 = lds4(stB + oU + 5 * L::U_B);   // 0 where not updated
        u1 = make_float4(fmaf(e1.x, c1.x, u1.x), fmaf(e1.y, c1.y, u1.y), fmaf(e1.z, c1.z, u1.z), fmaf(e1.w, c1.w, u1.w));
        u2 = make_float4(fmaf(e2.x, c2.x, u2.x), fmaf(e2.y, c2.y, u2.y), fmaf(e2.z, c2.z, u2.z), fmaf(e2.w, c2.w, u2.w));
        u3 = make_float4(fmaf(e3.x, c3.x, u3.x), fmaf(e3.y, c3.y, u3.y), fmaf(e3.z, c3.z, u3.z), fmaf(e3.w, c3.w, u3.w));
      }
      st4(W1, u1); st4(W2, u2); st4(W3, u3);
    }
    W1 += g.PS; W2 += g.PS; W3 += g.PS;
    psx0 += psx_step; psx1 += psx_step; psy0 += psy_step; psy1 += psy_step;
    // plane k is done with its ring B stage and with the oldest plane of its z stencil
    __syncwarp();
    if (lane == 0) { mbar_arrive(emptyB + qb); mbar_arrive(emptyA + qfirst); }
    if (++qb == DB) { qb = 0; phb ^= 1; }
    if (++qfirst == DA) qfirst = 0;
    if (++qlead == DA) { qlead = 0; phlead ^= 1; }
#pragma unroll
    for (int m = 0; m < 2 * R - 1; ++m) so[m] = so[m + 1];
    so[2 * R - 1] = qlead * L::STA_B;
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// fp32 tensor (x fastest): dims {P1, N2, N3[, nw]}, zero fill outside, box {bx, by, 1[, 1]}
int make_map(CUtensorMap *m, const float *base, const emm_grid *g, int nw, int bx, int by) {
  EncodeTiledFn enc = encode_fn();
  if (!enc) return fail(EMM_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
  const cuuint32_t rank = nw > 0 ? 4 : 3;
  const cuuint64_t dims[4] = {(cuuint64_t)g->P1, (cuuint64_t)g->N[1], (cuuint64_t)g->N[2], (cuuint64_t)(nw > 0 ? nw : 1)};
  const cuuint64_t strides[3] = {(cuuint64_t)g->P1 * 4, (cuuint64_t)g->P1 * g->N[1] * 4, (cuuint64_t)g->P1 * g->N[1] * g->N[2] * 4};
  const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1, 1}, es[4] = {1, 1, 1, 1};
  const CUresult rc = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, rank, const_cast<float *>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (rc != CUDA_SUCCESS) return fail(EMM_ECUDA, "cuTensorMapEncodeTiled failed (%d) for a %d x %d box", (int)rc, bx, by);
  return 0;
}

constexpr int kPrefetch = 2;

template <int R, bool IS_H>
int launch_tile_r(const TileMaps &tm, const DevGrid &dg, const DevState &s, dim3 grid, cudaStream_t st, int kc, int nchunks, int chunk0, int sel,
                  int bufA, int bufU) {
  using L = TileLayout<R, IS_H, kPrefetch>;
  auto kern = k_tile<R, IS_H, kPrefetch>;
  int dev = 0;
  cudaGetDevice(&dev);
  static unsigned long long configured = 0;            // bit per device ordinal (the attribute is per device)
  if (dev < 64 && !(configured >> dev & 1)) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L::SMEM) != cudaSuccess)
      return fail(EMM_ECUDA, "k_tile: cannot reserve %d bytes of shared memory", L::SMEM);
    configured |= 1ull << dev;
  } else if (dev >= 64) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L::SMEM);
  }
  kern<<<grid, NTHREADS, L::SMEM, st>>>(tm, dg, s, kc, nchunks, chunk0, sel, bufA, bufU);
  return 0;
}

}  // namespace

// tensor maps of the run's field rings and of dt/eps; called by emm_run_begin once the per-run region is laid out
int tile_make_maps(emm_grid *g, const DevState &s) {
  g->tile_ok = false;
  for (int c = 0; c < 3; ++c) { g->tile_base[0][c] = s.E[c]; g->tile_base[1][c] = s.H[c]; }     // buffer 0 of the field rings
  g->tile_hstride = s.hstride;
  const int R = g->r;
  if (g->P1 < TX || g->N[1] < TY + 2 * R) return 0;          // tiny grids keep the per-thread kernel
  const int nw = s.nbuf * s.nsrc, HY = TY + 2 * R - 1;
  int rc;
  for (int e = 0; e < 2; ++e) {                              // e = 0: E kernel (A = H, U = E), 1: H kernel (A = E, U = H)
    TileMaps &tm = g->tile_maps[e];
    float *const *A = e ? s.E : s.H, *const *U = e ? s.H : s.E;
    if ((rc = make_map(&tm.A1, A[0], g, nw, TX, HY)) || (rc = make_map(&tm.A2, A[1], g, nw, WX, TY)) || (rc = make_map(&tm.A3, A[2], g, nw, WX, HY)) ||
        (rc = make_map(&tm.U1, U[0], g, nw, TX, TY)) || (rc = make_map(&tm.U2, U[1], g, nw, TX, TY)) || (rc = make_map(&tm.U3, U[2], g, nw, TX, TY)))
      return rc;
    for (int c = 0; c < 3; ++c)
      if ((rc = make_map(c == 0 ? &tm.C1 : c == 1 ? &tm.C2 : &tm.C3, g->T.ce[c], g, 0, TX, TY))) return rc;
  }
  g->tile_ok = true;
  return 0;
}

// the accumulator-free update of the z chunks [chunk0, chunk0 + nchunks) through the tile pipeline
// (dg: the grid's device view, with klo = first plane of the part of the grid this launch covers)
int launch_tile(emm_grid *g, const DevGrid &dg, const DevState &s, int is_h, int kc, int nchunks, int chunk0, int sel, cudaStream_t st) {
  // which buffers of the rings the launch reads (the pointers of this launch against the ring bases)
  const float *a = is_h ? s.E[0] : s.H[0], *u = is_h ? s.H[0] : s.E[0];
  const int bufA = (int)((a - g->tile_base[is_h ? 0 : 1][0]) / g->tile_hstride), bufU = (int)((u - g->tile_base[is_h ? 1 : 0][0]) / g->tile_hstride);
  dim3 grid((dg.N1 + TX - 1) / TX, (dg.N2 + TY - 1) / TY, nchunks * s.nsrc);
  if (grid.z > 65535) return fail(EMM_EINVAL, "launch_tile: too many z chunks x sources");
  const TileMaps &tm = g->tile_maps[is_h ? 1 : 0];
  int rc = 0;
  if (is_h) {
    if (dg.r == 1) rc = launch_tile_r<1, true>(tm, dg, s, grid, st, kc, nchunks, chunk0, sel, bufA, bufU);
    else if (dg.r == 2) rc = launch_tile_r<2, true>(tm, dg, s, grid, st, kc, nchunks, chunk0, sel, bufA, bufU);
    else rc = launch_tile_r<3, true>(tm, dg, s, grid, st, kc, nchunks, chunk0, sel, bufA, bufU);
  } else {
    if (dg.r == 1) rc = launch_tile_r<1, false>(tm, dg, s, grid, st, kc, nchunks, chunk0, sel, bufA, bufU);
    else if (dg.r == 2) rc = launch_tile_r<2, false>(tm, dg, s, grid, st, kc, nchunks, chunk0, sel, bufA, bufU);
    else rc = launch_tile_r<3, false>(tm, dg, s, grid, st, kc, nchunks, chunk0, sel, bufA, bufU);
  }
  return rc;
}

void tile_dims(int *tx, int *ty) { *tx = TX; *ty = TY; }

}  // namespace emm
