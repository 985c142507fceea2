// emm_kernels.cu -- the per-time-step CUDA kernels of libemm_b200.so (sm_100a).
//
// One template, k_update<R, NF, IS_H>, is both fused passes of Algorithm 1:
//   IS_H = 0:  curl H (Eq. 14) + CPML psi (Eq. 22-24) + E += dt/eps * curl (Eq. 8) + DTFT of the new E
//   IS_H = 1:  DTFT of the old H (Eq. 25) + curl E (Eq. 13) + CPML psi + H -= dt/mu * curl
// so no curl arrays are written and the DTFT costs no extra field read (the paper's five separate
// kernels, Fig. 10).  Both curls have the same shape
//   (D2 A3 - D3 A2,  D3 A1 - D1 A3,  D1 A2 - D2 A1)
// with A = H and the D- tables, or A = E and the D+ tables whose stencil is shifted by one node.
//
// Mapping: a thread owns 4 consecutive x nodes (128-bit loads/stores) of one y row and marches along z
// over a chunk of planes, keeping the 2R z-neighbour planes of A1 and A2 in a register queue; x and y
// neighbours come through L1/L2 (rows are 128-byte aligned).  The DTFT accumulators are streamed with
// evict-first loads/stores: they are the dominant HBM traffic (96*nf of 84+96*nf bytes per node-step).
#include <cstdio>
#include <algorithm>
#include <cstdlib>

#include "emm_device.cuh"

namespace emm {

// DTFT of 4 nodes of one component into NF accumulators (Eq. 25): F[f] += u * tw[f]
template <int NF>
__device__ __forceinline__ void dtft4(float2 *F0, size_t fstride, float4 u, const float2 (&tw)[NF > 0 ? NF : 1]) {
  float4 a[NF > 0 ? NF : 1][2];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const float *p = reinterpret_cast<const float *>(F0 + f * fstride);
    a[f][0] = ldcs4(p);
    a[f][1] = ldcs4(p + 4);
  }
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    a[f][0].x = fmaf(u.x, tw[f].x, a[f][0].x); a[f][0].y = fmaf(u.x, tw[f].y, a[f][0].y);
    a[f][0].z = fmaf(u.y, tw[f].x, a[f][0].z); a[f][0].w = fmaf(u.y, tw[f].y, a[f][0].w);
    a[f][1].x = fmaf(u.z, tw[f].x, a[f][1].x); a[f][1].y = fmaf(u.z, tw[f].y, a[f][1].y);
    a[f][1].z = fmaf(u.w, tw[f].x, a[f][1].z); a[f][1].w = fmaf(u.w, tw[f].y, a[f][1].w);
    float *p = reinterpret_cast<float *>(F0 + f * fstride);
    stcs4(p, a[f][0]);
    stcs4(p + 4, a[f][1]);
  }
}

// runtime-nf fallback (one frequency at a time)
__device__ __forceinline__ void dtft4_rt(float2 *F0, size_t fstride, float4 u, const float2 *tw, int nf) {
  for (int f = 0; f < nf; ++f) {
    const float2 t = __ldg(tw + f);
    float *p = reinterpret_cast<float *>(F0 + f * fstride);
    float4 a0 = ldcs4(p), a1 = ldcs4(p + 4);
    a0.x = fmaf(u.x, t.x, a0.x); a0.y = fmaf(u.x, t.y, a0.y); a0.z = fmaf(u.y, t.x, a0.z); a0.w = fmaf(u.y, t.y, a0.w);
    a1.x = fmaf(u.z, t.x, a1.x); a1.y = fmaf(u.z, t.y, a1.y); a1.z = fmaf(u.w, t.x, a1.z); a1.w = fmaf(u.w, t.y, a1.w);
    stcs4(p, a0);
    stcs4(p + 4, a1);
  }
}

// 16-byte asynchronous global->shared copy (LDGSTS): no register is held while it is in flight.  `.ca` on purpose:
// the two 16-byte halves of a thread's 32-byte accumulator quad are fetched by two instructions that touch the
// same sectors; through L1 the second one hits, with `.cg` (L1 bypass) every sector is pulled from L2 twice
// (measured on cfg4: 6.03 ms/step with .cg vs 5.02 ms/step with .ca).
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_2() { asm volatile("cp.async.wait_group 2;" ::: "memory"); }

// Accumulators of one plane staged in shared memory: slot j of thread t sits at sm[j*128 + t] (conflict-free
// LDS.128).  Each thread only ever touches its own slots, so no block barrier is needed: the thread waits for
// its own cp.async group.  Slot order: ((c*NF + f)*2 + h), h = first / second pair of nodes of the quad.
template <int NF>
__device__ __forceinline__ void stage_plane(float4 *sm, const float2 *Fk, size_t fstride, size_t cstride) {
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const float *p = reinterpret_cast<const float *>(Fk + c * cstride + f * fstride);
      cp_async16(sm + ((c * NF + f) * 2 + 0) * 128, p);
      cp_async16(sm + ((c * NF + f) * 2 + 1) * 128, p + 4);
    }
}

// one component only (the three components are separate commit groups, see the kernel)
template <int NF>
__device__ __forceinline__ void stage_component(float4 *sm, int c, const float2 *Fkc, size_t fstride) {
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const float *p = reinterpret_cast<const float *>(Fkc + f * fstride);
    cp_async16(sm + ((c * NF + f) * 2 + 0) * 128, p);
    cp_async16(sm + ((c * NF + f) * 2 + 1) * 128, p + 4);
  }
}

// DTFT of one component from the staged accumulators: F[f] += u * tw[f], result streamed back to global
template <int NF>
__device__ __forceinline__ void dtft4_staged(const float4 *sm, int c, float2 *F0, size_t fstride, float4 u,
                                             const float2 (&tw)[NF > 0 ? NF : 1]) {
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    float4 a0 = sm[((c * NF + f) * 2 + 0) * 128], a1 = sm[((c * NF + f) * 2 + 1) * 128];
    a0.x = fmaf(u.x, tw[f].x, a0.x); a0.y = fmaf(u.x, tw[f].y, a0.y); a0.z = fmaf(u.y, tw[f].x, a0.z); a0.w = fmaf(u.y, tw[f].y, a0.w);
    a1.x = fmaf(u.z, tw[f].x, a1.x); a1.y = fmaf(u.z, tw[f].y, a1.y); a1.z = fmaf(u.w, tw[f].x, a1.z); a1.w = fmaf(u.w, tw[f].y, a1.w);
    float *p = reinterpret_cast<float *>(F0 + f * fstride);
    stcs4(p, a0);
    stcs4(p + 4, a1);
  }
}

// Two consecutive terms of Eq. 25 in one read-modify-write of the accumulators (paired DTFT): the
// update kernel holds the field before (uo) and after (un) its own update, i.e. the DTFT operands of two consecutive
// steps.  F = fma(un, tb, fma(uo, ta, F)): the same two fused multiply-adds, in the same order, as two single-term passes.
// kNHS: history levels a grouped-DTFT pass can take besides the old and the new field of its own update (group <= kNHS + 2)
constexpr int kNHS = kGroupMax - 2;
// smh: the thread's staged history quads of this component (levels 0..nh-1, oldest first), twh: their twiddles
// [nh][nf] in global memory (uniform loads).  Order of the fused multiply-adds = order of the terms in time.
template <int NF>
__device__ __forceinline__ void dtft4_staged2(const float4 *sm, int c, float2 *F0, size_t fstride, float4 uo, float4 un,
                                              const float2 (&ta)[NF > 0 ? NF : 1], const float2 (&tb)[NF > 0 ? NF : 1],
                                              const float4 *smh, const float2 *__restrict__ twh, const int nh, const int nf) {
  float4 uh[kNHS];
#pragma unroll
  for (int l = 0; l < kNHS; ++l) uh[l] = l < nh ? smh[l * 128] : zero4();
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    float4 a0 = sm[((c * NF + f) * 2 + 0) * 128], a1 = sm[((c * NF + f) * 2 + 1) * 128];
#pragma unroll
    for (int l = 0; l < kNHS; ++l)
      if (l < nh) {
        const float2 t = __ldg(twh + l * nf + f);
        a0.x = fmaf(uh[l].x, t.x, a0.x); a0.y = fmaf(uh[l].x, t.y, a0.y); a0.z = fmaf(uh[l].y, t.x, a0.z); a0.w = fmaf(uh[l].y, t.y, a0.w);
        a1.x = fmaf(uh[l].z, t.x, a1.x); a1.y = fmaf(uh[l].z, t.y, a1.y); a1.z = fmaf(uh[l].w, t.x, a1.z); a1.w = fmaf(uh[l].w, t.y, a1.w);
      }
    a0.x = fmaf(uo.x, ta[f].x, a0.x); a0.y = fmaf(uo.x, ta[f].y, a0.y); a0.z = fmaf(uo.y, ta[f].x, a0.z); a0.w = fmaf(uo.y, ta[f].y, a0.w);
    a1.x = fmaf(uo.z, ta[f].x, a1.x); a1.y = fmaf(uo.z, ta[f].y, a1.y); a1.z = fmaf(uo.w, ta[f].x, a1.z); a1.w = fmaf(uo.w, ta[f].y, a1.w);
    a0.x = fmaf(un.x, tb[f].x, a0.x); a0.y = fmaf(un.x, tb[f].y, a0.y); a0.z = fmaf(un.y, tb[f].x, a0.z); a0.w = fmaf(un.y, tb[f].y, a0.w);
    a1.x = fmaf(un.z, tb[f].x, a1.x); a1.y = fmaf(un.z, tb[f].y, a1.y); a1.z = fmaf(un.w, tb[f].x, a1.z); a1.w = fmaf(un.w, tb[f].y, a1.w);
    float *p = reinterpret_cast<float *>(F0 + f * fstride);
    stcs4(p, a0);
    stcs4(p + 4, a1);
  }
}

// Blocks per SM the register allocation is aimed at.  Measured on B200 (profiles/r1_kernel_experiments.md): with
// many frequencies (>= 4: 48+ KB of staged accumulators per block) two fat blocks per SM win -- no register cap,
// and the unified L1 keeps ~100 KB for the neighbour rows; with fewer frequencies three blocks win.
template <int NF> constexpr int update_min_blocks() { return NF >= 4 ? 2 : 3; }

// PAIR: the closing pass of a DTFT group (NF >= 1, staged).  The H kernel of step `it` holds old H
// (term it) and new H (term it+1), the E kernel of step `it` old E (term it-1) and new E (term it) [R6]; with `harg` = nh
// history levels (earlier buffers of the field ring the steps of the group update through) the pass takes nh + 2 consecutive
// terms of Eq. 25 in one read-modify-write of the accumulators, oldest first.
template <int R, int NF, bool IS_H, bool PAIR = false>
__global__ void __launch_bounds__(128, update_min_blocks<NF>()) k_update(const DevGrid g, const DevState s, const int kc, const int nchunks, const int chunk0, const int sel, const int harg) {
  constexpr int O = IS_H ? 1 : 0;            // D+ stencils start one node later than D- (Eq. 13 vs 14)
  const int src = blockIdx.z / nchunks, chunk = chunk0 + blockIdx.z - src * nchunks;   // this launch covers chunks [chunk0, chunk0 + nchunks)
  if (s.done[src]) return;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  if (i0 >= g.N1 || j < R || j > g.N2 - 1 - R) return;
  const int kbeg = g.klo + chunk * kc;
  const int kend = min(kbeg + kc, g.N3 - R);
  if (kbeg >= kend) return;
  const int it = *s.it;
  // DTFT decimation runs two instances per pass: sel 1 = the accumulator-free one, for the steps that skip the DTFT;
  // sel 2 = the DTFT one, for the steps that contribute; the instance whose turn it is not exits here (sel 0: no split)
  // sel 3 = accumulator-free, unconditionally (the step of a DTFT pair in which this kernel takes no term)
  if ((sel == 1 || sel == 2) && ((sel == 2) != (it % s.dft_every == 0))) return;

  const float *A1 = (IS_H ? s.E[0] : s.H[0]) + (size_t)src * g.VS;
  const float *A2 = (IS_H ? s.E[1] : s.H[1]) + (size_t)src * g.VS;
  const float *A3 = (IS_H ? s.E[2] : s.H[2]) + (size_t)src * g.VS;
  const float *U1 = (IS_H ? s.H[0] : s.E[0]) + (size_t)src * g.VS;
  const float *U2 = (IS_H ? s.H[1] : s.E[1]) + (size_t)src * g.VS;
  const float *U3 = (IS_H ? s.H[2] : s.E[2]) + (size_t)src * g.VS;
  // where the updated field goes: in place, or (inside a DTFT group of more than two steps) the next buffer of the ring
  float *const *Uo = IS_H ? s.Ho : s.Eo;
  float *W1 = (Uo[0] ? Uo[0] : (IS_H ? s.H[0] : s.E[0])) + (size_t)src * g.VS;
  float *W2 = (Uo[1] ? Uo[1] : (IS_H ? s.H[1] : s.E[1])) + (size_t)src * g.VS;
  float *W3 = (Uo[2] ? Uo[2] : (IS_H ? s.H[2] : s.E[2])) + (size_t)src * g.VS;
  const float *tx = IS_H ? g.cp[0] : g.cm[0];
  const float *ty = IS_H ? g.cp[1] : g.cm[1];
  const float *tz = IS_H ? g.cp[2] : g.cm[2];

  // x coefficients of the thread's 4 nodes.  The accumulator-free instance (register-capped at 3 blocks per SM) parks them
  // in private shared-memory slots and re-reads them where the x derivatives are formed (LDS.128, no bank conflicts:
  // slot q of thread t at [q*128 + t]); that frees 8R registers for loads in flight.
  constexpr bool CXS = NF == 0;
  constexpr int NCX = (8 * R + 3) / 4;                 // float4 slots for 4 nodes x 2R coefficients
  extern __shared__ float4 sm_dyn[];
  float4 *smC = sm_dyn + (threadIdx.y * blockDim.x + threadIdx.x);
  float cx[4][2 * R], cy[2 * R];
  if constexpr (CXS) {
    static_assert((8 * R) % 4 == 0, "4 nodes x 2R coefficients fill whole float4 slots");
    const float4 *src4 = reinterpret_cast<const float4 *>(tx + (size_t)i0 * 2 * R);    // 4 nodes x 2R floats, 16-byte aligned
#pragma unroll
    for (int q = 0; q < NCX; ++q) smC[q * 128] = __ldg(src4 + q);
  } else {
#pragma unroll
    for (int n = 0; n < 4; ++n)
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) cx[n][m] = __ldg(tx + (size_t)(i0 + n) * 2 * R + m);
  }
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) cy[m] = __ldg(ty + (size_t)j * 2 * R + m);

  // per-node update mask (outermost R layers are never updated, L563)
  bool upd[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) upd[n] = (i0 + n >= R) && (i0 + n <= g.N1 - 1 - R);
  const bool has_l = i0 >= 4, has_r = i0 + 4 < g.P1;

  // CPML bookkeeping that does not depend on k
  const int sj = slab_of(j, g.N2, g.nb, 1);
  const bool xq = (i0 < g.nb) || (i0 + 3 > g.N1 - 1 - g.nb);
  const float *ta[3] = {IS_H ? g.ap[0] : g.am[0], IS_H ? g.ap[1] : g.am[1], IS_H ? g.ap[2] : g.am[2]};
  const float *tb[3] = {IS_H ? g.bp[0] : g.bm[0], IS_H ? g.bp[1] : g.bm[1], IS_H ? g.bp[2] : g.bm[2]};
  float ay = 0.f, by = 0.f;
  if (sj >= 0) { ay = __ldg(ta[1] + sj); by = __ldg(tb[1] + sj); }
  const int KI = IS_H ? 1 : 0;
  float *psx0 = s.psx[KI][0] + (size_t)src * g.N3 * g.N2 * g.XS, *psx1 = s.psx[KI][1] + (size_t)src * g.N3 * g.N2 * g.XS;
  float *psy0 = s.psy[KI][0] + (size_t)src * g.N3 * 2 * g.nb * g.P1, *psy1 = s.psy[KI][1] + (size_t)src * g.N3 * 2 * g.nb * g.P1;
  float *psz0 = s.psz[KI][0] + (size_t)src * 2 * g.nb * g.PS, *psz1 = s.psz[KI][1] + (size_t)src * 2 * g.nb * g.PS;

  // DTFT bookkeeping
  const int nf = s.nf;
  const bool dft_xy = (sel != 1) && (sel != 3) && (nf > 0) && (it % s.dft_every == 0) &&        // DTFT decimation: this step contributes or not
                      (j >= g.blo[1]) && (j <= g.bhi[1]) && (i0 + 3 >= g.blo[0]) && (i0 <= g.bhi[0]);
  const size_t fstride = (size_t)6 * g.NZB * g.PS;      // float2 elements between frequencies
  float2 *Fsrc = s.F + (size_t)src * nf * fstride + (size_t)(IS_H ? 3 : 0) * g.NZB * g.PS;
  const float2 *twp = (IS_H ? s.twH : s.twE) + (size_t)(PAIR && !IS_H ? it - 1 : it) * nf;    // PAIR: first of the two terms
  float2 tw[NF > 0 ? NF : 1], tw2[PAIR && NF > 0 ? NF : 1];
#pragma unroll
  for (int f = 0; f < NF; ++f) tw[f] = __ldg(twp + f);
  if constexpr (PAIR) {
#pragma unroll
    for (int f = 0; f < NF; ++f) tw2[f] = __ldg(twp + nf + f);
  }

  const size_t row = (size_t)j * g.P1 + i0;
  // z queues of A1, A2: planes k-R+O .. k+R-1+O
  float4 q1[2 * R], q2[2 * R];
#pragma unroll
  for (int m = 1; m < 2 * R; ++m) {
    const size_t o = (size_t)(kbeg - R + O + m - 1) * g.PS + row;
    q1[m] = ld4(A1 + o);
    q2[m] = ld4(A2 + o);
  }

  constexpr bool STAGED = NF > 0;
  static_assert(!PAIR || STAGED, "the closing pass of a DTFT group needs staged accumulators");
  float4 *smF = smC;                                   // DTFT instances: the dynamic shared memory holds the staged accumulators
  const size_t cstride = (size_t)g.NZB * g.PS;
  // Grouped DTFT.  harg (PAIR instance) = number nh of history levels it takes besides its own old
  // and new field: whole earlier buffers of the ring, oldest first; their quads are staged with the accumulators of the
  // component, in slots behind them.
  const int nh = PAIR ? harg : 0;
  const float *hs[3] = {nullptr, nullptr, nullptr};
  if constexpr (PAIR) {
#pragma unroll
    for (int c = 0; c < 3; ++c) hs[c] = s.hist[IS_H ? 1 : 0][c] + (size_t)src * g.VS;
  }
  constexpr int HB = 3 * (NF > 0 ? NF : 0) * 2;        // first history slot in shared memory
  auto stage_history = [&](int c, int k) {
    if constexpr (PAIR) {
#pragma unroll
      for (int l = 0; l < kNHS; ++l)
        if (l < nh) cp_async16(smF + (HB + c * nh + l) * 128, hs[c] + (size_t)l * s.hstride + (size_t)k * g.PS + row);
    }
  };
  // The accumulators of the three components are three commit groups, consumed in issue order and re-issued for
  // the next plane as soon as their slots are free: every copy gets almost a whole plane of lead time, and
  // `cp.async.wait_group 2` before each use leaves exactly the two younger groups pending.
  if constexpr (STAGED) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      if (dft_xy && kbeg >= g.blo[2] && kbeg <= g.bhi[2]) {
        stage_component<NF>(smF, c, Fsrc + (size_t)(kbeg - g.blo[2]) * g.PS + row + c * cstride, fstride);
        stage_history(c, kbeg);
      }
      cp_async_commit();
    }
  }

  for (int k = kbeg; k < kend; ++k) {
    const size_t c0 = (size_t)k * g.PS + row;
    // pull the next plane's streaming operands into L2 while this plane is being worked on (no registers held)
    if (k + 1 < kend) {
      const size_t c1 = c0 + g.PS;
      prefetch_l2(U1 + c1); prefetch_l2(U2 + c1); prefetch_l2(U3 + c1);
      if (!IS_H) { prefetch_l2(g.ce[0] + c1); prefetch_l2(g.ce[1] + c1); prefetch_l2(g.ce[2] + c1); }
      prefetch_l2(A3 + c1);
      prefetch_l2(A1 + (size_t)(k + R + O) * g.PS + row); prefetch_l2(A2 + (size_t)(k + R + O) * g.PS + row);
      // CPML memory variables of the next plane (slab threads only): their loads sit behind the derivative they
      // update, so without this they are a second, DRAM-long round trip per plane
      if (xq) { const size_t pn = ((size_t)(k + 1) * g.N2 + j) * g.XS; prefetch_l2(psx0 + pn); prefetch_l2(psx1 + pn); }
      if (sj >= 0) { const size_t pn = ((size_t)(k + 1) * 2 * g.nb + sj) * g.P1 + i0; prefetch_l2(psy0 + pn); prefetch_l2(psy1 + pn); }
      const int skn = slab_of(k + 1, g.N3, g.nb, g.zslab_lo);
      if (skn >= 0) { const size_t pn = (size_t)skn * g.PS + row; prefetch_l2(psz0 + pn); prefetch_l2(psz1 + pn); }
      if (!STAGED && dft_xy && k + 1 >= g.blo[2] && k + 1 <= g.bhi[2]) {
        const float2 *Fn = Fsrc + (size_t)(k + 1 - g.blo[2]) * g.PS + row;
        const size_t cs = (size_t)g.NZB * g.PS;
        for (int f = 0; f < nf; ++f) {
          prefetch_l2(Fn + f * fstride); prefetch_l2(Fn + f * fstride + cs); prefetch_l2(Fn + f * fstride + 2 * cs);
        }
      }
    }
#pragma unroll
    for (int m = 0; m < 2 * R - 1; ++m) { q1[m] = q1[m + 1]; q2[m] = q2[m + 1]; }
    {
      const size_t o = (size_t)(k + R - 1 + O) * g.PS + row;
      q1[2 * R - 1] = ld4(A1 + o);
      q2[2 * R - 1] = ld4(A2 + o);
    }
    float cz[2 * R];
#pragma unroll
    for (int m = 0; m < 2 * R; ++m) cz[m] = __ldg(tz + (size_t)k * 2 * R + m);
    // issue the loads of the fields being updated (and dt/eps) together with the stencil loads: one dependent
    // memory round trip per plane instead of two
    float4 u1 = ld4(U1 + c0), u2 = ld4(U2 + c0), u3 = ld4(U3 + c0);
    float4 e1 = zero4(), e2 = zero4(), e3 = zero4();
    if (!IS_H) { e1 = ld4(g.ce[0] + c0); e2 = ld4(g.ce[1] + c0); e3 = ld4(g.ce[2] + c0); }
    const float4 a1c = q1[R - O], a2c = q2[R - O];      // plane k of A1, A2
    const float4 a3c = ld4(A3 + c0);

    // z derivatives (listing L212-236)
    float4 D3A1 = zero4(), D3A2 = zero4();
#pragma unroll
    for (int m = 0; m < 2 * R; ++m) { D3A1 = fma4(cz[m], q1[m], D3A1); D3A2 = fma4(cz[m], q2[m], D3A2); }
    // y derivatives: rows j-R+O+m of plane k
    float4 D2A3 = zero4(), D2A1 = zero4();
#pragma unroll
    for (int m = 0; m < 2 * R; ++m) {
      const int dj = m - R + O;
      const float4 v3 = dj == 0 ? a3c : ld4(A3 + c0 + (ptrdiff_t)dj * g.P1);
      const float4 v1 = dj == 0 ? a1c : ld4(A1 + c0 + (ptrdiff_t)dj * g.P1);
      D2A3 = fma4(cy[m], v3, D2A3);
      D2A1 = fma4(cy[m], v1, D2A1);
    }
    // x derivatives from 12-wide windows
    float4 D1A3, D1A2;
    {
      float w[12];
      if constexpr (CXS) {
#pragma unroll
        for (int q = 0; q < NCX; ++q) {
          const float4 v = smC[q * 128];
          (&cx[0][0])[4 * q] = v.x; (&cx[0][0])[4 * q + 1] = v.y; (&cx[0][0])[4 * q + 2] = v.z; (&cx[0][0])[4 * q + 3] = v.w;
        }
      }
      window(w, has_l ? ld4(A3 + c0 - 4) : zero4(), a3c, has_r ? ld4(A3 + c0 + 4) : zero4());
      D1A3 = ddx<R, O>(w, cx);
      window(w, has_l ? ld4(A2 + c0 - 4) : zero4(), a2c, has_r ? ld4(A2 + c0 + 4) : zero4());
      D1A2 = ddx<R, O>(w, cx);
    }

    // CPML memory variables (only inside the slabs)
    if (xq) {
      float d3[4] = {D1A3.x, D1A3.y, D1A3.z, D1A3.w}, d2[4] = {D1A2.x, D1A2.y, D1A2.z, D1A2.w};
      const size_t pr = ((size_t)k * g.N2 + j) * g.XS;
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        const int si = (i0 + n < g.N1) ? slab_of(i0 + n, g.N1, g.nb, 1) : -1;
        if (si >= 0) {
          const float a = __ldg(ta[0] + si), b = __ldg(tb[0] + si);
          float p = fmaf(b, psx0[pr + si], a * d3[n]); psx0[pr + si] = p; d3[n] += p;
          p = fmaf(b, psx1[pr + si], a * d2[n]); psx1[pr + si] = p; d2[n] += p;
        }
      }
      D1A3 = make_float4(d3[0], d3[1], d3[2], d3[3]);
      D1A2 = make_float4(d2[0], d2[1], d2[2], d2[3]);
    }
    if (sj >= 0) {
      const size_t po = ((size_t)k * 2 * g.nb + sj) * g.P1 + i0;
      cpml4(psy0 + po, ay, by, D2A3);
      cpml4(psy1 + po, ay, by, D2A1);
    }
    const int sk = slab_of(k, g.N3, g.nb, g.zslab_lo);
    if (sk >= 0) {
      const float a = __ldg(ta[2] + sk), b = __ldg(tb[2] + sk);
      const size_t po = (size_t)sk * g.PS + row;
      cpml4(psz0 + po, a, b, D3A2);
      cpml4(psz1 + po, a, b, D3A1);
    }

    // curl (L338-346)
    const float4 c1 = sub4(D2A3, D3A2), c2 = sub4(D3A1, D1A3), c3 = sub4(D1A2, D2A1);
    const bool dft = dft_xy && k >= g.blo[2] && k <= g.bhi[2];
    float2 *Fk = Fsrc + (size_t)(k - g.blo[2]) * g.PS + row;
    // one component: wait for its staged accumulators, add u * twiddle, stream out, refill the slots for plane k+1
    auto dtft_staged_component = [&](int c, float4 u, float4 un = zero4()) {
      cp_async_wait_2();
      if (dft) {
        if constexpr (PAIR) dtft4_staged2<NF>(smF, c, Fk + c * cstride, fstride, u, un, tw, tw2, smF + (HB + c * nh) * 128, twp - (size_t)nh * nf, nh, nf);
        else dtft4_staged<NF>(smF, c, Fk + c * cstride, fstride, u, tw);
      }
      if (k + 1 < kend && dft_xy && k + 1 >= g.blo[2] && k + 1 <= g.bhi[2]) {
        stage_component<NF>(smF, c, Fk + g.PS + c * cstride, fstride);
        stage_history(c, k + 1);
      }
      cp_async_commit();
    };

    const float4 o1 = u1, o2 = u2, o3 = u3;      // the fields before this update (PAIR: first of the two DTFT terms)
    if (IS_H) {
      // old H sits at t = it*dt, the time level of J (Eq. 8; [R6])
      if constexpr (PAIR) {}
      else if constexpr (STAGED) { dtft_staged_component(0, u1); dtft_staged_component(1, u2); dtft_staged_component(2, u3); }
      else if (dft) {
        if constexpr (NF > 0) { dtft4<NF>(Fk, fstride, u1, tw); dtft4<NF>(Fk + cstride, fstride, u2, tw); dtft4<NF>(Fk + 2 * cstride, fstride, u3, tw); }
        else { dtft4_rt(Fk, fstride, u1, twp, nf); dtft4_rt(Fk + cstride, fstride, u2, twp, nf); dtft4_rt(Fk + 2 * cstride, fstride, u3, twp, nf); }
      }
      const float m0 = upd[0] ? g.dtmu : 0.f, m1 = upd[1] ? g.dtmu : 0.f, m2 = upd[2] ? g.dtmu : 0.f, m3 = upd[3] ? g.dtmu : 0.f;
      u1 = make_float4(fmaf(-m0, c1.x, u1.x), fmaf(-m1, c1.y, u1.y), fmaf(-m2, c1.z, u1.z), fmaf(-m3, c1.w, u1.w));
      u2 = make_float4(fmaf(-m0, c2.x, u2.x), fmaf(-m1, c2.y, u2.y), fmaf(-m2, c2.z, u2.z), fmaf(-m3, c2.w, u2.w));
      u3 = make_float4(fmaf(-m0, c3.x, u3.x), fmaf(-m1, c3.y, u3.y), fmaf(-m2, c3.z, u3.z), fmaf(-m3, c3.w, u3.w));
      st4(W1 + c0, u1); st4(W2 + c0, u2); st4(W3 + c0, u3);
      // PAIR: old H is term it, new H is term it+1 (the old H of the next step)
      if constexpr (PAIR) { dtft_staged_component(0, o1, u1); dtft_staged_component(1, o2, u2); dtft_staged_component(2, o3, u3); }
    } else {
      u1 = make_float4(fmaf(e1.x, c1.x, u1.x), fmaf(e1.y, c1.y, u1.y), fmaf(e1.z, c1.z, u1.z), fmaf(e1.w, c1.w, u1.w));
      u2 = make_float4(fmaf(e2.x, c2.x, u2.x), fmaf(e2.y, c2.y, u2.y), fmaf(e2.z, c2.z, u2.z), fmaf(e2.w, c2.w, u2.w));
      u3 = make_float4(fmaf(e3.x, c3.x, u3.x), fmaf(e3.y, c3.y, u3.y), fmaf(e3.z, c3.z, u3.z), fmaf(e3.w, c3.w, u3.w));
      st4(W1 + c0, u1); st4(W2 + c0, u2); st4(W3 + c0, u3);
      // new E sits at t = (it+1/2)*dt [R6]; PAIR: old E is term it-1, new E is term it
      if constexpr (PAIR) { dtft_staged_component(0, o1, u1); dtft_staged_component(1, o2, u2); dtft_staged_component(2, o3, u3); }
      else if constexpr (STAGED) { dtft_staged_component(0, u1); dtft_staged_component(1, u2); dtft_staged_component(2, u3); }
      else if (dft) {
        if constexpr (NF > 0) { dtft4<NF>(Fk, fstride, u1, tw); dtft4<NF>(Fk + cstride, fstride, u2, tw); dtft4<NF>(Fk + 2 * cstride, fstride, u3, tw); }
        else { dtft4_rt(Fk, fstride, u1, twp, nf); dtft4_rt(Fk + cstride, fstride, u2, twp, nf); dtft4_rt(Fk + 2 * cstride, fstride, u3, twp, nf); }
      }
    }
  }
}

// ---- source injection (Eq. 8, [R7]): electric dipoles E_c[node] -= s(it dt) * (dt/eps W_c)[node] before the E
// update; magnetic dipoles H_c[node] -= s((it+1/2) dt) * (dt/mu W_c)[node] after the H update and its boundary ----
__global__ void k_inject(const DevGrid g, const DevState s, const int *__restrict__ off, const int *__restrict__ idx,
                         const float *__restrict__ w, const int magnetic, const int pairfix) {
  const int src = blockIdx.x;
  if (s.done[src] || s.src_mag[src] != magnetic) return;
  const int it = *s.it;
  const float st = magnetic ? s.wavh[it] : s.wav[it];
  // Paired DTFT: the two-term kernel sees the injected nodes at the wrong side of this injection for one of its
  // terms -- electric: the E kernel of this step reads (E - st w) as the old E of term it-1; magnetic: the H kernel
  // of this step took the new H of term it+1 before (- st w) was added.  The missing product goes into F here.
  const float2 *twf = magnetic ? s.twH + (size_t)(it + 1) * s.nf : s.twE + (size_t)(it - 1) * s.nf;
  const float sg = magnetic ? -1.f : 1.f;
  const size_t fstride = (size_t)6 * g.NZB * g.PS;
  for (int c = 0; c < 3; ++c) {
    float *U = (magnetic ? s.H[c] : s.E[c]) + (size_t)src * g.VS;
    float2 *F = s.F + (size_t)src * s.nf * fstride + (size_t)(c + (magnetic ? 3 : 0)) * g.NZB * g.PS;
    for (int n = off[src * 3 + c] + threadIdx.x; n < off[src * 3 + c + 1]; n += blockDim.x) {
      U[idx[n]] = fmaf(-st, w[n], U[idx[n]]);        // one rounding, with or without pairfix
      if (pairfix) {
        const float d = __fmul_rn(st, w[n]);
        const int k = idx[n] / (int)g.PS, rem = idx[n] - k * (int)g.PS, j = rem / g.P1, i = rem - j * g.P1;
        if (k >= g.blo[2] && k <= g.bhi[2] && j >= g.blo[1] && j <= g.bhi[1] && i >= g.blo[0] && i <= g.bhi[0])
          for (int f = 0; f < s.nf; ++f) {
            float2 &a = F[f * fstride + (size_t)(k - g.blo[2]) * g.PS + rem];
            a.x = fmaf(sg * d, twf[f].x, a.x);
            a.y = fmaf(sg * d, twf[f].y, a.y);
          }
      }
    }
  }
}

// ---- check set: separate fp64 accumulators of the lowest frequency, fed by the fp32 fields [R9] ----
__global__ void k_check_acc(const DevGrid g, const DevState s, const int *__restrict__ cidx, const int nchk,
                            double2 *__restrict__ C, const double2 *__restrict__ twE, const double2 *__restrict__ twH) {
  const int src = blockIdx.z, c = blockIdx.y;
  if (s.done[src]) return;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= nchk) return;
  const int it = *s.it;
  const float *fld = (c < 3 ? s.E[c] : s.H[c - 3]) + (size_t)src * g.VS;
  const double u = (double)fld[cidx[p]];
  const double2 t = c < 3 ? twE[it] : twH[it];
  double2 &a = C[((size_t)src * 6 + c) * nchk + p];
  a.x += u * t.x;
  a.y += u * t.y;
}

// The same sums for the m steps of a DTFT group in one pass: launched between the E and the H update
// of the last step of the group, when the field ring still holds every level -- E after step l (term l) in buffer
// (l+1) mod m, H before step l (term l) in buffer l.  Each accumulator receives the same fp64 operations in the same
// (time) order as with one launch per step; *s.it is the index of the last step of the group.
__global__ void k_check_acc_group(const DevGrid g, const DevState s, const int *__restrict__ cidx, const int nchk, double2 *__restrict__ C,
                                  const double2 *__restrict__ twE, const double2 *__restrict__ twH, const float *const baseE0,
                                  const float *const baseE1, const float *const baseE2, const float *const baseH0, const float *const baseH1,
                                  const float *const baseH2, const int m) {
  const int src = blockIdx.z, c = blockIdx.y;
  if (s.done[src]) return;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= nchk) return;
  const int it0 = *s.it - (m - 1);
  const float *base = c == 0 ? baseE0 : c == 1 ? baseE1 : c == 2 ? baseE2 : c == 3 ? baseH0 : c == 4 ? baseH1 : baseH2;
  const float *fld = base + (size_t)src * g.VS + cidx[p];
  const double2 *tw = (c < 3 ? twE : twH) + it0;
  double2 a = C[((size_t)src * 6 + c) * nchk + p];
  for (int l = 0; l < m; ++l) {
    const int buf = c < 3 ? (l + 1 == m ? 0 : l + 1) : l;
    const double u = (double)fld[(size_t)buf * s.hstride];
    const double2 t = tw[l];
    a.x += u * t.x;
    a.y += u * t.y;
  }
  C[((size_t)src * 6 + c) * nchk + p] = a;
}

// ---- receivers-only DTFT: Eq. 25 at the nodes of the receivers' interpolation stencils only, fp64 sums of the fp32
// fields, every frequency.  Runs where k_check_acc runs: after the E update (E at (it+1/2) dt) and before the H update
// (H at it dt), [R6]. ----
__global__ void k_rec_acc(const DevGrid g, const DevState s, const int *__restrict__ ridx, const int nn, const int nf,
                          double2 *__restrict__ RA, const double2 *__restrict__ twE, const double2 *__restrict__ twH) {
  const int src = blockIdx.z, c = blockIdx.y;
  if (s.done[src]) return;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= nn) return;
  const int it = *s.it;
  if (it % s.dft_every != 0) return;
  const float *fld = (c < 3 ? s.E[c] : s.H[c - 3]) + (size_t)src * g.VS;
  const double u = (double)fld[ridx[(size_t)c * nn + p]];
  const double2 *tw = (c < 3 ? twE : twH) + (size_t)it * nf;
  for (int f = 0; f < nf; ++f) {
    double2 &a = RA[(((size_t)src * nf + f) * 6 + c) * nn + p];
    a.x += u * tw[f].x;
    a.y += u * tw[f].y;
  }
}

// relative change since the previous check: warp shuffle + block reduction; every block leaves its partial sums in a slot
// of its own and k_check_final adds them in a fixed order, so that the integer outcome (the step count) does not depend
// on the order in which the blocks happen to finish
__global__ void k_check_reduce(const DevState s, const int nchk, const double2 *__restrict__ C, double2 *__restrict__ Cprev,
                               double *__restrict__ part) {
  const int src = blockIdx.z, c = blockIdx.y;
  if (s.done[src]) return;
  double num = 0.0, den = 0.0;
  const size_t base = ((size_t)src * 6 + c) * nchk;
  for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < nchk; p += gridDim.x * blockDim.x) {
    const double2 a = C[base + p], b = Cprev[base + p];
    const double dx = a.x - b.x, dy = a.y - b.y;
    num += dx * dx + dy * dy;
    den += a.x * a.x + a.y * a.y;
    Cprev[base + p] = a;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    num += __shfl_xor_sync(0xffffffffu, num, o);
    den += __shfl_xor_sync(0xffffffffu, den, o);
  }
  __shared__ double sn[32], sd[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) { sn[wid] = num; sd[wid] = den; }
  __syncthreads();
  if (wid == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    num = lane < nw ? sn[lane] : 0.0;
    den = lane < nw ? sd[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      num += __shfl_xor_sync(0xffffffffu, num, o);
      den += __shfl_xor_sync(0xffffffffu, den, o);
    }
    if (lane == 0) {
      part[(((size_t)src * 6 + c) * 2 + 0) * kCheckBlocks + blockIdx.x] = num;
      part[(((size_t)src * 6 + c) * 2 + 1) * kCheckBlocks + blockIdx.x] = den;
    }
  }
}

// decision per source; runs before k_step_end of the same step so *it is the index of that step
__global__ void k_check_final(const DevState s, const double *__restrict__ part, const int nblk, double *__restrict__ delta,
                              int *__restrict__ nsteps, int *__restrict__ status, const int it_min, const double tol, const int stop_enabled) {
  const int src = blockIdx.x * blockDim.x + threadIdx.x;
  if (src >= s.nsrc || s.done[src]) return;
  const int it = *s.it;
  double sum[4] = {0.0, 0.0, 0.0, 0.0};                    // num E, den E, num H, den H: components, then blocks, in order
  for (int c = 0; c < 6; ++c)
    for (int q = 0; q < 2; ++q)
      for (int b = 0; b < nblk; ++b) sum[(c / 3) * 2 + q] += part[(((size_t)src * 6 + c) * 2 + q) * kCheckBlocks + b];
  const double nE = sum[0], dE = sum[1], nH = sum[2], dH = sum[3];
  nsteps[src] = it + 1;
  if (!isfinite(nE) || !isfinite(dE) || !isfinite(nH) || !isfinite(dH)) {
    status[src] = EMM_ENAN;
    s.done[src] = 1;
    return;
  }
  const double qE = dE > 0 ? sqrt(nE / dE) : nan(""), qH = dH > 0 ? sqrt(nH / dH) : nan("");
  delta[src * 2 + 0] = qE;
  delta[src * 2 + 1] = qH;
  if (stop_enabled && it >= it_min && dE > 0 && dH > 0 && qE < tol && qH < tol) s.done[src] = 1;
}

__global__ void k_step_end(const DevState s) { *s.it += 1; }

// receivers: interpolate the accumulators to the receiver positions, sum_n w_n F[node_n] in fp64 over the np^3 nodes of
// each component's stencil (weights = tensor product of the 1-D weights, Eq. 9-12); one warp per (receiver, component,
// frequency, source).  Reads the full-grid accumulators, or the receivers-only sums RA when nf_rec > 0.  Eq. 7 (the
// division by the source spectrum) is applied on the host.
__global__ void k_rec_interp(const DevGrid g, const DevState s, const int *__restrict__ ridx, const double *__restrict__ rw,
                             const double2 *__restrict__ RA, const int nf, const int nrec, const int np3, const int sparse,
                             double2 *__restrict__ out) {
  const int q = blockIdx.x, c = blockIdx.y % 6, f = blockIdx.y / 6, src = blockIdx.z;
  const size_t nn = (size_t)nrec * np3, base = (size_t)c * nn + (size_t)q * np3;
  double ax = 0.0, ay = 0.0;
  for (int n = threadIdx.x; n < np3; n += 32) {
    double2 v;
    if (sparse) {
      v = RA[(((size_t)src * nf + f) * 6 + c) * nn + (size_t)q * np3 + n];
    } else {
      const int t = ridx[base + n];                      // node index in the padded volume
      const int k = t / (int)g.PS, rem = t - k * (int)g.PS;
      const float2 F = s.F[((((size_t)src * nf + f) * 6 + c) * g.NZB + (k - g.blo[2])) * g.PS + rem];
      v = make_double2((double)F.x, (double)F.y);
    }
    const double w = rw[base + n];
    ax += w * v.x;
    ay += w * v.y;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ax += __shfl_xor_sync(0xffffffffu, ax, o);
    ay += __shfl_xor_sync(0xffffffffu, ay, o);
  }
  if (threadIdx.x == 0) out[(((size_t)src * nf + f) * nrec + q) * 6 + c] = make_double2(ax, ay);
}

// ---------------------------------------------------------------------------------------------------
#define EMM_LAUNCH_CHECK(g, what)                                                      \
  do {                                                                                 \
    cudaError_t e_ = cudaGetLastError();                                               \
    if (e_ != cudaSuccess) return fail(EMM_ECUDA, "%s: %s", what, cudaGetErrorString(e_)); \
    (g)->launches++;                                                                   \
  } while (0)

// unrolled-NF instantiations stage one plane of accumulators per thread in dynamic shared memory
template <int R, int NF, bool IS_H, bool PAIR = false>
static void launch_one(const DevGrid &dg, const DevState &s, dim3 grid, dim3 block, cudaStream_t st, int kc, int nchunks, int chunk0, int sel, int harg) {
  // staged accumulators + (grouped DTFT) the history quads of the levels this pass takes: sized per launch, so that a
  // small group does not pay shared memory (= L1) for the largest one
  const size_t smem = (size_t)(3 * NF * 2 + (PAIR ? 3 * harg : 0)) * 128 * sizeof(float4);
  const size_t smem_max = (size_t)(3 * NF * 2 + (PAIR ? 3 * kNHS : 0)) * 128 * sizeof(float4);
  if (smem_max > 48 * 1024) {
    // the attribute belongs to the (function, device) pair: one bit per device ordinal, set on first use there
    static unsigned long long configured = 0;
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev >= 64 || !(configured >> dev & 1)) {
      cudaFuncSetAttribute(k_update<R, NF, IS_H, PAIR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
      if (dev < 64) configured |= 1ull << dev;
    }
  }
  k_update<R, NF, IS_H, PAIR><<<grid, block, smem, st>>>(dg, s, kc, nchunks, chunk0, sel, harg);
}

// two-term instances of the paired DTFT (1..kPairMaxNF frequencies)
template <int R, bool IS_H>
static void launch_update_pair(const DevGrid &dg, const DevState &s, int nf, dim3 grid, dim3 block, cudaStream_t st, int kc, int nchunks, int chunk0, int harg) {
  switch (nf) {
    case 1: launch_one<R, 1, IS_H, true>(dg, s, grid, block, st, kc, nchunks, chunk0, 0, harg); break;
    case 2: launch_one<R, 2, IS_H, true>(dg, s, grid, block, st, kc, nchunks, chunk0, 0, harg); break;
    case 3: launch_one<R, 3, IS_H, true>(dg, s, grid, block, st, kc, nchunks, chunk0, 0, harg); break;
    case 4: launch_one<R, 4, IS_H, true>(dg, s, grid, block, st, kc, nchunks, chunk0, 0, harg); break;
    default: launch_one<R, 5, IS_H, true>(dg, s, grid, block, st, kc, nchunks, chunk0, 0, harg); break;
  }
}

template <int R, bool IS_H>
static void launch_update_nf(const DevGrid &dg, const DevState &s, int nf, dim3 grid, dim3 block, cudaStream_t st, int kc, int nchunks, int chunk0, int sel, int harg) {
  switch (nf) {
    case 0: k_update<R, 0, IS_H><<<grid, block, (size_t)2 * R * 128 * sizeof(float4), st>>>(dg, s, kc, nchunks, chunk0, sel, harg); break;
    case 1: launch_one<R, 1, IS_H>(dg, s, grid, block, st, kc, nchunks, chunk0, sel, -1); break;
    case 2: launch_one<R, 2, IS_H>(dg, s, grid, block, st, kc, nchunks, chunk0, sel, -1); break;
    case 3: launch_one<R, 3, IS_H>(dg, s, grid, block, st, kc, nchunks, chunk0, sel, -1); break;
    case 4: launch_one<R, 4, IS_H>(dg, s, grid, block, st, kc, nchunks, chunk0, sel, -1); break;
    case 5: launch_one<R, 5, IS_H>(dg, s, grid, block, st, kc, nchunks, chunk0, sel, -1); break;
    default: k_update<R, -1, IS_H><<<grid, block, 0, st>>>(dg, s, kc, nchunks, chunk0, sel, harg); break;
  }
}

// part: 0 = every z chunk, 1 = only the chunks next to the air-water plane (their stencils read the ghost planes),
// 2 = all the others.  Parts 1 and 2 can run on different streams (emm_run.cu overlaps the boundary with part 2).
// mode: 0 = one DTFT term per step (and DTFT decimation); paired DTFT: 1 = the step in which this kernel takes no
// term (accumulator-free instance), 2 = the step in which it takes two (PAIR instance)
// harg: mode 2 = history levels (earlier buffers of the ring) the closing pass takes; unused in the other modes
int launch_update(emm_grid *g, const DevState &s, int is_h, int part, int mode, int harg, cudaStream_t st) {
  const int quads = g->dg.P1 / 4;
  // Split of the updated planes for the overlap with the air-water boundary (part 1 = surface, 2 = bulk, 0 = everything):
  // the surface part is the r + 1 planes whose z stencils reach the ghost planes, one thin chunk -- it heads the chain
  // surface update -> boundary -> surface update of the other field, so it is kept as short as it can be; the bulk is the
  // rest, in chunks of kc planes counted from its own first plane (the kernels take the first plane from DevGrid::klo).
  const int nk_all = g->dg.N3 - g->dg.r - g->dg.klo;  // updated planes
  const int ks = part == 0 ? 0 : std::min(nk_all, g->dg.r + 1);
  DevGrid dg = g->dg;
  if (part == 2) dg.klo += ks;
  const int nk = part == 0 ? nk_all : (part == 1 ? ks : nk_all - ks);
  if (nk <= 0) return 0;
  // launch one instance (nf = accumulators it is compiled for) over the chunks of `part`
  auto launch = [&](int nf, int sel, bool pair = false) -> int {
    if (nf == 0 && !pair && g->tile_ok) {
      // accumulator-free instance: the TMA tile pipeline (emm_tile.cu), same z-chunk scheme with its own tile shape
      int tx, ty, kc = 16;
      tile_dims(&tx, &ty);
      const long long xy = (long long)((dg.N1 + tx - 1) / tx) * ((dg.N2 + ty - 1) / ty) * s.nsrc;
      // (kc <= 32 = kMaxKC of emm_tile.cu).  Shorter chunks = more blocks and a shorter march per block, against more z-halo
      // planes re-read per chunk: down to 8 planes while the grid holds fewer than 12 blocks per SM, below that only while it
      // holds fewer than 6 (measured: cfg3 16 -> 8 planes 0.385 -> 0.373 ms, cfg2 8 -> 4 planes 0.144 -> 0.158 ms, cfg1 4 -> 2
      // planes 0.0356 -> 0.0320 ms per step)
      while (kc > 8 && xy * ((nk + kc - 1) / kc) < 148 * 12) kc /= 2;
      while (kc > 2 && xy * ((nk + kc - 1) / kc) < 148 * 6) kc /= 2;
      if (part == 1) kc = ks;
      const int nchunks = (nk + kc - 1) / kc;
      const int rc = launch_tile(g, dg, s, is_h, kc, nchunks, 0, sel, st);
      if (rc) return rc;
      EMM_LAUNCH_CHECK(g, is_h ? "k_tile<H>" : "k_tile<E>");
      return 0;
    }
    // block: TX quads wide, 128 threads.  With accumulators: 16 or 32 quads, whichever wastes fewer lanes (long
    // contiguous accumulator rows); without: 8 quads x 16 rows, more y reuse in L1 (profiles/r1_kernel_experiments.md)
    int TX = 16;
    if (((quads + 31) / 32) * 32 <= ((quads + 15) / 16) * 16) TX = 32;
    if (nf == 0 || quads <= 8) TX = 8;
    const int TY = 128 / TX;
    // planes per z chunk: 16 on large grids; fewer on small ones so that the grid still holds ~8 blocks per SM
    // (each block marches its planes one after the other, so a sparse grid is latency-bound)
    int kc = 16;
    {
      const long long xy = (long long)((quads + TX - 1) / TX) * ((dg.N2 + TY - 1) / TY) * s.nsrc;
      while (kc > 2 && xy * ((nk + kc - 1) / kc) < 148 * 8) kc /= 2;
    }
    if (part == 1) kc = ks;
    const int nchunks = (nk + kc - 1) / kc, chunk0 = 0;
    dim3 block(TX, TY, 1), grid((quads + TX - 1) / TX, (dg.N2 + TY - 1) / TY, nchunks * s.nsrc);
    if (grid.z > 65535) return fail(EMM_EINVAL, "launch_update: too many z chunks x sources");
    if (pair) {
      if (is_h) {
        if (dg.r == 1) launch_update_pair<1, true>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, harg);
        else if (dg.r == 2) launch_update_pair<2, true>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, harg);
        else launch_update_pair<3, true>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, harg);
      } else {
        if (dg.r == 1) launch_update_pair<1, false>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, harg);
        else if (dg.r == 2) launch_update_pair<2, false>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, harg);
        else launch_update_pair<3, false>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, harg);
      }
    } else if (is_h) {
      if (dg.r == 1) launch_update_nf<1, true>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, sel, sel == 3 ? harg : -1);
      else if (dg.r == 2) launch_update_nf<2, true>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, sel, sel == 3 ? harg : -1);
      else launch_update_nf<3, true>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, sel, sel == 3 ? harg : -1);
    } else {
      if (dg.r == 1) launch_update_nf<1, false>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, sel, sel == 3 ? harg : -1);
      else if (dg.r == 2) launch_update_nf<2, false>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, sel, sel == 3 ? harg : -1);
      else launch_update_nf<3, false>(dg, s, nf, grid, block, st, kc, nchunks, chunk0, sel, sel == 3 ? harg : -1);
    }
    EMM_LAUNCH_CHECK(g, is_h ? "k_update<H>" : "k_update<E>");
    return 0;
  };
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (g->prof) {
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return fail(EMM_ECUDA, "cudaEventCreate failed");
    cudaEventRecord(e0, st);
  }
  int rc;
  if (mode == 1) {
    if ((rc = launch(0, 3))) return rc;
  } else if (mode == 2) {
    if ((rc = launch(s.nf, 0, true))) return rc;
  } else if (s.nf > 0 && s.dft_every > 1) {
    // DTFT decimation: most steps take no accumulator at all.  Both instances are launched every step (the step index
    // lives on the device, so that a captured graph can be replayed); the one whose turn it is not exits at once.
    if ((rc = launch(0, 1)) || (rc = launch(s.nf, 2))) return rc;
  } else {
    if ((rc = launch(s.nf, 0))) return rc;
  }
  if (g->prof) {
    cudaEventRecord(e1, st);
    g->prof_ev.push_back(e0);
    g->prof_ev.push_back(e1);
    g->prof_kind.push_back(is_h + 2 * mode);
  }
  return 0;
}

int launch_inject(emm_grid *g, const DevState &s, const DevRun &r, int magnetic, int pairfix) {
  k_inject<<<s.nsrc, 128, 0, g->stream>>>(g->dg, s, r.src_off, r.src_idx, r.src_w, magnetic, pairfix);
  EMM_LAUNCH_CHECK(g, "k_inject");
  return 0;
}

int launch_check_acc(emm_grid *g, const DevState &s, const DevRun &r) {
  if (r.nchk <= 0) return 0;
  dim3 grid((r.nchk + 255) / 256, 6, s.nsrc);
  k_check_acc<<<grid, 256, 0, g->stream>>>(g->dg, s, r.chk_idx, r.nchk, r.C, r.twE64, r.twH64);
  EMM_LAUNCH_CHECK(g, "k_check_acc");
  return 0;
}

int launch_rec_acc(emm_grid *g, const DevState &s, const DevRun &r) {
  if (r.nf_rec <= 0 || r.nrec_nodes <= 0) return 0;
  dim3 grid((r.nrec_nodes + 255) / 256, 6, s.nsrc);
  k_rec_acc<<<grid, 256, 0, g->stream>>>(g->dg, s, r.rec_idx, r.nrec_nodes, r.nf_rec, r.RA, r.twEf, r.twHf);
  EMM_LAUNCH_CHECK(g, "k_rec_acc");
  return 0;
}

int launch_check_acc_group(emm_grid *g, const DevState &s, const DevRun &r, int m) {
  if (r.nchk <= 0) return 0;
  dim3 grid((r.nchk + 255) / 256, 6, s.nsrc);
  k_check_acc_group<<<grid, 256, 0, g->stream>>>(g->dg, s, r.chk_idx, r.nchk, r.C, r.twE64, r.twH64, g->tile_base[0][0], g->tile_base[0][1],
                                                 g->tile_base[0][2], g->tile_base[1][0], g->tile_base[1][1], g->tile_base[1][2], m);
  EMM_LAUNCH_CHECK(g, "k_check_acc_group");
  return 0;
}

int launch_check(emm_grid *g, const DevState &s, const DevRun &r, int it_min, double tol, int stop_enabled) {
  int nb = (r.nchk + 255) / 256;
  if (nb > kCheckBlocks) nb = kCheckBlocks;
  if (nb < 1) nb = 1;
  dim3 grid(nb, 6, s.nsrc);
  k_check_reduce<<<grid, 256, 0, g->stream>>>(s, r.nchk, r.C, r.Cprev, r.red_part);
  EMM_LAUNCH_CHECK(g, "k_check_reduce");
  k_check_final<<<(s.nsrc + 31) / 32, 32, 0, g->stream>>>(s, r.red_part, nb, r.delta, r.nsteps, r.status, it_min, tol, stop_enabled);
  EMM_LAUNCH_CHECK(g, "k_check_final");
  return 0;
}

int launch_step_end(emm_grid *g, const DevState &s) {
  k_step_end<<<1, 1, 0, g->stream>>>(s);
  EMM_LAUNCH_CHECK(g, "k_step_end");
  return 0;
}

int launch_rec_interp(emm_grid *g, const DevState &s, const DevRun &r, int nf, int nrec, int np3) {
  if (nrec <= 0 || nf <= 0) return 0;
  dim3 grid(nrec, 6 * nf, s.nsrc);
  if (grid.y > 65535) return fail(EMM_EINVAL, "launch_rec_interp: too many frequencies");
  k_rec_interp<<<grid, 32, 0, g->stream>>>(g->dg, s, r.rec_idx, r.rec_w, r.RA, nf, nrec, np3, r.nf_rec > 0 ? 1 : 0, r.rec_out);
  EMM_LAUNCH_CHECK(g, "k_rec_interp");
  return 0;
}

}  // namespace emm
