// emm_sens.cu -- sensitivity (Frechet) kernel of an electric-field datum with respect to the cell conductivities
// (gradient accumulation for inversion; PAPER.md L11, L825 name inversion as the purpose of the
// full-grid frequency-domain fields and give no formula: DESIGN.md [R14]).
//
// For a transmitter a and a unit dipole b at the receiver, both electric, the datum d = dir_b . G^EE(receiver; a) changes
// with the effective conductivity of an E node n by  V(n) G_c(n; a) G_c(n; b)  (reciprocity; G = sc F_E / J', Eq. 7).  The
// effective conductivity of a node is the area-weighted mean of the four cells around its edge (Eq. 26, [R3]) and V(n) is
// the product of the cell width along the edge and the two dual widths across it ([R7]); the dual widths are the
// denominators of the area weights, so the share of a cell in a node times the node volume is a quarter of the CELL
// volume, for every node and every spacing:
//
//   d d / d sigma_h[cell] = V_cell/4 * sum over the 4 x-edges and the 4 y-edges of the cell of  G_c(edge; a) G_c(edge; b)
//   d d / d sigma_v[cell] = V_cell/4 * sum over the 4 z-edges of the cell of                     G_3(edge; a) G_3(edge; b)
//
// with only the edges whose node lies inside the DTFT box [R11] (accumulators exist nowhere else).  Padding cells count
// towards the model cell they replicate [R1]; the air layer above z = 0 is not a model parameter.  One thread per model
// cell gathers its own padded cells and edges in a fixed order (no atomics: the result does not depend on scheduling);
// products and sums in fp64 from the fp32 accumulators.
#include "emm_kernels.cuh"

namespace emm {
namespace {

struct SensArgs {
  const float2 *Fa[3], *Fb[3];    // E accumulators of the chosen frequency, [NZB][N2][P1] each
  const double *xn[3];            // padded node coordinates [N+1]
  int N[3], lo[3], nc[3], blo[3], bhi[3];
  int P1;
  long long PS;
  int air;                        // 1: the cells above index lo[2] are air
  double2 scale;                  // sc^2 / (J'_a J'_b) / 4
  int ck0, nlayers;               // cell layers [ck0, ck0 + nlayers) of the model go to out[0 .. nlayers)
  double2 *out_h, *out_v;         // [nlayers][ny][nx]
};

__device__ __forceinline__ void cmac(double2 &acc, const float2 a, const float2 b) {
  acc.x += (double)a.x * (double)b.x - (double)a.y * (double)b.y;
  acc.y += (double)a.x * (double)b.y + (double)a.y * (double)b.x;
}

__global__ void __launch_bounds__(128) k_sensitivity(const SensArgs A) {
  const int ci = blockIdx.x * blockDim.x + threadIdx.x;
  const int cj = blockIdx.y;
  const int layer = blockIdx.z;
  if (ci >= A.nc[0]) return;
  const int cc[3] = {ci, cj, A.ck0 + layer};
  // padded cells that replicate this model cell, cut down to those with an edge node in the DTFT box
  int qlo[3], qhi[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    qlo[a] = cc[a] == 0 ? 0 : cc[a] + A.lo[a];
    qhi[a] = cc[a] == A.nc[a] - 1 ? A.N[a] - 1 : cc[a] + A.lo[a];
    if (a == 2 && A.air && cc[a] == 0) qlo[a] = A.lo[a];
    qlo[a] = max(qlo[a], A.blo[a] - 1);
    qhi[a] = min(qhi[a], A.bhi[a]);
  }
  double2 sh = make_double2(0.0, 0.0), sv = make_double2(0.0, 0.0);
  for (int q2 = qlo[2]; q2 <= qhi[2]; ++q2)
    for (int q1 = qlo[1]; q1 <= qhi[1]; ++q1)
      for (int q0 = qlo[0]; q0 <= qhi[0]; ++q0) {
        const int q[3] = {q0, q1, q2};
        const double vc = (A.xn[0][q0 + 1] - A.xn[0][q0]) * (A.xn[1][q1 + 1] - A.xn[1][q1]) * (A.xn[2][q2 + 1] - A.xn[2][q2]);
        double2 eh = make_double2(0.0, 0.0), ev = make_double2(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const int a1 = (c + 1) % 3, a2 = (c + 2) % 3;
          if (q[c] < A.blo[c] || q[c] > A.bhi[c]) continue;            // the edge's own node index along the edge
#pragma unroll
          for (int e1 = 0; e1 < 2; ++e1)
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2) {
              int n[3];
              n[c] = q[c];
              n[a1] = q[a1] + e1;
              n[a2] = q[a2] + e2;
              if (n[a1] < A.blo[a1] || n[a1] > A.bhi[a1] || n[a2] < A.blo[a2] || n[a2] > A.bhi[a2]) continue;
              const long long at = (long long)(n[2] - A.blo[2]) * A.PS + (long long)n[1] * A.P1 + n[0];
              cmac(c == 2 ? ev : eh, A.Fa[c][at], A.Fb[c][at]);
            }
        }
        sh.x += vc * eh.x; sh.y += vc * eh.y;
        sv.x += vc * ev.x; sv.y += vc * ev.y;
      }
  const size_t o = ((size_t)layer * A.nc[1] + cj) * A.nc[0] + ci;
  A.out_h[o] = make_double2(A.scale.x * sh.x - A.scale.y * sh.y, A.scale.x * sh.y + A.scale.y * sh.x);
  A.out_v[o] = make_double2(A.scale.x * sv.x - A.scale.y * sv.y, A.scale.x * sv.y + A.scale.y * sv.x);
}

}  // namespace

// cell layers [ck0, ck0 + nlayers) of the kernel of sources (isrc, iadj), frequency ifreq, into d_h / d_v [nlayers][ny][nx]
int launch_sensitivity(emm_grid *g, const DevState &s, int isrc, int iadj, int ifreq, double scale_re, double scale_im, int ck0,
                       int nlayers, double2 *d_h, double2 *d_v) {
  SensArgs A{};
  const size_t comp = (size_t)g->dg.NZB * g->dg.PS;
  for (int c = 0; c < 3; ++c) {
    A.Fa[c] = s.F + (((size_t)isrc * s.nf + ifreq) * 6 + c) * comp;
    A.Fb[c] = s.F + (((size_t)iadj * s.nf + ifreq) * 6 + c) * comp;
    A.xn[c] = g->T.xn[c];
    A.N[c] = g->N[c];
    A.lo[c] = g->lo[c];
    A.nc[c] = g->nc[c];
    A.blo[c] = g->blo[c];
    A.bhi[c] = g->bhi[c];
  }
  A.P1 = g->P1;
  A.PS = g->dg.PS;
  A.air = g->top == EMM_TOP_AIR;
  A.scale = make_double2(scale_re, scale_im);
  A.ck0 = ck0;
  A.nlayers = nlayers;
  A.out_h = d_h;
  A.out_v = d_v;
  const dim3 grid((g->nc[0] + 127) / 128, g->nc[1], nlayers);
  k_sensitivity<<<grid, 128, 0, g->stream>>>(A);
  ++g->launches;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(EMM_ECUDA, "k_sensitivity launch: %s", cudaGetErrorString(e));
  return 0;
}

}  // namespace emm
