// emm_kernels.cuh -- launch wrappers implemented in emm_kernels.cu / emm_air.cu.
#pragma once
#include "emm_internal.h"

namespace emm {

// host-visible description of the per-run device buffers that are not in DevState
struct DevRun {
  // sources
  int *src_off = nullptr;      // [nsrc*3+1] offsets into src_idx / src_w (component-major per source)
  int *src_idx = nullptr;      // node index inside one source's volume
  float *src_w = nullptr;      // dt/eps * W (c-6)
  long long *cell_idx = nullptr;  // [nsrc*3*np^3*4] raw cells around the source nodes (effective medium at the sources)
  int *cell_which = nullptr;
  float *cell_val = nullptr;
  // check set
  int *chk_idx = nullptr;
  int nchk = 0;
  double2 *C = nullptr, *Cprev = nullptr;   // [nsrc][6][nchk]
  double2 *twE64 = nullptr, *twH64 = nullptr;  // [max_steps] lowest frequency, fp64
  double *red_part = nullptr;  // [nsrc][6][2][kCheckBlocks] per-block partial sums of the check (summed in a fixed order)
  float *cpml[3][4] = {{nullptr, nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr, nullptr}};   // [axis]: a-, b-, a+, b+
  double *delta = nullptr;     // [nsrc][2]
  int *nsteps = nullptr;       // [nsrc]
  int *status = nullptr;       // [nsrc]
  // receivers
  int *rec_idx = nullptr;      // [6][nrec*np^3]
  double *rec_w = nullptr;     // [6][nrec*np^3] interpolation weights (tensor products)
  double2 *rec_out = nullptr;  // [nsrc][nf][nrec][6] accumulators interpolated to the receivers
  int nrec_nodes = 0;
  // receivers-only DTFT (emm_run_opts.sparse_dft): fp64 accumulators at the receiver stencil nodes
  double2 *RA = nullptr;       // [nsrc][nf][6][nrec*np^3]
  double2 *twEf = nullptr, *twHf = nullptr;   // [max_steps][nf] twiddles of every frequency, fp64
  int nf_rec = 0;              // number of frequencies in RA (0: mode off)
  // air boundary scratch: complex planes [1 + r][M2][M1] (plane route) or sep_air_scratch() elements (separable route)
  float2 *air = nullptr;
  void *sp_ws[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // cuFFT work areas of the separable route
  // emm_sensitivity: [2][sens_layers][ny][nx] (d/d sigma_h, d/d sigma_v) of the cell layers in flight
  double2 *sens = nullptr;
  int sens_layers = 0;
};

// one E (is_h=0) or H (is_h=1) update of every unfinished source: curl + CPML + update + DTFT
// mode: 0 = one DTFT term per step; paired DTFT: 1 = accumulator-free step of this kernel, 2 = its two-term step
// harg: mode 2 = number of history levels (earlier buffers of the ring) the closing pass takes; unused otherwise
int launch_update(emm_grid *g, const DevState &s, int is_h, int part, int mode, int harg, cudaStream_t st);
// tile pipeline of the accumulator-free update (emm_tile.cu): descriptors for a run's field rings; one launch over z chunks
int tile_make_maps(emm_grid *g, const DevState &s);
int launch_tile(emm_grid *g, const DevGrid &dg, const DevState &s, int is_h, int kc, int nchunks, int chunk0, int sel, cudaStream_t st);
void tile_dims(int *tx, int *ty);
constexpr int kCheckBlocks = 148;   // blocks per (source, component) of the convergence reduction
constexpr int kPairMaxNF = 5;       // grouped-DTFT instances exist for 1..5 frequencies (the staged, unrolled ones)
#ifndef EMM_GROUP_MAX
#define EMM_GROUP_MAX 8
#endif
constexpr int kGroupMax = EMM_GROUP_MAX;   // largest DTFT group (terms per accumulator pass): history levels + old + new
// default group: measured on B200 (profiles/r1_grouped_dtft.md) -- 8 with 4-5 frequencies (2 blocks per SM), 6 with 1-3
// (3 blocks per SM: the staged history quads of a larger group cost the shared memory of the third block)
inline int default_dtft_group(int nf) { return nf >= 4 ? (kGroupMax < 8 ? kGroupMax : 8) : (kGroupMax < 6 ? kGroupMax : 6); }
// pairfix: also add the product the two-term kernel misses at the injected nodes (see k_inject)
int launch_inject(emm_grid *g, const DevState &s, const DevRun &r, int magnetic, int pairfix);
int launch_check_acc(emm_grid *g, const DevState &s, const DevRun &r);
// the same sums for the m steps of a DTFT group at once, from the levels the field ring still holds (oldest first)
int launch_check_acc_group(emm_grid *g, const DevState &s, const DevRun &r, int m);
int launch_rec_acc(emm_grid *g, const DevState &s, const DevRun &r);
int launch_check(emm_grid *g, const DevState &s, const DevRun &r, int it_min, double tol, int stop_enabled);
int launch_step_end(emm_grid *g, const DevState &s);
int launch_rec_interp(emm_grid *g, const DevState &s, const DevRun &r, int nf, int nrec, int np3);
// air-water boundary (Eq. 17-21): ghost planes of Ex,Ey (is_h=0) or Hx,Hy (is_h=1)
int launch_air(emm_grid *g, const DevState &s, const DevRun &r, int is_h, cudaStream_t st);
// separable route of the same boundary for non-uniform x-y (emm_air_sep.cu); launch_air dispatches to it when g->sep_air
int launch_air_sep(emm_grid *g, const DevState &s, const DevRun &r, int is_h, cudaStream_t st);
// one-launch route for a uniform x-y plane that fits the shared memory of a thread-block cluster (emm_air_cluster.cu);
// air_cluster_plan picks the cluster size on the current device (0: does not fit), launch_air dispatches when g->air_cluster
int air_cluster_plan(emm_grid *g);
int launch_air_cluster(emm_grid *g, const DevState &s, const DevRun &r, int is_h, cudaStream_t st);
size_t sep_air_scratch(const emm_grid *g, int nsrc);
int sep_air_make_plans(emm_grid *g, int nsrc);
// model: effective medium (Eq. 26) -> min sigma (for Eq. 15) and dt/eps
int launch_model_scan(emm_grid *g, const float *d_sh, const float *d_sv, unsigned long long *d_out /* [7] */);
int launch_gather_cells(emm_grid *g, const float *d_sh, const float *d_sv, const long long *d_idx, const int *d_which, int n, float *d_out);
int launch_sigma_min(emm_grid *g, const float *d_sh, const float *d_sv, double *d_min);
int launch_make_ce(emm_grid *g, const float *d_sh, const float *d_sv, double scale);
// sensitivity kernel of an E-field datum (emm_sens.cu): cell layers [ck0, ck0 + nlayers) into d_h / d_v [nlayers][ny][nx]
constexpr int kSensLayers = 8;
int launch_sensitivity(emm_grid *g, const DevState &s, int isrc, int iadj, int ifreq, double scale_re, double scale_im, int ck0,
                       int nlayers, double2 *d_h, double2 *d_v);

}  // namespace emm
