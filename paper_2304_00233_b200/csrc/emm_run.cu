// emm_run.cu -- device binding, emm_model_set and the run driver (Algorithm 1).
// Host code only prepares tables (fp64) and enqueues kernels; no field arithmetic happens on the host.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "emm_kernels.cuh"

namespace emm {

bool make_stencil(const double *S, int n, double t, int p, int lo_ok, int hi_ok, bool clamp, Stencil1 *st);

struct Run {
  int nsrc = 0, nf = 0, nrec = 0, np = 4;
  std::vector<double> freqs;
  std::vector<std::complex<double>> wp;     // omega' (Eq. 4)
  int fmin = 0;
  double fmax = 0, beta = 0, t0 = 0, tol = 1e-6;
  int max_steps = 0, fixed_steps = 0, check_every = 100, check_set = EMM_CHECK_FACES;
  int it_min = 0, it_host = 0, table_steps = 0, dtft_every = 1;
  bool sparse = false;                   // receivers-only DTFT (emm_run_opts.sparse_dft)
  bool chk_grouped = false;              // check-set sums taken once per DTFT group from the field ring (no injected node in the set)
  int group = 1;                         // grouped DTFT: terms of Eq. 25 per accumulator pass (emm_run_opts.dtft_pair); 1 = one per step
  std::vector<double> wav, wavh;            // s(it dt), s((it+1/2) dt) rounded to fp32 (what the device injects)
  std::vector<int> mag;                     // [nsrc] 1 = magnetic dipole
  bool any_mag = false, any_el = false;
  std::vector<Stencil1> rst;                // [nrec][6][3]
  std::vector<int> nsteps, done, status;
  DevState ds{};
  DevRun dr{};
  int nrec_nodes = 0;
  // one CUDA graph = check_every consecutive steps (captured once, replayed; the kernels read the step index
  // from device memory, so replays need no parameter update)
  cudaGraphExec_t chunk_graph = nullptr;
  bool graph_failed = false;
  long long kernels_per_chunk = 0;
  ~Run() { if (chunk_graph) cudaGraphExecDestroy(chunk_graph); }
};

#define CU(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return fail(EMM_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));        \
  } while (0)

static size_t vol(const emm_grid *g) { return (size_t)g->P1 * g->N[1] * g->N[2]; }

// cuFFT plans of the air boundary; their work areas are carved from the caller's workspace
static int ensure_plans(emm_grid *g) {
  if (g->top != EMM_TOP_AIR || g->have_plans) return 0;
  // non-uniform x-y: separable route with batched 1-D transforms (emm_air_sep.cu) unless the grid asks for the
  // plane-sized one (emm_grid_opts.air_route)
  g->sep_air = !g->uniform_xy && g->air_route != 1;
  if (g->sep_air) {             // its plans are batched over the sources of a run: made by emm_workspace_bytes / emm_run_begin
    g->have_plans = true;
    return 0;
  }
  int n[2] = {g->M2, g->M1};
  cufftHandle *pl[3] = {&g->plan_fwd, &g->plan_inv_e, &g->plan_inv_h};
  const int batch[3] = {1, g->r - 1, g->r};
  for (int q = 0; q < 3; ++q) {
    g->fft_ws[q] = 0;
    if (batch[q] < 1) continue;
    if (cufftCreate(pl[q]) != CUFFT_SUCCESS) return fail(EMM_ECUDA, "cufftCreate failed (no CUDA device?)");
    cufftSetAutoAllocation(*pl[q], 0);
    if (cufftMakePlanMany(*pl[q], 2, n, nullptr, 1, g->M1 * g->M2, nullptr, 1, g->M1 * g->M2, CUFFT_C2C, batch[q],
                          &g->fft_ws[q]) != CUFFT_SUCCESS)
      return fail(EMM_ECUDA, "cufftMakePlanMany failed for a %d x %d plane", g->M2, g->M1);
  }
  g->have_plans = true;
  return 0;
}

// per-grid region: FD tables, node coordinates, dt/eps, air-boundary tables, cuFFT work areas
static void layout_fixed(emm_grid *g, Arena &A) {
  const int r2 = 2 * g->r;
  for (int a = 0; a < 3; ++a) {
    const size_t n = (size_t)std::max(g->N[a], a == 0 ? g->P1 : 0) + 4;
    g->T.cm[a] = A.take<float>(n * r2);
    g->T.cp[a] = A.take<float>(n * r2);
    g->T.xn[a] = A.take<double>((size_t)g->N[a] + 1);
  }
  for (int c = 0; c < 3; ++c) g->T.ce[c] = A.take<float>(vol(g));
  g->T.sig_h = A.take<float>((size_t)g->nc[0] * g->nc[1] * g->nc[2]);
  g->T.sig_v = A.take<float>((size_t)g->nc[0] * g->nc[1] * g->nc[2]);
  if (g->top == EMM_TOP_AIR) {
    g->T.kx = A.take<float>(g->M1);
    g->T.ky = A.take<float>(g->M2);
    g->T.tw1 = A.take<float2>(g->M1);
    g->T.tw2 = A.take<float2>(g->M2);
    if (!g->uniform_xy)
      for (int a = 0; a < 2; ++a)
        for (int l = 0; l < 2; ++l) {
          const int M = a == 0 ? g->M1 : g->M2;
          g->T.ta_start[a][l] = A.take<int>(M);
          g->T.ta_w[a][l] = A.take<float>((size_t)4 * M);
          g->T.fa_start[a][l] = A.take<int>(g->N[a]);
          g->T.fa_w[a][l] = A.take<float>((size_t)4 * g->N[a]);
        }
    for (int q = 0; q < 3; ++q) g->T.fft_ws[q] = A.take<char>(g->fft_ws[q] + 256);
  }
}

static size_t chk_count(const emm_grid *g, int check_set) {
  const size_t n0 = g->bhi[0] - g->blo[0] + 1, n1 = g->bhi[1] - g->blo[1] + 1, n2 = g->bhi[2] - g->blo[2] + 1;
  if (check_set == EMM_CHECK_CORNERS) return 8;
  if (check_set == EMM_CHECK_FULL) return n0 * n1 * n2;
  const size_t i0 = n0 > 2 ? n0 - 2 : 0, i1 = n1 > 2 ? n1 - 2 : 0, i2 = n2 > 2 ? n2 - 2 : 0;
  return n0 * n1 * n2 - i0 * i1 * i2;
}

// per-run region
// nf = frequencies with full-grid accumulators, nf_rec = frequencies kept at the receiver stencils only (one of the two is 0)
static void layout_run(emm_grid *g, Arena &A, int nsrc, int nf, int nf_rec, int table_steps, int nrec, size_t nchk, int nslots, DevState &s, DevRun &r) {
  const size_t V = vol(g), PS = (size_t)g->P1 * g->N[1];
  const int np = std::max(2 * g->r, 4);
  const size_t np3 = (size_t)np * np * np;
  // fields: a ring of nbuf buffers per component (nbuf = 1 unless the run groups more than two DTFT terms); buffer 0 is
  // where the fields live outside such a group
  const int nbuf = nslots > 0 ? nslots + 2 : 1;
  for (int c = 0; c < 3; ++c) { s.E[c] = A.take<float>(V * nsrc * nbuf); s.H[c] = A.take<float>(V * nsrc * nbuf); }
  for (int c = 0; c < 3; ++c) { s.Eo[c] = s.Ho[c] = nullptr; s.hist[0][c] = s.hist[1][c] = nullptr; }
  s.nbuf = nbuf;
  s.hstride = (long long)V * nsrc;
  for (int k = 0; k < 2; ++k)
    for (int q = 0; q < 2; ++q) {
      s.psx[k][q] = A.take<float>((size_t)nsrc * g->N[2] * g->N[1] * g->XS);
      s.psy[k][q] = A.take<float>((size_t)nsrc * g->N[2] * 2 * g->nb * g->P1);
      s.psz[k][q] = A.take<float>((size_t)nsrc * 2 * g->nb * PS);
    }
  const size_t nzb = g->bhi[2] - g->blo[2] + 1;
  s.F = A.take<float2>((size_t)nsrc * nf * 6 * nzb * PS);

  s.twE = A.take<float2>((size_t)table_steps * nf);
  s.twH = A.take<float2>((size_t)table_steps * nf);
  s.wav = A.take<float>(table_steps);
  s.wavh = A.take<float>(table_steps);
  s.src_mag = A.take<int>(nsrc);
  s.it = A.take<int>(1);
  s.done = A.take<int>(nsrc);
  s.nf = nf;
  s.nsrc = nsrc;
  r.src_off = A.take<int>((size_t)nsrc * 3 + 1);
  r.src_idx = A.take<int>((size_t)nsrc * 3 * np3);
  r.src_w = A.take<float>((size_t)nsrc * 3 * np3);
  r.cell_idx = A.take<long long>((size_t)nsrc * 3 * np3 * 4);
  r.cell_which = A.take<int>((size_t)nsrc * 3 * np3 * 4);
  r.cell_val = A.take<float>((size_t)nsrc * 3 * np3 * 4);
  r.chk_idx = A.take<int>(nchk);
  r.nchk = (int)nchk;
  r.C = A.take<double2>((size_t)nsrc * 6 * nchk);
  r.Cprev = A.take<double2>((size_t)nsrc * 6 * nchk);
  r.twE64 = A.take<double2>(table_steps);
  r.twH64 = A.take<double2>(table_steps);
  r.delta = A.take<double>((size_t)nsrc * 2);
  r.nsteps = A.take<int>(nsrc);
  r.status = A.take<int>(nsrc);
  r.rec_idx = A.take<int>((size_t)6 * nrec * np3);
  r.rec_w = A.take<double>((size_t)6 * nrec * np3);
  r.rec_out = A.take<double2>((size_t)nsrc * (nf + nf_rec) * nrec * 6);
  r.nf_rec = nf_rec;
  r.RA = A.take<double2>((size_t)nsrc * nf_rec * 6 * nrec * np3);
  r.twEf = A.take<double2>((size_t)table_steps * nf_rec);
  r.twHf = A.take<double2>((size_t)table_steps * nf_rec);
  if (g->top == EMM_TOP_AIR)   // FFT planes [1 + r][M2][M1] + (non-uniform x-y) the x-interpolated rows [N2][M1]
    r.air = A.take<float2>(g->sep_air ? sep_air_scratch(g, nsrc) : (size_t)(1 + g->r) * g->M1 * g->M2 + (g->uniform_xy ? 0 : (size_t)g->N[1] * g->M1));
  if (g->top == EMM_TOP_AIR && g->sep_air)
    for (int q = 0; q < 8; ++q) r.sp_ws[q] = A.take<char>(g->sp_ws[q] + 256);
  for (int a = 0; a < 3; ++a)            // CPML coefficients (Eq. 24) at node and half-node positions
    for (int q = 0; q < 4; ++q) r.cpml[a][q] = A.take<float>(2 * g->nb);
  r.red_part = A.take<double>((size_t)nsrc * 6 * 2 * kCheckBlocks);
  // emm_sensitivity: the kernel leaves the device a few cell layers at a time (two sources with full-grid accumulators needed)
  r.sens_layers = nf > 0 && nsrc >= 2 ? std::min(g->nc[2], kSensLayers) : 0;
  r.sens = A.take<double2>((size_t)2 * r.sens_layers * g->nc[1] * g->nc[0]);
}

template <class T>
static int upload(emm_grid *g, T *dst, const std::vector<T> &v) {
  if (v.empty()) return 0;
  CU(cudaMemcpyAsync(dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, g->stream));
  CU(cudaStreamSynchronize(g->stream));    // v may be a temporary (pageable memory)
  return 0;
}

static void free_run(emm_grid *g) {
  delete g->run;
  g->run = nullptr;
}

}  // namespace emm

using namespace emm;

extern "C" void emm_grid_destroy(emm_grid *g) {
  if (!g) return;
  free_run(g);
  for (cudaEvent_t e : g->prof_ev) cudaEventDestroy(e);
  for (cudaEvent_t e : g->ev) if (e) cudaEventDestroy(e);
  if (g->stream_b) cudaStreamDestroy(g->stream_b);
  if (g->have_plans) {
    if (g->plan_fwd) cufftDestroy(g->plan_fwd);
    if (g->plan_inv_e) cufftDestroy(g->plan_inv_e);
    if (g->plan_inv_h) cufftDestroy(g->plan_inv_h);
    for (cufftHandle h : g->sp) if (h) cufftDestroy(h);
  }
  delete g;
}

extern "C" size_t emm_workspace_bytes(emm_grid *g, int nsrc, int nfreq, int max_steps, int nrec, int dtft_pair) {
  if (!g || nsrc < 1 || nfreq < 0 || nrec < 0) { fail(EMM_EINVAL, "emm_workspace_bytes: bad arguments"); return 0; }
  if (ensure_plans(g)) return 0;
  if (g->sep_air && sep_air_make_plans(g, nsrc)) return 0;
  if (max_steps <= 0) max_steps = 100000;
  const DevTables keep = g->T;       // dry-run layout: the live grid's pointers are restored below
  Arena A;
  layout_fixed(g, A);
  const size_t fixed = A.off;
  DevState s{};
  DevRun r{};
  // full-grid accumulators with the field ring of the DTFT group the runs will ask for (emm_run_opts.dtft_pair; a run that
  // asks for a larger group than fits gets the largest that does), or the receivers-only layout: whichever is larger
  const int group = dtft_pair < 0 || nfreq < 1 || nfreq > kPairMaxNF ? 1 : std::min(kGroupMax, dtft_pair >= 2 ? dtft_pair : default_dtft_group(nfreq));
  layout_run(g, A, nsrc, nfreq, 0, max_steps + 1, nrec, chk_count(g, EMM_CHECK_FACES), group > 2 ? group - 2 : 0, s, r);
  const size_t full = A.off;
  A.off = fixed;
  layout_run(g, A, nsrc, 0, nfreq, max_steps + 1, nrec, chk_count(g, EMM_CHECK_FACES), 0, s, r);
  g->T = keep;
  return std::max(std::max(full, A.off), fixed + 1024) + 4096;       // emm_model_set keeps a few scalars behind the per-grid region
}

extern "C" int emm_bind_device(emm_grid *g, void *d_workspace, size_t bytes, void *cuda_stream) {
  if (!g || !d_workspace) return fail(EMM_EINVAL, "emm_bind_device: null argument");
  if (reinterpret_cast<uintptr_t>(d_workspace) % 256) return fail(EMM_EINVAL, "emm_bind_device: workspace must be 256-byte aligned");
  int rc = ensure_plans(g);
  if (rc) return rc;
  free_run(g);
  g->have_model = false;
  g->d_ws = d_workspace;
  g->ws_bytes = bytes;
  g->stream = static_cast<cudaStream_t>(cuda_stream);
  if (!g->stream_b) {
    // highest priority: the boundary chain is short and on the critical path of the step; its blocks must get the
    // next free SM slots while the bulk update (thousands of blocks on the main stream) is draining
    int prio_lo = 0, prio_hi = 0;
    CU(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    CU(cudaStreamCreateWithPriority(&g->stream_b, cudaStreamNonBlocking, prio_hi));
    for (cudaEvent_t &e : g->ev) CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  Arena A;
  A.base = static_cast<char *>(d_workspace);
  A.cap = bytes;
  A.dry = false;
  layout_fixed(g, A);
  if (A.overflow) return fail(EMM_ENOMEM, "emm_bind_device: workspace of %zu bytes too small (grid tables need %zu)", bytes, A.off);
  g->fixed_bytes = A.off;
  // upload the per-grid tables
  const int r2 = 2 * g->r;
  for (int a = 0; a < 3; ++a) {
    const size_t n = (size_t)std::max(g->N[a], a == 0 ? g->P1 : 0) + 4;
    std::vector<float> m(n * r2, 0.f), p(n * r2, 0.f);
    for (size_t t = 0; t < (size_t)g->N[a] * r2; ++t) { m[t] = (float)g->cm[a][t]; p[t] = (float)g->cp[a][t]; }
    if ((rc = upload(g, g->T.cm[a], m)) || (rc = upload(g, g->T.cp[a], p)) || (rc = upload(g, g->T.xn[a], g->xn[a]))) return rc;
  }
  if (g->top == EMM_TOP_AIR) {
    for (int a = 0; a < 2; ++a) {
      const int M = a == 0 ? g->M1 : g->M2;
      const double d = a == 0 ? g->dxa : g->dya;
      std::vector<float> k(M);
      for (int n = 0; n < M; ++n) k[n] = (float)(2.0 * kPi * (double)(n <= M / 2 ? n : n - M) / ((double)M * d));
      if ((rc = upload(g, a == 0 ? g->T.kx : g->T.ky, k))) return rc;
      std::vector<float2> tw(M);
      for (int n = 0; n < M; ++n) tw[n] = make_float2((float)std::cos(2.0 * kPi * n / M), (float)-std::sin(2.0 * kPi * n / M));
      if ((rc = upload(g, a == 0 ? g->T.tw1 : g->T.tw2, tw))) return rc;
      if (!g->uniform_xy)
        for (int l = 0; l < 2; ++l) {
          std::vector<int> st(M), sf(g->N[a]);
          std::vector<float> wt((size_t)4 * M), wf((size_t)4 * g->N[a]);
          for (int m = 0; m < M; ++m) { st[m] = g->toaux[a][l][m].start; for (int q = 0; q < 4; ++q) wt[4 * m + q] = (float)g->toaux[a][l][m].w[q]; }
          for (int i = 0; i < g->N[a]; ++i) { sf[i] = g->fromaux[a][l][i].start; for (int q = 0; q < 4; ++q) wf[4 * i + q] = (float)g->fromaux[a][l][i].w[q]; }
          if ((rc = upload(g, g->T.ta_start[a][l], st)) || (rc = upload(g, g->T.ta_w[a][l], wt)) ||
              (rc = upload(g, g->T.fa_start[a][l], sf)) || (rc = upload(g, g->T.fa_w[a][l], wf))) return rc;
        }
    }
    air_cluster_plan(g);
    cufftHandle pl[3] = {g->plan_fwd, g->plan_inv_e, g->plan_inv_h};
    const int batch[3] = {1, g->r - 1, g->r};
    for (int q = 0; q < 3; ++q) {
      if (batch[q] < 1 || g->sep_air) continue;
      if (cufftSetStream(pl[q], g->stream_b) != CUFFT_SUCCESS || cufftSetWorkArea(pl[q], g->T.fft_ws[q]) != CUFFT_SUCCESS)
        return fail(EMM_ECUDA, "cufftSetStream/cufftSetWorkArea failed");
    }
  }
  // device view of the grid (CPML and dt/eps pointers are completed later)
  DevGrid &d = g->dg;
  d = DevGrid{};
  d.N1 = g->N[0]; d.N2 = g->N[1]; d.N3 = g->N[2]; d.P1 = g->P1;
  d.PS = (long long)g->P1 * g->N[1];
  d.VS = d.PS * g->N[2];
  d.r = g->r; d.nb = g->nb; d.klo = g->klo;
  d.zslab_lo = g->top == EMM_TOP_CPML;
  for (int a = 0; a < 3; ++a) { d.blo[a] = g->blo[a]; d.bhi[a] = g->bhi[a]; d.cm[a] = g->T.cm[a]; d.cp[a] = g->T.cp[a]; d.ce[a] = g->T.ce[a]; }
  d.NZB = g->bhi[2] - g->blo[2] + 1;
  d.XS = g->XS;
  g->bound = true;
  return 0;
}

// Medium (Eq. 26, [R3]) and time step (Eq. 15-16, [R4]); effective medium evaluated on the device.
extern "C" int emm_model_set(emm_grid *g, const float *sigma_h, const float *sigma_v) {
  if (!g || !sigma_h) return fail(EMM_EINVAL, "emm_model_set: null argument");
  if (!g->bound) return fail(EMM_ECUDA, "emm_model_set: no device workspace bound (emm_bind_device)");
  free_run(g);
  g->have_model = false;
  const size_t nc = (size_t)g->nc[0] * g->nc[1] * g->nc[2];
  g->vti = sigma_v != nullptr;
  // the raw model stays resident in the per-grid region (emm_run_begin reads the cells around the source nodes);
  // validation, slab minima, effective medium and dt/eps are device passes over it: the host never walks the model
  float *d_sh = g->T.sig_h, *d_sv = sigma_v ? g->T.sig_v : g->T.sig_h;
  Arena A;
  A.base = static_cast<char *>(g->d_ws); A.cap = g->ws_bytes; A.dry = false; A.off = g->fixed_bytes;
  double *d_min = A.take<double>(1);
  unsigned long long *d_scan = A.take<unsigned long long>(7);
  if (A.overflow) return fail(EMM_ENOMEM, "emm_model_set: workspace too small");
  CU(cudaMemcpyAsync(d_sh, sigma_h, nc * sizeof(float), cudaMemcpyHostToDevice, g->stream));
  if (sigma_v) CU(cudaMemcpyAsync(d_sv, sigma_v, nc * sizeof(float), cudaMemcpyHostToDevice, g->stream));
  const unsigned long long inf_bits = 0x7ff0000000000000ULL;
  unsigned long long scan[7] = {inf_bits, inf_bits, inf_bits, inf_bits, inf_bits, inf_bits, 0ULL};
  CU(cudaMemcpyAsync(d_min, &inf_bits, sizeof inf_bits, cudaMemcpyHostToDevice, g->stream));
  CU(cudaMemcpyAsync(d_scan, scan, sizeof scan, cudaMemcpyHostToDevice, g->stream));
  int rc = launch_model_scan(g, d_sh, sigma_v ? d_sv : nullptr, d_scan);
  if (rc) return rc;
  if ((rc = launch_sigma_min(g, d_sh, d_sv, d_min))) return rc;
  double smin = 0;
  CU(cudaMemcpyAsync(&smin, d_min, sizeof smin, cudaMemcpyDeviceToHost, g->stream));
  CU(cudaMemcpyAsync(scan, d_scan, sizeof scan, cudaMemcpyDeviceToHost, g->stream));
  CU(cudaStreamSynchronize(g->stream));
  if (scan[6] != 0) return fail(EMM_EINVAL, "emm_model_set: sigma_h and sigma_v must be finite and > 0 (%llu cells are not)", scan[6]);
  if (!(smin > 0) || !std::isfinite(smin)) return fail(EMM_EINVAL, "emm_model_set: non-positive effective conductivity at an updated node");
  g->smin = smin;
  const double vmax = 1.0 / std::sqrt(kMu0 * smin / (2 * g->w0));                       // v = 1/sqrt(mu eps), eps = sigma/(2 w0)
  const double eta = 0.5 * vmax * std::sqrt(g->Dmax[0] * g->Dmax[0] + g->Dmax[1] * g->Dmax[1] + g->Dmax[2] * g->Dmax[2]);
  g->dt = g->cfl / eta;                                                                  // Eq. 15
  if ((rc = launch_make_ce(g, d_sh, d_sv, g->dt * 2 * g->w0))) return rc;
  CU(cudaStreamSynchronize(g->stream));
  g->dg.dtmu = (float)(g->dt / kMu0);
  // CPML reference speed per face = fastest padded cell inside the slab [R5]
  for (int a = 0; a < 3; ++a)
    for (int side = 0; side < 2; ++side) {
      if (a == 2 && side == 0 && g->top == EMM_TOP_AIR) { g->vref[a][side] = 0; continue; }
      double smn;
      std::memcpy(&smn, &scan[2 * a + side], sizeof smn);
      g->vref[a][side] = 1.0 / std::sqrt(kMu0 * smn / (2 * g->w0));
    }
  g->have_model = true;
  return 0;
}

// ---------------------------------------------------------------------------------------------------
namespace emm {

// effective conductivity of E component c at node (i,j,k), same rule as the device pass ([R3]): the four raw cells
// sharing the component's edge (index < 0: air above z = 0) and their area weights; sigma_bar = sum w s / sum w
static void sigma_bar_cells(const emm_grid *g, int c, int i, int j, int k, long long *cell, int *which, double *w) {
  const int idx[3] = {i, j, k};
  const int a1 = (c + 1) % 3, a2 = (c + 2) % 3;        // the two transverse axes
  int n = 0;
  for (int d1 = -1; d1 <= 0; ++d1)
    for (int d2 = -1; d2 <= 0; ++d2, ++n) {
      int q[3] = {idx[0], idx[1], idx[2]};
      q[a1] = std::max(idx[a1] + d1, 0);
      q[a2] = std::max(idx[a2] + d2, 0);
      w[n] = (g->xn[a1][q[a1] + 1] - g->xn[a1][q[a1]]) * (g->xn[a2][q[a2] + 1] - g->xn[a2][q[a2]]);
      int ci = q[0] - g->lo[0], cj = q[1] - g->lo[1], ck = q[2] - g->lo[2];
      which[n] = (c == 2 && g->vti) ? 1 : 0;
      if (g->top == EMM_TOP_AIR && ck < 0) { cell[n] = -1; continue; }
      ci = std::min(std::max(ci, 0), g->nc[0] - 1);
      cj = std::min(std::max(cj, 0), g->nc[1] - 1);
      ck = std::min(std::max(ck, 0), g->nc[2] - 1);
      cell[n] = (long long)ci + (long long)g->nc[0] * ((long long)cj + (long long)g->nc[1] * (long long)ck);
    }
}

static double node_width(const emm_grid *g, int a, int half, int i) {
  return half ? g->xn[a][i + 1] - g->xn[a][i] : g->xh[a][i] - g->xh[a][i - 1];
}

// CPML recursion coefficients (Eq. 24) of one axis, written from reading [R5]: kappa = 1; damping d = d0 s^2 with
// s = (depth into the layer) / (layer thickness) and d0 = 3 v_ref ln(1000) / (2 thickness) (theoretical reflection 1e-3);
// frequency shift alpha = pi (fmax/2) (1 - s), never negative; b = exp(-(d + alpha) dt), a = d (b - 1) / (d + alpha) and
// a = 0 where d = 0.  Depth is measured at the derivative's own location: the node for D-, the half node for D+.
// Slab entry e < nb belongs to the low face (index e), e >= nb to the high face, mirrored (index N-1-(e-nb)), L324-326.
static void cpml_tables(const emm_grid *g, int a, double fmax, std::vector<float> &am, std::vector<float> &bm,
                        std::vector<float> &ap, std::vector<float> &bp) {
  const int N = g->N[a], nb = g->nb;
  const std::vector<double> &xn = g->xn[a], &xh = g->xh[a];
  am.assign(2 * nb, 0.f); ap.assign(2 * nb, 0.f); bm.assign(2 * nb, 1.f); bp.assign(2 * nb, 1.f);
  auto coefficients = [&](double depth, double thickness, double vref, float &a_out, float &b_out) {
    const double s = std::max(depth / thickness, 0.0);
    const double d = 1.5 * vref * std::log(1000.0) / thickness * s * s;
    const double alpha = std::max(kPi * 0.5 * fmax * (1.0 - s), 0.0);
    const double rate = d + alpha;
    b_out = (float)std::exp(-rate * g->dt);
    a_out = d > 0 ? (float)(d / rate * std::expm1(-rate * g->dt)) : 0.f;
  };
  for (int e = 0; e < 2 * nb; ++e) {
    const bool high = e >= nb;
    if (!high && a == 2 && g->top == EMM_TOP_AIR) continue;           // no CPML at the surface (L292)
    const int i = high ? N - 1 - (e - nb) : e;
    // the layer is the outermost nb cells counted from the last updated-side node: [x_0, x_nb] or [x_{N-1-nb}, x_{N-1}]
    const double inner = high ? xn[N - 1 - nb] : xn[nb], outer = high ? xn[N - 1] : xn[0];
    const double thickness = std::fabs(outer - inner), vref = g->vref[a][high ? 1 : 0];
    coefficients(high ? xn[i] - inner : inner - xn[i], thickness, vref, am[e], bm[e]);
    coefficients(high ? xh[i] - inner : inner - xh[i], thickness, vref, ap[e], bp[e]);
  }
}

// source spectrum of Eq. 7: J'(w') = sum s(it dt) e^{i w' it dt}; a magnetic source is centred in the H update,
// M'(w') = sum s((it+1/2) dt) e^{i w' (it+1/2) dt} [R6]; only the terms the DTFT took (decimation)
static std::complex<double> source_spectrum(const emm_grid *g, const Run *R, int s, int f) {
  const std::complex<double> I(0, 1);
  std::complex<double> J = 0;
  for (int it = 0; it < R->nsteps[s]; it += R->dtft_every)
    J += R->mag[s] ? R->wavh[it] * std::exp(I * R->wp[f] * (((double)it + 0.5) * g->dt))
                   : R->wav[it] * std::exp(I * R->wp[f] * ((double)it * g->dt));
  return J;
}

static int enqueue_steps_raw(emm_grid *g, int n) {
  Run *R = g->run;
  int rc;
  int gpos = 0, gsize = 0;                   // grouped DTFT: position in / size of the current group of steps
  for (int q = 0; q < n; ++q) {
    if (R->it_host >= R->table_steps) return fail(EMM_EINVAL, "run: step %d beyond the twiddle table (max_steps)", R->it_host);
    cudaStream_t M = g->stream, B = g->stream_b;
    // Paired DTFT: the steps of this batch are taken two by two.  In the first step of a pair the H kernel adds the terms
    // it and it+1 of F_H (old and new H) and the E kernel none; in the second the E kernel adds the terms it-1 and it of
    // F_E (old and new E) and the H kernel none; a left-over last step takes its single terms as usual.  A batch never
    // crosses a convergence check (enqueue_steps), so every sum is complete where it is read.
    int me = 0, mh = 0, he = -1, hh = -1, fix_e = 0;
    int chk_m = 1;                           // check-set sums: 1 = this step's term now, 0 = later with its group, m = the whole group now
    // s1: injection + E update; s2: E boundary, check set, H update; s3: H boundary, magnetic injection, check
    DevState s1 = R->ds, s2 = R->ds, s3 = R->ds;
    if (R->group > 1) {
      if (gpos >= gsize) {                   // open the next group of this batch: up to `group` steps, at least 2
        gpos = 0;
        gsize = std::min(std::min(R->group, n - q), R->table_steps - R->it_host);
        if (gsize < 2) gsize = 1;
      }
      if (gsize >= 2) {
        // Position p of a group of m steps.  The E kernel closes the group at p = m-1 with m terms: its old E (term m-2),
        // its new E (term m-1) and the m-2 levels before; the H kernel closes it at p = m-2: old H (term m-2), new H
        // (term m-1).  m = 2: the pair of two-term passes, in place.  m > 2: step p reads buffer p of the ring and writes
        // buffer p+1 (the last step writes buffer 0), so that E after step l (term l) stays in buffer l+1 and H before
        // step l (term l) in buffer l until the closing pass has taken them.
        const int m = gsize, p = gpos;
        if (p == m - 1) { me = 2; he = m - 2; } else me = 1;
        if (p == m - 2) { mh = 2; hh = m - 2; } else mh = 1;
        // the electric injection of step p lands in the buffer that holds term p-1 (closing pass: its old E): the missing
        // product goes into the accumulators with the injection
        fix_e = p >= 1;
        if (m > 2 && R->chk_grouped) chk_m = p == m - 1 ? m : 0;
        if (m > 2) {
          const size_t bs = (size_t)R->ds.hstride;
          const int pn = (p + 1) % m;
          for (int c = 0; c < 3; ++c) {
            float *Ein = R->ds.E[c] + p * bs, *Eout = R->ds.E[c] + pn * bs, *Hin = R->ds.H[c] + p * bs, *Hout = R->ds.H[c] + pn * bs;
            s1.E[c] = Ein; s1.Eo[c] = Eout; s1.H[c] = Hin;
            s2.E[c] = Eout; s2.H[c] = Hin; s2.Ho[c] = Hout;
            s3.E[c] = Eout; s3.H[c] = Hout;
            s1.hist[0][c] = R->ds.E[c] + bs;          // E terms 0 .. m-3 sit in buffers 1 .. m-2
            s2.hist[1][c] = R->ds.H[c];               // H terms 0 .. m-3 sit in buffers 0 .. m-3
          }
        }
      }
      ++gpos;
    }
    if (R->any_el && (rc = launch_inject(g, s1, R->dr, 0, fix_e))) return rc;     // Alg. 1 L477 (before the update: same sum)
    if (g->top != EMM_TOP_AIR) {
      if ((rc = launch_update(g, s1, 0, 0, me, he, M))) return rc;                 // L476-479 + E part of L483
      if ((rc = chk_m == 1 ? launch_check_acc(g, s2, R->dr) : chk_m > 1 ? launch_check_acc_group(g, s2, R->dr, chk_m) : 0)) return rc;   // check-set part of L483
      if ((rc = launch_rec_acc(g, s2, R->dr))) return rc;
      if ((rc = launch_update(g, s2, 1, 0, mh, hh, M))) return rc;                 // H part of L483 + L486-489
    } else if (g->prof) {
      // one thing after the other (per-kernel timing): the boundary still runs on its own stream
      if ((rc = launch_update(g, s1, 0, 0, me, he, M))) return rc;
      CU(cudaEventRecord(g->ev[0], M)); CU(cudaStreamWaitEvent(B, g->ev[0], 0));
      if ((rc = launch_air(g, s2, R->dr, 0, B))) return rc;                // L481
      CU(cudaEventRecord(g->ev[1], B)); CU(cudaStreamWaitEvent(M, g->ev[1], 0));
      if ((rc = chk_m == 1 ? launch_check_acc(g, s2, R->dr) : chk_m > 1 ? launch_check_acc_group(g, s2, R->dr, chk_m) : 0)) return rc;
      if ((rc = launch_rec_acc(g, s2, R->dr))) return rc;
      if ((rc = launch_update(g, s2, 1, 0, mh, hh, M))) return rc;
      CU(cudaEventRecord(g->ev[2], M)); CU(cudaStreamWaitEvent(B, g->ev[2], 0));
      if ((rc = launch_air(g, s3, R->dr, 1, B))) return rc;                // L491
      CU(cudaEventRecord(g->ev[3], B)); CU(cudaStreamWaitEvent(M, g->ev[3], 0));
    } else {
      // The boundary only feeds the z chunks next to the surface: those chunks and the FFT boundary form a short
      // chain on the helper stream while the bulk of the grid is updated on the main stream (fork/join per step).
      CU(cudaEventRecord(g->ev[0], M)); CU(cudaStreamWaitEvent(B, g->ev[0], 0));      // fork (after the injection)
      if ((rc = launch_update(g, s1, 0, 1, me, he, B))) return rc;                 // E, surface chunks
      CU(cudaEventRecord(g->ev[1], B));
      if ((rc = launch_air(g, s2, R->dr, 0, B))) return rc;                // L481
      if ((rc = launch_update(g, s1, 0, 2, me, he, M))) return rc;                 // E, bulk
      CU(cudaEventRecord(g->ev[2], M));
      CU(cudaStreamWaitEvent(M, g->ev[1], 0));                                // H bulk and the check set read surface-chunk E
      if ((rc = chk_m == 1 ? launch_check_acc(g, s2, R->dr) : chk_m > 1 ? launch_check_acc_group(g, s2, R->dr, chk_m) : 0)) return rc;
      if ((rc = launch_rec_acc(g, s2, R->dr))) return rc;
      CU(cudaEventRecord(g->ev[4], M));
      if ((rc = launch_update(g, s2, 1, 2, mh, hh, M))) return rc;                 // H, bulk
      CU(cudaStreamWaitEvent(B, g->ev[2], 0)); CU(cudaStreamWaitEvent(B, g->ev[4], 0));
      if ((rc = launch_update(g, s2, 1, 1, mh, hh, B))) return rc;                 // H, surface chunks (after bulk E, check set, ghost E)
      if ((rc = launch_air(g, s3, R->dr, 1, B))) return rc;                // L491
      CU(cudaEventRecord(g->ev[3], B)); CU(cudaStreamWaitEvent(M, g->ev[3], 0));      // join
    }
    if (R->any_mag && (rc = launch_inject(g, s3, R->dr, 1, mh == 2))) return rc;    // L488, after the H update and its boundary
    if (R->nf > 0 && (R->it_host + 1) % R->check_every == 0 &&
        (rc = launch_check(g, s3, R->dr, R->it_min, R->tol, R->fixed_steps ? 0 : 1))) return rc;   // L493-498
    if ((rc = launch_step_end(g, R->ds))) return rc;
    R->it_host++;
  }
  return 0;
}

// Whole chunks of check_every steps go through a CUDA graph (launch-bound on small grids: ~10 launches per
// step); the first chunk (first-use set-up of the kernels), the ragged rest, and everything while per-kernel
// profiling is on, are launched directly.
static int enqueue_steps(emm_grid *g, int n) {
  Run *R = g->run;
  int rc;
  while (n > 0) {
    const int ce = R->check_every;
    const bool whole = !g->prof && !R->graph_failed && R->it_host >= ce && R->it_host % ce == 0 && n >= ce && R->it_host + ce <= R->table_steps;
    if (!whole) {
      const int m = std::min(n, ce - R->it_host % ce);
      if ((rc = enqueue_steps_raw(g, m))) return rc;
      n -= m;
      continue;
    }
    if (!R->chunk_graph) {
      cudaGraph_t graph = nullptr;
      const int it_save = R->it_host;
      const long long launches_save = g->launches;
      if (cudaStreamBeginCapture(g->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); R->graph_failed = true; continue; }
      rc = enqueue_steps_raw(g, ce);
      const cudaError_t e = cudaStreamEndCapture(g->stream, &graph);
      R->it_host = it_save;
      R->kernels_per_chunk = g->launches - launches_save;
      g->launches = launches_save;
      if (rc || e != cudaSuccess || !graph || cudaGraphInstantiate(&R->chunk_graph, graph, 0) != cudaSuccess) {
        cudaGetLastError();
        if (graph) cudaGraphDestroy(graph);
        R->chunk_graph = nullptr;
        R->graph_failed = true;          // fall back to direct launches (same kernels, same order)
        continue;
      }
      cudaGraphDestroy(graph);
    }
    if (cudaGraphLaunch(R->chunk_graph, g->stream) != cudaSuccess) return fail(EMM_ECUDA, "cudaGraphLaunch failed: %s", cudaGetErrorString(cudaGetLastError()));
    g->launches += R->kernels_per_chunk;
    R->it_host += ce;
    n -= ce;
  }
  return 0;
}

static int fetch_flags(emm_grid *g) {
  Run *R = g->run;
  std::vector<int> dn(R->nsrc), ns(R->nsrc), stt(R->nsrc);
  CU(cudaMemcpyAsync(dn.data(), R->ds.done, sizeof(int) * R->nsrc, cudaMemcpyDeviceToHost, g->stream));
  CU(cudaMemcpyAsync(ns.data(), R->dr.nsteps, sizeof(int) * R->nsrc, cudaMemcpyDeviceToHost, g->stream));
  CU(cudaMemcpyAsync(stt.data(), R->dr.status, sizeof(int) * R->nsrc, cudaMemcpyDeviceToHost, g->stream));
  CU(cudaStreamSynchronize(g->stream));
  for (int s = 0; s < R->nsrc; ++s) {
    if (dn[s] && !R->done[s]) { R->done[s] = 1; R->nsteps[s] = ns[s]; R->status[s] = stt[s]; }
    if (!R->done[s]) R->nsteps[s] = R->it_host;
  }
  return 0;
}

}  // namespace emm

extern "C" int emm_run_begin(emm_grid *g, const emm_src *src, int nsrc, const double *freqs, int nf, const double *rec, int nrec,
                             const emm_run_opts *o) {
  if (!g || !src || !freqs || !o || (nrec > 0 && !rec)) return fail(EMM_EINVAL, "emm_run_begin: null argument");
  if (!g->bound) return fail(EMM_ECUDA, "emm_run_begin: no device workspace bound");
  if (!g->have_model) return fail(EMM_EINVAL, "emm_run_begin: emm_model_set not called");
  if (nsrc < 1 || nf < 0 || nrec < 0) return fail(EMM_EINVAL, "emm_run_begin: bad counts");
  if (nf == 0 && (o->fixed_steps <= 0 || nrec > 0))   // pure time stepping (no DTFT): nothing to converge on or to return
    return fail(EMM_EINVAL, "emm_run_begin: nfreq = 0 needs fixed_steps > 0 and no receivers");
  free_run(g);
  Run *R = new (std::nothrow) Run();
  if (!R) return fail(EMM_ENOMEM, "emm_run_begin: out of memory");
  g->run = R;
  const int r = g->r, nb = g->nb;
  int rc = 0;
  try {
    R->nsrc = nsrc; R->nf = nf; R->nrec = nrec;
    R->max_steps = o->max_steps > 0 ? o->max_steps : 100000;
    R->fixed_steps = o->fixed_steps > 0 ? o->fixed_steps : 0;
    R->tol = o->tol > 0 ? o->tol : 1e-6;
    R->check_every = o->check_every > 0 ? o->check_every : 100;
    R->check_set = o->check_set;
    R->dtft_every = o->dtft_every > 1 ? o->dtft_every : 1;
    R->sparse = o->sparse_dft != 0 && nf > 0;
    {
      const bool can = o->dtft_pair >= 0 && nf >= 1 && nf <= kPairMaxNF && !R->sparse && o->dtft_every >= 0 && o->dtft_every <= 1;
      R->group = !can ? 1 : std::min(kGroupMax, o->dtft_pair >= 2 ? o->dtft_pair : default_dtft_group(nf));
    }
    if (R->check_set < 0 || R->check_set > 2) { free_run(g); return fail(EMM_EINVAL, "emm_run_begin: bad check_set"); }
    R->table_steps = (R->fixed_steps ? R->fixed_steps : R->max_steps) + 1;
    double fhi = 0;
    for (int f = 0; f < nf; ++f) {
      if (!(freqs[f] > 0) || !std::isfinite(freqs[f])) { free_run(g); return fail(EMM_EINVAL, "emm_run_begin: frequencies must be > 0"); }
      R->freqs.push_back(freqs[f]);
      R->wp.push_back(std::complex<double>(1.0, 1.0) * std::sqrt(2 * kPi * freqs[f] * g->w0));   // Eq. 4
      fhi = std::max(fhi, freqs[f]);
      if (freqs[f] < freqs[R->fmin]) R->fmin = f;
    }
    if (nf == 0) fhi = 1.0;
    R->fmax = o->fmax > 0 ? o->fmax : 4.0 * std::sqrt(fhi * g->f0);         // [R8]
    if (o->dtft_every < 0) {   // automatic: the largest m whose sampling rate clears the wavelet band
      const double m = std::floor(1.0 / (g->dt * (3.0 * R->fmax + 2.0 * std::sqrt(fhi * g->f0))));
      R->dtft_every = m > 1 ? (m > 1000 ? 1000 : (int)m) : 1;
    }
    R->beta = kPi * R->fmax * R->fmax;
    R->t0 = kPi / R->fmax;
    R->np = std::max(2 * r, 4);
    const int np = R->np;
    const size_t np3 = (size_t)np * np * np;
    R->it_min = 0;
    while (!((double)R->it_min * g->dt >= 2.0 * R->t0)) R->it_min++;        // [R9]
    R->nsteps.assign(nsrc, 0); R->done.assign(nsrc, 0); R->status.assign(nsrc, 0);

    // receivers (L167-178, L640)
    R->rst.resize((size_t)std::max(nrec, 1) * 18);
    for (int q = 0; q < nrec; ++q) for (int c = 0; c < 6; ++c) for (int a = 0; a < 3; ++a) {
      const double *S = kLat[c][a] ? g->xh[a].data() : g->xn[a].data();
      const double p = rec[3 * q + a];
      if (p < g->xn[a][g->lo[a]] || p > g->xn[a][g->lo[a] + g->nc[a]] ||
          !make_stencil(S, g->N[a], p, np, a == 2 ? g->klo : r, g->N[a] - 1 - r, false, &R->rst[((size_t)q * 6 + c) * 3 + a])) {
        free_run(g); return fail(EMM_EINVAL, "emm_run_begin: receiver %d outside the interior", q);
      }
      const Stencil1 &st = R->rst[((size_t)q * 6 + c) * 3 + a];
      if (st.start < g->blo[a] || st.start + np - 1 > g->bhi[a]) { free_run(g); return fail(EMM_EINVAL, "emm_run_begin: receiver %d stencil leaves the DFT box", q); }
    }
    // check set [R9]
    std::vector<int> chk;
    if (nf > 0)
      for (int k = g->blo[2]; k <= g->bhi[2]; ++k) for (int j = g->blo[1]; j <= g->bhi[1]; ++j) {
        const bool ej = j == g->blo[1] || j == g->bhi[1], ek = k == g->blo[2] || k == g->bhi[2];
        const size_t rowbase = ((size_t)k * g->N[1] + j) * g->P1;
        // whole row when the row lies on a face (or for the full set); otherwise only its two end nodes can qualify
        const bool whole = R->check_set == EMM_CHECK_FULL || (R->check_set == EMM_CHECK_FACES && (ej || ek));
        if (whole) {
          for (int i = g->blo[0]; i <= g->bhi[0]; ++i) chk.push_back((int)(rowbase + i));
        } else if (R->check_set == EMM_CHECK_FACES || (ej && ek)) {      // corners: only rows with ej && ek
          chk.push_back((int)(rowbase + g->blo[0]));
          if (g->bhi[0] != g->blo[0]) chk.push_back((int)(rowbase + g->bhi[0]));
        }
      }
    // workspace layout
    if (g->top == EMM_TOP_AIR && g->sep_air && (rc = sep_air_make_plans(g, nsrc))) { free_run(g); return rc; }
    Arena A;
    A.base = static_cast<char *>(g->d_ws); A.cap = g->ws_bytes; A.dry = false; A.off = g->fixed_bytes;
    layout_run(g, A, nsrc, R->sparse ? 0 : nf, R->sparse ? nf : 0, R->table_steps, nrec, chk.size(), R->group > 2 ? R->group - 2 : 0, R->ds, R->dr);
    while (A.overflow && R->group > 2) {     // a workspace without room for all the history copies: the largest group that fits
      R->group--;
      A.off = g->fixed_bytes;
      A.overflow = false;
      layout_run(g, A, nsrc, R->sparse ? 0 : nf, R->sparse ? nf : 0, R->table_steps, nrec, chk.size(), R->group - 2, R->ds, R->dr);
    }
    if (g->top == EMM_TOP_AIR && g->sep_air && !A.overflow)
      for (int q = 0; q < 8; ++q)
        if (g->sp[q] && (cufftSetStream(g->sp[q], g->stream_b) != CUFFT_SUCCESS || cufftSetWorkArea(g->sp[q], R->dr.sp_ws[q]) != CUFFT_SUCCESS)) {
          free_run(g);
          return fail(EMM_ECUDA, "cufftSetStream/cufftSetWorkArea failed");
        }
    R->ds.dft_every = R->dtft_every;
    if (!A.overflow && (rc = tile_make_maps(g, R->ds))) { free_run(g); return rc; }
    if (A.overflow) { size_t need = A.off; free_run(g); return fail(EMM_ENOMEM, "emm_run_begin: workspace too small (%zu bytes needed)", need); }
    // zero the whole run region (fields, psi, accumulators, flags)
    CU(cudaMemsetAsync(static_cast<char *>(g->d_ws) + g->fixed_bytes, 0, A.off - g->fixed_bytes, g->stream));

    // wavelet and twiddles (fp64 -> fp32), [R6]/[R8]
    const int T = R->table_steps;
    std::vector<float> wav(T);
    const int nfg = R->sparse ? 0 : nf, nfr = R->sparse ? nf : 0;      // frequencies on the grid / at the receivers only
    std::vector<float2> twE((size_t)T * nfg), twH((size_t)T * nfg);
    std::vector<double2> twE64(T), twH64(T), twEf((size_t)T * nfr), twHf((size_t)T * nfr);
    R->wav.resize(T);
    R->wavh.resize(T);
    std::vector<float> wavh(T);
    for (int it = 0; it < T; ++it) {
      const double t = (double)it * g->dt, u = t - R->t0;
      wav[it] = (float)(-2.0 * R->beta * u * std::sqrt(R->beta / kPi) * std::exp(-R->beta * u * u));
      R->wav[it] = (double)wav[it];
      const double uh = t + 0.5 * g->dt - R->t0;
      wavh[it] = (float)(-2.0 * R->beta * uh * std::sqrt(R->beta / kPi) * std::exp(-R->beta * uh * uh));
      R->wavh[it] = (double)wavh[it];
      for (int f = 0; f < nf; ++f) {
        const std::complex<double> I(0, 1);
        const std::complex<double> h = std::exp(I * R->wp[f] * t), e = std::exp(I * R->wp[f] * (((double)it + 0.5) * g->dt));
        if (R->sparse) {
          twHf[(size_t)it * nf + f] = make_double2(h.real(), h.imag());
          twEf[(size_t)it * nf + f] = make_double2(e.real(), e.imag());
        } else {
          twH[(size_t)it * nf + f] = make_float2((float)h.real(), (float)h.imag());
          twE[(size_t)it * nf + f] = make_float2((float)e.real(), (float)e.imag());
        }
        if (f == R->fmin) { twH64[it] = make_double2(h.real(), h.imag()); twE64[it] = make_double2(e.real(), e.imag()); }
      }
    }
    if ((rc = upload(g, const_cast<float *>(R->ds.wavh), wavh))) { free_run(g); return rc; }
    if ((rc = upload(g, const_cast<float *>(R->ds.wav), wav)) || (rc = upload(g, const_cast<float2 *>(R->ds.twE), twE)) ||
        (rc = upload(g, const_cast<float2 *>(R->ds.twH), twH)) || (rc = upload(g, R->dr.twE64, twE64)) ||
        (rc = upload(g, R->dr.twH64, twH64)) || (rc = upload(g, R->dr.chk_idx, chk)) ||
        (rc = upload(g, R->dr.twEf, twEf)) || (rc = upload(g, R->dr.twHf, twHf))) { free_run(g); return rc; }

    // CPML tables
    DevGrid &d = g->dg;
    for (int a = 0; a < 3; ++a) {
      std::vector<float> am, bm, ap, bp;
      cpml_tables(g, a, R->fmax, am, bm, ap, bp);
      float *const *t = R->dr.cpml[a];
      if ((rc = upload(g, t[0], am)) || (rc = upload(g, t[1], bm)) || (rc = upload(g, t[2], ap)) || (rc = upload(g, t[3], bp))) { free_run(g); return rc; }
      d.am[a] = t[0]; d.bm[a] = t[1]; d.ap[a] = t[2]; d.bp[a] = t[3];
    }

    // sources: W_c = dir_c w_x w_y w_z / V on the component's lattice, premultiplied by dt/eps ([R7])
    std::vector<int> soff(nsrc * 3 + 1, 0), sidx, cwhich;
    std::vector<float> sw;
    std::vector<long long> cidx;
    std::vector<double> cwgt, sWd;
    for (int s = 0; s < nsrc; ++s) {
      const double *dir = src[s].dir, *pos = src[s].pos;
      if (src[s].type != 0 && src[s].type != 1) { free_run(g); return fail(EMM_EINVAL, "emm_run_begin: source %d has an unknown type", s); }
      const bool mag = src[s].type == 1;
      R->mag.push_back(mag ? 1 : 0);
      (mag ? R->any_mag : R->any_el) = true;
      const double dn = std::sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
      if (!(dn > 0) || !std::isfinite(dn)) { free_run(g); return fail(EMM_EINVAL, "emm_run_begin: source %d has zero direction", s); }
      for (int c = 0; c < 3; ++c) {
        soff[s * 3 + c] = (int)sidx.size();
        if (dir[c] == 0.0) continue;
        const int cl = c + (mag ? 3 : 0);                 // lattice of E_c or of H_c
        Stencil1 st[3];
        for (int a = 0; a < 3; ++a) {
          const double *S = kLat[cl][a] ? g->xh[a].data() : g->xn[a].data();
          if (pos[a] < g->xn[a][g->lo[a]] || pos[a] > g->xn[a][g->lo[a] + g->nc[a]] ||
              !make_stencil(S, g->N[a], pos[a], np, a == 2 ? g->klo : r, g->N[a] - 1 - r, false, &st[a])) {
            free_run(g); return fail(EMM_EINVAL, "emm_run_begin: source %d outside the interior", s);
          }
        }
        for (int c3 = 0; c3 < np; ++c3) for (int c2 = 0; c2 < np; ++c2) for (int c1 = 0; c1 < np; ++c1) {
          const int i = st[0].start + c1, j = st[1].start + c2, k = st[2].start + c3;
          const double V = node_width(g, 0, kLat[cl][0], i) * node_width(g, 1, kLat[cl][1], j) * node_width(g, 2, kLat[cl][2], k);
          const double W = dir[c] / dn * st[0].w[c1] * st[1].w[c2] * st[2].w[c3] / V;
          // dt/mu, or dt/eps from the effective conductivity at the node (cells fetched from the device below)
          long long cell[4] = {-1, -1, -1, -1};
          int which[4] = {0, 0, 0, 0};
          double cw[4] = {0, 0, 0, 0};
          if (!mag) sigma_bar_cells(g, c, i, j, k, cell, which, cw);
          for (int n4 = 0; n4 < 4; ++n4) { cidx.push_back(cell[n4]); cwhich.push_back(which[n4]); cwgt.push_back(mag ? -1.0 : cw[n4]); }
          sidx.push_back((int)(((size_t)k * g->N[1] + j) * g->P1 + i));
          sWd.push_back(W);
        }
      }
      soff[s * 3 + 3] = (int)sidx.size();
    }
    for (int s = 0; s < nsrc; ++s) for (int c = 0; c < 3; ++c) if (soff[s * 3 + c + 1] < soff[s * 3 + c]) soff[s * 3 + c + 1] = soff[s * 3 + c];
    (void)np3;
    if (!cidx.empty()) {
      std::vector<float> cval(cidx.size());
      if ((rc = upload(g, R->dr.cell_idx, cidx)) || (rc = upload(g, R->dr.cell_which, cwhich)) ||
          (rc = launch_gather_cells(g, g->T.sig_h, g->vti ? g->T.sig_v : g->T.sig_h, R->dr.cell_idx, R->dr.cell_which, (int)cidx.size(), R->dr.cell_val))) {
        free_run(g); return rc;
      }
      CU(cudaMemcpyAsync(cval.data(), R->dr.cell_val, cval.size() * sizeof(float), cudaMemcpyDeviceToHost, g->stream));
      CU(cudaStreamSynchronize(g->stream));
      for (size_t n = 0; n < sWd.size(); ++n) {
        double ce = g->dt / kMu0;                                               // magnetic: dt/mu
        if (cwgt[4 * n] >= 0.0) {
          double num = 0, den = 0;
          for (int n4 = 0; n4 < 4; ++n4) { num += (double)cval[4 * n + n4] * cwgt[4 * n + n4]; den += cwgt[4 * n + n4]; }
          ce = g->dt * 2 * g->w0 / (num / den);                                 // electric: dt/eps
        }
        sw.push_back((float)(ce * sWd[n]));
      }
    }
    // check-set sums once per DTFT group (k_check_acc_group) read earlier levels of the field ring, into which later
    // electric injections have already been added at the source nodes: only when no source node is in the check set
    R->chk_grouped = R->group > 2 && R->check_set != EMM_CHECK_FULL;
    for (size_t n = 0; n < sidx.size() && R->chk_grouped; ++n)
      if (std::binary_search(chk.begin(), chk.end(), sidx[n])) R->chk_grouped = false;
    if ((rc = upload(g, const_cast<int *>(R->ds.src_mag), R->mag))) { free_run(g); return rc; }
    if ((rc = upload(g, R->dr.src_off, soff)) || (rc = upload(g, R->dr.src_idx, sidx)) || (rc = upload(g, R->dr.src_w, sw))) { free_run(g); return rc; }

    // receiver gather list
    std::vector<int> ridx((size_t)6 * nrec * np3);
    std::vector<double> rwgt((size_t)6 * nrec * np3);
    R->nrec_nodes = (int)(nrec * np3);
    R->dr.nrec_nodes = R->nrec_nodes;
    for (int c = 0; c < 6; ++c) for (int q = 0; q < nrec; ++q) {
      const Stencil1 *st = &R->rst[((size_t)q * 6 + c) * 3];
      size_t n = 0;
      for (int c3 = 0; c3 < np; ++c3) for (int c2 = 0; c2 < np; ++c2) for (int c1 = 0; c1 < np; ++c1)
      {
        rwgt[((size_t)c * nrec + q) * np3 + n] = st[0].w[c1] * st[1].w[c2] * st[2].w[c3];
        ridx[((size_t)c * nrec + q) * np3 + n++] = (int)(((size_t)(st[2].start + c3) * g->N[1] + st[1].start + c2) * g->P1 + st[0].start + c1);
      }
    }
    if ((rc = upload(g, R->dr.rec_idx, ridx)) || (rc = upload(g, R->dr.rec_w, rwgt))) { free_run(g); return rc; }
    CU(cudaStreamSynchronize(g->stream));
  } catch (const std::bad_alloc &) {
    free_run(g);
    return fail(EMM_ENOMEM, "emm_run_begin: out of memory");
  }
  return 0;
}

extern "C" int emm_run_enqueue(emm_grid *g, int n) {
  if (!g || !g->run) return fail(EMM_EINVAL, "emm_run_enqueue: no run in progress");
  return enqueue_steps(g, n);
}

extern "C" int emm_run_steps(emm_grid *g, int n, int *nsteps, int *all_done) {
  if (!g || !g->run) return fail(EMM_EINVAL, "emm_run_steps: no run in progress");
  Run *R = g->run;
  int rc = 0, left = n;
  bool alldone = false, noconv = false;
  while (left > 0 && !alldone) {
    int chunk = std::min(left, R->check_every - R->it_host % R->check_every);      // stop at every check
    if (R->fixed_steps) chunk = std::min(chunk, R->fixed_steps - R->it_host);
    else chunk = std::min(chunk, R->max_steps - R->it_host);
    if (chunk > 0) {
      if ((rc = enqueue_steps(g, chunk))) return rc;
      left -= chunk;
    }
    if ((rc = fetch_flags(g))) return rc;
    alldone = true;
    for (int s = 0; s < R->nsrc; ++s) alldone = alldone && R->done[s];
    if (R->fixed_steps && R->it_host >= R->fixed_steps) { for (int s = 0; s < R->nsrc; ++s) R->done[s] = 1; alldone = true; }
    if (!R->fixed_steps && R->it_host >= R->max_steps && !alldone) { noconv = true; for (int s = 0; s < R->nsrc; ++s) R->done[s] = 1; alldone = true; }
    if (chunk <= 0) break;
  }
  if (left <= 0 && !alldone) { if ((rc = fetch_flags(g))) return rc; }
  for (int s = 0; s < R->nsrc; ++s) if (nsteps) nsteps[s] = R->nsteps[s];
  if (all_done) *all_done = alldone ? 1 : 0;
  for (int s = 0; s < R->nsrc; ++s) if (R->status[s] == EMM_ENAN) return fail(EMM_ENAN, "emm_run_steps: non-finite field (source %d)", s);
  if (noconv) return fail(EMM_ENOCONV, "emm_run_steps: max_steps reached before convergence");
  return 0;
}

// compute_green_function + extract_emf (Alg. 1): receiver interpolation in fp64 on the device (k_rec_interp),
// Eq. 7 in fp64 on the host
extern "C" int emm_run_end(emm_grid *g, double *out_, int *nsteps) {
  if (!g || !g->run) return fail(EMM_EINVAL, "emm_run_end: no run in progress");
  Run *R = g->run;
  int rc;
  if ((rc = fetch_flags(g))) return rc;
  for (int s = 0; s < R->nsrc; ++s) if (nsteps) nsteps[s] = R->nsteps[s];
  if (!out_ || R->nrec == 0) return 0;
  const int nf = R->nf, np = R->np;
  const size_t np3 = (size_t)np * np * np;
  // accumulators interpolated to the receivers on the device (from the full-grid F, or from the receivers-only sums)
  if ((rc = launch_rec_interp(g, R->ds, R->dr, nf, R->nrec, (int)np3))) return rc;
  std::vector<double2> val((size_t)R->nsrc * nf * R->nrec * 6);
  CU(cudaMemcpyAsync(val.data(), R->dr.rec_out, val.size() * sizeof(double2), cudaMemcpyDeviceToHost, g->stream));
  CU(cudaStreamSynchronize(g->stream));
  std::complex<double> *out = reinterpret_cast<std::complex<double> *>(out_);
  const std::complex<double> I(0, 1);
  for (int s = 0; s < R->nsrc; ++s)
    for (int f = 0; f < nf; ++f) {
      const std::complex<double> Jw = source_spectrum(g, R, s, f);
      const std::complex<double> sc = std::sqrt(-I * 2.0 * kPi * R->freqs[f] / (2 * g->w0));   // Eq. 7a, principal root
      for (int q = 0; q < R->nrec; ++q)
        for (int c = 0; c < 6; ++c) {
          const double2 v = val[(((size_t)s * nf + f) * R->nrec + q) * 6 + c];
          std::complex<double> G = std::complex<double>(v.x, v.y) / Jw;         // Eq. 7b
          if (!R->mag[s] && c < 3) G *= sc;                                    // electric source: G^EE = sc F_E/J'
          if (R->mag[s] && c >= 3) G /= sc;                                    // magnetic source: G^HM = F_H/(sc M')
          out[(((size_t)s * nf + f) * R->nrec + q) * 6 + c] = G;
        }
    }
  return 0;
}

extern "C" int emm_run(emm_grid *g, const emm_src *src, int nsrc, const double *freqs, int nf, const double *rec, int nrec,
                       const emm_run_opts *o, double *out, int *nsteps) {
  if (!g || !src || nsrc < 1 || !o) return fail(EMM_EINVAL, "emm_run: bad arguments");
  const int group = o->batched ? nsrc : 1;
  int worst = 0;
  for (int s0 = 0; s0 < nsrc; s0 += group) {
    int rc = emm_run_begin(g, src + s0, group, freqs, nf, rec, nrec, o);
    if (rc) return rc;
    int done = 0;
    std::vector<int> ns(group, 0);
    while (!done) {
      rc = emm_run_steps(g, g->run->check_every, ns.data(), &done);
      if (rc == EMM_ENOCONV) { worst = rc; break; }
      if (rc) return rc;
    }
    rc = emm_run_end(g, out ? out + (size_t)s0 * nf * nrec * 12 : nullptr, ns.data());
    if (rc) return rc;
    if (nsteps) for (int s = 0; s < group; ++s) nsteps[s0 + s] = ns[s];
  }
  if (worst) return fail(worst, "emm_run: max_steps reached before convergence");
  return 0;
}

extern "C" int emm_get(emm_grid *g, int isrc, int what, int ifreq, void *host_out) {
  if (!g || !host_out) return fail(EMM_EINVAL, "emm_get: null argument");
  if (!g->bound) return fail(EMM_ECUDA, "emm_get: no device workspace bound");
  const int N1 = g->N[0], N2 = g->N[1], N3 = g->N[2], P1 = g->P1;
  if (what >= EMM_GET_CE1 && what <= EMM_GET_CE3) {
    if (!g->have_model) return fail(EMM_EINVAL, "emm_get: no model");
    CU(cudaMemcpy2DAsync(host_out, (size_t)N1 * 4, g->T.ce[what - EMM_GET_CE1], (size_t)P1 * 4, (size_t)N1 * 4, (size_t)N2 * N3,
                         cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    return 0;
  }
  Run *R = g->run;
  if (!R || isrc < 0 || isrc >= R->nsrc) return fail(EMM_EINVAL, "emm_get: no run state for that source");
  if (what >= EMM_GET_E1 && what <= EMM_GET_H3) {
    const float *p = (what < EMM_GET_H1 ? R->ds.E[what] : R->ds.H[what - EMM_GET_H1]) + (size_t)isrc * g->dg.VS;
    CU(cudaMemcpy2DAsync(host_out, (size_t)N1 * 4, p, (size_t)P1 * 4, (size_t)N1 * 4, (size_t)N2 * N3, cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    return 0;
  }
  if (what >= EMM_GET_F_E1 && what <= EMM_GET_F_H3) {
    if (ifreq < 0 || ifreq >= R->nf) return fail(EMM_EINVAL, "emm_get: bad ifreq");
    if (R->sparse) return fail(EMM_EINVAL, "emm_get: no full-grid accumulators in a receivers-only run (sparse_dft)");
    const int c = what - EMM_GET_F_E1;
    float2 *o = static_cast<float2 *>(host_out);
    std::memset(o, 0, sizeof(float2) * (size_t)N1 * N2 * N3);
    const float2 *F = R->ds.F + (((size_t)isrc * R->nf + ifreq) * 6 + c) * g->dg.NZB * g->dg.PS;
    CU(cudaMemcpy2DAsync(o + (size_t)g->blo[2] * N2 * N1, (size_t)N1 * 8, F, (size_t)P1 * 8, (size_t)N1 * 8, (size_t)N2 * g->dg.NZB,
                         cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    for (int k = g->blo[2]; k <= g->bhi[2]; ++k) for (int j = 0; j < N2; ++j) {
      float2 *row = o + ((size_t)k * N2 + j) * N1;
      const bool jin = j >= g->blo[1] && j <= g->bhi[1];
      for (int i = 0; i < N1; ++i) if (!jin || i < g->blo[0] || i > g->bhi[0]) row[i] = make_float2(0.f, 0.f);
    }
    return 0;
  }
  if (what == EMM_GET_JW) {
    int rc = fetch_flags(g);
    if (rc) return rc;
    std::complex<double> *o = static_cast<std::complex<double> *>(host_out);
    const std::complex<double> I(0, 1);
    for (int f = 0; f < R->nf; ++f) o[f] = source_spectrum(g, R, isrc, f);
    return 0;
  }
  if (what == EMM_GET_DTFT_GROUP) {
    *static_cast<int *>(host_out) = R->group;
    return 0;
  }
  if (what == EMM_GET_CHECK_N) {
    *static_cast<int *>(host_out) = R->dr.nchk;
    return 0;
  }
  if (what == EMM_GET_CHECK_ACC) {
    if (R->dr.nchk <= 0) return fail(EMM_EINVAL, "emm_get: this run has no check set");
    CU(cudaMemcpyAsync(host_out, R->dr.C + (size_t)isrc * 6 * R->dr.nchk, sizeof(double2) * 6 * R->dr.nchk, cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    return 0;
  }
  if (what == EMM_GET_DELTA) {
    CU(cudaMemcpyAsync(host_out, R->dr.delta + 2 * isrc, 2 * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    return 0;
  }
  return fail(EMM_EINVAL, "emm_get: unknown item %d", what);
}

// Sensitivity kernel of an electric-field datum with respect to the cell conductivities (DESIGN.md [R14]):
// Eq. 7 scaling of the two sources' accumulators on the host (fp64), the gather over edges and padded cells on the device
// (emm_sens.cu), a few cell layers at a time through the run's scratch.
extern "C" int emm_sensitivity(emm_grid *g, int isrc, int iadj, int ifreq, double *out_h, double *out_v) {
  if (!g || !g->run || !out_h || !out_v) return fail(EMM_EINVAL, "emm_sensitivity: no run in progress or null output");
  Run *R = g->run;
  if (isrc < 0 || isrc >= R->nsrc || iadj < 0 || iadj >= R->nsrc || ifreq < 0 || ifreq >= R->nf)
    return fail(EMM_EINVAL, "emm_sensitivity: bad source or frequency index");
  if (R->sparse || R->ds.nf < 1) return fail(EMM_EINVAL, "emm_sensitivity: needs full-grid accumulators (sparse_dft = 0)");
  if (R->mag[isrc] || R->mag[iadj]) return fail(EMM_EINVAL, "emm_sensitivity: electric sources only");
  if (R->dtft_every != 1) return fail(EMM_EINVAL, "emm_sensitivity: needs every term of the DTFT (dtft_every = 1)");
  if (R->dr.sens_layers < 1) return fail(EMM_EINVAL, "emm_sensitivity: the run holds a single source (transmitter and receiver dipole must be resident together)");
  int rc;
  if ((rc = fetch_flags(g))) return rc;
  const std::complex<double> I(0, 1);
  const std::complex<double> sc = std::sqrt(-I * 2.0 * kPi * R->freqs[ifreq] / (2 * g->w0));   // Eq. 7a, principal root
  const std::complex<double> scale = (sc / source_spectrum(g, R, isrc, ifreq)) * (sc / source_spectrum(g, R, iadj, ifreq)) * 0.25;
  const size_t layer = (size_t)g->nc[0] * g->nc[1];
  double2 *dh = R->dr.sens, *dv = R->dr.sens + (size_t)R->dr.sens_layers * layer;
  for (int k = 0; k < g->nc[2]; k += R->dr.sens_layers) {
    const int n = std::min(R->dr.sens_layers, g->nc[2] - k);
    if ((rc = launch_sensitivity(g, R->ds, isrc, iadj, ifreq, scale.real(), scale.imag(), k, n, dh, dv))) return rc;
    CU(cudaMemcpyAsync(out_h + 2 * (size_t)k * layer, dh, sizeof(double2) * n * layer, cudaMemcpyDeviceToHost, g->stream));
    CU(cudaMemcpyAsync(out_v + 2 * (size_t)k * layer, dv, sizeof(double2) * n * layer, cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
  }
  return 0;
}

// ---- optional per-kernel timing (bench evidence for the roofline of the dominant kernel) ----
extern "C" int emm_profile(emm_grid *g, int enable) {
  if (!g) return fail(EMM_EINVAL, "emm_profile: null grid");
  for (cudaEvent_t e : g->prof_ev) cudaEventDestroy(e);
  g->prof_ev.clear();
  g->prof_kind.clear();
  g->prof = enable != 0;
  return 0;
}

extern "C" int emm_profile_read(emm_grid *g, double *ms, int *counts) {
  if (!g || !ms || !counts) return fail(EMM_EINVAL, "emm_profile_read: null argument");
  CU(cudaStreamSynchronize(g->stream));
  for (int q = 0; q < 6; ++q) { ms[q] = 0.0; counts[q] = 0; }
  for (size_t q = 0; q < g->prof_kind.size(); ++q) {
    float t = 0.f;
    CU(cudaEventElapsedTime(&t, g->prof_ev[2 * q], g->prof_ev[2 * q + 1]));
    ms[g->prof_kind[q]] += t;
    counts[g->prof_kind[q]]++;
  }
  for (cudaEvent_t e : g->prof_ev) cudaEventDestroy(e);
  g->prof_ev.clear();
  g->prof_kind.clear();
  return 0;
}
