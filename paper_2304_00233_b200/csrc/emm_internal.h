// emm_internal.h -- internal types of libemm_b200.so (not part of the ABI; see include/emm.h).
//
// Host side keeps everything in double (grid, FD tables, CPML, wavelet, twiddles, Eq. 7); the device
// holds fp32 fields/accumulators.  Citations are PAPER.md line numbers; [Rn] = DESIGN.md readings.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cufft.h>

#include <complex>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/emm.h"

namespace emm {

constexpr double kMu0 = 4e-7 * 3.14159265358979323846;
constexpr double kPi = 3.14159265358979323846;
constexpr int kMaxR = 3;
constexpr int kMaxNF = 16;

int fail(int code, const char *fmt, ...);

// Yee lattice of component c (Ex,Ey,Ez,Hx,Hy,Hz) along axis a: 1 = half nodes, 0 = nodes [R2]
constexpr int kLat[6][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};

struct Stencil1 { int start; double w[8]; };

// ---- bump allocator over the caller's device workspace (dry-run mode computes sizes only) ----
struct Arena {
  char *base = nullptr;
  size_t cap = 0, off = 0;
  bool dry = true;
  bool overflow = false;
  template <class T> T *take(size_t n) {
    size_t bytes = (n * sizeof(T) + 255) & ~size_t(255);
    size_t at = off;
    off += bytes;
    if (dry) return nullptr;
    if (off > cap) { overflow = true; return nullptr; }
    return reinterpret_cast<T *>(base + at);
  }
};

// ---- device-side view handed to the kernels by value ----
struct DevGrid {
  int N1, N2, N3, P1;          // padded dims and x pitch (floats)
  long long PS, VS;            // plane stride P1*N2, volume stride PS*N3
  int r, nb;
  int klo;                     // first updated z index (= r)
  int zslab_lo;                // 1: CPML slab at low z exists (top=CPML)
  int blo[3], bhi[3];          // DTFT box, inclusive
  int NZB;                     // bhi[2]-blo[2]+1
  int XS;                      // x-slab row length (2*nb rounded up to 4)
  const float *cm[3], *cp[3];  // FD tables [N][2r]
  const float *am[3], *bm[3], *ap[3], *bp[3];  // CPML tables [2*nb]
  const float *ce[3];          // dt/eps [N3][N2][P1]
  float dtmu;                  // dt/mu0
};

struct DevState {              // per run; arrays carry a leading source dimension
  float *E[3], *H[3];          // [nsrc][N3][N2][P1]
  float *psx[2][2];            // [E/H kernel][2]: x-slab psi [nsrc][N3][N2][XS]
  float *psy[2][2];            // y-slab psi [nsrc][N3][2nb][P1]
  float *psz[2][2];            // z-slab psi [nsrc][2nb][N2][P1]
  float2 *F;                   // [nsrc][nf][6][NZB][N2][P1]
  // Grouped DTFT: inside a group of m > 2 steps the fields are updated out of place through a ring
  // of nbuf buffers per component ([nbuf][nsrc][N3][N2][P1], E[c]/H[c] of the run = buffer 0), so that earlier time levels
  // stay readable for the pass that closes the group.  Per launch: E/H = the buffers holding the current fields, Eo/Ho =
  // where the update kernel writes (nullptr: in place), hist = first history level of the closing pass, hstride = floats
  // between consecutive levels.
  float *Eo[3], *Ho[3];
  const float *hist[2][3];
  long long hstride;
  int nbuf;
  const float2 *twE, *twH;     // [max_steps][nf]
  const float *wav;            // [max_steps] s(it dt): electric sources
  const float *wavh;           // [max_steps] s((it+1/2) dt): magnetic sources
  const int *src_mag;          // [nsrc] 1 = magnetic dipole
  int *it;                     // device step counter
  int *done;                   // [nsrc]
  int nf, nsrc;
  int dft_every;               // DTFT decimation: accumulate only when it % dft_every == 0 (1 = every step)
};

struct DevTables {             // device pointers of the per-grid region
  float *ce[3], *cm[3], *cp[3];
  float *sig_h, *sig_v;        // raw per-cell model [nz][ny][nx] as given to emm_model_set (resident: effective medium at the source nodes)
  double *xn[3];
  int *ta_start[2][2], *fa_start[2][2];   // [axis][lattice]: lattice -> aux plane, aux plane -> lattice
  float *ta_w[2][2], *fa_w[2][2];
  float *kx, *ky;                          // signed wavenumbers of the FFT plane
  float2 *tw1, *tw2;                       // e^{-2 pi i k/M1}, e^{-2 pi i k/M2}: twiddles of the cluster route (emm_air_cluster.cu)
  void *fft_ws[3];
};

// TMA descriptors of one accumulator-free update kernel (emm_tile.cu): the three stencil fields with the halo each one
// needs, the three updated fields, dt/eps (E kernel only).  Passed to the kernel by value (__grid_constant__).
struct TileMaps { CUtensorMap A1, A2, A3, U1, U2, U3, C1, C2, C3; };

struct Run;

}  // namespace emm

struct emm_grid {
  // options
  int r = 1, nb = 0, ne = 0, top = 0, air_route = 0;
  double f0 = 1, w0 = 0, cfl = 0.99, aux_dx = 0;
  int nc[3] = {0, 0, 0}, N[3] = {0, 0, 0}, lo[3] = {0, 0, 0};
  std::vector<double> xn[3], xh[3];      // padded nodes [N+1], half nodes [N]
  std::vector<double> cm[3], cp[3];      // [N][2r]
  double Dmax[3] = {0, 0, 0};
  int k0 = -1, klo = 1, uniform_xy = 0;
  int blo[3] = {0, 0, 0}, bhi[3] = {0, 0, 0};
  int P1 = 0, XS = 0;
  // air boundary
  int M1 = 0, M2 = 0;
  int air_cluster = 0;                   // uniform x-y: cluster size of the one-launch boundary (emm_air_cluster.cu), 0 = library route
  int air_cluster_lg = 0;                // ... and the ghost levels it holds in shared memory at a time
  bool sep_air = false;                  // non-uniform x-y: separable route (emm_air_sep.cu) instead of plane-sized 2-D transforms
  double dxa = 0, dya = 0;
  std::vector<emm::Stencil1> toaux[2][2], fromaux[2][2];
  // model
  bool have_model = false;
  bool vti = false;
  double dt = 0, smin = 0;
  // device
  void *d_ws = nullptr;
  size_t ws_bytes = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t stream_b = nullptr;       // helper stream of the air-water boundary (created by emm_bind_device)
  cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // fork/join events between the two streams
  bool bound = false;
  size_t fixed_bytes = 0;                // arena offset after the per-grid (model) region
  emm::DevGrid dg{};
  emm::DevTables T{};                    // per-grid device tables (fixed region of the workspace)
  cufftHandle plan_fwd = 0, plan_inv_e = 0, plan_inv_h = 0;
  bool have_plans = false;
  size_t fft_ws[3] = {0, 0, 0};             // cuFFT work-area bytes: forward, inverse (E), inverse (H)
  cufftHandle sp[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // separable route: batched 1-D plans (emm_air_sep.cu)
  size_t sp_ws[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  int sp_nsrc = 0;                       // number of sources the plans in sp[] are batched for
  double vref[3][2] = {{0, 0}, {0, 0}, {0, 0}};   // CPML reference speed per face [R5]
  emm::Run *run = nullptr;
  // tile pipeline of the accumulator-free update (emm_tile.cu): descriptors of the current run's field rings
  bool tile_ok = false;
  emm::TileMaps tile_maps[2];            // [0] E kernel, [1] H kernel
  const float *tile_base[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};   // buffer 0 of the E / H rings
  long long tile_hstride = 1;
  long long launches = 0;
  // optional per-kernel timing of the two fused update kernels (CUDA events on the bound stream)
  bool prof = false;
  std::vector<cudaEvent_t> prof_ev;      // pairs: start, stop
  std::vector<int> prof_kind;            // 0 = E kernel, 1 = H kernel
};
