/* emm.h -- C ABI of libemm_b200.so: B200-native fictitious-wave-domain 3-D CSEM FDTD.
 *
 * The calls follow the paper's statement of the problem (arxiv 2304.00233; citations are
 * /root/reference/PAPER.md line numbers): a rectilinear non-uniform grid (L402-443, L644-660), a
 * conductivity model (L662-668, Eq. 26), and a survey of sources, frequencies and receivers
 * (L622-642, L670-680) for which the library returns the complex frequency-domain Green's
 * functions at the receivers (Eq. 7; output columns of L688-711).
 *
 * Conventions.  SI units; z positive downward (L646-649); arrays are x-fastest, a[k][j][i]
 * (L514).  Every pointer argument is a HOST pointer unless its name starts with `d_`.  Arrays
 * passed in are copied before the call returns; output buffers are caller-allocated.  Handles are
 * opaque and released only by emm_grid_destroy.  All time stepping runs in CUDA kernels on the
 * device memory and stream bound with emm_bind_device (PyTorch owns both); there is no CPU
 * fallback: without a bound workspace the run calls return EMM_ECUDA.
 *
 * Every function returns 0 on success or a negative EMM_E* code; it never throws, exits or
 * prints.  emm_last_error() returns a thread-local message for the last failure.
 */
#ifndef EMM_H
#define EMM_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

#define EMM_EINVAL  (-1) /* bad dims, non-monotone coordinates, sigma<=0, rd not in {1,2,3}, source or
                            receiver outside the interior, bad option                                */
#define EMM_ENOMEM  (-2) /* host allocation failed or bound workspace too small                      */
#define EMM_ECUDA   (-3) /* CUDA/cuFFT error, or no device workspace bound                            */
#define EMM_ENOCONV (-4) /* max_steps reached before convergence (outputs are still written)         */
#define EMM_ENAN    (-5) /* non-finite field detected by the convergence check                        */

#define EMM_TOP_CPML 0   /* CPML on the top face too (whole-space problems)                           */
#define EMM_TOP_AIR  1   /* air-water boundary at the first z node (Eq. 17-21)              */

#define EMM_CHECK_CORNERS 0 /* 8 corners of the non-CPML box (L528, Fig. 2)                           */
#define EMM_CHECK_FACES   1 /* its six faces ("the boundaries of the computing volume", L387)         */
#define EMM_CHECK_FULL    2 /* whole box (Yang 2021, L528)                                            */

typedef struct emm_grid emm_grid;

typedef struct {
  int rd;        /* half length of the FD operator, 1..3 => order 2*rd (L200, L684)                    */
  int nb;        /* CPML cells per face (L305, L686)                                                   */
  int ne;        /* buffer cells between CPML and interior (L686); <0 => rd+5                          */
  int top;       /* EMM_TOP_*                                                                          */
  double f0;     /* omega0 = 2*pi*f0 of the fictitious transform sigma = 2*omega0*eps (L47); <=0 => 1  */
  double cfl;    /* dt = cfl/eta (Eq. 15-16); <=0 => 0.99                                        */
  double aux_dx; /* spacing of the auxiliary uniform plane used by the air boundary when x-y is
                    non-uniform (L288); <=0 => smallest horizontal spacing                             */
  int air_route; /* air boundary on a non-uniform x-y grid: 0 = separable route (interpolation and transform one
                    axis at a time, batched 1-D transforms; default), 1 = plane-sized route (interpolate to the whole
                    auxiliary plane, 2-D transforms): the same linear map up to rounding order, about twice the
                    work; kept as the cross-check of the separable route.  On a uniform x-y grid: 0 = the whole boundary in
                    one launch per pass by a thread-block cluster that holds the plane in shared memory (hand-written
                    transforms; planes up to about 280 x 280, larger ones take the library route), 1 = library route
                    (pack, 2-D cuFFT, filter, 2-D cuFFT, unpack): the same linear map up to rounding order.          */
} emm_grid_opts;

typedef struct {
  double pos[3]; /* x,y,z of the point dipole (anywhere inside the model, L640)                        */
  double dir[3]; /* polarisation of the dipole (normalised internally)                                 */
  int type;      /* 0: electric dipole J (Eq. 8, inject_electric_src_fwd L457); 1: magnetic dipole M
                    (Eq. 8, inject_magnetic_src_fwd).  Outputs for type 1 are G^EM = E/M and G^HM = H/M
                    (same transformation as Eq. 7: E' = E, M' = M, H' = sqrt(-i w/2 w0) H, Eq. 4)            */
} emm_src;

typedef struct {
  int max_steps;   /* cap on time steps; <=0 => 100000                                                 */
  int fixed_steps; /* >0: run exactly this many steps and skip the convergence stop                    */
  double tol;      /* relative change of the lowest-frequency accumulators over check_every steps
                      below which the run stops (L385-387); <=0 => 1e-6                                 */
  int check_every; /* <=0 => 100 (L458)                                                                */
  int check_set;   /* EMM_CHECK_*                                                                      */
  double fmax;     /* source wavelet parameter; <=0 => 4*sqrt(max f * f0)                              */
  int batched;     /* 1: advance all sources in one launch per kernel (they share grid and
                      coefficients); 0: one source after the other                                     */
  int dtft_every;  /* m > 1: DTFT decimation -- only every m-th term of the sums of Eq. 25 is taken for the fields
                      and J' (the small check set keeps every term: the stopping rule does not depend on m).  The fictitious wave field is band-limited far below 1/(2 m dt)
                      (dt is set by the fastest cell, L251-260), so G = F/J' changes by ~1e-9 while the dominant
                      accumulator traffic drops by (1 - 1/m).  0, 1: every step, as the paper does (L454);
                      < 0: the largest safe m = floor(1/(dt (3 fmax + 2 sqrt(max f * f0))))                      */
  int sparse_dft;  /* 1: receivers-only DTFT -- the sums of Eq. 25 are kept only at the nodes of the receivers'
                      interpolation stencils (fp64 accumulators fed by the fp32 fields) and on the check set; no
                      full-grid accumulator exists (emm_get of EMM_GET_F_* fails with EMM_EINVAL), the update kernels
                      run without the 96*nf B/node term.  Same sums at those nodes, so emm_run returns the same
                      Green's functions and step counts; for runs that only want receiver data.
                      0: accumulators for every frequency on the whole DTFT box, as the paper does (L454)            */
  int dtft_pair;   /* Grouped DTFT: every term of Eq. 25 is taken, m consecutive terms per read-modify-write of the
                      accumulators.  An update kernel holds the field before and after its own update, i.e. the DTFT
                      operands of two consecutive steps (L372: old H of steps it and it+1; new E of steps it-1 and it);
                      the m-2 earlier levels of a group stay readable because inside a group the fields are updated out
                      of place through a ring of m buffers; the pass that closes the group reads them (12 B/node each).  Each accumulator gets the same
                      fused multiply-adds in the same order as with one term per step, at 1/m of the 96*nf B/node
                      traffic.  Groups never cross a convergence check or the end of an emm_run_steps/emm_run_enqueue
                      batch (shorter groups and single steps fill the rest), so accumulators are complete whenever they
                      can be read.  Applies to 1..5 frequencies with full-grid accumulators and dtft_every <= 1; otherwise
                      ignored.  0: default m (8 with 4-5 frequencies, 6 with 1-3); 2..8: that m (2 = pairs, no copies);
                      -1: one term per step in every step, as the paper's kernels do (L454, L880-884).  The workspace
                      holds (m-1)*6 more field-sized arrays per source for the ring; a workspace without room for them
                      gets the largest m that fits.                                                                  */
} emm_run_opts;

/* integer grid facts for emm_grid_info(): */
enum { EMM_I_N1 = 0, EMM_I_N2, EMM_I_N3,          /* padded array dims n?pad (L305-312)                  */
       EMM_I_LO1, EMM_I_LO2, EMM_I_LO3,           /* padding cells on the low side of each axis          */
       EMM_I_K0,                                  /* z index of the air-water plane, -1 without          */
       EMM_I_UNIFORM_XY,
       EMM_I_BOX_LO1, EMM_I_BOX_LO2, EMM_I_BOX_LO3, /* DTFT box = padded grid minus CPML (L365-370)     */
       EMM_I_BOX_HI1, EMM_I_BOX_HI2, EMM_I_BOX_HI3, /* inclusive                                         */
       EMM_I_AUX_M1, EMM_I_AUX_M2,                /* FFT plane of the air boundary                       */
       EMM_I_PITCH,                               /* floats per x row in device memory                   */
       EMM_I_AIR_CLUSTER,                         /* CTAs of the cluster that runs the air boundary in one launch
                                                     (uniform x-y, after emm_bind_device); 0 = library / separable route */
       EMM_I_COUNT };

/* items for emm_get(): state of the run in progress / last finished run */
enum { EMM_GET_E1 = 0, EMM_GET_E2, EMM_GET_E3, EMM_GET_H1, EMM_GET_H2, EMM_GET_H3,
                                   /* float [N3][N2][N1]: time-domain fields after the last step        */
       EMM_GET_F_E1 = 10, EMM_GET_F_E2, EMM_GET_F_E3, EMM_GET_F_H1, EMM_GET_F_H2, EMM_GET_F_H3,
                                   /* float complex [N3][N2][N1] (re,im pairs): DTFT accumulator of
                                      frequency `ifreq` (Eq. 25), zero outside the DTFT box              */
       EMM_GET_CE1 = 20, EMM_GET_CE2, EMM_GET_CE3, /* float [N3][N2][N1]: dt/eps of each E component   */
       EMM_GET_JW = 30,            /* double complex [nfreq]: J'(omega') accumulated so far (Eq. 7)     */
       EMM_GET_DELTA = 31,         /* double [2]: relative change of E and H accumulators at the last
                                      convergence check                                                  */
       EMM_GET_DTFT_GROUP = 32,    /* int: terms of Eq. 25 per accumulator pass in this run (1, or the m of dtft_pair) */
       EMM_GET_CHECK_N = 33,       /* int: number of points of the check set of this run [R9]                  */
       EMM_GET_CHECK_ACC = 34      /* double complex [6][EMM_GET_CHECK_N]: the fp64 check-set accumulators of the lowest
                                      frequency (Ex,Ey,Ez,Hx,Hy,Hz), complete up to the last step taken          */
};

/* ---- host-side pieces of the method (also the diagnostic surface) ------------------------------- */

/* Optimal geometric grid, Eq. 27-29 / L402-443: n intervals over length len, first interval dx.
 * x_out: n+1 node coordinates starting at 0; q_out (may be NULL): the stretching ratio.             */
int emm_nugrid(int n, double len, double dx, double *x_out, double *q_out);

/* Interpolation (row 0) and first-derivative (row 1) weights of `npts` arbitrary nodes for the
 * point x0, by Vandermonde inversion (Eq. 9-12).  Either output may be NULL.                */
int emm_fd_weights(int npts, const double *nodes, double x0, double *w_interp, double *w_deriv);

/* Acquisition geometry of the paper's source / receiver files (L632-640: x, y, z, azimuth, dip in rad).  The paper
 * gives the columns but no formula; reading [R13]: azimuth from +x towards +y, dip from the horizontal
 * towards +z (z is positive downward, L646), so dir = (cos dip cos az, cos dip sin az, sin dip), a unit vector.
 * emm_dipole_direction: the `dir` of an emm_src with that orientation.  emm_receiver_channels: what a receiver
 * dipole with that orientation records, chan[q] = (sum_c dir_c G_E[q][c], sum_c dir_c G_H[q][c]) for n receivers;
 * g6: complex double [n][6] as returned by emm_run for one source and frequency, chan: complex double [n][2].
 * Host, fp64.                                                                                            */
int emm_dipole_direction(double azimuth, double dip, double *dir /* [3] */);
int emm_receiver_channels(const double *g6, int n, const double *azimuth /* [n] */, const double *dip /* [n] */, double *chan);

/* ---- problem set-up --------------------------------------------------------------------------------- */

/* Node coordinates of the model (n?1 = cells+1 values each, strictly increasing).  Builds the padded
 * grid (L305-312), the per-node D+/D- coefficient tables (Eq. 13-14) and the air-boundary plan.      */
int emm_grid_create(const double *x, int nx1, const double *y, int ny1, const double *z, int nz1,
                    const emm_grid_opts *opts, emm_grid **out);
void emm_grid_destroy(emm_grid *g);
int emm_grid_info(const emm_grid *g, int *ints /* EMM_I_COUNT */, double *dt /* 0 before emm_model_set */);
int emm_grid_coords(const emm_grid *g, int axis, double *nodes_out /* padded nodes, n?pad+1 */);
int emm_grid_fdcoef(const emm_grid *g, int axis, int plus, double *out /* [n?pad][2*rd] */);

/* Device memory and stream (both owned by the caller, e.g. a torch uint8 tensor and the current torch
 * stream).  emm_workspace_bytes: bytes needed for nsrc simultaneously resident sources, nfreq
 * frequencies, up to max_steps steps and nrec receivers with check_set <= EMM_CHECK_FACES (0 on error), in either
 * DTFT mode (full-grid accumulators with the field ring of the group `dtft_pair` stands for, see emm_run_opts, or
 * receivers only).  The first call creates the grid's cuFFT plans, hence the non-const handle.
 * The workspace must be 256-byte aligned and stay alive while the grid is used; binding it uploads
 * the per-grid tables and invalidates any earlier model.                                             */
size_t emm_workspace_bytes(emm_grid *g, int nsrc, int nfreq, int max_steps, int nrec, int dtft_pair);
int emm_bind_device(emm_grid *g, void *d_workspace, size_t bytes, void *cuda_stream);

/* Per-cell conductivity [nz][ny][nx] (S/m, finite, >0); sigma_v NULL => isotropic (VTI otherwise, L43).
 * Does the padding, the effective medium at each E component (Eq. 26), sigma -> fictitious
 * permittivity (L47), the time step (Eq. 15-16) and uploads dt/eps.  Needs a bound workspace.        */
int emm_model_set(emm_grid *g, const float *sigma_h, const float *sigma_v);

/* ---- the run (Algorithm 1) ------------------------------------------------------------------ */

/* One call: every source stepped to convergence (or fixed_steps).
 * out:    double complex [nsrc][nfreq][nrec][6] as (re,im) pairs: Green's functions Ex,Ey,Ez,Hx,Hy,Hz
 *         per unit dipole moment (Eq. 7); nsteps: [nsrc] steps executed.
 * nfreq = 0 (pure time stepping, no DTFT) is accepted with fixed_steps > 0 and nrec = 0 (timing runs).  */
int emm_run(emm_grid *g, const emm_src *src, int nsrc, const double *freqs_hz, int nfreq,
            const double *rec_xyz, int nrec, const emm_run_opts *opts, double *out, int *nsteps);

/* Split-phase form of the same loop for device-resident stepping: begin uploads the tables and zeroes
 * the state of all nsrc sources (resident together); steps enqueues n more iterations of lines 9-23
 * for every unfinished source and returns after the stream has drained; end applies Eq. 7 and
 * gathers the receivers.  emm_run_enqueue only enqueues (no host sync) and is meant for timing.      */
int emm_run_begin(emm_grid *g, const emm_src *src, int nsrc, const double *freqs_hz, int nfreq,
                  const double *rec_xyz, int nrec, const emm_run_opts *opts);
int emm_run_steps(emm_grid *g, int n, int *nsteps /* [nsrc] */, int *all_done);
int emm_run_enqueue(emm_grid *g, int n);
int emm_run_end(emm_grid *g, double *out, int *nsteps);
int emm_get(emm_grid *g, int isrc, int what, int ifreq, void *host_out);

/* Sensitivity (Frechet) kernel of a measured electric field with respect to the cell conductivities: what the full-grid
 * frequency-domain fields are accumulated for (inversion is the stated purpose; the paper gives no
 * formula, DESIGN.md [R14] states the one used).  Needs a run in progress (between emm_run_begin and emm_run_end) with
 * full-grid accumulators (sparse_dft = 0, dtft_every = 1) that holds two electric sources resident together: `isrc` = the
 * transmitter, `iadj` = a unit dipole at the receiver, polarised along the receiver channel.  For the datum
 * d = sum_c dir_c G^EE_c(receiver; transmitter) of frequency `ifreq`:
 *   out_h[cell] = d d / d sigma_h[cell],  out_v[cell] = d d / d sigma_v[cell]
 * HOST buffers, double complex [nz][ny][nx] as (re,im) pairs, caller-owned, overwritten.  Each value is the cell volume / 4
 * times the sum, over the cell's four edges per direction, of the product of the two sources' Green's functions (Eq. 7) at
 * the edge node: x and y edges into sigma_h, z edges into sigma_v; edge nodes outside the DTFT box do not count, padding
 * cells count towards the model cell they replicate.  fp64 products of the fp32 accumulators, a fixed summation order.
 * Errors: EMM_EINVAL (no run, magnetic source, receivers-only or decimated DTFT, a run with one source, bad index).      */
int emm_sensitivity(emm_grid *g, int isrc, int iadj, int ifreq, double *out_h, double *out_v);

/* Optional timing of the two fused update kernels: emm_profile(g,1) brackets every later launch of the
 * E and H update kernel with CUDA events on the bound stream; emm_profile_read drains the stream and
 * returns the summed durations and launch counts, then resets.  ms[6], counts[6]: {E, H} one-term (or decimated)
 * instances, {E, H} accumulator-free steps of a DTFT pair, {E, H} two-term steps of a DTFT pair.      */
int emm_profile(emm_grid *g, int enable);
int emm_profile_read(emm_grid *g, double *ms, int *counts);

/* ---- an entry point that allocates nothing -------------------------------------------------------------------------
 * The convergence measure of the run (L385-387, DESIGN.md [R9]) as a stand-alone call for callers that cannot call
 * cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation):
 *   delta[s][0] = || now - prev ||_2 / || now ||_2 over the three E components of source s, delta[s][1] the same over H,
 *   NaN where the denominator is 0.
 * It is a variant of the run driver's reduction kernels (warp shuffle + block reduction, per-block partial sums in scratch
 * memory, added in a fixed order); its scratch is a file-scope device array inside the library, 222 KB, held by every GPU
 * that loads the library until the process exits.  No cudaMalloc, cudaFree or allocating library routine is called.
 *   d_acc_now, d_acc_prev  DEVICE pointers, double complex [nsrc][6][nchk] as (re,im) pairs: the check-set accumulators now
 *                          and at the previous check (not modified)
 *   d_delta                DEVICE pointer, double [nsrc][2], written by kernels enqueued on cuda_stream (no host sync)
 * Limits: nsrc <= EMM_CHECK_STATIC_MAX_NSRC, nchk <= EMM_CHECK_STATIC_MAX_NCHK; larger sizes are rejected with EMM_EINVAL.
 * All calls share the one scratch array, which keeps the last call's contents; every slot a call reads it has written
 * itself, so nothing is cleared.  Calls that overlap on the GPU (two streams, two host threads) race on it: keep them on
 * one stream.  The device current at the call is the one used.                                                        */
#define EMM_CHECK_STATIC_MAX_NSRC 16
#define EMM_CHECK_STATIC_MAX_NCHK (1 << 27)
int emm_check_delta_static(const double *d_acc_now, const double *d_acc_prev, int nchk, int nsrc, double *d_delta, void *cuda_stream);

/* number of kernel launches issued by this library since the grid was created (bench evidence) */
long long emm_launch_count(const emm_grid *g);

const char *emm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
