/* emm_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, double-precision CPU restatement of the libEMM method
 * (arxiv 2304.00233, /root/reference/PAPER.md): fictitious-wave-domain FDTD
 * time stepping on a non-uniform staggered grid with CPML, the FFT air-water
 * boundary condition, source injection, on-the-fly DTFT and a convergence
 * check.  It follows Algorithm 1 step by step with naive
 * loops; nothing here is blocked, fused or reordered.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this library.  It shares no code with the
 * CUDA path under paper_2304_00233_b200/ (own header, own symbols `emmo_*`).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see DESIGN.md section
 * "Oracle, pins and parity tolerances".  Layered models with the air-water
 * boundary are pinned against a semi-analytic layered-earth solution
 * (tests/layered1d.py).  Physical accuracy on the 3-D models (configs[2..4])
 * is *parity unpinned*: no finite-element / integral-equation solver in the
 * container; they rest on the pins of the scheme's parts.
 *
 * All functions return 0 on success and a negative EMMO_E* code otherwise;
 * emmo_last_error() gives a message.  Arrays passed in are copied; output
 * buffers are caller-allocated.  SI units, z positive downward (L646-649),
 * x fastest: a[k][j][i] (L514).
 */
#ifndef EMM_ORACLE_H
#define EMM_ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

#define EMMO_EINVAL  (-1)
#define EMMO_ENOMEM  (-2)
#define EMMO_ENOCONV (-4)
#define EMMO_ENAN    (-5)

#define EMMO_TOP_CPML 0
#define EMMO_TOP_AIR  1

#define EMMO_CHECK_CORNERS 0
#define EMMO_CHECK_FACES   1
#define EMMO_CHECK_FULL    2

typedef struct emmo_grid emmo_grid;

typedef struct {
  int rd;          /* half stencil length r = 1,2,3 (L684)                      */
  int nb;          /* CPML cells per face (L305)                                */
  int ne;          /* buffer cells; <0 => rd+5 (L686)                           */
  int top;         /* EMMO_TOP_AIR (Eq.17-21) or EMMO_TOP_CPML                  */
  double f0;       /* omega0 = 2*pi*f0 (L47); <=0 => 1 Hz                       */
  double cfl;      /* dt = cfl/eta (Eq.15); <=0 => 0.99                   */
  double aux_dx;   /* auxiliary uniform plane spacing for NU x-y; <=0 => min    */
} emmo_grid_opts;

typedef struct {
  double pos[3]; double dir[3];
  int type;        /* 0: electric dipole J (Eq. 8); 1: magnetic dipole M (Eq. 8, inject_magnetic_src_fwd L457) */
} emmo_src;

typedef struct {
  int max_steps;    /* hard cap; <=0 => 100000                                  */
  int fixed_steps;  /* >0: run exactly this many steps, no convergence stop     */
  double tol;       /* <=0 => 1e-6                                              */
  int check_every;  /* <=0 => 100 (L458)                                        */
  int check_set;    /* EMMO_CHECK_*                                             */
  double fmax;      /* wavelet parameter; <=0 => 4*sqrt(max f * f0)             */
  int sparse_dft;   /* 1: accumulate only on receiver stencils (+check set)     */
  int dtft_every;   /* m > 1: take only every m-th term of the DTFT sums (Eq. 25) of the fields and of J'; the
                       check set keeps every term, so the stopping rule does not depend on m; 0, 1: every step;
                       < 0: the largest safe m = floor(1/(dt (3 fmax + 2 sqrt(max f * f0))))                   */
} emmo_run_opts;

/* grid info indices for emmo_grid_info(): ints */
enum { EMMO_I_N1 = 0, EMMO_I_N2, EMMO_I_N3, EMMO_I_LO1, EMMO_I_LO2, EMMO_I_LO3,
       EMMO_I_K0, EMMO_I_UNIFORM_XY, EMMO_I_BOX_LO1, EMMO_I_BOX_LO2, EMMO_I_BOX_LO3,
       EMMO_I_BOX_HI1, EMMO_I_BOX_HI2, EMMO_I_BOX_HI3, EMMO_I_AUX_M1, EMMO_I_AUX_M2,
       EMMO_I_COUNT };

/* `what` codes for emmo_get(): */
enum { EMMO_GET_E1 = 0, EMMO_GET_E2, EMMO_GET_E3, EMMO_GET_H1, EMMO_GET_H2, EMMO_GET_H3, /* double[N3][N2][N1] */
       EMMO_GET_F_E1 = 10, EMMO_GET_F_E2, EMMO_GET_F_E3, EMMO_GET_F_H1, EMMO_GET_F_H2, EMMO_GET_F_H3, /* complex double [N3][N2][N1], zero outside the DFT set; needs ifreq */
       EMMO_GET_CE1 = 20, EMMO_GET_CE2, EMMO_GET_CE3,      /* dt/eps per component, double[N3][N2][N1] */
       EMMO_GET_JW = 30,                                   /* complex double [nfreq]: J'(omega') so far */
       EMMO_GET_DELTA = 31,                                /* double[2]: delta_E, delta_H of the last check */
       EMMO_GET_CPML = 40                                  /* double [4][2*nb] of axis `ifreq` (0,1,2): a and b of Eq. 24 at the node
                                                              positions (D-), then a and b at the half-node positions (D+); slab
                                                              index as L324-326 (low face 0..nb-1, high face mirrored nb..2nb-1)     */
};

/* Eq.27-29 / listing L421-443: geometric grid, n intervals, total length len, first interval dx. */
int emmo_nugrid(int n, double len, double dx, double *x_out /* n+1 */, double *q_out);

/* Eq.10-12 / listing L130-146: weights of the npts nodes for f(x0) (row 0) and f'(x0) (row 1). */
int emmo_fd_weights(int npts, const double *nodes, double x0, double *w_interp, double *w_deriv);

/* test surface: in-place 2-D DFT of a[n2][n1] (complex double as re,im pairs); sign=-1 forward
 * (includes 1/(n1*n2)), sign=+1 inverse (no factor).  Convention f(x)=sum F(k) e^{+ikx} (Eq.32). */
int emmo_fft2(double *a, int n1, int n2, int sign);

int emmo_grid_create(const double *x, int nx1, const double *y, int ny1, const double *z, int nz1,
                     const emmo_grid_opts *o, emmo_grid **out);
void emmo_grid_destroy(emmo_grid *g);
int emmo_grid_info(const emmo_grid *g, int *ints /* EMMO_I_COUNT */, double *dt /* 0 until model set */);
int emmo_grid_coords(const emmo_grid *g, int axis, double *nodes_out /* N+1 padded node coordinates */);
int emmo_grid_fdcoef(const emmo_grid *g, int axis, int plus, double *out /* [N][2r] */);

/* per-cell conductivity [nz][ny][nx]; sigma_v NULL => isotropic. (Eq.26, Eq.15-16) */
int emmo_model_set(emmo_grid *g, const float *sigma_h, const float *sigma_v);

/* One-shot: runs every source to convergence (or fixed_steps).
 * out: complex double [nsrc][nfreq][nrec][6] (Ex,Ey,Ez,Hx,Hy,Hz Green's functions, Eq.7); nsteps: [nsrc]. */
int emmo_run(emmo_grid *g, const emmo_src *src, int nsrc, const double *freqs_hz, int nfreq,
             const double *rec_xyz, int nrec, const emmo_run_opts *o, double *out, int *nsteps);

/* Split-phase form of the same loop, state kept in the handle (used for field parity and timing). */
int emmo_run_begin(emmo_grid *g, const emmo_src *src, int nsrc, const double *freqs_hz, int nfreq,
                   const double *rec_xyz, int nrec, const emmo_run_opts *o);
int emmo_run_steps(emmo_grid *g, int n, int *nsteps /* [nsrc] steps executed so far */, int *all_done);
int emmo_run_end(emmo_grid *g, double *out, int *nsteps);
int emmo_get(emmo_grid *g, int isrc, int what, int ifreq, void *host_out);

/* Sensitivity (Frechet) kernel of a measured electric field with respect to the cell conductivities -- what the
 * full-grid frequency-domain fields are kept for (inversion is the stated perspective; the paper
 * gives no formula, DESIGN.md [R14] states the one used).  Needs a run in progress with full-grid accumulators
 * (sparse_dft = 0) holding two electric sources: `isrc` = the transmitter, `iadj` = a unit dipole at the receiver,
 * polarised along the receiver channel.  For the datum d = sum_c dir_c G^EE_c(receiver; transmitter) of frequency ifreq:
 *   out_h[cell] = d d / d sigma_h[cell],  out_v[cell] = d d / d sigma_v[cell]   (complex double [nz][ny][nx] each),
 * = sum over the E nodes n whose effective conductivity (Eq. 26, [R3]) contains the cell:
 *   (d sigma_bar_c(n) / d sigma[cell]) * V(n) * G_c(n; transmitter) * G_c(n; receiver dipole),
 * G = Green's functions on the grid (Eq. 7), V(n) = node volume of the component's lattice ([R7]); sigma_h collects the
 * x and y components, sigma_v the z component.  Padding cells count towards the model cell they replicate.            */
int emmo_sensitivity(emmo_grid *g, int isrc, int iadj, int ifreq, double *out_h, double *out_v);

const char *emmo_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
