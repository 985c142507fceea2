/* emm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.  See emm_oracle.h.
 *
 * Double-precision, loop-by-loop restatement of the libEMM time-stepping method
 * (/root/reference/PAPER.md).  Each function cites the passage it follows; readings
 * of silent/garbled passages are listed in DESIGN.md ("Readings") and referenced here
 * as [R1]..[R12].  OpenMP pragmas only spread the outermost loops over threads; they do
 * not change the arithmetic of any node.
 */
#include "emm_oracle.h"
#include <complex.h>
#include <math.h>
#include <stdarg.h>
#include <stddef.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;
#define MU0 (4e-7 * M_PI)

static __thread char g_err[512];
static int fail(int code, const char *fmt, ...) {
  va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap);
  return code;
}
const char *emmo_last_error(void) { return g_err; }

/* ------------------------------------------------------------------------------------------ */
/* Vandermonde solve V^T(x0..xn) a = f.  PAPER.md listing L130-146 (Golub Alg. 4.6.1), braces  */
/* restored, double instead of float.                                                          */
static void vandermonde(int n, const double *x, double *a, const double *f) {
  int i, k;
  for (i = 0; i <= n; ++i) a[i] = f[i];
  for (k = 0; k < n; k++)
    for (i = n; i > k; i--) a[i] = (a[i] - a[i - 1]) / (x[i] - x[i - k - 1]);
  for (k = n - 1; k >= 0; k--)
    for (i = k; i < n; i++) a[i] -= a[i + 1] * x[k];
}

/* Eq. 12 (L173-176): feed unit vectors, column j of [V^T]^-1 comes out; row 0 = interpolation
 * weights, row 1 = first-derivative weights (Eq. 9-11, a_i = f^(i)/i!).                        */
int emmo_fd_weights(int npts, const double *nodes, double x0, double *w_interp, double *w_deriv) {
  if (npts < 2 || npts > 16 || !nodes) return fail(EMMO_EINVAL, "fd_weights: bad npts");
  double off[16], f[16], a[16];
  for (int i = 0; i < npts; i++) off[i] = nodes[i] - x0;
  for (int j = 0; j < npts; j++) {
    for (int i = 0; i < npts; i++) f[i] = (i == j) ? 1.0 : 0.0;
    vandermonde(npts - 1, off, a, f);
    if (w_interp) w_interp[j] = a[0];
    if (w_deriv) w_deriv[j] = a[1];
  }
  return 0;
}

/* Eq. 27-29, listing L421-443 (fixed-point iteration q <- (L/dx (q-1) + 1)^(1/n)).            */
int emmo_nugrid(int n, double len, double dx, double *x, double *q_out) {
  if (n < 1 || !(len > 0) || !(dx > 0) || !x) return fail(EMMO_EINVAL, "nugrid: bad arguments");
  if (fabs(n * dx - len) < 1e-12 * len) { /* listing L430 (absolute 1e-15 there; relative here) */
    for (int i = 0; i <= n; i++) x[i] = i * dx;
    if (q_out) *q_out = 1.0;
    return 0;
  }
  if (n * dx > len) return fail(EMMO_EINVAL, "nugrid: n*dx > len has no root q>1");
  double q = 1.1, qq;
  for (int iter = 0; iter < 100000; iter++) {
    qq = pow(len * (q - 1.) / dx + 1., 1. / n);
    if (fabs(qq - q) < 1e-15) { q = qq; break; }
    q = qq;
  }
  x[0] = 0;
  for (int i = 1; i <= n; i++) x[i] = (pow(q, i) - 1.) * dx / (q - 1.);
  if (q_out) *q_out = q;
  return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Plain mixed-radix DFT (decimation in time, any length; prime factors handled by the          */
/* definition).  Library-primitive step of the air-wave boundary (L282-288, L524).             */
typedef struct { int n; cplx *w; /* w[j] = exp(-2 pi i j / n) */ } fftplan;

static int fftplan_init(fftplan *p, int n) {
  p->n = n;
  p->w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
  if (!p->w) return -1;
  for (int j = 0; j < n; j++) p->w[j] = cexp(-2.0 * M_PI * I * (double)j / (double)n);
  return 0;
}
static void fftplan_free(fftplan *p) { free(p->w); p->w = NULL; }

static int smallest_factor(int n) {
  for (int p = 2; p * p <= n; p++) if (n % p == 0) return p;
  return n;
}

/* FB lines are transformed together: element t of line c sits at v[t*FB + c] (re) / vi[...] (im), so that every
 * inner loop runs over the FB lines with one twiddle factor.  Per line this is the plain recursion
 *   out[k + j m] = sum_q W_n^{q (k + j m)} sub_q[k],   sub_q = transform of in[q], in[q + p], ...   (n = p m, p prime)
 * with the sum over q taken in order q = 0..p-1; length n, W = exp(-2 pi i/n) (sign < 0) or its conjugate.      */
#define FB 16
static void fft_rec(const fftplan *pl, const double *inr, const double *ini, int stride, double *outr, double *outi,
                    int n, int sign, double *tr, double *ti) {
  if (n == 1) {
    for (int c = 0; c < FB; c++) { outr[c] = inr[c]; outi[c] = ini[c]; }
    return;
  }
  int p = smallest_factor(n), m = n / p;
  for (int q = 0; q < p; q++)
    fft_rec(pl, inr + (size_t)q * stride * FB, ini + (size_t)q * stride * FB, stride * p, outr + (size_t)q * m * FB,
            outi + (size_t)q * m * FB, m, sign, tr, ti);
  int step = pl->n / n; /* W_n^a = w[a*step] */
  const double sg = sign > 0 ? -1.0 : 1.0;       /* sign > 0: conjugate twiddles */
  for (int k = 0; k < m; k++) {
    for (int j = 0; j < p; j++) {
      int kk = k + j * m;
      double *ar = tr + (size_t)kk * FB, *ai = ti + (size_t)kk * FB;
      for (int c = 0; c < FB; c++) { ar[c] = 0; ai[c] = 0; }
      int a = 0;                                 /* (q * kk) mod n, carried from q to q + 1 */
      for (int q = 0; q < p; q++) {
        const double wr = creal(pl->w[(size_t)a * step]), wi = sg * cimag(pl->w[(size_t)a * step]);
        const double *xr = outr + ((size_t)q * m + k) * FB, *xi = outi + ((size_t)q * m + k) * FB;
#pragma omp simd
        for (int c = 0; c < FB; c++) {
          ar[c] += wr * xr[c] - wi * xi[c];
          ai[c] += wr * xi[c] + wi * xr[c];
        }
        a += kk; if (a >= n) a -= n;
      }
    }
  }
  /* second pass needed because out[q*m+k] for all q are inputs of all j */
  memcpy(outr, tr, sizeof(double) * (size_t)n * FB);
  memcpy(outi, ti, sizeof(double) * (size_t)n * FB);
}

/* nl lines of length n of a[], element stride es, line stride ls, transformed in place, FB lines at a time */
static int fft_lines(cplx *a, int n, size_t es, int nl, size_t ls, int sign, const fftplan *pl) {
  int err = 0;
#pragma omp parallel
  {
    double *buf = (double *)malloc(sizeof(double) * 6 * (size_t)n * FB);
    if (!buf) {
#pragma omp atomic write
      err = 1;
    } else {
      double *inr = buf, *ini = buf + (size_t)n * FB, *outr = buf + 2 * (size_t)n * FB, *outi = buf + 3 * (size_t)n * FB,
             *tr = buf + 4 * (size_t)n * FB, *ti = buf + 5 * (size_t)n * FB;
#pragma omp for schedule(dynamic, 1)
      for (int l0 = 0; l0 < nl; l0 += FB) {
        const int nc = nl - l0 < FB ? nl - l0 : FB;
        for (int t = 0; t < n; t++)
          for (int c = 0; c < FB; c++) {
            const cplx v = c < nc ? a[(size_t)(l0 + c) * ls + (size_t)t * es] : 0;
            inr[(size_t)t * FB + c] = creal(v); ini[(size_t)t * FB + c] = cimag(v);
          }
        fft_rec(pl, inr, ini, 1, outr, outi, n, sign, tr, ti);
        for (int t = 0; t < n; t++)
          for (int c = 0; c < nc; c++) a[(size_t)(l0 + c) * ls + (size_t)t * es] = outr[(size_t)t * FB + c] + I * outi[(size_t)t * FB + c];
      }
      free(buf);
    }
  }
  return err ? -1 : 0;
}

/* 2-D transform of a[n2][n1] in place.  sign=-1: F(k) = 1/(n1 n2) sum f e^{-ikx}; sign=+1:     */
/* f = sum F e^{+ikx}  (convention of Eq. 32).                                           */
static int fft2_inplace(cplx *a, int n1, int n2, int sign, const fftplan *p1, const fftplan *p2) {
  if (fft_lines(a, n1, 1, n2, (size_t)n1, sign, p1)) return -1;      /* rows    */
  if (fft_lines(a, n2, (size_t)n1, n1, 1, sign, p2)) return -1;      /* columns */
  if (sign < 0) {
    double s = 1.0 / ((double)n1 * (double)n2);
#pragma omp parallel for schedule(static)
    for (int j = 0; j < n2; j++) for (int i = 0; i < n1; i++) a[(size_t)j * n1 + i] *= s;
  }
  return 0;
}

int emmo_fft2(double *a, int n1, int n2, int sign) {
  if (!a || n1 < 1 || n2 < 1) return fail(EMMO_EINVAL, "fft2: bad arguments");
  fftplan p1, p2;
  if (fftplan_init(&p1, n1)) return fail(EMMO_ENOMEM, "fft2: out of memory");
  if (fftplan_init(&p2, n2)) { fftplan_free(&p1); return fail(EMMO_ENOMEM, "fft2: out of memory"); }
  int rc = fft2_inplace((cplx *)a, n1, n2, sign, &p1, &p2);
  fftplan_free(&p1); fftplan_free(&p2);
  return rc ? fail(EMMO_ENOMEM, "fft2: out of memory") : 0;
}

/* ------------------------------------------------------------------------------------------ */
typedef struct {           /* one source's time-stepping state */
  double *E[3], *H[3];
  double *psiE[6];         /* memory variables of the 6 H-derivatives used by the E update:
                              0:D1H3 1:D1H2 (x slabs) 2:D2H3 3:D2H1 (y) 4:D3H2 5:D3H1 (z)       */
  double *psiH[6];         /* of the 6 E-derivatives: 0:D1E3 1:D1E2 2:D2E3 3:D2E1 4:D3E2 5:D3E1 */
  int nsn[3]; size_t *sidx[3]; double *sw[3]; /* source nodes and weights W_c (c-6)            */
  int magnetic;            /* 1: the weights live on the H lattices and M is injected into H   */
  cplx *F;                 /* [(c*nf+f)*ndft + p], c = 0..5 (E1..H3)                            */
  cplx *Jw;                /* [nf] J'(omega')                                                   */
  cplx *Cnow, *Cprev;      /* [6][nchk] check-set accumulators, lowest frequency               */
  double delta[2];
  int nsteps, done;
} srcstate;

typedef struct { int start; double w[8]; } stencil1;

typedef struct {
  int nsrc, nf, nrec;
  double *freqs; cplx *wp;         /* omega' = (1+i) sqrt(omega omega0), Eq. 4                  */
  int fmin;                        /* index of the lowest frequency (L387)                      */
  double fmax, beta, t0;
  int max_steps, fixed_steps, check_every, check_set, sparse, dtft_every; double tol;
  size_t ndft; size_t *dft_idx;    /* sorted node indices carrying DFT accumulators             */
  size_t nchk; size_t *chk_idx;
  int np;                          /* interpolation points per axis, max(2r,4) (c-6)            */
  stencil1 *rst;                   /* [nrec][6][3]                                              */
  double *am[3], *bm[3], *ap[3], *bp[3]; /* CPML a,b at node (D-) and half-node (D+) positions  */
  srcstate *s;
} runstate;

struct emmo_grid {
  int r, nb, ne, top; double f0, w0, cfl, aux_dx;
  int nc[3], N[3], lo[3];
  double *xn[3], *xh[3];           /* padded nodes [N+1], half nodes [N]                        */
  double *cm[3], *cp[3];           /* D-, D+ coefficients [N][2r]                               */
  double Dmax[3];
  int k0, klo, uniform_xy;
  int blo[3], bhi[3];              /* DFT box, inclusive                                        */
  /* model */
  int have_model; double *sh, *sv; /* padded cell conductivities [N3][N2][N1]                   */
  double *ce[3]; double dt;
  /* air-wave boundary */
  int M1, M2; double dxa, dya;     /* transform plane                                           */
  fftplan p1, p2; int have_plans;
  stencil1 *toaux[2][2];           /* [axis][lattice 0=node 1=half][M]: lattice -> aux          */
  stencil1 *fromaux[2][2];         /* [axis][lattice][N]: aux -> lattice                        */
  runstate *run;
};

#define IDX(g, i, j, k) ((size_t)(i) + (size_t)(g)->N[0] * ((size_t)(j) + (size_t)(g)->N[1] * (size_t)(k)))

static int is_smooth7(int n) {
  for (int p = 2; p <= 7; p++) while (n % p == 0) n /= p;
  return n == 1;
}
static int smooth_up(int n) { while (!is_smooth7(n)) n++; return n; }

static int axis_uniform(const double *x, int n1) {
  double d0 = x[1] - x[0];
  for (int i = 1; i < n1 - 1; i++) if (fabs((x[i + 1] - x[i]) - d0) > 1e-9 * d0) return 0;
  return 1;
}

/* interpolation stencil of p points on lattice S[0..n-1] around target t (c-6 / L167-178):     */
/* i0 = last lattice point <= t, points i0-p/2+1 .. i0+p/2, weights = row 0 of Eq. 11.          */
static int lattice_stencil(const double *S, int n, double t, int p, int lo_ok, stencil1 *st) {
  if (!(t >= S[0]) || !(t <= S[n - 1])) return -1;
  int i0 = 0;
  while (i0 + 1 < n && S[i0 + 1] <= t) i0++;
  if (i0 == n - 1) i0 = n - 2;
  int start = i0 - p / 2 + 1;
  if (start < lo_ok || start + p - 1 > n - 1) return -1;
  st->start = start;
  emmo_fd_weights(p, S + start, t, st->w, NULL);
  return 0;
}

/* same, but the stencil is shifted to stay inside [0,n-1] and targets outside the lattice get  */
/* zero weights (used only by the auxiliary-plane air boundary, [R10]).                         */
static void lattice_stencil_clamped(const double *S, int n, double t, int p, stencil1 *st) {
  memset(st, 0, sizeof *st);
  if (!(t >= S[0]) || !(t <= S[n - 1])) return;
  int i0 = 0;
  while (i0 + 1 < n && S[i0 + 1] <= t) i0++;
  if (i0 == n - 1) i0 = n - 2;
  int start = i0 - p / 2 + 1;
  if (start < 0) start = 0;
  if (start + p - 1 > n - 1) start = n - p;
  st->start = start;
  emmo_fd_weights(p, S + start, t, st->w, NULL);
}

static void free_airbc(emmo_grid *g) {
  if (g->have_plans) { fftplan_free(&g->p1); fftplan_free(&g->p2); g->have_plans = 0; }
  for (int a = 0; a < 2; a++) for (int l = 0; l < 2; l++) {
    free(g->toaux[a][l]); g->toaux[a][l] = NULL;
    free(g->fromaux[a][l]); g->fromaux[a][l] = NULL;
  }
}

static void free_run(emmo_grid *g);

void emmo_grid_destroy(emmo_grid *g) {
  if (!g) return;
  free_run(g);
  free_airbc(g);
  for (int a = 0; a < 3; a++) { free(g->xn[a]); free(g->xh[a]); free(g->cm[a]); free(g->cp[a]); free(g->ce[a]); }
  free(g->sh); free(g->sv);
  free(g);
}

/* Grid: padding (L305-312, [R1]), Yee placement ([R2]), D+/D- tables (Eq. 13-14).    */
int emmo_grid_create(const double *x, int nx1, const double *y, int ny1, const double *z, int nz1,
                     const emmo_grid_opts *o, emmo_grid **out) {
  if (!x || !y || !z || !o || !out) return fail(EMMO_EINVAL, "grid_create: null argument");
  if (o->rd < 1 || o->rd > 3) return fail(EMMO_EINVAL, "grid_create: rd must be 1,2,3 (L684)");
  if (o->nb < 1) return fail(EMMO_EINVAL, "grid_create: nb must be >= 1");
  if (o->top != EMMO_TOP_AIR && o->top != EMMO_TOP_CPML) return fail(EMMO_EINVAL, "grid_create: bad top");
  const double *u[3] = {x, y, z}; int n1s[3] = {nx1, ny1, nz1};
  for (int a = 0; a < 3; a++) {
    if (n1s[a] < 3) return fail(EMMO_EINVAL, "grid_create: need at least 2 cells per axis");
    for (int i = 0; i + 1 < n1s[a]; i++)
      if (!(u[a][i + 1] > u[a][i]) || !isfinite(u[a][i]) || !isfinite(u[a][i + 1]))
        return fail(EMMO_EINVAL, "grid_create: axis %d coordinates not strictly increasing", a);
  }
  emmo_grid *g = (emmo_grid *)calloc(1, sizeof *g);
  if (!g) return fail(EMMO_ENOMEM, "grid_create: out of memory");
  g->r = o->rd; g->nb = o->nb; g->ne = o->ne < 0 ? o->rd + 5 : o->ne; g->top = o->top;
  g->f0 = o->f0 > 0 ? o->f0 : 1.0; g->w0 = 2 * M_PI * g->f0;
  g->cfl = o->cfl > 0 ? o->cfl : 0.99; g->aux_dx = o->aux_dx;
  int r = g->r, nbe = g->nb + g->ne;
  if (g->ne < r) { free(g); return fail(EMMO_EINVAL, "grid_create: ne must be >= rd (L686)"); }
  g->uniform_xy = axis_uniform(x, nx1) && axis_uniform(y, ny1);
  for (int a = 0; a < 3; a++) {
    g->nc[a] = n1s[a] - 1;
    int lo = nbe, hi = nbe;
    if (a == 2 && g->top == EMMO_TOP_AIR) lo = r;           /* [R1]: r ghost planes above z=0 */
    int N = g->nc[a] + lo + hi;
    if (a < 2 && g->top == EMMO_TOP_AIR && g->uniform_xy) N = smooth_up(N); /* [R1] FFT-friendly */
    g->lo[a] = lo; g->N[a] = N;
    g->xn[a] = (double *)malloc(sizeof(double) * (size_t)(N + 1));
    g->xh[a] = (double *)malloc(sizeof(double) * (size_t)N);
    g->cm[a] = (double *)calloc((size_t)N * 2 * r, sizeof(double));
    g->cp[a] = (double *)calloc((size_t)N * 2 * r, sizeof(double));
    if (!g->xn[a] || !g->xh[a] || !g->cm[a] || !g->cp[a]) { emmo_grid_destroy(g); return fail(EMMO_ENOMEM, "grid_create: out of memory"); }
    double dlo = u[a][1] - u[a][0], dhi = u[a][g->nc[a]] - u[a][g->nc[a] - 1];
    for (int i = 0; i <= N; i++) {                          /* [R1]: edge spacing held constant */
      int c = i - lo;
      if (c < 0) g->xn[a][i] = u[a][0] + c * dlo;
      else if (c > g->nc[a]) g->xn[a][i] = u[a][g->nc[a]] + (c - g->nc[a]) * dhi;
      else g->xn[a][i] = u[a][c];
    }
    for (int i = 0; i < N; i++) g->xh[a][i] = 0.5 * (g->xn[a][i] + g->xn[a][i + 1]); /* [R2] midpoint */
    /* Eq. 14: D- at x_i from half nodes xh[i-r .. i+r-1]; Eq. 13: D+ at xh_i from nodes x[i-r+1 .. i+r] */
    g->Dmax[a] = 0;
    for (int i = r; i <= N - 1 - r; i++) {
      emmo_fd_weights(2 * r, g->xh[a] + (i - r), g->xn[a][i], NULL, g->cm[a] + (size_t)i * 2 * r);
      emmo_fd_weights(2 * r, g->xn[a] + (i - r + 1), g->xh[a][i], NULL, g->cp[a] + (size_t)i * 2 * r);
      double sm = 0, sp = 0;
      for (int m = 0; m < 2 * r; m++) { sm += fabs(g->cm[a][(size_t)i * 2 * r + m]); sp += fabs(g->cp[a][(size_t)i * 2 * r + m]); }
      if (sm > g->Dmax[a]) g->Dmax[a] = sm;                 /* Eq. 16 */
      if (sp > g->Dmax[a]) g->Dmax[a] = sp;
    }
  }
  g->k0 = g->top == EMMO_TOP_AIR ? r : -1;
  g->klo = r;
  for (int a = 0; a < 3; a++) { g->blo[a] = g->nb; g->bhi[a] = g->N[a] - 1 - g->nb; } /* L365-370, [R11] */
  if (g->top == EMMO_TOP_AIR) g->blo[2] = g->k0;
  /* air-wave transform plane ([R10]) */
  if (g->top == EMMO_TOP_AIR) {
    if (g->uniform_xy) {
      g->M1 = g->N[0]; g->M2 = g->N[1];
      g->dxa = g->xn[0][1] - g->xn[0][0]; g->dya = g->xn[1][1] - g->xn[1][0];
    } else {
      double dmin[2];
      for (int a = 0; a < 2; a++) {
        dmin[a] = u[a][1] - u[a][0];
        for (int i = 0; i + 1 < n1s[a]; i++) if (u[a][i + 1] - u[a][i] < dmin[a]) dmin[a] = u[a][i + 1] - u[a][i];
      }
      g->dxa = g->aux_dx > 0 ? g->aux_dx : dmin[0];
      g->dya = g->aux_dx > 0 ? g->aux_dx : dmin[1];
      g->M1 = smooth_up((int)floor((g->xn[0][g->N[0]] - g->xn[0][0]) / g->dxa) + 2);
      g->M2 = smooth_up((int)floor((g->xn[1][g->N[1]] - g->xn[1][0]) / g->dya) + 2);
      for (int a = 0; a < 2; a++) {
        int M = a == 0 ? g->M1 : g->M2; double da = a == 0 ? g->dxa : g->dya;
        double *xa = (double *)malloc(sizeof(double) * (size_t)M);
        if (!xa) { emmo_grid_destroy(g); return fail(EMMO_ENOMEM, "grid_create: out of memory"); }
        for (int m = 0; m < M; m++) xa[m] = g->xn[a][0] + m * da;
        for (int l = 0; l < 2; l++) {
          const double *S = l ? g->xh[a] : g->xn[a];
          g->toaux[a][l] = (stencil1 *)malloc(sizeof(stencil1) * (size_t)M);
          g->fromaux[a][l] = (stencil1 *)malloc(sizeof(stencil1) * (size_t)g->N[a]);
          if (!g->toaux[a][l] || !g->fromaux[a][l]) { free(xa); emmo_grid_destroy(g); return fail(EMMO_ENOMEM, "grid_create: out of memory"); }
          for (int m = 0; m < M; m++) lattice_stencil_clamped(S, g->N[a], xa[m], 4, &g->toaux[a][l][m]);
          for (int i = 0; i < g->N[a]; i++) lattice_stencil_clamped(xa, M, S[i], 4, &g->fromaux[a][l][i]);
        }
        free(xa);
      }
    }
    if (fftplan_init(&g->p1, g->M1) || fftplan_init(&g->p2, g->M2)) { emmo_grid_destroy(g); return fail(EMMO_ENOMEM, "grid_create: out of memory"); }
    g->have_plans = 1;
  }
  *out = g;
  return 0;
}

int emmo_grid_info(const emmo_grid *g, int *ints, double *dt) {
  if (!g) return fail(EMMO_EINVAL, "grid_info: null grid");
  if (ints) {
    for (int a = 0; a < 3; a++) {
      ints[EMMO_I_N1 + a] = g->N[a]; ints[EMMO_I_LO1 + a] = g->lo[a];
      ints[EMMO_I_BOX_LO1 + a] = g->blo[a]; ints[EMMO_I_BOX_HI1 + a] = g->bhi[a];
    }
    ints[EMMO_I_K0] = g->k0; ints[EMMO_I_UNIFORM_XY] = g->uniform_xy;
    ints[EMMO_I_AUX_M1] = g->M1; ints[EMMO_I_AUX_M2] = g->M2;
  }
  if (dt) *dt = g->have_model ? g->dt : 0.0;
  return 0;
}
int emmo_grid_coords(const emmo_grid *g, int axis, double *nodes_out) {
  if (!g || axis < 0 || axis > 2 || !nodes_out) return fail(EMMO_EINVAL, "grid_coords: bad arguments");
  memcpy(nodes_out, g->xn[axis], sizeof(double) * (size_t)(g->N[axis] + 1));
  return 0;
}
int emmo_grid_fdcoef(const emmo_grid *g, int axis, int plus, double *out) {
  if (!g || axis < 0 || axis > 2 || !out) return fail(EMMO_EINVAL, "grid_fdcoef: bad arguments");
  memcpy(out, plus ? g->cp[axis] : g->cm[axis], sizeof(double) * (size_t)g->N[axis] * 2 * g->r);
  return 0;
}

/* Medium (Eq. 26, [R3]) and time step (Eq. 15-16, [R4]).                            */
int emmo_model_set(emmo_grid *g, const float *sigma_h, const float *sigma_v) {
  if (!g || !sigma_h) return fail(EMMO_EINVAL, "model_set: null argument");
  free_run(g);
  const int N1 = g->N[0], N2 = g->N[1], N3 = g->N[2], r = g->r;
  size_t ncell_in = (size_t)g->nc[0] * g->nc[1] * g->nc[2];
  for (size_t t = 0; t < ncell_in; t++) {
    if (!(sigma_h[t] > 0) || !isfinite(sigma_h[t])) return fail(EMMO_EINVAL, "model_set: sigma_h must be finite and > 0");
    if (sigma_v && (!(sigma_v[t] > 0) || !isfinite(sigma_v[t]))) return fail(EMMO_EINVAL, "model_set: sigma_v must be finite and > 0");
  }
  size_t N = (size_t)N1 * N2 * N3;
  if (!g->sh) g->sh = (double *)malloc(sizeof(double) * N);
  if (!g->sv) g->sv = (double *)malloc(sizeof(double) * N);
  for (int c = 0; c < 3; c++) if (!g->ce[c]) g->ce[c] = (double *)malloc(sizeof(double) * N);
  if (!g->sh || !g->sv || !g->ce[0] || !g->ce[1] || !g->ce[2]) return fail(EMMO_ENOMEM, "model_set: out of memory");
  /* [R3] padded cells: replicate the edge cell; cells above z=0 are air (sigma = 0) when top=AIR */
  for (int k = 0; k < N3; k++) for (int j = 0; j < N2; j++) for (int i = 0; i < N1; i++) {
    int ci = i - g->lo[0], cj = j - g->lo[1], ck = k - g->lo[2];
    double a, b;
    if (g->top == EMMO_TOP_AIR && ck < 0) { a = 0; b = 0; }
    else {
      ci = ci < 0 ? 0 : (ci > g->nc[0] - 1 ? g->nc[0] - 1 : ci);
      cj = cj < 0 ? 0 : (cj > g->nc[1] - 1 ? g->nc[1] - 1 : cj);
      ck = ck < 0 ? 0 : (ck > g->nc[2] - 1 ? g->nc[2] - 1 : ck);
      size_t t = (size_t)ci + (size_t)g->nc[0] * ((size_t)cj + (size_t)g->nc[1] * (size_t)ck);
      a = sigma_h[t]; b = sigma_v ? sigma_v[t] : sigma_h[t];
    }
    g->sh[IDX(g, i, j, k)] = a; g->sv[IDX(g, i, j, k)] = b;
  }
  /* [R3] effective conductivity at each E component = area-weighted arithmetic mean of the four
   * cells sharing its edge (tangential component, "resistors in parallel", L400).  Stored
   * temporarily in ce[]; converted to dt/eps below.                                            */
  const double *X = g->xn[0], *Y = g->xn[1], *Z = g->xn[2];
  double smin = INFINITY;
  for (int k = 0; k < N3; k++) for (int j = 0; j < N2; j++) for (int i = 0; i < N1; i++) {
    int im = i > 0 ? i - 1 : 0, jm = j > 0 ? j - 1 : 0, km = k > 0 ? k - 1 : 0;
    double dx0 = X[im + 1] - X[im], dx1 = X[i + 1] - X[i];
    double dy0 = Y[jm + 1] - Y[jm], dy1 = Y[j + 1] - Y[j];
    double dz0 = Z[km + 1] - Z[km], dz1 = Z[k + 1] - Z[k];
    double s11 = (g->sh[IDX(g, i, jm, km)] * dy0 * dz0 + g->sh[IDX(g, i, j, km)] * dy1 * dz0 +
                  g->sh[IDX(g, i, jm, k)] * dy0 * dz1 + g->sh[IDX(g, i, j, k)] * dy1 * dz1) / ((dy0 + dy1) * (dz0 + dz1));
    double s22 = (g->sh[IDX(g, im, j, km)] * dx0 * dz0 + g->sh[IDX(g, i, j, km)] * dx1 * dz0 +
                  g->sh[IDX(g, im, j, k)] * dx0 * dz1 + g->sh[IDX(g, i, j, k)] * dx1 * dz1) / ((dx0 + dx1) * (dz0 + dz1));
    double s33 = (g->sv[IDX(g, im, jm, k)] * dx0 * dy0 + g->sv[IDX(g, i, jm, k)] * dx1 * dy0 +
                  g->sv[IDX(g, im, j, k)] * dx0 * dy1 + g->sv[IDX(g, i, j, k)] * dx1 * dy1) / ((dx0 + dx1) * (dy0 + dy1));
    int upd = i >= r && i <= N1 - 1 - r && j >= r && j <= N2 - 1 - r && k >= g->klo && k <= N3 - 1 - r;
    size_t t = IDX(g, i, j, k);
    g->ce[0][t] = upd ? s11 : 0; g->ce[1][t] = upd ? s22 : 0; g->ce[2][t] = upd ? s33 : 0;
    if (upd) {
      if (s11 < smin) smin = s11;
      if (s22 < smin) smin = s22;
      if (s33 < smin) smin = s33;
    }
  }
  if (!(smin > 0)) return fail(EMMO_EINVAL, "model_set: non-positive effective conductivity at an updated node");
  /* Eq. 15-16: eta = 1/2 vmax sqrt(sum Dmax^2), v = 1/sqrt(mu eps), eps = sigma/(2 omega0) (L47) */
  double vmax = 1.0 / sqrt(MU0 * smin / (2 * g->w0));
  double eta = 0.5 * vmax * sqrt(g->Dmax[0] * g->Dmax[0] + g->Dmax[1] * g->Dmax[1] + g->Dmax[2] * g->Dmax[2]);
  g->dt = g->cfl / eta;
  for (int c = 0; c < 3; c++)
    for (size_t t = 0; t < N; t++) g->ce[c][t] = g->ce[c][t] > 0 ? g->dt * 2 * g->w0 / g->ce[c][t] : 0.0;
  g->have_model = 1;
  return 0;
}

/* ------------------------------------------------------------------------------------------ */
static void free_run(emmo_grid *g) {
  runstate *R = g->run;
  if (!R) return;
  if (R->s) for (int s = 0; s < R->nsrc; s++) {
    srcstate *S = &R->s[s];
    for (int c = 0; c < 3; c++) { free(S->E[c]); free(S->H[c]); free(S->sidx[c]); free(S->sw[c]); }
    for (int q = 0; q < 6; q++) { free(S->psiE[q]); free(S->psiH[q]); }
    free(S->F); free(S->Jw); free(S->Cnow); free(S->Cprev);
  }
  free(R->s); free(R->freqs); free(R->wp); free(R->dft_idx); free(R->chk_idx); free(R->rst);
  for (int a = 0; a < 3; a++) { free(R->am[a]); free(R->bm[a]); free(R->ap[a]); free(R->bp[a]); }
  free(R);
  g->run = NULL;
}

/* lattice of component c (0..5 = Ex,Ey,Ez,Hx,Hy,Hz) along axis a: 1 = half nodes, 0 = nodes [R2] */
static const int LAT[6][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};

static int cmp_size(const void *a, const void *b) {
  size_t x = *(const size_t *)a, y = *(const size_t *)b;
  return x < y ? -1 : x > y;
}
static size_t uniq(size_t *v, size_t n) {
  if (!n) return 0;
  qsort(v, n, sizeof(size_t), cmp_size);
  size_t m = 1;
  for (size_t t = 1; t < n; t++) if (v[t] != v[m - 1]) v[m++] = v[t];
  return m;
}
static long find_idx(const size_t *v, size_t n, size_t key) {
  size_t lo = 0, hi = n;
  while (lo < hi) { size_t mid = (lo + hi) / 2; if (v[mid] < key) lo = mid + 1; else hi = mid; }
  return (lo < n && v[lo] == key) ? (long)lo : -1;
}

/* first derivative of a Gaussian, [R8] */
static double wavelet(const runstate *R, double t) {
  double u = t - R->t0;
  return -2.0 * R->beta * u * sqrt(R->beta / M_PI) * exp(-R->beta * u * u);
}

/* CPML coefficients, Eq. 24 (L302) with the profile of [R5].  pos = location of the derivative. */
static void cpml_tables(const emmo_grid *g, int a, double fmax, const double vref[2], double *am, double *bm, double *ap, double *bp) {
  const int N = g->N[a], nb = g->nb;
  const double Rc = 1e-3, dt = g->dt;
  const double *X = g->xn[a], *XH = g->xh[a];
  for (int ii = 0; ii < 2 * nb; ii++) { am[ii] = ap[ii] = 0; bm[ii] = bp[ii] = 1; }
  for (int side = 0; side < 2; side++) {
    if (a == 2 && side == 0 && g->top == EMMO_TOP_AIR) continue;   /* no CPML at the top (L292) */
    double x_in = side == 0 ? X[nb] : X[N - 1 - nb];
    double L = side == 0 ? X[nb] - X[0] : X[N - 1] - X[N - 1 - nb];
    double d0 = -3.0 * vref[side] * log(Rc) / (2.0 * L);
    for (int q = 0; q < nb; q++) {
      int i = side == 0 ? q : N - 1 - q;       /* mirrored index as in L324-326 */
      int ii = side == 0 ? q : nb + q;
      for (int half = 0; half < 2; half++) {
        double p = half ? XH[i] : X[i];
        double xi = side == 0 ? x_in - p : p - x_in;
        if (xi < 0) xi = 0;
        double d = d0 * (xi / L) * (xi / L);
        double al = M_PI * (fmax / 2) * (1 - xi / L); if (al < 0) al = 0;
        double b = exp(-(d + al) * dt);          /* kappa = 1 */
        double aa = d > 0 ? d / (d + al) * (b - 1) : 0.0;
        if (half) { ap[ii] = aa; bp[ii] = b; } else { am[ii] = aa; bm[ii] = b; }
      }
    }
  }
}

/* slab index of i along axis a (-1 = interior): L317-333 */
static inline int slab(const emmo_grid *g, int a, int i) {
  if (i < g->nb) return (a == 2 && g->top == EMMO_TOP_AIR) ? -1 : i;
  if (i > g->N[a] - 1 - g->nb) return g->nb + (g->N[a] - 1 - i);
  return -1;
}

static double node_width(const emmo_grid *g, int a, int lat, int i) {
  if (lat) return g->xn[a][i + 1] - g->xn[a][i];
  return g->xh[a][i] - g->xh[a][i - 1];
}

int emmo_run_begin(emmo_grid *g, const emmo_src *src, int nsrc, const double *freqs, int nf,
                   const double *rec, int nrec, const emmo_run_opts *o) {
  if (!g || !src || !freqs || !o || (nrec > 0 && !rec)) return fail(EMMO_EINVAL, "run_begin: null argument");
  if (!g->have_model) return fail(EMMO_EINVAL, "run_begin: emmo_model_set not called");
  if (nsrc < 1 || nf < 1 || nrec < 0) return fail(EMMO_EINVAL, "run_begin: bad counts");
  free_run(g);
  runstate *R = (runstate *)calloc(1, sizeof *R);
  if (!R) return fail(EMMO_ENOMEM, "run_begin: out of memory");
  g->run = R;
  const int N1 = g->N[0], N2 = g->N[1], N3 = g->N[2], r = g->r, nb = g->nb;
  const size_t N = (size_t)N1 * N2 * N3;
  R->nsrc = nsrc; R->nf = nf; R->nrec = nrec;
  R->max_steps = o->max_steps > 0 ? o->max_steps : 100000;
  R->fixed_steps = o->fixed_steps > 0 ? o->fixed_steps : 0;
  R->tol = o->tol > 0 ? o->tol : 1e-6;
  R->check_every = o->check_every > 0 ? o->check_every : 100;
  R->check_set = o->check_set; R->sparse = o->sparse_dft;
  R->dtft_every = o->dtft_every > 1 ? o->dtft_every : 1;      /* < 0: automatic, set once fmax is known */
  if (R->check_set < 0 || R->check_set > 2) { free_run(g); return fail(EMMO_EINVAL, "run_begin: bad check_set"); }
  R->freqs = (double *)malloc(sizeof(double) * nf); R->wp = (cplx *)malloc(sizeof(cplx) * nf);
  if (!R->freqs || !R->wp) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
  double fhi = 0; R->fmin = 0;
  for (int f = 0; f < nf; f++) {
    if (!(freqs[f] > 0) || !isfinite(freqs[f])) { free_run(g); return fail(EMMO_EINVAL, "run_begin: frequencies must be > 0"); }
    R->freqs[f] = freqs[f];
    R->wp[f] = (1.0 + I) * sqrt(2 * M_PI * freqs[f] * g->w0);       /* Eq. 4 */
    if (freqs[f] > fhi) fhi = freqs[f];
    if (freqs[f] < freqs[R->fmin]) R->fmin = f;
  }
  R->fmax = o->fmax > 0 ? o->fmax : 4.0 * sqrt(fhi * g->f0);        /* [R8] */
  R->beta = M_PI * R->fmax * R->fmax; R->t0 = M_PI / R->fmax;
  if (o->dtft_every < 0) {  /* largest m whose sampling rate 1/(m dt) still clears the wavelet band (3 fmax) plus the
                               band the DTFT looks at (sqrt(f f0)) twice over: aliasing below ~1e-9 */
    double m = floor(1.0 / (g->dt * (3.0 * R->fmax + 2.0 * sqrt(fhi * g->f0))));
    R->dtft_every = m > 1 ? (m > 1000 ? 1000 : (int)m) : 1;
  }
  R->np = 2 * r > 4 ? 2 * r : 4;
  /* CPML tables; v_ref per face = fastest padded cell inside that slab [R5] */
  for (int a = 0; a < 3; a++) {
    R->am[a] = (double *)malloc(sizeof(double) * 2 * nb); R->bm[a] = (double *)malloc(sizeof(double) * 2 * nb);
    R->ap[a] = (double *)malloc(sizeof(double) * 2 * nb); R->bp[a] = (double *)malloc(sizeof(double) * 2 * nb);
    if (!R->am[a] || !R->bm[a] || !R->ap[a] || !R->bp[a]) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
    double vref[2] = {0, 0};
    for (int k = 0; k < N3; k++) for (int j = 0; j < N2; j++) for (int i = 0; i < N1; i++) {
      int ia = a == 0 ? i : a == 1 ? j : k;
      int side = ia < nb ? 0 : (ia >= g->N[a] - nb ? 1 : -1);
      if (side < 0) continue;
      double s = fmin(g->sh[IDX(g, i, j, k)], g->sv[IDX(g, i, j, k)]);
      if (!(s > 0)) continue;
      double v = 1.0 / sqrt(MU0 * s / (2 * g->w0));
      if (v > vref[side]) vref[side] = v;
    }
    cpml_tables(g, a, R->fmax, vref, R->am[a], R->bm[a], R->ap[a], R->bp[a]);
  }
  /* receivers: tensor product of 1-D interpolation stencils on each component's lattice (L167-178, L640) */
  R->rst = (stencil1 *)calloc((size_t)(nrec > 0 ? nrec : 1) * 6 * 3, sizeof(stencil1));
  if (!R->rst) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
  for (int q = 0; q < nrec; q++) for (int c = 0; c < 6; c++) for (int a = 0; a < 3; a++) {
    const double *S = LAT[c][a] ? g->xh[a] : g->xn[a];
    int lo_ok = (a == 2) ? g->klo : r;
    if (rec[3 * q + a] < g->xn[a][g->lo[a]] || rec[3 * q + a] > g->xn[a][g->lo[a] + g->nc[a]] ||
        lattice_stencil(S, g->N[a], rec[3 * q + a], R->np, lo_ok, &R->rst[((size_t)q * 6 + c) * 3 + a]) ||
        R->rst[((size_t)q * 6 + c) * 3 + a].start + R->np - 1 > g->N[a] - 1 - r) {
      free_run(g); return fail(EMMO_EINVAL, "run_begin: receiver %d outside the interior", q);
    }
  }
  /* DFT set [R11]: the non-CPML box (L365-370), or receiver stencils only (sparse mode) */
  if (!R->sparse) {
    R->ndft = (size_t)(g->bhi[0] - g->blo[0] + 1) * (g->bhi[1] - g->blo[1] + 1) * (g->bhi[2] - g->blo[2] + 1);
    R->dft_idx = (size_t *)malloc(sizeof(size_t) * R->ndft);
    if (!R->dft_idx) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
    size_t p = 0;
    for (int k = g->blo[2]; k <= g->bhi[2]; k++) for (int j = g->blo[1]; j <= g->bhi[1]; j++) for (int i = g->blo[0]; i <= g->bhi[0]; i++)
      R->dft_idx[p++] = IDX(g, i, j, k);
  } else {
    size_t np3 = (size_t)R->np * R->np * R->np, cap = (size_t)nrec * 6 * np3 + 1, p = 0;
    R->dft_idx = (size_t *)malloc(sizeof(size_t) * cap);
    if (!R->dft_idx) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
    for (int q = 0; q < nrec; q++) for (int c = 0; c < 6; c++) {
      stencil1 *st = &R->rst[((size_t)q * 6 + c) * 3];
      for (int c3 = 0; c3 < R->np; c3++) for (int c2 = 0; c2 < R->np; c2++) for (int c1 = 0; c1 < R->np; c1++)
        R->dft_idx[p++] = IDX(g, st[0].start + c1, st[1].start + c2, st[2].start + c3);
    }
    R->ndft = uniq(R->dft_idx, p);
  }
  /* check set [R9] */
  {
    size_t cap = 0, p = 0;
    int b0[3] = {g->blo[0], g->blo[1], g->blo[2]}, b1[3] = {g->bhi[0], g->bhi[1], g->bhi[2]};
    if (R->check_set == EMMO_CHECK_CORNERS) cap = 8;
    else cap = (size_t)(b1[0] - b0[0] + 1) * (b1[1] - b0[1] + 1) * (b1[2] - b0[2] + 1);
    R->chk_idx = (size_t *)malloc(sizeof(size_t) * cap);
    if (!R->chk_idx) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
    for (int k = b0[2]; k <= b1[2]; k++) for (int j = b0[1]; j <= b1[1]; j++) for (int i = b0[0]; i <= b1[0]; i++) {
      int ei = (i == b0[0] || i == b1[0]), ej = (j == b0[1] || j == b1[1]), ek = (k == b0[2] || k == b1[2]);
      int take = R->check_set == EMMO_CHECK_FULL ? 1 : R->check_set == EMMO_CHECK_FACES ? (ei || ej || ek) : (ei && ej && ek);
      if (take) R->chk_idx[p++] = IDX(g, i, j, k);
    }
    R->nchk = p;
  }
  /* per-source state */
  R->s = (srcstate *)calloc(nsrc, sizeof(srcstate));
  if (!R->s) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
  for (int s = 0; s < nsrc; s++) {
    srcstate *S = &R->s[s];
    for (int c = 0; c < 3; c++) {
      S->E[c] = (double *)calloc(N, sizeof(double)); S->H[c] = (double *)calloc(N, sizeof(double));
      if (!S->E[c] || !S->H[c]) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
    }
    for (int q = 0; q < 6; q++) {
      S->psiE[q] = (double *)calloc(N, sizeof(double)); S->psiH[q] = (double *)calloc(N, sizeof(double));
      if (!S->psiE[q] || !S->psiH[q]) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
    }
    S->F = (cplx *)calloc((size_t)6 * nf * R->ndft + 1, sizeof(cplx));
    S->Jw = (cplx *)calloc(nf, sizeof(cplx));
    S->Cnow = (cplx *)calloc(6 * R->nchk + 1, sizeof(cplx)); S->Cprev = (cplx *)calloc(6 * R->nchk + 1, sizeof(cplx));
    if (!S->F || !S->Jw || !S->Cnow || !S->Cprev) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
    S->delta[0] = S->delta[1] = NAN;
    /* source weights W_c = dir_c * wx wy wz / V_node on the component's own lattice [R7] */
    double dn = sqrt(src[s].dir[0] * src[s].dir[0] + src[s].dir[1] * src[s].dir[1] + src[s].dir[2] * src[s].dir[2]);
    if (!(dn > 0) || !isfinite(dn)) { free_run(g); return fail(EMMO_EINVAL, "run_begin: source %d has zero direction", s); }
    S->magnetic = src[s].type == 1;
    if (src[s].type != 0 && src[s].type != 1) { free_run(g); return fail(EMMO_EINVAL, "run_begin: source %d has an unknown type", s); }
    for (int c = 0; c < 3; c++) {
      const int cl = c + (S->magnetic ? 3 : 0);         /* lattice of E_c or of H_c */
      S->nsn[c] = 0;
      if (src[s].dir[c] == 0.0) continue;
      stencil1 st[3];
      for (int a = 0; a < 3; a++) {
        const double *L = LAT[cl][a] ? g->xh[a] : g->xn[a];
        int lo_ok = (a == 2) ? g->klo : r;
        if (src[s].pos[a] < g->xn[a][g->lo[a]] || src[s].pos[a] > g->xn[a][g->lo[a] + g->nc[a]] ||
            lattice_stencil(L, g->N[a], src[s].pos[a], R->np, lo_ok, &st[a]) || st[a].start + R->np - 1 > g->N[a] - 1 - r) {
          free_run(g); return fail(EMMO_EINVAL, "run_begin: source %d outside the interior", s);
        }
      }
      size_t np3 = (size_t)R->np * R->np * R->np;
      S->sidx[c] = (size_t *)malloc(sizeof(size_t) * np3); S->sw[c] = (double *)malloc(sizeof(double) * np3);
      if (!S->sidx[c] || !S->sw[c]) { free_run(g); return fail(EMMO_ENOMEM, "run_begin: out of memory"); }
      int n = 0;
      for (int c3 = 0; c3 < R->np; c3++) for (int c2 = 0; c2 < R->np; c2++) for (int c1 = 0; c1 < R->np; c1++) {
        int i = st[0].start + c1, j = st[1].start + c2, k = st[2].start + c3;
        double V = node_width(g, 0, LAT[cl][0], i) * node_width(g, 1, LAT[cl][1], j) * node_width(g, 2, LAT[cl][2], k);
        S->sidx[c][n] = IDX(g, i, j, k);
        S->sw[c][n] = src[s].dir[c] / dn * st[0].w[c1] * st[1].w[c2] * st[2].w[c3] / V;
        n++;
      }
      S->nsn[c] = n;
    }
  }
  return 0;
}

/* ---- one E update: fdtd_curlH + CPML + inject_electric_src_fwd + fdtd_update_E (Alg. 1) ---- */
static void update_E(const emmo_grid *g, const runstate *R, srcstate *S, double st) {
  const int N1 = g->N[0], N2 = g->N[1], N3 = g->N[2], r = g->r, r2 = 2 * g->r;
  const size_t s1 = 1, s2 = (size_t)N1, s3 = (size_t)N1 * N2;
  const double *H1 = S->H[0], *H2 = S->H[1], *H3 = S->H[2];
  const double *c1 = g->cm[0], *c2 = g->cm[1], *c3 = g->cm[2];
#pragma omp parallel for schedule(static)
  for (int k = g->klo; k <= N3 - 1 - r; k++) {
    int sk = slab(g, 2, k);
    for (int j = r; j <= N2 - 1 - r; j++) {
      int sj = slab(g, 1, j);
      for (int i = r; i <= N1 - 1 - r; i++) {
        size_t t = IDX(g, i, j, k);
        double D2H3 = 0, D3H2 = 0, D3H1 = 0, D1H3 = 0, D1H2 = 0, D2H1 = 0;
        for (int m = 0; m < r2; m++) {                 /* Eq. 14; index pattern of L212-236 */
          ptrdiff_t o = (ptrdiff_t)m - r;
          D1H3 += c1[(size_t)i * r2 + m] * H3[t + o * (ptrdiff_t)s1];
          D1H2 += c1[(size_t)i * r2 + m] * H2[t + o * (ptrdiff_t)s1];
          D2H3 += c2[(size_t)j * r2 + m] * H3[t + o * (ptrdiff_t)s2];
          D2H1 += c2[(size_t)j * r2 + m] * H1[t + o * (ptrdiff_t)s2];
          D3H2 += c3[(size_t)k * r2 + m] * H2[t + o * (ptrdiff_t)s3];
          D3H1 += c3[(size_t)k * r2 + m] * H1[t + o * (ptrdiff_t)s3];
        }
        int si = slab(g, 0, i);                        /* Eq. 22-23; listing L317-333 */
        if (si >= 0) {
          S->psiE[0][t] = R->bm[0][si] * S->psiE[0][t] + R->am[0][si] * D1H3; D1H3 += S->psiE[0][t];
          S->psiE[1][t] = R->bm[0][si] * S->psiE[1][t] + R->am[0][si] * D1H2; D1H2 += S->psiE[1][t];
        }
        if (sj >= 0) {
          S->psiE[2][t] = R->bm[1][sj] * S->psiE[2][t] + R->am[1][sj] * D2H3; D2H3 += S->psiE[2][t];
          S->psiE[3][t] = R->bm[1][sj] * S->psiE[3][t] + R->am[1][sj] * D2H1; D2H1 += S->psiE[3][t];
        }
        if (sk >= 0) {
          S->psiE[4][t] = R->bm[2][sk] * S->psiE[4][t] + R->am[2][sk] * D3H2; D3H2 += S->psiE[4][t];
          S->psiE[5][t] = R->bm[2][sk] * S->psiE[5][t] + R->am[2][sk] * D3H1; D3H1 += S->psiE[5][t];
        }
        /* curl (L338-346) and update (Eq. 8, listing L591-593; ce = dt/eps) */
        S->E[0][t] += g->ce[0][t] * (D2H3 - D3H2);
        S->E[1][t] += g->ce[1][t] * (D3H1 - D1H3);
        S->E[2][t] += g->ce[2][t] * (D1H2 - D2H1);
      }
    }
  }
  /* source term -dt/eps * J, J = s(t) W  (Eq. 8) */
  if (!S->magnetic) for (int c = 0; c < 3; c++)
    for (int n = 0; n < S->nsn[c]; n++) S->E[c][S->sidx[c][n]] -= g->ce[c][S->sidx[c][n]] * st * S->sw[c][n];
}

/* ---- one H update: fdtd_curlE + CPML + fdtd_update_H (Alg. 1), M = 0 ---- */
static void update_H(const emmo_grid *g, const runstate *R, srcstate *S) {
  const int N1 = g->N[0], N2 = g->N[1], N3 = g->N[2], r = g->r, r2 = 2 * g->r;
  const size_t s1 = 1, s2 = (size_t)N1, s3 = (size_t)N1 * N2;
  const double *E1 = S->E[0], *E2 = S->E[1], *E3 = S->E[2];
  const double *c1 = g->cp[0], *c2 = g->cp[1], *c3 = g->cp[2];
  const double dtmu = g->dt / MU0;
#pragma omp parallel for schedule(static)
  for (int k = g->klo; k <= N3 - 1 - r; k++) {
    int sk = slab(g, 2, k);
    for (int j = r; j <= N2 - 1 - r; j++) {
      int sj = slab(g, 1, j);
      for (int i = r; i <= N1 - 1 - r; i++) {
        size_t t = IDX(g, i, j, k);
        double D2E3 = 0, D3E2 = 0, D3E1 = 0, D1E3 = 0, D1E2 = 0, D2E1 = 0;
        for (int m = 0; m < r2; m++) {                 /* Eq. 13: nodes i-r+1 .. i+r */
          ptrdiff_t o = (ptrdiff_t)m - r + 1;
          D1E3 += c1[(size_t)i * r2 + m] * E3[t + o * (ptrdiff_t)s1];
          D1E2 += c1[(size_t)i * r2 + m] * E2[t + o * (ptrdiff_t)s1];
          D2E3 += c2[(size_t)j * r2 + m] * E3[t + o * (ptrdiff_t)s2];
          D2E1 += c2[(size_t)j * r2 + m] * E1[t + o * (ptrdiff_t)s2];
          D3E2 += c3[(size_t)k * r2 + m] * E2[t + o * (ptrdiff_t)s3];
          D3E1 += c3[(size_t)k * r2 + m] * E1[t + o * (ptrdiff_t)s3];
        }
        int si = slab(g, 0, i);
        if (si >= 0) {
          S->psiH[0][t] = R->bp[0][si] * S->psiH[0][t] + R->ap[0][si] * D1E3; D1E3 += S->psiH[0][t];
          S->psiH[1][t] = R->bp[0][si] * S->psiH[1][t] + R->ap[0][si] * D1E2; D1E2 += S->psiH[1][t];
        }
        if (sj >= 0) {
          S->psiH[2][t] = R->bp[1][sj] * S->psiH[2][t] + R->ap[1][sj] * D2E3; D2E3 += S->psiH[2][t];
          S->psiH[3][t] = R->bp[1][sj] * S->psiH[3][t] + R->ap[1][sj] * D2E1; D2E1 += S->psiH[3][t];
        }
        if (sk >= 0) {
          S->psiH[4][t] = R->bp[2][sk] * S->psiH[4][t] + R->ap[2][sk] * D3E2; D3E2 += S->psiH[4][t];
          S->psiH[5][t] = R->bp[2][sk] * S->psiH[5][t] + R->ap[2][sk] * D3E1; D3E1 += S->psiH[5][t];
        }
        S->H[0][t] -= dtmu * (D2E3 - D3E2);            /* Eq. 8 */
        S->H[1][t] -= dtmu * (D3E1 - D1E3);
        S->H[2][t] -= dtmu * (D1E2 - D2E1);
      }
    }
  }
}

/* ---- air-water boundary (Eq. 17-21, [R10]) ---- */
static inline double wavenum(int n, int M, double d) { /* signed wavenumber of bin n */
  int s = n <= M / 2 ? n : n - M;
  return 2.0 * M_PI * (double)s / ((double)M * d);
}
static inline int is_nyquist(int n, int M) { return (M % 2 == 0) && n == M / 2; }

/* plane of component c at level k -> transform plane (complex) */
static void plane_to_aux(const emmo_grid *g, const double *fld, int c, int k, cplx *A) {
  const int N1 = g->N[0], M1 = g->M1, M2 = g->M2;
  if (g->uniform_xy) {
    for (int j = 0; j < M2; j++) for (int i = 0; i < M1; i++) A[(size_t)j * M1 + i] = fld[IDX(g, i, j, k)];
    return;
  }
  const stencil1 *sx = g->toaux[0][LAT[c][0]], *sy = g->toaux[1][LAT[c][1]];
#pragma omp parallel for schedule(static)
  for (int n = 0; n < M2; n++) for (int m = 0; m < M1; m++) {
    double acc = 0;
    for (int b = 0; b < 4; b++) for (int a = 0; a < 4; a++)
      acc += sy[n].w[b] * sx[m].w[a] * fld[(size_t)(sx[m].start + a) + (size_t)N1 * ((size_t)(sy[n].start + b) + (size_t)g->N[1] * (size_t)k)];
    A[(size_t)n * M1 + m] = acc;
  }
}
/* real part of the transform plane -> plane of component c at level k */
static void aux_to_plane(const emmo_grid *g, const cplx *A, double *fld, int c, int k) {
  const int N1 = g->N[0], N2 = g->N[1], M1 = g->M1;
  if (g->uniform_xy) {
    for (int j = 0; j < N2; j++) for (int i = 0; i < N1; i++) fld[IDX(g, i, j, k)] = creal(A[(size_t)j * M1 + i]);
    return;
  }
  const stencil1 *sx = g->fromaux[0][LAT[c][0]], *sy = g->fromaux[1][LAT[c][1]];
#pragma omp parallel for schedule(static)
  for (int j = 0; j < N2; j++) for (int i = 0; i < N1; i++) {
    double acc = 0;
    for (int b = 0; b < 4; b++) for (int a = 0; a < 4; a++)
      acc += sy[j].w[b] * sx[i].w[a] * creal(A[(size_t)(sy[j].start + b) * M1 + (size_t)(sx[i].start + a)]);
    fld[IDX(g, i, j, k)] = acc;
  }
}

/* Eq. 21: Laplace E = 0 above the surface => E^(kx,ky,-h) = e^{-k_h h} E^(kx,ky,0) for Ex, Ey. */
static int airwave_bc_update_E(const emmo_grid *g, srcstate *S) {
  const int M1 = g->M1, M2 = g->M2, r = g->r, k0 = g->k0;
  if (r < 2) return 0;
  size_t M = (size_t)M1 * M2;
  cplx *A = (cplx *)malloc(sizeof(cplx) * M), *B = (cplx *)malloc(sizeof(cplx) * M);
  if (!A || !B) { free(A); free(B); return -1; }
  for (int c = 0; c < 2; c++) {
    plane_to_aux(g, S->E[c], c, k0, A);
    if (fft2_inplace(A, M1, M2, -1, &g->p1, &g->p2)) { free(A); free(B); return -1; }
    for (int m = 1; m <= r - 1; m++) {
      double h = g->xn[2][k0] - g->xn[2][k0 - m];
#pragma omp parallel for schedule(static)
      for (int n2 = 0; n2 < M2; n2++) for (int n1 = 0; n1 < M1; n1++) {
        double kx = wavenum(n1, M1, g->dxa), ky = wavenum(n2, M2, g->dya), kh = sqrt(kx * kx + ky * ky);
        B[(size_t)n2 * M1 + n1] = A[(size_t)n2 * M1 + n1] * exp(-kh * h);
      }
      if (fft2_inplace(B, M1, M2, +1, &g->p1, &g->p2)) { free(A); free(B); return -1; }
      aux_to_plane(g, B, S->E[c], c, k0 - m);
    }
  }
  free(A); free(B);
  return 0;
}

/* Eq. 20: Hx = i kx/k_h Hz, Hy = i ky/k_h Hz, continued upward with e^{-k_h h}; on the uniform
 * grid the half-cell shift between the Hz lattice and the Hx / Hy lattices is a phase factor.  */
static int airwave_bc_update_H(const emmo_grid *g, srcstate *S) {
  const int M1 = g->M1, M2 = g->M2, r = g->r, k0 = g->k0;
  size_t M = (size_t)M1 * M2;
  cplx *A = (cplx *)malloc(sizeof(cplx) * M), *B = (cplx *)malloc(sizeof(cplx) * M);
  if (!A || !B) { free(A); free(B); return -1; }
  plane_to_aux(g, S->H[2], 5, k0, A);
  if (fft2_inplace(A, M1, M2, -1, &g->p1, &g->p2)) { free(A); free(B); return -1; }
  for (int m = 1; m <= r; m++) {
    double h = g->xn[2][k0] - g->xh[2][k0 - m];
    for (int comp = 0; comp < 2; comp++) {            /* 0: Hx (uses kx), 1: Hy (uses ky) */
#pragma omp parallel for schedule(static)
      for (int n2 = 0; n2 < M2; n2++) for (int n1 = 0; n1 < M1; n1++) {
        double kx = wavenum(n1, M1, g->dxa), ky = wavenum(n2, M2, g->dya), kh = sqrt(kx * kx + ky * ky);
        double ka = comp == 0 ? kx : ky, da = comp == 0 ? g->dxa : g->dya;
        int nyq = comp == 0 ? is_nyquist(n1, M1) : is_nyquist(n2, M2);
        cplx f = 0;
        if (kh > 0 && !nyq) {
          f = I * ka / kh * exp(-kh * h);
          if (g->uniform_xy) f *= cexp(-I * ka * da / 2);
        }
        B[(size_t)n2 * M1 + n1] = A[(size_t)n2 * M1 + n1] * f;
      }
      if (fft2_inplace(B, M1, M2, +1, &g->p1, &g->p2)) { free(A); free(B); return -1; }
      aux_to_plane(g, B, S->H[comp], 3 + comp, k0 - m);
    }
  }
  free(A); free(B);
  return 0;
}

/* ---- DTFT (Eq. 25, listing L361-381) with the time levels of [R6] ---- */
static void dtft_emf(const emmo_grid *g, const runstate *R, srcstate *S, int it, double st) {
  const int nf = R->nf;
  const int fields = (it % R->dtft_every) == 0;   /* decimation: fields and J' take every m-th term; the check set
                                                     (cheap) takes every term so that the stopping rule is unchanged */
  for (int f = 0; f < nf; f++) {
    cplx twH = cexp(I * R->wp[f] * ((double)it * g->dt));          /* H and J at t = it dt       */
    cplx twE = cexp(I * R->wp[f] * (((double)it + 0.5) * g->dt));  /* updated E at (it+1/2) dt   */
    /* source spectrum: J sits at t = it dt; M is centred in the H update, at (it+1/2) dt [R6] */
    if (fields) S->Jw[f] += S->magnetic ? wavelet(R, ((double)it + 0.5) * g->dt) * twE : st * twH;
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < (fields ? R->ndft : 0); p++) {
      size_t t = R->dft_idx[p];
      for (int c = 0; c < 3; c++) {
        S->F[((size_t)c * nf + f) * R->ndft + p] += S->E[c][t] * twE;
        S->F[((size_t)(3 + c) * nf + f) * R->ndft + p] += S->H[c][t] * twH;
      }
    }
    if (f == R->fmin) {
      for (size_t p = 0; p < R->nchk; p++) {
        size_t t = R->chk_idx[p];
        for (int c = 0; c < 3; c++) {
          S->Cnow[(size_t)c * R->nchk + p] += S->E[c][t] * twE;
          S->Cnow[(size_t)(3 + c) * R->nchk + p] += S->H[c][t] * twH;
        }
      }
    }
  }
}

/* ---- check_convergence (L385-387, L458, [R9]); returns 1 converged, 0 not, -1 NaN ---- */
static int check_convergence(const emmo_grid *g, const runstate *R, srcstate *S, int it) {
  double num[2] = {0, 0}, den[2] = {0, 0};
  for (int c = 0; c < 6; c++) for (size_t p = 0; p < R->nchk; p++) {
    cplx a = S->Cnow[(size_t)c * R->nchk + p], d = a - S->Cprev[(size_t)c * R->nchk + p];
    num[c / 3] += creal(d) * creal(d) + cimag(d) * cimag(d);
    den[c / 3] += creal(a) * creal(a) + cimag(a) * cimag(a);
  }
  memcpy(S->Cprev, S->Cnow, sizeof(cplx) * 6 * R->nchk);
  if (!isfinite(num[0]) || !isfinite(num[1]) || !isfinite(den[0]) || !isfinite(den[1])) return -1;
  S->delta[0] = den[0] > 0 ? sqrt(num[0] / den[0]) : NAN;
  S->delta[1] = den[1] > 0 ? sqrt(num[1] / den[1]) : NAN;
  if (R->fixed_steps) return 0;
  if (!((double)it * g->dt >= 2.0 * R->t0)) return 0;
  if (!(den[0] > 0) || !(den[1] > 0)) return 0;         /* 0/0: nothing arrived yet */
  return (S->delta[0] < R->tol && S->delta[1] < R->tol) ? 1 : 0;
}

/* Algorithm 1 lines 9-23 for n more iterations of every unfinished source. */
int emmo_run_steps(emmo_grid *g, int n, int *nsteps, int *all_done) {
  if (!g || !g->run) return fail(EMMO_EINVAL, "run_steps: no run in progress");
  runstate *R = g->run;
  int rc = 0;
  for (int s = 0; s < R->nsrc; s++) {
    srcstate *S = &R->s[s];
    for (int q = 0; q < n && !S->done; q++) {
      int it = S->nsteps;
      double st = wavelet(R, (double)it * g->dt);
      update_E(g, R, S, st);                                              /* L476-479 */
      if (g->top == EMMO_TOP_AIR && airwave_bc_update_E(g, S)) return fail(EMMO_ENOMEM, "run_steps: out of memory");
      dtft_emf(g, R, S, it, st);                                          /* L483 */
      update_H(g, R, S);                                                  /* L486-489 */
      if (g->top == EMMO_TOP_AIR && airwave_bc_update_H(g, S)) return fail(EMMO_ENOMEM, "run_steps: out of memory");
      if (S->magnetic) {                                                  /* inject_magnetic_src_fwd (L488): -dt/mu * M^{n+1/2} */
        const double sm = wavelet(R, ((double)it + 0.5) * g->dt);
        for (int c = 0; c < 3; c++)
          for (int n = 0; n < S->nsn[c]; n++) S->H[c][S->sidx[c][n]] -= g->dt / MU0 * sm * S->sw[c][n];
      }
      S->nsteps = it + 1;
      if ((it + 1) % R->check_every == 0) {                               /* L493-498, [R9] */
        int cv = check_convergence(g, R, S, it);
        if (cv < 0) { S->done = 1; rc = EMMO_ENAN; }
        else if (cv > 0) S->done = 1;
      }
      if (R->fixed_steps && S->nsteps >= R->fixed_steps) S->done = 1;
      if (!R->fixed_steps && S->nsteps >= R->max_steps && !S->done) { S->done = 1; if (!rc) rc = EMMO_ENOCONV; }
    }
  }
  int ad = 1;
  for (int s = 0; s < R->nsrc; s++) { if (nsteps) nsteps[s] = R->s[s].nsteps; if (!R->s[s].done) ad = 0; }
  if (all_done) *all_done = ad;
  if (rc == EMMO_ENAN) return fail(rc, "run_steps: non-finite field");
  if (rc == EMMO_ENOCONV) return fail(rc, "run_steps: max_steps reached before convergence");
  return 0;
}

/* compute_green_function + extract_emf (Alg. 1): Eq. 7 and receiver interpolation. */
int emmo_run_end(emmo_grid *g, double *out_, int *nsteps) {
  if (!g || !g->run) return fail(EMMO_EINVAL, "run_end: no run in progress");
  runstate *R = g->run;
  cplx *out = (cplx *)out_;
  const int nf = R->nf, np = R->np;
  for (int s = 0; s < R->nsrc; s++) {
    srcstate *S = &R->s[s];
    if (nsteps) nsteps[s] = S->nsteps;
    if (!out) continue;
    for (int f = 0; f < nf; f++) for (int q = 0; q < R->nrec; q++) for (int c = 0; c < 6; c++) {
      const stencil1 *st = &R->rst[((size_t)q * 6 + c) * 3];
      cplx acc = 0;
      for (int c3 = 0; c3 < np; c3++) for (int c2 = 0; c2 < np; c2++) for (int c1 = 0; c1 < np; c1++) {
        size_t t = IDX(g, st[0].start + c1, st[1].start + c2, st[2].start + c3);
        long p = find_idx(R->dft_idx, R->ndft, t);
        if (p < 0) return fail(EMMO_EINVAL, "run_end: receiver %d stencil leaves the DFT box", q);
        acc += st[0].w[c1] * st[1].w[c2] * st[2].w[c3] * S->F[((size_t)c * nf + f) * R->ndft + (size_t)p];
      }
      /* Eq. 4 + Eq. 7: E' = E, M' = M, H' = sq H, J' = sq J with sq = sqrt(-i w / 2 w0) (principal root):
         electric source G^EE = sq F_E/J', G^HE = F_H/J'; magnetic source G^EM = F_E/M', G^HM = F_H/(sq M') */
      cplx G = acc / S->Jw[f];
      const cplx sq = csqrt(-I * 2 * M_PI * R->freqs[f] / (2 * g->w0));
      if (!S->magnetic && c < 3) G *= sq;
      if (S->magnetic && c >= 3) G /= sq;
      out[(((size_t)s * nf + f) * R->nrec + q) * 6 + c] = G;
    }
  }
  return 0;
}

int emmo_run(emmo_grid *g, const emmo_src *src, int nsrc, const double *freqs, int nf,
             const double *rec, int nrec, const emmo_run_opts *o, double *out, int *nsteps) {
  if (!g || !src || nsrc < 1 || !o) return fail(EMMO_EINVAL, "run: bad arguments");
  int worst = 0;
  for (int s = 0; s < nsrc; s++) {          /* one source at a time (L630: sources are independent) */
    int rc = emmo_run_begin(g, src + s, 1, freqs, nf, rec, nrec, o);
    if (rc) return rc;
    int done = 0, ns = 0;
    while (!done) {
      rc = emmo_run_steps(g, g->run->check_every, &ns, &done);
      if (rc == EMMO_ENOCONV) { worst = rc; break; }
      if (rc) { free_run(g); return rc; }
    }
    rc = emmo_run_end(g, out ? out + (size_t)s * nf * nrec * 6 * 2 : NULL, &ns);
    if (nsteps) nsteps[s] = ns;
    if (rc) { free_run(g); return rc; }
    if (s + 1 < nsrc) free_run(g);
  }
  if (worst) return fail(worst, "run: max_steps reached before convergence");
  return 0;
}

int emmo_get(emmo_grid *g, int isrc, int what, int ifreq, void *host_out) {
  if (!g || !host_out) return fail(EMMO_EINVAL, "get: null argument");
  const size_t N = (size_t)g->N[0] * g->N[1] * g->N[2];
  if (what >= EMMO_GET_CE1 && what <= EMMO_GET_CE3) {
    if (!g->have_model) return fail(EMMO_EINVAL, "get: no model");
    memcpy(host_out, g->ce[what - EMMO_GET_CE1], sizeof(double) * N);
    return 0;
  }
  runstate *R = g->run;
  if (!R || isrc < 0 || isrc >= R->nsrc) return fail(EMMO_EINVAL, "get: no run state for that source");
  srcstate *S = &R->s[isrc];
  if (what >= EMMO_GET_E1 && what <= EMMO_GET_H3) {
    const double *p = what < EMMO_GET_H1 ? S->E[what] : S->H[what - EMMO_GET_H1];
    memcpy(host_out, p, sizeof(double) * N);
    return 0;
  }
  if (what >= EMMO_GET_F_E1 && what <= EMMO_GET_F_H3) {
    if (ifreq < 0 || ifreq >= R->nf) return fail(EMMO_EINVAL, "get: bad ifreq");
    int c = what - EMMO_GET_F_E1;
    cplx *o = (cplx *)host_out;
    memset(o, 0, sizeof(cplx) * N);
    for (size_t p = 0; p < R->ndft; p++) o[R->dft_idx[p]] = S->F[((size_t)c * R->nf + ifreq) * R->ndft + p];
    return 0;
  }
  if (what == EMMO_GET_CPML) {       /* read-out of the tables of cpml_tables(); ifreq carries the axis */
    if (ifreq < 0 || ifreq > 2) return fail(EMMO_EINVAL, "get: bad axis");
    double *o = (double *)host_out;
    const int n = 2 * g->nb;
    memcpy(o, R->am[ifreq], sizeof(double) * n); memcpy(o + n, R->bm[ifreq], sizeof(double) * n);
    memcpy(o + 2 * n, R->ap[ifreq], sizeof(double) * n); memcpy(o + 3 * n, R->bp[ifreq], sizeof(double) * n);
    return 0;
  }
  if (what == EMMO_GET_JW) { memcpy(host_out, S->Jw, sizeof(cplx) * R->nf); return 0; }
  if (what == EMMO_GET_DELTA) { memcpy(host_out, S->delta, sizeof(double) * 2); return 0; }
  return fail(EMMO_EINVAL, "get: unknown item %d", what);
}

/* ------------------------------------------------------------------------------------------ */
/* Sensitivity kernel, DESIGN.md [R14].  The diffusive equations (Eq. 1) read curl H - sigma E = J, so a change
 * d sigma of the medium acts on the field E like the source current d sigma * E: the datum changes by
 *   d d = integral G(receiver; x) d sigma(x) E(x) dV,  G(receiver; x) = G(x; receiver) by reciprocity.
 * On the grid sigma enters only through the effective conductivities sigma_bar_c of the E nodes (model_set, [R3]),
 * so the derivative with respect to one cell is the chain rule over the nodes whose average contains that cell;
 * the volume element of node n is the V(n) of the source injection [R7].  Plain scatter loop, node by node.     */
int emmo_sensitivity(emmo_grid *g, int isrc, int iadj, int ifreq, double *out_h_, double *out_v_) {
  if (!g || !g->run || !out_h_ || !out_v_) return fail(EMMO_EINVAL, "sensitivity: no run in progress or null output");
  runstate *R = g->run;
  if (isrc < 0 || isrc >= R->nsrc || iadj < 0 || iadj >= R->nsrc || ifreq < 0 || ifreq >= R->nf) return fail(EMMO_EINVAL, "sensitivity: bad source or frequency index");
  if (R->sparse) return fail(EMMO_EINVAL, "sensitivity: needs full-grid accumulators (sparse_dft = 0)");
  const srcstate *Sa = &R->s[isrc], *Sb = &R->s[iadj];
  if (Sa->magnetic || Sb->magnetic) return fail(EMMO_EINVAL, "sensitivity: electric sources only");
  if (R->dtft_every != 1) return fail(EMMO_EINVAL, "sensitivity: needs every term of the DTFT");
  cplx *out_h = (cplx *)out_h_, *out_v = (cplx *)out_v_;
  const int nx = g->nc[0], ny = g->nc[1], nz = g->nc[2], nf = R->nf;
  const size_t ncell = (size_t)nx * ny * nz;
  for (size_t t = 0; t < ncell; t++) { out_h[t] = 0; out_v[t] = 0; }
  const cplx sq = csqrt(-I * 2 * M_PI * R->freqs[ifreq] / (2 * g->w0));       /* Eq. 7a: G^EE = sq F_E / J' */
  const cplx ga = sq / Sa->Jw[ifreq], gb = sq / Sb->Jw[ifreq];
  const double *X[3] = {g->xn[0], g->xn[1], g->xn[2]};
  for (size_t p = 0; p < R->ndft; p++) {
    const size_t t = R->dft_idx[p];
    const int i = (int)(t % (size_t)g->N[0]), j = (int)((t / (size_t)g->N[0]) % (size_t)g->N[1]), k = (int)(t / ((size_t)g->N[0] * g->N[1]));
    const int idx[3] = {i, j, k};
    for (int c = 0; c < 3; c++) {
      const cplx P = (ga * Sa->F[((size_t)c * nf + ifreq) * R->ndft + p]) * (gb * Sb->F[((size_t)c * nf + ifreq) * R->ndft + p]);
      if (P == 0) continue;
      const double V = node_width(g, 0, LAT[c][0], i) * node_width(g, 1, LAT[c][1], j) * node_width(g, 2, LAT[c][2], k);
      /* the four cells sharing the edge of component c at this node, and their area weights: as in emmo_model_set */
      const int a1 = (c + 1) % 3, a2 = (c + 2) % 3;
      double w[4], wsum = 0; int q1[4], q2[4];
      for (int d1 = -1, n = 0; d1 <= 0; d1++) for (int d2 = -1; d2 <= 0; d2++, n++) {
        q1[n] = idx[a1] + d1 > 0 ? idx[a1] + d1 : 0;
        q2[n] = idx[a2] + d2 > 0 ? idx[a2] + d2 : 0;
        w[n] = (X[a1][q1[n] + 1] - X[a1][q1[n]]) * (X[a2][q2[n] + 1] - X[a2][q2[n]]);
      }
      /* the denominator of the average is (d0 + d1) of either transverse axis */
      {
        const int m1 = idx[a1] > 0 ? idx[a1] - 1 : 0, m2 = idx[a2] > 0 ? idx[a2] - 1 : 0;
        wsum = ((X[a1][m1 + 1] - X[a1][m1]) + (X[a1][idx[a1] + 1] - X[a1][idx[a1]])) * ((X[a2][m2 + 1] - X[a2][m2]) + (X[a2][idx[a2] + 1] - X[a2][idx[a2]]));
      }
      for (int n = 0; n < 4; n++) {
        int q[3]; q[c] = idx[c]; q[a1] = q1[n]; q[a2] = q2[n];
        int ci = q[0] - g->lo[0], cj = q[1] - g->lo[1], ck = q[2] - g->lo[2];
        if (g->top == EMMO_TOP_AIR && ck < 0) continue;                       /* air above the surface: not a model parameter */
        ci = ci < 0 ? 0 : (ci > nx - 1 ? nx - 1 : ci);                        /* padding replicates the edge cell [R1] */
        cj = cj < 0 ? 0 : (cj > ny - 1 ? ny - 1 : cj);
        ck = ck < 0 ? 0 : (ck > nz - 1 ? nz - 1 : ck);
        const size_t cell = (size_t)ci + (size_t)nx * ((size_t)cj + (size_t)ny * (size_t)ck);
        if (c == 2) out_v[cell] += w[n] / wsum * V * P; else out_h[cell] += w[n] / wsum * V * P;
      }
    }
  }
  return 0;
}
