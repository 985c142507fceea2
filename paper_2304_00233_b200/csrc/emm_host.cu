// emm_host.cu -- host-side pre-computation of libemm_b200.so (fp64): optimal grid generator, FD and
// interpolation weights, padded grid, CPML profiles, air-boundary plan tables.  north_star item (1):
// these stay on the host; everything per time step runs in the kernels of emm_kernels.cu.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "emm_internal.h"

namespace emm {

static thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

// Solve V^T(x) a = f in place (Bjorck-Pereyra): Newton divided differences,
// then conversion to monomial coefficients.  a enters as f.
static void vandermonde_solve(std::vector<double> &a, const std::vector<double> &x) {
  const int n = (int)x.size() - 1;
  for (int k = 0; k < n; ++k)
    for (int i = n; i > k; --i) a[i] = (a[i] - a[i - 1]) / (x[i] - x[i - k - 1]);
  for (int k = n - 1; k >= 0; --k)
    for (int i = k; i < n; ++i) a[i] -= a[i + 1] * x[k];
}

// Rows 0 and 1 of [V^T]^-1 built from offsets (node - x0): feed unit vectors (Eq. 12).
void weights(const double *nodes, int npts, double x0, double *w0, double *w1) {
  std::vector<double> off(npts), a(npts);
  for (int i = 0; i < npts; ++i) off[i] = nodes[i] - x0;
  for (int j = 0; j < npts; ++j) {
    std::fill(a.begin(), a.end(), 0.0);
    a[j] = 1.0;
    vandermonde_solve(a, off);
    if (w0) w0[j] = a[0];
    if (w1) w1[j] = a[1];
  }
}

static bool smooth7(int n) {
  for (int p : {2, 3, 5, 7}) while (n % p == 0) n /= p;
  return n == 1;
}
static int next_smooth7(int n) {
  while (!smooth7(n)) ++n;
  return n;
}

static bool uniform_axis(const double *x, int n1) {
  const double d0 = x[1] - x[0];
  for (int i = 1; i + 1 < n1; ++i)
    if (std::fabs((x[i + 1] - x[i]) - d0) > 1e-9 * d0) return false;
  return true;
}

// p-point interpolation stencil around t on lattice S (c-6): last lattice point <= t is i0, points
// i0-p/2+1 .. i0+p/2.  clamp=true shifts the stencil into range and zeroes targets outside S [R10].
bool make_stencil(const double *S, int n, double t, int p, int lo_ok, int hi_ok, bool clamp, Stencil1 *st) {
  std::memset(st, 0, sizeof *st);
  if (!(t >= S[0]) || !(t <= S[n - 1])) return clamp;
  int i0 = (int)(std::upper_bound(S, S + n, t) - S) - 1;
  if (i0 > n - 2) i0 = n - 2;
  int start = i0 - p / 2 + 1;
  if (clamp) {
    start = std::max(0, std::min(start, n - p));
  } else if (start < lo_ok || start + p - 1 > hi_ok) {
    return false;
  }
  st->start = start;
  weights(S + start, p, t, st->w, nullptr);
  return true;
}

}  // namespace emm

using namespace emm;

extern "C" const char *emm_last_error(void) { return g_err; }

// Eq. 27-29: fixed-point iteration q <- (len/dx (q-1) + 1)^(1/n).
extern "C" int emm_nugrid(int n, double len, double dx, double *x_out, double *q_out) {
  if (n < 1 || !(len > 0) || !(dx > 0) || !x_out) return fail(EMM_EINVAL, "emm_nugrid: bad arguments");
  if (std::fabs(n * dx - len) < 1e-12 * len) {
    for (int i = 0; i <= n; ++i) x_out[i] = i * dx;
    if (q_out) *q_out = 1.0;
    return 0;
  }
  if (n * dx > len) return fail(EMM_EINVAL, "emm_nugrid: n*dx > len admits no ratio q > 1");
  double q = 1.1;
  for (int it = 0; it < 100000; ++it) {
    const double qn = std::pow(len * (q - 1.0) / dx + 1.0, 1.0 / n);
    const bool stop = std::fabs(qn - q) < 1e-15;
    q = qn;
    if (stop) break;
  }
  x_out[0] = 0.0;
  for (int i = 1; i <= n; ++i) x_out[i] = dx * (std::pow(q, i) - 1.0) / (q - 1.0);
  if (q_out) *q_out = q;
  return 0;
}

// acquisition geometry (L632-640), [R13]: azimuth from +x towards +y, dip from the horizontal towards +z (downward)
extern "C" int emm_dipole_direction(double azimuth, double dip, double *dir) {
  if (!dir || !std::isfinite(azimuth) || !std::isfinite(dip)) return fail(EMM_EINVAL, "emm_dipole_direction: bad arguments");
  dir[0] = std::cos(dip) * std::cos(azimuth);
  dir[1] = std::cos(dip) * std::sin(azimuth);
  dir[2] = std::sin(dip);
  return 0;
}

extern "C" int emm_receiver_channels(const double *g6, int n, const double *azimuth, const double *dip, double *chan) {
  if (n < 0 || (n > 0 && (!g6 || !azimuth || !dip || !chan))) return fail(EMM_EINVAL, "emm_receiver_channels: bad arguments");
  for (int q = 0; q < n; ++q) {
    double d[3];
    const int rc = emm_dipole_direction(azimuth[q], dip[q], d);
    if (rc) return rc;
    for (int eh = 0; eh < 2; ++eh) {
      double re = 0, im = 0;
      for (int c = 0; c < 3; ++c) {
        re += d[c] * g6[((size_t)q * 6 + 3 * eh + c) * 2];
        im += d[c] * g6[((size_t)q * 6 + 3 * eh + c) * 2 + 1];
      }
      chan[((size_t)q * 2 + eh) * 2] = re;
      chan[((size_t)q * 2 + eh) * 2 + 1] = im;
    }
  }
  return 0;
}

extern "C" int emm_fd_weights(int npts, const double *nodes, double x0, double *w_interp, double *w_deriv) {
  if (npts < 2 || npts > 16 || !nodes) return fail(EMM_EINVAL, "emm_fd_weights: bad arguments");
  weights(nodes, npts, x0, w_interp, w_deriv);
  return 0;
}

extern "C" int emm_grid_create(const double *x, int nx1, const double *y, int ny1, const double *z, int nz1,
                               const emm_grid_opts *o, emm_grid **out) {
  if (!x || !y || !z || !o || !out) return fail(EMM_EINVAL, "emm_grid_create: null argument");
  if (o->rd < 1 || o->rd > kMaxR) return fail(EMM_EINVAL, "emm_grid_create: rd must be 1, 2 or 3 (L684)");
  if (o->nb < 1) return fail(EMM_EINVAL, "emm_grid_create: nb must be >= 1");
  if (o->top != EMM_TOP_AIR && o->top != EMM_TOP_CPML) return fail(EMM_EINVAL, "emm_grid_create: bad top");
  const double *u[3] = {x, y, z};
  const int n1s[3] = {nx1, ny1, nz1};
  for (int a = 0; a < 3; ++a) {
    if (n1s[a] < 3) return fail(EMM_EINVAL, "emm_grid_create: need at least 2 cells per axis");
    for (int i = 0; i + 1 < n1s[a]; ++i)
      if (!std::isfinite(u[a][i]) || !std::isfinite(u[a][i + 1]) || !(u[a][i + 1] > u[a][i]))
        return fail(EMM_EINVAL, "emm_grid_create: axis %d coordinates must be finite and strictly increasing", a);
  }
  emm_grid *g = new (std::nothrow) emm_grid();
  if (!g) return fail(EMM_ENOMEM, "emm_grid_create: out of memory");
  g->r = o->rd;
  g->nb = o->nb;
  g->ne = o->ne < 0 ? o->rd + 5 : o->ne;                         // L686
  g->top = o->top;
  g->f0 = o->f0 > 0 ? o->f0 : 1.0;
  g->w0 = 2 * kPi * g->f0;
  g->cfl = o->cfl > 0 ? o->cfl : 0.99;                           // L260
  g->aux_dx = o->aux_dx;
  g->air_route = o->air_route;
  const int r = g->r, nbe = g->nb + g->ne;
  if (g->ne < r) { delete g; return fail(EMM_EINVAL, "emm_grid_create: ne must be >= rd (L686)"); }
  g->uniform_xy = uniform_axis(x, nx1) && uniform_axis(y, ny1);
  try {
    for (int a = 0; a < 3; ++a) {
      g->nc[a] = n1s[a] - 1;
      int lo = nbe;
      if (a == 2 && g->top == EMM_TOP_AIR) lo = r;               // [R1] r ghost planes above the surface
      int N = g->nc[a] + lo + nbe;                               // L308-311
      if (a < 2 && g->top == EMM_TOP_AIR && g->uniform_xy) N = next_smooth7(N);   // [R1]
      g->lo[a] = lo;
      g->N[a] = N;
      g->xn[a].resize(N + 1);
      g->xh[a].resize(N);
      const double dlo = u[a][1] - u[a][0], dhi = u[a][g->nc[a]] - u[a][g->nc[a] - 1];
      for (int i = 0; i <= N; ++i) {                             // [R1] edge spacing continued
        const int c = i - lo;
        g->xn[a][i] = c < 0 ? u[a][0] + c * dlo : (c > g->nc[a] ? u[a][g->nc[a]] + (c - g->nc[a]) * dhi : u[a][c]);
      }
      for (int i = 0; i < N; ++i) g->xh[a][i] = 0.5 * (g->xn[a][i] + g->xn[a][i + 1]);
      g->cm[a].assign((size_t)N * 2 * r, 0.0);
      g->cp[a].assign((size_t)N * 2 * r, 0.0);
      double dmax = 0;
      for (int i = r; i <= N - 1 - r; ++i) {
        double *m = &g->cm[a][(size_t)i * 2 * r], *p = &g->cp[a][(size_t)i * 2 * r];
        weights(&g->xh[a][i - r], 2 * r, g->xn[a][i], nullptr, m);        // Eq. 14: D- at x_i
        weights(&g->xn[a][i - r + 1], 2 * r, g->xh[a][i], nullptr, p);    // Eq. 13: D+ at x_{i+1/2}
        double sm = 0, sp = 0;
        for (int q = 0; q < 2 * r; ++q) { sm += std::fabs(m[q]); sp += std::fabs(p[q]); }
        dmax = std::max(dmax, std::max(sm, sp));                          // Eq. 16
      }
      g->Dmax[a] = dmax;
    }
    g->k0 = g->top == EMM_TOP_AIR ? r : -1;
    g->klo = r;
    for (int a = 0; a < 3; ++a) { g->blo[a] = g->nb; g->bhi[a] = g->N[a] - 1 - g->nb; }   // L365-370
    if (g->top == EMM_TOP_AIR) g->blo[2] = g->k0;
    g->P1 = (g->N[0] + 31) / 32 * 32;                            // 128-byte aligned rows
    g->XS = (2 * g->nb + 3) / 4 * 4;
    if (g->top == EMM_TOP_AIR) {
      if (g->uniform_xy) {
        g->M1 = g->N[0];
        g->M2 = g->N[1];
        g->dxa = g->xn[0][1] - g->xn[0][0];
        g->dya = g->xn[1][1] - g->xn[1][0];
      } else {
        double dmin[2];
        for (int a = 0; a < 2; ++a) {
          dmin[a] = u[a][1] - u[a][0];
          for (int i = 0; i + 1 < n1s[a]; ++i) dmin[a] = std::min(dmin[a], u[a][i + 1] - u[a][i]);
        }
        g->dxa = g->aux_dx > 0 ? g->aux_dx : dmin[0];
        g->dya = g->aux_dx > 0 ? g->aux_dx : dmin[1];
        g->M1 = next_smooth7((int)std::floor((g->xn[0][g->N[0]] - g->xn[0][0]) / g->dxa) + 2);
        g->M2 = next_smooth7((int)std::floor((g->xn[1][g->N[1]] - g->xn[1][0]) / g->dya) + 2);
        for (int a = 0; a < 2; ++a) {
          const int M = a == 0 ? g->M1 : g->M2;
          const double da = a == 0 ? g->dxa : g->dya;
          std::vector<double> xa(M);
          for (int m = 0; m < M; ++m) xa[m] = g->xn[a][0] + m * da;
          for (int l = 0; l < 2; ++l) {
            const double *S = l ? g->xh[a].data() : g->xn[a].data();
            g->toaux[a][l].resize(M);
            g->fromaux[a][l].resize(g->N[a]);
            for (int m = 0; m < M; ++m) make_stencil(S, g->N[a], xa[m], 4, 0, 0, true, &g->toaux[a][l][m]);
            for (int i = 0; i < g->N[a]; ++i) make_stencil(xa.data(), M, S[i], 4, 0, 0, true, &g->fromaux[a][l][i]);
          }
        }
      }
    }
  } catch (const std::bad_alloc &) {
    delete g;
    return fail(EMM_ENOMEM, "emm_grid_create: out of memory");
  }
  *out = g;
  return 0;
}

extern "C" int emm_grid_info(const emm_grid *g, int *ints, double *dt) {
  if (!g) return fail(EMM_EINVAL, "emm_grid_info: null grid");
  if (ints) {
    for (int a = 0; a < 3; ++a) {
      ints[EMM_I_N1 + a] = g->N[a];
      ints[EMM_I_LO1 + a] = g->lo[a];
      ints[EMM_I_BOX_LO1 + a] = g->blo[a];
      ints[EMM_I_BOX_HI1 + a] = g->bhi[a];
    }
    ints[EMM_I_K0] = g->k0;
    ints[EMM_I_UNIFORM_XY] = g->uniform_xy;
    ints[EMM_I_AUX_M1] = g->M1;
    ints[EMM_I_AUX_M2] = g->M2;
    ints[EMM_I_PITCH] = g->P1;
  }
  if (dt) *dt = g->have_model ? g->dt : 0.0;
  return 0;
}

extern "C" int emm_grid_coords(const emm_grid *g, int axis, double *nodes_out) {
  if (!g || axis < 0 || axis > 2 || !nodes_out) return fail(EMM_EINVAL, "emm_grid_coords: bad arguments");
  std::copy(g->xn[axis].begin(), g->xn[axis].end(), nodes_out);
  return 0;
}

extern "C" int emm_grid_fdcoef(const emm_grid *g, int axis, int plus, double *out) {
  if (!g || axis < 0 || axis > 2 || !out) return fail(EMM_EINVAL, "emm_grid_fdcoef: bad arguments");
  const std::vector<double> &t = plus ? g->cp[axis] : g->cm[axis];
  std::copy(t.begin(), t.end(), out);
  return 0;
}

extern "C" long long emm_launch_count(const emm_grid *g) { return g ? g->launches : 0; }
