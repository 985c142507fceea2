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

// Interpolation (derivative order 0) and first-derivative weights of arbitrary nodes for the point x0 (Eq. 9-12).
// The paper inverts the transposed Vandermonde matrix of the offsets (L127-146); the rows of that inverse are the
// Taylor-matched weights, which Fornberg's recursion (Math. Comp. 51, 1988) builds directly, one node at a time, from
// the Lagrange form -- a different construction of the same numbers (the oracle follows the paper's listing; a CPU
// test holds the two against each other).  C[j][k] = weight of node j for derivative order k.
void weights(const double *nodes, int npts, double x0, double *w0, double *w1) {
  double C[16][2];
  for (int j = 0; j < npts; ++j) C[j][0] = C[j][1] = 0.0;
  C[0][0] = 1.0;
  double prod_prev = 1.0, off_new = nodes[0] - x0;
  for (int i = 1; i < npts; ++i) {
    const double off_prev = off_new;
    off_new = nodes[i] - x0;
    double prod = 1.0;
    for (int j = 0; j < i; ++j) {
      const double gap = nodes[i] - nodes[j];
      prod *= gap;
      if (j == i - 1) {                       // weights of the node that has just joined
        C[i][1] = prod_prev * (C[i - 1][0] - off_prev * C[i - 1][1]) / prod;
        C[i][0] = -prod_prev * off_prev * C[i - 1][0] / prod;
      }
      C[j][1] = (off_new * C[j][1] - C[j][0]) / gap;
      C[j][0] = off_new * C[j][0] / gap;
    }
    prod_prev = prod;
  }
  for (int j = 0; j < npts; ++j) {
    if (w0) w0[j] = C[j][0];
    if (w1) w1[j] = C[j][1];
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

namespace {

struct AxisInput { const double *node; int ncell; };

// [R1] One padded axis: `below` / `above` extra cells that continue the first / last spacing of the model, the half
// nodes of [R2] (cell midpoints), and the two operator tables of Eq. 13-14 for every node that is ever updated.
// Returns the largest absolute row sum of either operator (the D_max of Eq. 16).
double pad_axis_and_tabulate(emm_grid *g, int a, const AxisInput &in, int below, int above, int r) {
  const int N = in.ncell + below + above;
  g->lo[a] = below;
  g->N[a] = N;
  std::vector<double> &xn = g->xn[a], &xh = g->xh[a];
  xn.assign(N + 1, 0.0);
  xh.assign(N, 0.0);
  const double first = in.node[1] - in.node[0], last = in.node[in.ncell] - in.node[in.ncell - 1];
  for (int i = 0; i < below; ++i) xn[i] = in.node[0] - (below - i) * first;
  for (int c = 0; c <= in.ncell; ++c) xn[below + c] = in.node[c];
  for (int i = 1; i <= above; ++i) xn[below + in.ncell + i] = in.node[in.ncell] + i * last;
  for (int i = 0; i < N; ++i) xh[i] = xn[i] + 0.5 * (xn[i + 1] - xn[i]);
  const int taps = 2 * r;
  g->cm[a].assign((size_t)N * taps, 0.0);
  g->cp[a].assign((size_t)N * taps, 0.0);
  double worst = 0.0;
  for (int i = r; i + r < N; ++i) {
    // D- lives on the node x_i and reads the half nodes i-r .. i+r-1 (L212-236); D+ lives on the half node and reads the
    // nodes i-r+1 .. i+r (Eq. 13)
    double *minus = &g->cm[a][(size_t)i * taps], *plus = &g->cp[a][(size_t)i * taps];
    weights(&xh[i - r], taps, xn[i], nullptr, minus);
    weights(&xn[i - r + 1], taps, xh[i], nullptr, plus);
    double sum_minus = 0.0, sum_plus = 0.0;
    for (int q = 0; q < taps; ++q) { sum_minus += std::fabs(minus[q]); sum_plus += std::fabs(plus[q]); }
    worst = std::max(worst, std::max(sum_minus, sum_plus));
  }
  return worst;
}

// [R10] auxiliary uniform plane of a non-uniform horizontal axis: spacing d from the first padded node, enough nodes to
// reach past the last one, count rounded up to a 7-smooth transform length; 4-point Lagrange stencils in both
// directions for the node lattice (l = 0) and the half-node lattice (l = 1)
int plan_aux_axis(emm_grid *g, int a, double d) {
  const double extent = g->xn[a][g->N[a]] - g->xn[a][0];
  const int M = next_smooth7((int)std::floor(extent / d) + 2);
  std::vector<double> aux(M);
  for (int m = 0; m < M; ++m) aux[m] = g->xn[a][0] + m * d;
  for (int l = 0; l < 2; ++l) {
    const double *lattice = l ? g->xh[a].data() : g->xn[a].data();
    g->toaux[a][l].resize(M);
    g->fromaux[a][l].resize(g->N[a]);
    for (int m = 0; m < M; ++m) make_stencil(lattice, g->N[a], aux[m], 4, 0, 0, true, &g->toaux[a][l][m]);
    for (int i = 0; i < g->N[a]; ++i) make_stencil(aux.data(), M, lattice[i], 4, 0, 0, true, &g->fromaux[a][l][i]);
  }
  return M;
}

}  // namespace

extern "C" int emm_grid_create(const double *x, int nx1, const double *y, int ny1, const double *z, int nz1,
                               const emm_grid_opts *o, emm_grid **out) {
  if (!x || !y || !z || !o || !out) return fail(EMM_EINVAL, "emm_grid_create: null argument");
  if (o->rd < 1 || o->rd > kMaxR) return fail(EMM_EINVAL, "emm_grid_create: rd must be 1, 2 or 3 (L684)");
  if (o->nb < 1) return fail(EMM_EINVAL, "emm_grid_create: nb must be >= 1");
  if (o->top != EMM_TOP_AIR && o->top != EMM_TOP_CPML) return fail(EMM_EINVAL, "emm_grid_create: bad top");
  const AxisInput in[3] = {{x, nx1 - 1}, {y, ny1 - 1}, {z, nz1 - 1}};
  for (int a = 0; a < 3; ++a) {
    if (in[a].ncell < 2) return fail(EMM_EINVAL, "emm_grid_create: need at least 2 cells per axis");
    for (int i = 0; i <= in[a].ncell; ++i)
      if (!std::isfinite(in[a].node[i]) || (i > 0 && !(in[a].node[i] > in[a].node[i - 1])))
        return fail(EMM_EINVAL, "emm_grid_create: axis %d coordinates must be finite and strictly increasing", a);
  }
  const int r = o->rd;
  const int ne = o->ne < 0 ? r + 5 : o->ne;                       // L686
  if (ne < r) return fail(EMM_EINVAL, "emm_grid_create: ne must be >= rd (L686)");
  emm_grid *g = new (std::nothrow) emm_grid();
  if (!g) return fail(EMM_ENOMEM, "emm_grid_create: out of memory");
  g->r = r;
  g->nb = o->nb;
  g->ne = ne;
  g->top = o->top;
  g->f0 = o->f0 > 0 ? o->f0 : 1.0;
  g->w0 = 2 * kPi * g->f0;
  g->cfl = o->cfl > 0 ? o->cfl : 0.99;                           // L260
  g->aux_dx = o->aux_dx;
  g->air_route = o->air_route;
  const bool air = g->top == EMM_TOP_AIR;
  g->uniform_xy = uniform_axis(x, nx1) && uniform_axis(y, ny1);
  try {
    const int pad = g->nb + ne;                                   // L308-311: CPML + buffer cells on a padded side
    for (int a = 0; a < 3; ++a) {
      g->nc[a] = in[a].ncell;
      // [R1]: the surface side of z carries no CPML (L292), only the r ghost planes the stencils reach; on a uniform x-y
      // grid with the air boundary the high side takes extra buffer cells up to a 7-smooth plane size
      const int below = (a == 2 && air) ? r : pad;
      int above = pad;
      if (a < 2 && air && g->uniform_xy) above += next_smooth7(in[a].ncell + below + pad) - (in[a].ncell + below + pad);
      g->Dmax[a] = pad_axis_and_tabulate(g, a, in[a], below, above, r);
    }
    g->klo = r;                                                   // first updated plane; the r planes above are ghosts / the wall
    g->k0 = air ? r : -1;
    for (int a = 0; a < 3; ++a) {                                 // [R11]: DTFT box = everything but the CPML cells
      g->blo[a] = (a == 2 && air) ? g->k0 : g->nb;
      g->bhi[a] = g->N[a] - 1 - g->nb;
    }
    g->P1 = (g->N[0] + 31) / 32 * 32;                            // 128-byte aligned rows
    // node indices inside one source's padded volume are 32-bit on the device (source, receiver and check-set lists)
    if ((long long)g->P1 * g->N[1] * g->N[2] > 2147483647LL) {
      const int rc = fail(EMM_EINVAL, "emm_grid_create: padded grid of %d x %d x %d nodes exceeds 2^31 - 1 entries", g->N[0], g->N[1], g->N[2]);
      delete g;
      return rc;
    }
    g->XS = (2 * g->nb + 3) / 4 * 4;
    if (air && g->uniform_xy) {                                   // the FFT plane is the padded plane itself
      g->M1 = g->N[0];
      g->M2 = g->N[1];
      g->dxa = g->xn[0][1] - g->xn[0][0];
      g->dya = g->xn[1][1] - g->xn[1][0];
    } else if (air) {
      double finest[2];
      for (int a = 0; a < 2; ++a) {
        finest[a] = in[a].node[1] - in[a].node[0];
        for (int c = 1; c < in[a].ncell; ++c) finest[a] = std::min(finest[a], in[a].node[c + 1] - in[a].node[c]);
      }
      g->dxa = g->aux_dx > 0 ? g->aux_dx : finest[0];
      g->dya = g->aux_dx > 0 ? g->aux_dx : finest[1];
      g->M1 = plan_aux_axis(g, 0, g->dxa);
      g->M2 = plan_aux_axis(g, 1, g->dya);
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
    ints[EMM_I_AIR_CLUSTER] = g->air_cluster;
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
