/*
 * ctr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the EP-TV CT reconstruction hot path of
 * Tian, Jia, Yuan, Pan, Jiang, "GPU-based Low Dose CT Reconstruction via
 * Edge-preserving Total Variation Regularization",
 * following the readings O1..O10 / S1..S23 of SURVEY.md section 8(c) and S24 (restated in
 * DESIGN.md).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  It shares no code, header, table or
 * constant with paper_1009_2288_b200/csrc (the CUDA path) and neither includes
 * the other.
 *
 * Every function cites the passage it follows as PAPER.md:<line>.
 * Pins (tests/test_oracle_pins.py): P against box chords, a brute-force dense
 * matrix and analytic ellipse integrals; P^T against the dense transpose and the
 * adjoint identity; CGLS against numpy.linalg.lstsq, hand iterations and the Krylov-subspace
 * minimiser built without a CG recurrence; A2/A3 against hand-evaluated 4x4 (2D) and
 * 3x3x3 (3D, all three face axes) examples, direct numpy restatements of A3 on every face axis,
 * central differences of the energy along columns of every axis (strides, 1/ndim at 3), axis
 * permutations and invariants; sigma against a sort; Armijo against its inequality.
 * PARITY UNPINNED: A2 (orc_gradient) beyond those special cases -- it is a
 * definition, not a theorem -- and the composed orc_reconstruct result.
 *
 * Layouts: image [nz][ny][nx] (x fastest; nz = 1 for a 2D slice), sinogram
 * [nviews][nv][nu] (nv = 1 in 2D), face planes w / N0^2 [ndim][nz][ny][nx] with
 * plane A holding the face between voxel p and p+e_A at p (last index along A: 0).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int ndim, nx, ny, nz;
  double dx, dy, dz, cx, cy, cz;
  int nviews;
  double theta0, dtheta;
  const double* angles; /* optional [nviews] override, may be NULL */
  int nu, nv;
  double du, dv, u_off, v_off, dso, dsd;
  int det_type; /* 0 flat, 1 arc */
} orc_geom;

typedef struct {
  int n_outer, n_cgls, n_gd;
  double lambda, sigma_quantile, eps, armijo_t0, armijo_rho, armijo_c;
  int armijo_max, weights_mode, positivity;
  int reorth; /* S24: 1 = CGLS with re-orthogonalised gradients (default), 0 = recurrence as printed */
} orc_params;

/* ------------------------------------------------------------------ O1 geometry
 * PAPER.md:85-89 (fan beam, p_ij = intersection length), :217 (distances), App. III
 * A6 :484 (ray direction (cos(beta+theta), sin(beta+theta))).                       */
static double view_angle(const orc_geom* g, int k) {
  return g->angles ? g->angles[k] : g->theta0 + g->dtheta * (double)k;
}

void orc_ray(const orc_geom* g, int k, int b, int a, double S[3], double D[3]) {
  double th = view_angle(g, k), c = cos(th), s = sin(th);
  double t = ((double)a - (g->nu - 1) / 2.0 + g->u_off) * g->du;
  double v = ((double)b - (g->nv - 1) / 2.0 + g->v_off) * g->dv;
  S[0] = -g->dso * c; S[1] = -g->dso * s; S[2] = 0.0;
  if (g->det_type == 0) {
    D[0] = (g->dsd - g->dso) * c - t * s;
    D[1] = (g->dsd - g->dso) * s + t * c;
  } else {
    double beta = t / g->dsd;
    D[0] = S[0] + g->dsd * cos(th + beta);
    D[1] = S[1] + g->dsd * sin(th + beta);
  }
  D[2] = v;
}

/* ------------------------------------------------------------------ O2 ray tracing
 * p_ij = length of the intersection of ray i with pixel j (Siddon 1985).
 * Written as the definition: clip S->D to the image box, cut it at every interior grid
 * plane it crosses, and give each piece to the voxel that contains its midpoint.     */
typedef void (*seg_fn)(void* ctx, long voxel, double len);

static int crossings(double S, double dir, double lo, double d, int n, double amin, double amax,
                     double* out) {
  /* parameters alpha in (amin, amax) at which the ray crosses lo + i*d, i = 1..n-1, ascending */
  int cnt = 0;
  if (dir == 0.0) return 0;
  if (dir > 0.0) {
    for (int i = 1; i < n; ++i) {
      double al = (lo + i * d - S) / dir;
      if (al > amin && al < amax) out[cnt++] = al;
    }
  } else {
    for (int i = n - 1; i >= 1; --i) {
      double al = (lo + i * d - S) / dir;
      if (al > amin && al < amax) out[cnt++] = al;
    }
  }
  return cnt;
}

static void trace(const orc_geom* g, const double S[3], const double D[3], seg_fn fn, void* ctx,
                  double* scratch /* 2*(nx+ny+nz)+8 doubles */) {
  const int n[3] = {g->nx, g->ny, g->nz};
  const double d[3] = {g->dx, g->dy, g->dz};
  const double ctr[3] = {g->cx, g->cy, g->cz};
  double lo[3], hi[3], dir[3];
  double amin = 0.0, amax = 1.0;
  for (int ax = 0; ax < 3; ++ax) {
    lo[ax] = ctr[ax] - n[ax] * d[ax] / 2.0;
    hi[ax] = lo[ax] + n[ax] * d[ax];
    dir[ax] = D[ax] - S[ax];
    if (dir[ax] == 0.0) {
      if (S[ax] < lo[ax] || S[ax] >= hi[ax]) return; /* half-open cells */
    } else {
      double a1 = (lo[ax] - S[ax]) / dir[ax], a2 = (hi[ax] - S[ax]) / dir[ax];
      double en = a1 < a2 ? a1 : a2, ex = a1 < a2 ? a2 : a1;
      if (en > amin) amin = en;
      if (ex < amax) amax = ex;
    }
  }
  if (!(amin < amax)) return;
  const double len_total = sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);

  /* crossing lists per axis (each ascending), then a 3-way merge */
  double* lst[3];
  int cnt[3];
  lst[0] = scratch;
  lst[1] = lst[0] + n[0];
  lst[2] = lst[1] + n[1];
  double* al = lst[2] + n[2];
  for (int ax = 0; ax < 3; ++ax)
    cnt[ax] = crossings(S[ax], dir[ax], lo[ax], d[ax], n[ax], amin, amax, lst[ax]);
  int m = 0, p[3] = {0, 0, 0};
  al[m++] = amin;
  for (;;) {
    int best = -1;
    for (int ax = 0; ax < 3; ++ax)
      if (p[ax] < cnt[ax] && (best < 0 || lst[ax][p[ax]] < lst[best][p[best]])) best = ax;
    if (best < 0) break;
    al[m++] = lst[best][p[best]++];
  }
  al[m++] = amax;

  for (int q = 0; q + 1 < m; ++q) {
    double a0 = al[q], a1 = al[q + 1];
    double len = (a1 - a0) * len_total;
    if (!(len > 0.0)) continue;
    double am = 0.5 * (a0 + a1);
    long idx[3];
    for (int ax = 0; ax < 3; ++ax) {
      double pos = (dir[ax] == 0.0) ? S[ax] : S[ax] + am * dir[ax];
      long i = (long)floor((pos - lo[ax]) / d[ax]);
      if (i < 0) i = 0;
      if (i > n[ax] - 1) i = n[ax] - 1;
      idx[ax] = i;
    }
    fn(ctx, (idx[2] * g->ny + idx[1]) * g->nx + idx[0], len);
  }
}

static size_t scratch_len(const orc_geom* g) { return 2 * (size_t)(g->nx + g->ny + g->nz) + 8; }

typedef struct { const double* img; double acc; } fwd_ctx;
static void fwd_seg(void* c, long v, double len) { fwd_ctx* x = (fwd_ctx*)c; x->acc += len * x->img[v]; }

/* y = P f  (Eq. 1; one ray at a time) */
void orc_forward(const orc_geom* g, const double* img, double* sino) {
  const long nrays = (long)g->nviews * g->nv * g->nu;
#pragma omp parallel
  {
    double* scratch = (double*)malloc(scratch_len(g) * sizeof(double));
#pragma omp for schedule(dynamic, 64)
    for (long r = 0; r < nrays; ++r) {
      int a = (int)(r % g->nu), b = (int)((r / g->nu) % g->nv), k = (int)(r / ((long)g->nu * g->nv));
      double S[3], D[3];
      orc_ray(g, k, b, a, S, D);
      fwd_ctx c = {img, 0.0};
      trace(g, S, D, fwd_seg, &c, scratch);
      sino[r] = c.acc;
    }
    free(scratch);
  }
}

typedef struct { double* img; double y; } bwd_ctx;
static void bwd_seg(void* c, long v, double len) { bwd_ctx* x = (bwd_ctx*)c; x->img[v] += len * x->y; }

/* f = P^T y as the ray-driven SCATTER of PAPER.md:193 ("updating its pixel values along all
 * the ray lines"): the exact transpose by construction.  Views are split over threads, each
 * with a private image; the private images are added in thread order.                       */
void orc_back(const orc_geom* g, const double* sino, double* img) {
  const long nvox = (long)g->nx * g->ny * g->nz;
  int nth = 1;
#ifdef _OPENMP
  nth = omp_get_max_threads();
  if (nth > 16) nth = 16;
  if (nth > g->nviews) nth = g->nviews;
#endif
  double* priv = (double*)calloc((size_t)nth * nvox, sizeof(double));
#pragma omp parallel num_threads(nth)
  {
    int t = 0;
#ifdef _OPENMP
    t = omp_get_thread_num();
#endif
    double* mine = priv + (size_t)t * nvox;
    double* scratch = (double*)malloc(scratch_len(g) * sizeof(double));
    int k0 = (int)((long)g->nviews * t / nth), k1 = (int)((long)g->nviews * (t + 1) / nth);
    for (int k = k0; k < k1; ++k)
      for (int b = 0; b < g->nv; ++b)
        for (int a = 0; a < g->nu; ++a) {
          double S[3], D[3];
          orc_ray(g, k, b, a, S, D);
          bwd_ctx c = {mine, sino[((long)k * g->nv + b) * g->nu + a]};
          if (c.y != 0.0) trace(g, S, D, bwd_seg, &c, scratch);
        }
    free(scratch);
  }
  memset(img, 0, nvox * sizeof(double));
  for (int t = 0; t < nth; ++t) {
    const double* mine = priv + (size_t)t * nvox;
#pragma omp parallel for schedule(static)
    for (long v = 0; v < nvox; ++v) img[v] += mine[v];
  }
  free(priv);
}

/* Explicit matrix row (for the tiny brute-force tests): lengths of ray (k,b,a) in every voxel */
void orc_matrix_row(const orc_geom* g, int k, int b, int a, double* row /* [nz*ny*nx], zeroed here */) {
  const long nvox = (long)g->nx * g->ny * g->nz;
  double S[3], D[3];
  double* scratch = (double*)malloc(scratch_len(g) * sizeof(double));
  memset(row, 0, nvox * sizeof(double));
  orc_ray(g, k, b, a, S, D);
  bwd_ctx c = {row, 1.0};
  trace(g, S, D, bwd_seg, &c, scratch);
  free(scratch);
}

/* ------------------------------------------------------------------ O4 CGLS
 * PAPER.md:414-440 (Appendix I), steps 1-5, warm start u0 = f^(k), M = n_iter iterations
 * (reading S3); a zero denominator stops the iteration (reading S4).
 *
 * reorth = 0: the five steps exactly as printed.
 * reorth = 1 (reading S24, used by orc_reconstruct): the same five steps, and after each
 * g = P^T r the components of g along the earlier gradients P^T r^(0..m) are removed (modified
 * Gram-Schmidt). In exact arithmetic those components are zero -- the gradients of CG are
 * mutually orthogonal (Hestenes & Stiefel 1952, the paper's reference for CGLS) --
 * so both variants define the same iterate: the minimiser of ||P u - y|| over
 * u0 + span{(P^T P)^i P^T r0, i < M}. In floating point the printed recurrence loses that
 * orthogonality after the dominant singular direction has converged; from then on its result
 * moves by ~1e-2 relative under a 1e-14 perturbation of y (fp64, M = 15, measured: DESIGN.md S24),
 * i.e. it is not a usable reference. With the projection the result is reproducible to ~1e-11.   */
static double dot(const double* a, const double* b, long n) {
  double s = 0.0;
  for (long i = 0; i < n; ++i) s += a[i] * b[i];
  return s;
}

void orc_cgls(const orc_geom* g, const double* y, double* u /* in: x0, out: u^(M) */, int n_iter, int reorth) {
  const long nvox = (long)g->nx * g->ny * g->nz, nray = (long)g->nviews * g->nv * g->nu;
  double* r = (double*)malloc(nray * sizeof(double));
  double* q = (double*)malloc(nray * sizeof(double));
  double* s = (double*)malloc(nvox * sizeof(double));
  double* gr = (double*)malloc(nvox * sizeof(double));
  double* basis = reorth ? (double*)malloc((size_t)(n_iter + 1) * nvox * sizeof(double)) : NULL;
  int nb = 0;                                             /* normalised earlier gradients kept      */
  orc_forward(g, u, q);                                   /* r0 = y - P u0        (:420) */
  for (long i = 0; i < nray; ++i) r[i] = y[i] - q[i];
  orc_back(g, r, gr);                                     /* s0 = P^T r0          (:420) */
  memcpy(s, gr, nvox * sizeof(double));
  double gamma = dot(gr, gr, nvox);                       /* ||P^T r||^2                 */
  if (reorth && gamma > 0.0) {
    double inv = 1.0 / sqrt(gamma);
    for (long i = 0; i < nvox; ++i) basis[i] = gr[i] * inv;
    nb = 1;
  }
  for (int m = 0; m < n_iter; ++m) {
    orc_forward(g, s, q);                                 /* P s                         */
    double delta = dot(q, q, nray);
    if (gamma == 0.0 || delta == 0.0) break;              /* S4                          */
    double a = gamma / delta;                             /* step 1               (:423) */
    for (long i = 0; i < nvox; ++i) u[i] += a * s[i];     /* step 2               (:426) */
    for (long i = 0; i < nray; ++i) r[i] -= a * q[i];     /* step 3               (:429) */
    orc_back(g, r, gr);                                   /* P^T r^(m+1)                 */
    if (reorth)                                           /* S24: enforce g _|_ earlier gradients */
      for (int p = 0; p < nb; ++p) {
        const double* bp = basis + (size_t)p * nvox;
        double c = dot(bp, gr, nvox);
        for (long i = 0; i < nvox; ++i) gr[i] -= c * bp[i];
      }
    double gamma1 = dot(gr, gr, nvox);
    if (reorth && gamma1 > 0.0) {
      double inv = 1.0 / sqrt(gamma1);
      double* bp = basis + (size_t)nb * nvox;
      for (long i = 0; i < nvox; ++i) bp[i] = gr[i] * inv;
      ++nb;
    }
    double b = gamma1 / gamma;                            /* step 4               (:432) */
    for (long i = 0; i < nvox; ++i) s[i] = gr[i] + b * s[i]; /* step 5            (:435) */
    gamma = gamma1;
  }
  free(r); free(q); free(s); free(gr); free(basis);
}

/* ------------------------------------------------------------------ O5 face magnitudes
 * PAPER.md:458-461 (A3): ||f_{i+1/2,j}||_TV^2 = (f_{i+1,j}-f_{i,j})^2
 *   + 1/2 (f_{i+1/2,j+1}-f_{i+1/2,j})^2 + 1/2 (f_{i+1/2,j}-f_{i+1/2,j-1})^2,
 *   f_{i+1/2,j} = (f_{i+1,j}+f_{i,j})/2; other axes by index symmetry (S8); indices outside
 * the image are clamped (replicate border, reading S12); 3D adds the second transverse axis
 * (S22).  Raw differences in grid units, as printed.                                         */
static double at(const double* f, const int n[3], int i, int j, int k) {
  if (i < 0) i = 0; if (i > n[0] - 1) i = n[0] - 1;
  if (j < 0) j = 0; if (j > n[1] - 1) j = n[1] - 1;
  if (k < 0) k = 0; if (k > n[2] - 1) k = n[2] - 1;
  return f[((long)k * n[1] + j) * n[0] + i];
}

static double face_n0sq(const double* f, const int n[3], int ndim, int A, int i, int j, int k) {
  int p[3] = {i, j, k};
  int e[3] = {0, 0, 0};
  e[A] = 1;
  double d = at(f, n, i + e[0], j + e[1], k + e[2]) - at(f, n, i, j, k);
  double s = d * d;
  for (int T = 0; T < ndim; ++T) {
    if (T == A) continue;
    double m[3];
    for (int o = -1; o <= 1; ++o) {
      int q[3] = {p[0], p[1], p[2]};
      q[T] += o;
      m[o + 1] = 0.5 * (at(f, n, q[0] + e[0], q[1] + e[1], q[2] + e[2]) + at(f, n, q[0], q[1], q[2]));
    }
    s += 0.5 * (m[2] - m[1]) * (m[2] - m[1]) + 0.5 * (m[1] - m[0]) * (m[1] - m[0]);
  }
  return s;
}

/* N0^2 on every interior face; border faces (last index along A) hold 0 */
void orc_face_mag2(int ndim, int nx, int ny, int nz, const double* f, double* n0sq /* [ndim][nz][ny][nx] */) {
  const int n[3] = {nx, ny, nz};
  const long nvox = (long)nx * ny * nz;
  for (int A = 0; A < ndim; ++A)
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          int p[3] = {i, j, k};
          long v = ((long)k * ny + j) * nx + i;
          n0sq[A * nvox + v] = (p[A] < n[A] - 1) ? face_n0sq(f, n, ndim, A, i, j, k) : 0.0;
        }
}

/* ------------------------------------------------------------------ O6 sigma
 * sigma set "according to the histogram of the gradient magnitude" so that a
 * fixed percentage of the values lies on one side of it; readings S9/S10: the exact
 * q-quantile (k = ceil(q |S|)-th smallest) of the interior-face magnitudes N0, floored at eps. */
static int cmp_double(const void* a, const void* b) {
  double x = *(const double*)a, y = *(const double*)b;
  return (x > y) - (x < y);
}

double orc_sigma(int ndim, int nx, int ny, int nz, const double* n0sq, double q, double eps) {
  const int n[3] = {nx, ny, nz};
  const long nvox = (long)nx * ny * nz;
  long cnt = 0;
  double* S = (double*)malloc((size_t)ndim * nvox * sizeof(double));
  for (int A = 0; A < ndim; ++A)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          int p[3] = {i, j, k};
          if (p[A] < n[A] - 1) S[cnt++] = sqrt(n0sq[A * nvox + ((long)k * ny + j) * nx + i]);
        }
  if (cnt == 0) { free(S); return eps; }
  qsort(S, (size_t)cnt, sizeof(double), cmp_double);
  long kth = (long)ceil(q * (double)cnt);
  if (kth < 1) kth = 1;
  if (kth > cnt) kth = cnt;
  double sig = S[kth - 1];
  free(S);
  return sig > eps ? sig : eps;
}

/* ------------------------------------------------------------------ O7 weights
 * PAPER.md:462 (A3): omega_face = exp(-N0^2 / sigma^2); weights_mode 1 = plain TV, omega = 1
 * (PAPER.md:392).  Border faces hold 0 (they carry no flux, S12).                              */
void orc_weights(int ndim, int nx, int ny, int nz, const double* n0sq, double sigma, int mode, double* w) {
  const int n[3] = {nx, ny, nz};
  const long nvox = (long)nx * ny * nz;
  for (int A = 0; A < ndim; ++A)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          int p[3] = {i, j, k};
          long v = A * nvox + ((long)k * ny + j) * nx + i;
          if (p[A] >= n[A] - 1) w[v] = 0.0;
          else w[v] = mode == 1 ? 1.0 : exp(-n0sq[v] / (sigma * sigma));
        }
}

/* ------------------------------------------------------------------ O8 gradient
 * PAPER.md:151 Eq. 9: g = lambda (f - v) + dJ/df;  PAPER.md:453 (A2):
 * dJ/df_{i,j} ~ -[ w_{i+1/2,j}(f_{i+1,j}-f_{i,j})/||f_{i+1/2,j}||_TV
 *                 - w_{i-1/2,j}(f_{i,j}-f_{i-1,j})/||f_{i-1/2,j}||_TV ] - [same in j].
 * omega is an input (frozen, no d omega/df term: Eq. 10 :153, :372); ||.||_TV is evaluated at
 * the current f with sqrt(N0^2 + eps^2) (reading S11); border faces carry zero flux (S12).     */
void orc_gradient(int ndim, int nx, int ny, int nz, const double* f, const double* v,
                  const double* w, double lambda, double eps, double* grad) {
  const int n[3] = {nx, ny, nz};
  const long nvox = (long)nx * ny * nz;
  double* flux = (double*)malloc((size_t)ndim * nvox * sizeof(double));
  for (int A = 0; A < ndim; ++A)
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          int p[3] = {i, j, k}, e[3] = {0, 0, 0};
          e[A] = 1;
          long idx = ((long)k * ny + j) * nx + i;
          if (p[A] >= n[A] - 1) { flux[A * nvox + idx] = 0.0; continue; }
          double d = at(f, n, i + e[0], j + e[1], k + e[2]) - at(f, n, i, j, k);
          double n0 = face_n0sq(f, n, ndim, A, i, j, k);
          flux[A * nvox + idx] = w[A * nvox + idx] * d / sqrt(n0 + eps * eps);
        }
  const long stride[3] = {1, nx, (long)nx * ny};
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        int p[3] = {i, j, k};
        long idx = ((long)k * ny + j) * nx + i;
        double gv = lambda * (f[idx] - v[idx]);
        for (int A = 0; A < ndim; ++A) {
          double fp = flux[A * nvox + idx];
          double fm = p[A] > 0 ? flux[A * nvox + idx - stride[A]] : 0.0;
          gv -= fp - fm;
        }
        grad[idx] = gv;
      }
  free(flux);
}

/* ------------------------------------------------------------------ O9 energy + Armijo sweep
 * (P2) of PAPER.md:144 Eq. 8 with omega frozen: E(f) = lambda/2 ||f-v||^2 + (1/ndim) sum_faces
 * omega (sqrt(N0^2(f)+eps^2) - eps).  PAPER.md:149: inexact line search along -g by Armijo's
 * rule; constants are reading S14: t = t0 rho^k, accept the first k < armijo_max with
 * E(f - t g) <= E(f) - c t ||g||^2, otherwise leave f unchanged.                               */
double orc_energy(int ndim, int nx, int ny, int nz, const double* f, const double* v,
                  const double* w, double lambda, double eps) {
  const int n[3] = {nx, ny, nz};
  const long nvox = (long)nx * ny * nz;
  double fid = 0.0, tv = 0.0;
  for (long i = 0; i < nvox; ++i) fid += (f[i] - v[i]) * (f[i] - v[i]);
  for (int A = 0; A < ndim; ++A)
#pragma omp parallel for schedule(static) reduction(+ : tv)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          int p[3] = {i, j, k};
          if (p[A] >= n[A] - 1) continue;
          long idx = A * nvox + ((long)k * ny + j) * nx + i;
          tv += w[idx] * (sqrt(face_n0sq(f, n, ndim, A, i, j, k) + eps * eps) - eps);
        }
  return 0.5 * lambda * fid + tv / (double)ndim;
}

/* One GD sweep given frozen w.  Returns the accepted k (or -1); out[0]=E0, out[1]=G, out[2]=t */
int orc_eptv_step(int ndim, int nx, int ny, int nz, double* f, const double* v, const double* w,
                  double lambda, const orc_params* p, double* out) {
  const long nvox = (long)nx * ny * nz;
  double* g = (double*)malloc(nvox * sizeof(double));
  double* trial = (double*)malloc(nvox * sizeof(double));
  orc_gradient(ndim, nx, ny, nz, f, v, w, lambda, p->eps, g);
  double G = dot(g, g, nvox);
  double E0 = orc_energy(ndim, nx, ny, nz, f, v, w, lambda, p->eps);
  int acc = -1;
  double t = 0.0;
  for (int k = 0; k < p->armijo_max; ++k) {
    t = p->armijo_t0 * pow(p->armijo_rho, (double)k);
    for (long i = 0; i < nvox; ++i) trial[i] = f[i] - t * g[i];
    double E = orc_energy(ndim, nx, ny, nz, trial, v, w, lambda, p->eps);
    if (E <= E0 - p->armijo_c * t * G) { acc = k; break; }
  }
  if (acc >= 0) memcpy(f, trial, nvox * sizeof(double));
  if (out) { out[0] = E0; out[1] = G; out[2] = acc >= 0 ? t : 0.0; }
  free(g); free(trial);
  return acc;
}

/* weight update of one sweep: O5 -> O6 -> O7.  Returns sigma. */
double orc_update_weights(int ndim, int nx, int ny, int nz, const double* f, double q, double eps,
                          int mode, double* w) {
  const long nvox = (long)nx * ny * nz;
  double* n0 = (double*)malloc((size_t)ndim * nvox * sizeof(double));
  orc_face_mag2(ndim, nx, ny, nz, f, n0);
  double sig = orc_sigma(ndim, nx, ny, nz, n0, q, eps);
  orc_weights(ndim, nx, ny, nz, n0, sig, mode, w);
  free(n0);
  return sig;
}

/* ------------------------------------------------------------------ O10 outer loop
 * PAPER.md:159-173 (EPTV Algorithm box; readings S2, S13, S15, S16, S18): f = 0; repeat n_outer
 * times { v = CGLS(y, x0 = f, n_cgls); f = v; n_gd x (weights -> Armijo sweep); f = max(f,0) }.
 * log: per sweep [sigma, k, E0, G] (4 doubles per sweep, n_outer*n_gd sweeps), may be NULL.
 * w_out [ndim][nz][ny][nx] receives the last weights, may be NULL.                             */
void orc_reconstruct(const orc_geom* g, const double* sino, const orc_params* p, double* f,
                     double* w_out, double* log) {
  const long nvox = (long)g->nx * g->ny * g->nz;
  double* v = (double*)malloc(nvox * sizeof(double));
  double* w = (double*)malloc((size_t)g->ndim * nvox * sizeof(double));
  memset(f, 0, nvox * sizeof(double));
  memset(w, 0, (size_t)g->ndim * nvox * sizeof(double));
  for (int it = 0; it < p->n_outer; ++it) {
    orc_cgls(g, sino, f, p->n_cgls, p->reorth);           /* Step 1 (:171), S24 */
    memcpy(v, f, nvox * sizeof(double));
    for (int s = 0; s < p->n_gd; ++s) {                   /* Step 2 (:172) */
      double sig = orc_update_weights(g->ndim, g->nx, g->ny, g->nz, f, p->sigma_quantile, p->eps,
                                      p->weights_mode, w);
      double out[3];
      int k = orc_eptv_step(g->ndim, g->nx, g->ny, g->nz, f, v, w, p->lambda, p, out);
      if (log) {
        double* l = log + 4 * ((long)it * p->n_gd + s);
        l[0] = sig; l[1] = (double)k; l[2] = out[0]; l[3] = out[1];
      }
    }
    if (p->positivity)                                    /* Step 3 (:173) */
      for (long i = 0; i < nvox; ++i) if (f[i] < 0.0) f[i] = 0.0;
  }
  if (w_out) memcpy(w_out, w, (size_t)g->ndim * nvox * sizeof(double));
  free(v); free(w);
}

/* ------------------------------------------------------------------------------------------------
 * NEXT-1: the paper's own "GPU-friendly" backprojector, Eq. (11) (derivation App. III
 * :467-493), 2D only:
 *     [P^T y](u*,v*) = (du_pix dv_pix / dbeta) * sum_theta y^theta(beta*) / l(u*,v*)
 * (u*,v*) = pixel CENTRE, l = distance source -> pixel, beta* = fan angle of the line source -> pixel
 * measured from the central ray, y^theta(beta*) by LINEAR interpolation between the two nearest detector
 * units (:197, last sentence); a pixel whose beta* falls outside the outermost unit centres gets 0 from
 * that view (reading S26). ARC detector (the paper's, :217): units equally spaced in beta,
 * dbeta = du/dsd. FLAT detector (BASELINE.json's configs; not in the paper): the same formula after the
 * change of variable t = dsd tan(beta): the unit at t* subtends dbeta(beta*) = du cos^2(beta*) / dsd.
 * An approximate adjoint only: the paper reports |<f,P^T y> - <Pf,y>| below 1 % (:493).
 * ------------------------------------------------------------------------------------------------ */
void orc_back_eq11(const orc_geom* g, const double* sino /* [nviews][nu] */, double* img /* [ny][nx] */) {
  const double xlo = g->cx - g->nx * g->dx / 2.0, ylo = g->cy - g->ny * g->dy / 2.0;
  for (int j = 0; j < g->ny; ++j) {
    for (int i = 0; i < g->nx; ++i) {
      const double px = xlo + (i + 0.5) * g->dx, py = ylo + (j + 0.5) * g->dy;
      double sum = 0.0;
      for (int k = 0; k < g->nviews; ++k) {
        const double th = view_angle(g, k), c = cos(th), s = sin(th);
        const double rx = px + g->dso * c, ry = py + g->dso * s; /* pixel - source, source = -dso (c, s) */
        const double along = rx * c + ry * s, lateral = -rx * s + ry * c;
        const double l = sqrt(rx * rx + ry * ry);
        const double beta = atan2(lateral, along);
        double bstar, dbeta;
        if (g->det_type == 1) {
          bstar = beta * g->dsd / g->du + (g->nu - 1) / 2.0 - g->u_off;
          dbeta = g->du / g->dsd;
        } else {
          bstar = g->dsd * tan(beta) / g->du + (g->nu - 1) / 2.0 - g->u_off;
          dbeta = g->du * cos(beta) * cos(beta) / g->dsd;
        }
        if (!(bstar >= 0.0) || !(bstar <= (double)(g->nu - 1))) continue;
        int b0 = (int)floor(bstar);
        if (b0 > g->nu - 2) b0 = g->nu - 2;
        if (b0 < 0) b0 = 0;
        const double fr = bstar - b0;
        const double y = g->nu > 1 ? (1.0 - fr) * sino[(long)k * g->nu + b0] + fr * sino[(long)k * g->nu + b0 + 1]
                                   : sino[(long)k * g->nu];
        sum += y / (l * dbeta);
      }
      img[(long)j * g->nx + i] = g->dx * g->dy * sum;
    }
  }
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
