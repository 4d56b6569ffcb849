/*
 * osiv_oracle.c -- float64 CPU ORACLE for the ordered-subset TV statistical iteration
 * of arxiv 1903.10088 ("Fast Statistical Iterative Reconstruction for MVCT in TomoTherapy").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or constant with the CUDA path under paper_1903_10088_b200/csrc/.
 *
 * It is deliberately plain and slow: every step follows the paper (PAPER.md line numbers
 * below) in the paper's order; where the paper is silent the reading of SURVEY.md section 8(c)
 * (C1..C12) is taken and restated in DESIGN.md.  The only concession to run time is
 * "#pragma omp parallel for" on outermost loops over independent rays / pixels; no blocking,
 * fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   chord weight      : brute-force polygon clipping written independently in the test  (P1)
 *   forward           : A*1 = chord of the ray in the whole grid square; analytic ellipse
 *                       line integrals; rotation / mirror symmetries                     (P2,P3,P5)
 *   forward/back pair : <Ax,y> = <x,A^T y> to 1e-12 (ray loop vs. pixel gather), and both
 *                       against the all-pairs brute force                               (P4)
 *   TV gradient       : central finite differences of TV_eps, sum of gradient = 0       (P6)
 *   likelihood grad.  : finite differences of L/b_ref                                   (P7)
 *   step scale tau    : power iteration ||A_S^T A_S|| / L_geo in (0.9, 1.0)              (P8)
 *   whole loop        : noise-free, beta=0 convergence to the true image; step-rule
 *                       behaviour of PAPER.md:140                                        (P9,P10)
 *   final image on NOISY data vs. truth: PARITY UNPINNED (depends on the noise realisation;
 *                       only sanity-checked), as stated in DESIGN.md.
 *
 * Units: lengths mm, attenuation 1/mm, angles rad.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t nx, ny;          /* image size; pixel (ix,iy) centre = ((ix-(nx-1)/2)*pixel, (iy-(ny-1)/2)*pixel) */
    double  pixel_mm;
    int32_t n_views, n_channels;
    double  sad_mm;          /* source-to-isocentre distance */
    double  dgamma_rad;      /* channel pitch; <=0 -> 2*asin(R_FOV/SAD)/C, R_FOV = min(nx,ny)*pixel/2  (C1) */
    double  channel_offset;  /* gamma_c = (c-(C-1)/2+off)*dgamma */
    double  theta0_rad;      /* theta_v = theta0 + 2*pi*v/V */
    int32_t model;           /* system matrix: 0 = exact chord length (C2); 1 = Joseph's interpolating model */
    int32_t _pad;
} oracle_geometry;

typedef struct {
    double  beta;            /* TV weight (C7) */
    int32_t n_subsets, n_iters;
    double  mu0;             /* homogeneous initial image */
    double  lambda0, lambda_up, lambda_down, lambda_min;   /* PAPER.md:100-108 Eq.4-5 (+floor, C10) */
    double  kappa;           /* step scale (C6) */
    double  tv_eps;          /* TV smoothing (C9) */
    int32_t return_best;
    int32_t monitor_mode;    /* which earlier D Eq. 4-5 compare D(n) with: 0 = D(n-1), the previous iteration (C10);
                                1 = D(n-M), the same subset one pass earlier (reading G3; lambda(n) = lambda0 for n < M) */
    const double* forced_lambda;   /* NULL or n_iters values replayed instead of Eq. 4-5 */
} oracle_params;

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- C1 geometry (the paper gives no geometry, BASELINE.json supplies it) ---- */

double oracle_dgamma(const oracle_geometry* g) {
    if (g->dgamma_rad > 0.0) return g->dgamma_rad;
    int nmin = g->nx < g->ny ? g->nx : g->ny;
    double rfov = 0.5 * nmin * g->pixel_mm;
    return 2.0 * asin(rfov / g->sad_mm) / g->n_channels;
}

static double view_angle(const oracle_geometry* g, int v) {
    return g->theta0_rad + 2.0 * M_PI * (double)v / (double)g->n_views;
}

static double channel_angle(const oracle_geometry* g, int c) {
    return ((double)c - 0.5 * (g->n_channels - 1) + g->channel_offset) * oracle_dgamma(g);
}

/* ray (v,c): from the source s = SAD(cos th, sin th) in direction d = -(cos(th+ga), sin(th+ga)) */
void oracle_ray(const oracle_geometry* g, int v, int c, double* sx, double* sy, double* dx, double* dy) {
    double th = view_angle(g, v), ga = channel_angle(g, c);
    *sx = g->sad_mm * cos(th);
    *sy = g->sad_mm * sin(th);
    *dx = -cos(th + ga);
    *dy = -sin(th + ga);
}

static double pix_x(const oracle_geometry* g, int ix) { return ((double)ix - 0.5 * (g->nx - 1)) * g->pixel_mm; }
static double pix_y(const oracle_geometry* g, int iy) { return ((double)iy - 0.5 * (g->ny - 1)) * g->pixel_mm; }

/* ---- C2 system matrix: exact length of a zero-width ray inside a square pixel ----
 * closed form in the perpendicular distance p of the pixel centre from the ray:
 * trapezoid of full half-width hi=(u+w)/2, flat half-width lo=|u-w|/2, height h=D/max(|dx|,|dy|),
 * u=|dx|D, w=|dy|D. */
static double chord_closed_form(double dx, double dy, double delta, double p) {
    double adx = fabs(dx), ady = fabs(dy), ap = fabs(p);
    double u = adx * delta, w = ady * delta;
    double hi = 0.5 * (u + w), lo = 0.5 * fabs(u - w);
    double h = delta / (adx > ady ? adx : ady);
    if (ap <= lo) return h;
    if (ap < hi)  return h * (hi - ap) / (hi - lo);
    return 0.0;
}

/* ---- second system matrix: Joseph's model.  The ray is sampled once on every image line of its
 * major axis (rows if |dy| >= |dx|, else columns), at the line's centre; the sample is the linear interpolation of
 * the line's two pixels next to the crossing, times the path length per line h = D/max(|dx|,|dy|).  As a function of
 * the perpendicular distance p of a pixel centre from the ray: the in-line distance between the centre and the
 * crossing is |p|/max(|dx|,|dy|), so a = h * max(0, 1 - |p| / (D*max(|dx|,|dy|))). ---- */
static double joseph_closed_form(double dx, double dy, double delta, double p) {
    double m = fabs(dx) > fabs(dy) ? fabs(dx) : fabs(dy);
    double t = 1.0 - fabs(p) / (delta * m);
    return t > 0.0 ? (delta / m) * t : 0.0;
}

static double weight_closed_form(int model, double dx, double dy, double delta, double p) {
    return model == 1 ? joseph_closed_form(dx, dy, delta, p) : chord_closed_form(dx, dy, delta, p);
}

/* a(i,r) for ray i=(v,c), pixel r=(ix,iy) */
double oracle_weight(const oracle_geometry* g, int v, int c, int ix, int iy) {
    double sx, sy, dx, dy;
    oracle_ray(g, v, c, &sx, &sy, &dx, &dy);
    double px = pix_x(g, ix), py = pix_y(g, iy);
    double p = (px - sx) * dy - (py - sy) * dx;      /* signed distance of the pixel centre from the ray */
    return weight_closed_form(g->model, dx, dy, g->pixel_mm, p);
}

static int subset_views(const oracle_geometry* g, int subset, int n_subsets) {
    return subset < 0 ? g->n_views : g->n_views / n_subsets;
}
static int subset_view(int j, int subset, int n_subsets) {
    return subset < 0 ? j : subset + j * n_subsets;       /* C11: S_m = {v : v mod M = m} */
}

/* ray geometry of one view subset, evaluated once per call with exactly oracle_ray()'s expressions
 * (a cache of C1, nothing more: the trigonometric calls would otherwise dominate the run time) */
typedef struct { int nv, C; double *sx, *sy, *dx, *dy; } ray_table;

static ray_table ray_table_make(const oracle_geometry* g, int subset, int n_subsets) {
    ray_table t;
    t.nv = subset_views(g, subset, n_subsets); t.C = g->n_channels;
    t.sx = (double*)malloc(sizeof(double) * t.nv);
    t.sy = (double*)malloc(sizeof(double) * t.nv);
    t.dx = (double*)malloc(sizeof(double) * (size_t)t.nv * t.C);
    t.dy = (double*)malloc(sizeof(double) * (size_t)t.nv * t.C);
    for (int j = 0; j < t.nv; ++j)
        for (int c = 0; c < t.C; ++c)
            oracle_ray(g, subset_view(j, subset, n_subsets), c, &t.sx[j], &t.sy[j],
                       &t.dx[(size_t)j * t.C + c], &t.dy[(size_t)j * t.C + c]);
    return t;
}
static void ray_table_free(ray_table* t) { free(t->sx); free(t->sy); free(t->dx); free(t->dy); }

/* ---- C3 forward: l_i = sum_r a(i,r) mu_r, ray loop.  sino is compact [V_S][C]. ---- */
void oracle_forward(const oracle_geometry* g, const double* img, double* sino, int subset, int n_subsets) {
    ray_table t = ray_table_make(g, subset, n_subsets);
    const int nv = t.nv, C = t.C;
    const double delta = g->pixel_mm;
    const double xleft = -0.5 * g->nx * delta, ybot = -0.5 * g->ny * delta;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < nv * C; ++k) {
        int j = k / C;
        double sx = t.sx[j], sy = t.sy[j], dx = t.dx[k], dy = t.dy[k];
        double sum = 0.0;
        if (fabs(dy) >= fabs(dx)) {
            /* the ray crosses every pixel row once; inside a row strip it deviates at most D/2 in x
             * from its position at the row centre, so it can only touch pixels ixc-1..ixc+1 (Joseph: the two pixel
             * centres next to the crossing at the row centre are among these three) */
            for (int iy = 0; iy < g->ny; ++iy) {
                double y = pix_y(g, iy);
                double x = sx + (y - sy) / dy * dx;
                int ixc = (int)floor((x - xleft) / delta);
                for (int ix = ixc - 1; ix <= ixc + 1; ++ix) {
                    if (ix < 0 || ix >= g->nx) continue;
                    double p = (pix_x(g, ix) - sx) * dy - (y - sy) * dx;
                    sum += weight_closed_form(g->model, dx, dy, delta, p) * img[(size_t)iy * g->nx + ix];
                }
            }
        } else {
            for (int ix = 0; ix < g->nx; ++ix) {
                double x = pix_x(g, ix);
                double y = sy + (x - sx) / dx * dy;
                int iyc = (int)floor((y - ybot) / delta);
                for (int iy = iyc - 1; iy <= iyc + 1; ++iy) {
                    if (iy < 0 || iy >= g->ny) continue;
                    double p = (x - sx) * dy - (pix_y(g, iy) - sy) * dx;
                    sum += weight_closed_form(g->model, dx, dy, delta, p) * img[(size_t)iy * g->nx + ix];
                }
            }
        }
        sino[k] = sum;
    }
    ray_table_free(&t);
}

/* all-pairs forward: every ray against every pixel (tiny inputs only) */
void oracle_forward_brute(const oracle_geometry* g, const double* img, double* sino, int subset, int n_subsets) {
    const int nv = subset_views(g, subset, n_subsets), C = g->n_channels;
    for (int k = 0; k < nv * C; ++k) {
        int j = k / C, c = k % C, v = subset_view(j, subset, n_subsets);
        double sum = 0.0;
        for (int iy = 0; iy < g->ny; ++iy)
            for (int ix = 0; ix < g->nx; ++ix)
                sum += oracle_weight(g, v, c, ix, iy) * img[(size_t)iy * g->nx + ix];
        sino[k] = sum;
    }
}

/* candidate half-range K of C3: a pixel (half-diagonal D/sqrt2) can only be touched by channels within
 * K of the channel coordinate of its centre; ray spacing at the pixel is >= (SAD-R_max)*dgamma */
int oracle_candidate_K(const oracle_geometry* g) {
    double rmax = 0.5 * g->pixel_mm * sqrt((double)g->nx * g->nx + (double)g->ny * g->ny);
    double spacing = (g->sad_mm - rmax) * oracle_dgamma(g);
    /* Joseph: a pixel is touched by rays within D*max(|dx|,|dy|) <= D of its centre */
    double reach = g->model == 1 ? g->pixel_mm : g->pixel_mm / sqrt(2.0);
    return (int)ceil(reach / spacing) + 1;
}

/* ---- C3 back: g_r = sum_{i in S} a(i,r) r_i, gather per pixel ---- */
void oracle_backward(const oracle_geometry* g, const double* sino, double* img, int subset, int n_subsets) {
    ray_table t = ray_table_make(g, subset, n_subsets);
    const int nv = t.nv, C = t.C;
    const double dgam = oracle_dgamma(g);
    const int K = oracle_candidate_K(g);
    #pragma omp parallel for schedule(dynamic, 64)
    for (int r = 0; r < g->nx * g->ny; ++r) {
        int iy = r / g->nx, ix = r % g->nx;
        double px = pix_x(g, ix), py = pix_y(g, iy);
        double sum = 0.0;
        for (int j = 0; j < nv; ++j) {
            double th = view_angle(g, subset_view(j, subset, n_subsets));
            double sx = t.sx[j], sy = t.sy[j];
            /* the ray through the pixel centre has th+gamma = direction of (s - P) */
            double gam = atan2(sy - py, sx - px) - th;
            gam = remainder(gam, 2.0 * M_PI);                        /* wrap to [-pi, pi] */
            double cstar = gam / dgam + 0.5 * (C - 1) - g->channel_offset;
            int c0 = (int)floor(cstar);
            for (int c = c0 - K; c <= c0 + K + 1; ++c) {
                if (c < 0 || c >= C) continue;
                double dx = t.dx[(size_t)j * C + c], dy = t.dy[(size_t)j * C + c];
                double p = (px - sx) * dy - (py - sy) * dx;
                sum += weight_closed_form(g->model, dx, dy, g->pixel_mm, p) * sino[(size_t)j * C + c];
            }
        }
        img[r] = sum;
    }
    ray_table_free(&t);
}

void oracle_backward_brute(const oracle_geometry* g, const double* sino, double* img, int subset, int n_subsets) {
    const int nv = subset_views(g, subset, n_subsets), C = g->n_channels;
    for (int iy = 0; iy < g->ny; ++iy)
        for (int ix = 0; ix < g->nx; ++ix) {
            double sum = 0.0;
            for (int j = 0; j < nv; ++j)
                for (int c = 0; c < C; ++c)
                    sum += oracle_weight(g, subset_view(j, subset, n_subsets), c, ix, iy) * sino[(size_t)j * C + c];
            img[(size_t)iy * g->nx + ix] = sum;
        }
}

/* ---- C8 total variation: isotropic, forward differences, replicate border, smoothed by eps ---- */
static double tv_cell(const double* mu, int nx, int ny, int x, int y, double eps) {
    double c = mu[(size_t)y * nx + x];
    double dxv = (x + 1 < nx) ? mu[(size_t)y * nx + x + 1] - c : 0.0;
    double dyv = (y + 1 < ny) ? mu[(size_t)(y + 1) * nx + x] - c : 0.0;
    return sqrt(eps * eps + dxv * dxv + dyv * dyv);
}

double oracle_tv_value(const double* mu, int nx, int ny, double eps) {
    double s = 0.0;
    for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) s += tv_cell(mu, nx, ny, x, y, eps);
    return s;
}

/* dTV/dmu_{x,y} = (mu-mu_{x-1,y})/t_{x-1,y} + (mu-mu_{x,y-1})/t_{x,y-1} - (mu_{x+1,y}+mu_{x,y+1}-2mu)/t_{x,y},
 * out-of-range terms dropped (C8) */
void oracle_tv_grad(const double* mu, double* grad, int nx, int ny, double eps) {
    #pragma omp parallel for
    for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
            double c = mu[(size_t)y * nx + x], s = 0.0;
            if (x > 0) s += (c - mu[(size_t)y * nx + x - 1]) / tv_cell(mu, nx, ny, x - 1, y, eps);
            if (y > 0) s += (c - mu[(size_t)(y - 1) * nx + x]) / tv_cell(mu, nx, ny, x, y - 1, eps);
            double dxv = (x + 1 < nx) ? mu[(size_t)y * nx + x + 1] - c : 0.0;
            double dyv = (y + 1 < ny) ? mu[(size_t)(y + 1) * nx + x] - c : 0.0;
            s -= (dxv + dyv) / tv_cell(mu, nx, ny, x, y, eps);
            grad[(size_t)y * nx + x] = s;
        }
}

static double blank_of(const double* blank, double blank_scalar, int c) { return blank ? blank[c] : blank_scalar; }

static double blank_ref(const double* blank, double blank_scalar, int C) {
    if (!blank) return blank_scalar;
    double s = 0.0;
    for (int c = 0; c < C; ++c) s += blank[c];
    return s / C;
}

/* ---- C4: L(mu)/b_ref over one subset, L = sum_i (y_i ln ybar_i - ybar_i), ybar_i = b_i exp(-[A mu]_i)
 * ("photon statistics at the detector obeys the Poisson distribution") ---- */
double oracle_loglik(const oracle_geometry* g, const double* img, const double* counts /*[V][C]*/,
                     const double* blank, double blank_scalar, int subset, int n_subsets) {
    const int nv = subset_views(g, subset, n_subsets), C = g->n_channels;
    double* l = (double*)malloc(sizeof(double) * nv * C);
    oracle_forward(g, img, l, subset, n_subsets);
    double bref = blank_ref(blank, blank_scalar, C), s = 0.0;
    for (int j = 0; j < nv; ++j)
        for (int c = 0; c < C; ++c) {
            double b = blank_of(blank, blank_scalar, c);
            double y = counts[(size_t)subset_view(j, subset, n_subsets) * C + c];
            double ybar = b * exp(-l[(size_t)j * C + c]);
            s += y * log(ybar) - ybar;
        }
    free(l);
    return s / bref;
}

/* r_i = (ybar_i - y_i)/b_ref on the subset (compact), and the monitor
 * D = sum_i (l_i - p_i)^2, p_i = ln(b_i / max(y_i,1))  (C5; "square of difference between a
 * reprojection and a projection") */
double oracle_residual(const oracle_geometry* g, const double* l, const double* counts, const double* blank,
                       double blank_scalar, int subset, int n_subsets, double* resid) {
    const int nv = subset_views(g, subset, n_subsets), C = g->n_channels;
    double bref = blank_ref(blank, blank_scalar, C), D = 0.0;
    for (int j = 0; j < nv; ++j)
        for (int c = 0; c < C; ++c) {
            double b = blank_of(blank, blank_scalar, c);
            double y = counts[(size_t)subset_view(j, subset, n_subsets) * C + c];
            double li = l[(size_t)j * C + c];
            double ybar = b * exp(-li);
            resid[(size_t)j * C + c] = (ybar - y) / bref;
            double p = log(b / (y > 1.0 ? y : 1.0));
            D += (li - p) * (li - p);
        }
    return D;
}

/* tau_S = kappa * delta_iso / (V_S N Delta^3), delta_iso = SAD*dgamma, N = max(nx,ny)   (C6) */
double oracle_tau(const oracle_geometry* g, int n_subsets, double kappa) {
    int N = g->nx > g->ny ? g->nx : g->ny;
    double vs = (double)(g->n_views / n_subsets), d = g->pixel_mm;
    return kappa * g->sad_mm * oracle_dgamma(g) / (vs * N * d * d * d);
}

/* ---- the iteration: PAPER.md:74 Eq.3, :100-108 Eq.4-5, :114 initial image, :118 ordered subsets and
 * alpha x thinning, :63 positivity, :140 minimum-of-oscillation image.  Readings C5,C6,C10-C12. ----
 * counts [V][C]; blank NULL (-> scalar) or [C]; img_out [ny][nx]; trace NULL or [n_iters][2] = (D, lambda).
 * returns 0, or -3 if the monitor became non-finite. */
int oracle_reconstruct(const oracle_geometry* g, const double* counts, const double* blank, double blank_scalar,
                       const oracle_params* prm, double* img_out, double* trace) {
    const int M = prm->n_subsets, C = g->n_channels, nv = g->n_views / M;
    const size_t npix = (size_t)g->nx * g->ny, nray = (size_t)nv * C;
    double* mu    = (double*)malloc(sizeof(double) * npix);
    double* best  = (double*)malloc(sizeof(double) * npix);
    double* grad  = (double*)malloc(sizeof(double) * npix);
    double* tvg   = (double*)malloc(sizeof(double) * npix);
    double* l     = (double*)malloc(sizeof(double) * nray);
    double* resid = (double*)malloc(sizeof(double) * nray);
    const double tau = oracle_tau(g, M, prm->kappa);
    double lambda = prm->lambda0, Dprev = 0.0, Dbest = INFINITY;
    double* Dsub  = (double*)malloc(sizeof(double) * M);      /* monitor_mode 1: D of each subset's last visit */
    int status = 0;

    for (size_t r = 0; r < npix; ++r) mu[r] = prm->mu0;
    memcpy(best, mu, sizeof(double) * npix);

    for (int n = 0; n < prm->n_iters; ++n) {
        int m = n % M;                                                        /* PAPER.md:118, C11 */
        oracle_forward(g, mu, l, m, M);                                       /* "reprojection" */
        double D = oracle_residual(g, l, counts, blank, blank_scalar, m, M, resid);
        if (!isfinite(D)) status = -3;
        if (prm->forced_lambda) lambda = prm->forced_lambda[n];
        else if (n < (prm->monitor_mode ? M : 1)) lambda = prm->lambda0;
        else if (D < (prm->monitor_mode ? Dsub[m] : Dprev)) lambda = lambda + prm->lambda_up;   /* Eq. 4 */
        else { lambda = lambda - prm->lambda_down;                            /* Eq. 5 */
               if (lambda < prm->lambda_min) lambda = prm->lambda_min; }      /* floor, C10 */
        Dprev = D;
        Dsub[m] = D;
        if (trace) { trace[2 * n] = D; trace[2 * n + 1] = lambda; }
        if (prm->return_best && D < Dbest) { Dbest = D; memcpy(best, mu, sizeof(double) * npix); }
        oracle_backward(g, resid, grad, m, M);                                /* "estimation" */
        oracle_tv_grad(mu, tvg, g->nx, g->ny, prm->tv_eps);
        for (size_t r = 0; r < npix; ++r) {                                   /* Eq. 3 + mu > 0 */
            double u = mu[r] + lambda * tau * (grad[r] - (prm->beta / M) * tvg[r]);
            mu[r] = u > 0.0 ? u : 0.0;
        }
    }
    if (prm->return_best) {
        /* the final iterate competes too: one extra reprojection with the subset that would come next (C12) */
        int m = prm->n_iters % M;
        oracle_forward(g, mu, l, m, M);
        double D = oracle_residual(g, l, counts, blank, blank_scalar, m, M, resid);
        if (D < Dbest) memcpy(best, mu, sizeof(double) * npix);
        memcpy(img_out, best, sizeof(double) * npix);
    } else {
        memcpy(img_out, mu, sizeof(double) * npix);
    }
    free(mu); free(best); free(grad); free(tvg); free(l); free(resid); free(Dsub);
    return status;
}

/* ======================================================================================================
 * Stack of slices (readings H1-H3): TomoTherapy acquires helically
 * (PAPER.md:51), so neighbouring slices see the gantry at shifted angles and belong to one volume.
 *   H1  slice s of S is a 2-D fan slice whose view j was taken at gantry angle theta0 + 2*pi*(j + k*s)/V:
 *       the couch advances one slice every k views (view_shift = k, an integer number of views).
 *   H2  the prior is the 3-D smoothed isotropic TV  sum_{x,y,s} sqrt(eps^2 + dx^2 + dy^2 + Dz^2),
 *       Dz = w_z * (mu_{s+1} - mu_s), forward differences, 0 across the volume's border (w_z = tv_z).
 *   H3  every slice keeps its own monitor D_s (its own data) and its own step lambda_s by Eq. 4-5; all slices
 *       are updated together from mu(n) (the coupling enters only through the TV gradient).
 * ====================================================================================================== */
static double tv3_cell(const double* mu, int nx, int ny, int S, int x, int y, int s, double eps, double wz) {
    const size_t np = (size_t)nx * ny;
    double c = mu[s * np + (size_t)y * nx + x];
    double dxv = (x + 1 < nx) ? mu[s * np + (size_t)y * nx + x + 1] - c : 0.0;
    double dyv = (y + 1 < ny) ? mu[s * np + (size_t)(y + 1) * nx + x] - c : 0.0;
    double dzv = (s + 1 < S) ? wz * (mu[(s + 1) * np + (size_t)y * nx + x] - c) : 0.0;
    return sqrt(eps * eps + dxv * dxv + dyv * dyv + dzv * dzv);
}

double oracle_tv3_value(const double* mu, int nx, int ny, int S, double eps, double wz) {
    double t = 0.0;
    for (int s = 0; s < S; ++s)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) t += tv3_cell(mu, nx, ny, S, x, y, s, eps, wz);
    return t;
}

/* d/dmu_{x,y,s}: own cell -(dx + dy + w_z*Dz)/t, cell (x-1,y,s) +dx/t, cell (x,y-1,s) +dy/t,
 * cell (x,y,s-1) +w_z*Dz/t; out-of-range terms dropped */
void oracle_tv3_grad(const double* mu, double* grad, int nx, int ny, int S, double eps, double wz) {
    const size_t np = (size_t)nx * ny;
    #pragma omp parallel for collapse(2)
    for (int s = 0; s < S; ++s)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const size_t o = s * np + (size_t)y * nx + x;
                double c = mu[o], g = 0.0;
                if (x > 0) g += (c - mu[o - 1]) / tv3_cell(mu, nx, ny, S, x - 1, y, s, eps, wz);
                if (y > 0) g += (c - mu[o - nx]) / tv3_cell(mu, nx, ny, S, x, y - 1, s, eps, wz);
                if (s > 0) g += wz * wz * (c - mu[o - np]) / tv3_cell(mu, nx, ny, S, x, y, s - 1, eps, wz);
                double dxv = (x + 1 < nx) ? mu[o + 1] - c : 0.0;
                double dyv = (y + 1 < ny) ? mu[o + nx] - c : 0.0;
                double dzv = (s + 1 < S) ? wz * (mu[o + np] - c) : 0.0;
                g -= (dxv + dyv + wz * dzv) / tv3_cell(mu, nx, ny, S, x, y, s, eps, wz);
                grad[o] = g;
            }
}

/* counts [S][V][C]; img_out [S][ny][nx]; trace NULL or [S][n_iters][2].  view_shift = k (H1), tv_z = w_z (H2;
 * 0 = the 2-D prior slice by slice).  return_best and forced_lambda are not offered for stacks. */
int oracle_reconstruct_stack(const oracle_geometry* g, int S, const double* counts, const double* blank,
                             double blank_scalar, const oracle_params* prm, int view_shift, double tv_z,
                             double* img_out, double* trace) {
    const int M = prm->n_subsets, C = g->n_channels, nv = g->n_views / M, N = prm->n_iters;
    const size_t npix = (size_t)g->nx * g->ny, nray = (size_t)nv * C, nsino = (size_t)g->n_views * C;
    double* mu    = (double*)malloc(sizeof(double) * npix * S);
    double* nxt   = (double*)malloc(sizeof(double) * npix * S);
    double* tvg   = (double*)malloc(sizeof(double) * npix * S);
    double* grad  = (double*)malloc(sizeof(double) * npix);
    double* l     = (double*)malloc(sizeof(double) * nray);
    double* resid = (double*)malloc(sizeof(double) * nray);
    double* lambda = (double*)malloc(sizeof(double) * S);
    double* Dprev  = (double*)malloc(sizeof(double) * S);
    double* Dsub   = (double*)malloc(sizeof(double) * S * M);
    const double tau = oracle_tau(g, M, prm->kappa);
    int status = 0;
    for (size_t r = 0; r < npix * S; ++r) mu[r] = prm->mu0;
    for (int s = 0; s < S; ++s) { lambda[s] = prm->lambda0; Dprev[s] = 0.0; }

    for (int n = 0; n < N; ++n) {
        const int m = n % M;
        if (tv_z > 0.0) oracle_tv3_grad(mu, tvg, g->nx, g->ny, S, prm->tv_eps, tv_z);
        else for (int s = 0; s < S; ++s) oracle_tv_grad(mu + s * npix, tvg + s * npix, g->nx, g->ny, prm->tv_eps);
        for (int s = 0; s < S; ++s) {
            oracle_geometry gs = *g;                                           /* H1: the gantry angle of slice s */
            gs.theta0_rad = g->theta0_rad + 2.0 * M_PI * (double)view_shift * (double)s / (double)g->n_views;
            const double* mus = mu + s * npix;
            oracle_forward(&gs, mus, l, m, M);
            double D = oracle_residual(&gs, l, counts + s * nsino, blank, blank_scalar, m, M, resid);
            if (!isfinite(D)) status = -3;
            double lam = lambda[s];
            if (n < (prm->monitor_mode ? M : 1)) lam = prm->lambda0;
            else if (D < (prm->monitor_mode ? Dsub[s * M + m] : Dprev[s])) lam = lam + prm->lambda_up;
            else { lam = lam - prm->lambda_down; if (lam < prm->lambda_min) lam = prm->lambda_min; }
            lambda[s] = lam; Dprev[s] = D; Dsub[s * M + m] = D;
            if (trace) { trace[((size_t)s * N + n) * 2] = D; trace[((size_t)s * N + n) * 2 + 1] = lam; }
            oracle_backward(&gs, resid, grad, m, M);
            for (size_t r = 0; r < npix; ++r) {
                double u = mus[r] + lam * tau * (grad[r] - (prm->beta / M) * tvg[s * npix + r]);
                nxt[s * npix + r] = u > 0.0 ? u : 0.0;
            }
        }
        double* t = mu; mu = nxt; nxt = t;
    }
    memcpy(img_out, mu, sizeof(double) * npix * S);
    free(mu); free(nxt); free(tvg); free(grad); free(l); free(resid); free(lambda); free(Dprev); free(Dsub);
    return status;
}
