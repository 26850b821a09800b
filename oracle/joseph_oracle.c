/*
 * joseph_oracle.c -- float64 CPU ORACLE for Joseph's projector (non-TOF, TOF sinogram,
 * TOF listmode) and listmode OSEM.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares
 * no code with the CUDA path (paper_2212_12519_b200/csrc) and neither includes the other.
 *
 * It follows the method of PAPER.md section 2.1 step by step, in the paper's order, with the
 * readings A1..A14 of SURVEY.md section 8(c) where the paper is silent (all listed in DESIGN.md).
 * All arithmetic is IEEE double.  Coordinates may be given as float32 (the arrays the GPU
 * gets; promoted exactly) or float64 (for pin tests).
 *
 * Parity pins (tests/test_oracle_pins.py): chord closed forms C1-C3, library interpolant L,
 * dense-matrix transpose M, adjointness ADJ, brute-force exact intersection BF, worked
 * examples W, TOF bin sum T1, TOF point source T2 (against numerical quadrature), LM == sinogram
 * column T3, symmetries S, degenerate D, OSEM count preservation O.
 * "parity unpinned" (pure conventions, fixed by nothing in the paper): A3 tie direction,
 * A9 TOF index origin / sign, A14 subset rule and guards.
 *
 * Notation: image f[i0,i1,i2], C order, axis 2 fastest; n = dims,
 * v = voxel size (mm), o = world coordinate of the centre of voxel [0,0,0]; LOR from s to e,
 * d = e - s, L = |d|, p = principal axis, q1 < q2 the other two axes.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC joseph_oracle.c -o liboracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t n[3];
    double o[3];
    double v[3];
} geom_t;

typedef struct {
    double delta;    /* TOF bin width (mm) */
    double sigma;    /* TOF resolution, standard deviation (mm) */
    double nsig;     /* truncation in sigmas (PAPER.md:78 -> 3) */
    int32_t nbins;   /* number of sinogram TOF bins */
    double coff;     /* centre offset (mm) */
} tof_t;

/* the six coordinate arrays, float32 or float64 */
typedef struct {
    const void *c[6]; /* xs ys zs xe ye ze */
    int is_f64;
} lors_t;

static inline double coord(const lors_t *l, int which, int64_t j)
{
    return l->is_f64 ? ((const double *)l->c[which])[j] : (double)((const float *)l->c[which])[j];
}

/* ---- per-LOR set-up: A1 (degenerate), A2/A3 (principal axis), A6 (cf) ------------------ */
typedef struct {
    double s[3], d[3];
    double L, cf;
    int p, q1, q2;
    int degenerate;
} ray_t;

static void ray_setup(const lors_t *l, int64_t j, const geom_t *g, ray_t *r)
{
    double e[3];
    for (int a = 0; a < 3; a++) {
        r->s[a] = coord(l, a, j);
        e[a] = coord(l, 3 + a, j);
        r->d[a] = e[a] - r->s[a]; /* exact in double for float32 inputs */
    }
    /* A1: zero-length LOR contributes nothing */
    r->degenerate = (r->d[0] == 0.0 && r->d[1] == 0.0 && r->d[2] == 0.0);
    /* A2: "the principal direction in the image that is most parallel to the ray"
       = argmax_a |d_a|;  A3: ties -> lowest axis index */
    int p = 0;
    if (fabs(r->d[1]) > fabs(r->d[p])) p = 1;
    if (fabs(r->d[2]) > fabs(r->d[p])) p = 2;
    r->p = p;
    r->q1 = (p == 0) ? 1 : 0;
    r->q2 = (p == 2) ? 1 : 2;
    r->L = sqrt(r->d[0] * r->d[0] + r->d[1] * r->d[1] + r->d[2] * r->d[2]);
    /* A6: "corrected for the incidence angle": path length between two
       consecutive planes of axis p */
    r->cf = r->degenerate ? 0.0 : g->v[p] * r->L / fabs(r->d[p]);
}

/* ---- one plane: A4 (plane, segment rule), A5 (crossing point, 4 neighbours) ------------ */
typedef struct {
    double t;        /* ray parameter of the crossing, 0 at s, 1 at e */
    int64_t k1, k2;  /* floor of the crossing point in voxel units along q1, q2 */
    double w1[2], w2[2]; /* bilinear weights (1-phi, phi) along q1, q2 */
} cross_t;

/* returns 0 if plane i is not crossed by the segment or the 4 neighbours are all outside */
static int plane_cross(const ray_t *r, const geom_t *g, int i, cross_t *c)
{
    const int p = r->p, q1 = r->q1, q2 = r->q2;
    /* A4: planes are the voxel-centre planes x_p = o_p + i v_p */
    double t = (g->o[p] + (double)i * g->v[p] - r->s[p]) / r->d[p];
    if (!(t >= 0.0 && t <= 1.0)) return 0; /* the LOR is the closed segment [s, e] */
    /* A5: "the intersection point between the ray and the plane" in voxel units */
    double u1 = (r->s[q1] + t * r->d[q1] - g->o[q1]) / g->v[q1];
    double u2 = (r->s[q2] + t * r->d[q2] - g->o[q2]) / g->v[q2];
    double f1 = floor(u1), f2 = floor(u2);
    /* neighbours k and k+1; if both are outside [0, n-1] nothing contributes (zero padding) */
    if (f1 < -1.0 || f1 > (double)(g->n[q1] - 1)) return 0;
    if (f2 < -1.0 || f2 > (double)(g->n[q2] - 1)) return 0;
    c->t = t;
    c->k1 = (int64_t)f1;
    c->k2 = (int64_t)f2;
    c->w1[1] = u1 - f1; c->w1[0] = 1.0 - c->w1[1];
    c->w2[1] = u2 - f2; c->w2[0] = 1.0 - c->w2[1];
    return 1;
}

/* linear index of voxel with index i along p, a along q1, b along q2; -1 if outside */
static inline int64_t vox_index(const ray_t *r, const geom_t *g, int i, int64_t a, int64_t b)
{
    if (a < 0 || a >= g->n[r->q1] || b < 0 || b >= g->n[r->q2]) return -1;
    int64_t idx[3];
    idx[r->p] = i; idx[r->q1] = a; idx[r->q2] = b;
    return (idx[0] * g->n[1] + idx[1]) * (int64_t)g->n[2] + idx[2];
}

/* A5: bilinear interpolation of the four nearest neighbours, zero outside the image */
static double plane_value(const ray_t *r, const geom_t *g, int i, const cross_t *c, const double *f)
{
    double val = 0.0;
    for (int a = 0; a < 2; a++)
        for (int b = 0; b < 2; b++) {
            int64_t idx = vox_index(r, g, i, c->k1 + a, c->k2 + b);
            if (idx >= 0) val += c->w1[a] * c->w2[b] * f[idx];
        }
    return val;
}

/* A7: adjoint of plane_value: img[...] += w1 w2 x */
static void plane_scatter(const ray_t *r, const geom_t *g, int i, const cross_t *c, double x, double *img)
{
    for (int a = 0; a < 2; a++)
        for (int b = 0; b < 2; b++) {
            int64_t idx = vox_index(r, g, i, c->k1 + a, c->k2 + b);
            if (idx >= 0) img[idx] += c->w1[a] * c->w2[b] * x;
        }
}

/* ---- TOF: A8 (coordinate), A10 (kernel) ------------------------------------------------- */
/* A8: signed distance of the crossing point from the LOR midpoint, positive towards e */
static inline double tof_tau(const ray_t *r, const tof_t *tf, double t)
{
    return (t - 0.5) * r->L - tf->coff;
}

static inline double clampd(double x, double lo, double hi)
{
    return x < lo ? lo : (x > hi ? hi : x);
}

/* A10: Gaussian (sigma) truncated at +-nsig sigma, integrated over the bin [c-delta/2, c+delta/2]
   as seen from position tau: "the difference of two error functions".
   No renormalisation. */
static double tof_weight(const tof_t *tf, double tau, double c)
{
    const double lim = tf->nsig * tf->sigma;
    double hi = clampd(c + 0.5 * tf->delta - tau, -lim, lim);
    double lo = clampd(c - 0.5 * tf->delta - tau, -lim, lim);
    const double sc = 1.0 / (tf->sigma * sqrt(2.0));
    return 0.5 * (erf(hi * sc) - erf(lo * sc));
}

/* A9: centre of sinogram bin k */
static inline double sino_bin_centre(const tof_t *tf, int k)
{
    return ((double)k - 0.5 * (double)(tf->nbins - 1)) * tf->delta;
}

/* ---- per-LOR operators ----------------------------------------------------------------- */
static double lor_fwd(const lors_t *l, int64_t j, const geom_t *g, const double *f)
{
    ray_t r; cross_t c;
    ray_setup(l, j, g, &r);
    if (r.degenerate) return 0.0;
    double sum = 0.0;
    for (int i = 0; i < g->n[r.p]; i++)
        if (plane_cross(&r, g, i, &c)) sum += plane_value(&r, g, i, &c, f);
    return r.cf * sum; /* A6 */
}

static void lor_back(const lors_t *l, int64_t j, const geom_t *g, double y, double *img)
{
    ray_t r; cross_t c;
    ray_setup(l, j, g, &r);
    if (r.degenerate) return;
    for (int i = 0; i < g->n[r.p]; i++)
        if (plane_cross(&r, g, i, &c)) plane_scatter(&r, g, i, &c, r.cf * y, img);
}

/* A11: all sinogram bins of one LOR; out[k], k = 0..nbins-1 */
static void lor_fwd_tof_sino(const lors_t *l, int64_t j, const geom_t *g, const tof_t *tf,
                             const double *f, double *out)
{
    ray_t r; cross_t c;
    for (int k = 0; k < tf->nbins; k++) out[k] = 0.0;
    ray_setup(l, j, g, &r);
    if (r.degenerate) return;
    for (int i = 0; i < g->n[r.p]; i++) {
        if (!plane_cross(&r, g, i, &c)) continue;
        double val = plane_value(&r, g, i, &c, f);
        double tau = tof_tau(&r, tf, c.t);
        for (int k = 0; k < tf->nbins; k++)
            out[k] += val * tof_weight(tf, tau, sino_bin_centre(tf, k));
    }
    for (int k = 0; k < tf->nbins; k++) out[k] *= r.cf;
}

static void lor_back_tof_sino(const lors_t *l, int64_t j, const geom_t *g, const tof_t *tf,
                              const double *y /*[nbins]*/, double *img)
{
    ray_t r; cross_t c;
    ray_setup(l, j, g, &r);
    if (r.degenerate) return;
    for (int i = 0; i < g->n[r.p]; i++) {
        if (!plane_cross(&r, g, i, &c)) continue;
        double tau = tof_tau(&r, tf, c.t);
        double x = 0.0;
        for (int k = 0; k < tf->nbins; k++)
            x += y[k] * tof_weight(tf, tau, sino_bin_centre(tf, k));
        plane_scatter(&r, g, i, &c, r.cf * x, img);
    }
}

/* A12: one listmode TOF bin it (signed, 0 = bin centred on the LOR midpoint) */
static double lor_fwd_tof_lm(const lors_t *l, int64_t j, const geom_t *g, const tof_t *tf,
                             int it, const double *f)
{
    ray_t r; cross_t c;
    ray_setup(l, j, g, &r);
    if (r.degenerate) return 0.0;
    const double centre = (double)it * tf->delta;
    double sum = 0.0;
    for (int i = 0; i < g->n[r.p]; i++) {
        if (!plane_cross(&r, g, i, &c)) continue;
        sum += plane_value(&r, g, i, &c, f) * tof_weight(tf, tof_tau(&r, tf, c.t), centre);
    }
    return r.cf * sum;
}

static void lor_back_tof_lm(const lors_t *l, int64_t j, const geom_t *g, const tof_t *tf,
                            int it, double y, double *img)
{
    ray_t r; cross_t c;
    ray_setup(l, j, g, &r);
    if (r.degenerate) return;
    const double centre = (double)it * tf->delta;
    for (int i = 0; i < g->n[r.p]; i++) {
        if (!plane_cross(&r, g, i, &c)) continue;
        double w = tof_weight(tf, tof_tau(&r, tf, c.t), centre);
        plane_scatter(&r, g, i, &c, r.cf * y * w, img);
    }
}

/* ---- helpers --------------------------------------------------------------------------- */
static int64_t nvox(const geom_t *g) { return (int64_t)g->n[0] * g->n[1] * g->n[2]; }

static int check_geom(const geom_t *g)
{
    for (int a = 0; a < 3; a++)
        if (g->n[a] <= 0 || !(g->v[a] > 0.0)) return -2;
    return 0;
}

static int check_tof(const tof_t *tf)
{
    if (tf->nbins < 1 || !(tf->sigma > 0.0) || !(tf->delta > 0.0) || !(tf->nsig > 0.0)) return -2;
    return 0;
}

static int max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int this_thread(void)
{
#ifdef _OPENMP
    return omp_get_thread_num();
#else
    return 0;
#endif
}

/* thread-private images reduced in thread order: deterministic for a given thread count */
static double *alloc_private(const geom_t *g, int nt)
{
    return (double *)calloc((size_t)nt * (size_t)nvox(g), sizeof(double));
}

static void reduce_private(const geom_t *g, int nt, const double *priv, double *img)
{
    const int64_t nv = nvox(g);
#pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < nv; x++) {
        double acc = 0.0;
        for (int t = 0; t < nt; t++) acc += priv[(size_t)t * nv + x];
        img[x] += acc;
    }
}

/* ---- exported C ABI (host pointers, double outputs) ------------------------------------ */
/* All LOR loops take (first, stride, count): LOR indices first, first+stride, ... (count of them);
   outputs / inputs y are indexed by the same LOR index j.  Plain calls use (0, 1, n). */

int orc_num_threads(void) { return max_threads(); }

int orc_classify(const lors_t *l, int64_t n, const geom_t *g, uint8_t *axis)
{
    if (!l || !g || (n > 0 && !axis)) return -1;
    if (n < 0) return -2;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; j++) {
        ray_t r;
        ray_setup(l, j, g, &r);
        axis[j] = (uint8_t)r.p;
    }
    return 0;
}

int orc_fwd(const lors_t *l, int64_t first, int64_t stride, int64_t count, const geom_t *g,
            const double *f, double *p)
{
    if (!l || !g || !f || (count > 0 && !p)) return -1;
    if (count < 0 || stride < 1 || check_geom(g)) return -2;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t c = 0; c < count; c++) {
        int64_t j = first + c * stride;
        p[j] = lor_fwd(l, j, g, f);
    }
    return 0;
}

int orc_back(const lors_t *l, int64_t first, int64_t stride, int64_t count, const geom_t *g,
             const double *y, double *img)
{
    if (!l || !g || !img || (count > 0 && !y)) return -1;
    if (count < 0 || stride < 1 || check_geom(g)) return -2;
    const int nt = max_threads();
    double *priv = alloc_private(g, nt);
    if (!priv) return -3;
    const int64_t nv = nvox(g);
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < count; c++) {
        int64_t j = first + c * stride;
        lor_back(l, j, g, y[j], priv + (size_t)this_thread() * nv);
    }
    reduce_private(g, nt, priv, img);
    free(priv);
    return 0;
}

int orc_fwd_tof_sino(const lors_t *l, int64_t first, int64_t stride, int64_t count,
                     const geom_t *g, const tof_t *tf, const double *f, double *p /*[n][nbins]*/)
{
    if (!l || !g || !tf || !f || (count > 0 && !p)) return -1;
    if (count < 0 || stride < 1 || check_geom(g) || check_tof(tf)) return -2;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t c = 0; c < count; c++) {
        int64_t j = first + c * stride;
        lor_fwd_tof_sino(l, j, g, tf, f, p + j * tf->nbins);
    }
    return 0;
}

int orc_back_tof_sino(const lors_t *l, int64_t first, int64_t stride, int64_t count,
                      const geom_t *g, const tof_t *tf, const double *y /*[n][nbins]*/, double *img)
{
    if (!l || !g || !tf || !img || (count > 0 && !y)) return -1;
    if (count < 0 || stride < 1 || check_geom(g) || check_tof(tf)) return -2;
    const int nt = max_threads();
    double *priv = alloc_private(g, nt);
    if (!priv) return -3;
    const int64_t nv = nvox(g);
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < count; c++) {
        int64_t j = first + c * stride;
        lor_back_tof_sino(l, j, g, tf, y + j * tf->nbins, priv + (size_t)this_thread() * nv);
    }
    reduce_private(g, nt, priv, img);
    free(priv);
    return 0;
}

int orc_fwd_tof_lm(const lors_t *l, const int16_t *tofbin, int64_t first, int64_t stride,
                   int64_t count, const geom_t *g, const tof_t *tf, const double *f, double *p)
{
    if (!l || !g || !tf || !f || (count > 0 && (!p || !tofbin))) return -1;
    if (count < 0 || stride < 1 || check_geom(g) || check_tof(tf)) return -2;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t c = 0; c < count; c++) {
        int64_t j = first + c * stride;
        p[j] = lor_fwd_tof_lm(l, j, g, tf, (int)tofbin[j], f);
    }
    return 0;
}

int orc_back_tof_lm(const lors_t *l, const int16_t *tofbin, int64_t first, int64_t stride,
                    int64_t count, const geom_t *g, const tof_t *tf, const double *y, double *img)
{
    if (!l || !g || !tf || !img || (count > 0 && (!y || !tofbin))) return -1;
    if (count < 0 || stride < 1 || check_geom(g) || check_tof(tf)) return -2;
    const int nt = max_threads();
    double *priv = alloc_private(g, nt);
    if (!priv) return -3;
    const int64_t nv = nvox(g);
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < count; c++) {
        int64_t j = first + c * stride;
        lor_back_tof_lm(l, j, g, tf, (int)tofbin[j], y[j], priv + (size_t)this_thread() * nv);
    }
    reduce_private(g, nt, priv, img);
    free(priv);
    return 0;
}

/* A14: listmode OSEM (standard OSEM, PAPER.md:193 ref. 39), no attenuation,
   contamination or resolution model (BASELINE.json configs[4]).
   subset m = events {e : e mod n_subsets == m}, m = 0..n_subsets-1 in order;
   ybar_e = (A x)_e;  r_e = 1/ybar_e if ybar_e > 1e-9 else 0;  b = A_m^T r;
   x <- x * b * n_subsets / sens where sens > 0, else 0.
   img: in = start image, out = result.  ybar_last (optional, [n]) receives the last forward
   projection of every event (used by the count-preservation pin O). */
int orc_lm_osem(const lors_t *l, const int16_t *tofbin, int64_t n, const geom_t *g, const tof_t *tf,
                const double *sens, double *img, int n_subsets, int n_iter, double *ybar_last)
{
    if (!l || !g || !tf || !sens || !img || (n > 0 && !tofbin)) return -1;
    if (n < 0 || n_subsets < 1 || n_iter < 0 || check_geom(g) || check_tof(tf)) return -2;
    const int64_t nv = nvox(g);
    double *ybar = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *b = (double *)malloc(sizeof(double) * (size_t)nv);
    if (!ybar || !b) { free(ybar); free(b); return -3; }
    int rc = 0;
    for (int it = 0; it < n_iter && !rc; it++) {
        for (int m = 0; m < n_subsets && !rc; m++) {
            if (m >= n) { /* empty subset: b = 0 */ }
            int64_t count = (n > m) ? (n - m + n_subsets - 1) / n_subsets : 0;
            rc = orc_fwd_tof_lm(l, tofbin, m, n_subsets, count, g, tf, img, ybar);
            if (rc) break;
            for (int64_t c = 0; c < count; c++) {
                int64_t j = m + c * (int64_t)n_subsets;
                if (ybar_last) ybar_last[j] = ybar[j];
                ybar[j] = (ybar[j] > 1e-9) ? 1.0 / ybar[j] : 0.0;
            }
            memset(b, 0, sizeof(double) * (size_t)nv);
            rc = orc_back_tof_lm(l, tofbin, m, n_subsets, count, g, tf, ybar, b);
            if (rc) break;
            for (int64_t x = 0; x < nv; x++)
                img[x] = (sens[x] > 0.0) ? img[x] * b[x] * (double)n_subsets / sens[x] : 0.0;
        }
    }
    free(ybar);
    free(b);
    return rc;
}

/* ---- image-based resolution model ------------------------------------
   PAPER.md:94: "a shift-invariant image-based resolution model was used, including a 3D isotropic
   Gaussian kernel of 4.5 mm FWHM"; 68 Gaussian convolutions per iteration of 34 subsets,
   i.e. one before every forward and one after every back projection.  The paper fixes nothing else;
   readings (R1-R3):
   R1  K[k0,k1,k2] = g_0[k0] g_1[k1] g_2[k2],  g_a[k] = exp(-(k v_a)^2 / (2 sigma^2)) / sum_k' (same),
       |k| <= r_a = ceil(n_sigmas sigma / v_a)  (truncated like the TOF kernel, normalised per axis);
   R2  voxels outside the image count as zero, so the operator is symmetric (G = G^T);
   R3  OSEM: ybar = A (G x), b = G (A^T r), x <- x b n_subsets / sens  (sens supplied by the caller).
   The convolution is written out as the plain triple sum (no separable passes). */
static int gauss_taps(double sigma_mm, double nsig, double v, double **taps, int *radius)
{
    int r = (int)ceil(nsig * sigma_mm / v);
    if (r < 0) r = 0;
    double *g = (double *)malloc(sizeof(double) * (size_t)(2 * r + 1));
    if (!g) return -3;
    double sum = 0.0;
    for (int k = -r; k <= r; k++) {
        double x = (double)k * v / sigma_mm;
        g[k + r] = exp(-0.5 * x * x);
        sum += g[k + r];
    }
    for (int k = 0; k <= 2 * r; k++) g[k] /= sum;
    *taps = g;
    *radius = r;
    return 0;
}

int orc_gauss3d(const double *in, double *out, const geom_t *g, double sigma_mm, double nsig)
{
    if (!in || !out || !g) return -1;
    if (check_geom(g) || !(sigma_mm > 0.0) || !(nsig > 0.0)) return -2;
    double *t[3] = {0, 0, 0};
    int r[3];
    for (int a = 0; a < 3; a++)
        if (gauss_taps(sigma_mm, nsig, g->v[a], &t[a], &r[a])) { free(t[0]); free(t[1]); free(t[2]); return -3; }
    const int n0 = g->n[0], n1 = g->n[1], n2 = g->n[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (int i0 = 0; i0 < n0; i0++)
        for (int i1 = 0; i1 < n1; i1++)
            for (int i2 = 0; i2 < n2; i2++) {
                double acc = 0.0;
                for (int k0 = -r[0]; k0 <= r[0]; k0++) {
                    int j0 = i0 - k0;
                    if (j0 < 0 || j0 >= n0) continue;
                    for (int k1 = -r[1]; k1 <= r[1]; k1++) {
                        int j1 = i1 - k1;
                        if (j1 < 0 || j1 >= n1) continue;
                        for (int k2 = -r[2]; k2 <= r[2]; k2++) {
                            int j2 = i2 - k2;
                            if (j2 < 0 || j2 >= n2) continue;
                            acc += t[0][k0 + r[0]] * t[1][k1 + r[1]] * t[2][k2 + r[2]] *
                                   in[((int64_t)j0 * n1 + j1) * n2 + j2];
                        }
                    }
                }
                out[((int64_t)i0 * n1 + i1) * n2 + i2] = acc;
            }
    free(t[0]); free(t[1]); free(t[2]);
    return 0;
}

/* listmode OSEM with the resolution model (reading R3); otherwise identical to orc_lm_osem */
int orc_lm_osem_res(const lors_t *l, const int16_t *tofbin, int64_t n, const geom_t *g, const tof_t *tf,
                    const double *sens, double *img, int n_subsets, int n_iter, double res_sigma_mm, double res_nsig)
{
    if (!l || !g || !tf || !sens || !img || (n > 0 && !tofbin)) return -1;
    if (n < 0 || n_subsets < 1 || n_iter < 0 || check_geom(g) || check_tof(tf)) return -2;
    const int64_t nv = nvox(g);
    double *ybar = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double *b = (double *)malloc(sizeof(double) * (size_t)nv);
    double *xb = (double *)malloc(sizeof(double) * (size_t)nv);
    double *gb = (double *)malloc(sizeof(double) * (size_t)nv);
    if (!ybar || !b || !xb || !gb) { free(ybar); free(b); free(xb); free(gb); return -3; }
    int rc = 0;
    for (int it = 0; it < n_iter && !rc; it++) {
        for (int m = 0; m < n_subsets && !rc; m++) {
            int64_t count = (n > m) ? (n - m + n_subsets - 1) / n_subsets : 0;
            rc = orc_gauss3d(img, xb, g, res_sigma_mm, res_nsig);
            if (rc) break;
            rc = orc_fwd_tof_lm(l, tofbin, m, n_subsets, count, g, tf, xb, ybar);
            if (rc) break;
            for (int64_t c = 0; c < count; c++) {
                int64_t j = m + c * (int64_t)n_subsets;
                ybar[j] = (ybar[j] > 1e-9) ? 1.0 / ybar[j] : 0.0;
            }
            memset(b, 0, sizeof(double) * (size_t)nv);
            rc = orc_back_tof_lm(l, tofbin, m, n_subsets, count, g, tf, ybar, b);
            if (rc) break;
            rc = orc_gauss3d(b, gb, g, res_sigma_mm, res_nsig);
            if (rc) break;
            for (int64_t x = 0; x < nv; x++)
                img[x] = (sens[x] > 0.0) ? img[x] * gb[x] * (double)n_subsets / sens[x] : 0.0;
        }
    }
    free(ybar); free(b); free(xb); free(gb);
    return rc;
}
