/*
 * tl_oracle.c -- FP64 CPU ORACLE for the batched lens-model likelihood.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant with the CUDA path under paper_2503_08586_b200/csrc/.
 *
 * What it is: the plain definition of the forward model of arxiv 2503.08586 (TinyLensGpu),
 * written out with pixel loops in double precision, in the paper's order and notation.  There
 * is no blocking, fusion or reordering.  Citations are PAPER.md:<line> (+ equation); where
 * the paper is silent the reading is SURVEY.md 8(c) G<k>, repeated in DESIGN.md "Readings".
 *
 * Pinned (tests/test_oracle_pins.py, -m "not gpu") against closed forms, invariants, library
 * routines and brute force: every exported function below has at least one pin, so nothing
 * here is "parity unpinned".  The conventions G4, G5, G10, G13 are choices, not facts; the
 * pins check the code implements the choice.
 *
 * Parameter row (float, widened exactly to double), P = 7 + 7*n_lens_light + 7*n_source:
 *   theta_E, e1, e2, cx, cy, gamma1, gamma2,
 *   [mass_model = EPL only: the slope gamma of Eq. 12, making P one larger,]
 *   then per Sersic (lens light first, then sources): I_e, r_e, n, e1, e2, cx, cy.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liboracle.so tl_oracle.c -lm   (no -ffast-math)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_EDGE_EXTEND 0
#define ORC_EDGE_ZERO 1

typedef struct {
    int32_t ny, nx;
    double pix_scale;
    int32_t supersample;
    int32_t n_lens_light;
    int32_t n_source;
    int32_t edge_mode;
    int32_t mass_model;      /* 0 = SIE (gamma = 2), 1 = EPL: the row carries the slope gamma at index 7 */
} orc_config;

#define ORC_MASS_SIE 0
#define ORC_MASS_EPL 1
/* parameters of the lens block: theta_E, e1, e2, cx, cy, gamma1, gamma2 [, gamma (EPL)] */
static int lens_np(const orc_config *cfg) { return 7 + (cfg->mass_model == ORC_MASS_EPL ? 1 : 0); }

/* ------------------------------------------------------------------ Eq. 9: b_n
 * PAPER.md:137-141 Eq. 9:  Gamma(2n) = 2 gamma(2n, b_n), i.e. P(2n, b_n) = 1/2 with P the
 * regularised lower incomplete gamma function.  gamma(a,x) by its power series
 *   gamma(a,x) = x^a e^{-x} sum_{k>=0} x^k / (a (a+1) ... (a+k)),
 * always in its fast regime here because the root lies below a = 2n.  Root by bisection.
 */
double orc_gammainc_p(double a, double x)
{
    if (x <= 0.0) return 0.0;
    double term = 1.0 / a, sum = term;
    for (int k = 1; k < 100000; ++k) {
        term *= x / (a + k);
        sum += term;
        if (term < sum * 1e-17) break;
    }
    return sum * exp(a * log(x) - x - lgamma(a));
}

double orc_bn(double n)
{
    double a = 2.0 * n;
    double lo = 0.0, hi = a > 1.0 ? a : 1.0;     /* the median of Gamma(a,1) is below max(a,1)... */
    while (orc_gammainc_p(a, hi) < 0.5) hi *= 2.0; /* ...and this loop makes the bracket unconditional */
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (orc_gammainc_p(a, mid) < 0.5) lo = mid; else hi = mid;
        if (hi - lo <= 1e-16 * hi) break;
    }
    return 0.5 * (lo + hi);
}

/* ------------------------------------------------------------------ Eq. 11 inverse
 * PAPER.md:150-154 Eq. 11: (e1,e2) = (1-q)/(1+q) (cos 2phi, sin 2phi).  Inverse (G3):
 * e = hypot(e1,e2), q = (1-e)/(1+e), phi = atan2(e2,e1)/2.  phi is the major-axis direction,
 * counter-clockwise from +x (G2).
 */
void orc_shape(double e1, double e2, double *q, double *phi)
{
    double e = hypot(e1, e2);
    *q = (1.0 - e) / (1.0 + e);
    *phi = 0.5 * atan2(e2, e1);
}

/* ------------------------------------------------------------------ Eq. 12 (gamma = 2): SIE
 * PAPER.md:156-160 Eq. 12 with gamma = 2 and R -> R_p of Eq. 10 ("extended to a two-
 * dimensional elliptical distribution ... similar to the light profile"), Kormann et al.
 * 1994 cited, no formula printed (G1):
 *   kappa = theta_E / (2 sqrt(q x'^2 + y'^2 / q))        in the frame rotated by phi,
 *   psi = sqrt(q^2 x'^2 + y'^2),  q' = sqrt((1-q)(1+q)),
 *   alpha_x' = theta_E sqrt(q) (x'/psi) A(q' x'/psi),  A(z) = atan(z)/z,
 *   alpha_y' = theta_E sqrt(q) (y'/psi) H(q' y'/psi),  H(z) = atanh(z)/z,
 * A, H -> 1 as z -> 0 (series below |z| < 1e-4), alpha = 0 at psi = 0 (G6).
 */
static double fn_A(double z)
{
    if (fabs(z) < 1e-4) { double z2 = z * z; return 1.0 - z2 / 3.0 + z2 * z2 / 5.0; }
    return atan(z) / z;
}
static double fn_H(double z)
{
    if (fabs(z) < 1e-4) { double z2 = z * z; return 1.0 + z2 / 3.0 + z2 * z2 / 5.0; }
    return atanh(z) / z;
}

void orc_sie_deflection(double theta_e, double q, double phi, double cx, double cy,
                        double x, double y, double *ax, double *ay)
{
    double c = cos(phi), s = sin(phi);
    double dx = x - cx, dy = y - cy;
    double xp = dx * c + dy * s;
    double yp = -dx * s + dy * c;
    double psi = sqrt(q * q * xp * xp + yp * yp);
    if (psi == 0.0) { *ax = 0.0; *ay = 0.0; return; }
    double qp = sqrt((1.0 - q) * (1.0 + q));
    double axp = theta_e * sqrt(q) * (xp / psi) * fn_A(qp * xp / psi);
    double ayp = theta_e * sqrt(q) * (yp / psi) * fn_H(qp * yp / psi);
    *ax = axp * c - ayp * s;
    *ay = axp * s + ayp * c;
}

/* ------------------------------------------------------------------ Eq. 12 (general gamma): EPL
 * PAPER.md:156-160 Eq. 12, kappa(R) = (3-gamma)/2 (theta_E/R)^(gamma-1), made elliptical as the
 * SIE above (R -> R_p of Eq. 10; reading G22), deflection after Tessore & Metcalf
 * (2015), which the paper cites and does not print.  With t = gamma - 1, the elliptical radius
 * and angle  R = sqrt(q^2 x'^2 + y'^2),  R cos(phi) = q x',  R sin(phi) = y',  b = theta_E sqrt(q)
 * (so that kappa = (2-t)/2 (b/R)^t), and f = (1-q)/(1+q), the complex deflection is
 *   alpha_x' + i alpha_y' = 2b/(1+q) (b/R)^(t-1) Omega,
 *   Omega = sum_{n>=0} Omega_n,  Omega_0 = e^{i phi},
 *   Omega_n = -f (2n - (2-t)) / (2n + (2-t)) e^{2 i phi} Omega_{n-1}
 * (their angular series of 2F1(1, t/2; 2 - t/2; -f e^{2 i phi})), summed in their order until a
 * term falls below 1e-18 of the sum.  alpha = 0 at R = 0.  Valid for 0 < t < 2.             */
void orc_epl_deflection(double theta_e, double gamma, double q, double phi, double cx, double cy,
                        double x, double y, double *ax, double *ay)
{
    double c = cos(phi), s = sin(phi);
    double dx = x - cx, dy = y - cy;
    double xp = dx * c + dy * s;
    double yp = -dx * s + dy * c;
    double R = sqrt(q * q * xp * xp + yp * yp);
    if (R == 0.0 || theta_e == 0.0) { *ax = 0.0; *ay = 0.0; return; }
    double t = gamma - 1.0, b = theta_e * sqrt(q), f = (1.0 - q) / (1.0 + q);
    double cph = q * xp / R, sph = yp / R;                    /* e^{i phi} */
    double c2 = cph * cph - sph * sph, s2 = 2.0 * cph * sph;  /* e^{2 i phi} */
    double on_re = cph, on_im = sph, sum_re = on_re, sum_im = on_im;
    for (int n = 1; n < 100000; ++n) {
        double fac = -f * (2.0 * n - (2.0 - t)) / (2.0 * n + (2.0 - t));
        double re = fac * (c2 * on_re - s2 * on_im), im = fac * (c2 * on_im + s2 * on_re);
        on_re = re; on_im = im;
        sum_re += re; sum_im += im;
        if (hypot(re, im) < 1e-18 * hypot(sum_re, sum_im)) break;
    }
    double pre = 2.0 * b / (1.0 + q) * pow(b / R, t - 1.0);
    double axp = pre * sum_re, ayp = pre * sum_im;
    *ax = axp * c - ayp * s;
    *ay = axp * s + ayp * c;
}

/* PAPER.md:160-162 Eq. 13, :187-190 Eq. 14: psi_ext = -1/2 gamma theta^2 cos 2(phi - phi_ext)
 * = -1/2 [gamma1 (x^2 - y^2) + 2 gamma2 x y] about the image origin (G4, G5);
 * alpha = grad psi_ext.                                                                   */
void orc_shear_deflection(double g1, double g2, double x, double y, double *ax, double *ay)
{
    *ax = -(g1 * x + g2 * y);
    *ay = -(g2 * x - g1 * y);
}

/* PAPER.md:133-137 Eq. 8 with R -> R_p of PAPER.md:141-150 Eq. 10. */
double orc_sersic(double i_e, double r_e, double n, double bn, double q, double phi,
                  double cx, double cy, double x, double y)
{
    double c = cos(phi), s = sin(phi);
    double x1 = (x - cx) * c + (y - cy) * s;
    double x2 = -(x - cx) * s + (y - cy) * c;
    double rp = sqrt(x1 * x1 * q + x2 * x2 / q);
    return i_e * exp(-bn * (pow(rp / r_e, 1.0 / n) - 1.0));
}

/* ------------------------------------------------------------------ validity (boundary rule)
 * include/tinylens.h: hypot(e1,e2) >= 1, theta_E < 0, r_e <= 0, n <= 0 or any non-finite
 * value makes the row physically invalid: logL = -inf, image = NaN.  EPL: also a slope outside
 * 1 < gamma < 3, where the deflection of Eq. 12 does not exist.                             */
int orc_row_valid(const orc_config *cfg, const float *row)
{
    int ncomp = cfg->n_lens_light + cfg->n_source;
    int LP = lens_np(cfg), P = LP + 7 * ncomp;
    for (int i = 0; i < P; ++i) if (!isfinite((double)row[i])) return 0;
    if (row[0] < 0.0f) return 0;
    if (hypot((double)row[1], (double)row[2]) >= 1.0) return 0;
    if (cfg->mass_model == ORC_MASS_EPL && !(row[7] > 1.0f && row[7] < 3.0f)) return 0;   /* 0 < t < 2 */
    for (int k = 0; k < ncomp; ++k) {
        const float *s = row + LP + 7 * k;
        if (!(s[1] > 0.0f) || !(s[2] > 0.0f)) return 0;
        if (hypot((double)s[3], (double)s[4]) >= 1.0) return 0;
    }
    return 1;
}

static int halo_of(const orc_config *cfg, int K) { return cfg->edge_mode == ORC_EDGE_EXTEND ? (K - 1) / 2 : 0; }

/* ------------------------------------------------------------------ Eq. 1, 2 + supersample + bin
 * Ideal (unblurred) image on the extended native grid (ny+2g) x (nx+2g), g = halo in EXTEND
 * mode, 0 in ZERO mode (G10).  Grid (G13): native pixel (i,j), i = row, centre
 *   x_j = (j - g - (nx-1)/2) s,  y_i = (i - g - (ny-1)/2) s,   s = pix_scale,
 * sub-sample (a,b): x = x_j + ((b+1/2)/S - 1/2) s, y = y_i + ((a+1/2)/S - 1/2) s.
 * Sample value (Eq. 2): sum of lens-light Sersics at theta plus source Sersics
 * at beta = theta - alpha (Eq. 1).  Native pixel = mean of S^2 samples
 * (G9).
 */
void orc_ideal_image(const orc_config *cfg, int g, const float *row, double *img)
{
    int S = cfg->supersample, ny = cfg->ny, nx = cfg->nx;
    int hy = ny + 2 * g, wx = nx + 2 * g;
    double s = cfg->pix_scale;
    double theta_e = row[0], q, phi;
    orc_shape(row[1], row[2], &q, &phi);
    double lcx = row[3], lcy = row[4], g1 = row[5], g2 = row[6];
    int ncomp = cfg->n_lens_light + cfg->n_source, LP = lens_np(cfg);
    int epl = cfg->mass_model == ORC_MASS_EPL;
    double slope = epl ? (double)row[7] : 2.0;
    double cq[8], cphi[8], cbn[8];
    for (int k = 0; k < ncomp && k < 8; ++k) {
        const float *c = row + LP + 7 * k;
        orc_shape(c[3], c[4], &cq[k], &cphi[k]);
        cbn[k] = orc_bn(c[2]);
    }
    for (int i = 0; i < hy; ++i) {
        double yi = (i - g - (ny - 1) / 2.0) * s;
        for (int j = 0; j < wx; ++j) {
            double xj = (j - g - (nx - 1) / 2.0) * s;
            double acc = 0.0;
            for (int a = 0; a < S; ++a) {
                double y = yi + ((a + 0.5) / S - 0.5) * s;
                for (int b = 0; b < S; ++b) {
                    double x = xj + ((b + 0.5) / S - 0.5) * s;
                    double ax, ay, sx, sy;
                    if (epl) orc_epl_deflection(theta_e, slope, q, phi, lcx, lcy, x, y, &ax, &ay);
                    else orc_sie_deflection(theta_e, q, phi, lcx, lcy, x, y, &ax, &ay);
                    orc_shear_deflection(g1, g2, x, y, &sx, &sy);
                    double bx = x - (ax + sx), by = y - (ay + sy);          /* Eq. 1 */
                    double v = 0.0;
                    for (int k = 0; k < ncomp; ++k) {
                        const float *c = row + LP + 7 * k;
                        int is_lens = k < cfg->n_lens_light;
                        v += orc_sersic(c[0], c[1], c[2], cbn[k], cq[k], cphi[k], c[5], c[6],
                                        is_lens ? x : bx, is_lens ? y : by);  /* Eq. 2 */
                    }
                    acc += v;
                }
            }
            img[(size_t)i * wx + j] = acc / (double)(S * S);
        }
    }
}

/* ------------------------------------------------------------------ Eq. 3: PSF convolution
 * PAPER.md:67-71 Eq. 3, true convolution, kernel used as given (G11):
 *   Im[i,j] = sum_{a,b} K[a,b] I[i-(a-h), j-(b-h)],  h = (K-1)/2,
 * I indexed in native pixels; img holds native index -g..n-1+g (g = h for EXTEND, so every
 * tap is inside; g = 0 for ZERO, taps outside the cutout read 0) (G10).
 */
void orc_convolve(int ny, int nx, int g, const double *img, const float *psf, int K, double *out)
{
    int h = (K - 1) / 2, wx = nx + 2 * g, hy = ny + 2 * g;
    for (int i = 0; i < ny; ++i)
        for (int j = 0; j < nx; ++j) {
            double acc = 0.0;
            for (int a = 0; a < K; ++a)
                for (int b = 0; b < K; ++b) {
                    int ii = i - (a - h) + g, jj = j - (b - h) + g;
                    if (ii < 0 || ii >= hy || jj < 0 || jj >= wx) continue;
                    acc += (double)psf[a * K + b] * img[(size_t)ii * wx + jj];
                }
            out[(size_t)i * nx + j] = acc;
        }
}

/* Whole forward model for one row: I^m [ny][nx].  Returns 0 for an invalid row
 * (image filled with NaN), 1 otherwise.                                                    */
int orc_render(const orc_config *cfg, const float *psf, int K, const float *row, double *image)
{
    size_t n = (size_t)cfg->ny * cfg->nx;
    if (!orc_row_valid(cfg, row)) { for (size_t i = 0; i < n; ++i) image[i] = NAN; return 0; }
    int g = halo_of(cfg, K);
    double *ext = (double *)malloc(sizeof(double) * (size_t)(cfg->ny + 2 * g) * (cfg->nx + 2 * g));
    orc_ideal_image(cfg, g, row, ext);
    orc_convolve(cfg->ny, cfg->nx, g, ext, psf, K, image);
    free(ext);
    return 1;
}

/* ------------------------------------------------------------------ Eq. 5: Gaussian likelihood
 * PAPER.md:80-84 Eq. 5: logL = -1/2 sum_i [ (d_i - Im_i)^2 / sigma_i^2 + ln(2 pi sigma_i^2) ]
 * (normalisation included, G12), Kahan-summed.                                             */
double orc_loglike_from_image(const double *image, const float *data, const float *noise, size_t n)
{
    double sum = 0.0, comp = 0.0;
    for (size_t i = 0; i < n; ++i) {
        double sg = noise[i], r = ((double)data[i] - image[i]) / sg;
        double t = r * r + log(2.0 * M_PI * sg * sg);
        double yk = t - comp, tk = sum + yk;
        comp = (tk - sum) - yk;
        sum = tk;
    }
    return -0.5 * sum;
}

double orc_chi2_from_image(const double *image, const float *data, const float *noise, size_t n)
{
    double sum = 0.0, comp = 0.0;
    for (size_t i = 0; i < n; ++i) {
        double r = ((double)data[i] - image[i]) / (double)noise[i];
        double yk = r * r - comp, tk = sum + yk;
        comp = (tk - sum) - yk;
        sum = tk;
    }
    return sum;
}

double orc_loglike(const orc_config *cfg, const float *psf, int K, const float *data,
                   const float *noise, const float *row)
{
    size_t n = (size_t)cfg->ny * cfg->nx;
    double *image = (double *)malloc(sizeof(double) * n);
    double r;
    if (!orc_render(cfg, psf, K, row, image)) r = -INFINITY;
    else r = orc_loglike_from_image(image, data, noise, n);
    free(image);
    return r;
}

/* ------------------------------------------------------------------ batches (rows independent)
 * n_lens > 1: psf/data/noise hold n_lens blocks, row r belongs to lens r / (B / n_lens).
 * OpenMP over rows; `threads` <= 0 means the OpenMP default.  Returns threads used.        */
int orc_loglike_batch(const orc_config *cfg, int n_lens, const float *psf, int K, const float *data,
                      const float *noise, const float *rows, int64_t B, double *logl, int threads)
{
    int P = lens_np(cfg) + 7 * (cfg->n_lens_light + cfg->n_source);
    size_t n = (size_t)cfg->ny * cfg->nx;
    int64_t per = B / (n_lens > 0 ? n_lens : 1);
    int used = 1;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < B; ++r) {
            int64_t l = n_lens > 1 ? r / per : 0;
            logl[r] = orc_loglike(cfg, psf + (size_t)l * K * K, K, data + l * n, noise + l * n,
                                  rows + r * P);
        }
    }
#else
    for (int64_t r = 0; r < B; ++r) {
        int64_t l = n_lens > 1 ? r / per : 0;
        logl[r] = orc_loglike(cfg, psf + (size_t)l * K * K, K, data + l * n, noise + l * n, rows + r * P);
    }
#endif
    return used;
}

int orc_render_batch(const orc_config *cfg, int n_lens, const float *psf, int K, const float *rows,
                     int64_t B, double *images, int threads)
{
    int P = lens_np(cfg) + 7 * (cfg->n_lens_light + cfg->n_source);
    size_t n = (size_t)cfg->ny * cfg->nx;
    int64_t per = B / (n_lens > 0 ? n_lens : 1);
    int used = 1;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < B; ++r) {
            int64_t l = n_lens > 1 ? r / per : 0;
            orc_render(cfg, psf + (size_t)l * K * K, K, rows + r * P, images + r * n);
        }
    }
#else
    for (int64_t r = 0; r < B; ++r) {
        int64_t l = n_lens > 1 ? r / per : 0;
        orc_render(cfg, psf + (size_t)l * K * K, K, rows + r * P, images + r * n);
    }
#endif
    return used;
}

/* ================================================================== NEXT-1: linear amplitudes
 * PAPER.md:86-93 Eq. 6 and :97-129 Eq. 7 (section 2.3): for given non-linear parameters the
 * amplitudes s of the N_l + N_s light profiles enter linearly, d = M s + n with M = B [L_l | L_s]
 * (column k = blurred image of component k at unit amplitude), and the likelihood is evaluated
 * at the s >= 0 that minimises || (M s - d) / n ||^2 (squared 2-norm).  The
 * paper solves this NNLS problem with the Bro & De Jong iteration; its result is the unique
 * minimiser of a convex problem, so the oracle writes the definition out: with at most three
 * components, every support set (which amplitudes are > 0) is tried, the normal equations are
 * solved on it, and the feasible candidate with the smallest penalty wins.  The I_e entries of
 * the row are ignored.
 */
int orc_component_images(const orc_config *cfg, const float *psf, int K, const float *row, double *M)
{
    int C = cfg->n_lens_light + cfg->n_source, LP = lens_np(cfg), P = LP + 7 * C;
    size_t n = (size_t)cfg->ny * cfg->nx;
    float tmp[8 + 7 * 8];
    for (int k = 0; k < C; ++k) {
        memcpy(tmp, row, sizeof(float) * (size_t)P);
        for (int j = 0; j < C; ++j) tmp[LP + 7 * j] = (j == k) ? 1.0f : 0.0f;     /* unit amplitude */
        if (!orc_render(cfg, psf, K, tmp, M + (size_t)k * n)) return 0;
    }
    return 1;
}

/* minimise s'G s - 2 b's over s >= 0 (n <= 4) by enumeration of the supports */
void orc_nnls_small(int n, const double *G, const double *b, double *s_out)
{
    double best = 0.0;                                   /* empty support: s = 0, penalty change 0 */
    for (int i = 0; i < n; ++i) s_out[i] = 0.0;
    for (int mask = 1; mask < (1 << n); ++mask) {
        int idx[4], m = 0;
        for (int i = 0; i < n; ++i) if (mask & (1 << i)) idx[m++] = i;
        double A[4][5];
        for (int r = 0; r < m; ++r) {
            for (int c = 0; c < m; ++c) A[r][c] = G[idx[r] * n + idx[c]];
            A[r][m] = b[idx[r]];
        }
        int singular = 0;
        for (int c = 0; c < m && !singular; ++c) {       /* Gaussian elimination, partial pivoting */
            int p = c;
            for (int r = c + 1; r < m; ++r) if (fabs(A[r][c]) > fabs(A[p][c])) p = r;
            if (!(fabs(A[p][c]) > 1e-300)) { singular = 1; break; }
            if (p != c) for (int k = 0; k <= m; ++k) { double t = A[c][k]; A[c][k] = A[p][k]; A[p][k] = t; }
            for (int r = c + 1; r < m; ++r) {
                double f = A[r][c] / A[c][c];
                for (int k = c; k <= m; ++k) A[r][k] -= f * A[c][k];
            }
        }
        if (singular) continue;
        double x[4];
        for (int r = m - 1; r >= 0; --r) {
            double t = A[r][m];
            for (int k = r + 1; k < m; ++k) t -= A[r][k] * x[k];
            x[r] = t / A[r][r];
        }
        int feasible = 1;
        double f = 0.0;
        for (int r = 0; r < m; ++r) { if (!(x[r] >= 0.0)) feasible = 0; f -= b[idx[r]] * x[r]; }
        if (feasible && f < best) {                      /* at a stationary point s'Gs - 2b's = -b's */
            best = f;
            for (int i = 0; i < n; ++i) s_out[i] = 0.0;
            for (int r = 0; r < m; ++r) s_out[idx[r]] = x[r];
        }
    }
}

double orc_loglike_linear(const orc_config *cfg, const float *psf, int K, const float *data,
                          const float *noise, const float *row, double *amps)
{
    int C = cfg->n_lens_light + cfg->n_source;
    size_t n = (size_t)cfg->ny * cfg->nx;
    for (int k = 0; k < C; ++k) if (amps) amps[k] = NAN;
    /* the amplitudes are not parameters here: validity is judged with them set to one */
    float tmp[8 + 7 * 8];
    memcpy(tmp, row, sizeof(float) * (size_t)(lens_np(cfg) + 7 * C));
    for (int j = 0; j < C; ++j) tmp[lens_np(cfg) + 7 * j] = 1.0f;
    if (!orc_row_valid(cfg, tmp)) return -INFINITY;
    double *M = (double *)malloc(sizeof(double) * n * (size_t)C);
    double *model = (double *)malloc(sizeof(double) * n);
    orc_component_images(cfg, psf, K, tmp, M);
    double G[16], b[4], s[4];
    for (int k = 0; k < C; ++k) {
        double bk = 0.0;
        for (size_t i = 0; i < n; ++i) bk += M[k * n + i] * (double)data[i] / ((double)noise[i] * noise[i]);
        b[k] = bk;
        for (int l = 0; l < C; ++l) {
            double g = 0.0;
            for (size_t i = 0; i < n; ++i) g += M[k * n + i] * M[l * n + i] / ((double)noise[i] * noise[i]);
            G[k * C + l] = g;
        }
    }
    orc_nnls_small(C, G, b, s);
    for (size_t i = 0; i < n; ++i) {
        double m = 0.0;
        for (int k = 0; k < C; ++k) m += s[k] * M[k * n + i];
        model[i] = m;
    }
    double ll = orc_loglike_from_image(model, data, noise, n);     /* Eq. 5 at the optimal amplitudes (Eq. 6) */
    if (amps) for (int k = 0; k < C; ++k) amps[k] = s[k];
    free(M); free(model);
    return ll;
}

int orc_loglike_linear_batch(const orc_config *cfg, int n_lens, const float *psf, int K, const float *data,
                             const float *noise, const float *rows, int64_t B, double *logl, double *amps, int threads)
{
    int C = cfg->n_lens_light + cfg->n_source, LP = lens_np(cfg), P = LP + 7 * C;
    size_t n = (size_t)cfg->ny * cfg->nx;
    int64_t per = B / (n_lens > 0 ? n_lens : 1);
    int used = 1;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < B; ++r) {
            int64_t l = n_lens > 1 ? r / per : 0;
            logl[r] = orc_loglike_linear(cfg, psf + (size_t)l * K * K, K, data + l * n, noise + l * n,
                                         rows + r * P, amps ? amps + r * C : NULL);
        }
    }
#else
    for (int64_t r = 0; r < B; ++r) {
        int64_t l = n_lens > 1 ? r / per : 0;
        logl[r] = orc_loglike_linear(cfg, psf + (size_t)l * K * K, K, data + l * n, noise + l * n,
                                     rows + r * P, amps ? amps + r * C : NULL);
    }
#endif
    return used;
}

/* ================================================================== NEXT-3: MGE lens light
 * PAPER.md:291-293 (section 4.3): "we have implemented the Multiple Gaussian Expansion (MGE)
 * model, which can describe arbitrary radial profiles ... in lens galaxies".  The paper gives
 * no formula; reading G23: the lens light is a sum of n_g elliptical Gaussians on
 * the ellipses R_p of PAPER.md:143-148 Eq. 10, sharing one centre and one (q, phi),
 *     I_l(theta) = sum_k a_k exp( -R_p(theta)^2 / (2 sigma_k^2) ),
 * with fixed dispersions sigma_k (arcsec) and amplitudes a_k >= 0 that are linear parameters
 * (PAPER.md:86-93 Eq. 6, :97-129 Eq. 7): together with the N_s source amplitudes they are the
 * non-negative least-squares minimiser of || (M s - d) / n ||^2, M = B [G_1 .. G_ng | L_s],
 * and logL is Eq. 5 at that optimum.
 *
 * The row is the usual one with n_lens_light = 1; of the lens-light block only e1, e2, cx, cy
 * (entries 3..6) are read -- I_e, r_e, n (0..2) are ignored.  The I_e of the sources is ignored
 * too (as in orc_loglike_linear).
 *
 * NNLS by its definition, as orc_nnls_small: every support is tried, the normal equations are
 * solved on it, and of the feasible candidates the one with the smallest penalty
 * s'Gs - 2b's (evaluated explicitly) wins.  2^n supports: the oracle takes n <= 16 columns.
 */
#define ORC_MGE_MAXCOL 16

/* one elliptical Gaussian of unit central brightness on the ellipses of Eq. 10 */
double orc_gauss(double sigma, double q, double phi, double cx, double cy, double x, double y)
{
    double c = cos(phi), s = sin(phi);
    double x1 = (x - cx) * c + (y - cy) * s;
    double x2 = -(x - cx) * s + (y - cy) * c;
    double rp2 = x1 * x1 * q + x2 * x2 / q;
    return exp(-rp2 / (2.0 * sigma * sigma));
}

/* validity for the MGE call: lens block and sources as orc_row_valid (source I_e ignored),
 * lens-light block: only its shape and centre are read                                    */
int orc_mge_row_valid(const orc_config *cfg, const float *row)
{
    if (cfg->n_lens_light != 1) return 0;
    int LP = lens_np(cfg), ncomp = 1 + cfg->n_source;
    for (int i = 0; i < LP; ++i) if (!isfinite((double)row[i])) return 0;
    if (row[0] < 0.0f) return 0;
    if (hypot((double)row[1], (double)row[2]) >= 1.0) return 0;
    if (cfg->mass_model == ORC_MASS_EPL && !(row[7] > 1.0f && row[7] < 3.0f)) return 0;
    const float *l = row + LP;
    for (int i = 3; i < 7; ++i) if (!isfinite((double)l[i])) return 0;
    if (hypot((double)l[3], (double)l[4]) >= 1.0) return 0;
    for (int k = 1; k < ncomp; ++k) {
        const float *s = row + LP + 7 * k;
        for (int i = 1; i < 7; ++i) if (!isfinite((double)s[i])) return 0;
        if (!(s[1] > 0.0f) || !(s[2] > 0.0f)) return 0;
        if (hypot((double)s[3], (double)s[4]) >= 1.0) return 0;
    }
    return 1;
}

/* columns of M: n_gauss blurred unit-amplitude Gaussians, then the N_s blurred unit-amplitude
 * sources.  M[(n_gauss + n_source)][ny*nx].  Returns 0 for an invalid row.                  */
int orc_mge_component_images(const orc_config *cfg, const float *psf, int K, const float *row,
                             const float *sigmas, int n_gauss, double *M)
{
    if (!orc_mge_row_valid(cfg, row)) return 0;
    int LP = lens_np(cfg), S = cfg->supersample, ny = cfg->ny, nx = cfg->nx;
    size_t n = (size_t)ny * nx;
    int g = halo_of(cfg, K), hy = ny + 2 * g, wx = nx + 2 * g;
    double s = cfg->pix_scale, q, phi;
    const float *l = row + LP;
    orc_shape(l[3], l[4], &q, &phi);
    double *ext = (double *)malloc(sizeof(double) * (size_t)hy * wx);
    for (int k = 0; k < n_gauss; ++k) {
        for (int i = 0; i < hy; ++i) {
            double yi = (i - g - (ny - 1) / 2.0) * s;
            for (int j = 0; j < wx; ++j) {
                double xj = (j - g - (nx - 1) / 2.0) * s;
                double acc = 0.0;
                for (int a = 0; a < S; ++a) {
                    double y = yi + ((a + 0.5) / S - 0.5) * s;
                    for (int b = 0; b < S; ++b) {
                        double x = xj + ((b + 0.5) / S - 0.5) * s;
                        acc += orc_gauss((double)sigmas[k], q, phi, l[5], l[6], x, y);
                    }
                }
                ext[(size_t)i * wx + j] = acc / (double)(S * S);             /* bin: mean */
            }
        }
        orc_convolve(ny, nx, g, ext, psf, K, M + (size_t)k * n);            /* Eq. 3 */
    }
    free(ext);
    /* sources through the plain forward model: a harmless lens-light Sersic of amplitude 0 */
    float tmp[8 + 7 * 8];
    int P = LP + 7 * (1 + cfg->n_source);
    for (int ks = 0; ks < cfg->n_source; ++ks) {
        memcpy(tmp, row, sizeof(float) * (size_t)P);
        tmp[LP + 0] = 0.0f; tmp[LP + 1] = 1.0f; tmp[LP + 2] = 1.0f;
        for (int j = 0; j < cfg->n_source; ++j) tmp[LP + 7 * (1 + j)] = (j == ks) ? 1.0f : 0.0f;
        if (!orc_render(cfg, psf, K, tmp, M + (size_t)(n_gauss + ks) * n)) return 0;
    }
    return 1;
}

/* minimise s'G s - 2 b's over s >= 0, n <= ORC_MGE_MAXCOL, by enumeration of the supports */
void orc_nnls_enum(int n, const double *G, const double *b, double *s_out)
{
    double best = 0.0;                                   /* empty support: s = 0 */
    for (int i = 0; i < n; ++i) s_out[i] = 0.0;
    if (n > ORC_MGE_MAXCOL) { for (int i = 0; i < n; ++i) s_out[i] = NAN; return; }
    for (long mask = 1; mask < (1L << n); ++mask) {
        int idx[ORC_MGE_MAXCOL], m = 0;
        for (int i = 0; i < n; ++i) if (mask & (1L << i)) idx[m++] = i;
        double A[ORC_MGE_MAXCOL][ORC_MGE_MAXCOL + 1];
        for (int r = 0; r < m; ++r) {
            for (int c = 0; c < m; ++c) A[r][c] = G[idx[r] * n + idx[c]];
            A[r][m] = b[idx[r]];
        }
        int singular = 0;
        for (int c = 0; c < m && !singular; ++c) {       /* Gaussian elimination, partial pivoting */
            int p = c;
            for (int r = c + 1; r < m; ++r) if (fabs(A[r][c]) > fabs(A[p][c])) p = r;
            if (!(fabs(A[p][c]) > 1e-300)) { singular = 1; break; }
            if (p != c) for (int k = 0; k <= m; ++k) { double t = A[c][k]; A[c][k] = A[p][k]; A[p][k] = t; }
            for (int r = c + 1; r < m; ++r) {
                double f = A[r][c] / A[c][c];
                for (int k = c; k <= m; ++k) A[r][k] -= f * A[c][k];
            }
        }
        if (singular) continue;
        double x[ORC_MGE_MAXCOL];
        int feasible = 1;
        for (int r = m - 1; r >= 0; --r) {
            double t = A[r][m];
            for (int k = r + 1; k < m; ++k) t -= A[r][k] * x[k];
            x[r] = t / A[r][r];
        }
        for (int r = 0; r < m; ++r) if (!(x[r] >= 0.0)) feasible = 0;
        if (!feasible) continue;
        double f = 0.0;                                  /* the penalty itself, not its stationary form */
        for (int r = 0; r < m; ++r) {
            double gx = 0.0;
            for (int c = 0; c < m; ++c) gx += G[idx[r] * n + idx[c]] * x[c];
            f += x[r] * (gx - 2.0 * b[idx[r]]);
        }
        if (f < best) {
            best = f;
            for (int i = 0; i < n; ++i) s_out[i] = 0.0;
            for (int r = 0; r < m; ++r) s_out[idx[r]] = x[r];
        }
    }
}

double orc_loglike_mge(const orc_config *cfg, const float *psf, int K, const float *data, const float *noise,
                       const float *row, const float *sigmas, int n_gauss, double *amps)
{
    int C = n_gauss + cfg->n_source;
    size_t n = (size_t)cfg->ny * cfg->nx;
    for (int k = 0; k < C; ++k) if (amps) amps[k] = NAN;
    if (C > ORC_MGE_MAXCOL || !orc_mge_row_valid(cfg, row)) return -INFINITY;
    double *M = (double *)malloc(sizeof(double) * n * (size_t)C);
    double *model = (double *)malloc(sizeof(double) * n);
    orc_mge_component_images(cfg, psf, K, row, sigmas, n_gauss, M);
    double G[ORC_MGE_MAXCOL * ORC_MGE_MAXCOL], b[ORC_MGE_MAXCOL], s[ORC_MGE_MAXCOL];
    for (int k = 0; k < C; ++k) {
        double bk = 0.0;
        for (size_t i = 0; i < n; ++i) bk += M[k * n + i] * (double)data[i] / ((double)noise[i] * noise[i]);
        b[k] = bk;
        for (int l = 0; l < C; ++l) {
            double gg = 0.0;
            for (size_t i = 0; i < n; ++i) gg += M[k * n + i] * M[l * n + i] / ((double)noise[i] * noise[i]);
            G[k * C + l] = gg;
        }
    }
    orc_nnls_enum(C, G, b, s);
    for (size_t i = 0; i < n; ++i) {
        double m = 0.0;
        for (int k = 0; k < C; ++k) m += s[k] * M[k * n + i];
        model[i] = m;
    }
    double ll = orc_loglike_from_image(model, data, noise, n);     /* Eq. 5 at the optimal amplitudes (Eq. 6) */
    if (amps) for (int k = 0; k < C; ++k) amps[k] = s[k];
    free(M); free(model);
    return ll;
}

int orc_loglike_mge_batch(const orc_config *cfg, int n_lens, const float *psf, int K, const float *data,
                          const float *noise, const float *rows, int64_t B, const float *sigmas, int n_gauss,
                          double *logl, double *amps, int threads)
{
    int C = n_gauss + cfg->n_source, P = lens_np(cfg) + 7 * (1 + cfg->n_source);
    size_t n = (size_t)cfg->ny * cfg->nx;
    int64_t per = B / (n_lens > 0 ? n_lens : 1);
    int used = 1;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < B; ++r) {
            int64_t l = n_lens > 1 ? r / per : 0;
            logl[r] = orc_loglike_mge(cfg, psf + (size_t)l * K * K, K, data + l * n, noise + l * n,
                                      rows + r * P, sigmas, n_gauss, amps ? amps + r * C : NULL);
        }
    }
#else
    for (int64_t r = 0; r < B; ++r) {
        int64_t l = n_lens > 1 ? r / per : 0;
        logl[r] = orc_loglike_mge(cfg, psf + (size_t)l * K * K, K, data + l * n, noise + l * n,
                                  rows + r * P, sigmas, n_gauss, amps ? amps + r * C : NULL);
    }
#endif
    return used;
}
