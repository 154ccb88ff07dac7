/*
 * jpet_oracle.c - plain fp64 CPU oracle for the list-mode MLEM iteration of arXiv:1502.07478
 * ("GPU accelerated image reconstruction in a two-strip J-PET tomograph").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header, table or
 * helper with paper_1502_07478_b200/csrc (the CUDA path) and neither includes the other.
 *
 * It is written to be checked against the paper by eye: every function cites the passage it follows and
 * uses the paper's notation (tilde quantities carry the suffix _t).  No blocking, fusion, factoring of
 * common sub-expressions across pixels, or reordering beyond what the paper states.  The only
 * parallelism is the paper's own CPU scheme: OpenMP over events, one private rho_new per thread, summed
 * after the loop.
 *
 * Readings of the paper where it is garbled or silent are the R-numbers of SURVEY.md section 8(c),
 * listed again in DESIGN.md ("Readings").  Pins for every function: tests/test_oracle_*.py.
 * Parity status: all functions pinned (none "parity unpinned"); what stays unpinned is only whether
 * Eq. 7 models the real detector, which no synthetic test can decide.
 *
 * Geometry: image plane (y, z); strips are the segments y = +R ("u") and y = -R ("d"), |z| <= L/2
 * (PAPER.md:34-40, :52, :77).  Lengths in mm.  Pixel (iy, iz) has its centre at
 *   y = (iy - (n_y-1)/2) * pixel,  z = (iz - (n_z-1)/2) * pixel     (row-major, z fastest).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define JO_PI 3.14159265358979323846264338327950288

/* ---- pixel centres (SURVEY.md 8(b) grid convention; "center of pixel i") ---------------- */
static double jo_pixel_y(int iy, int n_y, double pixel) { return ((double)iy - 0.5 * (double)(n_y - 1)) * pixel; }
static double jo_pixel_z(int iz, int n_z, double pixel) { return ((double)iz - 0.5 * (double)(n_z - 1)) * pixel; }

/* ---- Eq. 1: path difference of an emission at (e_y, e_z) whose photons hit z_u, z_d ----- */
double jo_eq1_delta_l(double e_y, double e_z, double z_u, double z_d, double R)
{
    return sqrt((R - e_y) * (R - e_y) + (z_u - e_z) * (z_u - e_z))
         - sqrt((R + e_y) * (R + e_y) + (z_d - e_z) * (z_d - e_z));
}

/* ---- Eq. 2, first forms; R-bar == R (R1), the "y" in the z~ line is y~ (R3) ---------
 * out = { tan(theta~), y~, z~ }                                                                         */
void jo_eq2(double z_u_t, double z_d_t, double dl_t, double R, double out[3])
{
    double tan_t = (z_u_t - z_d_t) / (2.0 * R);
    double y_t = -0.5 * dl_t / sqrt(1.0 + tan_t * tan_t);
    double z_t = 0.5 * (z_u_t + z_d_t + 2.0 * y_t * tan_t);
    out[0] = tan_t;
    out[1] = y_t;
    out[2] = z_t;
}

/* ---- Eq. 4: sensitivity of the point (y, z); negative values (points no LOR through
 * both strips can see) are clamped to 0 (R13).                                                          */
double jo_sensitivity(double y, double z, double R, double L)
{
    double hi1 = (0.5 * L - z) / (R - y);
    double hi2 = (0.5 * L + z) / (R + y);
    double lo1 = -(0.5 * L + z) / (R - y);
    double lo2 = (-0.5 * L + z) / (R + y);
    double s = (atan(fmin(hi1, hi2)) - atan(fmax(lo1, lo2))) / JO_PI;
    return s > 0.0 ? s : 0.0;
}

void jo_sensitivity_image(double R, double L, int n_y, int n_z, double pixel, double *s)
{
    for (int iy = 0; iy < n_y; ++iy)
        for (int iz = 0; iz < n_z; ++iz)
            s[(size_t)iy * n_z + iz] = jo_sensitivity(jo_pixel_y(iy, n_y, pixel), jo_pixel_z(iz, n_z, pixel), R, L);
}

/* ---- Eq. 12: the off-diagonal coefficient gamma of C^-1 --------------
 * The paper prints the general form and then sets gamma = 0; 0 is the default here too.
 * A process-wide setting, like the a3 coefficient of the tests: set it before an iteration, not during one. */
static double jo_gamma = 0.0;
void jo_set_gamma(double gamma) { jo_gamma = gamma; }
double jo_get_gamma(void) { return jo_gamma; }

/* ---- sigma_z as a function of the hit position (reading R22) ---------------------
 * C^-1 "depends on the z~u and z~d ... Experimentally we have found this dependence to be quite weak
 * on the order of 10% from the center (lowest) to the edge (highest)".  The paper gives no functional form; the
 * reading is  sigma_z(z) = sigma_z (1 + eta min(1, (2 z / L)^2)):  lowest at the strip centre, (1 + eta) sigma_z at
 * and beyond the strip ends, eta = 0.1 for the paper's 10 %.  eta = 0 (default) is the constant sigma_z the paper
 * works with.  Process-wide like gamma.                                                                      */
static double jo_sz_eta = 0.0;
void jo_set_sigma_z_edge(double eta) { jo_sz_eta = eta; }
double jo_get_sigma_z_edge(void) { return jo_sz_eta; }

double jo_sigma_z_at(double z_hit, double L, double sigma_z)
{
    double q = 2.0 * z_hit / L;
    q = q * q;
    if (q > 1.0) q = 1.0;
    return sigma_z * (1.0 + jo_sz_eta * q);
}

/* ---- Eq. 12 for one event: 1/sigma_z^2 taken at the event's own hit positions ------------------ */
void jo_cinv(double z_u_t, double z_d_t, double L, double sigma_z, double sigma_dl, double Cinv[3][3])
{
    double su = jo_sigma_z_at(z_u_t, L, sigma_z), sd = jo_sigma_z_at(z_d_t, L, sigma_z);
    const double g = jo_gamma;
    Cinv[0][0] = 1.0 / (su * su); Cinv[0][1] = 0.0;             Cinv[0][2] = g;
    Cinv[1][0] = 0.0;             Cinv[1][1] = 1.0 / (sd * sd); Cinv[1][2] = -g;
    Cinv[2][0] = g;               Cinv[2][1] = -g;              Cinv[2][2] = 1.0 / (sigma_dl * sigma_dl);
}

/* b of Eq. 10 for a pixel at offset (dy, dz) from the reconstructed point */
static void jo_vec_b(double dy, double dz, double tan_t, double b[3])
{
    double icos = sqrt(1.0 + tan_t * tan_t);
    b[0] = dz - dy * tan_t;
    b[1] = dz - dy * tan_t;
    b[2] = -2.0 * dy * icos;
}

/* b C^-1 b with the full matrix ("this term defines an 3 sigma ellipse") */
double jo_bCb_c(double dy, double dz, double tan_t, const double Cinv[3][3])
{
    double b[3], q = 0.0;
    jo_vec_b(dy, dz, tan_t, b);
    for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l) q += b[k] * Cinv[k][l] * b[l];
    return q;
}

/* ---- b C^-1 b (first line of B.3) ------------------------------------------------------
 * b = (u, u, -2 dy / cos) has equal first and second components (Eq. 10), so the gamma terms of Eq. 12,
 * 2 gamma (b1 - b2) b3, vanish: B.3 and the 3-sigma ellipse do not depend on gamma.                      */
double jo_bCb(double dy, double dz, double tan_t, double sigma_z, double sigma_dl)
{
    double cos2 = 1.0 / (1.0 + tan_t * tan_t);
    double u = dz - dy * tan_t;
    return 2.0 * u * u / (sigma_z * sigma_z) + 4.0 * dy * dy / (sigma_dl * sigma_dl * cos2);
}

/* ---- Eq. 7-12: reconstruction kernel P(e~ | pixel at (y, z)) ----------------------
 * Vectors o, a, b are Eq. 8, 9, 10 written out; C^-1 is the matrix of Eq. 12 with gamma = jo_gamma (0 unless
 * set: the paper's diagonal case).  a3_coef multiplies the third component of a: 2 gives a = d e/d theta (default, R5),
 * 1 gives Eq. 9 exactly as printed.  Prefactor: det^(1/2) of the INVERSE covariance over 2 pi^2 (R4).
 * No truncation here: the 3-sigma rule is applied by the caller.                                        */
double jo_kernel_c(double y, double z, double tan_t, double y_t, double z_t, double R, const double Cinv[3][3], double a3_coef)
{
    double dy = y - y_t;                       /* Eq. 11 */
    double dz = z - z_t;
    double icos = sqrt(1.0 + tan_t * tan_t);   /* cos^-1(theta~) */
    double icos2 = icos * icos;                /* cos^-2(theta~) */

    double o[3], a[3], b[3];
    o[0] = -(dy + y_t - R) * tan_t * icos2;                       /* Eq. 8 */
    o[1] = -(dy + y_t + R) * tan_t * icos2;
    o[2] = -(dy + y_t) * icos * (1.0 + 2.0 * tan_t * tan_t);
    a[0] = -(dy + y_t - R) * icos2;                               /* Eq. 9 */
    a[1] = -(dy + y_t + R) * icos2;
    a[2] = -a3_coef * (dy + y_t) * icos * tan_t;
    b[0] = dz - dy * tan_t;                                       /* Eq. 10 */
    b[1] = dz - dy * tan_t;
    b[2] = -2.0 * dy * icos;

    double aCa = 0.0, oCb = 0.0, bCb = 0.0, bCa = 0.0;
    for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l) {
            aCa += a[k] * Cinv[k][l] * a[l];
            oCb += o[k] * Cinv[k][l] * b[l];
            bCb += b[k] * Cinv[k][l] * b[l];
            bCa += b[k] * Cinv[k][l] * a[l];
        }
    double D = aCa + 2.0 * oCb;
    if (!(D > 0.0)) return 0.0;                                   /* R17 */
    double det_Cinv = Cinv[0][0] * (Cinv[1][1] * Cinv[2][2] - Cinv[1][2] * Cinv[2][1])
                    - Cinv[0][1] * (Cinv[1][0] * Cinv[2][2] - Cinv[1][2] * Cinv[2][0])
                    + Cinv[0][2] * (Cinv[1][0] * Cinv[2][1] - Cinv[1][1] * Cinv[2][0]);
    if (!(det_Cinv > 0.0)) return 0.0;                             /* gamma too large: C^-1 not positive definite */
    double sqrt_det_Cinv = sqrt(det_Cinv);
    return sqrt_det_Cinv / (2.0 * JO_PI * JO_PI * sqrt(D)) * exp(-0.5 * (bCb - bCa * bCa / D));   /* Eq. 7 */
}

/* the same with the constant matrix of Eq. 12: sigma_z everywhere, gamma = jo_gamma */
double jo_kernel(double y, double z, double tan_t, double y_t, double z_t,
                 double R, double sigma_z, double sigma_dl, double a3_coef)
{
    const double g = jo_gamma;
    double Cinv[3][3] = { { 1.0 / (sigma_z * sigma_z), 0.0, g },                     /* Eq. 12 */
                          { 0.0, 1.0 / (sigma_z * sigma_z), -g },
                          { g, -g, 1.0 / (sigma_dl * sigma_dl) } };
    return jo_kernel_c(y, z, tan_t, y_t, z_t, R, Cinv, a3_coef);
}

/* ---- the integral that Eq. 7 approximates (reading R15: emission angle uniform on (-pi/2, pi/2)) ------
 *   P_exact(e~ | y, z) = int dtheta / pi  N(e~; e(y, z, theta), C),
 * e(y, z, theta) = (z + (R - y) tan, z - (R + y) tan, -2 y / cos): where the photons of an emission at (y, z) along theta
 * hit the strips and their path difference (Eq. 1 on the LOR); N the normal density with inverse
 * covariance Cinv.  Composite trapezoid rule with n_theta nodes over the open interval.  e_t = (z_u~, z_d~, dl~).  */
double jo_kernel_exact(double y, double z, const double e_t[3], double R, const double Cinv[3][3], int n_theta)
{
    double det_Cinv = Cinv[0][0] * (Cinv[1][1] * Cinv[2][2] - Cinv[1][2] * Cinv[2][1])
                    - Cinv[0][1] * (Cinv[1][0] * Cinv[2][2] - Cinv[1][2] * Cinv[2][0])
                    + Cinv[0][2] * (Cinv[1][0] * Cinv[2][1] - Cinv[1][1] * Cinv[2][0]);
    if (!(det_Cinv > 0.0) || n_theta < 2) return 0.0;
    const double norm = sqrt(det_Cinv) / pow(2.0 * JO_PI, 1.5);
    const double lo = -0.5 * JO_PI + 1e-9, hi = 0.5 * JO_PI - 1e-9, h = (hi - lo) / (double)(n_theta - 1);
    double sum = 0.0;
    for (int k = 0; k < n_theta; ++k) {
        double theta = lo + h * (double)k;
        double e[3] = { z + (R - y) * tan(theta), z - (R + y) * tan(theta), -2.0 * y / cos(theta) };
        double d[3] = { e[0] - e_t[0], e[1] - e_t[1], e[2] - e_t[2] };
        double chi2 = 0.0;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) chi2 += d[a] * Cinv[a][b] * d[b];
        double f = norm * exp(-0.5 * chi2);
        sum += (k == 0 || k == n_theta - 1) ? 0.5 * f : f;
    }
    return sum * h / JO_PI;
}

static int jo_exact_nodes = 0;          /* > 0: jo_mlem_iterate uses jo_kernel_exact with that many nodes instead of Eq. 7 */
void jo_set_exact_kernel(int n_theta) { jo_exact_nodes = n_theta; }
int jo_get_exact_kernel(void) { return jo_exact_nodes; }

/* ---- convenience for quadrature tests: P(e~_j | pixel (y, z)) for many events (double [n][3]) ---------
 * Eq. 2 then Eq. 7 per event; inside3s[j] = 1 when the pixel centre is inside event j's 3-sigma ellipse. */
void jo_kernel_events(const double *events, int64_t n, double y, double z, double R, double sigma_z,
                      double sigma_dl, double a3_coef, double *P_out, unsigned char *inside3s)
{
    for (int64_t j = 0; j < n; ++j) {
        double e[3];
        jo_eq2(events[3 * j + 0], events[3 * j + 1], events[3 * j + 2], R, e);
        P_out[j] = jo_kernel(y, z, e[0], e[1], e[2], R, sigma_z, sigma_dl, a3_coef);
        if (inside3s) inside3s[j] = jo_bCb(y - e[1], z - e[2], e[0], sigma_z, sigma_dl) <= 9.0;
    }
}

/* ---- Appendix B: circumscribed half-extents of the 3-sigma ellipse ----------------
 * Ellipse A dy^2 + 2 C dy dz + B dz^2 = 3^2 with A, B, C read off B.3 (R8, R9).  out = { h_y, h_z }.   */
void jo_bbox_half_extents(double tan_t, double sigma_z, double sigma_dl, double out[2])
{
    double icos2 = 1.0 + tan_t * tan_t;
    double A = 2.0 * tan_t * tan_t / (sigma_z * sigma_z) + 4.0 * icos2 / (sigma_dl * sigma_dl);
    double B = 2.0 / (sigma_z * sigma_z);
    double C = -2.0 * tan_t / (sigma_z * sigma_z);
    out[0] = 3.0 / sqrt(A - C * C / B);                            /* B.2 */
    out[1] = 3.0 / sqrt(B - C * C / A);
}

/* the same for a general matrix: A, B, C of the ellipse A dy^2 + 2 C dy dz + B dz^2 = 9 read off the quadratic form
 * b C^-1 b itself (B.3 is that form written out for the constant diagonal matrix) */
void jo_bbox_half_extents_c(double tan_t, const double Cinv[3][3], double out[2])
{
    double A = jo_bCb_c(1.0, 0.0, tan_t, Cinv);
    double B = jo_bCb_c(0.0, 1.0, tan_t, Cinv);
    double C = 0.5 * (jo_bCb_c(1.0, 1.0, tan_t, Cinv) - A - B);
    out[0] = 3.0 / sqrt(A - C * C / B);                            /* B.2 */
    out[1] = 3.0 / sqrt(B - C * C / A);
}

/* ---- Listing 1 with Eq. 3's s(i) in the denominator (R11, R12) --------------------
 * One MLEM iteration.
 *   events   : float32 [n][3] = (z_u~, z_d~, dl~), the very array the GPU gets, widened to double here
 *   rho_in   : double [n_y*n_z];  rho_out: double [n_y*n_z]
 *   brute    : 0 = loop over the clipped bounding box (Listing 1), 1 = scan the whole image; both apply
 *              the same centre-in-ellipse test  b C^-1 b <= 9  (R8, R10) and must agree
 *   counters : n_evals = sum over events of |ellipse(e_j)|, n_skipped = events with an empty pixel set
 *              or a non-positive / non-finite denominator (R16)
 * Steps (SURVEY.md 8(c) algorithm):  w = s*rho;  per event: Eq. 2, pixel set, P, denominator = sum P*w,
 * rho_new[i] += P_i / denominator;  finally rho_out = rho_in * rho_new where s > 0, else 0.
 * Returns 0, or -1 on allocation failure / bad arguments.                                               */
int jo_mlem_iterate(const float *events, int64_t n, double R, double L, double sigma_z, double sigma_dl,
                    int n_y, int n_z, double pixel, double a3_coef, const double *rho_in, double *rho_out,
                    int brute, int n_threads, uint64_t *n_evals_out, uint64_t *n_skipped_out)
{
    if (n < 0 || n_y <= 0 || n_z <= 0 || !(pixel > 0.0) || !rho_in || !rho_out || (n > 0 && !events)) return -1;
    const size_t M = (size_t)n_y * (size_t)n_z;
    double *s = (double *)malloc(M * sizeof(double));
    double *w = (double *)malloc(M * sizeof(double));
    if (!s || !w) { free(s); free(w); return -1; }
    jo_sensitivity_image(R, L, n_y, n_z, pixel, s);
    for (size_t i = 0; i < M; ++i) w[i] = s[i] * rho_in[i];

#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
#else
    n_threads = 1;
#endif
    double *rho_new_all = (double *)calloc(M * (size_t)n_threads, sizeof(double));   /* Listing 1 lines 1-3 */
    if (!rho_new_all) { free(s); free(w); return -1; }
    uint64_t n_evals = 0, n_skipped = 0;
    int failed = 0;

#ifdef _OPENMP
#pragma omp parallel num_threads(n_threads) reduction(+ : n_evals, n_skipped) reduction(| : failed)
#endif
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        double *rho_new = rho_new_all + (size_t)tid * M;           /* private copy */
        size_t cap = 1024;
        double *kernel = (double *)malloc(cap * sizeof(double));    /* Listing 1: kernel[i] cache */
        int *pix = (int *)malloc(cap * sizeof(int));
        if (!kernel || !pix) failed = 1;

#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t j = 0; j < n; ++j) {                           /* Listing 1 line 4 */
            if (failed) continue;
            double e[3];
            jo_eq2((double)events[3 * j + 0], (double)events[3 * j + 1], (double)events[3 * j + 2], R, e);
            double tan_t = e[0], y_t = e[1], z_t = e[2];
            if (!isfinite(tan_t) || !isfinite(y_t) || !isfinite(z_t)) { n_skipped++; continue; }
            double e_t[3] = { (double)events[3 * j + 0], (double)events[3 * j + 1], (double)events[3 * j + 2] };
            double Cinv[3][3];
            jo_cinv(e_t[0], e_t[1], L, sigma_z, sigma_dl, Cinv);     /* Eq. 12 at this event's hit positions */

            int iy0 = 0, iy1 = n_y - 1, iz0 = 0, iz1 = n_z - 1;
            if (!brute) {                                           /* bounding box in pixel space */
                double h[2];
                jo_bbox_half_extents_c(tan_t, Cinv, h);
                double fy0 = ceil((y_t - h[0]) / pixel + 0.5 * (double)(n_y - 1));
                double fy1 = floor((y_t + h[0]) / pixel + 0.5 * (double)(n_y - 1));
                double fz0 = ceil((z_t - h[1]) / pixel + 0.5 * (double)(n_z - 1));
                double fz1 = floor((z_t + h[1]) / pixel + 0.5 * (double)(n_z - 1));
                if (fy0 > (double)iy0) iy0 = fy0 > (double)n_y ? n_y : (int)fy0;
                if (fy1 < (double)iy1) iy1 = fy1 < -1.0 ? -1 : (int)fy1;
                if (fz0 > (double)iz0) iz0 = fz0 > (double)n_z ? n_z : (int)fz0;
                if (fz1 < (double)iz1) iz1 = fz1 < -1.0 ? -1 : (int)fz1;
            }

            double denominator = 0.0;                               /* Listing 1 line 5 */
            size_t cnt = 0;
            for (int iy = iy0; iy <= iy1; ++iy) {                   /* Listing 1 line 6 */
                for (int iz = iz0; iz <= iz1; ++iz) {
                    double y = jo_pixel_y(iy, n_y, pixel), z = jo_pixel_z(iz, n_z, pixel);
                    if (!(jo_bCb_c(y - y_t, z - z_t, tan_t, Cinv) <= 9.0)) continue;   /* centre inside 3 sigma */
                    if (cnt == cap) {
                        cap *= 2;
                        double *k2 = (double *)realloc(kernel, cap * sizeof(double));
                        int *p2 = (int *)realloc(pix, cap * sizeof(int));
                        if (k2) kernel = k2;
                        if (p2) pix = p2;
                        if (!k2 || !p2) { failed = 1; break; }
                    }
                    int i = iy * n_z + iz;
                    kernel[cnt] = jo_exact_nodes > 0 ? jo_kernel_exact(y, z, e_t, R, Cinv, jo_exact_nodes)
                                                     : jo_kernel_c(y, z, tan_t, y_t, z_t, R, Cinv, a3_coef);   /* line 7 */
                    pix[cnt] = i;
                    denominator += kernel[cnt] * w[i];              /* line 8, with s(i) of Eq. 3 */
                    cnt++;
                }
                if (failed) break;
            }
            if (failed) continue;
            n_evals += cnt;
            if (cnt == 0 || !(denominator > 0.0) || !isfinite(denominator)) { n_skipped++; continue; }   /* R16 */
            for (size_t c = 0; c < cnt; ++c)                        /* lines 10-11; rho(i) pulled out (R11) */
                rho_new[pix[c]] += kernel[c] / denominator;
        }
        free(kernel);
        free(pix);
    }

    if (!failed) {
        for (size_t i = 0; i < M; ++i) {                            /* sum of the thread copies */
            double acc = 0.0;
            for (int t = 0; t < n_threads; ++t) acc += rho_new_all[(size_t)t * M + i];
            rho_out[i] = s[i] > 0.0 ? rho_in[i] * acc : 0.0;        /* Eq. 3; masked where s = 0 (R13) */
        }
        if (n_evals_out) *n_evals_out = n_evals;
        if (n_skipped_out) *n_skipped_out = n_skipped;
    }
    free(rho_new_all);
    free(s);
    free(w);
    return failed ? -1 : 0;
}

/* ---- n_iter iterations from rho_init (NULL => all ones, R18); counters are those of the LAST iteration */
int jo_reconstruct(const float *events, int64_t n, double R, double L, double sigma_z, double sigma_dl,
                   int n_y, int n_z, double pixel, double a3_coef, const double *rho_init, double *rho_out,
                   int n_iter, int n_threads, uint64_t *n_evals_out, uint64_t *n_skipped_out)
{
    if (n_iter < 0 || n_y <= 0 || n_z <= 0 || !rho_out) return -1;
    const size_t M = (size_t)n_y * (size_t)n_z;
    double *cur = (double *)malloc(M * sizeof(double));
    if (!cur) return -1;
    for (size_t i = 0; i < M; ++i) cur[i] = rho_init ? rho_init[i] : 1.0;
    int rc = 0;
    for (int it = 0; it < n_iter && rc == 0; ++it) {
        rc = jo_mlem_iterate(events, n, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, a3_coef, cur, rho_out,
                             0, n_threads, n_evals_out, n_skipped_out);
        memcpy(cur, rho_out, M * sizeof(double));
    }
    if (n_iter == 0) memcpy(rho_out, cur, M * sizeof(double));
    free(cur);
    return rc;
}

int jo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- direct reconstruction (Eq. 2; Fig. 4b): histogram of the reconstructed points ------------------
 * Every event is reconstructed to (y~, z~) with Eq. 2 (jo_eq2, fp64) and counted in the pixel that contains the point.
 * Pixel (iy, iz) covers [y_c - pixel/2, y_c + pixel/2) x [z_c - pixel/2, z_c + pixel/2) around its centre (y_c, z_c) of the
 * grid convention above, so in units of pixels from the lower edge of the grid the point has the coordinates
 *     c_y = y~ / pixel + n_y / 2,     c_z = z~ / pixel + n_z / 2
 * and lies in pixel (floor(c_y), floor(c_z)) when 0 <= c_y < n_y and 0 <= c_z < n_z; otherwise (or when a component of
 * the event is not finite) it is outside.  Nothing else: no precision is matched to any other implementation.  An fp32
 * implementation decides the same pixel except for points that lie within its rounding error of a pixel border; tests
 * that compare one with this function read the border distance from jo_direct_pixel_coords.
 * jo_direct_pixel_coords: coords[2 j] = c_y, coords[2 j + 1] = c_z of event j (NaN for a non-finite event).
 * jo_direct_histogram: hist (uint32 [n_y*n_z]) is INCREMENTED; returns the number of events outside.              */
void jo_direct_pixel_coords(const float *events, int64_t n, double R, int n_y, int n_z, double pixel, double *coords)
{
    for (int64_t j = 0; j < n; ++j) {
        double e[3];
        jo_eq2((double)events[3 * j + 0], (double)events[3 * j + 1], (double)events[3 * j + 2], R, e);
        const int finite = isfinite(e[0]) && isfinite(e[1]) && isfinite(e[2]);
        coords[2 * j + 0] = finite ? e[1] / pixel + 0.5 * (double)n_y : NAN;
        coords[2 * j + 1] = finite ? e[2] / pixel + 0.5 * (double)n_z : NAN;
    }
}

uint64_t jo_direct_histogram(const float *events, int64_t n, double R, int n_y, int n_z, double pixel, uint32_t *hist)
{
    uint64_t outside = 0;
    for (int64_t j = 0; j < n; ++j) {
        double c[2];
        jo_direct_pixel_coords(events + 3 * j, 1, R, n_y, n_z, pixel, c);
        if (!(c[0] >= 0.0 && c[0] < (double)n_y && c[1] >= 0.0 && c[1] < (double)n_z)) { outside++; continue; }   /* NaN: outside */
        hist[(size_t)floor(c[0]) * (size_t)n_z + (size_t)floor(c[1])] += 1u;
    }
    return outside;
}

/* ---- event simulation (recipe of SURVEY.md 8(d) / DESIGN.md section 5) -----------------------------
 * The same counter-based generator as the CUDA path, written out in fp64: event slot i draws from Philox4x32-10
 * (Salmon et al., SC'11: ten rounds of two 32x32 -> 64-bit multiplications, multipliers 0xD2511F53 / 0xCD9E8D57, key
 * increments 0x9E3779B9 / 0xBB67AE85) with key = (seed low, seed high) and counter = (slot low, slot high, attempt,
 * block).  A 32-bit word x becomes the uniform ((x >> 8) + 0.5) 2^-24.  Attempt a = 0, 1, ...:
 *   block 0 -> (u0, u1, u2, u3):  y = y0 + (y1 - y0) u0,  z = z0 + (z1 - z0) u1 in the phantom's bounding rectangle;
 *              accepted if u2 < intensity(y, z) / max intensity (first primitive in the list wins);
 *              theta = pi (u3 - 1/2); hits z_u = z + (R - y) tan, z_d = z - (R + y) tan; kept if both |.| <= L/2;
 *   block 1 -> (g0, g1, g2, g3):  Box-Muller  r0 = sqrt(-2 ln g0), r1 = sqrt(-2 ln g2):
 *              z_u~ = z_u + sigma_z r0 cos(2 pi g1),  z_d~ = z_d + sigma_z r0 sin(2 pi g1),
 *              dl~ = -2 y / cos(theta) + sigma_dl r1 cos(2 pi g3)                       (Eq. 1 on the LOR).
 * prims: double [n_prim][7] = (kind 0 ellipse / 1 box, cy, cz, hy, hz, phi_deg, intensity).  out: float32 [n][3].    */
static void jo_philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1)
{
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c[0], p1 = (uint64_t)0xCD9E8D57u * c[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1, n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}

static double jo_uniform24(uint32_t x) { return ((double)(x >> 8) + 0.5) / 16777216.0; }

static double jo_phantom_intensity(const double *prims, int n_prim, double y, double z)
{
    for (int k = 0; k < n_prim; ++k) {
        const double *q = prims + 7 * k;
        double phi = q[5] * JO_PI / 180.0, c = cos(phi), s = sin(phi);
        double dz = z - q[2], dy = y - q[1];
        double a = (c * dz + s * dy) / q[4], b = (-s * dz + c * dy) / q[3];
        int in = q[0] == 0.0 ? (a * a + b * b <= 1.0) : (fabs(a) <= 1.0 && fabs(b) <= 1.0);
        if (in) return q[6];
    }
    return 0.0;
}

int jo_generate_events(const double *prims, int n_prim, int64_t n, int64_t first, double R, double L, double sigma_z,
                       double sigma_dl, uint64_t seed, float *out)
{
    if (n_prim < 1 || n < 0 || !prims || (n > 0 && !out)) return -1;
    double y0 = 1e300, y1 = -1e300, z0 = 1e300, z1 = -1e300, rho_max = 0.0;
    for (int k = 0; k < n_prim; ++k) {                             /* bounding rectangle of the rotated primitives */
        const double *q = prims + 7 * k;
        double phi = q[5] * JO_PI / 180.0, c = fabs(cos(phi)), s = fabs(sin(phi)), ey, ez;
        if (q[0] == 0.0) { ez = hypot(q[4] * c, q[3] * s); ey = hypot(q[4] * s, q[3] * c); }
        else { ez = q[4] * c + q[3] * s; ey = q[4] * s + q[3] * c; }
        if (q[1] - ey < y0) y0 = q[1] - ey;
        if (q[1] + ey > y1) y1 = q[1] + ey;
        if (q[2] - ez < z0) z0 = q[2] - ez;
        if (q[2] + ez > z1) z1 = q[2] + ez;
        if (q[6] > rho_max) rho_max = q[6];
    }
    if (!(rho_max > 0.0)) return -1;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = 0; i < n; ++i) {
        const uint64_t slot = (uint64_t)first + (uint64_t)i;
        float zu = NAN, zd = NAN, dl = NAN;
        for (uint32_t a = 0; a < 65536u; ++a) {
            uint32_t c[4] = { (uint32_t)slot, (uint32_t)(slot >> 32), a, 0u };
            jo_philox4x32_10(c, k0, k1);
            double y = y0 + (y1 - y0) * jo_uniform24(c[0]), z = z0 + (z1 - z0) * jo_uniform24(c[1]);
            if (!(jo_uniform24(c[2]) < jo_phantom_intensity(prims, n_prim, y, z) / rho_max)) continue;
            double theta = JO_PI * (jo_uniform24(c[3]) - 0.5);
            double hu = z + (R - y) * tan(theta), hd = z - (R + y) * tan(theta);
            if (!(fabs(hu) <= 0.5 * L && fabs(hd) <= 0.5 * L)) continue;
            uint32_t g[4] = { (uint32_t)slot, (uint32_t)(slot >> 32), a, 1u };
            jo_philox4x32_10(g, k0, k1);
            double r0 = sqrt(-2.0 * log(jo_uniform24(g[0]))), r1 = sqrt(-2.0 * log(jo_uniform24(g[2])));
            zu = (float)(hu + sigma_z * r0 * cos(2.0 * JO_PI * jo_uniform24(g[1])));
            zd = (float)(hd + sigma_z * r0 * sin(2.0 * JO_PI * jo_uniform24(g[1])));
            dl = (float)(-2.0 * y / cos(theta) + sigma_dl * r1 * cos(2.0 * JO_PI * jo_uniform24(g[3])));
            break;
        }
        out[3 * i + 0] = zu; out[3 * i + 1] = zd; out[3 * i + 2] = dl;
    }
    return 0;
}

/* ---- conveniences for the tests: the exact integral for many events (double [n][3]) at one pixel, each with its own
 * matrix (jo_cinv); and the Philox block function on its own (known-answer test)                                 */
void jo_kernel_exact_events(const double *events, int64_t n, double y, double z, double R, double L, double sigma_z,
                            double sigma_dl, int n_theta, double *P_out)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t j = 0; j < n; ++j) {
        double Cinv[3][3];
        jo_cinv(events[3 * j + 0], events[3 * j + 1], L, sigma_z, sigma_dl, Cinv);
        P_out[j] = jo_kernel_exact(y, z, events + 3 * j, R, Cinv, n_theta);
    }
}

void jo_philox4x32_10_block(const uint32_t counter[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c[4] = { counter[0], counter[1], counter[2], counter[3] };
    jo_philox4x32_10(c, key[0], key[1]);
    for (int k = 0; k < 4; ++k) out[k] = c[k];
}
