/*
 * radon_oracle.c -- plain, slow, fp64 CPU oracle for the NUFFT-Radon hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  The product
 * (paper_1009_1380_b200/) never links, imports or executes anything in oracle/.
 * It shares no code, header, table or constant generator with the CUDA path.
 *
 * What it computes (citations are PAPER.md lines of arxiv 1009.1380 and the
 * readings S1..S17 listed in SURVEY.md section 8(c) / DESIGN.md section 4):
 *
 *   O-direct  the operator itself, written out as its definition:
 *             "perform a 2D FFT of x on a regular grid, and then interpolate
 *             the transform onto a polar grid before 1D inverse Fourier
 *             transforms are applied to interpolated points along the same
 *             radial lines" (section II).  The exact object the
 *             interpolation approximates is the image's DTFT sampled on radial
 *             lines (a non-uniform DFT), so the oracle evaluates that sum
 *             directly -- no FFT, no gridding, no table.
 *   O-dirichlet the same operator in closed form (periodic-sinc detector
 *             response), an independent second implementation used as a pin.
 *   O-ray     the continuous Radon line integral by ray sampling with bilinear
 *             interpolation (BASELINE.json north_star: "a direct Radon line
 *             integral by ray-sampling"): pins orientation/centre/scale only.
 *   O-grid    the two gridding sums printed with Fig. 5
 *             with a Kaiser-Bessel kernel K evaluated directly (no LUT):
 *               G_i(x_i,y_i) = sum_r G_r(x_r,y_r) K(x_r-x_i, y_r-y_i)   (:87)
 *               G_r(x_r,y_r) = sum_i D G(x_i,y_i) K(x_i-x_r, y_i-y_r)   (:85, D==1)
 *             plus the kernel, its Fourier transform (de-apodisation), I0.
 *
 * Geometry (readings S4-S8): pixel x[iy*N+ix], X = ix-c, Y = iy-c, c = N/2
 * (integer division); theta_a = pi*a/n_angles; detector bin s has t = s-c_d,
 * radial frequency index k has j = k-c_d, c_d = n/2 (integer division);
 * t = X cos(theta) + Y sin(theta).
 *
 * Pins (tests/test_oracle_pins.py): every function here is pinned; see the
 * table in DESIGN.md section 3.  No function is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC radon_oracle.c -o liboracle.so -lm
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------------- */
/* O-direct step 1: non-uniform DFT of the  */
/* image on the polar set.  F[a,k] = sum_{iy,ix} x[iy,ix] *                   */
/*        exp(-i (2 pi j / n) (X cos theta_a + Y sin theta_a)).               */
/* Evaluates only the listed output samples m = a*n_det + k (idx), so a       */
/* subset costs proportionally less; idx == NULL means all M outputs.         */
/* x is real (xi == NULL) or complex (xr + i xi).                             */
/* ------------------------------------------------------------------------- */
void odirect_ndft2(const double *xr, const double *xi, int N, int n_angles, int n_det,
                   const long long *idx, long long n_idx, double *Fr, double *Fi)
{
    const int c = N / 2, cd = n_det / 2;
    const long long M = (long long)n_angles * n_det;
    const long long cnt = idx ? n_idx : M;
#pragma omp parallel for schedule(dynamic, 16)
    for (long long q = 0; q < cnt; ++q) {
        const long long m = idx ? idx[q] : q;
        const int a = (int)(m / n_det), k = (int)(m % n_det);
        const double theta = M_PI * (double)a / (double)n_angles;
        const double ct = cos(theta), st = sin(theta);
        const double w = 2.0 * M_PI * (double)(k - cd) / (double)n_det;
        double sr = 0.0, si = 0.0;
        for (int iy = 0; iy < N; ++iy) {
            const double Y = (double)(iy - c);
            for (int ix = 0; ix < N; ++ix) {
                const double X = (double)(ix - c);
                const double ph = -w * (X * ct + Y * st);
                const double cr = cos(ph), ci = sin(ph);
                const double vr = xr[(size_t)iy * N + ix];
                if (xi) {
                    const double vi = xi[(size_t)iy * N + ix];
                    sr += vr * cr - vi * ci;
                    si += vr * ci + vi * cr;
                } else {
                    sr += vr * cr;
                    si += vr * ci;
                }
            }
        }
        Fr[q] = sr;
        Fi[q] = si;
    }
}

/* Conjugate transpose of odirect_ndft2 on arbitrary complex polar input:     */
/* z[iy,ix] = sum_{a,k} P[a,k] exp(+i (2 pi j/n)(X cos + Y sin)).             */
/* Evaluates the listed pixels p = iy*N+ix (pix == NULL: all).                */
void odirect_ndft1(const double *Pr, const double *Pi, int N, int n_angles, int n_det,
                   const long long *pix, long long n_pix, double *zr, double *zi)
{
    const int c = N / 2, cd = n_det / 2;
    const long long cnt = pix ? n_pix : (long long)N * N;
#pragma omp parallel for schedule(dynamic, 16)
    for (long long q = 0; q < cnt; ++q) {
        const long long p = pix ? pix[q] : q;
        const double X = (double)((int)(p % N) - c), Y = (double)((int)(p / N) - c);
        double sr = 0.0, si = 0.0;
        for (int a = 0; a < n_angles; ++a) {
            const double theta = M_PI * (double)a / (double)n_angles;
            const double tau = X * cos(theta) + Y * sin(theta);
            for (int k = 0; k < n_det; ++k) {
                const double ph = 2.0 * M_PI * (double)(k - cd) / (double)n_det * tau;
                const double cr = cos(ph), ci = sin(ph);
                const double vr = Pr[(size_t)a * n_det + k], vi = Pi[(size_t)a * n_det + k];
                sr += vr * cr - vi * ci;
                si += vr * ci + vi * cr;
            }
        }
        zr[q] = sr;
        zi[q] = si;
    }
}

/* ------------------------------------------------------------------------- */
/* O-direct forward y = Radon{x}:     */
/*   S[a,s] = Re{ (1/n) sum_k F[a,k] exp(+i 2 pi j t_s / n) }                 */
/* evaluated for the listed sinogram entries q = a*n_det + s (NULL: all).     */
/* For each needed angle the whole radial line F[a,:] is computed first       */
/* (step 1), then the 1-D inverse DFT along that line (step 2).               */
/* ------------------------------------------------------------------------- */
void odirect_forward(const double *x, int N, int n_angles, int n_det,
                     const long long *idx, long long n_idx, double *S)
{
    const int cd = n_det / 2;
    const long long M = (long long)n_angles * n_det;
    const long long cnt = idx ? n_idx : M;
    /* which angles are needed */
    char *need = (char *)calloc((size_t)n_angles, 1);
    for (long long q = 0; q < cnt; ++q) need[(idx ? idx[q] : q) / n_det] = 1;
    double *Fr = (double *)malloc(sizeof(double) * (size_t)M);
    double *Fi = (double *)malloc(sizeof(double) * (size_t)M);
    /* list of line samples to evaluate */
    long long nl = 0;
    for (int a = 0; a < n_angles; ++a) nl += need[a] ? n_det : 0;
    long long *lidx = (long long *)malloc(sizeof(long long) * (size_t)(nl ? nl : 1));
    double *tr = (double *)malloc(sizeof(double) * (size_t)(nl ? nl : 1));
    double *ti = (double *)malloc(sizeof(double) * (size_t)(nl ? nl : 1));
    nl = 0;
    for (int a = 0; a < n_angles; ++a)
        if (need[a])
            for (int k = 0; k < n_det; ++k) lidx[nl++] = (long long)a * n_det + k;
    odirect_ndft2(x, NULL, N, n_angles, n_det, lidx, nl, tr, ti);
    for (long long i = 0; i < nl; ++i) {
        Fr[lidx[i]] = tr[i];
        Fi[lidx[i]] = ti[i];
    }
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < cnt; ++q) {
        const long long m = idx ? idx[q] : q;
        const int a = (int)(m / n_det), s = (int)(m % n_det);
        const double t = (double)(s - cd);
        double acc = 0.0;
        for (int k = 0; k < n_det; ++k) {
            const double ph = 2.0 * M_PI * (double)(k - cd) * t / (double)n_det;
            /* real part of F * exp(+i ph) */
            acc += Fr[(size_t)a * n_det + k] * cos(ph) - Fi[(size_t)a * n_det + k] * sin(ph);
        }
        S[q] = acc / (double)n_det;
    }
    free(need); free(Fr); free(Fi); free(lidx); free(tr); free(ti);
}

/* ------------------------------------------------------------------------- */
/* O-direct adjoint x~ = Radon^T{y} (exact transpose of   */
/* odirect_forward; PAPER.md:85 with D == 1 is its fast approximation):       */
/*   Yh[a,k] = (1/n) sum_s y[a,s] exp(-i 2 pi j t_s / n)                      */
/*   x~[iy,ix] = Re{ sum_{a,k} Yh[a,k] exp(+i (2 pi j/n)(X cos + Y sin)) }    */
/* evaluated for the listed pixels (NULL: all).                               */
/* ------------------------------------------------------------------------- */
void odirect_adjoint(const double *y, int N, int n_angles, int n_det,
                     const long long *pix, long long n_pix, double *xt)
{
    const int cd = n_det / 2;
    const long long M = (long long)n_angles * n_det;
    double *Yr = (double *)malloc(sizeof(double) * (size_t)M);
    double *Yi = (double *)malloc(sizeof(double) * (size_t)M);
#pragma omp parallel for schedule(static)
    for (long long m = 0; m < M; ++m) {
        const int a = (int)(m / n_det), k = (int)(m % n_det);
        double sr = 0.0, si = 0.0;
        for (int s = 0; s < n_det; ++s) {
            const double ph = -2.0 * M_PI * (double)(k - cd) * (double)(s - cd) / (double)n_det;
            const double v = y[(size_t)a * n_det + s];
            sr += v * cos(ph);
            si += v * sin(ph);
        }
        Yr[m] = sr / (double)n_det;
        Yi[m] = si / (double)n_det;
    }
    const long long cnt = pix ? n_pix : (long long)N * N;
    double *zr = (double *)malloc(sizeof(double) * (size_t)cnt);
    double *zi = (double *)malloc(sizeof(double) * (size_t)cnt);
    odirect_ndft1(Yr, Yi, N, n_angles, n_det, pix, n_pix, zr, zi);
    for (long long q = 0; q < cnt; ++q) xt[q] = zr[q];
    free(Yr); free(Yi); free(zr); free(zi);
}

/* ------------------------------------------------------------------------- */
/* O-dirichlet: closed form of the same operator ("Equivalent    */
/* closed form"): summing the geometric series over k in step 2 gives         */
/*   S[a,s] = sum_pix x[pix] D_n(t_s - tau),  tau = X cos + Y sin,            */
/*   D_n(u) = sin(pi u) / (n sin(pi u / n))                  (n odd)          */
/*          = sin(pi u) cos(pi u / n) / (n sin(pi u / n))    (n even, Re{})   */
/*          = 1 when u == 0 (mod n).                                          */
/* ------------------------------------------------------------------------- */
static double dirichlet(double u, int n)
{
    const double un = u / (double)n;
    const double r = un - floor(un + 0.5);          /* u/n reduced to [-1/2,1/2) */
    const double sn = sin(M_PI * r);
    if (fabs(sn) < 1e-14) {
        /* u = 0 mod n: limit of the ratio (sign handled by the reduced u) */
        return 1.0;
    }
    /* sin(pi u) with u reduced consistently: u = n*(r + integer) */
    const double ured = r * (double)n;
    /* sin(pi u) = sin(pi (ured + n*q)) ; for integer q: = sin(pi ured) * (-1)^(n q)
       and sin(pi u/n) = sin(pi r) * (-1)^q ; cos(pi u/n) = cos(pi r) (-1)^q.
       odd n : ratio sign (-1)^(nq)/(-1)^q = 1.  even n: numerator sign 1,
       cos sign (-1)^q, denominator sign (-1)^q -> 1.  So use reduced values. */
    if (n & 1) return sin(M_PI * ured) / ((double)n * sn);
    return sin(M_PI * ured) * cos(M_PI * r) / ((double)n * sn);
}

void odirichlet_forward(const double *x, int N, int n_angles, int n_det, double *S)
{
    const int c = N / 2, cd = n_det / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int a = 0; a < n_angles; ++a) {
        const double theta = M_PI * (double)a / (double)n_angles;
        const double ct = cos(theta), st = sin(theta);
        for (int s = 0; s < n_det; ++s) {
            const double t = (double)(s - cd);
            double acc = 0.0;
            for (int iy = 0; iy < N; ++iy)
                for (int ix = 0; ix < N; ++ix) {
                    const double v = x[(size_t)iy * N + ix];
                    if (v != 0.0) acc += v * dirichlet(t - ((ix - c) * ct + (iy - c) * st), n_det);
                }
            S[(size_t)a * n_det + s] = acc;
        }
    }
}

/* Closed-form evaluation of listed outputs only (used at BASELINE.json's full  */
/* sizes, where the double sum of odirect_forward needs a whole radial line    */
/* -- n_det * N^2 terms -- per sampled angle): N^2 terms per listed entry.      */
void odirichlet_forward_subset(const double *x, int N, int n_angles, int n_det,
                               const long long *idx, long long n_idx, double *S)
{
    const int c = N / 2, cd = n_det / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (long long q = 0; q < n_idx; ++q) {
        const int a = (int)(idx[q] / n_det), s = (int)(idx[q] % n_det);
        const double theta = M_PI * (double)a / (double)n_angles;
        const double ct = cos(theta), st = sin(theta), t = (double)(s - cd);
        double acc = 0.0;
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                const double v = x[(size_t)iy * N + ix];
                if (v != 0.0) acc += v * dirichlet(t - ((ix - c) * ct + (iy - c) * st), n_det);
            }
        S[q] = acc;
    }
}

/* Transpose in closed form: x~[pix] = sum_{a,s} y[a,s] D_n(t_s - tau_a(pix)),  */
/* M terms per listed pixel (pix == NULL: all pixels).                          */
void odirichlet_adjoint(const double *y, int N, int n_angles, int n_det,
                        const long long *pix, long long n_pix, double *xt)
{
    const int c = N / 2, cd = n_det / 2;
    const long long cnt = pix ? n_pix : (long long)N * N;
#pragma omp parallel for schedule(dynamic, 1)
    for (long long q = 0; q < cnt; ++q) {
        const long long p = pix ? pix[q] : q;
        const double X = (double)((int)(p % N) - c), Y = (double)((int)(p / N) - c);
        double acc = 0.0;
        for (int a = 0; a < n_angles; ++a) {
            const double theta = M_PI * (double)a / (double)n_angles;
            const double tau = X * cos(theta) + Y * sin(theta);
            for (int s = 0; s < n_det; ++s) {
                const double v = y[(size_t)a * n_det + s];
                if (v != 0.0) acc += v * dirichlet((double)(s - cd) - tau, n_det);
            }
        }
        xt[q] = acc;
    }
}

/* ------------------------------------------------------------------------- */
/* O-ray (north_star; SURVEY 8(c) "O-ray"): line integral by ray sampling.    */
/*   L[a,s] = h sum_q bilinear(x; c + t cos - u_q sin, c + t sin + u_q cos),  */
/*   u_q = -N + (q + 1/2) h, h = step, q = 0 .. 2N/h - 1, zero outside.       */
/* ------------------------------------------------------------------------- */
static double bilinear(const double *x, int N, double px, double py)
{
    const double fx = floor(px), fy = floor(py);
    const int ix = (int)fx, iy = (int)fy;
    const double ax = px - fx, ay = py - fy;
    double v = 0.0;
    for (int dy = 0; dy < 2; ++dy)
        for (int dx = 0; dx < 2; ++dx) {
            const int jx = ix + dx, jy = iy + dy;
            if (jx < 0 || jy < 0 || jx >= N || jy >= N) continue;
            v += x[(size_t)jy * N + jx] * (dx ? ax : 1.0 - ax) * (dy ? ay : 1.0 - ay);
        }
    return v;
}

void oray_forward(const double *x, int N, int n_angles, int n_det, double h, double *L)
{
    const int c = N / 2, cd = n_det / 2;
    const long long nq = (long long)floor(2.0 * N / h + 0.5);
#pragma omp parallel for schedule(dynamic, 1)
    for (int a = 0; a < n_angles; ++a) {
        const double theta = M_PI * (double)a / (double)n_angles;
        const double ct = cos(theta), st = sin(theta);
        for (int s = 0; s < n_det; ++s) {
            const double t = (double)(s - cd);
            double acc = 0.0;
            for (long long q = 0; q < nq; ++q) {
                const double u = -(double)N + ((double)q + 0.5) * h;
                acc += bilinear(x, N, c + t * ct - u * st, c + t * st + u * ct);
            }
            L[(size_t)a * n_det + s] = acc * h;
        }
    }
}

/* ------------------------------------------------------------------------- */
/* Kaiser-Bessel kernel (reading S1/S2: the paper names no kernel, cites      */
/* Jackson et al. [3] PAPER.md:77; north_star fixes Kaiser-Bessel W, sigma).  */
/*   I0(z)  = sum_m (z^2/4)^m / (m!)^2                                        */
/*   beta   = pi sqrt((W/sigma)^2 (sigma - 1/2)^2 - 0.8)                      */
/*   phi(u) = I0(beta sqrt(1 - (2u/W)^2)) / I0(beta), |u| <= W/2, else 0      */
/*   phihat(xi) = int phi(u) exp(-i 2 pi xi u) du                             */
/*          = (W/I0(beta)) sinh(sqrt(beta^2 - (pi W xi)^2)) / sqrt(...)       */
/*            (sin(...)/... when the radicand is negative)                    */
/* ------------------------------------------------------------------------- */
double okb_i0(double z)
{
    const double q = 0.25 * z * z;
    double term = 1.0, sum = 1.0;
    for (int m = 1; m < 500; ++m) {
        term *= q / ((double)m * (double)m);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

double okb_beta(int W, double sigma)
{
    const double r = (double)W / sigma * (sigma - 0.5);
    return M_PI * sqrt(r * r - 0.8);
}

double okb_phi(double u, int W, double beta)
{
    const double t = 2.0 * u / (double)W;
    const double a = 1.0 - t * t;
    if (a < 0.0) return 0.0;
    return okb_i0(beta * sqrt(a)) / okb_i0(beta);
}

double okb_phihat(double xi, int W, double beta)
{
    const double a = M_PI * (double)W * xi;
    const double r = beta * beta - a * a;
    const double scale = (double)W / okb_i0(beta);
    if (r > 0.0) {
        const double q = sqrt(r);
        return scale * sinh(q) / q;
    } else if (r < 0.0) {
        const double q = sqrt(-r);
        return scale * sin(q) / q;
    }
    return scale;
}

/* Polar sample position on the oversampled grid (Fourier-    */
/* slice PAPER.md:51): kappa(a,k) = (G j / n)(cos theta_a, sin theta_a).      */
static void polar_kappa(int a, int k, int n_angles, int n_det, int G, double *kx, double *ky)
{
    const double theta = M_PI * (double)a / (double)n_angles;
    const double rho = (double)G * (double)(k - n_det / 2) / (double)n_det;
    /* theta = pi/2 (a = n_angles/2): the mathematical values cos = 0, sin = 1.  libm's       */
    /* cos(M_PI/2) = 6.1e-17 would push kappa_x off the exact tie of the tap rule S3           */
    /* (x0 = ceil(kappa - W/2)) in a direction that depends on the sign of j.    */
    const double c = (2 * a == n_angles) ? 0.0 : cos(theta);
    const double s = (2 * a == n_angles) ? 1.0 : sin(theta);
    *kx = rho * c;
    *ky = rho * s;
}

static int imod(int a, int m)
{
    int r = a % m;
    return r < 0 ? r + m : r;
}

/* ------------------------------------------------------------------------- */
/* O-grid inverse gridding:                                      */
/*   G_i(x_i,y_i) = sum_{x_r,y_r} G_r(x_r,y_r) K(x_r - x_i, y_r - y_i)        */
/* with K(dx,dy) = phi(dx) phi(dy), the sum running over the W x W regular    */
/* positions x_r = x0 .. x0+W-1, x0 = ceil(kappa_x - W/2) (reading S3),       */
/* indices taken mod G (reading S12).  Grid layout: centred, cell             */
/* grid[cy*G + cx] holds frequency (cx - G/2, cy - G/2) (include/radon.h).    */
/* ------------------------------------------------------------------------- */
void ogrid_interp(const double *gr, const double *gi, int G, int n_angles, int n_det,
                  int W, double beta, double *pr, double *pi)
{
    const long long M = (long long)n_angles * n_det;
#pragma omp parallel for schedule(static)
    for (long long m = 0; m < M; ++m) {
        double kx, ky;
        polar_kappa((int)(m / n_det), (int)(m % n_det), n_angles, n_det, G, &kx, &ky);
        const int x0 = (int)ceil(kx - 0.5 * W), y0 = (int)ceil(ky - 0.5 * W);
        double sr = 0.0, si = 0.0;
        for (int ly = 0; ly < W; ++ly)
            for (int lx = 0; lx < W; ++lx) {
                const int xr = x0 + lx, yr = y0 + ly;
                const double K = okb_phi((double)xr - kx, W, beta) * okb_phi((double)yr - ky, W, beta);
                const size_t cell = (size_t)imod(yr + G / 2, G) * G + imod(xr + G / 2, G);
                sr += gr[cell] * K;
                si += gi[cell] * K;
            }
        pr[m] = sr;
        pi[m] = si;
    }
}

/* O-grid gridding, PAPER.md:85 with D == 1 (reading S11):                    */
/*   G_r(x_r,y_r) = sum_{x_i,y_i} G(x_i,y_i) K(x_i - x_r, y_i - y_r)          */
/* over the same taps; serial accumulation in sample order.                   */
void ogrid_grid(const double *pr, const double *pi, int G, int n_angles, int n_det,
                int W, double beta, double *gr, double *gi)
{
    const long long M = (long long)n_angles * n_det;
    for (size_t i = 0; i < (size_t)G * G; ++i) gr[i] = gi[i] = 0.0;
    for (long long m = 0; m < M; ++m) {
        double kx, ky;
        polar_kappa((int)(m / n_det), (int)(m % n_det), n_angles, n_det, G, &kx, &ky);
        const int x0 = (int)ceil(kx - 0.5 * W), y0 = (int)ceil(ky - 0.5 * W);
        for (int ly = 0; ly < W; ++ly)
            for (int lx = 0; lx < W; ++lx) {
                const int xr = x0 + lx, yr = y0 + ly;
                const double K = okb_phi(kx - (double)xr, W, beta) * okb_phi(ky - (double)yr, W, beta);
                const size_t cell = (size_t)imod(yr + G / 2, G) * G + imod(xr + G / 2, G);
                gr[cell] += pr[m] * K;
                gi[cell] += pi[m] * K;
            }
    }
}

/* ------------------------------------------------------------------------- */
/* O-density: the density compensation printed with Fig. 5,     */
/*   D(x_i,y_i) = 1 / sum_j K(x_i - x_j, y_i - y_j),                          */
/* the sum running over ALL polar samples j (j = i included: K(0,0) = 1), with */
/* the same separable Kaiser-Bessel kernel K(dx,dy) = phi(dx) phi(dy) on the   */
/* oversampled grid's coordinates (kappa, polar_kappa above).  */
/* is a garbled duplicate of the same formula (reading S11).                   */
/* brute != 0: the double sum exactly as printed, every one of the M^2 terms.  */
/* brute == 0: the same sum without the terms that are exactly zero: K vanishes */
/* outside |dy| < W/2, so the samples are sorted by their y coordinate and, for */
/* sample i, only the contiguous run of the sorted list with |ky_i - ky_j| <   */
/* W/2 is visited (found by bisection; a 1-D sort-and-scan, no cell buckets).   */
/* No wrap mod G: eq. :89 as printed has none.                                  */
static const double *g_sort_key;
static int cmp_by_key(const void *a, const void *b)
{
    const double x = g_sort_key[*(const long long *)a], y = g_sort_key[*(const long long *)b];
    return (x > y) - (x < y);
}

void odensity(int n_angles, int n_det, int G, int W, double beta, int brute, double *D)
{
    const long long M = (long long)n_angles * n_det;
    double *kx = (double *)malloc(sizeof(double) * (size_t)M), *ky = (double *)malloc(sizeof(double) * (size_t)M);
    for (long long m = 0; m < M; ++m)
        polar_kappa((int)(m / n_det), (int)(m % n_det), n_angles, n_det, G, &kx[m], &ky[m]);
    if (brute) {
#pragma omp parallel for schedule(dynamic, 64)
        for (long long i = 0; i < M; ++i) {
            double s = 0.0;
            for (long long j = 0; j < M; ++j)
                s += okb_phi(kx[i] - kx[j], W, beta) * okb_phi(ky[i] - ky[j], W, beta);
            D[i] = 1.0 / s;
        }
    } else {
        long long *by_y = (long long *)malloc(sizeof(long long) * (size_t)M);
        double *ys = (double *)malloc(sizeof(double) * (size_t)M);
        for (long long m = 0; m < M; ++m) by_y[m] = m;
        g_sort_key = ky;
        qsort(by_y, (size_t)M, sizeof(long long), cmp_by_key);
        for (long long m = 0; m < M; ++m) ys[m] = ky[by_y[m]];
        const double hw = 0.5 * (double)W;
#pragma omp parallel for schedule(dynamic, 64)
        for (long long i = 0; i < M; ++i) {
            /* first sorted position with ys >= ky_i - W/2 */
            long long lo = 0, hi = M;
            const double ymin = ky[i] - hw - 1e-9;   /* slack: okb_phi itself decides the support */
            while (lo < hi) {
                const long long mid = (lo + hi) / 2;
                if (ys[mid] < ymin) lo = mid + 1; else hi = mid;
            }
            double s = 0.0;
            for (long long q = lo; q < M && ys[q] <= ky[i] + hw + 1e-9; ++q) {
                const long long j = by_y[q];
                const double dx = kx[i] - kx[j];
                if (fabs(dx) > hw + 1e-9) continue;    /* phi(dx) == 0 there */
                s += okb_phi(dx, W, beta) * okb_phi(ky[i] - ky[j], W, beta);
            }
            D[i] = 1.0 / s;
        }
        free(by_y); free(ys);
    }
    free(kx); free(ky);
}
