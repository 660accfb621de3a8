/*
 * hb_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU oracle for the
 * hybrid-beamline push of arXiv 2402.17248 (Sandberg et al., PASC'24).
 *
 * This file is the parity oracle.  It shares no code, header, table or constant with
 * the CUDA library (paper_2402_17248_b200/csrc).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  The product path
 * never calls it.
 *
 * Citations: "P:NN" = /root/reference/PAPER.md line NN; "R1..R10", "G1..G17" = the
 * readings listed in DESIGN.md (the paper is silent on the element maps and on the
 * s<->t conversion; it delegates them to ImpactX).
 *
 * Conventions (R1): per particle, at fixed s:  x, y [m];  px = Px/p0,
 * py = Py/p0;  t = c (T_arrival - T_ref) [m];  pt = -(E - E_ref)/(p0 c).
 * All arrays are fp64, one contiguous array per coordinate (SoA), updated in place.
 * Every function is the plain definition evaluated one particle at a time, one
 * element / one layer at a time; OpenMP only distributes particles over threads.
 *
 * Pins (tests/test_oracle_pins.py, all CPU): drift(L)drift(-L)=id; Jacobians vs the
 * closed-form 6x6 of R2-R4; M^T S M = S; quad(k->0), sbend(theta->0) -> drift; De Moivre
 * closed form of N FODO cells and the printed cell matrices; Sigma_out = M Sigma_in M^T;
 * emittance / det Sigma conservation; s->t->s round trip and first-order limits;
 * identity-initialised MLPs; dense numpy mat-vec brute force on 8 particles;
 * hand-computed moments of an 8-particle set.
 * Whole-config end-to-end values: parity unpinned beyond this oracle (no external
 * implementation or printed value exists).
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* R1: reference particle from kinetic energy T and rest energy mc^2 (both MeV). */
void orc_reference(double kinetic_MeV, double rest_MeV, double *gamma0, double *bg0, double *beta0)
{
    double g = 1.0 + kinetic_MeV / rest_MeV;
    double bg = sqrt(g * g - 1.0);
    *gamma0 = g;
    *bg0 = bg;
    *beta0 = bg / g;
}

/* R2: drift of length L.  x' = x + L px; y' = y + L py; t' = t + L pt/(beta0 gamma0)^2. */
void orc_drift(double *x, double *px, double *y, double *py, double *t, double *pt,
               long n, double L, double bg0)
{
    long i;
    (void)px; (void)py;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        x[i] = x[i] + L * px[i];
        y[i] = y[i] + L * py[i];
        t[i] = t[i] + L * pt[i] / (bg0 * bg0);
    }
}

/* R2x (NEXT-3): drift of length L WITHOUT the paraxial / first-order expansion of R2.  In the coordinates
 * of R1 the total momentum and energy of a particle, in units of p0 and p0 c, are
 *     E/(p0 c) = 1/beta0 - pt,      pz = sqrt( (1/beta0 - pt)^2 - 1/(beta0 gamma0)^2 - px^2 - py^2 )
 * (pz: longitudinal momentum / p0).  A free particle moves on a straight line with slopes px/pz, py/pz and takes the
 * time L (E/(p0 c))/pz (in units of 1/c) to advance by L in s, the reference L/beta0:
 *     x' = x + L px/pz,   y' = y + L py/pz,   t' = t + L ( (1/beta0 - pt)/pz - 1/beta0 ).
 * First order in (px, py, pt) this is R2. */
void orc_drift_exact(double *x, double *px, double *y, double *py, double *t, double *pt,
                     long n, double L, double bg0)
{
    long i;
    const double g0 = sqrt(1.0 + bg0 * bg0), b0 = bg0 / g0;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        const double e = 1.0 / b0 - pt[i];
        const double pz = sqrt(e * e - 1.0 / (bg0 * bg0) - px[i] * px[i] - py[i] * py[i]);
        x[i] = x[i] + L * px[i] / pz;
        y[i] = y[i] + L * py[i] / pz;
        t[i] = t[i] + L * (e / pz - 1.0 / b0);
    }
}

/* R3x (NEXT-3, "chromatic effects"): thick quadrupole whose focusing depends on the particle's momentum.
 * With 1+delta = |p|/p0 = sqrt((1/beta0 - pt)^2 - 1/(beta0 gamma0)^2) and e = E/(p0 c) = 1/beta0 - pt, the paraxial
 * Hamiltonian of the quadrupole for an off-momentum particle is
 *     H = -(1+delta) + (px^2 + py^2)/(2(1+delta)) + k (x^2 - y^2)/2 - pt/beta0
 * so  x' = px/(1+delta), px' = -k x  (omega^2 = k/(1+delta): "k -> k/(1+delta)"),  y likewise with -k, and
 *     t' = dH/dpt = e/(1+delta) - 1/beta0 + e (px^2 + py^2) / (2 (1+delta)^3).
 * chr_plane advances one plane over L and returns  integral_0^L p(s)^2 ds  (closed form of the harmonic motion). */
static double chr_plane(double *u, double *pu, double L, double k_plane, double d1 /* 1+delta */)
{
    const double u0 = *u, p0 = *pu;
    double A = p0, B, I;
    if (k_plane > 0.0) {
        const double w = sqrt(k_plane / d1), c = cos(w * L), sn = sin(w * L);
        B = -w * d1 * u0;                         /* p(s) = A cos(ws) + B sin(ws) */
        *u = c * u0 + sn / (w * d1) * p0;
        *pu = B * sn + A * c;
        I = 0.5 * (A * A + B * B) * L + (A * A - B * B) * sin(2.0 * w * L) / (4.0 * w)
            + A * B * (1.0 - cos(2.0 * w * L)) / (2.0 * w);
    } else if (k_plane < 0.0) {
        const double w = sqrt(-k_plane / d1), c = cosh(w * L), sn = sinh(w * L);
        B = w * d1 * u0;                          /* p(s) = A cosh(ws) + B sinh(ws) */
        *u = c * u0 + sn / (w * d1) * p0;
        *pu = B * sn + A * c;
        I = 0.5 * (A * A - B * B) * L + (A * A + B * B) * sinh(2.0 * w * L) / (4.0 * w)
            + A * B * (cosh(2.0 * w * L) - 1.0) / (2.0 * w);
    } else {
        *u = u0 + L * p0 / d1;
        I = p0 * p0 * L;
    }
    return I;
}

void orc_quad_chromatic(double *x, double *px, double *y, double *py, double *t, double *pt,
                        long n, double L, double k, double bg0)
{
    long i;
    const double g0 = sqrt(1.0 + bg0 * bg0), b0 = bg0 / g0;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        const double e = 1.0 / b0 - pt[i];
        const double d1 = sqrt(e * e - 1.0 / (bg0 * bg0));
        const double Ix = chr_plane(&x[i], &px[i], L, k, d1);
        const double Iy = chr_plane(&y[i], &py[i], L, -k, d1);
        t[i] = t[i] + L * (e / d1 - 1.0 / b0) + e * (Ix + Iy) / (2.0 * d1 * d1 * d1);
    }
}

/* R5x (NEXT-3): thin multipole kick of order m (1 = dipole, 2 = quadrupole, 3 = sextupole, ...) with integrated
 * normal / skew strengths kn, ks [m^-(m-1)]:  px - i py  -=  (kn + i ks) (x + i y)^(m-1) / (m-1)!   (the usual complex
 * form; m = 2, ks = 0:  px -= kn x,  py += kn y,  the thin limit of R3).  Positions and (t, pt) unchanged. */
void orc_multipole(double *x, double *px, double *y, double *py, double *t, double *pt,
                   long n, int m, double kn, double ks)
{
    long i;
    int j;
    double fact = 1.0;
    (void)t; (void)pt;
    for (j = 2; j < m; ++j) fact *= (double)j;
#pragma omp parallel for schedule(static) private(j)
    for (i = 0; i < n; ++i) {
        double zr = 1.0, zi = 0.0;                /* (x + i y)^(m-1) */
        for (j = 1; j < m; ++j) {
            const double r = zr * x[i] - zi * y[i], im = zr * y[i] + zi * x[i];
            zr = r; zi = im;
        }
        px[i] = px[i] - (kn * zr - ks * zi) / fact;
        py[i] = py[i] + (kn * zi + ks * zr) / fact;
    }
}

/* one transverse plane of a thick quadrupole, R3 */
static void quad_plane(double *u, double *pu, double L, double k_plane)
{
    /* k_plane > 0: focusing in this plane; < 0: defocusing; == 0: drift */
    double u0 = *u, p0 = *pu;
    if (k_plane > 0.0) {
        double w = sqrt(k_plane);
        *u = cos(w * L) * u0 + sin(w * L) / w * p0;
        *pu = -w * sin(w * L) * u0 + cos(w * L) * p0;
    } else if (k_plane < 0.0) {
        double w = sqrt(-k_plane);
        *u = cosh(w * L) * u0 + sinh(w * L) / w * p0;
        *pu = w * sinh(w * L) * u0 + cosh(w * L) * p0;
    } else {
        *u = u0 + L * p0;
    }
}

/* R3: thick quadrupole, length L, strength k [m^-2]; k>0 focuses x and defocuses y. */
void orc_quad(double *x, double *px, double *y, double *py, double *t, double *pt,
              long n, double L, double k, double bg0)
{
    long i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        quad_plane(&x[i], &px[i], L, k);
        quad_plane(&y[i], &py[i], L, -k);
        t[i] = t[i] + L * pt[i] / (bg0 * bg0);
    }
}

/* R3b (NEXT-2): thick axisymmetric linear (plasma) lens, length L, strength k [m^-2]:
 * x'' = -k x and y'' = -k y, i.e. k > 0 focuses BOTH planes (k < 0 defocuses both, k = 0 is a drift);
 * longitudinally a drift.  The paper sets k from the beam moments with an expression of its ref. [31] that it
 * does not print: here k is an input. */
void orc_plens(double *x, double *px, double *y, double *py, double *t, double *pt,
               long n, double L, double k, double bg0)
{
    long i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        quad_plane(&x[i], &px[i], L, k);
        quad_plane(&y[i], &py[i], L, k);
        t[i] = t[i] + L * pt[i] / (bg0 * bg0);
    }
}

/* R4: sector bend, arc length L, bend angle theta (signed), rho = L/theta. */
void orc_sbend(double *x, double *px, double *y, double *py, double *t, double *pt,
               long n, double L, double theta, double bg0)
{
    long i;
    double g0, b0, rho, s, c;
    if (theta == 0.0) {
        orc_drift(x, px, y, py, t, pt, n, L, bg0);
        return;
    }
    g0 = sqrt(1.0 + bg0 * bg0);
    b0 = bg0 / g0;
    rho = L / theta;
    s = sin(theta);
    c = cos(theta);
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double x0 = x[i], px0 = px[i], t0 = t[i], d = pt[i];
        x[i] = c * x0 + rho * s * px0 - (rho / b0) * (1.0 - c) * d;
        px[i] = -(s / rho) * x0 + c * px0 - (s / b0) * d;
        y[i] = y[i] + L * py[i];
        t[i] = t0 + (s / b0) * x0 + (rho / b0) * (1.0 - c) * px0 + rho * (-theta + s / (b0 * b0)) * d;
    }
}

/* R6 to_t: s-coordinates (x,px,y,py,t,pt), reference (bg0) -> fixed-time vector
 * (x_t, y_t, z_t, ux, uy, uz), written to six separate output arrays. */
void orc_to_t(const double *x, const double *px, const double *y, const double *py,
              const double *t, const double *pt, long n, double bg0,
              double *xt, double *yt, double *zt, double *ux, double *uy, double *uz)
{
    long i;
    double g0 = sqrt(1.0 + bg0 * bg0);
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double vx = px[i] * bg0;
        double vy = py[i] * bg0;
        double g = g0 - pt[i] * bg0;
        double vz = sqrt(g * g - 1.0 - vx * vx - vy * vy);
        xt[i] = x[i] - (vx / g) * t[i];
        yt[i] = y[i] - (vy / g) * t[i];
        zt[i] = -(vz / g) * t[i];
        ux[i] = vx;
        uy[i] = vy;
        uz[i] = vz;
    }
}

/* R6 to_s: fixed-time vector (z already relative to the new reference) -> s-coordinates
 * about the new reference (bg1). */
void orc_to_s(const double *xt, const double *yt, const double *zt, const double *ux,
              const double *uy, const double *uz, long n, double bg1,
              double *x, double *px, double *y, double *py, double *t, double *pt)
{
    long i;
    double g1 = sqrt(1.0 + bg1 * bg1);
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double g = sqrt(1.0 + ux[i] * ux[i] + uy[i] * uy[i] + uz[i] * uz[i]);
        x[i] = xt[i] - (ux[i] / uz[i]) * zt[i];
        y[i] = yt[i] - (uy[i] / uz[i]) * zt[i];
        t[i] = -zt[i] * g / uz[i];
        px[i] = ux[i] / bg1;
        py[i] = uy[i] / bg1;
        pt[i] = -(g - g1) / bg1;
    }
}

/* activation codes: 0 identity, 1 ReLU (Eq. 1), 2 PReLU slope a (Eq. 2), 3 tanh */
static double activate(double z, int act, double a)
{
    switch (act) {
    case 1: return z >= 0.0 ? z : 0.0;
    case 2: return z >= 0.0 ? z : a * z;
    case 3: return tanh(z);
    default: return z;
    }
}

/* R8 + R9 (Eq. 3): per particle v (6 values, one from each of the six
 * input arrays) -> (v - mu_in)/sd_in -> L_0, sigma, ..., L_l -> * sd_out + mu_out,
 * written in place.  W: concatenated row-major [out][in] matrices; b: concatenated biases;
 * widths: n_linear+1 entries (6, H, ..., H, 6); prelu_a: n_linear-1 slopes (or NULL). */
void orc_surrogate(double *v0, double *v1, double *v2, double *v3, double *v4, double *v5,
                   long n, int n_linear, const int *widths, const double *W, const double *b,
                   int act, const double *prelu_a,
                   const double *mu_in, const double *sd_in,
                   const double *mu_out, const double *sd_out)
{
    long i;
    int maxw = 0, l;
    double *vv[6];
    vv[0] = v0; vv[1] = v1; vv[2] = v2; vv[3] = v3; vv[4] = v4; vv[5] = v5;
    for (l = 0; l <= n_linear; ++l)
        if (widths[l] > maxw) maxw = widths[l];
#pragma omp parallel
    {
        double *h = (double *)malloc(sizeof(double) * (size_t)maxw);
        double *g = (double *)malloc(sizeof(double) * (size_t)maxw);
#pragma omp for schedule(static)
        for (i = 0; i < n; ++i) {
            const double *Wl = W;
            const double *bl = b;
            int j, o, ll;
            for (j = 0; j < 6; ++j) h[j] = (vv[j][i] - mu_in[j]) / sd_in[j];
            for (ll = 0; ll < n_linear; ++ll) {
                int fin = widths[ll], fout = widths[ll + 1];
                for (o = 0; o < fout; ++o) {
                    double acc = 0.0;
                    for (j = 0; j < fin; ++j) acc += Wl[(size_t)o * fin + j] * h[j];
                    acc += bl[o];
                    if (ll < n_linear - 1)
                        acc = activate(acc, act, prelu_a ? prelu_a[ll] : 0.0);
                    g[o] = acc;
                }
                { double *tmp = h; h = g; g = tmp; }
                Wl += (size_t)fin * fout;
                bl += fout;
            }
            for (j = 0; j < 6; ++j) vv[j][i] = h[j] * sd_out[j] + mu_out[j];
        }
        free(h);
        free(g);
    }
}

/* R10 (G11): uniform weights, 1/N, centred, two-pass.
 * out[0..5] = means; out[6..26] = upper triangle of the covariance, row-major. */
void orc_moments(const double *v0, const double *v1, const double *v2, const double *v3,
                 const double *v4, const double *v5, long n, double *out27)
{
    const double *vv[6];
    double m[6];
    int j, k, idx;
    long i;
    vv[0] = v0; vv[1] = v1; vv[2] = v2; vv[3] = v3; vv[4] = v4; vv[5] = v5;
    for (j = 0; j < 6; ++j) {
        double s = 0.0;
        for (i = 0; i < n; ++i) s += vv[j][i];
        m[j] = n > 0 ? s / (double)n : 0.0;
        out27[j] = m[j];
    }
    idx = 6;
    for (j = 0; j < 6; ++j)
        for (k = j; k < 6; ++k) {
            double s = 0.0;
            for (i = 0; i < n; ++i) s += (vv[j][i] - m[j]) * (vv[k][i] - m[k]);
            out27[idx++] = n > 0 ? s / (double)n : 0.0;
        }
}
