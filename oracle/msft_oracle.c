/*
 * msft_oracle.c -- FP64 CPU ORACLE for the MSFT forward simulation (arXiv 2202.03411).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with the
 * CUDA path under paper_2202_03411_b200/csrc and is deliberately plain: direct summation,
 * no FFT, no BLAS, no blocking or fusion beyond what the definition states.
 *
 * What it computes (BASELINE.json north_star; Eq. 2-9):
 *
 *   dn_j(x,y)  = delta + i beta                                  (Eq. 7; input)
 *   C_j(x,y)   = sum_{l<j} dn_l(x,y)                             (exclusive: Eq. 9 E_{s=0}=E_0,
 *                                                                 PAPER.md:129-131; Blocks 8->9,
 *                                                                 PAPER.md:158-160)
 *   rho_j(x,y) = f(dn_j) exp(i k dz C_j) dV                      (Eq. 6, 8, 9)
 *                f(c) = c (LINEAR, north_star) | c (2 - c) (N2M1: n^2-1 up to sign/conj, Eq. 5)
 *   A(p)       = sum_j sum_y sum_x rho_j(x,y) exp(i (qx x_i + qy y_i + qz z_j))   (Eq. 2, 4)
 *   I(p)       = |A(p)|^2                                        (Block 11 :164)
 *   q(p)       = k (s_p - z^),  s_p = (u, v, 1)/r                (Eq. 3; north_star)
 *
 * Sign convention: north_star's (dn = delta + i beta, q = k(s - z^)), the exact complex
 * conjugate of the paper's (n = 1 - delta + i beta, q = k0 - k): A = -conj(A_paper), same I.
 * oracle/eq9_literal.py follows the paper's signs and slice loop literally; tests pin the two
 * against each other (pin P7).
 *
 * Pins (tests/test_oracle_pins.py): P1 direct == tables; P2 closed-form absorbing cuboid;
 * P3 forward pixel; P4 Born sphere form factor; P5 D4 symmetry; P6 translation invariance;
 * P7 literal Eq. 9; P8 numpy.fft on the DFT grid; P9 one/two voxels; P10 N2M1 vs LINEAR;
 * P11 orientation by 90-degree turns.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libmsft_oracle.so msft_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_RHO_LINEAR 0
#define ORACLE_RHO_N2M1 1

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* centred voxel coordinate (SURVEY 8c-6 / DESIGN.md R6) */
static double centre(int i, int n, double d) { return ((double)i - 0.5 * (double)(n - 1)) * d; }

/*
 * q-map (Eq. 3; north_star "q = k(s_pixel - z^)"; R9, R10).
 * Flat detector at unit distance, perpendicular to the beam, npx x npy square pixels whose
 * outer edge mid-points sit at theta_max; pixel centres at half-integer offsets.
 * q[3*p + {0,1,2}], p = iy*npx + ix.  qz by the cancellation-free form -k(u^2+v^2)/(r(r+1)).
 */
void oracle_qmap(int npx, int npy, double theta_max_deg, double cx, double cy, double lambda, double *q) {
    const double k = 2.0 * M_PI / lambda;
    const double pitch = 2.0 * tan(theta_max_deg * M_PI / 180.0) / (double)npx;
    for (int iy = 0; iy < npy; ++iy)
        for (int ix = 0; ix < npx; ++ix) {
            double u = ((double)ix + 0.5 - 0.5 * (double)npx + cx) * pitch;
            double v = ((double)iy + 0.5 - 0.5 * (double)npy + cy) * pitch;
            double r = sqrt(u * u + v * v + 1.0);
            double *o = q + 3 * ((size_t)iy * npx + ix);
            o[0] = k * u / r;
            o[1] = k * v / r;
            o[2] = -k * (u * u + v * v) / (r * (r + 1.0));
        }
}

/*
 * Orientation (Block 5 "render at the proper spatial coordinates"; Fig. 6,
 * PAPER.md:289; R11).  quat = (w,x,y,z), unit, body->beam: r_beam = R r_body.
 * The beam-frame grid (same dims, same voxel) samples the body-frame grid at
 * r_body = R^T r_beam by trilinear interpolation in FP64, zero outside, rounded to FP32.
 */
void oracle_orient(const float *dn_in, int nx, int ny, int nz, double dx, double dy, double dz,
                   const double *quat, float *dn_out) {
    const double w = quat[0], a = quat[1], b = quat[2], c = quat[3];
    /* rotation matrix R (body->beam) */
    const double R[3][3] = {
        {1 - 2 * (b * b + c * c), 2 * (a * b - w * c), 2 * (a * c + w * b)},
        {2 * (a * b + w * c), 1 - 2 * (a * a + c * c), 2 * (b * c - w * a)},
        {2 * (a * c - w * b), 2 * (b * c + w * a), 1 - 2 * (a * a + b * b)}};
#pragma omp parallel for schedule(static)
    for (int iz = 0; iz < nz; ++iz)
        for (int iy = 0; iy < ny; ++iy)
            for (int ix = 0; ix < nx; ++ix) {
                const double xb = centre(ix, nx, dx), yb = centre(iy, ny, dy), zb = centre(iz, nz, dz);
                /* r_body = R^T r_beam */
                const double xo = R[0][0] * xb + R[1][0] * yb + R[2][0] * zb;
                const double yo = R[0][1] * xb + R[1][1] * yb + R[2][1] * zb;
                const double zo = R[0][2] * xb + R[1][2] * yb + R[2][2] * zb;
                const double fx = xo / dx + 0.5 * (double)(nx - 1);
                const double fy = yo / dy + 0.5 * (double)(ny - 1);
                const double fz = zo / dz + 0.5 * (double)(nz - 1);
                const double flx = floor(fx), fly = floor(fy), flz = floor(fz);
                const int x0 = (int)flx, y0 = (int)fly, z0 = (int)flz;
                const double tx = fx - flx, ty = fy - fly, tz = fz - flz;
                double acc[2] = {0.0, 0.0};
                for (int cz = 0; cz < 2; ++cz)
                    for (int cy = 0; cy < 2; ++cy)
                        for (int cxx = 0; cxx < 2; ++cxx) {
                            const int xi = x0 + cxx, yi = y0 + cy, zi = z0 + cz;
                            if (xi < 0 || xi >= nx || yi < 0 || yi >= ny || zi < 0 || zi >= nz) continue;
                            const double wgt = (cxx ? tx : 1.0 - tx) * (cy ? ty : 1.0 - ty) * (cz ? tz : 1.0 - tz);
                            const float *s = dn_in + 2 * (((size_t)zi * ny + yi) * nx + xi);
                            acc[0] += wgt * (double)s[0];
                            acc[1] += wgt * (double)s[1];
                        }
                float *o = dn_out + 2 * (((size_t)iz * ny + iy) * nx + ix);
                o[0] = (float)acc[0];
                o[1] = (float)acc[1];
            }
}

/*
 * Effective scattering strength of every voxel (Eq. 6, 8, 9):
 * exclusive prefix along z of dn = delta + i beta, transmission T = exp(i k dz C), strength
 * rho = f(dn) T dV.  rho[2*(((z*ny)+y)*nx+x) + {0,1}] = (Re, Im).
 */
void oracle_effective_strength(const float *dn, int nx, int ny, int nz, double dx, double dy, double dz,
                               double lambda, int rho_mode, double *rho) {
    const double k = 2.0 * M_PI / lambda;
    const double dV = dx * dy * dz;
    for (int iy = 0; iy < ny; ++iy)
        for (int ix = 0; ix < nx; ++ix) {
            double Cre = 0.0, Cim = 0.0; /* C_0 = 0: slice 0 sees E_0 */
            for (int iz = 0; iz < nz; ++iz) {
                const size_t v = ((size_t)iz * ny + iy) * nx + ix;
                const double d = (double)dn[2 * v], b = (double)dn[2 * v + 1];
                /* T = exp(i k dz (Cre + i Cim)) = exp(-k dz Cim) (cos(k dz Cre) + i sin(k dz Cre)) */
                const double mag = exp(-k * dz * Cim);
                const double Tre = mag * cos(k * dz * Cre), Tim = mag * sin(k * dz * Cre);
                double fre, fim;
                if (rho_mode == ORACLE_RHO_N2M1) { /* c (2 - c), c = d + i b */
                    fre = d * (2.0 - d) + b * b;
                    fim = b * (2.0 - d) - d * b;
                } else {
                    fre = d;
                    fim = b;
                }
                rho[2 * v] = (fre * Tre - fim * Tim) * dV;
                rho[2 * v + 1] = (fre * Tim + fim * Tre) * dV;
                Cre += d;
                Cim += b;
            }
        }
}

/*
 * O1: the definition, one sincos of the full phase per term (Eq. 1-2).
 * A[2*p + {0,1}].  Small cases only.
 */
void oracle_amplitude_direct(const double *rho, int nx, int ny, int nz, double dx, double dy, double dz,
                             const double *q, int64_t npix, double *A) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t p = 0; p < npix; ++p) {
        const double qx = q[3 * p], qy = q[3 * p + 1], qz = q[3 * p + 2];
        double are = 0.0, aim = 0.0;
        for (int iz = 0; iz < nz; ++iz)
            for (int iy = 0; iy < ny; ++iy)
                for (int ix = 0; ix < nx; ++ix) {
                    const size_t v = ((size_t)iz * ny + iy) * nx + ix;
                    const double rr = rho[2 * v], ri = rho[2 * v + 1];
                    if (rr == 0.0 && ri == 0.0) continue;
                    const double ph = qx * centre(ix, nx, dx) + qy * centre(iy, ny, dy) + qz * centre(iz, nz, dz);
                    const double c = cos(ph), s = sin(ph);
                    are += rr * c - ri * s;
                    aim += rr * s + ri * c;
                }
        A[2 * p] = are;
        A[2 * p + 1] = aim;
    }
}

/*
 * O2: the same triple sum with the phase factor written as the product of three per-pixel
 * 1-D FP64 tables e^{i qx x_i} e^{i qy y_i} e^{i qz z_j} (Eq. 2's split).
 * Still a direct summation over every voxel (exact zeros skipped); OpenMP over pixels.
 */
void oracle_amplitude_tables(const double *rho, int nx, int ny, int nz, double dx, double dy, double dz,
                             const double *q, int64_t npix, double *A) {
#pragma omp parallel
    {
        double *ex = (double *)malloc(sizeof(double) * 2 * (size_t)nx);
        double *ey = (double *)malloc(sizeof(double) * 2 * (size_t)ny);
        double *ez = (double *)malloc(sizeof(double) * 2 * (size_t)nz);
#pragma omp for schedule(dynamic, 4)
        for (int64_t p = 0; p < npix; ++p) {
            const double qx = q[3 * p], qy = q[3 * p + 1], qz = q[3 * p + 2];
            for (int i = 0; i < nx; ++i) { double ph = qx * centre(i, nx, dx); ex[2 * i] = cos(ph); ex[2 * i + 1] = sin(ph); }
            for (int i = 0; i < ny; ++i) { double ph = qy * centre(i, ny, dy); ey[2 * i] = cos(ph); ey[2 * i + 1] = sin(ph); }
            for (int i = 0; i < nz; ++i) { double ph = qz * centre(i, nz, dz); ez[2 * i] = cos(ph); ez[2 * i + 1] = sin(ph); }
            double are = 0.0, aim = 0.0;
            for (int iz = 0; iz < nz; ++iz) {
                double sre = 0.0, sim = 0.0; /* slice sum  sum_y e^{i qy y} sum_x rho e^{i qx x} */
                for (int iy = 0; iy < ny; ++iy) {
                    const double *row = rho + 2 * (((size_t)iz * ny + iy) * nx);
                    double rre = 0.0, rim = 0.0;
                    for (int ix = 0; ix < nx; ++ix) {
                        const double rr = row[2 * ix], ri = row[2 * ix + 1];
                        if (rr == 0.0 && ri == 0.0) continue;
                        rre += rr * ex[2 * ix] - ri * ex[2 * ix + 1];
                        rim += rr * ex[2 * ix + 1] + ri * ex[2 * ix];
                    }
                    sre += rre * ey[2 * iy] - rim * ey[2 * iy + 1];
                    sim += rre * ey[2 * iy + 1] + rim * ey[2 * iy];
                }
                are += sre * ez[2 * iz] - sim * ez[2 * iz + 1];
                aim += sre * ez[2 * iz + 1] + sim * ez[2 * iz];
            }
            A[2 * p] = are;
            A[2 * p + 1] = aim;
        }
        free(ex);
        free(ey);
        free(ez);
    }
}

/*
 * Whole path for one grid: [orient ->] effective strength -> amplitude at the given q list ->
 * intensity.  quat may be NULL (identity: no resampling).  method 0 = tables (O2), 1 = direct (O1).
 * A_out (2*npix) may be NULL.  Returns 0, or -1 if out of memory.
 */
int oracle_simulate_q(const float *dn, int nx, int ny, int nz, double dx, double dy, double dz,
                      double lambda, const double *quat, int rho_mode, const double *q, int64_t npix,
                      int method, double *I_out, double *A_out) {
    const size_t nvox = (size_t)nx * ny * nz;
    float *rot = NULL;
    const float *src = dn;
    if (quat) {
        rot = (float *)malloc(sizeof(float) * 2 * nvox);
        if (!rot) return -1;
        oracle_orient(dn, nx, ny, nz, dx, dy, dz, quat, rot);
        src = rot;
    }
    double *rho = (double *)malloc(sizeof(double) * 2 * nvox);
    double *A = (double *)malloc(sizeof(double) * 2 * (size_t)npix);
    if (!rho || !A) { free(rot); free(rho); free(A); return -1; }
    oracle_effective_strength(src, nx, ny, nz, dx, dy, dz, lambda, rho_mode, rho);
    if (method == 1) oracle_amplitude_direct(rho, nx, ny, nz, dx, dy, dz, q, npix, A);
    else oracle_amplitude_tables(rho, nx, ny, nz, dx, dy, dz, q, npix, A);
    for (int64_t p = 0; p < npix; ++p) I_out[p] = A[2 * p] * A[2 * p] + A[2 * p + 1] * A[2 * p + 1];
    if (A_out) memcpy(A_out, A, sizeof(double) * 2 * (size_t)npix);
    free(rot);
    free(rho);
    free(A);
    return 0;
}
