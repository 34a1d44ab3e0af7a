// render_kernels.cu -- shape rendering on the GPU (Block 5 of Fig. 4; shape models PAPER.md:279-281,
// 405-425): Ellipsoid, SphericalHarmonics, RadialMap, VolumeMap -> (delta, beta) grid, rendered directly
// in the beam frame at r_body = R^T r_beam (no resampling step), binary voxelisation at voxel centres, all FP64.
// Readings R18-R21 of DESIGN.md.  One thread per voxel, x fastest (coalesced 8-byte stores); the shapes of a batch are rendered by ONE
// launch per ~30 KB of descriptors (blockIdx.y = shape): the descriptors travel as a __grid_constant__ kernel parameter (no device
// allocation, no host buffer that must outlive the call), the harmonic coefficients of all shapes of a launch in one pool.
#include <cmath>
#include <utility>

#include "internal.h"

namespace scatman {

constexpr int kMaxCoef = 96;

struct RenderArgs {
    int kind;
    float delta, beta;
    int nx, ny, nz;
    double dx, dy, dz;
    double Rt[9];            // row-major R^T: r_body = Rt r_beam
    double a, b, c;          // ellipsoid: 1 / semi-axis
    int ncoef, coef0;        // spherical harmonics: value = sum cn[coef0 + i] P_{l}^{|m|}(cos theta) {1, cos m phi, sin m phi}, i < ncoef
    double r_lo, r_hi;       // every voxel with |r| < r_lo is inside, with |r| > r_hi outside
    double r2_in, r2_out;    // any kind: |r|^2 < r2_in is inside, |r|^2 > r2_out outside, without rotating (-1 / +inf: no such sphere)
    int nlat, nlon;          // radial map
    const double *radii;
    int nvx, nvy, nvz;       // volume map
    const unsigned char *vol;
    double vdx;
};

// The shapes of one launch: descriptors + the pooled harmonic coefficients (sorted per shape by (|m|, l)); < 32 KB of kernel parameters.
constexpr int kBatchShapes = 88, kPoolCoef = 1024;
struct RenderBatch {
    int n;
    RenderArgs a[kBatchShapes];
    double cn[kPoolCoef];                 // c * N_lm * (m != 0 ? sqrt 2 : 1)
    signed char l[kPoolCoef], m[kPoolCoef];   // m as given (sign selects cos / sin)
};
static_assert(sizeof(RenderBatch) <= 32700, "kernel parameters are limited to 32764 bytes");

__constant__ double c_rcp[40];   // 1 / n, n = 1 .. 39 (l <= 32); filled by render_init_device

// R(theta, phi) = sum_i cn[i] P_{l_i}^{|m_i|}(cos theta) {1 | cos |m| phi | sin |m| phi}, the triplets sorted by (|m|, l):
// P_m^m and (cos m phi, sin m phi) advance with m, P_l^m by the upward recurrence in l
//   (l + 1 - m) P_{l+1}^m = (2l + 1) x P_l^m - (l + m) P_{l-1}^m        (Condon-Shortley phase, Eq. 10),
// so one voxel costs O(l_max^2) FP64 operations and no trigonometric call.
__device__ double sh_radius(const RenderArgs &A, const double *__restrict__ Acn, const signed char *__restrict__ Al,
                            const signed char *__restrict__ Am, double ct, double cphi, double sphi) {
    const double st = sqrt(fmax(0.0, 1.0 - ct * ct));
    double R = 0.0, pmm = 1.0, cm = 1.0, sm = 0.0;
    int am = 0, i = 0;
    while (i < A.ncoef) {
        const int target = Am[i] < 0 ? -Am[i] : Am[i];
        while (am < target) {
            ++am;
            pmm = -pmm * (double)(2 * am - 1) * st;
            const double t = cm * cphi - sm * sphi;
            sm = sm * cphi + cm * sphi;
            cm = t;
        }
        double pl = pmm, pl_prev = 0.0;
        int lcur = am;
        while (i < A.ncoef && (Am[i] < 0 ? -Am[i] : Am[i]) == am) {
            const int l = Al[i];
            while (lcur < l) {
                // (an FP64 division costs ~40 instructions; 1 / n comes from a table, one rounding more than the quotient,
                // far inside the surface-tie margin of the rendering)
                const double pn = ((double)(2 * lcur + 1) * ct * pl - (double)(lcur + am) * pl_prev) * c_rcp[lcur + 1 - am];
                pl_prev = pl;
                pl = pn;
                ++lcur;
            }
            const double ang = Am[i] > 0 ? cm : (Am[i] < 0 ? sm : 1.0);
            R = fma(Acn[i] * pl, ang, R);
            ++i;
        }
    }
    return R;
}

__global__ void render_kernel(const __grid_constant__ RenderBatch Bt, float2 *__restrict__ out) {
    const double kPi = 3.14159265358979323846;
    const RenderArgs &A = Bt.a[blockIdx.y];
    const size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t nvox = (size_t)A.nx * A.ny * A.nz;
    if (v >= nvox) return;
    out += (size_t)blockIdx.y * nvox;
    int ix, iy, iz;
    if (nvox <= 0x7fffffffull) {   // 32-bit divisions (the usual case)
        const unsigned v32 = (unsigned)v, row = v32 / (unsigned)A.nx;
        ix = (int)(v32 - row * (unsigned)A.nx);
        iz = (int)(row / (unsigned)A.ny);
        iy = (int)(row - (unsigned)iz * (unsigned)A.ny);
    } else {
        ix = (int)(v % A.nx); iy = (int)((v / A.nx) % A.ny); iz = (int)(v / ((size_t)A.nx * A.ny));
    }
    const double x = ((double)ix - 0.5 * (double)(A.nx - 1)) * A.dx;
    const double y = ((double)iy - 0.5 * (double)(A.ny - 1)) * A.dy;
    const double z = ((double)iz - 0.5 * (double)(A.nz - 1)) * A.dz;
    // |r| does not change under the rotation: voxels inside the shape's inscribed sphere or outside its circumscribed one are
    // decided from x^2 + y^2 + z^2 alone (most of a grid); the margins of 1e-12 leave every close call to the full test below,
    // so the rendering is voxel for voxel what the full test gives.
    const double r2 = x * x + y * y + z * z;
    if (r2 > A.r2_out || r2 < A.r2_in) {
        out[v] = r2 < A.r2_in ? make_float2(A.delta, A.beta) : make_float2(0.f, 0.f);
        return;
    }
    const double xb = A.Rt[0] * x + A.Rt[1] * y + A.Rt[2] * z;
    const double yb = A.Rt[3] * x + A.Rt[4] * y + A.Rt[5] * z;
    const double zb = A.Rt[6] * x + A.Rt[7] * y + A.Rt[8] * z;
    bool inside = false;
    if (A.kind == SCATMAN_SHAPE_ELLIPSOID) {
        const double u = xb * A.a, w = yb * A.b, t = zb * A.c;   // A.a, A.b, A.c hold the reciprocal semi-axes
        inside = u * u + w * w + t * t <= 1.0;
    } else if (A.kind == SCATMAN_SHAPE_SPHERICAL_HARMONICS) {
        const double r = sqrt(xb * xb + yb * yb + zb * zb);
        if (r < A.r_lo) inside = true;
        else if (r <= A.r_hi) {
            const double ir = r > 0.0 ? 1.0 / r : 0.0;
            const double ct = r > 0.0 ? zb * ir : 1.0;
            const double rho = sqrt(xb * xb + yb * yb);
            const double irho = rho > 0.0 ? 1.0 / rho : 0.0;
            const double cphi = rho > 0.0 ? xb * irho : 1.0, sphi = yb * irho;   // phi = atan2(y, x)
            const double R = sh_radius(A, Bt.cn + A.coef0, Bt.l + A.coef0, Bt.m + A.coef0, ct, cphi, sphi);
            inside = r <= R;
        }
    } else if (A.kind == SCATMAN_SHAPE_RADIAL_MAP) {
        const double r = sqrt(xb * xb + yb * yb + zb * zb);
        const double sl = r > 0.0 ? fmin(1.0, fmax(-1.0, zb / r)) : 0.0;
        const double lat = asin(sl);
        double lon = atan2(yb, xb);
        if (lon < 0.0) lon += 2.0 * kPi;
        const double fi = fmin(fmax((lat + 0.5 * kPi) / (kPi / (double)A.nlat), 0.0), (double)(A.nlat - 1));
        const double fj = lon / (2.0 * kPi / (double)A.nlon);
        const int i0 = min((int)floor(fi), A.nlat - 1), i1 = min(i0 + 1, A.nlat - 1);
        const double ti = fi - (double)i0;
        const double j0f = floor(fj), tj = fj - j0f;
        const int j0 = (((int)j0f % A.nlon) + A.nlon) % A.nlon, j1 = (j0 + 1) % A.nlon;
        const double lo = A.radii[(size_t)i0 * A.nlon + j0] * (1.0 - tj) + A.radii[(size_t)i0 * A.nlon + j1] * tj;
        const double hi = A.radii[(size_t)i1 * A.nlon + j0] * (1.0 - tj) + A.radii[(size_t)i1 * A.nlon + j1] * tj;
        inside = r <= lo * (1.0 - ti) + hi * ti;
    } else {
        const double fx = xb * A.vdx + 0.5 * (double)A.nvx, fy = yb * A.vdx + 0.5 * (double)A.nvy,
                     fz = zb * A.vdx + 0.5 * (double)A.nvz;   // A.vdx holds 1 / cell size
        const double cx = floor(fx), cy = floor(fy), cz = floor(fz);
        if (cx >= 0.0 && cx < (double)A.nvx && cy >= 0.0 && cy < (double)A.nvy && cz >= 0.0 && cz < (double)A.nvz)
            inside = A.vol[((size_t)cz * A.nvy + (size_t)cy) * A.nvx + (size_t)cx] != 0;
    }
    out[v] = inside ? make_float2(A.delta, A.beta) : make_float2(0.f, 0.f);
}

cudaError_t render_init_device() {   // per device (scatman_create)
    double rcp[40];
    rcp[0] = 0.0;
    for (int n = 1; n < 40; ++n) rcp[n] = 1.0 / (double)n;
    return cudaMemcpyToSymbol(c_rcp, rcp, sizeof(rcp));
}

static double factorial_d(int n) {
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= (double)i;
    return f;
}

// Fills descriptor A (and, for harmonics, coefficients at coef0 of the pool arrays).  0 ok, 1 bad argument.
static int fill_render_args(const scatman_shape &s, const scatman_grid &g, RenderArgs &A, double *Acn, signed char *Al, signed char *Am) {
    const double kPi = 3.14159265358979323846;
    A = RenderArgs{};
    A.r2_in = -1.0;
    A.r2_out = INFINITY;
    A.kind = s.kind;
    A.delta = s.delta;
    A.beta = s.beta;
    A.nx = g.nx; A.ny = g.ny; A.nz = g.nz;
    A.dx = g.dx; A.dy = g.dy; A.dz = g.dz;
    const double w = s.quat[0], a = s.quat[1], b = s.quat[2], c = s.quat[3];
    if (!(std::fabs(w * w + a * a + b * b + c * c - 1.0) <= 2e-6)) return 1;
    const double R[9] = {1 - 2 * (b * b + c * c), 2 * (a * b - w * c),     2 * (a * c + w * b),
                         2 * (a * b + w * c),     1 - 2 * (a * a + c * c), 2 * (b * c - w * a),
                         2 * (a * c - w * b),     2 * (b * c + w * a),     1 - 2 * (a * a + b * b)};
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) A.Rt[3 * i + j] = R[3 * j + i];
    switch (s.kind) {
        case SCATMAN_SHAPE_ELLIPSOID:
            if (!(s.a > 0.0 && s.b > 0.0 && s.c > 0.0)) return 1;
            A.a = 1.0 / s.a; A.b = 1.0 / s.b; A.c = 1.0 / s.c;
            {
                const double rmin = std::fmin(s.a, std::fmin(s.b, s.c)), rmax = std::fmax(s.a, std::fmax(s.b, s.c));
                A.r2_in = rmin * rmin * (1.0 - 1e-12);
                A.r2_out = rmax * rmax * (1.0 + 1e-12);
            }
            break;
        case SCATMAN_SHAPE_SPHERICAL_HARMONICS: {
            if (s.ncoef < 1 || s.ncoef > kMaxCoef || !s.h_coef) return 1;
            // |sum_m c_lm Y_lm| <= sqrt(sum_m c_lm^2) sqrt((2l+1)/4pi) (addition theorem): brackets R around its l = 0 part
            double norm2[33] = {0};
            double r00 = 0.0;
            for (int i = 0; i < s.ncoef; ++i) {
                const int l = (int)s.h_coef[3 * i], m = (int)s.h_coef[3 * i + 1];
                const double cv = s.h_coef[3 * i + 2];
                if ((double)l != s.h_coef[3 * i] || (double)m != s.h_coef[3 * i + 1] || l < 0 || l > 32 || m < -l || m > l ||
                    !std::isfinite(cv))
                    return 1;
                const int am = m < 0 ? -m : m;
                const double n = std::sqrt((2 * l + 1) / (4 * kPi) * factorial_d(l - am) / factorial_d(l + am));
                Al[i] = (signed char)l;
                Am[i] = (signed char)m;
                Acn[i] = cv * n * (m != 0 ? std::sqrt(2.0) : 1.0);
                if (l == 0) r00 += cv * n;
                else norm2[l] += cv * cv;
            }
            double bound = 0.0;
            for (int l = 1; l <= 32; ++l) bound += std::sqrt(norm2[l]) * std::sqrt((2 * l + 1) / (4 * kPi));
            A.ncoef = s.ncoef;
            for (int i = 1; i < A.ncoef; ++i)   // insertion sort by (|m|, l): the order sh_radius walks
                for (int j = i; j > 0; --j) {
                    const int ka = (Am[j] < 0 ? -Am[j] : Am[j]) * 64 + Al[j];
                    const int kb = (Am[j - 1] < 0 ? -Am[j - 1] : Am[j - 1]) * 64 + Al[j - 1];
                    if (ka >= kb) break;
                    std::swap(Al[j], Al[j - 1]);
                    std::swap(Am[j], Am[j - 1]);
                    std::swap(Acn[j], Acn[j - 1]);
                }
            A.r_lo = (r00 - bound) * (1.0 - 1e-9) - 1e-300;
            A.r_hi = (r00 + bound) * (1.0 + 1e-9) + 1e-300;
            A.r2_in = A.r_lo > 0.0 ? A.r_lo * A.r_lo * (1.0 - 1e-12) : -1.0;
            A.r2_out = A.r_hi > 0.0 ? A.r_hi * A.r_hi * (1.0 + 1e-12) : 0.0;   // r_hi <= 0: the radius is nowhere positive
            break;
        }
        case SCATMAN_SHAPE_RADIAL_MAP:
            if (s.nlat < 1 || s.nlon < 1 || !s.d_radii) return 1;
            A.nlat = s.nlat; A.nlon = s.nlon; A.radii = s.d_radii;
            break;
        case SCATMAN_SHAPE_VOLUME_MAP:
            if (s.nvx < 1 || s.nvy < 1 || s.nvz < 1 || !s.d_volume || !(s.vdx > 0.0)) return 1;
            A.nvx = s.nvx; A.nvy = s.nvy; A.nvz = s.nvz; A.vol = s.d_volume; A.vdx = 1.0 / s.vdx;
            A.r2_out = 0.25 * s.vdx * s.vdx * ((double)s.nvx * s.nvx + (double)s.nvy * s.nvy + (double)s.nvz * s.nvz) * (1.0 + 1e-12);
            break;
        default: return 1;
    }
    return 0;
}

// Renders h_shapes[0 .. batch) into d_dn[batch][nz][ny][nx][2]: one launch per RenderBatch of descriptors.
// Returns 0, or 1 + the index of the first bad descriptor; *err = the CUDA status; *nlaunch = kernels launched.
int launch_render_batch(const scatman_shape *h_shapes, int batch, const scatman_grid &g, float *d_dn, cudaStream_t st, cudaError_t *err,
                        int *nlaunch) {
    *err = cudaSuccess;
    *nlaunch = 0;
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    static thread_local RenderBatch Bt;       // 31 KB: not on the stack
    int b = 0;
    while (b < batch) {
        const int first = b;
        int pool = 0;
        Bt.n = 0;
        while (b < batch && Bt.n < kBatchShapes) {
            const scatman_shape &s = h_shapes[b];
            const int nc = s.kind == SCATMAN_SHAPE_SPHERICAL_HARMONICS ? s.ncoef : 0;
            if (nc < 0 || nc > kMaxCoef) return 1 + b;
            if (pool + nc > kPoolCoef) break;
            if (fill_render_args(s, g, Bt.a[Bt.n], Bt.cn + pool, Bt.l + pool, Bt.m + pool)) return 1 + b;
            Bt.a[Bt.n].coef0 = pool;
            pool += nc;
            ++Bt.n;
            ++b;
        }
        render_kernel<<<dim3((unsigned)((nvox + 255) / 256), (unsigned)Bt.n), 256, 0, st>>>(Bt, (float2 *)d_dn + (size_t)first * nvox);
        ++*nlaunch;
        *err = cudaGetLastError();
        if (*err != cudaSuccess) return 0;
    }
    return 0;
}

}  // namespace scatman
