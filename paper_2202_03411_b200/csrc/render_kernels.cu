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
    int dense_L;             // 4, 6, 8: cn[coef0 ...] holds the dense cos | sin tables of sh_radius_dense<dense_L> instead (0: the triplets)
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

// The same sum for harmonics up to degree L <= 8 from DENSE coefficient tables -- cc / cs[p(m, l)] = the cos (or m = 0) and sin
// coefficients of the pair (l, m >= 0), pairs enumerated m-major (p = 0: (0,0), 1: (1,0) ... L: (L,0), L+1: (1,1) ...), zeros where
// the shape has no such triplet -- as straight-line code: the loops below unroll completely, the recurrence factors
// (2l-1)/(l-m), (l+m-1)/(l-m) and (2m-1) are compile-time constants, nothing is indexed by data.  (The walker above spends most of
// its time in loop control and in loads of l, m from the parameter bank, not in arithmetic: profiles/r02_orient_render.md.)
template <int L>
__device__ __forceinline__ double sh_radius_dense(const double *__restrict__ cc, const double *__restrict__ cs, double ct, double st,
                                                   double cphi, double sphi) {
    double R = 0.0, pmm = 1.0, cm = 1.0, sm = 0.0;
    int p = 0;
#pragma unroll
    for (int m = 0; m <= L; ++m) {
        if (m > 0) {
            pmm = -pmm * (double)(2 * m - 1) * st;
            const double t = cm * cphi - sm * sphi;
            sm = sm * cphi + cm * sphi;
            cm = t;
        }
        double pl = pmm, pl_prev = 0.0, S = 0.0, T = 0.0;
#pragma unroll
        for (int l = m; l <= L; ++l) {
            if (l > m) {
                const double pn = (double)(2 * l - 1) / (double)(l - m) * ct * pl - (double)(l + m - 1) / (double)(l - m) * pl_prev;
                pl_prev = pl;
                pl = pn;
            }
            S = fma(cc[p], pl, S);
            if (m > 0) T = fma(cs[p], pl, T);
            ++p;
        }
        R = fma(S, cm, R);
        if (m > 0) R = fma(T, sm, R);
    }
    return R;
}
__host__ __device__ constexpr int sh_pairs(int L) { return (L + 1) * (L + 2) / 2; }

// Is the voxel centre (x, y, z) (beam frame) inside shape A?  The full test, after the sphere tests of the caller.
__device__ bool render_inside(const RenderBatch &Bt, const RenderArgs &A, double x, double y, double z) {
    const double kPi = 3.14159265358979323846;
    const double xb = A.Rt[0] * x + A.Rt[1] * y + A.Rt[2] * z;
    const double yb = A.Rt[3] * x + A.Rt[4] * y + A.Rt[5] * z;
    const double zb = A.Rt[6] * x + A.Rt[7] * y + A.Rt[8] * z;
    if (A.kind == SCATMAN_SHAPE_ELLIPSOID) {
        const double u = xb * A.a, w = yb * A.b, t = zb * A.c;   // A.a, A.b, A.c hold the reciprocal semi-axes
        return u * u + w * w + t * t <= 1.0;
    }
    if (A.kind == SCATMAN_SHAPE_SPHERICAL_HARMONICS) {
        // two reciprocal square roots instead of three square roots and two divisions (each ~30 FP64 instructions): r = r^2 / r,
        // cos theta = z / r, sin theta = rho / r, (cos phi, sin phi) = (x, y) / rho
        const double rho2 = xb * xb + yb * yb, r2 = rho2 + zb * zb;
        const double ir = r2 > 0.0 ? rsqrt(r2) : 0.0;
        const double r = r2 * ir;
        if (r < A.r_lo) return true;
        if (r > A.r_hi) return false;
        const double ct = r2 > 0.0 ? zb * ir : 1.0;
        const double irho = rho2 > 0.0 ? rsqrt(rho2) : 0.0;
        const double cphi = rho2 > 0.0 ? xb * irho : 1.0, sphi = yb * irho;   // phi = atan2(y, x)
        double R;
        if (A.dense_L > 0) {
            const double st = rho2 * irho * ir;
            const double *cc = Bt.cn + A.coef0;
            if (A.dense_L == 4) R = sh_radius_dense<4>(cc, cc + sh_pairs(4), ct, st, cphi, sphi);
            else if (A.dense_L == 6) R = sh_radius_dense<6>(cc, cc + sh_pairs(6), ct, st, cphi, sphi);
            else R = sh_radius_dense<8>(cc, cc + sh_pairs(8), ct, st, cphi, sphi);
        } else {
            R = sh_radius(A, Bt.cn + A.coef0, Bt.l + A.coef0, Bt.m + A.coef0, ct, cphi, sphi);
        }
        return r <= R;
    }
    if (A.kind == SCATMAN_SHAPE_RADIAL_MAP) {
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
        return r <= lo * (1.0 - ti) + hi * ti;
    }
    const double fx = xb * A.vdx + 0.5 * (double)A.nvx, fy = yb * A.vdx + 0.5 * (double)A.nvy,
                 fz = zb * A.vdx + 0.5 * (double)A.nvz;   // A.vdx holds 1 / cell size
    const double cx = floor(fx), cy = floor(fy), cz = floor(fz);
    if (cx >= 0.0 && cx < (double)A.nvx && cy >= 0.0 && cy < (double)A.nvy && cz >= 0.0 && cz < (double)A.nvz)
        return A.vol[((size_t)cz * A.nvy + (size_t)cy) * A.nvx + (size_t)cx] != 0;
    return false;
}

// A WARP renders a run of up to 128 consecutive x of EIGHT consecutive rows (y .. y + 7, one z) of one shape (blockIdx.y): lane i takes
// x0 + i, x0 + i + 32, ..., so that every store of the warp is 256 contiguous bytes; the index arithmetic of a work item (integer
// divisions, the descriptor's fields from the parameter bank) is done once per 8 x 128 voxels -- with one row per warp it was most
// of the ~230 instructions that a row outside the shape cost, and those rows are most of a grid; a row that misses the shape's
// circumscribed sphere altogether is zero-filled without looking at its voxels.
// tilemap != null: SPARSE output for launch_sep_tc_prefix_prep, as launch_orient's -- a tile of 16 x 4 x 4 voxels whose nearest point to
// the centre lies outside the circumscribed sphere is not written at all, tilemap[shape][z / 4][y / 4][x / 16] = 0 says so (every row of
// a tile takes the same decision: it depends on the tile's indices only).
constexpr int kRenderRun = 128, kRenderRows = 8;
// min of coordinate^2 over cells i0 .. i0 + len - 1.  FP32: the decision only has to be the same in every row of a tile (it is a
// function of the tile's indices) and must never drop a tile that holds a voxel inside the sphere -- the sphere is widened by 1e-5.
__device__ __forceinline__ float nearest_sq(int i0, int n, float d, int len) {
    const float a = ((float)i0 - 0.5f * (float)(n - 1)) * d, b = a + (float)(len - 1) * d;
    return a > 0.f ? a * a : (b < 0.f ? b * b : 0.f);
}
__global__ void __launch_bounds__(256)
render_kernel(const __grid_constant__ RenderBatch Bt, float2 *__restrict__ out, unsigned char *__restrict__ tilemap) {
    const RenderArgs &A = Bt.a[blockIdx.y];
    const int lane = threadIdx.x & 31;
    const unsigned runs = (unsigned)(A.nx + kRenderRun - 1) / kRenderRun;      // runs per row
    const unsigned ygroups = (unsigned)(A.ny + kRenderRows - 1) / kRenderRows;
    const unsigned long long w = (unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);   // work item
    const unsigned long long ngroups = (unsigned long long)ygroups * A.nz;     // < 2^32 (ny <= 8192, nz <= 65535)
    if (w >= ngroups * runs) return;
    unsigned grp, run;                                                         // (a 64-bit division costs ~70 instructions: only if needed)
    if (runs == 1) { grp = (unsigned)w; run = 0; }
    else if (w <= 0xffffffffull) { grp = (unsigned)w / runs; run = (unsigned)w - grp * runs; }
    else { grp = (unsigned)(w / runs); run = (unsigned)(w - (unsigned long long)grp * runs); }
    const int iz = (int)(grp / ygroups), iy0 = (int)(grp - (unsigned)iz * ygroups) * kRenderRows;
    const int x0 = (int)run * kRenderRun, x1 = min(A.nx, x0 + kRenderRun);
    const int nx = A.nx, ny = A.ny;
    const double dx = A.dx, dy = A.dy, r2_out = A.r2_out, r2_in = A.r2_in;
    const double z = ((double)iz - 0.5 * (double)(A.nz - 1)) * A.dz;
    const float2 vac = make_float2(0.f, 0.f), mat = make_float2(A.delta, A.beta);
    float2 *dst = out + ((size_t)blockIdx.y * A.nz + iz) * ((size_t)nx * ny) + (size_t)iy0 * nx;
    // sparse output: the tiles' decisions
    const int nbx = (nx + 15) / 16;
    const float fdx = (float)dx, r2o = (float)r2_out * 1.00001f;
    const float tz2 = tilemap ? nearest_sq(iz & ~3, A.nz, (float)A.dz, 4) : 0.f;
    unsigned char *tm = tilemap ? tilemap + (((size_t)blockIdx.y * ((A.nz + 3) / 4) + (iz >> 2)) * ((ny + 3) / 4) + (iy0 >> 2)) * nbx : nullptr;
    float tyz2 = 0.f;
    bool rows_out = false;
#pragma unroll 1
    for (int r = 0; r < kRenderRows && iy0 + r < ny; ++r, dst += nx) {
        const int iy = iy0 + r;
        const double y = ((double)iy - 0.5 * (double)(ny - 1)) * dy;
        // |r| does not change under the rotation: voxels inside the shape's inscribed sphere or outside its circumscribed one are
        // decided from x^2 + y^2 + z^2 alone (most of a grid); the margins of 1e-12 leave every close call to the full test,
        // so the rendering is voxel for voxel what the full test gives.
        const double yz2 = y * y + z * z;
        if (tilemap) {
            if ((r & 3) == 0) {                          // a new row of tiles (iy0 is a multiple of 8)
                tyz2 = nearest_sq(iy, ny, (float)dy, 4) + tz2;
                rows_out = tyz2 > r2o;                   // every tile of these rows lies outside the sphere (most rows of most grids)
                if ((iz & 3) == 0) {                     // the first row of its tiles writes their map bytes: lane = tile of the run
                    const int tx = (x0 >> 4) + lane;
                    if (tx < nbx && tx * 16 < x1)
                        tm[(size_t)(r >> 2) * nbx + tx] = !rows_out && !(nearest_sq(tx * 16, nx, fdx, 16) + tyz2 > r2o) ? 1 : 0;
                }
            }
            if (rows_out) continue;
        } else if (yz2 > r2_out) {
            for (int ix = x0 + lane; ix < x1; ix += 32) dst[ix] = vac;
            continue;
        }
#pragma unroll 1
        for (int ix = x0 + lane; ix < x1; ix += 32) {
            if (tilemap && nearest_sq(ix & ~15, nx, fdx, 16) + tyz2 > r2o) continue;      // the tile cannot hold material: not written
            const double x = ((double)ix - 0.5 * (double)(nx - 1)) * dx;
            const double r2 = x * x + yz2;
            bool inside;
            if (r2 > r2_out) inside = false;
            else if (r2 < r2_in) inside = true;
            else inside = render_inside(Bt, A, x, y, z);
            dst[ix] = inside ? mat : vac;
        }
    }
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

// Slots of the coefficient pool a harmonics shape takes: the dense tables of sh_radius_dense (degrees <= 8) or its triplets.
static int sh_dense_degree(const scatman_shape &s) {
    int lmax = 0;
    for (int i = 0; i < s.ncoef; ++i) {
        const double l = s.h_coef[3 * i];
        if (!(l >= 0.0 && l <= 32.0)) return 0;      // (rejected by fill_render_args)
        lmax = (int)l > lmax ? (int)l : lmax;
    }
    return lmax <= 4 ? 4 : lmax <= 6 ? 6 : lmax <= 8 ? 8 : 0;
}
static int sh_pool_need(const scatman_shape &s) {
    if (s.ncoef < 1 || s.ncoef > kMaxCoef || !s.h_coef) return -1;
    const int L = sh_dense_degree(s);
    return L ? 2 * sh_pairs(L) : s.ncoef;
}

// Fills descriptor A (and, for harmonics, coefficients at coef0 of the pool arrays).  0 ok, 1 bad argument.
static int fill_render_args(const scatman_shape &s, const scatman_grid &g, RenderArgs &A, double *Acn_pool, signed char *Al, signed char *Am) {
    double *Acn = Acn_pool;
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
            const int L = sh_dense_degree(s);
            double tcn[kMaxCoef];
            signed char tl[kMaxCoef], tm[kMaxCoef];
            if (L) { Acn = tcn; Al = tl; Am = tm; }   // the triplets are scattered into the dense tables below
            double *pool_cn = L ? Acn_pool : nullptr;
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
            if (L) {
                const int np = sh_pairs(L);
                for (int i = 0; i < 2 * np; ++i) pool_cn[i] = 0.0;
                for (int i = 0; i < s.ncoef; ++i) {
                    const int l = Al[i], m = Am[i], am = m < 0 ? -m : m;
                    const int pi = am * (L + 1) - am * (am - 1) / 2 + (l - am);      // m-major enumeration of the pairs (l, m >= 0)
                    pool_cn[(m < 0 ? np : 0) + pi] += Acn[i];
                }
                A.dense_L = L;
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
                        int *nlaunch, unsigned char *d_tilemap) {
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
            const int nc = s.kind == SCATMAN_SHAPE_SPHERICAL_HARMONICS ? sh_pool_need(s) : 0;
            if (nc < 0) return 1 + b;
            if (pool + nc > kPoolCoef) break;
            if (fill_render_args(s, g, Bt.a[Bt.n], Bt.cn + pool, Bt.l + pool, Bt.m + pool)) return 1 + b;
            Bt.a[Bt.n].coef0 = pool;
            pool += nc;
            ++Bt.n;
            ++b;
        }
        const size_t nruns = (size_t)((g.ny + kRenderRows - 1) / kRenderRows) * g.nz * ((g.nx + kRenderRun - 1) / kRenderRun);      // one warp each
        const size_t tiles = (size_t)((g.nz + 3) / 4) * ((g.ny + 3) / 4) * ((g.nx + 15) / 16);
        render_kernel<<<dim3((unsigned)((nruns + 7) / 8), (unsigned)Bt.n), 256, 0, st>>>(Bt, (float2 *)d_dn + (size_t)first * nvox,
                                                                                      d_tilemap ? d_tilemap + (size_t)first * tiles : nullptr);
        ++*nlaunch;
        *err = cudaGetLastError();
        if (*err != cudaSuccess) return 0;
    }
    return 0;
}

}  // namespace scatman
