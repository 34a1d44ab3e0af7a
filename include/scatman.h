/*
 * scatman.h -- C ABI of libscatman: B200-native (sm_100a) MSFT forward simulation.
 *
 * The method: "The Scatman", arXiv 2202.03411 (reference text: PAPER.md), Multi-Slice Fourier
 * Transform.  For every detector pixel p with Ewald-sphere momentum transfer q(p) (Eq. 3,
 * PAPER.md:80-83) the library evaluates directly
 *
 *     A(p) = sum_j e^{i qz z_j} sum_{x,y} rho~_j(x,y) e^{i (qx x + qy y)}        (Eq. 2/4)
 *     rho~_j = f(dn_j) exp(i k dz sum_{l<j} dn_l) dV,  dn = delta + i beta         (Eq. 6-9)
 *     I(p) = |A(p)|^2                                                             (Block 11)
 *
 * in the sign convention of BASELINE.json's north_star (the complex conjugate of the paper's;
 * same intensity, reading R3).
 *
 * Conventions common to every entry point
 *   - Pointers named d_* are DEVICE pointers (16-byte aligned), h_* are HOST pointers.
 *   - The caller owns every device buffer, including the workspace; the library allocates no
 *     device memory in the d_* entry points (only scatman_simulate*_host keep a device arena in the
 *     context).  Inputs are never modified.
 *   - All device work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  No host synchronisation happens unless stated.
 *   - Every function returns a scatman_status.  No exceptions, no abort, NO CPU FALLBACK: without a
 *     compute-capability 10.x device scatman_create fails with SCATMAN_UNSUPPORTED_DEVICE.
 *   - Device data are not validated (no NaN / range checks).
 *   - Lengths (voxel size, lambda) share one arbitrary unit; k = 2 pi / lambda.
 *   - Grid layout: dn[b][iz][iy][ix][2] = (delta, beta) FP32 in the paper's sense (n = 1 - delta + i beta,
 *     Eq. 7), ix fastest, z = beam axis, slice iz = 0 is hit first.  Voxel centres at
 *     x_i = (i - (nx-1)/2) dx etc. (R6).  One slice per z-layer, slice thickness dz (R8).
 *   - Output: I[b][iy][ix] FP32 (ix fastest), units length^6 (dV^2 scale, R1).
 */
#ifndef SCATMAN_H_
#define SCATMAN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct scatman_ctx scatman_ctx; /* opaque; one per device; not thread-safe */

typedef enum {
    SCATMAN_OK = 0,
    SCATMAN_INVALID_ARGUMENT = 1,   /* null pointer, non-positive dims, lambda <= 0, theta_max outside (0,90),
                                       batch < 1, |quat| not 1 within 1e-6, unknown enum value */
    SCATMAN_UNSUPPORTED_DEVICE = 2, /* no CUDA device, or compute capability != 10.x */
    SCATMAN_WORKSPACE_TOO_SMALL = 3,
    SCATMAN_CUDA_ERROR = 4,         /* message via scatman_last_error */
    SCATMAN_NOT_IMPLEMENTED = 5
} scatman_status;

/* Voxel grid: z = beam axis, x fastest. */
typedef struct {
    int32_t nx, ny, nz;
    double dx, dy, dz;
} scatman_grid;

/* Flat detector perpendicular to the beam at unit distance, npx x npy square pixels; the mid-points of
 * its outer edges in x sit at scattering angle theta_max (R9).  (cx, cy) shifts the detector centre off
 * the axis, in pixels.  Pixel (ix, iy) has u = (ix + 1/2 - npx/2 + cx) pitch, v likewise with npy, cy;
 * pitch = 2 tan(theta_max) / npx. */
typedef struct {
    int32_t npx, npy;
    double theta_max_deg;
    double cx, cy;
} scatman_detector;

enum { SCATMAN_RHO_LINEAR = 0, /* f(c) = c        : north_star's contrast dn = delta + i beta   */
       SCATMAN_RHO_N2M1 = 1 }; /* f(c) = c (2 - c): the paper's n^2 - 1 (Eq. 5/9), conjugated */

enum { SCATMAN_METHOD_AUTO = 0,        /* = TENSOR */
       SCATMAN_METHOD_TENSOR = 1,      /* tcgen05 split-precision contraction + fused epilogue */
       SCATMAN_METHOD_SIMT_SINCOS = 2, /* CUDA-core variant: one sincos of the full phase per term */
       SCATMAN_METHOD_SIMT_TABLE = 3 };/* CUDA-core variant: FP32 FMA GEMM per slice against per-pixel phase tables */

enum { SCATMAN_PRECISION_AUTO = 0,     /* = FP16X3 */
       SCATMAN_PRECISION_FP16X3 = 1 }; /* A = Ah + Al, B = Bh + Bl in FP16; AhBh + AlBh + AhBl, FP32 accumulate */

typedef struct {
    int32_t rho_mode;
    int32_t method;
    int32_t precision;
    uint32_t flags; /* SCATMAN_FLAG_* bits; unknown bits are an error */
} scatman_options;

/* Tensor path only: run the contraction with one CTA per work item (tcgen05 cta_group::1, UMMA 128x128) instead of
 * the default CTA pairs (cta_group::2, UMMA 256x128, each CTA holding half of every B tile).  Same results up to
 * summation order; kept for comparison and as the smaller-cluster variant. */
#define SCATMAN_FLAG_SINGLE_CTA 1u
/* Tensor path only: also count the work the contraction really issues (one extra small kernel), for
 * scatman_last_issued_blocks.  The contraction skips 16-y steps of a (slice, 128-x tile, 128-y group) unit whose
 * rho~ values are all zero and narrows every unit to the range of its non-empty 16-x blocks. */
#define SCATMAN_FLAG_COUNT_ISSUED 2u
/* Every scatman_simulate* entry point: reuse the phase tables of the previous call.  The q-map (a1) and the phase tables (a3;
 * the window-corrected tables of the NUFFT route, the Ex / Ey tables of the separable route) depend only on the grid geometry,
 * lambda and the detector ("once per detector / lambda"); they sit at the start of the workspace, at offsets that do not depend
 * on the batch.  With this flag the caller PROMISES that the workspace (same pointer) has not been written since the previous
 * scatman_simulate* call on this context, and that explicit q arrays (d_q, d_qx, d_qy: same pointers) still hold the same
 * values.  The library checks that grid, voxel size, lambda, detector / q pointers, method and workspace pointer equal those of
 * the previous call and rebuilds the tables whenever anything differs, so the flag never changes a result: outputs are
 * bit-identical with and without it.  It saves the table kernels (cfg3, pixel route: 0.54 GB of tables per call). */
#define SCATMAN_FLAG_REUSE_TABLES 4u

/* Create / destroy a context on CUDA device `device`.  Fails with SCATMAN_UNSUPPORTED_DEVICE unless the
 * device is compute capability 10.x.  scatman_destroy(NULL) is SCATMAN_OK. */
int scatman_create(scatman_ctx **out, int device);
int scatman_destroy(scatman_ctx *ctx);

/* Bytes of workspace scatman_simulate / scatman_simulate_q need for this problem (any orientation).
 * npix = npx*npy for scatman_simulate.  opts may be NULL (all AUTO). */
int scatman_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int64_t npix, int32_t batch,
                            const scatman_options *opts, size_t *bytes);

/* Step a1, q-map (Eq. 3; north_star (1)): detector pixels -> Ewald-sphere
 * q = k (s_pixel - z^), FP64, d_q[p][3] with p = iy*npx + ix; qz = -k (u^2+v^2) / (r (r+1)) (R10). */
int scatman_qmap(scatman_ctx *ctx, const scatman_detector *det, double lambda, double *d_q, void *cuda_stream);

/* Step a0, orientation (Block 5; Fig. 6; R11): beam-frame grid = trilinear
 * resample (FP64 coordinates, zero outside) of the body-frame grid at r_body = R^T r_beam, same dims.
 * h_quat[b][4] = (w,x,y,z) unit quaternion, body -> beam; read on the host before return.
 * d_dn_out must not alias d_dn_in.  d_ws: scatman_orient_workspace_bytes(batch) bytes (rotation matrices and the
 * bounding boxes of the non-vacuum voxels), 16-byte aligned, owned by the caller like every device buffer. */
int scatman_orient_workspace_bytes(scatman_ctx *ctx, int32_t batch, size_t *bytes);
int scatman_orient(scatman_ctx *ctx, const float *d_dn_in, const scatman_grid *grid, const double *h_quat,
                   int32_t batch, void *d_ws, size_t ws_bytes, float *d_dn_out, void *cuda_stream);

/* Step a2, column prefix (Eq. 6/8/9; north_star (2)): effective scattering strength
 * d_rho[b][iz][iy][ix][2] = f(dn_j) exp(i k dz sum_{l<j} dn_l) as FP32 (Re, Im), WITHOUT the dV factor.
 * The prefix runs in FP64. */
int scatman_effective_strength(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                               int32_t rho_mode, int32_t batch, float *d_rho, void *cuda_stream);

/* The whole hot path a0-a6 (north_star (1)-(5)): `batch` grids of identical dims -> `batch` intensity
 * patterns on the flat detector.  h_quat may be NULL (identity for every item: a0 skipped).
 * d_I[b][npy][npx] FP32.  d_ws/ws_bytes: workspace of at least scatman_workspace_bytes(). */
int scatman_simulate(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                     const scatman_detector *det, const double *h_quat, int32_t batch,
                     const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream);

/* Same path minus a1, at an explicit list of momentum transfers d_q[npix][3] (FP64, device):
 * for tests (q = 0, FFT-grid q's) and non-flat detectors.  d_I[b][npix]. */
int scatman_simulate_q(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                       const double *d_q, int64_t npix, const double *h_quat, int32_t batch,
                       const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream);

/* The separable route (the paper's own evaluation points: Block 6 of Fig. 4 transforms every slice on a
 * uniform (qx, qy) grid): the detector is a TENSOR GRID of transverse momentum transfers, pixel (a, b)
 * at (qx[a], qy[b], qz) with qz = -(k - sqrt(k^2 - qx^2 - qy^2)) on the Ewald sphere (Eq. 3-4, in
 * north_star's sign), so the slice transform factors into two small complex GEMMs per slice instead of the
 * (pixel x voxel) contraction -- npx-fold less arithmetic.  Same a0 / a2 steps, same conventions and output scale as
 * scatman_simulate; grid points with qx^2 + qy^2 > k^2 (no scattering direction) get I = 0.
 * d_qx[npx], d_qy[npy]: FP64 device arrays (any values, e.g. the DFT grid 2 pi m / (N dx)).  d_I[b][npy][npx].
 * opts: rho_mode; method AUTO / TENSOR = both GEMMs on tcgen05 tensor cores with the FP16x3 split (grids with nx > 1024
 * use the CUDA-core stages), SIMT_TABLE = FP32 CUDA-core GEMMs; SIMT_SINCOS is INVALID_ARGUMENT here; precision and
 * flags other than SCATMAN_FLAG_REUSE_TABLES are ignored.  The workspace size depends on the method: pass the same opts to both calls. */
int scatman_qgrid_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int32_t npx, int32_t npy, int32_t batch,
                                  const scatman_options *opts, size_t *bytes);
int scatman_simulate_qgrid(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                           const double *d_qx, int32_t npx, const double *d_qy, int32_t npy, const double *h_quat,
                           int32_t batch, const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I,
                           void *cuda_stream);

/* The flat detector by a 3-D type-2 non-uniform Fourier transform ("a type-2 NUFFT for the flat detector"):
 * the SAME result as scatman_simulate -- A(p) = sum_r rho~(r) e^{i q(p).r} at every pixel's Ewald-sphere q (Eq. 2-4,
 * PAPER.md:68-87), same a0 / a1 / a2 steps, conventions and output scale -- but rho~ is first transformed onto a small uniform
 * (gz, gy, gx) grid covering the detector's q range (three FP64 complex GEMMs: slices, columns, rows; spacing 2 pi / (2 N d),
 * Kaiser-Bessel pre-correction) and every pixel is then interpolated from its 10^3 nearest grid points.  The window's
 * aliasing error is < 1e-8 of sum |rho~| dV per pixel; all sums are FP64 (the uniform-grid values are stored FP32 for the
 * interpolation, a rounding relative to the local amplitude), so north_star's tolerances against the direct
 * sum hold (tests/test_gpu_nufft.py).  Work ~ N_vox * nqz + ... instead of N_vox * N_pix: ~1000x fewer multiply-adds.
 * opts: rho_mode and SCATMAN_FLAG_REUSE_TABLES (method, precision, other flags ignored).  d_I[b][npy][npx].  The workspace depends on lambda and the
 * detector (they fix the q range): scatman_nufft_workspace_bytes with the same arguments. */
int scatman_nufft_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, double lambda, const scatman_detector *det,
                                  int32_t batch, size_t *bytes);
/* nq[3] = points per axis (x, y, z) of the uniform grid the route transforms onto (for work counts). */
int scatman_nufft_grid_dims(scatman_ctx *ctx, const scatman_grid *grid, double lambda, const scatman_detector *det,
                            int32_t *nq);
int scatman_simulate_nufft(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                           const scatman_detector *det, const double *h_quat, int32_t batch, const scatman_options *opts,
                           void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream);

/* End to end with HOST buffers (bench.py's e2e leg), one entry point per route: h_dn[batch][nz][ny][nx][2] in, h_I out, both
 * in host memory (pinned for full copy bandwidth and for the overlap below; pageable memory works, serially).  The batch is cut
 * into chunks of ~256 MB of input; the upload of chunk c + 1, the kernels of chunk c and the download of chunk c - 1 run
 * concurrently on three streams of the context, so for a batch of several chunks the call costs max(copy, compute) per chunk
 * instead of their sum.  The phase tables are built once and reused by every chunk and by later calls with the same geometry.
 * These entry points alone own device memory: a grow-only arena kept in the context until scatman_destroy.  They return
 * after h_I is complete (synchronous).  h_quat[batch][4] or NULL; h_qx[npx], h_qy[npy] are host arrays.
 * scatman_last_launch_count then counts the kernels of all chunks. */
int scatman_simulate_host(scatman_ctx *ctx, const float *h_dn, const scatman_grid *grid, double lambda,
                          const scatman_detector *det, const double *h_quat, int32_t batch,
                          const scatman_options *opts, float *h_I);
int scatman_simulate_nufft_host(scatman_ctx *ctx, const float *h_dn, const scatman_grid *grid, double lambda,
                                const scatman_detector *det, const double *h_quat, int32_t batch,
                                const scatman_options *opts, float *h_I);
int scatman_simulate_qgrid_host(scatman_ctx *ctx, const float *h_dn, const scatman_grid *grid, double lambda,
                                const double *h_qx, int32_t npx, const double *h_qy, int32_t npy, const double *h_quat,
                                int32_t batch, const scatman_options *opts, float *h_I);

/* ---- Forward-fitting pieces (simulate, compare with the measured pattern, improve) -------
 * scatman_discrepancy: one number per simulated pattern instead of an image.  d_I[batch][npix] FP32 simulated patterns;
 * d_M measured pattern(s), FP32: m_stride = 0 -> one pattern d_M[npix] for every item, m_stride = npix -> d_M[batch][npix];
 * d_mask[npix] bytes (0 = pixel ignored: detector gaps, beam stop, angular window) or NULL = all pixels; d_out[batch] FP64.
 *   SCATMAN_LOSS_L2_NORMALISED     sum_p w (I / S_I - M / S_M)^2, S = sum_p w (.): each pattern divided by its integral over
 *                                  the masked region, the normalisation of the paper's Fig. 5 (reading R22)
 *   SCATMAN_LOSS_POISSON_DEVIANCE  2 sum_p w [M log(M / mu) - (M - mu)], mu = (S_M / S_I) I: deviance of measured counts
 *                                  against the scale-fitted simulation (M log M = 0 at M = 0; +inf where mu = 0 < M) (R24)
 * FP64 accumulation, deterministic.  d_ws: scatman_fit_workspace_bytes(npix, batch) bytes.  Asynchronous on cuda_stream. */
enum { SCATMAN_LOSS_L2_NORMALISED = 0, SCATMAN_LOSS_POISSON_DEVIANCE = 1 };
int scatman_fit_workspace_bytes(scatman_ctx *ctx, int64_t npix, int32_t batch, size_t *bytes);
int scatman_discrepancy(scatman_ctx *ctx, const float *d_I, const float *d_M, int64_t m_stride, const uint8_t *d_mask,
                        int64_t npix, int32_t batch, int32_t metric, void *d_ws, size_t ws_bytes, double *d_out,
                        void *cuda_stream);

/* scatman_discrepancy for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same kernels and the same result, bit for bit, with the scratch in a static device array of
 * SCATMAN_STATIC_SCRATCH_BYTES inside the library instead of a caller's workspace.  The call allocates nothing, on the host
 * side of CUDA or the device.  Limits and rules:
 *   - scatman_fit_workspace_bytes(npix, batch) must not exceed SCATMAN_STATIC_SCRATCH_BYTES (1 MiB: e.g. 256 patterns of up
 *     to 2.7 M pixels, or 4096 of 128 k); beyond that the call fails with SCATMAN_WORKSPACE_TOO_SMALL and a message naming both
 *     numbers, and nothing is launched.
 *   - every GPU that loads the library holds the array until the process exits; ALL calls on a device share it, from any
 *     context or stream.  It keeps the last call's contents (each call overwrites what it reads: nothing needs clearing), so
 *     two calls that overlap on the GPU (different streams, or graphs replayed concurrently) race: serialise them.
 *   - the array's device address is resolved per device in scatman_create (cudaGetSymbolAddress with that device current);
 *     if that failed, this call returns SCATMAN_CUDA_ERROR with the reason and every other entry point is unaffected.
 * Arguments as scatman_discrepancy, without d_ws / ws_bytes.  Asynchronous on cuda_stream. */
#define SCATMAN_STATIC_SCRATCH_BYTES (1u << 20)
int scatman_discrepancy_static(scatman_ctx *ctx, const float *d_I, const float *d_M, int64_t m_stride, const uint8_t *d_mask,
                               int64_t npix, int32_t batch, int32_t metric, double *d_out, void *cuda_stream);

/* The Ideal detector ("even a perfect real-life detector is subjected to Poisson statistics of photons";
 * the paper's photon estimate is in its unavailable supplement, so the caller states it, reading R23): d_counts[b][p] =
 * Poisson(h_photons[b] * I[b][p] / sum_p I[b][p]) as FP32 integers, h_photons[batch] = expected detected photons per pattern
 * (host, read before return).  Draws come from Philox-4x32-10 with counter (p low word, p high word, b, draw) and key = seed:
 * a pixel's count depends only on (its mean, p, b, seed).  Means below 10 use inversion on one uniform, larger ones
 * Hoermann's transformed rejection (PTRS).  An all-zero pattern gives all-zero counts.  Same workspace as above. */
int scatman_ideal_detector(scatman_ctx *ctx, const float *d_I, int64_t npix, int32_t batch, const double *h_photons,
                           uint64_t seed, void *d_ws, size_t ws_bytes, float *d_counts, void *cuda_stream);

/* Number of kernels the last scatman_simulate* call on this context launched (for bench accounting). */
int scatman_last_launch_count(scatman_ctx *ctx, int32_t *count);

/* Device time of the contraction kernel (step a4+a5) of the last scatman_simulate* call, measured with
 * CUDA events on the call's stream.  Synchronises on the end event.  -1 if none was recorded. */
int scatman_last_contraction_ms(scatman_ctx *ctx, float *ms);

/* ---- Shape rendering (Block 5 of Fig. 4, "render the slice at the proper spatial coordinates"; shape
 * models of PAPER.md:245-259, 405-425; readings R18-R21 of DESIGN.md) ----------------------------------------------
 * A shape is rendered directly in the beam frame: voxel centre r_beam goes to r_body = R^T r_beam (R from `quat`,
 * body -> beam, as in scatman_orient) and the voxel becomes (delta, beta) if r_body is inside the shape, else (0, 0):
 * binary voxelisation at voxel centres, evaluated in FP64.  The rendered grid is already oriented, so it is passed to
 * scatman_simulate with h_quat = NULL.
 *   ELLIPSOID            (x/a)^2 + (y/b)^2 + (z/c)^2 <= 1, semi-axes a, b, c along body x, y, z.
 *   SPHERICAL_HARMONICS  |r| <= R(theta, phi) = sum over the triplets (l, m, c) of c * Y_lm, theta =
 *                        polar angle from body +z, phi = atan2(y, x); Y_lm = REAL orthonormal harmonics with Eq. 10's
 *                        normalisation and Condon-Shortley phase: m = 0: Y_l^0; m > 0: sqrt2 Re Y_l^m; m < 0:
 *                        sqrt2 Im Y_l^|m|.  A sphere of radius r is the single triplet (0, 0, r sqrt(4 pi)).
 *                        h_coef[ncoef][3] = (l, m, c) as doubles on the HOST, ncoef <= 96, l <= 32.
 *   RADIAL_MAP           |r| <= R(lat, lon), bilinear in d_radii[nlat][nlon] (FP64, DEVICE): sample (i, j) sits at
 *                        latitude -pi/2 + i pi/nlat and longitude j 2pi/nlon (the paper's 4 x 4 example),
 *                        periodic in longitude, latitudes above the last sample hold the last row;
 *                        lat = asin(z/|r|), lon = atan2(y, x) mod 2pi.
 *   VOLUME_MAP           d_volume[nvz][nvy][nvx] bytes (DEVICE, non-zero = inside): cubic cells of side vdx centred on
 *                        the origin; inside if the cell containing r_body is set.
 * Fields of other kinds are ignored. */
enum { SCATMAN_SHAPE_ELLIPSOID = 0, SCATMAN_SHAPE_SPHERICAL_HARMONICS = 1, SCATMAN_SHAPE_RADIAL_MAP = 2,
       SCATMAN_SHAPE_VOLUME_MAP = 3 };

typedef struct {
    int32_t kind;
    float delta, beta;       /* n = 1 - delta + i beta inside the shape (Eq. 7) */
    double quat[4];          /* (w, x, y, z) unit quaternion, body -> beam; {1, 0, 0, 0} = identity */
    double a, b, c;          /* ELLIPSOID */
    int32_t ncoef;           /* SPHERICAL_HARMONICS */
    const double *h_coef;
    int32_t nlat, nlon;      /* RADIAL_MAP */
    const double *d_radii;
    int32_t nvx, nvy, nvz;   /* VOLUME_MAP */
    const uint8_t *d_volume;
    double vdx;
} scatman_shape;

/* Render `batch` shapes (host array of descriptors, read before return) into d_dn[batch][nz][ny][nx][2] (device,
 * FP32 (delta, beta)), asynchronously on cuda_stream; one kernel launch per shape. */
int scatman_render(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid,
                   float *d_dn, void *cuda_stream);

/* Shapes in, patterns out (north_star (5), forward fitting: the candidates of an optimiser step are shape parameters, not
 * voxel grids): scatman_render into the workspace, then the whole path a1-a6 on the rendered (already oriented) grids.
 * Only the descriptors cross the host-device boundary.  d_I[batch][npy][npx].  Workspace: scatman_shapes_workspace_bytes. */
int scatman_shapes_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int64_t npix, int32_t batch,
                                   const scatman_options *opts, size_t *bytes);
int scatman_simulate_shapes(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid,
                            double lambda, const scatman_detector *det, const scatman_options *opts, void *d_ws,
                            size_t ws_bytes, float *d_I, void *cuda_stream);

/* The same from shape descriptors on the separable route: scatman_render followed by scatman_simulate_qgrid (shapes are
 * rendered in the beam frame, so a0 is skipped), for forward fitting against a detector that is a tensor grid of (qx, qy).
 * d_I[batch][npy][npx].  Workspace: scatman_shapes_qgrid_workspace_bytes with the same opts. */
int scatman_shapes_qgrid_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int32_t npx, int32_t npy, int32_t batch,
                                         const scatman_options *opts, size_t *bytes);
int scatman_simulate_shapes_qgrid(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid,
                                  double lambda, const double *d_qx, int32_t npx, const double *d_qy, int32_t npy,
                                  const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream);

/* The same from shape descriptors on the NUFFT route for the flat detector: scatman_render followed by scatman_simulate_nufft
 * (shapes are rendered in the beam frame, so a0 is skipped).  d_I[batch][npy][npx].  opts: rho_mode only. */
int scatman_shapes_nufft_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, double lambda, const scatman_detector *det,
                                         int32_t batch, size_t *bytes);
int scatman_simulate_shapes_nufft(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid,
                                  double lambda, const scatman_detector *det, const scatman_options *opts, void *d_ws,
                                  size_t ws_bytes, float *d_I, void *cuda_stream);

/* With SCATMAN_FLAG_COUNT_ISSUED: the number of 16-y x 16-x blocks of rho~ (256 voxels each) the contraction of the last
 * scatman_simulate* call multiplied against EVERY pixel, summed over slices and batch items; the dense count is
 * batch * nz * ceil(ny/16) * ceil(nx/16) blocks of the padded grid.  Issued tensor flop = blocks * 256 * npix_pad * 24.
 * Synchronises with the call's stream.  -1 if the last call did not count. */
int scatman_last_issued_blocks(scatman_ctx *ctx, int64_t *blocks);

const char *scatman_status_string(int status);
const char *scatman_last_error(scatman_ctx *ctx); /* never NULL; "" if none */
int scatman_version(void);                        /* major*10000 + minor*100 + patch */

#ifdef __cplusplus
}
#endif
#endif /* SCATMAN_H_ */
