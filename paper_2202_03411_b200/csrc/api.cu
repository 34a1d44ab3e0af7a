// api.cu -- the C ABI of libscatman (include/scatman.h): argument validation, workspace planning and the
// enqueue order of the hot path.  Host logic only; every step of the path runs in the kernels.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>

#include "internal.h"

using namespace scatman;

// What a set of phase tables was built for.  Tables live in the CALLER's workspace, ahead of everything that depends on the
// batch, so the key holds the workspace pointer and no batch size.
struct TableKey {
    int route = 0;                       // 1 pixel contraction, 2 separable q-grid, 3 NUFFT
    int32_t nx = 0, ny = 0, nz = 0;
    double dx = 0, dy = 0, dz = 0, lambda = 0;
    int32_t npx = 0, npy = 0;
    double theta = 0, cx = 0, cy = 0;
    int64_t npix = 0;
    int method = 0, ncta = 0;
    const void *q0 = nullptr, *q1 = nullptr;   // explicit q arrays (scatman_simulate_q, scatman_simulate_qgrid)
    const void *ws = nullptr;
    bool operator==(const TableKey &o) const {
        return route == o.route && nx == o.nx && ny == o.ny && nz == o.nz && dx == o.dx && dy == o.dy && dz == o.dz &&
               lambda == o.lambda && npx == o.npx && npy == o.npy && theta == o.theta && cx == o.cx && cy == o.cy &&
               npix == o.npix && method == o.method && ncta == o.ncta && q0 == o.q0 && q1 == o.q1 && ws == o.ws;
    }
};

struct scatman_ctx {
    int device = 0;
    int num_sms = 0;
    std::string last_error;
    int last_launches = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool ev_valid = false, ev_capturing = false;
    const unsigned long long *d_count = nullptr;   // issued-block counter of the last call (in its workspace)
    cudaStream_t count_stream = nullptr;
    // Phase tables of the last call (a1 q-map + a3 tables: functions of the detector, lambda and the grid geometry only,
    // "cacheable" in SURVEY section 3): what they were built for and where.  SCATMAN_FLAG_REUSE_TABLES skips rebuilding them.
    TableKey tables_key;
    bool tables_valid = false;
    // scatman_simulate*_host: device arena (grow-only) and the three streams / events of the copy-compute pipeline
    cudaStream_t host_stream = nullptr, in_stream = nullptr, out_stream = nullptr;
    cudaEvent_t in_ready[2] = {nullptr, nullptr}, in_free[2] = {nullptr, nullptr}, out_free[2] = {nullptr, nullptr};
    void *arena = nullptr;
    size_t arena_bytes = 0;
    std::vector<double> host_q;   // qx | qy of the last scatman_simulate_qgrid_host (its tables are valid for these values only)
    // scatman_discrepancy_static: this device's address of the library's static scratch array (null + the error if it could not
    // be resolved at set-up; only that entry point minds)
    double *fit_static = nullptr;
    cudaError_t fit_static_err = cudaSuccess;
};

namespace scatman {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Batch chunks x z splits of the tensor kernel: minimise waves * per-item length (in slices), where an
// item costs its slices plus ~2 slice-equivalents of fill (A load, pipeline ramp).
void tensor_schedule(const Plan &p, int num_sms, int *nchunks, int *nzs) {  // num_sms = concurrent workers (CTAs or CTA pairs)
    double best = 1e300;
    int bc = 1, bz = 1;
    const int max_z = p.nz < 16 ? p.nz : 16;
    const int max_c = p.batch < 64 ? p.batch : 64;
    for (int c = 1; c <= max_c; ++c) {
        const int bpc = (p.batch + c - 1) / c;
        const int cc = (p.batch + bpc - 1) / bpc;
        for (int z = 1; z <= max_z; ++z) {
            const long long items = (long long)cc * z * p.ngroups * (p.ntiles / p.t_ncta);
            const long long waves = (items + num_sms - 1) / num_sms;
            const double len = (double)bpc * (double)((p.nz + z - 1) / z) + 2.0;
            const double cost = (double)waves * len;
            if (cost < best * (1.0 - 1e-9)) { best = cost; bc = cc; bz = z; }
        }
    }
    *nchunks = bc;
    *nzs = bz;
}

static Plan make_plan(const scatman_grid &g, double lambda, int64_t npix, int batch, const scatman_options &o,
                      int num_sms) {
    Plan p;
    p.nx = g.nx; p.ny = g.ny; p.nz = g.nz; p.dx = g.dx; p.dy = g.dy; p.dz = g.dz; p.lambda = lambda;
    p.npix = npix; p.batch = batch; p.rho_mode = o.rho_mode;
    p.method = o.method == SCATMAN_METHOD_AUTO ? SCATMAN_METHOD_TENSOR : o.method;
    p.nvox = (int64_t)g.nx * g.ny * g.nz;
    p.nx_pad = (int)align_up(g.nx, kTileX);
    p.ny_pad = (int)align_up(g.ny, kBlockY);
    p.nyb = p.ny_pad / kBlockY;
    p.ngroups = (p.nyb + kGroupYB - 1) / kGroupYB;
    p.nxt = p.nx_pad / kTileX;
    p.nxa = p.nx_pad / kFine;
    p.ntiles = (int)((npix + kTileP - 1) / kTileP);
    p.t_ncta = (o.flags & SCATMAN_FLAG_SINGLE_CTA) ? 1 : 2;
    if (p.method == SCATMAN_METHOD_TENSOR && p.t_ncta == 2) p.ntiles = (p.ntiles + 1) / 2 * 2;  // whole CTA pairs
    p.npix_pad = (int64_t)p.ntiles * kTileP;
    if (p.method == SCATMAN_METHOD_TENSOR) {
        tensor_schedule(p, num_sms / p.t_ncta, &p.t_nchunks, &p.t_nzs);
        p.nsplit = p.ngroups * p.t_nzs;
    } else {
        p.nsplit = simt_zsplit(p, num_sms);
    }
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o2 = off; off = align_up(off + bytes, 1024); return o2; };
    // the phase tables first: their offsets and sizes do not depend on the batch (SCATMAN_FLAG_REUSE_TABLES)
    p.off_q = take(sizeof(double) * 3 * (size_t)npix);
    if (p.method == SCATMAN_METHOD_TENSOR) {
        p.off_A = take(sizeof(__half) * 4 * (size_t)p.npix_pad * p.ny_pad);
        p.off_anchor = take(sizeof(float2) * (size_t)p.ntiles * p.nxa * kTileP);
        p.off_fine = take(sizeof(float2) * (size_t)p.ntiles * kFine * kTileP);
        p.off_zturn = take(sizeof(unsigned long long) * (size_t)p.ntiles * kTileP);
    }
    p.off_rotmat = take(sizeof(double) * 9 * (size_t)batch);
    p.off_bbox = take(orient_scratch_bytes(p, batch));
    p.off_rot = take(sizeof(float) * 2 * (size_t)p.nvox * batch);
    p.off_rho = take(sizeof(float) * 2 * (size_t)p.nvox * batch);
    p.off_max = take(sizeof(unsigned) * (size_t)batch);
    p.off_ampscale = take(sizeof(float) * (size_t)batch);
    p.off_partial = take(sizeof(float2) * (size_t)batch * p.nsplit * (size_t)p.npix_pad);
    if (p.method == SCATMAN_METHOD_TENSOR) {
        p.off_B = take(sizeof(__half) * 4 * (size_t)p.nx_pad * p.ny_pad * (size_t)p.nz * batch);
        p.off_mask = take(sizeof(unsigned long long) * (size_t)batch * p.nz * p.nxt * p.ngroups);
        p.off_count = take(sizeof(unsigned long long));
    }
    if (p.method == SCATMAN_METHOD_SIMT_TABLE) {
        p.off_tab_y = take(sizeof(float2) * (size_t)npix * g.ny);
        p.off_tab_x = take(sizeof(float2) * (size_t)npix * g.nx);
        p.off_tab_z = take(sizeof(float2) * (size_t)npix * g.nz);
        p.off_flags = take((size_t)batch * g.nz * ((g.ny + 15) / 16));
    }
    p.total = off;
    return p;
}

}  // namespace scatman

// The contraction's CUDA events are skipped while the stream is being captured into a graph (an event recorded in a capture
// cannot be synchronised on or timed afterwards): scatman_last_contraction_ms then reports -1.
static bool stream_capturing(cudaStream_t st) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); return false; }
    return cs != cudaStreamCaptureStatusNone;
}
static void ev_begin(scatman_ctx *ctx, cudaStream_t st) {
    ctx->ev_capturing = stream_capturing(st);
    if (!ctx->ev_capturing) cudaEventRecord(ctx->ev0, st);
}
static void ev_end(scatman_ctx *ctx, cudaStream_t st) {
    if (!ctx->ev_capturing) { cudaEventRecord(ctx->ev1, st); ctx->ev_valid = true; }
}

// Checked build only (SCATMAN_CHECKED=1): wait for the stream after a stage and name the stage that failed.
#ifdef SCATMAN_CHECKED
#define SCATMAN_STAGE_CHECK(e, st, what)                                                             \
    do {                                                                                             \
        if ((e) == cudaSuccess) (e) = cudaStreamSynchronize(st);                                     \
        if ((e) != cudaSuccess) fprintf(stderr, "scatman checked build: stage '%s' failed: %s\n", what, cudaGetErrorString(e)); \
    } while (0)
#else
#define SCATMAN_STAGE_CHECK(e, st, what) ((void)0)
#endif

static int fail(scatman_ctx *ctx, int status, const std::string &msg) {
    if (ctx) ctx->last_error = msg;
    return status;
}
static int cuda_fail(scatman_ctx *ctx, cudaError_t e, const char *where) {
    return fail(ctx, SCATMAN_CUDA_ERROR, std::string(where) + ": " + cudaGetErrorString(e));
}

static bool valid_grid(const scatman_grid *g) {
    return g && g->nx > 0 && g->ny > 0 && g->nz > 0 && g->dx > 0 && g->dy > 0 && g->dz > 0 && std::isfinite(g->dx) &&
           std::isfinite(g->dy) && std::isfinite(g->dz) && g->nx <= 8192 && g->ny <= 8192 && g->nz <= 65535;
}
static bool valid_detector(const scatman_detector *d) {
    return d && d->npx > 0 && d->npy > 0 && d->theta_max_deg > 0.0 && d->theta_max_deg < 90.0 && std::isfinite(d->cx) &&
           std::isfinite(d->cy);
}
static bool valid_options(const scatman_options &o) {
    return (o.rho_mode == SCATMAN_RHO_LINEAR || o.rho_mode == SCATMAN_RHO_N2M1) && o.method >= 0 && o.method <= 3 &&
           o.precision >= 0 && o.precision <= 1 && (o.flags & ~(uint32_t)(SCATMAN_FLAG_SINGLE_CTA | SCATMAN_FLAG_COUNT_ISSUED | SCATMAN_FLAG_REUSE_TABLES)) == 0;
}
static bool valid_quats(const double *q, int batch) {
    for (int b = 0; b < batch; ++b) {
        double n2 = 0;
        for (int i = 0; i < 4; ++i) n2 += q[4 * b + i] * q[4 * b + i];
        if (!(std::fabs(n2 - 1.0) <= 2e-6)) return false;
    }
    return true;
}
// One thread per (x, y) column walks z in the fused prefix -> planes kernel (launch_sep_tc_prefix_prep): it beats strength + pack
// once a chunk's columns fill the SMs (measured: one item of 256^2 columns loses 22 us, one of 128^2 37 us; a chunk of 8 x 128^2 or
// more gains 8 %).
static bool fused_prefix_pays(const Plan &p, int chunk_items) { return (size_t)chunk_items * p.nx * p.ny >= (size_t)4 << 16; }

static bool all_identity(const double *q, int batch) {
    for (int b = 0; b < batch; ++b)
        if (std::fabs(q[4 * b]) != 1.0 || q[4 * b + 1] != 0.0 || q[4 * b + 2] != 0.0 || q[4 * b + 3] != 0.0) return false;
    return true;
}
static void quat_to_rotmat(const double *q, double *R) {
    const double w = q[0], a = q[1], b = q[2], c = q[3];
    R[0] = 1 - 2 * (b * b + c * c); R[1] = 2 * (a * b - w * c);     R[2] = 2 * (a * c + w * b);
    R[3] = 2 * (a * b + w * c);     R[4] = 1 - 2 * (a * a + c * c); R[5] = 2 * (b * c - w * a);
    R[6] = 2 * (a * c - w * b);     R[7] = 2 * (b * c + w * a);     R[8] = 1 - 2 * (a * a + b * b);
}

// Rotation matrices reach the device as kernel arguments (no host buffer outlives the call).
struct RotChunk {
    double r[32 * 9];
};
__global__ void store_rotmat_kernel(RotChunk c, int n, double *__restrict__ dst) {
    const int i = threadIdx.x;
    if (i < n * 9) dst[i] = c.r[i];
}
static cudaError_t upload_rotmats(const double *h_quat, int batch, double *d_rotmat, cudaStream_t st, int *nlaunch) {
    for (int b0 = 0; b0 < batch; b0 += 32) {
        RotChunk c;
        const int n = batch - b0 < 32 ? batch - b0 : 32;
        for (int i = 0; i < n; ++i) quat_to_rotmat(h_quat + 4 * (b0 + i), c.r + 9 * i);
        store_rotmat_kernel<<<1, 288, 0, st>>>(c, n, d_rotmat + 9 * b0);
        if (nlaunch) ++*nlaunch;
    }
    return cudaGetLastError();
}

// Extremes of grids the host already knows (rendered shapes: one (delta, beta) per item) reach the device as kernel arguments.
struct StatsChunk {
    unsigned v[3 * 256];
};
__global__ void store_stats_kernel(StatsChunk c, int n, unsigned *__restrict__ dst) {
    for (int i = threadIdx.x; i < 3 * n; i += blockDim.x) dst[i] = c.v[i];
}
static cudaError_t upload_stats(const float *h_stats, int batch, unsigned *d_stats, cudaStream_t st, int *nlaunch) {
    for (int b0 = 0; b0 < batch; b0 += 256) {
        StatsChunk c;
        const int n = batch - b0 < 256 ? batch - b0 : 256;
        for (int i = 0; i < 3 * n; ++i) std::memcpy(&c.v[i], &h_stats[3 * b0 + i], sizeof(unsigned));
        store_stats_kernel<<<1, 256, 0, st>>>(c, n, d_stats + 3 * b0);
        if (nlaunch) ++*nlaunch;
    }
    return cudaGetLastError();
}
static void shape_stats(const scatman_shape *h_shapes, int batch, std::vector<float> &stats) {
    stats.resize(3 * (size_t)batch);
    for (int b = 0; b < batch; ++b) {
        stats[3 * b] = std::fabs(h_shapes[b].delta);
        stats[3 * b + 1] = std::fabs(h_shapes[b].beta);
        stats[3 * b + 2] = h_shapes[b].beta < 0.f ? -h_shapes[b].beta : 0.f;
    }
}

extern "C" {

int scatman_version(void) { return 200; }

const char *scatman_status_string(int status) {
    switch (status) {
        case SCATMAN_OK: return "ok";
        case SCATMAN_INVALID_ARGUMENT: return "invalid argument";
        case SCATMAN_UNSUPPORTED_DEVICE: return "unsupported device (needs compute capability 10.x)";
        case SCATMAN_WORKSPACE_TOO_SMALL: return "workspace too small";
        case SCATMAN_CUDA_ERROR: return "CUDA error";
        case SCATMAN_NOT_IMPLEMENTED: return "not implemented";
        default: return "unknown status";
    }
}

const char *scatman_last_error(scatman_ctx *ctx) { return ctx ? ctx->last_error.c_str() : ""; }

int scatman_create(scatman_ctx **out, int device) {
    if (!out) return SCATMAN_INVALID_ARGUMENT;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count <= 0) {
        cudaGetLastError();
        return SCATMAN_UNSUPPORTED_DEVICE;
    }
    if (device < 0 || device >= count) return SCATMAN_INVALID_ARGUMENT;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return SCATMAN_CUDA_ERROR;
    if (prop.major != 10) return SCATMAN_UNSUPPORTED_DEVICE;
    if (cudaSetDevice(device) != cudaSuccess) return SCATMAN_CUDA_ERROR;
    scatman_ctx *ctx = new scatman_ctx();
    ctx->device = device;
    ctx->num_sms = prop.multiProcessorCount;
    if (cudaEventCreate(&ctx->ev0) != cudaSuccess || cudaEventCreate(&ctx->ev1) != cudaSuccess ||
        nufft_init_device() != cudaSuccess ||   // the NUFFT route's window polynomials -> constant memory of this device
        tensor_init_device() != cudaSuccess || sep_init_device() != cudaSuccess || sep_tc_init_device() != cudaSuccess ||
        nufft_tc_init_device() != cudaSuccess || render_init_device() != cudaSuccess) {
        delete ctx;
        return SCATMAN_CUDA_ERROR;
    }
    ctx->fit_static_err = fit_static_scratch(device, &ctx->fit_static);   // `device` is current
    if (ctx->fit_static_err != cudaSuccess) cudaGetLastError();
    *out = ctx;
    return SCATMAN_OK;
}

int scatman_destroy(scatman_ctx *ctx) {
    if (!ctx) return SCATMAN_OK;
    cudaSetDevice(ctx->device);
    if (ctx->arena) cudaFree(ctx->arena);
    if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
    if (ctx->in_stream) cudaStreamDestroy(ctx->in_stream);
    if (ctx->out_stream) cudaStreamDestroy(ctx->out_stream);
    for (int i = 0; i < 2; ++i) {
        if (ctx->in_ready[i]) cudaEventDestroy(ctx->in_ready[i]);
        if (ctx->in_free[i]) cudaEventDestroy(ctx->in_free[i]);
        if (ctx->out_free[i]) cudaEventDestroy(ctx->out_free[i]);
    }
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    delete ctx;
    return SCATMAN_OK;
}

int scatman_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int64_t npix, int32_t batch,
                            const scatman_options *opts, size_t *bytes) {
    if (!ctx || !bytes) return SCATMAN_INVALID_ARGUMENT;
    scatman_options o = opts ? *opts : scatman_options{0, 0, 0, 0};
    if (!valid_grid(grid) || npix < 1 || batch < 1 || !valid_options(o)) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    *bytes = make_plan(*grid, 1.0, npix, batch, o, ctx->num_sms).total;
    return SCATMAN_OK;
}

int scatman_qmap(scatman_ctx *ctx, const scatman_detector *det, double lambda, double *d_q, void *cuda_stream) {
    if (!ctx || !d_q || !valid_detector(det) || !(lambda > 0.0) || !std::isfinite(lambda))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    cudaSetDevice(ctx->device);
    cudaError_t e = launch_qmap(*det, lambda, d_q, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "qmap");
}

int scatman_orient_workspace_bytes(scatman_ctx *ctx, int32_t batch, size_t *bytes) {
    if (!ctx || !bytes) return SCATMAN_INVALID_ARGUMENT;
    if (batch < 1) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    *bytes = scatman::align_up(sizeof(double) * 9 * (size_t)batch, 256) + sizeof(int) * 6 * (size_t)batch;   // matrices + boxes
    return SCATMAN_OK;
}

int scatman_orient(scatman_ctx *ctx, const float *d_dn_in, const scatman_grid *grid, const double *h_quat,
                   int32_t batch, void *d_ws, size_t ws_bytes, float *d_dn_out, void *cuda_stream) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!d_dn_in || !d_dn_out || !d_ws || d_dn_in == d_dn_out || !valid_grid(grid) || !h_quat || batch < 1 ||
        !valid_quats(h_quat, batch) || ((uintptr_t)d_ws & 15))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    size_t need = 0;
    scatman_orient_workspace_bytes(ctx, batch, &need);
    if (ws_bytes < need) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    cudaSetDevice(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *d_rot = (double *)d_ws;
    int *d_bbox = (int *)((uint8_t *)d_ws + scatman::align_up(sizeof(double) * 9 * (size_t)batch, 256));
    Plan p;
    p.nx = grid->nx; p.ny = grid->ny; p.nz = grid->nz; p.dx = grid->dx; p.dy = grid->dy; p.dz = grid->dz;
    cudaError_t e = upload_rotmats(h_quat, batch, d_rot, st, nullptr);
    if (e == cudaSuccess) e = launch_orient(d_dn_in, p, d_rot, batch, d_dn_out, d_bbox, st);
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "orient");
}

int scatman_render(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid, float *d_dn,
                   void *cuda_stream) {
    if (!ctx || !h_shapes || !d_dn || !valid_grid(grid) || batch < 1) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    cudaSetDevice(ctx->device);
    if ((size_t)((uint64_t)grid->nx * grid->ny * grid->nz + 255) / 256 > 0x7fffffffull || batch > 65535)
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "grid or batch too large for one render launch");
    cudaError_t e = cudaSuccess;
    int nl = 0;
    const int bad = launch_render_batch(h_shapes, batch, *grid, d_dn, (cudaStream_t)cuda_stream, &e, &nl);
    if (bad) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad shape descriptor " + std::to_string(bad - 1));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "render");
    ctx->last_launches = nl;
    return SCATMAN_OK;
}

int scatman_effective_strength(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                               int32_t rho_mode, int32_t batch, float *d_rho, void *cuda_stream) {
    if (!ctx || !d_dn || !d_rho || !valid_grid(grid) || !(lambda > 0.0) || !std::isfinite(lambda) || batch < 1 ||
        (rho_mode != SCATMAN_RHO_LINEAR && rho_mode != SCATMAN_RHO_N2M1))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    cudaSetDevice(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Plan p;
    p.nx = grid->nx; p.ny = grid->ny; p.nz = grid->nz; p.dx = grid->dx; p.dy = grid->dy; p.dz = grid->dz;
    p.lambda = lambda; p.rho_mode = rho_mode;
    cudaError_t e = launch_strength(d_dn, p, batch, d_rho, nullptr, st);   // no per-item maximum wanted: no scratch needed
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "effective_strength");
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ hot path
// Enqueue order: [a1 q-map] -> [a0 orient] -> a2 prefix -> operand pack + a3 tables
// -> a4/a5 contraction -> |A|^2.  Nothing here waits for the device.
static int run_path(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                    const scatman_detector *det, const double *d_q_in, int64_t npix, const double *h_quat, int batch,
                    const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I, cudaStream_t st) {
    scatman_options o = opts ? *opts : scatman_options{0, 0, 0, 0};
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!d_dn || !d_I || !d_ws || !valid_grid(grid) || !(lambda > 0.0) || !std::isfinite(lambda) || batch < 1 ||
        npix < 1 || batch > 65535 || !valid_options(o) || (!det && !d_q_in) || (det && !valid_detector(det)))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    if (h_quat && !valid_quats(h_quat, batch)) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "quaternion is not unit");
    if (((uintptr_t)d_dn | (uintptr_t)d_ws | (uintptr_t)d_I) & 15)
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "device pointers must be 16-byte aligned");
    cudaSetDevice(ctx->device);
    const Plan p = make_plan(*grid, lambda, npix, batch, o, ctx->num_sms);
    if (ws_bytes < p.total) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    uint8_t *ws = (uint8_t *)d_ws;
    int nl = 0;
    cudaError_t e = cudaSuccess;
    ctx->ev_valid = false;
    ctx->d_count = nullptr;

    TableKey key;
    key.route = 1;
    key.nx = grid->nx; key.ny = grid->ny; key.nz = grid->nz; key.dx = grid->dx; key.dy = grid->dy; key.dz = grid->dz;
    key.lambda = lambda; key.npix = npix; key.method = p.method; key.ncta = p.t_ncta; key.q0 = d_q_in; key.ws = d_ws;
    if (det) { key.npx = det->npx; key.npy = det->npy; key.theta = det->theta_max_deg; key.cx = det->cx; key.cy = det->cy; }
    const bool reuse = (o.flags & SCATMAN_FLAG_REUSE_TABLES) && ctx->tables_valid && ctx->tables_key == key;
    ctx->tables_valid = false;
    const double *d_q = d_q_in;
    if (!d_q) {
        double *q = (double *)(ws + p.off_q);
        if (!reuse) {
            e = launch_qmap(*det, lambda, q, st);
            ++nl;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "qmap");
        }
        d_q = q;
    }
    const float *src = d_dn;
    if (h_quat && !all_identity(h_quat, batch)) {
        double *rm = (double *)(ws + p.off_rotmat);
        e = upload_rotmats(h_quat, batch, rm, st, &nl);
        if (e == cudaSuccess)
            e = launch_orient(d_dn, p, rm, batch, (float *)(ws + p.off_rot), (int *)(ws + p.off_bbox), st, nullptr, nullptr,
                              orient_occ_ptr(ws + p.off_bbox, p, batch));
        nl += 3;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "orient");
        src = (const float *)(ws + p.off_rot);
    }
    float *rho = (float *)(ws + p.off_rho);
    unsigned *maxbits = (unsigned *)(ws + p.off_max);
    e = launch_strength(src, p, batch, rho, maxbits, st);
    ++nl;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "strength");
    float2 *partial = (float2 *)(ws + p.off_partial);
    const double dV = p.dx * p.dy * p.dz;

    if (p.method == SCATMAN_METHOD_TENSOR) {
        float *ampscale = (float *)(ws + p.off_ampscale);
        e = launch_pack_b(rho, p, maxbits, ampscale, (__half *)(ws + p.off_B), (unsigned long long *)(ws + p.off_mask), st);
        ++nl;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "pack_b");
        if (o.flags & SCATMAN_FLAG_COUNT_ISSUED) {
            e = launch_count_issued((const unsigned long long *)(ws + p.off_mask), p, (unsigned long long *)(ws + p.off_count), st);
            ++nl;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "count_issued");
            ctx->d_count = (const unsigned long long *)(ws + p.off_count);
            ctx->count_stream = st;
        }
        if (!reuse) {
            e = launch_tables(d_q, p, (__half *)(ws + p.off_A), (float2 *)(ws + p.off_anchor), (float2 *)(ws + p.off_fine),
                              (unsigned long long *)(ws + p.off_zturn), st, &nl);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "tables");
        }
        TensorLaunch t;
        t.d_A = ws + p.off_A; t.d_B = ws + p.off_B;
        t.d_anchor = (const float2 *)(ws + p.off_anchor); t.d_fine = (const float2 *)(ws + p.off_fine);
        t.d_zturn = (const unsigned long long *)(ws + p.off_zturn); t.d_partial = partial;
        t.d_mask = (const unsigned long long *)(ws + p.off_mask); t.num_sms = ctx->num_sms;
        std::string err;
        ev_begin(ctx, st);
        e = launch_tensor(p, t, st, &err);
        ++nl;
        if (e != cudaSuccess) return err.empty() ? cuda_fail(ctx, e, "contract") : fail(ctx, SCATMAN_CUDA_ERROR, err);
        ev_end(ctx, st);
        e = launch_finalize(partial, p, ampscale, dV, d_I, st);
    } else if (p.method == SCATMAN_METHOD_SIMT_TABLE) {
        ev_begin(ctx, st);
        e = launch_simt_table(rho, d_q, p, (float2 *)(ws + p.off_tab_y), (float2 *)(ws + p.off_tab_x), (float2 *)(ws + p.off_tab_z),
                              ws + p.off_flags, partial, st, &nl);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "simt_table");
        ev_end(ctx, st);
        e = launch_finalize(partial, p, nullptr, dV, d_I, st);
    } else {
        ev_begin(ctx, st);
        e = launch_simt_sincos(rho, d_q, p, partial, st);
        ++nl;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "simt_sincos");
        ev_end(ctx, st);
        e = launch_finalize(partial, p, nullptr, dV, d_I, st);
    }
    ++nl;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "finalize");
    ctx->last_launches = nl;
    ctx->tables_key = key;
    ctx->tables_valid = true;
    return SCATMAN_OK;
}

extern "C" {

int scatman_simulate(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                     const scatman_detector *det, const double *h_quat, int32_t batch, const scatman_options *opts,
                     void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream) {
    if (!det) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "detector is null");
    if (!valid_detector(det)) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad detector");
    return run_path(ctx, d_dn, grid, lambda, det, nullptr, (int64_t)det->npx * det->npy, h_quat, batch, opts, d_ws,
                    ws_bytes, d_I, (cudaStream_t)cuda_stream);
}

int scatman_simulate_q(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda, const double *d_q,
                       int64_t npix, const double *h_quat, int32_t batch, const scatman_options *opts, void *d_ws,
                       size_t ws_bytes, float *d_I, void *cuda_stream) {
    if (!d_q) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "d_q is null");
    return run_path(ctx, d_dn, grid, lambda, nullptr, d_q, npix, h_quat, batch, opts, d_ws, ws_bytes, d_I,
                    (cudaStream_t)cuda_stream);
}

int scatman_shapes_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int64_t npix, int32_t batch,
                                   const scatman_options *opts, size_t *bytes) {
    size_t inner = 0;
    const int rc = scatman_workspace_bytes(ctx, grid, npix, batch, opts, &inner);
    if (rc != SCATMAN_OK) return rc;
    *bytes = scatman::align_up(sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz * batch, 1024) + inner;
    return SCATMAN_OK;
}

int scatman_simulate_shapes(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid,
                            double lambda, const scatman_detector *det, const scatman_options *opts, void *d_ws,
                            size_t ws_bytes, float *d_I, void *cuda_stream) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!h_shapes || !d_ws || !valid_grid(grid) || batch < 1 || !det || !valid_detector(det))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    const size_t dn_bytes = scatman::align_up(sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz * batch, 1024);
    if (ws_bytes < dn_bytes) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    float *d_dn = (float *)d_ws;
    int rc = scatman_render(ctx, h_shapes, batch, grid, d_dn, cuda_stream);
    if (rc != SCATMAN_OK) return rc;
    const int rendered = ctx->last_launches;
    rc = run_path(ctx, d_dn, grid, lambda, det, nullptr, (int64_t)det->npx * det->npy, nullptr, batch, opts,
                  (uint8_t *)d_ws + dn_bytes, ws_bytes - dn_bytes, d_I, (cudaStream_t)cuda_stream);
    if (rc == SCATMAN_OK) ctx->last_launches += rendered;
    return rc;
}

// ---- separable route: workspace layout -------------------------------------------------------------------------
struct SepPlan {
    Plan p;
    SepTcPlan tc;
    bool tensor = true;   // both GEMM stages on tcgen05 (method AUTO / TENSOR) or FP32 CUDA cores (SIMT_TABLE)
    bool fused_ok = false;   // tensor stages: a chunk is large enough for the fused prefix -> planes pass (fused_prefix_pays)
    int nzs = 1;
    size_t off_rotmat = 0, off_bbox = 0, off_rot = 0, off_rho = 0, off_max = 0, off_ex = 0, off_ey = 0, off_h = 0, off_flags = 0,
           off_partial = 0, off_eyp = 0, off_exp = 0, off_rp = 0, off_hp = 0, off_scale = 0, off_bounds = 0, off_stats = 0, off_tilemap = 0, off_layers = 0, total = 0;
};
static SepPlan make_sep_plan(const scatman_grid &g, double lambda, int npx, int npy, int batch, int rho_mode, int method,
                             int num_sms) {
    SepPlan sp;
    Plan &p = sp.p;
    p.nx = g.nx; p.ny = g.ny; p.nz = g.nz; p.dx = g.dx; p.dy = g.dy; p.dz = g.dz; p.lambda = lambda;
    p.npix = (int64_t)npx * npy; p.batch = batch; p.rho_mode = rho_mode;
    p.nvox = (int64_t)g.nx * g.ny * g.nz;
    sp.tensor = method != SCATMAN_METHOD_SIMT_TABLE && g.nx <= 1024 && g.ny <= 2048;   // stage X keeps an Ex tile of >= 16 columns resident; stage YZ's slice masks hold 32 64-y blocks
    sp.nzs = sep_zsplit(p, npx, npy, num_sms);
    if (sp.tensor) sp.tc = make_sep_tc_plan(p, npx, npy, num_sms);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o2 = off; off = scatman::align_up(off + bytes, 1024); return o2; };
    // the phase tables first: their offsets and sizes do not depend on the batch (SCATMAN_FLAG_REUSE_TABLES)
    if (sp.tensor) {
        sp.off_eyp = take(sizeof(__half) * 4 * (size_t)sp.tc.NPYP * sp.tc.NY);
        sp.off_exp = take(sizeof(__half) * 4 * (size_t)sp.tc.NPXP * sp.tc.NXP);
    } else {
        sp.off_ex = take(sizeof(float2) * (size_t)g.nx * npx);
        sp.off_ey = take(sizeof(float2) * (size_t)g.ny * npy);
    }
    sp.off_rotmat = take(sizeof(double) * 9 * (size_t)batch);
    sp.off_bbox = take(orient_scratch_bytes(p, batch));
    sp.off_rot = take(sizeof(float) * 2 * (size_t)p.nvox * batch);
    // FP32 rho~: always for the CUDA-core stages; for the tensor stages only where chunks are too small for the fused pass (when they
    // are not, strength + pack runs only on un-oriented input and borrows the orientation's buffer)
    sp.fused_ok = sp.tensor && fused_prefix_pays(p, batch < sp.tc.nb ? batch : sp.tc.nb);
    sp.off_rho = sp.fused_ok ? sp.off_rot : take(sizeof(float) * 2 * (size_t)p.nvox * batch);
    sp.off_max = take(sizeof(unsigned) * (size_t)batch);
    sp.off_stats = take(sizeof(unsigned) * 3 * (size_t)batch);
    if (sp.fused_ok) {   // sparse orientation / render output (launch_orient)
        sp.off_tilemap = take(orient_tilemap_bytes(p, batch));
        sp.off_layers = take(tile_layers_bytes(p, batch));
    }
    if (sp.tensor) {
        const SepTcPlan &t = sp.tc;
        sp.off_rp = take(sizeof(__half) * 4 * (size_t)t.nb * g.nz * t.NY * t.NXP);
        sp.off_hp = take(sizeof(__half) * 4 * (size_t)t.nb * g.nz * t.NPXP * t.NY);
        sp.off_flags = take((size_t)t.nb * g.nz * (t.NY / 64));
        sp.off_scale = take(sizeof(float) * (size_t)batch);
        sp.off_bounds = take(sizeof(int) * (size_t)((t.nsx + 1) + (size_t)t.nb * t.ng * (t.nzs + 1)));
        sp.off_partial = take(sizeof(float2) * (size_t)t.nb * t.nsplit * npx * npy);
    } else {
        sp.off_h = take(sizeof(float2) * (size_t)g.nz * g.ny * npx);
        sp.off_flags = take((size_t)g.nz * ((g.ny + 15) / 16));
        sp.off_partial = take(sizeof(float2) * (size_t)sp.nzs * npx * npy);
    }
    sp.total = off;
    return sp;
}

static bool valid_qgrid_method(int m) {
    return m == SCATMAN_METHOD_AUTO || m == SCATMAN_METHOD_TENSOR || m == SCATMAN_METHOD_SIMT_TABLE;
}

int scatman_qgrid_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int32_t npx, int32_t npy, int32_t batch,
                                  const scatman_options *opts, size_t *bytes) {
    if (!ctx || !bytes) return SCATMAN_INVALID_ARGUMENT;
    const int method = opts ? opts->method : SCATMAN_METHOD_AUTO;
    if (!valid_grid(grid) || npx < 1 || npy < 1 || batch < 1 || !valid_qgrid_method(method))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    *bytes = make_sep_plan(*grid, 1.0, npx, npy, batch, 0, method, ctx->num_sms).total;
    return SCATMAN_OK;
}

}  // extern "C"

// Renders h_shapes into d_dn on `st`; sparse (tile map at d_tilemap) if that is non-null.  SCATMAN_OK or the failure, *nl += launches.
static int render_into(scatman_ctx *ctx, const scatman_shape *h_shapes, int batch, const scatman_grid &grid, float *d_dn,
                       unsigned char *d_tilemap, cudaStream_t st, int *nl) {
    if ((size_t)((uint64_t)grid.nx * grid.ny * grid.nz + 255) / 256 > 0x7fffffffull || batch > 65535)
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "grid or batch too large for one render launch");
    cudaError_t e = cudaSuccess;
    int n = 0;
    const int bad = launch_render_batch(h_shapes, batch, grid, d_dn, st, &e, &n, d_tilemap);
    if (bad) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad shape descriptor " + std::to_string(bad - 1));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "render");
    *nl += n;
    return SCATMAN_OK;
}

// h_stats: extremes of the grids when the host knows them (rendered shapes), else null (measured on the device).
// h_shapes: non-null -> the grids are rendered into d_dn first (scatman_simulate_shapes_qgrid), sparsely when the fused prefix pass reads them.
static int qgrid_impl(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda, const double *d_qx,
                      int32_t npx, const double *d_qy, int32_t npy, const double *h_quat, int32_t batch,
                      const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream, const float *h_stats,
                      const scatman_shape *h_shapes = nullptr) {
    scatman_options o = opts ? *opts : scatman_options{0, 0, 0, 0};
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!d_dn || !d_I || !d_ws || !d_qx || !d_qy || !valid_grid(grid) || !(lambda > 0.0) || !std::isfinite(lambda) ||
        batch < 1 || batch > 65535 || npx < 1 || npy < 1 || (o.rho_mode != SCATMAN_RHO_LINEAR && o.rho_mode != SCATMAN_RHO_N2M1) ||
        !valid_qgrid_method(o.method))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    if (h_quat && !valid_quats(h_quat, batch)) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "quaternion is not unit");
    if (((uintptr_t)d_dn | (uintptr_t)d_ws | (uintptr_t)d_I) & 15)
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "device pointers must be 16-byte aligned");
    cudaSetDevice(ctx->device);
    const SepPlan sp = make_sep_plan(*grid, lambda, npx, npy, batch, o.rho_mode, o.method, ctx->num_sms);
    const Plan &p = sp.p;
    if (ws_bytes < sp.total) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint8_t *ws = (uint8_t *)d_ws;
    int nl = 0;
    cudaError_t e = cudaSuccess;
    ctx->ev_valid = false;
    ctx->d_count = nullptr;
    TableKey key;
    key.route = 2;
    key.nx = grid->nx; key.ny = grid->ny; key.nz = grid->nz; key.dx = grid->dx; key.dy = grid->dy; key.dz = grid->dz;
    key.lambda = lambda; key.npx = npx; key.npy = npy; key.method = sp.tensor ? 1 : 3; key.q0 = d_qx; key.q1 = d_qy; key.ws = d_ws;
    const bool reuse = (o.flags & SCATMAN_FLAG_REUSE_TABLES) && ctx->tables_valid && ctx->tables_key == key;
    ctx->tables_valid = false;
    const float *src = d_dn;
    unsigned *stats = (unsigned *)(ws + sp.off_stats);
    const bool oriented = h_quat && !all_identity(h_quat, batch);
    bool src_sparse = oriented;          // src is read through the tile map
    if (h_shapes) {
        src_sparse = sp.fused_ok;
        const int rc = render_into(ctx, h_shapes, batch, *grid, const_cast<float *>(d_dn), src_sparse ? ws + sp.off_tilemap : nullptr, st, &nl);
        if (rc != SCATMAN_OK) return rc;
    }
    if (oriented) {
        double *rm = (double *)(ws + sp.off_rotmat);
        e = upload_rotmats(h_quat, batch, rm, st, &nl);
        if (e == cudaSuccess)
            e = launch_orient(d_dn, p, rm, batch, (float *)(ws + sp.off_rot), (int *)(ws + sp.off_bbox), st,
                              sp.fused_ok ? stats : nullptr, sp.fused_ok ? ws + sp.off_tilemap : nullptr, orient_occ_ptr(ws + sp.off_bbox, p, batch));
        nl += 3;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "orient");
        src = (const float *)(ws + sp.off_rot);
    }
    // Tensor stages, two ways to the FP16 planes of rho~:  fused (prefix -> planes in one pass, the FP32 rho~ never exists; the scale
    // of the planes then comes from a bound of max |rho~| that needs the extremes of (delta, beta) BEFORE the prefix) when those
    // extremes are free -- a0's bounding-box pass measures them, the host knows them for rendered shapes -- and the chunk has
    // enough columns to fill the machine with one thread per column; else strength + pack (rho~ in FP32, in the buffer the
    // orientation does not use then), which is faster for single grids (profiles/r02_orient_render.md).
    const bool fused = sp.fused_ok && (oriented || h_stats);
    float *rho = (float *)(ws + sp.off_rho);
    unsigned *maxbits = (unsigned *)(ws + sp.off_max);
    if (fused) {
        if (h_stats) e = upload_stats(h_stats, batch, stats, st, &nl);
        if (e == cudaSuccess) e = launch_prefix_bound(stats, p, batch, maxbits, st);
        ++nl;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "prefix bound");
    } else {
        e = launch_strength(src, p, batch, rho, maxbits, st);
        ++nl;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "strength");
    }
    if (sp.tensor) {
        const SepTcPlan &t = sp.tc;
        __half *Eyp = (__half *)(ws + sp.off_eyp), *Exp = (__half *)(ws + sp.off_exp), *Rp = (__half *)(ws + sp.off_rp),
               *Hp = (__half *)(ws + sp.off_hp);
        float *ampscale = (float *)(ws + sp.off_scale);
        int *bounds = (int *)(ws + sp.off_bounds);
        if (!reuse) {
            e = launch_sep_tc_tables(d_qx, npx, d_qy, npy, p, t, Exp, Eyp, st);
            nl += 2;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "qgrid tables");
        }
        ev_begin(ctx, st);
        for (int b0 = 0; b0 < batch; b0 += t.nb) {   // a chunk of items per set of launches, stacked along z
            const int nb = batch - b0 < t.nb ? batch - b0 : t.nb;
            std::string err;
            e = fused ? launch_sep_tc_prefix_prep((const float2 *)src + (size_t)b0 * p.nvox, maxbits + b0, p, t, nb, Rp, ws + sp.off_flags,
                                                  bounds, ampscale + b0, st, false,
                                                  src_sparse ? ws + sp.off_tilemap + orient_tilemap_bytes(p, b0) : nullptr, ws + sp.off_layers)
                      : launch_sep_tc_prep((const float2 *)rho + (size_t)b0 * p.nvox, maxbits + b0, p, t, nb, Rp, ws + sp.off_flags, bounds,
                                           ampscale + b0, st);
            if (e == cudaSuccess) e = launch_sep_tc_x(p, t, Rp, Exp, ws + sp.off_flags, bounds, nb, Hp, ctx->num_sms, st, &err);
            if (e == cudaSuccess)
                e = launch_sep_tc_yz(p, t, Eyp, Hp, ws + sp.off_flags, bounds, nb, d_qx, npx, d_qy, npy,
                                     (float2 *)(ws + sp.off_partial), ctx->num_sms, st, &err);
            if (e == cudaSuccess)
                e = launch_sep_tc_finalize((const float2 *)(ws + sp.off_partial), d_qx, npx, d_qy, npy, p, t, nb, ampscale + b0,
                                           d_I + (size_t)b0 * npx * npy, st);
            nl += 6 + (fused && src_sparse ? 1 : 0);   // pack | prefix, scale, bounds, stage X, stage YZ, finalize (+ the tile map's layer reduction)
            if (e != cudaSuccess) return err.empty() ? cuda_fail(ctx, e, "qgrid stages") : fail(ctx, SCATMAN_CUDA_ERROR, err);
        }
    } else {
        float2 *Ex = (float2 *)(ws + sp.off_ex), *Ey = (float2 *)(ws + sp.off_ey);
        if (!reuse) {
            e = launch_sep_tables(d_qx, npx, d_qy, npy, p, Ex, Ey, st);
            nl += 2;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "qgrid tables");
        }
        ev_begin(ctx, st);
        for (int b = 0; b < batch; ++b) {
            e = launch_sep_item((const float2 *)rho + (size_t)b * p.nvox, p, Ex, Ey, d_qx, npx, d_qy, npy, sp.nzs,
                                (float2 *)(ws + sp.off_h), ws + sp.off_flags, (float2 *)(ws + sp.off_partial),
                                d_I + (size_t)b * npx * npy, st);
            nl += 4;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "qgrid stages");
        }
    }
    ev_end(ctx, st);
    ctx->last_launches = nl;
    ctx->tables_key = key;
    ctx->tables_valid = true;
    return SCATMAN_OK;
}

extern "C" {

int scatman_simulate_qgrid(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda, const double *d_qx,
                           int32_t npx, const double *d_qy, int32_t npy, const double *h_quat, int32_t batch,
                           const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream) {
    return qgrid_impl(ctx, d_dn, grid, lambda, d_qx, npx, d_qy, npy, h_quat, batch, opts, d_ws, ws_bytes, d_I, cuda_stream, nullptr);
}

int scatman_shapes_qgrid_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, int32_t npx, int32_t npy, int32_t batch,
                                         const scatman_options *opts, size_t *bytes) {
    size_t inner = 0;
    const int rc = scatman_qgrid_workspace_bytes(ctx, grid, npx, npy, batch, opts, &inner);
    if (rc != SCATMAN_OK) return rc;
    *bytes = scatman::align_up(sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz * batch, 1024) + inner;
    return SCATMAN_OK;
}

int scatman_simulate_shapes_qgrid(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid,
                                  double lambda, const double *d_qx, int32_t npx, const double *d_qy, int32_t npy,
                                  const scatman_options *opts, void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!h_shapes || !d_ws || !valid_grid(grid) || batch < 1) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    const size_t dn_bytes = scatman::align_up(sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz * batch, 1024);
    if (ws_bytes < dn_bytes) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    float *d_dn = (float *)d_ws;
    std::vector<float> stats;
    shape_stats(h_shapes, batch, stats);
    return qgrid_impl(ctx, d_dn, grid, lambda, d_qx, npx, d_qy, npy, nullptr, batch, opts, (uint8_t *)d_ws + dn_bytes,
                      ws_bytes - dn_bytes, d_I, cuda_stream, stats.data(), h_shapes);
}

// ---- flat detector by a 3-D type-2 NUFFT (nufft_kernels.cu) ----------------------------------------------------------
struct NufftLayout {
    Plan p;
    NufftPlan n;
    NufftTcPlan tc;      // the GEMM stages on tensor cores (tc.ok) ...
    bool fused_ok = false;   // as SepPlan::fused_ok
    bool tensor = false; // ... and whether this call uses them (method AUTO / TENSOR) or the FP64 CUDA-core stages (SIMT_TABLE)
    size_t off_rotmat = 0, off_bbox = 0, off_rot = 0, off_rho = 0, off_max = 0, off_q = 0, off_tz = 0, off_tx = 0, off_ty = 0,
           off_P = 0, off_H = 0, off_U = 0, total = 0;
    // tensor-core stages: table planes, rho~ planes, H planes, V planes, flags, z-split bounds, per-item scales
    size_t off_txp = 0, off_typ = 0, off_tzp = 0, off_rp = 0, off_hp = 0, off_vp = 0, off_flags = 0, off_bounds = 0, off_scale = 0, off_stats = 0, off_tilemap = 0, off_layers = 0;
    size_t hp_bytes = 0;
};
// Range of q over the detector (host, FP64, a1's formula): q_x and q_y are monotonic along u and v and extremal in the other
// coordinate on the rectangle's border; q_z <= 0 is monotonic in u^2 + v^2, so the border pixels plus q_z = 0 bound all three.
static NufftLayout make_nufft_layout(const scatman_grid &g, double lambda, const scatman_detector &det, int batch, int rho_mode,
                                     int method, int num_sms) {
    NufftLayout L;
    Plan &p = L.p;
    p.nx = g.nx; p.ny = g.ny; p.nz = g.nz; p.dx = g.dx; p.dy = g.dy; p.dz = g.dz; p.lambda = lambda;
    p.npix = (int64_t)det.npx * det.npy; p.batch = batch; p.rho_mode = rho_mode;
    p.nvox = (int64_t)g.nx * g.ny * g.nz;
    const double pi = 3.14159265358979323846;
    const double k = 2.0 * pi / lambda;
    const double pitch = 2.0 * tan(det.theta_max_deg * pi / 180.0) / (double)det.npx;
    double lo[3] = {1e300, 1e300, 0.0}, hi[3] = {-1e300, -1e300, 0.0};
    auto visit = [&](int ix, int iy) {
        const double u = ((double)ix + 0.5 - 0.5 * (double)det.npx + det.cx) * pitch;
        const double v = ((double)iy + 0.5 - 0.5 * (double)det.npy + det.cy) * pitch;
        const double s2 = u * u + v * v, r = sqrt(s2 + 1.0);
        const double q[3] = {k * u / r, k * v / r, -k * s2 / (r * (r + 1.0))};
        for (int d = 0; d < 3; ++d) { lo[d] = q[d] < lo[d] ? q[d] : lo[d]; hi[d] = q[d] > hi[d] ? q[d] : hi[d]; }
    };
    for (int ix = 0; ix < det.npx; ++ix) { visit(ix, 0); visit(ix, det.npy - 1); }
    for (int iy = 0; iy < det.npy; ++iy) { visit(0, iy); visit(det.npx - 1, iy); }
    // the axes u = 0 and v = 0 cross the rectangle where |q_x| (|q_y|) along an edge peaks: cover them by the nearest pixels
    for (int ix = 0; ix < det.npx; ++ix) {
        int iy = (int)floor(0.5 * det.npy - det.cy);
        for (int d = -1; d <= 1; ++d) if (iy + d >= 0 && iy + d < det.npy) visit(ix, iy + d);
    }
    for (int iy = 0; iy < det.npy; ++iy) {
        int ix = (int)floor(0.5 * det.npx - det.cx);
        for (int d = -1; d <= 1; ++d) if (ix + d >= 0 && ix + d < det.npx) visit(ix + d, iy);
    }
    const int N[3] = {g.nx, g.ny, g.nz};
    const double dd[3] = {g.dx, g.dy, g.dz};
    NufftAxis *ax[3] = {&L.n.ax, &L.n.ay, &L.n.az};
    for (int d = 0; d < 3; ++d) {
        const double h = 2.0 * pi / (2.0 * (double)N[d] * dd[d]);
        ax[d]->inv_h = 1.0 / h;
        const int m_lo = (int)floor(lo[d] / h - 0.5 * kNufftW) - 1;
        const int m_hi = (int)ceil(hi[d] / h + 0.5 * kNufftW) + 3;   // + 2: the interpolation's common window of W + 2 cells
        ax[d]->m_lo = m_lo;
        ax[d]->nq = m_hi - m_lo + 1;
    }
    // widest step between neighbouring pixels of a row, in grid cells: |dq/du| <= k on every axis (largest at the centre)
    {
        const double hmin = 2.0 * pi / (2.0 * fmax(fmax(g.nx * g.dx, g.ny * g.dy), g.nz * g.dz));
        L.n.pixel_cells = k * pitch / hmin;
    }
    // batch items per chunk (one set of launches each): at most 2 GB of stage-Z planes
    {
        const double per_item = 16.0 * (double)L.n.az.nq * g.ny * g.nx;
        int nb = (int)fmax(1.0, floor(2147483648.0 / per_item));
        if (nb > batch) nb = batch;
        if ((int64_t)nb * L.n.az.nq > 65535) nb = 65535 / L.n.az.nq > 0 ? 65535 / L.n.az.nq : 1;
        L.n.nb = nb;
    }
    L.tc = make_nufft_tc_plan(p, L.n, batch, num_sms);
    L.tensor = L.tc.ok && method != SCATMAN_METHOD_SIMT_TABLE;
    // Two layouts share the head (q-map, then the phase tables of the method in use: batch-independent, SCATMAN_FLAG_REUSE_TABLES);
    // the workspace size is the larger of the two so that one buffer serves both methods.
    size_t total[2] = {0, 0};
    for (int tensor = 0; tensor < 2; ++tensor) {
        if (tensor && !L.tc.ok) continue;
        const bool mine = (tensor != 0) == L.tensor;
        size_t off = 0;
        auto take = [&](size_t bytes) { size_t o2 = off; off = scatman::align_up(off + bytes, 1024); return o2; };
        const size_t o_q = take(sizeof(double) * 3 * (size_t)p.npix);
        if (mine) L.off_q = o_q;
        if (!tensor) {
            const size_t a = take(sizeof(double2) * (size_t)L.n.az.nq * g.nz), b = take(sizeof(double2) * (size_t)L.n.ax.nq * g.nx),
                         c = take(sizeof(double2) * (size_t)L.n.ay.nq * g.ny);
            if (mine) { L.off_tz = a; L.off_tx = b; L.off_ty = c; }
        } else {
            const NufftTcPlan &t = L.tc;
            const size_t a = take(sizeof(__half) * 4 * (size_t)t.NPXP * t.sep.NXP), b = take(sizeof(__half) * 4 * (size_t)t.NQYP * t.NY),
                         c = take(sizeof(__half) * 4 * (size_t)t.NQZP * t.NZP);
            if (mine) { L.off_txp = a; L.off_typ = b; L.off_tzp = c; }
        }
        const size_t o_rm = take(sizeof(double) * 9 * (size_t)batch), o_bb = take(orient_scratch_bytes(p, batch)),
                     o_rot = take(sizeof(float) * 2 * (size_t)p.nvox * batch),
                     o_rho = tensor && fused_prefix_pays(p, batch < L.tc.nb ? batch : L.tc.nb)   // see make_sep_plan
                                 ? o_rot : take(sizeof(float) * 2 * (size_t)p.nvox * batch),
                     o_max = take(sizeof(unsigned) * (size_t)batch), o_st = take(sizeof(unsigned) * 3 * (size_t)batch);
        if (mine) { L.off_rotmat = o_rm; L.off_bbox = o_bb; L.off_rot = o_rot; L.off_rho = o_rho; L.off_max = o_max; L.off_stats = o_st; L.fused_ok = tensor && o_rho == o_rot; }
        {
            const size_t o_tm = tensor && o_rho == o_rot ? take(orient_tilemap_bytes(p, batch)) : 0;
            const size_t o_ly = tensor && o_rho == o_rot ? take(tile_layers_bytes(p, batch)) : 0;
            if (mine) { L.off_tilemap = o_tm; L.off_layers = o_ly; }
        }
        if (!tensor) {
            const size_t a = take(sizeof(double2) * (size_t)L.n.nb * L.n.az.nq * g.ny * g.nx),
                         b = take(sizeof(double2) * (size_t)L.n.nb * L.n.az.nq * g.ny * L.n.ax.nq),
                         c = take(sizeof(float2) * (size_t)L.n.nb * L.n.az.nq * L.n.ay.nq * L.n.ax.nq);
            if (mine) { L.off_P = a; L.off_H = b; L.off_U = c; }
        } else {
            const NufftTcPlan &t = L.tc;
            const size_t slices = (size_t)t.nb * g.nz;
            const size_t hp = sizeof(__half) * 4 * slices * t.NPXP * t.NY;
            const size_t a = take(sizeof(__half) * 4 * slices * t.NY * t.sep.NXP), b = take(hp),
                         c = take(sizeof(__half) * 4 * (size_t)t.NPXP * t.NQYP * t.NZT), d = take(slices * (t.NY / 64)),
                         e2 = take(sizeof(int) * (size_t)((t.sep.nsx + 1) + (size_t)t.nb * t.sep.ng * (t.sep.nzs + 1))),
                         f = take(sizeof(float) * (size_t)batch),
                         u = take(sizeof(float2) * (size_t)t.nb * L.n.az.nq * L.n.ay.nq * L.n.ax.nq);
            if (mine) { L.off_rp = a; L.off_hp = b; L.hp_bytes = hp; L.off_vp = c; L.off_flags = d; L.off_bounds = e2; L.off_scale = f; L.off_U = u; }
        }
        total[tensor] = off;
    }
    L.total = total[0] > total[1] ? total[0] : total[1];
    return L;
}

int scatman_nufft_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, double lambda, const scatman_detector *det,
                                  int32_t batch, size_t *bytes) {
    if (!ctx || !bytes) return SCATMAN_INVALID_ARGUMENT;
    if (!valid_grid(grid) || !valid_detector(det) || !(lambda > 0.0) || !std::isfinite(lambda) || batch < 1)
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    *bytes = make_nufft_layout(*grid, lambda, *det, batch, 0, SCATMAN_METHOD_AUTO, ctx->num_sms).total;
    return SCATMAN_OK;
}

int scatman_nufft_grid_dims(scatman_ctx *ctx, const scatman_grid *grid, double lambda, const scatman_detector *det,
                            int32_t *nq) {
    if (!ctx || !nq) return SCATMAN_INVALID_ARGUMENT;
    if (!valid_grid(grid) || !valid_detector(det) || !(lambda > 0.0) || !std::isfinite(lambda))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    const NufftLayout L = make_nufft_layout(*grid, lambda, *det, 1, 0, SCATMAN_METHOD_AUTO, ctx->num_sms);
    nq[0] = L.n.ax.nq; nq[1] = L.n.ay.nq; nq[2] = L.n.az.nq;
    return SCATMAN_OK;
}

}  // extern "C"

static int nufft_impl(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                      const scatman_detector *det, const double *h_quat, int32_t batch, const scatman_options *opts,
                      void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream, const float *h_stats,
                      const scatman_shape *h_shapes = nullptr) {   // h_stats, h_shapes: see qgrid_impl
    scatman_options o = opts ? *opts : scatman_options{0, 0, 0, 0};
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!d_dn || !d_I || !d_ws || !valid_grid(grid) || !valid_detector(det) || !(lambda > 0.0) || !std::isfinite(lambda) ||
        batch < 1 || batch > 65535 || (o.rho_mode != SCATMAN_RHO_LINEAR && o.rho_mode != SCATMAN_RHO_N2M1) || !valid_qgrid_method(o.method))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    if (h_quat && !valid_quats(h_quat, batch)) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "quaternion is not unit");
    if (((uintptr_t)d_dn | (uintptr_t)d_ws | (uintptr_t)d_I) & 15)
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "device pointers must be 16-byte aligned");
    cudaSetDevice(ctx->device);
    const NufftLayout L = make_nufft_layout(*grid, lambda, *det, batch, o.rho_mode, o.method, ctx->num_sms);
    const Plan &p = L.p;
    if (ws_bytes < L.total) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint8_t *ws = (uint8_t *)d_ws;
    int nl = 0;
    ctx->ev_valid = false;
    ctx->d_count = nullptr;
    TableKey key;
    key.route = 3;
    key.nx = grid->nx; key.ny = grid->ny; key.nz = grid->nz; key.dx = grid->dx; key.dy = grid->dy; key.dz = grid->dz;
    key.lambda = lambda; key.npx = det->npx; key.npy = det->npy; key.theta = det->theta_max_deg; key.cx = det->cx; key.cy = det->cy;
    key.method = L.tensor ? 1 : 3;
    key.ws = d_ws;
    const bool reuse = (o.flags & SCATMAN_FLAG_REUSE_TABLES) && ctx->tables_valid && ctx->tables_key == key;
    ctx->tables_valid = false;
    double *q = (double *)(ws + L.off_q);
    cudaError_t e = cudaSuccess;
    if (!reuse) {
        e = launch_qmap(*det, lambda, q, st);
        ++nl;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "qmap");
    }
    const float *src = d_dn;
    unsigned *stats = (unsigned *)(ws + L.off_stats), *maxbits = (unsigned *)(ws + L.off_max);
    const bool oriented = h_quat && !all_identity(h_quat, batch);
    bool src_sparse = oriented;
    if (h_shapes) {
        src_sparse = L.fused_ok;
        const int rc = render_into(ctx, h_shapes, batch, *grid, const_cast<float *>(d_dn), src_sparse ? ws + L.off_tilemap : nullptr, st, &nl);
        if (rc != SCATMAN_OK) return rc;
    }
    if (oriented) {
        double *rm = (double *)(ws + L.off_rotmat);
        e = upload_rotmats(h_quat, batch, rm, st, &nl);
        if (e == cudaSuccess)
            e = launch_orient(d_dn, p, rm, batch, (float *)(ws + L.off_rot), (int *)(ws + L.off_bbox), st,
                              L.fused_ok ? stats : nullptr, L.fused_ok ? ws + L.off_tilemap : nullptr, orient_occ_ptr(ws + L.off_bbox, p, batch));
        nl += 3;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "orient");
        src = (const float *)(ws + L.off_rot);
    }
    const bool fused = L.fused_ok && (oriented || h_stats);   // see qgrid_impl
    float *rho = (float *)(ws + L.off_rho);
    if (fused) {
        if (h_stats) e = upload_stats(h_stats, batch, stats, st, &nl);
        if (e == cudaSuccess) e = launch_prefix_bound(stats, p, batch, maxbits, st);
        ++nl;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "prefix bound");
    } else {
        e = launch_strength(src, p, batch, rho, maxbits, st);
        ++nl;
        if (e != cudaSuccess) return cuda_fail(ctx, e, "strength");
    }
    if (L.tensor) {
        // GEMM stages on tcgen05 (nufft_tensor_kernels.cu): pack -> stage X (the separable route's) -> stage Y -> stage Z -> interpolation
        const NufftTcPlan &t = L.tc;
        __half *Txp = (__half *)(ws + L.off_txp), *Typ = (__half *)(ws + L.off_typ), *Tzp = (__half *)(ws + L.off_tzp);
        __half *Rp = (__half *)(ws + L.off_rp), *Hp = (__half *)(ws + L.off_hp), *Vp = (__half *)(ws + L.off_vp);
        float *ampscale = (float *)(ws + L.off_scale);
        int *bounds = (int *)(ws + L.off_bounds);
        float2 *U = (float2 *)(ws + L.off_U);
        if (!reuse) {
            e = launch_nufft_tc_tables(p, L.n, t, Txp, Typ, Tzp, st);
            nl += 3;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "nufft tables");
        }
        int Ly = 0;
        while ((1 << Ly) < p.ny) ++Ly;
        ev_begin(ctx, st);
        for (int b0 = 0; b0 < batch; b0 += t.nb) {
            const int nb = batch - b0 < t.nb ? batch - b0 : t.nb;
            std::string err;
            e = fused ? launch_sep_tc_prefix_prep((const float2 *)src + (size_t)b0 * p.nvox, maxbits + b0, p, t.sep, nb, Rp, ws + L.off_flags,
                                                  bounds, ampscale + b0, st, true,
                                                  src_sparse ? ws + L.off_tilemap + orient_tilemap_bytes(p, b0) : nullptr, ws + L.off_layers)
                      : launch_sep_tc_prep((const float2 *)rho + (size_t)b0 * p.nvox, maxbits + b0, p, t.sep, nb, Rp, ws + L.off_flags, bounds,
                                           ampscale + b0, st, true);
            // stage X writes only the live 128-y tiles of H; stage Y reads whole slices: the rest must be zero
            SCATMAN_STAGE_CHECK(e, st, "nufft pack");
            // (when a slice is a single 128-y tile, stage Y zeroes the rows of unwritten slices itself: no pass over the 2 GB of H)
            if (e == cudaSuccess && nufft_tc_needs_h_memset(t))
                e = cudaMemsetAsync(Hp, 0, sizeof(__half) * 4 * (size_t)nb * p.nz * t.NPXP * t.NY, st);
            if (e == cudaSuccess) e = launch_sep_tc_x(p, t.sep, Rp, Txp, ws + L.off_flags, bounds, nb, Hp, ctx->num_sms, st, &err, L.n.ax.nq);
            SCATMAN_STAGE_CHECK(e, st, "nufft stage X");
            if (e == cudaSuccess) e = launch_nufft_tc_yz(p, L.n, t, nb, Hp, Typ, Tzp, Vp, U, ctx->num_sms, st, &err, ws + L.off_flags);
            SCATMAN_STAGE_CHECK(e, st, "nufft stages Y, Z");
            // amplitude = accumulator x (the separable route's per-item scale) / (2^10 of Tz x stage Y's 2^(-11 - Ly))
            if (e == cudaSuccess)
                e = launch_nufft_interp(p, L.n, nb, det->npx, det->npy, L.n.pixel_cells, q, U, ampscale + b0, ldexp(1.0, 1 + Ly),
                                        d_I + (size_t)b0 * p.npix, st);
            nl += 7 + (fused && src_sparse ? 1 : 0);   // pack | prefix, scale, bounds, stages X, Y, Z, interpolation (+ the tile map's layer reduction)
            if (e != cudaSuccess) return err.empty() ? cuda_fail(ctx, e, "nufft stages") : fail(ctx, SCATMAN_CUDA_ERROR, err);
        }
    } else {
        double2 *Tz = (double2 *)(ws + L.off_tz), *TxT = (double2 *)(ws + L.off_tx), *Ty = (double2 *)(ws + L.off_ty);
        if (!reuse) {
            e = launch_nufft_tables(p, L.n, Tz, TxT, Ty, st);
            nl += 3;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "nufft tables");
        }
        ev_begin(ctx, st);
        for (int b0 = 0; b0 < batch; b0 += L.n.nb) {   // a chunk of items per set of launches
            const int nb = batch - b0 < L.n.nb ? batch - b0 : L.n.nb;
            e = launch_nufft_chunk((const float2 *)rho + (size_t)b0 * p.nvox, p, L.n, nb, det->npx, det->npy, L.n.pixel_cells, Tz, TxT, Ty,
                                   q, (double2 *)(ws + L.off_P), (double2 *)(ws + L.off_H), (float2 *)(ws + L.off_U),
                                   d_I + (size_t)b0 * p.npix, st);
            nl += 4;
            if (e != cudaSuccess) return cuda_fail(ctx, e, "nufft stages");
        }
    }
    ev_end(ctx, st);
    ctx->last_launches = nl;
    ctx->tables_key = key;
    ctx->tables_valid = true;
    return SCATMAN_OK;
}

extern "C" {

int scatman_simulate_nufft(scatman_ctx *ctx, const float *d_dn, const scatman_grid *grid, double lambda,
                           const scatman_detector *det, const double *h_quat, int32_t batch, const scatman_options *opts,
                           void *d_ws, size_t ws_bytes, float *d_I, void *cuda_stream) {
    return nufft_impl(ctx, d_dn, grid, lambda, det, h_quat, batch, opts, d_ws, ws_bytes, d_I, cuda_stream, nullptr);
}

int scatman_shapes_nufft_workspace_bytes(scatman_ctx *ctx, const scatman_grid *grid, double lambda, const scatman_detector *det,
                                         int32_t batch, size_t *bytes) {
    size_t inner = 0;
    const int rc = scatman_nufft_workspace_bytes(ctx, grid, lambda, det, batch, &inner);
    if (rc != SCATMAN_OK) return rc;
    *bytes = scatman::align_up(sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz * batch, 1024) + inner;
    return SCATMAN_OK;
}

int scatman_simulate_shapes_nufft(scatman_ctx *ctx, const scatman_shape *h_shapes, int32_t batch, const scatman_grid *grid,
                                  double lambda, const scatman_detector *det, const scatman_options *opts, void *d_ws,
                                  size_t ws_bytes, float *d_I, void *cuda_stream) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!h_shapes || !d_ws || !valid_grid(grid) || batch < 1) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    const size_t dn_bytes = scatman::align_up(sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz * batch, 1024);
    if (ws_bytes < dn_bytes) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    float *d_dn = (float *)d_ws;
    std::vector<float> stats;
    shape_stats(h_shapes, batch, stats);
    return nufft_impl(ctx, d_dn, grid, lambda, det, nullptr, batch, opts, (uint8_t *)d_ws + dn_bytes, ws_bytes - dn_bytes, d_I, cuda_stream,
                      stats.data(), h_shapes);
}

// ---- forward-fitting pieces ---------------------------------------------------------------------------------------
int scatman_fit_workspace_bytes(scatman_ctx *ctx, int64_t npix, int32_t batch, size_t *bytes) {
    if (!ctx || !bytes) return SCATMAN_INVALID_ARGUMENT;
    if (npix < 1 || batch < 1 || batch > 65535) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    *bytes = fit_workspace_bytes(npix, batch);
    return SCATMAN_OK;
}

int scatman_discrepancy(scatman_ctx *ctx, const float *d_I, const float *d_M, int64_t m_stride, const uint8_t *d_mask,
                        int64_t npix, int32_t batch, int32_t metric, void *d_ws, size_t ws_bytes, double *d_out,
                        void *cuda_stream) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!d_I || !d_M || !d_ws || !d_out || npix < 1 || batch < 1 || batch > 65535 || (m_stride != 0 && m_stride != npix) ||
        (metric != SCATMAN_LOSS_L2_NORMALISED && metric != SCATMAN_LOSS_POISSON_DEVIANCE))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    if (((uintptr_t)d_ws | (uintptr_t)d_out) & 7) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "d_ws, d_out must be 8-byte aligned");
    if (ws_bytes < fit_workspace_bytes(npix, batch)) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    cudaSetDevice(ctx->device);
    cudaError_t e = launch_discrepancy(d_I, d_M, m_stride, d_mask, npix, batch, metric, (double *)d_ws, d_out,
                                       (cudaStream_t)cuda_stream);
    ctx->last_launches = fit_discrepancy_launches(npix, batch);
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "discrepancy");
}

// The same kernels as scatman_discrepancy on the library's static scratch array: no allocation anywhere on this path.
int scatman_discrepancy_static(scatman_ctx *ctx, const float *d_I, const float *d_M, int64_t m_stride, const uint8_t *d_mask,
                               int64_t npix, int32_t batch, int32_t metric, double *d_out, void *cuda_stream) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!d_I || !d_M || !d_out || npix < 1 || batch < 1 || batch > 65535 || (m_stride != 0 && m_stride != npix) ||
        (metric != SCATMAN_LOSS_L2_NORMALISED && metric != SCATMAN_LOSS_POISSON_DEVIANCE))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    if ((uintptr_t)d_out & 7) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "d_out must be 8-byte aligned");
    const size_t need = fit_workspace_bytes(npix, batch);
    if (need > (size_t)SCATMAN_STATIC_SCRATCH_BYTES)
        return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL,
                    "scatman_discrepancy_static: npix = " + std::to_string(npix) + ", batch = " + std::to_string(batch) + " need " +
                        std::to_string(need) + " bytes of scratch, the static array holds " +
                        std::to_string((size_t)SCATMAN_STATIC_SCRATCH_BYTES) + " (use scatman_discrepancy with a workspace)");
    if (!ctx->fit_static)
        return cuda_fail(ctx, ctx->fit_static_err != cudaSuccess ? ctx->fit_static_err : cudaErrorInvalidSymbol, "static scratch address");
    cudaSetDevice(ctx->device);
    // every word of the scratch that is read (partials, sums) is written first by this call's own kernels: nothing to clear
    cudaError_t e = launch_discrepancy(d_I, d_M, m_stride, d_mask, npix, batch, metric, ctx->fit_static, d_out, (cudaStream_t)cuda_stream);
    ctx->last_launches = fit_discrepancy_launches(npix, batch);
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "discrepancy (static scratch)");
}

int scatman_ideal_detector(scatman_ctx *ctx, const float *d_I, int64_t npix, int32_t batch, const double *h_photons,
                           uint64_t seed, void *d_ws, size_t ws_bytes, float *d_counts, void *cuda_stream) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    if (!d_I || !h_photons || !d_ws || !d_counts || npix < 1 || batch < 1 || batch > 65535)
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    for (int b = 0; b < batch; ++b)
        if (!(h_photons[b] >= 0.0) || !std::isfinite(h_photons[b])) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad photon number");
    if ((uintptr_t)d_ws & 7) return fail(ctx, SCATMAN_INVALID_ARGUMENT, "d_ws must be 8-byte aligned");
    if (ws_bytes < fit_workspace_bytes(npix, batch)) return fail(ctx, SCATMAN_WORKSPACE_TOO_SMALL, "workspace too small");
    cudaSetDevice(ctx->device);
    cudaError_t e = launch_ideal_detector(d_I, npix, batch, h_photons, seed, (double *)d_ws, d_counts, (cudaStream_t)cuda_stream);
    ctx->last_launches = 3;
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "ideal detector");
}

}  // extern "C"

// ---- host-buffer entry points: copy / compute pipeline ----------------------------------------------------------------
// The batch is cut into chunks; chunk c + 1 is uploaded on `in_stream` while chunk c computes on `host_stream` and the
// patterns of chunk c - 1 go back on `out_stream` (two input and two output buffers in the context's arena, one workspace:
// compute is serial).  Phase tables are built by the first chunk and reused by the others and by later calls with the same
// geometry (the arena belongs to the context, so nobody else can have touched them).
static int host_prepare(scatman_ctx *ctx) {
    if (ctx->host_stream) return SCATMAN_OK;
    cudaError_t e = cudaStreamCreateWithFlags(&ctx->host_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->in_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->out_stream, cudaStreamNonBlocking);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&ctx->in_ready[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->in_free[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->out_free[i], cudaEventDisableTiming);
    }
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "host pipeline setup");
}

static int host_chunk_items(size_t in_item_bytes, int batch) {
    // ~256 MB of input per chunk; a batch worth overlapping (>= 16 MB) is cut into at least two chunks
    size_t n = ((size_t)256 << 20) / (in_item_bytes ? in_item_bytes : 1);
    if (n < 1) n = 1;
    if (n > (size_t)batch) n = (size_t)batch;
    if (batch >= 2 && n == (size_t)batch && in_item_bytes * (size_t)batch >= ((size_t)16 << 20)) n = ((size_t)batch + 1) / 2;
    return (int)n;
}

// run(d_dn, b0, nb, d_ws, d_I, stream): enqueue the simulation of items [b0, b0 + nb) on `stream`
template <class Run>
static int host_pipeline(scatman_ctx *ctx, const float *h_dn, size_t in_item_bytes, float *h_I, size_t out_item_bytes, int batch,
                         int chunk, size_t ws_bytes, const void *h_extra, size_t extra_bytes, void **d_extra_out, Run run) {
    int rc = host_prepare(ctx);
    if (rc != SCATMAN_OK) return rc;
    const size_t ws_b = scatman::align_up(ws_bytes, 1024), ex_b = scatman::align_up(extra_bytes, 1024);
    const size_t in_b = scatman::align_up(in_item_bytes * (size_t)chunk, 1024), out_b = scatman::align_up(out_item_bytes * (size_t)chunk, 1024);
    const size_t need = ws_b + ex_b + 2 * in_b + 2 * out_b;
    cudaError_t e;
    if (need > ctx->arena_bytes) {
        if (ctx->arena) cudaFree(ctx->arena);
        ctx->arena = nullptr;
        ctx->arena_bytes = 0;
        ctx->tables_valid = false;
        if ((e = cudaMalloc(&ctx->arena, need)) != cudaSuccess) return cuda_fail(ctx, e, "arena cudaMalloc");
        ctx->arena_bytes = need;
    }
    uint8_t *a = (uint8_t *)ctx->arena;
    void *d_ws = a;
    uint8_t *d_extra = a + ws_b;
    uint8_t *d_in[2] = {a + ws_b + ex_b, a + ws_b + ex_b + in_b};
    uint8_t *d_out[2] = {a + ws_b + ex_b + 2 * in_b, a + ws_b + ex_b + 2 * in_b + out_b};
    if (d_extra_out) *d_extra_out = d_extra;
    if (extra_bytes && (e = cudaMemcpyAsync(d_extra, h_extra, extra_bytes, cudaMemcpyHostToDevice, ctx->in_stream)) != cudaSuccess)
        return cuda_fail(ctx, e, "H2D");
    int launches = 0;
    rc = SCATMAN_OK;
    e = cudaSuccess;
    for (int c = 0, b0 = 0; b0 < batch && rc == SCATMAN_OK && e == cudaSuccess; ++c, b0 += chunk) {
        const int nb = batch - b0 < chunk ? batch - b0 : chunk, buf = c & 1;
        if (c >= 2) e = cudaStreamWaitEvent(ctx->in_stream, ctx->in_free[buf], 0);      // the compute that read this buffer is done
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(d_in[buf], (const uint8_t *)h_dn + (size_t)b0 * in_item_bytes, (size_t)nb * in_item_bytes,
                                cudaMemcpyHostToDevice, ctx->in_stream);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->in_ready[buf], ctx->in_stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->host_stream, ctx->in_ready[buf], 0);
        if (e == cudaSuccess && c >= 2) e = cudaStreamWaitEvent(ctx->host_stream, ctx->out_free[buf], 0);   // its patterns have left
        if (e != cudaSuccess) break;
        rc = run((const float *)d_in[buf], b0, nb, d_ws, (float *)d_out[buf], ctx->host_stream);
        if (rc != SCATMAN_OK) break;
        launches += ctx->last_launches;
        e = cudaEventRecord(ctx->in_free[buf], ctx->host_stream);                       // input consumed = patterns ready
        if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->out_stream, ctx->in_free[buf], 0);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync((uint8_t *)h_I + (size_t)b0 * out_item_bytes, d_out[buf], (size_t)nb * out_item_bytes,
                                cudaMemcpyDeviceToHost, ctx->out_stream);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->out_free[buf], ctx->out_stream);
    }
    // nothing of this call is left in flight when it returns, whatever happened
    cudaError_t e1 = cudaStreamSynchronize(ctx->in_stream), e2 = cudaStreamSynchronize(ctx->host_stream),
                e3 = cudaStreamSynchronize(ctx->out_stream);
    if (rc != SCATMAN_OK) return rc;
    if (e == cudaSuccess) e = e1 != cudaSuccess ? e1 : e2 != cudaSuccess ? e2 : e3;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "host pipeline");
    ctx->last_launches = launches;
    return SCATMAN_OK;
}

extern "C" {

int scatman_simulate_host(scatman_ctx *ctx, const float *h_dn, const scatman_grid *grid, double lambda,
                          const scatman_detector *det, const double *h_quat, int32_t batch, const scatman_options *opts,
                          float *h_I) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    scatman_options o = opts ? *opts : scatman_options{0, 0, 0, 0};
    if (!h_dn || !h_I || !valid_grid(grid) || !valid_detector(det) || batch < 1 || batch > 65535 || !valid_options(o) || !(lambda > 0.0))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    cudaSetDevice(ctx->device);
    o.flags |= SCATMAN_FLAG_REUSE_TABLES;
    const int64_t npix = (int64_t)det->npx * det->npy;
    const size_t in_item = sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz, out_item = sizeof(float) * (size_t)npix;
    const int chunk = host_chunk_items(in_item, batch);
    size_t ws_bytes = make_plan(*grid, lambda, npix, chunk, o, ctx->num_sms).total;
    if (batch % chunk) {
        const size_t last = make_plan(*grid, lambda, npix, batch % chunk, o, ctx->num_sms).total;
        ws_bytes = last > ws_bytes ? last : ws_bytes;
    }
    return host_pipeline(ctx, h_dn, in_item, h_I, out_item, batch, chunk, ws_bytes, nullptr, 0, nullptr,
                         [&](const float *d_dn, int b0, int nb, void *d_ws, float *d_I, cudaStream_t st) {
                             return run_path(ctx, d_dn, grid, lambda, det, nullptr, npix, h_quat ? h_quat + 4 * (size_t)b0 : nullptr, nb,
                                             &o, d_ws, ws_bytes, d_I, st);
                         });
}

int scatman_simulate_nufft_host(scatman_ctx *ctx, const float *h_dn, const scatman_grid *grid, double lambda,
                                const scatman_detector *det, const double *h_quat, int32_t batch, const scatman_options *opts,
                                float *h_I) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    scatman_options o = opts ? *opts : scatman_options{0, 0, 0, 0};
    if (!h_dn || !h_I || !valid_grid(grid) || !valid_detector(det) || batch < 1 || batch > 65535 || !(lambda > 0.0) ||
        !std::isfinite(lambda) || (o.rho_mode != SCATMAN_RHO_LINEAR && o.rho_mode != SCATMAN_RHO_N2M1))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    cudaSetDevice(ctx->device);
    o.flags |= SCATMAN_FLAG_REUSE_TABLES;
    const int64_t npix = (int64_t)det->npx * det->npy;
    const size_t in_item = sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz, out_item = sizeof(float) * (size_t)npix;
    const int chunk = host_chunk_items(in_item, batch);
    size_t ws_bytes = make_nufft_layout(*grid, lambda, *det, chunk, o.rho_mode, o.method, ctx->num_sms).total;   // grows with the batch
    return host_pipeline(ctx, h_dn, in_item, h_I, out_item, batch, chunk, ws_bytes, nullptr, 0, nullptr,
                         [&](const float *d_dn, int b0, int nb, void *d_ws, float *d_I, cudaStream_t st) {
                             return scatman_simulate_nufft(ctx, d_dn, grid, lambda, det, h_quat ? h_quat + 4 * (size_t)b0 : nullptr, nb, &o,
                                                           d_ws, ws_bytes, d_I, (void *)st);
                         });
}

int scatman_simulate_qgrid_host(scatman_ctx *ctx, const float *h_dn, const scatman_grid *grid, double lambda, const double *h_qx,
                                int32_t npx, const double *h_qy, int32_t npy, const double *h_quat, int32_t batch,
                                const scatman_options *opts, float *h_I) {
    if (!ctx) return SCATMAN_INVALID_ARGUMENT;
    scatman_options o = opts ? *opts : scatman_options{0, 0, 0, 0};
    if (!h_dn || !h_I || !h_qx || !h_qy || !valid_grid(grid) || npx < 1 || npy < 1 || batch < 1 || batch > 65535 || !(lambda > 0.0) ||
        !std::isfinite(lambda) || (o.rho_mode != SCATMAN_RHO_LINEAR && o.rho_mode != SCATMAN_RHO_N2M1) || !valid_qgrid_method(o.method))
        return fail(ctx, SCATMAN_INVALID_ARGUMENT, "bad argument");
    cudaSetDevice(ctx->device);
    // the q arrays come from the host on every call: the tables are reused only if their VALUES are those of the last call
    std::vector<double> qv((size_t)npx + npy);
    std::memcpy(qv.data(), h_qx, sizeof(double) * npx);
    std::memcpy(qv.data() + npx, h_qy, sizeof(double) * npy);
    if (qv != ctx->host_q) ctx->tables_valid = false;
    o.flags |= SCATMAN_FLAG_REUSE_TABLES;
    const size_t in_item = sizeof(float) * 2 * (size_t)grid->nx * grid->ny * grid->nz, out_item = sizeof(float) * (size_t)npx * npy;
    const int chunk = host_chunk_items(in_item, batch);
    size_t ws_bytes = make_sep_plan(*grid, lambda, npx, npy, chunk, o.rho_mode, o.method, ctx->num_sms).total;
    if (batch % chunk) {
        const size_t last = make_sep_plan(*grid, lambda, npx, npy, batch % chunk, o.rho_mode, o.method, ctx->num_sms).total;
        ws_bytes = last > ws_bytes ? last : ws_bytes;
    }
    void *d_q = nullptr;
    const int rc = host_pipeline(ctx, h_dn, in_item, h_I, out_item, batch, chunk, ws_bytes, qv.data(), sizeof(double) * qv.size(), &d_q,
                                 [&](const float *d_dn, int b0, int nb, void *d_ws, float *d_I, cudaStream_t st) {
                                     const double *d_qx = (const double *)d_q, *d_qy = d_qx + npx;
                                     return scatman_simulate_qgrid(ctx, d_dn, grid, lambda, d_qx, npx, d_qy, npy,
                                                                   h_quat ? h_quat + 4 * (size_t)b0 : nullptr, nb, &o, d_ws, ws_bytes, d_I,
                                                                   (void *)st);
                                 });
    if (rc == SCATMAN_OK) ctx->host_q.swap(qv); else ctx->host_q.clear();
    return rc;
}

int scatman_last_launch_count(scatman_ctx *ctx, int32_t *count) {
    if (!ctx || !count) return SCATMAN_INVALID_ARGUMENT;
    *count = ctx->last_launches;
    return SCATMAN_OK;
}

int scatman_last_issued_blocks(scatman_ctx *ctx, int64_t *blocks) {
    if (!ctx || !blocks) return SCATMAN_INVALID_ARGUMENT;
    *blocks = -1;
    if (!ctx->d_count) return SCATMAN_OK;
    unsigned long long v = 0;
    cudaError_t e = cudaMemcpyAsync(&v, ctx->d_count, sizeof(v), cudaMemcpyDeviceToHost, ctx->count_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->count_stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "issued blocks");
    *blocks = (int64_t)v;
    return SCATMAN_OK;
}

int scatman_last_contraction_ms(scatman_ctx *ctx, float *ms) {
    if (!ctx || !ms) return SCATMAN_INVALID_ARGUMENT;
    *ms = -1.f;
    if (!ctx->ev_valid) return SCATMAN_OK;
    cudaError_t e = cudaEventSynchronize(ctx->ev1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, ctx->ev0, ctx->ev1);
    return e == cudaSuccess ? SCATMAN_OK : cuda_fail(ctx, e, "event");
}

}  // extern "C"
