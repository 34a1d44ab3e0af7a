// simt_kernels.cu -- step a7: the CUDA-core comparison variant of the contraction.
//
// SIMT_SINCOS evaluates the definition term by term (Eq. 1-2):
//     A(p) = sum_voxels rho~ * exp(i (qx x + qy y + qz z))
// with ONE sincos of the full phase per (voxel, pixel) term on the SFU (MUFU.SIN/COS) and an FP32
// complex FMA accumulate.  One thread per pixel, 128 pixels per CTA, the rho~ rows of a z-range
// streamed through shared memory (every thread reads the same voxel: LDS broadcast).
//
// Phase accuracy: phases reach ~300 rad, where FP32 q*x would carry ~2e-5 rad of error.  The phase is
// therefore kept in TURNS: the per-row part (qy y + qz z)/2pi is formed and range-reduced in FP64 once
// per row; the per-voxel part tx*xi uses a 12-bit head tx_hi so that tx_hi*xi is exact in FP32 and its
// fractional part is exact too; the tail tx_lo*xi is tiny.
#include "internal.h"

namespace scatman {

constexpr int kSimtThreads = 128;
constexpr int kSimtChunk = 2048;  // voxels (float2) per shared-memory chunk = 16 KB

__global__ void __launch_bounds__(kSimtThreads)
simt_sincos_kernel(const float2 *__restrict__ rho, const double *__restrict__ q, int nx, int ny, int nz, double dx,
                   double dy, double dz, int64_t npix, int64_t npix_pad, int nsplit, float2 *__restrict__ partial) {
    __shared__ float2 srow[kSimtChunk];
    const int tile = blockIdx.x, zs = blockIdx.y, b = blockIdx.z;  // batch <= 65535 (validated)
    const int64_t p = (int64_t)tile * kSimtThreads + threadIdx.x;
    const int64_t pc = p < npix ? p : npix - 1;
    const double inv2pi = 0.15915494309189533577;
    const double tx = q[3 * pc + 0] * dx * inv2pi, ty = q[3 * pc + 1] * dy * inv2pi, tz = q[3 * pc + 2] * dz * inv2pi;
    // 12-bit head of tx: exact products with half-integer |xi| <= 2^11
    const float txh = __uint_as_float(__float_as_uint((float)tx) & 0xfffff000u);
    const float txl = (float)(tx - (double)txh);
    const float cxo = 0.5f * (float)(nx - 1);
    const double cyo = 0.5 * (double)(ny - 1), czo = 0.5 * (double)(nz - 1);
    const int z0 = (int)(((int64_t)nz * zs) / nsplit), z1 = (int)(((int64_t)nz * (zs + 1)) / nsplit);
    const int rows_per_chunk = kSimtChunk / nx > 0 ? kSimtChunk / nx : 1;
    const float2 *vol = rho + (size_t)b * nx * ny * nz;
    float are = 0.f, aim = 0.f;
    const int64_t row_begin = (int64_t)z0 * ny, row_end = (int64_t)z1 * ny;
    for (int64_t r0 = row_begin; r0 < row_end; r0 += rows_per_chunk) {
        const int nrows = (int)((row_end - r0) < rows_per_chunk ? (row_end - r0) : rows_per_chunk);
        // x may exceed the chunk for nx > kSimtChunk: loop x segments
        for (int xs = 0; xs < nx; xs += kSimtChunk) {
            const int xw = (nx - xs) < kSimtChunk ? (nx - xs) : kSimtChunk;
            __syncthreads();
            for (int i = threadIdx.x; i < nrows * xw; i += kSimtThreads) {
                const int rr = i / xw, xx = i - rr * xw;
                srow[i] = __ldg(vol + (size_t)(r0 + rr) * nx + xs + xx);
            }
            __syncthreads();
            for (int rr = 0; rr < nrows; ++rr) {
                const int64_t row = r0 + rr;
                const int iz = (int)(row / ny), iy = (int)(row - (int64_t)iz * ny);
                double base = ty * ((double)iy - cyo) + tz * ((double)iz - czo);
                base -= rint(base);
                const float basef = (float)base;
                float sre = 0.f, sim = 0.f;
                const float2 *s = srow + rr * xw;
                float xi = (float)xs - cxo;
#pragma unroll 4
                for (int xx = 0; xx < xw; ++xx, xi += 1.f) {
                    const float2 v = s[xx];
                    float u = txh * xi;          // exact
                    u -= rintf(u);               // exact fractional part
                    float t = fmaf(txl, xi, u + basef);
                    t -= rintf(t);
                    const float ang = 6.283185307179586f * t;
                    const float sn = __sinf(ang), cs = __cosf(ang);
                    sre = fmaf(v.x, cs, sre);
                    sre = fmaf(-v.y, sn, sre);
                    sim = fmaf(v.x, sn, sim);
                    sim = fmaf(v.y, cs, sim);
                }
                are += sre;
                aim += sim;
            }
        }
    }
    if (p < npix) partial[((size_t)b * nsplit + zs) * npix_pad + p] = make_float2(are, aim);
}

int simt_zsplit(const Plan &p, int num_sms) {
    // enough CTAs for ~8 per SM; never more splits than slices
    const int64_t want = (int64_t)num_sms * 8;
    int64_t zs = (want + (int64_t)p.ntiles * p.batch - 1) / ((int64_t)p.ntiles * p.batch);
    if (zs < 1) zs = 1;
    if (zs > p.nz) zs = p.nz;
    if (zs > 64) zs = 64;
    return (int)zs;
}

cudaError_t launch_simt_sincos(const float *d_rho, const double *d_q, const Plan &p, float2 *d_partial,
                               cudaStream_t st) {
    dim3 grid(p.ntiles, p.nsplit, p.batch);
    simt_sincos_kernel<<<grid, kSimtThreads, 0, st>>>((const float2 *)d_rho, d_q, p.nx, p.ny, p.nz, p.dx, p.dy, p.dz,
                                                      p.npix, p.npix_pad, p.nsplit, d_partial);
    return cudaGetLastError();
}

}  // namespace scatman
