// prep_kernels.cu -- the HBM-bound steps around the contraction: a1 q-map, a0 orient, a2 column prefix,
// operand packing, a3 phase tables, and the |A|^2 finalize.  All FP64 where a phase is formed.
#include "internal.h"

namespace scatman {

__device__ __forceinline__ double centre(int i, int n, double d) { return ((double)i - 0.5 * (double)(n - 1)) * d; }

// ------------------------------------------------------------------------------------------------ a1
// Eq. 3 in north_star's form q = k (s_pixel - z^): flat detector at unit distance.
__global__ void qmap_kernel(int npx, int npy, double pitch, double cx, double cy, double k, double *__restrict__ q) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= (int64_t)npx * npy) return;
    const int ix = (int)(p % npx), iy = (int)(p / npx);
    const double u = ((double)ix + 0.5 - 0.5 * (double)npx + cx) * pitch;
    const double v = ((double)iy + 0.5 - 0.5 * (double)npy + cy) * pitch;
    const double s2 = u * u + v * v;
    const double r = sqrt(s2 + 1.0);
    q[3 * p + 0] = k * u / r;
    q[3 * p + 1] = k * v / r;
    q[3 * p + 2] = -k * s2 / (r * (r + 1.0));  // = k (1/r - 1) without the cancellation (R10)
}

cudaError_t launch_qmap(const scatman_detector &det, double lambda, double *d_q, cudaStream_t st) {
    const int64_t npix = (int64_t)det.npx * det.npy;
    const double pitch = 2.0 * tan(det.theta_max_deg * 3.14159265358979323846 / 180.0) / (double)det.npx;
    const double k = 2.0 * 3.14159265358979323846 / lambda;
    qmap_kernel<<<(unsigned)((npix + 255) / 256), 256, 0, st>>>(det.npx, det.npy, pitch, det.cx, det.cy, k, d_q);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ a0
// Block 5 / Fig. 6: beam-frame voxel <- trilinear sample of the body-frame grid at
// r_body = R^T r_beam.  rotmat[b][9] row-major R (body -> beam).  One thread per beam-frame voxel.
// Bounding box (voxel indices, inclusive) of the non-vacuum voxels of every body-frame grid: bbox[b] = {x0, y0, z0, x1, y1, z1},
// initialised by the launcher to {INT_MAX x3, -1 x3}.  One block per (b, z) slice.  The resampling below gathers 8 corners
// along a slanted line (its cost is cache wavefronts, not bytes); beam-frame voxels that land outside this box are vacuum
// without looking.
// Per-item extremes of a grid: stats[b] = {max |delta|, max |beta|, max(0, -beta)} as FP32 bit patterns (non-negative floats order
// like their bits, so atomicMax works; zeroed by the launcher).  They bound |rho~| BEFORE the prefix runs (prefix_bound_kernel),
// which lets the separable and NUFFT routes write their FP16 operand planes straight from the prefix kernel.
struct Extremes {
    float d = 0.f, b = 0.f, nb = 0.f;
    __device__ __forceinline__ void see(float delta, float beta) {
        d = fmaxf(d, fabsf(delta));
        b = fmaxf(b, fabsf(beta));
        nb = fmaxf(nb, -beta);
    }
    __device__ __forceinline__ void reduce_warp() {   // whole warps call this
        for (int off = 16; off > 0; off >>= 1) {
            d = fmaxf(d, __shfl_xor_sync(0xffffffffu, d, off));
            b = fmaxf(b, __shfl_xor_sync(0xffffffffu, b, off));
            nb = fmaxf(nb, __shfl_xor_sync(0xffffffffu, nb, off));
        }
    }
    __device__ __forceinline__ void store(unsigned *__restrict__ stats) const {
        if (d > 0.f) atomicMax(stats + 0, __float_as_uint(d));
        if (b > 0.f) atomicMax(stats + 1, __float_as_uint(b));
        if (nb > 0.f) atomicMax(stats + 2, __float_as_uint(nb));
    }
};

// occ != null: also a coarse occupancy map for orient_kernel, occ[b][nz/4 + 1][ny/4 + 1][nx/4 + 1] bytes: byte (p >> 2) of every axis is
// set for p = m and p = m + 1 of every non-vacuum voxel m, so that the 2x2x2 interpolation cell with first corner c holds material
// only if the byte of (c + 1) >> 2 is set -- one cached byte instead of eight gathered corners for the vacuum inside the box.
constexpr int kOccSliceCap = 4096;   // bytes of a slice's map in shared memory (grids up to ~250 x 250)
__global__ void __launch_bounds__(256)
bbox_kernel(const float2 *__restrict__ in, int nx, int ny, int nz, int *__restrict__ bbox, unsigned *__restrict__ stats,
            unsigned char *__restrict__ occ) {
    const int iz = blockIdx.x % nz, b = blockIdx.x / nz;
    __shared__ unsigned char socc[kOccSliceCap];
    const int nbx8 = nx / 4 + 1, nby8 = ny / 4 + 1;
    if (occ) {
        for (int i = threadIdx.x; i < nbx8 * nby8; i += 256) socc[i] = 0;
        __syncthreads();
    }
    const float2 *src = in + ((size_t)b * nz + iz) * (size_t)nx * ny;
    int x0 = 0x7fffffff, y0 = 0x7fffffff, x1 = -1, y1 = -1;
    Extremes ex;
    const int n = nx * ny;
    // two voxels per 16-byte load (slices start 16-byte aligned when nx ny is even; the odd case takes the scalar path), four
    // loads in flight per thread: the pass is bound by HBM bandwidth, not by load latency
    auto seen = [&](int e) {
        const int x = e % nx, y = e / nx;
        x0 = min(x0, x); x1 = max(x1, x);
        y0 = min(y0, y); y1 = max(y1, y);
        if (occ) {
            const int xa = x >> 2, xb = (x + 1) >> 2, ya = (y >> 2) * nbx8, yb = ((y + 1) >> 2) * nbx8;
            socc[ya + xa] = 1;
            if (xb != xa) socc[ya + xb] = 1;
            if (yb != ya) { socc[yb + xa] = 1; if (xb != xa) socc[yb + xb] = 1; }
        }
    };
    if ((n & 1) == 0) {
        const float4 *src4 = (const float4 *)src;
        // gridDim.y blocks share a slice (single grids: nz blocks alone would leave SMs idle; never with the occupancy map)
        const int n2 = (int)((long long)(n >> 1) * (blockIdx.y + 1) / gridDim.y);
        for (int e0 = (int)((long long)(n >> 1) * blockIdx.y / gridDim.y) + threadIdx.x; e0 < n2; e0 += 4 * 256) {
            float4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) v[u] = e0 + u * 256 < n2 ? __ldg(src4 + e0 + u * 256) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (v[u].x != 0.f || v[u].y != 0.f) seen(2 * (e0 + u * 256));
                if (v[u].z != 0.f || v[u].w != 0.f) seen(2 * (e0 + u * 256) + 1);
                ex.see(v[u].x, v[u].y);
                ex.see(v[u].z, v[u].w);
            }
        }
    } else {
        const int n1 = (int)((long long)n * (blockIdx.y + 1) / gridDim.y);
        for (int e = (int)((long long)n * blockIdx.y / gridDim.y) + threadIdx.x; e < n1; e += 256) {
            const float2 v = __ldg(src + e);
            if (v.x != 0.f || v.y != 0.f) seen(e);
            ex.see(v.x, v.y);
        }
    }
    // warp -> block -> one set of atomics per block (a slice's eight warps hitting the same words serialise in L2 otherwise)
    for (int off = 16; off > 0; off >>= 1) {
        x0 = min(x0, __shfl_xor_sync(0xffffffffu, x0, off));
        y0 = min(y0, __shfl_xor_sync(0xffffffffu, y0, off));
        x1 = max(x1, __shfl_xor_sync(0xffffffffu, x1, off));
        y1 = max(y1, __shfl_xor_sync(0xffffffffu, y1, off));
    }
    ex.reduce_warp();
    __shared__ int sbox[8][4];
    __shared__ float sext[8][3];
    const int warp = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) {
        sbox[warp][0] = x0; sbox[warp][1] = y0; sbox[warp][2] = x1; sbox[warp][3] = y1;
        sext[warp][0] = ex.d; sext[warp][1] = ex.b; sext[warp][2] = ex.nb;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) {
            x0 = min(x0, sbox[w][0]); y0 = min(y0, sbox[w][1]);
            x1 = max(x1, sbox[w][2]); y1 = max(y1, sbox[w][3]);
            ex.d = fmaxf(ex.d, sext[w][0]); ex.b = fmaxf(ex.b, sext[w][1]); ex.nb = fmaxf(ex.nb, sext[w][2]);
        }
        if (x1 >= 0) {
            int *o = bbox + 6 * b;
            atomicMin(o + 0, x0); atomicMin(o + 1, y0); atomicMin(o + 2, iz);
            atomicMax(o + 3, x1); atomicMax(o + 4, y1); atomicMax(o + 5, iz);
            if (stats) ex.store(stats + 3 * b);
        }
    }
    if (occ) {   // (the block barrier above orders the slice map)
        const int za = iz >> 2, zb = (iz + 1) >> 2;
        unsigned char *o = occ + (size_t)b * (nz / 4 + 1) * nby8 * nbx8;
        for (int i = threadIdx.x; i < nbx8 * nby8; i += 256)
            if (socc[i]) {
                o[(size_t)za * nby8 * nbx8 + i] = 1;
                if (zb != za) o[(size_t)zb * nby8 * nbx8 + i] = 1;
            }
    }
}

__global__ void bbox_init_kernel(int *__restrict__ bbox, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) bbox[i] = (i % 6) < 3 ? 0x7fffffff : -1;
}

// Output voxels are handled in TILES of 16 x 4 x 4 (256 threads, one voxel each) so that the 2x2x2 source cells of a tile share
// cache lines for any rotation (row-shaped tiles gather along a slanted line and read 30x more sectors than they use).
// A block owns one layer of tiles (fixed item b and tile row bz) and walks it in chunks of 256 tiles: first every thread decides
// for ONE tile whether it can hold material at all -- the tile's image in the body frame is a parallelepiped whose extent along
// each body axis follows from three signed edge vectors, compared with the box of non-vacuum voxels widened by the interpolation
// cell -- and leaves the tile's origin in the body frame, its offset in the slice and its extent in shared memory; the live tiles
// are compacted (ballot); then the block resamples the live tiles -- a voxel's body-frame index is its tile's origin plus a
// per-thread constant: no index division, no integer -> FP64 conversion (the XU pipe's 4 lanes per scheduler were the limit) --
// and, for dense output, zero-fills the others with 16-byte stores.
// tilemap != null: SPARSE output -- the other tiles are not written at all; tilemap[b][bz][tile] = 1 for the written tiles that received
// material (see internal.h).
// (One launch-sized block per tile, each loading the rotation and the box and deciding on its own, was bound by that start-up
// latency, not by arithmetic or bytes: profiles/r02_orient_render.md.)
__device__ __forceinline__ void floor_split(double f, int &i, double &t) {   // f = i + t, i = floor(f), |f| < 2^31: FP64 adds only
    const double kMagic = 6755399441055744.0;                              // 1.5 * 2^52: f + kMagic holds round(f) in its low word
    const double r = f + kMagic;
    double n = r - kMagic;
    i = __double2loint(r);
    if (n > f) { n -= 1.0; --i; }
    t = f - n;
}

__global__ void __launch_bounds__(256, 4)   // 64 registers: four CTAs per SM (at 100 registers two CTAs left the issue slots half empty)
orient_kernel(const float2 *__restrict__ in, int nx, int ny, int nz, double dx, double dy, double dz, double3 inv,
              const double *__restrict__ rotmat, const int *__restrict__ bbox, float2 *__restrict__ out, unsigned char *__restrict__ tilemap,
              const unsigned char *__restrict__ occ8) {
    const int nbx = (nx + 15) / 16, nby = (ny + 3) / 4, nbz = (nz + 3) / 4;
    const int bz = blockIdx.x % nbz, b = blockIdx.x / nbz;
    __shared__ double sR[9];
    __shared__ int sbb[6];
    __shared__ double sbd[6];              // the box of non-vacuum voxels widened by one cell: lo - 1 (x, y, z), hi + 1
    __shared__ double tile_f[256][3];      // body-frame index of the tile's first voxel
    __shared__ int tile_off[256];          // offset of that voxel in its slice
    __shared__ unsigned char tile_ext[256];   // (extent - 1) of the tile along x | along y << 4 (ragged edges)
    __shared__ unsigned char hit[256];
    __shared__ unsigned char occ[256];     // sparse output: the tile received a non-vacuum voxel
    __shared__ unsigned short live[256];   // the chunk's tiles that can hold material, in order
    __shared__ int wcount[8];
    if (threadIdx.x < 9) sR[threadIdx.x] = rotmat[9 * b + threadIdx.x];
    if (threadIdx.x >= 32 && threadIdx.x < 38) {
        const int k = threadIdx.x - 32, v = bbox[6 * b + k];
        sbb[k] = v;
        sbd[k] = (double)(k < 3 ? v - 1 : v + 1);
    }
    __syncthreads();
    const double *R = sR;
    // fractional body-frame index of beam-frame voxel (ix, iy, iz): f = origin + ix ex + iy ey + iz ez (one row of R^T per axis);
    // kept in shared memory (the registers go to the resampling loop)
    __shared__ double sE[12];              // ex[3], ey[3], ez[3], origin[3]
    if (threadIdx.x < 9) {
        const int row = threadIdx.x / 3, d = threadIdx.x % 3;
        sE[threadIdx.x] = R[threadIdx.x] * (row == 0 ? dx : row == 1 ? dy : dz) * (d == 0 ? inv.x : d == 1 ? inv.y : inv.z);
    } else if (threadIdx.x < 12) {
        const int d = threadIdx.x - 9;
        const double xb0 = centre(0, nx, dx), yb0 = centre(0, ny, dy), zb0 = centre(0, nz, dz);
        sE[threadIdx.x] = (R[d] * xb0 + R[3 + d] * yb0 + R[6 + d] * zb0) * (d == 0 ? inv.x : d == 1 ? inv.y : inv.z) +
                          0.5 * (double)((d == 0 ? nx : d == 1 ? ny : nz) - 1);
    }
    __syncthreads();
    const double *ex = sE, *ey = sE + 3, *ez = sE + 6;
    const int lx = threadIdx.x & 15, ly = (threadIdx.x >> 4) & 3, lz = threadIdx.x >> 6;
    const int iz = bz * 4 + lz;
    const int wz = min(3, nz - 1 - bz * 4);                         // tile extent - 1 along z
    const bool empty = sbb[3] < 0;                                  // an all-vacuum item
    const float2 *src = in + (size_t)b * nx * ny * nz;
    const int nbx8 = nx / 4 + 1, nby8 = ny / 4 + 1;
    const unsigned char *occb = occ8 ? occ8 + (size_t)b * (nz / 4 + 1) * nby8 * nbx8 : nullptr;   // bbox_kernel's coarse occupancy map
    float2 *dstb = out + (size_t)b * nx * ny * nz;
    float2 *dstt = dstb + ((size_t)iz * ny + ly) * nx + lx;         // + tile_off
    // this thread's voxel relative to its tile's first one, in body-frame index units
    const double lo0 = (double)lx * ex[0] + (double)ly * ey[0] + (double)lz * ez[0];
    const double lo1 = (double)lx * ex[1] + (double)ly * ey[1] + (double)lz * ez[1];
    const double lo2 = (double)lx * ex[2] + (double)ly * ey[2] + (double)lz * ez[2];
    // gridDim.y blocks share a layer (single grids: a layer per block leaves most SMs without one)
    const int ntile = (int)(((long long)nbx * nby * (blockIdx.y + 1)) / gridDim.y);
    for (int t0 = (int)(((long long)nbx * nby * blockIdx.y) / gridDim.y); t0 < ntile; t0 += 256) {
        int nlive;
        {   // phase 1: thread t decides tile t0 + t
            const int t = t0 + threadIdx.x;
            bool h = false;
            if (t < ntile) {
                const int bx = t % nbx, by = t / nbx;
                const int wx = min(15, nx - 1 - bx * 16), wy = min(3, ny - 1 - by * 4);
                h = !empty;
                int qlo[3], qhi[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const double f0 = sE[9 + d] + (double)(bx * 16) * ex[d] + (double)(by * 4) * ey[d] + (double)(bz * 4) * ez[d];
                    tile_f[threadIdx.x][d] = f0;
                    const double sx = (double)wx * ex[d], sy = (double)wy * ey[d], sz = (double)wz * ez[d];
                    const double lo = f0 + fmin(sx, 0.0) + fmin(sy, 0.0) + fmin(sz, 0.0);
                    const double hi = f0 + fmax(sx, 0.0) + fmax(sy, 0.0) + fmax(sz, 0.0);
                    // the per-voxel test below is f > bb_lo - 1 && f < bb_hi + 1; a slack of 1e-9 voxels covers the rounding of this
                    // bound against the per-voxel evaluation (a wrongly kept tile only costs time)
                    if (hi <= sbd[d] - 1e-9 || lo >= sbd[3 + d] + 1e-9) h = false;
                    // blocks of the coarse occupancy map that the first corners of the tile's cells fall into (slack as above)
                    const int nd = d == 0 ? nx : d == 1 ? ny : nz;
                    qlo[d] = max(0, (int)floor(lo - 1e-9) + 1) >> 2;
                    qhi[d] = min(nd, (int)floor(hi + 1e-9) + 1) >> 2;
                }
                if (h && occb) {   // no occupied block among them: no cell of the tile holds material
                    unsigned any = 0;      // (no early exit: the loads are independent and stay in flight together)
                    for (int qz = qlo[2]; qz <= qhi[2]; ++qz)
                        for (int qy = qlo[1]; qy <= qhi[1]; ++qy) {
                            const unsigned char *row = occb + ((size_t)qz * nby8 + qy) * nbx8;
                            for (int qx = qlo[0]; qx <= qhi[0]; ++qx) any |= __ldg(row + qx);
                        }
                    h = any != 0;
                }
                tile_off[threadIdx.x] = by * 4 * nx + bx * 16;
                tile_ext[threadIdx.x] = (unsigned char)(wx | (wy << 4));
            }
            hit[threadIdx.x] = h ? 1 : 0;
            occ[threadIdx.x] = 0;
            // compact the live tiles (ballot + warp counts): the resampling loop below visits only those
            const unsigned bal = __ballot_sync(0xffffffffu, h);
            if ((threadIdx.x & 31) == 0) wcount[threadIdx.x >> 5] = __popc(bal);
            __syncthreads();
            int before = 0, total = 0;
#pragma unroll
            for (int w = 0; w < 8; ++w) {
                before += w < (int)(threadIdx.x >> 5) ? wcount[w] : 0;
                total += wcount[w];
            }
            if (h) live[before + __popc(bal & ((1u << (threadIdx.x & 31)) - 1u))] = (unsigned short)threadIdx.x;
            nlive = total;
        }
        __syncthreads();
        if (!tilemap) {
            // dense output: zero-fill the tiles that cannot hold material, a 128-byte tile row per 8 threads (16-byte stores when
            // the rows are 16-byte aligned, i.e. nx is even)
            const int tend = min(256, ntile - t0);
            for (int e = threadIdx.x; e < tend * 128; e += 256) {
                const int tt = e >> 7, r = (e >> 3) & 15, c = e & 7;       // tile, row of the tile (ly + 4 lz), 2-voxel chunk
                if (hit[tt]) continue;
                const int ext = tile_ext[tt];
                const int cx = 2 * c, cy = r & 3, izr = bz * 4 + (r >> 2);
                if (cx > (ext & 15) || cy > (ext >> 4) || izr >= nz) continue;
                float2 *d2 = dstb + ((size_t)izr * ny + cy) * nx + tile_off[tt] + cx;
                if ((nx & 1) == 0) *reinterpret_cast<float4 *>(d2) = make_float4(0.f, 0.f, 0.f, 0.f);
                else {
                    d2[0] = make_float2(0.f, 0.f);
                    if (cx + 1 <= (ext & 15)) d2[1] = make_float2(0.f, 0.f);
                }
            }
        }
        if (iz < nz) {
            for (int li = 0; li < nlive; ++li) {
                const int tt = live[li];
                const int ext = tile_ext[tt];
                if (lx > (ext & 15) || ly > (ext >> 4)) continue;
                const double fx = tile_f[tt][0] + lo0, fy = tile_f[tt][1] + lo1, fz = tile_f[tt][2] + lo2;
                float2 o = make_float2(0.f, 0.f);
                // the 2x2x2 cell holds material only if every coordinate lies within one voxel of the box of non-vacuum voxels
                if (fx > sbd[0] && fx < sbd[3] && fy > sbd[1] && fy < sbd[4] && fz > sbd[2] && fz < sbd[5]) {
                    int x0, y0, z0;
                    double tx, ty, tz;
                    floor_split(fx, x0, tx);
                    floor_split(fy, y0, ty);
                    floor_split(fz, z0, tz);
                    // the coarse map says whether the cell can hold material at all (z0 + 1 etc. lie in [0, n]: the box test above)
                    if (occb && !occb[(((z0 + 1) >> 2) * nby8 + ((y0 + 1) >> 2)) * nbx8 + ((x0 + 1) >> 2)]) {
                        dstt[tile_off[tt]] = o;
                        continue;
                    }
                    // Interior of the cell grid (the usual case): the eight corners without bounds tests.  If they all hold the same value
                    // -- deep inside a homogeneous particle, or in the vacuum around it -- the interpolated value IS that value (the
                    // weights sum to 1 within 1e-16, far below half an FP32 ulp), bit for bit what the weighted sum rounds to: skip it.
                    bool done = false;
                    if (x0 >= 0 && y0 >= 0 && z0 >= 0 && x0 + 1 < nx && y0 + 1 < ny && z0 + 1 < nz) {
                        const float2 *c0 = src + ((size_t)z0 * ny + y0) * nx + x0;
                        const size_t sy = (size_t)nx, sz = (size_t)nx * ny;
                        const float2 v000 = __ldg(c0), v001 = __ldg(c0 + 1), v010 = __ldg(c0 + sy), v011 = __ldg(c0 + sy + 1);
                        const float2 v100 = __ldg(c0 + sz), v101 = __ldg(c0 + sz + 1), v110 = __ldg(c0 + sz + sy), v111 = __ldg(c0 + sz + sy + 1);
                        const bool same = v001.x == v000.x && v001.y == v000.y && v010.x == v000.x && v010.y == v000.y && v011.x == v000.x &&
                                          v011.y == v000.y && v100.x == v000.x && v100.y == v000.y && v101.x == v000.x && v101.y == v000.y &&
                                          v110.x == v000.x && v110.y == v000.y && v111.x == v000.x && v111.y == v000.y;
                        if (same) {
                            o = v000;
                            done = true;
                        }
                    }
                    if (!done) {
                        const double wxx[2] = {1.0 - tx, tx}, wyy[2] = {1.0 - ty, ty}, wzz[2] = {1.0 - tz, tz};
                        double are = 0.0, aim = 0.0;
#pragma unroll
                        for (int cz = 0; cz < 2; ++cz) {
                            const int zi = z0 + cz;
                            if (zi < 0 || zi >= nz) continue;
#pragma unroll
                            for (int cy = 0; cy < 2; ++cy) {
                                const int yi = y0 + cy;
                                if (yi < 0 || yi >= ny) continue;
                                const double wyz = wyy[cy] * wzz[cz];
                                const float2 *row = src + ((size_t)zi * ny + yi) * nx;
#pragma unroll
                                for (int cx = 0; cx < 2; ++cx) {
                                    const int xi = x0 + cx;
                                    if (xi < 0 || xi >= nx) continue;
                                    const float2 v = __ldg(row + xi);
                                    if (v.x == 0.f && v.y == 0.f) continue;   // most of a grid is vacuum: skip the FP64 conversions
                                    const double w = wxx[cx] * wyz;
                                    are = fma(w, (double)v.x, are);
                                    aim = fma(w, (double)v.y, aim);
                                }
                            }
                        }
                        o = make_float2((float)are, (float)aim);
                    }
                }
                dstt[tile_off[tt]] = o;
                if (tilemap && (o.x != 0.f || o.y != 0.f)) occ[tt] = 1;
            }
        }
        __syncthreads();
        // the map says which tiles HOLD material, not merely which were written: the box test of phase 1 keeps about twice the tiles an
        // ellipsoid touches, and the prefix pass then skips the rest (and the layers they leave empty) as well
        if (tilemap && t0 + (int)threadIdx.x < ntile)
            tilemap[((size_t)b * nbz + bz) * ((size_t)nbx * nby) + t0 + threadIdx.x] = occ[threadIdx.x];
    }
}

// maxbits[b] = FP32 bits of an upper bound of max |component of rho~| of item b (without dV): |f(dn)| <= fb from the extremes, and
// |T_j| = exp(-k dz sum beta) <= exp(k dz nz max(0, -beta)) (1 for absorbing material, beta >= 0).  The bound only sets the FP16
// operand scale: it may be loose by orders of magnitude without costing accuracy that matters.
__global__ void prefix_bound_kernel(const unsigned *__restrict__ stats, int batch, int rho_mode, double kdz_nz, unsigned *__restrict__ maxbits) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    const double D = (double)__uint_as_float(stats[3 * b]), B = (double)__uint_as_float(stats[3 * b + 1]),
                 nb = (double)__uint_as_float(stats[3 * b + 2]);
    double fb = fmax(D, B);
    if (rho_mode == SCATMAN_RHO_N2M1) fb = fmax(D * (2.0 + D) + B * B, 2.0 * B * (1.0 + D));   // c (2 - c), c = delta + i beta
    double bound = fb * exp(fmin(kdz_nz * nb, 80.0));
    if (!(bound < 3.0e38)) bound = 3.0e38;
    maxbits[b] = __float_as_uint((float)bound);
}

cudaError_t launch_prefix_bound(const unsigned *d_stats, const Plan &p, int batch, unsigned *d_maxbits, cudaStream_t st) {
    const double kdz_nz = 2.0 * 3.14159265358979323846 / p.lambda * p.dz * (double)p.nz;
    prefix_bound_kernel<<<(batch + 127) / 128, 128, 0, st>>>(d_stats, batch, p.rho_mode, kdz_nz, d_maxbits);
    return cudaGetLastError();
}

cudaError_t launch_orient(const float *d_in, const Plan &p, const double *d_rotmat, int batch, float *d_out, int *d_bbox,
                          cudaStream_t st, unsigned *d_stats, unsigned char *d_tilemap, unsigned char *d_occ) {
    if (d_stats) {   // extremes of the body-frame grids: the trilinear samples of the beam-frame grid lie within them
        cudaError_t e = cudaMemsetAsync(d_stats, 0, sizeof(unsigned) * 3 * (size_t)batch, st);
        if (e != cudaSuccess) return e;
    }
    const size_t blocks = (size_t)((p.nz + 3) / 4) * batch;     // one block per layer of 16 x 4 x 4 tiles
    if (blocks > 0x7fffffffull || (size_t)p.nz * batch > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    bbox_init_kernel<<<(6 * batch + 255) / 256, 256, 0, st>>>(d_bbox, 6 * batch);
    // four resident blocks per SM; at least 16 tiles per block
    const int ntile = ((p.nx + 15) / 16) * ((p.ny + 3) / 4);
    int nsplit = (int)((4 * 148 + blocks - 1) / blocks);
    if (nsplit > ntile / 16) nsplit = ntile / 16;
    if (nsplit < 1) nsplit = 1;
    if (d_occ && orient_occ_bytes(p, batch) == 0) d_occ = nullptr;   // a slice's map does not fit shared memory
    if (nsplit > 1) d_occ = nullptr;   // single grids: the map's extra memset and look-ups cost the ~8 us they save on batches per item
    if (d_occ) {
        cudaError_t e = cudaMemsetAsync(d_occ, 0, orient_occ_bytes(p, batch), st);
        if (e != cudaSuccess) return e;
    }
    // slices shared by several blocks while there are fewer than two blocks per SM, each part at least 4096 voxels
    int parts = 1;
    if (!d_occ) {
        parts = (int)((2 * 148 + (size_t)p.nz * batch - 1) / ((size_t)p.nz * batch));
        const int most = (int)(((size_t)p.nx * p.ny) / 4096);
        if (parts > most) parts = most;
        if (parts < 1) parts = 1;
    }
    bbox_kernel<<<dim3((unsigned)(p.nz * batch), (unsigned)parts), 256, 0, st>>>((const float2 *)d_in, p.nx, p.ny, p.nz, d_bbox, d_stats, d_occ);
    orient_kernel<<<dim3((unsigned)blocks, (unsigned)nsplit), 256, 0, st>>>((const float2 *)d_in, p.nx, p.ny, p.nz, p.dx, p.dy, p.dz,
                                                   make_double3(1.0 / p.dx, 1.0 / p.dy, 1.0 / p.dz), d_rotmat, d_bbox,
                                                   (float2 *)d_out, d_tilemap, d_occ);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ a2
// Eq. 6/8/9: exclusive z-prefix C_j of dn = delta + i beta per (x,y) column in FP64,
// T_j = exp(i k dz C_j), rho~_j = f(dn_j) T_j (dV applied at the end).  One thread per column; x is the
// fast thread index so every slice access is coalesced.  Also reduces max |component| per batch item
// for the FP16 operand scale.
__global__ void strength_kernel(const float2 *__restrict__ dn, int nx, int ny, int nz, double kdz, int rho_mode,
                                float2 *__restrict__ rho, unsigned *__restrict__ maxbits) {
    const int ix = blockIdx.x * blockDim.x + threadIdx.x;
    const int iy = blockIdx.y, b = blockIdx.z;
    float vmax = 0.f;
    if (ix < nx) {
        const size_t plane = (size_t)nx * ny;
        const size_t base = (size_t)b * plane * nz + (size_t)iy * nx + ix;
        // T_j = exp(i k dz C_j) as a running FP64 product of the per-voxel factors g(dn) = exp(i k dz dn): exp of the
        // prefix sum, one complex multiplication per non-vacuum voxel.  The factor of the last (delta, beta) seen is kept, so a
        // homogeneous stretch of material costs no sincos / exp at all (each costs ~10x the product); a product of N factors
        // rounds N times (N 2^-53 relative), far below the FP32 the result is stored in.
        double Tre = 1.0, Tim = 0.0;
        double gre = 1.0, gim = 0.0;
        float ld = 0.f, lb = 0.f;          // the (delta, beta) of g; (0, 0) <-> g = 1
        // slices in batches of 8: the loads of a batch are independent of the running product, so they are all in flight
        // before the (serial) FP64 chain of the batch starts
        for (int iz0 = 0; iz0 < nz; iz0 += 8) {
            float2 cin[8];
#pragma unroll
            for (int i = 0; i < 8; ++i)
                cin[i] = iz0 + i < nz ? __ldg(dn + base + (size_t)(iz0 + i) * plane) : make_float2(0.f, 0.f);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (iz0 + i >= nz) break;
                const float2 c = cin[i];
                float2 o = make_float2(0.f, 0.f);
                if (c.x != 0.f || c.y != 0.f) {
                    const double d = (double)c.x, be = (double)c.y;
                    double fre = d, fim = be;
                    if (rho_mode == SCATMAN_RHO_N2M1) {  // c (2 - c)
                        fre = d * (2.0 - d) + be * be;
                        fim = 2.0 * be * (1.0 - d);
                    }
                    o.x = (float)(fre * Tre - fim * Tim);
                    o.y = (float)(fre * Tim + fim * Tre);
                    vmax = fmaxf(vmax, fmaxf(fabsf(o.x), fabsf(o.y)));
                    if (c.x != ld || c.y != lb) {
                        double s, co;
                        sincos(kdz * d, &s, &co);
                        const double mag = exp(-kdz * be);
                        gre = mag * co;
                        gim = mag * s;
                        ld = c.x;
                        lb = c.y;
                    }
                    const double t = Tre * gre - Tim * gim;
                    Tim = Tre * gim + Tim * gre;
                    Tre = t;
                }
                rho[base + (size_t)(iz0 + i) * plane] = o;
            }
        }
    }
    // block max -> one atomic per block (non-negative floats order like their bit patterns)
    for (int off = 16; off > 0; off >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, off));
    __shared__ float wmax[8];
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = vmax;
    __syncthreads();
    if (threadIdx.x == 0) {
        float m = 0.f;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) m = fmaxf(m, wmax[w]);
        if (m > 0.f && maxbits) atomicMax(maxbits + b, __float_as_uint(m));
    }
}

// The same for grids with so few columns that one thread per column leaves the GPU to a handful of warps, each walking its
// serial chain (128^3: 128 blocks of 128 threads; 32^3: 32 of 64): the column is cut into segments of ZPT slices, one warp of
// 32 columns per segment.  A thread holds its segment's voxels in registers, forms the product of their factors, the block
// exchanges the segment products through shared memory, every thread multiplies those of the segments below it (in order,
// <= 15 products) into its starting T and then writes its slices as strength_kernel does.  The running product is
// associated differently from the one-thread walk: ~nz 2^-53 relative either way.
constexpr int kSplitCols = 32;
constexpr int kSplitMaxSeg = 16;

template <int ZPT>
__global__ void __launch_bounds__(kSplitCols *kSplitMaxSeg)
strength_split_kernel(const float2 *__restrict__ dn, int nx, int ny, int nz, double kdz, int rho_mode, float2 *__restrict__ rho,
                      unsigned *__restrict__ maxbits) {
    __shared__ double2 segP[kSplitMaxSeg][kSplitCols];
    __shared__ float wmax[kSplitMaxSeg];
    const int cx = threadIdx.x & (kSplitCols - 1), seg = threadIdx.x / kSplitCols;
    const int ix = blockIdx.x * kSplitCols + cx, iy = blockIdx.y, b = blockIdx.z;
    const int z0 = seg * ZPT;
    const size_t plane = (size_t)nx * ny;
    const size_t base = (size_t)b * plane * nz + (size_t)iy * nx + ix;
    const bool col = ix < nx;
    float2 cin[ZPT];
#pragma unroll
    for (int i = 0; i < ZPT; ++i)
        cin[i] = col && z0 + i < nz ? __ldg(dn + base + (size_t)(z0 + i) * plane) : make_float2(0.f, 0.f);
    // the factor of the last (delta, beta) seen is kept across both walks: a homogeneous segment costs one sincos / exp
    double gre = 1.0, gim = 0.0;
    float ld = 0.f, lb = 0.f;
    auto factor = [&](const float2 c) {
        if (c.x != ld || c.y != lb) {
            double sn, co;
            sincos(kdz * (double)c.x, &sn, &co);
            const double mag = exp(-kdz * (double)c.y);
            gre = mag * co;
            gim = mag * sn;
            ld = c.x;
            lb = c.y;
        }
    };
    double Pre = 1.0, Pim = 0.0;
#pragma unroll
    for (int i = 0; i < ZPT; ++i) {
        const float2 c = cin[i];
        if (c.x != 0.f || c.y != 0.f) {
            factor(c);
            const double t = Pre * gre - Pim * gim;
            Pim = Pre * gim + Pim * gre;
            Pre = t;
        }
    }
    segP[seg][cx] = make_double2(Pre, Pim);
    __syncthreads();
    double Tre = 1.0, Tim = 0.0;
    for (int q = 0; q < seg; ++q) {
        const double2 pq = segP[q][cx];
        const double t = Tre * pq.x - Tim * pq.y;
        Tim = Tre * pq.y + Tim * pq.x;
        Tre = t;
    }
    float vmax = 0.f;
#pragma unroll
    for (int i = 0; i < ZPT; ++i) {
        if (!col || z0 + i >= nz) break;
        const float2 c = cin[i];
        float2 o = make_float2(0.f, 0.f);
        if (c.x != 0.f || c.y != 0.f) {
            const double d = (double)c.x, be = (double)c.y;
            double fre = d, fim = be;
            if (rho_mode == SCATMAN_RHO_N2M1) {  // c (2 - c)
                fre = d * (2.0 - d) + be * be;
                fim = 2.0 * be * (1.0 - d);
            }
            o.x = (float)(fre * Tre - fim * Tim);
            o.y = (float)(fre * Tim + fim * Tre);
            vmax = fmaxf(vmax, fmaxf(fabsf(o.x), fabsf(o.y)));
            factor(c);
            const double t = Tre * gre - Tim * gim;
            Tim = Tre * gim + Tim * gre;
            Tre = t;
        }
        rho[base + (size_t)(z0 + i) * plane] = o;
    }
    for (int off = 16; off > 0; off >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, off));
    if (cx == 0) wmax[seg] = vmax;
    __syncthreads();
    if (threadIdx.x == 0) {
        float m = 0.f;
        for (int w = 0; w < (int)(blockDim.x / kSplitCols); ++w) m = fmaxf(m, wmax[w]);
        if (m > 0.f && maxbits) atomicMax(maxbits + b, __float_as_uint(m));
    }
}

cudaError_t launch_strength(const float *d_dn, const Plan &p, int batch, float *d_rho, unsigned *d_maxbits,
                            cudaStream_t st) {
    if (d_maxbits) {   // nullptr: the caller does not want the per-item maximum (scatman_effective_strength)
        cudaError_t e = cudaMemsetAsync(d_maxbits, 0, sizeof(unsigned) * batch, st);
        if (e != cudaSuccess) return e;
    }
    const double kdz = 2.0 * 3.14159265358979323846 / p.lambda * p.dz;
    // few columns (below half a thread per lane slot of the GPU): cut the columns along z as well
    if ((size_t)p.nx * p.ny * batch <= 32768 && p.nz > 8 && p.nz <= 16 * kSplitMaxSeg) {
        const int zpt = p.nz <= 8 * kSplitMaxSeg ? 8 : 16, nseg = (p.nz + zpt - 1) / zpt;
        dim3 grid((p.nx + kSplitCols - 1) / kSplitCols, p.ny, batch);
        if (zpt == 8)
            strength_split_kernel<8><<<grid, kSplitCols * nseg, 0, st>>>((const float2 *)d_dn, p.nx, p.ny, p.nz, kdz, p.rho_mode,
                                                                         (float2 *)d_rho, d_maxbits);
        else
            strength_split_kernel<16><<<grid, kSplitCols * nseg, 0, st>>>((const float2 *)d_dn, p.nx, p.ny, p.nz, kdz, p.rho_mode,
                                                                          (float2 *)d_rho, d_maxbits);
        return cudaGetLastError();
    }
    const int threads = p.nx >= 128 ? 128 : 64;
    dim3 grid((p.nx + threads - 1) / threads, p.ny, batch);
    strength_kernel<<<grid, threads, 0, st>>>((const float2 *)d_dn, p.nx, p.ny, p.nz, kdz, p.rho_mode,
                                              (float2 *)d_rho, d_maxbits);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ operand B
// rho~ FP32 [b][z][y][x] -> FP16 split planes, scaled by sB[b] = 2^(13 - e) (max in [2^(e-1), 2^e)), laid out as
// the UMMA B operand wants to find it in shared memory, so that one TMA box of 256-byte rows is one k-step:
//   B[b][z][y16][xt][hg][plane][atom]      atom = 8 x-rows x 16 y of FP16 = 256 bytes, SWIZZLE_32B pattern applied
//   planes 0 Re_hi, 1 Re_lo, 2 Im_hi, 3 Im_lo;  x = 128 xt + 16 blk + 8 half + r  ->  hg = 8 half + blk, row r
// (each CTA of a pair owns one `half` of every 16-x block; a run of hg is then a contiguous x range in both).
// Inside an atom, row r is 32 bytes (y fastest = K-major) and its two 16-byte chunks are swapped when r >= 4.
// Also emits the occupancy word of every (slice, x tile, y group): bit 8*yi + xi = the 16-y x 16-x block is non-zero.
__device__ __forceinline__ float scale_from_maxbits(unsigned bits) {
    const float m = __uint_as_float(bits);
    if (!(m > 0.f)) return 1.f;
    int e;
    frexpf(m, &e);
    return ldexpf(1.f, kScaleBExp - e);
}

__global__ void pack_b_kernel(const float2 *__restrict__ rho, int nx, int ny, int nz, int nxt, int ny16, int ngroups,
                              const unsigned *__restrict__ maxbits, float *__restrict__ ampscale, float dV,
                              __half *__restrict__ B, unsigned long long *__restrict__ mask) {
    __shared__ float2 tile[32][33];
    const int bz = blockIdx.x;  // b*nz + z
    const int b = bz / nz;
    const float s = scale_from_maxbits(maxbits[b]);
    const int x0 = blockIdx.y * 32, y0 = blockIdx.z * 32;
    const int tx = threadIdx.x, ty = threadIdx.y;  // 32 x 8
    const float2 *src = rho + (size_t)bz * nx * ny;
    for (int r = ty; r < 32; r += 8) {
        const int y = y0 + r, x = x0 + tx;
        tile[r][tx] = (y < ny && x < nx) ? src[(size_t)y * nx + x] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    // one warp per atom: ty -> (x8 group ax = ty & 3, y16 block ay = ty >> 2); lane -> row r = tx / 4, 4 y from 4 (tx % 4)
    const int ax = ty & 3, ay = ty >> 2;
    const int r = tx >> 2, yq = (tx & 3) * 4;
    const int xl = ax * 8 + r, yl = ay * 16 + yq;
    __half h[4][4];   // [plane][y]
    bool any = false;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float2 v = tile[yl + i][xl];
        const float re = v.x * s, im = v.y * s;
        h[0][i] = __float2half_rn(re);
        h[1][i] = __float2half_rn(re - __half2float(h[0][i]));
        h[2][i] = __float2half_rn(im);
        h[3][i] = __float2half_rn(im - __half2float(h[2][i]));
        any |= ((__half_as_ushort(h[0][i]) | __half_as_ushort(h[1][i]) | __half_as_ushort(h[2][i]) |
                 __half_as_ushort(h[3][i])) & 0x7fffu) != 0;
    }
    const int x = x0 + ax * 8, y = y0 + ay * 16;          // first x / y of the atom
    const int xt = x / kTileX, blk = (x % kTileX) / 16, half = (x >> 3) & 1;
    const int y16 = y >> 4;
    if (y16 < ny16) {
        const size_t atom = ((((size_t)bz * ny16 + y16) * nxt + xt) * 16 + half * 8 + blk) * 4;   // x 256 bytes, + plane
        const int chunk = (yq >> 3) ^ (r >> 2);                                                 // SWIZZLE_32B
        const int off = r * 16 + chunk * 8 + (yq & 7);                                          // in FP16 elements
#pragma unroll
        for (int pl = 0; pl < 4; ++pl) {
            uint2 w;
            w.x = (uint32_t)__half_as_ushort(h[pl][0]) | ((uint32_t)__half_as_ushort(h[pl][1]) << 16);
            w.y = (uint32_t)__half_as_ushort(h[pl][2]) | ((uint32_t)__half_as_ushort(h[pl][3]) << 16);
            *(uint2 *)(B + (atom + pl) * 128 + off) = w;
        }
        if (__any_sync(0xffffffffu, any) && tx == 0) {
            const int yi = (y % (kGroupYB * kBlockY)) / 16;
            atomicOr(mask + ((size_t)bz * nxt + xt) * ngroups + y / (kGroupYB * kBlockY), 1ull << (8 * yi + blk));
        }
    }
    if (blockIdx.y == 0 && blockIdx.z == 0 && tx == 0 && ty == 0 && (bz % nz) == 0) ampscale[b] = dV / (kScaleA * s);
}

cudaError_t launch_pack_b(const float *d_rho, const Plan &p, const unsigned *d_maxbits, float *d_ampscale,
                          __half *d_B, unsigned long long *d_mask, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(d_mask, 0, sizeof(unsigned long long) * (size_t)p.batch * p.nz * p.nxt * p.ngroups, st);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)(p.batch * p.nz), p.nx_pad / 32, p.ny_pad / 32);
    pack_b_kernel<<<grid, dim3(32, 8), 0, st>>>((const float2 *)d_rho, p.nx, p.ny, p.nz, p.nxt, p.ny_pad / 16, p.ngroups,
                                                d_maxbits, d_ampscale, (float)(p.dx * p.dy * p.dz), d_B, d_mask);
    return cudaGetLastError();
}

// Work the contraction issues (scatman_last_issued_blocks): per occupancy word, (non-empty 16-y steps) x (length of the
// bounding range of non-empty 16-x blocks); a single CTA per item always runs the full 8 blocks of x.
__global__ void count_issued_kernel(const unsigned long long *__restrict__ mask, size_t n, int full_x,
                                    unsigned long long *__restrict__ count) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned v = 0;
    if (i < n) {
        const unsigned long long m = mask[i];
        if (m) {
            int ky = 0;
            unsigned ux = 0;
            for (int yi = 0; yi < 8; ++yi) {
                const unsigned b = (unsigned)(m >> (8 * yi)) & 0xffu;
                ky += b != 0;
                ux |= b;
            }
            const int xm = full_x ? 8 : (32 - __clz((int)ux)) - (__ffs((int)ux) - 1);
            v = (unsigned)(ky * xm);
        }
    }
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(count, (unsigned long long)v);
}

cudaError_t launch_count_issued(const unsigned long long *d_mask, const Plan &p, unsigned long long *d_count,
                                cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const size_t n = (size_t)p.batch * p.nz * p.nxt * p.ngroups;
    count_issued_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_mask, n, p.t_ncta == 1, d_count);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ a3
// Phase tables (Eq. 2's split), phases formed and evaluated in FP64 (R-precision):
//   A planes  fp16 [4][npix_pad][ny_pad]  = split(2^10 e^{i qy(p) y_i})   (the UMMA A operand)
//   anchor    float2 [tile][nxa][128]     = e^{i qx(p) x_{16 a}}
//   fine      float2 [tile][16][128]      = e^{i qx(p) b dx}
//   zturn     uint64 [tile][128]          = frac(qz(p) dz / 4 pi) as a 64-bit fixed-point fraction of a turn: the slice phase
//                                           e^{i qz z_j} is formed in the contraction's epilogue from it (no per-slice table)
// One thread = one pixel x 16 consecutive coordinates: FP64 sincos of the first phase and of the step, then the
// angle-addition recurrence in FP64 (15 complex products; the rounding it adds is ~1e-15, far below the FP32 / FP16-pair
// storage) -- an FP64 sincos per entry made these kernels FP64-throughput-bound.
__device__ __forceinline__ void phase_run16(double q, double x0, double step, double (&re)[16], double (&im)[16]) {
    double s0, c0, ss, cs;
    sincos(q * x0, &s0, &c0);
    sincos(q * step, &ss, &cs);
    re[0] = c0;
    im[0] = s0;
#pragma unroll
    for (int i = 1; i < 16; ++i) {
        re[i] = re[i - 1] * cs - im[i - 1] * ss;
        im[i] = re[i - 1] * ss + im[i - 1] * cs;
    }
}

__global__ void table_a_kernel(const double *__restrict__ q, int64_t npix, int64_t npix_pad, int ny, int ny_pad,
                               double dy, __half *__restrict__ A) {
    const int nrun = ny_pad / 16;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // run fastest: a warp writes 32 x 32 contiguous bytes
    if (t >= npix_pad * nrun) return;
    const int64_t p = t / nrun;
    const int y0 = (int)(t % nrun) * 16;
    double re[16], im[16];
    if (p < npix) phase_run16(q[3 * p + 1], centre(y0, ny, dy), dy, re, im);
    __align__(16) __half h[4][16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        float fr = 0.f, fi = 0.f;
        if (p < npix && y0 + i < ny) {
            fr = (float)(re[i] * (double)kScaleA);
            fi = (float)(im[i] * (double)kScaleA);
        }
        h[0][i] = __float2half_rn(fr);
        h[1][i] = __float2half_rn(fr - __half2float(h[0][i]));
        h[2][i] = __float2half_rn(fi);
        h[3][i] = __float2half_rn(fi - __half2float(h[2][i]));
    }
    const size_t plane = (size_t)npix_pad * ny_pad, o = (size_t)p * ny_pad + y0;
#pragma unroll
    for (int pl = 0; pl < 4; ++pl) {
        uint4 *dst = (uint4 *)(A + pl * plane + o);
        dst[0] = ((const uint4 *)h[pl])[0];
        dst[1] = ((const uint4 *)h[pl])[1];
    }
}

// anchor, fine and the slice-phase turn fraction in ONE launch: blockIdx.y ranges [0, ya) anchor runs, ya = fine, ya + 1 = zturn
__global__ void table_small_all_kernel(const double *__restrict__ q, int64_t npix, int nxa, int nx, double dx, double dz,
                                       int ya, float2 *__restrict__ anchor, float2 *__restrict__ fine,
                                       unsigned long long *__restrict__ zturn) {
    const int lane = threadIdx.x, tile = blockIdx.x;
    const int64_t p = (int64_t)tile * kTileP + lane;
    int y = blockIdx.y;
    if (y == ya + 1) {
        // t = qz dz / (4 pi) turns, reduced to [-1/2, 1/2) and stored as a 64-bit fixed-point fraction (two's complement wraps
        // like the phase does); FP64 carries 53 bits of it, far more than the 32 the epilogue keeps after the multiplication
        unsigned long long v = 0ull;
        if (p < npix) {
            double t = q[3 * p + 2] * dz * (0.25 / 3.14159265358979323846);
            t -= rint(t);
            v = (unsigned long long)(long long)rint(t * 18446744073709551616.0);   // 2^64; |t| <= 1/2 keeps it in int64 range
            if (t >= 0.5) v = 0x8000000000000000ull;
        }
        zturn[(size_t)tile * kTileP + lane] = v;
        return;
    }
    const bool is_fine = y == ya;
    if (is_fine) y = 0;
    const int count = is_fine ? kFine : nxa;
    float2 *out = is_fine ? fine : anchor;
    const int idx0 = y * 16;
    double re[16], im[16];
    if (p < npix) {
        if (!is_fine) phase_run16(q[3 * p + 0], centre(idx0 * kFine, nx, dx), dx * (double)kFine, re, im);
        else phase_run16(q[3 * p + 0], 0.0, dx, re, im);
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        if (idx0 + i >= count) break;
        const float2 v = p < npix ? make_float2((float)re[i], (float)im[i]) : make_float2(1.f, 0.f);
        out[((size_t)tile * count + idx0 + i) * kTileP + lane] = v;
    }
}

cudaError_t launch_tables(const double *d_q, const Plan &p, __half *d_A, float2 *d_anchor, float2 *d_fine,
                          unsigned long long *d_zturn, cudaStream_t st, int *nlaunch) {
    const int64_t nthreads_a = p.npix_pad * (p.ny_pad / 16);
    table_a_kernel<<<(unsigned)((nthreads_a + 127) / 128), 128, 0, st>>>(d_q, p.npix, p.npix_pad, p.ny, p.ny_pad, p.dy, d_A);
    const int ya = (p.nxa + 15) / 16;
    table_small_all_kernel<<<dim3(p.ntiles, ya + 2), kTileP, 0, st>>>(d_q, p.npix, p.nxa, p.nx, p.dx, p.dz, ya, d_anchor, d_fine, d_zturn);
    if (nlaunch) *nlaunch += 2;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ |A|^2
// Block 11: I = |sum of the partial amplitudes|^2 with the amplitude scale undone.
// partial float2 [b][nsplit][npix_pad]; ampscale[b] (device) or NULL -> dV.
__global__ void finalize_kernel(const float2 *__restrict__ partial, int64_t npix, int64_t npix_pad, int nsplit,
                                const float *__restrict__ ampscale, float dV, float *__restrict__ I) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    if (p >= npix) return;
    float re = 0.f, im = 0.f;
    for (int g = 0; g < nsplit; ++g) {
        const float2 v = partial[((size_t)b * nsplit + g) * npix_pad + p];
        re += v.x;
        im += v.y;
    }
    const float s = ampscale ? ampscale[b] : dV;
    re *= s;
    im *= s;
    I[(size_t)b * npix + p] = re * re + im * im;
}

cudaError_t launch_finalize(const float2 *d_partial, const Plan &p, const float *d_ampscale, double dV, float *d_I,
                            cudaStream_t st) {
    dim3 grid((unsigned)((p.npix + 255) / 256), p.batch);
    finalize_kernel<<<grid, 256, 0, st>>>(d_partial, p.npix, p.npix_pad, p.nsplit, d_ampscale, (float)dV, d_I);
    return cudaGetLastError();
}

}  // namespace scatman
