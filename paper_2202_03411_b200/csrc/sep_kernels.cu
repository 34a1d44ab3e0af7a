// sep_kernels.cu -- the separable route for detectors that are a tensor grid in (qx, qy): the paper's
// own evaluation points (Block 6 of Fig. 4 takes the 2-D DFT of every slice on a uniform (qx, qy) grid, PAPER.md:154,
// 146; cost model PAPER.md:435).  On such a grid the inner transform of Eq. 2/9 factors,
//     F_j[b, a] = sum_y e^{i qy[b] y} ( sum_x rho~_j[y, x] e^{i qx[a] x} ),
// into two small complex GEMMs per slice instead of one (pixel x voxel) contraction, N_p times less work:
//   stage X   H[(j, y), a] = sum_x rho~[(j, y), x] Ex[x, a]               one GEMM over all slices at once
//   stage YZ  A[b, a]     = sum_j e^{i qz(a, b) z_j} sum_y Ey[b, y] H[(j, y), a]   (Blocks 7-8 fused: the slice phase
//             is applied to the accumulator tile in registers, slices are summed in registers)
// with qz = -(k - sqrt(k^2 - qx^2 - qy^2)) on the Ewald sphere (Eq. 3-4, north_star's sign).
// FP32 CUDA-core GEMMs (64 x 64 x 16 tiles, 4 x 4 complex outputs per thread), FP64 phases.
#include "internal.h"

namespace scatman {

constexpr int kBM = 64, kBN = 64, kBK = 16;

__device__ __forceinline__ double centre_d(int i, int n, double d) { return ((double)i - 0.5 * (double)(n - 1)) * d; }

// E[i][a] = e^{i q[a] x_i} (transposed = false, a fastest) or E[a][i] (transposed = true, i fastest); FP64 phase
__global__ void sep_table_kernel(const double *__restrict__ q, int nq, int n, double d, int transposed,
                                 float2 *__restrict__ E) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)nq * n) return;
    int a, i;
    if (transposed) { a = (int)(t / n); i = (int)(t % n); }
    else { i = (int)(t / nq); a = (int)(t % nq); }
    double s, c;
    sincos(q[a] * centre_d(i, n, d), &s, &c);
    E[t] = make_float2((float)c, (float)s);
}

// One 64 x 64 complex output tile: acc[4][4] += A[m0.., k] B[k, n0..] over k in [0, K).  A row-major [M][lda] (k fastest),
// B row-major [K][ldb] (n fastest).  256 threads: thread (ty, tx) = (tid / 16, tid % 16) owns rows ty*4.. and cols tx*4..
struct TileSmem {
    float2 As[kBK][kBM + 2];
    float2 Bs[kBK][kBN + 2];
};

// kflag (optional): one byte per 16-k chunk, 0 = every B row of the chunk is zero -> the chunk is skipped (uniformly).
__device__ __forceinline__ int next_chunk(const unsigned char *kflag, int k0, int K) {
    if (kflag)
        while (k0 < K && kflag[k0 / kBK] == 0) k0 += kBK;
    return k0;
}

__device__ __forceinline__ void tile_gemm(const float2 *__restrict__ A, int lda, int M, int m0, const float2 *__restrict__ B,
                                          int ldb, int N, int n0, int K, const unsigned char *__restrict__ kflag, TileSmem &sm,
                                          float2 (&acc)[4][4]) {
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    // loader roles: A tile 64 rows x 16 k: thread -> row tid / 4, k = (tid % 4) * 4 .. +3;  B tile 16 k x 64 n: k = tid / 16, n = (tid % 16) * 4 .. +3
    const int ar = tid >> 2, ak = (tid & 3) * 4;
    const int bk = tid >> 4, bn = (tid & 15) * 4;
    float2 ra[4], rb[4];
    auto load = [&](int k0) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = m0 + ar, k = k0 + ak + i;
            ra[i] = (m < M && k < K) ? __ldg(A + (size_t)m * lda + k) : make_float2(0.f, 0.f);
            const int kk = k0 + bk, n = n0 + bn + i;
            rb[i] = (kk < K && n < N) ? __ldg(B + (size_t)kk * ldb + n) : make_float2(0.f, 0.f);
        }
    };
    int k0 = next_chunk(kflag, 0, K);
    if (k0 < K) load(k0);
    while (k0 < K) {
        __syncthreads();   // previous tile fully consumed
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            sm.As[ak + i][ar] = ra[i];
            sm.Bs[bk][bn + i] = rb[i];
        }
        __syncthreads();
        const int kn = next_chunk(kflag, k0 + kBK, K);
        if (kn < K) load(kn);   // next tile's global loads overlap this tile's FMAs
#pragma unroll
        for (int k = 0; k < kBK; ++k) {
            float2 a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                a[i] = sm.As[k][ty * 4 + i];
                b[i] = sm.Bs[k][tx * 4 + i];
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    acc[i][j].x = fmaf(a[i].x, b[j].x, acc[i][j].x);
                    acc[i][j].x = fmaf(-a[i].y, b[j].y, acc[i][j].x);
                    acc[i][j].y = fmaf(a[i].x, b[j].y, acc[i][j].y);
                    acc[i][j].y = fmaf(a[i].y, b[j].x, acc[i][j].y);
                }
        }
        k0 = kn;
    }
}

// flags[j][c] = 1 if any rho~ value of slice j, y rows [16c, 16c+16) is non-zero (one warp per chunk)
__global__ void sep_rowflags_kernel(const float2 *__restrict__ rho, int nx, int ny, int nz, int nyc,
                                    unsigned char *__restrict__ flags) {
    const int chunk = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (chunk >= nz * nyc) return;
    const int j = chunk / nyc, c = chunk % nyc;
    const int y0 = c * 16, y1 = min(ny, y0 + 16);
    const float2 *src = rho + ((size_t)j * ny + y0) * nx;
    const size_t n = (size_t)(y1 - y0) * nx;
    bool any = false;
    for (size_t e = lane; e < n; e += 32) {
        const float2 v = __ldg(src + e);
        any |= (v.x != 0.f) | (v.y != 0.f);
    }
    any = __any_sync(0xffffffffu, any);
    if (lane == 0) flags[chunk] = any ? 1 : 0;
}

// stage X: H[M][N] = rho[M][K] Ex[K][N]  (M = nz * ny, K = nx, N = npx).  Row tiles whose rho rows are all zero are not
// multiplied: H is written as zeros (vacuum rows are most of a grid).
__global__ void __launch_bounds__(256) sep_stage_x_kernel(const float2 *__restrict__ rho, const float2 *__restrict__ Ex, int M,
                                                          int K, int N, const unsigned char *__restrict__ rowflags,
                                                          float2 *__restrict__ H) {
    __shared__ TileSmem sm;
    __shared__ int s_any;
    const int m0 = blockIdx.x * kBM, n0 = blockIdx.y * kBN;
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    if (tid == 0) s_any = 0;
    __syncthreads();
    bool any = false;
    if (rowflags) {   // ny is a multiple of 16: the 16-row chunks of sep_rowflags_kernel are rows [16 c, 16 c + 16) of rho
        for (int c = 0; c < kBM / 16; ++c)
            if (m0 + 16 * c < M) any |= rowflags[m0 / 16 + c] != 0;
    } else {
        for (size_t e = tid; e < (size_t)kBM * K; e += 256) {
            const int m = m0 + (int)(e / K);
            if (m < M) {
                const float2 v = __ldg(rho + (size_t)m * K + (e % K));
                any |= (v.x != 0.f) | (v.y != 0.f);
            }
        }
    }
    if (any) s_any = 1;
    __syncthreads();
    float2 acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = make_float2(0.f, 0.f);
    if (s_any) tile_gemm(rho, K, M, m0, Ex, N, N, n0, K, nullptr, sm, acc);
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = m0 + ty * 4 + i, n = n0 + tx * 4 + j;
            if (m < M && n < N) H[(size_t)m * N + n] = acc[i][j];
        }
}

// stage YZ: partial[zs][b * npx + a] = sum over this z range of e^{i qz z_j} sum_y Ey[b][y] H[j][y][a].
// qz in turns per unit length: qzt = qz / 2pi, so the phase of slice j is sincospi(2 frac(qzt z_j)) with the reduction in FP64.
__global__ void __launch_bounds__(256, 2) sep_stage_yz_kernel(const float2 *__restrict__ Ey, const float2 *__restrict__ H,
                                                           const double *__restrict__ qx, const double *__restrict__ qy,
                                                           double k, int npx, int npy, int ny, int nz, double dz, int nzs,
                                                           const unsigned char *__restrict__ flags, int nyc,
                                                           float2 *__restrict__ partial) {
    __shared__ TileSmem sm;
    const int m0 = blockIdx.y * kBM, n0 = blockIdx.x * kBN, zs = blockIdx.z;
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int z0 = (int)(((long long)nz * zs) / nzs), z1 = (int)(((long long)nz * (zs + 1)) / nzs);
    // qz of this thread's 4 x 4 outputs, in turns per unit length, parked in shared memory (32 FP64 registers otherwise)
    extern __shared__ double s_qzt_raw[];
    double (*s_qzt)[256] = (double (*)[256])s_qzt_raw;   // [16][256], dynamic: 32 KB
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int b = m0 + ty * 4 + i, a = n0 + tx * 4 + j;
            double v = 0.0;
            if (b < npy && a < npx) {
                const double qxy2 = qx[a] * qx[a] + qy[b] * qy[b];
                const double kz2 = k * k - qxy2;
                // qz = -(k - sqrt(k^2 - qxy^2)) = -qxy^2 / (k + sqrt(k^2 - qxy^2)): no cancellation near forward
                v = kz2 >= 0.0 ? -qxy2 / (k + sqrt(kz2)) : 0.0;
            }
            s_qzt[i * 4 + j][tid] = v * (0.5 / 3.14159265358979323846);
        }
    float2 tot[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) tot[i][j] = make_float2(0.f, 0.f);
    // One pipeline over the non-vacuum (slice, 16-y chunk) pairs of the z range, c = (jz - z0) * nyc + chunk: the operand
    // tiles of the next pair (possibly of the next slice) are in flight while the current one is multiplied; when the slice
    // changes, the finished slice's tile gets its phase and joins the total.
    const int ar = tid >> 2, ak = (tid & 3) * 4;     // loader roles as in tile_gemm
    const int bk = tid >> 4, bn = (tid & 15) * 4;
    const int nc = (z1 - z0) * nyc;
    const unsigned char *fl = flags + (size_t)z0 * nyc;
    auto next_pair = [&](int c) {
        while (c < nc && fl[c] == 0) ++c;
        return c;
    };
    float2 ra[4], rb[4];
    auto load = [&](int c) {
        const int jz = z0 + c / nyc, k0 = (c % nyc) * kBK;
        const float2 *Hj = H + (size_t)jz * ny * npx;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = m0 + ar, kk = k0 + ak + i;
            ra[i] = (m < npy && kk < ny) ? __ldg(Ey + (size_t)m * ny + kk) : make_float2(0.f, 0.f);
            const int kb = k0 + bk, n = n0 + bn + i;
            rb[i] = (kb < ny && n < npx) ? __ldg(Hj + (size_t)kb * npx + n) : make_float2(0.f, 0.f);
        }
    };
    float2 acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = make_float2(0.f, 0.f);
    auto fold = [&](int jz) {   // Blocks 7-8: tot += e^{i qz z_j} acc, acc = 0
        const double zj = centre_d(jz, nz, dz);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                double t = s_qzt[i * 4 + j][tid] * zj;
                t -= rint(t);
                float sn, cs;
                sincospif(2.0f * (float)t, &sn, &cs);
                tot[i][j].x = fmaf(cs, acc[i][j].x, tot[i][j].x);
                tot[i][j].x = fmaf(-sn, acc[i][j].y, tot[i][j].x);
                tot[i][j].y = fmaf(cs, acc[i][j].y, tot[i][j].y);
                tot[i][j].y = fmaf(sn, acc[i][j].x, tot[i][j].y);
                acc[i][j] = make_float2(0.f, 0.f);
            }
    };
    int c = next_pair(0);
    if (c < nc) load(c);
    while (c < nc) {
        __syncthreads();   // previous tile fully consumed
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            sm.As[ak + i][ar] = ra[i];
            sm.Bs[bk][bn + i] = rb[i];
        }
        __syncthreads();
        const int cn = next_pair(c + 1);
        if (cn < nc) load(cn);
#pragma unroll
        for (int kk = 0; kk < kBK; ++kk) {
            float2 av[4], bv[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                av[i] = sm.As[kk][ty * 4 + i];
                bv[i] = sm.Bs[kk][tx * 4 + i];
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    acc[i][j].x = fmaf(av[i].x, bv[j].x, acc[i][j].x);
                    acc[i][j].x = fmaf(-av[i].y, bv[j].y, acc[i][j].x);
                    acc[i][j].y = fmaf(av[i].x, bv[j].y, acc[i][j].y);
                    acc[i][j].y = fmaf(av[i].y, bv[j].x, acc[i][j].y);
                }
        }
        if (cn >= nc || cn / nyc != c / nyc) fold(z0 + c / nyc);   // last pair of its slice
        c = cn;
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int b = m0 + ty * 4 + i, a = n0 + tx * 4 + j;
            if (b < npy && a < npx) partial[(size_t)zs * npx * npy + (size_t)b * npx + a] = tot[i][j];
        }
}

// I[b][a] = |dV sum of partials|^2; evanescent grid points (qx^2 + qy^2 > k^2: no scattering direction) give 0
__global__ void sep_finalize_kernel(const float2 *__restrict__ partial, const double *__restrict__ qx,
                                    const double *__restrict__ qy, double k, int npx, int npy, int nzs, float dV,
                                    float *__restrict__ I) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= (int64_t)npx * npy) return;
    const int a = (int)(p % npx), b = (int)(p / npx);
    float re = 0.f, im = 0.f;
    for (int s = 0; s < nzs; ++s) {
        const float2 v = partial[(size_t)s * npx * npy + p];
        re += v.x;
        im += v.y;
    }
    re *= dV;
    im *= dV;
    const bool real = qx[a] * qx[a] + qy[b] * qy[b] <= k * k;
    I[p] = real ? re * re + im * im : 0.f;
}

// ------------------------------------------------------------------------------------------------ SIMT_TABLE (a7)
// The CUDA-core counterpart of the tensor contraction for the flat detector ("FP32 FMA against 1-D phase
// tables"): per slice the same G_j[p, x] = sum_y My[p, y] rho~_j[y, x] as an FP32 complex GEMM on 64-pixel x 64-x tiles, the
// row-dot with Mx[p, x], the slice phase Mz[p, j] and the slice sum in registers.  Tables are per-pixel FP32 roundings of
// FP64 phases.  Vacuum y chunks are skipped like in the separable route.
__global__ void pixel_table_kernel(const double *__restrict__ q, int comp, int64_t npix, int n, double d,
                                   float2 *__restrict__ out) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= npix * n) return;
    const int64_t p = t / n;
    const int i = (int)(t % n);
    double s, c;
    sincos(q[3 * p + comp] * centre_d(i, n, d), &s, &c);
    out[t] = make_float2((float)c, (float)s);
}

__global__ void __launch_bounds__(256) simt_table_kernel(const float2 *__restrict__ My, const float2 *__restrict__ Mx,
                                                         const float2 *__restrict__ Mz, const float2 *__restrict__ rho,
                                                         const unsigned char *__restrict__ flags, int64_t npix,
                                                         int64_t npix_pad, int nx, int ny, int nz, int nyc, int nsplit,
                                                         float2 *__restrict__ partial) {
    __shared__ TileSmem sm;
    const int64_t m0 = (int64_t)blockIdx.x * kBM;
    const int zs = blockIdx.y, b = blockIdx.z;
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const int z0 = (int)(((long long)nz * zs) / nsplit), z1 = (int)(((long long)nz * (zs + 1)) / nsplit);
    const float2 *vol = rho + (size_t)b * nx * ny * nz;
    const unsigned char *fl = flags + (size_t)b * nz * nyc;
    // tile_gemm addresses rows with int: shift the table pointers to this tile
    const float2 *My_t = My + (size_t)m0 * ny;
    const int rows = (int)((npix - m0) < kBM ? (npix - m0) : kBM);
    float2 tot[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) tot[i] = make_float2(0.f, 0.f);
    for (int j = z0; j < z1; ++j) {
        bool has = false;
        for (int c = 0; c < nyc; ++c) has |= fl[(size_t)j * nyc + c] != 0;
        if (!has) continue;   // vacuum slice (uniform over the block)
        float2 f[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) f[i] = make_float2(0.f, 0.f);
        for (int x0 = 0; x0 < nx; x0 += kBN) {
            float2 acc[4][4];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) acc[i][jj] = make_float2(0.f, 0.f);
            tile_gemm(My_t, ny, rows, 0, vol + (size_t)j * ny * nx, nx, nx, x0, ny, fl + (size_t)j * nyc, sm, acc);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int r = ty * 4 + i;
                if (r >= rows) continue;
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    const int x = x0 + tx * 4 + jj;
                    if (x >= nx) continue;
                    const float2 w = __ldg(Mx + (size_t)(m0 + r) * nx + x);
                    f[i].x = fmaf(acc[i][jj].x, w.x, f[i].x);
                    f[i].x = fmaf(-acc[i][jj].y, w.y, f[i].x);
                    f[i].y = fmaf(acc[i][jj].x, w.y, f[i].y);
                    f[i].y = fmaf(acc[i][jj].y, w.x, f[i].y);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
#pragma unroll
            for (int off = 8; off > 0; off >>= 1) {   // the 16 threads of a row group hold the 64 x of the tile
                f[i].x += __shfl_xor_sync(0xffffffffu, f[i].x, off, 16);
                f[i].y += __shfl_xor_sync(0xffffffffu, f[i].y, off, 16);
            }
            const int r = ty * 4 + i;
            if (r < rows) {
                const float2 w = __ldg(Mz + (size_t)(m0 + r) * nz + j);
                tot[i].x = fmaf(w.x, f[i].x, tot[i].x);
                tot[i].x = fmaf(-w.y, f[i].y, tot[i].x);
                tot[i].y = fmaf(w.x, f[i].y, tot[i].y);
                tot[i].y = fmaf(w.y, f[i].x, tot[i].y);
            }
        }
    }
    if (tx == 0)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int r = ty * 4 + i;
            if (r < rows) partial[((size_t)b * nsplit + zs) * npix_pad + m0 + r] = tot[i];
        }
}

cudaError_t launch_simt_table(const float *d_rho, const double *d_q, const Plan &p, float2 *d_My, float2 *d_Mx, float2 *d_Mz,
                              unsigned char *d_flags, float2 *d_partial, cudaStream_t st, int *nlaunch) {
    const int nyc = (p.ny + 15) / 16;
    const int64_t ey = p.npix * p.ny, ex = p.npix * p.nx, ez = p.npix * p.nz;
    pixel_table_kernel<<<(unsigned)((ey + 255) / 256), 256, 0, st>>>(d_q, 1, p.npix, p.ny, p.dy, d_My);
    pixel_table_kernel<<<(unsigned)((ex + 255) / 256), 256, 0, st>>>(d_q, 0, p.npix, p.nx, p.dx, d_Mx);
    pixel_table_kernel<<<(unsigned)((ez + 255) / 256), 256, 0, st>>>(d_q, 2, p.npix, p.nz, p.dz, d_Mz);
    for (int b = 0; b < p.batch; ++b)
        sep_rowflags_kernel<<<(unsigned)((p.nz * nyc + 7) / 8), 256, 0, st>>>((const float2 *)d_rho + (size_t)b * p.nvox, p.nx, p.ny,
                                                                            p.nz, nyc, d_flags + (size_t)b * p.nz * nyc);
    dim3 grid((unsigned)((p.npix + kBM - 1) / kBM), p.nsplit, p.batch);
    simt_table_kernel<<<grid, 256, 0, st>>>(d_My, d_Mx, d_Mz, (const float2 *)d_rho, d_flags, p.npix, p.npix_pad, p.nx, p.ny, p.nz,
                                            nyc, p.nsplit, d_partial);
    if (nlaunch) *nlaunch += 4 + p.batch;
    return cudaGetLastError();
}

cudaError_t launch_sep_tables(const double *d_qx, int npx, const double *d_qy, int npy, const Plan &p, float2 *d_Ex,
                              float2 *d_Ey, cudaStream_t st) {
    const int64_t nxe = (int64_t)npx * p.nx, nye = (int64_t)npy * p.ny;
    sep_table_kernel<<<(unsigned)((nxe + 255) / 256), 256, 0, st>>>(d_qx, npx, p.nx, p.dx, 0, d_Ex);   // Ex[x][a]
    sep_table_kernel<<<(unsigned)((nye + 255) / 256), 256, 0, st>>>(d_qy, npy, p.ny, p.dy, 1, d_Ey);   // Ey[b][y]
    return cudaGetLastError();
}

int sep_zsplit(const Plan &p, int npx, int npy, int num_sms) {
    const int tiles = ((npx + kBN - 1) / kBN) * ((npy + kBM - 1) / kBM);
    int nzs = (2 * num_sms + tiles - 1) / tiles;
    if (nzs > p.nz) nzs = p.nz;
    if (nzs > 64) nzs = 64;
    return nzs < 1 ? 1 : nzs;
}

cudaError_t sep_init_device() {   // per device (scatman_create)
    return cudaFuncSetAttribute(sep_stage_yz_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * 256 * 8);
}

// one batch item: rho (FP32 complex [nz][ny][nx], without dV) -> I[npy][npx]
cudaError_t launch_sep_item(const float2 *d_rho, const Plan &p, const float2 *d_Ex, const float2 *d_Ey, const double *d_qx,
                            int npx, const double *d_qy, int npy, int nzs, float2 *d_H, unsigned char *d_flags,
                            float2 *d_partial, float *d_I, cudaStream_t st) {
    const int M = p.nz * p.ny;
    const int nyc = (p.ny + 15) / 16;
    const double k = 2.0 * 3.14159265358979323846 / p.lambda;
    sep_rowflags_kernel<<<(unsigned)((p.nz * nyc + 7) / 8), 256, 0, st>>>(d_rho, p.nx, p.ny, p.nz, nyc, d_flags);
    dim3 gx((M + kBM - 1) / kBM, (npx + kBN - 1) / kBN);
    sep_stage_x_kernel<<<gx, 256, 0, st>>>(d_rho, d_Ex, M, p.nx, npx, p.ny % 16 == 0 ? d_flags : nullptr, d_H);
    dim3 gy((npx + kBN - 1) / kBN, (npy + kBM - 1) / kBM, nzs);
    sep_stage_yz_kernel<<<gy, 256, 16 * 256 * 8, st>>>(d_Ey, d_H, d_qx, d_qy, k, npx, npy, p.ny, p.nz, p.dz, nzs, d_flags, nyc,
                                            d_partial);
    const int64_t npix = (int64_t)npx * npy;
    sep_finalize_kernel<<<(unsigned)((npix + 255) / 256), 256, 0, st>>>(d_partial, d_qx, d_qy, k, npx, npy, nzs,
                                                                        (float)(p.dx * p.dy * p.dz), d_I);
    return cudaGetLastError();
}

}  // namespace scatman
