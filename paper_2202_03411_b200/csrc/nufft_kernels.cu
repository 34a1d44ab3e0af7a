// nufft_kernels.cu -- flat-detector route by a 3-D type-2 non-uniform Fourier transform (second half).
//
// The pattern is still A(p) = sum_r rho~(r) e^{i q(p).r} at every pixel's Ewald-sphere q (Eq. 2/4), but the pixel x voxel
// contraction is replaced by
//   (1) a SEPARABLE transform of rho~ onto a small uniform (g_z, g_y, g_x) grid that covers the q's of the detector with a margin,
//       U[mz][my][mx] = sum_r c_z c_y c_x rho~(r) e^{i g_m . r}     -- three complex GEMMs (stage Z over slices, X over columns, Y over rows)
//   (2) an interpolation from that grid to each pixel with a Kaiser-Bessel window of W = 8 grid cells per axis,
//       A(p) = sum_{m near q(p)/h} phi(u_z - m_z) phi(u_y - m_y) phi(u_x - m_x) U[m],   u = q / h.
// Grid spacing h_d = 2 pi / (2 N_d d_d) (oversampling 2), pre-correction c_i = 1 / Phi(h x_i) with Phi the window's Fourier transform:
//   sum_m phi(u - m) e^{i m t} = sum_l Phi(t - 2 pi l) e^{i u (t - 2 pi l)}   (Poisson summation),   |t| = |h x_i| < pi / 2,
// so the l = 0 term is the wanted e^{i u t} and the l = +-1 aliases are below 2.4e-7 of it for W = 8, beta = pi sqrt(W^2 (3/4)^2 - 0.8).
// All sums, tables and window weights are FP64 on the CUDA cores (the work is ~3000x smaller than the pixel contraction: 1.2e9 complex MACs for
// 256^3 on 512^2 pixels against 4.4e12); only U is stored FP32 for the interpolation (see nufft_interp_kernel).  The only approximation beyond
// rounding is the window's, and the result meets the same tolerances against the oracle's direct sum (tests/test_gpu_nufft.py).
// Kernels: nufft_table_kernel (phase tables with the window correction folded in), nufft_zgemm_kernel (the three GEMM stages),
// nufft_interp_kernel<P> (P = 4, 3, 2, 1 pixels per thread); nufft_init_device fits the window's per-cell polynomials (host) once per device.
#include "internal.h"

namespace scatman {

double nufft_inv_i0_beta();

namespace {

constexpr int kW = kNufftW;                 // window width in grid cells
constexpr double kHalfW = 0.5 * kW;
constexpr double kPi = 3.14159265358979323846;

__host__ __device__ inline double kb_beta() { return kPi * sqrt(kHalfW * kHalfW * 2.25 - 0.8); }

// ---- tables: T[m][i] = c_i e^{i g_m x_i}, g_m x_i = pi (m_lo + m)(2 i - N + 1) / nf (exact integer phase), c_i = 1 / Phi(h x_i).
// transposed = 0: T[m][i] (A operand, K = i contiguous); 1: T[i][m] (B operand, N = m contiguous).
__global__ void nufft_table_kernel(int N, int nq, int m_lo, int transposed, double inv_i0b, double2 *__restrict__ T) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (int64_t)N * nq) return;
    int m, i;
    if (transposed) { m = (int)(e % nq); i = (int)(e / nq); } else { i = (int)(e % N); m = (int)(e / N); }
    const int nf = 2 * N;
    const int64_t c2 = 2 * i - N + 1;                       // 2 x_i / d
    int64_t t = ((int64_t)(m_lo + m) * c2) % (2 * (int64_t)nf);   // phase = pi t / nf, reduced exactly
    double s, c;
    sincospi((double)t / (double)nf, &s, &c);
    const double beta = kb_beta();
    const double theta = kPi * (double)c2 / (double)nf;     // h x_i in radians per grid cell, |theta| < pi / 2
    const double r = sqrt(beta * beta - kHalfW * kHalfW * theta * theta);
    const double Phi = 2.0 * kHalfW * sinh(r) / r * inv_i0b;
    const double corr = 1.0 / Phi;
    T[e] = make_double2(corr * c, corr * s);
}

// ---- complex FP64 GEMM: C[b] (M x N) = A[b] (M x K, K contiguous) * B[b] (K x N, N contiguous); 64 x 64 tiles, K steps of 16,
// 256 threads x (4 x 4) outputs at rows ty + 16 i, columns tx + 16 j (conflict-free 16-byte shared-memory reads).
constexpr int BN = 64, BK = 16;

__device__ inline double2 ld_c(const double2 *p) { return __ldg(p); }
__device__ inline double2 ld_c(const float2 *p) { const float2 v = __ldg(p); return make_double2((double)v.x, (double)v.y); }

// RM = rows per thread: the row tile is BM = 16 RM (32, 48 or 64), picked per GEMM (zgemm below).  Shared memory is double-buffered, so a
// K step costs ONE barrier: the tile of step s + 1 goes into the other buffer while slower warps still read step s.
// A K step whose streamed tile is all zero (vacuum: rho~, and the planes and rows made from it, are exact zeros outside the particle) adds
// nothing: the barrier doubles as a block-wide OR over "my part of the tile holds a non-zero", and the arithmetic is skipped.  ZERO_IN_A
// says which operand can be vacuum (stage X: the P planes are A; stages Z and Y: rho~ / H are B); the other one is a phase table.
__device__ inline void st_c(double2 *p, double2 v) { *p = v; }
__device__ inline void st_c(float2 *p, double2 v) { *p = make_float2((float)v.x, (float)v.y); }

template <typename TA, typename TB, typename TC, int RM, bool ZERO_IN_A>
__global__ void __launch_bounds__(256, RM <= 3 ? 2 : 1)
nufft_zgemm_kernel(const TA *__restrict__ A, const TB *__restrict__ B, TC *__restrict__ C, int M, int N, int K,
                   int64_t lda, int64_t ldb, int64_t ldc, int64_t strideA, int64_t strideB, int64_t strideC) {
    constexpr int BM = 16 * RM;
    extern __shared__ double2 zg_smem[];
    double2 (*As)[BK][BM + 1] = reinterpret_cast<double2 (*)[BK][BM + 1]>(zg_smem);                          // [2][BK][BM + 1]
    double2 (*Bs)[BK][BN] = reinterpret_cast<double2 (*)[BK][BN]>(zg_smem + 2 * BK * (BM + 1));              // [2][BK][BN]
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int n0 = blockIdx.x * BN, m0 = blockIdx.y * BM;
    A += (int64_t)blockIdx.z * strideA;
    B += (int64_t)blockIdx.z * strideB;
    C += (int64_t)blockIdx.z * strideC;
    double2 acc[RM][4];
#pragma unroll
    for (int i = 0; i < RM; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = make_double2(0.0, 0.0);
    double2 ra[RM], rb[4];
    auto fetch = [&](int k0) {
#pragma unroll
        for (int r = 0; r < RM; ++r) {
            const int idx = t + 256 * r;
            const int ak = idx & 15, am = idx >> 4;
            ra[r] = (m0 + am < M && k0 + ak < K) ? ld_c(A + (int64_t)(m0 + am) * lda + (k0 + ak)) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = t + 256 * r;
            const int bn = idx & 63, bk = idx >> 6;
            rb[r] = (n0 + bn < N && k0 + bk < K) ? ld_c(B + (int64_t)(k0 + bk) * ldb + (n0 + bn)) : make_double2(0.0, 0.0);
        }
    };
    fetch(0);
    int buf = 0;
    for (int k0 = 0; k0 < K; k0 += BK, buf ^= 1) {
        bool nz = false;
#pragma unroll
        for (int r = 0; r < RM; ++r) {
            const int idx = t + 256 * r;
            As[buf][idx & 15][idx >> 4] = ra[r];
            if (ZERO_IN_A) nz |= ra[r].x != 0.0 || ra[r].y != 0.0;
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = t + 256 * r;
            Bs[buf][idx >> 6][idx & 63] = rb[r];
            if (!ZERO_IN_A) nz |= rb[r].x != 0.0 || rb[r].y != 0.0;
        }
        const bool live = __syncthreads_or(nz) != 0;
        if (k0 + BK < K) fetch(k0 + BK);
        if (!live) continue;
#pragma unroll
        for (int k = 0; k < BK; ++k) {
            double2 a[RM], b[4];
#pragma unroll
            for (int i = 0; i < RM; ++i) a[i] = As[buf][k][ty + 16 * i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Bs[buf][k][tx + 16 * j];
#pragma unroll
            for (int i = 0; i < RM; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    acc[i][j].x = fma(a[i].x, b[j].x, acc[i][j].x);
                    acc[i][j].x = fma(-a[i].y, b[j].y, acc[i][j].x);
                    acc[i][j].y = fma(a[i].x, b[j].y, acc[i][j].y);
                    acc[i][j].y = fma(a[i].y, b[j].x, acc[i][j].y);
                }
        }
    }
#pragma unroll
    for (int i = 0; i < RM; ++i) {
        const int m = m0 + ty + 16 * i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = n0 + tx + 16 * j;
            if (n < N) st_c(C + (int64_t)m * ldc + n, acc[i][j]);
        }
    }
}

template <typename TA, typename TB, typename TC, int RM, bool ZERO_IN_A>
cudaError_t zgemm_rm(const TA *A, const TB *B, TC *C, int M, int N, int K, int64_t lda, int64_t ldb, int64_t ldc, int nbatch,
                     int64_t sA, int64_t sB, int64_t sC, cudaStream_t st) {
    constexpr int BM = 16 * RM;
    constexpr size_t smem = sizeof(double2) * 2 * BK * ((BM + 1) + BN);
    // (the dynamic shared-memory limit of every instantiation is raised once per device, nufft_init_device)
    // grid.y carries the row tiles (<= 65535), grid.z the batch (<= 65535, the callers' concern)
    for (int64_t m_base = 0; m_base < M; m_base += 65535LL * BM) {
        const int rows = (int)(M - m_base < 65535LL * BM ? M - m_base : 65535LL * BM);
        dim3 grid((N + BN - 1) / BN, (rows + BM - 1) / BM, nbatch);
        nufft_zgemm_kernel<TA, TB, TC, RM, ZERO_IN_A><<<grid, 256, smem, st>>>(A + m_base * lda, B, C + m_base * ldc, rows, N, K, lda, ldb, ldc,
                                                                          sA, sB, sC);
    }
    return cudaGetLastError();
}

template <typename TA, typename TB, typename TC, bool ZERO_IN_A>
cudaError_t zgemm(const TA *A, const TB *B, TC *C, int M, int N, int K, int64_t lda, int64_t ldb, int64_t ldc, int nbatch,
                  int64_t sA, int64_t sB, int64_t sC, cudaStream_t st) {
    // Row tile by a makespan estimate: resident sets of 148 x (2 CTAs of RM <= 3, or 1 of RM = 4) run one after the other and a
    // set takes ~ CTAs per SM x RM; ties go to the least padding, then to the taller tile.
    auto cost = [&](int rm) {
        const int64_t tiles = (int64_t)((M + 16 * rm - 1) / (16 * rm)) * ((N + BN - 1) / BN) * nbatch;
        const int cps = rm <= 3 ? 2 : 1;
        const int64_t sets = (tiles + 148 * cps - 1) / (148 * cps);
        return sets * cps * rm * 1000000 + (int64_t)((M + 16 * rm - 1) / (16 * rm)) * 16 * rm % 1000000 * 10 + (4 - rm);
    };
    const int64_t c2 = cost(2), c3 = cost(3), c4 = cost(4);
    if (c4 <= c3 && c4 <= c2) return zgemm_rm<TA, TB, TC, 4, ZERO_IN_A>(A, B, C, M, N, K, lda, ldb, ldc, nbatch, sA, sB, sC, st);
    if (c3 <= c2) return zgemm_rm<TA, TB, TC, 3, ZERO_IN_A>(A, B, C, M, N, K, lda, ldb, ldc, nbatch, sA, sB, sC, st);
    return zgemm_rm<TA, TB, TC, 2, ZERO_IN_A>(A, B, C, M, N, K, lda, ldb, ldc, nbatch, sA, sB, sC, st);
}

// ---- interpolation: A = sum over the W^3 nearest grid points, I = |A dV|^2 (Block 11).
// U is stored FP32 (the last GEMM stage rounds its accumulators on the way out): the window's weights are positive and A varies slowly
// over the window, so a value's 6e-8 relative rounding stays relative to the LOCAL amplitude (unlike an error made before the
// transforms, which would be relative to the whole particle).  The sums over x and y are FP32 (packed fma.rn.f32x2: (Re, Im) times a
// real weight), the sum over z and the intensity FP64; the weights are evaluated in FP64.
// A thread owns P = 2 (or 1) pixels that are neighbours along y: their windows overlap (a pixel is a fraction of a grid cell wide), so
// the thread walks ONE common window (W + 1 cells along x, W + 2 along y and z), loads every grid value once and applies it to both
// pixels with per-pixel weights (zero outside a pixel's own support) -- the kernel is bound by the shared-memory wavefronts of
// those loads.  A pair whose windows do not fit the common one (pixels more than a cell apart: coarse detectors) takes its pixels
// one by one.  Window weights of the y and z axes live in shared memory ([axis][pixel][cell][thread]).
// The window phi(s) = I0(beta sqrt(1 - (s / (W/2))^2)) / I0(beta) is entire in s^2, so on each of its W unit cells it is a polynomial
// to 2e-13 at degree 11 (Chebyshev fit on the host, nufft_init_device): the W weights of a point come from W Horner evaluations at
// the one offset t = m0 - (u - W/2) in [0, 1), weight of cell m0 + c = phi(W/2 - c - t) = sum_k c_kb[c][k] (2 t - 1)^k.
constexpr int kDeg = 11;
__constant__ double c_kb[kW][kDeg + 1];

__device__ inline void kb_weights(double u, int m0, double (&w)[kW]) {
    const double x = 2.0 * ((double)m0 - (u - kHalfW)) - 1.0;
#pragma unroll
    for (int c = 0; c < kW; ++c) {
        double v = c_kb[c][kDeg];
#pragma unroll
        for (int k = kDeg - 1; k >= 0; --k) v = fma(v, x, c_kb[c][k]);
        w[c] = v;
    }
}

// own[0..W) placed at cells shift..shift+W of a KU-cell window, zero elsewhere (static indices: selects, no local memory)
template <int KU>
__device__ inline double placed(const double (&own)[kW], int shift, int a) {
    double v = 0.0;
#pragma unroll
    for (int s = 0; s <= KU - kW; ++s)
        if (shift == s && a - s >= 0 && a - s < kW) v = own[a - s < 0 ? 0 : (a - s >= kW ? kW - 1 : a - s)];
    return v;
}

constexpr int kInterpThreads = 128;
constexpr int kTX = 16, kTY = 8;         // a block = 16 pixels along a detector row x 8 groups of P rows
constexpr int kTileCap = 3968;           // float2 elements of shared memory for the block's window of U (31 KB: with the 24 KB of weights
                                         // and the 1 KB the driver reserves per block, four blocks fit an SM)

// A block owns a TILE of 8 P x 8 pixels.  Its pixels' windows overlap heavily, so the block first copies the box of U that covers
// all of them into shared memory (coalesced, every thread loading: the whole box is in flight at once) and the per-thread sums
// then read shared memory -- the earlier version read U through L1 from a loop whose every iteration waited for an L2 round
// trip, with one wave of 8-12 warps per SM to hide it.  A tile whose box exceeds kTileCap (coarse detectors, where neighbouring
// pixels are cells apart) reads U from global memory as before.
template <int P>
__global__ void __launch_bounds__(kInterpThreads)
nufft_interp_kernel(const double *__restrict__ q, int npx, int npy, NufftAxis ax, NufftAxis ay, NufftAxis az,
                    const float2 *__restrict__ U, int64_t strideU, double dV, const float *__restrict__ ampscale,
                    float *__restrict__ I) {
    constexpr int KU = P > 1 ? kW + 2 : kW;              // common window along y, z: the thread's pixels are up to 1.9 cells apart
    constexpr int KX = P > 1 ? kW + 1 : kW;              // ... along x: neighbours along y sit at nearly the same q_x (< 1 cell apart)
    extern __shared__ float wsm[];                        // [2][P][KU][kInterpThreads] y and z weights (FP32), then the tile of U
    float2 *tile = reinterpret_cast<float2 *>(wsm + 2 * P * KU * kInterpThreads);
    __shared__ int red[8];                                // lo[3], hi[3], every thread's pixels share a window, any valid thread
    // A thread's P pixels are neighbours along y (same column ix), a half-warp = 16 consecutive ix of one row group: at the usual
    // pixel spacing (< 1 grid cell) its 16 lanes then read one run of <= 16 cells of a tile row per load -- one shared-memory
    // wavefront.  (P pixels along x and 8 x 4 thread groups per warp cost 3 wavefronts per load: the kernel's limit.)
    const int ngy = (npy + P - 1) / P;
    const int tiles_x = (npx + kTX - 1) / kTX;
    const int ix = (blockIdx.x % tiles_x) * kTX + (threadIdx.x % kTX), gy = (blockIdx.x / tiles_x) * kTY + threadIdx.x / kTX;
    const bool valid = ix < npx && gy < ngy;
    const int iy0 = gy * P;
    const int64_t p0 = (int64_t)iy0 * npx + ix;     // pixel j of the thread: p0 + j npx
    const int64_t npix = (int64_t)npx * npy;
    U += (int64_t)blockIdx.y * strideU;
    I += (int64_t)blockIdx.y * npix;
    if (ampscale) dV *= (double)__ldg(ampscale + blockIdx.y);   // tensor-core stages: U carries the item's operand scales
    const int np = valid ? (npy - iy0 < P ? npy - iy0 : P) : 0;
    double u[P][3];
    int m0[P][3], base[3], top[3];
    if (threadIdx.x == 0) {
        red[0] = red[1] = red[2] = 0x7fffffff;
        red[3] = red[4] = red[5] = -0x7fffffff;
        red[6] = 1;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int64_t p = valid ? p0 + (int64_t)(j < np ? j : 0) * npx : 0;     // threads past the detector's edge look at pixel 0 and stay out of the sums
        u[j][0] = q[3 * p + 0] * ax.inv_h; u[j][1] = q[3 * p + 1] * ay.inv_h; u[j][2] = q[3 * p + 2] * az.inv_h;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            m0[j][d] = (int)ceil(u[j][d] - kHalfW);
            base[d] = j == 0 ? m0[j][d] : min(base[d], m0[j][d]);
            top[d] = j == 0 ? m0[j][d] : max(top[d], m0[j][d]);
        }
    }
    const bool common = valid && top[0] - base[0] + kW <= KX && top[1] - base[1] + kW <= KU && top[2] - base[2] + kW <= KU;
    if (valid) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            atomicMin(&red[d], base[d]);
            // last cell the thread reads: along x every row is read over the whole common window of KX cells; along y and z
            // rows and planes whose weights are all zero are skipped, so only the pixels' own windows count
            atomicMax(&red[3 + d], d == 0 ? base[d] + KX - 1 : top[d] + kW - 1);
        }
        if (!common) atomicAnd(&red[6], 0);
    }
    __syncthreads();
    const int lo0 = red[0], lo1 = red[1], lo2 = red[2];
    const int e0 = red[3] - lo0 + 1, e1 = red[4] - lo1 + 1, e2 = red[5] - lo2 + 1;
    // the box must also lie inside the uniform grid (a thread's common window can reach 2 cells past its pixels' own windows)
    const bool tiled = red[6] != 0 && red[3] >= lo0 && (int64_t)e0 * e1 * e2 <= kTileCap && lo0 - ax.m_lo >= 0 && lo1 - ay.m_lo >= 0 &&
                       lo2 - az.m_lo >= 0 && red[3] - ax.m_lo < ax.nq && red[4] - ay.m_lo < ay.nq && red[5] - az.m_lo < az.nq;
    if (tiled) {
        const int rows = e1 * e2;
        for (int e = threadIdx.x; e < rows * e0; e += kInterpThreads) {
            const int x = e % e0, yz = e / e0;
            const int y = yz % e1, z = yz / e1;
            tile[e] = __ldg(U + ((int64_t)(lo2 - az.m_lo + z) * ay.nq + (lo1 - ay.m_lo + y)) * ax.nq + (lo0 - ax.m_lo + x));
        }
        __syncthreads();
    }
    if (!valid) return;
    auto wy = [&](int j, int b) -> float & { return wsm[((0 * P + j) * KU + b) * kInterpThreads + threadIdx.x]; };
    auto wz = [&](int j, int c) -> float & { return wsm[((1 * P + j) * KU + c) * kInterpThreads + threadIdx.x]; };
    if (common) {
        // The x weights and the row sums over x are FP32: a row sum of <= 9 terms of one sign pattern rounds at ~1e-7 of its own
        // magnitude, the same size as the FP32 rounding U already carries.
        // kept as (w, w) pairs: one packed fma.rn.f32x2 (sm_100) multiplies a grid value's (Re, Im) by the real weight
        float2 wx[P][KX];
#pragma unroll
        for (int j = 0; j < P; ++j) {
            double own[kW];
            kb_weights(u[j][0], m0[j][0], own);
#pragma unroll
            for (int a = 0; a < KX; ++a) {
                const float w = (float)placed<KX>(own, m0[j][0] - base[0], a);
                wx[j][a] = make_float2(w, w);
            }
            kb_weights(u[j][1], m0[j][1], own);
#pragma unroll
            for (int a = 0; a < KU; ++a) wy(j, a) = (float)placed<KU>(own, m0[j][1] - base[1], a);
            kb_weights(u[j][2], m0[j][2], own);
#pragma unroll
            for (int a = 0; a < KU; ++a) wz(j, a) = (float)placed<KU>(own, m0[j][2] - base[2], a);
        }
        // The window's rows: FP32 over x (above) and over y -- eight more roundings of 6e-8 each on sums of one plane, the size of the
        // rounding U already carries -- FP64 over z and for the intensity.  Called once with a pointer into the tile and once with one
        // into U, so that each copy of the loop uses its own address space (shared loads for the tile, not generic ones).
        double are[P], aim[P];
#pragma unroll
        for (int j = 0; j < P; ++j) are[j] = aim[j] = 0.0;
        auto walk = [&](const float2 *__restrict__ win, int sy, int sz) {   // strides < 2^31: a plane of the grid is a few 10^5 points
            for (int c = 0; c < KU; ++c) {
                float wzc[P];
                bool any = false;
#pragma unroll
                for (int j = 0; j < P; ++j) { wzc[j] = wz(j, c); any |= wzc[j] != 0.f; }
                if (!any) continue;
                float2 pl[P];
#pragma unroll
                for (int j = 0; j < P; ++j) pl[j] = make_float2(0.f, 0.f);
                for (int b = 0; b < KU; ++b) {
                    float wyb[P];
                    bool anyb = false;
#pragma unroll
                    for (int j = 0; j < P; ++j) { wyb[j] = wy(j, b); anyb |= wyb[j] != 0.f; }
                    if (!anyb) continue;
                    const float2 *row = win + c * sz + b * sy;
                    float2 v[KX];
#pragma unroll
                    for (int a = 0; a < KX; ++a) v[a] = row[a];
#pragma unroll
                    for (int j = 0; j < P; ++j) {
                        float2 ra = make_float2(0.f, 0.f), rb = make_float2(0.f, 0.f);   // two chains per pixel
#pragma unroll
                        for (int a = 0; a < KX; ++a) {
                            if (a & 1) rb = __ffma2_rn(wx[j][a], v[a], rb);
                            else ra = __ffma2_rn(wx[j][a], v[a], ra);
                        }
                        const float2 w2 = make_float2(wyb[j], wyb[j]);
                        pl[j] = __ffma2_rn(w2, ra, __ffma2_rn(w2, rb, pl[j]));
                    }
                }
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    are[j] = fma((double)wzc[j], (double)pl[j].x, are[j]);
                    aim[j] = fma((double)wzc[j], (double)pl[j].y, aim[j]);
                }
            }
        };
        if (tiled) walk(tile + ((base[2] - lo2) * e1 + (base[1] - lo1)) * e0 + (base[0] - lo0), e0, e0 * e1);
        else   // inside the grid by the plan's margins
            walk(U + ((int64_t)(base[2] - az.m_lo) * ay.nq + (base[1] - ay.m_lo)) * ax.nq + (base[0] - ax.m_lo), ax.nq, ax.nq * ay.nq);
#pragma unroll
        for (int j = 0; j < P; ++j)
            if (j < np) {
                const double re = are[j] * dV, im = aim[j] * dV;
                I[p0 + (int64_t)j * npx] = (float)(re * re + im * im);
            }
        return;
    }
    // pixels one by one, each with its own W-cell window
#pragma unroll
    for (int j = 0; j < P; ++j) {
        if (j >= np) break;
        double own[kW];
        float wx1[kW];
        kb_weights(u[j][0], m0[j][0], own);
#pragma unroll
        for (int a = 0; a < kW; ++a) wx1[a] = (float)own[a];
        kb_weights(u[j][1], m0[j][1], own);
#pragma unroll
        for (int a = 0; a < kW; ++a) wy(0, a) = (float)own[a];
        kb_weights(u[j][2], m0[j][2], own);
#pragma unroll
        for (int a = 0; a < kW; ++a) wz(0, a) = (float)own[a];
        const int ix = m0[j][0] - ax.m_lo, iyq = m0[j][1] - ay.m_lo, iz = m0[j][2] - az.m_lo;
        double are = 0.0, aim = 0.0;
        for (int c = 0; c < kW; ++c) {
            double pre = 0.0, pim = 0.0;
            for (int b = 0; b < kW; ++b) {
                const float2 *row = U + ((int64_t)(iz + c) * ay.nq + (iyq + b)) * ax.nq + ix;
                float rre = 0.f, rim = 0.f;
#pragma unroll
                for (int a = 0; a < kW; ++a) {
                    const float2 v = __ldg(row + a);
                    rre = fmaf(wx1[a], v.x, rre);
                    rim = fmaf(wx1[a], v.y, rim);
                }
                pre = fma((double)wy(0, b), (double)rre, pre);
                pim = fma((double)wy(0, b), (double)rim, pim);
            }
            are = fma((double)wz(0, c), pre, are);
            aim = fma((double)wz(0, c), pim, aim);
        }
        are *= dV;
        aim *= dV;
        I[p0 + (int64_t)j * npx] = (float)(are * are + aim * aim);
    }
}

template <int P>
cudaError_t launch_interp(const double *d_q, int npx, int npy, const NufftPlan &n, const float2 *d_U, int64_t strideU, int nb,
                          double dV, const float *d_ampscale, float *d_I, cudaStream_t st) {
    constexpr int KU = P > 1 ? kW + 2 : kW;
    const size_t smem = sizeof(float) * 2 * P * KU * kInterpThreads + sizeof(float2) * kTileCap;
    const int64_t tiles = (int64_t)((npx + kTX - 1) / kTX) * (((npy + P - 1) / P + kTY - 1) / kTY);
    dim3 grid((unsigned)tiles, nb);
    nufft_interp_kernel<P><<<grid, kInterpThreads, smem, st>>>(d_q, npx, npy, n.ax, n.ay, n.az, d_U, strideU, dV, d_ampscale, d_I);
    return cudaGetLastError();
}

}  // namespace

double nufft_inv_i0_beta() {
    // 1 / I0(beta) by the power series (host; one number handed to the kernels)
    const double beta = kb_beta();
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 200; ++k) {
        term *= (beta * 0.5 / k) * (beta * 0.5 / k);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    return 1.0 / sum;
}

// Chebyshev fit of the window on each unit cell (degree kDeg, nodes cos(pi (k + 1/2) / n)), rewritten in powers of x = 2 t - 1.
cudaError_t nufft_init_device() {
    static double coef[kW][kDeg + 1];
    static bool fitted = false;
    if (!fitted) {
        const double beta = kb_beta(), inv_i0b = nufft_inv_i0_beta();
        auto i0 = [](double x) {
            double term = 1.0, sum = 1.0;
            for (int k = 1; k < 300; ++k) {
                term *= (x * 0.5 / k) * (x * 0.5 / k);
                sum += term;
                if (term < 1e-18 * sum) break;
            }
            return sum;
        };
        constexpr int n = kDeg + 1;
        for (int c = 0; c < kW; ++c) {
            double f[n], cheb[n];
            for (int k = 0; k < n; ++k) {
                const double x = cos(kPi * (k + 0.5) / n);
                const double s = kHalfW - c - 0.5 * (x + 1.0);
                const double a = 1.0 - (s / kHalfW) * (s / kHalfW);
                f[k] = i0(beta * sqrt(a > 0.0 ? a : 0.0)) * inv_i0b;
            }
            for (int j = 0; j < n; ++j) {
                double acc = 0.0;
                for (int k = 0; k < n; ++k) acc += f[k] * cos(j * kPi * (k + 0.5) / n);
                cheb[j] = (j == 0 ? 1.0 : 2.0) / n * acc;
            }
            // sum_j cheb[j] T_j(x) in the monomial basis: T_0 = 1, T_1 = x, T_{j+1} = 2 x T_j - T_{j-1}
            double t0[n] = {1.0}, t1[n] = {0.0, 1.0}, mono[n] = {0.0};
            for (int k = 0; k < n; ++k) mono[k] = cheb[0] * t0[k] + (n > 1 ? cheb[1] * t1[k] : 0.0);
            for (int j = 2; j < n; ++j) {
                double t2[n];
                for (int k = 0; k < n; ++k) t2[k] = (k > 0 ? 2.0 * t1[k - 1] : 0.0) - t0[k];
                for (int k = 0; k < n; ++k) { mono[k] += cheb[j] * t2[k]; t0[k] = t1[k]; t1[k] = t2[k]; }
            }
            for (int k = 0; k < n; ++k) coef[c][k] = mono[k];
        }
        fitted = true;
    }
    cudaError_t e = cudaMemcpyToSymbol(c_kb, coef, sizeof(coef));
    auto smem_gemm = [](int rm) { return (int)(sizeof(double2) * 2 * BK * ((16 * rm + 1) + BN)); };
    auto smem_interp = [](int P) { return (int)(sizeof(float) * 2 * P * (P > 1 ? kW + 2 : kW) * kInterpThreads + sizeof(float2) * kTileCap); };
    const cudaFuncAttribute attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
#define SCATMAN_ZGEMM_ATTR(RM)                                                                                          \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(nufft_zgemm_kernel<double2, float2, double2, RM, false>, attr, smem_gemm(RM));   \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(nufft_zgemm_kernel<double2, double2, double2, RM, true>, attr, smem_gemm(RM));   \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(nufft_zgemm_kernel<double2, double2, float2, RM, false>, attr, smem_gemm(RM));
    SCATMAN_ZGEMM_ATTR(2)
    SCATMAN_ZGEMM_ATTR(3)
    SCATMAN_ZGEMM_ATTR(4)
#undef SCATMAN_ZGEMM_ATTR
    if (e == cudaSuccess) e = cudaFuncSetAttribute(nufft_interp_kernel<1>, attr, smem_interp(1));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(nufft_interp_kernel<2>, attr, smem_interp(2));
    return e;
}

cudaError_t launch_nufft_tables(const Plan &p, const NufftPlan &n, double2 *d_Tz, double2 *d_TxT, double2 *d_Ty, cudaStream_t st) {
    const double inv_i0b = nufft_inv_i0_beta();
    int64_t e = (int64_t)p.nz * n.az.nq;
    nufft_table_kernel<<<(unsigned)((e + 255) / 256), 256, 0, st>>>(p.nz, n.az.nq, n.az.m_lo, 0, inv_i0b, d_Tz);
    e = (int64_t)p.nx * n.ax.nq;
    nufft_table_kernel<<<(unsigned)((e + 255) / 256), 256, 0, st>>>(p.nx, n.ax.nq, n.ax.m_lo, 1, inv_i0b, d_TxT);
    e = (int64_t)p.ny * n.ay.nq;
    nufft_table_kernel<<<(unsigned)((e + 255) / 256), 256, 0, st>>>(p.ny, n.ay.nq, n.ay.m_lo, 0, inv_i0b, d_Ty);
    return cudaGetLastError();
}

// A chunk of nb batch items: rho~ [nb][nz][ny][nx] -> P [nb][nqz][ny][nx] -> H [nb][nqz][ny][nqx] -> U [nb][nqz][nqy][nqx] -> I [nb][npix].
// pixel_cells = the widest step between neighbouring pixels of a row, in grid cells of any axis (picks the pixels per thread).
cudaError_t launch_nufft_chunk(const float2 *d_rho, const Plan &p, const NufftPlan &n, int nb, int npx, int npy, double pixel_cells,
                               const double2 *d_Tz, const double2 *d_TxT, const double2 *d_Ty, const double *d_q, double2 *d_P,
                               double2 *d_H, float2 *d_U, float *d_I, cudaStream_t st) {
    const int64_t nyx = (int64_t)p.ny * p.nx;
    cudaError_t e = cudaSuccess;
    // stage Z, one GEMM per item: P_b (nqz x ny nx) = Tz (nqz x nz) * rho~_b (nz x ny nx)
    e = zgemm<double2, float2, double2, false>(d_Tz, d_rho, d_P, n.az.nq, (int)nyx, p.nz, p.nz, nyx, nyx, nb, 0, (int64_t)p.nz * nyx,
                               (int64_t)n.az.nq * nyx, st);
    if (e != cudaSuccess) return e;
    // stage X, all items and planes at once: H ((nb nqz ny) x nqx) = P ((nb nqz ny) x nx) * TxT (nx x nqx)
    const int64_t rows = (int64_t)nb * n.az.nq * p.ny;     // < 2^31: the chunk holds at most 2 GB of P
    e = zgemm<double2, double2, double2, true>(d_P, d_TxT, d_H, (int)rows, n.ax.nq, p.nx, p.nx, n.ax.nq, n.ax.nq, 1, 0, 0, 0, st);
    if (e != cudaSuccess) return e;
    // stage Y, one GEMM per (item, g_z plane): U_m (nqy x nqx) = Ty (nqy x ny) * H_m (ny x nqx)
    const int planes = nb * n.az.nq;
    for (int z0 = 0; z0 < planes; z0 += 65535) {
        const int nzb = planes - z0 < 65535 ? planes - z0 : 65535;
        e = zgemm<double2, double2, float2, false>(d_Ty, d_H + (int64_t)z0 * p.ny * n.ax.nq, d_U + (int64_t)z0 * n.ay.nq * n.ax.nq, n.ay.nq, n.ax.nq,
                                    p.ny, p.ny, n.ax.nq, n.ax.nq, nzb, 0, (int64_t)p.ny * n.ax.nq, (int64_t)n.ay.nq * n.ax.nq, st);
        if (e != cudaSuccess) return e;
    }
    return launch_nufft_interp(p, n, nb, npx, npy, pixel_cells, d_q, d_U, nullptr, p.dx * p.dy * p.dz, d_I, st);
}

cudaError_t launch_nufft_interp(const Plan &p, const NufftPlan &n, int nb, int npx, int npy, double pixel_cells, const double *d_q,
                                const float2 *d_U, const float *d_ampscale, double scale_mul, float *d_I, cudaStream_t st) {
    const int64_t strideU = (int64_t)n.az.nq * n.ay.nq * n.ax.nq;
    const double dV = scale_mul;
    (void)p;
    // P pixels share a window of W + 2 cells if their first cells differ by at most 2, i.e. if they lie within 2 grid cells of each other
    // on every axis: (P - 1) x pixel_cells < 2 (with a margin; a group that still does not fit takes its pixels one by one in the kernel)
    // (measured on B200: two pixels per thread and twice the threads beat four pixels per thread -- the same instruction count, but
    // the per-thread chains are half as long and twice as many warps hide them; profiles/r02_nufft_tensor.md)
    if (pixel_cells < 1.9) return launch_interp<2>(d_q, npx, npy, n, d_U, strideU, nb, dV, d_ampscale, d_I, st);
    return launch_interp<1>(d_q, npx, npy, n, d_U, strideU, nb, dV, d_ampscale, d_I, st);
}

}  // namespace scatman
