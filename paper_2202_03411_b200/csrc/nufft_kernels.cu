// nufft_kernels.cu -- flat-detector route by a 3-D type-2 non-uniform Fourier transform (second half).
//
// The pattern is still A(p) = sum_r rho~(r) e^{i q(p).r} at every pixel's Ewald-sphere q (Eq. 2/4), but the pixel x voxel
// contraction is replaced by
//   (1) a SEPARABLE transform of rho~ onto a small uniform (g_z, g_y, g_x) grid that covers the q's of the detector with a margin,
//       U[mz][my][mx] = sum_r c_z c_y c_x rho~(r) e^{i g_m . r}     -- three complex GEMMs (stage Z over slices, X over columns, Y over rows)
//   (2) an interpolation from that grid to each pixel with a Kaiser-Bessel window of W = 12 grid cells per axis,
//       A(p) = sum_{m near q(p)/h} phi(u_z - m_z) phi(u_y - m_y) phi(u_x - m_x) U[m],   u = q / h.
// Grid spacing h_d = 2 pi / (2 N_d d_d) (oversampling 2), pre-correction c_i = 1 / Phi(h x_i) with Phi the window's Fourier transform:
//   sum_m phi(u - m) e^{i m t} = sum_l Phi(t - 2 pi l) e^{i u (t - 2 pi l)}   (Poisson summation),   |t| = |h x_i| < pi / 2,
// so the l = 0 term is the wanted e^{i u t} and the l = +-1 aliases are below 1e-10 of it for W = 12, beta = pi sqrt(W^2 (3/4)^2 - 0.8).
// Everything is FP64 on the CUDA cores (the work is ~1000x smaller than the pixel contraction: 1.2e9 complex MACs for 256^3 on 512^2
// pixels against 4.4e12), so the only approximation is the window's and the result meets the same tolerances against the oracle.
#include "internal.h"

namespace scatman {

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
constexpr int BM = 64, BN = 64, BK = 16;

__device__ inline double2 ld_c(const double2 *p) { return __ldg(p); }
__device__ inline double2 ld_c(const float2 *p) { const float2 v = __ldg(p); return make_double2((double)v.x, (double)v.y); }

template <typename TA, typename TB>
__global__ void __launch_bounds__(256)
nufft_zgemm_kernel(const TA *__restrict__ A, const TB *__restrict__ B, double2 *__restrict__ C, int M, int N, int K,
                   int64_t lda, int64_t ldb, int64_t ldc, int64_t strideA, int64_t strideB, int64_t strideC) {
    __shared__ double2 As[BK][BM + 1];
    __shared__ double2 Bs[BK][BN];
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int n0 = blockIdx.x * BN, m0 = blockIdx.y * BM;
    A += (int64_t)blockIdx.z * strideA;
    B += (int64_t)blockIdx.z * strideB;
    C += (int64_t)blockIdx.z * strideC;
    double2 acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = make_double2(0.0, 0.0);
    double2 ra[4], rb[4];
    auto fetch = [&](int k0) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = t + 256 * r;
            const int ak = idx & 15, am = idx >> 4;
            ra[r] = (m0 + am < M && k0 + ak < K) ? ld_c(A + (int64_t)(m0 + am) * lda + (k0 + ak)) : make_double2(0.0, 0.0);
            const int bn = idx & 63, bk = idx >> 6;
            rb[r] = (n0 + bn < N && k0 + bk < K) ? ld_c(B + (int64_t)(k0 + bk) * ldb + (n0 + bn)) : make_double2(0.0, 0.0);
        }
    };
    fetch(0);
    for (int k0 = 0; k0 < K; k0 += BK) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = t + 256 * r;
            As[idx & 15][idx >> 4] = ra[r];
            Bs[idx >> 6][idx & 63] = rb[r];
        }
        __syncthreads();
        if (k0 + BK < K) fetch(k0 + BK);
#pragma unroll
        for (int k = 0; k < BK; ++k) {
            double2 a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[k][ty + 16 * i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Bs[k][tx + 16 * j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    acc[i][j].x = fma(a[i].x, b[j].x, acc[i][j].x);
                    acc[i][j].x = fma(-a[i].y, b[j].y, acc[i][j].x);
                    acc[i][j].y = fma(a[i].x, b[j].y, acc[i][j].y);
                    acc[i][j].y = fma(a[i].y, b[j].x, acc[i][j].y);
                }
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int m = m0 + ty + 16 * i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = n0 + tx + 16 * j;
            if (n < N) C[(int64_t)m * ldc + n] = acc[i][j];
        }
    }
}

template <typename TA, typename TB>
cudaError_t zgemm(const TA *A, const TB *B, double2 *C, int M, int N, int K, int64_t lda, int64_t ldb, int64_t ldc, int nbatch,
                  int64_t sA, int64_t sB, int64_t sC, cudaStream_t st) {
    // grid.y carries the row tiles (<= 65535: M <= 4 M rows), grid.z the batch
    for (int m_base = 0; m_base < M; m_base += 65535 * BM) {
        const int rows = M - m_base < 65535 * BM ? M - m_base : 65535 * BM;
        dim3 grid((N + BN - 1) / BN, (rows + BM - 1) / BM, nbatch);
        nufft_zgemm_kernel<TA, TB><<<grid, 256, 0, st>>>(A + (int64_t)m_base * lda, B, C + (int64_t)m_base * ldc, rows, N, K, lda, ldb,
                                                         ldc, sA, sB, sC);
    }
    return cudaGetLastError();
}

// ---- interpolation: one thread per pixel; A = sum over the W^3 nearest grid points, I = |A dV|^2 (Block 11).
__device__ inline double kb_phi(double s, double beta, double inv_i0b) {
    const double a = 1.0 - (s / kHalfW) * (s / kHalfW);
    return a > 0.0 ? cyl_bessel_i0(beta * sqrt(a)) * inv_i0b : (a == 0.0 ? inv_i0b : 0.0);
}

__global__ void __launch_bounds__(128)
nufft_interp_kernel(const double *__restrict__ q, int64_t npix, NufftAxis ax, NufftAxis ay, NufftAxis az,
                    const double2 *__restrict__ U, double inv_i0b, double dV, float *__restrict__ I) {
    __shared__ double wyz[2 * kW][128];
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npix) return;
    const double beta = kb_beta();
    const double ux = q[3 * p + 0] * ax.inv_h, uy = q[3 * p + 1] * ay.inv_h, uz = q[3 * p + 2] * az.inv_h;
    const int mx0 = (int)ceil(ux - kHalfW), my0 = (int)ceil(uy - kHalfW), mz0 = (int)ceil(uz - kHalfW);
    double wx[kW];
#pragma unroll
    for (int i = 0; i < kW; ++i) {
        wx[i] = kb_phi(ux - (double)(mx0 + i), beta, inv_i0b);
        wyz[i][threadIdx.x] = kb_phi(uy - (double)(my0 + i), beta, inv_i0b);
        wyz[kW + i][threadIdx.x] = kb_phi(uz - (double)(mz0 + i), beta, inv_i0b);
    }
    const int ix = mx0 - ax.m_lo, iy = my0 - ay.m_lo, iz = mz0 - az.m_lo;   // >= 0 and + kW <= nq by the margins of the plan
    double are = 0.0, aim = 0.0;
    for (int c = 0; c < kW; ++c) {
        const double wz = wyz[kW + c][threadIdx.x];
        double pre = 0.0, pim = 0.0;
        for (int b = 0; b < kW; ++b) {
            const double2 *row = U + ((int64_t)(iz + c) * ay.nq + (iy + b)) * ax.nq + ix;
            double rre = 0.0, rim = 0.0;
#pragma unroll
            for (int a = 0; a < kW; ++a) {
                const double2 v = __ldg(row + a);
                rre = fma(wx[a], v.x, rre);
                rim = fma(wx[a], v.y, rim);
            }
            const double wy = wyz[b][threadIdx.x];
            pre = fma(wy, rre, pre);
            pim = fma(wy, rim, pim);
        }
        are = fma(wz, pre, are);
        aim = fma(wz, pim, aim);
    }
    are *= dV;
    aim *= dV;
    I[p] = (float)(are * are + aim * aim);
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

// One batch item: rho~ [nz][ny][nx] -> P [nqz][ny][nx] -> H [nqz][ny][nqx] -> U [nqz][nqy][nqx] -> I [npix].
cudaError_t launch_nufft_item(const float2 *d_rho, const Plan &p, const NufftPlan &n, const double2 *d_Tz, const double2 *d_TxT,
                              const double2 *d_Ty, const double *d_q, double2 *d_P, double2 *d_H, double2 *d_U, float *d_I,
                              cudaStream_t st) {
    const int64_t nyx = (int64_t)p.ny * p.nx;
    cudaError_t e = cudaSuccess;
    // stage Z: P (nqz x ny nx) = Tz (nqz x nz) * rho~ (nz x ny nx); the column dimension is cut so that grid.x stays in range
    e = zgemm<double2, float2>(d_Tz, d_rho, d_P, n.az.nq, (int)nyx, p.nz, p.nz, nyx, nyx, 1, 0, 0, 0, st);
    if (e != cudaSuccess) return e;
    // stage X: H ((nqz ny) x nqx) = P ((nqz ny) x nx) * TxT (nx x nqx)
    e = zgemm<double2, double2>(d_P, d_TxT, d_H, n.az.nq * p.ny, n.ax.nq, p.nx, p.nx, n.ax.nq, n.ax.nq, 1, 0, 0, 0, st);
    if (e != cudaSuccess) return e;
    // stage Y, one GEMM per g_z plane: U_m (nqy x nqx) = Ty (nqy x ny) * H_m (ny x nqx)
    for (int z0 = 0; z0 < n.az.nq; z0 += 65535) {
        const int nzb = n.az.nq - z0 < 65535 ? n.az.nq - z0 : 65535;
        e = zgemm<double2, double2>(d_Ty, d_H + (int64_t)z0 * p.ny * n.ax.nq, d_U + (int64_t)z0 * n.ay.nq * n.ax.nq, n.ay.nq, n.ax.nq,
                                    p.ny, p.ny, n.ax.nq, n.ax.nq, nzb, 0, (int64_t)p.ny * n.ax.nq, (int64_t)n.ay.nq * n.ax.nq, st);
        if (e != cudaSuccess) return e;
    }
    nufft_interp_kernel<<<(unsigned)((p.npix + 127) / 128), 128, 0, st>>>(d_q, p.npix, n.ax, n.ay, n.az, d_U, nufft_inv_i0_beta(),
                                                                         p.dx * p.dy * p.dz, d_I);
    return cudaGetLastError();
}

}  // namespace scatman
