// fit_kernels.cu -- forward-fitting pieces on the device ("simulating its diffraction pattern,
// comparing it with the desired experimental data, and then iteratively improving the guess"):
//   * discrepancy between simulated patterns and a measured one, so that a fit step returns one number per candidate
//     instead of an image: the integral-normalised squared distance (the normalisation of Fig. 5) and the
//     scale-fitted Poisson deviance;
//   * the Ideal detector: Poisson counts with means n_photons * I / sum(I), drawn from Philox-4x32-10 with
//     the counter (pixel lo, pixel hi, item, draw) and the seed as key -- every pixel's draw is independent of the launch shape.
// HBM-bound: one or two passes over the patterns (4 B per pixel and item, + 4 B for the measured pattern, + 1 B mask),
// FP64 accumulation (free at this intensity), deterministic two-level sums (per-block partials, summed in index order).
#include <mutex>

#include "internal.h"

namespace scatman {

namespace {

constexpr int kFitThreads = 256;
constexpr int kFitChunk = 32768;  // pixels per block, fewer for problems that would not fill the GPU (fit_chunk)

__device__ __forceinline__ double block_sum(double v, double *s_red) {
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    __syncthreads();   // s_red may still be read from the previous call
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < kFitThreads / 32; ++w) t += s_red[w];
    return t;   // valid in thread 0
}

// One load slot of a thread: G consecutive pixels (4 as one 16-byte load of each pattern and one 4-byte load of the mask when
// the pixel count, the stride of M and the three addresses allow it, else 1).  The loads of a slot do not wait for one another.
template <bool kVec>
struct FitSlot {
    static constexpr int G = kVec ? 4 : 1;
    float i[G], m[G];
    bool on[G];
    __device__ __forceinline__ void load(const float *Ib, const float *Mb, const unsigned char *mask, int64_t p, bool in) {
        if constexpr (kVec) {
            const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
            const float4 vi = in ? __ldg((const float4 *)(Ib + p)) : z;
            const float4 vm = in && Mb ? __ldg((const float4 *)(Mb + p)) : z;
            const unsigned w = in ? (mask ? __ldg((const unsigned *)(mask + p)) : 0x01010101u) : 0u;
            i[0] = vi.x, i[1] = vi.y, i[2] = vi.z, i[3] = vi.w;
            m[0] = vm.x, m[1] = vm.y, m[2] = vm.z, m[3] = vm.w;
#pragma unroll
            for (int j = 0; j < 4; ++j) on[j] = ((w >> (8 * j)) & 0xffu) != 0u;
        } else {
            const unsigned char w = in ? (mask ? mask[p] : (unsigned char)1) : (unsigned char)0;
            i[0] = in ? Ib[p] : 0.f;
            m[0] = in && Mb ? Mb[p] : 0.f;
            on[0] = w != 0;
        }
    }
};

}  // namespace

// pass 1: partial[b][chunk][5] = sums over the chunk of w I, w M, w I^2, w M^2, w I M
template <bool kVec>
__global__ void __launch_bounds__(kFitThreads, 4) fit_sums_kernel(const float *__restrict__ I, const float *__restrict__ M,
                                                               int64_t m_stride, const unsigned char *__restrict__ mask,
                                                               int64_t npix, int nchunk, int chunk_px, double *__restrict__ partial) {
    __shared__ double s_red[5 * kFitThreads / 32];
    const int b = blockIdx.y, chunk = blockIdx.x;
    const float *Ib = I + (size_t)b * npix;
    const float *Mb = M ? M + (size_t)b * m_stride : nullptr;
    double a[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    const int64_t p1 = min((int64_t)(chunk + 1) * chunk_px, npix);
    constexpr int G = FitSlot<kVec>::G;
    for (int64_t p0 = (int64_t)chunk * chunk_px + threadIdx.x * G; p0 < p1; p0 += 4 * kFitThreads * G) {
        FitSlot<kVec> s[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {   // four independent slots in flight per thread; the mask is applied afterwards
            const int64_t p = p0 + k * kFitThreads * G;
            s[k].load(Ib, Mb, mask, p, p < p1);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int j = 0; j < G; ++j) {
                const double i = s[k].on[j] ? (double)s[k].i[j] : 0.0, m = s[k].on[j] ? (double)s[k].m[j] : 0.0;
                a[0] += i;
                a[1] += m;
                a[2] += i * i;
                a[3] += m * m;
                a[4] += i * m;
            }
    }
    // the five sums through one shared-memory stage
#pragma unroll
    for (int k = 0; k < 5; ++k)
        for (int off = 16; off > 0; off >>= 1) a[k] += __shfl_xor_sync(0xffffffffu, a[k], off);
    if ((threadIdx.x & 31) == 0)
#pragma unroll
        for (int k = 0; k < 5; ++k) s_red[(threadIdx.x >> 5) * 5 + k] = a[k];
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0.0;
        for (int w = 0; w < kFitThreads / 32; ++w) t += s_red[w * 5 + threadIdx.x];
        partial[((size_t)b * nchunk + chunk) * 5 + threadIdx.x] = t;
    }
}

// sums[b][5] = partials summed in chunk order (one warp per item would do; one thread is enough at these sizes)
__global__ void fit_reduce_kernel(const double *__restrict__ partial, int nchunk, int nk, int batch, double *__restrict__ sums) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= batch * nk) return;
    const int b = t / nk, k = t % nk;
    double s = 0.0;
    for (int c = 0; c < nchunk; ++c) s += partial[((size_t)b * nchunk + c) * nk + k];
    sums[t] = s;
}

// L2: D = sum w (I / S_I - M / S_M)^2 = S_II / S_I^2 - 2 S_IM / (S_I S_M) + S_MM / S_M^2 would cancel catastrophically
// for close patterns, so the squared differences are summed directly in a second pass (same cost: HBM-bound).
// metric 0: w (I / S_I - M / S_M)^2; metric 1: 2 w [M log(M / (c I)) - (M - c I)], c = S_M / S_I
template <bool kVec>
__global__ void __launch_bounds__(kFitThreads, 3) fit_metric_kernel(const float *__restrict__ I, const float *__restrict__ M,
                                                                 int64_t m_stride, const unsigned char *__restrict__ mask,
                                                                 int64_t npix, int nchunk, int chunk_px, int metric,
                                                                 const double *__restrict__ sums,
                                                                 const double *__restrict__ partial1, double *__restrict__ partial) {
    __shared__ double s_red[kFitThreads / 32];
    const int b = blockIdx.y, chunk = blockIdx.x;
    const float *Ib = I + (size_t)b * npix;
    const float *Mb = M + (size_t)b * m_stride;
    double SI, SM;
    if (partial1) {   // few chunks per item: every block adds pass 1's partial sums itself, in fit_reduce_kernel's order
        SI = 0.0, SM = 0.0;
        for (int c1 = 0; c1 < nchunk; ++c1) {
            SI += partial1[((size_t)b * nchunk + c1) * 5 + 0];
            SM += partial1[((size_t)b * nchunk + c1) * 5 + 1];
        }
    } else {
        SI = sums[b * 5 + 0], SM = sums[b * 5 + 1];
    }
    const double c = SM / SI, rSI = 1.0 / SI, rSM = 1.0 / SM;
    double acc = 0.0;
    const int64_t p1 = min((int64_t)(chunk + 1) * chunk_px, npix);
    constexpr int G = FitSlot<kVec>::G;
    for (int64_t p0 = (int64_t)chunk * chunk_px + threadIdx.x * G; p0 < p1; p0 += 4 * kFitThreads * G) {
        FitSlot<kVec> s[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int64_t p = p0 + k * kFitThreads * G;
            s[k].load(Ib, Mb, mask, p, p < p1);
        }
        if (metric == SCATMAN_LOSS_L2_NORMALISED) {
#pragma unroll
            for (int k = 0; k < 4; ++k)
#pragma unroll
                for (int j = 0; j < G; ++j) {
                    // no FMA contraction: identical patterns give exactly 0; a masked pixel adds an exact 0
                    const double d = __dmul_rn((double)s[k].i[j], rSI) - __dmul_rn((double)s[k].m[j], rSM);
                    acc += s[k].on[j] ? d * d : 0.0;
                }
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
#pragma unroll
                for (int j = 0; j < G; ++j) {
                    if (!s[k].on[j]) continue;
                    const double i = (double)s[k].i[j], m = (double)s[k].m[j];
                    const double mu = c * i;
                    acc += 2.0 * ((m > 0.0 ? m * log(m / mu) : 0.0) - (m - mu));
                }
        }
    }
    const double t = block_sum(acc, s_red);
    if (threadIdx.x == 0) partial[(size_t)b * nchunk + chunk] = t;
}

// ---- Ideal detector -----------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t &o0, uint32_t &o1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    o0 = c0;
    o1 = c1;
}

__device__ __forceinline__ void uniforms(uint64_t p, uint32_t b, uint32_t draw, uint64_t seed, double &u, double &v) {
    uint32_t x0, x1;
    philox4x32_10((uint32_t)p, (uint32_t)(p >> 32), b, draw, (uint32_t)seed, (uint32_t)(seed >> 32), x0, x1);
    u = ((double)x0 + 0.5) * 2.3283064365386963e-10;   // 2^-32
    v = ((double)x1 + 0.5) * 2.3283064365386963e-10;
}

// Poisson(lam): inversion by sequential search below 10, Hoermann's transformed rejection with squeeze (PTRS) from 10 on
__device__ double poisson_draw(double lam, uint64_t p, uint32_t b, uint64_t seed) {
    if (!(lam > 0.0)) return 0.0;
    double u, v;
    if (lam < 10.0) {
        uniforms(p, b, 0u, seed, u, v);
        int k = 0;
        double pk = exp(-lam), s = pk;
        while (u > s && k < 1000) {
            ++k;
            pk *= lam / (double)k;
            s += pk;
        }
        return (double)k;
    }
    const double slam = sqrt(lam), loglam = log(lam);
    const double bb = 0.931 + 2.53 * slam, a = -0.059 + 0.02483 * bb;
    const double invalpha = 1.1239 + 1.1328 / (bb - 3.4), vr = 0.9277 - 3.6224 / (bb - 2.0);
    for (uint32_t draw = 0;; ++draw) {
        uniforms(p, b, draw, seed, u, v);
        u -= 0.5;
        const double us = 0.5 - fabs(u);
        const double k = floor((2.0 * a / us + bb) * u + lam + 0.43);
        if (us >= 0.07 && v <= vr) return k;
        if (k < 0.0 || (us < 0.013 && v > us)) continue;
        if (log(v) + log(invalpha) - log(a / (us * us) + bb) <= -lam + k * loglam - lgamma(k + 1.0)) return k;
    }
}

__global__ void __launch_bounds__(kFitThreads) ideal_detector_kernel(const float *__restrict__ I, int64_t npix,
                                                                     const double *__restrict__ sums,
                                                                     const double *__restrict__ photons, uint64_t seed,
                                                                     float *__restrict__ counts) {
    const int b = blockIdx.y;
    const int64_t p = (int64_t)blockIdx.x * kFitThreads + threadIdx.x;
    if (p >= npix) return;
    const double S = sums[b * 5 + 0];
    double n = 0.0;
    if (S > 0.0) n = poisson_draw((double)I[(size_t)b * npix + p] * (photons[b] / S), (uint64_t)p, (uint32_t)b, seed);
    counts[(size_t)b * npix + p] = (float)n;
}

struct PhotonChunk {
    double v[256];
};
__global__ void store_photons_kernel(PhotonChunk c, int n, double *__restrict__ dst) {
    if ((int)threadIdx.x < n) dst[threadIdx.x] = c.v[threadIdx.x];
}

// ------------------------------------------------------------------------------------------------ host
// Pixels per block: 32768, but a block walks its chunk in steps of one load round trip each, so a problem with few such
// chunks (256 patterns of 256^2 pixels: 512) would run as one and a bit waves of long blocks.  Below four waves of blocks
// (148 SMs x 3 blocks) the chunk shrinks to 8192, then to 2048 (one step of a block).  The scratch stays below 512 KB there,
// so nothing that fitted the static array (scatman_discrepancy_static) with 32768-pixel chunks stops fitting.
int fit_chunk(int64_t npix, int batch) {
    const int64_t enough = 4 * 148 * 3;
    int chunk = kFitChunk;
    while (chunk > 2048 && (int64_t)batch * ((npix + chunk - 1) / chunk) < enough) chunk /= 4;
    return chunk;
}

int fit_nchunk(int64_t npix, int batch) {
    const int chunk = fit_chunk(npix, batch);
    return (int)((npix + chunk - 1) / chunk);
}

size_t fit_workspace_bytes(int64_t npix, int batch) {
    // partial[b][nchunk][5] + sums[b][5] + partial2[b][nchunk] + photons[b]
    return sizeof(double) * ((size_t)batch * fit_nchunk(npix, batch) * 6 + (size_t)batch * 6);
}

// ---- static scratch (scatman_discrepancy_static) ----------------------------------------------------------------------
// The scratch of the discrepancy kernels for callers that cannot allocate: a file-scope device array, held by every GPU
// that loads the library until the process exits.  In HOST code the name g_fit_static_scratch is a host-side stand-in, not
// a device address: kernels are handed the address cudaGetSymbolAddress returns for the CURRENT device, resolved once per
// device (call with that device current) and kept here.
static __device__ __align__(256) unsigned char g_fit_static_scratch[SCATMAN_STATIC_SCRATCH_BYTES];

cudaError_t fit_static_scratch(int device, double **d_ptr) {
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static double *resolved[kMaxDevices] = {};
    *d_ptr = nullptr;
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!resolved[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_fit_static_scratch);
        if (e != cudaSuccess) return e;
        resolved[device] = (double *)p;
    }
    *d_ptr = resolved[device];
    return cudaSuccess;
}

// 16-byte loads of the patterns and 4-byte loads of the mask: every item's row starts on such a boundary
static bool fit_vec_ok(const float *d_I, const float *d_M, int64_t m_stride, const unsigned char *d_mask, int64_t npix) {
    return (npix & 3) == 0 && (m_stride & 3) == 0 && (((uintptr_t)d_I | (uintptr_t)d_M) & 15) == 0 && ((uintptr_t)d_mask & 3) == 0;
}

cudaError_t launch_fit_sums(const float *d_I, const float *d_M, int64_t m_stride, const unsigned char *d_mask, int64_t npix,
                            int batch, double *d_ws, cudaStream_t st, bool reduce = true) {
    const int nchunk = fit_nchunk(npix, batch), chunk_px = fit_chunk(npix, batch);
    double *partial = d_ws, *sums = d_ws + (size_t)batch * nchunk * 5;
    if (fit_vec_ok(d_I, d_M, m_stride, d_mask, npix))
        fit_sums_kernel<true><<<dim3(nchunk, batch), kFitThreads, 0, st>>>(d_I, d_M, m_stride, d_mask, npix, nchunk, chunk_px, partial);
    else
        fit_sums_kernel<false><<<dim3(nchunk, batch), kFitThreads, 0, st>>>(d_I, d_M, m_stride, d_mask, npix, nchunk, chunk_px, partial);
    if (reduce) fit_reduce_kernel<<<(batch * 5 + 127) / 128, 128, 0, st>>>(partial, nchunk, 5, batch, sums);
    return cudaGetLastError();
}

// With at most this many chunks per item the metric kernel's blocks add pass 1's partial sums themselves (2 x nchunk FP64
// loads per block from L2) and the launch between the two passes goes.
constexpr int kFitFoldChunks = 32;

int fit_discrepancy_launches(int64_t npix, int batch) { return fit_nchunk(npix, batch) <= kFitFoldChunks ? 3 : 4; }

cudaError_t launch_discrepancy(const float *d_I, const float *d_M, int64_t m_stride, const unsigned char *d_mask, int64_t npix,
                               int batch, int metric, double *d_ws, double *d_out, cudaStream_t st) {
    const int nchunk = fit_nchunk(npix, batch), chunk_px = fit_chunk(npix, batch);
    const bool fold = nchunk <= kFitFoldChunks;
    cudaError_t e = launch_fit_sums(d_I, d_M, m_stride, d_mask, npix, batch, d_ws, st, !fold);
    if (e != cudaSuccess) return e;
    double *sums = d_ws + (size_t)batch * nchunk * 5, *partial2 = sums + (size_t)batch * 5;
    const double *partial1 = fold ? d_ws : nullptr;
    if (fit_vec_ok(d_I, d_M, m_stride, d_mask, npix))
        fit_metric_kernel<true><<<dim3(nchunk, batch), kFitThreads, 0, st>>>(d_I, d_M, m_stride, d_mask, npix, nchunk, chunk_px, metric, sums, partial1, partial2);
    else
        fit_metric_kernel<false><<<dim3(nchunk, batch), kFitThreads, 0, st>>>(d_I, d_M, m_stride, d_mask, npix, nchunk, chunk_px, metric, sums, partial1, partial2);
    fit_reduce_kernel<<<(batch + 127) / 128, 128, 0, st>>>(partial2, nchunk, 1, batch, d_out);
    return cudaGetLastError();
}

cudaError_t launch_ideal_detector(const float *d_I, int64_t npix, int batch, const double *h_photons, uint64_t seed, double *d_ws,
                                  float *d_counts, cudaStream_t st) {
    cudaError_t e = launch_fit_sums(d_I, nullptr, 0, nullptr, npix, batch, d_ws, st);
    if (e != cudaSuccess) return e;
    const int nchunk = fit_nchunk(npix, batch);
    double *sums = d_ws + (size_t)batch * nchunk * 5;
    double *photons = sums + (size_t)batch * 5 + (size_t)batch * nchunk;
    // the photon numbers travel as kernel arguments (read from h_photons before return whatever memory it is; capturable)
    for (int b0 = 0; b0 < batch; b0 += 256) {
        PhotonChunk c;
        const int n = batch - b0 < 256 ? batch - b0 : 256;
        for (int i = 0; i < n; ++i) c.v[i] = h_photons[b0 + i];
        store_photons_kernel<<<1, 256, 0, st>>>(c, n, photons + b0);
    }
    ideal_detector_kernel<<<dim3((unsigned)((npix + kFitThreads - 1) / kFitThreads), batch), kFitThreads, 0, st>>>(
        d_I, npix, sums, photons, seed, d_counts);
    return cudaGetLastError();
}

}  // namespace scatman
