// sep_tensor_kernels.cu -- the separable tensor-grid route (Block 6 of Fig. 4 transforms every slice on a
// uniform (qx, qy) grid) with both GEMM stages on tcgen05 tensor cores, FP16x3 split precision:
//   stage X   H_j[a, y]  = sum_x rho~_j[y, x] e^{i qx[a] x}                        (M = y rows, N = a columns, K = x)
//   stage YZ  A[b, a]    = sum_j e^{i qz(a,b) z_j} sum_y e^{i qy[b] y} H_j[a, y]   (K = y; Blocks 7-8 in the epilogue)
// Every operand is four FP16 planes (Re_hi, Re_lo, Im_hi, Im_lo) of a scaled FP32 value, K-major, fetched by TMA boxes of
// 64 K x rows with the 128-byte swizzle; a complex product is the 12 real MMAs AhBh + AlBh + AhBl of tensor_kernel.cu
// (the minus sign of Re = ArBr - AiBi is the instruction descriptor's negate-A bit).  Accumulators live in TMEM, FP32.
// Stage X's epilogue rescales H and splits it into the FP16 planes stage YZ reads; stage YZ's epilogue applies the slice
// phase e^{i qz(a,b) z_j} to the accumulator tile and sums over slices in registers.  Vacuum is skipped in 64-y blocks (byte
// flags); batch items are stacked along z; z splits are balanced on the device by live tiles.
// Kernels (selected by make_sep_tc_plan, covered by tests/test_gpu_qgrid.py):
//   stage X   tcg::cgemm_kernel<SepXPolicy<NX>>     CTA pairs, UMMA 256 x 2NX, Ex tile resident (NX = 64 / 32 / 16 for N_x <= 256 / 512 / 1024)
//   stage YZ  tcg::cgemm_kernel<SepYztPolicy<64>>   CTA pairs, transposed, Ey resident for all y (N_y <= 256)
//             sep_tc_yzs_kernel                     CTA pairs, both operands streamed (N_y <= 2048)
// Stage X and the transposed stage YZ are instances of ONE producer / issuer / epilogue pipeline (tc_cgemm.cuh), which also runs
// the NUFFT route's stages Y and Z; odd tile counts are handled by running the last tile twice in the pair, so no single-CTA
// variants exist.  Grids with N_x > 1024 or N_y > 2048 use the CUDA-core stages (sep_kernels.cu).
//
// Slice phase: qz z_j = 2 pi t (2j - nz + 1) with t = qz dz / (4 pi) turns; frac(t) is kept as a 32-bit fixed-point
// fraction of a turn, so the product with the integer (2j - nz + 1) wraps modulo one turn for free (error <= 512 * 2^-33
// turns = 4e-7 rad), and sin / cos come from the SFU on an argument in [-pi, pi) (absolute error ~4e-7).
#include <cuda.h>

#include <cstdio>
#include <cstdlib>

#include "internal.h"
#include "ptx_sm100.h"
#include "tc_cgemm.cuh"

namespace scatman {

bool encode_map(CUtensorMap *tm, const void *base, int rank, const cuuint64_t *dims, const cuuint64_t *strides,
                const cuuint32_t *box, CUtensorMapSwizzle swizzle);   // tensor_kernel.cu

namespace {

constexpr int kM = 128;              // UMMA M: rows of the A operand tile
constexpr int kKB = 64;              // K per block (one 128-byte swizzle row of FP16)
constexpr int kSlotA = kM * kKB * 2; // 16384: one plane, one K block of an A tile
constexpr int kThreadsTc = 384;      // warp 0 TMA, 1 and 3 MMA issuers, 2 TMEM, 4-11 epilogue
constexpr uint32_t kTmemColsTc = 512;

__device__ __forceinline__ double centre_t(int i, int n, double d) { return ((double)i - 0.5 * (double)(n - 1)) * d; }

__device__ __forceinline__ void split4(float re, float im, __half (&h)[4]) {
    h[0] = __float2half_rn(re);
    h[1] = __float2half_rn(re - __half2float(h[0]));
    h[2] = __float2half_rn(im);
    h[3] = __float2half_rn(im - __half2float(h[2]));
}

// The live units of a work item in issue order.  Unit n of the item is (slice z0 + n / ngw, 128-y group g0 + n % ngw); its two
// flag bytes say which of its 64-y blocks hold anything.  Warp-cooperative like tensor_kernel.cu's Units: each lane holds the
// flags of one of 32 consecutive units (the next 32 are already in flight), a ballot finds the next live one -- one L2 round
// trip per 32 units instead of one per unit in the critical path of every role.
struct LiveUnits {
    const unsigned char *fl;
    int nkb, z0, ngw, g0, total, base, lane;
    uint32_t cur, ahead, live;
    __device__ __forceinline__ uint32_t load(int n) const {
        if (n >= total) return 0u;
        const unsigned char *p = fl + (size_t)(z0 + n / ngw) * nkb + 2 * (g0 + n % ngw);
        return (uint32_t)__ldg(p) | ((uint32_t)__ldg(p + 1) << 1);
    }
    __device__ __forceinline__ void begin(const unsigned char *flags, int nkb_, int z0_, int z1, int ngw_, int g0_, int lane_) {
        fl = flags; nkb = nkb_; z0 = z0_; ngw = ngw_; g0 = g0_; lane = lane_;
        total = (z1 - z0_) * ngw_;
        base = 0;
        cur = load(lane);
        ahead = load(32 + lane);
        live = __ballot_sync(0xffffffffu, cur != 0u);
    }
    // next live unit: n = its index in the item, f = bit 0 / 1: first / second 64-y block non-empty; false at the end
    __device__ __forceinline__ bool next(int &n, uint32_t &f) {
        while (live == 0u) {
            base += 32;
            if (base >= total) return false;
            cur = ahead;
            ahead = load(base + 32 + lane);
            live = __ballot_sync(0xffffffffu, cur != 0u);
        }
        const int pos = __ffs((int)live) - 1;
        live &= live - 1;
        f = __shfl_sync(0xffffffffu, cur, pos);
        n = base + pos;
        return true;
    }
};

}  // namespace

// ------------------------------------------------------------------------------------------------ operands
// E planes fp16 [4][rows_pad][kpad] = split(2^10 e^{i q[r] c_i}), c_i centred coordinates; zero in the padding
__global__ void sep_tc_table_kernel(const double *__restrict__ q, int nq, int rows_pad, int n, int kpad, double d,
                                    __half *__restrict__ E) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)rows_pad * kpad) return;
    const int r = (int)(t / kpad), i = (int)(t % kpad);
    float re = 0.f, im = 0.f;
    if (r < nq && i < n) {
        double s, c;
        sincos(q[r] * centre_t(i, n, d), &s, &c);
        re = (float)(c * (double)kScaleA);
        im = (float)(s * (double)kScaleA);
    }
    __half h[4];
    split4(re, im, h);
    const size_t plane = (size_t)rows_pad * kpad;
#pragma unroll
    for (int pl = 0; pl < 4; ++pl) E[pl * plane + t] = h[pl];
}

// per item: sH = 2^(14 - e - L) (max |rho~ component| in [2^(e-1), 2^e), 2^L >= nx) is the scale H is stored with;
// ampscale = dV / (2^10 sH) takes the summed amplitude back to physical units
__global__ void sep_tc_scale_kernel(const unsigned *__restrict__ maxbits, int nb, int L, float dV, float *__restrict__ ampscale) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const float m = __uint_as_float(maxbits[b]);
    int e = 0;
    if (m > 0.f) frexpf(m, &e);
    ampscale[b] = dV / (kScaleA * ldexpf(1.f, 14 - e - L));
}

// rho~ FP32 [nb][nz][ny][nx] -> planes fp16 [4][nb * nz * NY][NXP] = split(sR[b] rho~), x fastest (K-major for stage X), zero
// in the padding; sR = 2^(13 - e) per item as in pack_b_kernel.  The items of a chunk are stacked along z: global slice
// jg = b nz + j.  Also raises flags64[j][y / 64] for every 64-y block holding a non-zero value
// (flags are cleared by a memset before).  One thread = 8 consecutive x of one row.
__global__ void sep_tc_pack_rho_kernel(const float2 *__restrict__ rho, int nx, int ny, int nz1, int nz, int NY, int NXP,
                                       const unsigned *__restrict__ maxbits, __half *__restrict__ R,
                                       unsigned char *__restrict__ flags) {   // nz1: slices per item, nz: of the chunk
    const int nx8 = NXP / 8;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)nz * NY * nx8) return;
    const int x0 = (int)(t % nx8) * 8;
    const int64_t row = t / nx8;
    const int y = (int)(row % NY), j = (int)(row / NY);
    const float m = __uint_as_float(maxbits[j / nz1]);
    int e = 0;
    if (m > 0.f) frexpf(m, &e);
    const float s = ldexpf(1.f, kScaleBExp - e);
    __align__(16) __half h[4][8];
    bool any = false;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float2 v = make_float2(0.f, 0.f);
        if (y < ny && x0 + i < nx) v = __ldg(rho + ((size_t)j * ny + y) * nx + x0 + i);
        any |= (v.x != 0.f) | (v.y != 0.f);
        __half q[4];
        split4(v.x * s, v.y * s, q);
#pragma unroll
        for (int pl = 0; pl < 4; ++pl) h[pl][i] = q[pl];
    }
    const size_t plane = (size_t)nz * NY * NXP, o = (size_t)row * NXP + x0;
#pragma unroll
    for (int pl = 0; pl < 4; ++pl) *(uint4 *)(R + pl * plane + o) = *(const uint4 *)h[pl];
    if (any) flags[(size_t)j * (NY / kKB) + y / kKB] = 1;
}

// Step a2 (Eq. 6/8/9) fused with the pack above: the exclusive z-prefix of strength_kernel (prep_kernels.cu: T_j
// as a running FP64 product of the per-voxel factors exp(i k dz dn), the factor of the last (delta, beta) seen reused) writes the
// scaled FP16 planes and the flags directly -- rho~ never goes to memory in FP32.  The scale 2^(13 - e) comes from an upper BOUND of
// max |rho~| known before the prefix runs (prefix_bound_kernel).  One thread = C adjacent columns (x .. x + C - 1, y) of one item,
// walking z, x fastest (sep_tc_prefix_planes_kernel below).
// layer_live[l] = any tile of layer l (four slices of one item) of the tile map was written
__global__ void tile_layers_kernel(const unsigned char *__restrict__ tilemap, int tiles, unsigned char *__restrict__ layer_live) {
    const unsigned char *t = tilemap + (size_t)blockIdx.x * tiles;
    int any = 0;
    for (int i = threadIdx.x; i < tiles; i += blockDim.x) any |= t[i];
    any = __syncthreads_or(any);
    if (threadIdx.x == 0) layer_live[blockIdx.x] = any ? 1 : 0;
}

constexpr int kPrefThreads = 128, kPrefStages = 3;
template <int C> struct PrefVec;                       // C columns of (delta, beta) / of one FP16 plane
template <> struct PrefVec<1> { using In = float2; using Out = unsigned short; };
template <> struct PrefVec<4> { using In = float4; using Out = uint2; };

// C = 4 columns per thread (two 16-byte copies per slice in, one 8-byte store per plane out; needs even nx) or C = 1 (any nx).
template <int C>
__global__ void __launch_bounds__(kPrefThreads, C == 1 ? 8 : 5)
sep_tc_prefix_planes_kernel(const float2 *__restrict__ dn, int nx, int ny, int nz1, int nb, int NY, int NXP, double kdz, int rho_mode,
                            const unsigned *__restrict__ maxbits, __half *__restrict__ R, unsigned char *__restrict__ flags,
                            const unsigned char *__restrict__ tilemap, const unsigned char *__restrict__ layer_live) {
    // The column's voxels reach the thread through a ring of cp.async stages in shared memory (every thread reads back only what it
    // copied itself: no barrier, only its own wait_group): two batches of slices are in flight while a third is worked on, and the
    // loop over the slices of a batch is NOT unrolled -- the unrolled register version (eight inlined FP64 sincos / exp) ran at
    // 128 registers, four warps per scheduler, and was bound by load latency at 45 % of the HBM rate; one column per thread with
    // 2-byte stores was then bound by the load/store instruction queue.
    constexpr int kBatch = C == 1 ? 8 : 3;             // 24 / 36 KB of shared memory: 8 / 5 blocks per SM
    constexpr int kCopies = C == 1 ? 1 : 2;            // cp.async per slice
    __shared__ __align__(16) float2 ring[kPrefStages][kBatch][kCopies][kPrefThreads][C / kCopies];
    const int ncg = NXP / C;                            // column groups of a row (NXP is a multiple of 64)
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int x = (t % ncg) * C, y = t / ncg, b = blockIdx.y;
    if (y >= NY) return;
    const float m = __uint_as_float(maxbits[b]);
    int e = 0;
    if (m > 0.f) frexpf(m, &e);
    const float s = ldexpf(1.f, kScaleBExp - e);
    const size_t plane = (size_t)nb * nz1 * NY * NXP;
    __half *out = R + ((size_t)b * nz1 * NY + y) * NXP + x;             // + j NY NXP per slice, + plane per plane
    const size_t ostride = (size_t)NY * NXP;
    const float2 *src = dn + (size_t)b * nx * ny * nz1 + (y < ny ? (size_t)y * nx : 0);
    const size_t sstride = (size_t)nx * ny;
    const int nkb = NY / kKB;
    unsigned char *fl = flags + (size_t)b * nz1 * nkb + y / kKB;
    const int nbatch = (nz1 + kBatch - 1) / kBatch;
    // Sparse input (launch_orient / the renderer with a tile map): tiles of 16 x 4 x 4 voxels that hold no material are not read -- the
    // copy is issued with source size 0, which zero-fills.  The thread's C columns lie in one tile column; the map byte of the
    // layer after the one being fetched is already in flight.
    // ... and a layer of four slices none of whose tiles holds material is not packed at all (no flag is raised for it, so no stage
    // reads its planes).
    const unsigned char *ll = layer_live ? layer_live + (size_t)b * ((nz1 + 3) / 4) : nullptr;
    const unsigned char *tmp = nullptr;      // map byte of the layer after the one being fetched
    size_t tm_stride = 0;
    unsigned char tm_cur = 1, tm_next = 1;
    int tm_left = 0;                         // layers after the current one
    bool okc[kCopies];                       // the copy's columns exist (C = 4: nx is even, a pair of columns is in or out as a whole)
#pragma unroll
    for (int c = 0; c < kCopies; ++c) okc[c] = y < ny && x + c * (C / kCopies) < nx;
    if (tilemap && okc[0]) {
        const int nbx = (nx + 15) / 16, nby = (ny + 3) / 4, layers = (nz1 + 3) / 4;
        tm_stride = (size_t)nbx * nby;
        tmp = tilemap + (size_t)b * layers * tm_stride + (size_t)(y >> 2) * nbx + (x >> 4);
        tm_next = __ldg(tmp);
        tm_left = layers;
    }
    // running state of the copies: next slice, its address for this thread's first column, the ring stage it goes to
    int fj = 0, fstage = 0;
    const float2 *fsrc = src + x;
    const uint32_t ring0 = (uint32_t)__cvta_generic_to_shared(&ring[0][0][0][threadIdx.x][0]);
    constexpr uint32_t kCopyBytes = kPrefThreads * (C / kCopies) * 8, kSliceBytes = kCopies * kCopyBytes, kStageBytes = kBatch * kSliceBytes;
    auto fetch = [&]() {   // the next batch -> the next stage; padding columns and slices past the end are zero-filled
#pragma unroll
        for (int i = 0; i < kBatch; ++i, ++fj, fsrc += sstride) {
            if (fj >= nz1) break;
            if (tmp && (fj & 3) == 0) {      // a new layer of tiles
                tm_cur = tm_next;
                --tm_left;
                tmp += tm_stride;
                if (tm_left > 0) tm_next = __ldg(tmp);
            }
#pragma unroll
            for (int c = 0; c < kCopies; ++c) {
                const bool ok = okc[c] && tm_cur;
                const float2 *g = ok ? fsrc + c * (C / kCopies) : src;
                const uint32_t d = ring0 + fstage * kStageBytes + i * kSliceBytes + c * kCopyBytes;
                if (C == 1) ptx::cp_async_8s(d, g, ok);
                else ptx::cp_async_16s(d, g, ok);
            }
        }
        fstage = fstage + 1 == kPrefStages ? 0 : fstage + 1;
        ptx::cp_async_commit();   // (an empty group past the end keeps the wait counts uniform)
    };
    fetch();
    fetch();
    double Tre[C], Tim[C], gre[C], gim[C];
    float ld[C], lb[C];
#pragma unroll
    for (int c = 0; c < C; ++c) { Tre[c] = 1.0; Tim[c] = 0.0; gre[c] = 1.0; gim[c] = 0.0; ld[c] = lb[c] = 0.f; }
    int pstage = 0;
    __half *dst = out;
    for (int k = 0; k < nbatch; ++k) {
        fetch();
        ptx::cp_async_wait<2>();   // batch k has landed
        const int jn = min(kBatch, nz1 - k * kBatch);
        const float2 *rs = &ring[pstage][0][0][threadIdx.x][0];
        pstage = pstage + 1 == kPrefStages ? 0 : pstage + 1;
        float2 v[C];
#pragma unroll 1
        for (int i = 0; i < jn; ++i, dst += ostride, rs += kSliceBytes / 8) {
            if (ll && !__ldg(ll + ((k * kBatch + i) >> 2))) continue;
#pragma unroll
            for (int c = 0; c < C; ++c) v[c] = rs[(c / (C / kCopies)) * (kCopyBytes / 8) + c % (C / kCopies)];
            bool any = false;
#pragma unroll
            for (int c = 0; c < C; ++c) any |= (v[c].x != 0.f) | (v[c].y != 0.f);
            typename PrefVec<C>::Out pk[4];
#pragma unroll
            for (int pl = 0; pl < 4; ++pl) pk[pl] = typename PrefVec<C>::Out();
            if (any) {   // (vacuum: rho~ = 0, T unchanged)
                __half h[C][4];
                bool live = false;
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    float ox = 0.f, oy = 0.f;
                    if (v[c].x != 0.f || v[c].y != 0.f) {
                        const double d = (double)v[c].x, be = (double)v[c].y;
                        double fre = d, fim = be;
                        if (rho_mode == SCATMAN_RHO_N2M1) {   // c (2 - c)
                            fre = d * (2.0 - d) + be * be;
                            fim = 2.0 * be * (1.0 - d);
                        }
                        ox = (float)(fre * Tre[c] - fim * Tim[c]);
                        oy = (float)(fre * Tim[c] + fim * Tre[c]);
                        if (v[c].x != ld[c] || v[c].y != lb[c]) {
                            double sn, co;
                            sincos(kdz * d, &sn, &co);
                            const double mag = exp(-kdz * be);
                            gre[c] = mag * co;
                            gim[c] = mag * sn;
                            ld[c] = v[c].x;
                            lb[c] = v[c].y;
                        }
                        const double t = Tre[c] * gre[c] - Tim[c] * gim[c];
                        Tim[c] = Tre[c] * gim[c] + Tim[c] * gre[c];
                        Tre[c] = t;
                    }
                    split4(ox * s, oy * s, h[c]);
                    live |= (ox != 0.f) | (oy != 0.f);
                }
#pragma unroll
                for (int pl = 0; pl < 4; ++pl) {
                    if constexpr (C == 1) {
                        pk[pl] = __half_as_ushort(h[0][pl]);
                    } else {
                        pk[pl].x = (unsigned)__half_as_ushort(h[0][pl]) | ((unsigned)__half_as_ushort(h[1][pl]) << 16);
                        pk[pl].y = (unsigned)__half_as_ushort(h[2][pl]) | ((unsigned)__half_as_ushort(h[3][pl]) << 16);
                    }
                }
                if (live) fl[(size_t)(k * kBatch + i) * nkb] = 1;
            }
#pragma unroll
            for (int pl = 0; pl < 4; ++pl) *reinterpret_cast<typename PrefVec<C>::Out *>(dst + pl * plane) = pk[pl];
        }
    }
}

// Balanced z splits.  Sequence 0 (stage X): weight of slice j = its live 128-y row tiles; sequence 1 + g (stage YZ, group g):
// its live 64-y blocks of that group.  bounds[seq][0..ns] cut [0, nz) into ns ranges of (almost) equal total weight, so that
// every work item of a stage carries the same number of live tiles whatever the particle's extent along the beam:
// bounds[s] = min { j in [0, nz] : E(j) >= target(s) }, E(j) = weight of the slices before j, target(s) = floor(total s / ns).
// One block of 1024 threads per sequence: every thread sums a contiguous run of slices (all flag loads of the block are in
// flight together), a block scan gives E at the run starts, and each thread then places the bounds that fall into its run.
// sequence 0: stage X over all nzt slices of the chunk; sequence 1 + b ngs + g: stage YZ of item b, group g (its nz1 slices).
// Bounds are GLOBAL slice indices (jbase + j).  nyz_seq = 0 skips the stage YZ sequences (the NUFFT route needs only stage X's).
constexpr int kBoundsThreads = 1024;
__global__ void __launch_bounds__(kBoundsThreads)
sep_tc_bounds_kernel(const unsigned char *__restrict__ flags, int nz1, int nzt, int nkb, int ng, int ngs, int gw,
                     int nsx, int nzs, int *__restrict__ bx, int *__restrict__ by) {   // ngs YZ groups of gw flags
    const int seq = blockIdx.x, tid = threadIdx.x;
    const int ns = seq == 0 ? nsx : nzs;
    int *out = seq == 0 ? bx : by + (size_t)(seq - 1) * (nzs + 1);
    const int gsel = seq == 0 ? 0 : (seq - 1) % ngs;
    const int jbase = seq == 0 ? 0 : ((seq - 1) / ngs) * nz1;
    const int nz = seq == 0 ? nzt : nz1;
    if (seq == 0 && nzt > 65536) {   // very many stacked slices: equal slice counts per range balance well enough
        for (int sidx = tid; sidx <= ns; sidx += kBoundsThreads) out[sidx] = (int)(((long long)nzt * sidx) / ns);
        return;
    }
    auto weight = [&](int j) -> unsigned {
        const unsigned char *fl = flags + (size_t)(jbase + j) * nkb;
        unsigned w = 0;
        if (seq == 0) {
            for (int g = 0; g < ng; ++g) w += (fl[2 * g] | fl[2 * g + 1]) != 0;
        } else {
            for (int q = 0; q < gw; ++q) w += fl[gw * gsel + q] != 0;
        }
        return w;
    };
    const int run = (nz + kBoundsThreads - 1) / kBoundsThreads;          // slices per thread
    const int j0 = min(tid * run, nz), j1 = min(j0 + run, nz);
    unsigned mine = 0;
    for (int j = j0; j < j1; ++j) mine += weight(j);
    // exclusive block scan of `mine` -> E(j0)
    __shared__ unsigned wsum[kBoundsThreads / 32];
    unsigned inc = mine;
    const int lane = tid & 31, wid = tid >> 5;
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned v = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += v;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    unsigned before = 0, tot = 0;
    for (int w = 0; w < kBoundsThreads / 32; ++w) {
        if (w < wid) before += wsum[w];
        tot += wsum[w];
    }
    const long long total = tot;
    auto target = [&](int sidx) { return (total * sidx) / ns; };
    long long E = (long long)before + (inc - mine);                      // E(j0)
    // slice j (or the weightless last slice j = nz) receives the bounds with E(j - 1) < target <= E(j), E(-1) = -1
    auto place = [&](int j, long long lo, long long hi) {
        if (lo >= hi) return;
        int sidx = total > 0 ? (int)(((lo + 1) * ns) / total) : 0;
        if (sidx > ns) sidx = ns;
        while (sidx > 0 && target(sidx - 1) > lo) --sidx;
        while (sidx < ns && target(sidx) <= lo) ++sidx;
        for (; sidx < ns && target(sidx) <= hi; ++sidx) out[sidx] = jbase + j;
    };
    // this thread's slices j0 .. j1-1: E(j) for j = j0 is E; E(j - 1) for j0 is E minus the weight of slice j0 - 1
    long long prev = j0 == 0 ? -1 : E - (long long)weight(j0 - 1);
    for (int j = j0; j < j1; ++j) {
        place(j, prev, E);
        prev = E;
        E += weight(j);
    }
    if (j0 < nz && j1 == nz) place(nz, prev, E);                         // the thread owning the last slice: E(nz) = total
    if (nz == 0 && tid == 0) place(0, -1, 0);
    if (tid == 0) out[ns] = jbase + nz;
}

// ------------------------------------------------------------------------------------------------ stage X
// H_j[a, y] = sum_x rho~_j[y, x] e^{i qx[a] x}: the streamed-A x resident-B pipeline of tc_cgemm.cuh.  A unit = one live 128-y row tile
// of a slice (rows y = TMEM lanes, K = x); the resident operand = NX rows per CTA of the Ex tile of 2 NX grid columns a
// (NX * NXP * 8 bytes <= 128 KB: NX = 64 / 32 / 16 for N_x <= 256 / 512 / 1024).  A work item = (column tile, balanced z range);
// the pair takes two consecutive live tiles (an odd last one is run twice, the peer's copy discarded).  The epilogue rescales the
// accumulator by the constant 2^(-9 - ceil(log2 N_x)) (|H| <= 2^14.5 whatever the data), splits it hi / lo and stores H as the
// planes [4][N_z][NPXP][NY], y fastest = K-major for stage YZ (a warp stores 32 consecutive y).
struct SepXParams {
    int nk;                                     // NXP / 64
    int nz, NY, NPXP, ng, nta, nsx, nkb;        // nta = tiles of 2 NX columns, nsx = z splits, nkb = NY / 64
    int ncols;                                  // columns a < ncols are stored (the NUFFT route's stage Y reads no others)
    float hscale;                               // 2^(-9 - L): accumulator (2^10 sR H) -> stored H (sH H)
    const unsigned char *flags;                 // [nz][nkb]
    const int *zb;                              // [nsx + 1] balanced z split bounds (sep_tc_bounds_kernel)
    __half *Hp;                                 // [4][nz][NPXP][NY]
};

template <int NX>
struct SepXPolicy {
    static constexpr int NB = NX;
    static constexpr bool kUnrollEpilogue = false;
    static constexpr int kEpilogueRegs = 0;
    using Params = SepXParams;
    struct Item {
        int ta, z0, z1;
    };
    __device__ static int nitems(const Params &P) { return P.nta * P.nsx; }
    __device__ static Item item(const Params &P, int index) {
        Item it;
        it.ta = index % P.nta;   // column tiles fastest: concurrent pairs stream the same rho~ tiles
        const int sp = index / P.nta;
        it.z0 = __ldg(P.zb + sp);
        it.z1 = __ldg(P.zb + sp + 1);
        return it;
    }
    __device__ static int b_row0(const Params &, const Item &it) { return it.ta * 2 * NX; }
    // unit id = slice * ng + 128-y group
    struct Units {
        LiveUnits lu;
        int base;
        __device__ void begin(const Params &P, const Item &it, int lane) {
            lu.begin(P.flags, P.nkb, it.z0, it.z1, P.ng, 0, lane);
            base = it.z0 * P.ng;
        }
        __device__ bool next(int &u0, int &u1, bool &dup, uint32_t &kmask) {
            kmask = 0xffffffffu;
            int n0, n1;
            uint32_t f;
            if (!lu.next(n0, f)) return false;
            dup = !lu.next(n1, f);
            u0 = base + n0;
            u1 = dup ? u0 : base + n1;
            return true;
        }
    };
    __device__ static void a_coords(const Params &P, const Item &, int unit, int kb, int (&c)[3]) {
        c[0] = kb * kKB;
        c[1] = (unit / P.ng) * P.NY + (unit % P.ng) * kM;
        c[2] = 0;
    }
    struct Epilogue {
        __half *dst;
        size_t plane;
        int ncol;            // columns of this thread's range that are stored
        __device__ void begin(const Params &P, const Item &, const tcg::EpiThread &) { plane = (size_t)P.nz * P.NPXP * P.NY; }
        __device__ void unit_begin(const Params &P, const Item &it, const tcg::EpiThread &et, int unit) {
            const int j = unit / P.ng, g = unit % P.ng;
            SCATMAN_ASSERT(j >= 0 && j < P.nz && it.ta * 2 * NX + et.col0 + NX <= P.NPXP && g * kM + kM <= P.NY);
            dst = P.Hp + ((size_t)j * P.NPXP + it.ta * 2 * NX + et.col0) * P.NY + g * kM + et.lane_row;
            ncol = P.ncols - (it.ta * 2 * NX + et.col0);
        }
        __device__ __forceinline__ void columns(const Params &P, const Item &, const tcg::EpiThread &, int, int c0,
                                                const uint32_t (&gre)[8], const uint32_t (&gim)[8]) {
            if (c0 >= ncol) return;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (c0 + i >= ncol) break;
                __half h[4];
                split4(__uint_as_float(gre[i]) * P.hscale, __uint_as_float(gim[i]) * P.hscale, h);
                __half *d = dst + (size_t)(c0 + i) * P.NY;
#pragma unroll
                for (int pl = 0; pl < 4; ++pl) d[pl * plane] = h[pl];
            }
        }
        __device__ void end(const Params &, const Item &, const tcg::EpiThread &) {}
    };
};

// ------------------------------------------------------------------------------------------------ stage YZ
struct SepYzParams {
    int nk;                       // NY / 64 (K blocks of the transposed form)
    int nz, nb, npx, npy, NY, NPXP, ng, nzs, ntb, nta, nkb;   // nz: slices per item, nb: items of the chunk, nkb = NY / 64; ntb / nta: 128-row b / a tiles
    int ntap, ntbn;               // transposed form: pairs of a tiles, tiles of 2 NB grid rows
    double k, dz;
    const double *qx, *qy;
    const unsigned char *flags;   // [nz][nkb]
    const int *zb;                // [nb][nzs + 1] balanced z split bounds (global slice indices) per item
    float2 *partial;              // [nb][nzs][npy][npx]
};

// ---- stage YZ with one accumulator per slice: both operands streamed -------------------------------------------------------
// With the Ey tile resident, a slice needs one accumulator pass PER 128-y group, and the per-element slice phase of the epilogue
// (two SFU calls for every accumulator element) then costs more than the group's MMAs: measured, the issuers wait 38 % of the
// kernel for an accumulator buffer.  Here a unit is a whole slice: every live 64-y block of it is one stage holding this CTA's
// Ey block (4 planes x 16 KB) AND its half of the H block (4 x 8 KB), 96 KB, two stages.  Ey is re-streamed for every slice (from
// L2: the tables are ~1 MB), which triples the L2 -> SM traffic and halves the epilogue work and the partial sums.  CTA pairs
// only (cta_group::2, UMMA 256 x 128 x 16), slices of at most 32 blocks (N_y <= 2048); other cases use sep_tc_yz128_kernel.
struct LiveSlices {   // the live slices of a z range with the bit mask of their live 64-y blocks, warp-cooperative as LiveUnits
    const unsigned char *fl;
    int nkb, z0, total, base, lane;
    uint32_t cur, ahead, live;
    __device__ __forceinline__ uint32_t load(int n) const {
        if (n >= total) return 0u;
        const unsigned char *p = fl + (size_t)(z0 + n) * nkb;
        uint32_t m = 0u;
        for (int kb = 0; kb < nkb; ++kb) m |= (uint32_t)(__ldg(p + kb) != 0) << kb;
        return m;
    }
    __device__ __forceinline__ void begin(const unsigned char *flags, int nkb_, int z0_, int z1, int lane_) {
        fl = flags; nkb = nkb_; z0 = z0_; lane = lane_;
        total = z1 - z0_;
        base = 0;
        cur = load(lane);
        ahead = load(32 + lane);
        live = __ballot_sync(0xffffffffu, cur != 0u);
    }
    __device__ __forceinline__ bool next(int &n, uint32_t &m) {
        while (live == 0u) {
            base += 32;
            if (base >= total) return false;
            cur = ahead;
            ahead = load(base + 32 + lane);
            live = __ballot_sync(0xffffffffu, cur != 0u);
        }
        const int pos = __ffs((int)live) - 1;
        live &= live - 1;
        m = __shfl_sync(0xffffffffu, cur, pos);
        n = base + pos;
        return true;
    }
};

__global__ void __launch_bounds__(kThreadsTc, 1)
sep_tc_yzs_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const SepYzParams P) {
    constexpr int kN = 128;
    constexpr int kPartA = 4 * kSlotA;                // 65536: this CTA's Ey block, four planes
    constexpr int kSlotB = kSlotA / 2;                // 8192: this CTA's half (64 rows) of one plane of an H block
    constexpr int kStage = kPartA + 4 * kSlotB;       // 98304
    constexpr int kStages = 2;
    constexpr int kNB = 2;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sS = smem;
    uint64_t *bars = (uint64_t *)(smem + kStages * kStage);
    uint64_t *s_full = bars + 0, *s_empty = s_full + kStages;
    uint64_t *t_full = s_empty + kStages, *t_empty = t_full + kNB, *first_done = t_empty + kNB;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + kNB);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    const bool leader = rank == 0;
    const int cluster_id = blockIdx.x / 2, nclusters = gridDim.x / 2;
    const int ntp = P.ntb / 2;
    const int nitems = ntp * P.nta * P.nzs * P.nb;   // item -> (tile pair tp, a tile, z split, batch item); no y groups

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(s_full + i, 1);
            ptx::mbar_init(s_empty + i, 2);
        }
        for (int i = 0; i < kNB; ++i) {
            ptx::mbar_init(t_full + i, 2);
            ptx::mbar_init(t_empty + i, 16);
            ptx::mbar_init(first_done + i, 1);
        }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) ptx::tmem_alloc_2sm(tmem_ptr, kTmemColsTc);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync_all();
    ptx::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);

    auto decode = [&](int item, int &tb, int &ta, int &sp, int &bi) {
        tb = (item % ntp) * 2 + (int)rank;
        item /= ntp;
        ta = item % P.nta;
        item /= P.nta;
        sp = item % P.nzs;
        bi = item / P.nzs;
    };
    auto zrange = [&](int bi, int sp, int &z0, int &z1) {   // global slice indices
        const int *zb = P.zb + (size_t)bi * (P.nzs + 1) + sp;
        z0 = __ldg(zb);
        z1 = __ldg(zb + 1);
    };

    if (warp < 4) {
      tcg::setmaxnreg_dec_48();
      if (warp == 0) {
        // ===================================================================== TMA producer (both CTAs)
        int slot = 0;
        uint32_t phase = 0;
        for (int item = cluster_id; item < nitems; item += nclusters) {
            int tb, ta, sp, bi;
            decode(item, tb, ta, sp, bi);
            int z0, z1;
            zrange(bi, sp, z0, z1);
            LiveSlices un;
            un.begin(P.flags, P.nkb, z0, z1, lane);
            int n;
            uint32_t m;
            while (un.next(n, m)) {
                const int j = z0 + n;
                for (int kb = 0; kb < P.nkb; ++kb) {
                    if (((m >> kb) & 1u) == 0u) continue;
                    ptx::mbar_wait(s_empty + slot, phase ^ 1);
                    if (ptx::elect_one()) {
                        if (leader) ptx::mbar_arrive_expect_tx(s_full + slot, (uint32_t)(2 * kStage));   // both CTAs' parts
                        uint8_t *st = sS + slot * kStage;
                        const int row = j * P.NPXP + ta * kN + (int)rank * (kN / 2);
#pragma unroll
                        for (int pl = 0; pl < 4; ++pl) {
                            ptx::tma_load_3d_2sm(st + pl * kSlotA, &tmA, s_full + slot, kb * kKB, tb * kM, pl);
                            ptx::tma_load_3d_2sm(st + kPartA + pl * kSlotB, &tmB, s_full + slot, kb * kKB, row, pl);
                        }
                    }
                    __syncwarp();
                    if (++slot == kStages) { slot = 0; phase ^= 1; }
                }
            }
        }
      } else if ((warp == 1 || warp == 3) && leader) {
        // ===================================================================== MMA issuers (leader; k-step ks belongs to issuer ks % 2)
        constexpr uint32_t idesc_pos = ptx::umma_idesc_f16(2 * kM, kN, false);
        constexpr uint32_t idesc_neg = ptx::umma_idesc_f16(2 * kM, kN, true);
        const uint64_t descS0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sS));
        constexpr uint64_t kA = kSlotA >> 4, kB = kSlotB >> 4, kSt = kStage >> 4, kPa = kPartA >> 4;
        const int iw = warp >> 1;
        int slot = 0;
        uint32_t phase = 0, u = 0;
        for (int item = cluster_id; item < nitems; item += nclusters) {
            int tb, ta, sp, bi;
            decode(item, tb, ta, sp, bi);
            int z0, z1;
            zrange(bi, sp, z0, z1);
            LiveSlices un;
            un.begin(P.flags, P.nkb, z0, z1, lane);
            int n;
            uint32_t m;
            while (un.next(n, m)) {
                const uint32_t buf = u % kNB, upar = (u / kNB) & 1;
                ptx::mbar_wait(t_empty + buf, upar ^ 1);
                ptx::tc_fence_after();
                const uint32_t d_re = tmem_base + buf * 256, d_im = d_re + 128;
                bool first = true;
                for (int kb = 0; kb < P.nkb; ++kb) {
                    if (((m >> kb) & 1u) == 0u) continue;
                    if (first && iw == 1) {   // D must have been initialised by issuer 0's first k-step
                        ptx::mbar_wait(first_done + buf, upar);
                        ptx::tc_fence_after();
                    }
                    ptx::mbar_wait(s_full + slot, phase);
                    ptx::tc_fence_after();
                    if (ptx::elect_one()) {
#pragma unroll
                        for (int kk = 0; kk < 2; ++kk) {
                            const int ks = 2 * kk + iw;
                            const uint64_t a_reh = descS0 + (uint64_t)slot * kSt + (uint64_t)(ks * 2);
                            const uint64_t a_rel = a_reh + kA, a_imh = a_rel + kA, a_iml = a_imh + kA;
                            const uint64_t b_reh = descS0 + (uint64_t)slot * kSt + kPa + (uint64_t)(ks * 2);
                            const uint64_t b_rel = b_reh + kB, b_imh = b_rel + kB, b_iml = b_imh + kB;
                            const uint32_t acc0 = (first && ks == 0) ? 0u : 1u;
                            ptx::umma_f16_2sm(d_re, a_reh, b_reh, idesc_pos, acc0);
                            ptx::umma_f16_2sm(d_im, a_imh, b_reh, idesc_pos, acc0);
                            ptx::umma_f16_2sm(d_re, a_rel, b_reh, idesc_pos, 1u);
                            ptx::umma_f16_2sm(d_im, a_iml, b_reh, idesc_pos, 1u);
                            ptx::umma_f16_2sm(d_re, a_reh, b_rel, idesc_pos, 1u);
                            ptx::umma_f16_2sm(d_im, a_imh, b_rel, idesc_pos, 1u);
                            ptx::umma_f16_2sm(d_re, a_imh, b_imh, idesc_neg, 1u);
                            ptx::umma_f16_2sm(d_im, a_reh, b_imh, idesc_pos, 1u);
                            ptx::umma_f16_2sm(d_re, a_iml, b_imh, idesc_neg, 1u);
                            ptx::umma_f16_2sm(d_im, a_rel, b_imh, idesc_pos, 1u);
                            ptx::umma_f16_2sm(d_re, a_imh, b_iml, idesc_neg, 1u);
                            ptx::umma_f16_2sm(d_im, a_reh, b_iml, idesc_pos, 1u);
                            if (first && iw == 0 && kk == 0) ptx::umma_commit_2sm(first_done + buf, (uint16_t)0x1);
                        }
                        ptx::umma_commit_2sm(s_empty + slot, (uint16_t)0x3);
                    }
                    __syncwarp();
                    first = false;
                    if (++slot == kStages) { slot = 0; phase ^= 1; }
                }
                if (ptx::elect_one()) ptx::umma_commit_2sm(t_full + buf, (uint16_t)0x3);
                __syncwarp();
                ++u;
            }
        }
      }
    } else {
        tcg::setmaxnreg_inc<224>();
        // ===================================================================== epilogue: Blocks 7-8, 64 columns per thread
        const int lg = warp & 3, ch = (warp - 4) >> 2;
        const uint32_t t_lane = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(ch * 64);
        uint32_t u = 0;
        for (int item = cluster_id; item < nitems; item += nclusters) {
            int tb, ta, sp, bi;
            decode(item, tb, ta, sp, bi);
            const int b = tb * kM + lg * 32 + lane;
            const int a0 = ta * kN + ch * 64;
            const double qyb = b < P.npy ? P.qy[b] : 0.0;
            uint32_t dph[64];
#pragma unroll
            for (int c = 0; c < 64; ++c) {
                const int a = a0 + c;
                double t = 0.0;
                if (a < P.npx && b < P.npy) {
                    const double qxa = P.qx[a];
                    const double qxy2 = qxa * qxa + qyb * qyb;
                    const double kz2 = P.k * P.k - qxy2;
                    const double qz = kz2 >= 0.0 ? -qxy2 / (P.k + sqrt(kz2)) : 0.0;
                    t = qz * P.dz * (0.25 / 3.14159265358979323846);
                    t -= rint(t);
                }
                dph[c] = (uint32_t)(long long)rint(t * 4294967296.0);
            }
            float2 tot[64];
#pragma unroll
            for (int c = 0; c < 64; ++c) tot[c] = make_float2(0.f, 0.f);
            int z0, z1;
            zrange(bi, sp, z0, z1);
            LiveSlices un;
            un.begin(P.flags, P.nkb, z0, z1, lane);
            int n;
            uint32_t m;
            while (un.next(n, m)) {
                const int j = z0 + n - bi * P.nz;
                const uint32_t buf = u % kNB, upar = (u / kNB) & 1;
                const uint32_t mult = (uint32_t)(2 * j - P.nz + 1);
                ptx::mbar_wait(t_full + buf, upar);
                ptx::tc_fence_after();
                const uint32_t t_re = t_lane + buf * 256, t_im = t_re + 128;
#pragma unroll
                for (int q8 = 0; q8 < 8; ++q8) {
                    uint32_t gre[8], gim[8];
                    ptx::tmem_ld8(t_re + q8 * 8, gre);
                    ptx::tmem_ld8(t_im + q8 * 8, gim);
                    ptx::tmem_ld_wait();
                    if (q8 == 7) {
                        ptx::tc_fence_before();
                        __syncwarp();
                        if (lane == 0) ptx::mbar_arrive_cluster(t_empty + buf, 0);   // the leader's barrier
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int c = q8 * 8 + i;
                        const float ang = (float)(int)(dph[c] * mult) * 1.4629180792671596e-9f;   // pi / 2^31
                        float sn, cs;
                        __sincosf(ang, &sn, &cs);
                        const float gr = __uint_as_float(gre[i]), gi = __uint_as_float(gim[i]);
                        tot[c].x = fmaf(cs, gr, tot[c].x);
                        tot[c].x = fmaf(-sn, gi, tot[c].x);
                        tot[c].y = fmaf(cs, gi, tot[c].y);
                        tot[c].y = fmaf(sn, gr, tot[c].y);
                    }
                }
                ++u;
            }
            if (b < P.npy) {
                float2 *dst = P.partial + (((size_t)bi * P.nzs + sp) * P.npy + b) * P.npx;
#pragma unroll
                for (int c = 0; c < 64; ++c)
                    if (a0 + c < P.npx) dst[a0 + c] = tot[c];
            }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync_all();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_2sm(tmem_base, kTmemColsTc);
    }
}

// ---- stage YZ transposed: D^T[a, b] = sum_y H_j[a, y] Ey[b, y], the Ey tile resident for ALL y -----------------------------
// The same pipeline (tc_cgemm.cuh): the streamed A operand is each CTA's own H tile (128 grid columns a = the TMEM lanes), the
// resident B operand this CTA's NB rows of the Ey tile of 2 NB grid rows b for every 64-y block (NB nkb 8 KB <= 128 KB: NB = 64 for
// N_y <= 256, the only instance built; NB = 32 for N_y <= 512 ran UMMA N = 64 and measured slower than the streamed form).  A work
// item = (pair of a tiles, b tile, z range, batch item); a unit = (live slice, a tile): the pair takes the two a tiles of the
// same slice (an odd last a tile is run twice and the copy discarded), and 64-y blocks of a slice that hold nothing are never
// loaded.  One accumulator per slice, so the epilogue -- Blocks 7-8: slice phase, sum over slices -- runs once per slice; its
// thread owns one column a and NB rows b: 2 NB running totals + NB phase fractions, hence the setmaxnreg re-split (224 registers).
template <int NB_>
struct SepYztPolicy {
    static constexpr int NB = NB_;
    static constexpr bool kUnrollEpilogue = true;
    static constexpr int kEpilogueRegs = 224;
    using Params = SepYzParams;
    struct Item {
        int ta0, tbn, sp, bi, z0, z1;
    };
    __device__ static int nitems(const Params &P) { return P.ntap * P.ntbn * P.nzs * P.nb; }
    __device__ static Item item(const Params &P, int index) {   // a pairs fastest: neighbours share the Ey tile
        Item it;
        it.ta0 = (index % P.ntap) * 2;
        index /= P.ntap;
        it.tbn = index % P.ntbn;
        index /= P.ntbn;
        it.sp = index % P.nzs;
        it.bi = index / P.nzs;
        const int *zb = P.zb + (size_t)it.bi * (P.nzs + 1) + it.sp;
        it.z0 = __ldg(zb);
        it.z1 = __ldg(zb + 1);
        return it;
    }
    __device__ static int b_row0(const Params &, const Item &it) { return it.tbn * 2 * NB; }
    // unit id = global slice * nta + a tile
    struct Units {
        LiveSlices ls;
        int z0, ta0, nta;
        __device__ void begin(const Params &P, const Item &it, int lane) {
            ls.begin(P.flags, P.nkb, it.z0, it.z1, lane);
            z0 = it.z0; ta0 = it.ta0; nta = P.nta;
        }
        __device__ bool next(int &u0, int &u1, bool &dup, uint32_t &kmask) {
            int n;
            if (!ls.next(n, kmask)) return false;
            u0 = (z0 + n) * nta + ta0;
            dup = ta0 + 1 >= nta;
            u1 = dup ? u0 : u0 + 1;
            return true;
        }
    };
    __device__ static void a_coords(const Params &P, const Item &, int unit, int kb, int (&c)[3]) {
        c[0] = kb * kKB;
        c[1] = (unit / P.nta) * P.NPXP + (unit % P.nta) * kM;
        c[2] = 0;
    }
    struct Epilogue {
        uint32_t dph[NB], mult;
        float2 tot[NB];
        int a, b0;
        __device__ __forceinline__ void begin(const Params &P, const Item &it, const tcg::EpiThread &et) {
            const int ta = it.ta0 + ((et.rank != 0 && it.ta0 + 1 < P.nta) ? 1 : 0);
            a = ta * kM + et.lane_row;
            b0 = it.tbn * 2 * NB + et.col0;
            const double qxa = a < P.npx ? P.qx[a] : 0.0;
#pragma unroll
            for (int c = 0; c < NB; ++c) {
                const int b = b0 + c;
                double t = 0.0;
                if (a < P.npx && b < P.npy) {
                    const double qyb = P.qy[b];
                    const double qxy2 = qxa * qxa + qyb * qyb;
                    const double kz2 = P.k * P.k - qxy2;
                    // qz = -(k - sqrt(k^2 - qxy^2)) = -qxy^2 / (k + sqrt(k^2 - qxy^2)): no cancellation near forward
                    const double qz = kz2 >= 0.0 ? -qxy2 / (P.k + sqrt(kz2)) : 0.0;
                    t = qz * P.dz * (0.25 / 3.14159265358979323846);
                    t -= rint(t);
                }
                dph[c] = (uint32_t)(long long)rint(t * 4294967296.0);
                tot[c] = make_float2(0.f, 0.f);
            }
        }
        __device__ __forceinline__ void unit_begin(const Params &P, const Item &it, const tcg::EpiThread &, int unit) {
            const int j = unit / P.nta - it.bi * P.nz;   // slice within its item
            SCATMAN_ASSERT(j >= 0 && j < P.nz && it.bi < P.nb && it.sp < P.nzs);
            mult = (uint32_t)(2 * j - P.nz + 1);
        }
        __device__ __forceinline__ void columns(const Params &, const Item &, const tcg::EpiThread &, int, int c0,
                                                const uint32_t (&gre)[8], const uint32_t (&gim)[8]) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int c = c0 + i;
                const float ang = (float)(int)(dph[c] * mult) * 1.4629180792671596e-9f;   // pi / 2^31
                float sn, cs;
                __sincosf(ang, &sn, &cs);
                const float gr = __uint_as_float(gre[i]), gi = __uint_as_float(gim[i]);
                tot[c].x = fmaf(cs, gr, tot[c].x);
                tot[c].x = fmaf(-sn, gi, tot[c].x);
                tot[c].y = fmaf(cs, gi, tot[c].y);
                tot[c].y = fmaf(sn, gr, tot[c].y);
            }
        }
        __device__ __forceinline__ void end(const Params &P, const Item &it, const tcg::EpiThread &et) {
            if (et.rank != 0 && it.ta0 + 1 >= P.nta) return;   // the peer repeated the leader's tile
            if (a < P.npx) {   // a warp stores 32 consecutive a of one grid row
                float2 *dst = P.partial + ((size_t)it.bi * P.nzs + it.sp) * P.npy * P.npx + a;
#pragma unroll
                for (int c = 0; c < NB; ++c)
                    if (b0 + c < P.npy) dst[(size_t)(b0 + c) * P.npx] = tot[c];
            }
        }
    };
};

// I[b][a] = |ampscale * sum of partials|^2; evanescent grid points (qx^2 + qy^2 > k^2: no scattering direction) give 0
__global__ void sep_tc_finalize_kernel(const float2 *__restrict__ partial, const double *__restrict__ qx,
                                       const double *__restrict__ qy, double k, int npx, int npy, int nsplit,
                                       const float *__restrict__ ampscale, float *__restrict__ I) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int item = blockIdx.y;
    const size_t npix = (size_t)npx * npy;
    if (p >= (int64_t)npix) return;
    const int a = (int)(p % npx), b = (int)(p / npx);
    const float2 *part = partial + (size_t)item * nsplit * npix;
    float re = 0.f, im = 0.f;
    for (int s = 0; s < nsplit; ++s) {
        const float2 v = part[(size_t)s * npix + p];
        re += v.x;
        im += v.y;
    }
    const float sc = ampscale[item];
    re *= sc;
    im *= sc;
    const bool real = qx[a] * qx[a] + qy[b] * qy[b] <= k * k;
    I[(size_t)item * npix + p] = real ? re * re + im * im : 0.f;
}

// ------------------------------------------------------------------------------------------------ host
SepTcPlan make_sep_tc_plan(const Plan &p, int npx, int npy, int num_sms) {
    SepTcPlan t;
    t.NY = (p.ny + 127) / 128 * 128;
    t.NXP = (p.nx + kKB - 1) / kKB * kKB;
    t.nyz = 128;                                  // stage YZ accumulator width (columns a per tile)
    t.NPXP = (npx + kM - 1) / kM * kM;            // whole 128-column tiles: stage X's tiles of 2 NX columns and stage YZ's a tiles divide it
    t.ng = t.NY / 128;
    int L = 0;
    while ((1 << L) < p.nx) ++L;
    t.L = L;
    // Stage YZ, in order of preference:
    //   transposed (SepYztPolicy<64>)  pairs of a tiles, Ey resident for all y: N_y <= 256
    //   streamed   (sep_tc_yzs_kernel) pairs of b tiles, both operands streamed: N_y <= 2048 (taller grids use the CUDA-core stages)
    t.yzt_nb = t.NY / kKB <= 4 ? 64 : 0;
    t.yz_t = t.yzt_nb != 0;
    t.yz_stream = true;                           // both forms: one accumulator per slice, z-split bounds and partial sums per item
    t.yz_ncta = 2;
    // the streamed form pairs b tiles: an odd count is padded by one all-zero tile of Ey rows
    t.NPYP = (npy + kM - 1) / kM * kM;
    if (!t.yz_t && (t.NPYP / kM) % 2 != 0) t.NPYP += kM;
    // items per chunk (stacked along z, one set of launches per chunk): as many as keep the H planes of a chunk under 4 GB
    const size_t h_item = (size_t)8 * p.nz * t.NPXP * t.NY;
    size_t nb = ((size_t)4 << 30) / (h_item ? h_item : 1);
    if (nb > (size_t)p.batch) nb = (size_t)p.batch;
    if (nb * p.nz > 60000) nb = 60000 / (size_t)p.nz;   // global slice index and TMA row coordinates stay small
    t.nb = nb < 1 ? 1 : (int)nb;
    // z splits: minimise waves x (slices per item + ~3 slice-equivalents of fill: Ey tile load, pipeline ramp, partial store)
    const int base = t.yz_t ? ((t.NPXP / kM + 1) / 2) * (t.NPYP / (2 * t.yzt_nb)) * t.nb : (t.NPYP / kM / 2) * (t.NPXP / t.nyz) * t.nb;
    const int workers = num_sms / 2;
    int best = 1;
    double best_cost = 1e300;
    const int max_z = p.nz < 32 ? p.nz : 32;
    for (int z = 1; z <= max_z; ++z) {
        const long long items = (long long)base * z;
        const long long waves = (items + workers - 1) / workers;
        const double cost = (double)waves * ((double)((p.nz + z - 1) / z) + 3.0);
        if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; best = z; }
    }
    t.nzs = best;
    t.nsplit = t.nzs;
    // stage X: a columns per resident Ex tile (NX * NXP * 8 bytes <= 128 KB), z splits for two balanced items per CTA pair
    t.NX = t.NXP <= 256 ? 64 : t.NXP <= 512 ? 32 : 16;
    t.x_ncta = 2;
    const int nta = t.NPXP / (2 * t.NX);
    int nsx = (2 * (num_sms / 2) + nta - 1) / nta;
    t.nsx = nsx < 1 ? 1 : nsx > p.nz * t.nb ? p.nz * t.nb : nsx;
    return t;
}

constexpr int kSmemYzs = 1024 + 2 * (4 * kSlotA + 4 * (kSlotA / 2)) + 256;   // streamed stage YZ: two stages of 96 KB

// Function attributes belong to a device's context: set for the CURRENT device by scatman_create.
cudaError_t sep_tc_init_device() {
    cudaError_t e = cudaFuncSetAttribute(sep_tc_yzs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemYzs);
    if (e == cudaSuccess) e = tcg::cgemm_init_device<SepYztPolicy<64>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<SepXPolicy<64>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<SepXPolicy<32>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<SepXPolicy<16>>();
    return e;
}

cudaError_t launch_sep_tc_tables(const double *d_qx, int npx, const double *d_qy, int npy, const Plan &p,
                                 const SepTcPlan &t, __half *d_Exp, __half *d_Eyp, cudaStream_t st) {
    const int64_t nye = (int64_t)t.NPYP * t.NY;
    sep_tc_table_kernel<<<(unsigned)((nye + 255) / 256), 256, 0, st>>>(d_qy, npy, t.NPYP, p.ny, t.NY, p.dy, d_Eyp);
    const int64_t nxe = (int64_t)t.NPXP * t.NXP;
    sep_tc_table_kernel<<<(unsigned)((nxe + 255) / 256), 256, 0, st>>>(d_qx, npx, t.NPXP, p.nx, t.NXP, p.dx, d_Exp);
    return cudaGetLastError();
}

cudaError_t launch_sep_tc_yz(const Plan &p, const SepTcPlan &t, const __half *d_Eyp, const __half *d_Hp,
                             const unsigned char *d_flags64, const int *d_bounds, int nb, const double *d_qx, int npx,
                             const double *d_qy, int npy, float2 *d_partial, int num_sms, cudaStream_t st, std::string *err) {
    SepYzParams P;
    P.nk = t.NY / kKB;
    P.nz = p.nz; P.nb = nb; P.npx = npx; P.npy = npy; P.NY = t.NY; P.NPXP = t.NPXP; P.ng = t.ng; P.nzs = t.nzs;
    P.ntb = t.NPYP / kM; P.nta = t.NPXP / kM; P.nkb = t.NY / kKB;
    P.ntap = (P.nta + 1) / 2;
    P.ntbn = t.yz_t ? t.NPYP / (2 * t.yzt_nb) : 0;
    P.k = 2.0 * 3.14159265358979323846 / p.lambda; P.dz = p.dz;
    P.qx = d_qx; P.qy = d_qy; P.flags = d_flags64; P.zb = d_bounds + (t.nsx + 1); P.partial = d_partial;
    const cuuint64_t hrows = (cuuint64_t)p.nz * nb * t.NPXP;
    CUtensorMap tmA, tmB;
    bool ok;
    if (t.yz_t) {
        // streamed operand: the H planes [4][slices NPXP][NY], box = 64 y x a whole 128-column a tile; resident: the Ey planes,
        // box = this CTA's NB rows of one 64-y block
        cuuint64_t dimsA[4] = {(cuuint64_t)t.NY, hrows, 1, 4};
        cuuint64_t stridesA[3] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * hrows * 2, (cuuint64_t)t.NY * hrows * 2};
        cuuint32_t boxA[4] = {(cuuint32_t)kKB, (cuuint32_t)kM, 1, 1};
        cuuint64_t dimsB[3] = {(cuuint64_t)t.NY, (cuuint64_t)t.NPYP, 4};
        cuuint64_t stridesB[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * (cuuint64_t)t.NPYP * 2};
        cuuint32_t boxB[3] = {(cuuint32_t)kKB, (cuuint32_t)t.yzt_nb, 1};
        ok = encode_map(&tmA, d_Hp, 4, dimsA, stridesA, boxA, CU_TENSOR_MAP_SWIZZLE_128B) &&
             encode_map(&tmB, d_Eyp, 3, dimsB, stridesB, boxB, CU_TENSOR_MAP_SWIZZLE_128B);
        if (!ok) {
            if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
            return cudaErrorUnknown;
        }
        return tcg::cgemm_launch<SepYztPolicy<64>>(tmA, tmB, P, P.ntap * P.ntbn * P.nzs * nb, num_sms, st);
    }
    {   // streamed form: A = Ey planes (box = a 128-row b tile), B = H planes (box = this CTA's 64 rows of an a tile)
        cuuint64_t dims[3] = {(cuuint64_t)t.NY, (cuuint64_t)t.NPYP, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * (cuuint64_t)t.NPYP * 2};
        cuuint32_t box[3] = {(cuuint32_t)kKB, (cuuint32_t)kM, 1};
        ok = encode_map(&tmA, d_Eyp, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (ok) {
        cuuint64_t dims[3] = {(cuuint64_t)t.NY, hrows, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * hrows * 2};
        cuuint32_t box[3] = {(cuuint32_t)kKB, (cuuint32_t)(t.nyz / 2), 1};
        ok = encode_map(&tmB, d_Hp, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (!ok) {
        if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
        return cudaErrorUnknown;
    }
    const int nit = (P.ntb / 2) * P.nta * P.nzs * nb, maxc = num_sms / 2;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(2 * (nit < maxc ? nit : maxc)));
    cfg.blockDim = dim3(kThreadsTc);
    cfg.dynamicSmemBytes = kSmemYzs;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, sep_tc_yzs_kernel, tmA, tmB, P);
}

cudaError_t launch_sep_tc_prefix_prep(const float2 *d_dn, const unsigned *d_maxbits, const Plan &p, const SepTcPlan &t, int nb,
                                      __half *d_Rp, unsigned char *d_flags64, int *d_bounds, float *d_ampscale, cudaStream_t st,
                                      bool x_only, const unsigned char *d_tilemap, unsigned char *d_layer_live) {
    const int nyb = t.NY / kKB, nzt = p.nz * nb;
    if (d_tilemap && d_layer_live) {
        const int layers = nb * ((p.nz + 3) / 4), tiles = ((p.ny + 3) / 4) * ((p.nx + 15) / 16);
        tile_layers_kernel<<<layers, 128, 0, st>>>(d_tilemap, tiles, d_layer_live);
    } else {
        d_layer_live = nullptr;
    }
    cudaError_t e = cudaMemsetAsync(d_flags64, 0, (size_t)nzt * nyb, st);
    if (e != cudaSuccess) return e;
    const double kdz = 2.0 * 3.14159265358979323846 / p.lambda * p.dz;
    if (p.nx % 2 == 0) {
        dim3 grid((unsigned)(((size_t)(t.NXP / 4) * t.NY + kPrefThreads - 1) / kPrefThreads), (unsigned)nb);
        sep_tc_prefix_planes_kernel<4><<<grid, kPrefThreads, 0, st>>>(d_dn, p.nx, p.ny, p.nz, nb, t.NY, t.NXP, kdz, p.rho_mode, d_maxbits,
                                                                    d_Rp, d_flags64, d_tilemap, d_layer_live);
    } else {
        dim3 grid((unsigned)(((size_t)t.NXP * t.NY + kPrefThreads - 1) / kPrefThreads), (unsigned)nb);
        sep_tc_prefix_planes_kernel<1><<<grid, kPrefThreads, 0, st>>>(d_dn, p.nx, p.ny, p.nz, nb, t.NY, t.NXP, kdz, p.rho_mode, d_maxbits,
                                                                    d_Rp, d_flags64, d_tilemap, d_layer_live);
    }
    sep_tc_scale_kernel<<<(nb + 127) / 128, 128, 0, st>>>(d_maxbits, nb, t.L, (float)(p.dx * p.dy * p.dz), d_ampscale);
    const int ngs = t.yz_stream ? 1 : t.ng, gw = t.yz_stream ? nyb : 2;
    sep_tc_bounds_kernel<<<x_only ? 1 : 1 + nb * ngs, kBoundsThreads, 0, st>>>(d_flags64, p.nz, nzt, nyb, t.ng, ngs, gw, t.nsx, t.nzs,
                                                                              d_bounds, d_bounds + (t.nsx + 1));
    return cudaGetLastError();
}

cudaError_t launch_sep_tc_prep(const float2 *d_rho, const unsigned *d_maxbits, const Plan &p, const SepTcPlan &t, int nb,
                               __half *d_Rp, unsigned char *d_flags64, int *d_bounds, float *d_ampscale, cudaStream_t st,
                               bool x_only) {
    const int nyb = t.NY / kKB, nzt = p.nz * nb;
    cudaError_t e = cudaMemsetAsync(d_flags64, 0, (size_t)nzt * nyb, st);
    if (e != cudaSuccess) return e;
    const int64_t nthreads = (int64_t)nzt * t.NY * (t.NXP / 8);
    sep_tc_pack_rho_kernel<<<(unsigned)((nthreads + 255) / 256), 256, 0, st>>>(d_rho, p.nx, p.ny, p.nz, nzt, t.NY, t.NXP, d_maxbits,
                                                                             d_Rp, d_flags64);
    sep_tc_scale_kernel<<<(nb + 127) / 128, 128, 0, st>>>(d_maxbits, nb, t.L, (float)(p.dx * p.dy * p.dz), d_ampscale);
    const int ngs = t.yz_stream ? 1 : t.ng, gw = t.yz_stream ? nyb : 2;   // stage YZ's z splits: per item, or per item and 128-y group
    sep_tc_bounds_kernel<<<x_only ? 1 : 1 + nb * ngs, kBoundsThreads, 0, st>>>(d_flags64, p.nz, nzt, nyb, t.ng, ngs, gw, t.nsx, t.nzs,
                                                                              d_bounds, d_bounds + (t.nsx + 1));
    return cudaGetLastError();
}

cudaError_t launch_sep_tc_x(const Plan &p, const SepTcPlan &t, const __half *d_Rp, const __half *d_Exp,
                            const unsigned char *d_flags64, const int *d_bounds, int nb, __half *d_Hp, int num_sms,
                            cudaStream_t st, std::string *err, int ncols) {
    CUtensorMap tmA, tmB;
    bool ok;
    {   // streamed: the rho~ planes [4][slices NY][NXP], box = 64 x of a 128-row tile
        const cuuint64_t rows = (cuuint64_t)p.nz * nb * t.NY;
        cuuint64_t dims[4] = {(cuuint64_t)t.NXP, rows, 1, 4};
        cuuint64_t strides[3] = {(cuuint64_t)t.NXP * 2, (cuuint64_t)t.NXP * rows * 2, (cuuint64_t)t.NXP * rows * 2};
        cuuint32_t box[4] = {(cuuint32_t)kKB, (cuuint32_t)kM, 1, 1};
        ok = encode_map(&tmA, d_Rp, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (ok) {   // resident: the Ex planes [4][NPXP][NXP], box = this CTA's NX rows of one 64-x block
        cuuint64_t dims[3] = {(cuuint64_t)t.NXP, (cuuint64_t)t.NPXP, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NXP * 2, (cuuint64_t)t.NXP * (cuuint64_t)t.NPXP * 2};
        cuuint32_t box[3] = {(cuuint32_t)kKB, (cuuint32_t)t.NX, 1};
        ok = encode_map(&tmB, d_Exp, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (!ok) {
        if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
        return cudaErrorUnknown;
    }
    SepXParams P;
    P.nk = t.NXP / kKB;
    P.nz = p.nz * nb; P.NY = t.NY; P.NPXP = t.NPXP; P.ng = t.ng; P.nta = t.NPXP / (2 * t.NX);
    P.nsx = t.nsx;
    P.nkb = t.NY / kKB;
    P.hscale = ldexpf(1.f, -9 - t.L);
    P.flags = d_flags64; P.zb = d_bounds; P.Hp = d_Hp;
    P.ncols = ncols > 0 && ncols < t.NPXP ? ncols : t.NPXP;
    const int nitems = P.nta * P.nsx;
    switch (t.NX) {
        case 64: return tcg::cgemm_launch<SepXPolicy<64>>(tmA, tmB, P, nitems, num_sms, st);
        case 32: return tcg::cgemm_launch<SepXPolicy<32>>(tmA, tmB, P, nitems, num_sms, st);
        default: return tcg::cgemm_launch<SepXPolicy<16>>(tmA, tmB, P, nitems, num_sms, st);
    }
}

cudaError_t launch_sep_tc_finalize(const float2 *d_partial, const double *d_qx, int npx, const double *d_qy, int npy,
                                   const Plan &p, const SepTcPlan &t, int nb, const float *d_ampscale, float *d_I,
                                   cudaStream_t st) {
    const int64_t npix = (int64_t)npx * npy;
    const double k = 2.0 * 3.14159265358979323846 / p.lambda;
    sep_tc_finalize_kernel<<<dim3((unsigned)((npix + 255) / 256), nb), 256, 0, st>>>(d_partial, d_qx, d_qy, k, npx, npy, t.nsplit,
                                                                                    d_ampscale, d_I);
    return cudaGetLastError();
}

}  // namespace scatman
