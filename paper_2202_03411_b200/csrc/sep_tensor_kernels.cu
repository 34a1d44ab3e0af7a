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
// Kernels (each is selected by make_sep_tc_plan and covered by tests/test_gpu_qgrid.py):
//   stage X   sep_tc_x2_kernel<NX>  CTA pairs, UMMA 256 x 2NX, Ex tile resident          | sep_tc_x_kernel<NX>  one CTA
//   stage YZ  sep_tc_yzt_kernel<64> CTA pairs, transposed, Ey resident for all y (N_y <= 256)
//             sep_tc_yzs_kernel     CTA pairs, both operands streamed (N_y <= 2048)
//             sep_tc_yz128_kernel   one CTA, Ey resident per 128-y group (any size)      | sep_tc_yz_kernel  grids of <= 64 columns
//
// Slice phase: qz z_j = 2 pi t (2j - nz + 1) with t = qz dz / (4 pi) turns; frac(t) is kept as a 32-bit fixed-point
// fraction of a turn, so the product with the integer (2j - nz + 1) wraps modulo one turn for free (error <= 512 * 2^-33
// turns = 4e-7 rad), and sin / cos come from the SFU on an argument in [-pi, pi) (absolute error ~4e-7).
#include <cuda.h>

#include <cstdio>
#include <cstdlib>

#include "internal.h"
#include "ptx_sm100.h"

namespace scatman {

bool encode_map(CUtensorMap *tm, const void *base, int rank, const cuuint64_t *dims, const cuuint64_t *strides,
                const cuuint32_t *box, CUtensorMapSwizzle swizzle);   // tensor_kernel.cu

namespace {

constexpr int kM = 128;              // UMMA M: rows of the A operand tile
constexpr int kKB = 64;              // K per block (one 128-byte swizzle row of FP16)
constexpr int kSlotA = kM * kKB * 2; // 16384: one plane, one K block of an A tile
constexpr int kNyz = 64;             // stage YZ: a columns per accumulator
constexpr int kThreadsTc = 384;      // warp 0 TMA, 1 and 3 MMA issuers, 2 TMEM, 4-11 epilogue
constexpr uint32_t kTmemColsTc = 512;
constexpr int kNBuf = 4;             // accumulator buffers (128 columns each: D_re 64 + D_im 64)

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

// Balanced z splits.  Sequence 0 (stage X): weight of slice j = its live 128-y row tiles; sequence 1 + g (stage YZ, group g):
// its live 64-y blocks of that group.  bounds[seq][0..ns] cut [0, nz) into ns ranges of (almost) equal total weight, so that
// every work item of a stage carries the same number of live tiles whatever the particle's extent along the beam:
// bounds[s] = min { j in [0, nz] : E(j) >= target(s) }, E(j) = weight of the slices before j, target(s) = floor(total s / ns).
// One block of 256 threads per sequence: every thread sums a contiguous run of slices (all flag loads of the block are in
// flight together), a block scan gives E at the run starts, and each thread then places the bounds that fall into its run.
// sequence 0: stage X over all nzt slices of the chunk; sequence 1 + b ngs + g: stage YZ of item b, group g (its nz1 slices).
// Bounds are GLOBAL slice indices (jbase + j).  nyz_seq = 0 skips the stage YZ sequences (the NUFFT route needs only stage X's).
constexpr int kBoundsThreads = 256;
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
struct SepXParams {
    int nz, NY, NPXP, ng, nkx, nta, nsx, nkb;   // nkx = NXP / 64, nta = a tiles of NX columns, nsx = z splits, nkb = NY / 64
    float hscale;                               // 2^(-9 - L): accumulator (2^10 sR H) -> stored H (sH H)
    const unsigned char *flags;                 // [nz][nkb]
    const int *zb;                              // [nsx + 1] balanced z split bounds (sep_tc_bounds_kernel)
    __half *Hp;                                 // [4][nz][NPXP][NY]
};

// NX = a columns per accumulator = rows of the resident Ex tile (NX * NXP * 8 bytes <= 128 KB)
template <int NX>
__global__ void __launch_bounds__(kThreadsTc, 1)
sep_tc_x_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const SepXParams P) {
    constexpr int kSmemE = 131072;                // resident Ex planes: [4][nkx][NX rows x 128 bytes]
    constexpr int kStages = 6;                    // ring of single-plane 64-x blocks of a rho~ row tile (16 KB each)
    constexpr int kBlkE = NX * kKB * 2;           // bytes of one plane, one K block of the Ex tile
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sE = smem;
    uint8_t *sR = smem + kSmemE;
    uint64_t *bars = (uint64_t *)(smem + kSmemE + kStages * kSlotA);
    uint64_t *e_full = bars + 0, *e_empty = bars + 1;
    uint64_t *r_full = bars + 2, *r_empty = r_full + kStages;
    uint64_t *t_full = r_empty + kStages, *t_empty = t_full + kNBuf, *first_done = t_empty + kNBuf;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + kNBuf);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nitems = P.nta * P.nsx;

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(e_full, 1);
        ptx::mbar_init(e_empty, 2);          // both MMA issuers
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(r_full + i, 1);
            ptx::mbar_init(r_empty + i, 2);
        }
        for (int i = 0; i < kNBuf; ++i) {
            ptx::mbar_init(t_full + i, 2);
            ptx::mbar_init(t_empty + i, 8);
            ptx::mbar_init(first_done + i, 1);
        }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) ptx::tmem_alloc(tmem_ptr, kTmemColsTc);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);

    // units of an item: (slice j of its z range, 128-y group g) with a non-empty 64-y block; u = (j - z0) * ng + g
    auto zrange = [&](int s, int &z0, int &z1) {
        z0 = __ldg(P.zb + s);
        z1 = __ldg(P.zb + s + 1);
    };

    if (warp == 0) {
        // ===================================================================== TMA producer
        int slot = 0;
        uint32_t phase = 0;
        int it_local = 0;
        for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it_local) {
            const int ta = item % P.nta, s = item / P.nta;   // a tiles fastest: concurrent CTAs stream the same rho~ tiles
            ptx::mbar_wait(e_empty, (uint32_t)((it_local & 1) ^ 1));
            if (ptx::elect_one()) {
                ptx::mbar_arrive_expect_tx(e_full, (uint32_t)(4 * P.nkx * kBlkE));
                for (int pl = 0; pl < 4; ++pl)
                    for (int kx = 0; kx < P.nkx; ++kx)
                        ptx::tma_load_3d(sE + (pl * P.nkx + kx) * kBlkE, &tmB, e_full, kx * kKB, ta * NX, pl);
            }
            __syncwarp();
            int z0, z1;
            zrange(s, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, P.ng, 0, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                    const int j = z0 + n / P.ng, g = n % P.ng;
                    for (int kx = 0; kx < P.nkx; ++kx)
                        for (int pl = 0; pl < 4; ++pl) {
                            ptx::mbar_wait(r_empty + slot, phase ^ 1);
                            if (ptx::elect_one()) {
                                ptx::mbar_arrive_expect_tx(r_full + slot, (uint32_t)kSlotA);
                                ptx::tma_load_3d(sR + slot * kSlotA, &tmA, r_full + slot, kx * kKB, j * P.NY + g * kM, pl);
                            }
                            __syncwarp();
                            if (++slot == kStages) { slot = 0; phase ^= 1; }
                        }
                }
        }
    } else if (warp == 1 || warp == 3) {
        // ===================================================================== MMA issuers
        // Two issuer warps share every stage: k-step ks belongs to issuer ks % 2.  At N = 64 a tcgen05.mma is bound by its
        // shared-memory operand fetch (48 cycles) and a single issuing thread exposes whatever it spends between stages
        // (measured 72-107 cycles per MMA with one issuer); two threads hide each other's gaps (as in tensor_kernel.cu).
        // The unit's first k-step (accumulate = 0) is issuer 0's; issuer 1 starts on the unit once it has completed.
        constexpr uint32_t idesc_pos = ptx::umma_idesc_f16(kM, NX, false);
        constexpr uint32_t idesc_neg = ptx::umma_idesc_f16(kM, NX, true);
        const uint64_t descR0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sR));
        const uint64_t descE0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sE));
        constexpr uint64_t kR = kSlotA >> 4, kE = kBlkE >> 4;
        const int iw = warp >> 1;   // issuer 0 = warp 1, issuer 1 = warp 3
        int slot = 0;
        uint32_t phase = 0, u = 0;
        int it_local = 0;
        for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it_local) {
            const int s = item / P.nta;
            ptx::mbar_wait(e_full, (uint32_t)(it_local & 1));
            ptx::tc_fence_after();
            const uint64_t kEpl = (uint64_t)P.nkx * kE;   // descriptor distance between Ex planes
            int z0, z1;
            zrange(s, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, P.ng, 0, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                    const uint32_t buf = u % kNBuf, upar = (u / kNBuf) & 1;
                    ptx::mbar_wait(t_empty + buf, upar ^ 1);
                    ptx::tc_fence_after();
                    const uint32_t d_re = tmem_base + buf * 128, d_im = d_re + 64;
                    for (int kx = 0; kx < P.nkx; ++kx)
                        for (int pl = 0; pl < 4; ++pl) {
                            if (iw == 1 && kx == 0 && pl == 0) {   // D must have been initialised by issuer 0
                                ptx::mbar_wait(first_done + buf, upar);
                                ptx::tc_fence_after();
                            }
                            ptx::mbar_wait(r_full + slot, phase);
                            ptx::tc_fence_after();
                            if (ptx::elect_one()) {
#pragma unroll
                                for (int kk = 0; kk < 2; ++kk) {
                                    const int ks = 2 * kk + iw;
                                    const uint64_t a = descR0 + (uint64_t)slot * kR + (uint64_t)(ks * 2);
                                    const uint64_t e_reh = descE0 + (uint64_t)kx * kE + (uint64_t)(ks * 2);
                                    const uint64_t e_rel = e_reh + kEpl, e_imh = e_rel + kEpl, e_iml = e_imh + kEpl;
                                    const uint32_t acc0 = (kx == 0 && ks == 0) ? 0u : 1u;
                                    // (Ar + i Ai)(Er + i Ei), A = rho~ plane of this stage, three split products AhEh + AlEh + AhEl
                                    if (pl == 0) {          // Re_hi
                                        ptx::umma_f16(d_re, a, e_reh, idesc_pos, acc0);
                                        ptx::umma_f16(d_im, a, e_imh, idesc_pos, acc0);
                                        ptx::umma_f16(d_re, a, e_rel, idesc_pos, 1u);
                                        ptx::umma_f16(d_im, a, e_iml, idesc_pos, 1u);
                                    } else if (pl == 1) {   // Re_lo
                                        ptx::umma_f16(d_re, a, e_reh, idesc_pos, 1u);
                                        ptx::umma_f16(d_im, a, e_imh, idesc_pos, 1u);
                                    } else if (pl == 2) {   // Im_hi
                                        ptx::umma_f16(d_re, a, e_imh, idesc_neg, 1u);
                                        ptx::umma_f16(d_im, a, e_reh, idesc_pos, 1u);
                                        ptx::umma_f16(d_re, a, e_iml, idesc_neg, 1u);
                                        ptx::umma_f16(d_im, a, e_rel, idesc_pos, 1u);
                                    } else {                // Im_lo
                                        ptx::umma_f16(d_re, a, e_imh, idesc_neg, 1u);
                                        ptx::umma_f16(d_im, a, e_reh, idesc_pos, 1u);
                                    }
                                    if (iw == 0 && kk == 0 && kx == 0 && pl == 0) ptx::umma_commit(first_done + buf);
                                }
                                ptx::umma_commit(r_empty + slot);
                            }
                            __syncwarp();
                            if (++slot == kStages) { slot = 0; phase ^= 1; }
                        }
                    if (ptx::elect_one()) ptx::umma_commit(t_full + buf);
                    __syncwarp();
                    ++u;
                }
            if (ptx::elect_one()) ptx::umma_commit(e_empty);
            __syncwarp();
        }
    } else if (warp >= 4) {
        // ===================================================================== epilogue: H -> FP16 planes [j][a][y]
        constexpr int kCols = NX / 2;                    // columns of this warp's half
        const int lg = warp & 3, ch = (warp - 4) >> 2;
        const uint32_t t_lane = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(ch * kCols);
        const size_t plane = (size_t)P.nz * P.NPXP * P.NY;
        uint32_t u = 0;
        for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
            const int ta = item % P.nta, s = item / P.nta;
            const int a0 = ta * NX + ch * kCols;
            int z0, z1;
            zrange(s, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, P.ng, 0, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                    const int j = z0 + n / P.ng, g = n % P.ng;
                    const uint32_t buf = u % kNBuf, upar = (u / kNBuf) & 1;
                    ptx::mbar_wait(t_full + buf, upar);
                    ptx::tc_fence_after();
                    const uint32_t t_re = t_lane + buf * 128, t_im = t_re + 64;
                    SCATMAN_ASSERT(j >= 0 && j < P.nz && a0 + kCols <= P.NPXP && g * kM + kM <= P.NY);
                    __half *dst = P.Hp + ((size_t)j * P.NPXP + a0) * P.NY + g * kM + lg * 32 + lane;
#pragma unroll 1
                    for (int c0 = 0; c0 < kCols; c0 += 8) {
                        uint32_t gre[8], gim[8];
                        ptx::tmem_ld8(t_re + c0, gre);
                        ptx::tmem_ld8(t_im + c0, gim);
                        ptx::tmem_ld_wait();
                        if (c0 + 8 >= kCols) {
                            ptx::tc_fence_before();
                            __syncwarp();
                            if (lane == 0) ptx::mbar_arrive(t_empty + buf);
                        }
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            __half h[4];
                            split4(__uint_as_float(gre[i]) * P.hscale, __uint_as_float(gim[i]) * P.hscale, h);
                            __half *d = dst + (size_t)(c0 + i) * P.NY;
#pragma unroll
                            for (int pl = 0; pl < 4; ++pl) d[pl * plane] = h[pl];
                        }
                    }
                    ++u;
                }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, kTmemColsTc);
    }
}

// ---- stage X on CTA pairs ------------------------------------------------------------------------------------------
// tcgen05 cta_group::2, UMMA 256 x 2NX x 16: the two CTAs of a pair take two consecutive live row tiles (each streams its own
// rho~ tile, 128 rows = its half of M) against the same 2 NX grid columns, of whose Ex tile each CTA keeps NX rows resident.
// Per SM an instruction then fetches 4 KB of A + 2 KB of B for 64 tensor cycles (N = 128) instead of 6 KB for 32 (N = 64 from
// one CTA, shared-memory bound at 48.7 cycles).  Stages hold two planes (Re hi + lo, then Im hi + lo: 24 MMAs per barrier round
// trip).  Each CTA converts and stores the H rows of its own tile; an odd last tile is run twice (the peer repeats the
// leader's tile and discards it).  Leader-side barriers as in tensor_kernel.cu.
template <int NX>
__global__ void __launch_bounds__(kThreadsTc, 1)
sep_tc_x2_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const SepXParams P) {
    constexpr int kN = 2 * NX;                    // accumulator columns
    constexpr int kSmemE = 131072;                // resident Ex planes of this CTA's NX columns: [4][nkx][NX rows x 128 bytes]
    constexpr int kStages = 3;                    // ring of two-plane 64-x blocks of this CTA's rho~ row tile (32 KB each)
    constexpr int kStage = 2 * kSlotA;
    constexpr int kBlkE = NX * kKB * 2;
    constexpr int kNB = 2;                        // accumulator buffers (D_re, D_im of up to 128 columns each)
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sE = smem;
    uint8_t *sR = smem + kSmemE;
    uint64_t *bars = (uint64_t *)(smem + kSmemE + kStages * kStage);
    uint64_t *e_full = bars + 0, *e_empty = bars + 1;
    uint64_t *r_full = bars + 2, *r_empty = r_full + kStages;
    uint64_t *t_full = r_empty + kStages, *t_empty = t_full + kNB, *first_done = t_empty + kNB;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + kNB);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    const bool leader = rank == 0;
    const int cluster_id = blockIdx.x / 2, nclusters = gridDim.x / 2;
    const int nitems = P.nta * P.nsx;             // nta = tiles of 2 NX columns

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(e_full, 1);
        ptx::mbar_init(e_empty, 2);
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(r_full + i, 1);
            ptx::mbar_init(r_empty + i, 2);
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

    auto zrange = [&](int s, int &z0, int &z1) {
        z0 = __ldg(P.zb + s);
        z1 = __ldg(P.zb + s + 1);
    };
    // the next pair of live units: n0 for the leader, n1 for the peer (n1 = n0 and dup = true when only one is left)
    auto next_pair = [&](LiveUnits &un, int &n0, int &n1, bool &dup) {
        uint32_t f;
        if (!un.next(n0, f)) return false;
        dup = !un.next(n1, f);
        if (dup) n1 = n0;
        return true;
    };

    if (warp == 0) {
        // ===================================================================== TMA producer (both CTAs)
        int slot = 0;
        uint32_t phase = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            const int ta = item % P.nta, s = item / P.nta;
            ptx::mbar_wait(e_empty, (uint32_t)((it_local & 1) ^ 1));
            if (ptx::elect_one()) {
                if (leader) ptx::mbar_arrive_expect_tx(e_full, (uint32_t)(2 * 4 * P.nkx * kBlkE));
                for (int pl = 0; pl < 4; ++pl)
                    for (int kx = 0; kx < P.nkx; ++kx)
                        ptx::tma_load_3d_2sm(sE + (pl * P.nkx + kx) * kBlkE, &tmB, e_full, kx * kKB, ta * kN + (int)rank * NX, pl);
            }
            __syncwarp();
            int z0, z1;
            zrange(s, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, P.ng, 0, lane);
            int n0, n1;
            bool dup;
            while (next_pair(un, n0, n1, dup)) {
                const int n = leader ? n0 : n1;
                const int j = z0 + n / P.ng, g = n % P.ng;
                for (int kx = 0; kx < P.nkx; ++kx)
                    for (int ph = 0; ph < 2; ++ph) {   // Re planes, Im planes
                        ptx::mbar_wait(r_empty + slot, phase ^ 1);
                        if (ptx::elect_one()) {
                            if (leader) ptx::mbar_arrive_expect_tx(r_full + slot, (uint32_t)(2 * kStage));
                            ptx::tma_load_3d_2sm(sR + slot * kStage, &tmA, r_full + slot, kx * kKB, j * P.NY + g * kM, 2 * ph);
                            ptx::tma_load_3d_2sm(sR + slot * kStage + kSlotA, &tmA, r_full + slot, kx * kKB, j * P.NY + g * kM, 2 * ph + 1);
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
        const uint64_t descR0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sR));
        const uint64_t descE0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sE));
        constexpr uint64_t kR = kSlotA >> 4, kSt = kStage >> 4, kE = kBlkE >> 4;
        const int iw = warp >> 1;
        int slot = 0;
        uint32_t phase = 0, u = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            const int s = item / P.nta;
            ptx::mbar_wait(e_full, (uint32_t)(it_local & 1));
            ptx::tc_fence_after();
            const uint64_t kEpl = (uint64_t)P.nkx * kE;
            int z0, z1;
            zrange(s, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, P.ng, 0, lane);
            int n0, n1;
            bool dup;
            while (next_pair(un, n0, n1, dup)) {
                const uint32_t buf = u % kNB, upar = (u / kNB) & 1;
                ptx::mbar_wait(t_empty + buf, upar ^ 1);
                ptx::tc_fence_after();
                const uint32_t d_re = tmem_base + buf * 256, d_im = d_re + 128;
                for (int kx = 0; kx < P.nkx; ++kx)
                    for (int ph = 0; ph < 2; ++ph) {
                        if (iw == 1 && kx == 0 && ph == 0) {   // D must have been initialised by issuer 0
                            ptx::mbar_wait(first_done + buf, upar);
                            ptx::tc_fence_after();
                        }
                        ptx::mbar_wait(r_full + slot, phase);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
#pragma unroll
                            for (int kk = 0; kk < 2; ++kk) {
                                const int ks = 2 * kk + iw;
                                const uint64_t a_hi = descR0 + (uint64_t)slot * kSt + (uint64_t)(ks * 2), a_lo = a_hi + kR;
                                const uint64_t e_reh = descE0 + (uint64_t)kx * kE + (uint64_t)(ks * 2);
                                const uint64_t e_rel = e_reh + kEpl, e_imh = e_rel + kEpl, e_iml = e_imh + kEpl;
                                const uint32_t acc0 = (kx == 0 && ph == 0 && ks == 0) ? 0u : 1u;
                                // (Ar + i Ai)(Er + i Ei), A = the rho~ planes of this stage, three split products AhEh + AlEh + AhEl
                                if (ph == 0) {   // Re hi, Re lo
                                    ptx::umma_f16_2sm(d_re, a_hi, e_reh, idesc_pos, acc0);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_imh, idesc_pos, acc0);
                                    ptx::umma_f16_2sm(d_re, a_hi, e_rel, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_iml, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_lo, e_reh, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_im, a_lo, e_imh, idesc_pos, 1u);
                                } else {         // Im hi, Im lo
                                    ptx::umma_f16_2sm(d_re, a_hi, e_imh, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_reh, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_hi, e_iml, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_rel, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_lo, e_imh, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_lo, e_reh, idesc_pos, 1u);
                                }
                                if (iw == 0 && kk == 0 && kx == 0 && ph == 0) ptx::umma_commit_2sm(first_done + buf, (uint16_t)0x1);
                            }
                            ptx::umma_commit_2sm(r_empty + slot, (uint16_t)0x3);
                        }
                        __syncwarp();
                        if (++slot == kStages) { slot = 0; phase ^= 1; }
                    }
                if (ptx::elect_one()) ptx::umma_commit_2sm(t_full + buf, (uint16_t)0x3);
                __syncwarp();
                ++u;
            }
            if (ptx::elect_one()) ptx::umma_commit_2sm(e_empty, (uint16_t)0x3);
            __syncwarp();
        }
    } else if (warp >= 4) {
        // ===================================================================== epilogue: H rows of this CTA's tile -> FP16 planes
        const int lg = warp & 3, ch = (warp - 4) >> 2;   // TMEM lane group; column half: [ch NX, +NX) of the 2 NX columns
        const uint32_t t_lane = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(ch * NX);
        const size_t plane = (size_t)P.nz * P.NPXP * P.NY;
        uint32_t u = 0;
        for (int item = cluster_id; item < nitems; item += nclusters) {
            const int ta = item % P.nta, s = item / P.nta;
            const int a0 = ta * kN + ch * NX;
            int z0, z1;
            zrange(s, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, P.ng, 0, lane);
            int n0, n1;
            bool dup;
            while (next_pair(un, n0, n1, dup)) {
                const int n = leader ? n0 : n1;
                const int j = z0 + n / P.ng, g = n % P.ng;
                const bool store = leader || !dup;
                const uint32_t buf = u % kNB, upar = (u / kNB) & 1;
                ptx::mbar_wait(t_full + buf, upar);
                ptx::tc_fence_after();
                const uint32_t t_re = t_lane + buf * 256, t_im = t_re + 128;
                SCATMAN_ASSERT(j >= 0 && j < P.nz && a0 + NX <= P.NPXP && g * kM + kM <= P.NY);
                __half *dst = P.Hp + ((size_t)j * P.NPXP + a0) * P.NY + g * kM + lg * 32 + lane;
#pragma unroll 1
                for (int c0 = 0; c0 < NX; c0 += 8) {
                    uint32_t gre[8], gim[8];
                    ptx::tmem_ld8(t_re + c0, gre);
                    ptx::tmem_ld8(t_im + c0, gim);
                    ptx::tmem_ld_wait();
                    if (c0 + 8 >= NX) {
                        ptx::tc_fence_before();
                        __syncwarp();
                        if (lane == 0) ptx::mbar_arrive_cluster(t_empty + buf, 0);   // the leader's barrier
                    }
                    if (store) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            __half h[4];
                            split4(__uint_as_float(gre[i]) * P.hscale, __uint_as_float(gim[i]) * P.hscale, h);
                            __half *d = dst + (size_t)(c0 + i) * P.NY;
#pragma unroll
                            for (int pl = 0; pl < 4; ++pl) d[pl * plane] = h[pl];
                        }
                    }
                }
                ++u;
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

// ------------------------------------------------------------------------------------------------ stage YZ
struct SepYzParams {
    int nz, nb, npx, npy, NY, NPXP, ng, nzs, ntb, nta, nkb;   // nz: slices per item, nb: items of the chunk, nkb = NY / 64
    double k, dz;
    const double *qx, *qy;
    const unsigned char *flags;   // [nz][nkb]
    const int *zb;                // [nb][ng][nzs + 1] balanced z split bounds (global slice indices) per item and 128-y group
    float2 *partial;              // [nb][ng * nzs][npy][npx]
};

struct YzItem {
    int tb, ta, g, s, b;
};
__device__ __forceinline__ YzItem yz_decode(int item, const SepYzParams &P) {
    YzItem it;
    it.tb = item % P.ntb;   // b tiles fastest: concurrent CTAs stream the same H tiles
    item /= P.ntb;
    it.ta = item % P.nta;
    item /= P.nta;
    it.g = item % P.ng;
    item /= P.ng;
    it.s = item % P.nzs;
    it.b = item / P.nzs;
    return it;
}

// items of the CTA-pair variant: a pair index replaces the b tile, this CTA's tile is NCTA tp + rank
template <int NCTA>
__device__ __forceinline__ YzItem yz_decode_n(int item, const SepYzParams &P, int rank) {
    YzItem it;
    const int ntp = P.ntb / NCTA;
    it.tb = (item % ntp) * NCTA + rank;
    item /= ntp;
    it.ta = item % P.nta;
    item /= P.nta;
    it.g = item % P.ng;
    item /= P.ng;
    it.s = item % P.nzs;
    it.b = item / P.nzs;
    return it;
}

__global__ void __launch_bounds__(kThreadsTc, 1)
sep_tc_yz_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const SepYzParams P) {
    constexpr int kSmemA = 4 * 2 * kSlotA;            // 131072: resident Ey planes of one b tile, one 128-y group
    constexpr int kStageB = 4 * kNyz * kKB * 2;       // 32768: four planes of one 64-y block of an H tile
    constexpr int kStages = 3;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sA = smem;
    uint8_t *sB = smem + kSmemA;
    uint64_t *bars = (uint64_t *)(smem + kSmemA + kStages * kStageB);
    uint64_t *a_full = bars + 0, *a_empty = bars + 1;
    uint64_t *b_full = bars + 2, *b_empty = b_full + kStages;
    uint64_t *t_full = b_empty + kStages, *t_empty = t_full + kNBuf, *first_done = t_empty + kNBuf;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + kNBuf);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nitems = P.ntb * P.nta * P.ng * P.nzs * P.nb;

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(a_full, 1);
        ptx::mbar_init(a_empty, 2);          // both MMA issuers
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(b_full + i, 1);
            ptx::mbar_init(b_empty + i, 2);
        }
        for (int i = 0; i < kNBuf; ++i) {
            ptx::mbar_init(t_full + i, 2);
            ptx::mbar_init(t_empty + i, 8);
            ptx::mbar_init(first_done + i, 1);
        }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) ptx::tmem_alloc(tmem_ptr, kTmemColsTc);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);

    auto zrange = [&](const YzItem &it, int &z0, int &z1) {   // global slice indices
        const int *zb = P.zb + (size_t)(it.b * P.ng + it.g) * (P.nzs + 1) + it.s;
        z0 = __ldg(zb);
        z1 = __ldg(zb + 1);
    };

    if (warp == 0) {
        // ===================================================================== TMA producer
        int slot = 0;
        uint32_t phase = 0;
        int it_local = 0;
        for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it_local) {
            const YzItem it = yz_decode(item, P);
            ptx::mbar_wait(a_empty, (uint32_t)((it_local & 1) ^ 1));
            if (ptx::elect_one()) {
                ptx::mbar_arrive_expect_tx(a_full, (uint32_t)kSmemA);
                for (int pl = 0; pl < 4; ++pl)
                    for (int kb = 0; kb < 2; ++kb)
                        ptx::tma_load_3d(sA + (pl * 2 + kb) * kSlotA, &tmA, a_full, (it.g * 2 + kb) * kKB, it.tb * kM, pl);
            }
            __syncwarp();
            int z0, z1;
            zrange(it, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, 1, it.g, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                const int j = z0 + n;
                for (int kb = 0; kb < 2; ++kb) {
                    if (((f >> kb) & 1u) == 0u) continue;
                    ptx::mbar_wait(b_empty + slot, phase ^ 1);
                    if (ptx::elect_one()) {
                        ptx::mbar_arrive_expect_tx(b_full + slot, (uint32_t)kStageB);
                        for (int pl = 0; pl < 4; ++pl)
                            ptx::tma_load_3d(sB + slot * kStageB + pl * (kStageB / 4), &tmB, b_full + slot,
                                             (it.g * 2 + kb) * kKB, j * P.NPXP + it.ta * kNyz, pl);
                    }
                    __syncwarp();
                    if (++slot == kStages) { slot = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1 || warp == 3) {
        // ===================================================================== MMA issuers (k-step ks belongs to issuer ks % 2)
        constexpr uint32_t idesc_pos = ptx::umma_idesc_f16(kM, kNyz, false);
        constexpr uint32_t idesc_neg = ptx::umma_idesc_f16(kM, kNyz, true);
        const uint64_t descA0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sA));
        const uint64_t descB0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sB));
        constexpr uint64_t kA = kSlotA >> 4, kBst = kStageB >> 4, kBpl = (kStageB / 4) >> 4;
        const int iw = warp >> 1;   // issuer 0 = warp 1, issuer 1 = warp 3
        int slot = 0;
        uint32_t phase = 0, u = 0;
        int it_local = 0;
        for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it_local) {
            const YzItem it = yz_decode(item, P);
            ptx::mbar_wait(a_full, (uint32_t)(it_local & 1));
            ptx::tc_fence_after();
            int z0, z1;
            zrange(it, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, 1, it.g, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                const uint32_t buf = u % kNBuf, upar = (u / kNBuf) & 1;
                ptx::mbar_wait(t_empty + buf, upar ^ 1);
                ptx::tc_fence_after();
                const uint32_t d_re = tmem_base + buf * 128, d_im = d_re + 64;
                bool first = true;
                for (int kb = 0; kb < 2; ++kb) {
                    if (((f >> kb) & 1u) == 0u) continue;
                    if (first && iw == 1) {   // D must have been initialised by issuer 0's first k-step
                        ptx::mbar_wait(first_done + buf, upar);
                        ptx::tc_fence_after();
                    }
                    ptx::mbar_wait(b_full + slot, phase);
                    ptx::tc_fence_after();
                    if (ptx::elect_one()) {
#pragma unroll
                        for (int kk = 0; kk < 2; ++kk) {
                            const int ks = 2 * kk + iw;
                            const uint64_t a_reh = descA0 + (uint64_t)kb * kA + (uint64_t)(ks * 2);
                            const uint64_t a_rel = a_reh + 2 * kA, a_imh = a_reh + 4 * kA, a_iml = a_reh + 6 * kA;
                            const uint64_t b_reh = descB0 + (uint64_t)slot * kBst + (uint64_t)(ks * 2);
                            const uint64_t b_rel = b_reh + kBpl, b_imh = b_rel + kBpl, b_iml = b_imh + kBpl;
                            const uint32_t acc0 = (first && ks == 0) ? 0u : 1u;
                            ptx::umma_f16(d_re, a_reh, b_reh, idesc_pos, acc0);
                            ptx::umma_f16(d_im, a_imh, b_reh, idesc_pos, acc0);
                            ptx::umma_f16(d_re, a_rel, b_reh, idesc_pos, 1u);
                            ptx::umma_f16(d_im, a_iml, b_reh, idesc_pos, 1u);
                            ptx::umma_f16(d_re, a_reh, b_rel, idesc_pos, 1u);
                            ptx::umma_f16(d_im, a_imh, b_rel, idesc_pos, 1u);
                            ptx::umma_f16(d_re, a_imh, b_imh, idesc_neg, 1u);
                            ptx::umma_f16(d_im, a_reh, b_imh, idesc_pos, 1u);
                            ptx::umma_f16(d_re, a_iml, b_imh, idesc_neg, 1u);
                            ptx::umma_f16(d_im, a_rel, b_imh, idesc_pos, 1u);
                            ptx::umma_f16(d_re, a_imh, b_iml, idesc_neg, 1u);
                            ptx::umma_f16(d_im, a_reh, b_iml, idesc_pos, 1u);
                            if (first && iw == 0 && kk == 0) ptx::umma_commit(first_done + buf);
                        }
                        ptx::umma_commit(b_empty + slot);
                    }
                    __syncwarp();
                    first = false;
                    if (++slot == kStages) { slot = 0; phase ^= 1; }
                }
                if (ptx::elect_one()) ptx::umma_commit(t_full + buf);
                __syncwarp();
                ++u;
            }
            if (ptx::elect_one()) ptx::umma_commit(a_empty);
            __syncwarp();
        }
    } else if (warp >= 4) {
        // ===================================================================== epilogue: Blocks 7-8
        const int lg = warp & 3, ch = (warp - 4) >> 2;   // TMEM lane group, column half
        const uint32_t t_lane = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(ch * 32);
        uint32_t u = 0;
        for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
            const YzItem it = yz_decode(item, P);
            const int b = it.tb * kM + lg * 32 + lane;
            const int a0 = it.ta * kNyz + ch * 32;
            const double qyb = b < P.npy ? P.qy[b] : 0.0;
            uint32_t dph[32];
#pragma unroll
            for (int c = 0; c < 32; ++c) {
                const int a = a0 + c;
                double t = 0.0;
                if (a < P.npx && b < P.npy) {
                    const double qxa = P.qx[a];
                    const double qxy2 = qxa * qxa + qyb * qyb;
                    const double kz2 = P.k * P.k - qxy2;
                    // qz = -(k - sqrt(k^2 - qxy^2)) = -qxy^2 / (k + sqrt(k^2 - qxy^2)): no cancellation near forward
                    const double qz = kz2 >= 0.0 ? -qxy2 / (P.k + sqrt(kz2)) : 0.0;
                    t = qz * P.dz * (0.25 / 3.14159265358979323846);
                    t -= rint(t);
                }
                dph[c] = (uint32_t)(long long)rint(t * 4294967296.0);
            }
            float2 tot[32];
#pragma unroll
            for (int c = 0; c < 32; ++c) tot[c] = make_float2(0.f, 0.f);
            int z0, z1;
            zrange(it, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, 1, it.g, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                const int j = z0 + n - it.b * P.nz;   // slice within its item
                const uint32_t buf = u % kNBuf, upar = (u / kNBuf) & 1;
                const uint32_t mult = (uint32_t)(2 * j - P.nz + 1);
                ptx::mbar_wait(t_full + buf, upar);
                ptx::tc_fence_after();
                const uint32_t t_re = t_lane + buf * 128, t_im = t_re + 64;
                uint32_t gre[2][8], gim[2][8];
                ptx::tmem_ld8(t_re, gre[0]);
                ptx::tmem_ld8(t_im, gim[0]);
                ptx::tmem_ld_wait();
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                    const int cur = q4 & 1, nxt = cur ^ 1;
                    if (q4 < 3) {
                        ptx::tmem_ld8(t_re + (q4 + 1) * 8, gre[nxt]);
                        ptx::tmem_ld8(t_im + (q4 + 1) * 8, gim[nxt]);
                    } else {
                        ptx::tc_fence_before();
                        __syncwarp();
                        if (lane == 0) ptx::mbar_arrive(t_empty + buf);   // every column of this warp has landed
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int c = q4 * 8 + i;
                        const float ang = (float)(int)(dph[c] * mult) * 1.4629180792671596e-9f;   // pi / 2^31
                        float sn, cs;
                        __sincosf(ang, &sn, &cs);
                        const float gr = __uint_as_float(gre[cur][i]), gi = __uint_as_float(gim[cur][i]);
                        tot[c].x = fmaf(cs, gr, tot[c].x);
                        tot[c].x = fmaf(-sn, gi, tot[c].x);
                        tot[c].y = fmaf(cs, gi, tot[c].y);
                        tot[c].y = fmaf(sn, gr, tot[c].y);
                    }
                    if (q4 < 3) ptx::tmem_ld_wait();
                }
                ++u;
            }
            if (b < P.npy) {
                float2 *dst = P.partial + (((size_t)it.b * P.ng * P.nzs + it.g * P.nzs + it.s) * P.npy + b) * P.npx;
#pragma unroll
                for (int c = 0; c < 32; ++c)
                    if (a0 + c < P.npx) dst[a0 + c] = tot[c];
            }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, kTmemColsTc);
    }
}

// ---- stage YZ with 128-column accumulators ------------------------------------------------------------------------
// Same work as sep_tc_yz_kernel with UMMA 128 x 128 x 16: at N = 128 the instruction's 64 tensor cycles cover its
// shared-memory operand fetch (8 KB), at N = 64 they do not (48.7 cycles for 32 of work).  H tiles of 128 columns stream
// plane by plane through a ring of 6 x 16 KB (as the rho~ tiles of stage X); two accumulator buffers of D_re, D_im x 128
// columns.  An epilogue thread now carries 64 columns: 128 running totals + 64 phase fractions, more than the 168 registers
// a 384-thread CTA gives each thread, so the register file is re-split with setmaxnreg: the producer / issuer warpgroup
// drops to 48 registers per thread, the two epilogue warpgroups rise to 224: 128 x 48 + 256 x 224 = 63488 <= the 384 x 168 =
// 64512 registers the CTA owns (an increase can only take what the CTA's own warps released, or it waits forever).
__device__ __forceinline__ void setmaxnreg_inc_224() { asm volatile("setmaxnreg.inc.sync.aligned.u32 224;"); }
__device__ __forceinline__ void setmaxnreg_dec_48() { asm volatile("setmaxnreg.dec.sync.aligned.u32 48;"); }

// NCTA = 2: a CTA pair per work item (tcgen05 cta_group::2, UMMA 256 x 128 x 16): each CTA owns one b tile (its Ey tile, its
// accumulators, its epilogue) and HALF of every H tile (64 of the 128 a rows), so an instruction fetches 4 KB of A + 2 KB of B
// per SM for its 64 tensor cycles -- at 128 B/clk that leaves the shared-memory port slack, where a single CTA (8 KB per 64
// cycles) has none and measured 54 % tensor-pipe activity.  The leader (rank 0) issues every MMA; full barriers live in the
// leader, empty barriers are signalled in both CTAs (the protocol of tensor_kernel.cu).
template <int NCTA>
__global__ void __launch_bounds__(kThreadsTc, 1)
sep_tc_yz128_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const SepYzParams P) {
    constexpr int kN = 128;
    constexpr int kSmemA = 4 * 2 * kSlotA;            // 131072: resident Ey planes of one b tile, one 128-y group
    constexpr int kSlotB = kSlotA / NCTA;             // this CTA's part of a single-plane 64-y block of an H tile (kN / NCTA rows)
    // A stage = G planes of one 64-y block.  A pair's halves are small enough for all four planes (48 MMAs per barrier round
    // trip); a single CTA streams plane by plane (8 or 4 MMAs per stage: the issue overhead shows).
    constexpr int kG = NCTA == 2 ? 4 : 1;
    constexpr int kStageB = kG * kSlotB;              // 32 KB (pair) / 16 KB (single)
    constexpr int kStages = NCTA == 2 ? 3 : 6;
    constexpr int kNB = 2;                            // accumulator buffers (256 columns each)
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sA = smem;
    uint8_t *sB = smem + kSmemA;
    uint64_t *bars = (uint64_t *)(smem + kSmemA + kStages * kStageB);
    uint64_t *a_full = bars + 0, *a_empty = bars + 1;
    uint64_t *b_full = bars + 2, *b_empty = b_full + kStages;
    uint64_t *t_full = b_empty + kStages, *t_empty = t_full + kNB, *first_done = t_empty + kNB;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + kNB);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = NCTA == 2 ? ptx::cluster_ctarank() : 0u;
    const bool leader = rank == 0;
    const int cluster_id = blockIdx.x / NCTA, nclusters = gridDim.x / NCTA;
    const int nitems = (P.ntb / NCTA) * P.nta * P.ng * P.nzs * P.nb;   // an item covers NCTA b tiles: tb = NCTA tp + rank

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(a_full, 1);
        ptx::mbar_init(a_empty, 2);
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(b_full + i, 1);
            ptx::mbar_init(b_empty + i, 2);
        }
        for (int i = 0; i < kNB; ++i) {
            ptx::mbar_init(t_full + i, 2);
            ptx::mbar_init(t_empty + i, 8 * NCTA);
            ptx::mbar_init(first_done + i, 1);
        }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) {
        if (NCTA == 2) ptx::tmem_alloc_2sm(tmem_ptr, kTmemColsTc);
        else ptx::tmem_alloc(tmem_ptr, kTmemColsTc);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (NCTA == 2) ptx::cluster_sync_all();   // peer barriers are initialised before anyone signals them
    ptx::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);

    auto zrange = [&](const YzItem &it, int &z0, int &z1) {
        const int *zb = P.zb + (size_t)(it.b * P.ng + it.g) * (P.nzs + 1) + it.s;
        z0 = __ldg(zb);
        z1 = __ldg(zb + 1);
    };

    if (warp < 4) {
      setmaxnreg_dec_48();
      if (warp == 0) {
        // ===================================================================== TMA producer
        int slot = 0;
        uint32_t phase = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            const YzItem it = yz_decode_n<NCTA>(item, P, (int)rank);
            ptx::mbar_wait(a_empty, (uint32_t)((it_local & 1) ^ 1));
            if (ptx::elect_one()) {
                if (leader) ptx::mbar_arrive_expect_tx(a_full, (uint32_t)(NCTA * kSmemA));
                for (int pl = 0; pl < 4; ++pl)
                    for (int kb = 0; kb < 2; ++kb) {
                        void *dst = sA + (pl * 2 + kb) * kSlotA;
                        if (NCTA == 2) ptx::tma_load_3d_2sm(dst, &tmA, a_full, (it.g * 2 + kb) * kKB, it.tb * kM, pl);
                        else ptx::tma_load_3d(dst, &tmA, a_full, (it.g * 2 + kb) * kKB, it.tb * kM, pl);
                    }
            }
            __syncwarp();
            int z0, z1;
            zrange(it, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, 1, it.g, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                const int j = z0 + n;
                for (int kb = 0; kb < 2; ++kb) {
                    if (((f >> kb) & 1u) == 0u) continue;
                    for (int pg = 0; pg < 4 / kG; ++pg) {
                        ptx::mbar_wait(b_empty + slot, phase ^ 1);
                        if (ptx::elect_one()) {
                            if (leader) ptx::mbar_arrive_expect_tx(b_full + slot, (uint32_t)(NCTA * kStageB));   // both halves land on the leader's barrier
                            const int row = j * P.NPXP + it.ta * kN + (int)rank * (kN / NCTA);
#pragma unroll
                            for (int q = 0; q < kG; ++q) {
                                void *dst = sB + slot * kStageB + q * kSlotB;
                                if (NCTA == 2) ptx::tma_load_3d_2sm(dst, &tmB, b_full + slot, (it.g * 2 + kb) * kKB, row, pg * kG + q);
                                else ptx::tma_load_3d(dst, &tmB, b_full + slot, (it.g * 2 + kb) * kKB, row, pg * kG + q);
                            }
                        }
                        __syncwarp();
                        if (++slot == kStages) { slot = 0; phase ^= 1; }
                    }
                }
            }
        }
      } else if ((warp == 1 || warp == 3) && leader) {
        // ===================================================================== MMA issuers (k-step ks belongs to issuer ks % 2)
        constexpr uint32_t idesc_pos = ptx::umma_idesc_f16(kM * NCTA, kN, false);
        constexpr uint32_t idesc_neg = ptx::umma_idesc_f16(kM * NCTA, kN, true);
        auto mma = [](uint32_t d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
            if (NCTA == 2) ptx::umma_f16_2sm(d, a, b, idesc, acc);
            else ptx::umma_f16(d, a, b, idesc, acc);
        };
        auto commit = [](uint64_t *bar) {         // in every CTA of the pair
            if (NCTA == 2) ptx::umma_commit_2sm(bar, (uint16_t)0x3);
            else ptx::umma_commit(bar);
        };
        auto commit_local = [](uint64_t *bar) {   // this (leader) CTA's barrier only
            if (NCTA == 2) ptx::umma_commit_2sm(bar, (uint16_t)0x1);
            else ptx::umma_commit(bar);
        };
        const uint64_t descA0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sA));
        const uint64_t descB0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sB));
        constexpr uint64_t kA = kSlotA >> 4, kB = kSlotB >> 4;
        const int iw = warp >> 1;
        int slot = 0;
        uint32_t phase = 0, u = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            const YzItem it = yz_decode_n<NCTA>(item, P, (int)rank);
            ptx::mbar_wait(a_full, (uint32_t)(it_local & 1));
            ptx::tc_fence_after();
            int z0, z1;
            zrange(it, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, 1, it.g, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                const uint32_t buf = u % kNB, upar = (u / kNB) & 1;
                ptx::mbar_wait(t_empty + buf, upar ^ 1);
                ptx::tc_fence_after();
                const uint32_t d_re = tmem_base + buf * 256, d_im = d_re + 128;
                bool first = true;
                for (int kb = 0; kb < 2; ++kb) {
                    if (((f >> kb) & 1u) == 0u) continue;
                    for (int pg = 0; pg < 4 / kG; ++pg) {
                        if (first && pg == 0 && iw == 1) {   // D must have been initialised by issuer 0's first k-step
                            ptx::mbar_wait(first_done + buf, upar);
                            ptx::tc_fence_after();
                        }
                        ptx::mbar_wait(b_full + slot, phase);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
#pragma unroll
                            for (int kk = 0; kk < 2; ++kk) {
                                const int ks = 2 * kk + iw;
                                const uint64_t a_reh = descA0 + (uint64_t)kb * kA + (uint64_t)(ks * 2);
                                const uint64_t a_rel = a_reh + 2 * kA, a_imh = a_reh + 4 * kA, a_iml = a_reh + 6 * kA;
#pragma unroll
                                for (int q = 0; q < kG; ++q) {
                                    const int pl = pg * kG + q;
                                    const uint64_t b = descB0 + (uint64_t)slot * (kStageB >> 4) + (uint64_t)q * kB + (uint64_t)(ks * 2);
                                    const uint32_t acc0 = (first && pl == 0 && ks == 0) ? 0u : 1u;
                                    // (Ar + i Ai)(Br + i Bi), B = H plane pl of this stage, three split products AhBh + AlBh + AhBl
                                    if (pl == 0) {          // B Re_hi
                                        mma(d_re, a_reh, b, idesc_pos, acc0);
                                        mma(d_im, a_imh, b, idesc_pos, acc0);
                                        mma(d_re, a_rel, b, idesc_pos, 1u);
                                        mma(d_im, a_iml, b, idesc_pos, 1u);
                                    } else if (pl == 1) {   // B Re_lo
                                        mma(d_re, a_reh, b, idesc_pos, 1u);
                                        mma(d_im, a_imh, b, idesc_pos, 1u);
                                    } else if (pl == 2) {   // B Im_hi
                                        mma(d_re, a_imh, b, idesc_neg, 1u);
                                        mma(d_im, a_reh, b, idesc_pos, 1u);
                                        mma(d_re, a_iml, b, idesc_neg, 1u);
                                        mma(d_im, a_rel, b, idesc_pos, 1u);
                                    } else {                // B Im_lo
                                        mma(d_re, a_imh, b, idesc_neg, 1u);
                                        mma(d_im, a_reh, b, idesc_pos, 1u);
                                    }
                                }
                                if (first && pg == 0 && iw == 0 && kk == 0) commit_local(first_done + buf);
                            }
                            commit(b_empty + slot);
                        }
                        __syncwarp();
                        if (++slot == kStages) { slot = 0; phase ^= 1; }
                    }
                    first = false;
                }
                if (ptx::elect_one()) commit(t_full + buf);
                __syncwarp();
                ++u;
            }
            if (ptx::elect_one()) commit(a_empty);
            __syncwarp();
        }
      }
    } else {
        setmaxnreg_inc_224();
        // ===================================================================== epilogue: Blocks 7-8, 64 columns per thread
        const int lg = warp & 3, ch = (warp - 4) >> 2;
        const uint32_t t_lane = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(ch * 64);
        uint32_t u = 0;
        for (int item = cluster_id; item < nitems; item += nclusters) {
            const YzItem it = yz_decode_n<NCTA>(item, P, (int)rank);
            const int b = it.tb * kM + lg * 32 + lane;
            const int a0 = it.ta * kN + ch * 64;
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
            zrange(it, z0, z1);
            LiveUnits un;
            un.begin(P.flags, P.nkb, z0, z1, 1, it.g, lane);
            int n;
            uint32_t f;
            while (un.next(n, f)) {
                const int j = z0 + n - it.b * P.nz;
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
                        if (lane == 0) {
                            if (NCTA == 2) ptx::mbar_arrive_cluster(t_empty + buf, 0);   // the leader's barrier
                            else ptx::mbar_arrive(t_empty + buf);
                        }
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
                float2 *dst = P.partial + (((size_t)it.b * P.ng * P.nzs + it.g * P.nzs + it.s) * P.npy + b) * P.npx;
#pragma unroll
                for (int c = 0; c < 64; ++c)
                    if (a0 + c < P.npx) dst[a0 + c] = tot[c];
            }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (NCTA == 2) ptx::cluster_sync_all();   // nobody leaves while the peer may still signal its barriers
    if (warp == 2) {
        ptx::tc_fence_after();
        if (NCTA == 2) ptx::tmem_dealloc_2sm(tmem_base, kTmemColsTc);
        else ptx::tmem_dealloc(tmem_base, kTmemColsTc);
    }
}

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
      setmaxnreg_dec_48();
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
        setmaxnreg_inc_224();
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
// The roles of sep_tc_x2_kernel: the streamed A operand is each CTA's own H tile (128 grid columns a = the TMEM lanes, two
// planes per stage), the resident B operand this CTA's NB rows of the Ey tile of 2 NB grid rows b, for every 64-y block
// (NB nkb 8 KB <= 128 KB: NB = 64 for N_y <= 256, the only instance built; NB = 32 for N_y <= 512 ran UMMA N = 64 and measured
// slower than the streamed form).  One accumulator per slice like sep_tc_yzs_kernel, but only H streams (2/3 of that kernel's
// L2 -> SM traffic).  The epilogue thread owns one column a and NB rows b.
template <int NB>
__global__ void __launch_bounds__(kThreadsTc, 1)
sep_tc_yzt_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const SepYzParams P) {
    constexpr int kN = 2 * NB;
    constexpr int kSmemE = 131072;                // resident Ey planes of this CTA's NB rows: [4][nkb][NB rows x 128 bytes]
    constexpr int kStages = 3;
    constexpr int kStage = 2 * kSlotA;            // two planes of one 64-y block of this CTA's H tile
    constexpr int kBlkE = NB * kKB * 2;
    constexpr int kNB = 2;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sE = smem;
    uint8_t *sH = smem + kSmemE;
    uint64_t *bars = (uint64_t *)(smem + kSmemE + kStages * kStage);
    uint64_t *e_full = bars + 0, *e_empty = bars + 1;
    uint64_t *h_full = bars + 2, *h_empty = h_full + kStages;
    uint64_t *t_full = h_empty + kStages, *t_empty = t_full + kNB, *first_done = t_empty + kNB;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + kNB);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    const bool leader = rank == 0;
    const int cluster_id = blockIdx.x / 2, nclusters = gridDim.x / 2;
    const int ntap = P.NPXP / (2 * kM);           // pairs of a tiles
    const int ntbn = P.ntb * kM / kN;             // tiles of 2 NB grid rows
    const int nitems = ntap * ntbn * P.nzs * P.nb;

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(e_full, 1);
        ptx::mbar_init(e_empty, 2);
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(h_full + i, 1);
            ptx::mbar_init(h_empty + i, 2);
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

    auto decode = [&](int item, int &ta, int &tbn, int &sp, int &bi) {   // a pairs fastest: neighbours share the Ey tile
        ta = (item % ntap) * 2 + (int)rank;
        item /= ntap;
        tbn = item % ntbn;
        item /= ntbn;
        sp = item % P.nzs;
        bi = item / P.nzs;
    };
    auto zrange = [&](int bi, int sp, int &z0, int &z1) {
        const int *zb = P.zb + (size_t)bi * (P.nzs + 1) + sp;
        z0 = __ldg(zb);
        z1 = __ldg(zb + 1);
    };

    if (warp < 4) {
      setmaxnreg_dec_48();
      if (warp == 0) {
        // ===================================================================== TMA producer (both CTAs)
        int slot = 0;
        uint32_t phase = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            int ta, tbn, sp, bi;
            decode(item, ta, tbn, sp, bi);
            ptx::mbar_wait(e_empty, (uint32_t)((it_local & 1) ^ 1));
            if (ptx::elect_one()) {
                if (leader) ptx::mbar_arrive_expect_tx(e_full, (uint32_t)(2 * 4 * P.nkb * kBlkE));
                for (int pl = 0; pl < 4; ++pl)
                    for (int kb = 0; kb < P.nkb; ++kb)
                        ptx::tma_load_3d_2sm(sE + (pl * P.nkb + kb) * kBlkE, &tmA, e_full, kb * kKB, tbn * kN + (int)rank * NB, pl);
            }
            __syncwarp();
            int z0, z1;
            zrange(bi, sp, z0, z1);
            LiveSlices un;
            un.begin(P.flags, P.nkb, z0, z1, lane);
            int n;
            uint32_t m;
            while (un.next(n, m)) {
                const int row = (z0 + n) * P.NPXP + ta * kM;
                for (int kb = 0; kb < P.nkb; ++kb) {
                    if (((m >> kb) & 1u) == 0u) continue;
                    for (int ph = 0; ph < 2; ++ph) {   // Re planes, Im planes
                        ptx::mbar_wait(h_empty + slot, phase ^ 1);
                        if (ptx::elect_one()) {
                            if (leader) ptx::mbar_arrive_expect_tx(h_full + slot, (uint32_t)(2 * kStage));
                            ptx::tma_load_3d_2sm(sH + slot * kStage, &tmB, h_full + slot, kb * kKB, row, 2 * ph);
                            ptx::tma_load_3d_2sm(sH + slot * kStage + kSlotA, &tmB, h_full + slot, kb * kKB, row, 2 * ph + 1);
                        }
                        __syncwarp();
                        if (++slot == kStages) { slot = 0; phase ^= 1; }
                    }
                }
            }
        }
      } else if ((warp == 1 || warp == 3) && leader) {
        // ===================================================================== MMA issuers (leader; k-step ks belongs to issuer ks % 2)
        constexpr uint32_t idesc_pos = ptx::umma_idesc_f16(2 * kM, kN, false);
        constexpr uint32_t idesc_neg = ptx::umma_idesc_f16(2 * kM, kN, true);
        const uint64_t descH0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sH));
        const uint64_t descE0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sE));
        constexpr uint64_t kR = kSlotA >> 4, kSt = kStage >> 4, kE = kBlkE >> 4;
        const int iw = warp >> 1;
        int slot = 0;
        uint32_t phase = 0, u = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            int ta, tbn, sp, bi;
            decode(item, ta, tbn, sp, bi);
            ptx::mbar_wait(e_full, (uint32_t)(it_local & 1));
            ptx::tc_fence_after();
            const uint64_t kEpl = (uint64_t)P.nkb * kE;   // descriptor distance between Ey planes
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
                    for (int ph = 0; ph < 2; ++ph) {
                        if (first && ph == 0 && iw == 1) {   // D must have been initialised by issuer 0
                            ptx::mbar_wait(first_done + buf, upar);
                            ptx::tc_fence_after();
                        }
                        ptx::mbar_wait(h_full + slot, phase);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
#pragma unroll
                            for (int kk = 0; kk < 2; ++kk) {
                                const int ks = 2 * kk + iw;
                                const uint64_t a_hi = descH0 + (uint64_t)slot * kSt + (uint64_t)(ks * 2), a_lo = a_hi + kR;
                                const uint64_t e_reh = descE0 + (uint64_t)kb * kE + (uint64_t)(ks * 2);
                                const uint64_t e_rel = e_reh + kEpl, e_imh = e_rel + kEpl, e_iml = e_imh + kEpl;
                                const uint32_t acc0 = (first && ph == 0 && ks == 0) ? 0u : 1u;
                                // (Hr + i Hi)(Er + i Ei), the H planes of this stage as A, three split products HhEh + HlEh + HhEl
                                if (ph == 0) {
                                    ptx::umma_f16_2sm(d_re, a_hi, e_reh, idesc_pos, acc0);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_imh, idesc_pos, acc0);
                                    ptx::umma_f16_2sm(d_re, a_hi, e_rel, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_iml, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_lo, e_reh, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_im, a_lo, e_imh, idesc_pos, 1u);
                                } else {
                                    ptx::umma_f16_2sm(d_re, a_hi, e_imh, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_reh, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_hi, e_iml, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, e_rel, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_lo, e_imh, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_lo, e_reh, idesc_pos, 1u);
                                }
                                if (first && ph == 0 && iw == 0 && kk == 0) ptx::umma_commit_2sm(first_done + buf, (uint16_t)0x1);
                            }
                            ptx::umma_commit_2sm(h_empty + slot, (uint16_t)0x3);
                        }
                        __syncwarp();
                        if (++slot == kStages) { slot = 0; phase ^= 1; }
                    }
                    first = false;
                }
                if (ptx::elect_one()) ptx::umma_commit_2sm(t_full + buf, (uint16_t)0x3);
                __syncwarp();
                ++u;
            }
            if (ptx::elect_one()) ptx::umma_commit_2sm(e_empty, (uint16_t)0x3);
            __syncwarp();
        }
      }
    } else {
        setmaxnreg_inc_224();
        // ===================================================================== epilogue: Blocks 7-8; thread = (column a, NB rows b)
        const int lg = warp & 3, ch = (warp - 4) >> 2;
        const uint32_t t_lane = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(ch * NB);
        uint32_t u = 0;
        for (int item = cluster_id; item < nitems; item += nclusters) {
            int ta, tbn, sp, bi;
            decode(item, ta, tbn, sp, bi);
            const int a = ta * kM + lg * 32 + lane;
            const int b0 = tbn * kN + ch * NB;
            const double qxa = a < P.npx ? P.qx[a] : 0.0;
            uint32_t dph[NB];
#pragma unroll
            for (int c = 0; c < NB; ++c) {
                const int b = b0 + c;
                double t = 0.0;
                if (a < P.npx && b < P.npy) {
                    const double qyb = P.qy[b];
                    const double qxy2 = qxa * qxa + qyb * qyb;
                    const double kz2 = P.k * P.k - qxy2;
                    const double qz = kz2 >= 0.0 ? -qxy2 / (P.k + sqrt(kz2)) : 0.0;
                    t = qz * P.dz * (0.25 / 3.14159265358979323846);
                    t -= rint(t);
                }
                dph[c] = (uint32_t)(long long)rint(t * 4294967296.0);
            }
            float2 tot[NB];
#pragma unroll
            for (int c = 0; c < NB; ++c) tot[c] = make_float2(0.f, 0.f);
            int z0, z1;
            zrange(bi, sp, z0, z1);
            LiveSlices un;
            un.begin(P.flags, P.nkb, z0, z1, lane);
            int n;
            uint32_t m;
            while (un.next(n, m)) {
                const int j = z0 + n - bi * P.nz;
                SCATMAN_ASSERT(j >= 0 && j < P.nz && bi < P.nb && sp < P.nzs);
                const uint32_t buf = u % kNB, upar = (u / kNB) & 1;
                const uint32_t mult = (uint32_t)(2 * j - P.nz + 1);
                ptx::mbar_wait(t_full + buf, upar);
                ptx::tc_fence_after();
                const uint32_t t_re = t_lane + buf * 256, t_im = t_re + 128;
#pragma unroll
                for (int q8 = 0; q8 < NB / 8; ++q8) {
                    uint32_t gre[8], gim[8];
                    ptx::tmem_ld8(t_re + q8 * 8, gre);
                    ptx::tmem_ld8(t_im + q8 * 8, gim);
                    ptx::tmem_ld_wait();
                    if (q8 == NB / 8 - 1) {
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
            if (a < P.npx) {   // a warp stores 32 consecutive a of one grid row
                float2 *dst = P.partial + ((size_t)bi * P.nzs + sp) * P.npy * P.npx + a;
#pragma unroll
                for (int c = 0; c < NB; ++c)
                    if (b0 + c < P.npy) dst[(size_t)(b0 + c) * P.npx] = tot[c];
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
    t.nyz = npx > kNyz ? 128 : kNyz;   // stage YZ accumulator width: 128 columns (full-rate UMMA) unless the grid is narrower
    t.NPXP = (npx + t.nyz - 1) / t.nyz * t.nyz;
    t.NPYP = (npy + kM - 1) / kM * kM;
    t.ng = t.NY / 128;
    int L = 0;
    while ((1 << L) < p.nx) ++L;
    t.L = L;
    // items per chunk (stacked along z, one set of launches per chunk): as many as keep the H planes of a chunk under 4 GB
    const size_t h_item = (size_t)8 * p.nz * t.NPXP * t.NY;
    size_t nb = ((size_t)4 << 30) / (h_item ? h_item : 1);
    if (nb > (size_t)p.batch) nb = (size_t)p.batch;
    if (nb * p.nz > 60000) nb = 60000 / (size_t)p.nz;   // global slice index and TMA row coordinates stay small
    t.nb = nb < 1 ? 1 : (int)nb;
    // z splits: minimise waves x (slices per item + ~3 slice-equivalents of fill: Ey tile load, pipeline ramp, partial store)
    // stage YZ runs on CTA pairs (UMMA 256 x 128) when it uses 128-column accumulators and the b tiles pair up
    // stage YZ variants, in order of preference (each needs its tiles to pair up for cta_group::2):
    //   sep_tc_yzt_kernel   pairs of a tiles, Ey resident for all y (N_y <= 256)
    //   sep_tc_yzs_kernel   pairs of b tiles, both operands streamed (N_y <= 2048)
    //   sep_tc_yz128_kernel one CTA, Ey resident per 128-y group, one accumulator per (slice, group): any size
    //   sep_tc_yz_kernel    the same with 64-column accumulators, for grids of at most 64 columns
    t.yz_stream = t.nyz == 128 && (t.NPYP / kM) % 2 == 0 && t.NY / kKB <= 32;
    t.yz_ncta = t.yz_stream ? 2 : 1;
    // transposed form (sep_tc_yzt_kernel): pairs of a tiles, the Ey tile of 2 NB rows resident for all y
    t.yzt_nb = t.NY / kKB <= 4 ? 64 : 0;   // (NB = 32 / 16 for taller grids run UMMA N = 64 / 32: measured slower than the streamed form)
    t.yz_t = t.nyz == 128 && (t.NPXP / kM) % 2 == 0 && t.yzt_nb != 0;
    if (t.yz_t) { t.yz_stream = true; t.yz_ncta = 2; }   // same bounds / partial layout as the streamed form
    const int base = t.yz_t ? (t.NPXP / (2 * kM)) * (t.NPYP / (2 * t.yzt_nb)) * t.nb
                            : (t.NPYP / kM / t.yz_ncta) * (t.NPXP / t.nyz) * (t.yz_stream ? 1 : t.ng) * t.nb;
    const int workers = num_sms / t.yz_ncta;
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
    t.nsplit = (t.yz_stream ? 1 : t.ng) * t.nzs;
    // stage X: a columns per resident Ex tile (NX * NXP * 8 bytes <= 128 KB), z splits for ~4 waves of a-tile items
    t.NX = t.NXP <= 256 ? 64 : t.NXP <= 512 ? 32 : 16;
    t.x_ncta = t.NPXP % (2 * t.NX) == 0 ? 2 : 1;   // CTA pairs (UMMA 256 x 2NX) when the column tiles pair up
    const int nta = t.NPXP / (t.NX * t.x_ncta);
    int nsx = (2 * (num_sms / t.x_ncta) + nta - 1) / nta;   // two balanced items per CTA (pair)
    t.nsx = nsx < 1 ? 1 : nsx > p.nz * t.nb ? p.nz * t.nb : nsx;
    return t;
}

constexpr int kSmemYz = 1024 + 4 * 2 * kSlotA + 3 * (4 * kNyz * kKB * 2) + 256;   // every stage YZ variant: 128 KB resident + 96 KB ring
constexpr int kSmemX = 1024 + 131072 + 6 * kSlotA + 256;                           // every stage X variant

// Function attributes belong to a device's context: set for the CURRENT device by scatman_create.
cudaError_t sep_tc_init_device() {
    const cudaFuncAttribute attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
    cudaError_t e = cudaFuncSetAttribute(sep_tc_yz_kernel, attr, kSmemYz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_yz128_kernel<1>, attr, kSmemYz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_yzs_kernel, attr, kSmemYz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_yzt_kernel<64>, attr, kSmemYz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_x_kernel<64>, attr, kSmemX);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_x_kernel<32>, attr, kSmemX);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_x_kernel<16>, attr, kSmemX);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_x2_kernel<64>, attr, kSmemX);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_x2_kernel<32>, attr, kSmemX);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sep_tc_x2_kernel<16>, attr, kSmemX);
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

template <int NCTA>
static cudaError_t launch_yz128_variant(const CUtensorMap &tmA, const CUtensorMap &tmB, const SepYzParams &P, int nitems, int num_sms,
                                        int smem, cudaStream_t st) {
    const int max_clusters = num_sms / NCTA;
    const int nclusters = nitems < max_clusters ? nitems : max_clusters;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(nclusters * NCTA));
    cfg.blockDim = dim3(kThreadsTc);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = NCTA;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, sep_tc_yz128_kernel<NCTA>, tmA, tmB, P);
}

cudaError_t launch_sep_tc_yz(const Plan &p, const SepTcPlan &t, const __half *d_Eyp, const __half *d_Hp,
                             const unsigned char *d_flags64, const int *d_bounds, int nb, const double *d_qx, int npx,
                             const double *d_qy, int npy, float2 *d_partial, int num_sms, cudaStream_t st, std::string *err) {
    constexpr int kSmem = kSmemYz;
    const int ncta = t.nyz == 128 ? t.yz_ncta : 1;
    CUtensorMap tmA, tmB;
    bool ok;
    {
        cuuint64_t dims[3] = {(cuuint64_t)t.NY, (cuuint64_t)t.NPYP, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * (cuuint64_t)t.NPYP * 2};
        cuuint32_t box[3] = {(cuuint32_t)kKB, (cuuint32_t)kM, 1};
        ok = encode_map(&tmA, d_Eyp, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (ok) {   // box = one CTA's rows of an H tile
        const cuuint64_t rows = (cuuint64_t)p.nz * nb * t.NPXP;
        cuuint64_t dims[3] = {(cuuint64_t)t.NY, rows, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * rows * 2};
        cuuint32_t box[3] = {(cuuint32_t)kKB, (cuuint32_t)(t.nyz / ncta), 1};
        ok = encode_map(&tmB, d_Hp, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (!ok) {
        if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
        return cudaErrorUnknown;
    }
    SepYzParams P;
    P.nz = p.nz; P.nb = nb; P.npx = npx; P.npy = npy; P.NY = t.NY; P.NPXP = t.NPXP; P.ng = t.ng; P.nzs = t.nzs;
    P.ntb = t.NPYP / kM; P.nta = t.NPXP / t.nyz; P.nkb = t.NY / kKB;
    P.k = 2.0 * 3.14159265358979323846 / p.lambda; P.dz = p.dz;
    P.qx = d_qx; P.qy = d_qy; P.flags = d_flags64; P.zb = d_bounds + (t.nsx + 1); P.partial = d_partial;
    if (t.yz_t) {
        // A map: the Ey planes, box = this CTA's NB rows of one 64-y block; B map: the H planes, box = a whole a tile
        cuuint64_t dimsA[3] = {(cuuint64_t)t.NY, (cuuint64_t)t.NPYP, 4};
        cuuint64_t stridesA[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * (cuuint64_t)t.NPYP * 2};
        cuuint32_t boxA[3] = {(cuuint32_t)kKB, (cuuint32_t)t.yzt_nb, 1};
        const cuuint64_t rows = (cuuint64_t)p.nz * nb * t.NPXP;
        cuuint64_t dimsB[3] = {(cuuint64_t)t.NY, rows, 4};
        cuuint64_t stridesB[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * rows * 2};
        cuuint32_t boxB[3] = {(cuuint32_t)kKB, (cuuint32_t)kM, 1};
        if (!encode_map(&tmA, d_Eyp, 3, dimsA, stridesA, boxA, CU_TENSOR_MAP_SWIZZLE_128B) ||
            !encode_map(&tmB, d_Hp, 3, dimsB, stridesB, boxB, CU_TENSOR_MAP_SWIZZLE_128B)) {
            if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
            return cudaErrorUnknown;
        }
        const int nit = (t.NPXP / (2 * kM)) * (t.NPYP / (2 * t.yzt_nb)) * P.nzs * nb, maxc = num_sms / 2;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(2 * (nit < maxc ? nit : maxc)));
        cfg.blockDim = dim3(kThreadsTc);
        cfg.dynamicSmemBytes = kSmem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, sep_tc_yzt_kernel<64>, tmA, tmB, P);
    }
    if (t.yz_stream) {
        const int nit = (P.ntb / 2) * P.nta * P.nzs * nb, maxc = num_sms / 2;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(2 * (nit < maxc ? nit : maxc)));
        cfg.blockDim = dim3(kThreadsTc);
        cfg.dynamicSmemBytes = kSmem;
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
    const int nitems = (P.ntb / ncta) * P.nta * P.ng * P.nzs * nb;
    if (t.nyz == 128) return launch_yz128_variant<1>(tmA, tmB, P, nitems, num_sms, kSmem, st);
    sep_tc_yz_kernel<<<nitems < num_sms ? nitems : num_sms, kThreadsTc, kSmem, st>>>(tmA, tmB, P);
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

template <int NX>
static cudaError_t launch_x_variant(const CUtensorMap &tmA, const CUtensorMap &tmB, const SepXParams &P, int num_sms,
                                    cudaStream_t st) {
    constexpr int kSmem = kSmemX;
    const int nitems = P.nta * P.nsx;
    sep_tc_x_kernel<NX><<<nitems < num_sms ? nitems : num_sms, kThreadsTc, kSmem, st>>>(tmA, tmB, P);
    return cudaGetLastError();
}

template <int NX>
static cudaError_t launch_x2_variant(const CUtensorMap &tmA, const CUtensorMap &tmB, const SepXParams &P, int num_sms,
                                     cudaStream_t st) {
    constexpr int kSmem = kSmemX;
    const int nitems = P.nta * P.nsx, max_clusters = num_sms / 2;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(2 * (nitems < max_clusters ? nitems : max_clusters)));
    cfg.blockDim = dim3(kThreadsTc);
    cfg.dynamicSmemBytes = kSmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, sep_tc_x2_kernel<NX>, tmA, tmB, P);
}

cudaError_t launch_sep_tc_x(const Plan &p, const SepTcPlan &t, const __half *d_Rp, const __half *d_Exp,
                            const unsigned char *d_flags64, const int *d_bounds, int nb, __half *d_Hp, int num_sms,
                            cudaStream_t st, std::string *err) {
    CUtensorMap tmA, tmB;
    bool ok;
    {
        const cuuint64_t rows = (cuuint64_t)p.nz * nb * t.NY;
        cuuint64_t dims[3] = {(cuuint64_t)t.NXP, rows, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NXP * 2, (cuuint64_t)t.NXP * rows * 2};
        cuuint32_t box[3] = {(cuuint32_t)kKB, (cuuint32_t)kM, 1};
        ok = encode_map(&tmA, d_Rp, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (ok) {
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
    P.nz = p.nz * nb; P.NY = t.NY; P.NPXP = t.NPXP; P.ng = t.ng; P.nkx = t.NXP / kKB; P.nta = t.NPXP / (t.NX * t.x_ncta);
    P.nsx = t.nsx;
    P.nkb = t.NY / kKB;
    P.hscale = ldexpf(1.f, -9 - t.L);
    P.flags = d_flags64; P.zb = d_bounds; P.Hp = d_Hp;
    if (t.x_ncta == 2) {
        switch (t.NX) {
            case 64: return launch_x2_variant<64>(tmA, tmB, P, num_sms, st);
            case 32: return launch_x2_variant<32>(tmA, tmB, P, num_sms, st);
            default: return launch_x2_variant<16>(tmA, tmB, P, num_sms, st);
        }
    }
    switch (t.NX) {
        case 64: return launch_x_variant<64>(tmA, tmB, P, num_sms, st);
        case 32: return launch_x_variant<32>(tmA, tmB, P, num_sms, st);
        default: return launch_x_variant<16>(tmA, tmB, P, num_sms, st);
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
