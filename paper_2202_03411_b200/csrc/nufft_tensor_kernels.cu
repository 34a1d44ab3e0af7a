// nufft_tensor_kernels.cu -- the three GEMM stages of the NUFFT route (nufft_kernels.cu) on tcgen05 tensor cores.
//
// The uniform-grid transform U[mz][my][mx] = sum_r c_z c_y c_x rho~(r) e^{i g_m . r} is separable: three complex GEMMs against
// window-corrected phase tables.  Here they run in the FP16x3 split precision of the other tensor-core kernels (every operand =
// four FP16 planes of a scaled FP32 value, AhBh + AlBh + AhBl, FP32 accumulation in TMEM), chained so that the TMEM lane (row)
// dimension of one stage is the contraction dimension of the next -- each epilogue then writes its result K-major for its
// successor with coalesced stores, and no transposition pass exists:
//   stage X  H[j][mx][y]  = sum_x rho~[j][y][x]  Tx[mx][x]     rows y   (sep_tc_x*_kernel of sep_tensor_kernels.cu, reused as it is)
//   stage Y  V[mx][my][j] = sum_y H[j][mx][y]    Ty[my][y]     rows j   (tc_cgemm.cuh, StageY)
//   stage Z  U[mz][my][mx] = sum_j V[mx][my][j]  Tz[mz][j]     rows mx  (tc_cgemm.cuh, StageZ; FP32 complex out, mx fastest)
// Batch items are stacked along j (global slice jg = b nz + j); only stage Z knows about items (its K range is one item's slices,
// the Tz planes are zero beyond nz).  Scales: rho~ planes 2^(13-e) per item, tables 2^10, H and V stored with constant
// power-of-two rescalings that keep them in FP16 range whatever the data (|H|, |V| <= 2^14.5); the interpolation undoes all of
// them with one factor per item.  Precision: each factor carries 22 bits; measured against the FP64 stages in
// tests/test_gpu_nufft.py and profiles/r02_nufft_tensor.md.
#include <cuda.h>

#include <cstdio>

#include "internal.h"
#include "ptx_sm100.h"
#include "tc_cgemm.cuh"

namespace scatman {

bool encode_map(CUtensorMap *tm, const void *base, int rank, const cuuint64_t *dims, const cuuint64_t *strides,
                const cuuint32_t *box, CUtensorMapSwizzle swizzle);   // tensor_kernel.cu
double nufft_inv_i0_beta();                                            // nufft_kernels.cu

namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr double kHalfW = 0.5 * kNufftW;
__host__ __device__ inline double kb_beta_tc() { return kPi * sqrt(kHalfW * kHalfW * 2.25 - 0.8); }

// T planes fp16 [4][rows_pad][kpad] = split(2^10 c_i e^{i g_m x_i}), the table of nufft_table_kernel (exact integer phase
// reduction, window correction c_i = 1 / Phi(h x_i)) as a K-major tensor-core operand; zero in the padding (rows >= nq, i >= N).
__global__ void nufft_tc_table_kernel(int N, int nq, int m_lo, int rows_pad, int kpad, double inv_i0b, __half *__restrict__ T) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (int64_t)rows_pad * kpad) return;
    const int m = (int)(e / kpad), i = (int)(e % kpad);
    float re = 0.f, im = 0.f;
    if (m < nq && i < N) {
        const int nf = 2 * N;
        const int64_t c2 = 2 * i - N + 1;
        const int64_t t = ((int64_t)(m_lo + m) * c2) % (2 * (int64_t)nf);
        double s, c;
        sincospi((double)t / (double)nf, &s, &c);
        const double beta = kb_beta_tc();
        const double theta = kPi * (double)c2 / (double)nf;
        const double r = sqrt(beta * beta - kHalfW * kHalfW * theta * theta);
        const double corr = (double)kScaleA / (2.0 * kHalfW * sinh(r) / r * inv_i0b);
        re = (float)(corr * c);
        im = (float)(corr * s);
    }
    __half h[4];
    tcg::split4h(re, im, h);
    const size_t plane = (size_t)rows_pad * kpad;
#pragma unroll
    for (int pl = 0; pl < 4; ++pl) T[pl * plane + e] = h[pl];
}

// ---- stage Y: rows = global slices jg (tiles of 128), K = y, columns = my; out V planes [4][NPXP][NQYP][NZT] (jg fastest)
struct YParams {
    int nk;                 // NY / 64
    int ntb, nunits, nsplit;
    int njt, ntot;          // j tiles of 128 slices; slices of the chunk (nb nz)
    int nz, NZI;            // slices per item; the same padded to 8: item b's slices sit at [b NZI, b NZI + nz) of a V row, so
                            // that stage Z's TMA boxes start 16-byte aligned (a box start that is not raises an illegal-instruction fault)
    int NQYP, NZT;          // padded columns; row length of V (nb NZI)
    int nqy;                // columns my < nqy are stored (stage Z reads no others)
    float hscale;           // accumulator -> stored V
    const unsigned char *flags;   // non-null (NY = 128 only): flags64[jg][2] of the separable pack; a slice with no flag set was not
                            // written by stage X at all -- its rows of H hold whatever was there and its rows of V are written as zeros
    __half *Vp;
    size_t plane;           // elements per V plane
};
struct GItem {
    int tb, u_begin, u_end;
};

template <int NB_>
struct StageY {
    static constexpr int NB = NB_;
    static constexpr bool kUnrollEpilogue = false;
    static constexpr int kEpilogueRegs = 0;
    using Params = YParams;
    using Item = GItem;
    __device__ static int nitems(const Params &P) { return P.ntb * P.nsplit; }
    __device__ static Item item(const Params &P, int index) {
        Item it;
        it.tb = index % P.ntb;   // column tiles fastest: concurrent pairs stream the same H tiles
        const int s = index / P.ntb;
        it.u_begin = (int)(((long long)P.nunits * s) / P.nsplit);
        it.u_end = (int)(((long long)P.nunits * (s + 1)) / P.nsplit);
        return it;
    }
    __device__ static int b_row0(const Params &, const Item &it) { return it.tb * 2 * NB; }
    struct Units : tcg::RangeUnits {
        __device__ void begin(const Params &, const Item &it, int) { set(it.u_begin, it.u_end); }
    };
    // unit = mx * njt + jt
    __device__ static void a_coords(const Params &P, const Item &, int unit, int kb, int (&c)[3]) {
        c[0] = kb * tcg::kKB;
        c[1] = (unit % P.njt) * tcg::kM;
        c[2] = unit / P.njt;
    }
    struct Epilogue {
        __device__ void begin(const Params &, const Item &, const tcg::EpiThread &) {}
        int jg, jv, mx;      // global slice; its position in a V row; uniform-grid column
        bool dead;           // the slice holds no material: stage X left its rows of H unwritten (row j of the product depends on row j only)
        __device__ void unit_begin(const Params &P, const Item &, const tcg::EpiThread &et, int unit) {
            jg = (unit % P.njt) * tcg::kM + et.lane_row;
            const int b = jg / P.nz;
            jv = b * P.NZI + (jg - b * P.nz);
            mx = unit / P.njt;
            dead = false;
            if (P.flags && jg < P.ntot) dead = (P.flags[2 * (size_t)jg] | P.flags[2 * (size_t)jg + 1]) == 0;
        }
        __device__ void columns(const Params &P, const Item &it, const tcg::EpiThread &et, int, int c0, const uint32_t (&gre)[8],
                                const uint32_t (&gim)[8]) {
            if (jg >= P.ntot) return;
            const int my0 = it.tb * 2 * NB + et.col0 + c0;
            SCATMAN_ASSERT(my0 + 8 <= P.NQYP && jv < P.NZT);
            __half *dst = P.Vp + ((size_t)mx * P.NQYP + my0) * P.NZT + jv;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (my0 + i >= P.nqy) break;
                __half h[4];
                tcg::split4h(dead ? 0.f : __uint_as_float(gre[i]) * P.hscale, dead ? 0.f : __uint_as_float(gim[i]) * P.hscale, h);
                __half *d = dst + (size_t)i * P.NZT;
#pragma unroll
                for (int pl = 0; pl < 4; ++pl) d[pl * P.plane] = h[pl];
            }
        }
        __device__ void end(const Params &, const Item &, const tcg::EpiThread &) {}
    };
};

// ---- stage Z: rows = mx (tiles of 128), K = the slices of ONE item, columns = mz; out U float2 [nb][nqz][nqy][nqx]
struct ZParams {
    int nk;                 // ceil(nz / 64)
    int ntb, nunits, nsplit;
    int nmt, nqx, nqy, nqz, NZI;   // NZI: stride between the items' slices in a V row (nz padded to 8)
    float2 *U;
};

template <int NB_>
struct StageZ {
    static constexpr int NB = NB_;
    static constexpr bool kUnrollEpilogue = false;
    static constexpr int kEpilogueRegs = 0;
    using Params = ZParams;
    using Item = GItem;
    __device__ static int nitems(const Params &P) { return P.ntb * P.nsplit; }
    __device__ static Item item(const Params &P, int index) {
        Item it;
        it.tb = index % P.ntb;
        const int s = index / P.ntb;
        it.u_begin = (int)(((long long)P.nunits * s) / P.nsplit);
        it.u_end = (int)(((long long)P.nunits * (s + 1)) / P.nsplit);
        return it;
    }
    __device__ static int b_row0(const Params &, const Item &it) { return it.tb * 2 * NB; }
    struct Units : tcg::RangeUnits {
        __device__ void begin(const Params &, const Item &it, int) { set(it.u_begin, it.u_end); }
    };
    // unit = (b * nqy + my) * nmt + mt; the K range of item b starts at its first global slice
    __device__ static void a_coords(const Params &P, const Item &, int unit, int kb, int (&c)[3]) {
        const int mt = unit % P.nmt, bm = unit / P.nmt;
        c[0] = (bm / P.nqy) * P.NZI + kb * tcg::kKB;
        c[1] = mt * tcg::kM;
        c[2] = bm % P.nqy;
    }
    struct Epilogue {
        __device__ void begin(const Params &, const Item &, const tcg::EpiThread &) {}
        int mx;
        float2 *base;
        __device__ void unit_begin(const Params &P, const Item &, const tcg::EpiThread &et, int unit) {
            const int mt = unit % P.nmt, bm = unit / P.nmt;
            mx = mt * tcg::kM + et.lane_row;
            const int b = bm / P.nqy, my = bm % P.nqy;
            base = P.U + (((size_t)b * P.nqz) * P.nqy + my) * P.nqx + mx;   // + mz nqy nqx
        }
        __device__ void columns(const Params &P, const Item &it, const tcg::EpiThread &et, int, int c0, const uint32_t (&gre)[8],
                                const uint32_t (&gim)[8]) {
            if (mx >= P.nqx) return;
            const int mz0 = it.tb * 2 * NB + et.col0 + c0;
#pragma unroll
            for (int i = 0; i < 8; ++i)
                if (mz0 + i < P.nqz)
                    base[(size_t)(mz0 + i) * P.nqy * P.nqx] = make_float2(__uint_as_float(gre[i]), __uint_as_float(gim[i]));
        }
        __device__ void end(const Params &, const Item &, const tcg::EpiThread &) {}
    };
};

// columns of B resident per CTA: the largest of 64 / 32 / 16 whose K fits (nk NB <= 256) and that does not pad the columns by a whole tile half
int pick_nb(int ncols, int nk) {
    const int cand[3] = {64, 32, 16};
    for (int i = 0; i < 3; ++i) {
        const int nb = cand[i];
        if (nk * nb > 256) continue;
        const int padded = (ncols + 2 * nb - 1) / (2 * nb) * (2 * nb);
        if (nb == 16 || padded - ncols < nb) return nb;
    }
    return 0;
}

int split_for(int ntb, int nunits, int num_sms) {
    int s = (2 * (num_sms / 2) + ntb - 1) / ntb;      // ~two items per CTA pair
    const int maxs = (nunits + 1) / 2;                // at least one unit pair per item
    if (s > maxs) s = maxs;
    return s < 1 ? 1 : s;
}

}  // namespace

cudaError_t nufft_tc_init_device() {
    cudaError_t e = tcg::cgemm_init_device<StageY<64>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<StageY<32>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<StageY<16>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<StageZ<64>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<StageZ<32>>();
    if (e == cudaSuccess) e = tcg::cgemm_init_device<StageZ<16>>();
    return e;
}

// Layout of the tensor-core stages for a chunk of items; ok = false when a dimension does not fit the resident operands
// (nx, ny or nz above 1024): the caller then uses the FP64 stages.
NufftTcPlan make_nufft_tc_plan(const Plan &p, const NufftPlan &n, int batch, int num_sms) {
    NufftTcPlan t;
    Plan q = p;
    q.batch = batch;
    t.sep = make_sep_tc_plan(q, n.ax.nq, n.ay.nq, num_sms);   // stage X = the separable route's stage X on nqx "pixels"
    t.NY = t.sep.NY;
    t.NPXP = t.sep.NPXP;
    t.nky = t.NY / tcg::kKB;
    t.nkz = (p.nz + tcg::kKB - 1) / tcg::kKB;
    t.NZP = t.nkz * tcg::kKB;
    t.nby = pick_nb(n.ay.nq, t.nky);
    t.nbz = pick_nb(n.az.nq, t.nkz);
    t.ok = p.nx <= 1024 && t.nby != 0 && t.nbz != 0;
    if (!t.ok) return t;
    t.NQYP = (n.ay.nq + 2 * t.nby - 1) / (2 * t.nby) * (2 * t.nby);
    t.NQZP = (n.az.nq + 2 * t.nbz - 1) / (2 * t.nbz) * (2 * t.nbz);
    // items per chunk: the separable plan's (H planes under 4 GB), further limited so that V stays under 2 GB
    int nb = t.sep.nb;
    const double v_item = 8.0 * (double)t.NPXP * t.NQYP * p.nz;
    while (nb > 1 && v_item * nb > 2147483648.0) --nb;
    t.nb = nb;
    t.NZI = (p.nz + 7) / 8 * 8;
    t.NZT = nb * t.NZI;
    return t;
}

cudaError_t launch_nufft_tc_tables(const Plan &p, const NufftPlan &n, const NufftTcPlan &t, __half *d_Tx, __half *d_Ty, __half *d_Tz,
                                   cudaStream_t st) {
    const double inv_i0b = nufft_inv_i0_beta();
    int64_t e = (int64_t)t.NPXP * t.sep.NXP;
    nufft_tc_table_kernel<<<(unsigned)((e + 255) / 256), 256, 0, st>>>(p.nx, n.ax.nq, n.ax.m_lo, t.NPXP, t.sep.NXP, inv_i0b, d_Tx);
    e = (int64_t)t.NQYP * t.NY;
    nufft_tc_table_kernel<<<(unsigned)((e + 255) / 256), 256, 0, st>>>(p.ny, n.ay.nq, n.ay.m_lo, t.NQYP, t.NY, inv_i0b, d_Ty);
    e = (int64_t)t.NQZP * t.NZP;
    nufft_tc_table_kernel<<<(unsigned)((e + 255) / 256), 256, 0, st>>>(p.nz, n.az.nq, n.az.m_lo, t.NQZP, t.NZP, inv_i0b, d_Tz);
    return cudaGetLastError();
}

template <int NB>
static cudaError_t run_stage_y(const CUtensorMap &tmA, const CUtensorMap &tmB, const YParams &P, int num_sms, cudaStream_t st) {
    return tcg::cgemm_launch<StageY<NB>>(tmA, tmB, P, P.ntb * P.nsplit, num_sms, st);
}
template <int NB>
static cudaError_t run_stage_z(const CUtensorMap &tmA, const CUtensorMap &tmB, const ZParams &P, int num_sms, cudaStream_t st) {
    return tcg::cgemm_launch<StageZ<NB>>(tmA, tmB, P, P.ntb * P.nsplit, num_sms, st);
}

// Stages Y and Z for a chunk of nb items whose H planes [4][nb nz][NPXP][NY] stage X has written.  The tiles stage X did not write
// (no material) must read as zero: the caller zeroes H first -- or, when a slice is one 128-y tile (NY = 128), passes the flags of
// the pack (d_flags64) and stage Y writes the rows of such slices as zeros whatever H holds (nufft_tc_needs_h_memset).
bool nufft_tc_needs_h_memset(const NufftTcPlan &t) { return t.NY != tcg::kM; }
cudaError_t launch_nufft_tc_yz(const Plan &p, const NufftPlan &n, const NufftTcPlan &t, int nb, const __half *d_Hp, const __half *d_Ty,
                               const __half *d_Tz, __half *d_Vp, float2 *d_U, int num_sms, cudaStream_t st, std::string *err,
                               const unsigned char *d_flags64) {
    const int ntot = nb * p.nz;
    const size_t h_plane = (size_t)ntot * t.NPXP * t.NY, v_plane = (size_t)t.NPXP * t.NQYP * t.NZT;
    CUtensorMap tmA, tmB;
    bool ok;
    {   // A of stage Y: H planes seen as (y, jg, mx, plane); a unit's box = 64 y x 128 slices of one mx
        cuuint64_t dims[4] = {(cuuint64_t)t.NY, (cuuint64_t)ntot, (cuuint64_t)t.NPXP, 4};
        cuuint64_t strides[3] = {(cuuint64_t)t.NPXP * t.NY * 2, (cuuint64_t)t.NY * 2, (cuuint64_t)h_plane * 2};
        cuuint32_t box[4] = {(cuuint32_t)tcg::kKB, (cuuint32_t)tcg::kM, 1, 1};
        ok = encode_map(&tmA, d_Hp, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (ok) {   // B of stage Y: Ty planes [4][NQYP][NY]; box = this CTA's NB rows of one 64-y block
        cuuint64_t dims[3] = {(cuuint64_t)t.NY, (cuuint64_t)t.NQYP, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NY * 2, (cuuint64_t)t.NY * t.NQYP * 2};
        cuuint32_t box[3] = {(cuuint32_t)tcg::kKB, (cuuint32_t)t.nby, 1};
        ok = encode_map(&tmB, d_Ty, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (!ok) {
        if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
        return cudaErrorUnknown;
    }
    YParams Y;
    Y.nk = t.nky;
    Y.ntb = t.NQYP / (2 * t.nby);
    Y.njt = (ntot + tcg::kM - 1) / tcg::kM;
    Y.nunits = n.ax.nq * Y.njt;
    Y.nsplit = split_for(Y.ntb, Y.nunits, num_sms);
    Y.ntot = ntot;
    Y.nz = p.nz;
    Y.NZI = t.NZI;
    Y.NQYP = t.NQYP;
    Y.nqy = n.ay.nq;
    Y.NZT = t.NZT;
    int Ly = 0;
    while ((1 << Ly) < p.ny) ++Ly;
    Y.hscale = ldexpf(1.f, -11 - Ly);     // |acc| <= 2^14.5 (H) x 2^10.5 (Ty) x 2^Ly  ->  |V| <= 2^14
    Y.Vp = d_Vp;
    Y.plane = v_plane;
    Y.flags = nufft_tc_needs_h_memset(t) ? nullptr : d_flags64;
    cudaError_t e = cudaSuccess;
    if (t.NZI != p.nz) {   // the padding between the items' slices is read by stage Z (against zero table entries): it must be finite
        e = cudaMemsetAsync(d_Vp, 0, sizeof(__half) * 4 * v_plane, st);
        if (e != cudaSuccess) return e;
    }
    e = t.nby == 64 ? run_stage_y<64>(tmA, tmB, Y, num_sms, st)
                  : t.nby == 32 ? run_stage_y<32>(tmA, tmB, Y, num_sms, st) : run_stage_y<16>(tmA, tmB, Y, num_sms, st);
#ifdef SCATMAN_CHECKED
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) fprintf(stderr, "scatman checked build: NUFFT stage Y failed: %s (nby %d nky %d ntb %d nunits %d nsplit %d)\n",
                                  cudaGetErrorString(e), t.nby, t.nky, Y.ntb, Y.nunits, Y.nsplit);
#endif
    if (e != cudaSuccess) return e;
    {   // A of stage Z: V planes seen as (slice position, mx, my, plane); box = 64 slices x 128 mx of one my
        cuuint64_t dims[4] = {(cuuint64_t)nb * t.NZI, (cuuint64_t)t.NPXP, (cuuint64_t)t.NQYP, 4};
        cuuint64_t strides[3] = {(cuuint64_t)t.NQYP * t.NZT * 2, (cuuint64_t)t.NZT * 2, (cuuint64_t)v_plane * 2};
        cuuint32_t box[4] = {(cuuint32_t)tcg::kKB, (cuuint32_t)tcg::kM, 1, 1};
        ok = encode_map(&tmA, d_Vp, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (ok) {   // B of stage Z: Tz planes [4][NQZP][NZP], zero for j >= nz
        cuuint64_t dims[3] = {(cuuint64_t)t.NZP, (cuuint64_t)t.NQZP, 4};
        cuuint64_t strides[2] = {(cuuint64_t)t.NZP * 2, (cuuint64_t)t.NZP * t.NQZP * 2};
        cuuint32_t box[3] = {(cuuint32_t)tcg::kKB, (cuuint32_t)t.nbz, 1};
        ok = encode_map(&tmB, d_Tz, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (!ok) {
        if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
        return cudaErrorUnknown;
    }
    ZParams Z;
    Z.nk = t.nkz;
    Z.ntb = t.NQZP / (2 * t.nbz);
    Z.nmt = (n.ax.nq + tcg::kM - 1) / tcg::kM;
    Z.nunits = nb * n.ay.nq * Z.nmt;
    Z.nsplit = split_for(Z.ntb, Z.nunits, num_sms);
    Z.nqx = n.ax.nq; Z.nqy = n.ay.nq; Z.nqz = n.az.nq; Z.NZI = t.NZI;
    Z.U = d_U;
    return t.nbz == 64 ? run_stage_z<64>(tmA, tmB, Z, num_sms, st)
         : t.nbz == 32 ? run_stage_z<32>(tmA, tmB, Z, num_sms, st) : run_stage_z<16>(tmA, tmB, Z, num_sms, st);
}

}  // namespace scatman
