// tc_cgemm.cuh -- one tcgen05 pipeline for "streamed A x resident B" complex GEMMs in FP16x3 split precision.
//
//     C[row, col] = sum_k A[row, k] B[col, k]          (complex; every operand = four FP16 planes Re_hi, Re_lo, Im_hi, Im_lo, K-major)
//
// A CTA PAIR (tcgen05 cta_group::2, UMMA 256 x 2NB x 16) runs a work item = (column tile of 2 NB columns, a range of units).
// A unit = one 128-row tile of A per CTA (the pair takes two consecutive units; an odd last one is run twice and the peer's
// copy discarded).  Each CTA streams its OWN row tile (two planes per stage: Re hi + lo, then Im hi + lo, 32 KB stages through a
// ring of three) against the same 2 NB columns, of whose B tile each CTA keeps NB rows resident for the whole item
// (4 planes x nk x NB x 128 bytes <= 128 KB: NB = 64 / 32 / 16 for K <= 256 / 512 / 1024).  The complex product is twelve real
// MMAs per k-step: AhBh + AlBh + AhBl for each of the four real products; the minus sign of Re = ArBr - AiBi is the
// instruction descriptor's negate-A bit.  FP32 accumulators D_re, D_im live in TMEM, two buffers, so the epilogue of unit u
// overlaps the MMAs of unit u + 1.
//
// Roles (384 threads): warp 0 TMA producer (both CTAs), warps 1 and 3 MMA issuers (leader CTA; k-step ks of a stage belongs
// to issuer ks % 2 -- at N <= 128 a tcgen05.mma is bound by its shared-memory operand fetch and one issuing thread exposes
// what it spends between stages; both issuers wait for every stage and both release it, so no parity can alias), warp 2 TMEM
// allocator, warps 4-11 epilogue (TMEM lane group = warp % 4, column half = (warp - 4) / 4).
//
// What the pipeline is used FOR is a policy class:
//     struct Policy {
//         static constexpr int NB;                       // columns of B resident per CTA
//         struct Params;                                 // kernel argument (plain data)
//         struct Item;                                   // decoded work item
//         struct Units;                                  // iterator over the units of an item, warp-cooperative
//         static int nitems(const Params &);
//         static Item item(const Params &, int index);
//         static int b_row0(const Params &, const Item &);                       // first B row (column of C) of the item's column tile
//         Units: void begin(const Params &, const Item &, int lane);
//                bool next(int &u0, int &u1, bool &dup, uint32_t &kmask);        // units of leader / peer, live 64-k blocks; false at the end
//         static constexpr bool kUnrollEpilogue;         // column loop of the epilogue fully unrolled (register-array accumulators)
//         static constexpr int kEpilogueRegs;            // 0, or registers per epilogue thread after setmaxnreg (the other warps drop to 48)
//         static void a_coords(const Params &, const Item &, int unit, int kb, int (&c)[3]);   // TMA coordinates {k, row, outer} of a 64-k block
//         struct Epilogue { begin(P, item, ...), unit(...), end(...) };          // see the users
//     };
// Users: sep_tensor_kernels.cu (stage X and the transposed stage YZ of the separable route), nufft_tensor_kernels.cu (stages Y
// and Z of the NUFFT route).
#pragma once
#include <cuda.h>

#include "internal.h"
#include "ptx_sm100.h"

namespace scatman {
namespace tcg {

constexpr int kM = 128;                 // rows of a unit's A tile = TMEM lanes
constexpr int kKB = 64;                 // K per block (one 128-byte swizzle row of FP16)
constexpr int kSlotA = kM * kKB * 2;    // 16384: one plane, one K block of an A tile
constexpr int kStage = 2 * kSlotA;      // a stage = two planes
constexpr int kStages = 3;
constexpr int kSmemB = 131072;          // resident B planes of this CTA
constexpr int kThreads = 384;
constexpr uint32_t kTmemCols = 512;
constexpr int kNBuf = 2;                // accumulator buffers (D_re, D_im of up to 128 columns each)
constexpr int kSmemTotal = 1024 + kSmemB + kStages * kStage + 256;

// What the epilogue warps know about themselves.
struct EpiThread {
    int lane_row;     // row of the unit's tile this thread owns (TMEM lane), 0..127
    int col0;         // first of the NB accumulator columns this thread reads
    uint32_t rank;    // CTA rank in the pair
};

// The register file is re-split when the epilogue needs more than the 168 registers a 384-thread CTA gives each thread: the
// producer / issuer warpgroup drops to 48, the two epilogue warpgroups rise to N: 128 x 48 + 256 x N must not exceed the
// 384 x 168 the CTA owns (an increase can only take what the CTA's own warps released, or it waits forever) -> N <= 224.
template <int N> __device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ void setmaxnreg_dec_48() { asm volatile("setmaxnreg.dec.sync.aligned.u32 48;"); }

template <class Policy>
__global__ void __launch_bounds__(kThreads, 1)
cgemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const typename Policy::Params P) {
    constexpr int NB = Policy::NB;
    constexpr int kN = 2 * NB;
    constexpr int kBlkB = NB * kKB * 2;       // bytes of one plane, one K block of this CTA's B rows
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sB = smem;
    uint8_t *sA = smem + kSmemB;
    uint64_t *bars = (uint64_t *)(smem + kSmemB + kStages * kStage);
    uint64_t *b_full = bars + 0, *b_empty = bars + 1;
    uint64_t *a_full = bars + 2, *a_empty = a_full + kStages;
    uint64_t *t_full = a_empty + kStages, *t_empty = t_full + kNBuf, *first_done = t_empty + kNBuf;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + kNBuf);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    const bool leader = rank == 0;
    const int cluster_id = blockIdx.x / 2, nclusters = gridDim.x / 2;
    const int nitems = Policy::nitems(P);
    const int nk = P.nk;

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(b_full, 1);
        ptx::mbar_init(b_empty, 2);            // both MMA issuers
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(a_full + i, 1);
            ptx::mbar_init(a_empty + i, 2);
        }
        for (int i = 0; i < kNBuf; ++i) {
            ptx::mbar_init(t_full + i, 2);
            ptx::mbar_init(t_empty + i, 16);   // 8 epilogue warps in each CTA
            ptx::mbar_init(first_done + i, 1);
        }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) ptx::tmem_alloc_2sm(tmem_ptr, kTmemCols);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync_all();                   // peer barriers are initialised before anyone signals them
    ptx::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);

    // (each role's code must be DOMINATED by its setmaxnreg: ptxas allots the raised register count only to such code)
    if (warp < 4) {
      if constexpr (Policy::kEpilogueRegs != 0) setmaxnreg_dec_48();
      if (warp == 0) {
        // ===================================================================== TMA producer (both CTAs)
        int slot = 0;
        uint32_t phase = 0;
        int it_local = 0;
        for (int index = cluster_id; index < nitems; index += nclusters, ++it_local) {
            const typename Policy::Item it = Policy::item(P, index);
            ptx::mbar_wait(b_empty, (uint32_t)((it_local & 1) ^ 1));
            if (ptx::elect_one()) {
                if (leader) ptx::mbar_arrive_expect_tx(b_full, (uint32_t)(2 * 4 * nk * kBlkB));
                const int row0 = Policy::b_row0(P, it) + (int)rank * NB;
                for (int pl = 0; pl < 4; ++pl)
                    for (int kb = 0; kb < nk; ++kb)
                        ptx::tma_load_3d_2sm(sB + (pl * nk + kb) * kBlkB, &tmB, b_full, kb * kKB, row0, pl);
            }
            __syncwarp();
            typename Policy::Units un;
            un.begin(P, it, lane);
            int u0, u1;
            bool dup;
            uint32_t kmask;
            while (un.next(u0, u1, dup, kmask)) {
                const int u = leader ? u0 : u1;
                for (int kb = 0; kb < nk; ++kb) {
                    if (((kmask >> kb) & 1u) == 0u) continue;   // a 64-k block that holds nothing: never loaded, never multiplied
                    int c[3];
                    Policy::a_coords(P, it, u, kb, c);
                    for (int ph = 0; ph < 2; ++ph) {   // Re planes, Im planes
                        ptx::mbar_wait(a_empty + slot, phase ^ 1);
                        if (ptx::elect_one()) {
                            if (leader) ptx::mbar_arrive_expect_tx(a_full + slot, (uint32_t)(2 * kStage));
                            ptx::tma_load_4d_2sm(sA + slot * kStage, &tmA, a_full + slot, c[0], c[1], c[2], 2 * ph);
                            ptx::tma_load_4d_2sm(sA + slot * kStage + kSlotA, &tmA, a_full + slot, c[0], c[1], c[2], 2 * ph + 1);
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
        const uint64_t descA0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sA));
        const uint64_t descB0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sB));
        constexpr uint64_t kA = kSlotA >> 4, kSt = kStage >> 4, kB = kBlkB >> 4;
        const int iw = warp >> 1;
        int slot = 0;
        uint32_t phase = 0, u = 0;
        int it_local = 0;
        for (int index = cluster_id; index < nitems; index += nclusters, ++it_local) {
            const typename Policy::Item it = Policy::item(P, index);
            ptx::mbar_wait(b_full, (uint32_t)(it_local & 1));
            ptx::tc_fence_after();
            const uint64_t kBpl = (uint64_t)nk * kB;   // descriptor distance between B planes
            typename Policy::Units un;
            un.begin(P, it, lane);
            int u0, u1;
            bool dup;
            uint32_t kmask;
            while (un.next(u0, u1, dup, kmask)) {
                const uint32_t buf = u % kNBuf, upar = (u / kNBuf) & 1;
                ptx::mbar_wait(t_empty + buf, upar ^ 1);
                ptx::tc_fence_after();
                const uint32_t d_re = tmem_base + buf * 256, d_im = d_re + 128;
                bool first = true;                             // the unit's first live k block
                for (int kb = 0; kb < nk; ++kb) {
                    if (((kmask >> kb) & 1u) == 0u) continue;
                    for (int ph = 0; ph < 2; ++ph) {
                        if (iw == 1 && first && ph == 0) {     // D must have been initialised by issuer 0
                            ptx::mbar_wait(first_done + buf, upar);
                            ptx::tc_fence_after();
                        }
                        ptx::mbar_wait(a_full + slot, phase);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
#pragma unroll
                            for (int kk = 0; kk < 2; ++kk) {
                                const int ks = 2 * kk + iw;
                                const uint64_t a_hi = descA0 + (uint64_t)slot * kSt + (uint64_t)(ks * 2), a_lo = a_hi + kA;
                                const uint64_t b_reh = descB0 + (uint64_t)kb * kB + (uint64_t)(ks * 2);
                                const uint64_t b_rel = b_reh + kBpl, b_imh = b_rel + kBpl, b_iml = b_imh + kBpl;
                                const uint32_t acc0 = (first && ph == 0 && ks == 0) ? 0u : 1u;
                                // (Ar + i Ai)(Br + i Bi) with the A planes of this stage: AhBh + AhBl + AlBh
                                if (ph == 0) {   // A Re hi, Re lo
                                    ptx::umma_f16_2sm(d_re, a_hi, b_reh, idesc_pos, acc0);
                                    ptx::umma_f16_2sm(d_im, a_hi, b_imh, idesc_pos, acc0);
                                    ptx::umma_f16_2sm(d_re, a_hi, b_rel, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, b_iml, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_lo, b_reh, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_im, a_lo, b_imh, idesc_pos, 1u);
                                } else {         // A Im hi, Im lo
                                    ptx::umma_f16_2sm(d_re, a_hi, b_imh, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, b_reh, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_hi, b_iml, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_hi, b_rel, idesc_pos, 1u);
                                    ptx::umma_f16_2sm(d_re, a_lo, b_imh, idesc_neg, 1u);
                                    ptx::umma_f16_2sm(d_im, a_lo, b_reh, idesc_pos, 1u);
                                }
                                if (iw == 0 && kk == 0 && first && ph == 0) ptx::umma_commit_2sm(first_done + buf, (uint16_t)0x1);
                            }
                            ptx::umma_commit_2sm(a_empty + slot, (uint16_t)0x3);
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
            if (ptx::elect_one()) ptx::umma_commit_2sm(b_empty, (uint16_t)0x3);
            __syncwarp();
        }
      }
    } else {
        if constexpr (Policy::kEpilogueRegs != 0) setmaxnreg_inc<Policy::kEpilogueRegs != 0 ? Policy::kEpilogueRegs : 168>();
        // ===================================================================== epilogue: this CTA's 128 rows x 2 NB columns
        const int lg = warp & 3, ch = (warp - 4) >> 2;     // TMEM lane group; column half [ch NB, +NB)
        const uint32_t t_lane = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(ch * NB);
        EpiThread et;
        et.lane_row = lg * 32 + lane;
        et.col0 = ch * NB;
        et.rank = rank;
        uint32_t u = 0;
        for (int index = cluster_id; index < nitems; index += nclusters) {
            const typename Policy::Item it = Policy::item(P, index);
            typename Policy::Epilogue epi;
            epi.begin(P, it, et);
            typename Policy::Units un;
            un.begin(P, it, lane);
            int u0, u1;
            bool dup;
            uint32_t kmask;
            while (un.next(u0, u1, dup, kmask)) {
                const int unit = leader ? u0 : u1;
                const bool keep = leader || !dup;
                const uint32_t buf = u % kNBuf, upar = (u / kNBuf) & 1;
                epi.unit_begin(P, it, et, unit);
                ptx::mbar_wait(t_full + buf, upar);
                ptx::tc_fence_after();
                const uint32_t t_re = t_lane + buf * 256, t_im = t_re + 128;
#define SCATMAN_EPILOGUE_EIGHT_COLUMNS(c0)                                                                            \
    {                                                                                                                    \
        uint32_t gre[8], gim[8];                                                                                         \
        ptx::tmem_ld8(t_re + (c0), gre);                                                                                 \
        ptx::tmem_ld8(t_im + (c0), gim);                                                                                 \
        ptx::tmem_ld_wait();                                                                                             \
        if ((c0) + 8 >= NB) { /* every column of this warp has landed: hand the buffer back */                           \
            ptx::tc_fence_before();                                                                                      \
            __syncwarp();                                                                                                \
            if (lane == 0) ptx::mbar_arrive_cluster(t_empty + buf, 0); /* the leader's barrier */                        \
        }                                                                                                                \
        if (keep) epi.columns(P, it, et, unit, (c0), gre, gim);                                                          \
    }
                if constexpr (Policy::kUnrollEpilogue) {   // register-array accumulators: every column index must be static
#pragma unroll
                    for (int c0 = 0; c0 < NB; c0 += 8) SCATMAN_EPILOGUE_EIGHT_COLUMNS(c0)
                } else {
#pragma unroll 1
                    for (int c0 = 0; c0 < NB; c0 += 8) SCATMAN_EPILOGUE_EIGHT_COLUMNS(c0)
                }
#undef SCATMAN_EPILOGUE_EIGHT_COLUMNS
                ++u;
            }
            epi.end(P, it, et);
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync_all();                   // nobody leaves while the peer may still signal its barriers
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_2sm(tmem_base, kTmemCols);
    }
}

template <class Policy>
inline cudaError_t cgemm_init_device() {
    return cudaFuncSetAttribute(cgemm_kernel<Policy>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemTotal);
}

template <class Policy>
inline cudaError_t cgemm_launch(const CUtensorMap &tmA, const CUtensorMap &tmB, const typename Policy::Params &P, int nitems,
                                int num_sms, cudaStream_t st) {
    const int max_clusters = num_sms / 2;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(2 * (nitems < max_clusters ? nitems : max_clusters)));
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemTotal;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, cgemm_kernel<Policy>, tmA, tmB, P);
}

// Units numbered 0 .. n-1 of a range [begin, end), handed out in pairs (leader, peer).
struct RangeUnits {
    int cur, end;
    __device__ __forceinline__ void set(int b, int e) { cur = b; end = e; }
    __device__ __forceinline__ bool next(int &u0, int &u1, bool &dup, uint32_t &kmask) {
        kmask = 0xffffffffu;
        if (cur >= end) return false;
        u0 = cur;
        dup = cur + 1 >= end;
        u1 = dup ? cur : cur + 1;
        cur += 2;
        return true;
    }
};

__device__ __forceinline__ void split4h(float re, float im, __half (&h)[4]) {
    h[0] = __float2half_rn(re);
    h[1] = __float2half_rn(re - __half2float(h[0]));
    h[2] = __float2half_rn(im);
    h[3] = __float2half_rn(im - __half2float(h[2]));
}

}  // namespace tcg
}  // namespace scatman
