// tensor_kernel.cu -- steps a4 + a5 + a6: the per-slice contraction on tcgen05 tensor cores with the fused
// slice-phase / accumulate epilogue (north_star (3), (4), (5); Eq. 2/9; Blocks 6-8,
// PAPER.md:154-160).
//
// Per work item a CTA owns 128 pixels (UMMA M) and one y-group (<= 128 y).  For every slice j and x-tile
// (128 x = UMMA N) it forms, in TMEM (FP32),
//     G_re[p,x] = sum_y  My_re[p,y] Rre_j[y,x] - My_im[p,y] Rim_j[y,x]
//     G_im[p,x] = sum_y  My_re[p,y] Rim_j[y,x] + My_im[p,y] Rre_j[y,x]
// where every FP32 factor is split into FP16 hi + lo and the product is AhBh + AlBh + AhBl (FP16x3;
// the minus sign is the instruction descriptor's negate-A bit).  The epilogue warps then read the
// accumulators (tcgen05.ld) and reduce them over x against e^{i qx x} = anchor[x/16] * fine[x%16],
// multiply by e^{i qz z_j} and accumulate over slices in FP32 registers (the fused epilogue).
//
// Roles: warp 0 lane 0 = TMA producer, warp 1 lane 0 = MMA issuer, warp 2 = TMEM allocator,
// warps 4-7 = epilogue (TMEM lane group = warp % 4).  Pipelines: A-resident (a_full/a_empty),
// B ring of kStagesB 16-KB slots (b_full/b_empty), two TMEM accumulator buffers (t_full/t_empty).
#include <cuda.h>

#include "internal.h"
#include "ptx_sm100.h"

namespace scatman {

constexpr int kSlotBytes = kTileP * kBlockY * 2;            // 16384: 128 rows x 128 bytes (one A K-block; one B tile)
constexpr int kSmemA = 4 * kGroupYB * kSlotBytes;           // 131072: resident A planes of one pixel tile
constexpr int kSmemB = 6 * kSlotBytes;                      // 98304: B ring (6 slots of 16 KB, or 12 of 8 KB per CTA of a pair)
constexpr int kSmemBar = 512;
constexpr int kSmemTotal = 1024 + kSmemA + kSmemB + kSmemBar;  // + alignment slack
constexpr int kThreads = 256;
constexpr uint32_t kTmemCols = 512;
constexpr int kMaxStagesB = 12;

size_t tensor_smem_bytes() { return kSmemTotal; }

#ifdef SCATMAN_TIMING
// debug-only cycle accounting (built by _work scripts with -DSCATMAN_TIMING; never in the product build)
__device__ long long g_timing[148 * 8];
#define TIMING_DECL(name) long long name = 0
#define TIMED_WAIT(acc, stmt) do { long long _t0 = clock64(); stmt; acc += clock64() - _t0; } while (0)
#else
#define TIMING_DECL(name)
#define TIMED_WAIT(acc, stmt) stmt
#endif

struct TensorParams {
    int nz, nxt, nyb, ngroups, ntiles, batch, nchunks, bpc, nzs, nxa;
    int64_t npix_pad;
    const float2 *anchor, *fine, *mz;
    const unsigned long long *mask;   // [batch][nz][nxt][ngroups]: bit 8*yi + xi = 16-y x 16-x block of rho~ is non-zero
    float2 *partial;
};

struct Item {
    int c, s, g, tp;
};
// item -> (batch chunk, z split, y group, tile pair); tile pair fastest so concurrent CTAs stream the same B
__device__ __forceinline__ Item decode_item(int item, const TensorParams &P, int ntp) {
    Item it;
    it.tp = item % ntp;
    item /= ntp;
    it.g = item % P.ngroups;
    item /= P.ngroups;
    it.s = item % P.nzs;
    it.c = item / P.nzs;
    return it;
}

// Units (batch item b, slice j, x tile xt) of a work item in issue order, with the occupancy word of each.
// Every role walks the same sequence and skips what the mask says is empty, so their pipelines stay in step.
struct Walk {
    int b, j, xt, b1, z0, z1, nxt;
    __device__ __forceinline__ bool valid() const { return b < b1; }
    __device__ __forceinline__ void next() {
        if (++xt == nxt) {
            xt = 0;
            if (++j == z1) { j = z0; ++b; }
        }
    }
};
__device__ __forceinline__ Walk walk_begin(const Item &it, const TensorParams &P) {
    Walk w;
    w.b = it.c * P.bpc;
    w.b1 = min(P.batch, w.b + P.bpc);
    w.z0 = (int)(((long long)P.nz * it.s) / P.nzs);
    w.z1 = (int)(((long long)P.nz * (it.s + 1)) / P.nzs);
    w.j = w.z0;
    w.xt = 0;
    w.nxt = P.nxt;
    return w;
}
__device__ __forceinline__ unsigned long long walk_mask(const Walk &w, const TensorParams &P, int g) {
    return w.valid() ? __ldg(P.mask + (((size_t)w.b * P.nz + w.j) * P.nxt + w.xt) * P.ngroups + g) : 0ull;
}

// NCTA = 1: one CTA per work item (cta_group::1, UMMA 128 x 128).
// NCTA = 2: a CTA pair per work item (cta_group::2, UMMA 256 x 128): each CTA owns its own 128-pixel tile (A resident in
//           its smem, D in its TMEM, its own epilogue) and HALF of every B tile (64 of the 128 x rows), so the B bytes
//           fetched and read from shared memory per CTA halve and the ring is twice as deep.  The leader (rank 0)
//           issues every MMA; full barriers live in the leader, empty barriers are signalled in both CTAs.
template <int NCTA>
__global__ void __launch_bounds__(kThreads, 1)
msft_contract_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                     const TensorParams P) {
    constexpr int kStagesB = 6 * NCTA;
    constexpr int kSlotB = kSlotBytes / NCTA;     // bytes of a B slot in one CTA
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sA = smem;
    uint8_t *sB = smem + kSmemA;
    uint64_t *bars = (uint64_t *)(smem + kSmemA + kSmemB);
    uint64_t *a_full = bars + 0, *a_empty = bars + 1;
    uint64_t *b_full = bars + 2, *b_empty = bars + 2 + kMaxStagesB;
    uint64_t *t_full = bars + 2 + 2 * kMaxStagesB, *t_empty = t_full + 2;
    uint32_t *tmem_ptr = (uint32_t *)(t_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = NCTA == 2 ? ptx::cluster_ctarank() : 0u;
    const int cluster_id = blockIdx.x / NCTA, nclusters = gridDim.x / NCTA;
    const int ntp = P.ntiles / NCTA;
    const int nitems = P.nchunks * P.nzs * P.ngroups * ntp;
    const bool leader = rank == 0;

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(a_full, 1);
        ptx::mbar_init(a_empty, 1);
        for (int i = 0; i < kStagesB; ++i) {
            ptx::mbar_init(b_full + i, 1);
            ptx::mbar_init(b_empty + i, 1);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(t_full + i, 1);
            ptx::mbar_init(t_empty + i, 4 * NCTA);
        }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) {
        if (NCTA == 2) ptx::tmem_alloc_2sm(tmem_ptr, kTmemCols);
        else ptx::tmem_alloc(tmem_ptr, kTmemCols);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (NCTA == 2) ptx::cluster_sync_all();   // peer barriers are initialised before anyone signals them
    ptx::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);  // provably warp-uniform

    if (warp == 0) {
        // ===================================================================== TMA producer (both CTAs of a pair)
        // The whole warp walks the loop (warp-uniform control flow); one elected lane issues.
        int slot = 0;
        uint32_t phase = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            const Item it = decode_item(item, P, ntp);
            const int tile = it.tp * NCTA + (int)rank;
            const int nybg = min(kGroupYB, P.nyb - it.g * kGroupYB);
            ptx::mbar_wait(a_empty, (uint32_t)((it_local & 1) ^ 1));
            if (ptx::elect_one()) {
                if (leader) ptx::mbar_arrive_expect_tx(a_full, (uint32_t)(NCTA * 4 * nybg * kSlotBytes));
                for (int pl = 0; pl < 4; ++pl)
                    for (int yb = 0; yb < nybg; ++yb) {
                        void *dst = sA + (pl * kGroupYB + yb) * kSlotBytes;
                        const int cy = (it.g * kGroupYB + yb) * kBlockY;
                        if (NCTA == 2) ptx::tma_load_3d_2sm(dst, &tmA, a_full, cy, tile * kTileP, pl);
                        else ptx::tma_load_3d(dst, &tmA, a_full, cy, tile * kTileP, pl);
                    }
            }
            __syncwarp();
            Walk w = walk_begin(it, P);
            unsigned long long m = walk_mask(w, P, it.g);
            while (w.valid()) {
                Walk wn = w;
                wn.next();
                const unsigned long long mn = walk_mask(wn, P, it.g);   // in flight while this unit is issued
                for (int yb = 0; yb < nybg; ++yb) {
                    if ((uint32_t)(m >> (32 * yb)) == 0u) continue;     // this 64-y block of the slice tile is empty
                    for (int pl = 0; pl < 4; ++pl) {
                        ptx::mbar_wait(b_empty + slot, phase ^ 1);
                        if (ptx::elect_one()) {
                            if (leader) ptx::mbar_arrive_expect_tx(b_full + slot, kSlotBytes);
                            void *dst = sB + slot * kSlotB;
                            const int cy = (it.g * kGroupYB + yb) * kBlockY;
                            const int cx = w.xt * kTileX + (int)rank * (kTileX / NCTA);
                            const int cp = (w.b * P.nz + w.j) * 4 + pl;
                            if (NCTA == 2) ptx::tma_load_3d_2sm(dst, &tmB, b_full + slot, cy, cx, cp);
                            else ptx::tma_load_3d(dst, &tmB, b_full + slot, cy, cx, cp);
                        }
                        __syncwarp();
                        if (++slot == kStagesB) { slot = 0; phase ^= 1; }
                    }
                }
                w = wn;
                m = mn;
            }
        }
    } else if (warp == 1) {
      if (leader) {
        // ===================================================================== MMA issuer (leader CTA only)
        // Warp-uniform loop; descriptors are uniform-register arithmetic; one elected lane issues the
        // tcgen05.mma / tcgen05.commit instructions.
        constexpr uint32_t idesc_pos = ptx::umma_idesc_f16(kTileP * NCTA, kTileX, false);
        constexpr uint32_t idesc_neg = ptx::umma_idesc_f16(kTileP * NCTA, kTileX, true);
        const uint64_t descA0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sA));
        const uint64_t descB0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sB));
        constexpr uint64_t kSlotDescA = kSlotBytes >> 4;
        constexpr uint64_t kSlotDescB = kSlotB >> 4;
        auto mma = [](uint32_t d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
            if (NCTA == 2) ptx::umma_f16_2sm(d, a, b, idesc, acc);
            else ptx::umma_f16(d, a, b, idesc, acc);
        };
        auto commit = [](uint64_t *bar) {
            if (NCTA == 2) ptx::umma_commit_2sm(bar, (uint16_t)0x3);
            else ptx::umma_commit(bar);
        };
        int slot = 0;
        uint32_t phase = 0;
        uint32_t u = 0;
        int it_local = 0;
        TIMING_DECL(w_tempty); TIMING_DECL(w_bfull); TIMING_DECL(w_afull);
#ifdef SCATMAN_TIMING
        const long long t_begin = clock64();
#endif
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            const Item it = decode_item(item, P, ntp);
            const int nybg = min(kGroupYB, P.nyb - it.g * kGroupYB);
            TIMED_WAIT(w_afull, ptx::mbar_wait(a_full, (uint32_t)(it_local & 1)));
            ptx::tc_fence_after();
            Walk w = walk_begin(it, P);
            unsigned long long m = walk_mask(w, P, it.g);
            while (w.valid()) {
                Walk wn = w;
                wn.next();
                const unsigned long long mn = walk_mask(wn, P, it.g);
                if (m != 0ull) {   // an all-zero unit adds nothing: no MMA, no accumulator hand-over
                    const uint32_t buf = u & 1;
                    TIMED_WAIT(w_tempty, ptx::mbar_wait(t_empty + buf, ((u >> 1) & 1) ^ 1));
                    ptx::tc_fence_after();
                    const uint32_t d_re = tmem_base + buf * 256, d_im = d_re + 128;
                    uint32_t started = 0u;   // 0 until the first k-step of this unit has initialised D_re and D_im
                    for (int yb = 0; yb < nybg; ++yb) {
                        const uint32_t occ = (uint32_t)(m >> (32 * yb));   // byte k = x-occupancy of 16-y step k
                        if (occ == 0u) continue;
                        // A-plane descriptors of this y-block: 0 Re_hi, 1 Re_lo, 2 Im_hi, 3 Im_lo
                        const uint64_t a_reh = descA0 + (uint64_t)(0 * kGroupYB + yb) * kSlotDescA;
                        const uint64_t a_rel = descA0 + (uint64_t)(1 * kGroupYB + yb) * kSlotDescA;
                        const uint64_t a_imh = descA0 + (uint64_t)(2 * kGroupYB + yb) * kSlotDescA;
                        const uint64_t a_iml = descA0 + (uint64_t)(3 * kGroupYB + yb) * kSlotDescA;
                        // ---- B = Re_hi
                        TIMED_WAIT(w_bfull, ptx::mbar_wait(b_full + slot, phase));
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            const uint64_t bd = descB0 + (uint64_t)slot * kSlotDescB;
                            uint32_t acc0 = started;
#pragma unroll
                            for (int k = 0; k < kBlockY / 16; ++k) {
                                if (((occ >> (8 * k)) & 0xffu) == 0u) continue;   // empty 16-y step
                                const uint64_t ko = (uint64_t)(k * 2);  // 16 fp16 = 32 bytes = 2 descriptor units
                                mma(d_re, a_reh + ko, bd + ko, idesc_pos, acc0);
                                mma(d_re, a_rel + ko, bd + ko, idesc_pos, 1u);
                                mma(d_im, a_imh + ko, bd + ko, idesc_pos, acc0);
                                mma(d_im, a_iml + ko, bd + ko, idesc_pos, 1u);
                                acc0 = 1u;
                            }
                            commit(b_empty + slot);
                        }
                        __syncwarp();
                        started = 1u;
                        if (++slot == kStagesB) { slot = 0; phase ^= 1; }
                        // ---- B = Re_lo
                        TIMED_WAIT(w_bfull, ptx::mbar_wait(b_full + slot, phase));
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            const uint64_t bd = descB0 + (uint64_t)slot * kSlotDescB;
#pragma unroll
                            for (int k = 0; k < kBlockY / 16; ++k) {
                                if (((occ >> (8 * k)) & 0xffu) == 0u) continue;
                                const uint64_t ko = (uint64_t)(k * 2);
                                mma(d_re, a_reh + ko, bd + ko, idesc_pos, 1u);
                                mma(d_im, a_imh + ko, bd + ko, idesc_pos, 1u);
                            }
                            commit(b_empty + slot);
                        }
                        __syncwarp();
                        if (++slot == kStagesB) { slot = 0; phase ^= 1; }
                        // ---- B = Im_hi
                        TIMED_WAIT(w_bfull, ptx::mbar_wait(b_full + slot, phase));
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            const uint64_t bd = descB0 + (uint64_t)slot * kSlotDescB;
#pragma unroll
                            for (int k = 0; k < kBlockY / 16; ++k) {
                                if (((occ >> (8 * k)) & 0xffu) == 0u) continue;
                                const uint64_t ko = (uint64_t)(k * 2);
                                mma(d_re, a_imh + ko, bd + ko, idesc_neg, 1u);
                                mma(d_re, a_iml + ko, bd + ko, idesc_neg, 1u);
                                mma(d_im, a_reh + ko, bd + ko, idesc_pos, 1u);
                                mma(d_im, a_rel + ko, bd + ko, idesc_pos, 1u);
                            }
                            commit(b_empty + slot);
                        }
                        __syncwarp();
                        if (++slot == kStagesB) { slot = 0; phase ^= 1; }
                        // ---- B = Im_lo
                        TIMED_WAIT(w_bfull, ptx::mbar_wait(b_full + slot, phase));
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            const uint64_t bd = descB0 + (uint64_t)slot * kSlotDescB;
#pragma unroll
                            for (int k = 0; k < kBlockY / 16; ++k) {
                                if (((occ >> (8 * k)) & 0xffu) == 0u) continue;
                                const uint64_t ko = (uint64_t)(k * 2);
                                mma(d_re, a_imh + ko, bd + ko, idesc_neg, 1u);
                                mma(d_im, a_reh + ko, bd + ko, idesc_pos, 1u);
                            }
                            commit(b_empty + slot);
                        }
                        __syncwarp();
                        if (++slot == kStagesB) { slot = 0; phase ^= 1; }
                    }
                    if (ptx::elect_one()) commit(t_full + buf);
                    __syncwarp();
                    ++u;
                }
                w = wn;
                m = mn;
            }
            if (ptx::elect_one()) commit(a_empty);
            __syncwarp();
        }
#ifdef SCATMAN_TIMING
        if (lane == 0) {
            g_timing[blockIdx.x * 8 + 0] = clock64() - t_begin;
            g_timing[blockIdx.x * 8 + 1] = w_tempty;
            g_timing[blockIdx.x * 8 + 2] = w_bfull;
            g_timing[blockIdx.x * 8 + 3] = w_afull;
        }
#endif
      }
    } else if (warp >= 4) {
        // ========================================================================= epilogue
        const int ew = warp & 3;
        const int el = ew * 32 + lane;  // pixel within the tile = TMEM lane
        const uint32_t lane_base = tmem_base + ((uint32_t)(ew * 32) << 16);
        uint32_t u = 0;
        TIMING_DECL(w_tfull);
#ifdef SCATMAN_TIMING
        const long long e_begin = clock64();
#endif
        for (int item = cluster_id; item < nitems; item += nclusters) {
            const Item it = decode_item(item, P, ntp);
            const int tile = it.tp * NCTA + (int)rank;
            const int b0 = it.c * P.bpc, b1 = min(P.batch, b0 + P.bpc);
            const int z0 = (int)(((long long)P.nz * it.s) / P.nzs), z1 = (int)(((long long)P.nz * (it.s + 1)) / P.nzs);
            float2 fine[kFine];
#pragma unroll
            for (int i = 0; i < kFine; ++i) fine[i] = __ldg(P.fine + ((size_t)tile * kFine + i) * kTileP + el);
            const float2 *anchor_t = P.anchor + (size_t)tile * P.nxa * kTileP + el;
            const float2 *mz_t = P.mz + (size_t)tile * P.nz * kTileP + el;
            Walk w = walk_begin(it, P);
            unsigned long long m_next = walk_mask(w, P, it.g);
            for (int b = b0; b < b1; ++b) {
                float acc_re = 0.f, acc_im = 0.f;
                for (int j = z0; j < z1; ++j) {
                    const float2 mz = __ldg(mz_t + (size_t)j * kTileP);
                    float f_re = 0.f, f_im = 0.f;
                    for (int xt = 0; xt < P.nxt; ++xt) {
                        const unsigned long long m = m_next;
                        w.next();
                        m_next = walk_mask(w, P, it.g);
                        if (m == 0ull) continue;   // empty unit: G = 0, nothing was issued for it
                        const uint32_t buf = u & 1;
                        float2 anc[kTileX / kFine];
#pragma unroll
                        for (int a = 0; a < kTileX / kFine; ++a)
                            anc[a] = __ldg(anchor_t + (size_t)(xt * (kTileX / kFine) + a) * kTileP);
                        TIMED_WAIT(w_tfull, ptx::mbar_wait(t_full + buf, (u >> 1) & 1));
                        ptx::tc_fence_after();
                        const uint32_t t_re = lane_base + buf * 256, t_im = t_re + 128;
                        // software-pipelined: the loads of block a+1 are in flight while block a is reduced; the
                        // accumulator buffer is handed back to the MMA warp as soon as its last column has landed
                        uint32_t gre[2][16], gim[2][16];
                        ptx::tmem_ld16(t_re, gre[0]);
                        ptx::tmem_ld16(t_im, gim[0]);
                        ptx::tmem_ld_wait_dep(gre[0]);
                        ptx::tmem_ld_wait_dep(gim[0]);
#pragma unroll
                        for (int a = 0; a < kTileX / kFine; ++a) {
                            const int cur = a & 1, nxt = cur ^ 1;
                            if (a + 1 < kTileX / kFine) {
                                ptx::tmem_ld16(t_re + (a + 1) * kFine, gre[nxt]);
                                ptx::tmem_ld16(t_im + (a + 1) * kFine, gim[nxt]);
                            } else {
                                ptx::tc_fence_before();
                                __syncwarp();
                                if (lane == 0) {
                                    if (NCTA == 2) ptx::mbar_arrive_cluster(t_empty + buf, 0);   // the leader's barrier
                                    else ptx::mbar_arrive(t_empty + buf);
                                }
                            }
                            float sra = 0.f, srb = 0.f, sia = 0.f, sib = 0.f;   // four independent FMA chains
#pragma unroll
                            for (int i = 0; i < kFine; ++i) {
                                const float gr = __uint_as_float(gre[cur][i]), gi = __uint_as_float(gim[cur][i]);
                                sra = fmaf(fine[i].x, gr, sra);
                                srb = fmaf(fine[i].y, gi, srb);
                                sia = fmaf(fine[i].x, gi, sia);
                                sib = fmaf(fine[i].y, gr, sib);
                            }
                            const float s_re = sra - srb, s_im = sia + sib;
                            f_re = fmaf(anc[a].x, s_re, f_re);
                            f_re = fmaf(-anc[a].y, s_im, f_re);
                            f_im = fmaf(anc[a].x, s_im, f_im);
                            f_im = fmaf(anc[a].y, s_re, f_im);
                            if (a + 1 < kTileX / kFine) {
                                ptx::tmem_ld_wait_dep(gre[nxt]);
                                ptx::tmem_ld_wait_dep(gim[nxt]);
                            }
                        }
                        ++u;
                    }
                    acc_re = fmaf(mz.x, f_re, acc_re);
                    acc_re = fmaf(-mz.y, f_im, acc_re);
                    acc_im = fmaf(mz.x, f_im, acc_im);
                    acc_im = fmaf(mz.y, f_re, acc_im);
                }
                P.partial[((size_t)b * (P.ngroups * P.nzs) + (it.g * P.nzs + it.s)) * P.npix_pad +
                          (size_t)tile * kTileP + el] = make_float2(acc_re, acc_im);
            }
        }
#ifdef SCATMAN_TIMING
        if (warp == 4 && lane == 0) {
            g_timing[blockIdx.x * 8 + 4] = clock64() - e_begin;
            g_timing[blockIdx.x * 8 + 5] = w_tfull;
            g_timing[blockIdx.x * 8 + 6] = u;
        }
#endif
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (NCTA == 2) ptx::cluster_sync_all();   // nobody leaves while the peer may still signal its barriers
    if (warp == 2) {
        ptx::tc_fence_after();
        if (NCTA == 2) ptx::tmem_dealloc_2sm(tmem_base, kTmemCols);
        else ptx::tmem_dealloc(tmem_base, kTmemCols);
    }
}

// ------------------------------------------------------------------------------------------------ host
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

static bool encode_planes(CUtensorMap *tm, const void *base, uint64_t inner, uint64_t rows, uint64_t planes,
                          uint32_t box_rows) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {inner, rows, planes};
    cuuint64_t strides[2] = {inner * 2, inner * rows * 2};
    cuuint32_t box[3] = {(cuuint32_t)kBlockY, box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void *>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int NCTA>
static cudaError_t launch_variant(const CUtensorMap &tmA, const CUtensorMap &tmB, const TensorParams &P, int num_sms,
                                  cudaStream_t st) {
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(msft_contract_kernel<NCTA>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             kSmemTotal);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int nitems = P.nchunks * P.nzs * P.ngroups * (P.ntiles / NCTA);
    const int max_clusters = num_sms / NCTA;
    const int nclusters = nitems < max_clusters ? nitems : max_clusters;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(nclusters * NCTA));
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemTotal;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = NCTA;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, msft_contract_kernel<NCTA>, tmA, tmB, P);
}

cudaError_t launch_tensor(const Plan &p, const TensorLaunch &t, cudaStream_t st, std::string *err) {
    const int ncta = p.t_ncta;
    CUtensorMap tmA, tmB;
    if (!encode_planes(&tmA, t.d_A, (uint64_t)p.ny_pad, (uint64_t)p.npix_pad, 4, kTileP) ||
        !encode_planes(&tmB, t.d_B, (uint64_t)p.ny_pad, (uint64_t)p.nx_pad, (uint64_t)p.batch * p.nz * 4,
                       kTileX / ncta)) {
        if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
        return cudaErrorUnknown;
    }
    TensorParams P;
    P.nz = p.nz; P.nxt = p.nxt; P.nyb = p.nyb; P.ngroups = p.ngroups; P.ntiles = p.ntiles; P.batch = p.batch;
    P.nzs = p.t_nzs;
    P.bpc = (p.batch + p.t_nchunks - 1) / p.t_nchunks;
    P.nchunks = (p.batch + P.bpc - 1) / P.bpc;
    P.nxa = p.nxa;
    P.npix_pad = p.npix_pad;
    P.anchor = t.d_anchor; P.fine = t.d_fine; P.mz = t.d_mz; P.partial = t.d_partial; P.mask = t.d_mask;
    return ncta == 2 ? launch_variant<2>(tmA, tmB, P, t.num_sms, st) : launch_variant<1>(tmA, tmB, P, t.num_sms, st);
}

#ifdef SCATMAN_TIMING
extern "C" int scatman_debug_timing(long long *h_out) {
    return (int)cudaMemcpyFromSymbol(h_out, g_timing, sizeof(long long) * 148 * 8);
}
#endif

}  // namespace scatman
