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
// Roles: warp 0 = TMA producer, warps 1 and 3 = MMA issuers (k-step n of a unit belongs to issuer n % 2), warp 2 = TMEM
// allocator, warps 4-7 = epilogue (TMEM lane group = warp % 4).  Pipelines: A-resident (a_full/a_empty), B ring of
// kStagesB slots (b_full[issuer]/b_empty), two TMEM accumulator buffers (t_full/t_empty), first_done orders issuer 1 behind the
// unit's first k-step.  Ordering between the two issuing threads (tcgen05.mma is ordered only within one thread): a
// unit's accumulator is initialised by issuer 0's first k-step and issuer 1 waits for its completion (first_done);
// after that both threads only ACCUMULATE into D, in whatever order their MMAs reach the tensor pipe -- results are
// reproducible to FP32 summation order, not bit for bit; both commit t_full (count 2), so the epilogue
// sees every MMA of both threads.  A B slot is filled for ONE issuer (the owner of its k-step) and signalled on that issuer's
// own full barrier, so each issuer sees every completion of the barriers it waits on and a parity can never alias.
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

struct TensorParams {
    int nz, nxt, nyb, ny16, ngroups, ntiles, batch, nchunks, bpc, nzs, nxa;
    int64_t npix_pad;
    const float2 *anchor, *fine;
    const unsigned long long *zturn;  // [tile][128]: frac(qz dz / 4 pi) of the pixel as a 64-bit fixed-point fraction of a turn
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

// The NON-EMPTY units (batch item b, slice j, x tile xt) of a work item in issue order, with the occupancy word of
// each.  Every role walks the same sequence, so their pipelines stay in step.  Warp-cooperative: each lane holds the
// occupancy word of one of 32 consecutive units (the next 32 are already in flight), a ballot finds the next
// non-empty one, a shuffle broadcasts it: one L2 round trip per 32 units instead of one per unit.
struct Units {
    int b0, z0, nzr, nxt, total, g, base, lane;
    unsigned long long cur, ahead;
    uint32_t live;
    const TensorParams *P;
    __device__ __forceinline__ void decode(int n, int &b, int &j, int &xt) const {
        xt = n % nxt;
        const int r = n / nxt;
        j = z0 + r % nzr;
        b = b0 + r / nzr;
    }
    __device__ __forceinline__ unsigned long long load(int n) const {
        if (n >= total) return 0ull;
        int b, j, xt;
        decode(n, b, j, xt);
        return __ldg(P->mask + (((size_t)b * P->nz + j) * P->nxt + xt) * P->ngroups + g);
    }
    __device__ __forceinline__ void begin(const Item &it, const TensorParams &Pr, int lane_) {
        P = &Pr;
        lane = lane_;
        g = it.g;
        b0 = it.c * Pr.bpc;
        const int b1 = min(Pr.batch, b0 + Pr.bpc);
        z0 = (int)(((long long)Pr.nz * it.s) / Pr.nzs);
        nzr = (int)(((long long)Pr.nz * (it.s + 1)) / Pr.nzs) - z0;
        nxt = Pr.nxt;
        total = (b1 - b0) * nzr * nxt;
        base = 0;
        cur = load(lane);
        ahead = load(32 + lane);
        live = __ballot_sync(0xffffffffu, cur != 0ull);
    }
    // occupancy word of the next non-empty unit only (the MMA issuer needs nothing else)
    __device__ __forceinline__ bool next_mask(unsigned long long &m) {
        while (live == 0u) {
            base += 32;
            if (base >= total) return false;
            cur = ahead;
            ahead = load(base + 32 + lane);
            live = __ballot_sync(0xffffffffu, cur != 0ull);
        }
        const int pos = __ffs((int)live) - 1;
        live &= live - 1;
        m = __shfl_sync(0xffffffffu, cur, pos);
        return true;
    }
    // next non-empty unit; false when the item is exhausted (warp-uniform result)
    __device__ __forceinline__ bool next(int &b, int &j, int &xt, unsigned long long &m) {
        while (live == 0u) {
            base += 32;
            if (base >= total) return false;
            cur = ahead;
            ahead = load(base + 32 + lane);
            live = __ballot_sync(0xffffffffu, cur != 0ull);
        }
        const int pos = __ffs((int)live) - 1;
        live &= live - 1;
        m = __shfl_sync(0xffffffffu, cur, pos);
        decode(base + pos, b, j, xt);
        return true;
    }
};

// x extent of a unit in 16-x blocks: [a, a + m) = bounding range of the non-empty blocks over the whole y group.
// CTA pairs run the unit's MMAs at N = 16 m (the B tile rows are stored so that a prefix of each CTA's half is a
// contiguous x range, see pack_b_kernel); a single CTA always runs the full tile.
template <int NCTA>
__device__ __forceinline__ void unit_range(unsigned long long m64, int &a, int &m) {
    if (NCTA == 1) { a = 0; m = kTileX / 16; return; }
    uint32_t v = (uint32_t)m64 | (uint32_t)(m64 >> 32);
    v |= v >> 16;
    v = (v | (v >> 8)) & 0xffu;
    a = __ffs((int)v) - 1;
    m = (32 - __clz((int)v)) - a;
}
struct TmapsB {
    CUtensorMap m[kTileX / 16];   // box heights 8, 16, ... rows per CTA of a pair (entry 7 = the full half / full tile)
};

// NCTA = 1: one CTA per work item (cta_group::1, UMMA 128 x 128).
// NCTA = 2: a CTA pair per work item (cta_group::2, UMMA 256 x 128): each CTA owns its own 128-pixel tile (A resident in
//           its smem, D in its TMEM, its own epilogue) and HALF of every B tile (64 of the 128 x rows), so the B bytes
//           fetched and read from shared memory per CTA halve and the ring is twice as deep.  The leader (rank 0)
//           issues every MMA; full barriers live in the leader, empty barriers are signalled in both CTAs.
template <int NCTA>
__global__ void __launch_bounds__(kThreads, 1)
msft_contract_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ TmapsB tmB,
                     const TensorParams P) {
    constexpr int kStagesB = 6 * NCTA;
    constexpr int kSlotB = kSlotBytes / NCTA;     // bytes of a B slot in one CTA
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *sA = smem;
    uint8_t *sB = smem + kSmemA;
    uint64_t *bars = (uint64_t *)(smem + kSmemA + kSmemB);
    uint64_t *a_full = bars + 0, *a_empty = bars + 1;
    // b_full[i][slot]: "slot filled" for a k-step owned by MMA issuer i.  Each issuer has its OWN full barriers: it waits on every
    // completion of each of them, in order, so a parity wait can never take an older pass for the current one (with one shared
    // barrier per slot an issuer saw only the passes of its own k-steps -- every other one where units have odd k-step counts --
    // and "pass R - 2 complete" is indistinguishable from "pass R complete" by parity).
    uint64_t *b_full = bars + 2, *b_empty = bars + 2 + 2 * kMaxStagesB;
    uint64_t *t_full = bars + 2 + 3 * kMaxStagesB, *t_empty = t_full + 2, *first_done = t_empty + 2;
    uint32_t *tmem_ptr = (uint32_t *)(first_done + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = NCTA == 2 ? ptx::cluster_ctarank() : 0u;
    const int cluster_id = blockIdx.x / NCTA, nclusters = gridDim.x / NCTA;
    const int ntp = P.ntiles / NCTA;
    const int nitems = P.nchunks * P.nzs * P.ngroups * ntp;
    const bool leader = rank == 0;

    if (warp == 0 && lane == 0) {
        ptx::tma_prefetch_desc(&tmA);
        for (int i = 0; i < kTileX / 16; ++i) ptx::tma_prefetch_desc(&tmB.m[i]);
    }
    if (warp == 1 && lane == 0) {
        ptx::mbar_init(a_full, 1);
        ptx::mbar_init(a_empty, 2);      // both MMA issuers
        for (int i = 0; i < kStagesB; ++i) {
            ptx::mbar_init(b_full + i, 1);
            ptx::mbar_init(b_full + kMaxStagesB + i, 1);
            ptx::mbar_init(b_empty + i, 1);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(t_full + i, 2);   // both MMA issuers
            ptx::mbar_init(first_done + i, 1);
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
                // the A tile of this cluster's next work item comes from HBM: start it towards L2 now
                if (item + nclusters < nitems) {
                    const Item nx = decode_item(item + nclusters, P, ntp);
                    const int ntile = nx.tp * NCTA + (int)rank;
                    const int nyn = min(kGroupYB, P.nyb - nx.g * kGroupYB);
                    for (int pl = 0; pl < 4; ++pl)
                        for (int yb = 0; yb < nyn; ++yb)
                            ptx::tma_prefetch_l2_3d(&tmA, (nx.g * kGroupYB + yb) * kBlockY, ntile * kTileP, pl);
                }
            }
            __syncwarp();
            Units un;
            un.begin(it, P, lane);
            int ub, uj, uxt;
            unsigned long long m;
            while (un.next(ub, uj, uxt, m)) {
                int xa, xm;
                unit_range<NCTA>(m, xa, xm);
                // one box = one 16-y step: {256-byte atom, 4 planes, xm x-groups of this CTA's half (16 for one CTA)}
                const CUtensorMap *tmb = &tmB.m[xm - 1];
                const uint32_t tx_bytes = NCTA == 2 ? (uint32_t)(2 * xm * 1024) : (uint32_t)kSlotBytes;
                int kidx = 0;                                                   // k-step index within the unit: its parity = the issuer that owns it
                for (int yi = 0; yi < 4 * nybg; ++yi) {
                    if (((uint32_t)(m >> (8 * yi)) & 0xffu) == 0u) continue;   // this 16-y step of the slice tile is empty
                    ptx::mbar_wait(b_empty + slot, phase ^ 1);
                    uint64_t *full = b_full + (kidx & 1) * kMaxStagesB + slot;
                    ++kidx;
                    if (ptx::elect_one()) {
                        if (leader) ptx::mbar_arrive_expect_tx(full, tx_bytes);
                        void *dst = sB + slot * kSlotB;
                        const int cg = uxt * 16 + (NCTA == 2 ? (int)rank * 8 + xa : 0);
                        const int cs = (ub * P.nz + uj) * P.ny16 + it.g * (kGroupYB * kBlockY / 16) + yi;
                        SCATMAN_ASSERT(xm >= 1 && xm <= 8 && xa >= 0 && xa + xm <= 8);
                        SCATMAN_ASSERT(ub < P.batch && uj < P.nz && cs < P.batch * P.nz * P.ny16 && cg + (NCTA == 2 ? xm : 16) <= P.nxt * 16);
                        if (NCTA == 2) ptx::tma_load_4d_2sm(dst, tmb, full, 0, 0, cg, cs);
                        else ptx::tma_load_4d(dst, tmb, full, 0, 0, cg, cs);
                    }
                    __syncwarp();
                    if (++slot == kStagesB) { slot = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1 || warp == 3) {
      if (leader) {
        // ===================================================================== MMA issuer (leader CTA only)
        // Warp-uniform loop; descriptors are uniform-register arithmetic; one elected lane issues the
        // tcgen05.mma / tcgen05.commit instructions.
        constexpr uint32_t idesc_pos0 = ptx::umma_idesc_f16(kTileP * NCTA, 0, false);   // N is set per unit
        constexpr uint32_t idesc_neg0 = ptx::umma_idesc_f16(kTileP * NCTA, 0, true);
        const uint64_t descA0 = ptx::umma_smem_desc_sw128(ptx::smem_u32(sA));
        const uint64_t descB0 = ptx::umma_smem_desc_sw32(ptx::smem_u32(sB), 1024);   // x groups 1 KB apart: 4 planes x 256 B
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
        auto commit_local = [](uint64_t *bar) {   // this (leader) CTA's barrier only
            if (NCTA == 2) ptx::umma_commit_2sm(bar, (uint16_t)0x1);
            else ptx::umma_commit(bar);
        };
        const int iw = warp >> 1;   // issuer 0 = warp 1, issuer 1 = warp 3
        int slot = 0;
        uint32_t full_phase = 0;                                   // bit s: parity of the next pass of my_full[s]
        uint64_t *my_full = b_full + iw * kMaxStagesB;
        uint32_t u = 0;
        int it_local = 0;
        for (int item = cluster_id; item < nitems; item += nclusters, ++it_local) {
            const Item it = decode_item(item, P, ntp);
            const int nybg = min(kGroupYB, P.nyb - it.g * kGroupYB);
            ptx::mbar_wait(a_full, (uint32_t)(it_local & 1));
            ptx::tc_fence_after();
            // All-zero units never appear: no MMA, no accumulator hand-over.
            // TWO issuers (warps 1 and 3) share every unit: k-step n of a unit belongs to issuer n % 2.  For N < 112 a
            // tcgen05.mma is bound by its shared-memory operand fetch and, measured, a single issuing thread then
            // exposes every cycle it spends between two k-steps (barrier poll, fences, descriptor arithmetic); two
            // threads hide each other's gaps.  The unit's first k-step (accumulate = 0) is issuer 0's; issuer 1 starts on
            // the unit only after that k-step has completed (first_done).  Both commit the accumulator (t_full counts 2).
            Units un;
            un.begin(it, P, lane);
            unsigned long long m;
            while (un.next_mask(m)) {
                {
                    const uint32_t buf = u & 1;
                    const uint32_t upar = (u >> 1) & 1;
                    ptx::mbar_wait(t_empty + buf, upar ^ 1);
                    ptx::tc_fence_after();
                    const uint32_t d_re = tmem_base + buf * 256, d_im = d_re + 128;
                    int xa, xm;
                    unit_range<NCTA>(m, xa, xm);
                    const uint32_t idesc_pos = idesc_pos0 | ((uint32_t)(2 * xm) << 17);   // N = 16 xm
                    const uint32_t idesc_neg = idesc_neg0 | ((uint32_t)(2 * xm) << 17);
                    constexpr uint64_t pstride = 256 >> 4;   // B planes of one x group are 256 bytes apart
                    int kidx = 0;            // k-step index within the unit
                    for (int yi = 0; yi < 4 * nybg; ++yi) {
                        if (((uint32_t)(m >> (8 * yi)) & 0xffu) == 0u) continue;   // empty 16-y step: never loaded
                        if ((kidx & 1) == iw) {
                            ptx::mbar_wait(my_full + slot, (full_phase >> slot) & 1u);   // this issuer's own barrier of the slot
                            full_phase ^= 1u << slot;
                            if (kidx == 1) {   // issuer 1's first k-step of the unit: D must have been initialised
                                ptx::mbar_wait(first_done + buf, upar);
                            }
                            ptx::tc_fence_after();
                            if (ptx::elect_one()) {
                                // A planes 0 Re_hi, 1 Re_lo, 2 Im_hi, 3 Im_lo of this k-step (32 bytes = 2 descriptor units per step)
                                const uint64_t a_reh = descA0 + (uint64_t)(yi >> 2) * kSlotDescA + (uint64_t)((yi & 3) * 2);
                                const uint64_t a_rel = a_reh + (uint64_t)(1 * kGroupYB) * kSlotDescA;
                                const uint64_t a_imh = a_reh + (uint64_t)(2 * kGroupYB) * kSlotDescA;
                                const uint64_t a_iml = a_reh + (uint64_t)(3 * kGroupYB) * kSlotDescA;
                                const uint64_t b_reh = descB0 + (uint64_t)slot * kSlotDescB;
                                const uint64_t b_rel = b_reh + pstride, b_imh = b_rel + pstride, b_iml = b_imh + pstride;
                                const uint32_t acc0 = kidx != 0 ? 1u : 0u;
                                mma(d_re, a_reh, b_reh, idesc_pos, acc0);
                                mma(d_im, a_imh, b_reh, idesc_pos, acc0);
                                mma(d_re, a_rel, b_reh, idesc_pos, 1u);
                                mma(d_im, a_iml, b_reh, idesc_pos, 1u);
                                mma(d_re, a_reh, b_rel, idesc_pos, 1u);
                                mma(d_im, a_imh, b_rel, idesc_pos, 1u);
                                mma(d_re, a_imh, b_imh, idesc_neg, 1u);
                                mma(d_im, a_reh, b_imh, idesc_pos, 1u);
                                mma(d_re, a_iml, b_imh, idesc_neg, 1u);
                                mma(d_im, a_rel, b_imh, idesc_pos, 1u);
                                mma(d_re, a_imh, b_iml, idesc_neg, 1u);
                                mma(d_im, a_reh, b_iml, idesc_pos, 1u);
                                commit(b_empty + slot);
                                if (kidx == 0) commit_local(first_done + buf);
                            }
                            __syncwarp();
                        }
                        ++kidx;
                        if (++slot == kStagesB) slot = 0;
                    }
                    if (ptx::elect_one()) commit(t_full + buf);
                    __syncwarp();
                    ++u;
                }
            }
            if (ptx::elect_one()) commit(a_empty);
            __syncwarp();
        }
      }
    } else if (warp >= 4) {
        // ========================================================================= epilogue
        const int ew = warp & 3;
        const int el = ew * 32 + lane;  // pixel within the tile = TMEM lane
        const uint32_t lane_base = tmem_base + ((uint32_t)(ew * 32) << 16);
        uint32_t u = 0;
        for (int item = cluster_id; item < nitems; item += nclusters) {
            const Item it = decode_item(item, P, ntp);
            const int tile = it.tp * NCTA + (int)rank;
            const int b0 = it.c * P.bpc, b1 = min(P.batch, b0 + P.bpc);
            float2 fine[kFine];
#pragma unroll
            for (int i = 0; i < kFine; ++i) fine[i] = __ldg(P.fine + ((size_t)tile * kFine + i) * kTileP + el);
            const float2 *anchor_t = P.anchor + (size_t)tile * P.nxa * kTileP + el;
            // slice phase e^{i qz z_j}, z_j = (j - (nz-1)/2) dz: qz z_j = 2 pi t (2j - nz + 1) with t = qz dz / 4 pi turns.  frac(t) is a
            // 64-bit fixed-point fraction of a turn, so the integer product wraps modulo one turn for free; its top 32 bits go
            // to the SFU as an angle in [-pi, pi) (error <= 2^-32 turn + 4e-7 rad of __sincosf, for any nz).
            const unsigned long long zt = __ldg(P.zturn + (size_t)tile * kTileP + el);
            SCATMAN_ASSERT(tile < P.ntiles && it.g < P.ngroups && it.s < P.nzs && b1 <= P.batch);
            float2 *partial_t = P.partial + (size_t)(it.g * P.nzs + it.s) * P.npix_pad + (size_t)tile * kTileP + el;
            const size_t partial_b = (size_t)(P.ngroups * P.nzs) * P.npix_pad;   // stride between batch items
            // Flat walk over the non-empty units; f = row-dot of the current slice, acc = amplitude of the current
            // batch item.  A slice change folds f into acc with e^{i qz z_j}; an item change stores acc.  Items with
            // no unit at all in this work item still get their (zero) partial written.
            Units un;
            un.begin(it, P, lane);
            int ub, uj, xt;
            unsigned long long m;
            int cb = b0, cj = -1;          // current batch item / slice (cj < 0: nothing pending)
            float2 mz = make_float2(0.f, 0.f);
            float acc_re = 0.f, acc_im = 0.f, f_re = 0.f, f_im = 0.f;
            {
                {
                    while (un.next(ub, uj, xt, m)) {
                        if (ub != cb || uj != cj) {
                            acc_re = fmaf(mz.x, f_re, acc_re);      // fold the finished slice (mz = 0 when none pending)
                            acc_re = fmaf(-mz.y, f_im, acc_re);
                            acc_im = fmaf(mz.x, f_im, acc_im);
                            acc_im = fmaf(mz.y, f_re, acc_im);
                            f_re = 0.f;
                            f_im = 0.f;
                            SCATMAN_ASSERT(ub >= cb && ub < b1 && uj >= 0 && uj < P.nz);
                            for (; cb < ub; ++cb) {                 // finished (or empty) batch items
                                partial_t[(size_t)cb * partial_b] = make_float2(acc_re, acc_im);
                                acc_re = 0.f;
                                acc_im = 0.f;
                            }
                            cj = uj;
                            const unsigned long long turn = zt * (unsigned long long)(long long)(2 * uj - P.nz + 1);
                            __sincosf((float)(int)(uint32_t)(turn >> 32) * 1.4629180792671596e-9f, &mz.y, &mz.x);   // pi / 2^31
                        }
                        const uint32_t buf = u & 1;
                        int xa, xm;
                        unit_range<NCTA>(m, xa, xm);   // the unit's accumulator holds x blocks [xa, xa + xm)
                        float2 anc[kTileX / kFine];
#pragma unroll
                        for (int a = 0; a < kTileX / kFine; ++a)
                            anc[a] = __ldg(anchor_t + (size_t)(xt * (kTileX / kFine) + min(xa + a, kTileX / kFine - 1)) * kTileP);
                        ptx::mbar_wait(t_full + buf, (u >> 1) & 1);
                        ptx::tc_fence_after();
                        const uint32_t t_re = lane_base + buf * 256, t_im = t_re + 128;
                        // Column layout of an accumulator (N = 16 xm): x block a = columns [8a, 8a+8) (its x 0..7) and
                        // [8 xm + 8a, +8) (its x 8..15): the two halves of B come from the two CTAs of the pair.
                        const uint32_t half = 8u * (uint32_t)xm;
                        // software-pipelined: the loads of block a+1 are in flight while block a is reduced; the
                        // accumulator buffer is handed back to the MMA warp as soon as its last column has landed
                        uint32_t gre[2][16], gim[2][16];
                        ptx::tmem_ld8(t_re, gre[0]);
                        ptx::tmem_ld8(t_re + half, gre[0] + 8);
                        ptx::tmem_ld8(t_im, gim[0]);
                        ptx::tmem_ld8(t_im + half, gim[0] + 8);
                        ptx::tmem_ld_wait_dep(gre[0]);
                        ptx::tmem_ld_wait_dep(gim[0]);
#pragma unroll
                        for (int a = 0; a < kTileX / kFine; ++a) {
                            if (a < xm) {   // warp-uniform
                                const int cur = a & 1, nxt = cur ^ 1;
                                const bool more = a + 1 < kTileX / kFine && a + 1 < xm;
                                if (more) {
                                    ptx::tmem_ld8(t_re + (a + 1) * 8, gre[nxt]);
                                    ptx::tmem_ld8(t_re + half + (a + 1) * 8, gre[nxt] + 8);
                                    ptx::tmem_ld8(t_im + (a + 1) * 8, gim[nxt]);
                                    ptx::tmem_ld8(t_im + half + (a + 1) * 8, gim[nxt] + 8);
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
                                if (more) {
                                    ptx::tmem_ld_wait_dep(gre[nxt]);
                                    ptx::tmem_ld_wait_dep(gim[nxt]);
                                }
                            }
                        }
                        ++u;
                    }
                }
            }
            acc_re = fmaf(mz.x, f_re, acc_re);
            acc_re = fmaf(-mz.y, f_im, acc_re);
            acc_im = fmaf(mz.x, f_im, acc_im);
            acc_im = fmaf(mz.y, f_re, acc_im);
            for (; cb < b1; ++cb) {
                partial_t[(size_t)cb * partial_b] = make_float2(acc_re, acc_im);
                acc_re = 0.f;
                acc_im = 0.f;
            }
        }
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

bool encode_map(CUtensorMap *tm, const void *base, int rank, const cuuint64_t *dims, const cuuint64_t *strides,
                       const cuuint32_t *box, CUtensorMapSwizzle swizzle) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, (cuuint32_t)rank, const_cast<void *>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Function attributes belong to a device's context: set for the CURRENT device by scatman_create (one context per device).
cudaError_t tensor_init_device() {
    cudaError_t e = cudaFuncSetAttribute(msft_contract_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemTotal);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(msft_contract_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemTotal);
    return e;
}

template <int NCTA>
static cudaError_t launch_variant(const CUtensorMap &tmA, const TmapsB &tmB, const TensorParams &P, int num_sms,
                                  cudaStream_t st) {
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
    CUtensorMap tmA;
    TmapsB tmB;
    // A: fp16 [4 planes][npix_pad][ny_pad], box = one 64-y K-block of a 128-pixel tile, 128-byte swizzle
    bool ok;
    {
        cuuint64_t dims[3] = {(cuuint64_t)p.ny_pad, (cuuint64_t)p.npix_pad, 4};
        cuuint64_t strides[2] = {(cuuint64_t)p.ny_pad * 2, (cuuint64_t)p.ny_pad * (cuuint64_t)p.npix_pad * 2};
        cuuint32_t box[3] = {(cuuint32_t)kBlockY, (cuuint32_t)kTileP, 1};
        ok = encode_map(&tmA, t.d_A, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    // B: fp16 [batch nz ny16][16 nxt x-groups][4 planes][128-element atom] (pack_b_kernel); box = one 16-y step of
    // i+1 x-groups (CTA pairs fetch only the groups of a unit's x range) or of the whole tile (single CTA)
    for (int i = 0; ok && i < kTileX / 16; ++i) {
        cuuint64_t dims[4] = {128, 4, (cuuint64_t)p.nxt * 16, (cuuint64_t)p.batch * p.nz * (p.ny_pad / 16)};
        cuuint64_t strides[3] = {256, 1024, (cuuint64_t)p.nxt * 16 * 1024};
        cuuint32_t box[4] = {128, 4, (cuuint32_t)(ncta == 2 ? i + 1 : 16), 1};
        ok = encode_map(&tmB.m[i], t.d_B, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_NONE);
    }
    if (!ok) {
        if (err) *err = "cuTensorMapEncodeTiled failed or is unavailable";
        return cudaErrorUnknown;
    }
    TensorParams P;
    P.nz = p.nz; P.nxt = p.nxt; P.nyb = p.nyb; P.ny16 = p.ny_pad / 16; P.ngroups = p.ngroups; P.ntiles = p.ntiles; P.batch = p.batch;
    P.nzs = p.t_nzs;
    P.bpc = (p.batch + p.t_nchunks - 1) / p.t_nchunks;
    P.nchunks = (p.batch + P.bpc - 1) / P.bpc;
    P.nxa = p.nxa;
    P.npix_pad = p.npix_pad;
    P.anchor = t.d_anchor; P.fine = t.d_fine; P.zturn = t.d_zturn; P.partial = t.d_partial; P.mask = t.d_mask;
    return ncta == 2 ? launch_variant<2>(tmA, tmB, P, t.num_sms, st) : launch_variant<1>(tmA, tmB, P, t.num_sms, st);
}


}  // namespace scatman
