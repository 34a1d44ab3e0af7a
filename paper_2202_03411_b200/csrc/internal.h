// internal.h -- shared declarations of libscatman's translation units (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cstddef>
#include <cstdint>
#include <string>

#include "../../include/scatman.h"

namespace scatman {

// ---- tile geometry of the tensor-core contraction (tensor_kernel.cu) ---------------------------
constexpr int kTileP = 128;     // pixels per CTA tile          = UMMA M
constexpr int kTileX = 128;     // x columns per accumulator    = UMMA N
constexpr int kBlockY = 64;     // y per smem K-block (64 fp16 = one 128-byte swizzle row)
constexpr int kGroupYB = 2;     // K-blocks of the A operand resident in smem per work item
constexpr int kFine = 16;       // x per anchor block in the epilogue row-dot
constexpr float kScaleA = 1024.0f;  // M_y tables are stored as 2^10 * e^{i qy y} (keeps the FP16 low part normal)
constexpr int kScaleBExp = 13;  // rho~ is scaled so that max |component| lies in [2^12, 2^13)

// Problem plan: every derived size and every workspace offset, computed on the host.
struct Plan {
    int nx = 0, ny = 0, nz = 0;
    double dx = 0, dy = 0, dz = 0, lambda = 0;
    int64_t npix = 0;
    int batch = 0;
    int rho_mode = 0, method = 0;
    int64_t nvox = 0;
    // padded sizes of the tensor path
    int nx_pad = 0, ny_pad = 0;   // multiples of kTileX / kBlockY
    int nyb = 0;                  // ny_pad / kBlockY
    int ngroups = 0;              // y-groups (work items per pixel tile and batch chunk)
    int nxt = 0;                  // x tiles
    int nxa = 0;                  // anchor blocks per row = nx_pad / kFine
    int ntiles = 0;               // pixel tiles
    int64_t npix_pad = 0;
    int nsplit = 0;               // partial sums per pixel (tensor: ngroups * t_nzs; simt: z splits)
    int t_nchunks = 1, t_nzs = 1; // tensor schedule: batch chunks and z splits per (tile, y-group)
    int t_ncta = 2;               // CTAs per work item: 2 = cta_group::2 pairs (default), 1 = single CTA
    // workspace offsets (bytes)
    size_t off_q = 0, off_rotmat = 0, off_rot = 0, off_rho = 0, off_max = 0, off_ampscale = 0, off_B = 0,
           off_A = 0, off_anchor = 0, off_fine = 0, off_zturn = 0, off_partial = 0, off_mask = 0, off_count = 0, off_bbox = 0, off_tab_y = 0, off_tab_x = 0, off_tab_z = 0, off_flags = 0, total = 0;
};

int simt_zsplit(const Plan &p, int num_sms);
void tensor_schedule(const Plan &p, int num_workers, int *nchunks, int *nzs);

// ---- kernels launchers (all asynchronous on `st`; return cudaGetLastError()) -------------------
cudaError_t launch_qmap(const scatman_detector &det, double lambda, double *d_q, cudaStream_t st);
cudaError_t launch_orient(const float *d_in, const Plan &p, const double *d_rotmat, int batch, float *d_out, int *d_bbox,
                          cudaStream_t st, unsigned *d_stats = nullptr,   // d_stats[batch][3]: also the extremes of the input, FP32 bits
                          unsigned char *d_tilemap = nullptr, unsigned char *d_occ = nullptr);   // d_occ: orient_occ_bytes() of scratch (coarse occupancy map)
// d_tilemap = null: d_out is written everywhere.  Else SPARSE output: only the 16 x 4 x 4-voxel tiles that can hold material are
// written, and d_tilemap[b][ceil(nz/4)][ceil(ny/4)][ceil(nx/16)] = 1 for those of them that received material -- the rest of d_out is left as it was (or holds zeros) and must be read
// as vacuum (launch_sep_tc_prefix_prep does)
inline size_t orient_tilemap_bytes(const Plan &p, int batch) {
    return (size_t)batch * ((p.nz + 3) / 4) * ((p.ny + 3) / 4) * ((p.nx + 15) / 16);
}
inline size_t tile_layers_bytes(const Plan &p, int batch) { return (size_t)batch * ((p.nz + 3) / 4); }
// bbox_kernel's coarse occupancy map for orient_kernel (4^3-voxel blocks); 0 = not used (a slice's map must fit 4 KB of shared memory)
inline size_t orient_occ_bytes(const Plan &p, int batch) {
    const size_t sl = (size_t)(p.nx / 4 + 1) * (p.ny / 4 + 1);
    return sl <= 4096 ? (size_t)batch * (p.nz / 4 + 1) * sl : 0;
}
// a0's scratch: the boxes [batch][6] followed by the occupancy map
inline size_t orient_scratch_bytes(const Plan &p, int batch) {
    return (sizeof(int) * 6 * (size_t)batch + 255) / 256 * 256 + orient_occ_bytes(p, batch);
}
inline unsigned char *orient_occ_ptr(void *d_bbox, const Plan &p, int batch) {
    return orient_occ_bytes(p, batch) ? (unsigned char *)d_bbox + (sizeof(int) * 6 * (size_t)batch + 255) / 256 * 256 : nullptr;
}
// the bound of max |rho~| per item that its extremes {max |delta|, max |beta|, max(0, -beta)} give (p.lambda, dz, nz, rho_mode)
cudaError_t launch_prefix_bound(const unsigned *d_stats, const Plan &p, int batch, unsigned *d_maxbits, cudaStream_t st);
cudaError_t launch_strength(const float *d_dn, const Plan &p, int batch, float *d_rho, unsigned *d_maxbits,
                            cudaStream_t st);
cudaError_t launch_pack_b(const float *d_rho, const Plan &p, const unsigned *d_maxbits, float *d_ampscale,
                          __half *d_B, unsigned long long *d_mask, cudaStream_t st);
cudaError_t launch_count_issued(const unsigned long long *d_mask, const Plan &p, unsigned long long *d_count,
                                cudaStream_t st);
cudaError_t launch_tables(const double *d_q, const Plan &p, __half *d_A, float2 *d_anchor, float2 *d_fine,
                          unsigned long long *d_zturn, cudaStream_t st, int *nlaunch);
cudaError_t launch_finalize(const float2 *d_partial, const Plan &p, const float *d_ampscale, double dV,
                            float *d_I, cudaStream_t st);
cudaError_t launch_simt_sincos(const float *d_rho, const double *d_q, const Plan &p, float2 *d_partial,
                               cudaStream_t st);
cudaError_t launch_simt_table(const float *d_rho, const double *d_q, const Plan &p, float2 *d_My, float2 *d_Mx, float2 *d_Mz,
                              unsigned char *d_flags, float2 *d_partial, cudaStream_t st, int *nlaunch);

cudaError_t launch_sep_tables(const double *d_qx, int npx, const double *d_qy, int npy, const Plan &p, float2 *d_Ex,
                              float2 *d_Ey, cudaStream_t st);
int sep_zsplit(const Plan &p, int npx, int npy, int num_sms);
cudaError_t launch_sep_item(const float2 *d_rho, const Plan &p, const float2 *d_Ex, const float2 *d_Ey, const double *d_qx,
                            int npx, const double *d_qy, int npy, int nzs, float2 *d_H, unsigned char *d_flags,
                            float2 *d_partial, float *d_I, cudaStream_t st);
// separable route on tensor cores (sep_tensor_kernels.cu)
struct SepTcPlan {
    int NY = 0, NXP = 0, NPXP = 0, NPYP = 0;   // padded y (x128), x (x64), grid columns (x128), grid rows (x128; x256 in the streamed form)
    int ng = 0, nzs = 1, nsplit = 1, L = 0;    // 128-y groups, z splits of stage YZ (= partial sums per point), ceil(log2 nx)
    int NX = 64, nsx = 1, x_ncta = 2;          // stage X: a columns per resident Ex tile, z splits, CTAs per work item (always pairs)
    int nyz = 128, yz_ncta = 2;                // stage YZ: a columns per tile, CTAs per work item (always pairs)
    bool yz_stream = true;                     // stage YZ keeps one accumulator per slice (both forms): bounds and partial sums per item
    bool yz_t = false;                         // stage YZ transposed, Ey resident for all y (SepYztPolicy<yzt_nb>); else sep_tc_yzs_kernel
    int yzt_nb = 0;
    int nb = 1;                                // batch items per chunk (stacked along z, one set of launches per chunk)
};
SepTcPlan make_sep_tc_plan(const Plan &p, int npx, int npy, int num_sms);
cudaError_t launch_sep_tc_tables(const double *d_qx, int npx, const double *d_qy, int npy, const Plan &p,
                                 const SepTcPlan &t, __half *d_Exp, __half *d_Eyp, cudaStream_t st);
// a2 fused with the operand pack: (delta, beta) grids -> FP16 planes of rho~ + flags + per-item scale + z-split bounds; d_maxbits = bounds of
// max |rho~| per item (launch_prefix_bound).  Replaces launch_strength + launch_sep_tc_prep on the routes that only need the planes.
cudaError_t launch_sep_tc_prefix_prep(const float2 *d_dn, const unsigned *d_maxbits, const Plan &p, const SepTcPlan &t, int nb,
                                      __half *d_Rp, unsigned char *d_flags64, int *d_bounds, float *d_ampscale, cudaStream_t st,
                                      bool x_only = false, const unsigned char *d_tilemap = nullptr,    // d_tilemap: of these nb items (launch_orient)
                                      unsigned char *d_layer_live = nullptr);   // scratch, nb ceil(nz / 4) bytes: with a tile map, layers without a written tile are not packed
cudaError_t launch_sep_tc_prep(const float2 *d_rho, const unsigned *d_maxbits, const Plan &p, const SepTcPlan &t, int nb,
                               __half *d_Rp, unsigned char *d_flags64, int *d_bounds, float *d_ampscale, cudaStream_t st,
                               bool x_only = false);   // x_only: z-split bounds of stage X only (the NUFFT route)
cudaError_t launch_sep_tc_x(const Plan &p, const SepTcPlan &t, const __half *d_Rp, const __half *d_Exp,
                            const unsigned char *d_flags64, const int *d_bounds, int nb, __half *d_Hp, int num_sms,
                            cudaStream_t st, std::string *err,
                            int ncols = 0);   // > 0: only columns a < ncols of H are stored (nobody reads the padding)
cudaError_t launch_sep_tc_yz(const Plan &p, const SepTcPlan &t, const __half *d_Eyp, const __half *d_Hp,
                             const unsigned char *d_flags64, const int *d_bounds, int nb, const double *d_qx, int npx,
                             const double *d_qy, int npy, float2 *d_partial, int num_sms, cudaStream_t st, std::string *err);
cudaError_t launch_sep_tc_finalize(const float2 *d_partial, const double *d_qx, int npx, const double *d_qy, int npy,
                                   const Plan &p, const SepTcPlan &t, int nb, const float *d_ampscale, float *d_I,
                                   cudaStream_t st);
int launch_render_batch(const scatman_shape *h_shapes, int batch, const scatman_grid &g, float *d_dn, cudaStream_t st,
                        cudaError_t *err, int *nlaunch,    // 0, or 1 + index of the first bad descriptor
                        unsigned char *d_tilemap = nullptr);   // non-null: sparse output + tile map, as launch_orient's

// flat-detector route by a 3-D type-2 NUFFT (nufft_kernels.cu)
constexpr int kNufftW = 8;                      // Kaiser-Bessel window width in grid cells (oversampling 2); R25
struct NufftAxis { int m_lo = 0, nq = 0; double inv_h = 0; };   // uniform grid g_m = (m_lo + m) h, m = 0..nq-1; inv_h = 1 / h
struct NufftPlan { NufftAxis ax, ay, az; int nb = 1; double pixel_cells = 0; };   // nb = batch items per chunk
cudaError_t nufft_init_device();   // once per device (scatman_create): uploads the window's piecewise polynomials
// per-device kernel attributes (dynamic shared memory limits) of the other translation units; called by scatman_create
cudaError_t tensor_init_device();
cudaError_t sep_init_device();
cudaError_t sep_tc_init_device();
cudaError_t render_init_device();
cudaError_t launch_nufft_tables(const Plan &p, const NufftPlan &n, double2 *d_Tz, double2 *d_TxT, double2 *d_Ty, cudaStream_t st);
cudaError_t launch_nufft_chunk(const float2 *d_rho, const Plan &p, const NufftPlan &n, int nb, int npx, int npy, double pixel_cells,
                               const double2 *d_Tz, const double2 *d_TxT, const double2 *d_Ty, const double *d_q, double2 *d_P,
                               double2 *d_H, float2 *d_U, float *d_I, cudaStream_t st);

// the NUFFT route's GEMM stages on tensor cores (nufft_tensor_kernels.cu)
struct NufftTcPlan {
    bool ok = false;                 // the grid fits the resident operands (nx, ny, nz <= 1024); else the FP64 stages run
    SepTcPlan sep;                   // stage X = the separable route's stage X on the nqx uniform-grid columns
    int NY = 0, NPXP = 0;            // padded y (x128) and uniform-grid columns, as in sep
    int nky = 0, nkz = 0, NZP = 0;   // 64-blocks of y and of one item's slices; padded slices of the Tz planes
    int nby = 0, nbz = 0;            // resident table rows per CTA in stages Y and Z (64 / 32 / 16)
    int NQYP = 0, NQZP = 0;          // padded uniform-grid rows and planes (multiples of 2 nby, 2 nbz)
    int nb = 1, NZI = 0, NZT = 0;    // items per chunk; slices per item padded to 8; row length of V (nb NZI)
};
NufftTcPlan make_nufft_tc_plan(const Plan &p, const NufftPlan &n, int batch, int num_sms);
cudaError_t nufft_tc_init_device();
cudaError_t launch_nufft_tc_tables(const Plan &p, const NufftPlan &n, const NufftTcPlan &t, __half *d_Tx, __half *d_Ty, __half *d_Tz,
                                   cudaStream_t st);
cudaError_t launch_nufft_tc_yz(const Plan &p, const NufftPlan &n, const NufftTcPlan &t, int nb, const __half *d_Hp, const __half *d_Ty,
                               const __half *d_Tz, __half *d_Vp, float2 *d_U, int num_sms, cudaStream_t st, std::string *err,
                               const unsigned char *d_flags64 = nullptr);
bool nufft_tc_needs_h_memset(const NufftTcPlan &t);   // false: pass d_flags64 above instead of zeroing the H planes
// interpolation of a chunk from U (FP32 complex [nb][nqz][nqy][nqx]); amplitude scale = ampscale[b] * scale_mul, or dV if ampscale is null
cudaError_t launch_nufft_interp(const Plan &p, const NufftPlan &n, int nb, int npx, int npy, double pixel_cells, const double *d_q,
                                const float2 *d_U, const float *d_ampscale, double scale_mul, float *d_I, cudaStream_t st);

// forward-fitting pieces (fit_kernels.cu)
size_t fit_workspace_bytes(int64_t npix, int batch);
int fit_discrepancy_launches(int64_t npix, int batch);   // 3 or 4: the sums of few chunks per item are added inside pass 2
cudaError_t launch_discrepancy(const float *d_I, const float *d_M, int64_t m_stride, const unsigned char *d_mask, int64_t npix,
                               int batch, int metric, double *d_ws, double *d_out, cudaStream_t st);
cudaError_t launch_ideal_detector(const float *d_I, int64_t npix, int batch, const double *h_photons, uint64_t seed, double *d_ws,
                                  float *d_counts, cudaStream_t st);
// device address, on `device` (which must be current), of the library's static scratch array (SCATMAN_STATIC_SCRATCH_BYTES;
// scatman_discrepancy_static): resolved with cudaGetSymbolAddress once per device
cudaError_t fit_static_scratch(int device, double **d_ptr);

// tensor path: tensor maps are encoded on the host through the driver entry point
struct TensorMaps;  // opaque here
struct TensorLaunch {
    const void *d_A;      // fp16 [4][npix_pad][ny_pad]
    const void *d_B;      // fp16 [batch][nz][4][nx_pad][ny_pad]
    const float2 *d_anchor, *d_fine;
    const unsigned long long *d_zturn;   // [tile][128] slice-phase turn fractions
    const unsigned long long *d_mask;  // occupancy [batch][nz][nxt][ngroups], bit 8*yi + xi: 16-y x 16-x block is non-zero
    float2 *d_partial;
    int num_sms;
};
cudaError_t launch_tensor(const Plan &p, const TensorLaunch &t, cudaStream_t st, std::string *err);
size_t tensor_smem_bytes();

}  // namespace scatman
