// rfa_internal.h -- host-side declarations shared by rfa_api.cpp (host logic, C ABI) and
// rfa_kernels.cu (sm_100a kernels + launchers).  Not part of the public boundary.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "rfa_device.cuh"

struct RfaGrid {
    int nx, ny, nz, batch;
    float wx, wy, wz;   // normalised 1/h^2 weights (sum = 1)
    float thr;          // necrosis threshold in theta = T - T_a
    float t_blood;
    int held_copy;      // 1: kernel variant in which warps of held voxels only copy their rows (Alg. 1 :313);
                        // chosen by rfa_create when >= 1/8 of the volume carries a held label (rfa_configure_held_copy overrides)
};

// Plan of the temporally blocked kernel for one launch geometry.
struct RfaTbPlan {
    int fused;                 // S: time steps per launch, 1..4
    int shape;                 // index into RFA_TB_SHAPE
    int tiles_x, tiles_y;      // xy tiling
    int nzc, zchunk;           // z chunks
    int n_items;               // batch * nzc * tiles_y * tiles_x
    int grid;                  // CTAs launched (persistent, static round-robin over items)
    int ok;                    // 0: this grid cannot use the blocked kernel
    int tma;                   // 1: the variant whose level-0 planes are staged by the Tensor Memory Accelerator
};

// tile shape of the blocked kernel per number of fused steps S (index 1..4): TX x TY threads, each owning
// one float4 column and RY rows -> BX = 4 TX by BY = RY TY voxels per plane; minb = CTAs per SM asked
// of the compiler (register cap).
struct RfaTbShape {
    int tx, ty, ry, minb;
};
#ifndef RFA_TX
#define RFA_TX 16
#endif
#ifndef RFA_TY
#define RFA_TY 16
#endif
#ifndef RFA_S1_RY
#define RFA_S1_RY 4
#define RFA_S1_MINB 2
#endif
#ifndef RFA_S2_RY
#define RFA_S2_RY 2
#define RFA_S2_MINB 2
#endif
#ifndef RFA_S3_RY
#define RFA_S3_RY 2
#define RFA_S3_MINB 2
#endif
#ifndef RFA_S4_RY
#define RFA_S4_RY 2
#define RFA_S4_MINB 2
#endif
// Two thread arrangements of the same 256-thread CTA, chosen per grid by the planner (fewest plane iterations):
//   shape 0  16 x 16 threads: tile 64 x 32  -- few y halo rows; the default on wide grids
//   shape 1  32 x  8 threads: tile 128 x 16 -- a whole 128-voxel row per tile (no x halo at all for nx <= 128:
//            the 128^3 planning-sweep volumes run 1.3x faster with it)
#define RFA_N_SHAPES 2
constexpr RfaTbShape RFA_TB_SHAPE[RFA_N_SHAPES][5] = {{{0, 0, 0, 0},
                                                       {RFA_TX, RFA_TY, RFA_S1_RY, RFA_S1_MINB},
                                                       {RFA_TX, RFA_TY, RFA_S2_RY, RFA_S2_MINB},
                                                       {RFA_TX, RFA_TY, RFA_S3_RY, RFA_S3_MINB},
                                                       {RFA_TX, RFA_TY, RFA_S4_RY, RFA_S4_MINB}},
                                                      {{0, 0, 0, 0},
                                                       {2 * RFA_TX, RFA_TY / 2, RFA_S1_RY, RFA_S1_MINB},
                                                       {2 * RFA_TX, RFA_TY / 2, RFA_S2_RY, RFA_S2_MINB},
                                                       {2 * RFA_TX, RFA_TY / 2, RFA_S3_RY, RFA_S3_MINB},
                                                       {2 * RFA_TX, RFA_TY / 2, RFA_S4_RY, RFA_S4_MINB}}};

// host-only planning (no CUDA calls): implemented in rfa_api.cpp, unit-tested on CPU
// resident_ctas: co-resident CTAs per shape (0 = this shape cannot run)
// tma = 1: plan for the TMA-staged variant (tiles start RY-aligned above the grid: one more halo row at S = 3)
RfaTbPlan rfa_plan_blocked(int nx, int ny, int nz, int batch, int fused, const int resident_ctas[RFA_N_SHAPES], int tma = 0);

// launchers (rfa_kernels.cu).  All asynchronous on `st`; return cudaGetLastError().
cudaError_t rfa_launch_table(const RfaTableHost &tbl, float *dst, cudaStream_t st);
// resid: fp16 residual image (rfa_device.cuh: rfa_advance), same indexing as theta
cudaError_t rfa_launch_init(const RfaGrid &g, const uint8_t *labels_dev, const float *theta0_by_label /*host, 16*/,
                            const float *k_by_label /*host, 16*/, float *theta, void *resid, uint8_t *state,
                            cudaStream_t st);
// label histogram of the uploaded volume (256 bins, device; zeroed by the call)
cudaError_t rfa_launch_label_hist(const RfaGrid &g, const uint8_t *labels_dev, unsigned long long *hist_dev, cudaStream_t st);
cudaError_t rfa_launch_needle(const RfaGrid &g, int scenario, const uint8_t *mask_dev /*may be null*/, int mode,
                              float theta_value, float *theta, void *resid, uint8_t *state, cudaStream_t st);
cudaError_t rfa_launch_set_temperature(const RfaGrid &g, int scenario, const float *t_dev, float *theta,
                                       void *resid, uint8_t *state, cudaStream_t st);
cudaError_t rfa_launch_get_temperature(const RfaGrid &g, int scenario, const float *theta, float *out_dev,
                                       cudaStream_t st);
cudaError_t rfa_launch_get_necrosis(const RfaGrid &g, int scenario, const uint8_t *state, uint8_t *out_dev,
                                    cudaStream_t st);
cudaError_t rfa_launch_warp(const RfaGrid &g, int scenario, const float *theta /*all scenarios*/, const float *disp_dev,
                            float scale, const float inv_h_mm[3], float *out_dev, cudaStream_t st);
// orthographic camera of rfa_render_zone, set up in fp64 on the host (include/rfa.h: rfa_view)
struct RfaRay {
    double c[3], e1[3], e2[3], w[3];   // volume centre (mm), image-plane basis, viewing direction (unit)
    double inv_h[3];                   // 1 / voxel spacing (1/mm)
    double R, pixel, step;             // half diagonal, pixel spacing, sample spacing (mm)
    int width, height, n_samples;
};
cudaError_t rfa_launch_render(const RfaGrid &g, int scenario, const RfaRay &ray, const float *theta /*all scenarios*/,
                              float iso_theta, float *tmax_dev, float *depth_dev /*may be null*/, cudaStream_t st);
cudaError_t rfa_launch_probe(const RfaGrid &g, int n, const long long *index_dev, const float *theta /*all scenarios*/,
                             float *out_dev, cudaStream_t st);
// ---- rfa_step_record_static: probe list and rows in a file-scope device array (rfa_noalloc.cu), no allocation anywhere ----
// begin: probe list (host) -> head of the array;  probe: the probe kernel into row `row`;  fetch: rows -> out (host or device).
// All asynchronous on `st`, all for the CURRENT device (the first of them on a device looks the array's address up).
cudaError_t rfa_static_record_begin(int n_probes, const long long *index_host, cudaStream_t st);
cudaError_t rfa_static_record_probe(const RfaGrid &g, int n_probes, const float *theta /*all scenarios*/, size_t row, cudaStream_t st);
cudaError_t rfa_static_record_fetch(float *out, size_t floats, cudaStream_t st);
cudaError_t rfa_launch_count(const RfaGrid &g, int scenario, const uint8_t *state, uint32_t label_held_mask,
                             unsigned long long *counters_dev /*2*/, cudaStream_t st);
// kap: null = Eq. 12 as printed; else device table [16][16] of Kf/K_c - 1 (conservative conduction, R-28)
cudaError_t rfa_launch_plain(const RfaGrid &g, const float *tin, float *tout, const void *rin, void *rout,
                             uint8_t *state, const float *tables, const float *kap, cudaStream_t st);
struct RfaTensorMap;
// map_theta_in / map_state: tensor maps (box = the plan's tile) of the input image and the state volume; used when plan.tma
cudaError_t rfa_launch_blocked(const RfaGrid &g, const RfaTbPlan &plan, const float *tin, float *tout,
                               const void *rin, void *rout, uint8_t *state, const float *tables, const float *kap,
                               const RfaTensorMap *map_theta_in, const RfaTensorMap *map_state, int res_prefetch,
                               unsigned long long *hot_ctr /*device: += hot warp-planes*/, cudaStream_t st);
// 1: a kernel variant that prefetches the level-0 residual rows of hot planes exists for this number of fused steps / staging
int rfa_blocked_has_prefetch(int fused, int tma);
void rfa_blocked_tile(int fused, int shape, int *bx, int *by);
// ---- one-step kernel staged by the Tensor Memory Accelerator (rfa_stream.cu) ----------------------------------------
// tile of one CTA: RFA_STREAM_BX x RFA_STREAM_BY voxels (8 warps x RFA_STREAM_RY rows, one float4 column per lane), a ring of
// RFA_STREAM_D shared-memory slots per CTA (D - 2 planes in flight).  Measured on the B200 (C4, us per step): 2 rows per
// warp 146, 4 rows 198-241, 1 row with 16 warps 152; ring depth 3 / 4 / 6 / 8: 164 / 152 / 163 / 168; 3 or 4 CTAs per SM
// 186-204: this memory system wants about two planes in flight per CTA and few concurrent streams, not more of either.
#define RFA_STREAM_BX 128
#ifndef RFA_STREAM_RY
#define RFA_STREAM_RY 2
#endif
#ifndef RFA_STREAM_NW
#define RFA_STREAM_NW 8                    // warps per CTA, each owning RFA_STREAM_RY rows of the tile
#endif
#define RFA_STREAM_BY (RFA_STREAM_NW * RFA_STREAM_RY)
#ifndef RFA_STREAM_D
#define RFA_STREAM_D 4
#endif
#ifndef RFA_STREAM_MINB
#define RFA_STREAM_MINB 2                  // CTAs per SM asked of the compiler (register cap)
#endif
struct alignas(64) RfaTensorMap {
    unsigned long long opaque[16];   // a CUtensorMap (cuda.h), kept opaque so that host code needs no driver header
};
// tensor maps of one fp32 image / of the packed state volume, both seen as (nx, ny, nz * batch); either output may be null.
// false: no TMA path for this grid (nx % 16 != 0) or no driver entry point
// general form: box_x x box_y x 1 elements of 4 (fp32 image) or 1 (state volume) bytes
bool rfa_make_tile_map(const RfaGrid &g, const void *base, int elem_bytes, int box_x, int box_y, RfaTensorMap *out);
bool rfa_stream_make_maps(const RfaGrid &g, const float *theta, const uint8_t *state, RfaTensorMap *map_theta, RfaTensorMap *map_state);
int rfa_stream_resident_ctas();
// plan fields used: tiles_x, tiles_y, nzc, zchunk, n_items, grid
RfaTbPlan rfa_plan_stream(int nx, int ny, int nz, int batch, int resident_ctas);
cudaError_t rfa_launch_stream(const RfaGrid &g, const RfaTbPlan &plan, const RfaTensorMap &map_theta_in, const RfaTensorMap &map_state,
                              float *tout, const void *rin, void *rout, uint8_t *state, const float *tables,
                              unsigned long long *work_ctr /*device, never reset*/, unsigned long long work_base /*its value at launch*/,
                              cudaStream_t st);

// resident CTAs of the blocked kernel on the current device for `fused` steps (occupancy * SM count);
// cons = 1: the conservative-conduction variant
int rfa_blocked_resident_ctas(int fused, int shape, int cons, int tma = 0);
