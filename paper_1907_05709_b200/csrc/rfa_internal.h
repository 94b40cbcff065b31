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
RfaTbPlan rfa_plan_blocked(int nx, int ny, int nz, int batch, int fused, const int resident_ctas[RFA_N_SHAPES]);

// launchers (rfa_kernels.cu).  All asynchronous on `st`; return cudaGetLastError().
cudaError_t rfa_launch_table(const RfaTableHost &tbl, float *dst, cudaStream_t st);
// resid: fp16 residual image (rfa_device.cuh: rfa_advance), same indexing as theta
cudaError_t rfa_launch_init(const RfaGrid &g, const uint8_t *labels_dev, const float *theta0_by_label /*host, 16*/,
                            const float *k_by_label /*host, 16*/, float *theta, void *resid, uint8_t *state,
                            cudaStream_t st);
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
cudaError_t rfa_launch_count(const RfaGrid &g, int scenario, const uint8_t *state, uint32_t label_held_mask,
                             unsigned long long *counters_dev /*2*/, cudaStream_t st);
// kap: null = Eq. 12 as printed; else device table [16][16] of Kf/K_c - 1 (conservative conduction, R-28)
cudaError_t rfa_launch_plain(const RfaGrid &g, const float *tin, float *tout, const void *rin, void *rout,
                             uint8_t *state, const float *tables, const float *kap, cudaStream_t st);
cudaError_t rfa_launch_blocked(const RfaGrid &g, const RfaTbPlan &plan, const float *tin, float *tout,
                               const void *rin, void *rout, uint8_t *state, const float *tables, const float *kap,
                               cudaStream_t st);
// resident CTAs of the blocked kernel on the current device for `fused` steps (occupancy * SM count)
int rfa_blocked_resident_ctas(int fused, int shape);
