// rfa_kernels.cu -- sm_100a kernels of librfa.so.
//
//   rfa_plain_kernel     one thread per voxel, one time step per launch (any grid size)
//   rfa_blocked_kernel   the hot path: 2.5D z-sweep, S fused time steps per launch
//   + small set-up / read-back kernels (init, needle, set/get temperature, necrosis, count)
//
// Every stepping kernel evaluates rfa_update() (rfa_device.cuh) with the same operands in the same
// order, so all variants produce bit-identical fields.
#include <cstdio>

#include "rfa_internal.h"

// ------------------------------------------------------------------------------------------------
// small helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

// ------------------------------------------------------------------------------------------------
// set-up / read-back kernels
// ------------------------------------------------------------------------------------------------
__global__ void rfa_table_kernel(RfaTableHost tbl, float *dst)
{
    int e = threadIdx.x;
    if (e < RFA_TABLE_N) {
        dst[e] = tbl.a[e];
        dst[RFA_TABLE_N + e] = tbl.nk[e];
        dst[2 * RFA_TABLE_N + e] = tbl.qa[e];
    }
}

struct Theta0 {
    float v[32];
};

// label -> initial temperature image: theta = t_init[label] - T_a, state = label id,
// necrosis on the initial state (R-14).  One launch covers all scenarios.
__global__ void rfa_init_kernel(size_t nvox, int batch, const uint8_t *__restrict__ labels, Theta0 t0, float thr,
                                float *__restrict__ theta, uint8_t *__restrict__ state)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvox) return;
    unsigned l = labels[v] & RFA_ST_LABEL;
    float t = t0.v[l];
    unsigned st = l | (t >= thr ? RFA_ST_NECRO : 0u);
    for (int b = 0; b < batch; ++b) {
        theta[(size_t)b * nvox + v] = t;
        state[(size_t)b * nvox + v] = (uint8_t)st;
    }
}

// needle placement for one scenario (R-15, R-16, R-17)
__global__ void rfa_needle_kernel(size_t nvox, const uint8_t *__restrict__ mask, int mode, float theta_value,
                                  float thr, float *__restrict__ theta, uint8_t *__restrict__ state)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvox) return;
    unsigned st = state[v] & ~(RFA_ST_DIRICHLET | RFA_ST_POWER);       // release the old needle
    if (mode != 0 && mask[v]) {
        if (mode == 1) {
            st |= RFA_ST_DIRICHLET;
            theta[v] = theta_value;
            if (theta_value >= thr) st |= RFA_ST_NECRO;
        } else {
            st |= RFA_ST_POWER;
        }
    }
    state[v] = (uint8_t)st;
}

__global__ void rfa_set_temperature_kernel(size_t nvox, const float *__restrict__ t_c, float t_blood, float thr,
                                           float *__restrict__ theta, uint8_t *__restrict__ state)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvox) return;
    float t = __fsub_rn(t_c[v], t_blood);
    theta[v] = t;
    if (t >= thr) state[v] |= RFA_ST_NECRO;
}

__global__ void rfa_get_temperature_kernel(size_t nvox, const float *__restrict__ theta, float t_blood,
                                           float *__restrict__ out)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v < nvox) out[v] = __fadd_rn(theta[v], t_blood);
}

__global__ void rfa_get_necrosis_kernel(size_t nvox, const uint8_t *__restrict__ state, uint8_t *__restrict__ out)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v < nvox) out[v] = state[v] >> 7;
}

__global__ void rfa_count_kernel(size_t nvox, const uint8_t *__restrict__ state, uint32_t label_held_mask,
                                 unsigned long long *counters)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned all = 0, tissue = 0;
    if (v < nvox) {
        unsigned st = state[v];
        if (st & RFA_ST_NECRO) {
            all = 1;
            bool needle = (st & (RFA_ST_DIRICHLET | RFA_ST_POWER)) != 0;
            bool held_label = (label_held_mask >> (st & RFA_ST_LABEL)) & 1u;
            tissue = (!needle && !held_label) ? 1u : 0u;
        }
    }
    unsigned a = __reduce_add_sync(0xffffffffu, all);
    unsigned t = __reduce_add_sync(0xffffffffu, tissue);
    if ((threadIdx.x & 31) == 0) {
        if (a) atomicAdd(&counters[0], (unsigned long long)a);
        if (t) atomicAdd(&counters[1], (unsigned long long)t);
    }
}

// ------------------------------------------------------------------------------------------------
// plain kernel: Alg. 1 literally -- "for all voxel", one thread each
// ------------------------------------------------------------------------------------------------
__global__ void rfa_plain_kernel(RfaGrid g, const float *__restrict__ tin, float *__restrict__ tout,
                                 uint8_t *__restrict__ state, const float *__restrict__ tables)
{
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    size_t gid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= nvox * (size_t)g.batch) return;
    const int b = (int)(gid / nvox);
    const size_t v = gid - (size_t)b * nvox;
    const int i = (int)(v % g.nx);
    const int j = (int)((v / g.nx) % g.ny);
    const int k = (int)(v / ((size_t)g.nx * g.ny));
    const float *T = tin + (size_t)b * nvox;
    const float *tab = tables + (size_t)b * 3 * RFA_TABLE_N;
    const size_t sx = 1, sy = g.nx, sz = (size_t)g.nx * g.ny;
    const float t = T[v];
    const float xm = i > 0 ? T[v - sx] : t;                     // zero flux: the voxel itself (R-7)
    const float xp = i < g.nx - 1 ? T[v + sx] : t;
    const float ym = j > 0 ? T[v - sy] : t;
    const float yp = j < g.ny - 1 ? T[v + sy] : t;
    const float zm = k > 0 ? T[v - sz] : t;
    const float zp = k < g.nz - 1 ? T[v + sz] : t;
    const unsigned st = state[gid];
    const unsigned e = st & RFA_ST_INDEX;
    const float r = rfa_update(t, xm, xp, ym, yp, zm, zp, __ldg(tab + e), __ldg(tab + RFA_TABLE_N + e),
                               __ldg(tab + 2 * RFA_TABLE_N + e), g.wx, g.wy, g.wz);
    tout[gid] = r;
    if (r >= g.thr && !(st & RFA_ST_NECRO)) state[gid] = (uint8_t)(st | RFA_ST_NECRO);
}

// ------------------------------------------------------------------------------------------------
// blocked kernel: 2.5D z-sweep with S fused time steps
// ------------------------------------------------------------------------------------------------
// Work item = (scenario, z chunk, y tile, x tile); a CTA of TX*TY threads owns a BX x BY xy tile
// (BX = 4 TX, BY = RY TY) and streams it along z.  Thread (tx,ty) owns the float4 column tx and the
// RY rows ty*RY.. of every plane.  For each fused level k = 1..S it keeps the previous and the centre
// plane of level k-1 in registers (the z queue); the next plane arrives from level k-1 in the same
// iteration, level 0 being the plane just landed from HBM (cp.async ring, thread-private slots).
// x neighbours come from warp shuffles, y neighbours across threads from a double-buffered shared
// exchange of each thread's first/last row -> one __syncthreads per plane.
//
// Halos: x tiles overlap by 8 columns (4 = one float4 per side, S <= 4), y tiles and z chunks carry
// S halo rows / planes per side.  At the outer y and z faces the halo is loaded MIRRORED
// (ghost -1 = row 0, -2 = row 1, ...), which reproduces the zero-flux replicate rule exactly through
// all S levels because the update is symmetric in (ym,yp) and (zm,zp) bit for bit.  At the outer x
// faces the replicate rule is applied directly (a select on the two edge lanes).
struct RfaTbParams {
    const float *tin;
    float *tout;
    uint8_t *state;
    const float *tables;
    int nx, ny, nz, batch;
    int nx4;
    float wx, wy, wz, thr;
    int tiles_x, tiles_y, nzc, zchunk, n_items;
};

template <int S, int TX, int TY, int RY>
struct TbCfg {
    static constexpr int NT = TX * TY;
    static constexpr int BX = 4 * TX;
    static constexpr int BY = RY * TY;
    static constexpr int PD = 2;              // prefetch distance (planes in flight)
    static constexpr int DT = PD + 1;         // temperature ring depth
    static constexpr int DS = PD + S + 1;     // state ring depth (level k reads plane i-k)
    static constexpr size_t RING_T = (size_t)DT * RY * NT * 16;
    static constexpr size_t EXCH = (size_t)S * 2 * 2 * NT * 16;
    static constexpr size_t RING_S = (size_t)DS * RY * NT * 4;
    static constexpr size_t TAB = 3 * RFA_TABLE_N * 4;
    static constexpr size_t SMEM = RING_T + EXCH + RING_S + TAB;
};

template <int S, int TX, int TY, int RY>
__global__ void __launch_bounds__(TX *TY, 1) rfa_blocked_kernel(const RfaTbParams P)
{
    using C = TbCfg<S, TX, TY, RY>;
    constexpr int NT = C::NT, BX = C::BX, BY = C::BY, PD = C::PD, DT = C::DT, DS = C::DS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *ringT = reinterpret_cast<float4 *>(smem_raw);                  // [DT][RY][NT]
    float4 *exch = reinterpret_cast<float4 *>(smem_raw + C::RING_T);       // [S][2 parity][2 top/bot][NT]
    uint32_t *ringS = reinterpret_cast<uint32_t *>(smem_raw + C::RING_T + C::EXCH);   // [DS][RY][NT]
    float *tab = reinterpret_cast<float *>(smem_raw + C::RING_T + C::EXCH + C::RING_S);   // [3][128]

    const int tid = threadIdx.x;
    const int tx = tid % TX, ty = tid / TX;
    const int up_tid = (ty > 0 ? ty - 1 : ty) * TX + tx;
    const int dn_tid = (ty < TY - 1 ? ty + 1 : ty) * TX + tx;

    for (int e = tid; e < S * 2 * 2 * NT; e += NT) exch[e] = make_float4(0.f, 0.f, 0.f, 0.f);

    const size_t plane4 = (size_t)P.ny * P.nx4;       // float4 (= state words) per plane
    int cur_b = -1;

    for (int item = blockIdx.x; item < P.n_items; item += gridDim.x) {
        int t = item;
        const int txi = t % P.tiles_x;
        t /= P.tiles_x;
        const int tyi = t % P.tiles_y;
        t /= P.tiles_y;
        const int zc = t % P.nzc;
        const int b = t / P.nzc;
        const int X0 = txi * (BX - 8);
        const int Y0 = -S + tyi * (BY - 2 * S);
        const int z0 = zc * P.zchunk;
        const int z1 = min(z0 + P.zchunk, P.nz);

        const int gx4 = X0 / 4 + tx;
        const int gx4c = min(gx4, P.nx4 - 1);
        const bool xl_self = (gx4 == 0);
        const bool xr_self = (gx4 == P.nx4 - 1);
        const bool col_ok = (gx4 < P.nx4) && !(tx == 0 && X0 > 0) && !(tx == TX - 1 && X0 + BX < P.nx);
        unsigned row_ok = 0;
        size_t row_src[RY], row_dst[RY];
#pragma unroll
        for (int r = 0; r < RY; ++r) {
            const int ly = ty * RY + r;
            const int gy = Y0 + ly;
            if (ly >= S && ly < BY - S && gy >= 0 && gy < P.ny && col_ok) row_ok |= 1u << r;
            row_src[r] = (size_t)rfa_reflect(gy, P.ny) * P.nx4 + gx4c;
            row_dst[r] = (size_t)min(max(gy, 0), P.ny - 1) * P.nx4 + gx4c;
        }
        const size_t base4 = (size_t)b * P.nz * plane4;
        const float4 *tin4 = reinterpret_cast<const float4 *>(P.tin) + base4;
        float4 *tout4 = reinterpret_cast<float4 *>(P.tout) + base4;
        uint32_t *st4 = reinterpret_cast<uint32_t *>(P.state) + base4;

        __syncthreads();                                   // previous item done with tab / exchange
        if (b != cur_b) {
            for (int e = tid; e < 3 * RFA_TABLE_N; e += NT) tab[e] = P.tables[(size_t)b * 3 * RFA_TABLE_N + e];
            cur_b = b;
        }

        float4 qm[S][RY], qc[S][RY];                       // z queue: previous / centre plane per level
        unsigned nbc[S];                                   // necrosis bits travelling with qc
#pragma unroll
        for (int k = 0; k < S; ++k) {
            nbc[k] = 0;
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                qm[k][r] = make_float4(0.f, 0.f, 0.f, 0.f);
                qc[k][r] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }

        const int niter = (z1 - z0) + 2 * S;
        auto issue = [&](int j) {
            const int zs = rfa_reflect(z0 - S + j, P.nz);
            const size_t pl = (size_t)zs * plane4;
            const int sT = j % DT, sS = j % DS;
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                cp_async16(&ringT[(sT * RY + r) * NT + tid], tin4 + pl + row_src[r]);
                cp_async4(&ringS[(sS * RY + r) * NT + tid], st4 + pl + row_src[r]);
            }
        };
#pragma unroll
        for (int j = 0; j < PD; ++j) {
            if (j < niter) issue(j);
            cp_async_commit();
        }

        for (int i = 0; i < niter; ++i) {
            if (i + PD < niter) issue(i + PD);
            cp_async_commit();
            cp_async_wait<PD>();
            __syncthreads();                               // exchange rows of iteration i-1 are visible

            const int par_w = i & 1, par_r = par_w ^ 1;
            float4 in[RY];
            unsigned nb_in = 0;
            {
                const int sT = i % DT;
#pragma unroll
                for (int r = 0; r < RY; ++r) in[r] = ringT[(sT * RY + r) * NT + tid];
            }
#pragma unroll
            for (int k = 0; k < S; ++k) {
                // publish first/last row of level-k input plane (it is the centre plane next iteration)
                exch[((k * 2 + par_w) * 2 + 0) * NT + tid] = in[0];
                exch[((k * 2 + par_w) * 2 + 1) * NT + tid] = in[RY - 1];
                const float4 above = exch[((k * 2 + par_r) * 2 + 1) * NT + up_tid];
                const float4 below = exch[((k * 2 + par_r) * 2 + 0) * NT + dn_tid];
                const int sS = (i - (k + 1) + 2 * DS) % DS;          // state of plane zin-(k+1)
                float4 o[RY];
                float mx = -3.0e38f;
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    const float4 c = qc[k][r];
                    const float4 u = (r == 0) ? above : qc[k][r - 1];
                    const float4 d = (r == RY - 1) ? below : qc[k][r + 1];
                    float left = __shfl_up_sync(0xffffffffu, c.w, 1, TX);
                    float right = __shfl_down_sync(0xffffffffu, c.x, 1, TX);
                    if (xl_self) left = c.x;               // zero flux at the outer x faces (R-7)
                    if (xr_self) right = c.w;
                    const uint32_t w = ringS[(sS * RY + r) * NT + tid];
                    const unsigned e0 = w & RFA_ST_INDEX, e1 = (w >> 8) & RFA_ST_INDEX,
                                   e2 = (w >> 16) & RFA_ST_INDEX, e3 = (w >> 24) & RFA_ST_INDEX;
                    const float4 zm = qm[k][r], zp = in[r];
                    o[r].x = rfa_update(c.x, left, c.y, u.x, d.x, zm.x, zp.x, tab[e0], tab[RFA_TABLE_N + e0],
                                        tab[2 * RFA_TABLE_N + e0], P.wx, P.wy, P.wz);
                    o[r].y = rfa_update(c.y, c.x, c.z, u.y, d.y, zm.y, zp.y, tab[e1], tab[RFA_TABLE_N + e1],
                                        tab[2 * RFA_TABLE_N + e1], P.wx, P.wy, P.wz);
                    o[r].z = rfa_update(c.z, c.y, c.w, u.z, d.z, zm.z, zp.z, tab[e2], tab[RFA_TABLE_N + e2],
                                        tab[2 * RFA_TABLE_N + e2], P.wx, P.wy, P.wz);
                    o[r].w = rfa_update(c.w, c.z, right, u.w, d.w, zm.w, zp.w, tab[e3], tab[RFA_TABLE_N + e3],
                                        tab[2 * RFA_TABLE_N + e3], P.wx, P.wy, P.wz);
                    mx = fmaxf(mx, fmaxf(fmaxf(o[r].x, o[r].y), fmaxf(o[r].z, o[r].w)));
                }
                unsigned nb_o = nbc[k];
                if (mx >= P.thr) {                         // rare: some voxel of this thread reached 60 C
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        nb_o |= (o[r].x >= P.thr ? 1u : 0u) << (4 * r);
                        nb_o |= (o[r].y >= P.thr ? 2u : 0u) << (4 * r);
                        nb_o |= (o[r].z >= P.thr ? 4u : 0u) << (4 * r);
                        nb_o |= (o[r].w >= P.thr ? 8u : 0u) << (4 * r);
                    }
                }
                nbc[k] = nb_in;
                nb_in = nb_o;
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    qm[k][r] = qc[k][r];
                    qc[k][r] = in[r];
                    in[r] = o[r];
                }
            }
            // `in` is now level S of plane z0 + (i - 2S)
            if (i >= 2 * S) {
                const size_t pl = (size_t)(z0 + i - 2 * S) * plane4;
                const int sS = (i - S + 2 * DS) % DS;
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    if (row_ok & (1u << r)) {
                        tout4[pl + row_dst[r]] = in[r];
                        const unsigned bits = (nb_in >> (4 * r)) & 0xfu;
                        if (bits) {
                            const uint32_t w = ringS[(sS * RY + r) * NT + tid];
                            const uint32_t nw = w | ((bits & 1u) << 7) | ((bits & 2u) << 14) | ((bits & 4u) << 21) |
                                                ((bits & 8u) << 28);
                            if (nw != w) st4[pl + row_dst[r]] = nw;
                        }
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
static inline unsigned blocks_for(size_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }

cudaError_t rfa_launch_table(const RfaTableHost &tbl, float *dst, cudaStream_t st)
{
    rfa_table_kernel<<<1, RFA_TABLE_N, 0, st>>>(tbl, dst);
    return cudaGetLastError();
}

cudaError_t rfa_launch_init(const RfaGrid &g, const uint8_t *labels_dev, const float *theta0_by_label, float *theta,
                            uint8_t *state, cudaStream_t st)
{
    Theta0 t0;
    for (int i = 0; i < 32; ++i) t0.v[i] = theta0_by_label[i];
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    rfa_init_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, g.batch, labels_dev, t0, g.thr, theta, state);
    return cudaGetLastError();
}

cudaError_t rfa_launch_needle(const RfaGrid &g, int scenario, const uint8_t *mask_dev, int mode, float theta_value,
                              float *theta, uint8_t *state, cudaStream_t st)
{
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    rfa_needle_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, mask_dev, mode, theta_value, g.thr,
                                                             theta + (size_t)scenario * nvox,
                                                             state + (size_t)scenario * nvox);
    return cudaGetLastError();
}

cudaError_t rfa_launch_set_temperature(const RfaGrid &g, int scenario, const float *t_dev, float *theta,
                                       uint8_t *state, cudaStream_t st)
{
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    rfa_set_temperature_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, t_dev, g.t_blood, g.thr,
                                                                      theta + (size_t)scenario * nvox,
                                                                      state + (size_t)scenario * nvox);
    return cudaGetLastError();
}

cudaError_t rfa_launch_get_temperature(const RfaGrid &g, int scenario, const float *theta, float *out_dev,
                                       cudaStream_t st)
{
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    rfa_get_temperature_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, theta + (size_t)scenario * nvox,
                                                                      g.t_blood, out_dev);
    return cudaGetLastError();
}

cudaError_t rfa_launch_get_necrosis(const RfaGrid &g, int scenario, const uint8_t *state, uint8_t *out_dev,
                                    cudaStream_t st)
{
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    rfa_get_necrosis_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, state + (size_t)scenario * nvox, out_dev);
    return cudaGetLastError();
}

cudaError_t rfa_launch_count(const RfaGrid &g, int scenario, const uint8_t *state, uint32_t label_held_mask,
                             unsigned long long *counters_dev, cudaStream_t st)
{
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    cudaError_t e = cudaMemsetAsync(counters_dev, 0, 2 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    rfa_count_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, state + (size_t)scenario * nvox, label_held_mask,
                                                            counters_dev);
    return cudaGetLastError();
}

cudaError_t rfa_launch_plain(const RfaGrid &g, const float *tin, float *tout, uint8_t *state, const float *tables,
                             cudaStream_t st)
{
    size_t n = (size_t)g.nx * g.ny * g.nz * g.batch;
    rfa_plain_kernel<<<blocks_for(n, 256), 256, 0, st>>>(g, tin, tout, state, tables);
    return cudaGetLastError();
}

template <int S>
static cudaError_t launch_blocked_s(const RfaTbParams &p, int grid, cudaStream_t st)
{
    using C = TbCfg<S, RFA_TB_TX, RFA_TB_TY, RFA_TB_RY>;
    auto kern = rfa_blocked_kernel<S, RFA_TB_TX, RFA_TB_TY, RFA_TB_RY>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    kern<<<grid, C::NT, C::SMEM, st>>>(p);
    return cudaGetLastError();
}

cudaError_t rfa_launch_blocked(const RfaGrid &g, const RfaTbPlan &plan, const float *tin, float *tout,
                               uint8_t *state, const float *tables, cudaStream_t st)
{
    RfaTbParams p;
    p.tin = tin;
    p.tout = tout;
    p.state = state;
    p.tables = tables;
    p.nx = g.nx;
    p.ny = g.ny;
    p.nz = g.nz;
    p.batch = g.batch;
    p.nx4 = g.nx / 4;
    p.wx = g.wx;
    p.wy = g.wy;
    p.wz = g.wz;
    p.thr = g.thr;
    p.tiles_x = plan.tiles_x;
    p.tiles_y = plan.tiles_y;
    p.nzc = plan.nzc;
    p.zchunk = plan.zchunk;
    p.n_items = plan.n_items;
    switch (plan.fused) {
    case 1: return launch_blocked_s<1>(p, plan.grid, st);
    case 2: return launch_blocked_s<2>(p, plan.grid, st);
    case 3: return launch_blocked_s<3>(p, plan.grid, st);
    case 4: return launch_blocked_s<4>(p, plan.grid, st);
    default: return cudaErrorInvalidValue;
    }
}

template <int S>
static int resident_s()
{
    using C = TbCfg<S, RFA_TB_TX, RFA_TB_TY, RFA_TB_RY>;
    auto kern = rfa_blocked_kernel<S, RFA_TB_TX, RFA_TB_TY, RFA_TB_RY>;
    int dev = 0, sms = 0, occ = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, C::NT, C::SMEM) != cudaSuccess) return 0;
    return sms * occ;
}

int rfa_blocked_resident_ctas(int fused)
{
    switch (fused) {
    case 1: return resident_s<1>();
    case 2: return resident_s<2>();
    case 3: return resident_s<3>();
    case 4: return resident_s<4>();
    default: return 0;
    }
}
