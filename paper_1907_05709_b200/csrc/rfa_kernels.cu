// rfa_kernels.cu -- sm_100a kernels of librfa.so.
//
//   rfa_plain_kernel     one thread per voxel, one time step per launch (any grid size)
//   rfa_blocked_kernel   the hot path: 2.5D z-sweep, S fused time steps per launch
//   + small set-up / read-back kernels (init, needle, set/get temperature, necrosis, count)
//
// Every stepping kernel evaluates rfa_bracket() + rfa_advance() (rfa_device.cuh) with the same operands
// in the same order, so all variants produce bit-identical fields.
#include <algorithm>
#include <atomic>
#include <cstdio>

#include <cuda_fp16.h>

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
__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gsrc)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gsrc) : "memory");
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
        dst[RFA_TABLE_N + e] = tbl.np[e];
        dst[2 * RFA_TABLE_N + e] = tbl.qa[e];
    }
}

struct LabelInfo {
    float theta0[RFA_NLABEL];       // initial theta = t_init - T_a per label
    float k[RFA_NLABEL];            // conductivity per label: equal K <=> no interface between two labels
};

// label -> initial temperature image: theta = t_init[label] - T_a, state = label id,
// necrosis on the initial state (R-14), interface bit = some in-grid face neighbour carries a
// label with a different K (R-28).  One launch covers all scenarios.
__global__ void rfa_init_kernel(int nx, int ny, int nz, int batch, const uint8_t *__restrict__ labels, LabelInfo li,
                                float thr, float *__restrict__ theta, __half *__restrict__ resid,
                                uint8_t *__restrict__ state)
{
    // grid = (x blocks, rows, planes): no integer division per voxel
    const size_t nvox = (size_t)nx * ny * nz;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    // the per-label constants are indexed by data: from shared memory (indexed out of the parameter bank, the divergent
    // lookups were serialised and the kernel took 3.7 ms for 67 M voxels)
    __shared__ float sk[RFA_NLABEL], st0[RFA_NLABEL];
    if (threadIdx.x < RFA_NLABEL) {
        sk[threadIdx.x] = li.k[threadIdx.x];
        st0[threadIdx.x] = li.theta0[threadIdx.x];
    }
    __syncthreads();
    if (i >= nx) return;
    const size_t sy = nx, sz = (size_t)nx * ny;
    const size_t v = (size_t)k * sz + (size_t)j * sy + i;
    unsigned l = labels[v] & RFA_ST_LABEL;
    const float kc = sk[l];
    bool iface = false;
    if (i > 0) iface |= sk[labels[v - 1] & RFA_ST_LABEL] != kc;
    if (i < nx - 1) iface |= sk[labels[v + 1] & RFA_ST_LABEL] != kc;
    if (j > 0) iface |= sk[labels[v - sy] & RFA_ST_LABEL] != kc;
    if (j < ny - 1) iface |= sk[labels[v + sy] & RFA_ST_LABEL] != kc;
    if (k > 0) iface |= sk[labels[v - sz] & RFA_ST_LABEL] != kc;
    if (k < nz - 1) iface |= sk[labels[v + sz] & RFA_ST_LABEL] != kc;
    float t = st0[l];
    unsigned st = l | (iface ? RFA_ST_IFACE : 0u) | (t >= thr ? RFA_ST_NECRO : 0u);
    for (int b = 0; b < batch; ++b) {
        theta[(size_t)b * nvox + v] = t;
        resid[(size_t)b * nvox + v] = __float2half_rn(0.f);
        state[(size_t)b * nvox + v] = (uint8_t)st;
    }
}

// histogram of the label ids of the uploaded volume (range check and held share in rfa_create; on the host this walk
// over the label volume was most of rfa_create's time): 16 bytes per thread, one shared-memory histogram per block
__global__ void rfa_label_hist_kernel(size_t nvox, const uint8_t *__restrict__ labels, unsigned long long *__restrict__ hist)
{
    __shared__ unsigned h[256];
    for (int e = threadIdx.x; e < 256; e += blockDim.x) h[e] = 0u;
    __syncthreads();
    const size_t n16 = nvox / 16, stride = (size_t)gridDim.x * blockDim.x;
    const uint4 *l16 = reinterpret_cast<const uint4 *>(labels);
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < n16; v += stride) {
        const uint4 w = l16[v];
        const unsigned ws[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            atomicAdd(&h[ws[c] & 0xffu], 1u);
            atomicAdd(&h[(ws[c] >> 8) & 0xffu], 1u);
            atomicAdd(&h[(ws[c] >> 16) & 0xffu], 1u);
            atomicAdd(&h[ws[c] >> 24], 1u);
        }
    }
    if (blockIdx.x == 0)
        for (size_t v = n16 * 16 + threadIdx.x; v < nvox; v += blockDim.x) atomicAdd(&h[labels[v]], 1u);
    __syncthreads();
    for (int e = threadIdx.x; e < 256; e += blockDim.x)
        if (h[e]) atomicAdd(&hist[e], (unsigned long long)h[e]);
}

// needle placement for one scenario (R-15, R-16, R-17)
__global__ void rfa_needle_kernel(size_t nvox, const uint8_t *__restrict__ mask, int mode, float theta_value,
                                  float thr, float *__restrict__ theta, __half *__restrict__ resid,
                                  uint8_t *__restrict__ state)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvox) return;
    unsigned st = state[v] & ~(RFA_ST_DIRICHLET | RFA_ST_POWER);       // release the old needle
    if (mode != 0 && mask[v]) {
        if (mode == 1) {
            st |= RFA_ST_DIRICHLET;
            theta[v] = theta_value;
            resid[v] = __float2half_rn(0.f);
            if (theta_value >= thr) st |= RFA_ST_NECRO;
        } else {
            st |= RFA_ST_POWER;
        }
    }
    state[v] = (uint8_t)st;
}

__global__ void rfa_set_temperature_kernel(size_t nvox, const float *__restrict__ t_c, float t_blood, float thr,
                                           float *__restrict__ theta, __half *__restrict__ resid,
                                           uint8_t *__restrict__ state)
{
    size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvox) return;
    float t = __fsub_rn(t_c[v], t_blood);
    theta[v] = t;
    resid[v] = __float2half_rn(0.f);
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


// probe read-out (Fig. 6): T at n flat voxel indices of the batched volume
__global__ void rfa_probe_kernel(int n, const long long *__restrict__ index, const float *__restrict__ theta,
                                 float t_blood, float *__restrict__ out)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) out[p] = __fadd_rn(theta[index[p]], t_blood);
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
                                 const __half *__restrict__ rin, __half *__restrict__ rout,
                                 uint8_t *__restrict__ state, const float *__restrict__ tables,
                                 const float *__restrict__ kap /* null: Eq. 12; else 16x16 Kf/K_c - 1 (R-28) */)
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
    float br = rfa_bracket(t, xm, xp, ym, yp, zm, zp, __ldg(tab + RFA_TABLE_N + e),
                           __ldg(tab + 2 * RFA_TABLE_N + e), g.wx, g.wy, g.wz);
    if (kap != nullptr && (st & RFA_ST_IFACE)) {
        // labels of the six face neighbours (a missing neighbour is the voxel itself: same K, factor 0)
        const uint8_t *S = state + (size_t)b * nvox;
        const unsigned lc = (st & RFA_ST_LABEL) * RFA_NLABEL;
        const unsigned lxm = i > 0 ? S[v - sx] : st, lxp = i < g.nx - 1 ? S[v + sx] : st;
        const unsigned lym = j > 0 ? S[v - sy] : st, lyp = j < g.ny - 1 ? S[v + sy] : st;
        const unsigned lzm = k > 0 ? S[v - sz] : st, lzp = k < g.nz - 1 ? S[v + sz] : st;
        br = __fadd_rn(br, rfa_face_correction(t, xm, xp, ym, yp, zm, zp, __ldg(kap + lc + (lxm & RFA_ST_LABEL)),
                                               __ldg(kap + lc + (lxp & RFA_ST_LABEL)), __ldg(kap + lc + (lym & RFA_ST_LABEL)),
                                               __ldg(kap + lc + (lyp & RFA_ST_LABEL)), __ldg(kap + lc + (lzm & RFA_ST_LABEL)),
                                               __ldg(kap + lc + (lzp & RFA_ST_LABEL)), g.wx, g.wy, g.wz));
    }
    float r, res;
    rfa_advance(t, __half2float(rin[gid]), __ldg(tab + e), br, r, res);
    tout[gid] = r;
    rout[gid] = __float2half_rn(res);
    if (r >= g.thr && !(st & RFA_ST_NECRO)) state[gid] = (uint8_t)(st | RFA_ST_NECRO);
}

// ------------------------------------------------------------------------------------------------
// blocked kernel: 2.5D z-sweep with S fused time steps
// ------------------------------------------------------------------------------------------------
// Work item = (scenario, z chunk, y tile, x tile); a CTA of TX*TY threads owns a BX x BY xy tile
// (BX = 4 TX, BY = RY TY) and streams it along z.  Thread (tx,ty) owns the float4 column tx and the
// RY rows ty*RY.. of every plane.  For each fused level k = 0..S-1 it keeps three planes of level k in
// registers (slots rotate with the iteration number mod 3; the plane loop is unrolled three times so
// the rotation costs no register moves): the plane that arrived this iteration (z+1), the centre
// plane (z) and the previous one (z-1).  Level 0 arrives from HBM through a thread-private cp.async
// ring; level k+1 of the centre plane is produced in the same iteration and is level k+1's arrival.
// x neighbours come from warp shuffles, y neighbours across threads from a double-buffered shared
// exchange of each thread's first/last row -> one __syncthreads per plane.
//
// The arithmetic runs two voxels per instruction (add.rn.f32x2 / fma.rn.f32x2 -> FADD2 / FFMA2) in
// exactly the rounding sequence of rfa_bracket()/rfa_advance().  Three code paths per (warp, level),
// chosen by two warp votes taken before the barrier:
//   cold + one label per thread   every voxel has |theta| < RFA_COMP_MIN (residual zero by definition):
//                                 coefficients fetched once per thread, theta' = theta + fma(a, g, 0)
//   cold + mixed labels           tissue interfaces: coefficients gathered per voxel
//   hot                           near the needle: compensated add in full; residuals come from the
//                                 fp16 residual image (level 0) or from the level below through shared memory
// All give bit-identical results to the plain kernel.
//
// Halos: x tiles overlap by 8 columns (4 = one float4 per side, S <= 4), y tiles and z chunks carry
// S halo rows / planes per side.  At the outer y and z faces the halo is loaded MIRRORED
// (ghost -1 = row 0, -2 = row 1, ...), which reproduces the zero-flux replicate rule exactly through
// all S levels because the update is symmetric in (ym,yp) and (zm,zp) bit for bit.  At the outer x
// faces the replicate rule is applied directly (a select on the two edge lanes).
struct alignas(64) RfaTbParams {
    RfaTensorMap tm_theta, tm_state;  // TMA variant: tensor maps of the input image and of the state volume (box = the tile)
    const float *tin;
    float *tout;
    const __half *rin;
    __half *rout;
    uint8_t *state;
    const float *tables;
    const float *kap;                 // conservative conduction: [16][16] Kf/K_c - 1; null = Eq. 12 as printed
    int nx, ny, nz, batch;
    int nx4;
    float wx, wy, wz, thr;
    int tiles_x, tiles_y, nzc, zchunk, n_items;
    int held_copy;                    // kernel variant: warps of held voxels only copy their rows (HELDCOPY)
    int res_prefetch;                 // kernel variant: level-0 residual rows of hot planes are prefetched (RPF)
    unsigned long long *hot_ctr;      // += warp-planes that took the compensated path at level 0 (never reset)
};

constexpr int rfa_pow2_at_least(int n) { return n <= 1 ? 1 : 2 * rfa_pow2_at_least((n + 1) / 2); }

template <int S, int TX, int TY, int RY, bool CONS = false, bool TMA = false, bool RPF = false>
struct TbCfg {
    static constexpr int NT = TX * TY;
    static constexpr int BX = 4 * TX;
    static constexpr int BY = RY * TY;
#ifndef RFA_S1_PD
#define RFA_S1_PD 1
#endif
    // prefetch distance (planes in flight): the one-step kernel is bound by memory latency, not by issue slots
    // (TMA variant: two planes in flight, a ring of three slots indexed by the iteration number mod 3 = the unrolled body)
    static constexpr int PD = TMA ? 2 : (S == 1 ? RFA_S1_PD : 1);
    static constexpr int DT = TMA ? 3 : rfa_pow2_at_least(PD + 1);          // temperature ring depth
    // state ring depth: level k reads plane i-k-1; the conservative mode also reads the planes i-k and i-k-2 and
    // the rows of the neighbouring threads (one extra slot keeps a thread one barrier ahead off them)
    static constexpr int DS = rfa_pow2_at_least(CONS ? PD + S + 3 : PD + S + 1);
    static constexpr int NR = S > 1 ? S - 1 : 1;                  // inter-level residual buffers
    static constexpr size_t RING_T = (size_t)DT * RY * NT * 16;
    static constexpr size_t EXCH = (size_t)S * 2 * 2 * NT * 16;
    // TMA variant: the copy engine wants the box of the byte volume to start on a 16-byte boundary in x (a box at x = 56
    // faults), while tiles start every BX - 8 voxels: the state box starts at the boundary at or below the tile and is 16 bytes wider
    static constexpr int SROW = TMA ? TX + 4 : TX;                // state words per tile row in shared memory
    static constexpr size_t RING_S = (size_t)DS * RY * TY * SROW * 4;
    static constexpr size_t RSM = S > 1 ? (size_t)NR * 2 * RY * NT * 8 : 0;
    static constexpr size_t TAB = 3 * RFA_TABLE_N * 4;
    static constexpr size_t KAP = CONS ? RFA_NLABEL * RFA_NLABEL * 4 : 0;
    static constexpr size_t BARS = TMA ? DT * 8 : 0;              // one mbarrier per temperature slot
    // level-0 residuals of hot rows are prefetched (cp.async, 8 bytes per row) one iteration ahead into a two-slot ring
    // instead of being loaded where they are used (the 3-step TMA variants have no shared memory left for it)
    // -- a kernel variant of its own (RPF): +12..14 % where a good part of the volume is hot (C3, C4F), -3 % where next to
    // nothing is (C4: the added code is not free in a kernel that already stalls on instruction fetch); the library picks
    // the variant from the share of hot warp-planes the kernels themselves count (rfa_api.cpp: advance)
    static constexpr bool RESPF = RPF && (!TMA || S == 2);
    static constexpr size_t RESQ = RESPF ? (size_t)2 * RY * NT * 8 : 0;
    static constexpr size_t SMEM = RING_T + EXCH + RING_S + RSM + TAB + KAP + RESQ + BARS;
    static constexpr int SR = ((S + RY - 1) / RY) * RY;           // TMA variant: halo rows above the first tile (a multiple of RY)
    static_assert(!TMA || (!CONS && S >= 2 && RY == 2), "TMA variant: Eq. 12 mode, S >= 2, two rows per thread");
};

#define RFA_MAX_DEVICES 64
#include "rfa_packed.cuh"
#include "rfa_tma.cuh"

// Conservative conduction, one row of four voxels (rfa_device.cuh: rfa_face_correction; R-28): g of
// every voxel whose interface bit is set gets the face correction added.  w = the row's state word, w?? = the
// state words of its six neighbour rows aligned byte for byte, kap = [16][16] face factors in shared memory.
// Inlined on purpose: a __noinline__ version (smaller SASS) was slower on the B200 (298 vs 380 GVox/s on C4):
// the call ABI forces spills in a kernel that already sits at the 128-register cap.
__device__ __forceinline__ float4 rfa_face_row(float4 g, const float4 c, const float4 u, const float4 d, const float4 zm,
                                            const float4 zp, const float left, const float right, const uint32_t w,
                                            const uint32_t wxm, const uint32_t wxp, const uint32_t wym,
                                            const uint32_t wyp, const uint32_t wzm, const uint32_t wzp,
                                            const float *kap, const float wx, const float wy, const float wz)
{
    float gg[4] = {g.x, g.y, g.z, g.w};
    const float tc[4] = {c.x, c.y, c.z, c.w}, txm[4] = {left, c.x, c.y, c.z}, txp[4] = {c.y, c.z, c.w, right},
                tym[4] = {u.x, u.y, u.z, u.w}, typ[4] = {d.x, d.y, d.z, d.w}, tzm[4] = {zm.x, zm.y, zm.z, zm.w},
                tzp[4] = {zp.x, zp.y, zp.z, zp.w};
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        if ((w >> (8 * v)) & RFA_ST_IFACE) {
            const float *kc = kap + ((w >> (8 * v)) & RFA_ST_LABEL) * RFA_NLABEL;
            gg[v] = __fadd_rn(gg[v], rfa_face_correction(tc[v], txm[v], txp[v], tym[v], typ[v], tzm[v], tzp[v],
                                                         kc[(wxm >> (8 * v)) & RFA_ST_LABEL], kc[(wxp >> (8 * v)) & RFA_ST_LABEL],
                                                         kc[(wym >> (8 * v)) & RFA_ST_LABEL], kc[(wyp >> (8 * v)) & RFA_ST_LABEL],
                                                         kc[(wzm >> (8 * v)) & RFA_ST_LABEL], kc[(wzp >> (8 * v)) & RFA_ST_LABEL],
                                                         wx, wy, wz));
        }
    }
    return make_float4(gg[0], gg[1], gg[2], gg[3]);
}

template <int I>
struct IC {
    static constexpr int value = I;
};

template <int S, int TX, int TY, int RY, int MINB, bool CONS, bool HELDCOPY, bool TMA, bool RPF>
__global__ void __launch_bounds__(TX *TY, MINB) rfa_blocked_kernel(const __grid_constant__ RfaTbParams P)
{
    using C = TbCfg<S, TX, TY, RY, CONS, TMA, RPF>;
    constexpr int NT = C::NT, BX = C::BX, BY = C::BY, PD = C::PD, DT = C::DT, DS = C::DS;
    static_assert(RY == 4 || RY == 2, "state words of a thread are read as one vector");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4 *ringT = reinterpret_cast<float4 *>(smem_raw);                                          // [DT][RY][NT]; TMA: [DT][BY][TX]
    float4 *exch = reinterpret_cast<float4 *>(smem_raw + C::RING_T);                               // [S][2 parity][2 top/bot][NT]
    uint32_t *ringS = reinterpret_cast<uint32_t *>(smem_raw + C::RING_T + C::EXCH);                // [DS][NT][RY]; TMA: [DS][BY][TX]
    uint2 *rsm = reinterpret_cast<uint2 *>(smem_raw + C::RING_T + C::EXCH + C::RING_S);            // [NR][2 parity][RY][NT]
    float *tab = reinterpret_cast<float *>(smem_raw + C::RING_T + C::EXCH + C::RING_S + C::RSM);   // [3][128]
    float *kap = tab + 3 * RFA_TABLE_N;                                                            // [16][16] (CONS)
    uint2 *resq = reinterpret_cast<uint2 *>(smem_raw + C::SMEM - C::BARS - C::RESQ);               // [2][RY][NT] (RESPF)
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + C::SMEM - C::BARS);                   // [DT] plane landed (TMA)

    const int tid = threadIdx.x;
    const int tx = tid % TX, ty = tid / TX;
    const int up_tid = (ty > 0 ? ty - 1 : ty) * TX + tx;
    const int dn_tid = (ty < TY - 1 ? ty + 1 : ty) * TX + tx;
    // shared-memory words of this thread's rows inside one ring slot (temperature: float4 units, state: 32-bit words)
    auto t_idx = [&](const int slot, const int r) { return TMA ? (slot * BY + ty * RY + r) * TX + tx : (slot * RY + r) * NT + tid; };
    int s_off = tx;                                          // TMA: word of this thread's column inside a state row (set per item)
    auto s_idx = [&](const int slot, const int r) { return TMA ? (slot * BY + ty * RY + r) * C::SROW + s_off : (slot * NT + tid) * RY + r; };
    if constexpr (TMA) {
        if (tid == 0) {
#pragma unroll
            for (int s = 0; s < DT; ++s) mbar_init(&full[s], 1);
            mbar_fence_init();
        }
    }
    unsigned phases = 0;                                     // TMA: bit s = parity of the next completion of full[s]

    for (int e = tid; e < S * 2 * 2 * NT; e += NT) exch[e] = make_float4(0.f, 0.f, 0.f, 0.f);
    if constexpr (CONS)
        for (int e = tid; e < RFA_NLABEL * RFA_NLABEL; e += NT) kap[e] = P.kap[e];

    const unsigned plane4 = (unsigned)(P.ny * P.nx4);       // float4 (= state words = residual quads) per plane
    const float wx = P.wx, wy = P.wy, wz = P.wz;
    const u64 wx2 = pk(wx, wx), wy2 = pk(wy, wy), wz2 = pk(wz, wz), m2 = pk(-2.0f, -2.0f), zero2 = pk(0.f, 0.f);
    const float thr = P.thr;
    const float thr_filter = fmaxf(thr, 0.0f);               // max|theta'| below this: no voxel can reach thr
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
        // TMA variant: the tile starts a multiple of RY rows above the grid, so that row 0 is some thread's first row and
        // (ny being a multiple of RY) row ny-1 some thread's last one: the zero-flux rule at the outer y faces is then a
        // matter of which exchange entry a thread reads (its own row instead of the neighbour's), not of mirrored loads
        const int Y0 = (TMA ? -C::SR : -S) + tyi * (BY - 2 * S);
        const int z0 = zc * P.zchunk;
        const int z1 = min(z0 + P.zchunk, P.nz);

        const int gx4 = X0 / 4 + tx;
        const int gx4c = min(gx4, P.nx4 - 1);
        const bool xl_self = (gx4 == 0);
        const bool xr_self = (gx4 == P.nx4 - 1);
        const bool col_ok = (gx4 < P.nx4) && !(tx == 0 && X0 > 0) && !(tx == TX - 1 && X0 + BX < P.nx);
        unsigned row_ok = 0;
        unsigned row_src[RY], row_dst[RY];               // float4 offsets inside one plane
#pragma unroll
        for (int r = 0; r < RY; ++r) {
            const int ly = ty * RY + r;
            const int gy = Y0 + ly;
            if (ly >= S && ly < BY - S && gy >= 0 && gy < P.ny && col_ok) row_ok |= 1u << r;
            row_src[r] = (unsigned)(rfa_reflect(gy, P.ny) * P.nx4 + gx4c);
            row_dst[r] = (unsigned)(min(max(gy, 0), P.ny - 1) * P.nx4 + gx4c);
        }
        // exchange entries of the rows above / below this thread's rows: [0] = a thread's first row, [1] = its last row
        int up_idx = NT + up_tid, dn_idx = dn_tid;
        if constexpr (TMA) {
            s_off = tx + (X0 & 15) / 4;
            const int gyf = Y0 + ty * RY;
            if (gyf == 0) up_idx = tid;                      // outer faces: the voxel itself (R-7)
            if (gyf + RY == P.ny) dn_idx = NT + tid;
        }
        // (b * nz < 2^31 is checked by the planner: one 32 x 32 -> 64-bit multiply, cheap to recompute where the compiler
        // prefers that to keeping five 64-bit pointers alive)
        const size_t base4 = (size_t)((unsigned)b * (unsigned)P.nz) * plane4;
        const float4 *tin4 = reinterpret_cast<const float4 *>(P.tin) + base4;
        float4 *tout4 = reinterpret_cast<float4 *>(P.tout) + base4;
        const uint2 *rin2 = reinterpret_cast<const uint2 *>(P.rin) + base4;
        uint2 *rout2 = reinterpret_cast<uint2 *>(P.rout) + base4;
        uint32_t *st4 = reinterpret_cast<uint32_t *>(P.state) + base4;

        __syncthreads();                                   // previous item done with tab / exchange
        if (b != cur_b) {
            for (int e = tid; e < 3 * RFA_TABLE_N; e += NT) tab[e] = P.tables[(size_t)b * 3 * RFA_TABLE_N + e];
            cur_b = b;
        }

        // q[k][slot][r]: three planes of level k (see the header comment); per plane: nbq = necrosis bits set
        // on the way up, hotq = some voxel of this thread has |theta| >= RFA_COMP_MIN, rvq = its residual
        // sits in rsm (levels >= 1; level 0 residuals live in the HBM residual image)
        float4 q[S][3][RY];
        unsigned nbq[S][3];
        bool hotq[S][3], rvq[S][3];
        unsigned hot_planes = 0;                         // warp-planes of this item on the compensated path at level 0
        bool coldq0[3] = {true, true, true};             // level 0: no thread of the warp has a hot voxel in the plane (the vote, taken on arrival)
#pragma unroll
        for (int k = 0; k < S; ++k)
#pragma unroll
            for (int s = 0; s < 3; ++s) {
                nbq[k][s] = 0;
                hotq[k][s] = false;
                rvq[k][s] = false;
#pragma unroll
                for (int r = 0; r < RY; ++r) q[k][s][r] = make_float4(0.f, 0.f, 0.f, 0.f);
            }

        const int niter = (z1 - z0) + 2 * S;
        auto issue = [&](int j) {
            const unsigned pl = (unsigned)rfa_reflect(z0 - S + j, P.nz) * plane4;
            const int sT = j & (DT - 1), sS = j & (DS - 1);
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                cp_async16(&ringT[(sT * RY + r) * NT + tid], tin4 + (pl + row_src[r]));
                cp_async4(&ringS[(sS * NT + tid) * RY + r], st4 + (pl + row_src[r]));
            }
        };
        // TMA variant: ONE thread hands plane j of the item (tile box at (X0, Y0), z mirrored at the outer faces) to the copy
        // engine; parts of the box outside the grid arrive as zeros and are never used by a voxel that is stored
        auto issue_tma = [&](const int j, const int sT) {
            const int pz = b * P.nz + rfa_reflect(z0 - S + j, P.nz);
            mbar_expect_tx(&full[sT], (uint32_t)(BX * BY * 4 + C::SROW * 4 * BY));
            tma_load_3d(ringT + sT * BY * TX, &P.tm_theta, &full[sT], X0, Y0, pz);
            tma_load_3d(ringS + (j & (DS - 1)) * BY * C::SROW, &P.tm_state, &full[sT], X0 & ~15, Y0, pz);
        };
        if constexpr (TMA) {
            if (tid == 0) {
                issue_tma(0, 0);
                issue_tma(1, 1);                             // niter >= 2 S + 1 > 2
            }
        } else {
#pragma unroll
            for (int j = 0; j < PD; ++j) {
                if (j < niter) issue(j);
                cp_async_commit();
            }
        }

        // one plane iteration; PH = i mod 3 selects the register slots at compile time; ts = i mod 3 is the ring slot of the
        // TMA variant (= PH in the unrolled loop, a run-time value in the rotated one)
        auto body = [&](auto ph, const int i, const int ts) {
            constexpr int PH = decltype(ph)::value;
            constexpr int CE = (PH + 2) % 3;               // centre plane slot
            constexpr int MI = (PH + 1) % 3;               // previous plane slot
            if constexpr (TMA) {
                mbar_wait(&full[ts], (phases >> ts) & 1u);
                phases ^= 1u << ts;
                if constexpr (C::RESPF) cp_async_wait<0>();          // residual rows of the centre plane (issued one iteration ago)
            } else {
                if (i + PD < niter) issue(i + PD);
                cp_async_commit();
                // all but the youngest group: this iteration's plane and (RESPF) last iteration's residual rows have landed
                static_assert(PD == 1, "the residual prefetch group sits between two plane groups");
                cp_async_wait<PD>();
            }
            {
                const int sT = TMA ? ts : (i & (DT - 1));
                float m = 0.f;
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    q[0][PH][r] = ringT[t_idx(sT, r)];
                    m = max_abs4(q[0][PH][r], m);
                }
                nbq[0][PH] = 0;
                hotq[0][PH] = m >= RFA_COMP_MIN;
                // the level-0 vote of the NEXT iteration, taken now: a warp-uniform flag, so the prefetch below costs a cold warp
                // one uniform branch
                if constexpr (C::RESPF) {
                    coldq0[PH] = __all_sync(0xffffffffu, !hotq[0][PH]);
                    // this plane is the centre plane of the next iteration: fetch the residuals of its hot rows now (cp.async,
                    // 8 bytes per row), so that the hot path finds them in shared memory instead of waiting for L2 in the
                    // middle of level 0 while the warp's whole CTA waits at the barrier
                    if (!coldq0[PH] && hotq[0][PH]) {
                        const unsigned pla = (unsigned)rfa_reflect(z0 - S + i, P.nz) * plane4;
#pragma unroll
                        for (int r = 0; r < RY; ++r) cp_async8(&resq[((i & 1) * RY + r) * NT + tid], rin2 + (pla + row_src[r]));
                        // a group of its own, committed by the hot threads only: cp.async groups are per thread, and for a
                        // thread that has one it sits between two plane groups, so the wait above covers it either way
                        cp_async_commit();
                    }
                }
            }
            // state words of the S centre planes and the two warp votes per level that pick the code path:
            // thread-private data, so all of it is issued before the barrier and overlaps the wait
            uint32_t sw[S][RY];
            bool uni[S], cold[S], ifc[S];
#pragma unroll
            for (int k = 0; k < S; ++k) {
                const int sS = (i - (k + 1)) & (DS - 1);
                if constexpr (TMA) {
#pragma unroll
                    for (int r = 0; r < RY; ++r) sw[k][r] = ringS[s_idx(sS, r)];
                } else if constexpr (RY == 4) {
                    const uint4 v = *reinterpret_cast<const uint4 *>(&ringS[(sS * NT + tid) * RY]);
                    sw[k][0] = v.x; sw[k][1] = v.y; sw[k][2] = v.z; sw[k][3] = v.w;
                } else {
                    const uint2 v = *reinterpret_cast<const uint2 *>(&ringS[(sS * NT + tid) * RY]);
                    sw[k][0] = v.x; sw[k][1] = v.y;
                }
                uint32_t diff = sw[k][0] ^ __byte_perm(sw[k][0], 0, 0);
#pragma unroll
                for (int r = 1; r < RY; ++r) diff |= sw[k][0] ^ sw[k][r];
                bool one = (diff & 0x6f6f6f6fu) == 0u;                           // one label per thread
                if constexpr (CONS) {                                            // ... and no interface voxel
                    uint32_t any = sw[k][0];
#pragma unroll
                    for (int r = 1; r < RY; ++r) any |= sw[k][r];
                    ifc[k] = __any_sync(0xffffffffu, (any & 0x10101010u) != 0u); // some voxel of the warp needs face terms
                    one = one && !ifc[k];
                }
                uni[k] = __all_sync(0xffffffffu, one);
                cold[k] = (C::RESPF && k == 0) ? coldq0[CE] : __all_sync(0xffffffffu, !hotq[k][CE]);   // all residuals are zero
            }
            __syncthreads();                               // exchange rows of iteration i-1 are visible
            if constexpr (TMA) {
                // every thread has taken plane i-1 out of its slot (and is done with state plane i-6): refill them
                if (tid == 0 && i + PD < niter) issue_tma(i + PD, ts + PD >= DT ? ts + PD - DT : ts + PD);
            }
            const int par_w = i & 1, par_r = par_w ^ 1;
            float4 out[RY];
            uint2 rout[RY];
            unsigned nb_out = 0;
            bool write_res = true;
#pragma unroll
            for (int k = 0; k < S; ++k) {
                // publish first/last row of the arriving level-k plane (it is the centre plane next iteration)
                exch[((k * 2 + par_w) * 2 + 0) * NT + tid] = q[k][PH][0];
                exch[((k * 2 + par_w) * 2 + 1) * NT + tid] = q[k][PH][RY - 1];
                // rows of the neighbouring threads (centre plane): fetched only by the paths that evaluate the bracket
                float4 above, below;
                auto load_rows = [&]() {
                    above = exch[(k * 2 + par_r) * 2 * NT + up_idx];
                    below = exch[(k * 2 + par_r) * 2 * NT + dn_idx];
                };
                float mx = 0.f;                            // max |theta'| over this thread's voxels
                float4 o[RY];

                // g = rfa_bracket() of the four voxels of row r, two voxels per instruction
                auto bracket_row = [&](const int r, const u64 n01, const u64 n23, const u64 q01, const u64 q23,
                                       u64 &t01, u64 &t23, u64 &g01, u64 &g23, const bool faces) {
                    const float4 c = q[k][CE][r];
                    const float4 u = (r == 0) ? above : q[k][CE][r > 0 ? r - 1 : 0];
                    const float4 d = (r == RY - 1) ? below : q[k][CE][r < RY - 1 ? r + 1 : r];
                    float left = __shfl_up_sync(0xffffffffu, c.w, 1, TX);
                    float right = __shfl_down_sync(0xffffffffu, c.x, 1, TX);
                    if (xl_self) left = c.x;               // zero flux at the outer x faces (R-7)
                    if (xr_self) right = c.w;
                    const float4 zm = q[k][MI][r], zp = q[k][PH][r];
                    t01 = pk(c.x, c.y);
                    t23 = pk(c.z, c.w);
                    const u64 sx01 = pk(__fadd_rn(left, c.y), __fadd_rn(c.x, c.z));
                    const u64 sx23 = pk(__fadd_rn(c.y, c.w), __fadd_rn(c.z, right));
                    const u64 sy01 = add2(pk(u.x, u.y), pk(d.x, d.y)), sy23 = add2(pk(u.z, u.w), pk(d.z, d.w));
                    const u64 sz01 = add2(pk(zm.x, zm.y), pk(zp.x, zp.y)), sz23 = add2(pk(zm.z, zm.w), pk(zp.z, zp.w));
                    const u64 l01 = fma2(wz2, sz01, fma2(wy2, sy01, fma2(wx2, sx01, fma2(n01, t01, q01))));
                    const u64 l23 = fma2(wz2, sz23, fma2(wy2, sy23, fma2(wx2, sx23, fma2(n23, t23, q23))));
                    g01 = fma2(m2, t01, l01);
                    g23 = fma2(m2, t23, l23);
                    if constexpr (CONS) {
                        if (faces) {
                            // conservative conduction (R-28): labels of the six face neighbours of the row's four
                            // voxels as byte-aligned words; rfa_face_correction() where the interface bit is set
                            const uint32_t w = sw[k][r];
                            const uint32_t wl = __shfl_up_sync(0xffffffffu, w, 1, TX), wr = __shfl_down_sync(0xffffffffu, w, 1, TX);
                            const uint32_t wxm = (w << 8) | (xl_self ? (w & 0xffu) : (wl >> 24));
                            const uint32_t wxp = (w >> 8) | (xr_self ? (w & 0xff000000u) : (wr << 24));
                            const int sC = (i - (k + 1)) & (DS - 1), sM = (i - (k + 2)) & (DS - 1), sP = (i - k) & (DS - 1);
                            const uint32_t wym = (r == 0) ? ringS[(sC * NT + up_tid) * RY + RY - 1] : sw[k][r > 0 ? r - 1 : 0];
                            const uint32_t wyp = (r == RY - 1) ? ringS[(sC * NT + dn_tid) * RY] : sw[k][r < RY - 1 ? r + 1 : r];
                            const uint32_t wzm = ringS[(sM * NT + tid) * RY + r], wzp = ringS[(sP * NT + tid) * RY + r];
                            if (w & 0x10101010u) {
                                float4 gg;
                                upk(g01, gg.x, gg.y);
                                upk(g23, gg.z, gg.w);
                                gg = rfa_face_row(gg, c, u, d, zm, zp, left, right, w, wxm, wxp, wym, wyp, wzm, wzp, kap, wx, wy, wz);
                                g01 = pk(gg.x, gg.y);
                                g23 = pk(gg.z, gg.w);
                            }
                        }
                    }
                };
                // per-voxel coefficients of row r (tissue interfaces, needle voxels)
                auto gather_row = [&](const int r, u64 &a01, u64 &a23, u64 &n01, u64 &n23, u64 &q01, u64 &q23) {
                    const uint32_t w = sw[k][r];
                    const unsigned e0 = w & RFA_ST_INDEX, e1 = (w >> 8) & RFA_ST_INDEX, e2 = (w >> 16) & RFA_ST_INDEX,
                                   e3 = (w >> 24) & RFA_ST_INDEX;
                    a01 = pk(tab[e0], tab[e1]);
                    a23 = pk(tab[e2], tab[e3]);
                    n01 = pk(tab[RFA_TABLE_N + e0], tab[RFA_TABLE_N + e1]);
                    n23 = pk(tab[RFA_TABLE_N + e2], tab[RFA_TABLE_N + e3]);
                    q01 = pk(tab[2 * RFA_TABLE_N + e0], tab[2 * RFA_TABLE_N + e1]);
                    q23 = pk(tab[2 * RFA_TABLE_N + e2], tab[2 * RFA_TABLE_N + e3]);
                };

                if (cold[k]) {
                    // rfa_advance() with r = 0:  theta' = theta + fma(a, g, 0)
                    if (uni[k]) {
                        const unsigned e = sw[k][0] & RFA_ST_INDEX;
                        const float a = tab[e], nk = tab[RFA_TABLE_N + e], qa = tab[2 * RFA_TABLE_N + e];
                        const u64 a2 = pk(a, a), n2 = pk(nk, nk), q2 = pk(qa, qa);
                        if (HELDCOPY && __all_sync(0xffffffffu, a == 0.f)) {
                            // every voxel of the warp is held (a = 0: exterior, vessel, Dirichlet needle): Alg. 1's
                            // else-branch, "copy the input voxel".  theta + fma(0, g, +0) = theta + (+0)
                            // for any finite g, so the bracket need not be evaluated; bit-identical to the full path
#pragma unroll
                            for (int r = 0; r < RY; ++r) {
                                const float4 c = q[k][CE][r];
                                upk(add2(pk(c.x, c.y), zero2), o[r].x, o[r].y);
                                upk(add2(pk(c.z, c.w), zero2), o[r].z, o[r].w);
                            }
                            // the copied rows are cold (|theta| < RFA_COMP_MIN, this branch) and stay what they are: their maximum
                            // matters only to a necrosis threshold below RFA_COMP_MIN (T_a within 1 C of 60 C)
                            if (thr_filter < RFA_COMP_MIN) {
#pragma unroll
                                for (int r = 0; r < RY; ++r) mx = max_abs4(o[r], mx);
                            }
                        } else {
                            load_rows();
#pragma unroll
                            for (int r = 0; r < RY; ++r) {
                                u64 t01, t23, g01, g23;
                                bracket_row(r, n2, n2, q2, q2, t01, t23, g01, g23, false);
                                upk(add2(t01, fma2(a2, g01, zero2)), o[r].x, o[r].y);
                                upk(add2(t23, fma2(a2, g23, zero2)), o[r].z, o[r].w);
                                mx = max_abs4(o[r], mx);
                            }
                        }
                    } else {
                        load_rows();
#pragma unroll
                        for (int r = 0; r < RY; ++r) {
                            u64 a01, a23, n01, n23, q01, q23, t01, t23, g01, g23;
                            gather_row(r, a01, a23, n01, n23, q01, q23);
                            bracket_row(r, n01, n23, q01, q23, t01, t23, g01, g23, CONS && ifc[k]);
                            upk(add2(t01, fma2(a01, g01, zero2)), o[r].x, o[r].y);
                            upk(add2(t23, fma2(a23, g23, zero2)), o[r].z, o[r].w);
                            mx = max_abs4(o[r], mx);
                        }
                    }
                    if (k + 1 < S) rvq[k + 1][PH] = false;
#pragma unroll
                    for (int r = 0; r < RY; ++r)
                        if (k + 1 == S) rout[r] = make_uint2(0u, 0u);
                    // A residual is read only where |theta| >= RFA_COMP_MIN at the start of a step (rfa_advance), i.e. where
                    // the output of the step before reaches it: rows that are cold before and after the last fused step
                    // need no residual store (whatever the image holds there is never looked at)
                    if (k + 1 == S) write_res = mx >= RFA_COMP_MIN;
                } else {
                    // rfa_advance() in full, two voxels per instruction (o - t and d - bv as exact-product FMAs)
                    const u64 neg1 = pk(-1.0f, -1.0f), mg = pk(RFA_COMP_MAGIC, RFA_COMP_MAGIC), nmg = pk(-RFA_COMP_MAGIC, -RFA_COMP_MAGIC);
                    const unsigned plc = (unsigned)rfa_reflect(z0 - S + i - 1, P.nz) * plane4;   // level-0 centre plane
                    if (k == 0) ++hot_planes;
                    load_rows();
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (hotq[k][CE]) {
                            if (k == 0) ri = unpack_h4(C::RESPF ? resq[(((i & 1) ^ 1) * RY + r) * NT + tid] : __ldg(rin2 + (plc + row_src[r])));
                            else if (rvq[k][CE]) ri = unpack_h4(rsm[(((k > 0 ? k - 1 : 0) * 2 + par_r) * RY + r) * NT + tid]);
                        }
                        u64 a01, a23, n01, n23, q01, q23, t01, t23, g01, g23;
                        gather_row(r, a01, a23, n01, n23, q01, q23);
                        bracket_row(r, n01, n23, q01, q23, t01, t23, g01, g23, CONS && ifc[k]);
                        const float4 c = q[k][CE][r];
                        const bool h0 = fabsf(c.x) >= RFA_COMP_MIN, h1 = fabsf(c.y) >= RFA_COMP_MIN,
                                   h2 = fabsf(c.z) >= RFA_COMP_MIN, h3 = fabsf(c.w) >= RFA_COMP_MIN;
                        const u64 r01 = pk(h0 ? ri.x : 0.f, h1 ? ri.y : 0.f), r23 = pk(h2 ? ri.z : 0.f, h3 ? ri.w : 0.f);
                        const u64 d01 = fma2(a01, g01, r01), d23 = fma2(a23, g23, r23);
                        const u64 o01 = add2(t01, d01), o23 = add2(t23, d23);
                        const u64 bv01 = fma2(t01, neg1, o01), bv23 = fma2(t23, neg1, o23);
                        const u64 e01 = fma2(bv01, neg1, d01), e23 = fma2(bv23, neg1, d23);
                        const u64 eq01 = add2(add2(e01, mg), nmg), eq23 = add2(add2(e23, mg), nmg);
                        upk(o01, o[r].x, o[r].y);
                        upk(o23, o[r].z, o[r].w);
                        mx = max_abs4(o[r], mx);
                        float4 ro;
                        upk(eq01, ro.x, ro.y);
                        upk(eq23, ro.z, ro.w);
                        const uint2 rp = pack_h4(h0 ? ro.x : 0.f, h1 ? ro.y : 0.f, h2 ? ro.z : 0.f, h3 ? ro.w : 0.f);
                        if (k + 1 < S) rsm[((k * 2 + par_w) * RY + r) * NT + tid] = rp;
                        else rout[r] = rp;
                    }
                    if (k + 1 < S) rvq[k + 1][PH] = true;
                }
                unsigned nb_o = nbq[k][CE];
                if (mx >= thr_filter) {                    // rare: some voxel of this thread may have reached 60 C
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        nb_o |= (o[r].x >= thr ? 1u : 0u) << (4 * r);
                        nb_o |= (o[r].y >= thr ? 2u : 0u) << (4 * r);
                        nb_o |= (o[r].z >= thr ? 4u : 0u) << (4 * r);
                        nb_o |= (o[r].w >= thr ? 8u : 0u) << (4 * r);
                    }
                }
                if (k + 1 < S) {
#pragma unroll
                    for (int r = 0; r < RY; ++r) q[(k + 1) % S][PH][r] = o[r];
                    nbq[(k + 1) % S][PH] = nb_o;
                    hotq[(k + 1) % S][PH] = mx >= RFA_COMP_MIN;
                } else {
#pragma unroll
                    for (int r = 0; r < RY; ++r) out[r] = o[r];
                    nb_out = nb_o;
                }
            }
            // `out` is level S of plane z0 + (i - 2S)
            if (i >= 2 * S) {
                const unsigned pl = (unsigned)(z0 + i - 2 * S) * plane4;
                const int sS = (i - S) & (DS - 1);
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    if (row_ok & (1u << r)) {
                        tout4[pl + row_dst[r]] = out[r];
                        if (write_res) rout2[pl + row_dst[r]] = rout[r];
                        const unsigned bits = (nb_out >> (4 * r)) & 0xfu;
                        if (bits) {
                            const uint32_t w = ringS[s_idx(sS, r)];
                            const uint32_t nw = w | ((bits & 1u) << 7) | ((bits & 2u) << 14) | ((bits & 4u) << 21) |
                                                ((bits & 8u) << 28);
                            if (nw != w) st4[pl + row_dst[r]] = nw;
                        }
                    }
                }
            }
        };

        if constexpr (!CONS && !(HELDCOPY && S >= 3)) {
            for (int i = 0;;) {
                body(IC<0>{}, i, 0);
                if (++i >= niter) break;
                body(IC<1>{}, i, 1);
                if (++i >= niter) break;
                body(IC<2>{}, i, 2);
                if (++i >= niter) break;
            }
        } else {
            // The conservative variant carries the face-term code in every mixed / hot path; unrolled three times
            // it is 185 KB of SASS and stalls on instruction fetch (ncu: no_instruction 1.47 per issue, 380 GVox/s).
            // One body and an explicit rotation of the plane registers instead: a third of the code, 48 moves more
            // (446 GVox/s).  The same holds for the held-copy variant at three fused steps, whose warps run two different
            // paths side by side (copy / bracket): unrolled, no_instruction is its largest stall (1.36 per issue) and C4
            // runs 786 GVox/s, rotated 806.  Without held-copy (no_instruction 0.47) and at two fused steps the unrolled
            // body wins (C4, S = 2: 728 vs 713), so those stay unrolled.
            int ts = 0;
#pragma unroll 1
            for (int i = 0; i < niter; ++i) {
                body(IC<2>{}, i, ts);                      // arrival in slot 2, centre 1, previous 0
                ts = ts == 2 ? 0 : ts + 1;
#pragma unroll
                for (int k = 0; k < S; ++k) {
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        q[k][0][r] = q[k][1][r];
                        q[k][1][r] = q[k][2][r];
                    }
                    nbq[k][0] = nbq[k][1];
                    nbq[k][1] = nbq[k][2];
                    hotq[k][0] = hotq[k][1];
                    hotq[k][1] = hotq[k][2];
                    rvq[k][0] = rvq[k][1];
                    rvq[k][1] = rvq[k][2];
                }
                coldq0[0] = coldq0[1];
                coldq0[1] = coldq0[2];
            }
        }
        // feedback for the host's choice of the RPF variant: one atomic per warp and item, only where something was hot
        if (hot_planes != 0u && (tid & 31) == 0) atomicAdd(P.hot_ctr, (unsigned long long)hot_planes);
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

cudaError_t rfa_launch_init(const RfaGrid &g, const uint8_t *labels_dev, const float *theta0_by_label,
                            const float *k_by_label, float *theta, void *resid, uint8_t *state, cudaStream_t st)
{
    LabelInfo li;
    for (int i = 0; i < RFA_NLABEL; ++i) {
        li.theta0[i] = theta0_by_label[i];
        li.k[i] = k_by_label[i];
    }
    if (g.ny > 65535 || g.nz > 65535) return cudaErrorInvalidValue;
    const int bs = g.nx >= 256 ? 256 : (g.nx >= 128 ? 128 : 64);
    const dim3 grid((unsigned)((g.nx + bs - 1) / bs), (unsigned)g.ny, (unsigned)g.nz);
    rfa_init_kernel<<<grid, bs, 0, st>>>(g.nx, g.ny, g.nz, g.batch, labels_dev, li, g.thr, theta, (__half *)resid, state);
    return cudaGetLastError();
}

cudaError_t rfa_launch_label_hist(const RfaGrid &g, const uint8_t *labels_dev, unsigned long long *hist_dev /*256, zeroed here*/,
                                  cudaStream_t st)
{
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    cudaError_t e = cudaMemsetAsync(hist_dev, 0, 256 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const unsigned blocks = (unsigned)std::min<size_t>((nvox / 16 + 255) / 256 + 1, 148 * 8);
    rfa_label_hist_kernel<<<blocks, 256, 0, st>>>(nvox, labels_dev, hist_dev);
    return cudaGetLastError();
}

cudaError_t rfa_launch_needle(const RfaGrid &g, int scenario, const uint8_t *mask_dev, int mode, float theta_value,
                              float *theta, void *resid, uint8_t *state, cudaStream_t st)
{
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    rfa_needle_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, mask_dev, mode, theta_value, g.thr,
                                                             theta + (size_t)scenario * nvox,
                                                             (__half *)resid + (size_t)scenario * nvox,
                                                             state + (size_t)scenario * nvox);
    return cudaGetLastError();
}

cudaError_t rfa_launch_set_temperature(const RfaGrid &g, int scenario, const float *t_dev, float *theta,
                                       void *resid, uint8_t *state, cudaStream_t st)
{
    size_t nvox = (size_t)g.nx * g.ny * g.nz;
    rfa_set_temperature_kernel<<<blocks_for(nvox, 256), 256, 0, st>>>(nvox, t_dev, g.t_blood, g.thr,
                                                                      theta + (size_t)scenario * nvox,
                                                                      (__half *)resid + (size_t)scenario * nvox,
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


cudaError_t rfa_launch_probe(const RfaGrid &g, int n, const long long *index_dev, const float *theta, float *out_dev,
                             cudaStream_t st)
{
    rfa_probe_kernel<<<blocks_for((size_t)n, 128), 128, 0, st>>>(n, index_dev, theta, g.t_blood, out_dev);
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

cudaError_t rfa_launch_plain(const RfaGrid &g, const float *tin, float *tout, const void *rin, void *rout,
                             uint8_t *state, const float *tables, const float *kap, cudaStream_t st)
{
    size_t n = (size_t)g.nx * g.ny * g.nz * g.batch;
    rfa_plain_kernel<<<blocks_for(n, 256), 256, 0, st>>>(g, tin, tout, (const __half *)rin, (__half *)rout, state, tables, kap);
    return cudaGetLastError();
}

template <int S, bool CONS, int SHAPE, bool HC = false, bool TMA = false, bool RPF = false>
struct TbKernel {
    static constexpr RfaTbShape sh = RFA_TB_SHAPE[SHAPE][S];
    using C = TbCfg<S, sh.tx, sh.ty, sh.ry, CONS, TMA, RPF>;
    static auto get() { return rfa_blocked_kernel<S, sh.tx, sh.ty, sh.ry, sh.minb, CONS, HC, TMA, RPF>; }
};

// the TMA variant exists for the Eq. 12 kernels with 2 or 3 fused steps (the ones the planner picks by default), the
// residual-prefetch variant for 2 and 3 fused steps (with TMA staging: 2)
template <int S, bool CONS>
constexpr bool rfa_has_tma() { return !CONS && (S == 2 || S == 3); }
template <int S, bool TMA>
constexpr bool rfa_has_rpf() { return TMA ? S == 2 : (S == 2 || S == 3); }

template <int S, bool CONS, int SHAPE, bool HC, bool TMA, bool RPF>
static cudaError_t launch_blocked_sc(const RfaTbParams &p, int grid, cudaStream_t st)
{
    using K = TbKernel<S, CONS, SHAPE, HC, TMA, RPF>;
    auto kern = K::get();
    // the dynamic shared-memory opt-in is a per-DEVICE function attribute: remember it per device ordinal
    static std::atomic<bool> attr_set[RFA_MAX_DEVICES];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= RFA_MAX_DEVICES || !attr_set[dev].load(std::memory_order_acquire)) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::C::SMEM);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < RFA_MAX_DEVICES) attr_set[dev].store(true, std::memory_order_release);
    }
    kern<<<grid, K::C::NT, K::C::SMEM, st>>>(p);
    return cudaGetLastError();
}

template <int S, bool CONS, int SHAPE, bool TMA>
static cudaError_t launch_blocked_r(const RfaTbParams &p, int grid, cudaStream_t st)
{
    const bool hc = p.held_copy != 0;
    if constexpr (rfa_has_rpf<S, TMA>()) {
        if (p.res_prefetch) return hc ? launch_blocked_sc<S, CONS, SHAPE, true, TMA, true>(p, grid, st) : launch_blocked_sc<S, CONS, SHAPE, false, TMA, true>(p, grid, st);
    }
    return hc ? launch_blocked_sc<S, CONS, SHAPE, true, TMA, false>(p, grid, st) : launch_blocked_sc<S, CONS, SHAPE, false, TMA, false>(p, grid, st);
}

template <int S, bool CONS, int SHAPE>
static cudaError_t launch_blocked_v(const RfaTbParams &p, int tma, int grid, cudaStream_t st)
{
    if constexpr (rfa_has_tma<S, CONS>()) {
        if (tma) return launch_blocked_r<S, CONS, SHAPE, true>(p, grid, st);
    } else {
        if (tma) return cudaErrorInvalidValue;
    }
    return launch_blocked_r<S, CONS, SHAPE, false>(p, grid, st);
}

template <int S>
static cudaError_t launch_blocked_s(const RfaTbParams &p, int shape, int tma, int grid, cudaStream_t st)
{
    const bool cons = p.kap != nullptr;
    if (shape == 0) return cons ? launch_blocked_v<S, true, 0>(p, tma, grid, st) : launch_blocked_v<S, false, 0>(p, tma, grid, st);
    return cons ? launch_blocked_v<S, true, 1>(p, tma, grid, st) : launch_blocked_v<S, false, 1>(p, tma, grid, st);
}

cudaError_t rfa_launch_blocked(const RfaGrid &g, const RfaTbPlan &plan, const float *tin, float *tout,
                               const void *rin, void *rout, uint8_t *state, const float *tables, const float *kap,
                               const RfaTensorMap *map_theta_in, const RfaTensorMap *map_state, int res_prefetch,
                               unsigned long long *hot_ctr, cudaStream_t st)
{
    RfaTbParams p{};
    if (plan.tma) {
        if (!map_theta_in || !map_state || kap) return cudaErrorInvalidValue;
        p.tm_theta = *map_theta_in;
        p.tm_state = *map_state;
    }
    if (!hot_ctr) return cudaErrorInvalidValue;
    p.res_prefetch = res_prefetch;
    p.hot_ctr = hot_ctr;
    p.kap = kap;
    p.tin = tin;
    p.tout = tout;
    p.rin = (const __half *)rin;
    p.rout = (__half *)rout;
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
    p.held_copy = g.held_copy;
    switch (plan.fused) {
    case 1: return launch_blocked_s<1>(p, plan.shape, plan.tma, plan.grid, st);
    case 2: return launch_blocked_s<2>(p, plan.shape, plan.tma, plan.grid, st);
    case 3: return launch_blocked_s<3>(p, plan.shape, plan.tma, plan.grid, st);
    case 4: return launch_blocked_s<4>(p, plan.shape, plan.tma, plan.grid, st);
    default: return cudaErrorInvalidValue;
    }
}

// occupancy of the variant with the largest shared-memory footprint (residual prefetch where it exists): the plan
// must hold for either choice of RPF
template <int S, int SHAPE, bool CONS, bool TMA>
static int resident_s()
{
    using K = TbKernel<S, CONS, SHAPE, false, TMA, rfa_has_rpf<S, TMA>()>;
    auto kern = K::get();
    int dev = 0, sms = 0, occ = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    // a shape that does not fit (shared memory, registers) yields 0 resident CTAs -> no plan for this S;
    // the failed query must not stay behind as the runtime's sticky "last error"
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::C::SMEM) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, K::C::NT, K::C::SMEM) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return sms * occ;
}

template <int S>
static int resident_sc(int shape, int cons, int tma)
{
    if (tma) {
        if constexpr (rfa_has_tma<S, false>()) {
            if (cons) return 0;
            return shape == 0 ? resident_s<S, 0, false, true>() : resident_s<S, 1, false, true>();
        } else {
            return 0;
        }
    }
    if (shape == 0) return cons ? resident_s<S, 0, true, false>() : resident_s<S, 0, false, false>();
    return cons ? resident_s<S, 1, true, false>() : resident_s<S, 1, false, false>();
}

int rfa_blocked_resident_ctas(int fused, int shape, int cons, int tma)
{
    switch (fused) {
    case 1: return resident_sc<1>(shape, cons, tma);
    case 2: return resident_sc<2>(shape, cons, tma);
    case 3: return resident_sc<3>(shape, cons, tma);
    case 4: return resident_sc<4>(shape, cons, tma);
    default: return 0;
    }
}

// does a residual-prefetch variant exist for this plan?
int rfa_blocked_has_prefetch(int fused, int tma) { return tma ? fused == 2 : (fused == 2 || fused == 3); }

// tile of the blocked kernel for `fused` steps and `shape`: the box of its TMA variant's tensor maps
void rfa_blocked_tile(int fused, int shape, int *bx, int *by)
{
    // (the box of the state volume is 16 bytes wider than bx: TbCfg::SROW)
    *bx = 4 * RFA_TB_SHAPE[shape][fused].tx;
    *by = RFA_TB_SHAPE[shape][fused].ry * RFA_TB_SHAPE[shape][fused].ty;
}
