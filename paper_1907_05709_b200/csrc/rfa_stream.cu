// rfa_stream.cu -- the one-time-step-per-launch kernel of librfa.so (Alg. 2's frame loop: "one time
// iteration (N=1) of Alg. 1" per displayed frame, :330), staged by the Tensor Memory Accelerator.
//
//   rfa_stream_kernel   one CTA (8 warps) owns a 128 x (8 RY) xy tile and streams it along z.  For every plane ONE elected
//                       thread issues two bulk tensor copies (cp.async.bulk.tensor.3d -> SASS UTMALDG): the fp32 tile with
//                       its halo (136 x (8 RY + 2) floats: one float4 column and one row per side) and the tile of packed
//                       state bytes, into a ring of D shared-memory slots; completion is counted on an mbarrier per slot,
//                       and each warp hands a slot back through a second mbarrier when it has read it -> no __syncthreads
//                       in the plane loop, the warps of a CTA drift up to D - 2 planes apart and the copy engine keeps
//                       D - 2 planes in flight per CTA (the one-step kernel is bound by memory latency, not by issue slots).
//                       Thread (lane, warp) owns one float4 column (16-byte loads and stores along x) and RY rows; the
//                       planes z-1, z, z+1 of its rows sit in a register queue (slots rotate, the plane loop is unrolled
//                       three times); the rows above / below and the x neighbours of the two edge voxels come from the
//                       shared-memory tile.  Out-of-bounds parts of a box are zero-filled by the copy engine; the zero-flux
//                       rule (missing neighbour := the voxel itself, R-7) is applied by selects on the outer faces.
//
// The arithmetic is rfa_bracket() + rfa_advance() of rfa_device.cuh in the packed two-voxel form of rfa_packed.cuh, with
// the same three code paths per warp as the temporally blocked kernel (cold + one label per thread, cold + mixed labels,
// hot = compensated add in full), so the field is bit-identical to every other kernel of the library.
#include <atomic>
#include <cstdio>

#include <cuda.h>

#include "rfa_internal.h"
#include "rfa_packed.cuh"
#include "rfa_tma.cuh"

// ------------------------------------------------------------------------------------------------
// kernel
// ------------------------------------------------------------------------------------------------
struct RfaStreamParams {
    float *tout;
    const __half *rin;
    __half *rout;
    uint8_t *state;
    const float *tables;
    int nx, ny, nz, batch, nx4;
    float wx, wy, wz, thr;
    int tiles_x, tiles_y, nzc, zchunk, n_items;
    unsigned long long *work_ctr;        // dynamic work distribution: items beyond the first of each CTA are drawn from here
    unsigned long long work_base;        // value of *work_ctr at launch (the counter is never reset: n_items draws per launch)
};

template <int RY, int D>
struct StreamCfg {
    static constexpr int NW = RFA_STREAM_NW, NT = 32 * NW;
    static constexpr int BX = RFA_STREAM_BX, BY = NW * RY;
    static constexpr int ROW4 = BX / 4 + 2;                       // float4 per shared-memory row (one halo float4 per side)
    static constexpr int SLOT_T = ((ROW4 * 16 * (BY + 2)) + 127) / 128 * 128;
    static constexpr int SLOT_S = BX * BY;                        // one packed state byte per voxel, no halo
    static constexpr uint32_t TX_BYTES = ROW4 * 16 * (BY + 2) + BX * BY;
    static constexpr int QI = 4;                                  // item hand-over queue producer -> consumers
    static constexpr size_t SMEM = (size_t)D * (SLOT_T + SLOT_S) + 3 * RFA_TABLE_N * 4 + 2 * D * 8 + QI * 4 + 128;
};

// g = rfa_bracket() of the four voxels of one row, two voxels per instruction (same rounding sequence as the scalar form)
__device__ __forceinline__ void rfa_bracket_row4(const float4 c, const float4 u, const float4 d, const float4 zm, const float4 zp,
                                                 const float left, const float right, const u64 n01, const u64 n23,
                                                 const u64 q01, const u64 q23, const u64 wx2, const u64 wy2, const u64 wz2,
                                                 u64 &t01, u64 &t23, u64 &g01, u64 &g23)
{
    const u64 m2 = pk(-2.0f, -2.0f);
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
}

template <int I>
struct IC {
    static constexpr int value = I;
};

template <int RY, int D, bool HELDCOPY>
__global__ void __launch_bounds__(32 * RFA_STREAM_NW, RFA_STREAM_MINB)
    rfa_stream_kernel(const __grid_constant__ CUtensorMap tmT, const __grid_constant__ CUtensorMap tmS, const RfaStreamParams P)
{
    using C = StreamCfg<RY, D>;
    constexpr int NW = C::NW, NT = C::NT, BX = C::BX, BY = C::BY, ROW4 = C::ROW4;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *ringT = smem_raw;                                                     // [D][BY + 2][ROW4] float4
    unsigned char *ringS = smem_raw + (size_t)D * C::SLOT_T;                             // [D][BY][BX] bytes
    float *tab = reinterpret_cast<float *>(ringS + (size_t)D * C::SLOT_S);               // [3][128]
    uint64_t *full = reinterpret_cast<uint64_t *>(tab + 3 * RFA_TABLE_N);                // [D] copy landed
    uint64_t *empty = full + D;                                                          // [D] all warps are done with the slot
    int *item_q = reinterpret_cast<int *>(empty + D);                                    // [QI] the k-th item of this CTA

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < D; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], NW);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const unsigned plane4 = (unsigned)(P.ny * P.nx4);
    const float wx = P.wx, wy = P.wy, wz = P.wz;
    const u64 wx2 = pk(wx, wx), wy2 = pk(wy, wy), wz2 = pk(wz, wz), zero2 = pk(0.f, 0.f);
    const float thr = P.thr;
    const float thr_filter = fmaxf(thr, 0.0f);

    // ---- producer (thread 0): a cursor over the planes of this CTA's items, kept D - 2 planes ahead of the consumers
    // (only thread 0 runs this; an item is decoded once, when the cursor enters it, so that the per-plane cost is a few
    // integer instructions and the two copies)
    // Work items are handed out dynamically: the first item of a CTA is its block index, further ones are drawn from a
    // global counter by the producer, ONE PLANE BEFORE it finishes the current item, and passed to the consumers through
    // item_q (written before the mbarrier of that plane is armed, so every thread that has waited for the plane sees it).
    int p_item = blockIdx.x, p_k = 0, p_j = 0, p_n = 0, p_cx = 0, p_cy = 0, p_cz = 0, p_zlo = 0, p_zhi = 0, p_next = 0;
    unsigned p_cnt = 0;
    auto enter_item = [&]() {
        if (p_item >= P.n_items) return;
        int t = p_item;
        const int txi = t % P.tiles_x;
        t /= P.tiles_x;
        const int tyi = t % P.tiles_y;
        t /= P.tiles_y;
        const int zc = t % P.nzc, b = t / P.nzc;
        const int z0 = zc * P.zchunk, z1 = min(z0 + P.zchunk, P.nz);
        p_cx = txi * BX;
        p_cy = tyi * BY;
        p_zlo = b * P.nz;                                   // plane coordinates of the scenario: [p_zlo, p_zhi]
        p_zhi = p_zlo + P.nz - 1;
        p_cz = p_zlo + z0 - 1;                              // plane of p_j = 0
        p_n = (z1 - z0) + 2;
        p_j = 0;
    };
    auto produce = [&]() {
        if (p_item >= P.n_items) return;
        if (p_j == p_n - 1) {                               // last plane of the item: draw the next item first
            p_next = (int)(atomicAdd(P.work_ctr, 1ull) - P.work_base) + (int)gridDim.x;
            item_q[(p_k + 1) % C::QI] = p_next;
        }
        const int slot = (int)(p_cnt % D);
        if (p_cnt >= (unsigned)D) mbar_wait(&empty[slot], ((p_cnt / D) - 1u) & 1u);       // the slot's previous plane is released
        const int pz = min(max(p_cz + p_j, p_zlo), p_zhi);                                // z faces: the plane itself (R-7)
        mbar_expect_tx(&full[slot], C::TX_BYTES);
        tma_load_3d(ringT + (size_t)slot * C::SLOT_T, &tmT, &full[slot], p_cx - 4, p_cy - 1, pz);
        tma_load_3d(ringS + (size_t)slot * C::SLOT_S, &tmS, &full[slot], p_cx, p_cy, pz);
        ++p_cnt;
        if (++p_j == p_n) {
            p_item = p_next;
            ++p_k;
            enter_item();
        }
    };
    if (tid == 0) {
        enter_item();
#pragma unroll
        for (int n = 0; n < D - 2; ++n) produce();
    }

    unsigned c_cnt = 0;                                    // planes consumed so far (all items)
    int cur_b = -1;
    int c_k = 0;                                           // items consumed so far
    for (int item = blockIdx.x; item < P.n_items; item = item_q[(++c_k) % C::QI]) {
        int t = item;
        const int txi = t % P.tiles_x;
        t /= P.tiles_x;
        const int tyi = t % P.tiles_y;
        t /= P.tiles_y;
        const int zc = t % P.nzc, b = t / P.nzc;
        const int z0 = zc * P.zchunk, z1 = min(z0 + P.zchunk, P.nz);
        const int gx4 = txi * (BX / 4) + lane;
        const bool col_ok = gx4 < P.nx4;
        const bool xl_self = gx4 == 0, xr_self = gx4 == P.nx4 - 1;
        const int gy0 = tyi * BY + warp * RY;              // first row of this warp
        const int r_last = P.ny - 1 - gy0;                 // row of this warp on the outer y face (>= RY: none of them)
        unsigned row_ok = 0;
#pragma unroll
        for (int r = 0; r < RY; ++r)
            if (gy0 + r < P.ny && col_ok) row_ok |= 1u << r;
        const unsigned row0 = (unsigned)(min(gy0, P.ny - 1) * P.nx4 + min(gx4, P.nx4 - 1));   // float4 offset of row 0 inside a plane
        const size_t base4 = (size_t)b * P.nz * plane4;
        float4 *tout4 = reinterpret_cast<float4 *>(P.tout) + base4;
        const uint2 *rin2 = reinterpret_cast<const uint2 *>(P.rin) + base4;
        uint2 *rout2 = reinterpret_cast<uint2 *>(P.rout) + base4;
        uint32_t *st4 = reinterpret_cast<uint32_t *>(P.state) + base4;

        if (b != cur_b) {                                  // per-scenario coefficient table (changes only in batched runs)
            __syncthreads();
            for (int e = tid; e < 3 * RFA_TABLE_N; e += NT) tab[e] = P.tables[(size_t)b * 3 * RFA_TABLE_N + e];
            __syncthreads();
            cur_b = b;
        }

        float4 q[3][RY];                                   // planes z-1, z, z+1 of this thread's rows (slots rotate)
        bool hotq[3] = {false, false, false};
#pragma unroll
        for (int s = 0; s < 3; ++s)
#pragma unroll
            for (int r = 0; r < RY; ++r) q[s][r] = make_float4(0.f, 0.f, 0.f, 0.f);

        const int niter = (z1 - z0) + 2;
        auto body = [&](auto ph, const int i) {
            constexpr int PH = decltype(ph)::value;        // arrival slot
            constexpr int CE = (PH + 2) % 3;               // centre plane
            constexpr int MI = (PH + 1) % 3;               // previous plane
            if (tid == 0) produce();
            const int slot = (int)(c_cnt % D);
            mbar_wait(&full[slot], (c_cnt / D) & 1u);
            {
                const float4 *rowp = reinterpret_cast<const float4 *>(ringT + (size_t)slot * C::SLOT_T) + (warp * RY + 1) * ROW4 + lane + 1;
                float m = 0.f;
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    q[PH][r] = rowp[r * ROW4];
                    m = max_abs4(q[PH][r], m);
                }
                hotq[PH] = m >= RFA_COMP_MIN;
                if (RY > 1 && r_last < RY - 1) {
                    // warp cut by the outer y face: its rows beyond the grid (zero-filled by the copy engine, never stored)
                    // take the last row's values, so that row r_last finds itself below (zero flux, R-7)
#pragma unroll
                    for (int r = 1; r < RY; ++r)
                        if (r > r_last) q[PH][r] = q[PH][r - 1];
                }
            }
            if (i >= 2) {
                // centre plane = plane z0 + i - 2, arrived one iteration ago
                const int slot_c = (int)((c_cnt - 1u) % D);
                const unsigned char *tileT = ringT + (size_t)slot_c * C::SLOT_T;
                const float4 *t4 = reinterpret_cast<const float4 *>(tileT);
                const float *t1 = reinterpret_cast<const float *>(tileT);
                const uint32_t *s4 = reinterpret_cast<const uint32_t *>(ringS + (size_t)slot_c * C::SLOT_S);
                uint32_t sw[RY];
#pragma unroll
                for (int r = 0; r < RY; ++r) sw[r] = s4[(warp * RY + r) * (BX / 4) + lane];
                uint32_t diff = sw[0] ^ __byte_perm(sw[0], 0, 0);
#pragma unroll
                for (int r = 1; r < RY; ++r) diff |= sw[0] ^ sw[r];
                const bool uni = __all_sync(0xffffffffu, (diff & 0x6f6f6f6fu) == 0u);      // one label per thread
                const bool cold = __all_sync(0xffffffffu, !hotq[CE]);                      // all residuals are zero
                // rows above / below this warp's rows and the x neighbours of the edge voxels, from the tile
                // (outer y faces: the voxel itself, R-7 -- warp-uniform, so these are two branches per plane, not selects per row)
                float4 above = q[CE][0], below = q[CE][RY - 1];
                if (gy0 != 0) above = t4[(warp * RY) * ROW4 + lane + 1];
                if (r_last > RY - 1) below = t4[(warp * RY + RY + 1) * ROW4 + lane + 1];
                float4 o[RY];
                uint2 ro[RY];
                float mx = 0.f;
                bool write_res = true;
                auto neighbours = [&](const int r, float4 &u, float4 &d, float &left, float &right) {
                    const float4 c = q[CE][r];
                    u = (r == 0) ? above : q[CE][r > 0 ? r - 1 : 0];
                    d = (r == RY - 1) ? below : q[CE][r < RY - 1 ? r + 1 : r];
                    const float *rowf = t1 + (warp * RY + r + 1) * (ROW4 * 4) + 4 * lane;
                    left = xl_self ? c.x : rowf[3];                            // ... and at the outer x faces
                    right = xr_self ? c.w : rowf[8];
                };
                auto gather_row = [&](const int r, u64 &a01, u64 &a23, u64 &n01, u64 &n23, u64 &q01, u64 &q23) {
                    const uint32_t w = sw[r];
                    const unsigned e0 = w & RFA_ST_INDEX, e1 = (w >> 8) & RFA_ST_INDEX, e2 = (w >> 16) & RFA_ST_INDEX,
                                   e3 = (w >> 24) & RFA_ST_INDEX;
                    a01 = pk(tab[e0], tab[e1]);
                    a23 = pk(tab[e2], tab[e3]);
                    n01 = pk(tab[RFA_TABLE_N + e0], tab[RFA_TABLE_N + e1]);
                    n23 = pk(tab[RFA_TABLE_N + e2], tab[RFA_TABLE_N + e3]);
                    q01 = pk(tab[2 * RFA_TABLE_N + e0], tab[2 * RFA_TABLE_N + e1]);
                    q23 = pk(tab[2 * RFA_TABLE_N + e2], tab[2 * RFA_TABLE_N + e3]);
                };
                if (cold) {
                    // rfa_advance() with r = 0:  theta' = theta + fma(a, g, 0)
                    if (uni) {
                        const unsigned e = sw[0] & RFA_ST_INDEX;
                        const float a = tab[e], nk = tab[RFA_TABLE_N + e], qa = tab[2 * RFA_TABLE_N + e];
                        const u64 a2 = pk(a, a), n2 = pk(nk, nk), q2 = pk(qa, qa);
                        if (HELDCOPY && __all_sync(0xffffffffu, a == 0.f)) {
                            // every voxel of the warp is held: Alg. 1's else-branch, "copy the input voxel";
                            // theta + fma(0, g, +0) = theta + (+0) for any finite g: bit-identical to the full path
#pragma unroll
                            for (int r = 0; r < RY; ++r) {
                                const float4 c = q[CE][r];
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
#pragma unroll
                            for (int r = 0; r < RY; ++r) {
                                float4 u, d;
                                float left, right;
                                neighbours(r, u, d, left, right);
                                u64 t01, t23, g01, g23;
                                rfa_bracket_row4(q[CE][r], u, d, q[MI][r], q[PH][r], left, right, n2, n2, q2, q2, wx2, wy2, wz2, t01, t23, g01, g23);
                                upk(add2(t01, fma2(a2, g01, zero2)), o[r].x, o[r].y);
                                upk(add2(t23, fma2(a2, g23, zero2)), o[r].z, o[r].w);
                                mx = max_abs4(o[r], mx);
                            }
                        }
                    } else {
#pragma unroll
                        for (int r = 0; r < RY; ++r) {
                            float4 u, d;
                            float left, right;
                            neighbours(r, u, d, left, right);
                            u64 a01, a23, n01, n23, q01, q23, t01, t23, g01, g23;
                            gather_row(r, a01, a23, n01, n23, q01, q23);
                            rfa_bracket_row4(q[CE][r], u, d, q[MI][r], q[PH][r], left, right, n01, n23, q01, q23, wx2, wy2, wz2, t01, t23, g01, g23);
                            upk(add2(t01, fma2(a01, g01, zero2)), o[r].x, o[r].y);
                            upk(add2(t23, fma2(a23, g23, zero2)), o[r].z, o[r].w);
                            mx = max_abs4(o[r], mx);
                        }
                    }
#pragma unroll
                    for (int r = 0; r < RY; ++r) ro[r] = make_uint2(0u, 0u);
                    // A residual is read only where |theta| >= RFA_COMP_MIN at the START of a step (rfa_advance), i.e. where
                    // this step's OUTPUT reaches it.  Rows that are cold before and after the step therefore need no
                    // residual store at all: whatever the image holds there is never looked at (2 of the 11 bytes per voxel).
                    write_res = mx >= RFA_COMP_MIN;
                } else {
                    // rfa_advance() in full, two voxels per instruction (o - t and d - bv as exact-product FMAs)
                    const u64 neg1 = pk(-1.0f, -1.0f), mg = pk(RFA_COMP_MAGIC, RFA_COMP_MAGIC), nmg = pk(-RFA_COMP_MAGIC, -RFA_COMP_MAGIC);
                    const unsigned plc = (unsigned)(z0 + i - 2) * plane4;
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (hotq[CE] && (row_ok & (1u << r))) ri = unpack_h4(__ldg(rin2 + (plc + row0 + r * P.nx4)));
                        float4 u, d;
                        float left, right;
                        neighbours(r, u, d, left, right);
                        u64 a01, a23, n01, n23, q01, q23, t01, t23, g01, g23;
                        gather_row(r, a01, a23, n01, n23, q01, q23);
                        rfa_bracket_row4(q[CE][r], u, d, q[MI][r], q[PH][r], left, right, n01, n23, q01, q23, wx2, wy2, wz2, t01, t23, g01, g23);
                        const float4 c = q[CE][r];
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
                        float4 rq;
                        upk(eq01, rq.x, rq.y);
                        upk(eq23, rq.z, rq.w);
                        ro[r] = pack_h4(h0 ? rq.x : 0.f, h1 ? rq.y : 0.f, h2 ? rq.z : 0.f, h3 ? rq.w : 0.f);
                    }
                }
                // sticky necrosis, and the stores: only voxels of the grid
                const unsigned pl = (unsigned)(z0 + i - 2) * plane4;
                const bool any_thr = mx >= thr_filter;    // rare: some voxel of this thread may have reached 60 C
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    if (row_ok & (1u << r)) {
                        const unsigned off = pl + row0 + r * P.nx4;
                        tout4[off] = o[r];
                        if (write_res) rout2[off] = ro[r];
                        if (any_thr) {
                            const uint32_t w = sw[r];
                            const uint32_t nw = w | (o[r].x >= thr ? 0x80u : 0u) | (o[r].y >= thr ? 0x8000u : 0u) |
                                                (o[r].z >= thr ? 0x800000u : 0u) | (o[r].w >= thr ? 0x80000000u : 0u);
                            if (nw != w) st4[off] = nw;
                        }
                    }
                }
            }
            // the slot of the previous plane is not read any more (its own rows went to registers on arrival)
            if (i >= 1) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[(c_cnt - 1u) % D]);
            }
            ++c_cnt;
        };
        for (int i = 0;;) {
            body(IC<0>{}, i);
            if (++i >= niter) break;
            body(IC<1>{}, i);
            if (++i >= niter) break;
            body(IC<2>{}, i);
            if (++i >= niter) break;
        }
        // the last plane of the item was only ever a z neighbour: release its slot too
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[(c_cnt - 1u) % D]);
    }
}

// ------------------------------------------------------------------------------------------------
// host side: tensor maps, occupancy, launch
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static std::atomic<EncodeTiledFn> cached{nullptr};
    EncodeTiledFn f = cached.load(std::memory_order_acquire);
    if (f) return f;
    void *p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess || !p) {
        cudaGetLastError();
        return nullptr;
    }
    f = (EncodeTiledFn)p;
    cached.store(f, std::memory_order_release);
    return f;
}

using SCfg = StreamCfg<RFA_STREAM_RY, RFA_STREAM_D>;
static_assert(sizeof(RfaTensorMap) == sizeof(CUtensorMap), "RfaTensorMap must hold a CUtensorMap");
static_assert(SCfg::BY == RFA_STREAM_BY, "tile height");

// tensor map of one fp32 image (elem_bytes 4) or of the packed state volume (elem_bytes 1), seen as (nx, ny, nz * batch),
// with a box of box_x x box_y x 1 elements
bool rfa_make_tile_map(const RfaGrid &g, const void *base, int elem_bytes, int box_x, int box_y, RfaTensorMap *out)
{
    EncodeTiledFn enc = encode_fn();
    if (!enc || !out || !base) return false;
    if ((g.nx % 16) != 0) return false;                     // row pitch of the byte volume must be a multiple of 16 bytes
    if ((long long)g.nz * g.batch > 0x7fffffffLL) return false;
    if (box_x < 1 || box_x > 256 || box_y < 1 || box_y > 256 || (box_x * elem_bytes) % 16 != 0) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz * g.batch};
    const cuuint32_t estr[3] = {1, 1, 1};
    const cuuint64_t str[2] = {(cuuint64_t)g.nx * elem_bytes, (cuuint64_t)g.nx * g.ny * elem_bytes};
    const cuuint32_t box[3] = {(cuuint32_t)box_x, (cuuint32_t)box_y, 1};
    return enc(reinterpret_cast<CUtensorMap *>(out), elem_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 3,
               const_cast<void *>(base), dims, str, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// the two maps of the one-step kernel: the fp32 tile with its halo, the state tile without
bool rfa_stream_make_maps(const RfaGrid &g, const float *theta, const uint8_t *state, RfaTensorMap *map_theta, RfaTensorMap *map_state)
{
    if (map_theta && !rfa_make_tile_map(g, theta, 4, SCfg::ROW4 * 4, SCfg::BY + 2, map_theta)) return false;
    if (map_state && !rfa_make_tile_map(g, state, 1, SCfg::BX, SCfg::BY, map_state)) return false;
    return true;
}

template <bool HC>
static cudaError_t stream_attr()
{
    static std::atomic<bool> attr_set[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !attr_set[dev].load(std::memory_order_acquire)) {
        e = cudaFuncSetAttribute(rfa_stream_kernel<RFA_STREAM_RY, RFA_STREAM_D, HC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SCfg::SMEM);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_set[dev].store(true, std::memory_order_release);
    }
    return cudaSuccess;
}

int rfa_stream_resident_ctas()
{
    int dev = 0, sms = 0, occ = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    if (stream_attr<false>() != cudaSuccess || stream_attr<true>() != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, rfa_stream_kernel<RFA_STREAM_RY, RFA_STREAM_D, true>, SCfg::NT, SCfg::SMEM) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return sms * occ;
}

cudaError_t rfa_launch_stream(const RfaGrid &g, const RfaTbPlan &plan, const RfaTensorMap &map_theta_in, const RfaTensorMap &map_state,
                              float *tout, const void *rin, void *rout, uint8_t *state, const float *tables,
                              unsigned long long *work_ctr, unsigned long long work_base, cudaStream_t st)
{
    RfaStreamParams p;
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
    p.work_ctr = work_ctr;
    p.work_base = work_base;
    const CUtensorMap &mt = reinterpret_cast<const CUtensorMap &>(map_theta_in), &ms = reinterpret_cast<const CUtensorMap &>(map_state);
    cudaError_t e = g.held_copy ? stream_attr<true>() : stream_attr<false>();
    if (e != cudaSuccess) return e;
    if (g.held_copy)
        rfa_stream_kernel<RFA_STREAM_RY, RFA_STREAM_D, true><<<plan.grid, SCfg::NT, SCfg::SMEM, st>>>(mt, ms, p);
    else
        rfa_stream_kernel<RFA_STREAM_RY, RFA_STREAM_D, false><<<plan.grid, SCfg::NT, SCfg::SMEM, st>>>(mt, ms, p);
    return cudaGetLastError();
}
