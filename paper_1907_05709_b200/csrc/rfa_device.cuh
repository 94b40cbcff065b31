// rfa_device.cuh -- the one per-voxel arithmetic every kernel of librfa.so shares, and the packed
// per-voxel state byte.  (Product code; the fp64 oracle under oracle/ shares nothing with this.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

// ---- packed state byte (one per voxel per scenario) ---------------------------------------------
//   bits 0..3  label id (<= 16 tissues, "voxel-wise" parameters)
//   bit  4     interface: some face neighbour carries a label with a different conductivity K (static,
//              set by rfa_init_kernel; only the conservative conduction mode looks at it, R-28)
//   bit  5     needle voxel, Dirichlet: held at its temperature (Alg. 1 :306)
//   bit  6     needle voxel, constant power source (R-17)
//   bit  7     necrotic: T reached 60 C at some step (sticky)
// bits 0..6 index the per-scenario coefficient table (128 entries; the interface bit does not change
// the coefficients).
#define RFA_ST_LABEL 0x0fu
#define RFA_ST_IFACE 0x10u
#define RFA_ST_DIRICHLET 0x20u
#define RFA_ST_POWER 0x40u
#define RFA_ST_NECRO 0x80u
#define RFA_ST_INDEX 0x7fu
#define RFA_TABLE_N 128
#define RFA_NLABEL 16

// Per-scenario coefficient table, three planes of RFA_TABLE_N floats each (fp64 on the host,
// rounded once):
//   a[e]   = dt K /(rho c_p) * W          W = 1/dx^2 + 1/dy^2 + 1/dz^2 (metres)      (0 for held entries)
//   np[e]  = -w_b c_b /(K W)              (0 for held entries)
//   qa[e]  = (Q_m + Q_power) / (K W)      (0 for held entries)
// and three global weights wx = (1/dx^2)/W, wy, wz, rounded to multiples of 2^-24 such that their
// fp32 values sum to exactly 1 (otherwise the cancellation
// wx sx + wy sy + wz sz - 2 theta leaves a systematic source ~ 1e-7 * 2 theta per step).
struct RfaTableHost {
    float a[RFA_TABLE_N];
    float np[RFA_TABLE_N];
    float qa[RFA_TABLE_N];
};

// One time step of one voxel.  theta = T - T_a.  Eq. 12 rearranged as
//   theta' = theta + a * g,    g = wx (xm+xp) + wy (ym+yp) + wz (zm+zp) - 2 theta + qa + np theta
// The "-2 theta" is applied with the exact constant 2 and the perfusion term separately, so no
// rounded coefficient multiplies the large cancelling terms.  Explicit intrinsics fix the rounding
// sequence, so every kernel variant is bit-identical (the blocked kernel evaluates the same sequence
// two voxels at a time with add.rn.f32x2 / fma.rn.f32x2).
__device__ __forceinline__ float rfa_bracket(float t, float xm, float xp, float ym, float yp, float zm, float zp,
                                             float np, float qa, float wx, float wy, float wz)
{
    const float sx = __fadd_rn(xm, xp);
    const float sy = __fadd_rn(ym, yp);
    const float sz = __fadd_rn(zm, zp);
    const float u = __fmaf_rn(np, t, qa);
    const float l = __fmaf_rn(wz, sz, __fmaf_rn(wy, sy, __fmaf_rn(wx, sx, u)));
    return __fmaf_rn(-2.0f, t, l);
}

// Conservative conduction (row f1, R-28): div(K grad T) of Eq. 9 with harmonic-mean
// face conductivities Kf = 2 K_c K_n / (K_c + K_n).  Written as a correction to the bracket of Eq. 12,
//   g_cons = g + sum_axis w_axis [ (Kf-/K_c - 1)(t- - t) + (Kf+/K_c - 1)(t+ - t) ],
// so that voxels whose six neighbours share their K (interface bit clear: almost all) run the unchanged
// sequence.  k?? = Kf/K_c - 1 from the 16x16 label-pair table (fp64 on the host, rounded once; exactly 0
// for equal K).  Applied if and only if the voxel's interface bit is set.
__device__ __forceinline__ float rfa_face_correction(float t, float xm, float xp, float ym, float yp, float zm,
                                                     float zp, float kxm, float kxp, float kym, float kyp,
                                                     float kzm, float kzp, float wx, float wy, float wz)
{
    // both products are rounded before they are added: the result is bit-symmetric under swapping the two sides of
    // an axis, like rfa_bracket, which is what lets the blocked kernel load mirrored y/z halos at the outer faces
    const float cx = __fadd_rn(__fmul_rn(kxm, __fsub_rn(xm, t)), __fmul_rn(kxp, __fsub_rn(xp, t)));
    const float cy = __fadd_rn(__fmul_rn(kym, __fsub_rn(ym, t)), __fmul_rn(kyp, __fsub_rn(yp, t)));
    const float cz = __fadd_rn(__fmul_rn(kzm, __fsub_rn(zm, t)), __fmul_rn(kzp, __fsub_rn(zp, t)));
    return __fmaf_rn(wz, cz, __fmaf_rn(wy, cy, __fmul_rn(wx, cx)));
}

// Compensated accumulation theta' = theta + a g.  With dt far below the
// stability bound the increment a*g of a slowly converging hot voxel is a fraction of ulp(theta); a
// plain round-to-nearest add drops it every step and the field stalls short of the oracle (measured:
// 1.8e-3 C on config 3 after 24000 steps).  So wherever |theta| >= RFA_COMP_MIN the rounding error of
// the add is carried to the next step as a residual r (Fast2Sum), quantised to multiples of 2^-24 C
// (exactly representable in the fp16 residual image for |theta| < 2048), which makes the stored pair
// (theta, r) a temperature with uniform 6e-8 C resolution.  Colder voxels carry r = 0: there fp32
// already resolves 1.2e-7 C or better.  A held voxel (a = 0, r = 0) returns theta bit-exactly (Eq. 13, Alg. 1 :313).
#define RFA_COMP_MIN 1.0f
#define RFA_COMP_MAGIC 0.75f      /* ulp(0.75) = 2^-24 */
__device__ __forceinline__ void rfa_advance(float t, float r_in, float a, float g, float &t_out, float &r_out)
{
    const bool hot = fabsf(t) >= RFA_COMP_MIN;
    const float r = hot ? r_in : 0.0f;
    const float d = __fmaf_rn(a, g, r);                 // increment + carried residual (small magnitudes)
    const float o = __fadd_rn(t, d);
    const float bv = __fsub_rn(o, t);                   // the part of d that made it into o (exact)
    const float e = __fsub_rn(d, bv);                   // what was rounded away
    const float eq = __fsub_rn(__fadd_rn(e, RFA_COMP_MAGIC), RFA_COMP_MAGIC);
    t_out = o;
    r_out = hot ? eq : 0.0f;
}

__device__ __forceinline__ int rfa_reflect(int j, int n)
{
    // mirror about the outer faces (ghost -1 -> 0, -2 -> 1, n -> n-1 ...), then clamp
    if (j < 0) j = -1 - j;
    if (j >= n) j = 2 * n - 1 - j;
    return min(max(j, 0), n - 1);
}
