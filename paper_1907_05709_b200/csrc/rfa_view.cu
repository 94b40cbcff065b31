// rfa_view.cu -- the two consumers of the temperature image in librfa.so (rows f3 / f4 of SURVEY.md 8(f)):
//
//   rfa_warp_kernel     breathing-motion warp, Eq. 14: out[v] = T(x_v + scale * u[v]), trilinear, clamped
//   rfa_render_kernel   headless view of the heat zone (Figs. 11-12): orthographic ray-march, one thread per pixel
//
// Both read the current image only.  Neither uses a graphics API.
#include "rfa_internal.h"

// ------------------------------------------------------------------------------------------------
// Eq. 14 warp
// ------------------------------------------------------------------------------------------------
// One axis of the sample position: the displacement d (in voxels) is clamped so that base + d stays inside [0, n-1]
// (bounds exact in fp32: small integers), then split into cell index and weight.  d keeps its own fp32 resolution: it
// is never added to the coordinate in floating point, so the interpolation weights carry the resolution of the (small)
// displacement, not of the coordinate.
__device__ __forceinline__ void rfa_warp_axis(int base, int n, float d, int &i0, int &step1, float &a)
{
    const float dc = fminf(fmaxf(d, -(float)base), (float)(n - 1 - base));
    const float f = floorf(dc);
    a = dc - f;
    i0 = base + (int)f;
    step1 = i0 < n - 1 ? 1 : 0;                    // i1 = min(i0 + 1, n - 1)
}

// Lanes own CONSECUTIVE voxels of a row (a warp-wide gather then touches one or two 128-byte lines; with four voxels per
// lane along x it touched four to five, and the L1 tag stage was the limiter: ncu l1tex 82 % busy at 198 GVoxel/s), each
// thread walks RFA_WARP_ROWS rows of the plane with everything unrolled (loads of all rows in flight), indices are 32-bit
// offsets from the scenario's image, and the block index gives (row block, plane): no integer division anywhere.
#define RFA_WARP_BX 128
#define RFA_WARP_BY 2
#define RFA_WARP_ROWS 4
__global__ void __launch_bounds__(RFA_WARP_BX *RFA_WARP_BY)
    rfa_warp_kernel(int nx, int ny, int nz, const float *__restrict__ theta, const float *__restrict__ disp, float sx, float sy,
                    float sz, float t_blood, float *__restrict__ out)
{
    const int i = blockIdx.x * RFA_WARP_BX + threadIdx.x;
    const int jb = (blockIdx.y * RFA_WARP_BY + threadIdx.y) * RFA_WARP_ROWS, k = blockIdx.z;
    if (i >= nx) return;
    const unsigned pitch = (unsigned)nx, plane = (unsigned)nx * (unsigned)ny;
    const size_t nvox = (size_t)plane * nz;
    const unsigned v0 = (unsigned)k * plane + (unsigned)jb * pitch + (unsigned)i;
    float ux[RFA_WARP_ROWS], uy[RFA_WARP_ROWS], uz[RFA_WARP_ROWS];
#pragma unroll
    for (int r = 0; r < RFA_WARP_ROWS; ++r) {
        const bool ok = jb + r < ny;
        const unsigned v = v0 + r * pitch;
        ux[r] = ok ? __ldcs(disp + v) : 0.f;       // streamed once: do not displace the image lines in L1 / L2
        uy[r] = ok ? __ldcs(disp + nvox + v) : 0.f;
        uz[r] = ok ? __ldcs(disp + 2 * nvox + v) : 0.f;
    }
#pragma unroll
    for (int r = 0; r < RFA_WARP_ROWS; ++r) {
        const int j = min(jb + r, ny - 1);
        int i0, j0, k0, di, dj, dk;
        float ax, ay, az;
        rfa_warp_axis(i, nx, ux[r] * sx, i0, di, ax);
        rfa_warp_axis(j, ny, uy[r] * sy, j0, dj, ay);
        rfa_warp_axis(k, nz, uz[r] * sz, k0, dk, az);
        // all eight offsets are formed in 32 bits and added to the image pointer once each (one IMAD.WIDE per load)
        const unsigned o000 = (unsigned)k0 * plane + (unsigned)j0 * pitch + (unsigned)i0, o100 = o000 + (unsigned)di;
        const unsigned o010 = o000 + (dj ? pitch : 0u), o110 = o010 + (unsigned)di;
        const unsigned o001 = o000 + (dk ? plane : 0u), o101 = o001 + (unsigned)di;
        const unsigned o011 = o001 + (dj ? pitch : 0u), o111 = o011 + (unsigned)di;
        const float c000 = __ldg(&theta[o000]), c100 = __ldg(&theta[o100]), c010 = __ldg(&theta[o010]), c110 = __ldg(&theta[o110]);
        const float c001 = __ldg(&theta[o001]), c101 = __ldg(&theta[o101]), c011 = __ldg(&theta[o011]), c111 = __ldg(&theta[o111]);
        const float x00 = fmaf(ax, c100 - c000, c000), x10 = fmaf(ax, c110 - c010, c010);
        const float x01 = fmaf(ax, c101 - c001, c001), x11 = fmaf(ax, c111 - c011, c011);
        const float y0 = fmaf(ay, x10 - x00, x00), y1 = fmaf(ay, x11 - x01, x01);
        const float t = fmaf(az, y1 - y0, y0) + t_blood;
        if (jb + r < ny) __stcs(out + v0 + r * pitch, t);
    }
}

cudaError_t rfa_launch_warp(const RfaGrid &g, int scenario, const float *theta, const float *disp_dev, float scale,
                            const float inv_h_mm[3], float *out_dev, cudaStream_t st)
{
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    if (nvox >= 0xffffffffull) return cudaErrorInvalidValue;       // 32-bit voxel offsets inside one scenario
    const float *th = theta + (size_t)scenario * nvox;
    const unsigned gy = (unsigned)((g.ny + RFA_WARP_BY * RFA_WARP_ROWS - 1) / (RFA_WARP_BY * RFA_WARP_ROWS));
    if (gy > 65535u || g.nz > 65535) return cudaErrorInvalidValue;
    const dim3 block(RFA_WARP_BX, RFA_WARP_BY, 1);
    const dim3 grid((unsigned)((g.nx + RFA_WARP_BX - 1) / RFA_WARP_BX), gy, (unsigned)g.nz);
    // mm -> voxels, scaled by the breathing amplitude of the phase
    rfa_warp_kernel<<<grid, block, 0, st>>>(g.nx, g.ny, g.nz, th, disp_dev, scale * inv_h_mm[0], scale * inv_h_mm[1],
                                            scale * inv_h_mm[2], g.t_blood, out_dev);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// heat-zone view
// ------------------------------------------------------------------------------------------------
// Samples q(m) = q0 + m dq in voxel coordinates, m = 0 .. n_samples-1; a sample counts if 0 <= q <= n-1 on all axes
// (include/rfa.h: rfa_render_zone, R-30).
//
// The ray is first clipped against the box of voxel centres (slab test in fp64), so the loop visits only the samples
// that can count -- on a 512 x 512 x 256 volume seen obliquely that is about a third of the 1136 samples of a ray.  The
// first and last RFA_RAY_EDGE samples of that range are evaluated with fp64 positions and the exact inside test; the
// samples between them lie at least RFA_RAY_EDGE - 1 steps inside the box and run in fp32: per axis the position is an
// integer cell plus a fraction in [0,1), advanced by dq with a carry, and re-anchored to the fp64 position every
// RFA_RAY_ANCHOR samples.  Between anchors the fraction drifts by at most RFA_RAY_ANCHOR * (ulp(1) + |dq| 2^-24)
// < 4e-6 voxel, i.e. < 2e-4 C at the 53 C/voxel gradient next to the needle (a coordinate of ~500 voxels carried in
// fp32 would cost 6e-5 voxel = 3e-3 C, outside the 1e-3 C bar: that is why the positions are not plain fp32).
#define RFA_RAY_EDGE 3
#define RFA_RAY_ANCHOR 16

struct RfaSampler {
    const float *theta;
    int nx, ny, nz;
    unsigned pitch, plane, dxs, dys, dzs;          // strides of the +1 neighbours (0 on an axis of one voxel)
    __device__ __forceinline__ float at(int i0, int j0, int k0, float ax, float ay, float az) const
    {
        const unsigned o000 = (unsigned)k0 * plane + (unsigned)j0 * pitch + (unsigned)i0, o100 = o000 + dxs;
        const unsigned o010 = o000 + dys, o110 = o010 + dxs, o001 = o000 + dzs, o101 = o001 + dxs, o011 = o001 + dys, o111 = o011 + dxs;
        const float c000 = __ldg(&theta[o000]), c100 = __ldg(&theta[o100]), c010 = __ldg(&theta[o010]), c110 = __ldg(&theta[o110]);
        const float c001 = __ldg(&theta[o001]), c101 = __ldg(&theta[o101]), c011 = __ldg(&theta[o011]), c111 = __ldg(&theta[o111]);
        const float x00 = fmaf(ax, c100 - c000, c000), x10 = fmaf(ax, c110 - c010, c010);
        const float x01 = fmaf(ax, c101 - c001, c001), x11 = fmaf(ax, c111 - c011, c011);
        const float y0 = fmaf(ay, x10 - x00, x00), y1 = fmaf(ay, x11 - x01, x01);
        return fmaf(az, y1 - y0, y0);
    }
};

__global__ void __launch_bounds__(128) rfa_render_kernel(RfaRay ray, int nx, int ny, int nz, const float *__restrict__ theta,
                                                         float t_blood, float iso_theta, float *__restrict__ tmax,
                                                         float *__restrict__ depth)
{
    const int px = blockIdx.x * blockDim.x + threadIdx.x, py = blockIdx.y * blockDim.y + threadIdx.y;
    if (px >= ray.width || py >= ray.height) return;
    const double u = (px - 0.5 * (ray.width - 1)) * ray.pixel, v = (py - 0.5 * (ray.height - 1)) * ray.pixel;
    const int n[3] = {nx, ny, nz};
    double q0[3], dq[3];
    // range of m whose samples can lie inside the box: lo <= m <= hi on every axis
    double lo = 0.0, hi = (double)(ray.n_samples - 1);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double o = ray.c[c] + u * ray.e1[c] + v * ray.e2[c] - ray.R * ray.w[c];
        q0[c] = o * ray.inv_h[c] - 0.5;
        dq[c] = ray.step * ray.w[c] * ray.inv_h[c];
        const double top = (double)(n[c] - 1);
        if (dq[c] > 0.0) {
            lo = fmax(lo, (0.0 - q0[c]) / dq[c]);
            hi = fmin(hi, (top - q0[c]) / dq[c]);
        } else if (dq[c] < 0.0) {
            lo = fmax(lo, (top - q0[c]) / dq[c]);
            hi = fmin(hi, (0.0 - q0[c]) / dq[c]);
        } else if (q0[c] < 0.0 || q0[c] > top) {
            hi = -1.0;                                 // parallel to this pair of faces and outside: no sample counts
        }
    }
    RfaSampler smp;
    smp.theta = theta;
    smp.nx = nx;
    smp.ny = ny;
    smp.nz = nz;
    smp.pitch = (unsigned)nx;
    smp.plane = (unsigned)nx * (unsigned)ny;
    smp.dxs = nx > 1 ? 1u : 0u;
    smp.dys = ny > 1 ? smp.pitch : 0u;
    smp.dzs = nz > 1 ? smp.plane : 0u;
    float best = -3.0e38f;
    int first = -1;
    // one sample with the fp64 position and the exact inside test (the definition, literally)
    auto exact = [&](const int m) {
        const double t = m * ray.step;
        double q[3];
        bool in = true;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double o = ray.c[c] + u * ray.e1[c] + v * ray.e2[c] - ray.R * ray.w[c];
            q[c] = (o + t * ray.w[c]) * ray.inv_h[c] - 0.5;
            in = in && q[c] >= 0.0 && q[c] <= (double)(n[c] - 1);
        }
        if (!in) return;
        const int i0 = min((int)q[0], max(nx - 2, 0)), j0 = min((int)q[1], max(ny - 2, 0)), k0 = min((int)q[2], max(nz - 2, 0));
        const float th = smp.at(i0, j0, k0, (float)(q[0] - i0), (float)(q[1] - j0), (float)(q[2] - k0));
        best = fmaxf(best, th);
        if (first < 0 && th >= iso_theta) first = m;
    };
    if (hi >= lo) {
        // one sample of slack on both sides covers the rounding of the two quotients
        const int mA = max((int)floor(lo) - 1, 0), mB = min((int)ceil(hi) + 1, ray.n_samples - 1);
        const int mI0 = mA + RFA_RAY_EDGE, mI1 = mB - RFA_RAY_EDGE;          // fp32 samples: mI0 <= m <= mI1
        for (int m = mA; m <= min(mI0 - 1, mB); ++m) exact(m);
        for (int ma = mI0; ma <= mI1; ma += RFA_RAY_ANCHOR) {
            int cell[3];
            float fr[3], df[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double q = q0[c] + (double)ma * dq[c];
                const double fl = floor(q);
                cell[c] = (int)fl;
                fr[c] = (float)(q - fl);
                df[c] = (float)dq[c];
            }
            const int cnt = min(RFA_RAY_ANCHOR, mI1 - ma + 1);
#pragma unroll 4
            for (int s = 0; s < cnt; ++s) {
                // cell indices kept inside the grid whatever the rounding did (a ray almost parallel to a face); the
                // weight then leaves [0,1] by the same few 1e-6, which the interpolation takes as it comes
                const int i0 = min(max(cell[0], 0), max(nx - 2, 0)), j0 = min(max(cell[1], 0), max(ny - 2, 0)),
                          k0 = min(max(cell[2], 0), max(nz - 2, 0));
                const float th = smp.at(i0, j0, k0, fr[0] + (float)(cell[0] - i0), fr[1] + (float)(cell[1] - j0),
                                        fr[2] + (float)(cell[2] - k0));
                best = fmaxf(best, th);
                if (first < 0 && th >= iso_theta) first = ma + s;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    fr[c] += df[c];
                    const float cf = floorf(fr[c]);
                    cell[c] += (int)cf;
                    fr[c] -= cf;
                }
            }
        }
        for (int m = max(mI1 + 1, mI0); m <= mB; ++m) exact(m);
    }
    const size_t pix = (size_t)py * ray.width + px;
    tmax[pix] = (best > -1.0e38f ? best : 0.f) + t_blood;
    if (depth) depth[pix] = first >= 0 ? (float)(first * ray.step) : -1.0f;
}

cudaError_t rfa_launch_render(const RfaGrid &g, int scenario, const RfaRay &ray, const float *theta, float iso_theta,
                              float *tmax_dev, float *depth_dev, cudaStream_t st)
{
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    if (nvox >= 0xffffffffull) return cudaErrorInvalidValue;       // 32-bit voxel offsets inside one scenario
    const dim3 block(16, 8, 1), grid((unsigned)((ray.width + 15) / 16), (unsigned)((ray.height + 7) / 8), 1);
    rfa_render_kernel<<<grid, block, 0, st>>>(ray, g.nx, g.ny, g.nz, theta + (size_t)scenario * nvox, g.t_blood, iso_theta,
                                              tmax_dev, depth_dev);
    return cudaGetLastError();
}
