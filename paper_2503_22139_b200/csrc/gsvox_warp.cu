// gsvox_warp.cu — SURVEY.md 8(f) rank 2: the warp  I(x,p) = I_ref(x + d(x,p))  (Eq. 2;
// :136 "we applied DVFs derived from the MBC motion model to yield time-resolved dynamic CBCTs"),
// batched over the B projections of a training batch, forward and backward.
//
// Readings W1-W4: trilinear interpolation of the voxel-centre samples; a corner outside
// the grid contributes 0; d is in world units, the sample sits at index u_k = i_k + d_k / h_k, its
// cell is floor(d_k / h_k) EXACTLY (see warp_cell), so positions far from the origin lose nothing to the
// magnitude of i_k; a non-finite displacement yields 0 and zero gradients.
//
// HBM/L2-bound gather.  One thread per output voxel, x fastest: the three d loads, the g load and
// the store are coalesced; the eight corner reads hit L1/L2 (I_ref is 33 MB at 256x256x128, inside
// the 126 MB L2, and neighbouring threads read neighbouring cells).  Algorithmic bytes per output
// voxel: forward 12 (d) + 4 (out) + 4/B (I_ref once per batch); backward 4 (g) + 12 (d) + 12
// (grad d) + 8/B (I_ref read, grad I_ref written) — the eight `red.global.add.f32` per voxel land
// in L2.
#include "gsvox_internal.cuh"

namespace gsvox {

constexpr int kWarpThreads = 256;

struct WarpGrid { int nx, ny, nz; float inv_hx, inv_hy, inv_hz; float hx, hy, hz; int inexact; };   // inexact: bit k set <=> 1/h_k is not a power of two

// One axis of the cell decision.  t = d * fp32(1/h) carries two fp32 roundings, |t - d/h| <= 2^-23 |t|, so
// floor(t) can differ from floor(d/h) only within that distance of a cell face.  The interpolant is continuous
// there, but its slope (grad d) is not, so such samples are settled exactly: the sign of the fused
// d - k h is the sign of the exact value (one rounding, never to the other side of 0), which tells whether
// k <= d/h < k + 1.  Rare branch (|t| >= 8 or a fraction within 2e-6 of 0 or 1); skipped altogether when 1/h
// is exact in fp32 (power-of-two spacing: t is then exact).
__device__ __forceinline__ void settle_cell(float d, float h, float t, float& fl, float& f)
{
    const float r0 = fmaf(-fl, h, d), r1 = fmaf(-(fl + 1.f), h, d);
    if (r0 < 0.f) fl -= 1.f; else if (r1 >= 0.f) fl += 1.f;
    f = fminf(fmaxf(t - fl, 0.f), 1.f);
}

// Cell of one sample: base corner (may be outside the grid) and fractions; false if non-finite or
// |t| >= 2^22 voxels.  floor -> int without a second conversion instruction: for |fl| < 2^22,
// fl + 1.5 * 2^23 holds the integer in its low mantissa bits.
__device__ __forceinline__ bool warp_cell(float dx, float dy, float dz, const WarpGrid& wg, int x, int y, int z,
                                          int& cx, int& cy, int& cz, float& fx, float& fy, float& fz)
{
    const float tx = __fmul_rn(dx, wg.inv_hx), ty = __fmul_rn(dy, wg.inv_hy), tz = __fmul_rn(dz, wg.inv_hz);
    // the comparison is false for NaN, so it rejects NaN and inf as well
    const bool ok = (fabsf(tx) < 4194304.f) && (fabsf(ty) < 4194304.f) && (fabsf(tz) < 4194304.f);
    float flx = floorf(tx), fly = floorf(ty), flz = floorf(tz);
    fx = tx - flx; fy = ty - fly; fz = tz - flz;
    if (wg.inexact && ok) {
        constexpr float kEps = 2.0e-6f, kBig = 8.f;                 // 2^-23 * 8 = 9.5e-7 < kEps
        if (wg.inexact & 1) if (fx < kEps || fx > 1.f - kEps || fabsf(tx) >= kBig) settle_cell(dx, wg.hx, tx, flx, fx);
        if (wg.inexact & 2) if (fy < kEps || fy > 1.f - kEps || fabsf(ty) >= kBig) settle_cell(dy, wg.hy, ty, fly, fy);
        if (wg.inexact & 4) if (fz < kEps || fz > 1.f - kEps || fabsf(tz) >= kBig) settle_cell(dz, wg.hz, tz, flz, fz);
    }
    fx = ok ? fx : 0.f; fy = ok ? fy : 0.f; fz = ok ? fz : 0.f;
    const int ix = __float_as_int(flx + 12582912.f) - 0x4B400000, iy = __float_as_int(fly + 12582912.f) - 0x4B400000;
    const int iz = __float_as_int(flz + 12582912.f) - 0x4B400000;
    cx = ok ? x + ix : x; cy = ok ? y + iy : y; cz = ok ? z + iz : z;
    return ok;
}

// Eight-corner gather of one sample; corners outside the grid read 0.  Cells wholly inside the grid
// (all but a boundary shell) take the path without bounds tests.
__device__ __forceinline__ float warp_sample(const float* __restrict__ iref, const WarpGrid& wg,
                                             int cx, int cy, int cz, float fx, float fy, float fz)
{
    if ((unsigned)cx < (unsigned)(wg.nx - 1) && (unsigned)cy < (unsigned)(wg.ny - 1) && (unsigned)cz < (unsigned)(wg.nz - 1)) {
        const float* p00 = iref + ((size_t)cz * wg.ny + cy) * wg.nx + cx;
        const float* p10 = p00 + wg.nx;
        const float* p01 = p00 + (size_t)wg.nx * wg.ny;
        const float* p11 = p01 + wg.nx;
        const float a0 = __ldg(p00), a1 = __ldg(p00 + 1), b0 = __ldg(p10), b1 = __ldg(p10 + 1);
        const float c0 = __ldg(p01), c1 = __ldg(p01 + 1), e0 = __ldg(p11), e1 = __ldg(p11 + 1);
        const float la = fmaf(fx, a1 - a0, a0), lb = fmaf(fx, b1 - b0, b0);
        const float lc = fmaf(fx, c1 - c0, c0), le = fmaf(fx, e1 - e0, e0);
        const float lo = fmaf(fy, lb - la, la), hi = fmaf(fy, le - lc, lc);
        return fmaf(fz, hi - lo, lo);
    }
    float acc = 0.f;
    #pragma unroll
    for (int az = 0; az < 2; ++az) {
        const int zz = cz + az;
        const float wz = az ? fz : 1.f - fz;
        #pragma unroll
        for (int ay = 0; ay < 2; ++ay) {
            const int yy = cy + ay;
            const float wyz = wz * (ay ? fy : 1.f - fy);
            const bool rowok = ((unsigned)zz < (unsigned)wg.nz) && ((unsigned)yy < (unsigned)wg.ny);
            const float* row = iref + ((size_t)(rowok ? zz : 0) * wg.ny + (rowok ? yy : 0)) * wg.nx;
            const float v0 = (rowok && (unsigned)cx < (unsigned)wg.nx) ? __ldg(row + cx) : 0.f;
            const float v1 = (rowok && (unsigned)(cx + 1) < (unsigned)wg.nx) ? __ldg(row + cx + 1) : 0.f;
            acc = fmaf(wyz, fmaf(fx, v1 - v0, v0), acc);
        }
    }
    return acc;
}

// A warp takes 32 * kWarpNJ consecutive voxels; lane l handles voxels l, l + 32, ... of them, so every load, store and
// corner gather of a warp touches neighbouring addresses (4 consecutive x per thread with 128-bit loads strides the
// gathers by 16 bytes, 16 sectors per gather instead of 5: 0.37 ms against 0.30 ms at 256x256x128, B = 8).  32-bit index
// arithmetic: V < 2^31 is checked on the host.
constexpr int kWarpNJ = 4;
#define WARP_BWD_NJ 2   // voxels per thread of the backward, 32 apart (measured 1: 0.96 / 0.71 ms, 2: 0.95 / 0.65, 4: 0.98 / 0.70; bench field / noise-free field)
__global__ void __launch_bounds__(kWarpThreads)
k_warp_forward(const float* __restrict__ iref, const float* __restrict__ dvf, WarpGrid wg, int B,
               float* __restrict__ out)
{
    const unsigned V = (unsigned)wg.nx * wg.ny * wg.nz;
    const unsigned gwarp = (blockIdx.x * kWarpThreads + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const unsigned v0 = gwarp * (32u * kWarpNJ) + lane;
    const int b = blockIdx.y;
    if (v0 >= V) return;
    const unsigned row = v0 / (unsigned)wg.nx;
    int x = (int)(v0 - row * wg.nx), z = (int)(row / (unsigned)wg.ny), y = (int)(row - (unsigned)z * wg.ny);
    const float* d = dvf + (size_t)b * 3 * V;
    float* o = out + (size_t)b * V;
    float dx[kWarpNJ], dy[kWarpNJ], dz[kWarpNJ];
    #pragma unroll
    for (int j = 0; j < kWarpNJ; ++j) {
        const unsigned v = v0 + 32u * j;
        const bool live = v < V;
        dx[j] = live ? __ldcs(d + v) : 0.f; dy[j] = live ? __ldcs(d + V + v) : 0.f; dz[j] = live ? __ldcs(d + 2 * (size_t)V + v) : 0.f;
    }
    #pragma unroll
    for (int j = 0; j < kWarpNJ; ++j) {
        const unsigned v = v0 + 32u * j;
        if (v < V) {
            int cx, cy, cz; float fx, fy, fz;
            const bool ok = warp_cell(dx[j], dy[j], dz[j], wg, x, y, z, cx, cy, cz, fx, fy, fz);
            __stcs(o + v, ok ? warp_sample(iref, wg, cx, cy, cz, fx, fy, fz) : 0.f);
        }
        x += 32;
        while (x >= wg.nx) { x -= wg.nx; if (++y >= wg.ny) { y = 0; ++z; } }
    }
}

__device__ __forceinline__ void red_add(float* addr, float v)
{
    asm volatile("red.global.add.f32 [%0], %1;" :: "l"(addr), "f"(v) : "memory");
}

// One thread per voxel, lanes along x, so the atomics of a warp are contiguous.  Neighbouring samples
// of a smooth DVF sit in neighbouring cells: lane l's right-hand corner is lane l+1's left-hand one.
// Those two contributions are merged with a shuffle before they leave the SM, which halves the
// `red.global.add.f32` count (8 -> ~4 per voxel); a lane keeps its own left-hand add only when its
// left neighbour did not take it.  (Four x per thread, as in the forward kernel, strides the
// atomics and measured 40 % slower.)
__global__ void __launch_bounds__(kWarpThreads)
k_warp_backward(const float* __restrict__ iref, const float* __restrict__ dvf, const float* __restrict__ gout,
                WarpGrid wg, int B, float* __restrict__ giref, float* __restrict__ gdvf)
{
    const unsigned V = (unsigned)wg.nx * wg.ny * wg.nz;
    const unsigned gwarp = (blockIdx.x * kWarpThreads + threadIdx.x) >> 5;
    const unsigned vfirst = gwarp * (32u * WARP_BWD_NJ) + (threadIdx.x & 31);
    const int b = blockIdx.y;
    if (gwarp * (32u * WARP_BWD_NJ) >= V) return;                   // whole warp out (warp-uniform)
    const unsigned row0 = min(vfirst, V - 1) / (unsigned)wg.nx;
    int x = (int)(min(vfirst, V - 1) - row0 * wg.nx), z = (int)(row0 / (unsigned)wg.ny), y = (int)(row0 - (unsigned)z * wg.ny);
    const float* d = dvf + (size_t)b * 3 * V;
    float dxs[WARP_BWD_NJ], dys[WARP_BWD_NJ], dzs[WARP_BWD_NJ], gs[WARP_BWD_NJ];
    #pragma unroll
    for (int j = 0; j < WARP_BWD_NJ; ++j) {
        const unsigned v = vfirst + 32u * j;
        const bool live = v < V;
        dxs[j] = live ? __ldcs(d + v) : 0.f; dys[j] = live ? __ldcs(d + V + v) : 0.f;
        dzs[j] = live ? __ldcs(d + 2 * (size_t)V + v) : 0.f; gs[j] = live ? __ldcs(gout + (size_t)b * V + v) : 0.f;
    }
    #pragma unroll
    for (int j = 0; j < WARP_BWD_NJ; ++j) {
    const unsigned v = vfirst + 32u * j;
    if (gwarp * (32u * WARP_BWD_NJ) + 32u * j >= V) break;          // warp-uniform
    const bool live = v < V;
    const float dx = dxs[j], dy = dys[j], dz = dzs[j];
    float g = gs[j];
    int cx, cy, cz; float fx, fy, fz;
    const bool ok = warp_cell(dx, dy, dz, wg, x, y, z, cx, cy, cz, fx, fy, fz) && live;
    // does lane+1 continue my cell row?  (same y,z cell, x cell one further, both valid)
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int ncx = __shfl_down_sync(full, cx, 1), ncy = __shfl_down_sync(full, cy, 1), ncz = __shfl_down_sync(full, cz, 1);
    const int nok = __shfl_down_sync(full, (int)ok, 1);
    const bool take_next = ok && nok && (lane < 31) && (ncx == cx + 1) && (ncy == cy) && (ncz == cz);
    const bool taken = __shfl_up_sync(full, (int)take_next, 1) && (lane > 0);       // my left add is done by lane-1
    if (!ok) g = 0.f;                                               // non-finite displacement: zero gradients
    float gx = 0.f, gy = 0.f, gz = 0.f;
    // all 32 cells wholly inside the grid (every warp but those at the rim): 32-bit offsets from one base, no bounds tests
    const bool interior = ok && (unsigned)cx < (unsigned)(wg.nx - 1) && (unsigned)cy < (unsigned)(wg.ny - 1) &&
                          (unsigned)cz < (unsigned)(wg.nz - 1);
    if (__all_sync(full, interior)) {
        const unsigned base = ((unsigned)cz * wg.ny + cy) * wg.nx + cx;
        const float* ip = iref + base;
        float* gp = giref + base;
        const int sy_ = wg.nx, sz_ = wg.nx * wg.ny;
        #pragma unroll
        for (int az = 0; az < 2; ++az) {
            const float wz = az ? fz : 1.f - fz, sz = az ? 1.f : -1.f;
            #pragma unroll
            for (int ay = 0; ay < 2; ++ay) {
                const float wy = ay ? fy : 1.f - fy, sy = ay ? 1.f : -1.f;
                const int off = az * sz_ + ay * sy_;
                const float v0 = __ldg(ip + off), v1 = __ldg(ip + off + 1);
                const float gwyz = g * wy * wz;
                const float a0 = gwyz * (1.f - fx);
                float a1 = gwyz * fx;
                const float na0 = __shfl_down_sync(full, a0, 1);
                if (take_next) a1 += na0;
                if (!taken) red_add(gp + off, a0);
                red_add(gp + off + 1, a1);
                const float lin = fmaf(fx, v1 - v0, v0);
                gx = fmaf(wy * wz, v1 - v0, gx);
                gy = fmaf(sy * wz, lin, gy);
                gz = fmaf(wy * sz, lin, gz);
            }
        }
    } else
    #pragma unroll
    for (int az = 0; az < 2; ++az) {
        const int zz = cz + az;
        const float wz = az ? fz : 1.f - fz, sz = az ? 1.f : -1.f;
        #pragma unroll
        for (int ay = 0; ay < 2; ++ay) {
            const int yy = cy + ay;
            const float wy = ay ? fy : 1.f - fy, sy = ay ? 1.f : -1.f;
            const bool rowok = ok && ((unsigned)zz < (unsigned)wg.nz) && ((unsigned)yy < (unsigned)wg.ny);
            const size_t rowoff = ((size_t)(rowok ? zz : 0) * wg.ny + (rowok ? yy : 0)) * wg.nx;
            const bool ok0 = rowok && (unsigned)cx < (unsigned)wg.nx, ok1 = rowok && (unsigned)(cx + 1) < (unsigned)wg.nx;
            const float v0 = ok0 ? __ldg(iref + rowoff + cx) : 0.f;
            const float v1 = ok1 ? __ldg(iref + rowoff + cx + 1) : 0.f;
            const float gwyz = g * wy * wz;
            const float a0 = gwyz * (1.f - fx);
            float a1 = gwyz * fx;
            const float na0 = __shfl_down_sync(full, a0, 1);          // lane+1's left-hand contribution, same address
            if (take_next) a1 += na0;
            if (ok0 && !taken) red_add(giref + rowoff + cx, a0);
            if (ok1) red_add(giref + rowoff + cx + 1, a1);
            const float lin = fmaf(fx, v1 - v0, v0);                  // interpolated along x
            gx = fmaf(wy * wz, v1 - v0, gx);
            gy = fmaf(sy * wz, lin, gy);
            gz = fmaf(wy * sz, lin, gz);
        }
    }
    if (live) {
        float* gd = gdvf + (size_t)b * 3 * V;
        __stcs(gd + v, g * gx * wg.inv_hx); __stcs(gd + V + v, g * gy * wg.inv_hy);
        __stcs(gd + 2 * (size_t)V + v, g * gz * wg.inv_hz);
    }
    x += 32;
    while (x >= wg.nx) { x -= wg.nx; if (++y >= wg.ny) { y = 0; ++z; } }
    }
}

}  // namespace gsvox

using namespace gsvox;

static int warp_grid(const gsvox_grid* g, int32_t B, WarpGrid* wg)
{
    if (!g || B < 1 || B > 65535) return GSVOX_EINVAL;
    for (int k = 0; k < 3; ++k)
        if (!(g->spacing[k] > 0.f) || g->dims[k] < 1 || g->dims[k] > GSVOX_MAX_DIM) return GSVOX_EINVAL;
    wg->nx = g->dims[0]; wg->ny = g->dims[1]; wg->nz = g->dims[2];
    wg->hx = g->spacing[0]; wg->hy = g->spacing[1]; wg->hz = g->spacing[2];
    wg->inv_hx = 1.f / g->spacing[0]; wg->inv_hy = 1.f / g->spacing[1]; wg->inv_hz = 1.f / g->spacing[2];
    wg->inexact = 0;
    for (int k = 0; k < 3; ++k) {
        int e; const float m = frexpf(g->spacing[k], &e);           // power of two <=> mantissa 0.5: then d * (1/h) is exact
        const float inv = 1.f / g->spacing[k];
        if (m != 0.5f || !(inv > 1.17549435e-38f) || !(inv < 3.0e38f)) wg->inexact |= 1 << k;
    }
    if ((long long)wg->nx * wg->ny * wg->nz >= (1LL << 31)) return GSVOX_ELIMIT;     // 32-bit voxel indices
    return GSVOX_OK;
}

extern "C" int gsvox_warp_forward(const float* iref, const float* dvf, const gsvox_grid* grid, int32_t B,
                                  float* out, void* stream)
{
    WarpGrid wg;
    int rc = warp_grid(grid, B, &wg);
    if (rc != GSVOX_OK) return rc;
    if (!iref || !dvf || !out) return GSVOX_EINVAL;
    const long long V = (long long)wg.nx * wg.ny * wg.nz;
    const long long per_cta = (long long)kWarpThreads * kWarpNJ;
    dim3 gridDim((unsigned)((V + per_cta - 1) / per_cta), (unsigned)B);
    k_warp_forward<<<gridDim, kWarpThreads, 0, (cudaStream_t)stream>>>(iref, dvf, wg, B, out);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

extern "C" int gsvox_warp_backward(const float* iref, const float* dvf, const gsvox_grid* grid, int32_t B,
                                   const float* grad_out, float* grad_iref, float* grad_dvf, void* stream)
{
    WarpGrid wg;
    int rc = warp_grid(grid, B, &wg);
    if (rc != GSVOX_OK) return rc;
    if (!iref || !dvf || !grad_out || !grad_iref || !grad_dvf) return GSVOX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const long long V = (long long)wg.nx * wg.ny * wg.nz;
    GSVOX_CUDA(cudaMemsetAsync(grad_iref, 0, sizeof(float) * (size_t)V, st));
    const long long per_cta = (long long)kWarpThreads * WARP_BWD_NJ;
    dim3 gridDim((unsigned)((V + per_cta - 1) / per_cta), (unsigned)B);
    k_warp_backward<<<gridDim, kWarpThreads, 0, st>>>(iref, dvf, grad_out, wg, B, grad_iref, grad_dvf);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}
