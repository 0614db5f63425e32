// gsvox_project.cu — SURVEY.md 8(f) rank 4: batched cone-beam forward projector and its transpose,
// ONE DISTINCT VOLUME PER GANTRY ANGLE (Eq. 12: P[I(x,p)]; "PMF-STGR
// requires a distinct DRR for each dynamic CBCT at each gantry angle, necessitating sequential
// projections across views ... future work could implement GPU-based parallelization to compute
// DRRs from multiple dynamic CBCTs simultaneously").  Eq. 6: I(r) = int sigma(r(t)) dt.
//
// Readings P1-P4: circular orbit about the axis through `iso` parallel to z,
// flat detector; Joseph's method — along the axis on which the ray direction is largest, one sample
// per voxel-centre plane, bilinear in the plane, zero outside, weight h_a |D| / |D_a|; per-ray
// constants in fp64 rounded to fp32, sample position fp32(u0 + fp32(m su)) without FMA (the oracle
// takes the same two roundings); backward = exact transpose.
//
// One thread per detector pixel, lanes along u.  Neighbouring rays hit neighbouring in-plane cells,
// so the four corner reads of a warp are contiguous when the in-plane fast axis is the memory-fast
// axis: true for y-dominant rays on the x-fastest volume, false for x-dominant rays (lanes then
// differ in y, one cache line each).  x-dominant rays therefore read a y-fastest copy of the volume
// (k_transpose_xy, 2 x 4V bytes per volume, < 10 % of the projector's time) — no texture units: point
// sampling must be exact and hardware filtering has 8-bit weights.  L1/L2-bound gather: per sample 4
// loads, algorithmic HBM bytes = 4V per volume + 4 per DRR pixel.
#include <cmath>
#include <mutex>
#include "gsvox_internal.cuh"

namespace gsvox {

constexpr int kProjMaxBatch = 64;
constexpr int kProjThreads = 128;

struct ProjParams {
    int n[3];                 // nx, ny, nz
    int nu, nv, B;
    double o[3], h[3];        // grid origin, spacing
    double iso[3];
    double sad, sdd, du, dv, off_u, off_v;
    double ca[kProjMaxBatch], sa[kProjMaxBatch];
    long long vol_stride;     // 0: one volume shared by all projections
};

struct Ray { int axis; float p0, ps, q0, qs, w; int m0, m1; };

// Per-ray constants, fp64 -> fp32 (reading P3).  In-plane axes (b, c) = the two other axes, ascending.
__device__ __forceinline__ Ray make_ray(const ProjParams& P, int b_, int iu, int iv)
{
    const double ca = P.ca[b_], sa = P.sa[b_];
    const double src[3] = { P.iso[0] + P.sad * ca, P.iso[1] + P.sad * sa, P.iso[2] };
    const double u = ((double)iu - (P.nu - 1) / 2.0) * P.du + P.off_u;
    const double v = ((double)iv - (P.nv - 1) / 2.0) * P.dv + P.off_v;
    const double D[3] = { -P.sdd * ca - u * sa, -P.sdd * sa + u * ca, v };
    const double ax = fabs(D[0]), ay = fabs(D[1]), az = fabs(D[2]);
    Ray r;
    r.axis = (ax >= ay && ax >= az) ? 0 : ((ay >= az) ? 1 : 2);
    const int a = r.axis, b = (a == 0) ? 1 : 0, c = (a == 2) ? 1 : 2;
    const double Da = D[a], rb = D[b] / Da, rc = D[c] / Da;
    const double norm = sqrt(D[0] * D[0] + D[1] * D[1] + D[2] * D[2]);
    r.p0 = (float)((src[b] - P.o[b] + (P.o[a] - src[a]) * rb) / P.h[b]);
    r.q0 = (float)((src[c] - P.o[c] + (P.o[a] - src[a]) * rc) / P.h[c]);
    r.ps = (float)((P.h[a] / P.h[b]) * rb);
    r.qs = (float)((P.h[a] / P.h[c]) * rc);
    r.w = (float)(P.h[a] * norm / fabs(Da));
    // planes on which the sample can touch the grid: -1 < p < n_b and -1 < q < n_c (superset, +-1 plane)
    float lo = 0.f, hi = (float)(P.n[a] - 1);
    const float p0[2] = { r.p0, r.q0 }, ps[2] = { r.ps, r.qs }, nn[2] = { (float)P.n[b], (float)P.n[c] };
    #pragma unroll
    for (int k = 0; k < 2; ++k) {
        if (fabsf(ps[k]) > 1e-12f) {
            const float t0 = (-1.f - p0[k]) / ps[k], t1 = (nn[k] - p0[k]) / ps[k];
            lo = fmaxf(lo, fminf(t0, t1) - 1.f); hi = fminf(hi, fmaxf(t0, t1) + 1.f);
        } else if (!(p0[k] > -1.f && p0[k] < nn[k])) hi = -1.f;
    }
    r.m0 = (lo <= hi) ? (int)floorf(lo) : 0;
    r.m1 = (lo <= hi) ? (int)ceilf(hi) : -1;
    r.m0 = max(r.m0, 0); r.m1 = min(r.m1, P.n[a] - 1);
    return r;
}

// Layout of the array a ray samples: x-dominant rays use the y-fastest copy.
struct Lay { long long sa, sb, sc; int nb, nc; };
__device__ __forceinline__ Lay make_lay(const ProjParams& P, int axis)
{
    const long long nx = P.n[0], ny = P.n[1];
    Lay L;
    if (axis == 0)      { L.sa = ny; L.sb = 1;  L.sc = nx * ny; L.nb = P.n[1]; L.nc = P.n[2]; }   // volT[z][x][y]: a = x, b = y, c = z
    else if (axis == 1) { L.sa = nx; L.sb = 1;  L.sc = nx * ny; L.nb = P.n[0]; L.nc = P.n[2]; }   // vol [z][y][x]: a = y, b = x, c = z
    else                { L.sa = nx * ny; L.sb = 1; L.sc = nx;  L.nb = P.n[0]; L.nc = P.n[1]; }   // vol: a = z, b = x, c = y
    return L;
}

__device__ __forceinline__ bool sample_cell(const Ray& r, int m, int& ib, int& ic, float& fb, float& fc)
{
    const float fm = (float)m;
    const float p = __fadd_rn(r.p0, __fmul_rn(fm, r.ps)), q = __fadd_rn(r.q0, __fmul_rn(fm, r.qs));
    const bool good = (fabsf(p) < 4194304.f) && (fabsf(q) < 4194304.f);
    const float pf = floorf(p), qf = floorf(q);
    fb = p - pf; fc = q - qf;
    ib = __float_as_int(pf + 12582912.f) - 0x4B400000; ic = __float_as_int(qf + 12582912.f) - 0x4B400000;
    return good;
}

// A latency-bound gather: full occupancy (16 CTAs x 4 warps, 32 registers, the per-ray constants spilled) beats the
// 46-register build at 10 CTAs (0.72 -> 0.58 ms; 12 CTAs 0.65).  The backward is issue-bound and loses with more CTAs.
__global__ void __launch_bounds__(kProjThreads, 16)
k_project_forward(const float* __restrict__ vol, const float* __restrict__ volT, ProjParams P, float* __restrict__ drr)
{
    const int iu = blockIdx.x * kProjThreads + threadIdx.x, iv = blockIdx.y, b_ = blockIdx.z;
    if (iu >= P.nu) return;
    const Ray r = make_ray(P, b_, iu, iv);
    const Lay L = make_lay(P, r.axis);
    const long long V = (long long)P.n[0] * P.n[1] * P.n[2];
    const float* base = ((r.axis == 0) ? volT + (long long)b_ * V : vol + (long long)b_ * P.vol_stride);
    // 32-bit offsets inside one volume (V < 2^31, checked on the host); cells wholly inside the plane
    // (all but the rim) take the path without bounds tests
    const int sa = (int)L.sa, sc = (int)L.sc, nb1 = L.nb - 1, nc1 = L.nc - 1;
    float acc = 0.f;
    #pragma unroll 4
    for (int m = r.m0; m <= r.m1; ++m) {
        int ib, ic; float fb, fc;
        const bool good = sample_cell(r, m, ib, ic, fb, fc);
        if ((unsigned)ib < (unsigned)nb1 && (unsigned)ic < (unsigned)nc1 && good) {
            const float* q0 = base + (m * sa + ic * sc + ib);
            const float v00 = __ldg(q0), v10 = __ldg(q0 + 1), v01 = __ldg(q0 + sc), v11 = __ldg(q0 + sc + 1);
            const float l0 = fmaf(fb, v10 - v00, v00), l1 = fmaf(fb, v11 - v01, v01);
            acc += fmaf(fc, l1 - l0, l0);
        } else if (good) {
            const bool b0 = (unsigned)ib <= (unsigned)nb1, b1 = (unsigned)(ib + 1) <= (unsigned)nb1;
            const bool c0 = (unsigned)ic <= (unsigned)nc1, c1 = (unsigned)(ic + 1) <= (unsigned)nc1;
            const float* r0 = base + (m * sa + (c0 ? ic : 0) * sc + ib);
            const float* r1 = base + (m * sa + (c1 ? ic + 1 : 0) * sc + ib);
            const float v00 = (b0 && c0) ? __ldg(r0) : 0.f, v10 = (b1 && c0) ? __ldg(r0 + 1) : 0.f;
            const float v01 = (b0 && c1) ? __ldg(r1) : 0.f, v11 = (b1 && c1) ? __ldg(r1 + 1) : 0.f;
            const float l0 = fmaf(fb, v10 - v00, v00), l1 = fmaf(fb, v11 - v01, v01);
            acc += fmaf(fc, l1 - l0, l0);
        }
    }
    drr[((long long)b_ * P.nv + iv) * P.nu + iu] = acc * r.w;
}

__device__ __forceinline__ void proj_red(float* addr, float v)
{
    asm volatile("red.global.add.f32 [%0], %1;" :: "l"(addr), "f"(v) : "memory");
}

// Transpose: every sample scatters g w {(1-fb)(1-fc), fb(1-fc), (1-fb)fc, fb fc} into its four corners;
// x-dominant rays scatter into the y-fastest scratch, folded back by k_transpose_add.
// Neighbouring detector pixels are ~0.26 voxel apart in the volume (0.776 mm pixels, magnification
// 1.5, 2 mm voxels), so runs of 3-4 consecutive lanes hit the SAME cell on a plane: their four corner
// contributions are summed by a segmented shuffle reduction (runs = maximal stretches of lanes with
// equal (ib, ic), split every CUT lanes so that log2(CUT) doubling steps suffice) and only the head of a
// run issues the atomics.  The kernel is bound by instruction issue, not by the atomics: merging PAIRS
// (CUT = 2, 4 shuffles) beats longer runs until ~4.5 lanes share a cell (host picks CUT, see below).
__device__ __forceinline__ void scatter4(float* __restrict__ base, const Lay& L, int m, int ib, int ic,
                                         float a00, float a10, float a01, float a11)
{
    float* pl = base + (long long)m * L.sa;
    const bool b0 = (unsigned)ib < (unsigned)L.nb, b1 = (unsigned)(ib + 1) < (unsigned)L.nb;
    const bool c0 = (unsigned)ic < (unsigned)L.nc, c1 = (unsigned)(ic + 1) < (unsigned)L.nc;
    float* r0 = pl + (long long)(c0 ? ic : 0) * L.sc + ib;
    float* r1 = pl + (long long)(c1 ? ic + 1 : 0) * L.sc + ib;
    if (b0 && c0) proj_red(r0, a00);
    if (b1 && c0) proj_red(r0 + 1, a10);
    if (b0 && c1) proj_red(r1, a01);
    if (b1 && c1) proj_red(r1 + 1, a11);
}

template <int CUT>
__global__ void __launch_bounds__(kProjThreads)
k_project_backward(const float* __restrict__ gdrr, ProjParams P, float* __restrict__ gvol, float* __restrict__ gvolT)
{
    const int iu = blockIdx.x * kProjThreads + threadIdx.x, iv = blockIdx.y, b_ = blockIdx.z;
    const bool live = iu < P.nu;
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const Ray r = make_ray(P, b_, live ? iu : P.nu - 1, iv);
    const Lay L = make_lay(P, r.axis);
    const long long V = (long long)P.n[0] * P.n[1] * P.n[2];
    float* base = ((r.axis == 0) ? gvolT : gvol) + (long long)b_ * V;
    const float g = live ? gdrr[((long long)b_ * P.nv + iv) * P.nu + iu] * r.w : 0.f;
    const bool uniform = __all_sync(full, r.axis == __shfl_sync(full, r.axis, 0));
    if (!uniform) {                                   // a warp that straddles a 45-degree diagonal: plain scatter
        if (g == 0.f) return;
        for (int m = r.m0; m <= r.m1; ++m) {
            int ib, ic; float fb, fc;
            if (!sample_cell(r, m, ib, ic, fb, fc)) continue;
            const float g0 = g * (1.f - fc), g1 = g * fc;
            scatter4(base, L, m, ib, ic, g0 * (1.f - fb), g0 * fb, g1 * (1.f - fb), g1 * fb);
        }
        return;
    }
    const int sa = (int)L.sa, sc = (int)L.sc, nb1 = L.nb - 1, nc1 = L.nc - 1;      // 32-bit offsets inside one volume, as in the forward
    int mlo = (live && r.m0 <= r.m1) ? r.m0 : 0x7fffffff, mhi = (live && r.m0 <= r.m1) ? r.m1 : -1;
    for (int o = 16; o > 0; o >>= 1) {
        mlo = min(mlo, __shfl_xor_sync(full, mlo, o));
        mhi = max(mhi, __shfl_xor_sync(full, mhi, o));
    }
    const bool on = live && g != 0.f;
    const int m0 = on ? r.m0 : 0x7fffffff, m1 = on ? r.m1 : -1;
    for (int m = mlo; m <= mhi; ++m) {
        int ib, ic; float fb, fc;
        const bool good = sample_cell(r, m, ib, ic, fb, fc);
        const bool act = good && m >= m0 && m <= m1;
        const int key = act ? (ic + 1) * 40000 + (ib + 1) : -1 - lane;          // dims <= 32760: no collision, no overflow
        const float g0 = act ? g * (1.f - fc) : 0.f, g1 = act ? g * fc : 0.f;
        float a00 = g0 * (1.f - fb), a10 = g0 * fb, a01 = g1 * (1.f - fb), a11 = g1 * fb;
        const int kprev = __shfl_up_sync(full, key, 1);
        const unsigned bmask = __ballot_sync(full, lane == 0 || key != kprev);   // run starts
        const int start = 31 - __clz(bmask & (0xffffffffu >> (31 - lane)));
        const bool head = ((lane - start) & (CUT - 1)) == 0;                     // runs are cut every CUT lanes
        const unsigned hmask = __ballot_sync(full, head);
        const unsigned ahead = ~((~hmask >> lane) >> 1);                         // heads strictly after this lane; ones beyond lane 31
        #pragma unroll
        for (int o = 1; o < CUT; o <<= 1) {
            const float v00 = __shfl_down_sync(full, a00, o), v10 = __shfl_down_sync(full, a10, o);
            const float v01 = __shfl_down_sync(full, a01, o), v11 = __shfl_down_sync(full, a11, o);
            if ((ahead & ((1u << o) - 1u)) == 0u) { a00 += v00; a10 += v10; a01 += v01; a11 += v11; }
        }
        if (head && act) {
            if ((unsigned)ib < (unsigned)nb1 && (unsigned)ic < (unsigned)nc1) {   // cell wholly inside the plane: no bounds tests
                float* q0 = base + (m * sa + ic * sc + ib);
                proj_red(q0, a00); proj_red(q0 + 1, a10); proj_red(q0 + sc, a01); proj_red(q0 + sc + 1, a11);
            } else scatter4(base, L, m, ib, ic, a00, a10, a01, a11);
        }
    }
}

// dst[b][z][x][y] = src[b][z][y][x]  (ADD: dst[b][z][y][x] += src[b][z][x][y] with the roles of nx, ny swapped).
// One CTA per 64 x 64 tile of one (b, z) slice, 1-D grid (slice-major).  VEC: nx, ny multiples of 4 and 16-byte
// aligned bases -> float4 global loads and stores (16 KB in flight per CTA); otherwise scalar with bounds tests.
constexpr int kTrTile = 64;
template <bool ADD, bool VEC>
__global__ void __launch_bounds__(256)
k_transpose_xy(const float* __restrict__ src, long long src_stride, int nx, int ny, int nz, int tiles_x, int tiles_y,
               float* __restrict__ dst)
{
    __shared__ float tile[kTrTile][kTrTile + 1];
    const int tid = threadIdx.x;
    const unsigned tiles = (unsigned)(tiles_x * tiles_y);
    const unsigned slice = blockIdx.x / tiles, tl = blockIdx.x % tiles;
    const int z = (int)(slice % (unsigned)nz), b_ = (int)(slice / (unsigned)nz);
    const int x0 = (int)(tl % (unsigned)tiles_x) * kTrTile, y0 = (int)(tl / (unsigned)tiles_x) * kTrTile;
    const long long V = (long long)nx * ny * nz;
    const float* s = src + (long long)b_ * src_stride + (long long)z * nx * ny;
    float* d = dst + (long long)b_ * V + (long long)z * nx * ny;
    if (VEC) {
        const int c4 = (tid & 15) * 4, r0 = tid >> 4;
        float4 v[4];
        #pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int y = y0 + r0 + 16 * i, x = x0 + c4;
            v[i] = (x < nx && y < ny) ? __ldg(reinterpret_cast<const float4*>(s + y * nx + x)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        #pragma unroll
        for (int i = 0; i < 4; ++i) {
            float* t = &tile[r0 + 16 * i][c4];
            t[0] = v[i].x; t[1] = v[i].y; t[2] = v[i].z; t[3] = v[i].w;
        }
        __syncthreads();
        float4 o[4];
        #pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int x = x0 + r0 + 16 * i, y = y0 + c4;
            if (ADD) o[i] = (x < nx && y < ny) ? *reinterpret_cast<const float4*>(d + x * ny + y) : make_float4(0.f, 0.f, 0.f, 0.f);
            else o[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        #pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int xr = r0 + 16 * i, x = x0 + xr, y = y0 + c4;
            if (x < nx && y < ny) {
                o[i].x += tile[c4][xr]; o[i].y += tile[c4 + 1][xr]; o[i].z += tile[c4 + 2][xr]; o[i].w += tile[c4 + 3][xr];
                *reinterpret_cast<float4*>(d + x * ny + y) = o[i];
            }
        }
    } else {
        const int tx = tid & 63, ty = tid >> 6;
        for (int j = ty; j < kTrTile; j += 4) {
            const int x = x0 + tx, y = y0 + j;
            tile[j][tx] = (x < nx && y < ny) ? s[y * nx + x] : 0.f;
        }
        __syncthreads();
        for (int j = ty; j < kTrTile; j += 4) {
            const int y = y0 + tx, x = x0 + j;
            if (x < nx && y < ny) {
                float* o = d + x * ny + y;
                if (ADD) *o += tile[tx][j]; else *o = tile[tx][j];
            }
        }
    }
}

}  // namespace gsvox

using namespace gsvox;

template <bool ADD>
static int launch_transpose(const float* src, long long src_stride, int nx, int ny, int nz, int B, float* dst, cudaStream_t st)
{
    const int tiles_x = (nx + kTrTile - 1) / kTrTile, tiles_y = (ny + kTrTile - 1) / kTrTile;
    const long long blocks = (long long)tiles_x * tiles_y * nz * B;
    if (blocks > 0x7fffffffLL) return GSVOX_ELIMIT;
    const bool vec = (nx % 4 == 0) && (ny % 4 == 0) && (src_stride % 4 == 0) &&
                     (((uintptr_t)src | (uintptr_t)dst) & 15u) == 0;
    if (vec) k_transpose_xy<ADD, true><<<(unsigned)blocks, 256, 0, st>>>(src, src_stride, nx, ny, nz, tiles_x, tiles_y, dst);
    else     k_transpose_xy<ADD, false><<<(unsigned)blocks, 256, 0, st>>>(src, src_stride, nx, ny, nz, tiles_x, tiles_y, dst);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

static int fill_params(const gsvox_grid* g, const gsvox_cone_geometry* c, const float* angles_host, int32_t B,
                       ProjParams* P)
{
    if (!g || !c || !angles_host || B < 1 || B > kProjMaxBatch) return GSVOX_EINVAL;
    for (int k = 0; k < 3; ++k) {
        if (!(g->spacing[k] > 0.f) || g->dims[k] < 1 || g->dims[k] > GSVOX_MAX_DIM) return GSVOX_EINVAL;
        P->n[k] = g->dims[k]; P->o[k] = (double)g->origin[k]; P->h[k] = (double)g->spacing[k]; P->iso[k] = (double)c->iso[k];
    }
    if ((long long)g->dims[0] * g->dims[1] * g->dims[2] >= (1LL << 31)) return GSVOX_ELIMIT;
    if (!(c->sad > 0.f) || !(c->sdd > 0.f) || c->nu < 1 || c->nv < 1 || c->nv > 65535 || !(c->du > 0.f) || !(c->dv > 0.f))
        return GSVOX_EINVAL;
    P->nu = c->nu; P->nv = c->nv; P->B = B;
    P->sad = c->sad; P->sdd = c->sdd; P->du = c->du; P->dv = c->dv; P->off_u = c->off_u; P->off_v = c->off_v;
    for (int b = 0; b < B; ++b) { P->ca[b] = cos((double)angles_host[b]); P->sa[b] = sin((double)angles_host[b]); }
    return GSVOX_OK;
}

extern "C" int gsvox_project_scratch_bytes(const gsvox_grid* grid, int32_t B, size_t* bytes)
{
    if (!grid || !bytes || B < 1 || B > kProjMaxBatch) return GSVOX_EINVAL;
    for (int k = 0; k < 3; ++k) if (grid->dims[k] < 1) return GSVOX_EINVAL;
    *bytes = sizeof(float) * (size_t)grid->dims[0] * grid->dims[1] * grid->dims[2] * (size_t)B;
    return GSVOX_OK;
}

extern "C" int gsvox_project_forward(const float* vol, int64_t vol_stride, const gsvox_grid* grid,
                                     const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                                     void* scratch, float* drr, void* stream)
{
    ProjParams P;
    int rc = fill_params(grid, geom, angles_host, B, &P);
    if (rc != GSVOX_OK) return rc;
    const long long V = (long long)P.n[0] * P.n[1] * P.n[2];
    if (!vol || !scratch || !drr || (vol_stride != 0 && vol_stride != V)) return GSVOX_EINVAL;
    P.vol_stride = vol_stride;
    cudaStream_t st = (cudaStream_t)stream;
    rc = launch_transpose<false>(vol, vol_stride, P.n[0], P.n[1], P.n[2], B, (float*)scratch, st);
    if (rc != GSVOX_OK) return rc;
    dim3 pg((P.nu + kProjThreads - 1) / kProjThreads, (unsigned)P.nv, (unsigned)B);
    k_project_forward<<<pg, kProjThreads, 0, st>>>(vol, (const float*)scratch, P, drr);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

extern "C" int gsvox_project_backward(const float* grad_drr, const gsvox_grid* grid,
                                      const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                                      void* scratch, float* grad_vol, void* stream)
{
    ProjParams P;
    int rc = fill_params(grid, geom, angles_host, B, &P);
    if (rc != GSVOX_OK) return rc;
    if (!grad_drr || !scratch || !grad_vol) return GSVOX_EINVAL;
    const long long V = (long long)P.n[0] * P.n[1] * P.n[2];
    P.vol_stride = V;
    cudaStream_t st = (cudaStream_t)stream;
    GSVOX_CUDA(cudaMemsetAsync(grad_vol, 0, sizeof(float) * (size_t)V * B, st));
    GSVOX_CUDA(cudaMemsetAsync(scratch, 0, sizeof(float) * (size_t)V * B, st));
    dim3 pg((P.nu + kProjThreads - 1) / kProjThreads, (unsigned)P.nv, (unsigned)B);
    // lanes (adjacent detector pixels) per in-plane cell at the isocentre; measured on a B200 at 8 x 512x384 rays:
    // ratio 0.97 / 1.45 / 1.93 / 3.02 / 3.87 -> merging pairs wins (2.69, 2.87, 3.17, 1.43, 1.08 ms; no merging 2.78,
    // 3.48, 3.84, 1.97, 1.68), ratio 4.83 / 6.04 / 7.73 -> runs of 4 win (0.83, 0.64, 0.52 ms); runs of 8 never win
    const double lanes_per_cell = fmin(P.h[0], P.h[1]) / (P.du * P.sad / P.sdd);
    if (lanes_per_cell >= 4.5) k_project_backward<4><<<pg, kProjThreads, 0, st>>>(grad_drr, P, grad_vol, (float*)scratch);
    else                       k_project_backward<2><<<pg, kProjThreads, 0, st>>>(grad_drr, P, grad_vol, (float*)scratch);
    GSVOX_CUDA(cudaGetLastError());
    // fold the y-fastest scratch back: grad_vol[z][y][x] += scratch[z][x][y]  (a transpose with nx, ny swapped)
    return launch_transpose<true>((const float*)scratch, V, P.n[1], P.n[0], P.n[2], B, grad_vol, st);
}

// ------------------------------------------------------------------------------------------
// gsvox_project_forward_static: the forward projector for callers that cannot allocate device memory (code under
// CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Same kernels as gsvox_project_forward; the
// y-fastest copy of the volumes lives in the file-scope array below instead of caller-owned scratch:
// GSVOX_PROJECT_STATIC_MAX_VOXELS floats = 16 MB, held by every GPU that loads the library until the process exits.
// The array's name is a host-side stand-in in host code, NOT a device address: its device address is looked up once
// per device (with that device current) by cudaGetSymbolAddress and cached here.  This entry point calls no
// cudaMalloc / cudaFree / allocating library routine.  All calls on one device share the array: it keeps the last
// call's contents (every call overwrites the B * V floats it reads, nothing has to start at zero), and two calls
// that overlap on the GPU (different streams, or graph branches) race on it.
// ------------------------------------------------------------------------------------------
static __device__ __align__(256) float g_project_static_scratch[GSVOX_PROJECT_STATIC_MAX_VOXELS];

constexpr int kProjStaticMaxDevices = 64;
static float* g_project_static_addr[kProjStaticMaxDevices];     // [device] -> device address of the array, 0 = not looked up yet
static std::mutex g_project_static_mu;

static int project_static_scratch(float** ptr)
{
    int dev = -1;
    GSVOX_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kProjStaticMaxDevices) return GSVOX_ELIMIT;
    std::lock_guard<std::mutex> lk(g_project_static_mu);
    if (!g_project_static_addr[dev]) {
        float* p = nullptr;
        GSVOX_CUDA(cudaGetSymbolAddress((void**)&p, g_project_static_scratch));
        if (!p) return GSVOX_ECUDA;
        g_project_static_addr[dev] = p;
    }
    *ptr = g_project_static_addr[dev];
    return GSVOX_OK;
}

extern "C" int gsvox_project_forward_static(const float* vol, int64_t vol_stride, const gsvox_grid* grid,
                                            const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                                            float* drr, void* stream)
{
    ProjParams P;
    int rc = fill_params(grid, geom, angles_host, B, &P);
    if (rc != GSVOX_OK) return rc;
    const long long V = (long long)P.n[0] * P.n[1] * P.n[2];
    if (!vol || !drr || (vol_stride != 0 && vol_stride != V)) return GSVOX_EINVAL;
    if (V * B > (long long)GSVOX_PROJECT_STATIC_MAX_VOXELS) return GSVOX_ELIMIT;      // beyond the built-in scratch
    float* scratch = nullptr;
    rc = project_static_scratch(&scratch);
    if (rc != GSVOX_OK) return rc;
    P.vol_stride = vol_stride;
    cudaStream_t st = (cudaStream_t)stream;
    rc = launch_transpose<false>(vol, vol_stride, P.n[0], P.n[1], P.n[2], B, scratch, st);
    if (rc != GSVOX_OK) return rc;
    dim3 pg((P.nu + kProjThreads - 1) / kProjThreads, (unsigned)P.nv, (unsigned)B);
    k_project_forward<<<pg, kProjThreads, 0, st>>>(vol, (const float*)scratch, P, drr);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}
