// gsvox_splat.cu — SURVEY.md 8(f) rank 3: Gaussian-splat X-ray rasterizer, forward and backward, batched
// over the gantry angles of a training batch (Eq. 6-9; Stage 1 = 5000 of the 7000
// iterations).
//
//   Eq. 8   Sigma~ = J W Sigma W^T J^T          (local affine approximation of the projective mapping)
//   Eq. 9   I(r) = sum_i rho^_i exp(-1/2 (x^ - p^_i)^T Sigma^_i^-1 (x^ - p^_i)),
//           Sigma^ = Sigma~[0:2,0:2],  rho^ = rho sqrt(2 pi |Sigma~| / |Sigma^|)
// Readings R1-R6 (the paper leaves phi, J, W to "scanner parameters"): the
// projector's scanner (P1); camera frame at the source with rows of W = (u, v, central ray);
// ray space phi(t) = (t0/t2, t1/t2, |t|); pixel = SDD x^ on the detector grid; cutoff = inclusive
// pixel box of the 3-sigma ellipse, decided in fp64; t2 <= 0 or degenerate -> skipped; backward
// with frozen boxes.
//
// Same machinery as the voxelizer, one dimension down: s1 per-(angle, Gaussian) 2D record in fp64
// (centre split into integer pixel + fp32 fraction, conic, amplitude, box) with the tile counts
// fused in; s2 exclusive scan (shared with a2) + scatter: counting sort of (tile, Gaussian) keys,
// 16x16-pixel tiles; s3 one CTA per (tile, angle), keys staged through shared memory, one thread
// per pixel, ex2.approx; s4 backward: the tile's upstream gradient in shared memory, ONE THREAD PER
// KEY walks box ∩ tile and reduces its six 2D gradients in registers, one vector atomic per key;
// s5 per-Gaussian chain rule through Sigma^-1, |Sigma~|/|Sigma^|, J(t), W, R(q), S in fp64, summed
// over the angles without atomics.
#include <cmath>
#include "gsvox_internal.cuh"

namespace gsvox {
constexpr float kSplatRecurrenceMaxA = 1.0f;   // footprints narrower than ~0.85 pixel along a row: one EX2 per pixel


constexpr int kSplatTile = 16;
constexpr int kSplatMaxBatch = 64;
constexpr double kSplatKappa = GSVOX_SIGMA_CUTOFF;

struct __align__(16) Splat2D {
    float cfu, cfv;        // fractional part of the centre in pixels, [-0.5, 0.5]
    float A, B;            // conic in pixel units, already times -log2(e)/2:  E = A dx^2 + 2 B dx dy + C dy^2 (base 2)
    float C, amp;
    int16_t ciu, civ;      // integer part of the centre (may be off the detector)
    int16_t u0, v0, u1, v1;   // inclusive pixel box; empty <=> u1 < u0
    float Bq, Dq;          // row form of the exponent: E = A (dx + Bq dy)^2 + Dq dy^2, Bq = B/A, Dq = -log2(e)/2 / Sigma^_vv
    int32_t pad;
};
static_assert(sizeof(Splat2D) == 48, "Splat2D must be 48 bytes");

// `stamp` is written by the LAST kernel of gsvox_splat_forward: magic + a digest of (n, B, nu, nv, key_capacity).  A
// backward or status call on a workspace without it (no forward yet, or a forward with other sizes: every sub-buffer
// would sit elsewhere) does nothing / reports GSVOX_ENOTREADY instead of reading garbage.
struct SplatStatus {
    unsigned long long keys_needed, pairs; unsigned int overflow, skipped;
    unsigned long long stamp;
    unsigned int drop_behind, drop_range, drop_empty, pad_;      // per (angle, Gaussian): t2 <= 0 | centre beyond +-30000 px | empty box
};
constexpr unsigned long long kSplatMagic = 0x67735370ull << 32;     // "gsSp"
static unsigned long long splat_stamp(long long n, int B, int nu, int nv, long long key_capacity)
{
    unsigned long long h = 1469598103934665603ull;
    const unsigned long long v[5] = { (unsigned long long)n, (unsigned long long)B, (unsigned long long)nu,
                                      (unsigned long long)nv, (unsigned long long)key_capacity };
    for (int i = 0; i < 5; ++i) { h ^= v[i]; h *= 1099511628211ull; }
    return kSplatMagic | (h & 0xffffffffull);
}

struct SplatParams {
    int n, B, nu, nv, ntx, nty;
    double sad, sdd, du, dv, off_u, off_v, iso[3];
    double ca[kSplatMaxBatch], sa[kSplatMaxBatch];
};

struct SplatWs {            // views into the caller's workspace
    SplatStatus* status; Splat2D* rec; uint32_t* bin_count; uint32_t* bin_start; uint32_t* partial;
    uint32_t* keys; float* acc; int nbins; size_t total;
};

// Everything Eq. 8-9 needs for one (angle, Gaussian), fp64.
struct SplatTerms {
    bool valid;
    int why;                 // when !valid: 1 degenerate parameters (any angle), 2 at or behind the source plane, 3 numerically singular
    double R[9], Sig[9], t[3], ell, T[9], St[9], det_t, det_h, amp_over_rho, P[3], dp, cu, cv;
};

__device__ __forceinline__ void mat3mul(const double* a, const double* b, double* c)
{
    #pragma unroll
    for (int i = 0; i < 3; ++i)
        #pragma unroll
        for (int j = 0; j < 3; ++j) c[3 * i + j] = a[3 * i] * b[j] + a[3 * i + 1] * b[3 + j] + a[3 * i + 2] * b[6 + j];
}

__device__ __forceinline__ void splat_W(const SplatParams& P, int b, double* W, double* src)
{
    const double ca = P.ca[b], sa = P.sa[b];
    W[0] = -sa; W[1] = ca;  W[2] = 0.0;       // u
    W[3] = 0.0; W[4] = 0.0; W[5] = 1.0;       // v
    W[6] = -ca; W[7] = -sa; W[8] = 0.0;       // central ray, source -> detector
    src[0] = P.iso[0] + P.sad * ca; src[1] = P.iso[1] + P.sad * sa; src[2] = P.iso[2];
}

__device__ void splat_terms(const SplatParams& P, int b, const float* __restrict__ pos, const float* __restrict__ scale,
                            const float* __restrict__ quat, int g, SplatTerms& o)
{
    const double p[3] = { pos[3 * g], pos[3 * g + 1], pos[3 * g + 2] };
    const double s[3] = { scale[3 * g], scale[3 * g + 1], scale[3 * g + 2] };
    const double q[4] = { quat[4 * g], quat[4 * g + 1], quat[4 * g + 2], quat[4 * g + 3] };
    o.valid = false; o.why = 1;
    bool bad = false;
    for (int k = 0; k < 3; ++k) bad |= !isfinite(p[k]) || !isfinite(s[k]) || !(s[k] > 0.0);
    for (int k = 0; k < 4; ++k) bad |= !isfinite(q[k]);
    const double n2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3];
    if (bad || !(n2 > 0.0)) return;
    const double nn = sqrt(n2), r = q[0] / nn, x = q[1] / nn, y = q[2] / nn, z = q[3] / nn;
    double* R = o.R;
    R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - r * z); R[2] = 2 * (x * z + r * y);
    R[3] = 2 * (x * y + r * z); R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - r * x);
    R[6] = 2 * (x * z - r * y); R[7] = 2 * (y * z + r * x); R[8] = 1 - 2 * (x * x + y * y);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            o.Sig[3 * i + j] = R[3 * i] * s[0] * s[0] * R[3 * j] + R[3 * i + 1] * s[1] * s[1] * R[3 * j + 1]
                             + R[3 * i + 2] * s[2] * s[2] * R[3 * j + 2];
    double W[9], src[3];
    splat_W(P, b, W, src);
    const double d[3] = { p[0] - src[0], p[1] - src[1], p[2] - src[2] };
    for (int i = 0; i < 3; ++i) o.t[i] = W[3 * i] * d[0] + W[3 * i + 1] * d[1] + W[3 * i + 2] * d[2];
    const double t0 = o.t[0], t1 = o.t[1], t2 = o.t[2];
    o.why = 2;
    if (!(t2 > 0.0)) return;                                   // R5: at or behind the source plane
    o.why = 3;
    o.ell = sqrt(t0 * t0 + t1 * t1 + t2 * t2);
    const double J[9] = { 1 / t2, 0, -t0 / (t2 * t2),  0, 1 / t2, -t1 / (t2 * t2),  t0 / o.ell, t1 / o.ell, t2 / o.ell };
    mat3mul(J, W, o.T);
    double TS[9], Tt[9];
    mat3mul(o.T, o.Sig, TS);
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Tt[3 * i + j] = o.T[3 * j + i];
    mat3mul(TS, Tt, o.St);
    const double* S = o.St;
    o.det_t = S[0] * (S[4] * S[8] - S[5] * S[7]) - S[1] * (S[3] * S[8] - S[5] * S[6]) + S[2] * (S[3] * S[7] - S[4] * S[6]);
    o.det_h = S[0] * S[4] - S[1] * S[1];
    const double ku = P.sdd / P.du, kv = P.sdd / P.dv;
    o.P[0] = S[0] * ku * ku; o.P[1] = S[1] * ku * kv; o.P[2] = S[4] * kv * kv;
    o.dp = o.P[0] * o.P[2] - o.P[1] * o.P[1];
    o.cu = (P.sdd * t0 / t2 - P.off_u) / P.du + (P.nu - 1) / 2.0;
    o.cv = (P.sdd * t1 / t2 - P.off_v) / P.dv + (P.nv - 1) / 2.0;
    if (!(o.det_t > 0.0) || !(o.det_h > 0.0) || !(o.dp > 0.0) || !isfinite(o.cu) || !isfinite(o.cv)) return;
    o.amp_over_rho = sqrt(2.0 * 3.14159265358979323846 * o.det_t / o.det_h);
    o.valid = true;
}

// s1: 2D record.  One thread per (angle, Gaussian).
__global__ void __launch_bounds__(128)
k_splat_pre(SplatParams P, const float* __restrict__ pos, const float* __restrict__ scale, const float* __restrict__ quat,
            const float* __restrict__ rho, Splat2D* __restrict__ rec, uint32_t* __restrict__ bin_count,
            SplatStatus* __restrict__ status)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = idx < (long long)P.n * P.B;
    const int b = live ? (int)(idx / P.n) : 0, g = live ? (int)(idx - (long long)b * P.n) : 0;
    unsigned long long my_pairs = 0ull;
    unsigned int my_skipped = 0u, my_drops = 0u;             // my_drops: behind | range << 10 | empty << 20 (per thread: 0/1 each)
    Splat2D r;
    r.cfu = r.cfv = r.A = r.B = r.C = r.amp = 0.f; r.ciu = r.civ = 0; r.u0 = r.v0 = 0; r.u1 = r.v1 = -1; r.Bq = r.Dq = 0.f; r.pad = 0;
    SplatTerms o;
    o.valid = false;
    if (live) splat_terms(P, b, pos, scale, quat, g, o);
    const double rh = live ? (double)rho[g] : 0.0;
    if (o.valid && isfinite(rh)) {
        const double ru = kSplatKappa * sqrt(o.P[0]), rv = kSplatKappa * sqrt(o.P[2]);
        double u0 = ceil(o.cu - ru), u1 = floor(o.cu + ru), v0 = ceil(o.cv - rv), v1 = floor(o.cv + rv);
        if (u0 < 0.0) u0 = 0.0; if (v0 < 0.0) v0 = 0.0;
        if (u1 > P.nu - 1.0) u1 = P.nu - 1.0; if (v1 > P.nv - 1.0) v1 = P.nv - 1.0;
        if (isfinite(ru) && isfinite(rv) && u1 >= u0 && v1 >= v0 && fabs(o.cu) <= 30000.0 && fabs(o.cv) <= 30000.0) {
            const double k2 = -0.72134752044448170368;           // -log2(e)/2
            r.A = (float)(k2 * o.P[2] / o.dp); r.B = (float)(-k2 * o.P[1] / o.dp); r.C = (float)(k2 * o.P[0] / o.dp);
            r.amp = (float)(rh * o.amp_over_rho);
            r.Bq = (float)(-o.P[1] / o.P[2]); r.Dq = (float)(k2 / o.P[2]);        // Schur complement: no cancellation
            const double ci = rint(o.cu), cj = rint(o.cv);       // |.| <= 30000 (R5): fits int16
            r.ciu = (int16_t)ci; r.civ = (int16_t)cj; r.cfu = (float)(o.cu - ci); r.cfv = (float)(o.cv - cj);
            r.u0 = (int16_t)u0; r.v0 = (int16_t)v0; r.u1 = (int16_t)u1; r.v1 = (int16_t)v1;
            my_pairs = (unsigned long long)((u1 - u0 + 1.0) * (v1 - v0 + 1.0));
        } else if (!(fabs(o.cu) <= 30000.0 && fabs(o.cv) <= 30000.0)) my_drops = 1u << 10;
        else my_drops = 1u << 20;
    } else if (live) {
        // degenerate Gaussians (and non-finite rho) are counted once, per-angle drops per (angle, Gaussian)
        if (o.why == 2 && isfinite(rh)) my_drops = 1u;
        else if (b == 0) my_skipped = 1u;
    }
    if (live) rec[idx] = r;
    // counters: warp -> CTA -> one atomic per CTA (per-item atomics on one address cost 0.15 ms)
    __shared__ unsigned long long s_pairs[4];
    __shared__ unsigned int s_skip[4], s_drop[4];
    for (int o2 = 16; o2 > 0; o2 >>= 1) {
        my_pairs += __shfl_xor_sync(0xffffffffu, my_pairs, o2);
        my_skipped += __shfl_xor_sync(0xffffffffu, my_skipped, o2);
        my_drops += __shfl_xor_sync(0xffffffffu, my_drops, o2);          // three 10-bit fields, <= 32 each per warp
    }
    if ((threadIdx.x & 31) == 0) { s_pairs[threadIdx.x >> 5] = my_pairs; s_skip[threadIdx.x >> 5] = my_skipped; s_drop[threadIdx.x >> 5] = my_drops; }
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned long long tp = s_pairs[0] + s_pairs[1] + s_pairs[2] + s_pairs[3];
        const unsigned int ts = s_skip[0] + s_skip[1] + s_skip[2] + s_skip[3];
        const unsigned int td = s_drop[0] + s_drop[1] + s_drop[2] + s_drop[3];
        if (tp) atomicAdd(&status->pairs, tp);
        if (ts) atomicAdd(&status->skipped, ts);
        if (td & 1023u) atomicAdd(&status->drop_behind, td & 1023u);
        if ((td >> 10) & 1023u) atomicAdd(&status->drop_range, (td >> 10) & 1023u);
        if (td >> 20) atomicAdd(&status->drop_empty, td >> 20);
    }
}

// s2: counting sort of (tile, angle, Gaussian) keys.  The detector has only a few hundred tiles, so plain
// global atomics pile up on a few thousand addresses (6.7e6 adds on 6144 counters: 0.41 ms).  Each CTA
// of 1024 (angle, Gaussian) items histograms its keys in shared memory instead (native integer
// atomics) and touches every global counter once.  MODE 0: counts.  MODE 1: the CTA reserves a
// range per tile with one global atomic, items take their rank inside it from shared memory;
// keys[slot] = angle * n + Gaussian.
constexpr int kSplatSortThreads = 1024;
constexpr int kSplatMaxTilesShared = 8192;          // 32 KB of shared counters; larger detectors fall back to global atomics

template <int MODE>
__global__ void __launch_bounds__(kSplatSortThreads)
k_splat_sort(SplatParams P, const Splat2D* __restrict__ rec, uint32_t* __restrict__ bin_count, uint32_t* __restrict__ keys,
             const SplatStatus* __restrict__ status)
{
    extern __shared__ uint32_t s_bins[];               // [tiles] counts, then (MODE 1) [tiles] global bases
    if (MODE == 1 && status->overflow) return;
    const int tiles = P.ntx * P.nty, b = blockIdx.y;
    const bool shared = tiles <= kSplatMaxTilesShared;
    uint32_t* gbin = bin_count + (size_t)b * tiles;
    const int g = blockIdx.x * kSplatSortThreads + threadIdx.x;
    int tx0 = 0, tx1 = -1, ty0 = 0, ty1 = -1;
    const uint32_t id = (uint32_t)((size_t)b * P.n + (g < P.n ? g : 0));
    if (g < P.n) {
        const int4 w = __ldg(reinterpret_cast<const int4*>(rec + id) + 1);     // C, amp, ciu|civ, u0|v0
        const int w2 = __ldg(reinterpret_cast<const int*>(rec + id) + 8);      // u1|v1
        const int u0 = (int16_t)(w.w & 0xffff), v0 = (int16_t)(w.w >> 16), u1 = (int16_t)(w2 & 0xffff), v1 = (int16_t)(w2 >> 16);
        if (u1 >= u0) { tx0 = u0 / kSplatTile; tx1 = u1 / kSplatTile; ty0 = v0 / kSplatTile; ty1 = v1 / kSplatTile; }
    }
    if (!shared) {
        for (int ty = ty0; ty <= ty1; ++ty)
            for (int tx = tx0; tx <= tx1; ++tx) {
                if (MODE == 0) atomicAdd(&gbin[ty * P.ntx + tx], 1u);
                else keys[atomicAdd(&gbin[ty * P.ntx + tx], 1u)] = id;
            }
        return;
    }
    for (int t = threadIdx.x; t < tiles; t += kSplatSortThreads) s_bins[t] = 0u;
    __syncthreads();
    if (MODE == 0) {
        for (int ty = ty0; ty <= ty1; ++ty)
            for (int tx = tx0; tx <= tx1; ++tx) atomicAdd(&s_bins[ty * P.ntx + tx], 1u);
        __syncthreads();
        for (int t = threadIdx.x; t < tiles; t += kSplatSortThreads)
            if (s_bins[t]) atomicAdd(&gbin[t], s_bins[t]);
    } else {
        uint32_t* s_base = s_bins + tiles;
        for (int ty = ty0; ty <= ty1; ++ty)
            for (int tx = tx0; tx <= tx1; ++tx) atomicAdd(&s_bins[ty * P.ntx + tx], 1u);
        __syncthreads();
        for (int t = threadIdx.x; t < tiles; t += kSplatSortThreads) {
            const uint32_t c = s_bins[t];
            s_base[t] = c ? atomicAdd(&gbin[t], c) : 0u;       // this CTA's range of the tile's key list
            s_bins[t] = 0u;
        }
        __syncthreads();
        for (int ty = ty0; ty <= ty1; ++ty)
            for (int tx = tx0; tx <= tx1; ++tx) {
                const int t = ty * P.ntx + tx;
                keys[s_base[t] + atomicAdd(&s_bins[t], 1u)] = id;
            }
    }
}

__device__ __forceinline__ float ex2s(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// s3: ONE WARP per (tile, angle); thread t owns the 8-pixel row segment (row t >> 1, columns 8 (t & 1) ..
// + 7) in registers.  Along a row the exponent is a parabola in x, E(x) = A (x - xs)^2 + Es with
// xs = cx - Bq dy, Es = Dq dy^2, so — as in a3 — the eight values come from a centre-out
// multiplicative recurrence: 3 ex2 + 2 FMUL + 5 FMUL2 + 4 FFMA2 per 8 pixels instead of 8 ex2 and 8 x 7
// flops (the per-pixel version of this kernel: 1.00 ms; this one: see DESIGN.md section 13).  Footprints
// narrower than ~0.85 pixel along x (A < -1) take one ex2 per pixel.  Keys are staged 32 at a time as
// 96-byte tile-local records: geometry, the row mask of box ∩ tile, and the amplitude times
// [column inside the box] for the 16 columns in the packed-pair order of the recurrence.
struct __align__(16) SplatTileRec {
    float cx, cy, A, Bq;       // centre relative to the tile origin
    float Dq, cc;              // cc = 2^(2A): ratio of successive ratios along x
    uint32_t rowmask, direct;
    float w[16];               // per segment: columns 3,4, 2,5, 1,6, 0,7 (+8 for the second segment)
};
static_assert(sizeof(SplatTileRec) == 96, "SplatTileRec must be 96 bytes");

#ifndef SPLAT_FWD_WARPS
#define SPLAT_FWD_WARPS 4   // measured: 1 warp 0.52 ms, 2: 0.45, 4: 0.40, 8: 0.40 (50 k Gaussians x 8 angles)
#endif
constexpr int kSplatFwdBatch = 32;
constexpr int kSplatFwdWarps = SPLAT_FWD_WARPS;   // warps of a CTA take the tile's key batches round-robin; partial tiles summed in smem

__global__ void __launch_bounds__(32 * kSplatFwdWarps)
k_splat_forward(SplatParams P, const Splat2D* __restrict__ rec, const uint32_t* __restrict__ bin_start,
                const uint32_t* __restrict__ keys, SplatStatus* __restrict__ status, unsigned long long stamp,
                float* __restrict__ drr)
{
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) status->stamp = stamp;     // the forward got this far
    __shared__ SplatTileRec s_recs[kSplatFwdWarps][kSplatFwdBatch];
    __shared__ float s_part[kSplatFwdWarps > 1 ? kSplatFwdWarps - 1 : 1][8][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tile = blockIdx.x, b = blockIdx.y;
    SplatTileRec* s_rec = s_recs[warp];
    const int tx = tile % P.ntx, ty = tile / P.ntx;
    const int ox = tx * kSplatTile, oy = ty * kSplatTile;
    const int row = lane >> 1, seg = lane & 1;
    const float fy = (float)row, fx3 = (float)(8 * seg + 3);
    const uint32_t rowbit = 1u << row;
    uint32_t kbeg = 0, kend = 0;
    if (!status->overflow) { kbeg = bin_start[b * P.ntx * P.nty + tile]; kend = bin_start[b * P.ntx * P.nty + tile + 1]; }
    float acc[8];                                          // acc[2j], acc[2j+1] = columns 3 - j, 4 + j of the segment
    #pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = 0.f;
    for (uint32_t base = kbeg + warp * kSplatFwdBatch; base < kend; base += kSplatFwdBatch * kSplatFwdWarps) {
        const int nb = (int)min((uint32_t)kSplatFwdBatch, kend - base);
        __syncwarp();
        if (lane < nb) {
            const Splat2D r = rec[keys[base + lane]];
            const int x0 = max(r.u0 - ox, 0), x1 = min(r.u1 - ox, kSplatTile - 1);
            const int y0 = max(r.v0 - oy, 0), y1 = min(r.v1 - oy, kSplatTile - 1);
            SplatTileRec& t = s_rec[lane];
            t.cx = (float)(r.ciu - ox) + r.cfu; t.cy = (float)(r.civ - oy) + r.cfv;
            t.A = r.A; t.Bq = r.Bq; t.Dq = r.Dq; t.cc = ex2s(2.f * r.A);
            t.rowmask = ((2u << y1) - (1u << y0)) & 0xffffu;
            t.direct = (-r.A > kSplatRecurrenceMaxA) ? 1u : 0u;
            const uint32_t xm = ((2u << x1) - (1u << x0)) & 0xffffu;
            // amplitude x [column in box] x c^{0,1,3,6} (pair j of the centre-out chain; direct keys: no c-power)
            const float c1 = t.direct ? 1.f : t.cc, c3 = c1 * c1 * c1;
            const float ak[4] = { r.amp, r.amp * c1, r.amp * c3, r.amp * (c3 * c3) };
            #pragma unroll
            for (int s2 = 0; s2 < 2; ++s2)
                #pragma unroll
                for (int j = 0; j < 4; ++j) {
                    t.w[8 * s2 + 2 * j] = (xm >> (8 * s2 + 3 - j)) & 1u ? ak[j] : 0.f;
                    t.w[8 * s2 + 2 * j + 1] = (xm >> (8 * s2 + 4 + j)) & 1u ? ak[j] : 0.f;
                }
        }
        __syncwarp();
        #pragma unroll 2
        for (int j = 0; j < nb; ++j) {
            const float4 g0 = *reinterpret_cast<const float4*>(&s_rec[j]);             // cx, cy, A, Bq
            const float4 g1 = *reinterpret_cast<const float4*>(&s_rec[j].Dq);          // Dq, cc, rowmask, direct
            const float4 wa = *reinterpret_cast<const float4*>(&s_rec[j].w[8 * seg]);
            const float4 wb = *reinterpret_cast<const float4*>(&s_rec[j].w[8 * seg + 4]);
            const float dy = fy - g0.y;
            const float xs = fmaf(-g0.w, dy, g0.x);                    // E(x) = A (x - xs)^2 + Es
            float Es = g1.x * dy * dy;
            Es = (__float_as_uint(g1.z) & rowbit) ? Es : -1.0e30f;     // rows outside the box contribute exact zeros
            const float negA = g0.z;
            f32x2 Pp[4];                                               // Pp[j] = (G[3-j], G[4+j]) of this segment
            if (__float_as_uint(g1.w) == 0u) {
                // E(x) = E3 + (x - 3) Lf + A (x - 3)(x - 4): G(x) = G3 rho^(x-3) c^((x-3)(x-4)/2), rho = 2^Lf, c = 2^2A; the
                // c-powers depend on the key and the column only and are staged into the weights (as in a3)
                const float t3 = fx3 - xs;
                const float nAt = negA * t3;
                const float Lf = fminf(fmaxf(fmaf(nAt, 2.0f, negA), -120.f), 120.f);   // 2^+-Lf finite; beyond, G3 is 0
                const float G3 = ex2s(fmaf(nAt, t3, Es));
                const float rf = ex2s(Lf), rb = ex2s(-Lf);
                const f32x2 R = pk2(rb, rf);
                Pp[0] = pk2(G3, G3 * rf);
                Pp[1] = mul2(Pp[0], R);
                Pp[2] = mul2(Pp[1], R);
                Pp[3] = mul2(Pp[2], R);
            } else {
                #pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float tl = fx3 - (float)q - xs, th = fx3 + 1.f + (float)q - xs;
                    Pp[q] = pk2(ex2s(fmaf(negA * tl, tl, Es)), ex2s(fmaf(negA * th, th, Es)));
                }
            }
            fma2_acc(acc[0], acc[1], Pp[0], pk2(wa.x, wa.y));
            fma2_acc(acc[2], acc[3], Pp[1], pk2(wa.z, wa.w));
            fma2_acc(acc[4], acc[5], Pp[2], pk2(wb.x, wb.y));
            fma2_acc(acc[6], acc[7], Pp[3], pk2(wb.z, wb.w));
        }
    }
    if (kSplatFwdWarps > 1) {
        if (warp > 0) {
            #pragma unroll
            for (int k = 0; k < 8; ++k) s_part[warp - 1][k][lane] = acc[k];
        }
        __syncthreads();
        if (warp > 0) return;
        #pragma unroll
        for (int w = 0; w < kSplatFwdWarps - 1; ++w)
            #pragma unroll
            for (int k = 0; k < 8; ++k) acc[k] += s_part[w][k][lane];
    }
    const int py = oy + row;
    if (py < P.nv) {
        float* o = drr + ((size_t)b * P.nv + py) * P.nu + ox + 8 * seg;
        #pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int xl = ox + 8 * seg + 3 - q, xh = ox + 8 * seg + 4 + q;
            if (xl < P.nu) o[3 - q] = acc[2 * q];
            if (xh < P.nu) o[4 + q] = acc[2 * q + 1];
        }
    }
}

// s4: one CTA (128 threads) per (tile, angle); the tile's upstream gradient in shared memory; ONE
// THREAD PER KEY walks box ∩ tile and reduces the six raw moments of g E about the centre in
// registers:  m = sum g E {1, dx, dy, dx^2, dx dy, dy^2};  one vector atomic set per key.
// The 32 keys of a warp should have similar trip counts: the CTA counting-sorts its keys, 1024 at a
// time, into 64 shape classes (rows/2 x columns/2 of box ∩ tile) in shared memory first (measured
// 16.9 of 32 lanes active unsorted).
constexpr int kSplatBwdThreads = 128;
constexpr int kSplatBwdChunk = 1024;

__global__ void __launch_bounds__(kSplatBwdThreads)
k_splat_backward(SplatParams P, const Splat2D* __restrict__ rec, const uint32_t* __restrict__ bin_start,
                 const uint32_t* __restrict__ keys, const SplatStatus* __restrict__ status, unsigned long long stamp,
                 const float* __restrict__ gdrr, float* __restrict__ acc)
{
    __shared__ float s_g[kSplatTile * kSplatTile];
    __shared__ uint32_t s_key[kSplatBwdChunk], s_sorted[kSplatBwdChunk];
    __shared__ uint8_t s_cls[kSplatBwdChunk];
    __shared__ uint32_t s_hist[64];
    if (status->overflow || status->stamp != stamp) return;
    const int tid = threadIdx.x, tile = blockIdx.x, b = blockIdx.y;
    const uint32_t kbeg = bin_start[b * P.ntx * P.nty + tile], kend = bin_start[b * P.ntx * P.nty + tile + 1];
    if (kbeg == kend) return;
    const int tx = tile % P.ntx, ty = tile / P.ntx;
    const int ox = tx * kSplatTile, oy = ty * kSplatTile;
    for (int e = tid; e < kSplatTile * kSplatTile; e += kSplatBwdThreads) {
        const int px = ox + (e & 15), py = oy + (e >> 4);
        s_g[e] = (px < P.nu && py < P.nv) ? __ldg(gdrr + ((size_t)b * P.nv + py) * P.nu + px) : 0.f;
    }
    for (uint32_t base = kbeg; base < kend; base += kSplatBwdChunk) {
        const int nc = (int)min((uint32_t)kSplatBwdChunk, kend - base);
        if (tid < 64) s_hist[tid] = 0u;
        __syncthreads();
        for (int i = tid; i < nc; i += kSplatBwdThreads) {
            const uint32_t id = keys[base + i];
            const int w1 = __ldg(reinterpret_cast<const int*>(rec + id) + 7), w2 = __ldg(reinterpret_cast<const int*>(rec + id) + 8);
            const int u0 = (int16_t)(w1 & 0xffff), v0 = (int16_t)(w1 >> 16), u1 = (int16_t)(w2 & 0xffff), v1 = (int16_t)(w2 >> 16);
            const int nx = min(u1 - ox, kSplatTile - 1) - max(u0 - ox, 0), ny = min(v1 - oy, kSplatTile - 1) - max(v0 - oy, 0);
            const int cls = ((ny >> 1) << 3) | (nx >> 1);
            s_key[i] = id; s_cls[i] = (uint8_t)cls;
            atomicAdd(&s_hist[cls], 1u);
        }
        __syncthreads();
        if (tid < 32) {                                         // exclusive scan of the 64 class counts
            const uint32_t a0 = s_hist[2 * tid], a1 = s_hist[2 * tid + 1];
            uint32_t inc = a0 + a1;
            for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (tid >= o) inc += t; }
            s_hist[2 * tid] = inc - a0 - a1; s_hist[2 * tid + 1] = inc - a1;
        }
        __syncthreads();
        for (int i = tid; i < nc; i += kSplatBwdThreads) s_sorted[atomicAdd(&s_hist[s_cls[i]], 1u)] = s_key[i];
        __syncthreads();
        for (int i = tid; i < nc; i += kSplatBwdThreads) {
            const uint32_t id = s_sorted[i];
            const float4* rp = reinterpret_cast<const float4*>(rec + id);
            const float4 a = __ldg(rp), c = __ldg(rp + 1);
            const int4 w = __ldg(reinterpret_cast<const int4*>(rp + 2));
            const float cfu = a.x, cfv = a.y, A = a.z;                                // c.y = amp (applied in s5)
            const float Bq = __int_as_float(w.y), Dq = __int_as_float(w.z);           // row form: E = A t^2 + Dq dy^2, t = dx + Bq dy
            const int ciu = (int16_t)(__float_as_int(c.z) & 0xffff), civ = (int16_t)(__float_as_int(c.z) >> 16);
            const int u0 = (int16_t)(__float_as_int(c.w) & 0xffff), v0 = (int16_t)(__float_as_int(c.w) >> 16);
            const int u1 = (int16_t)(w.x & 0xffff), v1 = (int16_t)(w.x >> 16);
            const int x0 = max(u0 - ox, 0), x1 = min(u1 - ox, kSplatTile - 1), y0 = max(v0 - oy, 0), y1 = min(v1 - oy, kSplatTile - 1);
            // Moments of g E about the centre in the SHEARED frame (t, dy), t = dx + Bq dy = distance from the row's ridge:
            // for an elongated footprint t is the transverse coordinate, and sum g E t^2 is summed directly instead of
            // being the small difference of raw dx/dy moments (fp32 raw moments lost (s_max/s_min)^2: a 34:1 needle seen
            // at 240:1 in 2D had its scale/quaternion gradients off by 1.7e-4).  s5 goes back to raw moments in fp64.
            float m0 = 0.f, mt = 0.f, my = 0.f, mtt = 0.f, mty = 0.f, myy = 0.f;
            for (int y = y0; y <= y1; ++y) {
                const float dy = (float)(oy + y - civ) - cfv;
                const float ey = Dq * dy * dy, sh = fmaf(Bq, dy, -cfu);
                float r0 = 0.f, r1 = 0.f, r2 = 0.f;               // row sums of g E {1, t, t^2}
                for (int x = x0; x <= x1; ++x) {
                    const float t = (float)(ox + x - ciu) + sh;
                    const float gE = s_g[y * kSplatTile + x] * ex2s(fmaf(A * t, t, ey));
                    r0 += gE; const float q = gE * t; r1 += q; r2 = fmaf(q, t, r2);
                }
                m0 += r0; mt += r1; mtt += r2;
                my = fmaf(dy, r0, my); mty = fmaf(dy, r1, mty); myy = fmaf(dy * dy, r0, myy);
            }
            float* dst = acc + (size_t)id * 8;
            asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(dst), "f"(m0), "f"(mt), "f"(my), "f"(mtt) : "memory");
            asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" :: "l"(dst + 4), "f"(mty), "f"(myy) : "memory");
        }
        __syncthreads();                                        // s_key / s_hist are reused by the next chunk
    }
}

// s5: chain rule, one thread per Gaussian, fp64, summed over the angles in a loop (no atomics).
// Upstream per (angle, Gaussian): the raw moments m = sum g E {1, dx, dy, dx^2, dx dy, dy^2} of s4.
//   value = amp E,  E = exp(-1/2 q),  q = A dx^2 + 2 B dx dy + C dy^2,  dx = iu - cu,  [A B; B C] = P^-1
//   dL/damp = m0;  dL/dA = -amp mxx / 2;  dL/dB = -amp mxy;  dL/dC = -amp myy / 2
//   dL/dcu = amp (A mx + B my);  dL/dcv = amp (B mx + C my)
// then back through P = K Sigma^ K, amp = rho sqrt(2 pi |Sigma~| / |Sigma^|), Sigma~ = T Sigma T^T,
// T = J(t) W, t = W (p - source), Sigma = R S^2 R^T, R(q / |q|).
__global__ void __launch_bounds__(128, 4)
k_splat_epilogue(SplatParams P, const float* __restrict__ pos, const float* __restrict__ scale, const float* __restrict__ quat,
                 const float* __restrict__ rho, const Splat2D* __restrict__ rec, const float* __restrict__ acc,
                 const SplatStatus* __restrict__ status, unsigned long long stamp,
                 float* __restrict__ grho, float* __restrict__ gpos, float* __restrict__ gscale, float* __restrict__ gquat)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= P.n) return;
    double d_rho = 0.0, d_p[3] = { 0, 0, 0 }, d_Sig[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };
    const double rh = (double)rho[g];
    SplatTerms o;
    o.valid = false;
    const bool ready = !status->overflow && status->stamp == stamp;      // else: zero gradients
    for (int b = 0; b < P.B && ready; ++b) {
        const size_t idx = (size_t)b * P.n + g;
        if (rec[idx].u1 < rec[idx].u0) continue;               // skipped or off the detector at this angle
        splat_terms(P, b, pos, scale, quat, g, o);
        if (!o.valid) continue;
        const float* m = acc + idx * 8;
        // sheared-frame moments (t = dx + Bq dy, with the Bq the kernel used) -> raw moments, in fp64
        const double bq = (double)rec[idx].Bq;
        const double m0 = m[0], my = m[2], myy = m[5];
        const double mx = m[1] - bq * my, mxy = m[4] - bq * myy, mxx = m[3] - 2.0 * bq * m[4] + bq * bq * myy;
        const double amp = rh * o.amp_over_rho;
        const double A = o.P[2] / o.dp, Bc = -o.P[1] / o.dp, C = o.P[0] / o.dp;
        const double g_amp = m0, gA = -0.5 * amp * mxx, gB = -amp * mxy, gC = -0.5 * amp * myy;
        const double g_cu = amp * (A * mx + Bc * my), g_cv = amp * (Bc * mx + C * my);
        d_rho += g_amp * o.amp_over_rho;
        // conic -> P:  GP = -Pinv Gc Pinv,  Gc = [[gA, gB/2], [gB/2, gC]]
        const double c00 = gA, c01 = 0.5 * gB, c11 = gC;
        const double x00 = A * c00 + Bc * c01, x01 = A * c01 + Bc * c11, x10 = Bc * c00 + C * c01, x11 = Bc * c01 + C * c11;
        const double GP00 = -(x00 * A + x01 * Bc), GP01 = -(x00 * Bc + x01 * C), GP11 = -(x10 * Bc + x11 * C);
        const double ku = P.sdd / P.du, kv = P.sdd / P.dv;
        double GS[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };           // symmetric matrix gradient wrt Sigma~
        GS[0] = GP00 * ku * ku; GS[4] = GP11 * kv * kv; GS[1] = GS[3] = GP01 * ku * kv;
        // amplitude: amp = rho sqrt(2 pi det_t / det_h)
        const double g_dett = g_amp * amp / (2.0 * o.det_t), g_deth = -g_amp * amp / (2.0 * o.det_h);
        const double* S = o.St;
        GS[0] += g_deth * S[4]; GS[4] += g_deth * S[0]; GS[1] -= g_deth * S[1]; GS[3] -= g_deth * S[1];
        // d det_t = adj(Sigma~) : d Sigma~   (adjugate = cofactors, Sigma~ symmetric)
        const double adj[9] = { S[4] * S[8] - S[5] * S[7], S[2] * S[7] - S[1] * S[8], S[1] * S[5] - S[2] * S[4],
                                S[5] * S[6] - S[3] * S[8], S[0] * S[8] - S[2] * S[6], S[2] * S[3] - S[0] * S[5],
                                S[3] * S[7] - S[4] * S[6], S[1] * S[6] - S[0] * S[7], S[0] * S[4] - S[1] * S[3] };
        for (int k = 0; k < 9; ++k) GS[k] += g_dett * adj[k];
        // Sigma~ = T Sigma T^T:  dL/dSigma += T^T GS T;  dL/dT = 2 GS T Sigma
        double Tt[9], GT[9], tmp[9], tmp2[9];
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Tt[3 * i + j] = o.T[3 * j + i];
        mat3mul(Tt, GS, tmp); mat3mul(tmp, o.T, tmp2);
        for (int k = 0; k < 9; ++k) d_Sig[k] += tmp2[k];
        mat3mul(GS, o.T, tmp); mat3mul(tmp, o.Sig, GT);
        for (int k = 0; k < 9; ++k) GT[k] *= 2.0;
        // T = J W:  dL/dJ = dL/dT W^T
        double W[9], src[3], Wt[9], GJ[9];
        splat_W(P, b, W, src);
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Wt[3 * i + j] = W[3 * j + i];
        mat3mul(GT, Wt, GJ);
        // J(t) and the centre (cu, cv) -> t
        const double t0 = o.t[0], t1 = o.t[1], t2 = o.t[2], l = o.ell, l3 = l * l * l, it2 = 1.0 / (t2 * t2), it3 = it2 / t2;
        double gt[3];
        gt[0] = -GJ[2] * it2 + GJ[6] * (1.0 / l - t0 * t0 / l3) - GJ[7] * t0 * t1 / l3 - GJ[8] * t0 * t2 / l3 + g_cu * ku / t2;
        gt[1] = -GJ[5] * it2 - GJ[6] * t0 * t1 / l3 + GJ[7] * (1.0 / l - t1 * t1 / l3) - GJ[8] * t1 * t2 / l3 + g_cv * kv / t2;
        gt[2] = -(GJ[0] + GJ[4]) * it2 + 2.0 * (GJ[2] * t0 + GJ[5] * t1) * it3 - (GJ[6] * t0 + GJ[7] * t1) * t2 / l3
              + GJ[8] * (1.0 / l - t2 * t2 / l3) - (g_cu * ku * t0 + g_cv * kv * t1) * it2;
        for (int k = 0; k < 3; ++k) d_p[k] += W[k] * gt[0] + W[3 + k] * gt[1] + W[6 + k] * gt[2];   // W^T gt
    }
    grho[g] = (float)d_rho;
    for (int k = 0; k < 3; ++k) gpos[3 * g + k] = (float)d_p[k];
    // Sigma = R S^2 R^T  (R, s from the parameters; independent of the angle)
    const double s[3] = { scale[3 * g], scale[3 * g + 1], scale[3 * g + 2] };
    const double q[4] = { quat[4 * g], quat[4 * g + 1], quat[4 * g + 2], quat[4 * g + 3] };
    const double n2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3];
    bool bad = !(n2 > 0.0) || !isfinite(n2);
    for (int k = 0; k < 3; ++k) bad |= !(s[k] > 0.0) || !isfinite(s[k]);
    if (bad) {
        for (int k = 0; k < 3; ++k) gscale[3 * g + k] = 0.f;
        for (int k = 0; k < 4; ++k) gquat[4 * g + k] = 0.f;
        return;
    }
    const double qn = sqrt(n2), r = q[0] / qn, x = q[1] / qn, y = q[2] / qn, z = q[3] / qn;
    const double R[9] = { 1 - 2 * (y * y + z * z), 2 * (x * y - r * z), 2 * (x * z + r * y),
                          2 * (x * y + r * z), 1 - 2 * (x * x + z * z), 2 * (y * z - r * x),
                          2 * (x * z - r * y), 2 * (y * z + r * x), 1 - 2 * (x * x + y * y) };
    // dL/ds_k = 2 s_k (R^T G R)_kk;  D_R = 2 G R S^2   (G = d_Sig, symmetric)
    double GR[9], DR[9];
    mat3mul(d_Sig, R, GR);
    for (int k = 0; k < 3; ++k) {
        const double d = R[k] * GR[k] + R[3 + k] * GR[3 + k] + R[6 + k] * GR[6 + k];
        gscale[3 * g + k] = (float)(2.0 * s[k] * d);
    }
    for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) DR[3 * i + k] = 2.0 * GR[3 * i + k] * s[k] * s[k];
    double gh[4];
    gh[0] = 2 * (-z * DR[1] + y * DR[2] + z * DR[3] - x * DR[5] - y * DR[6] + x * DR[7]);
    gh[1] = 2 * (y * DR[1] + z * DR[2] + y * DR[3] - 2 * x * DR[4] - r * DR[5] + z * DR[6] + r * DR[7] - 2 * x * DR[8]);
    gh[2] = 2 * (-2 * y * DR[0] + x * DR[1] + r * DR[2] + x * DR[3] + z * DR[5] - r * DR[6] + z * DR[7] - 2 * y * DR[8]);
    gh[3] = 2 * (-2 * z * DR[0] - r * DR[1] + x * DR[2] + r * DR[3] - 2 * z * DR[4] + y * DR[5] + x * DR[6] + y * DR[7]);
    const double qh[4] = { r, x, y, z };
    const double dot = qh[0] * gh[0] + qh[1] * gh[1] + qh[2] * gh[2] + qh[3] * gh[3];
    for (int k = 0; k < 4; ++k) gquat[4 * g + k] = (float)((gh[k] - qh[k] * dot) / qn);
}

}  // namespace gsvox

using namespace gsvox;

static size_t sup256(size_t v) { return (v + 255) & ~(size_t)255; }

static int splat_setup(int64_t n, const gsvox_cone_geometry* c, const float* angles_host, int32_t B,
                       int64_t key_capacity, void* workspace, size_t workspace_bytes, SplatParams* P, SplatWs* ws)
{
    if (!c || n < 0 || B < 1 || B > kSplatMaxBatch || key_capacity < 0) return GSVOX_EINVAL;
    if (!(c->sad > 0.f) || !(c->sdd > 0.f) || c->nu < 1 || c->nv < 1 || !(c->du > 0.f) || !(c->dv > 0.f)) return GSVOX_EINVAL;
    if (c->nu > GSVOX_MAX_DIM || c->nv > GSVOX_MAX_DIM || n * (int64_t)B > 0x7ffffff0LL || key_capacity > 0xfffffff0LL) return GSVOX_ELIMIT;
    P->n = (int)n; P->B = B; P->nu = c->nu; P->nv = c->nv;
    P->ntx = (c->nu + kSplatTile - 1) / kSplatTile; P->nty = (c->nv + kSplatTile - 1) / kSplatTile;
    P->sad = c->sad; P->sdd = c->sdd; P->du = c->du; P->dv = c->dv; P->off_u = c->off_u; P->off_v = c->off_v;
    for (int k = 0; k < 3; ++k) P->iso[k] = c->iso[k];
    if (angles_host) for (int b = 0; b < B; ++b) { P->ca[b] = cos((double)angles_host[b]); P->sa[b] = sin((double)angles_host[b]); }
    const long long nbins = (long long)P->ntx * P->nty * B;
    if (nbins > 0x7ffffff0LL || P->ntx * (long long)P->nty > 0x7fffffffLL) return GSVOX_ELIMIT;
    ws->nbins = (int)nbins;
    size_t off = 0;
    char* w = (char*)workspace;
    ws->status = (SplatStatus*)(w + off);  off += sup256(sizeof(SplatStatus));      // status and bin_count contiguous: one memset
    ws->bin_count = (uint32_t*)(w + off);  off += sup256(sizeof(uint32_t) * (size_t)(nbins + 1));
    ws->bin_start = (uint32_t*)(w + off);  off += sup256(sizeof(uint32_t) * (size_t)(nbins + 1));
    ws->partial = (uint32_t*)(w + off);    off += sup256(sizeof(uint32_t) * (size_t)((nbins + kScanItemsPerBlock - 1) / kScanItemsPerBlock + 1));
    ws->rec = (Splat2D*)(w + off);         off += sup256(sizeof(Splat2D) * (size_t)n * B);
    ws->keys = (uint32_t*)(w + off);       off += sup256(sizeof(uint32_t) * (size_t)key_capacity);
    ws->acc = (float*)(w + off);           off += sup256(sizeof(float) * 8 * (size_t)n * B);
    ws->total = off;
    if (workspace && (((uintptr_t)workspace & 255) || workspace_bytes < off)) return GSVOX_EWORKSPACE;
    return GSVOX_OK;
}

extern "C" int gsvox_splat_workspace_bytes(int64_t n, const gsvox_cone_geometry* geom, int32_t B,
                                           int64_t key_capacity, size_t* bytes)
{
    if (!bytes) return GSVOX_EINVAL;
    SplatParams P; SplatWs ws;
    int rc = splat_setup(n, geom, nullptr, B, key_capacity, nullptr, 0, &P, &ws);
    if (rc == GSVOX_OK) *bytes = ws.total;
    return rc;
}

extern "C" int gsvox_splat_forward(const float* pos, const float* scale, const float* quat, const float* rho,
                                   int64_t n, const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                                   void* workspace, size_t workspace_bytes, int64_t key_capacity,
                                   float* drr, void* stream)
{
    if (!workspace || !angles_host || !drr) return GSVOX_EINVAL;
    if (n > 0 && (!pos || !scale || !quat || !rho)) return GSVOX_EINVAL;
    SplatParams P; SplatWs ws;
    int rc = splat_setup(n, geom, angles_host, B, key_capacity, workspace, workspace_bytes, &P, &ws);
    if (rc != GSVOX_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    GSVOX_CUDA(cudaMemsetAsync(ws.status, 0, (size_t)((char*)ws.bin_count - (char*)ws.status) + sizeof(uint32_t) * (size_t)(ws.nbins + 1), st));
    const long long items = (long long)n * B;
    if (items > 0) {
        k_splat_pre<<<(unsigned)((items + 127) / 128), 128, 0, st>>>(P, pos, scale, quat, rho, ws.rec, ws.bin_count, ws.status);
        GSVOX_CUDA(cudaGetLastError());
    }
    const int tiles = P.ntx * P.nty;
    const size_t sort_smem = (tiles <= kSplatMaxTilesShared) ? sizeof(uint32_t) * 2 * (size_t)tiles : 0;
    dim3 sgrid((unsigned)((n + kSplatSortThreads - 1) / kSplatSortThreads), (unsigned)B);
    if (sort_smem > 48 * 1024) {
        GSVOX_CUDA(cudaFuncSetAttribute(k_splat_sort<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem));
        GSVOX_CUDA(cudaFuncSetAttribute(k_splat_sort<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem));
    }
    if (items > 0) {
        k_splat_sort<0><<<sgrid, kSplatSortThreads, sort_smem, st>>>(P, ws.rec, ws.bin_count, ws.keys, ws.status);
        GSVOX_CUDA(cudaGetLastError());
    }
    rc = launch_exclusive_scan(ws.bin_count, ws.nbins, ws.partial, ws.bin_start, &ws.status->keys_needed,
                               &ws.status->overflow, (unsigned long long)key_capacity, st);
    if (rc != GSVOX_OK) return rc;
    if (items > 0) {
        k_splat_sort<1><<<sgrid, kSplatSortThreads, sort_smem, st>>>(P, ws.rec, ws.bin_count, ws.keys, ws.status);
        GSVOX_CUDA(cudaGetLastError());
    }
    dim3 grid((unsigned)(P.ntx * P.nty), (unsigned)B);
    k_splat_forward<<<grid, 32 * kSplatFwdWarps, 0, st>>>(P, ws.rec, ws.bin_start, ws.keys, ws.status,
                                                          splat_stamp(n, B, P.nu, P.nv, key_capacity), drr);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

extern "C" int gsvox_splat_backward(const float* pos, const float* scale, const float* quat, const float* rho,
                                    int64_t n, const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                                    void* workspace, size_t workspace_bytes, int64_t key_capacity,
                                    const float* grad_drr, float* grad_rho, float* grad_pos, float* grad_scale,
                                    float* grad_quat, void* stream)
{
    if (!workspace || !angles_host || !grad_drr) return GSVOX_EINVAL;
    if (n > 0 && (!pos || !scale || !quat || !rho || !grad_rho || !grad_pos || !grad_scale || !grad_quat)) return GSVOX_EINVAL;
    SplatParams P; SplatWs ws;
    int rc = splat_setup(n, geom, angles_host, B, key_capacity, workspace, workspace_bytes, &P, &ws);
    if (rc != GSVOX_OK) return rc;
    if (n == 0) return GSVOX_OK;
    cudaStream_t st = (cudaStream_t)stream;
    GSVOX_CUDA(cudaMemsetAsync(ws.acc, 0, sizeof(float) * 8 * (size_t)n * B, st));
    dim3 grid((unsigned)(P.ntx * P.nty), (unsigned)B);
    const unsigned long long stamp = splat_stamp(n, B, P.nu, P.nv, key_capacity);
    k_splat_backward<<<grid, kSplatBwdThreads, 0, st>>>(P, ws.rec, ws.bin_start, ws.keys, ws.status, stamp, grad_drr, ws.acc);
    GSVOX_CUDA(cudaGetLastError());
    k_splat_epilogue<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(P, pos, scale, quat, rho, ws.rec, ws.acc, ws.status, stamp,
                                                                 grad_rho, grad_pos, grad_scale, grad_quat);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

extern "C" int gsvox_splat_status(const void* workspace, int64_t* keys_needed, int64_t* pairs, int32_t* overflow,
                                  int32_t* skipped, void* stream)
{
    if (!workspace) return GSVOX_EINVAL;
    SplatStatus h;
    cudaStream_t st = (cudaStream_t)stream;
    GSVOX_CUDA(cudaMemcpyAsync(&h, workspace, sizeof h, cudaMemcpyDeviceToHost, st));
    GSVOX_CUDA(cudaStreamSynchronize(st));
    if ((h.stamp >> 32) != (kSplatMagic >> 32)) return GSVOX_ENOTREADY;      // no gsvox_splat_forward completed on this workspace
    if (keys_needed) *keys_needed = (int64_t)h.keys_needed;
    if (pairs) *pairs = (int64_t)h.pairs;
    if (overflow) *overflow = (int32_t)h.overflow;
    if (skipped) *skipped = (int32_t)h.skipped;
    return GSVOX_OK;
}

extern "C" int gsvox_splat_drops(const void* workspace, int64_t* behind_source, int64_t* out_of_range, int64_t* empty_box,
                                 void* stream)
{
    if (!workspace) return GSVOX_EINVAL;
    SplatStatus h;
    cudaStream_t st = (cudaStream_t)stream;
    GSVOX_CUDA(cudaMemcpyAsync(&h, workspace, sizeof h, cudaMemcpyDeviceToHost, st));
    GSVOX_CUDA(cudaStreamSynchronize(st));
    if ((h.stamp >> 32) != (kSplatMagic >> 32)) return GSVOX_ENOTREADY;
    if (behind_source) *behind_source = (int64_t)h.drop_behind;
    if (out_of_range) *out_of_range = (int64_t)h.drop_range;
    if (empty_box) *empty_box = (int64_t)h.drop_empty;
    return GSVOX_OK;
}
