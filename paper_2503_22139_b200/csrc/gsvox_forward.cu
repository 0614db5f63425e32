// gsvox_forward.cu — step a3: per-brick forward accumulation (Eq. 5).
//
// Two kernels: k_forward<CH> (CH = 9: the motion-basis fields, channel groups of a wider C) described here, and
// k_forward_b1<CH> (CH = 1: the CBCT volume, the headline configuration; CH = 3: one DVF level) further down,
// which re-cuts the same row arithmetic around what actually limits it — operand delivery through shared memory.
// (Nine channels as three b1<3> passes measured slower than k_forward<9>: 0.75/1.0/0.98 vs 0.50/0.70/0.62 ms on
// config 3's levels; two rows x nine channels of accumulators do not fit a thread.)
//
// k_forward<CH>: one CTA of 64 threads per 8^3 brick; thread t owns the x-row (y = t&7, z = t>>3) of the brick,
// i.e. 8 consecutive voxels per channel, accumulated in registers and written once.  The brick's
// keys are staged 64 at a time into shared memory: each thread gathers one 64-byte Gaussian
// record (four LDG.128, L2-resident: a record is shared by ~20 bricks), rebases the centre to
// brick-local coordinates and derives the brick-local row masks (which of the 64 rows lie inside
// the Gaussian's box in y,z) and, for C = 1, the eight per-voxel weights w·[k inside the box in x],
// so that full and x-partial keys run the same branch-free code.  Warps then walk the staged
// batch; a warp whose 32 rows miss the box skips the key.
//
// Along a row the exponent of Eq. 4 is the parabola E(k) = Es - A (k - xs)^2 (base 2), with
// xs, Es from the LDL^T form of the record (sum of squares, no cancellation).  For A <= 1 the
// eight values are produced by a centre-out multiplicative recurrence from k = 3:
//     G(k+1) = G(k) r(k),  r(k+1) = r(k) c,  c = 2^(-2A)      (exact identity for a parabola)
// 3 MUFU.EX2 + 14 FMUL per row instead of 8 MUFU: the kernel is then FMA/issue bound, not
// MUFU bound (16 vs 128 lanes/clk/SM).  Narrow Gaussians (A > 1, under ~0.85 voxel along x)
// take the direct path, one EX2 per voxel: the recurrence would lose accuracy and could
// underflow there (error budget).  Direct keys are class 0 of the brick's
// key range, so which path a staged key takes is known from bin_start, not from its data.
#include "gsvox_internal.cuh"

namespace gsvox {

constexpr int kFwdThreads = 64;
constexpr int kFwdBatch = 64;      // keys staged per __syncthreads.  Measured on config 4: batch 32/48 and forcing
                                   // 24-32 resident CTAs (<= 40 / 32 registers) are 2-25 % slower than this.

__device__ __forceinline__ float ex2f(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Shared-memory record of a staged key (floats); pairs that feed packed (f32x2) instructions sit on
// even word offsets so that one LDS.128 delivers them as aligned register pairs:
//   0 cx  1 cy  2 cz  3 -A | 4 -l01  5 -l02  6 l12  7 -D1 | 8 -D2  9 (unused)  10 c  11 c
//   CH == 1: 12..19  w * [k inside the box in x] in the order k = 3,4, 2,5 | 1,6, 0,7
//   CH  > 1: 12 xmask, 13.. weights (scalar arithmetic: packed FFMA2 measured slower there)
// The brick-local row masks (one word per warp) live in a separate array.
template <int CH> struct FwdRec { static constexpr int kWords = (CH == 1) ? 20 : ((13 + CH + 3) & ~3); };

template <int CH>
__device__ __forceinline__ void stage_key(float* __restrict__ dst, uint32_t* __restrict__ mask0,
                                          uint32_t* __restrict__ mask1, const GsRec* __restrict__ rec,
                                          const float* __restrict__ weight, int wstride, int c0,
                                          uint32_t gid, int b0x, int b0y, int b0z)
{
    const float4* rp = reinterpret_cast<const float4*>(rec + gid);
    float4 a = __ldg(rp), b = __ldg(rp + 1), c = __ldg(rp + 2), d = __ldg(rp + 3);
    // a = cf.xyz, cexp | b = ci.xyz, negA | c = nl01, nl02, l12, nD1 | d = nD2, lo/hi packed
    int cix = __float_as_int(b.x), ciy = __float_as_int(b.y), ciz = __float_as_int(b.z);
    int w1 = __float_as_int(d.y), w2 = __float_as_int(d.z), w3 = __float_as_int(d.w);
    int lox = (int16_t)(w1 & 0xffff), loy = (int16_t)(w1 >> 16), loz = (int16_t)(w2 & 0xffff);
    int hix = (int16_t)(w2 >> 16), hiy = (int16_t)(w3 & 0xffff), hiz = (int16_t)(w3 >> 16);
    int x0 = max(lox - b0x, 0), x1 = min(hix - b0x, 7);
    int y0 = max(loy - b0y, 0), y1 = min(hiy - b0y, 7);
    int z0 = max(loz - b0z, 0), z1 = min(hiz - b0z, 7);
    uint32_t ym = ((2u << y1) - (1u << y0)) & 0xffu;               // bits y0..y1
    uint32_t zm = ((2u << z1) - (1u << z0)) & 0xffu;
    uint32_t xm = ((2u << x1) - (1u << x0)) & 0xffu;
    uint32_t rep = ym * 0x01010101u;                                // ym in all four bytes
    uint32_t sel0 = ((zm & 1u) ? 0xffu : 0u) | ((zm & 2u) ? 0xff00u : 0u) |
                    ((zm & 4u) ? 0xff0000u : 0u) | ((zm & 8u) ? 0xff000000u : 0u);
    uint32_t zh = zm >> 4;
    uint32_t sel1 = ((zh & 1u) ? 0xffu : 0u) | ((zh & 2u) ? 0xff00u : 0u) |
                    ((zh & 4u) ? 0xff0000u : 0u) | ((zh & 8u) ? 0xff000000u : 0u);
    *mask0 = rep & sel0;
    *mask1 = rep & sel1;
    float4* o = reinterpret_cast<float4*>(dst);
    o[0] = make_float4((float)(cix - b0x) + a.x, (float)(ciy - b0y) + a.y, (float)(ciz - b0z) + a.z, b.w);
    o[1] = make_float4(c.x, c.y, c.z, c.w);
    const float cc = fabsf(a.w);                                    // the sign bit is a2's cull flag
    o[2] = make_float4(d.x, 0.f, cc, cc);
    if (CH == 1) {
        const float w = __ldg(weight + (size_t)gid * wstride + c0);
        o[3] = make_float4((xm & 8u) ? w : 0.f, (xm & 16u) ? w : 0.f, (xm & 4u) ? w : 0.f, (xm & 32u) ? w : 0.f);
        o[4] = make_float4((xm & 2u) ? w : 0.f, (xm & 64u) ? w : 0.f, (xm & 1u) ? w : 0.f, (xm & 128u) ? w : 0.f);
    } else {
        dst[12] = __uint_as_float(xm);
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) dst[13 + ch] = __ldg(weight + (size_t)gid * wstride + c0 + ch);
    }
}

// One staged key against this thread's row.  DIRECT: one EX2 per voxel (narrow Gaussians).
// acc[ch][j] is the packed pair of voxels (3 - j, 4 + j): the two arms of the centre-out recurrence
// advance together, one FMUL2 per step.
template <int CH, bool DIRECT>
__device__ __forceinline__ void eval_key(const float* __restrict__ r, uint32_t mrow, uint32_t lanebit,
                                         float fy, float fz, float (&acc)[CH][8])
{
    if (mrow == 0u) return;                                         // none of this warp's 32 rows is in the box
    const float4 r0 = *reinterpret_cast<const float4*>(r);
    const float4 r1 = *reinterpret_cast<const float4*>(r + 4);
    const float4 r2 = *reinterpret_cast<const float4*>(r + 8);
    // row geometry: u2 = dz, u1 = dy + l12 dz, xs = cx - l01 dy - l02 dz
    const float dy = fy - r0.y, dz = fz - r0.z;
    const float u1 = fmaf(r1.z, dz, dy);
    const float xs = fmaf(r1.y, dz, fmaf(r1.x, dy, r0.x));
    float Es = fmaf(r2.x * dz, dz, (r1.w * u1) * u1);
    Es = (mrow & lanebit) ? Es : -1.0e30f;                          // rows outside the box contribute exact zeros
    const float negA = r0.w;
    if (CH == 1) {
        // packed pairs P[j] = (G[3-j], G[4+j]): the two arms of the centre-out recurrence advance together
        f32x2 P[4];
        if (!DIRECT) {
            const float t3 = 3.0f - xs;
            const float nAt = negA * t3;
            const float Lf = fminf(fmaf(nAt, 2.0f, negA), 120.f);  // E(4) - E(3), clamped: 0 * inf would be NaN
            const float Lb = fminf(fmaf(nAt, -2.0f, negA), 120.f); // E(2) - E(3)
            const f32x2 cc2 = pk2(r2.z, r2.w);
            const float G3 = ex2f(fmaf(nAt, t3, Es));
            const float rf = ex2f(Lf), rb = ex2f(Lb);
            const float G4 = G3 * rf;
            f32x2 R = pk2(rb, rf * r2.z);                           // (G2/G3, G5/G4)
            P[0] = pk2(G3, G4);
            P[1] = mul2(P[0], R); R = mul2(R, cc2);
            P[2] = mul2(P[1], R); R = mul2(R, cc2);
            P[3] = mul2(P[2], R);
        } else {
            #pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float tl = (float)(3 - j) - xs, th = (float)(4 + j) - xs;
                P[j] = pk2(ex2f(fmaf(negA * tl, tl, Es)), ex2f(fmaf(negA * th, th, Es)));
            }
        }
        const float4 wa = *reinterpret_cast<const float4*>(r + 12);
        const float4 wb = *reinterpret_cast<const float4*>(r + 16);
        fma2_acc(acc[0][0], acc[0][1], P[0], pk2(wa.x, wa.y));
        fma2_acc(acc[0][2], acc[0][3], P[1], pk2(wa.z, wa.w));
        fma2_acc(acc[0][4], acc[0][5], P[2], pk2(wb.x, wb.y));
        fma2_acc(acc[0][6], acc[0][7], P[3], pk2(wb.z, wb.w));
    } else {
        float G[8];
        if (!DIRECT) {
            const float t3 = 3.0f - xs;
            const float nAt = negA * t3;
            const float Lf = fminf(fmaf(nAt, 2.0f, negA), 120.f);
            const float Lb = fminf(fmaf(nAt, -2.0f, negA), 120.f);
            const float cc = r2.z;
            G[3] = ex2f(fmaf(nAt, t3, Es));
            float rf = ex2f(Lf), rb = ex2f(Lb);
            G[4] = G[3] * rf; rf *= cc; G[5] = G[4] * rf; rf *= cc; G[6] = G[5] * rf; rf *= cc; G[7] = G[6] * rf;
            G[2] = G[3] * rb; rb *= cc; G[1] = G[2] * rb; rb *= cc; G[0] = G[1] * rb;
        } else {
            #pragma unroll
            for (int k = 0; k < 8; ++k) { const float t = (float)k - xs; G[k] = ex2f(fmaf(negA * t, t, Es)); }
        }
        const uint32_t xm = __float_as_uint(r[12]);
        #pragma unroll
        for (int k = 0; k < 8; ++k) G[k] = (xm & (1u << k)) ? G[k] : 0.f;
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) {
            const float w = r[13 + ch];
            #pragma unroll
            for (int k = 0; k < 8; ++k) acc[ch][k] = fmaf(w, G[k], acc[ch][k]);
        }
    }
}

template <int CH, bool VEC>
__global__ void __launch_bounds__(kFwdThreads)
k_forward(const GsRec* __restrict__ rec, const uint32_t* __restrict__ bin_start,
          const uint32_t* __restrict__ keys, const DevStatus* __restrict__ status,
          const float* __restrict__ weight, int wstride, int c0,
          float* __restrict__ out, GridDev gd)
{
    constexpr int W = FwdRec<CH>::kWords;
    __shared__ __align__(16) float s_rec[2][kFwdBatch * W];
    __shared__ uint32_t s_mask[2][2][kFwdBatch];                    // [buffer][warp][key]

    const int tid = threadIdx.x;
    const int b = blockIdx.x + gd.slab0 * gd.nb[0] * gd.nb[1];      // bricks are z-major: a z-slab is a contiguous id range
    const int bx = b % gd.nb[0], by = (b / gd.nb[0]) % gd.nb[1], bz = b / (gd.nb[0] * gd.nb[1]);
    const int b0x = bx * kBrick, b0y = by * kBrick, b0z = bz * kBrick;
    const int ry = tid & 7, rz = tid >> 3;
    const float fy = (float)ry, fz = (float)rz;
    const int wsel = tid >> 5;
    const uint32_t lanebit = 1u << (tid & 31);

    float acc[CH][8];       // CH == 1: acc[0][2j], acc[0][2j+1] = voxels 3 - j, 4 + j (packed pair j); else x order
    #pragma unroll
    for (int ch = 0; ch < CH; ++ch)
        #pragma unroll
        for (int j = 0; j < 8; ++j) acc[ch][j] = 0.f;

    uint32_t kbeg = 0, kend = 0, kdirect = 0;
    if (!status->overflow) {
        kbeg = bin_start[b * kNumClasses]; kdirect = bin_start[b * kNumClasses + 1];
        kend = bin_start[(b + 1) * kNumClasses];
    }

    int buf = 0;
    for (uint32_t base = kbeg; base < kend; base += kFwdBatch, buf ^= 1) {
        float* sb = s_rec[buf];
        uint32_t k = base + tid;
        if (tid < kFwdBatch && k < kend) stage_key<CH>(sb + tid * W, &s_mask[buf][0][tid], &s_mask[buf][1][tid], rec, weight, wstride,
                                    c0, keys[k], b0x, b0y, b0z);
        __syncthreads();
        const uint32_t* mk = s_mask[buf][wsel];
        const int nb = (int)min((uint32_t)kFwdBatch, kend - base);
        const int nd = (kdirect > base) ? (int)min((uint32_t)nb, kdirect - base) : 0;   // class 0 comes first
        int j = 0;
        for (; j < nd; ++j) eval_key<CH, true>(sb + j * W, mk[j], lanebit, fy, fz, acc);
        #pragma unroll 2
        for (; j < nb; ++j) eval_key<CH, false>(sb + j * W, mk[j], lanebit, fy, fz, acc);
    }

    // write the row once (zeros for empty bricks); x fastest, [C, nz, ny, nx]
    const int gy = b0y + ry, gz = b0z + rz;
    if (gy < gd.dims[1] && gz < gd.dims[2]) {
        const size_t plane = (size_t)gd.dims[0] * gd.dims[1] * gd.dims[2];
        const size_t rowoff = ((size_t)gz * gd.dims[1] + gy) * gd.dims[0] + b0x;
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) {
            float v[8];
            #pragma unroll
            for (int j = 0; j < 4; ++j) {
                v[3 - j] = (CH == 1) ? acc[ch][2 * j] : acc[ch][3 - j];
                v[4 + j] = (CH == 1) ? acc[ch][2 * j + 1] : acc[ch][4 + j];
            }
            float* o = out + (size_t)(c0 + ch) * plane + rowoff;
            if (VEC) {
                if (b0x + 3 < gd.dims[0])
                    __stcs(reinterpret_cast<float4*>(o), make_float4(v[0], v[1], v[2], v[3]));
                if (b0x + 7 < gd.dims[0])
                    __stcs(reinterpret_cast<float4*>(o) + 1, make_float4(v[4], v[5], v[6], v[7]));
            } else {
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2)
                    if (b0x + k2 < gd.dims[0]) o[k2] = v[k2];
            }
        }
    }
}


// ==========================================================================================
// C = 1 and C = 3 fast path: one WARP per brick, two rows per thread.
//
// What binds k_forward above is not arithmetic but operand delivery: every key costs each of the brick's two
// warps ~21 words through LDS, and a warp-wide LDS.128 occupies the SM's one shared-memory return path for
// 2-4 cycles whether or not all lanes read the same address (ncu: l1tex 85-94 % busy, mio_throttle the
// top stall; a first pair-of-keys kernel that halved the instruction count ran SLOWER for that reason).
// Here a key's 20 words are loaded once per brick: the warp covers all 64 rows, thread (y, z) owning the
// rows (y, z) and (y, z + 4).  The row setup runs once for both rows in packed f32x2 instructions whose
// key operands are scalar registers broadcast to both halves (SASS: the .F32 operand form), so the staged
// record needs no interleaving; the three exponents per row then feed the centre-out recurrence of
// k_forward.  Per key: 5 LDS.128, ~12 setup + 2 x 13 row instructions, 6 EX2; shared-memory path, issue slots and
// the FP32 pipe (packed instructions take two pipe cycles) are about equally busy.  The batch's 64-byte records arrive
// by cp.async, issued one batch ahead; single-warp CTAs need no
// __syncthreads, 32 of them are resident per SM.
// Keys are staged class by class — slow | both z-halves | lower half only | upper half only — so each class runs
// its own branch-free loop (a half no row of which lies in the box is never evaluated).  "Slow" keys take a scalar route: direct-exponential keys (A > 1, class 0) and keys
// whose first ratio 2^Lf, 2^Lb could overflow on some row of the brick (A (1 + 2 max|t3|) >= 120: the fast
// path has no clamp — such rows hold nothing but zeros, yet inf * 0 must not be formed).
// ==========================================================================================
constexpr int kB1Batch = 32;
constexpr int kB1Words = 20;                        // staged record (C = 1); also the stride of the raw copy (16 words, padded): conflict-free 128-bit per-lane access
// CH > 1 (the motion-basis fields, groups of three channels): words 12..19 hold the key-and-k factor alone,
// km_k = [k inside the box in x] (fast keys: * c^{0,0,1,1,3,3,6,6}), words 20.. the CH weights; 28 words keep the
// per-lane 128-bit staging stores conflict-free (stride 24 would map eight lanes onto four bank groups).
template <int CH> struct B1Rec { static constexpr int kWords = (CH == 1) ? kB1Words : 28; };

__device__ __forceinline__ void red_add_v4f(float* addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void cp_async16(uint32_t saddr, const void* g)
{ asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" :: "r"(saddr), "l"(g) : "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// staged record (floats):  0 cx3  1 ncy  2 ncz  3 negA | 4 l01  5 l02  6 l12  7 nD1 | 8 nD2  9 +-c  10 mask(z 0..3)  11 mask(z 4..7)
//                          12..19  w * [k inside the box in x] (fast keys: * c^{0,0,1,1,3,3,6,6}) in the order k = 3,4, 2,5 | 1,6, 0,7
// cx3 = 3 - cx, ncy = -cy, ncz = -cz, l01 = +l01, l02 = +l02:  t3 = 3 - xs = cx3 + l01 dy + l02 dz.

// One row from its two exponents: E3 (value at k = 3) and Lf = E(4) - E(3).  The row is the parabola
// E(k) = E3 + (k - 3) Lf - A (k - 3)(k - 4), so  G(k) = G3 rho^(k-3) c^((k-3)(k-4)/2),  rho = 2^Lf, c = 2^-2A:
// a plain geometric sequence times a factor that depends on the key and k only — staged into the weights
// (w'_k = w [k in box] c^{0,0,1,1,3,3,6,6} in the centre-out order).  One FMUL + three FMUL2 for eight values.
// G3 rho^(k-3) never overflows for A <= 1: its exponent is Es - A (t3 +- ...)^2 + 12 A <= 12.
__device__ __forceinline__ void recur_accumulate(float E3, float Lf, const float4 wa, const float4 wb, float (&acc)[8])
{
    const float G3 = ex2f(E3), rf = ex2f(Lf), rb = ex2f(-Lf);
    const float G4 = G3 * rf;
    const f32x2 R = pk2(rb, rf);
    const f32x2 P0 = pk2(G3, G4);
    const f32x2 P1 = mul2(P0, R);
    const f32x2 P2 = mul2(P1, R);
    const f32x2 P3 = mul2(P2, R);
    fma2_acc(acc[0], acc[1], P0, pk2(wa.x, wa.y));
    fma2_acc(acc[2], acc[3], P1, pk2(wa.z, wa.w));
    fma2_acc(acc[4], acc[5], P2, pk2(wb.x, wb.y));
    fma2_acc(acc[6], acc[7], P3, pk2(wb.z, wb.w));
}

// CH > 1: the same eight values, times km (four more FMUL2), then one broadcast weight per channel.
template <int CH>
__device__ __forceinline__ void recur_accumulate_ch(float E3, float Lf, const float4 ka, const float4 kb,
                                                    const float (&w)[CH], float (&acc)[CH][8])
{
    const float G3 = ex2f(E3), rf = ex2f(Lf), rb = ex2f(-Lf);
    const float G4 = G3 * rf;
    const f32x2 R = pk2(rb, rf);
    const f32x2 P0 = pk2(G3, G4);
    const f32x2 P1 = mul2(P0, R);
    const f32x2 P2 = mul2(P1, R);
    const f32x2 P3 = mul2(P2, R);
    const f32x2 Q0 = mul2(P0, pk2(ka.x, ka.y)), Q1 = mul2(P1, pk2(ka.z, ka.w));
    const f32x2 Q2 = mul2(P2, pk2(kb.x, kb.y)), Q3 = mul2(P3, pk2(kb.z, kb.w));
    #pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
        const f32x2 wv = pk2(w[ch], w[ch]);
        fma2_acc(acc[ch][0], acc[ch][1], Q0, wv);
        fma2_acc(acc[ch][2], acc[ch][3], Q1, wv);
        fma2_acc(acc[ch][4], acc[ch][5], Q2, wv);
        fma2_acc(acc[ch][6], acc[ch][7], Q3, wv);
    }
}

template <int CH> struct B1W { float w[CH == 1 ? 1 : CH]; };
template <int CH>
__device__ __forceinline__ B1W<CH> load_w(const float* __restrict__ r)
{
    B1W<CH> o;
    if constexpr (CH == 1) o.w[0] = 0.f;
    else {
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) o.w[ch] = r[20 + ch];
    }
    return o;
}
template <int CH>
__device__ __forceinline__ void row_accumulate(float E3, float Lf, const float4 wa, const float4 wb, const B1W<CH>& w,
                                               float (&acc)[CH][8])
{
    if constexpr (CH == 1) recur_accumulate(E3, Lf, wa, wb, acc[0]);
    else recur_accumulate_ch<CH>(E3, Lf, wa, wb, w.w, acc);
}

// One row of a slow key, scalar.
template <int CH>
__device__ __forceinline__ void eval_row_slow(const float* __restrict__ r, bool inrow, float fy, float fz, float (&acc)[CH][8])
{
    const float dy = fy + r[1], dz = fz + r[2];
    const float negA = r[3];
    const float u1 = fmaf(r[6], dz, dy);
    const float t3 = fmaf(r[5], dz, fmaf(r[4], dy, r[0]));
    float Es = fmaf(r[8] * dz, dz, (r[7] * u1) * u1);
    Es = inrow ? Es : -1.0e30f;
    float G[8];                                                     // order 3,4,2,5,1,6,0,7
    if (-negA > kRecurrenceMaxA) {
        #pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float tl = t3 - (float)j, th = t3 + (float)(1 + j);          // (3 - j) - xs, (4 + j) - xs
            G[2 * j] = ex2f(fmaf(negA * tl, tl, Es)); G[2 * j + 1] = ex2f(fmaf(negA * th, th, Es));
        }
    } else {
        const float cc = fabsf(r[9]);
        const float nAt = negA * t3;
        float rf = ex2f(fminf(fmaf(nAt, 2.0f, negA), 120.f)), rb = ex2f(fminf(fmaf(nAt, -2.0f, negA), 120.f));
        G[0] = ex2f(fmaf(nAt, t3, Es));
        G[1] = G[0] * rf; rf *= cc; G[3] = G[1] * rf; rf *= cc; G[5] = G[3] * rf; rf *= cc; G[7] = G[5] * rf;
        G[2] = G[0] * rb; rb *= cc; G[4] = G[2] * rb; rb *= cc; G[6] = G[4] * rb;
    }
    if constexpr (CH == 1) {
        #pragma unroll
        for (int k = 0; k < 8; ++k) acc[0][k] = fmaf(G[k], r[12 + k], acc[0][k]);
    } else {
        #pragma unroll
        for (int k = 0; k < 8; ++k) G[k] *= r[12 + k];
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) {
            const float w = r[20 + ch];
            #pragma unroll
            for (int k = 0; k < 8; ++k) acc[ch][k] = fmaf(G[k], w, acc[ch][k]);
        }
    }
}

// A slow key (direct exponentials, or a recurrence that needs its clamps): scalar, row by row.
template <int CH>
__device__ __forceinline__ void eval_key_slow(const float* __restrict__ r, uint32_t lanebit, float fy, float fz,
                                              float (&acc0)[CH][8], float (&acc1)[CH][8])
{
    const uint32_t m0 = __float_as_uint(r[10]), m1 = __float_as_uint(r[11]);
    if (m0) eval_row_slow<CH>(r, (m0 & lanebit) != 0u, fy, fz, acc0);
    if (m1) eval_row_slow<CH>(r, (m1 & lanebit) != 0u, fy, fz + 4.0f, acc1);
}

// A fast key that reaches both z-halves: setup of both rows at once, (row z, row z + 4) in the two halves of
// a packed register, the key's scalars broadcast.
template <int CH>
__device__ __forceinline__ void eval_key_both(const float* __restrict__ r, uint32_t lanebit, float fy, f32x2 fz2,
                                              float (&acc0)[CH][8], float (&acc1)[CH][8])
{
    const float4 q0 = *reinterpret_cast<const float4*>(r);
    const float4 q1 = *reinterpret_cast<const float4*>(r + 4);
    const float4 q2 = *reinterpret_cast<const float4*>(r + 8);
    const float4 wa = *reinterpret_cast<const float4*>(r + 12);
    const float4 wb = *reinterpret_cast<const float4*>(r + 16);
    const float dy = fy + q0.y;
    const f32x2 dz = add2(fz2, pk2(q0.z, q0.z));
    const f32x2 u1 = fma2(pk2(q1.z, q1.z), dz, pk2(dy, dy));
    const float tA = fmaf(q1.x, dy, q0.x);
    const f32x2 t3 = fma2(pk2(q1.y, q1.y), dz, pk2(tA, tA));
    const f32x2 Es = fma2(mul2(pk2(q2.x, q2.x), dz), dz, mul2(mul2(pk2(q1.w, q1.w), u1), u1));
    const f32x2 negA = pk2(q0.w, q0.w);
    const f32x2 nAt = mul2(negA, t3);
    const f32x2 E3 = fma2(nAt, t3, Es);
    const f32x2 Lf = fma2(nAt, pk2(2.0f, 2.0f), negA);
    float E3a, E3b, Lfa, Lfb;
    upk2(E3, E3a, E3b); upk2(Lf, Lfa, Lfb);
    E3a = (__float_as_uint(q2.z) & lanebit) ? E3a : -1.0e30f;        // rows outside the box contribute exact zeros
    E3b = (__float_as_uint(q2.w) & lanebit) ? E3b : -1.0e30f;
    const B1W<CH> w = load_w<CH>(r);
    row_accumulate<CH>(E3a, Lfa, wa, wb, w, acc0);
    row_accumulate<CH>(E3b, Lfb, wa, wb, w, acc1);
}

// A fast key that reaches one z-half only: one row per thread, scalar setup.  HI: the half z = 4..7.
template <int CH, bool HI>
__device__ __forceinline__ void eval_key_half(const float* __restrict__ r, uint32_t lanebit, float fy, float fzh,
                                              float (&acc)[CH][8])
{
    const float4 q0 = *reinterpret_cast<const float4*>(r);
    const float4 q1 = *reinterpret_cast<const float4*>(r + 4);
    const float4 q2 = *reinterpret_cast<const float4*>(r + 8);
    const float4 wa = *reinterpret_cast<const float4*>(r + 12);
    const float4 wb = *reinterpret_cast<const float4*>(r + 16);
    const float dy = fy + q0.y, dz = fzh + q0.z;
    const float u1 = fmaf(q1.z, dz, dy);
    const float t3 = fmaf(q1.y, dz, fmaf(q1.x, dy, q0.x));
    const float Es = fmaf(q2.x * dz, dz, (q1.w * u1) * u1);
    const float nAt = q0.w * t3;
    float E3 = fmaf(nAt, t3, Es);
    const float Lf = fmaf(nAt, 2.0f, q0.w);
    E3 = (__float_as_uint(HI ? q2.w : q2.z) & lanebit) ? E3 : -1.0e30f;
    row_accumulate<CH>(E3, Lf, wa, wb, load_w<CH>(r), acc);
}

// Keys [kbeg, kend) of brick b.  ADD = false: the brick's rows are stored (segment 0; zeros for an empty brick);
// ADD = true: a later segment of a hot brick, added atomically to what segment 0 stored.
template <int CH, bool VEC, bool ADD>
__device__ __forceinline__ void b1_brick(const GsRec* __restrict__ rec, const uint32_t* __restrict__ keys,
                                         const float* __restrict__ weight, int wstride, int c0, float* __restrict__ out,
                                         const GridDev& gd, float* __restrict__ s_raw, float* __restrict__ s_rec,
                                         int b, uint32_t kbeg, uint32_t kend)
{
    const int lane = threadIdx.x;
    const int bx = b % gd.nb[0], by = (b / gd.nb[0]) % gd.nb[1], bz = b / (gd.nb[0] * gd.nb[1]);
    const int b0x = bx * kBrick, b0y = by * kBrick, b0z = bz * kBrick;
    const int ry = lane & 7, rz = lane >> 3;                        // rows (ry, rz) and (ry, rz + 4)
    const float fy = (float)ry, fz = (float)rz;
    const f32x2 fz2 = pk2(fz, fz + 4.0f);
    const uint32_t lanebit = 1u << lane;

    constexpr int KW = B1Rec<CH>::kWords;
    float acc0[CH][8], acc1[CH][8];                 // acc[ch][2j], acc[ch][2j+1] = voxels 3 - j, 4 + j
    #pragma unroll
    for (int ch = 0; ch < CH; ++ch)
        #pragma unroll
        for (int j = 0; j < 8; ++j) { acc0[ch][j] = 0.f; acc1[ch][j] = 0.f; }

    const uint32_t raw_addr = (uint32_t)__cvta_generic_to_shared(s_raw + lane * kB1Words);
    auto fetch = [&](uint32_t gid) {                // this lane's record -> s_raw, asynchronously
        const char* rp = reinterpret_cast<const char*>(rec + gid);
        cp_async16(raw_addr, rp); cp_async16(raw_addr + 16, rp + 16);
        cp_async16(raw_addr + 32, rp + 32); cp_async16(raw_addr + 48, rp + 48);
    };
    uint32_t gid_next = 0;
    float w_cur[CH], w_next[CH];
    #pragma unroll
    for (int ch = 0; ch < CH; ++ch) { w_cur[ch] = 0.f; w_next[ch] = 0.f; }
    if (kbeg + lane < kend) {
        const uint32_t gid = keys[kbeg + lane];
        fetch(gid);
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) w_cur[ch] = __ldg(weight + (size_t)gid * wstride + c0 + ch);
    }
    cp_async_commit();
    if (kbeg + kB1Batch + lane < kend) gid_next = keys[kbeg + kB1Batch + lane];

    for (uint32_t base = kbeg; base < kend; base += kB1Batch) {
        cp_async_wait_all();
        __syncwarp();                               // the previous batch's records have been read by every lane
        // ---- stage: lane l turns key l into brick-local form and classifies it; keys are stored class by class
        //      (slow | both halves | lower half only | upper half only) so that each class runs a branch-free loop
        int cls = -1;
        float4 o0, o1, o2, o3, o4, o5;
        if (base + lane < kend) {
            const float4* rp = reinterpret_cast<const float4*>(s_raw + lane * kB1Words);
            const float4 a = rp[0], bq = rp[1], c = rp[2], d = rp[3];
            const float w = (CH == 1) ? w_cur[0] : 1.0f;          // CH > 1: words 12..19 carry km alone
            const int w1i = __float_as_int(d.y), w2i = __float_as_int(d.z), w3i = __float_as_int(d.w);
            const int lox = (int16_t)(w1i & 0xffff), loy = (int16_t)(w1i >> 16), loz = (int16_t)(w2i & 0xffff);
            const int hix = (int16_t)(w2i >> 16), hiy = (int16_t)(w3i & 0xffff), hiz = (int16_t)(w3i >> 16);
            const int x0 = max(lox - b0x, 0), x1 = min(hix - b0x, 7);
            const int y0 = max(loy - b0y, 0), y1 = min(hiy - b0y, 7);
            const int z0 = max(loz - b0z, 0), z1 = min(hiz - b0z, 7);
            const uint32_t ym = ((2u << y1) - (1u << y0)) & 0xffu;
            const uint32_t zm = ((2u << z1) - (1u << z0)) & 0xffu;
            const uint32_t xm = ((2u << x1) - (1u << x0)) & 0xffu;
            const uint32_t rep = ym * 0x01010101u;
            const uint32_t sel0 = ((zm & 1u) ? 0xffu : 0u) | ((zm & 2u) ? 0xff00u : 0u) |
                                  ((zm & 4u) ? 0xff0000u : 0u) | ((zm & 8u) ? 0xff000000u : 0u);
            const uint32_t zh = zm >> 4;
            const uint32_t sel1 = ((zh & 1u) ? 0xffu : 0u) | ((zh & 2u) ? 0xff00u : 0u) |
                                  ((zh & 4u) ? 0xff0000u : 0u) | ((zh & 8u) ? 0xff000000u : 0u);
            const float cx = (float)(__float_as_int(bq.x) - b0x) + a.x;
            const float cy = (float)(__float_as_int(bq.y) - b0y) + a.y;
            const float cz = (float)(__float_as_int(bq.z) - b0z) + a.z;
            const float cx3 = 3.0f - cx, negA = bq.w, l01 = -c.x, l02 = -c.y;
            // largest |t3| over the 64 rows: dy in [-cy, 7 - cy], dz in [-cz, 7 - cz]
            const float t3max = fabsf(cx3) + fabsf(l01) * fmaxf(fabsf(cy), fabsf(7.0f - cy)) +
                                fabsf(l02) * fmaxf(fabsf(cz), fabsf(7.0f - cz));
            const bool slow = (-negA > kRecurrenceMaxA) || !(-negA * fmaf(2.0f, t3max, 1.0f) < 120.f);
            const float cc = fabsf(a.w);
            cls = slow ? 0 : ((zm & 0x0fu) == 0u ? 3 : ((zm & 0xf0u) == 0u ? 2 : 1));
            o0 = make_float4(cx3, -cy, -cz, negA);
            o1 = make_float4(l01, l02, c.z, c.w);
            o2 = make_float4(d.x, cc, __uint_as_float(rep & sel0), __uint_as_float(rep & sel1));
            // fast keys: the key-and-k part of the row profile, c^((k-3)(k-4)/2), goes into the weights (recur_accumulate)
            const float w1 = slow ? w : w * cc, c3 = cc * cc * cc, w3 = slow ? w : w * c3, w6 = slow ? w : w * (c3 * c3);
            o3 = make_float4((xm & 8u) ? w : 0.f, (xm & 16u) ? w : 0.f, (xm & 4u) ? w1 : 0.f, (xm & 32u) ? w1 : 0.f);
            o4 = make_float4((xm & 2u) ? w3 : 0.f, (xm & 64u) ? w3 : 0.f, (xm & 1u) ? w6 : 0.f, (xm & 128u) ? w6 : 0.f);
            if constexpr (CH > 1) o5 = make_float4(w_cur[0], w_cur[1], w_cur[2 % CH], 0.f);
        }
        const uint32_t b0 = __ballot_sync(0xffffffffu, cls == 0), b1 = __ballot_sync(0xffffffffu, cls == 1),
                       b2 = __ballot_sync(0xffffffffu, cls == 2), b3 = __ballot_sync(0xffffffffu, cls == 3);
        const int n0 = __popc(b0), n1 = n0 + __popc(b1), n2 = n1 + __popc(b2), n3 = n2 + __popc(b3);
        if (cls >= 0) {
            const uint32_t mine = cls == 0 ? b0 : (cls == 1 ? b1 : (cls == 2 ? b2 : b3));
            const int slot = (cls == 0 ? 0 : (cls == 1 ? n0 : (cls == 2 ? n1 : n2))) + __popc(mine & (lanebit - 1u));
            float4* o = reinterpret_cast<float4*>(s_rec + slot * KW);
            o[0] = o0; o[1] = o1; o[2] = o2; o[3] = o3; o[4] = o4;
            if constexpr (CH > 1) o[5] = o5;
        }
        __syncwarp();
        // next batch's records on their way while this one is evaluated
        if (base + kB1Batch + lane < kend) {
            fetch(gid_next);
            #pragma unroll
            for (int ch = 0; ch < CH; ++ch) w_next[ch] = __ldg(weight + (size_t)gid_next * wstride + c0 + ch);
        }
        cp_async_commit();
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) w_cur[ch] = w_next[ch];
        if (base + 2 * kB1Batch + lane < kend) gid_next = keys[base + 2 * kB1Batch + lane];
        int j = 0;
        for (; j < n0; ++j) eval_key_slow<CH>(s_rec + j * KW, lanebit, fy, fz, acc0, acc1);
        if constexpr (CH > 1) {
            for (; j + 1 < n1; j += 2) {
                eval_key_both<CH>(s_rec + j * KW, lanebit, fy, fz2, acc0, acc1);
                eval_key_both<CH>(s_rec + (j + 1) * KW, lanebit, fy, fz2, acc0, acc1);
            }
        }
        #pragma unroll 1
        for (; j < n1; ++j) eval_key_both<CH>(s_rec + j * KW, lanebit, fy, fz2, acc0, acc1);
        #pragma unroll 1
        for (; j < n2; ++j) eval_key_half<CH, false>(s_rec + j * KW, lanebit, fy, fz, acc0);
        #pragma unroll 1
        for (; j < n3; ++j) eval_key_half<CH, true>(s_rec + j * KW, lanebit, fy, fz + 4.0f, acc1);
    }

    // write (or add) the two rows; x fastest
    const size_t plane = (size_t)gd.dims[0] * gd.dims[1] * gd.dims[2];
    #pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int gy = b0y + ry, gz = b0z + rz + 4 * h;
        if (gy < gd.dims[1] && gz < gd.dims[2]) {
            const size_t rowoff = ((size_t)gz * gd.dims[1] + gy) * gd.dims[0] + b0x;
            #pragma unroll
            for (int ch = 0; ch < CH; ++ch) {
            float v[8];
            #pragma unroll
            for (int j = 0; j < 4; ++j) { v[3 - j] = h ? acc1[ch][2 * j] : acc0[ch][2 * j]; v[4 + j] = h ? acc1[ch][2 * j + 1] : acc0[ch][2 * j + 1]; }
            float* o = out + (size_t)(c0 + ch) * plane + rowoff;
            if (VEC) {
                if (ADD) {
                    if (b0x + 3 < gd.dims[0]) red_add_v4f(o, v[0], v[1], v[2], v[3]);
                    if (b0x + 7 < gd.dims[0]) red_add_v4f(o + 4, v[4], v[5], v[6], v[7]);
                } else {
                    if (b0x + 3 < gd.dims[0]) __stcs(reinterpret_cast<float4*>(o), make_float4(v[0], v[1], v[2], v[3]));
                    if (b0x + 7 < gd.dims[0]) __stcs(reinterpret_cast<float4*>(o) + 1, make_float4(v[4], v[5], v[6], v[7]));
                }
            } else {
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2)
                    if (b0x + k2 < gd.dims[0]) { if (ADD) atomicAdd(o + k2, v[k2]); else o[k2] = v[k2]; }
            }
            }
        }
    }
}

// First launch: one warp per brick, segment 0 of its key range.
template <int CH, bool VEC>
__global__ void __launch_bounds__(32, CH == 1 ? 32 : 16)
k_forward_b1(const GsRec* __restrict__ rec, const uint32_t* __restrict__ bin_start,
             const uint32_t* __restrict__ keys, const DevStatus* __restrict__ status,
             const float* __restrict__ weight, int wstride, int c0,
             float* __restrict__ out, GridDev gd, uint32_t max_keys)
{
    __shared__ __align__(16) float s_raw[kB1Batch * kB1Words];
    __shared__ __align__(16) float s_rec[kB1Batch * B1Rec<CH>::kWords];
    const int b = blockIdx.x + gd.slab0 * gd.nb[0] * gd.nb[1];
    uint32_t kbeg = 0, kend = 0;
    if (!status->overflow) {
        kbeg = bin_start[b * kNumClasses];
        kend = bin_start[(b + 1) * kNumClasses];
        if (kend - kbeg > max_keys) kend = kbeg + max_keys;         // kSplitKeys; deterministic mode: the whole range
    }
    b1_brick<CH, VEC, false>(rec, keys, weight, wstride, c0, out, gd, s_raw, s_rec, b, kbeg, kend);
}

// Second launch: the later segments of hot bricks, a fixed grid striding over a2's item list.
template <int CH, bool VEC>
__global__ void __launch_bounds__(32, CH == 1 ? 32 : 16)
k_forward_b1_extra(const GsRec* __restrict__ rec, const uint32_t* __restrict__ bin_start,
                   const uint32_t* __restrict__ keys, const DevStatus* __restrict__ status,
                   const uint2* __restrict__ split_list, int split_cap,
                   const float* __restrict__ weight, int wstride, int c0,
                   float* __restrict__ out, GridDev gd)
{
    __shared__ __align__(16) float s_raw[kB1Batch * kB1Words];
    __shared__ __align__(16) float s_rec[kB1Batch * B1Rec<CH>::kWords];
    if (status->overflow) return;
    const uint32_t nitems = min(status->nsplit, (uint32_t)split_cap);
    for (uint32_t i = blockIdx.x; i < nitems; i += gridDim.x) {
        const uint2 item = split_list[i];
        const uint32_t kbeg = bin_start[item.x * kNumClasses] + item.y * (uint32_t)kSplitKeys;
        const uint32_t kend = min(bin_start[(item.x + 1) * kNumClasses], kbeg + (uint32_t)kSplitKeys);
        __syncwarp();
        b1_brick<CH, VEC, true>(rec, keys, weight, wstride, c0, out, gd, s_raw, s_rec, (int)item.x, kbeg, kend);
    }
}

template <int CH>
static int launch_fwd_b1(gsvox_plan* p, const float* weight, int C, int c0, float* out, cudaStream_t st)
{
    static_assert(CH == 1 || CH == 3, "b1 staging carries one or three weights");
    LaunchScope ls(p, GSVOX_K_FORWARD, st);
    const bool vec = (p->gd.dims[0] % 4 == 0) && (((uintptr_t)out & 15) == 0);
    const int nblocks = (p->gd.slab1 - p->gd.slab0) * p->gd.nb[0] * p->gd.nb[1];
    if (nblocks <= 0) return GSVOX_OK;
    // deterministic mode: one warp walks its brick's whole key list in the sorted order, no second launch, no atomics
    const uint32_t max_keys = p->deterministic ? 0xffffffffu : (uint32_t)kSplitKeys;
    if (vec) k_forward_b1<CH, true><<<nblocks, 32, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, weight, C, c0, out, p->gd, max_keys);
    else     k_forward_b1<CH, false><<<nblocks, 32, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, weight, C, c0, out, p->gd, max_keys);
    GSVOX_CUDA(cudaGetLastError());
    if (p->deterministic) return GSVOX_OK;
    p->launches[GSVOX_K_FORWARD] += 1;               // the hot-brick launch
    // single-warp CTAs: 32 resident per SM at C = 1 (64 registers), 16 at C = 3
    constexpr int xgrid = (CH == 1) ? 2 * kSplitGrid : kSplitGrid;
    if (vec) k_forward_b1_extra<CH, true><<<xgrid, 32, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, p->split_list,
                                                                     p->split_cap, weight, C, c0, out, p->gd);
    else     k_forward_b1_extra<CH, false><<<xgrid, 32, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, p->split_list,
                                                                      p->split_cap, weight, C, c0, out, p->gd);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

template <int CH>
static int launch_fwd_ch(gsvox_plan* p, const float* weight, int C, int c0, float* out, cudaStream_t st)
{
    LaunchScope ls(p, GSVOX_K_FORWARD, st);
    bool vec = (p->gd.dims[0] % 4 == 0) && (((uintptr_t)out & 15) == 0);
    const int nblocks = (p->gd.slab1 - p->gd.slab0) * p->gd.nb[0] * p->gd.nb[1];
    if (nblocks <= 0) return GSVOX_OK;
    if (vec)
        k_forward<CH, true><<<nblocks, kFwdThreads, 0, st>>>(p->rec, p->bin_start, p->keys, p->status,
                                                                   weight, C, c0, out, p->gd);
    else
        k_forward<CH, false><<<nblocks, kFwdThreads, 0, st>>>(p->rec, p->bin_start, p->keys, p->status,
                                                                    weight, C, c0, out, p->gd);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

int launch_forward(gsvox_plan* p, const float* weight, int channels, float* out, cudaStream_t st)
{
    // channel groups of 9, 3, 1: C = 9 (motion-basis fields) and C = 1 (CBCT) are single launches
    int c0 = 0, rc = GSVOX_OK;
    while (c0 < channels && rc == GSVOX_OK) {
        int left = channels - c0;
        if (left >= 9)      { rc = launch_fwd_ch<9>(p, weight, channels, c0, out, st); c0 += 9; }
        else if (left >= 3) { rc = launch_fwd_b1<3>(p, weight, channels, c0, out, st); c0 += 3; }
        else                { rc = launch_fwd_b1<1>(p, weight, channels, c0, out, st); c0 += 1; }
    }
    return rc;
}

}  // namespace gsvox
