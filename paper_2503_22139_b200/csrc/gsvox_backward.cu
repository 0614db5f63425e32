// gsvox_backward.cu — step a4: per-brick backward (gradients of Eq. 5).
//
// One CTA (128 threads) per 8^3 brick.  The brick's upstream-gradient tile (CH x 512 floats) is
// staged in shared memory; then every THREAD takes one (brick, Gaussian) key and walks the rows
// of box ∩ brick itself, so the reduction over voxels that the gradient needs happens in
// registers: no cross-lane traffic, no shared-memory atomics.  Keys arrive sorted by class inside
// the brick (gsvox_internal.cuh, key_class): the 32 keys of a warp have similar row counts and the
// same code path, which is what keeps the lanes of a warp busy (measured 15/32 active lanes with
// unsorted keys).
//
// Per row: G recomputed exactly as in a3, a_k = (sum_c g_c w_c) G_k, and the three x-moments
//     U0,U1,U2 = sum_k a_k {1, u0, u0^2},  u0 = k - xs,
// from which every first and second moment of u = L^T d follows (u1, u2 = dz are constant along a
// row; M = L D L^T).  Moments are kept in this u frame because sqrt(D) u is an orthogonal rotation
// of the whitened coordinates S^-1 R^T d: fp32 sums then lose nothing to the anisotropy of the
// Gaussian (a world-frame d d^T sum loses (s_max/s_min)^2).  Per key: vector reductions
// (red.global.add.v4.f32) of the 9 moments + C weight gradients into
//     acc[g][...] = { m_u0,m_u1,m_u2, m_00,m_01,m_02,m_11,m_12,m_22, dw_0..dw_{C-1} }  (index units).
// a5 (gsvox_epilogue.cu) turns acc into dL/dp, dL/ds, dL/dq.
#include "gsvox_internal.cuh"

namespace gsvox {

constexpr int kBwdThreads = 128;
// A CTA of the first launch takes up to 4 segments of kSplitKeys keys (16 keys per thread); dense-but-even fields
// (config 3: ~1000 keys in every brick) then run as one launch, only truly hot bricks spill into the second.
constexpr int kBwdMainSegments = 4;
constexpr int kZSwizzleCH = 9;           // channel groups this wide also swizzle the gradient tile by the slice z (backward_brick)

__device__ __forceinline__ float ex2b(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};"
                 :: "l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__device__ __forceinline__ float4 lds_v4(uint32_t saddr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
    return v;
}

// Geometry of one key, brick-local.
struct KeyGeom {
    float cx, cy, cz, negA, nl01, nl02, l12, nD1, nD2, cc;
    int y0, z0, ny, nrows;
    uint32_t xm;
    bool direct;
};

struct Moments { float b0, bu0, bu1, bu2, b00, b01, b02, b11, b12, b22; };

// Walk the rows of one key.  MODE 0: the warp's keys all take the geometric chain; 1: all take one EX2 per voxel (narrow
// Gaussians, class 0); 2: both kinds in this warp — ONE row loop, the lanes part only for the eight G values.  (Two loops
// one after the other cost the warp rows_direct x 100 + rows_chain x 85 instructions; config 5's needle-only bricks hold
// 17..64 keys, 5 % of them direct, so nearly every warp there paid both: ncu counted 15.5 of 32 lanes active.)
// sbase is the shared-window byte address of the gradient tile.
template <int CH, bool SINGLE, int MODE>
__device__ __forceinline__ void walk_rows(const KeyGeom& kg, uint32_t sbase, const float (&wv)[CH],
                                          Moments& m, float (&dw)[CH])
{
    float dy = (float)kg.y0 - kg.cy, dz = (float)kg.z0 - kg.cz;
    const float dy0 = dy;
    float km[8];                                                    // [k in box] c^((k-3)(k-4)/2), c = 2^-2A
    {
        const float c1 = kg.cc, c3 = c1 * c1 * c1, c6 = c3 * c3;
        const float kk[8] = { c6, c3, c1, 1.f, 1.f, c1, c3, c6 };
        #pragma unroll
        for (int k = 0; k < 8; ++k)
            km[k] = (MODE != 1 && (kg.xm & (1u << k))) ? ((MODE == 2 && kg.direct) ? 1.f : kk[k]) : 0.f;
    }
    // byte address of the row in the tile (CH = 9: its offset inside the tile, the z swizzle below works on that)
    uint32_t gaddr = (CH >= kZSwizzleCH ? 0u : sbase) + ((((kg.z0 << 3) + kg.y0) << 3) << 2);
    const uint32_t wrapstep = (uint32_t)(9 - kg.ny) << 5;              // last y of a slice -> y0 of the next
    int yc = kg.ny;
    for (int r = kg.nrows; r > 0; --r) {
        const float u1 = fmaf(kg.l12, dz, dy);
        const float xs = fmaf(kg.nl02, dz, fmaf(kg.nl01, dy, kg.cx));
        const float Es = fmaf(kg.nD2 * dz, dz, (kg.nD1 * u1) * u1);
        float G[8];
        if (MODE == 0 || (MODE == 2 && !kg.direct)) {
            // the row is the parabola E(k) = E3 + (k - 3) Lf - A (k - 3)(k - 4):  G(k) = G3 rho^(k-3) c^((k-3)(k-4)/2).
            // The geometric part is chained here (7 FMUL); the key-and-k part, together with the x mask of the box,
            // sits in km[k] (per key, hoisted out of the row loop) — as in a3, where it sits in the staged weights.
            const float t3 = 3.0f - xs;
            const float nAt = kg.negA * t3;
            const float Lf = fminf(fmaxf(fmaf(nAt, 2.0f, kg.negA), -120.f), 120.f);      // 2^+-Lf stay finite; beyond, G3 is 0
            G[3] = ex2b(fmaf(nAt, t3, Es));
            const float rf = ex2b(Lf), rb = ex2b(-Lf);
            G[4] = G[3] * rf; G[5] = G[4] * rf; G[6] = G[5] * rf; G[7] = G[6] * rf;
            G[2] = G[3] * rb; G[1] = G[2] * rb; G[0] = G[1] * rb;
            if (MODE == 0) {
                #pragma unroll
                for (int k = 0; k < 8; ++k) G[k] *= km[k];
            }
        } else {
            #pragma unroll
            for (int k = 0; k < 8; ++k) { const float t = (float)k - xs; G[k] = ex2b(fmaf(kg.negA * t, t, Es)); }
            if (MODE == 1) {
                #pragma unroll
                for (int k = 0; k < 8; ++k) G[k] = (kg.xm & (1u << k)) ? G[k] : 0.f;      // voxels outside the box in x
            }
        }
        if (MODE == 2) {                                            // km: the chain's factors, or the bare x mask of a direct key
            #pragma unroll
            for (int k = 0; k < 8; ++k) G[k] *= km[k];
        }
        // a_k = (sum_c g_c w_c) G_k  (w factored out when SINGLE)
        float av[8];
        if (SINGLE) {
            const float4 g0 = lds_v4(gaddr), g1 = lds_v4(gaddr + 16);
            av[0] = g0.x * G[0]; av[1] = g0.y * G[1]; av[2] = g0.z * G[2]; av[3] = g0.w * G[3];
            av[4] = g1.x * G[4]; av[5] = g1.y * G[5]; av[6] = g1.z * G[6]; av[7] = g1.w * G[7];
        } else {
            // rows with y >= 4 hold their halves swapped when CH > 1 (stage loop); a lone channel of a wider C keeps the plain layout
            // (bits 8..10 of the offset inside the tile are the slice z)
            const uint32_t ga0 = (CH >= kZSwizzleCH) ? (sbase + (gaddr ^ ((gaddr >> 3) & 16u) ^ ((gaddr >> 4) & 0x70u)))
                               : ((CH > 1) ? (gaddr ^ ((gaddr >> 3) & 16u)) : gaddr), ga1 = ga0 ^ 16u;
            if (CH >= 3) {
                // packed pairs of neighbouring voxels: 8 FFMA2 + 2 per channel instead of 16 FFMA (a4 at C = 3 is issue-bound; C = 9 gains 3 % on full-brick keys)
                const f32x2 G2[4] = { pk2(G[0], G[1]), pk2(G[2], G[3]), pk2(G[4], G[5]), pk2(G[6], G[7]) };
                f32x2 a2[4];
                #pragma unroll
                for (int ch = 0; ch < CH; ++ch) {
                    const float4 g0 = lds_v4(ga0 + ch * kBrickVox * 4), g1 = lds_v4(ga1 + ch * kBrickVox * 4);
                    const f32x2 gp[4] = { pk2(g0.x, g0.y), pk2(g0.z, g0.w), pk2(g1.x, g1.y), pk2(g1.z, g1.w) };
                    const f32x2 w2 = pk2(wv[ch], wv[ch]);
                    f32x2 d2 = mul2(gp[0], G2[0]);
                    #pragma unroll
                    for (int j = 1; j < 4; ++j) d2 = fma2(gp[j], G2[j], d2);
                    #pragma unroll
                    for (int j = 0; j < 4; ++j) a2[j] = (ch == 0) ? mul2(gp[j], w2) : fma2(gp[j], w2, a2[j]);
                    float dl, dh; upk2(d2, dl, dh);
                    dw[ch] += dl + dh;
                }
                #pragma unroll
                for (int j = 0; j < 4; ++j) { a2[j] = mul2(a2[j], G2[j]); upk2(a2[j], av[2 * j], av[2 * j + 1]); }
            } else {
            #pragma unroll
            for (int k = 0; k < 8; ++k) av[k] = 0.f;
            #pragma unroll
            for (int ch = 0; ch < CH; ++ch) {
                const float4 g0 = lds_v4(ga0 + ch * kBrickVox * 4), g1 = lds_v4(ga1 + ch * kBrickVox * 4);
                const float gv[8] = { g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w };
                float d = 0.f;
                #pragma unroll
                for (int k = 0; k < 8; ++k) { d = fmaf(gv[k], G[k], d); av[k] = fmaf(gv[k], wv[ch], av[k]); }
                dw[ch] += d;
            }
            #pragma unroll
            for (int k = 0; k < 8; ++k) av[k] *= G[k];
            }
        }
        // x-moments about xs
        float U0, U1, U2;
        if (MODE == 0) {
            // about the brick-local index, then shifted (wide profile: mild cancellation only)
            U0 = av[0]; float S1 = 0.f, S2 = 0.f;
            #pragma unroll
            for (int k = 1; k < 8; ++k) { U0 += av[k]; S1 = fmaf(av[k], (float)k, S1); S2 = fmaf(av[k], (float)(k * k), S2); }
            U1 = fmaf(-xs, U0, S1);
            U2 = fmaf(xs, fmaf(xs, U0, -2.0f * S1), S2);
        } else {
            U0 = 0.f; U1 = 0.f; U2 = 0.f;
            #pragma unroll
            for (int k = 0; k < 8; ++k) { const float u = (float)k - xs, au = av[k] * u; U0 += av[k]; U1 += au; U2 = fmaf(au, u, U2); }
        }
        // row moments -> key moments in the u frame
        const float u1U0 = u1 * U0, dzU0 = dz * U0;
        m.b0 += U0; m.bu0 += U1; m.b00 += U2;
        m.bu1 += u1U0; m.bu2 += dzU0;
        m.b01 = fmaf(u1, U1, m.b01); m.b02 = fmaf(dz, U1, m.b02);
        m.b11 = fmaf(u1, u1U0, m.b11); m.b12 = fmaf(dz, u1U0, m.b12); m.b22 = fmaf(dz, dzU0, m.b22);
        // next row: y fastest inside the box, then z
        --yc;
        const bool wrap = (yc == 0);
        dy = wrap ? dy0 : dy + 1.0f;
        dz = wrap ? dz + 1.0f : dz;
        gaddr += wrap ? wrapstep : 32u;
        yc = wrap ? kg.ny : yc;
    }
}

// Keys [kbeg, kend) of brick b (a whole brick, or one kSplitKeys segment of a hot one): gradient tile, then thread per key.
template <int CH, bool SINGLE>
__device__ __forceinline__ void backward_brick(const GsRec* __restrict__ rec, const uint32_t* __restrict__ keys,
                                               const float* __restrict__ weight, int wstride, int c0,
                                               const float* __restrict__ grad_out, float* __restrict__ acc, int astride,
                                               const GridDev& gd, float* __restrict__ s_g, int b, uint32_t kbeg, uint32_t kend)
{
    const int tid = threadIdx.x;
    const int bx = b % gd.nb[0], by = (b / gd.nb[0]) % gd.nb[1], bz = b / (gd.nb[0] * gd.nb[1]);
    const int b0x = bx * kBrick, b0y = by * kBrick, b0z = bz * kBrick;

    // stage the gradient tile, zero outside the grid
    {
        const size_t plane = (size_t)gd.dims[0] * gd.dims[1] * gd.dims[2];
        for (int e = tid; e < CH * kBrickVox; e += kBwdThreads) {
            int ch = e >> 9, v = e & 511, x = v & 7, y = (v >> 3) & 7, z = v >> 6;
            int gx = b0x + x, gy = b0y + y, gz = b0z + z;
            float val = 0.f;
            if (gx < gd.dims[0] && gy < gd.dims[1] && gz < gd.dims[2])
                val = __ldg(grad_out + (size_t)(c0 + ch) * plane + ((size_t)gz * gd.dims[1] + gy) * gd.dims[0] + gx);
            // 16-byte chunk c = 2 row + half goes to chunk c ^ (bit 2 of y): the eight rows y = 0..7 of a slice then start in
            // eight different bank groups, not four (thread-per-key LDS.128 of different rows: ncu counted 48 % of the
            // shared-memory wavefronts of k_backward<9> as bank conflicts, on a kernel whose l1tex pipe was 95 % busy)
            // (C = 1 keeps the plain layout: it is issue-bound, and the two extra address instructions per row cost it 4 %)
            // and to chunk ^ z: rows of equal y in different slices (keys of full y extent whose boxes start at different z
            // walk in step) no longer share a bank group either
            // (CH = 9 only: levels of full-brick keys pay 2 % for the extra address arithmetic, config 3 level 3 gains 11 %;
            //  C = 3 is issue-bound and loses 1.5 % with it)
            s_g[CH >= kZSwizzleCH ? ((e & ~63) | (((((y << 1) | (x >> 2)) ^ ((y >> 2) & 1) ^ z) & 15) << 2) | (x & 3))
                                  : (CH > 1 ? ((e & ~7) | ((x & 4) ^ (y & 4)) | (x & 3)) : e)] = val;
        }
    }
    __syncthreads();

    const uint32_t nkeys = kend - kbeg;
    const uint32_t lane = tid & 31u;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_g);
    for (uint32_t wbase = tid & ~31u; wbase < nkeys; wbase += kBwdThreads) {     // warp-uniform trip count
        const bool active = wbase + lane < nkeys;
        KeyGeom kg;
        kg.nrows = 0; kg.ny = 1; kg.y0 = 0; kg.z0 = 0; kg.xm = 0xffu; kg.direct = false;
        kg.cx = kg.cy = kg.cz = kg.negA = kg.nl01 = kg.nl02 = kg.l12 = kg.nD1 = kg.nD2 = 0.f; kg.cc = 1.f;
        uint32_t gid = 0;
        float wv[CH];
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) wv[ch] = 0.f;
        if (active) {
            gid = keys[kbeg + wbase + lane];
            const float4* rp = reinterpret_cast<const float4*>(rec + gid);
            const float4 ra = __ldg(rp), rb4 = __ldg(rp + 1), rc = __ldg(rp + 2), rd = __ldg(rp + 3);
            const int w1 = __float_as_int(rd.y), w2 = __float_as_int(rd.z), w3 = __float_as_int(rd.w);
            const int lox = (int16_t)(w1 & 0xffff), loy = (int16_t)(w1 >> 16), loz = (int16_t)(w2 & 0xffff);
            const int hix = (int16_t)(w2 >> 16), hiy = (int16_t)(w3 & 0xffff), hiz = (int16_t)(w3 >> 16);
            const int x0 = max(lox - b0x, 0), x1 = min(hix - b0x, 7);
            const int y0 = max(loy - b0y, 0), y1 = min(hiy - b0y, 7);
            const int z0 = max(loz - b0z, 0), z1 = min(hiz - b0z, 7);
            kg.xm = ((2u << x1) - (1u << x0)) & 0xffu;
            kg.cx = (float)(__float_as_int(rb4.x) - b0x) + ra.x;
            kg.cy = (float)(__float_as_int(rb4.y) - b0y) + ra.y;
            kg.cz = (float)(__float_as_int(rb4.z) - b0z) + ra.z;
            kg.negA = rb4.w; kg.nl01 = rc.x; kg.nl02 = rc.y; kg.l12 = rc.z; kg.nD1 = rc.w; kg.nD2 = rd.x; kg.cc = fabsf(ra.w);
            kg.direct = (-kg.negA > kRecurrenceMaxA);
            kg.y0 = y0; kg.z0 = z0; kg.ny = y1 - y0 + 1; kg.nrows = kg.ny * (z1 - z0 + 1);
            #pragma unroll
            for (int ch = 0; ch < CH; ++ch) wv[ch] = __ldg(weight + (size_t)gid * wstride + c0 + ch);
        }
        Moments m = { 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f };
        float dw[CH];
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) dw[ch] = 0.f;

        // class 0 (direct) keys sit at the front of the brick's range: at most one warp of a brick holds both kinds
        // (the loop over wbase has a warp-uniform trip count: whole warps arrive here)
        const bool any_direct = __any_sync(0xffffffffu, kg.direct && kg.nrows > 0);
        const bool any_chain = __any_sync(0xffffffffu, !kg.direct && kg.nrows > 0);
        if (any_direct && any_chain) walk_rows<CH, SINGLE, 2>(kg, sbase, wv, m, dw);
        else if (any_direct)         walk_rows<CH, SINGLE, 1>(kg, sbase, wv, m, dw);
        else                         walk_rows<CH, SINGLE, 0>(kg, sbase, wv, m, dw);

        if (active) {
            float* dst = acc + (size_t)gid * astride;
            if (SINGLE) {
                // moments of a = w g G; dw = sum g G
                const float w = wv[0];
                red_add_v4(dst, w * m.bu0, w * m.bu1, w * m.bu2, w * m.b00);
                red_add_v4(dst + 4, w * m.b01, w * m.b02, w * m.b11, w * m.b12);
                red_add_v4(dst + 8, w * m.b22, m.b0, 0.f, 0.f);
            } else {
                red_add_v4(dst, m.bu0, m.bu1, m.bu2, m.b00);
                red_add_v4(dst + 4, m.b01, m.b02, m.b11, m.b12);
                atomicAdd(dst + 8, m.b22);
                #pragma unroll
                for (int ch = 0; ch < CH; ++ch) atomicAdd(dst + 9 + c0 + ch, dw[ch]);
            }
        }
    }
}

// First launch: one CTA per brick, segment 0 of its key range.
template <int CH, bool SINGLE>
__global__ void __launch_bounds__(kBwdThreads)
k_backward(const GsRec* __restrict__ rec, const uint32_t* __restrict__ bin_start,
           const uint32_t* __restrict__ keys, const DevStatus* __restrict__ status,
           const float* __restrict__ weight, int wstride, int c0,
           const float* __restrict__ grad_out, float* __restrict__ acc, int astride, GridDev gd)
{
    __shared__ __align__(256) float s_g[CH * kBrickVox];
    if (status->overflow) return;
    const int b = blockIdx.x + gd.slab0 * gd.nb[0] * gd.nb[1];      // z-slab of this plan
    const uint32_t kbeg = bin_start[b * kNumClasses];
    const uint32_t kend = min(bin_start[(b + 1) * kNumClasses], kbeg + (uint32_t)(kBwdMainSegments * kSplitKeys));
    if (kbeg == kend) return;
    backward_brick<CH, SINGLE>(rec, keys, weight, wstride, c0, grad_out, acc, astride, gd, s_g, b, kbeg, kend);
}

// Second launch: the later segments of hot bricks (a2's item list), a fixed grid striding over the items.
template <int CH, bool SINGLE>
__global__ void __launch_bounds__(kBwdThreads)
k_backward_extra(const GsRec* __restrict__ rec, const uint32_t* __restrict__ bin_start,
                 const uint32_t* __restrict__ keys, const DevStatus* __restrict__ status,
                 const uint2* __restrict__ split_list, int split_cap,
                 const float* __restrict__ weight, int wstride, int c0,
                 const float* __restrict__ grad_out, float* __restrict__ acc, int astride, GridDev gd)
{
    __shared__ __align__(256) float s_g[CH * kBrickVox];
    if (status->overflow) return;
    const uint32_t nitems = min(status->nsplit, (uint32_t)split_cap);
    for (uint32_t i = blockIdx.x; i < nitems; i += gridDim.x) {
        const uint2 item = split_list[i];
        if (item.y < (uint32_t)kBwdMainSegments) continue;          // the first launch took these (CTA-uniform)
        const uint32_t kbeg = bin_start[item.x * kNumClasses] + item.y * (uint32_t)kSplitKeys;
        const uint32_t kend = min(bin_start[(item.x + 1) * kNumClasses], kbeg + (uint32_t)kSplitKeys);
        __syncthreads();                                            // the previous item's tile is no longer read
        backward_brick<CH, SINGLE>(rec, keys, weight, wstride, c0, grad_out, acc, astride, gd, s_g, (int)item.x, kbeg, kend);
    }
}

template <int CH, bool SINGLE>
static int launch_bwd_ch(gsvox_plan* p, const float* weight, int C, int c0, const float* grad_out,
                         int astride, cudaStream_t st)
{
    const int nblocks = (p->gd.slab1 - p->gd.slab0) * p->gd.nb[0] * p->gd.nb[1];
    if (nblocks <= 0) return GSVOX_OK;
    LaunchScope ls(p, GSVOX_K_BACKWARD, st);
    k_backward<CH, SINGLE><<<nblocks, kBwdThreads, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, weight,
                                                                  C, c0, grad_out, p->acc, astride, p->gd);
    GSVOX_CUDA(cudaGetLastError());
    p->launches[GSVOX_K_BACKWARD] += 1;              // the hot-brick launch
    k_backward_extra<CH, SINGLE><<<kSplitGrid / 2, kBwdThreads, 0, st>>>(p->rec, p->bin_start, p->keys, p->status,
                                                                         p->split_list, p->split_cap, weight, C, c0,
                                                                         grad_out, p->acc, astride, p->gd);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

int launch_backward_accumulate(gsvox_plan* p, const float* weight, int channels, const float* grad_out,
                               cudaStream_t st)
{
    const int astride = acc_stride(channels);
    { LaunchScope ls(p, GSVOX_K_MEMSET, st);
      GSVOX_CUDA(cudaMemsetAsync(p->acc, 0, sizeof(float) * (size_t)p->n * astride, st)); }
    int c0 = 0, rc = GSVOX_OK;
    if (channels == 1) rc = launch_bwd_ch<1, true>(p, weight, channels, 0, grad_out, astride, st);
    else {
        // multi-channel: groups of 9 / 3 / 1; the a-moments of the groups add up in acc
        while (c0 < channels && rc == GSVOX_OK) {
            int left = channels - c0;
            if (left >= 9)      { rc = launch_bwd_ch<9, false>(p, weight, channels, c0, grad_out, astride, st); c0 += 9; }
            else if (left >= 3) { rc = launch_bwd_ch<3, false>(p, weight, channels, c0, grad_out, astride, st); c0 += 3; }
            else                { rc = launch_bwd_ch<1, false>(p, weight, channels, c0, grad_out, astride, st); c0 += 1; }
        }
    }
    return rc;
}

// C = 1, for gsvox_step_host: a4 in pieces.  Piece `part` of `nparts` covers a contiguous range of brick layers (whole
// z-slices of the gradient volume), so it can start as soon as THAT part of the upstream gradient has arrived on the
// device; the caller waits on the matching copy event before each call.  part 0 zeroes the accumulators, the last part
// also runs the hot-brick launch (which reads any part of the gradient).
void backward_part_layers(const gsvox_plan* p, int part, int nparts, int* z0, int* z1)
{
    const int nl = p->gd.slab1 - p->gd.slab0;
    *z0 = p->gd.slab0 + (int)((long long)nl * part / nparts);
    *z1 = p->gd.slab0 + (int)((long long)nl * (part + 1) / nparts);
}

int launch_backward_part(gsvox_plan* p, const float* weight, const float* grad_out, int part, int nparts, cudaStream_t st)
{
    const int astride = acc_stride(1);
    if (part == 0) {
        LaunchScope ls(p, GSVOX_K_MEMSET, st);
        GSVOX_CUDA(cudaMemsetAsync(p->acc, 0, sizeof(float) * (size_t)p->n * astride, st));
    }
    int z0, z1;
    backward_part_layers(p, part, nparts, &z0, &z1);
    GridDev gd = p->gd;
    gd.slab0 = z0; gd.slab1 = z1;
    const int nblocks = (z1 - z0) * gd.nb[0] * gd.nb[1];
    LaunchScope ls(p, GSVOX_K_BACKWARD, st);
    if (nblocks > 0) {
        k_backward<1, true><<<nblocks, kBwdThreads, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, weight, 1, 0, grad_out,
                                                             p->acc, astride, gd);
        GSVOX_CUDA(cudaGetLastError());
    }
    if (part == nparts - 1) {
        k_backward_extra<1, true><<<kSplitGrid / 2, kBwdThreads, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, p->split_list,
                                                                         p->split_cap, weight, 1, 0, grad_out, p->acc, astride, p->gd);
        GSVOX_CUDA(cudaGetLastError());
    }
    return GSVOX_OK;
}

int launch_backward(gsvox_plan* p, const float* weight, int channels, const float* grad_out,
                    float* gw, float* gp, float* gs, float* gq, cudaStream_t st)
{
    int rc = launch_backward_accumulate(p, weight, channels, grad_out, st);
    if (rc != GSVOX_OK) return rc;
    return launch_epilogue(p, channels, gw, gp, gs, gq, st);
}

}  // namespace gsvox
