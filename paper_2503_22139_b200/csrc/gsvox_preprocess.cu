// gsvox_preprocess.cu — steps a1 (per-Gaussian geometry) and a2 (brick binning).
//
// a1  k_preprocess: one thread per Gaussian, fp64.  Follows DESIGN.md "forward definition"
//     steps 1-5 (Eq. 4; Sigma = R S S^T R^T per north_star).  The box bounds use
//     the operation order of reading A5 with explicitly rounded intrinsics (__dmul_rn, ...),
//     so no FMA contraction can change an integer bound.
// a2  counting sort of (brick, Gaussian) keys by (brick, class): k_keys<0> -> exclusive
//     scan -> k_keys<1>.  Order inside a brick is whatever the atomics produce (sums are order
//     independent within tolerance, reading A13).
#include "gsvox_internal.cuh"

namespace gsvox {

constexpr float kCullQ = 64.0f;
constexpr double kCullBoxRatio = 8.0;     // config 4's 6:1 Gaussians stay below 7.6: the test costs them nothing

__device__ __forceinline__ bool finite_d(double v) { return isfinite(v); }

__global__ void __launch_bounds__(256, 3)
k_preprocess(const float* __restrict__ pos, const float* __restrict__ scale,
             const float* __restrict__ quat, int n, GridDev gd,
             GsRec* __restrict__ rec, GsAux* __restrict__ aux, DevStatus* __restrict__ status)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long my_pairs = 0; unsigned int my_skipped = 0;
    if (i < n) {
        double p[3], s[3], q[4];
        for (int k = 0; k < 3; ++k) { p[k] = (double)pos[3 * i + k]; s[k] = (double)scale[3 * i + k]; }
        for (int k = 0; k < 4; ++k) q[k] = (double)quat[4 * i + k];
        bool bad = false;
        for (int k = 0; k < 3; ++k) bad |= !finite_d(p[k]) || !finite_d(s[k]) || !(s[k] > 0.0);
        for (int k = 0; k < 4; ++k) bad |= !finite_d(q[k]);
        bad |= (q[0] == 0.0 && q[1] == 0.0 && q[2] == 0.0 && q[3] == 0.0);

        GsAux a;
        for (int k = 0; k < 4; ++k) a.q[k] = (float)q[k];
        for (int k = 0; k < 3; ++k) a.s[k] = (float)s[k];
        a.valid = bad ? 0u : 1u;
        aux[i] = a;

        GsRec r;
        r.cf[0] = r.cf[1] = r.cf[2] = 0.f; r.cexp = 1.f; r.ci[0] = r.ci[1] = r.ci[2] = 0;
        r.negA = r.nl01 = r.nl02 = r.l12 = r.nD1 = r.nD2 = 0.f;
        r.lo[0] = r.lo[1] = r.lo[2] = 0; r.hi[0] = r.hi[1] = r.hi[2] = -1;
        if (bad) { my_skipped = 1; }
        else {
            // step 1: normalise (reading A5 order: ((r*r + x*x) + y*y) + z*z)
            double n2 = __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(q[0], q[0]), __dmul_rn(q[1], q[1])),
                                            __dmul_rn(q[2], q[2])), __dmul_rn(q[3], q[3]));
            double nn = __dsqrt_rn(n2);
            double qr = __ddiv_rn(q[0], nn), qx = __ddiv_rn(q[1], nn),
                   qy = __ddiv_rn(q[2], nn), qz = __ddiv_rn(q[3], nn);
            // step 2: rotation matrix, entries as written in the definition
            double R[9];
            #define MUL __dmul_rn
            #define ADD __dadd_rn
            #define SUB __dsub_rn
            R[0] = SUB(1.0, MUL(2.0, ADD(MUL(qy, qy), MUL(qz, qz))));
            R[1] = MUL(2.0, SUB(MUL(qx, qy), MUL(qr, qz)));
            R[2] = MUL(2.0, ADD(MUL(qx, qz), MUL(qr, qy)));
            R[3] = MUL(2.0, ADD(MUL(qx, qy), MUL(qr, qz)));
            R[4] = SUB(1.0, MUL(2.0, ADD(MUL(qx, qx), MUL(qz, qz))));
            R[5] = MUL(2.0, SUB(MUL(qy, qz), MUL(qr, qx)));
            R[6] = MUL(2.0, SUB(MUL(qx, qz), MUL(qr, qy)));
            R[7] = MUL(2.0, ADD(MUL(qy, qz), MUL(qr, qx)));
            R[8] = SUB(1.0, MUL(2.0, ADD(MUL(qx, qx), MUL(qy, qy))));
            // steps 4-5: r_k = 3 sqrt(Sigma_kk), integer box clipped to the grid
            double s0 = MUL(s[0], s[0]), s1 = MUL(s[1], s[1]), s2 = MUL(s[2], s[2]);
            bool empty = false; int lo[3], hi[3];
            double rprod = 1.0;
            #pragma unroll
            for (int k = 0; k < 3; ++k) {
                double Skk = ADD(ADD(MUL(MUL(R[3 * k], R[3 * k]), s0),
                                     MUL(MUL(R[3 * k + 1], R[3 * k + 1]), s1)),
                                 MUL(MUL(R[3 * k + 2], R[3 * k + 2]), s2));
                double rk = MUL(GSVOX_SIGMA_CUTOFF, __dsqrt_rn(Skk));
                rprod *= rk;
                double l = ceil(__ddiv_rn(SUB(SUB(p[k], rk), gd.origin[k]), gd.spacing[k]));
                double h = floor(__ddiv_rn(SUB(ADD(p[k], rk), gd.origin[k]), gd.spacing[k]));
                double top = (double)(gd.dims[k] - 1);
                if (l < 0.0) l = 0.0;
                if (h > top) h = top;
                if (!(h >= l)) { empty = true; lo[k] = 0; hi[k] = -1; }
                else { lo[k] = (int)l; hi[k] = (int)h; }
            }
            #undef MUL
            #undef ADD
            #undef SUB
            if (!empty) {
                my_pairs = (unsigned long long)(hi[0] - lo[0] + 1) * (unsigned long long)(hi[1] - lo[1] + 1)
                         * (unsigned long long)(hi[2] - lo[2] + 1);
                // step 3 in index units: M = H R diag(1/s^2) R^T H, H = diag(spacing)
                double is2[3] = { 1.0 / s0, 1.0 / s1, 1.0 / s2 };
                double M[6]; int t = 0;
                for (int a2 = 0; a2 < 3; ++a2)
                    for (int b = a2; b < 3; ++b) {
                        double acc = 0.0;
                        for (int j = 0; j < 3; ++j) acc += R[3 * a2 + j] * is2[j] * R[3 * b + j];
                        M[t++] = acc * gd.spacing[a2] * gd.spacing[b];      // xx xy xz yy yz zz
                    }
                // LDL^T, x eliminated first (x is the row direction of a3/a4)
                const double k2 = 0.72134752044448170368;                  // log2(e)/2
                double D0 = M[0], l01 = M[1] / D0, l02 = M[2] / D0;
                double D1 = M[3] - M[1] * l01;
                double l12 = (M[4] - M[1] * l02) / D1;
                double D2 = M[5] - M[2] * l02 - l12 * l12 * D1;
                if (!(D1 > 0.0)) { D1 = 0.0; l12 = 0.0; }                   // rounding guard
                if (!(D2 > 0.0)) D2 = 0.0;
                r.negA = (float)(-k2 * D0); r.nl01 = (float)(-l01); r.nl02 = (float)(-l02);
                r.l12 = (float)l12; r.nD1 = (float)(-k2 * D1); r.nD2 = (float)(-k2 * D2);
                r.cexp = (float)exp2(-2.0 * k2 * D0);
                // a2 cull flag in the sign bit of cexp (readers take fabsf): the box holds > 8x the volume of
                // the box of the unrotated 3-sigma ellipsoid, i.e. it is mostly empty space (thin and rotated)
                const double kap3 = GSVOX_SIGMA_CUTOFF * GSVOX_SIGMA_CUTOFF * GSVOX_SIGMA_CUTOFF;
                if (rprod > kCullBoxRatio * kap3 * s[0] * s[1] * s[2]) r.cexp = -r.cexp;
                for (int k = 0; k < 3; ++k) {
                    double c = (p[k] - gd.origin[k]) / gd.spacing[k];
                    double ci = rint(c);
                    if (ci > 1073741824.0) ci = 1073741824.0;
                    if (ci < -1073741824.0) ci = -1073741824.0;
                    r.ci[k] = (int)ci; r.cf[k] = (float)(c - ci);
                    r.lo[k] = (int16_t)lo[k]; r.hi[k] = (int16_t)hi[k];
                }
            }
        }
        rec[i] = r;
    }
    // block-level totals -> one atomic per block
    __shared__ unsigned long long sh_pairs[8]; __shared__ unsigned int sh_skip[8];
    for (int o = 16; o > 0; o >>= 1) {
        my_pairs += __shfl_xor_sync(0xffffffffu, my_pairs, o);
        my_skipped += __shfl_xor_sync(0xffffffffu, my_skipped, o);
    }
    int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { sh_pairs[w] = my_pairs; sh_skip[w] = my_skipped; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long tp = 0; unsigned int ts = 0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { tp += sh_pairs[k]; ts += sh_skip[k]; }
        if (tp) atomicAdd(&status->pairs, tp);
        if (ts) atomicAdd(&status->skipped, ts);
    }
}

// ------------------------------------------------------------------------------------------
// a2: keys.  A warp walks the bricks of the boxes of its (up to 32) Gaussians as one flat list (k_keys below).
// MODE 0: count keys per (brick, class) bin.  MODE 1: claim a slot per key and write the Gaussian id.
//
// Negligible keys are dropped (reading A15; SURVEY.md section 7 hard part 7): the axis-aligned box
// of a thin rotated Gaussian is mostly empty space (config 5's needles: 91 % of all pairs, 0.8 % of
// them with q < 9).  For a brick, in the Gaussian's principal frame t = S^-1 R^T (x - p), each t_k is
// linear in x, so over the brick it spans centre_k +- half_k with half_k = sum_j |R_jk| h_j 3.5 / s_k,
// and q = |t|^2 >= sum_k max(|centre_k| - half_k, 0)^2.  A key is kept unless that lower bound
// exceeds kCullQ = 64: every dropped term is below w e^-32 = 1.3e-14 w, far inside the forward
// tolerance even with 1e5 keys per brick.  Both passes take the decision with the same code on the
// same data.  Dropped keys and the pairs of kept keys (P_exec) are counted in DevStatus.  Only Gaussians
// flagged by a1 (box volume > 8x the unrotated ellipsoid box: thin AND rotated) run the test, the rest
// pay nothing (unflagged: 0.23 ms of binning at config 4; testing every key cost 0.31 ms).
// ------------------------------------------------------------------------------------------

// The brick test of one flagged Gaussian, in two parts.  cull_setup (once per Gaussian and pass): each principal
// coordinate t_k of a brick centre is affine in the brick's offset (tx, ty, tz) from the first brick of the box,
//     c_k = c0_k + tx ax_k + ty ay_k + tz az_k,     and spans +- half_k over the brick;
// 15 floats, kept in shared memory (one set per warp).  key_negligible (per brick): 9 FMA + 3 x 4.
// (Round 1 rebuilt R from the quaternion for every brick: ~70 instructions per test, 2.9e7 tests per pass at config 5.)
__device__ __forceinline__ void cull_setup(const GsRec* __restrict__ rec, const GsAux* __restrict__ aux, int g,
                                           float h0, float h1, float h2, int bx0, int by0, int bz0, float* __restrict__ cq)
{
    const int4* rp = reinterpret_cast<const int4*>(rec + g);
    const int4 w0 = __ldg(rp), w1 = __ldg(rp + 1);                        // cf, cexp | ci, negA
    const float4 qa = __ldg(reinterpret_cast<const float4*>(aux + g));
    const float4 sa = __ldg(reinterpret_cast<const float4*>(aux + g) + 1);
    const float qn = rsqrtf(qa.x * qa.x + qa.y * qa.y + qa.z * qa.z + qa.w * qa.w);
    const float r = qa.x * qn, x = qa.y * qn, y = qa.z * qn, z = qa.w * qn;
    // rows of R scaled by the spacing: t_k = (1/s_k) sum_j R_jk h_j (x_j - c_j) in index units
    const float Rm[9] = { (1.f - 2.f * (y * y + z * z)) * h0, 2.f * (x * y - r * z) * h0, 2.f * (x * z + r * y) * h0,
                          2.f * (x * y + r * z) * h1, (1.f - 2.f * (x * x + z * z)) * h1, 2.f * (y * z - r * x) * h1,
                          2.f * (x * z - r * y) * h2, 2.f * (y * z + r * x) * h2, (1.f - 2.f * (x * x + y * y)) * h2 };
    const float is[3] = { 1.f / sa.x, 1.f / sa.y, 1.f / sa.z };
    const float d0 = (float)(8 * bx0 - w1.x) + (3.5f - __int_as_float(w0.x));      // centre of the first brick
    const float d1 = (float)(8 * by0 - w1.y) + (3.5f - __int_as_float(w0.y));
    const float d2 = (float)(8 * bz0 - w1.z) + (3.5f - __int_as_float(w0.z));
    #pragma unroll
    for (int k = 0; k < 3; ++k) {
        cq[5 * k + 0] = (Rm[k] * d0 + Rm[3 + k] * d1 + Rm[6 + k] * d2) * is[k];
        cq[5 * k + 1] = 8.f * Rm[k] * is[k]; cq[5 * k + 2] = 8.f * Rm[3 + k] * is[k]; cq[5 * k + 3] = 8.f * Rm[6 + k] * is[k];
        cq[5 * k + 4] = 3.5f * (fabsf(Rm[k]) + fabsf(Rm[3 + k]) + fabsf(Rm[6 + k])) * is[k];
    }
}

__device__ __forceinline__ bool key_negligible(const float* __restrict__ cq, int tx, int ty, int tz)
{
    const float fx = (float)tx, fy = (float)ty, fz = (float)tz;
    float qmin = 0.f;
    #pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float c = fmaf(fz, cq[5 * k + 3], fmaf(fy, cq[5 * k + 2], fmaf(fx, cq[5 * k + 1], cq[5 * k])));
        const float dist = fmaxf(fabsf(c) - cq[5 * k + 4], 0.f);
        qmin = fmaf(dist, dist, qmin);
    }
    return qmin > kCullQ;
}

// One WARP takes 32 consecutive Gaussians and walks the keys of all of them as ONE flat list, 32 keys per trip:
// lane l decodes Gaussian l (box, brick range, key count), the live ones are compacted into a shared-memory table
// (8 words each) with the exclusive prefix sum of their key counts, and key j of the list belongs to the last
// entry whose start is <= j.  Per trip that owner is found without a search: the starts that fall inside the
// trip's window [j0, j0 + 32) are OR-ed into a 32-bit mask (redux.sync), so
//     owner(lane) = #(starts <= j0) - 1 + popc(mask & bits 1..lane).
// Every lane then has a key in every trip but the last, whatever the mix of box sizes (round 2's first scheme gave each
// Gaussian 8 lanes: ncu counted 17 of 32 lanes active and 131 thread instructions per key, the decode replicated
// eight times; the count pass was issue-bound at 81 %, not atomics-bound).
constexpr int kKeysThreads = 128;
constexpr int kKeysWarps = kKeysThreads / 32;

struct KeyOwner {                      // 8 words in shared memory
    int w_lo, w_mid, w_hi;             // the record's packed int16 box: lox|loy, loz|hix, hiy|hiz
    int b01;                           // bx0 | by0 << 16 | direct << 31
    int b2g;                           // bz0 | lane << 16
    int exy;                           // ex | ey << 16
    float inv_ex, inv_ey;
};

// Bin of key t of an owner: (brick, class).  t -> (tx, ty, tz) by reciprocal multiplies with a +-1 fix-up
// (exact while t < 2^23; larger boxes take the parked route below).
__device__ __forceinline__ int owner_bin(const KeyOwner& o, int t, const GridDev& gd)
{
    const int ex = o.exy & 0xffff, ey = o.exy >> 16;
    int r = (int)(__int2float_rz(t) * o.inv_ex), tx = t - r * ex;
    if (tx >= ex) { ++r; tx -= ex; }
    if (tx < 0) { --r; tx += ex; }
    int tz = (int)(__int2float_rz(r) * o.inv_ey), ty = r - tz * ey;
    if (ty >= ey) { ++tz; ty -= ey; }
    if (ty < 0) { --tz; ty += ey; }
    const int bx = (o.b01 & 0x7fff) + tx, by = ((o.b01 >> 16) & 0x7fff) + ty, bz = (o.b2g & 0xffff) + tz;
    const int loy = o.w_lo >> 16, loz = (int16_t)(o.w_mid & 0xffff), hiy = (int16_t)(o.w_hi & 0xffff), hiz = o.w_hi >> 16;
    const int y0 = max(loy - 8 * by, 0), y1 = min(hiy - 8 * by, 7), z0 = max(loz - 8 * bz, 0), z1 = min(hiz - 8 * bz, 7);
    return ((bz * gd.nb[1] + by) * gd.nb[0] + bx) * kNumClasses + key_class(o.b01 < 0, 0, 7, y0, y1, z0, z1);
}

template <int MODE>
__global__ void __launch_bounds__(kKeysThreads, 10)
k_keys(const GsRec* __restrict__ rec, const GsAux* __restrict__ aux, int n, int gw, GridDev gd,
       uint32_t* __restrict__ bin_count, uint32_t* __restrict__ keys, DevStatus* __restrict__ status,
       const uint32_t* __restrict__ bin_start, uint2* __restrict__ split_list, int split_cap)
{
    if (MODE == 1 && status->overflow) return;
    if (MODE == 1) {
        // the scan is done: list the key-range segments beyond the first of every hot brick (kSplitKeys)
        const int b_lo = gd.slab0 * gd.nb[0] * gd.nb[1], b_hi = gd.slab1 * gd.nb[0] * gd.nb[1];
        for (int b = b_lo + blockIdx.x * blockDim.x + threadIdx.x; b < b_hi; b += gridDim.x * blockDim.x) {
            const uint32_t nk = bin_start[(b + 1) * kNumClasses] - bin_start[b * kNumClasses];
            if (nk > (uint32_t)kSplitKeys) {
                const uint32_t extra = (nk - 1u) / (uint32_t)kSplitKeys;
                const uint32_t at = atomicAdd(&status->nsplit, extra);
                for (uint32_t sgm = 0; sgm < extra; ++sgm)
                    if (at + sgm < (uint32_t)split_cap) split_list[at + sgm] = make_uint2((uint32_t)b, sgm + 1u);
            }
        }
    }
    __shared__ __align__(16) KeyOwner s_own[kKeysWarps][32];
    __shared__ int s_start[kKeysWarps][32];
    __shared__ float s_cull[kKeysWarps][16];
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, wq = threadIdx.x >> 5;
    const int wbase = (blockIdx.x * kKeysWarps + wq) * gw;      // this warp's gw (a power of two <= 32) Gaussians
    const int g = wbase + lane;
    unsigned long long my_pairs = 0ull;
    unsigned int my_culled = 0u;

    // ---- decode Gaussian `lane`
    int total = 0;
    bool park = false;
    KeyOwner me;
    me.w_lo = me.w_mid = 0; me.w_hi = -1; me.b01 = 0; me.b2g = lane << 16; me.exy = 1 | (1 << 16); me.inv_ex = me.inv_ey = 1.f;
    if (lane < gw && g < n) {
        const int4* rp = reinterpret_cast<const int4*>(rec + g);
        const int4 w3 = __ldg(rp + 3);                      // bytes 48..63: nD2, lo[3], hi[3]
        const bool direct = -__int_as_float(__ldg(rp + 1).w) > kRecurrenceMaxA;      // negA at byte 28
        const int lox = (int16_t)(w3.y & 0xffff), loy = w3.y >> 16, loz = (int16_t)(w3.z & 0xffff);
        const int hix = w3.z >> 16, hiy = (int16_t)(w3.w & 0xffff), hiz = w3.w >> 16;
        if (hix >= lox) {
            const int bx0 = lox >> 3, by0 = loy >> 3, bz0 = max(loz >> 3, gd.slab0);          // z-slab of this plan only
            const int ex = (hix >> 3) - bx0 + 1, ey = (hiy >> 3) - by0 + 1;
            const int ez = min(hiz >> 3, gd.slab1 - 1) - bz0 + 1;
            if (ez > 0) {
                const int tot = ex * ey * ez;                 // < 2^31: nbricks is an int
                const bool cullable = (tot > 1) && (__ldg(reinterpret_cast<const int*>(rec + g) + 3) < 0);   // sign bit of cexp
                park = cullable || tot >= (1 << 23);
                total = park ? 0 : tot;
                me.w_lo = w3.y; me.w_mid = w3.z; me.w_hi = w3.w;
                me.b01 = bx0 | (by0 << 16) | (direct ? (int)0x80000000u : 0);
                me.b2g = bz0 | (lane << 16);
                me.exy = ex | (ey << 16);
                me.inv_ex = __frcp_rn((float)ex); me.inv_ey = __frcp_rn((float)ey);
                if (MODE == 0 && !park) {                   // every key of an unflagged Gaussian is kept: P_exec = its box (in this slab)
                    const int zl = max(loz, 8 * gd.slab0), zh = min(hiz, 8 * gd.slab1 - 1);
                    my_pairs = (unsigned long long)((hix - lox + 1) * (hiy - loy + 1)) * (unsigned long long)(zh - zl + 1);
                }
            }
        }
    }
    // ---- compact the live Gaussians, prefix-sum their key counts
    const unsigned live_mask = __ballot_sync(full, total > 0);
    const int nlive = __popc(live_mask);
    int incl = total;
    #pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(full, incl, o); if (lane >= o) incl += v; }
    const int T = __shfl_sync(full, incl, 31);
    if (total > 0) {
        const int c = __popc(live_mask & ((1u << lane) - 1u));
        int4* dst = reinterpret_cast<int4*>(&s_own[wq][c]);
        dst[0] = make_int4(me.w_lo, me.w_mid, me.w_hi, me.b01);
        dst[1] = make_int4(me.b2g, me.exy, __float_as_int(me.inv_ex), __float_as_int(me.inv_ey));
        s_start[wq][c] = incl - total;
    }
    unsigned parked = __ballot_sync(full, park);
    __syncwarp();
    const int start_c = (lane < nlive) ? s_start[wq][lane] : 0x7fffffff;
    // ---- the flat key list, 32 keys per trip (scatter pass: two trips at once, so that both slot-returning atomics
    //      of a lane are in flight before the stores)
    constexpr int kTrips = (MODE == 0) ? 1 : 2;
    for (int j0 = 0; j0 < T; j0 += 32 * kTrips) {
        int bin[kTrips], gid[kTrips];
        #pragma unroll
        for (int u = 0; u < kTrips; ++u) {
            const int jb = j0 + 32 * u, j = jb + lane;
            const unsigned m = __reduce_or_sync(full, (start_c > jb && start_c < jb + 32) ? (1u << (start_c - jb)) : 0u);
            const int first = __popc(__ballot_sync(full, start_c <= jb)) - 1;
            bin[u] = -1; gid[u] = 0;
            if (j < T) {
                const int owner = first + __popc(m & (0xffffffffu >> (31 - lane)));
                const int4* src = reinterpret_cast<const int4*>(&s_own[wq][owner]);
                const int4 a = src[0], b = src[1];
                KeyOwner o;
                o.w_lo = a.x; o.w_mid = a.y; o.w_hi = a.z; o.b01 = a.w; o.b2g = b.x; o.exy = b.y;
                o.inv_ex = __int_as_float(b.z); o.inv_ey = __int_as_float(b.w);
                bin[u] = owner_bin(o, j - s_start[wq][owner], gd);
                gid[u] = wbase + (o.b2g >> 16);
            }
        }
        if (MODE == 0) {
            if (bin[0] >= 0) atomicAdd(&bin_count[bin[0]], 1u);
        } else {
            uint32_t slot[kTrips];
            #pragma unroll
            for (int u = 0; u < kTrips; ++u) slot[u] = (bin[u] >= 0) ? atomicAdd(&bin_count[bin[u]], 1u) : 0u;
            #pragma unroll
            for (int u = 0; u < kTrips; ++u) if (bin[u] >= 0) keys[slot[u]] = (uint32_t)gid[u];
        }
    }
    // ---- the parked Gaussians of this warp (flagged needles: boxes of hundreds of bricks, most of them culled; and
    //      boxes of 2^23 bricks or more), one after another, 32 bricks per trip
    while (parked) {                                     // warp-uniform
        const int pl = __ffs(parked) - 1;
        parked &= parked - 1u;
        const int pg = wbase + pl;
        const int4* rp = reinterpret_cast<const int4*>(rec + pg);
        const int4 w3 = __ldg(rp + 3);
        const bool pdirect = -__int_as_float(__ldg(rp + 1).w) > kRecurrenceMaxA;
        const bool flagged = __ldg(reinterpret_cast<const int*>(rec + pg) + 3) < 0;
        const int lox = (int16_t)(w3.y & 0xffff), loy = w3.y >> 16, loz = (int16_t)(w3.z & 0xffff);
        const int hix = w3.z >> 16, hiy = (int16_t)(w3.w & 0xffff), hiz = w3.w >> 16;
        const int bx0 = lox >> 3, by0 = loy >> 3, bz0 = max(loz >> 3, gd.slab0);
        const int pex = (hix >> 3) - bx0 + 1, pey = (hiy >> 3) - by0 + 1;
        const int ptotal = pex * pey * (min(hiz >> 3, gd.slab1 - 1) - bz0 + 1);      // < 2^31: nbricks is an int
        if (flagged) {
            if (lane == 0) cull_setup(rec, aux, pg, (float)gd.spacing[0], (float)gd.spacing[1], (float)gd.spacing[2],
                                      bx0, by0, bz0, s_cull[wq]);
            __syncwarp();
        }
        const float* cq = s_cull[wq];
        for (int t = lane; t < ptotal; t += 32) {
            const int tx = t % pex, r = t / pex, ty = r % pey, tz = r / pey;
            if (flagged && key_negligible(cq, tx, ty, tz)) { my_culled += 1u; continue; }
            const int bx = bx0 + tx, by = by0 + ty, bz = bz0 + tz;
            const int x0 = max(lox - 8 * bx, 0), x1 = min(hix - 8 * bx, 7), y0 = max(loy - 8 * by, 0), y1 = min(hiy - 8 * by, 7);
            const int z0 = max(loz - 8 * bz, 0), z1 = min(hiz - 8 * bz, 7);
            if (MODE == 0) my_pairs += (unsigned long long)((x1 - x0 + 1) * (y1 - y0 + 1) * (z1 - z0 + 1));
            const int bin = ((bz * gd.nb[1] + by) * gd.nb[0] + bx) * kNumClasses + key_class(pdirect, x0, x1, y0, y1, z0, z1);
            if (MODE == 0) atomicAdd(&bin_count[bin], 1u);
            else keys[atomicAdd(&bin_count[bin], 1u)] = (uint32_t)pg;
        }
        __syncwarp();                                    // s_cull is rewritten for the next parked Gaussian
    }
    if (MODE == 0) {
        // P_exec and the culled count: warp -> ONE global atomic pair per warp that has something to add
        for (int o = 16; o > 0; o >>= 1) {
            my_pairs += __shfl_xor_sync(full, my_pairs, o);
            my_culled += __shfl_xor_sync(full, my_culled, o);
        }
        if (lane == 0) {
            if (my_pairs) atomicAdd(&status->pairs_exec, my_pairs);
            if (my_culled) atomicAdd(&status->culled, (unsigned long long)my_culled);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Exclusive scan over the nbins counters: reduce, then apply (each tile sums the tile totals before it); beyond
// kScanFusedTiles tiles a single-block scan of the tile totals runs in between.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_scan_reduce(const uint32_t* __restrict__ cnt, int nbins, uint32_t* __restrict__ partial)
{
    int base = blockIdx.x * kScanItemsPerBlock;
    uint32_t s = 0;
    for (int k = threadIdx.x; k < kScanItemsPerBlock; k += 256) {
        int idx = base + k;
        if (idx < nbins) s += cnt[idx];
    }
    __shared__ uint32_t sh[8];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t t = 0; for (int k = 0; k < 8; ++k) t += sh[k]; partial[blockIdx.x] = t; }
}

__global__ void __launch_bounds__(1024)
k_scan_partials(uint32_t* __restrict__ partial, int nblocks, unsigned long long* __restrict__ keys_needed,
                unsigned int* __restrict__ overflow,
                unsigned long long key_capacity)
{
    // single block: serial-per-thread chunks + warp scans; nblocks is small (<= a few thousand)
    __shared__ unsigned long long sh[1024];
    int per = (nblocks + 1023) / 1024;
    int b0 = threadIdx.x * per;
    unsigned long long s = 0;
    for (int k = 0; k < per; ++k) if (b0 + k < nblocks) s += partial[b0 + k];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        unsigned long long v = (threadIdx.x >= o) ? sh[threadIdx.x - o] : 0ull;
        __syncthreads();
        sh[threadIdx.x] += v;
        __syncthreads();
    }
    unsigned long long run = sh[threadIdx.x] - s;           // exclusive prefix of this chunk
    for (int k = 0; k < per; ++k)
        if (b0 + k < nblocks) { uint32_t v = partial[b0 + k]; partial[b0 + k] = (uint32_t)run; run += v; }
    if (threadIdx.x == 1023) {
        unsigned long long total = sh[1023];
        *keys_needed = total;
        *overflow = (total > key_capacity || total > 0xfffffff0ull) ? 1u : 0u;
    }
}

// SUMMED = false: partial[] already holds the exclusive prefix of the tile sums (k_scan_partials ran).
// SUMMED = true: partial[] holds the tile sums themselves and every CTA adds up the ones before it (two launches
// instead of three; quadratic in the tile count, so only for up to kScanFusedTiles tiles); the last CTA reports the total.
constexpr int kScanFusedTiles = 4096;
template <bool SUMMED>
__global__ void __launch_bounds__(256)
k_scan_apply(uint32_t* __restrict__ cnt, int nbins, const uint32_t* __restrict__ partial,
             uint32_t* __restrict__ start, unsigned long long* __restrict__ keys_needed,
             unsigned int* __restrict__ overflow, unsigned long long key_capacity)
{
    // 256 threads x 8 consecutive items; counts are replaced by write cursors (= start)
    __shared__ uint32_t sh[8];
    __shared__ unsigned long long sh_off[8];
    unsigned long long tile_off = 0ull;
    if (SUMMED) {
        unsigned long long a = 0ull;
        for (int k = threadIdx.x; k < (int)blockIdx.x; k += 256) a += partial[k];
        for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if ((threadIdx.x & 31) == 0) sh_off[threadIdx.x >> 5] = a;
        __syncthreads();
        #pragma unroll
        for (int k = 0; k < 8; ++k) tile_off += sh_off[k];
    } else {
        tile_off = partial[blockIdx.x];
    }
    int base = blockIdx.x * kScanItemsPerBlock + threadIdx.x * 8;
    uint32_t v[8]; uint32_t s = 0;
    #pragma unroll
    for (int k = 0; k < 8; ++k) { v[k] = (base + k < nbins) ? cnt[base + k] : 0u; s += v[k]; }
    uint32_t inc = s;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) sh[w] = inc;
    __syncthreads();
    uint32_t woff = 0;
    for (int k = 0; k < w; ++k) woff += sh[k];
    uint32_t run = (uint32_t)tile_off + woff + inc - s;       // 32-bit cursors: a total beyond 2^32 - 16 is an overflow
    #pragma unroll
    for (int k = 0; k < 8; ++k) {
        if (base + k < nbins) { start[base + k] = run; cnt[base + k] = run; }
        run += v[k];
    }
    // sentinel start[nbins] = total
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 255) {
        start[nbins] = run;
        if (SUMMED) {
            uint32_t mine = 0;
            for (int k = 0; k < 8; ++k) mine += sh[k];
            const unsigned long long total = tile_off + mine;
            *keys_needed = total;
            *overflow = (total > key_capacity || total > 0xfffffff0ull) ? 1u : 0u;
        }
    }
}

// cnt[nbins] -> start[nbins + 1] (exclusive scan, start[nbins] = total); cnt is overwritten by the same
// offsets (write cursors for the scatter pass); *keys_needed = total, *overflow = total > capacity.
// partial: scratch of ceil(nbins / kScanItemsPerBlock) + 1 words.  Shared by the voxelizer and the rasterizer.
int launch_exclusive_scan(uint32_t* cnt, int nbins, uint32_t* partial, uint32_t* start,
                          unsigned long long* keys_needed, unsigned int* overflow,
                          unsigned long long key_capacity, cudaStream_t st)
{
    const int sblocks = (nbins + kScanItemsPerBlock - 1) / kScanItemsPerBlock;
    k_scan_reduce<<<sblocks, 256, 0, st>>>(cnt, nbins, partial);
    if (sblocks <= kScanFusedTiles) {
        k_scan_apply<true><<<sblocks, 256, 0, st>>>(cnt, nbins, partial, start, keys_needed, overflow, key_capacity);
    } else {
        k_scan_partials<<<1, 1024, 0, st>>>(partial, sblocks, keys_needed, overflow, key_capacity);
        k_scan_apply<false><<<sblocks, 256, 0, st>>>(cnt, nbins, partial, start, keys_needed, overflow, key_capacity);
    }
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

// ------------------------------------------------------------------------------------------
// Deterministic mode (gsvox_plan_set_deterministic; SURVEY section 7 hard part 3, section 4 test 6): the counting
// sort leaves the keys of a (brick, class) bin in whatever order the atomics produced.  Here every bin is sorted by
// Gaussian id, in place: the bin is loaded into shared memory, every key counts the smaller ones (ids are unique
// inside a bin), and is written to that rank.  k_sort_bins: one CTA per brick, bins up to kSortSmall keys (config 4:
// 18 keys per bin on average).  k_sort_bins_large: the longer bins of hot bricks (one item of the split list per
// brick), up to kSortLarge keys in 200 KB of shared memory; anything longer stays unsorted and is counted.
// ------------------------------------------------------------------------------------------
constexpr int kSortSmall = 4096, kSortLarge = 51200;

template <int THREADS>
__device__ __forceinline__ void sort_bin_in_place(uint32_t* __restrict__ keys, uint32_t beg, uint32_t len, uint32_t* s_keys)
{
    for (uint32_t i = threadIdx.x; i < len; i += THREADS) s_keys[i] = keys[beg + i];
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < len; i += THREADS) {
        const uint32_t mine = s_keys[i];
        uint32_t rank = 0;
        for (uint32_t j = 0; j < len; ++j) rank += (s_keys[j] < mine) ? 1u : 0u;
        keys[beg + rank] = mine;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(128)
k_sort_bins(const uint32_t* __restrict__ bin_start, uint32_t* __restrict__ keys, const DevStatus* __restrict__ status, GridDev gd)
{
    __shared__ uint32_t s_keys[kSortSmall];
    if (status->overflow) return;
    const int b = blockIdx.x + gd.slab0 * gd.nb[0] * gd.nb[1];
    for (int c = 0; c < kNumClasses; ++c) {
        const uint32_t beg = bin_start[b * kNumClasses + c], len = bin_start[b * kNumClasses + c + 1] - beg;
        if (len >= 2u && len <= (uint32_t)kSortSmall) sort_bin_in_place<128>(keys, beg, len, s_keys);     // CTA-uniform
    }
}

__global__ void __launch_bounds__(1024)
k_sort_bins_large(const uint32_t* __restrict__ bin_start, uint32_t* __restrict__ keys, DevStatus* __restrict__ status,
                  const uint2* __restrict__ split_list, int split_cap)
{
    extern __shared__ uint32_t s_big[];
    if (status->overflow) return;
    const uint32_t nitems = min(status->nsplit, (uint32_t)split_cap);
    for (uint32_t i = blockIdx.x; i < nitems; i += gridDim.x) {
        const uint2 item = split_list[i];
        if (item.y != 1u) continue;                          // one item per hot brick does the brick
        for (int c = 0; c < kNumClasses; ++c) {
            const uint32_t beg = bin_start[item.x * kNumClasses + c], len = bin_start[item.x * kNumClasses + c + 1] - beg;
            if (len <= (uint32_t)kSortSmall) continue;
            if (len <= (uint32_t)kSortLarge) sort_bin_in_place<1024>(keys, beg, len, s_big);
            else if (threadIdx.x == 0) atomicAdd(&status->unsorted, 1u);
        }
    }
}

int launch_sort_bins(gsvox_plan* p, cudaStream_t st)
{
    const int nblocks = (p->gd.slab1 - p->gd.slab0) * p->gd.nb[0] * p->gd.nb[1];
    if (nblocks <= 0) return GSVOX_OK;
    LaunchScope ls(p, GSVOX_K_SCATTER, st);
    k_sort_bins<<<nblocks, 128, 0, st>>>(p->bin_start, p->keys, p->status, p->gd);
    GSVOX_CUDA(cudaGetLastError());
    const size_t smem = sizeof(uint32_t) * (size_t)kSortLarge;
    GSVOX_CUDA(cudaFuncSetAttribute(k_sort_bins_large, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_sort_bins_large<<<148, 1024, smem, st>>>(p->bin_start, p->keys, p->status, p->split_list, p->split_cap);
    GSVOX_CUDA(cudaGetLastError());
    p->launches[GSVOX_K_SCATTER] += 1;
    return GSVOX_OK;
}

int launch_preprocess(gsvox_plan* p, const float* pos, const float* scale, const float* quat,
                      int64_t n, cudaStream_t st)
{
    { LaunchScope ls(p, GSVOX_K_MEMSET, st);        // status block + bin counters, contiguous in the workspace
      size_t bytes = (size_t)((char*)p->bin_count - (char*)p->status) + sizeof(uint32_t) * (size_t)(p->nbins + 1);
      GSVOX_CUDA(cudaMemsetAsync(p->status, 0, bytes, st)); }
    if (n > 0) {
        LaunchScope ls(p, GSVOX_K_PREPROCESS, st);
        int blocks = (int)((n + 255) / 256);
        k_preprocess<<<blocks, 256, 0, st>>>(pos, scale, quat, (int)n, p->gd, p->rec, p->aux, p->status);
        GSVOX_CUDA(cudaGetLastError());
    }
    return GSVOX_OK;
}

int launch_binning(gsvox_plan* p, int64_t n, cudaStream_t st)
{
    // Gaussians per warp: 32 when that still leaves >= 8192 warps, fewer otherwise, down to one warp per Gaussian
    // (measured count + scatter: config 4, 500 k Gaussians x 20 keys, 0.188 / 0.195 / 0.214 / 0.256 ms at 32 / 16 / 8 / 4;
    //  config 3 level 1, 1000 Gaussians x 1336 keys, 0.91 / 0.25 / 0.138 / 0.065 ms at 32 / 8 / 4 / 1;
    //  level 3, 64 k x 31 keys, 0.069 / 0.062 / 0.073 at 32 / 4 / 2)
    int gw = 32;
    while (gw > 1 && n / gw < 8192) gw >>= 1;
    const int64_t kwarps = (n + gw - 1) / gw;
    const int kblocks = (int)((kwarps + kKeysWarps - 1) / kKeysWarps);
    if (n > 0) {
        LaunchScope ls(p, GSVOX_K_COUNT, st);
        k_keys<0><<<kblocks, kKeysThreads, 0, st>>>(p->rec, p->aux, (int)n, gw, p->gd, p->bin_count, p->keys, p->status,
                                           p->bin_start, p->split_list, p->split_cap);
        GSVOX_CUDA(cudaGetLastError());
    }
    { LaunchScope ls(p, GSVOX_K_SCAN, st);
      int rc = launch_exclusive_scan(p->bin_count, p->nbins, p->scan_partial, p->bin_start, &p->status->keys_needed,
                                     &p->status->overflow, (unsigned long long)p->key_capacity, st);
      p->launches[GSVOX_K_SCAN] += ((p->nbins + kScanItemsPerBlock - 1) / kScanItemsPerBlock <= kScanFusedTiles) ? 1 : 2;   // two or three kernels
      if (rc != GSVOX_OK) return rc; }
    if (n > 0) {
        LaunchScope ls(p, GSVOX_K_SCATTER, st);
        k_keys<1><<<kblocks, kKeysThreads, 0, st>>>(p->rec, p->aux, (int)n, gw, p->gd, p->bin_count, p->keys, p->status,
                                           p->bin_start, p->split_list, p->split_cap);
        GSVOX_CUDA(cudaGetLastError());
        if (p->deterministic) { int rc = launch_sort_bins(p, st); if (rc != GSVOX_OK) return rc; }
    }
    return GSVOX_OK;
}

}  // namespace gsvox
