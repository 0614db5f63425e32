// gsvox_backward.cu — steps a4 (per-brick backward) and a5 (per-Gaussian chain rule).
//
// a4  One CTA per 8^3 brick.  The brick's upstream-gradient tile (CH x 512 floats) is staged in
//     shared memory; then every THREAD takes one (brick, Gaussian) key and walks the rows of
//     box ∩ brick itself, so the reduction over voxels that the gradient needs happens in
//     registers with no cross-lane traffic.  Per row it forms the three x-moments
//     U0,U1,U2 = sum_k a_k {1, u0, u0^2},  a_k = (sum_c g_c w_c) G_k,  u0 = k - xs, from which
//     every first and second moment of u = L^T d follows (u1, u2 are constant along a row;
//     M = L D L^T).  Moments are kept in this u frame because sqrt(D) u is an orthogonal
//     rotation of the whitened coordinates S^-1 R^T d: fp32 sums then lose nothing to the
//     anisotropy of the Gaussian (a world-frame d d^T sum loses (s_max/s_min)^2).  Per key it
//     issues vector reductions (red.global.add.v4.f32) of the 9 moments + C weight gradients
//     into acc[g][...] = { m_u0,m_u1,m_u2, m_00,m_01,m_02,m_11,m_12,m_22, dw_0..dw_{C-1} },
//     index units.  G is recomputed exactly as in a3.
// a5  k_epilogue: one thread per Gaussian, fp64: d = L^-T u, dL/dp = M S1, D_M = -1/2 S2, then
//     dL/ds, dL/dq through R(q/|q|) as in DESIGN.md "backward definition".
#include "gsvox_internal.cuh"

namespace gsvox {

constexpr int kBwdThreads = 128;
constexpr float kRecurrenceMaxA_b = 1.0f;

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

template <int CH, bool SINGLE>
__global__ void __launch_bounds__(kBwdThreads)
k_backward(const GsRec* __restrict__ rec, const uint32_t* __restrict__ bin_start,
           const uint32_t* __restrict__ keys, const DevStatus* __restrict__ status,
           const float* __restrict__ weight, int wstride, int c0,
           const float* __restrict__ grad_out, float* __restrict__ acc, int astride, GridDev gd)
{
    __shared__ __align__(16) float s_g[CH * kBrickVox];
    if (status->overflow) return;
    const int b = blockIdx.x;
    const uint32_t kbeg = bin_start[b], kend = bin_start[b + 1];
    if (kbeg == kend) return;
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
            s_g[e] = val;
        }
    }
    __syncthreads();

    for (uint32_t k = kbeg + tid; k < kend; k += kBwdThreads) {
        const uint32_t gid = keys[k];
        const float4* rp = reinterpret_cast<const float4*>(rec + gid);
        const float4 ra = __ldg(rp), rb4 = __ldg(rp + 1), rc = __ldg(rp + 2), rd = __ldg(rp + 3);
        const int w1 = __float_as_int(rd.y), w2 = __float_as_int(rd.z), w3 = __float_as_int(rd.w);
        const int lox = (int16_t)(w1 & 0xffff), loy = (int16_t)(w1 >> 16), loz = (int16_t)(w2 & 0xffff);
        const int hix = (int16_t)(w2 >> 16), hiy = (int16_t)(w3 & 0xffff), hiz = (int16_t)(w3 >> 16);
        const int x0 = max(lox - b0x, 0), x1 = min(hix - b0x, 7);
        const int y0 = max(loy - b0y, 0), y1 = min(hiy - b0y, 7);
        const int z0 = max(loz - b0z, 0), z1 = min(hiz - b0z, 7);
        const uint32_t xm = ((2u << x1) - (1u << x0)) & 0xffu;
        const float cx = (float)(__float_as_int(rb4.x) - b0x) + ra.x;
        const float cy = (float)(__float_as_int(rb4.y) - b0y) + ra.y;
        const float cz = (float)(__float_as_int(rb4.z) - b0z) + ra.z;
        const float negA = rb4.w, nl01 = rc.x, nl02 = rc.y, l12 = rc.z, nD1 = rc.w, nD2 = rd.x, cc = ra.w;
        const bool direct = (-negA > kRecurrenceMaxA_b);
        float wv[CH];
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) wv[ch] = __ldg(weight + (size_t)gid * wstride + c0 + ch);

        float b0 = 0.f, bu0 = 0.f, bu1 = 0.f, bu2 = 0.f, b00 = 0.f, b01 = 0.f, b02 = 0.f, b11 = 0.f, b12 = 0.f, b22 = 0.f;
        float dw[CH];
        #pragma unroll
        for (int ch = 0; ch < CH; ++ch) dw[ch] = 0.f;

        int y = y0, z = z0;
        const int nrows = (y1 - y0 + 1) * (z1 - z0 + 1);
        for (int r = 0; r < nrows; ++r) {
            const float dy = (float)y - cy, dz = (float)z - cz;
            const float u1 = fmaf(l12, dz, dy);
            const float xs = fmaf(nl02, dz, fmaf(nl01, dy, cx));
            const float Es = fmaf(nD2 * dz, dz, (nD1 * u1) * u1);
            float G[8];
            if (!direct) {
                const float t3 = 3.0f - xs;
                const float nAt = negA * t3;
                G[3] = ex2b(fmaf(nAt, t3, Es));
                float rf = ex2b(fminf(fmaf(nAt, 2.0f, negA), 120.f));
                float rbk = ex2b(fminf(fmaf(nAt, -2.0f, negA), 120.f));
                G[4] = G[3] * rf; rf *= cc; G[5] = G[4] * rf; rf *= cc; G[6] = G[5] * rf; rf *= cc; G[7] = G[6] * rf;
                G[2] = G[3] * rbk; rbk *= cc; G[1] = G[2] * rbk; rbk *= cc; G[0] = G[1] * rbk;
            } else {
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) { const float t = (float)k2 - xs; G[k2] = ex2b(fmaf(negA * t, t, Es)); }
            }
            #pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) G[k2] = (xm & (1u << k2)) ? G[k2] : 0.f;

            // a_k = (sum_c g_c w_c) G_k for the 8 voxels of the row (w factored out when SINGLE)
            const float* grow = s_g + ((z << 3) + y) * 8;
            float av[8];
            if (SINGLE) {
                const float4 g0 = *reinterpret_cast<const float4*>(grow);
                const float4 g1 = *reinterpret_cast<const float4*>(grow + 4);
                const float gv[8] = { g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w };
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) av[k2] = gv[k2] * G[k2];
            } else {
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) av[k2] = 0.f;
                #pragma unroll
                for (int ch = 0; ch < CH; ++ch) {
                    const float4 g0 = *reinterpret_cast<const float4*>(grow + ch * kBrickVox);
                    const float4 g1 = *reinterpret_cast<const float4*>(grow + ch * kBrickVox + 4);
                    const float gv[8] = { g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w };
                    float d = 0.f;
                    #pragma unroll
                    for (int k2 = 0; k2 < 8; ++k2) { d = fmaf(gv[k2], G[k2], d); av[k2] = fmaf(gv[k2], wv[ch], av[k2]); }
                    dw[ch] += d;
                }
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) av[k2] *= G[k2];
            }
            // x-moments about xs: U0 = sum a, U1 = sum a u0, U2 = sum a u0^2, u0 = k - xs
            float U0 = 0.f, U1 = 0.f, U2 = 0.f;
            if (!direct) {
                // about the brick-local index, then shifted (profile is wide: mild cancellation)
                float S1 = 0.f, S2 = 0.f;
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) {
                    U0 += av[k2]; S1 = fmaf(av[k2], (float)k2, S1); S2 = fmaf(av[k2], (float)(k2 * k2), S2);
                }
                U1 = fmaf(-xs, U0, S1);
                U2 = fmaf(xs, fmaf(xs, U0, -2.0f * S1), S2);
            } else {
                // narrow profile: accumulate about xs directly
                #pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) {
                    const float u = (float)k2 - xs, au = av[k2] * u;
                    U0 += av[k2]; U1 += au; U2 = fmaf(au, u, U2);
                }
            }
            // row moments -> key moments in the u frame (u1, u2 = dz constant along the row)
            const float u1U0 = u1 * U0, dzU0 = dz * U0;
            b0 += U0; bu0 += U1; b00 += U2;
            bu1 += u1U0; bu2 += dzU0;
            b01 = fmaf(u1, U1, b01); b02 = fmaf(dz, U1, b02);
            b11 = fmaf(u1, u1U0, b11); b12 = fmaf(dz, u1U0, b12); b22 = fmaf(dz, dzU0, b22);
            if (++y > y1) { y = y0; ++z; }
        }
        float* dst = acc + (size_t)gid * astride;
        if (SINGLE) {
            // moments of a = w g G; dw = sum g G
            const float w = wv[0];
            red_add_v4(dst, w * bu0, w * bu1, w * bu2, w * b00);
            red_add_v4(dst + 4, w * b01, w * b02, w * b11, w * b12);
            red_add_v4(dst + 8, w * b22, b0, 0.f, 0.f);
        } else {
            red_add_v4(dst, bu0, bu1, bu2, b00);
            red_add_v4(dst + 4, b01, b02, b11, b12);
            atomicAdd(dst + 8, b22);
            #pragma unroll
            for (int ch = 0; ch < CH; ++ch) atomicAdd(dst + 9 + c0 + ch, dw[ch]);
        }
    }
}

// ------------------------------------------------------------------------------------------
// a5: chain rule, one thread per Gaussian, fp64 (negligible cost; keeps the rounding of the
// kernel's fp32 sums the only fp32 error in the gradients).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_epilogue(const GsAux* __restrict__ aux, const GsRec* __restrict__ rec, const float* __restrict__ acc, int astride, int n, int C,
           GridDev gd, const DevStatus* __restrict__ status,
           float* __restrict__ gw, float* __restrict__ gp, float* __restrict__ gs, float* __restrict__ gq)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const GsAux a = aux[i];
    const bool dead = (a.valid == 0u) || (status->overflow != 0u);
    const float* m = acc + (size_t)i * astride;
    for (int c = 0; c < C; ++c) gw[(size_t)i * C + c] = dead ? 0.f : m[9 + c];
    if (dead) {
        for (int k = 0; k < 3; ++k) { gp[3 * i + k] = 0.f; gs[3 * i + k] = 0.f; }
        for (int k = 0; k < 4; ++k) gq[4 * i + k] = 0.f;
        return;
    }
    const double h[3] = { gd.spacing[0], gd.spacing[1], gd.spacing[2] };
    // u-frame -> index-frame moments: d = T u, T = L^-T (unit upper triangular), with the
    // fp32 l's the kernel used; then world units: S1 = H T mu, S2 = H T B T^T H
    const GsRec rc = rec[i];
    const double l01 = -(double)rc.nl01, l02 = -(double)rc.nl02, l12 = (double)rc.l12;
    const double T[9] = { 1.0, -l01, l01 * l12 - l02,   0.0, 1.0, -l12,   0.0, 0.0, 1.0 };
    const double mu[3] = { m[0], m[1], m[2] };
    const double B[9] = { m[3], m[4], m[5],   m[4], m[6], m[7],   m[5], m[7], m[8] };
    double S1[3], TB[9], S2[9];
    for (int a2 = 0; a2 < 3; ++a2) {
        S1[a2] = (T[3 * a2] * mu[0] + T[3 * a2 + 1] * mu[1] + T[3 * a2 + 2] * mu[2]) * h[a2];
        for (int k = 0; k < 3; ++k)
            TB[3 * a2 + k] = T[3 * a2] * B[k] + T[3 * a2 + 1] * B[3 + k] + T[3 * a2 + 2] * B[6 + k];
    }
    for (int a2 = 0; a2 < 3; ++a2)
        for (int k = 0; k < 3; ++k)
            S2[3 * a2 + k] = (TB[3 * a2] * T[3 * k] + TB[3 * a2 + 1] * T[3 * k + 1] + TB[3 * a2 + 2] * T[3 * k + 2])
                             * h[a2] * h[k];
    double q[4] = { a.q[0], a.q[1], a.q[2], a.q[3] }, s[3] = { a.s[0], a.s[1], a.s[2] };
    double qn = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    double r = q[0] / qn, x = q[1] / qn, y = q[2] / qn, z = q[3] / qn;
    double R[9] = { 1 - 2 * (y * y + z * z), 2 * (x * y - r * z), 2 * (x * z + r * y),
                    2 * (x * y + r * z), 1 - 2 * (x * x + z * z), 2 * (y * z - r * x),
                    2 * (x * z - r * y), 2 * (y * z + r * x), 1 - 2 * (x * x + y * y) };
    double is2[3] = { 1.0 / (s[0] * s[0]), 1.0 / (s[1] * s[1]), 1.0 / (s[2] * s[2]) };
    // dL/dp = M S1, M = R diag(1/s^2) R^T : t = R^T S1, scaled, rotated back
    double t[3];
    for (int k = 0; k < 3; ++k) t[k] = (R[k] * S1[0] + R[3 + k] * S1[1] + R[6 + k] * S1[2]) * is2[k];
    for (int a2 = 0; a2 < 3; ++a2) gp[3 * i + a2] = (float)(R[3 * a2] * t[0] + R[3 * a2 + 1] * t[1] + R[3 * a2 + 2] * t[2]);
    // D_M = -1/2 S2;  P = D_M R
    double P[9];
    for (int a2 = 0; a2 < 3; ++a2)
        for (int k = 0; k < 3; ++k)
            P[3 * a2 + k] = -0.5 * (S2[3 * a2] * R[k] + S2[3 * a2 + 1] * R[3 + k] + S2[3 * a2 + 2] * R[6 + k]);
    // dL/ds_k = -2 (R^T D_M R)_kk / s_k^3
    for (int k = 0; k < 3; ++k) {
        double d = R[k] * P[k] + R[3 + k] * P[3 + k] + R[6 + k] * P[6 + k];
        gs[3 * i + k] = (float)(-2.0 * d * is2[k] / s[k]);
    }
    // D_R = 2 D_M R diag(1/s^2);  dL/dq^_j = <dR/dq^_j, D_R>
    double DR[9];
    for (int a2 = 0; a2 < 3; ++a2) for (int k = 0; k < 3; ++k) DR[3 * a2 + k] = 2.0 * P[3 * a2 + k] * is2[k];
    double gh[4];
    gh[0] = 2 * (-z * DR[1] + y * DR[2] + z * DR[3] - x * DR[5] - y * DR[6] + x * DR[7]);
    gh[1] = 2 * (y * DR[1] + z * DR[2] + y * DR[3] - 2 * x * DR[4] - r * DR[5] + z * DR[6] + r * DR[7] - 2 * x * DR[8]);
    gh[2] = 2 * (-2 * y * DR[0] + x * DR[1] + r * DR[2] + x * DR[3] + z * DR[5] - r * DR[6] + z * DR[7] - 2 * y * DR[8]);
    gh[3] = 2 * (-2 * z * DR[0] - r * DR[1] + x * DR[2] + r * DR[3] - 2 * z * DR[4] + y * DR[5] + x * DR[6] + y * DR[7]);
    double qh[4] = { r, x, y, z };
    double dot = qh[0] * gh[0] + qh[1] * gh[1] + qh[2] * gh[2] + qh[3] * gh[3];
    for (int k = 0; k < 4; ++k) gq[4 * i + k] = (float)((gh[k] - qh[k] * dot) / qn);
}

template <int CH, bool SINGLE>
static int launch_bwd_ch(gsvox_plan* p, const float* weight, int C, int c0, const float* grad_out,
                         int astride, cudaStream_t st)
{
    LaunchScope ls(p, GSVOX_K_BACKWARD, st);
    k_backward<CH, SINGLE><<<p->nbins, kBwdThreads, 0, st>>>(p->rec, p->bin_start, p->keys, p->status, weight, C, c0,
                                                     grad_out, p->acc, astride, p->gd);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

int launch_backward(gsvox_plan* p, const float* weight, int channels, const float* grad_out,
                    float* gw, float* gp, float* gs, float* gq, cudaStream_t st)
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
    if (rc != GSVOX_OK) return rc;
    { LaunchScope ls(p, GSVOX_K_EPILOGUE, st);
      int blocks = (int)((p->n + 255) / 256);
      k_epilogue<<<blocks, 256, 0, st>>>(p->aux, p->rec, p->acc, astride, (int)p->n, channels, p->gd, p->status, gw, gp, gs, gq);
      GSVOX_CUDA(cudaGetLastError()); }
    return GSVOX_OK;
}

}  // namespace gsvox
