// gsvox_dvf.cu — SURVEY.md 8(f) rank 1: motion-basis components -> deformation vector fields in
// one pass (Eq. 3, d(x,p) = sum_i w_i(p) e_i(x); :106 three levels x three Cartesian
// directions = nine MBC volumes; :141 coefficients w_{i,k}(p) per projection p).
//
// Voxelization is linear in the per-Gaussian value, so
//     d_k(x,p_b) = sum_i w_{i,k}(p_b) sum_{j in level i} f_{j,k} G_j(x) = sum_j [w_{l(j),k}(p_b) f_{j,k}] G_j(x):
// the three levels are ONE Gaussian set voxelized once with the C = 3B per-Gaussian weights
// m_{j,(b,k)} = w_{l(j),k}(p_b) f_{j,k}.  The nine MBC volumes are never written or re-read per
// projection; G_j(x) is evaluated once per channel group of 9 instead of once per MBC volume and
// projection.  k_dvf_mix forms m (a few MB); a3/a4/a5 do the rest; k_dvf_unmix maps dL/dm back to
// dL/df and dL/dw.
#include "gsvox_internal.cuh"

namespace gsvox {

__global__ void __launch_bounds__(256)
k_dvf_mix(const float* __restrict__ feat, const int32_t* __restrict__ level, const float* __restrict__ coef,
          int n, int B, int L, float* __restrict__ mixed)
{
    const int C = 3 * B;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)n * C) return;
    const int j = (int)(idx / C), c = (int)(idx - (long long)j * C);
    const int b = c / 3, k = c - 3 * b;
    const int l = level[j];
    float v = 0.f;
    if (l >= 0 && l < L) v = coef[(b * L + l) * 3 + k] * feat[3 * j + k];      // out-of-range level: no contribution
    mixed[idx] = v;
}

// One thread per Gaussian.  dL/df[j,k] = sum_b w[b,l,k] gm[j,(b,k)];
// dL/dw[b,l,k] = sum_{j in level l} f[j,k] gm[j,(b,k)]: warp-shuffle sums per level, one atomic per warp.
__global__ void __launch_bounds__(256)
k_dvf_unmix(const float* __restrict__ feat, const int32_t* __restrict__ level, const float* __restrict__ coef,
            const float* __restrict__ gmixed, int n, int B, int L,
            float* __restrict__ gfeat, float* __restrict__ gcoef)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = j < n;
    const int C = 3 * B;
    int l = -1;
    float f[3] = { 0.f, 0.f, 0.f }, gf[3] = { 0.f, 0.f, 0.f };
    if (live) {
        l = level[j];
        if (l < 0 || l >= L) l = -1;
        #pragma unroll
        for (int k = 0; k < 3; ++k) f[k] = feat[3 * j + k];
    }
    const int lane = threadIdx.x & 31;
    for (int b = 0; b < B; ++b) {
        #pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float g = (live && l >= 0) ? gmixed[(size_t)j * C + 3 * b + k] : 0.f;
            if (l >= 0) gf[k] = fmaf(coef[(b * L + l) * 3 + k], g, gf[k]);
            const float t = f[k] * g;
            for (int ll = 0; ll < L; ++ll) {
                float s = (l == ll) ? t : 0.f;
                for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
                if (lane == 0 && s != 0.f) atomicAdd(&gcoef[(b * L + ll) * 3 + k], s);
            }
        }
    }
    if (live) {
        #pragma unroll
        for (int k = 0; k < 3; ++k) gfeat[3 * j + k] = gf[k];
    }
}

}  // namespace gsvox

using namespace gsvox;

static int dvf_args_ok(const gsvox_plan* p, int32_t B, int32_t L)
{
    if (!p || B < 1 || L < 1 || L > 64) return GSVOX_EINVAL;
    if ((int64_t)3 * B > p->max_channels) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    return GSVOX_OK;
}

static int launch_mix(gsvox_plan* p, const float* feat, const int32_t* level, const float* coef,
                      int B, int L, float* mixed, cudaStream_t st)
{
    LaunchScope ls(p, GSVOX_K_DVF, st);
    const long long total = (long long)p->n * 3 * B;
    k_dvf_mix<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(feat, level, coef, (int)p->n, B, L, mixed);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

extern "C" int gsvox_dvf_forward(gsvox_plan* p, const float* feat, const int32_t* level, const float* coef,
                                 int32_t B, int32_t L, float* mixed, float* dvf, void* stream)
{
    int rc = dvf_args_ok(p, B, L);
    if (rc != GSVOX_OK) return rc;
    if (!dvf || !coef) return GSVOX_EINVAL;
    if (p->n > 0 && (!feat || !level || !mixed)) return GSVOX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->n > 0) { rc = launch_mix(p, feat, level, coef, B, L, mixed, st); if (rc != GSVOX_OK) return rc; }
    return launch_forward(p, mixed, 3 * B, dvf, st);
}

extern "C" int gsvox_dvf_backward(gsvox_plan* p, const float* feat, const int32_t* level, const float* coef,
                                  int32_t B, int32_t L, float* mixed, const float* grad_dvf, float* grad_mixed,
                                  float* grad_feat, float* grad_coef, float* grad_pos, float* grad_scale,
                                  float* grad_quat, void* stream)
{
    int rc = dvf_args_ok(p, B, L);
    if (rc != GSVOX_OK) return rc;
    if (!coef || !grad_coef) return GSVOX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    { LaunchScope ls(p, GSVOX_K_MEMSET, st);
      GSVOX_CUDA(cudaMemsetAsync(grad_coef, 0, sizeof(float) * (size_t)B * L * 3, st)); }
    if (p->n == 0) return GSVOX_OK;
    if (!feat || !level || !mixed || !grad_dvf || !grad_mixed || !grad_feat || !grad_pos || !grad_scale || !grad_quat)
        return GSVOX_EINVAL;
    rc = launch_mix(p, feat, level, coef, B, L, mixed, st);           // recomputed: coef may have changed since forward
    if (rc != GSVOX_OK) return rc;
    rc = launch_backward(p, mixed, 3 * B, grad_dvf, grad_mixed, grad_pos, grad_scale, grad_quat, st);
    if (rc != GSVOX_OK) return rc;
    LaunchScope ls(p, GSVOX_K_DVF, st);
    k_dvf_unmix<<<(unsigned)((p->n + 255) / 256), 256, 0, st>>>(feat, level, coef, grad_mixed, (int)p->n, B, L,
                                                                 grad_feat, grad_coef);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

// ---------------------------------------------------------------------------------------------
// Two-stage form of the same map, for batches: e = the L x 3 MBC volumes (each level voxelized
// with its own plan, C = 3; BASELINE config 3: "each level voxelized separately"), then
//     dvf[b,k,v] = sum_i coef[b,i,k] e[i,k,v]                                   (Eq. 3)
// The voxelizer is ALU-bound, so for B > 1 projections evaluating G once per level and combining
// the nine volumes B times (HBM-bound, 4 V (3L + 3B) bytes) beats folding the coefficients into
// 3B weight channels, which re-evaluates the exponentials per channel group (measured: DESIGN.md).
// ---------------------------------------------------------------------------------------------
namespace gsvox {

constexpr int kMaxLevels = GSVOX_MAX_LEVELS;
constexpr int kCombThreads = 256;

__device__ __forceinline__ float4 ldg4(const float* p, long long v, long long V)
{
    if (v + 3 < V && ((reinterpret_cast<uintptr_t>(p + v) & 15) == 0)) return __ldg(reinterpret_cast<const float4*>(p + v));
    float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
    if (v < V) r.x = __ldg(p + v);
    if (v + 1 < V) r.y = __ldg(p + v + 1);
    if (v + 2 < V) r.z = __ldg(p + v + 2);
    if (v + 3 < V) r.w = __ldg(p + v + 3);
    return r;
}

__device__ __forceinline__ void stcs4(float* p, long long v, long long V, float4 r)
{
    if (v + 3 < V && ((reinterpret_cast<uintptr_t>(p + v) & 15) == 0)) { __stcs(reinterpret_cast<float4*>(p + v), r); return; }
    if (v < V) p[v] = r.x;
    if (v + 1 < V) p[v + 1] = r.y;
    if (v + 2 < V) p[v + 2] = r.z;
    if (v + 3 < V) p[v + 3] = r.w;
}

// grid = (voxel quads, 3 axes).  Reads the L volumes of axis k once, writes B volumes.
__global__ void __launch_bounds__(kCombThreads)
k_mbc_combine(const float* __restrict__ e, const float* __restrict__ coef, int B, int L, long long V,
              float* __restrict__ dvf)
{
    extern __shared__ float s_coef[];                     // [B][L] for this axis
    const int k = blockIdx.y;
    for (int t = threadIdx.x; t < B * L; t += kCombThreads) s_coef[t] = coef[t * 3 + k];
    __syncthreads();
    const long long v = ((long long)blockIdx.x * kCombThreads + threadIdx.x) * 4;
    if (v >= V) return;
    float4 ev[kMaxLevels];
    #pragma unroll
    for (int i = 0; i < kMaxLevels; ++i)
        ev[i] = (i < L) ? ldg4(e + ((size_t)i * 3 + k) * V, v, V) : make_float4(0.f, 0.f, 0.f, 0.f);
    for (int b = 0; b < B; ++b) {
        float4 d = make_float4(0.f, 0.f, 0.f, 0.f);
        #pragma unroll
        for (int i = 0; i < kMaxLevels; ++i) {
            if (i < L) {
                const float c = s_coef[b * L + i];
                d.x = fmaf(c, ev[i].x, d.x); d.y = fmaf(c, ev[i].y, d.y);
                d.z = fmaf(c, ev[i].z, d.z); d.w = fmaf(c, ev[i].w, d.w);
            }
        }
        stcs4(dvf + ((size_t)b * 3 + k) * V, v, V, d);
    }
}

// grid = (persistent voxel-quad strips, 3 axes).  One pass over grad_dvf and e:
//   grad_e[i,k,v] = sum_b coef[b,i,k] g[b,k,v]            (written once)
//   grad_coef[b,i,k] = sum_v g[b,k,v] e[i,k,v]            (registers -> warp -> block -> one atomic)
// VEC: V % 4 == 0 and 16-byte aligned bases, so every access is one branch-free 128-bit
// instruction and the loads of a chunk of 8 projections are issued back to back (the first
// version tested alignment per load and ptxas serialised the loads behind the branches: 3.0 of
// 6.5 TB/s).  Projections b >= B are clamped to B-1 for the address and carry zero coefficients.
template <int BT, bool VEC>
__global__ void __launch_bounds__(kCombThreads)
k_mbc_combine_bwd(const float* __restrict__ e, const float* __restrict__ coef, const float* __restrict__ g,
                  int B, int L, long long V, float* __restrict__ grad_e, float* __restrict__ grad_coef)
{
    extern __shared__ float s_mem[];                      // [BT][kMaxLevels] coefficients, then [8 warps][BT][kMaxLevels]
    float* s_coef = s_mem;
    float* s_red = s_mem + BT * kMaxLevels;
    const int k = blockIdx.y;
    for (int t = threadIdx.x; t < BT * kMaxLevels; t += kCombThreads) {
        const int b = t / kMaxLevels, i = t - b * kMaxLevels;
        s_coef[t] = (b < B && i < L) ? coef[(b * L + i) * 3 + k] : 0.f;
    }
    __syncthreads();
    float part[BT][kMaxLevels];
    #pragma unroll
    for (int b = 0; b < BT; ++b)
        #pragma unroll
        for (int i = 0; i < kMaxLevels; ++i) part[b][i] = 0.f;
    const long long nquads = (V + 3) / 4;
    for (long long qd = (long long)blockIdx.x * kCombThreads + threadIdx.x; qd < nquads;
         qd += (long long)gridDim.x * kCombThreads) {
        const long long v = qd * 4;
        float4 ev[kMaxLevels], ge[kMaxLevels];
        #pragma unroll
        for (int i = 0; i < kMaxLevels; ++i) {
            const float* src = e + ((size_t)min(i, L - 1) * 3 + k) * V;
            ev[i] = VEC ? __ldg(reinterpret_cast<const float4*>(src + v)) : ldg4(src, v, V);
            ge[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        #pragma unroll
        for (int c0 = 0; c0 < BT; c0 += 8) {
            float4 gv[8];
            #pragma unroll
            for (int bb = 0; bb < 8; ++bb) {
                const float* src = g + ((size_t)min(c0 + bb, B - 1) * 3 + k) * V;
                gv[bb] = VEC ? __ldg(reinterpret_cast<const float4*>(src + v)) : ldg4(src, v, V);
            }
            #pragma unroll
            for (int bb = 0; bb < 8; ++bb) {
                #pragma unroll
                for (int i = 0; i < kMaxLevels; ++i) {
                    const float c = s_coef[(c0 + bb) * kMaxLevels + i];
                    ge[i].x = fmaf(c, gv[bb].x, ge[i].x); ge[i].y = fmaf(c, gv[bb].y, ge[i].y);
                    ge[i].z = fmaf(c, gv[bb].z, ge[i].z); ge[i].w = fmaf(c, gv[bb].w, ge[i].w);
                    part[c0 + bb][i] += (gv[bb].x * ev[i].x + gv[bb].y * ev[i].y) + (gv[bb].z * ev[i].z + gv[bb].w * ev[i].w);
                }
            }
        }
        #pragma unroll
        for (int i = 0; i < kMaxLevels; ++i) {
            if (i < L) {
                float* dst = grad_e + ((size_t)i * 3 + k) * V;
                if (VEC) __stcs(reinterpret_cast<float4*>(dst + v), ge[i]); else stcs4(dst, v, V, ge[i]);
            }
        }
    }
    // reduce the B x L partial dot products over the block
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    #pragma unroll
    for (int b = 0; b < BT; ++b)
        #pragma unroll
        for (int i = 0; i < kMaxLevels; ++i) {
            float s = part[b][i];
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) s_red[(w * BT + b) * kMaxLevels + i] = s;
        }
    __syncthreads();
    for (int t = threadIdx.x; t < BT * kMaxLevels; t += kCombThreads) {
        const int b = t / kMaxLevels, i = t - b * kMaxLevels;
        if (b < B && i < L) {
            float s = 0.f;
            for (int ww = 0; ww < kCombThreads / 32; ++ww) s += s_red[(ww * BT + b) * kMaxLevels + i];
            atomicAdd(&grad_coef[(b * L + i) * 3 + k], s);
        }
    }
}

}  // namespace gsvox

static int comb_args_ok(int32_t B, int32_t L, int64_t V)
{
    if (B < 1 || B > GSVOX_MAX_CHANNELS / 3 || L < 1 || L > GSVOX_MAX_LEVELS || V < 1) return GSVOX_EINVAL;
    return GSVOX_OK;
}

extern "C" int gsvox_mbc_combine_forward(const float* e, const float* coef, int32_t B, int32_t L,
                                         int64_t V, float* dvf, void* stream)
{
    int rc = comb_args_ok(B, L, V);
    if (rc != GSVOX_OK) return rc;
    if (!e || !coef || !dvf) return GSVOX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const long long nquads = (V + 3) / 4;
    dim3 grid((unsigned)((nquads + kCombThreads - 1) / kCombThreads), 3);
    k_mbc_combine<<<grid, kCombThreads, sizeof(float) * B * L, st>>>(e, coef, B, L, (long long)V, dvf);
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}

extern "C" int gsvox_mbc_combine_backward(const float* e, const float* coef, const float* grad_dvf,
                                          int32_t B, int32_t L, int64_t V, float* grad_e, float* grad_coef,
                                          void* stream)
{
    int rc = comb_args_ok(B, L, V);
    if (rc != GSVOX_OK) return rc;
    if (!e || !coef || !grad_dvf || !grad_e || !grad_coef) return GSVOX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    GSVOX_CUDA(cudaMemsetAsync(grad_coef, 0, sizeof(float) * (size_t)B * L * 3, st));
    int dev = 0, sms = 0;
    GSVOX_CUDA(cudaGetDevice(&dev));
    GSVOX_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const long long nquads = (V + 3) / 4;
    long long want = (nquads + kCombThreads - 1) / kCombThreads;
    // persistent strips: about 2 CTAs per SM and axis keep the per-block atomics few
    long long cap = (long long)sms * 2;
    dim3 grid((unsigned)(want < cap ? want : cap), 3);
    const bool vec = (V % 4 == 0) && ((((uintptr_t)e | (uintptr_t)grad_dvf | (uintptr_t)grad_e) & 15) == 0);
    const int bt = (B <= 8) ? 8 : 32;
    const size_t sh = sizeof(float) * ((size_t)bt * kMaxLevels * (1 + kCombThreads / 32));
    #define GSVOX_COMB_LAUNCH(BT_, VEC_) k_mbc_combine_bwd<BT_, VEC_><<<grid, kCombThreads, sh, st>>>( \
        e, coef, grad_dvf, B, L, (long long)V, grad_e, grad_coef)
    if (bt == 8) { if (vec) GSVOX_COMB_LAUNCH(8, true); else GSVOX_COMB_LAUNCH(8, false); }
    else         { if (vec) GSVOX_COMB_LAUNCH(32, true); else GSVOX_COMB_LAUNCH(32, false); }
    #undef GSVOX_COMB_LAUNCH
    GSVOX_CUDA(cudaGetLastError());
    return GSVOX_OK;
}
