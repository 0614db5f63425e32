// gsvox_host.cu — the synchronising calls of the C ABI: status, parity read-backs, timings,
// and the host-buffer end-to-end step (bench.py's e2e leg).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#include "gsvox_internal.cuh"

using namespace gsvox;

constexpr int kStepParts = 4;       // pieces of the upstream gradient in gsvox_step_host (C = 1)

static void drain(gsvox_plan* p)
{
    for (int i = 0; i < p->n_pending; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p->pending[i].a, p->pending[i].b) == cudaSuccess)
            p->ms[p->pending[i].kind] += (double)ms;
        cudaEventDestroy(p->pending[i].a); cudaEventDestroy(p->pending[i].b);
    }
    p->n_pending = 0;
}

extern "C" int gsvox_plan_status(gsvox_plan* p, gsvox_status* status, void* stream)
{
    if (!p || !status) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    cudaStream_t st = (cudaStream_t)stream;
    DevStatus h;
    GSVOX_CUDA(cudaMemcpyAsync(&h, p->status, sizeof h, cudaMemcpyDeviceToHost, st));
    GSVOX_CUDA(cudaStreamSynchronize(st));
    status->keys_needed = (int64_t)h.keys_needed;
    status->pairs = (int64_t)h.pairs;
    status->skipped_gaussians = (int32_t)h.skipped;
    status->overflow = (int32_t)h.overflow;
    status->culled_keys = (int64_t)h.culled;
    status->pairs_exec = (int64_t)h.pairs_exec;
    return GSVOX_OK;
}

extern "C" int gsvox_plan_unsorted_bins(gsvox_plan* p, int64_t* unsorted_bins, void* stream)
{
    if (!p || !unsorted_bins) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    cudaStream_t st = (cudaStream_t)stream;
    DevStatus h;
    GSVOX_CUDA(cudaMemcpyAsync(&h, p->status, sizeof h, cudaMemcpyDeviceToHost, st));
    GSVOX_CUDA(cudaStreamSynchronize(st));
    *unsorted_bins = p->deterministic ? (int64_t)h.unsorted : -1;
    return GSVOX_OK;
}

extern "C" int gsvox_plan_geometry_host(gsvox_plan* p, int32_t* box_host, float* minv_host, void* stream)
{
    if (!p) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    cudaStream_t st = (cudaStream_t)stream;
    size_t n = (size_t)p->n;
    std::vector<GsRec> h(n);
    if (n) GSVOX_CUDA(cudaMemcpyAsync(h.data(), p->rec, n * sizeof(GsRec), cudaMemcpyDeviceToHost, st));
    GSVOX_CUDA(cudaStreamSynchronize(st));
    const double k2 = 0.72134752044448170368;
    for (size_t i = 0; i < n; ++i) {
        const GsRec& r = h[i];
        bool empty = r.hi[0] < r.lo[0];
        if (box_host) {
            for (int k = 0; k < 3; ++k) {
                box_host[6 * i + k] = empty ? 0 : r.lo[k];
                box_host[6 * i + 3 + k] = empty ? -1 : r.hi[k];
            }
        }
        if (minv_host) {
            // undo the LDL^T factorisation: M = L D L^T with unit-lower L
            double D0 = -r.negA / k2, D1 = -r.nD1 / k2, D2 = -r.nD2 / k2;
            double l01 = -r.nl01, l02 = -r.nl02, l12 = r.l12;
            float* m = minv_host + 6 * i;
            m[0] = (float)D0; m[1] = (float)(D0 * l01); m[2] = (float)(D0 * l02);
            m[3] = (float)(D1 + D0 * l01 * l01);
            m[4] = (float)(D1 * l12 + D0 * l01 * l02);
            m[5] = (float)(D2 + D1 * l12 * l12 + D0 * l02 * l02);
            if (empty) for (int k = 0; k < 6; ++k) m[k] = 0.f;
        }
    }
    return GSVOX_OK;
}

extern "C" int gsvox_plan_bins_host(gsvox_plan* p, int64_t* brick_start_host, int32_t* key_gaussian_host,
                                    int64_t key_host_capacity, void* stream)
{
    if (!p || !brick_start_host) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<uint32_t> hs((size_t)p->nbins + 1);
    GSVOX_CUDA(cudaMemcpyAsync(hs.data(), p->bin_start, hs.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    GSVOX_CUDA(cudaStreamSynchronize(st));
    for (int i = 0; i <= p->gd.nbricks; ++i) brick_start_host[i] = (int64_t)hs[(size_t)i * kNumClasses];
    int64_t total = (int64_t)hs[p->nbins];
    if (key_gaussian_host) {
        if (total > key_host_capacity || total > p->key_capacity) return GSVOX_EWORKSPACE;
        if (total) GSVOX_CUDA(cudaMemcpyAsync(key_gaussian_host, p->keys, (size_t)total * sizeof(uint32_t),
                                              cudaMemcpyDeviceToHost, st));
        GSVOX_CUDA(cudaStreamSynchronize(st));
    }
    return GSVOX_OK;
}

extern "C" int gsvox_plan_set_timing(gsvox_plan* p, int32_t enabled)
{
    if (!p) return GSVOX_EINVAL;
    p->timing = enabled ? 1 : 0;
    return GSVOX_OK;
}

extern "C" int gsvox_plan_timings(gsvox_plan* p, double* ms, int64_t* launches, int32_t reset, void* stream)
{
    if (!p) return GSVOX_EINVAL;
    GSVOX_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    drain(p);
    for (int k = 0; k < GSVOX_K_COUNT_KINDS; ++k) {
        if (ms) ms[k] = p->ms[k];
        if (launches) launches[k] = p->launches[k];
        if (reset) { p->ms[k] = 0.0; p->launches[k] = 0; }
    }
    return GSVOX_OK;
}

// --------------------------------------------------------------------- host-buffer step
struct Staging { size_t pos, scale, quat, weight, vol_out, vol_grad, gw, gp, gs, gq, total; };

static size_t up256(size_t v) { return (v + 255) & ~(size_t)255; }

static int staging_layout(int64_t n_max, int32_t C, const gsvox_grid* g, Staging* S)
{
    if (!g || n_max < 0 || C < 1 || C > GSVOX_MAX_CHANNELS) return GSVOX_EINVAL;
    for (int k = 0; k < 3; ++k) if (g->dims[k] < 1) return GSVOX_EINVAL;
    size_t V = (size_t)g->dims[0] * g->dims[1] * g->dims[2];
    size_t n = (size_t)n_max, off = 0;
    S->pos = off;      off += up256(n * 3 * 4);
    S->scale = off;    off += up256(n * 3 * 4);
    S->quat = off;     off += up256(n * 4 * 4);
    S->weight = off;   off += up256(n * C * 4);
    S->vol_out = off;  off += up256(V * C * 4);
    S->vol_grad = off; off += up256(V * C * 4);
    S->gw = off;       off += up256(n * C * 4);
    S->gp = off;       off += up256(n * 3 * 4);
    S->gs = off;       off += up256(n * 3 * 4);
    S->gq = off;       off += up256(n * 4 * 4);
    S->total = off;
    return GSVOX_OK;
}

extern "C" int gsvox_host_staging_bytes(int64_t n_max, int32_t max_channels, const gsvox_grid* grid, size_t* bytes)
{
    if (!bytes) return GSVOX_EINVAL;
    Staging S;
    int rc = staging_layout(n_max, max_channels, grid, &S);
    if (rc == GSVOX_OK) *bytes = S.total;
    return rc;
}

static int step_host_enqueue(gsvox_plan* p, void* staging, size_t staging_bytes,
                             const float* pos_h, const float* scale_h, const float* quat_h,
                             const float* weight_h, int64_t n, int32_t C,
                             const float* grad_out_h, float* out_h,
                             float* gw_h, float* gp_h, float* gs_h, float* gq_h, void* stream);

extern "C" int gsvox_step_host(gsvox_plan* p, void* staging, size_t staging_bytes,
                               const float* pos_h, const float* scale_h, const float* quat_h,
                               const float* weight_h, int64_t n, int32_t C,
                               const float* grad_out_h, float* out_h,
                               float* gw_h, float* gp_h, float* gs_h, float* gq_h, void* stream)
{
    int rc = step_host_enqueue(p, staging, staging_bytes, pos_h, scale_h, quat_h, weight_h, n, C, grad_out_h, out_h,
                               gw_h, gp_h, gs_h, gq_h, stream);
    if (rc != GSVOX_OK && p && p->side_ready) {
        // an error after the first enqueue: copies that reference the caller's host buffers may still be in flight
        // on the two copy streams and on the caller's stream — drain them before control returns
        cudaStreamSynchronize(p->side[0]); cudaStreamSynchronize(p->side[1]);
        cudaStreamSynchronize((cudaStream_t)stream);
        (void)cudaGetLastError();
    }
    return rc;
}

static int step_host_enqueue(gsvox_plan* p, void* staging, size_t staging_bytes,
                             const float* pos_h, const float* scale_h, const float* quat_h,
                             const float* weight_h, int64_t n, int32_t C,
                             const float* grad_out_h, float* out_h,
                             float* gw_h, float* gp_h, float* gs_h, float* gq_h, void* stream)
{
    if (!p || !staging || n < 0 || n > p->n_max || C < 1 || C > p->max_channels) return GSVOX_EINVAL;
    // a z-slab plan writes its own brick layers only: the whole-volume copy below would hand out the rest unwritten
    if (p->gd.slab0 != 0 || p->gd.slab1 != p->gd.nb[2]) return GSVOX_EINVAL;
    if (n > 0 && (!pos_h || !scale_h || !quat_h || !weight_h)) return GSVOX_EINVAL;
    if (grad_out_h && n > 0 && (!gw_h || !gp_h || !gs_h || !gq_h)) return GSVOX_EINVAL;
    Staging S;
    int rc = staging_layout(p->n_max, p->max_channels, &p->grid, &S);
    if (rc != GSVOX_OK) return rc;
    if (((uintptr_t)staging & 255) || staging_bytes < S.total) return GSVOX_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    char* d = (char*)staging;
    size_t V = (size_t)p->grid.dims[0] * p->grid.dims[1] * p->grid.dims[2];
    size_t nn = (size_t)n;
    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    // Two copy streams keep both DMA engines busy beside the kernels: the upstream gradient (the
    // large H2D) travels while a1-a3 run, the volume (the large D2H) while a4-a5 run.
    if (!p->side_ready) {
        for (int i = 0; i < 2; ++i) GSVOX_CUDA(cudaStreamCreateWithFlags(&p->side[i], cudaStreamNonBlocking));
        for (int i = 0; i < 4 + kStepParts; ++i) GSVOX_CUDA(cudaEventCreateWithFlags(&p->side_ev[i], cudaEventDisableTiming));
        p->side_ready = 1;
    }
    cudaStream_t up = p->side[0], down = p->side[1];
    cudaEvent_t ev_begin = p->side_ev[0], ev_grad = p->side_ev[1], ev_fwd = p->side_ev[2], ev_out = p->side_ev[3];
    GSVOX_CUDA(cudaEventRecord(ev_begin, st));                 // the copy streams start after the caller's earlier work
    if (nn) {
        GSVOX_CUDA(cudaMemcpyAsync(d + S.pos, pos_h, nn * 12, H2D, st));
        GSVOX_CUDA(cudaMemcpyAsync(d + S.scale, scale_h, nn * 12, H2D, st));
        GSVOX_CUDA(cudaMemcpyAsync(d + S.quat, quat_h, nn * 16, H2D, st));
        GSVOX_CUDA(cudaMemcpyAsync(d + S.weight, weight_h, nn * C * 4, H2D, st));
    }
    // C = 1: the upstream gradient travels in kStepParts pieces of whole brick layers, and a4 runs piece by piece as they
    // arrive (the upload of 67 MB at config 4 takes longer than a1-a3; a4 used to wait for all of it)
    const bool parts = grad_out_h && C == 1 && nn > 0 && p->gd.nb[2] >= kStepParts;
    if (grad_out_h) {
        GSVOX_CUDA(cudaStreamWaitEvent(up, ev_begin, 0));
        if (parts) {
            const size_t slice = (size_t)p->grid.dims[0] * p->grid.dims[1];
            for (int k = 0; k < kStepParts; ++k) {
                int z0, z1;
                backward_part_layers(p, k, kStepParts, &z0, &z1);
                const size_t v0 = slice * (size_t)std::min(z0 * kBrick, p->grid.dims[2]), v1 = slice * (size_t)std::min(z1 * kBrick, p->grid.dims[2]);
                if (v1 > v0) GSVOX_CUDA(cudaMemcpyAsync(d + S.vol_grad + 4 * v0, grad_out_h + v0, 4 * (v1 - v0), H2D, up));
                GSVOX_CUDA(cudaEventRecord(p->side_ev[4 + k], up));
            }
        } else {
            GSVOX_CUDA(cudaMemcpyAsync(d + S.vol_grad, grad_out_h, V * C * 4, H2D, up));
        }
        GSVOX_CUDA(cudaEventRecord(ev_grad, up));
    }
    rc = gsvox_preprocess(p, (float*)(d + S.pos), (float*)(d + S.scale), (float*)(d + S.quat), n, stream);
    if (rc != GSVOX_OK) return rc;
    rc = gsvox_forward(p, (float*)(d + S.weight), C, (float*)(d + S.vol_out), stream);
    if (rc != GSVOX_OK) return rc;
    if (out_h) {
        GSVOX_CUDA(cudaEventRecord(ev_fwd, st));
        GSVOX_CUDA(cudaStreamWaitEvent(down, ev_fwd, 0));
        GSVOX_CUDA(cudaMemcpyAsync(out_h, d + S.vol_out, V * C * 4, D2H, down));
        GSVOX_CUDA(cudaEventRecord(ev_out, down));
    }
    if (grad_out_h && !parts) GSVOX_CUDA(cudaStreamWaitEvent(st, ev_grad, 0));
    if (grad_out_h && nn) {
        if (parts) {
            for (int k = 0; k < kStepParts; ++k) {
                GSVOX_CUDA(cudaStreamWaitEvent(st, p->side_ev[4 + k], 0));
                rc = launch_backward_part(p, (float*)(d + S.weight), (float*)(d + S.vol_grad), k, kStepParts, st);
                if (rc != GSVOX_OK) return rc;
            }
            rc = launch_epilogue(p, 1, (float*)(d + S.gw), (float*)(d + S.gp), (float*)(d + S.gs), (float*)(d + S.gq), st);
        } else {
            rc = gsvox_backward(p, (float*)(d + S.weight), C, (float*)(d + S.vol_grad), (float*)(d + S.gw),
                                (float*)(d + S.gp), (float*)(d + S.gs), (float*)(d + S.gq), stream);
        }
        if (rc != GSVOX_OK) return rc;
        GSVOX_CUDA(cudaMemcpyAsync(gw_h, d + S.gw, nn * C * 4, D2H, st));
        GSVOX_CUDA(cudaMemcpyAsync(gp_h, d + S.gp, nn * 12, D2H, st));
        GSVOX_CUDA(cudaMemcpyAsync(gs_h, d + S.gs, nn * 12, D2H, st));
        GSVOX_CUDA(cudaMemcpyAsync(gq_h, d + S.gq, nn * 16, D2H, st));
    }
    if (out_h) GSVOX_CUDA(cudaStreamWaitEvent(st, ev_out, 0));
    GSVOX_CUDA(cudaStreamSynchronize(st));
    return GSVOX_OK;
}

extern "C" const char* gsvox_error_string(int code)
{
    switch (code) {
        case GSVOX_OK: return "ok";
        case GSVOX_EINVAL: return "invalid argument";
        case GSVOX_EWORKSPACE: return "workspace too small or misaligned";
        case GSVOX_ECUDA: return "CUDA error (see gsvox_last_cuda_error)";
        case GSVOX_ENOTREADY: return "gsvox_preprocess has not been called on this plan";
        case GSVOX_ELIMIT: return "size beyond library limits";
        default: return "unknown error";
    }
}

extern "C" int gsvox_version(void) { return 100; }
