// gsvox_api.cu — host side of the C ABI declared in include/gsvox.h: argument checks,
// workspace carving, plan bookkeeping, status/read-back calls, event timing, host-buffer step.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include "gsvox_internal.cuh"

using namespace gsvox;

static thread_local char g_cuda_err[512] = "";

int gsvox::cuda_fail(cudaError_t e, const char* what)
{
    snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    (void)cudaGetLastError();     // clear the sticky-free error state
    return GSVOX_ECUDA;
}

// ---------------------------------------------------------------------------- timing
gsvox::LaunchScope::LaunchScope(gsvox_plan* plan, int kind_, cudaStream_t s)
    : p(plan), kind(kind_), st(s), a(nullptr), b(nullptr), timed(false)
{
    p->launches[kind] += 1;
    if (p->timing) {
        if (cudaEventCreate(&a) == cudaSuccess && cudaEventCreate(&b) == cudaSuccess) {
            timed = true;
            cudaEventRecord(a, st);
        }
    }
}

gsvox::LaunchScope::~LaunchScope()
{
    if (!timed) return;
    cudaEventRecord(b, st);
    if (p->n_pending == p->cap_pending) {
        int cap = p->cap_pending ? 2 * p->cap_pending : 256;
        void* np = realloc(p->pending, sizeof(gsvox_plan::Pending) * (size_t)cap);
        if (!np) { cudaEventDestroy(a); cudaEventDestroy(b); return; }
        p->pending = (gsvox_plan::Pending*)np; p->cap_pending = cap;
    }
    p->pending[p->n_pending++] = { a, b, kind };
}

extern "C" const char* gsvox_last_cuda_error(void) { return g_cuda_err; }

// ------------------------------------------------------------------- workspace layout
static bool grid_ok(const gsvox_grid* g)
{
    if (!g) return false;
    for (int k = 0; k < 3; ++k) {
        if (!(g->spacing[k] > 0.f) || !std::isfinite(g->spacing[k]) || !std::isfinite(g->origin[k])) return false;
        if (g->dims[k] < 1) return false;
    }
    return true;
}

struct Layout { size_t status, rec, aux, bin_count, bin_start, scan_partial, keys, split, acc, total; int nbins, nbricks, nb[3], split_cap; };

static size_t up256(size_t v) { return (v + 255) & ~(size_t)255; }

static int make_layout(int64_t n_max, int32_t max_channels, const gsvox_grid* g, int64_t key_capacity, Layout* L)
{
    if (!grid_ok(g) || n_max < 0 || key_capacity < 0) return GSVOX_EINVAL;
    if (max_channels < 1 || max_channels > GSVOX_MAX_CHANNELS) return GSVOX_EINVAL;
    for (int k = 0; k < 3; ++k) if (g->dims[k] > GSVOX_MAX_DIM) return GSVOX_ELIMIT;
    if (n_max > 0x7ffffff0LL / 8 || key_capacity > 0xfffffff0LL) return GSVOX_ELIMIT;
    int64_t nbins = 1;
    for (int k = 0; k < 3; ++k) { L->nb[k] = (g->dims[k] + kBrick - 1) / kBrick; nbins *= L->nb[k]; }
    L->nbricks = (int)nbins;
    nbins *= kNumClasses;
    if (nbins > 0x7ffffff0LL) return GSVOX_ELIMIT;
    L->nbins = (int)nbins;
    size_t off = 0;
    L->status = off;       off += up256(sizeof(DevStatus));          // status and bin_count are contiguous:
    L->bin_count = off;    off += up256(sizeof(uint32_t) * (size_t)(nbins + 1));   // one memset clears both
    L->rec = off;          off += up256(sizeof(GsRec) * (size_t)n_max);
    L->aux = off;          off += up256(sizeof(GsAux) * (size_t)n_max);
    L->bin_start = off;    off += up256(sizeof(uint32_t) * (size_t)(nbins + 1));
    size_t sblocks = (size_t)((nbins + kScanItemsPerBlock - 1) / kScanItemsPerBlock);
    L->scan_partial = off; off += up256(sizeof(uint32_t) * (sblocks + 1));
    L->keys = off;         off += up256(sizeof(uint32_t) * (size_t)key_capacity);
    L->split_cap = (int)(key_capacity / kSplitKeys) + 1;              // sum over bricks of floor(keys / kSplitKeys) <= this
    L->split = off;        off += up256(sizeof(uint2) * (size_t)L->split_cap);
    L->acc = off;          off += up256(sizeof(float) * (size_t)n_max * (size_t)acc_stride(max_channels));
    L->total = off;
    return GSVOX_OK;
}

extern "C" int gsvox_workspace_bytes(int64_t n_max, int32_t max_channels, const gsvox_grid* grid,
                                     int64_t key_capacity, size_t* bytes)
{
    if (!bytes) return GSVOX_EINVAL;
    Layout L;
    int rc = make_layout(n_max, max_channels, grid, key_capacity, &L);
    if (rc != GSVOX_OK) return rc;
    *bytes = L.total;
    return GSVOX_OK;
}

extern "C" int gsvox_plan_create(int64_t n_max, int32_t max_channels, const gsvox_grid* grid,
                                 int64_t key_capacity, void* workspace, size_t workspace_bytes,
                                 gsvox_plan** plan)
{
    if (!plan) return GSVOX_EINVAL;
    *plan = nullptr;
    Layout L;
    int rc = make_layout(n_max, max_channels, grid, key_capacity, &L);
    if (rc != GSVOX_OK) return rc;
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < L.total) return GSVOX_EWORKSPACE;
    gsvox_plan* p = new (std::nothrow) gsvox_plan();
    if (!p) return GSVOX_EINVAL;
    memset(p, 0, sizeof *p);
    p->grid = *grid;
    for (int k = 0; k < 3; ++k) {
        p->gd.origin[k] = (double)grid->origin[k]; p->gd.spacing[k] = (double)grid->spacing[k];
        p->gd.dims[k] = grid->dims[k]; p->gd.nb[k] = L.nb[k];
    }
    p->gd.nbricks = L.nbricks;
    p->gd.slab0 = 0; p->gd.slab1 = L.nb[2];
    p->n_max = n_max; p->max_channels = max_channels; p->key_capacity = key_capacity; p->n = -1;
    char* w = (char*)workspace;
    p->status = (DevStatus*)(w + L.status); p->rec = (GsRec*)(w + L.rec); p->aux = (GsAux*)(w + L.aux);
    p->bin_count = (uint32_t*)(w + L.bin_count); p->bin_start = (uint32_t*)(w + L.bin_start);
    p->scan_partial = (uint32_t*)(w + L.scan_partial); p->keys = (uint32_t*)(w + L.keys);
    p->acc = (float*)(w + L.acc);
    p->split_list = (uint2*)(w + L.split); p->split_cap = L.split_cap;
    p->nbins = L.nbins;
    *plan = p;
    return GSVOX_OK;
}

extern "C" void gsvox_plan_destroy(gsvox_plan* p)
{
    if (!p) return;
    for (int i = 0; i < p->n_pending; ++i) { cudaEventDestroy(p->pending[i].a); cudaEventDestroy(p->pending[i].b); }
    free(p->pending);
    if (p->side_ready) {
        for (int i = 0; i < 2; ++i) cudaStreamDestroy(p->side[i]);
        for (int i = 0; i < 4 + 8; ++i) if (p->side_ev[i]) cudaEventDestroy(p->side_ev[i]);
    }
    delete p;
}

// --------------------------------------------------------------------------- hot path
extern "C" int gsvox_preprocess(gsvox_plan* p, const float* pos, const float* scale, const float* quat,
                                int64_t n, void* stream)
{
    if (!p || n < 0 || n > p->n_max) return GSVOX_EINVAL;
    if (n > 0 && (!pos || !scale || !quat)) return GSVOX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = launch_preprocess(p, pos, scale, quat, n, st);
    if (rc != GSVOX_OK) return rc;
    rc = launch_binning(p, n, st);
    if (rc != GSVOX_OK) return rc;
    p->n = n;
    return GSVOX_OK;
}

extern "C" int gsvox_forward(gsvox_plan* p, const float* weight, int32_t channels, float* out, void* stream)
{
    if (!p || !out || channels < 1 || channels > p->max_channels) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    if (p->n > 0 && !weight) return GSVOX_EINVAL;
    return launch_forward(p, weight, channels, out, (cudaStream_t)stream);
}

extern "C" int gsvox_backward(gsvox_plan* p, const float* weight, int32_t channels, const float* grad_out,
                              float* gw, float* gp, float* gs, float* gq, void* stream)
{
    if (!p || channels < 1 || channels > p->max_channels) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    if (p->n == 0) return GSVOX_OK;
    if (!weight || !grad_out || !gw || !gp || !gs || !gq) return GSVOX_EINVAL;
    return launch_backward(p, weight, channels, grad_out, gw, gp, gs, gq, (cudaStream_t)stream);
}

extern "C" int gsvox_plan_set_deterministic(gsvox_plan* p, int32_t enabled)
{
    if (!p) return GSVOX_EINVAL;
    p->deterministic = enabled ? 1 : 0;
    p->n = -1;                                   // the binning in the workspace was made in the other mode
    return GSVOX_OK;
}

// ------------------------------------------------------------------ multi-GPU z-slabs
extern "C" int gsvox_plan_set_slab(gsvox_plan* p, int32_t bz_begin, int32_t bz_end)
{
    if (!p || bz_begin < 0 || bz_end < bz_begin || bz_end > p->gd.nb[2]) return GSVOX_EINVAL;
    p->gd.slab0 = bz_begin; p->gd.slab1 = bz_end;
    p->n = -1;                                   // the binning of the previous slab is stale
    return GSVOX_OK;
}

extern "C" int gsvox_backward_accumulate(gsvox_plan* p, const float* weight, int32_t channels,
                                         const float* grad_out, void* stream)
{
    if (!p || channels < 1 || channels > p->max_channels) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    if (p->n == 0) return GSVOX_OK;
    if (!weight || !grad_out) return GSVOX_EINVAL;
    return launch_backward_accumulate(p, weight, channels, grad_out, (cudaStream_t)stream);
}

extern "C" int gsvox_backward_finish(gsvox_plan* p, int32_t channels, float* gw, float* gp, float* gs,
                                     float* gq, void* stream)
{
    if (!p || channels < 1 || channels > p->max_channels) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    if (p->n == 0) return GSVOX_OK;
    if (!gw || !gp || !gs || !gq) return GSVOX_EINVAL;
    return launch_epilogue(p, channels, gw, gp, gs, gq, (cudaStream_t)stream);
}

extern "C" int gsvox_plan_accumulators(gsvox_plan* p, int32_t channels, float** acc, int64_t* count)
{
    if (!p || !acc || !count || channels < 1 || channels > p->max_channels) return GSVOX_EINVAL;
    if (p->n < 0) return GSVOX_ENOTREADY;
    *acc = p->acc;
    *count = p->n * (int64_t)acc_stride(channels);
    return GSVOX_OK;
}
