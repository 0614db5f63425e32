// gsvox_internal.cuh — shared declarations of the CUDA path (sm_100a only).
// Not part of the public boundary (include/gsvox.h) and never seen by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/gsvox.h"

namespace gsvox {

// ------------------------------------------------------------------------------------------
// Per-Gaussian geometry record written by a1 (k_preprocess), 64 B, read by a3/a4 with four
// 16-byte loads.  Index space: voxel (i,j,k) sits at integer coordinates (i,j,k).
//   centre   = ci + cf   (integer part + fp32 fraction in [-0.5,0.5]: brick-local coordinates
//              (ci - brick_origin) + cf then carry ~1e-7 voxel of error whatever the grid size)
//   exponent (base 2) of Eq. 4 through the LDL^T factorisation of M_idx = H Sigma^-1 H:
//              E = -( A u0^2 + D1 u1^2 + D2 u2^2 ),  u2 = dz, u1 = dy + l12 dz,
//              u0 = dx + l01 dy + l02 dz,  A = kappa2*M00, kappa2 = log2(e)/2
//            a sum of squares: no cancellation for needle-like Gaussians (kernels)
//   cexp     = 2^(-2A), rounded from fp64: ratio of successive ratios along an x-row; its SIGN BIT is
//              a2's cull flag (thin rotated Gaussian: run the per-brick negligibility test); use fabsf
//   box      = inclusive voxel box (reading A5), int16; empty <=> hi[0] < lo[0]
// ------------------------------------------------------------------------------------------
struct __align__(16) GsRec {
    float   cf[3];      //  0
    float   cexp;       // 12
    int32_t ci[3];      // 16
    float   negA;       // 28   -A
    float   nl01, nl02; // 32   -l01, -l02
    float   l12;        // 40
    float   nD1, nD2;   // 44   -D1, -D2 (already times kappa2)
    int16_t lo[3];      // 52
    int16_t hi[3];      // 58
};
static_assert(sizeof(GsRec) == 64, "GsRec must be 64 bytes");

// What a5 (chain rule) needs from the inputs, copied so that the caller's arrays need not
// outlive gsvox_preprocess().
struct __align__(16) GsAux {
    float q[4];
    float s[3];
    uint32_t valid;     // 0 = skipped (degenerate input)
};
static_assert(sizeof(GsAux) == 32, "GsAux must be 32 bytes");

// Device-resident counters of one preprocess.
struct DevStatus {
    unsigned long long keys_needed;
    unsigned long long pairs;
    unsigned int skipped;
    unsigned int overflow;
    unsigned long long culled;        // keys dropped by the conservative q_min > 64 test (reading A15)
    unsigned long long pairs_exec;    // P_exec: pairs of the kept keys
    unsigned int nsplit;              // extra key-range segments of hot bricks (entries of the split list)
    unsigned int unsorted;            // deterministic mode: (brick, class) bins too long to be sorted by Gaussian id
};

struct GridDev {
    double origin[3];
    double spacing[3];
    int dims[3];
    int nb[3];          // bricks per axis
    int nbricks;
    int slab0, slab1;   // brick layers [slab0, slab1) along z this plan works on (multi-GPU z-slabs; default all)
};

constexpr int kBrick = GSVOX_BRICK;
constexpr int kBrickVox = kBrick * kBrick * kBrick;
constexpr int kScanItemsPerBlock = 2048;     // k_scan_*: 256 threads x 8 items
// Rows with A > kRecurrenceMaxA (narrower than ~0.54 voxel along x, conditional sigma) take one EX2 per voxel; the
// others the multiplicative recurrence.  2.5 is what the recurrence's own safety argument allows: the start value
// G(3) can underflow while another voxel of the row is still above 2^-20 only if (106 - 16 A)^2 / (64 A) < 20, i.e.
// A > 2.8; the un-damped geometric chain of a3 peaks at 2^(12 A) = 2^30.  (Round 1 used 1.0: config 5's blobs,
// scales log-uniform 0.5-2, then had 38 % direct keys at ~3x the cost; at 2.5 it is 5 %.)
constexpr float kRecurrenceMaxA = 2.5f;
// Hot bricks (SURVEY section 7 hard part 6; config 5: 1.9e4 keys in one brick against a mean of ~100): a brick's CTA
// of a3 (C = 1) and a4 walks at most kSplitKeys keys, segment 0 of the brick's key range; the segments beyond are
// listed by a2 as (brick, segment) items and worked off by a second, grid-stride launch whose CTAs accumulate
// atomically (a3: red.global.add into the volume the first launch wrote; a4 accumulates atomically anyway).
// No CTA then carries more than kSplitKeys keys, whatever the density.
constexpr int kSplitKeys = 512;
constexpr int kSplitGrid = 148 * 16;         // CTAs of the second launch (each strides over the item list)

// Bins of the counting sort are (brick, class): inside a brick, keys are ordered so that the 32
// keys a backward warp works on have similar trip counts (a4 runs one THREAD per key and walks
// the rows of box ∩ brick).  class 0: direct-exponential keys (A > kRecurrenceMaxA); 1..16: by
// decreasing row count in steps of 4 rows.  Measured lane occupancy of a4 on config 4: 0.48
// unsorted, 0.73 with 8 row classes split by x-fullness, 0.90 (simulated) with 16 row classes.
constexpr int kNumClasses = 17;
__host__ __device__ __forceinline__ int key_class(bool direct, int x0, int x1, int y0, int y1, int z0, int z1)
{
    (void)x0; (void)x1;
    if (direct) return 0;
    const int nrows = (y1 - y0 + 1) * (z1 - z0 + 1);
    return 16 - ((nrows - 1) >> 2);
}

inline __host__ __device__ int acc_stride(int channels) { return (9 + channels + 3) & ~3; }

#ifdef __CUDACC__
// Packed fp32 pairs (sm_100 family FFMA2/FMUL2/FADD2): one issue slot for two lanes of work.  a3/a4
// are issue-bound (profiles/r1b), so halving the instruction count of the per-voxel arithmetic is
// what the packed forms buy; the FP32 pipe rate itself is unchanged (gsvox_probe_peaks).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{ f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float& lo, float& hi)
{ asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{ f32x2 r; asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{ f32x2 r; asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{ f32x2 r; asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
// c += a * b in place: ties the accumulator to one register pair (the three-operand form lets
// ptxas pick a fresh destination and copy back across the key loop's reconvergence points).
__device__ __forceinline__ void fma2_acc(f32x2& c, f32x2 a, f32x2 b)
{ asm("fma.rn.ftz.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b)); }
// Same with the accumulator held as two scalar registers.
__device__ __forceinline__ void fma2_acc(float& clo, float& chi, f32x2 a, f32x2 b)
{
    asm("{\n\t.reg .b64 c;\n\tmov.b64 c, {%0, %1};\n\tfma.rn.ftz.f32x2 c, %2, %3, c;\n\tmov.b64 {%0, %1}, c;\n\t}"
        : "+f"(clo), "+f"(chi) : "l"(a), "l"(b));
}
#endif

}  // namespace gsvox

// The host-side plan (opaque in the public header).
struct gsvox_plan {
    gsvox_grid grid;
    gsvox::GridDev gd;
    int64_t n_max;
    int32_t max_channels;
    int64_t key_capacity;
    int64_t n;                 // Gaussians of the latest preprocess, -1 before the first
    // device pointers, all inside the caller's workspace
    gsvox::DevStatus* status;
    gsvox::GsRec* rec;
    gsvox::GsAux* aux;
    uint32_t* bin_count;       // [nbins+1]  counts, then write cursors; nbins = nbricks * kNumClasses
    uint32_t* bin_start;       // [nbins+1]  exclusive scan of counts
    uint32_t* scan_partial;    // [scan blocks]
    uint32_t* keys;            // [key_capacity] Gaussian id per key, grouped by brick
    uint2* split_list;         // [split_cap] (brick, segment >= 1) items of hot bricks
    int split_cap;
    float* acc;                // [n_max * acc_stride(max_channels)] backward accumulators
    int nbins;
    // timing
    int timing;
    double ms[GSVOX_K_COUNT_KINDS];
    int64_t launches[GSVOX_K_COUNT_KINDS];
    struct Pending { cudaEvent_t a, b; int kind; };
    Pending* pending;
    int n_pending, cap_pending;
    // gsvox_step_host: copy streams (H2D of the upstream gradient, D2H of the volume) and their events, created lazily
    cudaStream_t side[2];
    cudaEvent_t side_ev[4 + 8];    // [4..]: arrival of the upstream-gradient parts (gsvox_step_host, C = 1)
    int side_ready;
    int deterministic;         // gsvox_plan_set_deterministic: keys of every bin sorted by Gaussian id, a3 without atomics
};

namespace gsvox {

// RAII bracket around one kernel launch: counts it and, when timing is on, records events.
struct LaunchScope {
    gsvox_plan* p; int kind; cudaStream_t st; cudaEvent_t a, b; bool timed;
    LaunchScope(gsvox_plan* plan, int kind_, cudaStream_t s);
    ~LaunchScope();
};

int cuda_fail(cudaError_t e, const char* what);          // records text, returns GSVOX_ECUDA
#define GSVOX_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) \
        return gsvox::cuda_fail(e__, #call); } while (0)

// stage entry points implemented in the other .cu files
int launch_preprocess(gsvox_plan* p, const float* pos, const float* scale, const float* quat,
                      int64_t n, cudaStream_t st);
int launch_binning(gsvox_plan* p, int64_t n, cudaStream_t st);
int launch_sort_bins(gsvox_plan* p, cudaStream_t st);
int launch_exclusive_scan(uint32_t* cnt, int nbins, uint32_t* partial, uint32_t* start,
                          unsigned long long* keys_needed, unsigned int* overflow,
                          unsigned long long key_capacity, cudaStream_t st);
int launch_forward(gsvox_plan* p, const float* weight, int channels, float* out, cudaStream_t st);
int launch_backward(gsvox_plan* p, const float* weight, int channels, const float* grad_out,
                    float* gw, float* gp, float* gs, float* gq, cudaStream_t st);
int launch_backward_accumulate(gsvox_plan* p, const float* weight, int channels, const float* grad_out,
                               cudaStream_t st);
void backward_part_layers(const gsvox_plan* p, int part, int nparts, int* z0, int* z1);
int launch_backward_part(gsvox_plan* p, const float* weight, const float* grad_out, int part, int nparts, cudaStream_t st);
int launch_epilogue(gsvox_plan* p, int channels, float* gw, float* gp, float* gs, float* gq, cudaStream_t st);

}  // namespace gsvox
