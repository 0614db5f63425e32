/*
 * gsvox.h — C ABI of the B200-native differentiable 3D Gaussian voxelizer.
 *
 * The operation (PAPER.md = /root/reference/PAPER.md):
 *   Eq. 4   G_i(x) = w_i exp(-1/2 (x-p_i)^T Sigma_i^-1 (x-p_i))
 *   Eq. 5   out(x) = sum_i G_i(x)                     ("voxelization")
 *   PAPER.md:104          differentiable wrt every Gaussian parameter
 *   PAPER.md:106-108      signed, multi-channel values (motion-basis components)
 *   PAPER.md:128-130,136  arbitrary sub-grids and resolutions (origin/spacing/dims)
 * with Sigma_i = R(q_i) diag(s_i)^2 R(q_i)^T and each Gaussian cut off at the axis-aligned
 * bounding box of its 3-sigma ellipsoid (BASELINE.json north_star; DESIGN.md readings
 * A1-A16).  Backward treats that box as frozen.
 *
 * Conventions
 *   - Every `const float*` / `float*` below is a DEVICE pointer unless the name ends in
 *     `_host`.  The caller owns all buffers; the library never allocates or frees device
 *     memory.  All device work is enqueued on `stream` (a cudaStream_t passed as void*);
 *     gsvox_preprocess / gsvox_forward / gsvox_backward never synchronise with the host.
 *   - Layouts: pos [n,3], scale [n,3], quat [n,4] = (w,x,y,z) (need not be normalised),
 *     weight [n,C], volumes [C,nz,ny,nx] with x fastest, all fp32, densely packed.
 *   - Voxel (i,j,k) has its CENTRE at origin + (i*hx, j*hy, k*hz).
 *   - A Gaussian with a non-finite parameter, a scale <= 0 or a zero quaternion is
 *     skipped: it contributes nothing and all its gradients are 0.
 *   - Return value: GSVOX_OK (0) or a negative error code; gsvox_error_string() names it.
 *     Conditions only the device can see (key capacity exceeded) set a flag in the plan:
 *     forward/backward then write zeros and gsvox_plan_status() reports the overflow.
 *   - A plan is bound to one workspace and one grid.  gsvox_preprocess() may be called
 *     any number of times on it (every training step); forward/backward use the geometry
 *     of the latest preprocess.  Distinct plans may be used from distinct threads/streams.
 */
#ifndef GSVOX_H
#define GSVOX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GSVOX_OK            0
#define GSVOX_EINVAL       -1   /* null pointer, n < 0, dims < 1, spacing <= 0, C out of range */
#define GSVOX_EWORKSPACE   -2   /* workspace too small or misaligned                          */
#define GSVOX_ECUDA        -3   /* a CUDA runtime call or launch failed                       */
#define GSVOX_ENOTREADY    -4   /* forward/backward before preprocess                         */
#define GSVOX_ELIMIT       -5   /* size beyond the library limits below                       */

#define GSVOX_MAX_CHANNELS  96          /* 1 <= C <= 96 (3 axes x 32 projections) */
#define GSVOX_MAX_DIM       32760       /* per-axis voxel count                               */
#define GSVOX_MAX_LEVELS    4           /* MBC levels of the two-stage combine (the paper uses 3) */
#define GSVOX_BRICK         8           /* bricks are 8x8x8 voxels                            */
#define GSVOX_SIGMA_CUTOFF  3.0         /* fixed (north_star)                                 */

typedef struct {
    float   origin[3];   /* world position of the centre of voxel (0,0,0), order x,y,z      */
    float   spacing[3];  /* world units per voxel along x,y,z, > 0                           */
    int32_t dims[3];     /* nx, ny, nz                                                        */
} gsvox_grid;

typedef struct gsvox_plan gsvox_plan;   /* opaque host object; device state lives in the workspace */

/* Size of the device workspace for up to n_max Gaussians, channels C <= max_channels and at most
 * key_capacity (brick, Gaussian) keys.  A key is one Gaussian touching one 8^3 brick; if a
 * preprocess needs more than key_capacity keys the plan overflows (see gsvox_plan_status).   */
int gsvox_workspace_bytes(int64_t n_max, int32_t max_channels, const gsvox_grid* grid,
                          int64_t key_capacity, size_t* bytes);

/* Create a plan over caller-owned device memory `workspace` (256-byte aligned, at least
 * gsvox_workspace_bytes() long).  No device work is enqueued.                                 */
int gsvox_plan_create(int64_t n_max, int32_t max_channels, const gsvox_grid* grid,
                      int64_t key_capacity, void* workspace, size_t workspace_bytes,
                      gsvox_plan** plan);
void gsvox_plan_destroy(gsvox_plan* plan);

/* Steps a1+a2: per-Gaussian inverse covariance and voxel box (Eq. 4's Sigma^-1,
 * reading A5 for the box), then brick binning: per-brick lists of the Gaussians whose box
 * meets the brick.  n <= n_max.                                                              */
int gsvox_preprocess(gsvox_plan* plan, const float* pos, const float* scale, const float* quat,
                     int64_t n, void* stream);

/* Step a3: out[c,k,j,i] = sum_i w_ic exp(-1/2 d^T Sigma_i^-1 d) over the Gaussians whose box
 * holds voxel (i,j,k) (Eq. 5).  `out` is OVERWRITTEN, zeros where no Gaussian reaches.        */
int gsvox_forward(gsvox_plan* plan, const float* weight, int32_t channels, float* out,
                  void* stream);

/* Steps a4+a5: given grad_out = dL/dout, write dL/dweight [n,C], dL/dpos [n,3],
 * dL/dscale [n,3], dL/dquat [n,4] (wrt the unnormalised quaternion).  All four OVERWRITTEN.
 * fp32 atomics make the last bits run-to-run dependent.                                       */
int gsvox_backward(gsvox_plan* plan, const float* weight, int32_t channels,
                   const float* grad_out, float* grad_weight, float* grad_pos,
                   float* grad_scale, float* grad_quat, void* stream);

/* Device-side outcome of the latest preprocess.  SYNCHRONISES `stream`.
 *   keys_needed        number of (brick, Gaussian) keys the input produces
 *   overflow           1 if keys_needed > key_capacity (forward/backward wrote zeros)
 *   skipped_gaussians  degenerate inputs that were skipped
 *   pairs              P_def: (Gaussian, voxel) pairs inside the cutoff = sum of box volumes
 *   culled_keys        (brick, Gaussian) keys of the boxes that were NOT emitted because a conservative
 *                      lower bound of the exponent over the brick shows every term of the key below
 *                      w e^-32 (reading A15; thin rotated Gaussians); keys_needed excludes them
 *   pairs_exec         P_exec: pairs of the emitted keys (what forward/backward evaluate), this slab */
typedef struct {
    int64_t keys_needed;
    int64_t pairs;
    int32_t skipped_gaussians;
    int32_t overflow;
    int64_t culled_keys;
    int64_t pairs_exec;
} gsvox_status;
int gsvox_plan_status(gsvox_plan* plan, gsvox_status* status, void* stream);

/* Deterministic forward (SURVEY.md section 7 hard part 3).  By default the keys of a (brick, class) bin stand in
 * the order the binning's atomics produced, so two preprocess calls on the same inputs may sum a voxel's terms in
 * different orders (results agree to ~1e-7 relative, not bit for bit).  With `enabled` != 0, gsvox_preprocess
 * additionally sorts every bin by Gaussian id (two more launches) and gsvox_forward walks each brick's whole key
 * list in one CTA without atomics: the forward output is then bitwise identical from run to run and from plan to
 * plan, at the price of the sort (0.22 ms at config 4, 2.9 ms at config 5) and of no hot-brick splitting in a3 (config 5 forward 1.36 -> 2.48 ms).  The backward keeps
 * its fp32 atomics (gradients repeatable to ~1e-6 relative, north_star allows it).  Takes effect at the next
 * gsvox_preprocess (until then forward/backward return GSVOX_ENOTREADY).  Bins longer than 51200 keys are left
 * unsorted and counted: gsvox_plan_unsorted_bins (SYNCHRONISES; -1 when the mode is off).                      */
int gsvox_plan_set_deterministic(gsvox_plan* plan, int32_t enabled);
int gsvox_plan_unsorted_bins(gsvox_plan* plan, int64_t* unsorted_bins, void* stream);

/* Debug/parity read-back of the latest preprocess (SYNCHRONISES): integer voxel boxes
 * box_host [n,6] = lo_x,lo_y,lo_z,hi_x,hi_y,hi_z inclusive (0,0,0,-1,-1,-1 when empty or
 * skipped) and the inverse covariance in index units minv_host [n,6] = xx,xy,xz,yy,yz,zz
 * (M_idx = H M_world H, H = diag(spacing)).  Either pointer may be NULL.  HOST pointers.     */
int gsvox_plan_geometry_host(gsvox_plan* plan, int32_t* box_host, float* minv_host, void* stream);

/* Debug/parity read-back of the binning (SYNCHRONISES).  HOST pointers.
 *   brick_start_host [nbricks+1]  CSR offsets into the key array, brick id = (bz*nby+by)*nbx+bx
 *   key_gaussian_host [keys]      Gaussian id of every key, grouped by brick (any order within) */
int gsvox_plan_bins_host(gsvox_plan* plan, int64_t* brick_start_host, int32_t* key_gaussian_host,
                         int64_t key_host_capacity, void* stream);

/* Per-kernel CUDA-event timing.  When enabled every kernel launched by the three calls above
 * is bracketed by events on `stream`; gsvox_plan_timings() SYNCHRONISES and returns the
 * accumulated milliseconds and launch counts since the last reset, indexed by GSVOX_K_*.     */
enum {
    GSVOX_K_PREPROCESS = 0,   /* a1  per-Gaussian record + box                   */
    GSVOX_K_COUNT,            /* a2  keys per bin                                 */
    GSVOX_K_SCAN,             /* a2  exclusive scan over bins                     */
    GSVOX_K_SCATTER,          /* a2  write keys                                   */
    GSVOX_K_FORWARD,          /* a3                                               */
    GSVOX_K_BACKWARD,         /* a4                                               */
    GSVOX_K_EPILOGUE,         /* a5  chain rule to scale/quat/pos                 */
    GSVOX_K_MEMSET,           /* zero-fills issued by the library                 */
    GSVOX_K_DVF,              /* 8(f)-1 coefficient mixing / un-mixing            */
    GSVOX_K_COUNT_KINDS
};
int gsvox_plan_set_timing(gsvox_plan* plan, int32_t enabled);
int gsvox_plan_timings(gsvox_plan* plan, double* ms /*[GSVOX_K_COUNT_KINDS]*/,
                       int64_t* launches /*[GSVOX_K_COUNT_KINDS]*/, int32_t reset, void* stream);

/* End-to-end step on HOST buffers (bench.py's e2e leg): copies pos/scale/quat/weight/grad_out
 * host->device, runs preprocess + forward + backward, copies out and the four gradients
 * device->host, all on `stream`, then SYNCHRONISES.  `staging` is caller-owned device memory of
 * at least gsvox_host_staging_bytes(); host buffers should be pinned.  out_host may be NULL
 * (skip the volume read-back) and grad_out_host may be NULL (forward only).  The upstream gradient
 * is uploaded and the volume downloaded on two copy streams owned by the plan, overlapped with the
 * kernels (both ordered after work already enqueued on `stream`); for C = 1 the gradient travels in four pieces of whole
 * brick layers and a4 runs piece by piece as they arrive.  What the library creates behind the caller's
 * back, all of it HOST-side and owned by the plan: the plan object itself (gsvox_plan_create: heap), and on the first
 * gsvox_step_host two non-blocking CUDA streams and eight events (destroyed by gsvox_plan_destroy); never device
 * memory.  Errors: GSVOX_EINVAL for a plan restricted to a z-slab (gsvox_plan_set_slab: it writes its own brick
 * layers only); on any error after the first copy was enqueued the call drains `stream` and both copy streams
 * before it returns, so no copy still references the caller's host buffers.                            */
int gsvox_host_staging_bytes(int64_t n_max, int32_t max_channels, const gsvox_grid* grid, size_t* bytes);
int gsvox_step_host(gsvox_plan* plan, void* staging, size_t staging_bytes,
                    const float* pos_host, const float* scale_host, const float* quat_host,
                    const float* weight_host, int64_t n, int32_t channels,
                    const float* grad_out_host, float* out_host,
                    float* grad_weight_host, float* grad_pos_host, float* grad_scale_host,
                    float* grad_quat_host, void* stream);

/* ---- Multi-GPU z-slabs ------------------------------------
 * One process per GPU; every rank holds all Gaussian parameters and owns a contiguous range of
 * brick layers along z.  gsvox_plan_set_slab restricts a2/a3/a4 of this plan to brick layers
 * [bz_begin, bz_end) (0 <= bz_begin <= bz_end <= ceil(nz/8); an empty range is allowed); call it
 * before gsvox_preprocess.  Forward then writes only the voxels of its slab (no collective: the
 * slabs are disjoint).  Backward is split so that the caller can sum the per-Gaussian accumulators
 * over ranks (NCCL all-reduce on the buffer gsvox_plan_accumulators returns) between the two halves:
 *     gsvox_backward_accumulate  ->  all-reduce(acc, count floats, sum)  ->  gsvox_backward_finish
 * gsvox_backward = accumulate + finish on one GPU.  status.pairs stays the whole-grid P_def;
 * status.keys_needed counts the slab's keys.                                                    */
int gsvox_plan_set_slab(gsvox_plan* plan, int32_t bz_begin, int32_t bz_end);
int gsvox_backward_accumulate(gsvox_plan* plan, const float* weight, int32_t channels,
                              const float* grad_out, void* stream);
int gsvox_backward_finish(gsvox_plan* plan, int32_t channels, float* grad_weight, float* grad_pos,
                          float* grad_scale, float* grad_quat, void* stream);
/* DEVICE pointer to the [n, round4(9 + C)] fp32 accumulators of the latest preprocess and their
 * number (the all-reduce payload: 24 MB at config 4).  HOST output pointers.                     */
int gsvox_plan_accumulators(gsvox_plan* plan, int32_t channels, float** acc, int64_t* count);

/* ---- motion-basis components -> deformation vector fields, fused ----
 * PAPER.md:58-61 (Eq. 3)  d(x,p) = sum_i w_i(p) e_i(x);  PAPER.md:106: three spatial levels i, each
 * with one MBC volume per Cartesian direction k (nine volumes), each level its own Gaussian set;
 * the motion encoder yields nine coefficients w_{i,k}(p) per projection p.
 *   e_{i,k}(x) = sum_{j in level i} feat[j,k] G_j(x)   (Eq. 5, signed values)
 *   dvf[b,k,x] = sum_i coef[b,i,k] e_{i,k}(x)           for the B projections of a batch.
 * The plan holds the geometry of ALL levels as one Gaussian set (gsvox_preprocess once per step);
 * level[j] in 0..L-1 names the level of Gaussian j (other values: the Gaussian contributes
 * nothing).  The nine MBC volumes are never materialised: the coefficients are folded into
 * per-Gaussian weights mixed[j, 3b+k] = coef[b,level[j],k] feat[j,k] and the set is voxelized once
 * with C = 3B channels (the plan needs max_channels >= 3B).
 *   feat [n,3], level [n] int32, coef [B,L,3], mixed [n,3B] (caller-owned scratch, overwritten),
 *   dvf [B,3,nz,ny,nx] OVERWRITTEN.  All DEVICE pointers.  No host synchronisation.            */
int gsvox_dvf_forward(gsvox_plan* plan, const float* feat, const int32_t* level, const float* coef,
                      int32_t B, int32_t L, float* mixed, float* dvf, void* stream);
/* Backward of the above for grad_dvf = dL/ddvf [B,3,nz,ny,nx]: writes dL/dfeat [n,3],
 * dL/dcoef [B,L,3], dL/dpos [n,3], dL/dscale [n,3], dL/dquat [n,4] (all OVERWRITTEN).
 * grad_mixed [n,3B] is caller-owned scratch (overwritten); mixed is recomputed from coef.       */
int gsvox_dvf_backward(gsvox_plan* plan, const float* feat, const int32_t* level, const float* coef,
                       int32_t B, int32_t L, float* mixed, const float* grad_dvf, float* grad_mixed,
                       float* grad_feat, float* grad_coef, float* grad_pos, float* grad_scale,
                       float* grad_quat, void* stream);

/* Two-stage form of the same map for batches of projections (BASELINE config 3: "each level
 * voxelized separately"): e [L,3,V] are the MBC volumes (gsvox_forward with C = 3 on one plan per
 * level, V = nx*ny*nz), coef [B,L,3]:
 *     dvf[b,k,v] = sum_i coef[b,i,k] e[i,k,v]                                    (Eq. 3)
 * HBM-bound: 4 V (3L + 3B) algorithmic bytes.  The voxelizer is ALU-bound, so for B > 1 this form
 * (exponentials evaluated once per level) is the fast one; gsvox_dvf_forward re-evaluates them per
 * group of 9 channels and is the single-projection path (measured).
 * 1 <= B <= 32, 1 <= L <= GSVOX_MAX_LEVELS.  All DEVICE pointers; outputs OVERWRITTEN.          */
int gsvox_mbc_combine_forward(const float* e, const float* coef, int32_t B, int32_t L, int64_t V,
                              float* dvf, void* stream);
/* Backward: grad_e[i,k,v] = sum_b coef[b,i,k] grad_dvf[b,k,v] (feed it to gsvox_backward of level
 * i) and grad_coef[b,i,k] = sum_v grad_dvf[b,k,v] e[i,k,v], in one pass over grad_dvf and e:
 * 4 V (3B + 6L) algorithmic bytes.                                                              */
int gsvox_mbc_combine_backward(const float* e, const float* coef, const float* grad_dvf, int32_t B,
                               int32_t L, int64_t V, float* grad_e, float* grad_coef, void* stream);

/* ---- the warp (Eq. 2) -------------------------------------
 *     out[b, v] = I_ref(x_v + d[b, :, v]),   b = 0..B-1 projections of a batch
 * iref [nz,ny,nx]; dvf [B,3,nz,ny,nx] with components in the order x,y,z and in WORLD units (the
 * unit of grid->spacing; grid->origin cancels); out [B,nz,ny,nx] OVERWRITTEN.  Trilinear
 * interpolation of the voxel-centre samples, corners outside the grid read 0, a non-finite
 * displacement yields 0 (readings W1-W4).  All DEVICE pointers, no host sync.        */
int gsvox_warp_forward(const float* iref, const float* dvf, const gsvox_grid* grid, int32_t B,
                       float* out, void* stream);
/* Backward for grad_out = dL/dout [B,nz,ny,nx]: grad_iref [nz,ny,nx] (OVERWRITTEN; summed over the
 * batch with fp32 atomics, so run-to-run dependent in the last bits) and grad_dvf [B,3,nz,ny,nx]
 * (OVERWRITTEN), the exact derivative of the piecewise-trilinear interpolant.                   */
int gsvox_warp_backward(const float* iref, const float* dvf, const gsvox_grid* grid, int32_t B,
                        const float* grad_out, float* grad_iref, float* grad_dvf, void* stream);

/* ---- batched cone-beam projector, one distinct volume per gantry angle ----
 * PAPER.md:141 (Eq. 12) P[I(x,p)]; "PMF-STGR requires a distinct DRR for each dynamic
 * CBCT at each gantry angle ... future work could implement GPU-based parallelization to compute DRRs
 * from multiple dynamic CBCTs simultaneously"; Eq. 6: I(r) = int sigma(r(t)) dt; Table I: SAD, SDD,
 * detector size and pixel pitch.  Geometry (reading P1): circular orbit about the axis through `iso`
 * parallel to z; at gantry angle a the source sits at iso + sad (cos a, sin a, 0); flat detector
 * perpendicular to the central ray at distance sdd from the source; u = (-sin a, cos a, 0),
 * v = (0, 0, 1); pixel (iu, iv) centre at det_centre + ((iu - (nu-1)/2) du + off_u) u
 * + ((iv - (nv-1)/2) dv + off_v) v.  Line integral by Joseph's method (reading P2).              */
typedef struct {
    float   sad, sdd;        /* source-to-axis and source-to-detector distance, world units          */
    int32_t nu, nv;          /* detector pixels along u (in the orbit plane) and v (along the axis)   */
    float   du, dv;          /* pixel pitch                                                            */
    float   off_u, off_v;    /* detector offset (half-fan acquisitions)                                */
    float   iso[3];          /* a point of the rotation axis, world units                              */
} gsvox_cone_geometry;
/* scratch: caller-owned DEVICE memory of gsvox_project_scratch_bytes() (a y-fastest copy of the B
 * volumes, so that rays running mostly along x read contiguously).  1 <= B <= 64 per call.          */
int gsvox_project_scratch_bytes(const gsvox_grid* grid, int32_t B, size_t* bytes);
/* drr[b, iv, iu] = line integral of volume b along the ray source(angles_host[b]) -> pixel (iu, iv).
 * vol [B,nz,ny,nx] with vol_stride = nx*ny*nz, or ONE volume shared by all angles with vol_stride =
 * 0 (the conventional case); angles_host [B] radians, a HOST pointer; drr [B,nv,nu] OVERWRITTEN.    */
int gsvox_project_forward(const float* vol, int64_t vol_stride, const gsvox_grid* grid,
                          const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                          void* scratch, float* drr, void* stream);
/* The same forward projection for callers that cannot allocate device memory (code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc): no scratch argument, the y-fastest copy of the volumes lives
 * in a 16 MB array built into the library (every GPU that loads the library holds it until the process exits).
 * Limit: B * nx * ny * nz <= GSVOX_PROJECT_STATIC_MAX_VOXELS (one 200x200x100 volume; four of
 * 128x128x64), else GSVOX_ELIMIT and nothing is enqueued.  Calls no cudaMalloc / cudaFree / allocating routine;
 * the first call on a device looks the array's address up (cudaGetSymbolAddress), so make that call outside a
 * capture.  All calls on one device SHARE the array: calls that overlap on the GPU (different streams, parallel
 * graph branches) race on it; calls ordered on one stream do not.  Everything else as gsvox_project_forward,
 * whose results it reproduces bit for bit.                                                                 */
#define GSVOX_PROJECT_STATIC_MAX_VOXELS 4194304
int gsvox_project_forward_static(const float* vol, int64_t vol_stride, const gsvox_grid* grid,
                                 const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                                 float* drr, void* stream);
/* Exact transpose: grad_vol[b] = P_b^T grad_drr[b], grad_vol [B,nz,ny,nx] OVERWRITTEN (fp32 atomics). */
int gsvox_project_backward(const float* grad_drr, const gsvox_grid* grid, const gsvox_cone_geometry* geom,
                           const float* angles_host, int32_t B, void* scratch, float* grad_vol, void* stream);

/* ---- Gaussian-splat X-ray rasterizer (Eq. 6-9) ---------------
 * drr[b, iv, iu] = sum_i rho^_i exp(-1/2 (x^ - p^_i)^T Sigma^_i^-1 (x^ - p^_i))  for gantry angle b, with
 * Sigma~ = J W Sigma W^T J^T (Eq. 8), Sigma^ = Sigma~[0:2,0:2], rho^ = rho sqrt(2 pi |Sigma~| / |Sigma^|)
 * (Eq. 9).  Scanner = gsvox_cone_geometry (reading R1 = P1); camera frame at the source, rows of W =
 * (u, v, central ray); ray space phi(t) = (t0/t2, t1/t2, |t|) (R2); cutoff = inclusive pixel box of the
 * 3-sigma ellipse (R4); Gaussians at or behind the source plane, or degenerate, are skipped (R5).
 * pos [n,3], scale [n,3], quat [n,4] (w,x,y,z), rho [n]: DEVICE pointers in WORLD units; angles_host
 * [B] radians, HOST pointer, 1 <= B <= 64; drr [B,nv,nu] OVERWRITTEN.  workspace: caller-owned
 * DEVICE memory, 256-byte aligned, gsvox_splat_workspace_bytes() long; key_capacity bounds the number
 * of (16x16 tile, angle, Gaussian) keys: beyond it the call writes zeros and gsvox_splat_status
 * reports overflow and the capacity needed.  No host synchronisation.                            */
int gsvox_splat_workspace_bytes(int64_t n, const gsvox_cone_geometry* geom, int32_t B,
                                int64_t key_capacity, size_t* bytes);
int gsvox_splat_forward(const float* pos, const float* scale, const float* quat, const float* rho,
                        int64_t n, const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                        void* workspace, size_t workspace_bytes, int64_t key_capacity,
                        float* drr, void* stream);
/* Backward for grad_drr = dL/ddrr [B,nv,nu], boxes frozen (R6).  MUST follow gsvox_splat_forward
 * with the same inputs, geometry, angles and workspace (it reuses the 2D records and the tile
 * lists).  grad_rho [n], grad_pos [n,3], grad_scale [n,3], grad_quat [n,4] OVERWRITTEN.  The forward
 * leaves a stamp (magic + digest of n, B, nu, nv, key_capacity) in the workspace; a backward on a
 * workspace without the matching stamp (no forward yet, other sizes) touches none of the lists and
 * writes ZERO gradients — the condition lives on the device, so it is reported by gsvox_splat_status
 * (GSVOX_ENOTREADY), not by this call's return value.                                              */
int gsvox_splat_backward(const float* pos, const float* scale, const float* quat, const float* rho,
                         int64_t n, const gsvox_cone_geometry* geom, const float* angles_host, int32_t B,
                         void* workspace, size_t workspace_bytes, int64_t key_capacity,
                         const float* grad_drr, float* grad_rho, float* grad_pos, float* grad_scale,
                         float* grad_quat, void* stream);
/* Outcome of the latest gsvox_splat_forward on this workspace (SYNCHRONISES): keys needed, pairs
 * inside the cutoff over all angles, overflow flag, Gaussians skipped as degenerate (non-finite
 * parameter, scale <= 0, zero quaternion: counted once, whatever the number of angles).  HOST outputs.
 * GSVOX_ENOTREADY if no forward has completed on this workspace (zero it before the first use).
 * gsvox_splat_drops: per (angle, Gaussian) items that contribute nothing at that angle although the
 * Gaussian is valid (R5) — at or behind the source plane, centre more than 30000 pixels from the
 * detector origin, footprint box empty after clipping to the detector.                            */
int gsvox_splat_drops(const void* workspace, int64_t* behind_source, int64_t* out_of_range, int64_t* empty_box,
                      void* stream);
int gsvox_splat_status(const void* workspace, int64_t* keys_needed, int64_t* pairs, int32_t* overflow,
                       int32_t* skipped, void* stream);

const char* gsvox_error_string(int code);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char* gsvox_last_cuda_error(void);
int gsvox_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GSVOX_H */
