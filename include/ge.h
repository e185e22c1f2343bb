/*
 * ge.h -- C ABI of libge: the time-marching loop of the group-explicit (GE)
 * finite-difference scheme of arXiv 1310.3422 for U_t = laplace(U), on one
 * NVIDIA B200 (sm_100a).  Every step of the path runs in libge's own CUDA
 * kernels; there is no CPU fallback.
 *
 * The method (citations are PAPER.md lines; DESIGN.md lists the readings):
 *   - grid: N interior nodes 1..N per axis, nodes 0 and N+1 Dirichlet and
 *     constant in time, h = 1/(N+1), r = tau/h^2
 *   - one LEVEL advances every node by tau.  phase = level mod 2.
 *   - 1-D, group_k = 1 ("two-point groups"): the nodes are split into pairs
 *     (i,i+1), left members at i = 1+phase (mod 2); each pair's 2x2 implicit
 *     block is solved in closed form from the four previous-level values
 *     u_{i-1}..u_{i+2} -- Eqs (3),(4), with prefactor 1/(1+2r);
 *     a pair with a boundary member updates its interior member by Saul'yev's
 *     Eq (1)/(2) with the boundary value as new-level neighbour
 *     (PAPER.md:70-78, :142, :148).  The pattern alternates between levels
 *     (PAPER.md:92, :140-150).
 *   - 1-D, group_k = k >= 2 (the paper's general scheme): node classes
 *     c = (i - phase*k) mod 2k: c = 2k-1 / 0 are the left / right member of a pair (Eqs (3),(4)),
 *     c = 1..k-1 follow by Saul'yev's Eq (1) in ascending order, c = k..2k-2 by Eq (2) in
 *     descending order; sweeps that reach a boundary read it.
 *   - 3-D (reading R-3D, same construction as 2-D): 2x2x2 eight-point groups anchored at
 *     (1+phase) mod 2 in every axis, 8x8 block solved in closed form (Walsh modes of the cube).
 *   - 2-D (reading R-2D; the paper only claims the extension,
 *     PAPER.md:134, :228): 2x2 four-point groups anchored at (1+phase, 1+phase)
 *     (mod 2) -- diagonal shift --, in-group links implicit, out-of-group links
 *     explicit, 4x4 block solved in closed form; groups cut by an edge keep
 *     their interior members.
 *
 * Conventions
 *   - All functions return GE_OK (0) or a negative ge_status.  None throws.
 *     None synchronises the stream except ge_run_host (see there).
 *   - "device pointer": memory of the current CUDA device, owned by the
 *     caller, holding INTERIOR nodes only, contiguous, row-major:
 *     1-D [batch][nx], 2-D [ny][nx] (x fastest).  16-byte alignment of the
 *     base pointer selects the vectorised kernels; any alignment is accepted.
 *   - ge_stream_t is a cudaStream_t (CUstream); 0 = the legacy default stream.
 *   - A plan is used from one host thread and one stream at a time.
 *   - Determinism: same inputs and plan settings give bit-identical output.
 */
#ifndef GE_H_
#define GE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ge_plan ge_plan;                 /* opaque, owned by the library */
typedef struct CUstream_st *ge_stream_t;        /* == cudaStream_t              */

typedef enum { GE_F32 = 0, GE_F64 = 1 } ge_dtype;

typedef enum {
    GE_KERNEL_AUTO = 0,       /* library picks per shape; 2-D grids below 24 MB of
                                 state: PER_STEP (a blocked launch has a latency floor a small grid does not repay) */
    GE_KERNEL_PER_STEP = 1,   /* A: one launch per level, one HBM round trip per level              */
    GE_KERNEL_TEMPORAL = 2,   /* B: tb levels per launch in registers/SMEM, halo-redundant tiles    */
    GE_KERNEL_PERSISTENT = 3  /* C: state stays in registers for the whole run, one launch (1-D): a rod
                                 per CTA (batched rods), or one rod spread over the whole chip by a
                                 cooperative launch whose tiles meet every tb levels; shapes that do not
                                 fit on the chip fall back to B (GE_INFO_KERNEL tells)                  */
} ge_kernel;

typedef enum {
    GE_OK = 0,
    GE_EINVAL = -1,           /* bad argument; nothing was enqueued                   */
    GE_ENOMEM = -2,           /* host or device allocation failed                     */
    GE_ECUDA = -3,            /* a CUDA call failed; ge_strerror appends its message  */
    GE_EUNSUPPORTED = -4      /* valid request the GPU path does not implement (group_k > 2048) */
} ge_status;

typedef struct {
    int32_t   dim;        /* 1, 2 or 3 (3: 2x2x2 groups, strategy A only)       */
    int64_t   nx, ny;     /* interior nodes per axis, >= 1 (ny must be 1 when dim == 1)                */
    int64_t   batch;      /* independent 1-D rods, >= 1 (must be 1 when dim == 2)                      */
    int32_t   dtype;      /* ge_dtype: arithmetic and storage type of u                                */
    int32_t   group_k;    /* 1 = two-point groups (2x2 groups in 2-D); 2..2048 = PAPER.md:82 sub-domain
                             length k (1-D only; the paper's runs use 16): confluence pairs every 2k nodes
                             joined by Saul'yev sweeps; strategy A (one launch per level), or C when a
                             rod fits in one CTA's shared memory (AUTO / PERSISTENT)                  */
    const double *r;      /* HOST array, `batch` entries (dim 2: 1 entry), finite, > 0; copied         */
    const double *bc_lo;  /* HOST array: 1-D `batch` entries, u at node 0;   2-D {x_lo, y_lo}; 3-D {x_lo, y_lo, z_lo} */
    const double *bc_hi;  /* HOST array: 1-D `batch` entries, u at node N+1; 2-D {x_hi, y_hi}; 3-D {x_hi, y_hi, z_hi} */
    int32_t   kernel;     /* ge_kernel                                                                 */
    int32_t   tb;         /* levels per launch for TEMPORAL (0 = auto; any value >= 1, both starting
                             phases are handled in-kernel); levels between two meetings of the tiles for
                             PERSISTENT on one long rod (0 = the largest the halo allows)              */
    int64_t   nz;         /* interior nodes along z (dim == 3; must be 0 or 1 otherwise); layout [nz][ny][nx] */
} ge_desc;

/* Create a plan: validates desc, uploads per-rod coefficients (r, r/(1+2r), r/(1+r), ... computed in
 * fp64 on the host and rounded once to dtype) and allocates one scratch level of the state's size on the
 * current device.  `stream` orders the uploads.  The level counter starts at 0 (phase 0 first,
 * PAPER.md:92, :142).  *out is set only on GE_OK.  desc and its arrays may be freed on return. */
int ge_plan_create(ge_plan **out, const ge_desc *desc, ge_stream_t stream);

/* One level: u_out = level(u_in) with phase = level & 1, then level += 1.
 * u_in, u_out: device pointers, batch*nx (1-D) or ny*nx (2-D) elements of dtype, u_in != u_out, no
 * overlap.  Always one launch of the per-level kernel (strategy A) whatever desc.kernel says.
 * GE_EINVAL if the plan's dim does not match or a pointer is null/misaligned for dtype. */
int ge_step_1d(ge_plan *p, const void *u_in, void *u_out, ge_stream_t stream);
int ge_step_2d(ge_plan *p, const void *u_in, void *u_out, ge_stream_t stream);
int ge_step_3d(ge_plan *p, const void *u_in, void *u_out, ge_stream_t stream);

/* One level of a single rod (batch == 1, group_k == 1) with NON-CONSTANT problem data (SURVEY.md 8(f)
 * NEXT-3, reading R-N3; the paper's model problem has neither):
 * u_t = u_xx + f(x,t) with boundary values that move in time.
 *   tau_f: device pointer, nx elements of dtype, tau_f[i] = tau * f(x_{i+1}, t*) (the time point t*
 *          is the caller's choice, e.g. the middle of the level), or NULL for no source;
 *   bc4:   HOST array {lo_old, lo_new, hi_old, hi_new}: the values of nodes 0 and N+1 at the old and
 *          at the new level (the plan's constant boundary values are not used).
 * Otherwise as ge_step_1d (phase = level & 1, level += 1, one launch).  GE_EINVAL for batch > 1 or
 * dim == 2, GE_EUNSUPPORTED for group_k >= 2. */
int ge_step_1d_src(ge_plan *p, const void *u_in, void *u_out, const void *tau_f, const double *bc4,
                   ge_stream_t stream);

/* One level of a single rod (batch == 1, group_k == 1) with VARIABLE DIFFUSIVITY (DESIGN.md
 * reading R-VAR; the paper's coefficient is constant): u_t = (a(x) u_x)_x in flux form.
 *   rl: device pointer, nx + 1 elements of dtype: rl[j] = tau * a(x_{j+1/2}) / h^2 > 0 for the link between nodes j
 *       and j+1, j = 0 .. N (the plan's own r is not used; the boundary values are the plan's).
 * Otherwise as ge_step_1d (batch == 1).  ge_run_var: `steps` such levels in place, temporally blocked (20 levels per HBM
 * round trip: a tile's state, link numbers and pair factors in registers, ge_temporal_src.cuh -- rows of whole
 * 16-byte vectors holding a tile --, else the window and its link numbers in shared memory, 16 levels, ge_window.cuh;
 * GE_TUNE_SRC_FORM), batched rods included: rl is then [batch][nx + 1].  GE_EINVAL for dim != 1 or a null / misaligned pointer (ge_step_1d_var: also batch > 1),
 * GE_EUNSUPPORTED for group_k >= 2. */
int ge_step_1d_var(ge_plan *p, const void *u_in, void *u_out, const void *rl, ge_stream_t stream);
int ge_run_var(ge_plan *p, void *u, int64_t steps, const void *rl, ge_stream_t stream);

/* `steps` >= 0 levels with a source term and moving boundary values in place (group_k == 1; result in u, level += steps):
 *   tau_f:          device pointer or NULL.  f_level_stride == 0: ONE STATIONARY source, [batch][nx] elements, used at
 *                   every level -- the run is temporally blocked (20 levels per HBM round trip: a tile's state and
 *                   source in registers, ge_temporal_src.cuh -- rows of whole 16-byte vectors holding a tile --, else
 *                   the window and its source in shared memory, 16 levels, ge_window.cuh; GE_TUNE_SRC_FORM), batched rods
 *                   included (per-rod r);
 *                   f_level_stride >= nx: level n of the run reads tau_f + n * f_level_stride (`steps` rows) -- one
 *                   launch of ge_step_1d_src per level, batch must be 1;
 *   bc_lo_t, bc_hi_t: HOST arrays, [batch][steps + 1] entries: the values of nodes 0 and N+1 of every rod at the run's
 *                   levels 0 .. steps (entry n is the old-level value of step n and the new-level value of step n-1).
 * GE_EINVAL for dim != 1, a non-finite boundary value, 0 < f_level_stride < nx or f_level_stride > 0 with batch > 1;
 * GE_EUNSUPPORTED for group_k >= 2.  Nothing is enqueued on an argument error.  Synchronises `stream` once (the
 * boundary values are staged through a host buffer of the call). */
int ge_run_src(ge_plan *p, void *u, int64_t steps, const void *tau_f, int64_t f_level_stride,
               const double *bc_lo_t, const double *bc_hi_t, ge_stream_t stream);

/* `steps` >= 0 levels in place: on completion of the enqueued work u holds level (level0+steps) and
 * the plan's level counter has advanced by `steps`.  The plan's scratch level is used for
 * ping-ponging; the strategy is the plan's (AUTO/PER_STEP/TEMPORAL/PERSISTENT).  steps == 0 is a no-op. */
int ge_run(ge_plan *p, void *u, int64_t steps, ge_stream_t stream);

/* End-to-end variant with HOST buffers: copies u_host (batch*nx or ny*nx elements, ideally pinned)
 * to a plan-owned device buffer, runs `steps` levels, copies the result back into u_host and
 * synchronises `stream` before returning.  One long rod (dim 1, batch 1, nx >= 2^23) is cut into chunks
 * of 2^22 nodes that carry 2*steps+8 extra nodes per side -- more than the dependency cone of `steps`
 * levels -- and are marched independently through a three-slot pipeline (upload, compute and download of
 * neighbouring chunks overlap; u_host should be pinned for that); the result is bit-identical.  Batched rods
 * (batch >= 64, >= 8 MiB) travel through the same pipeline in eight groups of rods. */
int ge_run_host(ge_plan *p, void *u_host, int64_t steps, ge_stream_t stream);

/* Level counter (checkpoint/resume: state = (u, level)). */
int ge_plan_get_level(const ge_plan *p, int64_t *level);
int ge_plan_set_level(ge_plan *p, int64_t level);          /* level >= 0 */

/* Introspection for the benchmark harness.  `what`: */
enum {
    GE_INFO_KERNEL = 0,        /* ge_kernel actually selected for ge_run                          */
    GE_INFO_TB = 1,            /* levels per launch of the temporal kernel (0 if not used)        */
    GE_INFO_LAUNCHES = 2,      /* kernels launched through this plan so far                       */
    GE_INFO_TILE_VALID = 3,    /* valid outputs per tile of the temporal kernel (per axis)        */
    GE_INFO_TILE_LOADED = 4,   /* elements loaded per tile of the temporal kernel (per axis)      */
    GE_INFO_RESIDENT_PATH = 5, /* strategy C: 0 not in use, 1 rod per CTA, 2 one rod on the whole chip,
                                  3 group_k >= 2: rod per CTA, resident in shared memory               */
    GE_INFO_RESIDENT_C = 6,    /* strategy C: values per lane                                     */
    GE_INFO_RESIDENT_WARPS = 7,/* path 1: warps per rod; path 2: tiles (warps) in the launch      */
    GE_INFO_RESIDENT_CAPACITY = 8, /* path 2: co-resident tiles the device offers                 */
    GE_INFO_RESIDENT_TB = 9,   /* path 2: levels between two meetings                             */
    GE_INFO_MEETINGS = 10,     /* path 2: meetings (halo exchanges) performed so far              */
    GE_INFO_TEMPORAL_C = 12,   /* values per lane of the 1-D temporal kernel in use (18 / 36: TMA-staged)   */
    GE_INFO_SYNC_FAULT = 11    /* path 2: 1 if a tile ever gave up waiting for a neighbour (the result
                                  is then invalid); SYNCHRONISES the last stream used              */
};
int ge_plan_info(const ge_plan *p, int32_t what, int64_t *value);

/* Tuning knobs of the temporally blocked kernel (benchmark sweeps; defaults are picked at create).
 * GE_EINVAL for a value the kernels are not instantiated for; nothing is enqueued. */
enum {
    GE_TUNE_TEMPORAL_C = 0,    /* values per lane of the 1-D temporal kernel: 8, 16, 32 (f64) / 16, 32, 64 (f32):
                                  warp-per-tile kernel; 18, 22, 26 (f64) / 36, 44, 52 (f32): TMA-staged persistent kernel, 22 / 52 the
                                  default for rods of >= 2 tiles, 8 / 16 for shorter rods (needs nx >= 32 * value)          */
    GE_TUNE_TB = 1,            /* levels per launch, or between meetings on path 2 (1-D: >= 1, clamped to the largest the tile allows;
                                  2-D: one of the compiled-in block lengths 4, 6, 8; 6 needs the strip kernel)                            */
    GE_TUNE_SEG_PAIRS = 2,     /* 2-D temporal kernel: output row pairs per warp segment (default 67 f32, 56 f64; fewer, down to
                                  16, on grids that would not give every SM its 16 warps)                              */
    GE_TUNE_RESIDENT_C = 3,    /* strategy C: values per lane (f64: 2..64, f32: 4..128, powers of two; one
                                  long rod: 16, 32, 64 (f64) / 32, 64, 128 (f32)); may synchronise and reallocate      */
    GE_TUNE_HALO_LANES = 4,    /* path 2: halo lanes per side, 1..8, default 2 (tb <= lanes * C); may synchronise */
    GE_TUNE_STRIP_COOP = 6,    /* 2-D strip kernel: warps of a CTA that share ONE strip and exchange their edge columns
                                  every level through shared memory and named barriers instead of each recomputing
                                  tb stale columns per side (0 = a warp per strip; 4, 8; needs tb = 6 and
                                  nx >= value * 32 * columns per lane)                                              */
    GE_TUNE_FORM_3D = 7,       /* 3-D per-level kernels: 1 (default) = streaming kernel for the full groups + shell kernel
                                  for the groups cut by a face (one or two launches per level) where rows are a multiple
                                  of 16 bytes and the buffers aligned, a thread per group elsewhere; 0 = a thread per
                                  group always; 2 = the streaming kernel always (its scalar form on other rows)           */
    GE_TUNE_SRC_FORM = 9,      /* ge_run_src with a stationary source, ge_run_var: 1 = the state and tau*f / the links of a tile in registers (default;
                                  rows of whole aligned vectors holding at least one tile of 256 / 512 nodes), 0 = windows in
                                  shared memory (any row)                                                                  */
    GE_TUNE_K_FORM = 8,        /* group_k >= 2, TEMPORAL: 1 = units of 2k nodes held in registers for tb levels + the two ends of the
                                  rod recomputed by the shared-memory kernel (default where compiled: k = 2, 4, 8, 16, fp32 also 32),
                                  0 = windows in shared memory throughout                                                  */
    GE_TUNE_SYNC_MODE = 5      /* path 2, how the tiles meet: 0 = neighbour flags (data, release fence, flag per
                                  tile, acquire), 1 = grid-wide barrier (cooperative groups), 2 = neighbour
                                  flag-in-data lines (no fence, no separate flag), 3 = the same lines published
                                  every tb/2 levels and consumed every other time, the CTAs that share an SM
                                  taking opposite turns (needs tb >= 8); 4, 5, 6, 7 = thread-block CLUSTERS of 2, 4, 8,
                                  16 CTAs: shared memory (the CTA's own or, through distributed shared memory, the
                                  adjacent CTA's) and the cluster's hardware barrier inside a cluster, mode 2's lines
                                  between clusters; GE_EINVAL when the rod cannot stay resident with clusters of that
                                  size; default 1, the fastest measured                                              */
};
int ge_plan_tune(ge_plan *p, int32_t what, int64_t value);

/* Measurement helper, not part of the path ("64 fp64 lanes -- assumption, measure with an FMA
 * microbenchmark"): enqueues ONE launch of a kernel in which each of 2048 threads per SM runs 8 independent
 * chains of `iters` dependent fused multiply-adds of `dtype` (ge_dtype), and stores in *flops the
 * floating-point operations of that launch (an FMA counts 2).  The caller times the launch with events on
 * `stream`; flops / seconds is the sustained FFMA / DFMA rate of the chip at the clock it holds.
 * sink: device pointer to at least 8 writable bytes (never written in practice).  GE_EINVAL for a bad
 * dtype, iters < 1 or a null pointer. */
int ge_fma_probe(int32_t dtype, int64_t iters, void *sink, double *flops, ge_stream_t stream);
/* The same with a choice of operand pattern: variant 0 = ge_fma_probe (x <- x*a + b, a and b shared by all chains: the
 * pipe's own rate), 1 = three DISTINCT registers per FMA (x <- x*y_c + z_c, y and z per chain), which is what the
 * arithmetic of the kernels looks like to the register file.  GE_EINVAL for any other variant. */
int ge_fma_probe_ex(int32_t dtype, int32_t variant, int64_t iters, void *sink, double *flops, ge_stream_t stream);

/* ---- an entry point that allocates NOTHING (for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it; a ge_plan allocates its coefficient block and the second
 * copy of the state) ----
 * ge_run_1d_static: `steps` levels of the 1-D scheme with two-point groups (strategy A,
 * ge1d_level_kernel, the arithmetic of ge_run on a plan with kernel = per_step, bit for bit), one rod, from level
 * `level0` (phase = level & 1), Dirichlet values bc_lo / bc_hi, r = tau/h^2.
 *   u_in, u_out: DEVICE pointers to nx elements of `dtype` (ge_dtype), aligned to the element size, owned by the
 *     caller, not overlapping; u_in is only read.  steps = 0 copies u_in to u_out.
 *   The second copy of the state and the coefficient block live in a file-scope device array of
 *   GE_STATIC_MAX_BYTES + 256 bytes that EVERY GPU which loads the library holds until the process exits.
 *   nx * sizeof(element) > GE_STATIC_MAX_BYTES (nx > 524288 in f64, 1048576 in f32) is rejected with GE_EINVAL and
 *   nothing is enqueued; ge_static_error gives the text.
 *   All calls share that array and find the previous call's contents in it (nothing in it needs to start at zero:
 *   every call rewrites what it reads).  Calls that OVERLAP on the GPU -- two streams, two host threads -- race;
 *   order them on one stream or with events.
 *   No cudaMalloc / cudaFree / allocating routine is called; the only set-up is one cudaGetSymbolAddress per
 *   device, at the first call on that device (ge_static_limit does it too: call it ahead of a capture).
 *   Enqueues 1 + steps launches on `stream` and returns without synchronising.
 * ge_static_limit: *max_nodes = the largest nx ge_run_1d_static takes for `dtype` (and the per-device set-up).
 * ge_static_error: copies the calling thread's last ge_run_1d_static / ge_static_limit message ("ok" after a
 *   success) into buf[cap], NUL-terminated; GE_EINVAL for a null buf or cap < 1. */
#define GE_STATIC_MAX_BYTES (4 * 1024 * 1024)
int ge_run_1d_static(int32_t dtype, const void *u_in, void *u_out, int64_t nx, int64_t steps, int64_t level0,
                     double r, double bc_lo, double bc_hi, ge_stream_t stream);
int ge_static_limit(int32_t dtype, int64_t *max_nodes);
int ge_static_error(char *buf, int64_t cap);

/* Frees the plan's device buffers (stream-ordered on the stream last used) and the plan. */
int ge_plan_destroy(ge_plan *p);

/* Static description of a status; after GE_ECUDA it includes the last CUDA error string seen by
 * the calling thread. */
const char *ge_strerror(int status);

/* Library version: major*10000 + minor*100 + patch. */
int ge_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GE_H_ */
