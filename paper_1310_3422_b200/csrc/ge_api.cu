// ge_api.cu -- the C ABI of libge (include/ge.h): plan, validation, strategy
// selection and kernel dispatch.  No torch types, no CPU fallback: every level
// is computed by the CUDA kernels in this directory.
#include "../../include/ge.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>     // header-only NVTX v3: ranges around ge_run / ge_run_host

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "ge_common.cuh"
#include "ge_level.cuh"
#include "ge_temporal_src.cuh"
#include "ge_temporal.cuh"
#include "ge_temporal2d.cuh"
#include "ge_resident.cuh"
#include "ge_stream.cuh"
#include "ge_dispatch.h"
#include "ge_level_k.cuh"
#include "ge_level_src.cuh"
#include "ge_probe.cuh"
#include "ge_tail.cuh"
#include "ge_level_var.cuh"
#include "ge_window.cuh"

// (measured on a 2^27 rod, GLUPS source / variable diffusivity: fp64 C = 16 2326 / 1793, C = 8 2943 / 2455;
// fp32 C = 32 4584 / 2781, C = 16 4794 / 4737, C = 8 4436 / 4359)
#ifndef GE_SRC_C_F64
#define GE_SRC_C_F64 8
#endif
#ifndef GE_SRC_C_F32
#define GE_SRC_C_F32 16          // values per lane of the fp32 register kernels for non-constant data
#endif

namespace {

thread_local char g_errbuf[512];
thread_local cudaError_t g_last_cuda = cudaSuccess;

#define GE_CUDA(expr)                                   \
    do {                                                \
        cudaError_t e__ = (expr);                       \
        if (e__ != cudaSuccess) {                       \
            g_last_cuda = e__;                          \
            return e__ == cudaErrorMemoryAllocation ? GE_ENOMEM : GE_ECUDA; \
        }                                               \
    } while (0)

inline size_t elem_size(int dtype) { return dtype == GE_F64 ? 8 : 4; }

// NVTX range for the lifetime of the object (a no-op unless a profiler has injected itself)
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

}  // namespace

struct ge_plan {
    int32_t dim, dtype, group_k, kernel, tb;
    int32_t tc;               // values per lane of the temporal kernel (18 f64 / 36 f32: the TMA-staged one)
    int32_t stream_ctas;      // persistent grid of the TMA-staged kernel (0: not queried yet)
    int32_t hp;               // 2-D temporal kernel: output row pairs per segment
    int64_t nx, ny, nz, batch;
    int64_t count;            // elements of the state
    int64_t level;
    int64_t launches;
    int device;
    void* coef;               // device: Coef1<T>[batch] or Coef2<T>[1]
    void* scratch;            // device: one level
    void* hostpath;           // device: state buffer for ge_run_host (lazy)
    cudaStream_t last_stream;
    int sm_count;
    // strategy C (ge_resident.cuh)
    int32_t res_path;         // 0 none, 1 rod per CTA, 2 one rod on the whole chip
    int32_t res_c, res_w;     // values per lane, warps per rod (path 1)
    int32_t res_hl;           // halo lanes per side (path 2)
    int32_t res_tb;           // levels between two meetings (path 2)
    int32_t res_sync;         // kSyncFlags / kSyncGrid (path 2)
    int64_t res_tiles;        // tiles (warps) of path 2
    int64_t res_capacity;     // co-resident tiles the device offers for path 2
    void* res_xbuf;           // device: exchange buffer of path 2
    unsigned* res_flags;      // device: one flag per tile, + the fault word at [res_tiles]
    unsigned res_epoch;       // value every flag holds between launches
    int64_t meetings;         // meetings of the persistent kernel so far (info)
    // ge_run_host pipeline (one long rod): per slot a stream, a device buffer and cached sub-plans
    struct HostSlot { cudaStream_t stream; void* buf; size_t cap; cudaEvent_t h2d_done; ge_plan* sub[4]; int64_t sub_len[4]; };
    HostSlot* slots;          // kHostSlots entries (lazy)
    ge_desc host_desc;        // shape of this plan for the sub-plans (r, boundary values below)
    double host_r, host_lo, host_hi;
    int32_t strip_attr_tb;    // strip-kernel instantiation (tb*16 + coop) whose function attributes are set on this device (0: none)
    cudaStream_t aux3d;       // 3-D: side stream of the shell kernel, with its fork / join events (lazy)
    cudaEvent_t ev3d[2];
    int32_t src_form;         // ge_run_src, stationary source: 1 registers (ge_temporal_src.cuh, default), 0 shared-memory windows
    int32_t kform;            // k >= 2 blocked kernel: 1 register-resident units + end windows (default), 0 shared-memory windows
    int32_t form3d;           // 3-D per-level form: 1 streaming + shell kernels (default), 0 a thread per group
    int32_t strip_coop;       // warps that share one strip of the 2-D strip kernel (0: a warp per strip)
    bool levelk_attr;         // function attributes of the k >= 2 kernel are set on this device
    bool rodk_attr;           // ... and of its shared-memory-resident form
    bool temporalk_attr;      // ... and of its temporally blocked form
    bool win_attr;            // ... and of the window kernels (source term / variable diffusivity)
    void* bc_dev;             // device: boundary values level by level of a ge_run_src call (grown on demand)
    size_t bc_cap;
};

namespace {

template <typename T>
int upload_coef(ge_plan* p, const ge_desc* d, cudaStream_t s) {
    if (p->dim == 1) {
        std::vector<ge::Coef1<T>> h((size_t)p->batch);
        for (int64_t b = 0; b < p->batch; ++b) {
            const double r = d->r[b];
            h[b].r = (T)r;
            h[b].g = (T)(r / (1.0 + 2.0 * r));
            h[b].e = (T)(r / (1.0 + r));
            h[b].lo = (T)d->bc_lo[b];
            h[b].hi = (T)d->bc_hi[b];
            h[b].pad[0] = h[b].pad[1] = h[b].pad[2] = (T)0;
        }
        GE_CUDA(cudaMalloc(&p->coef, h.size() * sizeof(ge::Coef1<T>)));
        GE_CUDA(cudaMemcpyAsync(p->coef, h.data(), h.size() * sizeof(ge::Coef1<T>), cudaMemcpyHostToDevice, s));
        GE_CUDA(cudaStreamSynchronize(s));   // h is a stack-owned staging buffer
    } else if (p->dim == 3) {
        ge::Coef3<T> h;
        std::memset(&h, 0, sizeof(h));
        const double r = d->r[0];
        h.r = (T)r;
        h.c1 = (T)(2.0 * r / (1.0 + 2.0 * r) / 8.0);
        h.c2 = (T)(4.0 * r / (1.0 + 4.0 * r) / 8.0);
        h.c3 = (T)(6.0 * r / (1.0 + 6.0 * r) / 8.0);
        h.q1 = (T)(r / (1.0 + r) / 4.0);
        h.q2 = (T)(3.0 * r / (1.0 + 3.0 * r) / 4.0);
        h.q3 = (T)(5.0 * r / (1.0 + 5.0 * r) / 4.0);
        for (int ax = 0; ax < 3; ++ax) { h.lo[ax] = (T)d->bc_lo[ax]; h.hi[ax] = (T)d->bc_hi[ax]; }
        GE_CUDA(cudaMalloc(&p->coef, sizeof(h)));
        GE_CUDA(cudaMemcpyAsync(p->coef, &h, sizeof(h), cudaMemcpyHostToDevice, s));
        GE_CUDA(cudaStreamSynchronize(s));
    } else {
        ge::Coef2<T> h;
        std::memset(&h, 0, sizeof(h));
        const double r = d->r[0];
        h.r = (T)r;
        h.g2 = (T)(r / (1.0 + 2.0 * r));
        h.g4 = (T)(r / (1.0 + 4.0 * r));
        h.h1 = (T)(r / (2.0 * (1.0 + r)));
        h.h3 = (T)(3.0 * r / (2.0 * (1.0 + 3.0 * r)));
        h.xlo = (T)d->bc_lo[0]; h.ylo = (T)d->bc_lo[1];
        h.xhi = (T)d->bc_hi[0]; h.yhi = (T)d->bc_hi[1];
        GE_CUDA(cudaMalloc(&p->coef, sizeof(h)));
        GE_CUDA(cudaMemcpyAsync(p->coef, &h, sizeof(h), cudaMemcpyHostToDevice, s));
        GE_CUDA(cudaStreamSynchronize(s));
    }
    return GE_OK;
}

// ---- strategy A launches ---------------------------------------------------
template <typename T>
int launch_level_1d(ge_plan* p, const void* uin, void* uout, int phase, cudaStream_t s) {
    constexpr int V = ge::VecOf<T>::V;
    constexpr int ITER = 4;
    const bool vec = (p->nx % V == 0) && (((uintptr_t)uin | (uintptr_t)uout) % 16 == 0);
    const int64_t nvec = vec ? p->nx / V : p->nx;
    const int64_t per_block = (int64_t)ge::kLevelThreads * ITER;
    dim3 grid((unsigned)((nvec + per_block - 1) / per_block), (unsigned)(p->batch < 65535 ? p->batch : 65535));
    dim3 block(ge::kLevelThreads);
    auto* c = (const ge::Coef1<T>*)p->coef;
    auto* in = (const T*)uin;
    auto* out = (T*)uout;
    if (vec) {
        if (phase == 0) ge::ge1d_level_kernel<T, V, 0, ITER><<<grid, block, 0, s>>>(in, out, p->nx, p->batch, c);
        else            ge::ge1d_level_kernel<T, V, 1, ITER><<<grid, block, 0, s>>>(in, out, p->nx, p->batch, c);
    } else {
        if (phase == 0) ge::ge1d_level_kernel<T, 1, 0, ITER><<<grid, block, 0, s>>>(in, out, p->nx, p->batch, c);
        else            ge::ge1d_level_kernel<T, 1, 1, ITER><<<grid, block, 0, s>>>(in, out, p->nx, p->batch, c);
    }
    GE_CUDA(cudaGetLastError());
    p->launches += 1;
    return GE_OK;
}

template <typename T>
int launch_level_2d(ge_plan* p, const void* uin, void* uout, int phase, cudaStream_t s) {
    constexpr int NV = ge::VecOf<T>::V;
    constexpr int V = 4;                               // columns per thread: one float4, two double2
    const bool aligned = (((uintptr_t)uin | (uintptr_t)uout) % 16 == 0);
    const int v = aligned && p->nx % V == 0 ? V : (aligned && p->nx % NV == 0 ? NV : 1);
    // rows that are not whole aligned vectors: V columns per thread all the same, element by element
    const int64_t nvec = v == 1 ? (p->nx + V - 1) / V : p->nx / v;
    const int64_t npair = (p->ny + phase) / 2 + 1;      // anchor rows -phase, 2-phase, ... <= ny-1
    dim3 grid((unsigned)((nvec + ge::kLevel2dBx - 1) / ge::kLevel2dBx),
              (unsigned)((npair + ge::kLevel2dBy - 1) / ge::kLevel2dBy));
    dim3 block(ge::kLevel2dBx, ge::kLevel2dBy);
    auto* c = (const ge::Coef2<T>*)p->coef;
    auto* in = (const T*)uin;
    auto* out = (T*)uout;
    if (v == V) {
        if (phase == 0) ge::ge2d_level_kernel<T, V, 0><<<grid, block, 0, s>>>(in, out, p->nx, p->ny, c);
        else            ge::ge2d_level_kernel<T, V, 1><<<grid, block, 0, s>>>(in, out, p->nx, p->ny, c);
    } else if (v == NV) {
        if (phase == 0) ge::ge2d_level_kernel<T, NV, 0><<<grid, block, 0, s>>>(in, out, p->nx, p->ny, c);
        else            ge::ge2d_level_kernel<T, NV, 1><<<grid, block, 0, s>>>(in, out, p->nx, p->ny, c);
    } else {
        if (phase == 0) ge::ge2d_level_kernel<T, V, 0, false><<<grid, block, 0, s>>>(in, out, p->nx, p->ny, c);
        else            ge::ge2d_level_kernel<T, V, 1, false><<<grid, block, 0, s>>>(in, out, p->nx, p->ny, c);
    }
    GE_CUDA(cudaGetLastError());
    p->launches += 1;
    return GE_OK;
}

// ---- strategy A for sub-domain length k >= 2 (ge_level_k.cuh) ----
constexpr size_t kLevelKSmemBudget = 96 * 1024;
constexpr int kMaxGroupK = 2048;          // a unit of 2k+1 values (twice) must fit the shared-memory budget

template <typename T>
int launch_level_k(ge_plan* p, const void* uin, void* uout, int phase, cudaStream_t s) {
    const ge::LevelKGeom g = ge::level_k_geom(p->group_k, phase, p->nx, sizeof(T), kLevelKSmemBudget);
    if (g.upc < 1) return GE_EUNSUPPORTED;
    const size_t smem = ge::level_k_smem(g, sizeof(T));
    if (!p->levelk_attr) {
        GE_CUDA(cudaFuncSetAttribute(ge::ge1d_level_k_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)(kLevelKSmemBudget + 64)));
        p->levelk_attr = true;
    }
    dim3 grid((unsigned)((g.units + g.upc - 1) / g.upc), (unsigned)(p->batch < 65535 ? p->batch : 65535));
    ge::ge1d_level_k_kernel<T><<<grid, ge::kLevelKThreads, smem, s>>>((const T*)uin, (T*)uout, p->nx, p->batch,
                                                                      (const ge::Coef1<T>*)p->coef, g);
    GE_CUDA(cudaGetLastError());
    p->launches += 1;
    return GE_OK;
}

// strategy B for k >= 2: `levels` <= tb levels per launch on tiles of the rod (ge1d_temporal_k_kernel)
#ifndef GE_TK_SMEM_KB
#define GE_TK_SMEM_KB 64
#endif
constexpr size_t kTemporalKSmemBudget = GE_TK_SMEM_KB * 1024;
bool temporal_k_ok(const ge_plan* p, int tb) {
    return p->dim == 1 && p->group_k >= 2 && tb >= 1 &&
           ge::temporal_k_geom(p->group_k, tb, p->nx, elem_size(p->dtype), kTemporalKSmemBudget).valid > 0;
}
// the register-resident form (ge_unit_k.cuh) + the shared-memory kernel on the two ends of the rod
int64_t unit_k_end_len(const ge_plan* p) { return (int64_t)p->tb * (p->group_k + 1) + 4 * p->group_k + 8; }
bool unit_k_ok(const ge_plan* p, const void* u) {
    const int V = p->dtype == GE_F64 ? 2 : 4;
    if (p->dim != 1 || !ge::unit_k_compiled(p->dtype, p->group_k) || !p->kform) return false;
    if (((uintptr_t)u % 16) || ((uintptr_t)p->scratch % 16) || (p->batch > 1 && p->nx % V)) return false;
    if (p->batch > 65535 || p->nx < 4 * unit_k_end_len(p)) return false;
    return ge::unit_k_valid_lanes(p->group_k, p->tb) >= 64 &&
           ge::temporal_k_ends_geom(p->group_k, p->tb, unit_k_end_len(p), elem_size(p->dtype)).valid > 0;
}
template <typename T>
int launch_unit_k(ge_plan* p, const void* uin, void* uout, int levels, cudaStream_t s) {
    const int phase = (int)(p->level & 1);
    cudaError_t e = ge::unit_k_dispatch(p->dtype, p->group_k, uin, uout, p->nx, p->batch, p->coef, p->tb, phase, levels, s);
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    const ge::TemporalKGeom g = ge::temporal_k_ends_geom(p->group_k, p->tb, unit_k_end_len(p), sizeof(T));
    if (!p->temporalk_attr) {
        GE_CUDA(cudaFuncSetAttribute(ge::ge1d_temporal_k_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)(kTemporalKSmemBudget + 1024)));
        GE_CUDA(cudaFuncSetAttribute(ge::ge1d_temporal_k_kernel<T>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        p->temporalk_attr = true;
    }
    dim3 grid(2, (unsigned)(p->batch < 65535 ? p->batch : 65535));
    ge::ge1d_temporal_k_kernel<T><<<grid, g.threads, g.smem, s>>>((const T*)uin, (T*)uout, p->nx, p->batch,
                                                                  (const ge::Coef1<T>*)p->coef, g, phase, levels);
    GE_CUDA(cudaGetLastError());
    p->launches += 2;
    p->level += levels;
    return GE_OK;
}

template <typename T>
int launch_temporal_k(ge_plan* p, const void* uin, void* uout, int levels, cudaStream_t s) {
    if (unit_k_ok(p, uin) && unit_k_ok(p, uout)) return launch_unit_k<T>(p, uin, uout, levels, s);
    const ge::TemporalKGeom g = ge::temporal_k_geom(p->group_k, p->tb, p->nx, sizeof(T), kTemporalKSmemBudget);
    if (g.valid <= 0 || levels < 1 || levels > p->tb) return GE_EINVAL;
    if (!p->temporalk_attr) {
        GE_CUDA(cudaFuncSetAttribute(ge::ge1d_temporal_k_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)(kTemporalKSmemBudget + 1024)));
        GE_CUDA(cudaFuncSetAttribute(ge::ge1d_temporal_k_kernel<T>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        p->temporalk_attr = true;
    }
    dim3 grid((unsigned)g.tiles, (unsigned)(p->batch < 65535 ? p->batch : 65535));
    ge::ge1d_temporal_k_kernel<T><<<grid, g.threads, g.smem, s>>>((const T*)uin, (T*)uout, p->nx, p->batch,
                                                                  (const ge::Coef1<T>*)p->coef, g, (int)(p->level & 1), levels);
    GE_CUDA(cudaGetLastError());
    p->launches += 1;
    p->level += levels;
    return GE_OK;
}

// strategy C for k >= 2: the rod resident in shared memory, one launch for the whole run (res_path 3)
constexpr size_t kRodKSmemMax = 200 * 1024;
bool rod_k_fits(const ge_plan* p) {
    if (p->dim != 1 || p->group_k < 2 || p->nx >= (1 << 24)) return false;
    const ge::RodKGeom g = ge::rod_k_geom(p->group_k, p->nx, elem_size(p->dtype));
    return g.threads > 0 && g.smem <= kRodKSmemMax;
}
template <typename T>
int launch_rod_k_resident(ge_plan* p, void* u, int64_t steps, cudaStream_t s) {
    const ge::RodKGeom g = ge::rod_k_geom(p->group_k, p->nx, sizeof(T));
    if (!p->rodk_attr) {
        GE_CUDA(cudaFuncSetAttribute(ge::ge1d_rod_k_resident_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)kRodKSmemMax));
        p->rodk_attr = true;
    }
    const unsigned grid = (unsigned)(p->batch < (1 << 30) ? p->batch : (1 << 30));
    ge::ge1d_rod_k_resident_kernel<T><<<grid, g.threads, g.smem, s>>>((T*)u, p->nx, p->batch,
                                                                      (const ge::Coef1<T>*)p->coef, p->group_k,
                                                                      (int)(p->level & 1), steps);
    GE_CUDA(cudaGetLastError());
    p->launches += 1;
    p->level += steps;
    return GE_OK;
}

int launch_level(ge_plan* p, const void* uin, void* uout, cudaStream_t s) {
    const int phase = (int)(p->level & 1);
    int rc;
    if (p->dim == 1 && p->group_k >= 2)
        rc = p->dtype == GE_F64 ? launch_level_k<double>(p, uin, uout, phase, s)
                                : launch_level_k<float>(p, uin, uout, phase, s);
    else if (p->dim == 3) {
        // the streaming form (deep groups) + shell, unless the grid is too small to have deep groups worth a launch
        const int form = p->form3d && p->nx >= 8 && p->ny >= 8 && p->nz >= 8 ? p->form3d : 0;
        int n = 0;
        if (form != 0 && !p->aux3d) {        // side stream of the shell kernel (lazy; a failure just keeps everything on s)
            int prio_least = 0, prio_greatest = 0;           // GE_S3D_MODE 2: the side stream carries the streaming kernel, ahead of the shell
            cudaDeviceGetStreamPriorityRange(&prio_least, &prio_greatest);
            if (cudaStreamCreateWithPriority(&p->aux3d, cudaStreamNonBlocking, GE_S3D_MODE == 2 ? prio_greatest : prio_least) != cudaSuccess ||
                cudaEventCreateWithFlags(&p->ev3d[0], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&p->ev3d[1], cudaEventDisableTiming) != cudaSuccess) {
                cudaGetLastError();
                if (p->aux3d) cudaStreamDestroy(p->aux3d);
                p->aux3d = nullptr; p->ev3d[0] = p->ev3d[1] = nullptr;
            }
        }
        const cudaError_t e = ge::level3d_dispatch(p->dtype, form, uin, uout, p->nx, p->ny, p->nz, p->coef, phase, p->sm_count, s, &n,
                                                   p->aux3d, p->ev3d[0], p->ev3d[1]);
        if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
        p->launches += n;
        rc = GE_OK;
    }
    else if (p->dim == 1) rc = p->dtype == GE_F64 ? launch_level_1d<double>(p, uin, uout, phase, s)
                                             : launch_level_1d<float>(p, uin, uout, phase, s);
    else             rc = p->dtype == GE_F64 ? launch_level_2d<double>(p, uin, uout, phase, s)
                                             : launch_level_2d<float>(p, uin, uout, phase, s);
    if (rc == GE_OK) p->level += 1;
    return rc;
}

// persistent grid of the TMA-staged kernel: queried once per plan and tile width
template <typename T, int C>
cudaError_t stream_dispatch(ge_plan* p, const T* in, T* out, const ge::Coef1<T>* c, int tb, int phase, cudaStream_t s) {
    if (p->stream_ctas == 0) {
        int per_sm = 0;
        auto* fn = &ge::ge1d_stream_kernel<T, C>;
        cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e == cudaSuccess && ge::stream_smem_bytes<T, C>() > 48 * 1024)
            e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ge::stream_smem_bytes<T, C>());
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, ge::kStreamWarps * 32, ge::stream_smem_bytes<T, C>());
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorInvalidConfiguration;
        p->stream_ctas = per_sm * p->sm_count;
    }
    return ge::stream1d_launch<T, C>(in, out, p->nx, p->batch, c, tb, phase, p->stream_ctas, s);
}

// ---- strategy B launch (1-D): tb levels from the plan's current level (any phase) ----
template <typename T>
int launch_temporal_1d(ge_plan* p, const void* uin, void* uout, int tb, cudaStream_t s) {
    const int phase = (int)(p->level & 1);
    auto* in = (const T*)uin;
    auto* out = (T*)uout;
    auto* c = (const ge::Coef1<T>*)p->coef;
    cudaError_t e;
    constexpr int C0 = 16 / (int)sizeof(T) * 4;     // 8 (f64) / 16 (f32)
    // rods of at least one tile take the drift-free kernels, shorter ones the generic (drifting) one
    const bool df = p->nx >= 32 * (int64_t)p->tc;
    // the TMA-staged kernel: lane strides of 144 / 176 / 208 bytes (odd multiples of 16: conflict-free)
    constexpr int CS = 144 / (int)sizeof(T), CS2 = 176 / (int)sizeof(T), CS3 = 208 / (int)sizeof(T);
    switch (p->tc) {
        case CS: case CS2: case CS3: {
            if (!df) return GE_EINVAL;
            e = p->tc == CS ? stream_dispatch<T, CS>(p, in, out, c, tb, phase, s)
              : p->tc == CS2 ? stream_dispatch<T, CS2>(p, in, out, c, tb, phase, s)
                             : stream_dispatch<T, CS3>(p, in, out, c, tb, phase, s);
            break;
        }
        case C0:
            e = df ? ge::temporal1d_launch<T, C0>(in, out, p->nx, p->batch, c, tb, phase, s)
                   : ge::temporal1d_generic_launch<T, C0>(in, out, p->nx, p->batch, c, tb, phase, s);
            break;
        case 2 * C0:
            e = df ? ge::temporal1d_launch<T, 2 * C0>(in, out, p->nx, p->batch, c, tb, phase, s)
                   : ge::temporal1d_generic_launch<T, 2 * C0>(in, out, p->nx, p->batch, c, tb, phase, s);
            break;
        case 4 * C0:
            e = df ? ge::temporal1d_launch<T, 4 * C0>(in, out, p->nx, p->batch, c, tb, phase, s)
                   : ge::temporal1d_generic_launch<T, 4 * C0>(in, out, p->nx, p->batch, c, tb, phase, s);
            break;
        default: return GE_EINVAL;
    }
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    p->launches += 1;
    p->level += tb;
    return GE_OK;
}

// ---- strategy B launch (2-D): plan->tb levels (a compiled-in block length) from the current level ----
template <typename T>
int launch_temporal_2d(ge_plan* p, const void* uin, void* uout, cudaStream_t s) {
    const int phase = (int)(p->level & 1);
    auto* in = (const T*)uin;
    auto* out = (T*)uout;
    auto* c = (const ge::Coef2<T>*)p->coef;
    cudaError_t e;
    switch (p->tb) {
        case 4: e = ge::temporal2d_launch<T, 4, 4>(in, out, p->nx, p->ny, c, phase, p->hp, s); break;
        case 8: e = ge::temporal2d_launch<T, 4, 8>(in, out, p->nx, p->ny, c, phase, p->hp, s); break;
        default: return GE_EINVAL;
    }
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    p->launches += 1;
    p->level += p->tb;
    return GE_OK;
}
// ---- strategy B launch (2-D, drift-free strips; ge_strip2d.cu): plan->tb levels from the current PHASE-1 level ----
bool strip2d_ok(const ge_plan* p) {
    return p->dim == 2 && p->nx % 4 == 0 && p->nx >= 32 * ge::strip2d_columns_per_lane(p->dtype);
}
// COOP warps of a CTA share one strip (GE_TUNE_STRIP_COOP): the grid must hold at least one such strip
bool strip2d_coop_ok(const ge_plan* p, int64_t coop) {
    return coop == 0 || (strip2d_ok(p) && ge::strip2d_coop_compiled(p->dtype, p->tb, (int)coop) &&
                         p->nx >= coop * 32 * ge::strip2d_columns_per_lane(p->dtype));
}

int launch_strip_2d(ge_plan* p, const void* uin, void* uout, cudaStream_t s) {
    if (!ge::strip2d_tb_compiled(p->tb)) return GE_EINVAL;
    const int coop = strip2d_coop_ok(p, p->strip_coop) ? p->strip_coop : 0;
    const int key = p->tb * 16 + coop;
    bool configured = p->strip_attr_tb == key;
    const cudaError_t e = ge::strip2d_dispatch(p->dtype, p->tb, coop, uin, uout, p->nx, p->ny, p->coef, p->hp, configured, s);
    if (configured) p->strip_attr_tb = key;
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    p->launches += 1;
    p->level += p->tb;
    return GE_OK;
}
// block lengths: 4, 8 everywhere; 6 only where the strip kernel runs
bool temporal2d_tb_ok(const ge_plan* p, int64_t tb) { return tb == 4 || tb == 8 || (tb == 6 && strip2d_ok(p)); }

// A single rod whose length is not a multiple of the vector: the blocked kernel marches the prefix of
// nx - nx % V nodes, ge1d_tail_kernel recomputes the end piece (ge_tail.cuh).  Returns the prefix length, or 0.
int64_t temporal_prefix(const ge_plan* p, const void* u) {
    const int V = p->dtype == GE_F64 ? 2 : 4;
    if (p->dim != 1 || p->group_k != 1 || p->batch != 1 || p->nx % V == 0) return 0;
    if (((uintptr_t)u % 16) || ((uintptr_t)p->scratch % 16)) return 0;
    const int64_t np = p->nx - p->nx % V;
    // the window of the end piece (4 tb + 4 + tail, tb may grow by 2 in ge_run's schedule) must fit, and the
    // prefix must still be a rod the blocked kernels take
    if (4 * ((int64_t)p->tb + 2) + 8 + V > ge::kTailMaxLen || np < 8 * ((int64_t)p->tb + 2) + 64) return 0;
    return np;
}
template <typename T>
int launch_tail(ge_plan* p, const void* uin, void* uout, int64_t np, int phase0, int levels, cudaStream_t s) {
    int64_t w0 = np - 4 * (int64_t)levels - 4;
    w0 -= w0 & 1;
    const int64_t o0 = np - 2 * (int64_t)levels - 2;
    ge::ge1d_tail_kernel<T><<<1, ge::kTailThreads, 0, s>>>((const T*)uin, (T*)uout, p->nx, (const ge::Coef1<T>*)p->coef,
                                                            w0, o0, phase0, levels);
    GE_CUDA(cudaGetLastError());
    p->launches += 1;
    return GE_OK;
}

bool temporal_ok(const ge_plan* p, const void* u) {
    if (p->dim == 2 && (p->nx >= (1 << 30) || p->ny >= (1 << 30))) return false;
    const int V = p->dtype == GE_F64 ? 2 : 4;
    return p->nx % V == 0 && ((uintptr_t)u % 16 == 0) && ((uintptr_t)p->scratch % 16 == 0);
}

// Rows the aligned kernels do not take (batched rods with nx % V != 0, unaligned pointers): the warp-per-tile kernel
// with coalesced scalar accesses transposed through shared memory (ge_temporal.cuh, UA).
template <typename T>
int launch_temporal_1d_unaligned(ge_plan* p, const void* uin, void* uout, int tb, cudaStream_t s) {
    const int phase = (int)(p->level & 1);
    auto* in = (const T*)uin;
    auto* out = (T*)uout;
    auto* c = (const ge::Coef1<T>*)p->coef;
    constexpr int C0 = 16 / (int)sizeof(T) * 4;     // 8 (f64) / 16 (f32)
    if (tb < 1 || tb > ge::temporal1d_max_tb(C0)) return GE_EINVAL;
    // 16 values per lane in either precision (measured on a 2^27 rod: fp64 C = 16 3546 GLUPS, C = 8 3291; fp32 C = 16
    // 4775, C = 32 3914 -- 175 registers)
    const bool big = sizeof(T) == 8 && p->nx >= 128 * (int64_t)C0;
    const cudaError_t e = big ? ge::temporal1d_unaligned_launch<T, 2 * C0>(in, out, p->nx, p->batch, c, tb, phase, s)
                              : ge::temporal1d_unaligned_launch<T, C0>(in, out, p->nx, p->batch, c, tb, phase, s);
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    p->launches += 1;
    p->level += tb;
    return GE_OK;
}

int stream_tc(int dtype) { return dtype == GE_F64 ? 22 : 52; }     // measured on C4 / C3
bool is_stream_tc(int dtype, int64_t tc) { const int64_t b = dtype == GE_F64 ? 8 : 4; return tc * b == 144 || tc * b == 176 || tc * b == 208; }
// the TMA-staged kernel when the rod holds at least two tiles, else the warp-per-tile one
int default_tc(int dtype, int64_t nx) {
    // (shorter rods: 64 bytes per lane -- 65536 rods of 1032 nodes, tb 20: fp64 3347 GLUPS at 8 per lane against 3001
    // at 16, fp32 5255 at 16 against 4089 at 32)
    return nx >= 2 * 32 * (int64_t)stream_tc(dtype) ? stream_tc(dtype) : (dtype == GE_F64 ? 8 : 16);
}
int clamp_tb(const ge_plan* p, int64_t tb) {
    const int mx = ge::temporal1d_max_tb(p->tc);
    return (int)(tb > mx ? mx : tb);
}

// ---- strategy C (ge_resident.cuh) ------------------------------------------
// Values per lane the resident kernels are instantiated for (ascending).
template <typename T> struct ResidentC;
// (the two smallest serve short batched rods -- a rod of 100 nodes in 25 lanes of one warp; the whole-chip kernel
// takes the three largest)
constexpr int kResidentCs = 6;
template <> struct ResidentC<float>  { static constexpr int n = kResidentCs; static constexpr int c[kResidentCs] = {4, 8, 16, 32, 64, 128}; };
template <> struct ResidentC<double> { static constexpr int n = kResidentCs; static constexpr int c[kResidentCs] = {2, 4, 8, 16, 32, 64}; };
constexpr int kRodMaxWarps = 8;

inline const int* resident_c_list(int dtype) { return dtype == GE_F64 ? ResidentC<double>::c : ResidentC<float>::c; }

// Path 1 geometry: a rod of nx nodes in one CTA.  Prefers one warp (no barrier) with as many lanes
// in use as possible, then the largest C with the fewest warps.  `want_c` != 0 pins C.
bool rod_resident_pick(int dtype, int64_t nx, int want_c, int* c_out, int* w_out) {
    const int* cs = resident_c_list(dtype);
    if (nx % 2) return false;
    if (want_c) {
        bool known = false;
        for (int i = 0; i < kResidentCs; ++i) known |= cs[i] == want_c;
        if (!known || nx % want_c) return false;
        const int64_t lanes = nx / want_c;
        int w = 1;
        while (32 * w < lanes) w *= 2;
        if (w > kRodMaxWarps) return false;
        *c_out = want_c; *w_out = w;
        return true;
    }
    for (int i = 0; i < kResidentCs; ++i)
        if (nx % cs[i] == 0 && nx / cs[i] <= 32) { *c_out = cs[i]; *w_out = 1; return true; }
    for (int i = kResidentCs - 1; i >= 0; --i) {
        if (nx % cs[i]) continue;
        const int64_t lanes = nx / cs[i];
        int w = 1;
        while (32 * w < lanes) w *= 2;
        if (w <= kRodMaxWarps) { *c_out = cs[i]; *w_out = w; return true; }
    }
    return false;
}

template <typename T, int C>
cudaError_t rod_resident_dispatch_w(ge_plan* p, T* u, int phase0, int64_t steps, cudaStream_t s) {
    auto* c = (const ge::Coef1<T>*)p->coef;
    switch (p->res_w) {
        case 1: return ge::rod_resident_launch<T, C, 1>(u, p->nx, p->batch, c, phase0, steps, s);
        case 2: return ge::rod_resident_launch<T, C, 2>(u, p->nx, p->batch, c, phase0, steps, s);
        case 4: return ge::rod_resident_launch<T, C, 4>(u, p->nx, p->batch, c, phase0, steps, s);
        case 8: return ge::rod_resident_launch<T, C, 8>(u, p->nx, p->batch, c, phase0, steps, s);
        default: return cudaErrorInvalidValue;
    }
}

template <typename T>
int launch_rod_resident(ge_plan* p, void* u, int64_t steps, cudaStream_t s) {
    const int phase0 = (int)(p->level & 1);
    constexpr const int* cs = ResidentC<T>::c;
    cudaError_t e = cudaErrorInvalidValue;
    if (p->res_c == cs[0]) e = rod_resident_dispatch_w<T, cs[0]>(p, (T*)u, phase0, steps, s);
    else if (p->res_c == cs[1]) e = rod_resident_dispatch_w<T, cs[1]>(p, (T*)u, phase0, steps, s);
    else if (p->res_c == cs[2]) e = rod_resident_dispatch_w<T, cs[2]>(p, (T*)u, phase0, steps, s);
    else if (p->res_c == cs[3]) e = rod_resident_dispatch_w<T, cs[3]>(p, (T*)u, phase0, steps, s);
    else if (p->res_c == cs[4]) e = rod_resident_dispatch_w<T, cs[4]>(p, (T*)u, phase0, steps, s);
    else if (p->res_c == cs[5]) e = rod_resident_dispatch_w<T, cs[5]>(p, (T*)u, phase0, steps, s);
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    p->launches += 1;
    p->level += steps;
    return GE_OK;
}

// Path 2: the grid-resident kernel is instantiated for the three largest C of the dtype.
template <typename T, int C>
const void* grid_resident_fn(bool cl) {
    return cl ? (const void*)&ge::ge1d_grid_resident_kernel<T, C, true> : (const void*)&ge::ge1d_grid_resident_kernel<T, C, false>;
}

// cl: the instantiation whose tiles meet inside thread-block clusters (sync modes 4 .. 7)
const void* grid_resident_fn_for(int dtype, int c, bool cl = false) {
    if (dtype == GE_F64) {
        if (c == 16) return grid_resident_fn<double, 16>(cl);
        if (c == 32) return grid_resident_fn<double, 32>(cl);
        if (c == 64) return grid_resident_fn<double, 64>(cl);
    } else {
        if (c == 32) return grid_resident_fn<float, 32>(cl);
        if (c == 64) return grid_resident_fn<float, 64>(cl);
        if (c == 128) return grid_resident_fn<float, 128>(cl);
    }
    return nullptr;
}

// Launch geometry of the cluster form: CTAs rounded up to whole clusters, the shared-memory exchange buffer
// (2 parities x kGridWarps tiles x 2 sides x hl*C), cooperative + cluster attributes.
struct ClusterLaunch {
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[2];
};
int cluster_launch_config(const ge_plan* p, int sync_mode, cudaStream_t s, ClusterLaunch* cl, const void** fn_out) {
    const int cs = ge::sync_cluster_size(sync_mode);
    const void* fn = grid_resident_fn_for(p->dtype, p->res_c, true);
    if (!fn || cs < 2) return GE_EINVAL;
    const size_t smem = (size_t)2 * ge::kGridWarps * 2 * p->res_hl * p->res_c * elem_size(p->dtype);
    if (smem > 48 * 1024) GE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (cs > 8) GE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    unsigned ctas = (unsigned)((p->res_tiles + ge::kGridWarps - 1) / ge::kGridWarps);
    ctas = (ctas + cs - 1) / cs * cs;
    std::memset(cl, 0, sizeof(*cl));
    cl->cfg.gridDim = dim3(ctas);
    cl->cfg.blockDim = dim3(32 * ge::kGridWarps);
    cl->cfg.dynamicSmemBytes = smem;
    cl->cfg.stream = s;
    cl->attr[0].id = cudaLaunchAttributeClusterDimension;
    cl->attr[0].val.clusterDim.x = (unsigned)cs; cl->attr[0].val.clusterDim.y = 1; cl->attr[0].val.clusterDim.z = 1;
    cl->attr[1].id = cudaLaunchAttributeCooperative;
    cl->attr[1].val.cooperative = 1;
    cl->cfg.attrs = cl->attr;
    cl->cfg.numAttrs = 2;
    *fn_out = fn;
    return GE_OK;
}
// can the whole rod be resident when its CTAs come in clusters of this size?
int cluster_mode_fits(const ge_plan* p, int sync_mode, bool* fits) {
    ClusterLaunch cl;
    const void* fn = nullptr;
    *fits = false;
    const int rc = cluster_launch_config(p, sync_mode, nullptr, &cl, &fn);
    if (rc != GE_OK) return rc;
    cl.cfg.numAttrs = 1;                                  // the occupancy query takes the cluster shape only
    int nclusters = 0;
    const cudaError_t e = cudaOccupancyMaxActiveClusters(&nclusters, fn, &cl.cfg);
    if (e != cudaSuccess) { cudaGetLastError(); return GE_OK; }      // this cluster size is not available: does not fit
    *fits = (int64_t)nclusters * ge::sync_cluster_size(sync_mode) >= (int64_t)cl.cfg.gridDim.x;
    return GE_OK;
}

// (Re)derive path-2 geometry from res_c / res_hl / res_tb and (re)allocate its buffers.
// Returns GE_OK with res_path = 2 when the rod fits on the chip, GE_OK with res_path = 0 when not.
int grid_resident_configure(ge_plan* p) {
    p->res_path = 0;
    if (p->dim != 1 || p->batch != 1) return GE_OK;
    const void* fn = grid_resident_fn_for(p->dtype, p->res_c);
    if (!fn || p->nx % p->res_c) return GE_OK;
    if (p->res_hl < 1 || p->res_hl > 8) return GE_OK;
    const int64_t valid = (int64_t)(32 - 2 * p->res_hl) * p->res_c;
    const int64_t tiles = (p->nx + valid - 1) / valid;
    int coop = 0, per_sm = 0;
    GE_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, p->device));
    if (!coop) return GE_OK;
    GE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * ge::kGridWarps, 0));
    p->res_capacity = (int64_t)per_sm * p->sm_count * ge::kGridWarps;
    if (tiles > p->res_capacity) return GE_OK;
    int tb = p->res_tb > 0 ? p->res_tb : p->res_hl * p->res_c;
    if (tb > p->res_hl * p->res_c) tb = p->res_hl * p->res_c;
    tb -= tb % 2;
    if (tb < 2) return GE_OK;
    // buffers: exchange (2 parities x tiles x 2 sides x hl*C) and flags (+ fault word)
    GE_CUDA(cudaStreamSynchronize(p->last_stream));      // an earlier launch may still use the old ones
    cudaFree(p->res_xbuf); cudaFree(p->res_flags);
    p->res_xbuf = nullptr; p->res_flags = nullptr;
    // sized for the flag-in-data lines: 16 bytes per fp64 value (8 per fp32 value)
    const size_t xb = (size_t)ge::kLineSlots * tiles * 2 * p->res_hl * p->res_c * 2 * elem_size(p->dtype);
    GE_CUDA(cudaMalloc(&p->res_xbuf, xb));
    GE_CUDA(cudaMemset(p->res_xbuf, 0, xb));
    // flags[tiles], the fault word, and 256 per-SM arrival counters of the staggered mode
    GE_CUDA(cudaMalloc((void**)&p->res_flags, (size_t)(tiles + 1 + 256) * sizeof(unsigned)));
    GE_CUDA(cudaMemset(p->res_flags, 0, (size_t)(tiles + 1 + 256) * sizeof(unsigned)));
    p->res_epoch = 0;
    p->res_tiles = tiles;
    p->res_tb = tb;
    p->res_path = 2;
    if (ge::sync_cluster_size(p->res_sync) > 1) {        // a cluster mode chosen for the old geometry must still fit
        bool fits = false;
        const int rc = cluster_mode_fits(p, p->res_sync, &fits);
        if (rc != GE_OK || !fits) p->res_sync = ge::kSyncGrid;
    }
    return GE_OK;
}

int launch_grid_resident(ge_plan* p, void* u, int64_t steps, cudaStream_t s) {
    ge::GridResidentArgs a;
    a.nx = p->nx; a.ntiles = p->res_tiles; a.steps = steps; a.phase0 = (int)(p->level & 1);
    a.hl = p->res_hl; a.tb = p->res_tb; a.sync_mode = p->res_sync; a.epoch0 = p->res_epoch;
    void* xbuf = p->res_xbuf;
    void* coef = p->coef;
    unsigned* flags = p->res_flags;
    unsigned* fault = p->res_flags + p->res_tiles;
    if (p->res_sync == ge::kSyncStagger)
        GE_CUDA(cudaMemsetAsync(p->res_flags + p->res_tiles + 1, 0, 256 * sizeof(unsigned), s));
    void* args[] = {&u, &xbuf, &coef, &flags, &fault, &a};
    cudaError_t e;
    if (ge::sync_cluster_size(p->res_sync) > 1) {
        ClusterLaunch cl;
        const void* fn = nullptr;
        const int rc = cluster_launch_config(p, p->res_sync, s, &cl, &fn);
        if (rc != GE_OK) return rc;
        e = cudaLaunchKernelExC(&cl.cfg, fn, args);
    } else {
        const void* fn = grid_resident_fn_for(p->dtype, p->res_c);
        const unsigned ctas = (unsigned)((p->res_tiles + ge::kGridWarps - 1) / ge::kGridWarps);
        e = cudaLaunchCooperativeKernel(fn, dim3(ctas), dim3(32 * ge::kGridWarps), args, 0, s);
    }
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    const int64_t meet = ge::grid_resident_meetings(steps, a.phase0, a.tb);
    // every launch moves the epoch past all flag values / line tags it used (one extra meeting is held
    // by the flag-in-data mode when the run has none)
    p->res_epoch += (unsigned)(2 + (p->res_sync == ge::kSyncStagger ? ge::grid_resident_halves(steps, a.phase0, a.tb) : meet));
    p->meetings += meet;
    p->launches += 1;
    p->level += steps;
    return GE_OK;
}

// Decide the strategy-C path at plan creation / after a tuning call.
int resident_configure(ge_plan* p, int want_c) {
    if (p->group_k != 1) return GE_EUNSUPPORTED;       // two-point groups only (callers check; never silently k = 1)
    p->res_path = 0;
    if (p->dim != 1) return GE_OK;
    const int* cs = resident_c_list(p->dtype);
    int c = 0, w = 0;
    const bool rod = rod_resident_pick(p->dtype, p->nx, want_c, &c, &w);
    // one rod that needs more than one warp: spread it over the chip when it fits there
    if (p->batch == 1 && (!rod || w > 1)) {
        p->res_c = want_c ? want_c : cs[4];
        const int rc = grid_resident_configure(p);
        if (rc != GE_OK || p->res_path == 2) return rc;
    }
    if (rod) { p->res_path = 1; p->res_c = c; p->res_w = w; }
    return GE_OK;
}

bool resident_ok(const ge_plan* p, const void* u) {
    return p->res_path != 0 && ((uintptr_t)u % 16 == 0);
}

// ---- strategy B with non-constant data (ge_window.cuh): `levels` <= kWindowTb levels per launch ----
constexpr int kWindowTb = 16;
// (2^27 rod, GLUPS source / variable diffusivity at 8 / 12 / 16 / 20 / 24 levels per launch: fp64 2085 / 2735 / 2941 /
// 2933 / 2816 and 1546 / 2019 / 2449 / 2668 / 2693; fp32 3698 / 4293 / 4775 / 4998 / 4958 and 2485 / 3454 / 4739 / 5610 / 5747)
#ifndef GE_SRC_TB
#define GE_SRC_TB 20
#endif
constexpr int kSrcTb = GE_SRC_TB;        // levels per launch of the register kernels for non-constant data
template <typename T, bool SRC, bool VAR>
int launch_window(ge_plan* p, const void* uin, void* uout, const void* src, const void* rl, const void* bc, int64_t bc_lev,
                  int64_t bc_stride, int levels, cudaStream_t s) {
    const ge::WinGeom g = ge::win_geom(kWindowTb, p->nx);
    if (g.valid <= 0 || levels < 1 || levels > kWindowTb) return GE_EINVAL;
    auto* fn = ge::ge1d_window_kernel<T, SRC, VAR>;
    GE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ge::win_smem<T>()));
    GE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    dim3 grid((unsigned)g.tiles, (unsigned)(p->batch < 65535 ? p->batch : 65535));
    fn<<<grid, ge::kWinThreads, ge::win_smem<T>(), s>>>((const T*)uin, (T*)uout, (const T*)src, (const T*)rl, (const T*)bc, bc_lev,
                                                         bc_stride, p->nx, p->batch, (const ge::Coef1<T>*)p->coef, g,
                                                         (int)(p->level & 1), levels);
    GE_CUDA(cudaGetLastError());
    p->launches += 1;
    p->level += levels;
    return GE_OK;
}

int step_common(ge_plan* p, int dim, const void* uin, void* uout, cudaStream_t s) {
    if (!p || !uin || !uout || uin == uout || p->dim != dim) return GE_EINVAL;
    const size_t es = elem_size(p->dtype);
    if ((uintptr_t)uin % es || (uintptr_t)uout % es) return GE_EINVAL;
    const char* a = (const char*)uin; const char* b = (const char*)uout;
    const size_t bytes = (size_t)p->count * es;
    if ((a < b + bytes) && (b < a + bytes)) return GE_EINVAL;   // overlap
    p->last_stream = s;
    return launch_level(p, uin, uout, s);
}

}  // namespace

extern "C" {

int ge_version(void) { return 100; }

const char* ge_strerror(int status) {
    switch (status) {
        case GE_OK: return "ok";
        case GE_EINVAL: return "invalid argument";
        case GE_ENOMEM: return "out of memory";
        case GE_EUNSUPPORTED: return "unsupported on the GPU path (group_k > 2048: a unit does not fit in shared memory)";
        case GE_ECUDA:
            std::snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error: %s", cudaGetErrorString(g_last_cuda));
            return g_errbuf;
        default: return "unknown status";
    }
}

int ge_plan_create(ge_plan** out, const ge_desc* d, ge_stream_t stream) {
    if (!out || !d) return GE_EINVAL;
    if (d->dim != 1 && d->dim != 2 && d->dim != 3) return GE_EINVAL;
    if (d->nx < 1 || d->ny < 1 || d->batch < 1) return GE_EINVAL;
    if (d->dim == 3 && (d->nz < 1 || d->batch != 1 || d->nx >= (1 << 30) || d->ny >= (1 << 30) || d->nz >= (1 << 30))) return GE_EINVAL;
    if (d->dim != 3 && d->nz > 1) return GE_EINVAL;
    if (d->dim == 1 && d->ny != 1) return GE_EINVAL;
    if (d->dim == 2 && d->batch != 1) return GE_EINVAL;
    if (d->dtype != GE_F32 && d->dtype != GE_F64) return GE_EINVAL;
    if (d->group_k < 1) return GE_EINVAL;
    if (d->group_k >= 2 && d->dim >= 2) return GE_EINVAL;
    if (d->kernel < GE_KERNEL_AUTO || d->kernel > GE_KERNEL_PERSISTENT) return GE_EINVAL;
    if (d->tb < 0) return GE_EINVAL;
    if (!d->r || !d->bc_lo || !d->bc_hi) return GE_EINVAL;
    const int64_t nr = d->dim == 1 ? d->batch : 1;
    for (int64_t b = 0; b < nr; ++b)
        if (!(d->r[b] > 0.0) || !std::isfinite(d->r[b])) return GE_EINVAL;
    const int64_t nb = d->dim == 1 ? d->batch : d->dim;
    for (int64_t b = 0; b < nb; ++b)
        if (!std::isfinite(d->bc_lo[b]) || !std::isfinite(d->bc_hi[b])) return GE_EINVAL;
    if (d->group_k > kMaxGroupK) return GE_EUNSUPPORTED;

    ge_plan* p = new (std::nothrow) ge_plan();
    if (!p) return GE_ENOMEM;
    std::memset(p, 0, sizeof(*p));
    p->dim = d->dim; p->dtype = d->dtype; p->group_k = d->group_k;
    p->host_r = d->r[0]; p->host_lo = d->bc_lo[0]; p->host_hi = d->bc_hi[0];
    p->host_desc = *d;
    p->nx = d->nx; p->ny = d->ny; p->nz = d->dim == 3 ? d->nz : 1; p->batch = d->batch;
    p->count = d->dim == 1 ? d->batch * d->nx : d->ny * d->nx * p->nz;
    p->last_stream = (cudaStream_t)stream;
    int rc = GE_OK;
    cudaError_t ce = cudaGetDevice(&p->device);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    if (ce != cudaSuccess) { g_last_cuda = ce; delete p; return GE_ECUDA; }
    rc = p->dtype == GE_F64 ? upload_coef<double>(p, d, (cudaStream_t)stream)
                            : upload_coef<float>(p, d, (cudaStream_t)stream);
    if (rc == GE_OK) {
        ce = cudaMalloc(&p->scratch, (size_t)p->count * elem_size(p->dtype));
        if (ce != cudaSuccess) { g_last_cuda = ce; rc = ce == cudaErrorMemoryAllocation ? GE_ENOMEM : GE_ECUDA; }
    }
    if (rc != GE_OK) { cudaFree(p->coef); cudaFree(p->scratch); cudaGetLastError(); delete p; return rc; }

    // strategy selection: AUTO takes the resident kernels when the state fits on
    // the chip (1-D only), else the temporally blocked ones
    p->tb = 0;
    p->tc = default_tc(p->dtype, p->nx);
    p->hp = p->dtype == GE_F64 ? 56 : 67;   // measured on C5 (the rate depends on the segment count, and sharply)
    p->form3d = 1;
    p->kform = 1;
    p->src_form = 1;
    p->res_hl = 2;                 // measured on C2: 2 halo lanes, grid-wide meetings
    p->res_sync = ge::kSyncGrid;
    int kernel = d->kernel;
    if (d->group_k >= 2) {                                  // k >= 2 (ge_level_k.cuh): strategy A, or C when the rod fits in shared memory
        const bool want_c = kernel == GE_KERNEL_AUTO || kernel == GE_KERNEL_PERSISTENT;
        const bool want_b = kernel != GE_KERNEL_PER_STEP;
        // measured on the C4-shaped rod: 32 for the register-resident form, 16 for the shared-memory one
        const int tbk = d->tb > 0 ? d->tb : (ge::unit_k_compiled(d->dtype, d->group_k) ? 32 : 16);
        kernel = GE_KERNEL_PER_STEP;
        if (want_c && rod_k_fits(p)) { kernel = GE_KERNEL_PERSISTENT; p->res_path = 3; }
        else if (want_b && temporal_k_ok(p, tbk)) { kernel = GE_KERNEL_TEMPORAL; p->tb = tbk; }
    }
    if (d->dim == 3) kernel = GE_KERNEL_PER_STEP;          // 3-D: strategy A only (ge_level3d.cuh)
    if (d->group_k == 1 && (kernel == GE_KERNEL_AUTO || kernel == GE_KERNEL_PERSISTENT)) {
        p->res_tb = d->tb;
        rc = resident_configure(p, 0);
        if (rc != GE_OK) { cudaFree(p->coef); cudaFree(p->scratch); cudaFree(p->res_xbuf); cudaFree(p->res_flags); cudaGetLastError(); delete p; return rc; }
        kernel = p->res_path ? GE_KERNEL_PERSISTENT : GE_KERNEL_TEMPORAL;
    }
    // 2-D, AUTO: a blocked launch has a latency floor of 60 - 75 us (a warp marches its segment row pair by row pair
    // through tb stages) whatever the grid, a per-level launch costs 4 us or its HBM time: below 24 MB of state one
    // launch per level is faster (measured: fp32 2048^2 0.99 against 1.24 ms for 120 levels, 3072^2 1.63 against
    // 1.54; fp64 1024^2 0.86 against 1.22, 2048^2 1.85 against 1.40)
    if (d->dim == 2 && d->kernel == GE_KERNEL_AUTO && (int64_t)p->count * (int64_t)elem_size(p->dtype) < ((int64_t)24 << 20))
        kernel = GE_KERNEL_PER_STEP;
    p->kernel = kernel;
    const bool temporal_like = kernel == GE_KERNEL_TEMPORAL || kernel == GE_KERNEL_PERSISTENT;   // C falls back to B
    // measured on C4: the TMA-staged kernel is fp64-bound from tb ~ 12 on, best near 20
    if (temporal_like && d->dim == 1 && d->group_k == 1) p->tb = clamp_tb(p, d->tb > 0 ? d->tb : (is_stream_tc(p->dtype, p->tc) ? 20 : 24));   // (warp-per-tile, 65536 rods of 1032 nodes: fp64 3278 / 3348 / 3420 GLUPS at 16 / 20 / 24, fp32 5137 / 5255 / 5388)
    if (temporal_like && d->dim == 2) {
        p->tc = 4;
        p->tb = d->tb > 0 ? d->tb : (strip2d_ok(p) ? 6 : 8);   // measured on C5
        if (!temporal2d_tb_ok(p, p->tb)) { cudaFree(p->coef); cudaFree(p->scratch); delete p; return GE_EINVAL; }
        // segments: the C5 optimum (67 / 56 row pairs) leaves a smaller grid with too few warps -- 32 strips x 31
        // segments on 4096^2 fp32 --, so segments shrink until strips x segments give every SM ~28 warps, down to 16
        // pairs; GE_TUNE_SEG_PAIRS overrides
        if (strip2d_ok(p)) {
            const int64_t strips = (p->nx + 32 * ge::strip2d_columns_per_lane(p->dtype) - 1) / (32 * ge::strip2d_columns_per_lane(p->dtype));
            // (4096^2, 120 levels: fp32 2.30 / 2.16 / 1.88 ms at 67 / 32 / 16 pairs, fp64 2.56 / 2.42 / 2.62 at 56 / 32 / 16:
            // both optima hold ~28 warps per SM)
            const int64_t want = (int64_t)28 * p->sm_count;
            int64_t hp = (p->ny / 2) * strips / want;
            if (hp < 16) hp = 16;
            if (4 * hp < 3 * p->hp) p->hp = (int32_t)hp;         // (near the C5 optimum the rate is too sensitive to move)
        }
    }
    *out = p;
    return GE_OK;
}

int ge_step_1d(ge_plan* p, const void* u_in, void* u_out, ge_stream_t stream) {
    return step_common(p, 1, u_in, u_out, (cudaStream_t)stream);
}

int ge_step_1d_src(ge_plan* p, const void* u_in, void* u_out, const void* tau_f, const double* bc4,
                   ge_stream_t stream) {
    if (!p || !u_in || !u_out || u_in == u_out || !bc4 || p->dim != 1 || p->batch != 1) return GE_EINVAL;
    if (p->group_k != 1) return GE_EUNSUPPORTED;
    for (int i = 0; i < 4; ++i) if (!std::isfinite(bc4[i])) return GE_EINVAL;
    const size_t es = elem_size(p->dtype);
    if ((uintptr_t)u_in % es || (uintptr_t)u_out % es || (uintptr_t)tau_f % es) return GE_EINVAL;
    const char* a = (const char*)u_in; const char* b = (const char*)u_out;
    const size_t bytes = (size_t)p->count * es;
    if ((a < b + bytes) && (b < a + bytes)) return GE_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    p->last_stream = s;
    const int phase = (int)(p->level & 1);
    cudaError_t e;
    if (p->dtype == GE_F64) {
        const ge::SrcBc<double> bc{bc4[0], bc4[1], bc4[2], bc4[3]};
        e = ge::level_src_launch<double>((const double*)u_in, (double*)u_out, (const double*)tau_f, p->nx,
                                         (const ge::Coef1<double>*)p->coef, bc, phase, s);
    } else {
        const ge::SrcBc<float> bc{(float)bc4[0], (float)bc4[1], (float)bc4[2], (float)bc4[3]};
        e = ge::level_src_launch<float>((const float*)u_in, (float*)u_out, (const float*)tau_f, p->nx,
                                        (const ge::Coef1<float>*)p->coef, bc, phase, s);
    }
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    p->launches += 1;
    p->level += 1;
    return GE_OK;
}

int ge_step_1d_var(ge_plan* p, const void* u_in, void* u_out, const void* rl, ge_stream_t stream) {
    if (!p || !u_in || !u_out || u_in == u_out || !rl || p->dim != 1 || p->batch != 1) return GE_EINVAL;
    if (p->group_k != 1) return GE_EUNSUPPORTED;
    const size_t es = elem_size(p->dtype);
    if ((uintptr_t)u_in % es || (uintptr_t)u_out % es || (uintptr_t)rl % es) return GE_EINVAL;
    const char* a = (const char*)u_in; const char* b = (const char*)u_out;
    const size_t bytes = (size_t)p->count * es;
    if ((a < b + bytes) && (b < a + bytes)) return GE_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    p->last_stream = s;
    const int phase = (int)(p->level & 1);
    const cudaError_t e = p->dtype == GE_F64
        ? ge::level_var_launch<double>((const double*)u_in, (double*)u_out, (const double*)rl, p->nx, (const ge::Coef1<double>*)p->coef, phase, s)
        : ge::level_var_launch<float>((const float*)u_in, (float*)u_out, (const float*)rl, p->nx, (const ge::Coef1<float>*)p->coef, phase, s);
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    p->launches += 1;
    p->level += 1;
    return GE_OK;
}

int ge_run_var(ge_plan* p, void* u, int64_t steps, const void* rl, ge_stream_t stream) {
    if (!p || !u || steps < 0 || !rl || p->dim != 1) return GE_EINVAL;
    if (p->group_k != 1) return GE_EUNSUPPORTED;
    const size_t es = elem_size(p->dtype);
    if ((uintptr_t)u % es || (uintptr_t)rl % es) return GE_EINVAL;
    NvtxRange nvtx("ge_run_var");
    cudaStream_t s = (cudaStream_t)stream;
    p->last_stream = s;
    void* cur = u;
    void* oth = p->scratch;
    int64_t left = steps;
    // rows of whole aligned vectors that hold a tile: the register form (ge_temporal_src.cuh); anything else: windows in
    // shared memory (ge_window.cuh)
    const int V = p->dtype == GE_F64 ? 2 : 4, cvar = p->dtype == GE_F64 ? GE_SRC_C_F64 : GE_SRC_C_F32;
    const bool regs = p->nx % V == 0 && p->nx >= 32 * (int64_t)cvar && (uintptr_t)u % 16 == 0 && (uintptr_t)p->scratch % 16 == 0 &&
                      p->src_form != 0;
    while (left > 0) {
        // equal-sized blocks of at most kWindowTb levels, the link numbers resident beside the state
        const int tbmax = regs ? kSrcTb : kWindowTb;
        const int64_t nl = (left + tbmax - 1) / tbmax;
        const int lv = (int)((left + nl - 1) / nl);
        int rc;
        if (regs) {
            const int phase = (int)(p->level & 1);
            const cudaError_t e = p->dtype == GE_F64
                ? ge::temporal1d_var_launch<double, GE_SRC_C_F64>((const double*)cur, (double*)oth, (const double*)rl, p->nx, p->batch,
                                                        (const ge::Coef1<double>*)p->coef, lv, phase, s)
                : ge::temporal1d_var_launch<float, GE_SRC_C_F32>((const float*)cur, (float*)oth, (const float*)rl, p->nx, p->batch,
                                                       (const ge::Coef1<float>*)p->coef, lv, phase, s);
            if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
            p->launches += 1;
            p->level += lv;
            rc = GE_OK;
        } else
        rc = p->dtype == GE_F64 ? launch_window<double, false, true>(p, cur, oth, nullptr, rl, nullptr, 0, 0, lv, s)
                                : launch_window<float, false, true>(p, cur, oth, nullptr, rl, nullptr, 0, 0, lv, s);
        if (rc != GE_OK) return rc;
        left -= lv;
        void* t = cur; cur = oth; oth = t;
    }
    if (cur != u) GE_CUDA(cudaMemcpyAsync(u, cur, (size_t)p->count * es, cudaMemcpyDeviceToDevice, s));
    return GE_OK;
}

int ge_run_src(ge_plan* p, void* u, int64_t steps, const void* tau_f, int64_t f_level_stride, const double* bc_lo_t,
               const double* bc_hi_t, ge_stream_t stream) {
    if (!p || !u || steps < 0 || !bc_lo_t || !bc_hi_t || f_level_stride < 0 || p->dim != 1) return GE_EINVAL;
    if (p->group_k != 1) return GE_EUNSUPPORTED;
    const bool per_level = tau_f && f_level_stride != 0;
    if (per_level && (f_level_stride < p->nx || p->batch != 1)) return GE_EINVAL;
    const int64_t nb = p->batch * (steps + 1);
    for (int64_t n = 0; n < nb; ++n)
        if (!std::isfinite(bc_lo_t[n]) || !std::isfinite(bc_hi_t[n])) return GE_EINVAL;
    const size_t es = elem_size(p->dtype);
    if ((uintptr_t)u % es || (uintptr_t)tau_f % es) return GE_EINVAL;
    NvtxRange nvtx("ge_run_src");
    cudaStream_t s = (cudaStream_t)stream;
    p->last_stream = s;
    void* cur = u;
    void* oth = p->scratch;
    if (per_level) {
        // a different source array every level: one launch per level (ge_level_src.cuh)
        for (int64_t n = 0; n < steps; ++n) {
            const double bc4[4] = {bc_lo_t[n], bc_lo_t[n + 1], bc_hi_t[n], bc_hi_t[n + 1]};
            const void* f = (const char*)tau_f + (size_t)(n * f_level_stride) * es;
            const int rc = ge_step_1d_src(p, cur, oth, f, bc4, stream);
            if (rc != GE_OK) return rc;
            void* t = cur; cur = oth; oth = t;
        }
    } else if (steps > 0) {
        // stationary source (or none): blocked -- the boundary values of all levels go to the device first
        const size_t bytes = (size_t)nb * 2 * es;
        if (p->bc_cap < bytes) {
            GE_CUDA(cudaStreamSynchronize(s));                 // an earlier run may still read the old buffer
            cudaFree(p->bc_dev); p->bc_dev = nullptr; p->bc_cap = 0;
            GE_CUDA(cudaMalloc(&p->bc_dev, bytes));
            p->bc_cap = bytes;
        }
        if (p->dtype == GE_F64) {
            std::vector<double> h((size_t)nb * 2);
            for (int64_t n = 0; n < nb; ++n) { h[2 * n] = bc_lo_t[n]; h[2 * n + 1] = bc_hi_t[n]; }
            GE_CUDA(cudaMemcpyAsync(p->bc_dev, h.data(), bytes, cudaMemcpyHostToDevice, s));
            GE_CUDA(cudaStreamSynchronize(s));                 // h is a stack-owned staging buffer
        } else {
            std::vector<float> h((size_t)nb * 2);
            for (int64_t n = 0; n < nb; ++n) { h[2 * n] = (float)bc_lo_t[n]; h[2 * n + 1] = (float)bc_hi_t[n]; }
            GE_CUDA(cudaMemcpyAsync(p->bc_dev, h.data(), bytes, cudaMemcpyHostToDevice, s));
            GE_CUDA(cudaStreamSynchronize(s));
        }
        // rows of whole aligned vectors that hold a tile: the register form (ge_temporal_src.cuh); anything else: windows
        // in shared memory (ge_window.cuh)
        const int V = p->dtype == GE_F64 ? 2 : 4, csrc = p->dtype == GE_F64 ? GE_SRC_C_F64 : GE_SRC_C_F32;
        const bool regs = p->nx % V == 0 && p->nx >= 32 * (int64_t)csrc && (uintptr_t)u % 16 == 0 && (uintptr_t)p->scratch % 16 == 0 &&
                          (uintptr_t)tau_f % 16 == 0 && p->src_form != 0;
        int64_t left = steps, done = 0;
        while (left > 0) {
            const int tbmax = regs ? kSrcTb : kWindowTb;
            const int64_t nl = (left + tbmax - 1) / tbmax;
            const int lv = (int)((left + nl - 1) / nl);
            int rc;
            if (regs) {
                const int phase = (int)(p->level & 1);
                const cudaError_t e = p->dtype == GE_F64
                    ? ge::temporal1d_src_launch<double, GE_SRC_C_F64>((const double*)cur, (double*)oth, (const double*)tau_f, (const double*)p->bc_dev, done, steps + 1,
                                                            p->nx, p->batch, (const ge::Coef1<double>*)p->coef, lv, phase, s)
                    : ge::temporal1d_src_launch<float, GE_SRC_C_F32>((const float*)cur, (float*)oth, (const float*)tau_f, (const float*)p->bc_dev, done, steps + 1,
                                                           p->nx, p->batch, (const ge::Coef1<float>*)p->coef, lv, phase, s);
                if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
                p->launches += 1;
                p->level += lv;
                rc = GE_OK;
            } else
            rc = p->dtype == GE_F64 ? launch_window<double, true, false>(p, cur, oth, tau_f, nullptr, p->bc_dev, done, steps + 1, lv, s)
                                    : launch_window<float, true, false>(p, cur, oth, tau_f, nullptr, p->bc_dev, done, steps + 1, lv, s);
            if (rc != GE_OK) return rc;
            left -= lv; done += lv;
            void* t = cur; cur = oth; oth = t;
        }
    }
    if (cur != u) GE_CUDA(cudaMemcpyAsync(u, cur, (size_t)p->count * es, cudaMemcpyDeviceToDevice, s));
    return GE_OK;
}

int ge_step_2d(ge_plan* p, const void* u_in, void* u_out, ge_stream_t stream) {
    return step_common(p, 2, u_in, u_out, (cudaStream_t)stream);
}

int ge_step_3d(ge_plan* p, const void* u_in, void* u_out, ge_stream_t stream) {
    return step_common(p, 3, u_in, u_out, (cudaStream_t)stream);
}

// Levels of the next launch of strategy B in 1-D, `left` levels to go from level `level`.
static int temporal1d_block(int64_t left, int64_t level, int tb, int tc) {
    int tbn;
    if (tb % 2 == 0 && tb >= 4) {
        // blocks that start at an odd level and have an even length are pure R/L pairs: a run from
        // an even level opens with one block of tb-1 levels (in-lane level I first), a tail of one
        // or two levels joins the last block (which may then end with R + shift back)
        const int64_t nl = left > 2 ? (left - 2 + tb - 1) / tb : 1;   // launches to go (a block may take tb+2)
        int64_t q = (left + nl - 1) / nl;
        q += q & 1;
        tbn = (int)((level & 1) ? q : q - 1);
        if (tbn > left) tbn = (int)left;
        if (left - tbn <= 2 && left <= ge::temporal1d_max_tb(tc)) tbn = (int)left;
    } else {
        // equal-sized blocks: ceil(left / tb) launches of (almost) the same number of levels
        const int64_t nl = (left + tb - 1) / tb;
        tbn = (int)((left + nl - 1) / nl);
    }
    return tbn;
}
static int64_t temporal1d_launch_count(int64_t left, int64_t level, int tb, int tc) {
    int64_t n = 0;
    while (left > 0) { const int t = temporal1d_block(left, level, tb, tc); left -= t; level += t; ++n; }
    return n;
}
// The state ping-pongs between the caller's buffer and the plan's scratch level: an ODD number of launches leaves
// the result in the scratch level and costs a copy of the whole state.  Three or more launches: a block length up
// to a quarter larger (one launch fewer) or, failing that, smaller (one launch more: the price of the copy, no
// more) makes the count even.  Returns the block length to run with.
static int temporal1d_even_tb(int64_t left, int64_t level, int tb, int tc, int tb_max) {
    const int64_t n0 = temporal1d_launch_count(left, level, tb, tc);
    if (n0 < 3 || (n0 & 1) == 0) return tb;
    const int step = (tb % 2 == 0 && tb >= 4) ? 2 : 1;             // an even tb keeps the R/L block form
    int cap = tb + tb / 4;
    if (cap > tb_max) cap = tb_max;
    for (int t = tb + step; t <= cap; t += step)
        if ((temporal1d_launch_count(left, level, t, tc) & 1) == 0) return t;
    for (int t = tb - step; t >= 4 && 2 * t >= tb; t -= step)
        if ((temporal1d_launch_count(left, level, t, tc) & 1) == 0) return t;
    return tb;
}

int ge_run(ge_plan* p, void* u, int64_t steps, ge_stream_t stream) {
    if (!p || !u || steps < 0) return GE_EINVAL;
    NvtxRange nvtx("ge_run");
    const size_t es = elem_size(p->dtype);
    if ((uintptr_t)u % es) return GE_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    p->last_stream = s;
    void* cur = u;
    void* oth = p->scratch;
    int64_t left = steps;
    int rc = GE_OK;
    if (p->kernel == GE_KERNEL_PERSISTENT && p->res_path == 3) {
        if (steps == 0) return GE_OK;
        return p->dtype == GE_F64 ? launch_rod_k_resident<double>(p, u, steps, s)
                                  : launch_rod_k_resident<float>(p, u, steps, s);
    }
    if (p->kernel == GE_KERNEL_PERSISTENT && resident_ok(p, u)) {
        // strategy C: the whole run is one launch, in place
        if (steps == 0) return GE_OK;
        if (p->res_path == 1)
            return p->dtype == GE_F64 ? launch_rod_resident<double>(p, u, steps, s)
                                      : launch_rod_resident<float>(p, u, steps, s);
        return launch_grid_resident(p, u, steps, s);
    }
    const bool blocked = (p->kernel == GE_KERNEL_TEMPORAL || p->kernel == GE_KERNEL_PERSISTENT) && p->group_k == 1;
    const int64_t prefix = blocked ? temporal_prefix(p, u) : 0;
    const bool temporal_al = blocked && (prefix > 0 || temporal_ok(p, u));
    const bool unaligned = blocked && !temporal_al && p->dim == 1 && p->tb >= 1 && p->tb + 2 <= 64;
    const bool temporal = temporal_al || unaligned;
    const bool temporal_k = p->kernel == GE_KERNEL_TEMPORAL && p->group_k >= 2;
    int tb1d = p->tb;
    if (temporal && p->dim == 1) {
        // largest block the kernel of this run takes: the unaligned form has the smaller tiles, the end piece a window limit
        int tb_max = unaligned ? ge::temporal1d_max_tb(16 / (int)es * 4) - 2 : ge::temporal1d_max_tb(p->tc) - 2;
        if (prefix && tb_max > p->tb) tb_max = p->tb;
        tb1d = temporal1d_even_tb(left, p->level, p->tb, p->tc, tb_max);
    }
    while (left > 0 && rc == GE_OK) {
        if (temporal_k) {
            // equal-sized blocks of at most tb levels (any starting phase)
            const int64_t nl = (left + p->tb - 1) / p->tb;
            const int lv = (int)((left + nl - 1) / nl);
            rc = p->dtype == GE_F64 ? launch_temporal_k<double>(p, cur, oth, lv, s) : launch_temporal_k<float>(p, cur, oth, lv, s);
            left -= lv;
        } else if (temporal && p->dim == 2) {
            const bool strips = strip2d_ok(p);
            if (strips && left > p->tb && (p->level & 1) == 0) {
                // the strip kernel starts at a phase-1 level: one per-level launch first
                rc = launch_level(p, cur, oth, s);
                left -= 1;
            } else if (strips && left >= p->tb && (p->level & 1) == 1) {
                rc = launch_strip_2d(p, cur, oth, s);
                left -= p->tb;
            } else if (!strips && left >= p->tb) {
                rc = p->dtype == GE_F64 ? launch_temporal_2d<double>(p, cur, oth, s)
                                        : launch_temporal_2d<float>(p, cur, oth, s);
                left -= p->tb;
            } else {
                rc = launch_level(p, cur, oth, s);
                left -= 1;
            }
        } else if (temporal) {
            const int tbn = temporal1d_block(left, p->level, tb1d, p->tc);
            if (unaligned) {
                rc = p->dtype == GE_F64 ? launch_temporal_1d_unaligned<double>(p, cur, oth, tbn, s)
                                        : launch_temporal_1d_unaligned<float>(p, cur, oth, tbn, s);
            } else if (prefix) {
                // the prefix as a rod of its own (tile geometry and kernel choice follow its length), then the end piece
                const int64_t nx0 = p->nx;
                const int ph0 = (int)(p->level & 1);
                p->nx = prefix;
                rc = p->dtype == GE_F64 ? launch_temporal_1d<double>(p, cur, oth, tbn, s)
                                        : launch_temporal_1d<float>(p, cur, oth, tbn, s);
                p->nx = nx0;
                if (rc == GE_OK)
                    rc = p->dtype == GE_F64 ? launch_tail<double>(p, cur, oth, prefix, ph0, tbn, s)
                                            : launch_tail<float>(p, cur, oth, prefix, ph0, tbn, s);
            } else
            rc = p->dtype == GE_F64 ? launch_temporal_1d<double>(p, cur, oth, tbn, s)
                                    : launch_temporal_1d<float>(p, cur, oth, tbn, s);
            left -= tbn;
        } else {
            rc = launch_level(p, cur, oth, s);
            left -= 1;
        }
        void* t = cur; cur = oth; oth = t;
    }
    if (rc != GE_OK) return rc;
    if (cur != u) GE_CUDA(cudaMemcpyAsync(u, cur, (size_t)p->count * es, cudaMemcpyDeviceToDevice, s));
    return GE_OK;
}

// ge_run_host for one long rod: the rod is cut into chunks that are marched INDEPENDENTLY -- a chunk
// carries 2*steps+8 extra nodes per side, more than the dependency cone of `steps` levels (a two-point
// group reads u_{i-1}..u_{i+2}), so its interior comes out exactly as in the whole-rod
// run -- and the chunks travel through a three-slot pipeline: while chunk c is computed, chunk c+1 is
// on its way to the device and chunk c-1 on its way back.
constexpr int kHostSlots = 3;
#ifndef GE_HOST_CHUNK_LOG2
#define GE_HOST_CHUNK_LOG2 22
#endif
constexpr int64_t kHostChunk = (int64_t)1 << GE_HOST_CHUNK_LOG2;

static int host_pipeline(ge_plan* p, void* u_host, int64_t steps, cudaStream_t user) {
    const size_t es = elem_size(p->dtype);
    const int64_t halo = (2 * steps + 8 + 3) & ~(int64_t)3, nx = p->nx;    // a multiple of 4: chunks keep the vector kernels
    if (!p->slots) {
        p->slots = new (std::nothrow) ge_plan::HostSlot[kHostSlots]();
        if (!p->slots) return GE_ENOMEM;
        for (int i = 0; i < kHostSlots; ++i) {
            GE_CUDA(cudaStreamCreateWithFlags(&p->slots[i].stream, cudaStreamNonBlocking));
            GE_CUDA(cudaEventCreateWithFlags(&p->slots[i].h2d_done, cudaEventDisableTiming));
        }
    }
    cudaEvent_t start;
    GE_CUDA(cudaEventCreateWithFlags(&start, cudaEventDisableTiming));
    GE_CUDA(cudaEventRecord(start, user));
    for (int i = 0; i < kHostSlots; ++i) GE_CUDA(cudaStreamWaitEvent(p->slots[i].stream, start, 0));
    const int64_t nchunks = (nx + kHostChunk - 1) / kHostChunk;
    auto range = [&](int64_t c, int64_t& i0, int64_t& i1, int64_t& o0, int64_t& o1) {
        o0 = c * kHostChunk; o1 = o0 + kHostChunk < nx ? o0 + kHostChunk : nx;
        i0 = o0 - halo > 0 ? o0 - halo : 0; i1 = o1 + halo < nx ? o1 + halo : nx;
    };
    auto upload = [&](int64_t c) -> int {
        ge_plan::HostSlot& sl = p->slots[c % kHostSlots];
        int64_t i0, i1, o0, o1; range(c, i0, i1, o0, o1);
        const size_t bytes = (size_t)(i1 - i0) * es;
        if (sl.cap < bytes) { cudaFree(sl.buf); sl.buf = nullptr; sl.cap = 0; GE_CUDA(cudaMalloc(&sl.buf, bytes)); sl.cap = bytes; }
        GE_CUDA(cudaMemcpyAsync(sl.buf, (const char*)u_host + (size_t)i0 * es, bytes, cudaMemcpyHostToDevice, sl.stream));
        GE_CUDA(cudaEventRecord(sl.h2d_done, sl.stream));
        return GE_OK;
    };
    int rc = upload(0);
    for (int64_t c = 0; c < nchunks && rc == GE_OK; ++c) {
        ge_plan::HostSlot& sl = p->slots[c % kHostSlots];
        int64_t i0, i1, o0, o1; range(c, i0, i1, o0, o1);
        // sub-plan of this slot for this chunk shape: real boundary value where the chunk touches the rod's end
        const int kind = (i0 == 0 ? 1 : 0) | (i1 == nx ? 2 : 0);
        if (sl.sub[kind] && sl.sub_len[kind] != i1 - i0) { ge_plan_destroy(sl.sub[kind]); sl.sub[kind] = nullptr; }
        if (!sl.sub[kind]) {
            ge_desc d = p->host_desc;
            const double r = p->host_r, lo = (kind & 1) ? p->host_lo : 0.0, hi = (kind & 2) ? p->host_hi : 0.0;
            d.nx = i1 - i0; d.r = &r; d.bc_lo = &lo; d.bc_hi = &hi; d.kernel = p->kernel == GE_KERNEL_PER_STEP ? GE_KERNEL_PER_STEP : GE_KERNEL_TEMPORAL;
            d.tb = p->tb > 0 ? p->tb : 0;
            rc = ge_plan_create(&sl.sub[kind], &d, (ge_stream_t)sl.stream);
            if (rc != GE_OK) break;
            sl.sub_len[kind] = i1 - i0;
        }
        ge_plan* sub = sl.sub[kind];
        sub->level = p->level;
        rc = ge_run(sub, sl.buf, steps, (ge_stream_t)sl.stream);
        if (rc != GE_OK) break;
        p->launches += sub->launches; sub->launches = 0;
        // the next chunk reads host nodes this chunk is about to overwrite: upload it first
        if (c + 1 < nchunks) {
            // its slot's previous download (chunk c-2) is ordered before by the slot's stream
            rc = upload(c + 1);
            if (rc != GE_OK) break;
            GE_CUDA(cudaStreamWaitEvent(sl.stream, p->slots[(c + 1) % kHostSlots].h2d_done, 0));
        }
        // ... and so did the previous chunk (its upload is long done; make the order explicit)
        if (c >= 1) GE_CUDA(cudaStreamWaitEvent(sl.stream, p->slots[(c - 1) % kHostSlots].h2d_done, 0));
        GE_CUDA(cudaMemcpyAsync((char*)u_host + (size_t)o0 * es, (const char*)sl.buf + (size_t)(o0 - i0) * es,
                                (size_t)(o1 - o0) * es, cudaMemcpyDeviceToHost, sl.stream));
    }
    for (int i = 0; i < kHostSlots; ++i) {
        const cudaError_t e = cudaStreamSynchronize(p->slots[i].stream);
        if (e != cudaSuccess && rc == GE_OK) { g_last_cuda = e; rc = GE_ECUDA; }
    }
    cudaEventDestroy(start);
    if (rc == GE_OK) p->level += steps;
    return rc;
}

// ge_run_host for batched rods: the rods are independent, so the batch travels in groups of rods through the
// same three-slot pipeline (upload of group c+1 and download of group c-1 overlap the levels of group c).
// A group is run by pointing the plan at its slice of the state, the coefficient table and the scratch level.
static int host_pipeline_rods(ge_plan* p, void* u_host, int64_t steps, cudaStream_t user) {
    const size_t es = elem_size(p->dtype);
    const size_t coef_sz = p->dtype == GE_F64 ? sizeof(ge::Coef1<double>) : sizeof(ge::Coef1<float>);
    const int64_t groups = 8, per = (p->batch + groups - 1) / groups;
    if (!p->slots) {
        p->slots = new (std::nothrow) ge_plan::HostSlot[kHostSlots]();
        if (!p->slots) return GE_ENOMEM;
        for (int i = 0; i < kHostSlots; ++i) {
            GE_CUDA(cudaStreamCreateWithFlags(&p->slots[i].stream, cudaStreamNonBlocking));
            GE_CUDA(cudaEventCreateWithFlags(&p->slots[i].h2d_done, cudaEventDisableTiming));
        }
    }
    const size_t bytes = (size_t)p->count * es;
    if (!p->hostpath) GE_CUDA(cudaMalloc(&p->hostpath, bytes));
    cudaEvent_t start;
    GE_CUDA(cudaEventCreateWithFlags(&start, cudaEventDisableTiming));
    GE_CUDA(cudaEventRecord(start, user));
    for (int i = 0; i < kHostSlots; ++i) GE_CUDA(cudaStreamWaitEvent(p->slots[i].stream, start, 0));
    // the plan is pointed at one group at a time
    const int64_t batch0 = p->batch, count0 = p->count, level0 = p->level;
    void* const coef0 = p->coef; void* const scratch0 = p->scratch;
    int rc = GE_OK;
    int64_t c = 0;
    for (int64_t rod0 = 0; rod0 < batch0 && rc == GE_OK; rod0 += per, ++c) {
        const int64_t n = rod0 + per <= batch0 ? per : batch0 - rod0;
        cudaStream_t st = p->slots[c % kHostSlots].stream;
        const size_t off = (size_t)rod0 * p->nx * es, len = (size_t)n * p->nx * es;
        cudaError_t e = cudaMemcpyAsync((char*)p->hostpath + off, (const char*)u_host + off, len, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { g_last_cuda = e; rc = GE_ECUDA; break; }
        p->batch = n; p->count = n * p->nx; p->level = level0;
        p->coef = (char*)coef0 + (size_t)rod0 * coef_sz;
        p->scratch = (char*)scratch0 + off;
        rc = ge_run(p, (char*)p->hostpath + off, steps, (ge_stream_t)st);
        if (rc != GE_OK) break;
        e = cudaMemcpyAsync((char*)u_host + off, (const char*)p->hostpath + off, len, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) { g_last_cuda = e; rc = GE_ECUDA; }
    }
    p->batch = batch0; p->count = count0; p->coef = coef0; p->scratch = scratch0;
    for (int i = 0; i < kHostSlots; ++i) {
        const cudaError_t e = cudaStreamSynchronize(p->slots[i].stream);
        if (e != cudaSuccess && rc == GE_OK) { g_last_cuda = e; rc = GE_ECUDA; }
    }
    cudaEventDestroy(start);
    p->level = rc == GE_OK ? level0 + steps : level0;
    return rc;
}

int ge_run_host(ge_plan* p, void* u_host, int64_t steps, ge_stream_t stream) {
    if (!p || !u_host || steps < 0) return GE_EINVAL;
    NvtxRange nvtx("ge_run_host");
    cudaStream_t s = (cudaStream_t)stream;
    const size_t bytes = (size_t)p->count * elem_size(p->dtype);
    if (p->dim == 1 && p->batch == 1 && p->group_k == 1 && steps > 0 && p->nx >= 2 * kHostChunk &&
        2 * steps + 8 <= kHostChunk / 8) {
        p->last_stream = s;
        const int rc = host_pipeline(p, u_host, steps, s);
        if (rc != GE_OK) return rc;
        GE_CUDA(cudaStreamSynchronize(s));
        return GE_OK;
    }
    if (p->dim == 1 && p->batch >= 64 && steps > 0 && bytes >= ((size_t)8 << 20) && p->res_path != 2) {
        p->last_stream = s;
        const int rc = host_pipeline_rods(p, u_host, steps, s);
        if (rc != GE_OK) return rc;
        GE_CUDA(cudaStreamSynchronize(s));
        return GE_OK;
    }
    if (!p->hostpath) GE_CUDA(cudaMalloc(&p->hostpath, bytes));
    GE_CUDA(cudaMemcpyAsync(p->hostpath, u_host, bytes, cudaMemcpyHostToDevice, s));
    int rc = ge_run(p, p->hostpath, steps, stream);
    if (rc != GE_OK) return rc;
    GE_CUDA(cudaMemcpyAsync(u_host, p->hostpath, bytes, cudaMemcpyDeviceToHost, s));
    GE_CUDA(cudaStreamSynchronize(s));
    return GE_OK;
}

int ge_plan_get_level(const ge_plan* p, int64_t* level) {
    if (!p || !level) return GE_EINVAL;
    *level = p->level;
    return GE_OK;
}

int ge_plan_set_level(ge_plan* p, int64_t level) {
    if (!p || level < 0) return GE_EINVAL;
    p->level = level;
    return GE_OK;
}

int ge_plan_info(const ge_plan* p, int32_t what, int64_t* value) {
    if (!p || !value) return GE_EINVAL;
    switch (what) {
        case GE_INFO_KERNEL: *value = p->kernel; return GE_OK;
        case GE_INFO_TB: *value = p->tb; return GE_OK;
        case GE_INFO_LAUNCHES: *value = p->launches; return GE_OK;
        case GE_INFO_TILE_VALID:
        case GE_INFO_TILE_LOADED: {
            const int V = p->dtype == GE_F64 ? 2 : 4;
            int valid = 0, loaded = 0;
            if (p->kernel != GE_KERNEL_TEMPORAL) { }
            else if (p->dim == 1 && p->group_k >= 2) {
                const ge::TemporalKGeom g = ge::temporal_k_geom(p->group_k, p->tb, p->nx, elem_size(p->dtype), kTemporalKSmemBudget);
                valid = g.valid; loaded = g.window;
            }
            else if (p->dim == 1) { valid = ge::temporal1d_geom(p->tc, V, p->tb, 1).valid; loaded = 32 * p->tc; }
            else if (strip2d_ok(p))   // the kernel that runs: strips of (coop*)32*C columns, halo stale columns per side
                ge::strip2d_tile(p->dtype, p->tb, strip2d_coop_ok(p, p->strip_coop) ? p->strip_coop : 0, p->nx, p->ny, p->hp, &valid, &loaded);
            else { valid = ge::temporal2d_geom(p->tc, V, p->tb, 0, p->nx, p->ny, p->hp).valid; loaded = 32 * p->tc; }
            *value = what == GE_INFO_TILE_VALID ? valid : loaded;
            return GE_OK;
        }
        case GE_INFO_TEMPORAL_C: *value = p->kernel == GE_KERNEL_TEMPORAL && p->dim == 1 && p->group_k == 1 ? p->tc : 0; return GE_OK;
        case GE_INFO_RESIDENT_PATH: *value = p->kernel == GE_KERNEL_PERSISTENT ? p->res_path : 0; return GE_OK;
        case GE_INFO_RESIDENT_C: *value = p->res_path ? p->res_c : 0; return GE_OK;
        case GE_INFO_RESIDENT_WARPS:
            *value = p->res_path == 1 ? p->res_w : (p->res_path == 2 ? p->res_tiles : 0);
            return GE_OK;
        case GE_INFO_RESIDENT_CAPACITY: *value = p->res_path == 2 ? p->res_capacity : 0; return GE_OK;
        case GE_INFO_RESIDENT_TB: *value = p->res_path == 2 ? p->res_tb : 0; return GE_OK;
        case GE_INFO_MEETINGS: *value = p->meetings; return GE_OK;
        case GE_INFO_SYNC_FAULT: {
            *value = 0;
            if (p->res_path == 2 && p->res_flags) {
                unsigned f = 0;
                GE_CUDA(cudaStreamSynchronize(p->last_stream));
                GE_CUDA(cudaMemcpy(&f, p->res_flags + p->res_tiles, sizeof(f), cudaMemcpyDeviceToHost));
                *value = f;
            }
            return GE_OK;
        }
        default: return GE_EINVAL;
    }
}

int ge_plan_tune(ge_plan* p, int32_t what, int64_t value) {
    if (!p) return GE_EINVAL;
    switch (what) {
        case GE_TUNE_SEG_PAIRS:
            if (value < 1 || value > (1 << 20) || p->dim != 2) return GE_EINVAL;
            p->hp = (int32_t)value;
            return GE_OK;
        case GE_TUNE_K_FORM:
            if (p->group_k < 2 || (value != 0 && value != 1)) return GE_EINVAL;
            p->kform = (int32_t)value;
            return GE_OK;
        case GE_TUNE_SRC_FORM:
            if (p->dim != 1 || (value != 0 && value != 1)) return GE_EINVAL;
            p->src_form = (int32_t)value;
            return GE_OK;
        case GE_TUNE_FORM_3D:
            if (p->dim != 3 || value < 0 || value > 2) return GE_EINVAL;
            p->form3d = (int32_t)value;
            return GE_OK;
        case GE_TUNE_STRIP_COOP:
            if (p->dim != 2 || p->kernel != GE_KERNEL_TEMPORAL || (value != 0 && !strip2d_coop_ok(p, value))) return GE_EINVAL;
            p->strip_coop = (int32_t)value;
            return GE_OK;
        case GE_TUNE_TEMPORAL_C: {
            if (p->dim != 1 || p->group_k != 1) return GE_EINVAL;
            const int c0 = p->dtype == GE_F64 ? 8 : 16;
            if (is_stream_tc(p->dtype, value)) { if (p->nx < 32 * value) return GE_EINVAL; p->stream_ctas = 0; }
            else if (value != c0 && value != 2 * c0 && value != 4 * c0) return GE_EINVAL;
            p->tc = (int32_t)value;
            if (p->kernel == GE_KERNEL_TEMPORAL) p->tb = clamp_tb(p, p->tb);
            return GE_OK;
        }
        case GE_TUNE_RESIDENT_C: {
            // path 1: values per lane (warps follow); path 2: values per lane of a tile
            if (p->kernel != GE_KERNEL_PERSISTENT || value < 2 || value > 128) return GE_EINVAL;
            // the register-resident kernels are the k = 1 scheme; a k >= 2 plan stays on its shared-memory path
            if (p->group_k >= 2 || p->res_path == 3) return GE_EUNSUPPORTED;
            const int32_t path0 = p->res_path, c0 = p->res_c, w0 = p->res_w;
            p->res_tb = 0;                                     // back to the largest the new halo allows
            int rc = resident_configure(p, (int)value);
            if (rc != GE_OK) return rc;
            if (p->res_path == 0) {                            // not instantiated / does not fit: restore
                p->res_c = c0; p->res_w = w0;
                if (path0 == 2) { rc = grid_resident_configure(p); if (rc != GE_OK) return rc; }
                else p->res_path = path0;
                return GE_EINVAL;
            }
            return GE_OK;
        }
        case GE_TUNE_HALO_LANES: {
            if (p->kernel != GE_KERNEL_PERSISTENT || p->res_path != 2 || value < 1 || value > 8) return GE_EINVAL;
            const int32_t hl0 = p->res_hl, tb0 = p->res_tb;
            p->res_hl = (int32_t)value; p->res_tb = 0;
            int rc = grid_resident_configure(p);
            if (rc == GE_OK && p->res_path != 2) {
                p->res_hl = hl0; p->res_tb = tb0;
                rc = grid_resident_configure(p);
                return rc == GE_OK ? GE_EINVAL : rc;
            }
            return rc;
        }
        case GE_TUNE_SYNC_MODE:
            if (p->kernel != GE_KERNEL_PERSISTENT || p->res_path != 2) return GE_EINVAL;
            if (value < ge::kSyncFlags || value > ge::kSyncCluster16) return GE_EINVAL;
            if (value == ge::kSyncStagger && p->res_tb < 8) return GE_EINVAL;
            if (ge::sync_cluster_size((int)value) > 1) {         // clusters: the whole rod must still be co-resident
                bool fits = false;
                const int rc = cluster_mode_fits(p, (int)value, &fits);
                if (rc != GE_OK) return rc;
                if (!fits) return GE_EINVAL;
            }
            p->res_sync = (int32_t)value;
            return GE_OK;
        case GE_TUNE_TB:
            if (value < 1) return GE_EINVAL;
            if (p->kernel == GE_KERNEL_PERSISTENT && p->res_path == 2) {
                int64_t tb = value > (int64_t)p->res_hl * p->res_c ? (int64_t)p->res_hl * p->res_c : value;
                tb -= tb % 2;
                if (tb < 2 || (p->res_sync == ge::kSyncStagger && tb < 8)) return GE_EINVAL;
                p->res_tb = (int32_t)tb;
                return GE_OK;
            }
            if (p->kernel != GE_KERNEL_TEMPORAL) return GE_EINVAL;
            if (p->group_k >= 2) {
                if (!temporal_k_ok(p, (int)(value > 4096 ? 4096 : value))) return GE_EINVAL;
                p->tb = (int32_t)value;
                return GE_OK;
            }
            if (p->dim == 2) {
                if (!temporal2d_tb_ok(p, value)) return GE_EINVAL;
                p->tb = (int32_t)value;
                return GE_OK;
            }
            p->tb = clamp_tb(p, value);
            return GE_OK;
        default: return GE_EINVAL;
    }
}

int ge_fma_probe(int32_t dtype, int64_t iters, void* sink, double* flops, ge_stream_t stream) {
    return ge_fma_probe_ex(dtype, 0, iters, sink, flops, stream);
}

int ge_fma_probe_ex(int32_t dtype, int32_t variant, int64_t iters, void* sink, double* flops, ge_stream_t stream) {
    if ((dtype != GE_F32 && dtype != GE_F64) || iters < 1 || !sink || !flops || variant < 0 || variant > 1) return GE_EINVAL;
    int dev = 0, sms = 0;
    GE_CUDA(cudaGetDevice(&dev));
    GE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const cudaError_t e = dtype == GE_F64 ? ge::fma_probe_launch<double>((double*)sink, iters, sms, flops, (cudaStream_t)stream, variant == 1)
                                          : ge::fma_probe_launch<float>((float*)sink, iters, sms, flops, (cudaStream_t)stream, variant == 1);
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    return GE_OK;
}

int ge_plan_destroy(ge_plan* p) {
    if (!p) return GE_EINVAL;
    // stream-ordered with respect to the last stream used: wait for it, then free
    cudaError_t e = cudaStreamSynchronize(p->last_stream);
    cudaFree(p->coef);
    cudaFree(p->scratch);
    cudaFree(p->hostpath);
    cudaFree(p->res_xbuf);
    cudaFree(p->res_flags);
    cudaFree(p->bc_dev);
    if (p->aux3d) { cudaStreamSynchronize(p->aux3d); cudaStreamDestroy(p->aux3d); }
    if (p->ev3d[0]) cudaEventDestroy(p->ev3d[0]);
    if (p->ev3d[1]) cudaEventDestroy(p->ev3d[1]);
    if (p->slots) {
        for (int i = 0; i < kHostSlots; ++i) {
            for (int kd = 0; kd < 4; ++kd) if (p->slots[i].sub[kd]) ge_plan_destroy(p->slots[i].sub[kd]);
            cudaFree(p->slots[i].buf);
            if (p->slots[i].stream) cudaStreamDestroy(p->slots[i].stream);
            if (p->slots[i].h2d_done) cudaEventDestroy(p->slots[i].h2d_done);
        }
        delete[] p->slots;
    }
    delete p;
    if (e != cudaSuccess) { g_last_cuda = e; return GE_ECUDA; }
    return GE_OK;
}

}  // extern "C"
