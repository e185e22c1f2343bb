// ge_static.cu -- ONE entry point that allocates nothing: ge_run_1d_static (include/ge.h).
//
// Callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it) cannot create a ge_plan: a plan allocates its coefficient block and the second copy of the state the levels
// ping-pong through.  This file runs strategy A in 1-D (two-point groups; ge1d_level_kernel of
// ge_level.cuh, the arithmetic unchanged) with both of them in a file-scope device array of a fixed size: every
// GPU that loads the library holds kStaticBytes (4 MiB + 256 bytes) until the process exits.
//
//   * In HOST code the array's name is a host-side stand-in, not a device address.  The address the kernels get
//     comes from cudaGetSymbolAddress, asked once per device with that device current (static_base()).  Device code
//     (ge_static_coef_kernel) names the array directly.
//   * Every call shares the array and finds the previous call's contents in it.  Nothing in it has to start at
//     zero: the coefficient block is rewritten by every call, and every node of the state copy is written by a
//     level before a later level reads it.  Calls that OVERLAP on the GPU (two streams, two host threads) race.
//   * No cudaMalloc, cudaFree or allocating library routine is called: the coefficients travel as a kernel argument.
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/ge.h"
#include "ge_common.cuh"
#include "ge_level.cuh"

namespace {

constexpr size_t kStaticCoefBytes = 256;                       // the coefficient block, then the state copy
constexpr size_t kStaticStateBytes = (size_t)GE_STATIC_MAX_BYTES;
constexpr size_t kStaticBytes = kStaticCoefBytes + kStaticStateBytes;

static __device__ __align__(256) unsigned char ge_static_scratch[kStaticBytes];

template <typename T>
__global__ void ge_static_coef_kernel(const ge::Coef1<T> h) {
    static_assert(sizeof(ge::Coef1<T>) <= kStaticCoefBytes, "coefficient block");
    if (threadIdx.x == 0 && blockIdx.x == 0) *reinterpret_cast<ge::Coef1<T>*>(ge_static_scratch) = h;
}

thread_local char g_static_msg[320] = "ok";

int fail(int status, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(g_static_msg, sizeof(g_static_msg), fmt, ap);
    va_end(ap);
    return status;
}
int fail_cuda(const char* what, cudaError_t e) {
    return fail(GE_ECUDA, "ge_run_1d_static: %s failed: %s", what, cudaGetErrorString(e));
}

// device address of ge_static_scratch on the CURRENT device; asked once per device
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
unsigned char* g_static_base[kMaxDevices] = {};

int static_base(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda("cudaGetDevice", e);
    std::lock_guard<std::mutex> lock(g_static_mu);
    const bool cached = dev >= 0 && dev < kMaxDevices;
    if (cached && g_static_base[dev]) { *out = g_static_base[dev]; return GE_OK; }
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, ge_static_scratch);
    if (e != cudaSuccess) return fail_cuda("cudaGetSymbolAddress", e);
    if (!ptr || ((uintptr_t)ptr % 256) != 0) return fail(GE_ECUDA, "ge_run_1d_static: the scratch array has no usable device address");
    if (cached) g_static_base[dev] = (unsigned char*)ptr;
    *out = (unsigned char*)ptr;
    return GE_OK;
}

template <typename T>
cudaError_t static_level(const T* in, T* out, int64_t nx, const ge::Coef1<T>* c, int phase, cudaStream_t s) {
    constexpr int V = ge::VecOf<T>::V;
    constexpr int ITER = 4;
    const bool vec = (nx % V == 0) && (((uintptr_t)in | (uintptr_t)out) % 16 == 0);
    const int64_t nvec = vec ? nx / V : nx;
    const int64_t per_block = (int64_t)ge::kLevelThreads * ITER;
    dim3 grid((unsigned)((nvec + per_block - 1) / per_block), 1), block(ge::kLevelThreads);
    if (vec) {
        if (phase == 0) ge::ge1d_level_kernel<T, V, 0, ITER><<<grid, block, 0, s>>>(in, out, nx, 1, c);
        else            ge::ge1d_level_kernel<T, V, 1, ITER><<<grid, block, 0, s>>>(in, out, nx, 1, c);
    } else {
        if (phase == 0) ge::ge1d_level_kernel<T, 1, 0, ITER><<<grid, block, 0, s>>>(in, out, nx, 1, c);
        else            ge::ge1d_level_kernel<T, 1, 1, ITER><<<grid, block, 0, s>>>(in, out, nx, 1, c);
    }
    return cudaGetLastError();
}

template <typename T>
int static_run(const void* u_in, void* u_out, int64_t nx, int64_t steps, int64_t level0, double r, double bc_lo,
               double bc_hi, unsigned char* base, cudaStream_t s) {
    ge::Coef1<T> h;
    std::memset(&h, 0, sizeof(h));
    h.r = (T)r;                                   // as ge_plan_create computes them (ge_api.cu upload_coef)
    h.g = (T)(r / (1.0 + 2.0 * r));
    h.e = (T)(r / (1.0 + r));
    h.lo = (T)bc_lo;
    h.hi = (T)bc_hi;
    ge_static_coef_kernel<T><<<1, 32, 0, s>>>(h);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda("the coefficient kernel launch", e);
    const auto* coef = reinterpret_cast<const ge::Coef1<T>*>(base);
    T* tmp = reinterpret_cast<T*>(base + kStaticCoefBytes);
    T* out = static_cast<T*>(u_out);
    const T* src = static_cast<const T*>(u_in);
    // level i (0-based) of `steps` writes u_out when the levels after it are even in number, the scratch copy otherwise
    for (int64_t i = 0; i < steps; ++i) {
        T* dst = ((steps - 1 - i) % 2 == 0) ? out : tmp;
        e = static_level<T>(src, dst, nx, coef, (int)((level0 + i) & 1), s);
        if (e != cudaSuccess) return fail_cuda("a level kernel launch", e);
        src = dst;
    }
    return GE_OK;
}

}  // namespace

extern "C" {

int ge_static_limit(int32_t dtype, int64_t* max_nodes) {
    if (!max_nodes) return fail(GE_EINVAL, "ge_static_limit: max_nodes is null");
    if (dtype != GE_F32 && dtype != GE_F64) return fail(GE_EINVAL, "ge_static_limit: dtype %d is neither GE_F32 nor GE_F64", (int)dtype);
    unsigned char* base = nullptr;
    const int rc = static_base(&base);            // the per-device set-up, so that a caller can do it ahead of time
    if (rc != GE_OK) return rc;
    *max_nodes = (int64_t)(kStaticStateBytes / (dtype == GE_F64 ? 8 : 4));
    return GE_OK;
}

int ge_run_1d_static(int32_t dtype, const void* u_in, void* u_out, int64_t nx, int64_t steps, int64_t level0,
                     double r, double bc_lo, double bc_hi, ge_stream_t stream) {
    if (dtype != GE_F32 && dtype != GE_F64) return fail(GE_EINVAL, "ge_run_1d_static: dtype %d is neither GE_F32 nor GE_F64", (int)dtype);
    const size_t es = dtype == GE_F64 ? 8 : 4;
    if (!u_in || !u_out) return fail(GE_EINVAL, "ge_run_1d_static: u_in / u_out is null");
    if (((uintptr_t)u_in | (uintptr_t)u_out) % es) return fail(GE_EINVAL, "ge_run_1d_static: u_in / u_out is not aligned to the element size");
    if (nx < 1) return fail(GE_EINVAL, "ge_run_1d_static: nx = %lld, need nx >= 1", (long long)nx);
    const int64_t max_nodes = (int64_t)(kStaticStateBytes / es);
    if (nx > max_nodes)
        return fail(GE_EINVAL, "ge_run_1d_static: nx = %lld exceeds the static scratch array: at most %lld %s nodes (%zu bytes, "
                               "GE_STATIC_MAX_BYTES); use a ge_plan for larger rods",
                    (long long)nx, (long long)max_nodes, dtype == GE_F64 ? "f64" : "f32", kStaticStateBytes);
    if (steps < 0 || level0 < 0) return fail(GE_EINVAL, "ge_run_1d_static: steps and level0 must be >= 0");
    if (!(r > 0.0) || !std::isfinite(r) || !std::isfinite(bc_lo) || !std::isfinite(bc_hi))
        return fail(GE_EINVAL, "ge_run_1d_static: r must be finite and > 0, the boundary values finite");
    const uintptr_t a = (uintptr_t)u_in, b = (uintptr_t)u_out, bytes = (uintptr_t)nx * es;
    if (a < b + bytes && b < a + bytes) return fail(GE_EINVAL, "ge_run_1d_static: u_in and u_out overlap");
    unsigned char* base = nullptr;
    int rc = static_base(&base);
    if (rc != GE_OK) return rc;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    if (steps == 0) {
        const cudaError_t e = cudaMemcpyAsync(u_out, u_in, bytes, cudaMemcpyDeviceToDevice, s);
        if (e != cudaSuccess) return fail_cuda("cudaMemcpyAsync", e);
        return GE_OK;
    }
    rc = dtype == GE_F64 ? static_run<double>(u_in, u_out, nx, steps, level0, r, bc_lo, bc_hi, base, s)
                         : static_run<float>(u_in, u_out, nx, steps, level0, r, bc_lo, bc_hi, base, s);
    if (rc == GE_OK) std::snprintf(g_static_msg, sizeof(g_static_msg), "ok");
    return rc;
}

int ge_static_error(char* buf, int64_t cap) {
    if (!buf || cap < 1) return GE_EINVAL;
    std::snprintf(buf, (size_t)cap, "%s", g_static_msg);
    return GE_OK;
}

}  // extern "C"
