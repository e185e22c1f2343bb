// ge_stream3d.cu -- instantiations and dispatch of the 3-D kernels (ge_level3d.cuh, ge_stream3d.cuh).
#include "ge_dispatch.h"
#include "ge_stream3d.cuh"

namespace ge {

cudaError_t level3d_dispatch(int dtype, int form, const void* uin, void* uout, int64_t nx, int64_t ny, int64_t nz,
                             const void* coef, int phase, int sm_count, cudaStream_t s, int* launches, cudaStream_t aux, cudaEvent_t ev_in,
                             cudaEvent_t ev_out) {
    // form 1: the streaming kernel where its 16-byte form applies (rows of a multiple of the lane's piece, aligned
    // buffers); its scalar form loses to the thread-per-group kernel (258 x 256 x 256 fp32: 90 against 327 GLUPS),
    // so other shapes take that one.  form 2 forces the streaming kernel (tests of the scalar form).
    const int e = dtype == 1 ? 2 * S3Cfg<double>::ng : 2 * S3Cfg<float>::ng;
    const size_t es = dtype == 1 ? 8 : 4;
    const bool vec = nx % e == 0 && (((uintptr_t)uin | (uintptr_t)uout) % (e * es)) == 0;
    const bool stream = form == 2 || (form == 1 && vec);
    if (!stream) *launches = 1;
    if (dtype == 1)
        return stream ? stream3d_launch<double>((const double*)uin, (double*)uout, nx, ny, nz, (const Coef3<double>*)coef, phase, sm_count, s, launches, aux, ev_in, ev_out)
                      : level3d_launch<double>((const double*)uin, (double*)uout, nx, ny, nz, (const Coef3<double>*)coef, phase, s);
    return stream ? stream3d_launch<float>((const float*)uin, (float*)uout, nx, ny, nz, (const Coef3<float>*)coef, phase, sm_count, s, launches, aux, ev_in, ev_out)
                  : level3d_launch<float>((const float*)uin, (float*)uout, nx, ny, nz, (const Coef3<float>*)coef, phase, s);
}

}  // namespace ge
