// ge_stream3d.cu -- instantiations and dispatch of the 3-D kernels (ge_level3d.cuh, ge_stream3d.cuh).
#include "ge_dispatch.h"
#include "ge_stream3d.cuh"

namespace ge {

cudaError_t level3d_dispatch(int dtype, int form, const void* uin, void* uout, int64_t nx, int64_t ny, int64_t nz,
                             const void* coef, int phase, int sm_count, cudaStream_t s, int* launches, cudaStream_t aux, cudaEvent_t ev_in,
                             cudaEvent_t ev_out) {
    const bool stream = form == 1;
    if (!stream) *launches = 1;
    if (dtype == 1)
        return stream ? stream3d_launch<double>((const double*)uin, (double*)uout, nx, ny, nz, (const Coef3<double>*)coef, phase, sm_count, s, launches, aux, ev_in, ev_out)
                      : level3d_launch<double>((const double*)uin, (double*)uout, nx, ny, nz, (const Coef3<double>*)coef, phase, s);
    return stream ? stream3d_launch<float>((const float*)uin, (float*)uout, nx, ny, nz, (const Coef3<float>*)coef, phase, sm_count, s, launches, aux, ev_in, ev_out)
                  : level3d_launch<float>((const float*)uin, (float*)uout, nx, ny, nz, (const Coef3<float>*)coef, phase, s);
}

}  // namespace ge
