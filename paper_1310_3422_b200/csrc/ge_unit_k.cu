// ge_unit_k.cu -- instantiations and dispatch of the register-resident k >= 2 kernel (ge_unit_k.cuh).
#include "ge_dispatch.h"
#include "ge_unit_k.cuh"

namespace ge {

bool unit_k_compiled(int dtype, int k) {
    return k == 2 || k == 4 || k == 8 || k == 16 || (k == 32 && dtype == 0);
}

int unit_k_valid_lanes(int k, int tb) { return unit_k_geom(k, tb, 1).valid_lanes; }

template <typename T>
static cudaError_t dispatch_t(int k, const T* in, T* out, int64_t nx, int64_t batch, const Coef1<T>* c, int tb, int phase,
                              int levels, cudaStream_t s) {
    switch (k) {
        case 2: return unit_k_launch<T, 2>(in, out, nx, batch, c, tb, phase, levels, s);
        case 4: return unit_k_launch<T, 4>(in, out, nx, batch, c, tb, phase, levels, s);
        case 8: return unit_k_launch<T, 8>(in, out, nx, batch, c, tb, phase, levels, s);
        case 16: return unit_k_launch<T, 16>(in, out, nx, batch, c, tb, phase, levels, s);
        case 32: if constexpr (sizeof(T) == 4) return unit_k_launch<T, 32>(in, out, nx, batch, c, tb, phase, levels, s);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t unit_k_dispatch(int dtype, int k, const void* uin, void* uout, int64_t nx, int64_t batch, const void* coef,
                            int tb, int phase, int levels, cudaStream_t s) {
    return dtype == 1 ? dispatch_t<double>(k, (const double*)uin, (double*)uout, nx, batch, (const Coef1<double>*)coef, tb, phase, levels, s)
                      : dispatch_t<float>(k, (const float*)uin, (float*)uout, nx, batch, (const Coef1<float>*)coef, tb, phase, levels, s);
}

}  // namespace ge
