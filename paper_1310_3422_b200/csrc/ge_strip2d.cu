// ge_strip2d.cu -- instantiations and dispatch of the 2-D strip kernels (ge_strip2d.cuh).
#include "ge_dispatch.h"
#include "ge_strip2d.cuh"

namespace ge {

#ifndef GE_STRIP_C_F32
#define GE_STRIP_C_F32 4
#endif
#ifndef GE_STRIP_C_F64
#define GE_STRIP_C_F64 2
#endif
template <typename T> struct StripC { static constexpr int c = sizeof(T) == 8 ? GE_STRIP_C_F64 : GE_STRIP_C_F32; };

int strip2d_columns_per_lane(int dtype) { return dtype == 1 ? StripC<double>::c : StripC<float>::c; }
bool strip2d_tb_compiled(int tb) { return tb == 4 || tb == 6 || tb == 8; }
bool strip2d_coop_compiled(int dtype, int tb, int coop) {
    (void)dtype;
    return coop == 0 || (tb == 6 && (coop == 2 || coop == 4 || coop == 8));
}

void strip2d_tile(int dtype, int tb, int coop, int64_t nx, int64_t ny, int hp, int* valid, int* loaded) {
    const int c = strip2d_columns_per_lane(dtype), v = dtype == 1 ? 2 : 4;
    if (coop > 1) { *valid = strip2d_coop_geom(c, v, tb, coop, nx, ny, hp).valid; *loaded = coop * 32 * c; }
    else          { *valid = strip2d_geom(c, v, tb, nx, ny, hp).valid; *loaded = 32 * c; }
}

template <typename T>
static cudaError_t dispatch_t(int tb, int coop, const T* in, T* out, int64_t nx, int64_t ny, const Coef2<T>* c, int hp,
                              bool& configured, cudaStream_t s) {
    constexpr int C = StripC<T>::c;
    if (coop == 2 && tb == 6) return strip2d_coop_launch<T, C, 6, 2>(in, out, nx, ny, c, hp, configured, s);
    if (coop == 4 && tb == 6) return strip2d_coop_launch<T, C, 6, 4>(in, out, nx, ny, c, hp, configured, s);
    if (coop == 8 && tb == 6) return strip2d_coop_launch<T, C, 6, 8>(in, out, nx, ny, c, hp, configured, s);
    if (coop != 0) return cudaErrorInvalidValue;
    switch (tb) {
        case 4: return strip2d_launch<T, C, 4>(in, out, nx, ny, c, hp, configured, s);
        case 6: return strip2d_launch<T, C, 6>(in, out, nx, ny, c, hp, configured, s);
        case 8: return strip2d_launch<T, C, 8>(in, out, nx, ny, c, hp, configured, s);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t strip2d_dispatch(int dtype, int tb, int coop, const void* uin, void* uout, int64_t nx, int64_t ny,
                             const void* coef, int hp, bool& configured, cudaStream_t s) {
    return dtype == 1 ? dispatch_t<double>(tb, coop, (const double*)uin, (double*)uout, nx, ny, (const Coef2<double>*)coef, hp, configured, s)
                      : dispatch_t<float>(tb, coop, (const float*)uin, (float*)uout, nx, ny, (const Coef2<float>*)coef, hp, configured, s);
}

}  // namespace ge
