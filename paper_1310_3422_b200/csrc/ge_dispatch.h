// ge_dispatch.h -- non-template entry points of the kernel families that live in their own translation
// units (so that the families compile in parallel); called by ge_api.cu only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// 3-D: which of the two kernels of a level goes first and on which stream (ge_stream3d.cuh stream3d_launch)
#ifndef GE_S3D_MODE
#define GE_S3D_MODE 0
#endif

namespace ge {

// 2-D strip kernels (ge_strip2d.cu).  dtype: 0 = f32, 1 = f64 (ge_dtype).  coop: 0 = a warp per strip
// (ge2d_strip_kernel), 4 / 8 = that many warps of a CTA share one strip (ge2d_strip_coop_kernel).
// `configured`: the caller's per-plan flag for the function attributes of the instantiation last used.
cudaError_t strip2d_dispatch(int dtype, int tb, int coop, const void* uin, void* uout, int64_t nx, int64_t ny,
                             const void* coef, int hp, bool& configured, cudaStream_t s);
int strip2d_columns_per_lane(int dtype);                       // C of the instantiations for that dtype
bool strip2d_tb_compiled(int tb);                              // 4, 6, 8
bool strip2d_coop_compiled(int dtype, int tb, int coop);
// valid output columns per strip and columns a strip loads, for ge_plan_info
void strip2d_tile(int dtype, int tb, int coop, int64_t nx, int64_t ny, int hp, int* valid, int* loaded);

// Register-resident blocked kernel for sub-domain length k >= 2 (ge_unit_k.cu): `levels` <= tb levels from a level of
// phase `phase`; the two ends of the rod are NOT valid afterwards (the caller recomputes them).
bool unit_k_compiled(int dtype, int k);
int unit_k_valid_lanes(int k, int tb);            // units a tile of 256 lanes delivers (<= 0: tb too large)
cudaError_t unit_k_dispatch(int dtype, int k, const void* uin, void* uout, int64_t nx, int64_t batch, const void* coef,
                            int tb, int phase, int levels, cudaStream_t s);

// 3-D per-level kernels (ge_stream3d.cu).  form 0: a thread per group (ge3d_level_kernel); form 1: the streaming
// kernel for the deep groups + the shell kernel for the outermost layer (two launches; the shell on the stream
// `aux` between the events ev_in / ev_out when all three are given).
cudaError_t level3d_dispatch(int dtype, int form, const void* uin, void* uout, int64_t nx, int64_t ny, int64_t nz,
                             const void* coef, int phase, int sm_count, cudaStream_t s, int* launches,
                             cudaStream_t aux = nullptr, cudaEvent_t ev_in = nullptr, cudaEvent_t ev_out = nullptr);

}  // namespace ge
