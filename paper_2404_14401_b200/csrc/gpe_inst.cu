// gpe_inst.cu -- one translation unit per (dtype, N): compile with
//   -DGPE_T=float|double -DGPE_N=<64..2048> -DGPE_TAG=f|d
#include "gpe_kernels.cuh"
#include "gpe_dispatch.h"

#define GPE_CAT3_(a, b, c) a##b##_##c
#define GPE_CAT3(a, b, c) GPE_CAT3_(a, b, c)

namespace gpe {
extern const Ops<GPE_T> GPE_CAT3(ops_, GPE_TAG, GPE_N) = {
    &Launch<GPE_T, GPE_N>::row_fwd,
    &Launch<GPE_T, GPE_N>::row_inv,
    &Launch<GPE_T, GPE_N>::col,
    RowGeom<GPE_N>::RPC,
};
}  // namespace gpe
