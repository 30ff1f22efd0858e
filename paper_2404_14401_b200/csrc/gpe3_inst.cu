// gpe3_inst.cu -- the 3-D passes of one (dtype, N): compile with -DGPE_T=float|double -DGPE_N=<64..512> -DGPE_TAG=f|d
#include "gpe3_kernels.cuh"

#define GPE_CAT3_(a, b, c) a##b##_##c
#define GPE_CAT3(a, b, c) GPE_CAT3_(a, b, c)

namespace gpe {
extern const Ops3<GPE_T> GPE_CAT3(ops3_, GPE_TAG, GPE_N) = {
    &Launch3<GPE_T, GPE_N>::row,
    &Launch3<GPE_T, GPE_N>::col,
};
}  // namespace gpe
