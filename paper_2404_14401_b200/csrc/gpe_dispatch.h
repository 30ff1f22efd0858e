// gpe_dispatch.h -- table of per-(dtype, N) launchers.  Each (T, N) pair is compiled in its own
// translation unit (gpe_inst.cu with -DGPE_T/-DGPE_N/-DGPE_TAG) so the build parallelises.
#pragma once
#include "gpe_fft.cuh"
#include "gpe_types.h"

namespace gpe {

template <typename T> struct Ops {
    using A = StepArgs<T, cx<T>>;
    cudaError_t (*row_fwd)(const A &, bool imag, cudaStream_t);            // ny == N
    cudaError_t (*row_inv)(const A &, bool imag, cudaStream_t);            // ny == N
    cudaError_t (*col)(const A &, bool imag, int mode, cudaStream_t);      // nx == N
    int rows_per_cta;
    // paired complex64 hot path (gpe_pair.cuh); null when not built for this (dtype, N)
    cudaError_t (*p_row_fwd)(const A &, bool imag, cudaStream_t);
    cudaError_t (*p_row_inv)(const A &, bool imag, cudaStream_t);
    cudaError_t (*p_col)(const A &, bool imag, cudaStream_t);
    int p_rows_per_cta;
    // pass C of step n fused with pass A of step n+1 (the 2-pass form): both kernel families
    cudaError_t (*row_ca)(const A &, bool imag, cudaStream_t);
    cudaError_t (*p_row_ca)(const A &, bool imag, cudaStream_t);
    // small square grids: all steps of a call in one cluster kernel (gpe_chip.cuh); null above 256
    cudaError_t (*chip)(const A &, bool imag, long n_steps, cudaStream_t);
    bool (*chip_available)();
    int cols_per_cta, p_colpairs_per_cta;   // columns (column pairs) per CTA of pass B: number of its partial sums
};

#define GPE_DECL_OPS(N)                    \
    extern const Ops<float> ops_f_##N;     \
    extern const Ops<double> ops_d_##N;
GPE_DECL_OPS(64)
GPE_DECL_OPS(128)
GPE_DECL_OPS(256)
GPE_DECL_OPS(512)
GPE_DECL_OPS(1024)
GPE_DECL_OPS(2048)
#undef GPE_DECL_OPS

template <typename T> inline const Ops<T> *get_ops(int n);
template <> inline const Ops<float> *get_ops<float>(int n) {
    switch (n) {
    case 64: return &ops_f_64;   case 128: return &ops_f_128;   case 256: return &ops_f_256;
    case 512: return &ops_f_512; case 1024: return &ops_f_1024; case 2048: return &ops_f_2048;
    }
    return nullptr;
}
template <> inline const Ops<double> *get_ops<double>(int n) {
    switch (n) {
    case 64: return &ops_d_64;   case 128: return &ops_d_128;   case 256: return &ops_d_256;
    case 512: return &ops_d_512; case 1024: return &ops_d_1024; case 2048: return &ops_d_2048;
    }
    return nullptr;
}

}  // namespace gpe
