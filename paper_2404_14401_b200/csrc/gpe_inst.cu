// gpe_inst.cu -- one translation unit per (dtype, N): compile with
//   -DGPE_T=float|double -DGPE_N=<64..2048> -DGPE_TAG=f|d
#include "gpe_pair.cuh"
#include "gpe_chip.cuh"
#include "gpe_dispatch.h"

#define GPE_CAT3_(a, b, c) a##b##_##c
#define GPE_CAT3(a, b, c) GPE_CAT3_(a, b, c)

namespace gpe {
template <typename T, int N, bool ON = (sizeof(T) == 4 && N >= 128)> struct PairOps {
    static constexpr decltype(Ops<T>::p_row_fwd) row_fwd = nullptr;
    static constexpr decltype(Ops<T>::p_row_inv) row_inv = nullptr;
    static constexpr decltype(Ops<T>::p_col) col = nullptr;
    static constexpr decltype(Ops<T>::p_row_ca) row_ca = nullptr;
    static constexpr int rpc = 0;
    static constexpr int cpw = 0;
};
template <int N> struct PairOps<float, N, true> {
    static constexpr auto row_fwd = &LaunchP<N>::row_fwd;
    static constexpr auto row_inv = &LaunchP<N>::row_inv;
    static constexpr auto col = &LaunchP<N>::col;
    static constexpr auto row_ca = &LaunchP<N>::row_ca;
    static constexpr int rpc = RowGeomP<N>::RPC;
    static constexpr int cpw = ColGeomP<N>::CPW;
};
template <typename T, int N, bool ON = (N <= 256)> struct ChipOps {
    static constexpr decltype(Ops<T>::chip) run = nullptr;
    static constexpr decltype(Ops<T>::chip_available) available = nullptr;
};
template <typename T, int N> struct ChipOps<T, N, true> {
    static constexpr auto run = &LaunchChip<T, N>::run;
    static constexpr auto available = &LaunchChip<T, N>::available;
};
extern const Ops<GPE_T> GPE_CAT3(ops_, GPE_TAG, GPE_N) = {
    &Launch<GPE_T, GPE_N>::row_fwd,
    &Launch<GPE_T, GPE_N>::row_inv,
    &Launch<GPE_T, GPE_N>::col,
    RowGeom<GPE_N>::RPC,
    PairOps<GPE_T, GPE_N>::row_fwd,
    PairOps<GPE_T, GPE_N>::row_inv,
    PairOps<GPE_T, GPE_N>::col,
    PairOps<GPE_T, GPE_N>::rpc,
    &Launch<GPE_T, GPE_N>::row_ca,
    PairOps<GPE_T, GPE_N>::row_ca,
    ChipOps<GPE_T, GPE_N>::run,
    ChipOps<GPE_T, GPE_N>::available,
    ColGeom<GPE_T, GPE_N>::W,
    PairOps<GPE_T, GPE_N>::cpw,
};
}  // namespace gpe
