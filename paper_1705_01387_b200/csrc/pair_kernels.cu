// Second translation unit of libgpuqt.so: the instantiations of the opt-in two-steps-per-launch
// kernel (cheb_pair_kernel), compiled in parallel with gpuqt.cu to halve the build time.
#define GPUQT_PAIR_TU
#include "kernels.cuh"

namespace gpuqt {

namespace {
template <int MODE, int BB, int KK>
void* pair_fn(int hop) {
    if (KK > 0 && hop == kHopConst16) return (void*)cheb_pair_kernel<BB, (KK > 0 ? KK : 3), kHopConst16, MODE>;
    return hop == kHopComplex ? (void*)cheb_pair_kernel<BB, KK, kHopComplex, MODE>
           : hop == kHopConst ? (void*)cheb_pair_kernel<BB, KK, kHopConst, MODE>
                              : (void*)cheb_pair_kernel<BB, KK, kHopReal, MODE>;
}
template <int MODE, int BB>
void* pair_fn_k(int kt, int hop) {
    switch (kt) {
    case 3: return pair_fn<MODE, BB, 3>(hop);
    case 4: return pair_fn<MODE, BB, 4>(hop);
    case 6: return pair_fn<MODE, BB, 6>(hop);
    default: return pair_fn<MODE, BB, 0>(hop);
    }
}
template <int MODE>
void* pair_fn_b(int B, int kt, int hop) {
    switch (B) {
    case 1: return pair_fn_k<MODE, 1>(kt, hop);
    case 2: return pair_fn_k<MODE, 2>(kt, hop);
    case 4: return pair_fn_k<MODE, 4>(kt, hop);
    default: return pair_fn_k<MODE, 8>(kt, hop);
    }
}
}  // namespace

// host address of the cheb_pair_kernel instantiation for (mode, B, unrolled width or 0, Hop variant)
void* pair_kernel_fn(int mode, int B, int kt, int hop) {
    switch (mode) {
    case kModeDoubling: return pair_fn_b<kModeDoubling>(B, kt, hop);
    case kModeLeft: return pair_fn_b<kModeLeft>(B, kt, hop);
    case kModeEvolve: return pair_fn_b<kModeEvolve>(B, kt, hop);
    default: return pair_fn_b<kModeEvolveMsd>(B, kt, hop);
    }
}

}  // namespace gpuqt
