// The cheb_step_kernel instantiations, one translation unit per Mode (compiled with
// -DGPUQT_TU_MODE=0..3, in parallel, by paper_1705_01387_b200/build.py), plus the dispatcher in the
// translation unit of mode 0.
#define GPUQT_STEP_TU
#include "kernels.cuh"

#ifndef GPUQT_TU_MODE
#error "compile with -DGPUQT_TU_MODE=<0..3>"
#endif

namespace gpuqt {

namespace {
template <int MODE, int BB, int KK>
void* step_fn(int hop) {
    if (KK > 0 && hop == kHopConst16)      // 16-bit columns exist for the unrolled uniform tables only
        return (void*)cheb_step_kernel<BB, (KK > 0 ? KK : 3), kHopConst16, MODE>;
    if (KK > 0 && hop == kHopConst16P) return (void*)cheb_step_kernel<BB, (KK > 0 ? KK : 3), kHopConst16P, MODE>;
    if (KK > 0 && hop == kHopStencil)      // pattern-dictionary columns: unrolled uniform tables only
        return (void*)cheb_step_kernel<BB, (KK > 0 ? KK : 3), kHopStencil, MODE>;
    return hop == kHopComplex ? (void*)cheb_step_kernel<BB, KK, kHopComplex, MODE>
           : hop == kHopConst ? (void*)cheb_step_kernel<BB, KK, kHopConst, MODE>
                              : (void*)cheb_step_kernel<BB, KK, kHopReal, MODE>;
}
template <int MODE, int BB>
void* step_fn_k(int kt, int hop) {
    switch (kt) {
    case 2: return step_fn<MODE, BB, 2>(hop);
    case 3: return step_fn<MODE, BB, 3>(hop);
    case 4: return step_fn<MODE, BB, 4>(hop);
    case 6: return step_fn<MODE, BB, 6>(hop);
    default: return step_fn<MODE, BB, 0>(hop);
    }
}
template <int MODE>
void* step_fn_b(int B, int kt, int hop) {
    switch (B) {
    case 1: return step_fn_k<MODE, 1>(kt, hop);
    case 2: return step_fn_k<MODE, 2>(kt, hop);
    case 4: return step_fn_k<MODE, 4>(kt, hop);
    default: return step_fn_k<MODE, 8>(kt, hop);
    }
}
}  // namespace

#if GPUQT_TU_MODE == 0
void* step_kernel_fn_doubling(int B, int kt, int hop) { return step_fn_b<kModeDoubling>(B, kt, hop); }
void* step_kernel_fn_left(int B, int kt, int hop);
void* step_kernel_fn_evolve(int B, int kt, int hop);
void* step_kernel_fn_evolve_msd(int B, int kt, int hop);
// host address of the cheb_step_kernel instantiation for (mode, B, unrolled width or 0, Hop variant)
void* step_kernel_fn(int mode, int B, int kt, int hop) {
    switch (mode) {
    case kModeDoubling: return step_kernel_fn_doubling(B, kt, hop);
    case kModeLeft: return step_kernel_fn_left(B, kt, hop);
    case kModeEvolve: return step_kernel_fn_evolve(B, kt, hop);
    default: return step_kernel_fn_evolve_msd(B, kt, hop);
    }
}
#elif GPUQT_TU_MODE == 1
void* step_kernel_fn_left(int B, int kt, int hop) { return step_fn_b<kModeLeft>(B, kt, hop); }
#elif GPUQT_TU_MODE == 2
void* step_kernel_fn_evolve(int B, int kt, int hop) { return step_fn_b<kModeEvolve>(B, kt, hop); }
#else
void* step_kernel_fn_evolve_msd(int B, int kt, int hop) { return step_fn_b<kModeEvolveMsd>(B, kt, hop); }
#endif

}  // namespace gpuqt
