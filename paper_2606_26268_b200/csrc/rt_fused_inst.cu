// rt_fused_inst.cu — explicit instantiations of k_substep_fused, one part per translation unit:
//   nvcc -DRT_FUSED_PART=<0 .. RT_FUSED_PARTS-1> -c rt_fused_inst.cu
// (112 instantiations of a 128-register kernel take minutes in one unit; the parts compile side by side).
#include "rt_kernels_fused.cuh"
#include "rt_fused_inst.cuh"

#ifndef RT_FUSED_PART
#error "compile with -DRT_FUSED_PART=<n>"
#endif

namespace rtm1 {
#define RT_X(P, A, B, C_, D_, E_, F_, G_) RT_X_##P(A, B, C_, D_, E_, F_, G_)
#define RT_INST(A, B, C_, D_, E_, F_, G_)                                                                                  \
    template __global__ void k_substep_fused<A, B, C_, D_, E_, F_, G_>(const __grid_constant__ GridDev, const __grid_constant__ ParamsDev, const __grid_constant__ OpacDev, \
        const __grid_constant__ OpacDev, const __grid_constant__ OpacDev, const __grid_constant__ FusedArgs, const __grid_constant__ FusedMaps, int);
#define RT_SKIP(A, B, C_, D_, E_, F_, G_)
#if RT_FUSED_PART == 0
#define RT_X_0 RT_INST
#else
#define RT_X_0 RT_SKIP
#endif
#if RT_FUSED_PART == 1
#define RT_X_1 RT_INST
#else
#define RT_X_1 RT_SKIP
#endif
#if RT_FUSED_PART == 2
#define RT_X_2 RT_INST
#else
#define RT_X_2 RT_SKIP
#endif
#if RT_FUSED_PART == 3
#define RT_X_3 RT_INST
#else
#define RT_X_3 RT_SKIP
#endif
#if RT_FUSED_PART == 4
#define RT_X_4 RT_INST
#else
#define RT_X_4 RT_SKIP
#endif
#if RT_FUSED_PART == 5
#define RT_X_5 RT_INST
#else
#define RT_X_5 RT_SKIP
#endif
RT_FUSED_INSTANCES(RT_X)
}  // namespace rtm1
