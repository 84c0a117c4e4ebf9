// rt_fused_inst.cuh — the instantiations of k_substep_fused the launcher can select (rt_api.cu: launch_fused), as a list:
// X(part, HLL, THICK, CURVI, FEEDBACK, RUS, HASZ, VARFIX).  rt_fused_inst.cu instantiates the entries of one `part` per
// translation unit (the build compiles the parts side by side); rt_api.cu declares them all `extern template`.
#pragma once

#define RT_FUSED_PARTS 6
#define RT_FUSED_INSTANCES(X) \
    X(0, false, false, false, false, false, false, false) \
    X(1, false, false, false, false, false, false, true) \
    X(2, false, false, false, false, false, true, false) \
    X(3, false, false, false, false, false, true, true) \
    X(4, false, false, false, true, false, false, false) \
    X(5, false, false, false, true, false, false, true) \
    X(0, false, false, false, true, false, true, false) \
    X(1, false, false, false, true, false, true, true) \
    X(2, false, false, true, false, false, false, false) \
    X(3, false, false, true, false, false, false, true) \
    X(4, false, false, true, false, false, true, false) \
    X(5, false, false, true, false, false, true, true) \
    X(0, false, false, true, true, false, false, false) \
    X(1, false, false, true, true, false, false, true) \
    X(2, false, false, true, true, false, true, false) \
    X(3, false, false, true, true, false, true, true) \
    X(4, false, true, false, false, false, false, false) \
    X(5, false, true, false, false, false, false, true) \
    X(0, false, true, false, false, false, true, false) \
    X(1, false, true, false, false, false, true, true) \
    X(2, false, true, false, true, false, false, false) \
    X(3, false, true, false, true, false, false, true) \
    X(4, false, true, false, true, false, true, false) \
    X(5, false, true, false, true, false, true, true) \
    X(0, false, true, true, false, false, false, false) \
    X(1, false, true, true, false, false, false, true) \
    X(2, false, true, true, false, false, true, false) \
    X(3, false, true, true, false, false, true, true) \
    X(4, false, true, true, true, false, false, false) \
    X(5, false, true, true, true, false, false, true) \
    X(0, false, true, true, true, false, true, false) \
    X(1, false, true, true, true, false, true, true) \
    X(2, true, false, false, false, false, false, false) \
    X(3, true, false, false, false, false, false, true) \
    X(4, true, false, false, false, false, true, false) \
    X(5, true, false, false, false, false, true, true) \
    X(0, true, false, false, true, false, false, false) \
    X(1, true, false, false, true, false, false, true) \
    X(2, true, false, false, true, false, true, false) \
    X(3, true, false, false, true, false, true, true) \
    X(4, true, false, true, false, false, false, false) \
    X(5, true, false, true, false, false, false, true) \
    X(0, true, false, true, false, false, true, false) \
    X(1, true, false, true, false, false, true, true) \
    X(2, true, false, true, true, false, false, false) \
    X(3, true, false, true, true, false, false, true) \
    X(4, true, false, true, true, false, true, false) \
    X(5, true, false, true, true, false, true, true) \
    X(0, true, true, false, false, false, false, false) \
    X(1, true, true, false, false, false, false, true) \
    X(2, true, true, false, false, false, true, false) \
    X(3, true, true, false, false, false, true, true) \
    X(4, true, true, false, true, false, false, false) \
    X(5, true, true, false, true, false, false, true) \
    X(0, true, true, false, true, false, true, false) \
    X(1, true, true, false, true, false, true, true) \
    X(2, true, true, true, false, false, false, false) \
    X(3, true, true, true, false, false, false, true) \
    X(4, true, true, true, false, false, true, false) \
    X(5, true, true, true, false, false, true, true) \
    X(0, true, true, true, true, false, false, false) \
    X(1, true, true, true, true, false, false, true) \
    X(2, true, true, true, true, false, true, false) \
    X(3, true, true, true, true, false, true, true) \
    X(4, true, false, false, false, true, false, false) \
    X(5, true, false, false, false, true, true, false) \
    X(0, true, false, false, true, true, false, false) \
    X(1, true, false, false, true, true, true, false) \
    X(2, true, false, true, false, true, false, false) \
    X(3, true, false, true, false, true, true, false) \
    X(4, true, false, true, true, true, false, false) \
    X(5, true, false, true, true, true, true, false) \
    X(0, true, true, false, false, true, false, false) \
    X(1, true, true, false, false, true, true, false) \
    X(2, true, true, false, true, true, false, false) \
    X(3, true, true, false, true, true, true, false) \
    X(4, true, true, true, false, true, false, false) \
    X(5, true, true, true, false, true, true, false) \
    X(0, true, true, true, true, true, false, false) \
    X(1, true, true, true, true, true, true, false) 
