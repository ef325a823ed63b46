// mg_coarse_kernel.cuh -- single persistent CTA for the coarse levels (placeholder)
#pragma once
#include "mg_common.cuh"
namespace mg {
constexpr int kCoarseMaxLevels = 4;
struct CoarseArgs {
    int nlev;
    int n[kCoarseMaxLevels][3];
    double h2[kCoarseMaxLevels], ih2[kCoarseMaxLevels];
    const double *bx[kCoarseMaxLevels], *by[kCoarseMaxLevels], *bz[kCoarseMaxLevels];
    int bc[3];
    int nu1, nu2, coarse_sweeps;
    const double *f;
    double *p;
};
inline bool coarse_cta_fits(int (*)[3], int) { return false; }
inline int launch_coarse_cta(const CoarseArgs &, cudaStream_t) { return -1; }
} // namespace mg
