// taps.cuh -- sample coordinates and Kaiser-Bessel tap weights, shared by every gridding kernel.
#pragma once
#include "radon_internal.h"

namespace radon {

// =====================================================================================
// Sample coordinates and Kaiser-Bessel weights (shared by gather and scatter so that the
// two kernels use bit-identical tap positions and weights: exact transposes)
// =====================================================================================
template <int W>
struct Taps {
    float wx[W], wy[W];
};

// Polar sample (a,k) -> fractional offsets of its first tap: delta = x0 - (gx - W/2) in [0,1).
// fp64 on purpose (an fp32 product G*j/n*cos loses 2.6e-5 at G = 4096).
// d = cs[a] = (G/n)(cos theta_a, sin theta_a).
template <int W>
__device__ __forceinline__ void sample_taps_dir(const double2 d, const KbPoly &kp,
                                                int k, int cd, double halfG, Taps<W> &tp)
{
    const double jj = (double)(k - cd);
    const double gx = fma(jj, d.x, halfG) - 0.5 * W;
    const double gy = fma(jj, d.y, halfG) - 0.5 * W;
    const float dx = (float)(ceil(gx) - gx);
    const float dy = (float)(ceil(gy) - gy);
    kb_poly_weights(kp, dx, tp.wx);
    kb_poly_weights(kp, dy, tp.wy);
}

}  // namespace radon
