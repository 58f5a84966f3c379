// Device helpers of the exterior field (eq. 2, eq. 6, eq. 7), shared by scw_exterior.cu and the fused exterior-image
// kernel of scw_tc_synth.cu.
#pragma once
#include <cuda_runtime.h>

namespace scw {

// eq. 2 with the branch moved to Im >= 0 (Re >= 0 on the real axis); stable complex square root in fp64.
__device__ __forceinline__ double2 ext_sz(double n_re, double n_im, double sx, double sy)
{
    const double a = n_re * n_re - n_im * n_im - (sx * sx + sy * sy);
    double b = 2.0 * n_re * n_im;
    if (b == 0.0) b = 0.0;                                  // clears a negative zero
    const double r = hypot(a, b);
    double re, im;
    if (r == 0.0) return make_double2(0.0, 0.0);
    if (a >= 0.0) {
        re = sqrt(0.5 * (r + a));
        im = b / (2.0 * re);
    } else {
        im = sqrt(0.5 * (r - a));
        re = b / (2.0 * im);
    }
    if (im < 0.0 || (im == 0.0 && re < 0.0)) { re = -re; im = -im; }
    return make_double2(re, im);
}

// G(gamma, zref, z) = exp(i 2 pi gamma (z - zref) / lambda): phase in turns reduced exactly, fp64 throughout
__device__ __forceinline__ double2 ext_green(double2 g, double dz_over_lambda)
{
    double t = g.x * dz_over_lambda;
    t -= rint(t);
    double s, c;
    sincospi(2.0 * t, &s, &c);
    const double a = exp(-6.283185307179586476925 * g.y * dz_over_lambda);
    return make_double2(a * c, a * s);
}

__device__ __forceinline__ void ext_freq(int U, int Vn, int m, double lam_over_X, double lam_over_Y, double& sx, double& sy)
{
    const int v = m / U, u = m - v * U;                     // eq. 6 index map, u fastest
    sx = (double)(u - U / 2) * lam_over_X;
    sy = (double)(v - Vn / 2) * lam_over_Y;
}

}  // namespace scw
