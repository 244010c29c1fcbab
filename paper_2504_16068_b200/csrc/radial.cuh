// radial.cuh -- Bessel radial basis with polynomial cutoff (reading A8), shared by misc.cu (radial_forward /
// radial_backward) and env_kernels.cuh (the fused geometry kernels).
#pragma once
#include <cuda_runtime.h>

namespace allegro {

constexpr int kMaxBasis = 16;
constexpr double kPiD = 3.14159265358979323846264338327950288;

// Bessel basis times polynomial cutoff and its derivative w.r.t. |r|, evaluated in double for either dtype
// (the embedding is "largely in double-precision"); cost is per edge, not per channel.
//   x = r/rc, B_b = sqrt(2/rc) sin(b pi x)/r, u = 1 - 28x^6 + 48x^7 - 21x^8
// One sincos per edge; sin(b t), cos(b t) for b >= 2 by the angle-addition recurrence (error growth ~ b eps).
template <bool WANT_D>
__device__ __forceinline__ void radial_basis(double r, double rc, int nb, double* Bu, double* dBu) {
    const double x = r / rc;
    const double x2 = x * x, x5 = x2 * x2 * x, x6 = x5 * x, x7 = x6 * x, x8 = x7 * x;
    double u = 1.0 - 28.0 * x6 + 48.0 * x7 - 21.0 * x8;
    double du = (-168.0 * x5 + 336.0 * x6 - 168.0 * x7) / rc;
    if (x >= 1.0) { u = 0.0; du = 0.0; }
    const double pre = sqrt(2.0 / rc), ir = 1.0 / r;
    double s1, c1;
    sincospi(x, &s1, &c1);
    double sn = s1, cs = c1;
    for (int b = 1; b <= nb; ++b) {
        const double B = pre * sn * ir;
        Bu[b - 1] = B * u;
        if (WANT_D) {
            const double k = b * kPiD / rc;
            const double dB = pre * (k * cs * ir - sn * ir * ir);
            dBu[b - 1] = dB * u + B * du;
        }
        const double sn2 = sn * c1 + cs * s1;
        cs = cs * c1 - sn * s1;
        sn = sn2;
    }
}

}  // namespace allegro
