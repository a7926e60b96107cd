// pair64.h -- the pair interaction in IEEE double precision, shared by force64.cu (full-double
// pair loop) and fused.cu (predict-inside-the-loop kernel for a handful of active particles).
// Formulas: DESIGN.md R2 (force law), R5/R6 (self pair and coincident pairs contribute nothing).
#pragma once
#include "nb_internal.h"

namespace nb {

// 1/sqrt(s) to fp64 rounding: hardware approximation on the fp32-rounded argument + 2 Newton steps.
// Valid for s inside the normal fp32 range [S_MIN, ~3.4e38]: below it the fp32 argument would be
// flushed to zero (rsqrt = inf, NaN after the Newton steps), so pair64 treats s < S_MIN as s = 0
// (coincident, contributes nothing, R6); above it the approximation returns 0 (out of range,
// contributes nothing).  In length units: pairs closer than 1.1e-19 or farther than 1.8e19.
constexpr double S_MIN = 1.1754943508222875e-38;      // FLT_MIN
__device__ __forceinline__ double rsqrt64(double s)
{
    float y0;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(__double2float_rn(s)));
    double y = (double)y0;
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double e = fma(-(s * y), y, 1.0);      // 1 - s y^2
        y = fma(0.5 * y, e, y);
    }
    return y;
}

struct Acc64 {
    double ax, ay, az, jx, jy, jz, p;
};

template <bool JERK>
__device__ __forceinline__ void pair64(const double* xi, Acc64& A, double xj, double yj, double zj,
                                       double vxj, double vyj, double vzj, double mj, double e2, bool skip)
{
    const double dx = xj - xi[0], dy = yj - xi[1], dz = zj - xi[2];
    const double s = fma(dz, dz, fma(dy, dy, fma(dx, dx, e2)));
    double y = rsqrt64(s);
    y = (skip || !(s >= S_MIN)) ? 0.0 : y;             // self pair (R5) or coincident with eps2 = 0 (R6)
    const double y2 = y * y;
    const double mr = mj * y;
    const double mr3 = mr * y2;
    A.p -= mr;
    A.ax = fma(mr3, dx, A.ax);
    A.ay = fma(mr3, dy, A.ay);
    A.az = fma(mr3, dz, A.az);
    if (JERK) {
        const double wx = vxj - xi[3], wy = vyj - xi[4], wz = vzj - xi[5];
        const double rv = fma(dz, wz, fma(dy, wy, dx * wx));
        const double al = (y2 * -3.0) * rv;
        A.jx = fma(mr3, fma(al, dx, wx), A.jx);
        A.jy = fma(mr3, fma(al, dy, wy), A.jy);
        A.jz = fma(mr3, fma(al, dz, wz), A.jz);
    }
}

}  // namespace nb
