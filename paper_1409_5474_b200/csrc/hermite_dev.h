// hermite_dev.h -- device functions of the block-step layer shared by hermite.cu (one kernel per
// piece: nb_next_block, nb_correct) and steps.cu (all pieces in one persistent kernel: nb_steps), so
// that both take every decision with the same arithmetic.  Readings R12, R18..R21 of DESIGN.md.
#pragma once
#include "nb_internal.h"

namespace nb {

// order-preserving map double -> uint64 (so that atomicMin on integers is a min on doubles)
__device__ __forceinline__ unsigned long long key_of(double x)
{
    const long long b = __double_as_longlong(x);
    return (unsigned long long)(b ^ ((b >> 63) | (long long)0x8000000000000000ull));
}
__device__ __forceinline__ double of_key(unsigned long long k)
{
    const long long b = (long long)k;
    return __longlong_as_double(b ^ ((~b >> 63) | (long long)0x8000000000000000ull));
}

__device__ __forceinline__ double norm3(double x, double y, double z) { return sqrt(x * x + y * y + z * z); }

// Is t1 a multiple of p (p > 0)?  Steps are powers of two, so t1 / p is exact and the answer is
// "the quotient is an integer" -- the same truth value as fmod(t1, p) == 0 without its long loop;
// any other p (a step the caller set by hand) takes fmod.
__device__ __forceinline__ bool is_multiple(double t1, double p)
{
    const long long pb = __double_as_longlong(p);
    const int e = (int)(pb >> 52);            // biased exponent (p > 0: no sign bit)
    if ((pb & 0x000fffffffffffffll) == 0 && e > 523 && e < 1523) {      // 2^-500 < p = 2^k < 2^500
        const double q = t1 * __longlong_as_double(0x7fe0000000000000ll - pb);   // t1 * 2^-k, exact
        return q == rint(q) && fabs(q) < __longlong_as_double(0x7ff0000000000000ll);
    }
    return fmod(t1, p) == 0.0;
}

// R20: new power-of-two step after a step of d_old that ended at t1, given the wanted step w
__device__ __forceinline__ double block_rule(double d, double w, double t1, double dt_min, double dt_max)
{
    d = d < dt_min ? dt_min : d;      // a step that was never set (0) must not stay below the grid
    if (w < d) {
        while (d > w && d * 0.5 >= dt_min) d *= 0.5;
    } else if (w >= 2.0 * d && 2.0 * d <= dt_max && is_multiple(t1, 2.0 * d)) {
        d *= 2.0;
    }
    return d;
}

// The stored state of one particle that the corrector reads.
struct Stored {
    double x[3], v[3], a[3], j[3], t, dt;
};
__device__ __forceinline__ Stored load_stored(const StorePtrs& st, const double* __restrict__ dts, int64_t i)
{
    Stored s;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        s.x[c] = st.f[F_X + c][i];
        s.v[c] = st.f[F_VX + c][i];
        s.a[c] = st.f[F_AX + c][i];
        s.j[c] = st.f[F_JX + c][i];
    }
    s.t = st.f[F_T][i];
    s.dt = dts[i];
    return s;
}

// R12 + R18 + R19 + R20 for particle i, whose stored state is s0 and whose forces at t1 are (a1, j1):
// corrector, interpolated derivatives, Aarseth step, block rule; writes x1, v1, a1, j1, t = t1 and the
// new step into the j-store and returns the new step.  A zero step (h = 0: steps never set) or a NaN
// time would make a2, a3 NaN: the particle is left alone, bit 1 of the error latch is set (nb_sync ->
// NB_ERR_STATE) and the old step is returned.
__device__ __forceinline__ double correct_stored(const StorePtrs& st, double* __restrict__ dts, int64_t i,
                                                 const Stored& s0, double t1, const double* a1, const double* j1,
                                                 double eta, double dt_min, double dt_max, int* err)
{
    const double h = t1 - s0.t;
    if (!(h != 0.0)) {
        atomicOr(err, 2);
        return s0.dt;
    }
    double a2[3], a3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double x0 = s0.x[c], v0 = s0.v[c], a0 = s0.a[c], j0 = s0.j[c];
        const double v1 = v0 + (a0 + a1[c]) * (h / 2.0) + (j0 - j1[c]) * (h * h / 12.0);
        const double x1 = x0 + (v0 + v1) * (h / 2.0) + (a0 - a1[c]) * (h * h / 12.0);
        const double a2_0 = (-6.0 * (a0 - a1[c]) - h * (4.0 * j0 + 2.0 * j1[c])) / (h * h);
        a3[c] = (12.0 * (a0 - a1[c]) + 6.0 * h * (j0 + j1[c])) / (h * h * h);
        a2[c] = a2_0 + h * a3[c];
        st.f[F_X + c][i] = x1;
        st.f[F_VX + c][i] = v1;
        st.f[F_AX + c][i] = a1[c];
        st.f[F_JX + c][i] = j1[c];
    }
    const double na = norm3(a1[0], a1[1], a1[2]), nj = norm3(j1[0], j1[1], j1[2]);
    const double n2 = norm3(a2[0], a2[1], a2[2]), n3 = norm3(a3[0], a3[1], a3[2]);
    const double num = eta * (na * n2 + nj * nj), den = nj * n3 + n2 * n2;
    const double want = den > 0.0 ? sqrt(num / den) : __longlong_as_double(0x7ff0000000000000ll);
    const double d = block_rule(s0.dt, want, t1, dt_min, dt_max);
    st.f[F_T][i] = t1;
    dts[i] = d;
    return d;
}

__device__ __forceinline__ void correct_one(const StorePtrs& st, double* __restrict__ dts, int64_t i, double t1,
                                            const double* a1, const double* j1, double eta, double dt_min,
                                            double dt_max, int* err)
{
    const Stored s0 = load_stored(st, dts, i);
    correct_stored(st, dts, i, s0, t1, a1, j1, eta, dt_min, dt_max, err);
}

}  // namespace nb
