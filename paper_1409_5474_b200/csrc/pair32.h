// pair32.h -- the mixed-precision pair interaction and the reduction of partial forces, shared by the
// tile-streaming pair kernels (force.cu) and the direct few-i kernel (direct.cu).  Two consecutive j
// form the two lanes of every packed FP32 instruction (fma/add/mul .f32x2); position differences
// are two-float sums (>= 48 bits), everything after is fp32 (R2, R17).
#pragma once
#include "nb_internal.h"
#include "tma.h"

namespace nb {

struct IPart {            // one i-particle, negated and duplicated over both f32x2 lanes
    float2 nxh, nyh, nzh, nxl, nyl, nzl, nvx, nvy, nvz;
};
struct Acc32 {            // per-tile fp32 sums, lane 0 = even j, lane 1 = odd j
    float2 ax, ay, az, jx, jy, jz, p;
};

__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }

// One i against one pair of j's: 13 FADD2 + 14 FFMA2 + 6 FMUL2 + 2 MUFU (R2, R17).
// GUARD (calls with eps2 below EPS2_GUARD, eps2 == 0 among them): a pair whose s does not exceed
// eps2 -- r = 0 to fp32 precision: the self pair, or two particles at one place (R5, R6) -- gets
// rinv = 0 and so contributes nothing; the compare and select run on the ALU pipe, beside the FP32
// pipe the loop is bound by.
template <bool GUARD>
__device__ __forceinline__ void pair2(const IPart& I, Acc32& A, float2 xh, float2 yh, float2 zh,
                                      float2 xl, float2 yl, float2 zl, float2 vx, float2 vy,
                                      float2 vz, float2 m, float2 eps2, float2 m3)
{
    const float2 dx = __fadd2_rn(__fadd2_rn(xh, I.nxh), __fadd2_rn(xl, I.nxl));
    const float2 dy = __fadd2_rn(__fadd2_rn(yh, I.nyh), __fadd2_rn(yl, I.nyl));
    const float2 dz = __fadd2_rn(__fadd2_rn(zh, I.nzh), __fadd2_rn(zl, I.nzl));
    const float2 wx = __fadd2_rn(vx, I.nvx);
    const float2 wy = __fadd2_rn(vy, I.nvy);
    const float2 wz = __fadd2_rn(vz, I.nvz);
    float2 r2 = __ffma2_rn(dx, dx, eps2);
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dz, dz, r2);
    float2 rinv;
    rinv.x = rsqrt_fast(r2.x);
    rinv.y = rsqrt_fast(r2.y);
    if (GUARD) {
        rinv.x = r2.x > eps2.x ? rinv.x : 0.0f;
        rinv.y = r2.y > eps2.x ? rinv.y : 0.0f;
    }
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 mr = __fmul2_rn(m, rinv);
    const float2 mr3 = __fmul2_rn(mr, rinv2);
    float2 rv = __fmul2_rn(dx, wx);
    rv = __ffma2_rn(dy, wy, rv);
    rv = __ffma2_rn(dz, wz, rv);
    const float2 al = __fmul2_rn(__fmul2_rn(rinv2, m3), rv);      // -3 (r.w) / s
    A.p = __fadd2_rn(A.p, mr);
    A.ax = __ffma2_rn(mr3, dx, A.ax);
    A.ay = __ffma2_rn(mr3, dy, A.ay);
    A.az = __ffma2_rn(mr3, dz, A.az);
    A.jx = __ffma2_rn(mr3, __ffma2_rn(al, dx, wx), A.jx);
    A.jy = __ffma2_rn(mr3, __ffma2_rn(al, dy, wy), A.jy);
    A.jz = __ffma2_rn(mr3, __ffma2_rn(al, dz, wz), A.jz);
}

// acc + pot only (the kick of a bridge between two systems):
// 9 FADD2 + 6 FFMA2 + 3 FMUL2 + 1 FADD2 = 19 lane-ops per interaction, no velocities.
template <bool GUARD>
__device__ __forceinline__ void pair2_acc(const IPart& I, Acc32& A, float2 xh, float2 yh, float2 zh,
                                          float2 xl, float2 yl, float2 zl, float2 m, float2 eps2)
{
    const float2 dx = __fadd2_rn(__fadd2_rn(xh, I.nxh), __fadd2_rn(xl, I.nxl));
    const float2 dy = __fadd2_rn(__fadd2_rn(yh, I.nyh), __fadd2_rn(yl, I.nyl));
    const float2 dz = __fadd2_rn(__fadd2_rn(zh, I.nzh), __fadd2_rn(zl, I.nzl));
    float2 r2 = __ffma2_rn(dx, dx, eps2);
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dz, dz, r2);
    float2 rinv;
    rinv.x = rsqrt_fast(r2.x);
    rinv.y = rsqrt_fast(r2.y);
    if (GUARD) {
        rinv.x = r2.x > eps2.x ? rinv.x : 0.0f;
        rinv.y = r2.y > eps2.x ? rinv.y : 0.0f;
    }
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 mr = __fmul2_rn(m, rinv);
    const float2 mr3 = __fmul2_rn(mr, rinv2);
    A.p = __fadd2_rn(A.p, mr);
    A.ax = __ffma2_rn(mr3, dx, A.ax);
    A.ay = __ffma2_rn(mr3, dy, A.ay);
    A.az = __ffma2_rn(mr3, dz, A.az);
}

// One i against a quad of consecutive j (four floats of each tile array): two packed pairs.
template <bool JERK, bool GUARD>
__device__ __forceinline__ void quad(const IPart& I, Acc32& A, const float4* f, float2 eps2, float2 m3)
{
    if (!JERK) {
        pair2_acc<GUARD>(I, A, make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y),
                         make_float2(f[2].x, f[2].y), make_float2(f[3].x, f[3].y),
                         make_float2(f[4].x, f[4].y), make_float2(f[5].x, f[5].y),
                         make_float2(f[9].x, f[9].y), eps2);
        pair2_acc<GUARD>(I, A, make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w),
                         make_float2(f[2].z, f[2].w), make_float2(f[3].z, f[3].w),
                         make_float2(f[4].z, f[4].w), make_float2(f[5].z, f[5].w),
                         make_float2(f[9].z, f[9].w), eps2);
        return;
    }
    pair2<GUARD>(I, A, make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y),
                 make_float2(f[2].x, f[2].y), make_float2(f[3].x, f[3].y), make_float2(f[4].x, f[4].y),
                 make_float2(f[5].x, f[5].y), make_float2(f[6].x, f[6].y), make_float2(f[7].x, f[7].y),
                 make_float2(f[8].x, f[8].y), make_float2(f[9].x, f[9].y), eps2, m3);
    pair2<GUARD>(I, A, make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w),
                 make_float2(f[2].z, f[2].w), make_float2(f[3].z, f[3].w), make_float2(f[4].z, f[4].w),
                 make_float2(f[5].z, f[5].w), make_float2(f[6].z, f[6].w), make_float2(f[7].z, f[7].w),
                 make_float2(f[8].z, f[8].w), make_float2(f[9].z, f[9].w), eps2, m3);
}

template <bool JERK>
__device__ __forceinline__ void load_quad(float4* f, const float* T, int p)
{
#pragma unroll
    for (int c = 0; c < 10; ++c)
        if (JERK || c < 6 || c == 9) f[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
}

// Masked scalar pair, j given by value: a skipped pair gets rinv = 0, i.e. contributes nothing.
__device__ __forceinline__ void pair1_vals(const IPart& I, Acc32& A, float xh, float yh, float zh, float xl,
                                           float yl, float zl, float vx, float vy, float vz, float m, bool skip_pair,
                                           float eps2)
{
    const float dx = (xh + I.nxh.x) + (xl + I.nxl.x);
    const float dy = (yh + I.nyh.x) + (yl + I.nyl.x);
    const float dz = (zh + I.nzh.x) + (zl + I.nzl.x);
    const float wx = vx + I.nvx.x;
    const float wy = vy + I.nvy.x;
    const float wz = vz + I.nvz.x;
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
    const bool skip = skip_pair || !(r2 > 0.0f);
    const float rinv = skip ? 0.0f : rsqrt_fast(r2);
    const float rinv2 = rinv * rinv;
    const float mr = m * rinv;
    const float mr3 = mr * rinv2;
    const float rv = fmaf(dz, wz, fmaf(dy, wy, dx * wx));
    const float al = (rinv2 * -3.0f) * rv;
    A.p.x += mr;
    A.ax.x = fmaf(mr3, dx, A.ax.x);
    A.ay.x = fmaf(mr3, dy, A.ay.x);
    A.az.x = fmaf(mr3, dz, A.az.x);
    A.jx.x = fmaf(mr3, fmaf(al, dx, wx), A.jx.x);
    A.jy.x = fmaf(mr3, fmaf(al, dy, wy), A.jy.x);
    A.jz.x = fmaf(mr3, fmaf(al, dz, wz), A.jz.x);
}

// Masked scalar pair for the rare tiles that hold the i-particle itself, a flagged partner of a
// flagged i, or when eps2 == 0 (R5, R6, R7); j = entry p of the tile T in shared memory.
__device__ __forceinline__ void pair1_masked(const IPart& I, Acc32& A, const float* T, int p,
                                             bool skip_self, bool iflag, float eps2)
{
    const bool jflag = (__float_as_uint(T[P_FLAG * TJ + p]) & 1u) != 0;
    pair1_vals(I, A, T[P_XH * TJ + p], T[P_YH * TJ + p], T[P_ZH * TJ + p], T[P_XL * TJ + p], T[P_YL * TJ + p],
               T[P_ZL * TJ + p], T[P_VX * TJ + p], T[P_VY * TJ + p], T[P_VZ * TJ + p], T[P_M * TJ + p],
               skip_self || (iflag && jflag), eps2);
}

// R5 in the packed path.  The packed loop runs over whole tiles, so in the one tile that holds the
// index of an i-particle it evaluates the self pair: r = w = 0 exactly, nothing for acc and jerk,
// but m_i/eps for pot -- a term that can be orders of magnitude above the real ones (|pot| ~ 1 at
// m_i/eps = 1e4), and an fp32 sum that holds it rounds them away.  So that tile's pot lane (the
// even or the odd j of the thread's share, whichever holds the self index) is summed again here
// without the self pair and replaces the polluted lane; the caller makes sure the lane held
// nothing else.  At most 64 scalar terms, once per i-particle per call.
__device__ __forceinline__ float pot_lane(const IPart& I, const float* T, int jlane, int jsh, int self, float eps2)
{
    float ps = 0.0f;
    const int nq = (TJ / 4) >> jsh;           // my j-quads of the tile: jlane, jlane + jl, ..
#pragma unroll 1
    for (int q = 0; q < nq; ++q) {
#pragma unroll
        for (int e = 0; e < 4; e += 2) {
            const int k = 4 * (jlane + (q << jsh)) + (self & 1) + e;
            const float dx = (T[P_XH * TJ + k] + I.nxh.x) + (T[P_XL * TJ + k] + I.nxl.x);
            const float dy = (T[P_YH * TJ + k] + I.nyh.x) + (T[P_YL * TJ + k] + I.nyl.x);
            const float dz = (T[P_ZH * TJ + k] + I.nzh.x) + (T[P_ZL * TJ + k] + I.nzl.x);
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
            const float mr = T[P_M * TJ + k] * rsqrt_fast(r2);
            ps += (k == self) ? 0.0f : mr;
        }
    }
    return ps;
}

// S = distance between the 7 sums of one i: 1 when they sit in registers, FORCE_THREADS when they
// sit in shared memory (the all-i kernel keeps them there: 28 registers fewer, 4 CTAs per SM)
template <int S, bool JERK>
__device__ __forceinline__ void flush(Acc32& A, double* d)
{
    d[0 * S] += (double)(A.ax.x + A.ax.y);
    d[1 * S] += (double)(A.ay.x + A.ay.y);
    d[2 * S] += (double)(A.az.x + A.az.y);
    if (JERK) {
        d[3 * S] += (double)(A.jx.x + A.jx.y);
        d[4 * S] += (double)(A.jy.x + A.jy.y);
        d[5 * S] += (double)(A.jz.x + A.jz.y);
    }
    d[6 * S] -= (double)(A.p.x + A.p.y);
    A.ax = A.ay = A.az = A.jx = A.jy = A.jz = A.p = make_float2(0.f, 0.f);
}

// a4/a5 for one i-particle: sum the S partials in a fixed order (deterministic, R9), add the
// unsoftened flagged-flagged pair terms in fp64 straight from the j-store (R7), NaN for a rejected
// index, store SoA.  WARP: the 32 lanes of a warp stride over the partials (fixed butterfly) -- for
// the few-i calls, whose many j-subsets would otherwise be summed by one thread; else one thread.
// IFAST (with WARP): the partials are laid out [c][subset][i] (part_i_fastest) -- the tail rows of a call
// whose other rows are summed one per thread; a compile-time choice, so that the in-kernel reductions of
// the few-i, direct and fused kernels keep their code (a run-time select here cost them 2 - 10 us)
template <bool WARP, bool IFAST = false>
__device__ __forceinline__ void reduce_row(const ReduceArgs& R, int k, int lane)
{
    double o[NOUT];
    if (R.atomic_mode) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            o[c] = R.acc[(int64_t)c * R.ni + k];
            o[3 + c] = R.jrk[(int64_t)c * R.ni + k];
        }
        o[6] = R.pot[k];
    } else {
#pragma unroll
        for (int c = 0; c < NOUT; ++c) o[c] = 0.0;
        const bool in_b = k >= R.kA;
        const double* part = in_b ? R.part_b : R.part;
        const int64_t stride = in_b ? R.ni_pad_b : R.ni_pad;
        const int kl = in_b ? k - R.kA : k, ns = in_b ? R.splits_b : R.splits;
        if (WARP) {
            // four partials per lane and component in flight: the loop is all load latency
            for (int s0 = 0; s0 < ns; s0 += 128) {
                double v[4][NOUT];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int s = s0 + q * 32 + lane;
#pragma unroll
                    for (int c = 0; c < NOUT; ++c)
                        v[q][c] = s < ns ? __ldcg(part + (IFAST ? ((int64_t)c * ns + s) * stride + kl
                                                                : ((int64_t)c * stride + kl) * ns + s))
                                         : 0.0;
                }
#pragma unroll
                for (int q = 0; q < 4; ++q)
#pragma unroll
                    for (int c = 0; c < NOUT; ++c) o[c] += v[q][c];
            }
#pragma unroll
            for (int c = 0; c < NOUT; ++c)
#pragma unroll
                for (int w = 16; w >= 1; w >>= 1) o[c] += __shfl_xor_sync(0xffffffffu, o[c], w);
        } else {
            // element (c, s) of my row is at base + c * cs + s * ss in either layout.  Eight subsets are
            // requested before the first is added (56 loads in flight; one subset at a time the loop is all
            // load latency: 0.45 us per subset, 47 us of a 380 us call at N = 65536, N_i = 4352, S = 103);
            // the additions keep their order (R9)
            const int64_t cs = stride * ns, ss = R.part_i_fastest ? stride : 1;
            const double* base = part + (R.part_i_fastest ? (int64_t)kl : (int64_t)kl * ns);
            int s = 0;
            for (; s + 8 <= ns; s += 8) {
                double v[8][NOUT];
#pragma unroll
                for (int q = 0; q < 8; ++q)
#pragma unroll
                    for (int c = 0; c < NOUT; ++c) v[q][c] = __ldcg(base + c * cs + (s + q) * ss);
#pragma unroll
                for (int q = 0; q < 8; ++q)
#pragma unroll
                    for (int c = 0; c < NOUT; ++c) o[c] += v[q][c];
            }
            for (; s < ns; ++s) {
#pragma unroll
                for (int c = 0; c < NOUT; ++c) o[c] += __ldcg(base + c * cs + s * ss);
            }
        }
    }
    if (WARP && lane != 0) return;
    // who is particle k: a member of the j-set by index (nb_force), or given by value, possibly with
    // the index of the member it is and its flag (nb_force_ext_ids), or by value only (nb_force_ext)
    const bool by_value = R.i_list == nullptr;
    const int i = by_value ? (R.ext_self ? R.ext_self[k] : -1) : R.i_list[k];
    const bool flagged = R.nflag > 0 && (by_value ? (R.ext_flags && (R.ext_flags[k] & 1))
                                                  : (i >= 0 && i < R.n && (R.flags[i] & 1)));
    if (!by_value && (i < 0 || i >= R.n)) {
#pragma unroll
        for (int c = 0; c < NOUT; ++c) o[c] = __longlong_as_double(0x7ff8000000000000LL);
    } else if (flagged && (R.nflag > 1 || by_value)) {
        double xi[3], vi[3];
        if (by_value) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                xi[c] = R.ext_x[(int64_t)c * R.ni + k];
                vi[c] = R.ext_v[(int64_t)c * R.ni + k];
            }
        } else {
            const double dti = R.t_pred - R.store.f[F_T][i];
#pragma unroll
            for (int c = 0; c < 3; ++c)
                predict1(R.store.f[F_X + c][i], R.store.f[F_VX + c][i], R.store.f[F_AX + c][i],
                         R.store.f[F_JX + c][i], dti, xi[c], vi[c]);
        }
        for (int q = 0; q < R.nflag; ++q) {
            const int j = R.flag_list[q];
            if (j == i) continue;
            double r[3], w[3];
            const double dtj = R.t_pred - R.store.f[F_T][j];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double xj, vj;
                predict1(R.store.f[F_X + c][j], R.store.f[F_VX + c][j], R.store.f[F_AX + c][j],
                         R.store.f[F_JX + c][j], dtj, xj, vj);
                r[c] = xj - xi[c];
                w[c] = vj - vi[c];
            }
            const double s2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
            if (s2 == 0.0) continue;
            const double rinv = 1.0 / sqrt(s2), rinv2 = rinv * rinv;
            const double mr = R.store.f[F_M][j] * rinv, mr3 = mr * rinv2;
            const double b = 3.0 * (r[0] * w[0] + r[1] * w[1] + r[2] * w[2]) * rinv2;
            o[6] -= mr;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                o[c] += mr3 * r[c];
                o[3 + c] += mr3 * (w[c] - b * r[c]);
            }
        }
    } else if (R.atomic_mode) {
        return;   // sums are already in place
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        R.acc[(int64_t)c * R.ni + k] = o[c];
        if (R.jrk) R.jrk[(int64_t)c * R.ni + k] = o[3 + c];
    }
    R.pot[k] = o[6];
}

}  // namespace nb
