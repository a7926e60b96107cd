// force6.cu -- the 6th-order variant of the pair loop: acc, jerk, SNAP and pot (
// PAPER.md:35 "high >= 4th order integrators with individual time stepping").
//
// A 6th-order Hermite scheme corrects with the second derivative of the acceleration as well.  For
// a pair with r = x_j - x_i, w = v_j - v_i, b = a_j - a_i and s = r.r + eps2 (reading R22 of
// DESIGN.md; the paper prints no formula):
//     al = (r.w)/s ,  be = (w.w + r.b)/s + al^2
//     A = m r s^-3/2 ;  J = m w s^-3/2 - 3 al A ;  S = m b s^-3/2 - 6 al J - 3 be A
// so the kernel needs the accelerations of i and j next to positions and velocities: with
// nb_set_order(ctx, 6) the predictor also writes tiles of 14 floats per particle (two-float position,
// velocity, predicted acceleration a + jerk dt, mass, flag: 56 B), which this kernel streams.
//
// Same mapping as force.cu's all-i kernel (CTA = 128 threads x 2 i-particles in registers, one
// j-subset, tiles brought in by 1-D bulk copies into an mbarrier ring, packed f32x2 arithmetic with two
// consecutive j per instruction, fp32 sums over one tile then fp64 in shared memory, partial sums
// [10][N_i][S] + a reduction kernel).  64 FP32 lane-operations per interaction instead of 33, so the
// ceiling is half that of the 4th-order kernel in interactions per second.  Every pair is masked
// inside the packed loop (compare + select on the ALU pipe, free beside the FP32 pipe): the self pair
// by index (R5), s = 0 (R6), flagged-flagged pairs (R7, added back unsoftened in fp64 by the
// reduction, straight from the j-store).
#include "nb_internal.h"
#include "tma.h"
#include "pdl.h"

namespace nb {

namespace {

constexpr int NOUT6 = 10;                     // ax ay az jx jy jz sx sy sz pot
constexpr int STG6 = 4;

struct I6 {               // one i-particle, negated
    float xh[3], xl[3], v[3], a[3];
};
struct A6 {               // per-tile fp32 sums, lane 0 = even j, lane 1 = odd j
    float2 a[3], j[3], s[3], p;
};

__device__ __forceinline__ float2 dup6(float a) { return make_float2(a, a); }

// One i against a pair of consecutive j (indices jq, jq + 1 inside the tile).
__device__ __forceinline__ void pair6(const I6& I, A6& A, const float2* f, float2 eps2, int self, int jq,
                                      bool iflag)
{
    float2 d[3], w[3], b[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        d[c] = __fadd2_rn(__fadd2_rn(f[c], dup6(I.xh[c])), __fadd2_rn(f[3 + c], dup6(I.xl[c])));
        w[c] = __fadd2_rn(f[6 + c], dup6(I.v[c]));
        b[c] = __fadd2_rn(f[9 + c], dup6(I.a[c]));
    }
    float2 r2 = __ffma2_rn(d[0], d[0], eps2);
    r2 = __ffma2_rn(d[1], d[1], r2);
    r2 = __ffma2_rn(d[2], d[2], r2);
    float2 rinv;
    rinv.x = rsqrt_fast(r2.x);
    rinv.y = rsqrt_fast(r2.y);
    // masks: self pair (R5), s == 0 (R6), flagged-flagged (R7: redone unsoftened by the reduction)
    const bool fx = iflag && (__float_as_uint(f[13].x) & 1u), fy = iflag && (__float_as_uint(f[13].y) & 1u);
    rinv.x = (self == jq || !(r2.x > 0.0f) || fx) ? 0.0f : rinv.x;
    rinv.y = (self == jq + 1 || !(r2.y > 0.0f) || fy) ? 0.0f : rinv.y;
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 mr = __fmul2_rn(f[12], rinv);
    const float2 mr3 = __fmul2_rn(mr, rinv2);
    float2 rv = __fmul2_rn(d[0], w[0]);
    rv = __ffma2_rn(d[1], w[1], rv);
    rv = __ffma2_rn(d[2], w[2], rv);
    float2 q = __fmul2_rn(w[0], w[0]);
    q = __ffma2_rn(w[1], w[1], q);
    q = __ffma2_rn(w[2], w[2], q);
    q = __ffma2_rn(d[0], b[0], q);
    q = __ffma2_rn(d[1], b[1], q);
    q = __ffma2_rn(d[2], b[2], q);
    const float2 al = __fmul2_rn(rv, rinv2);
    const float2 be = __ffma2_rn(al, al, __fmul2_rn(q, rinv2));
    const float2 c1 = __fmul2_rn(al, dup6(-3.0f));
    const float2 c2 = __fadd2_rn(c1, c1);
    const float2 c3 = __fmul2_rn(be, dup6(-3.0f));
    A.p = __fadd2_rn(A.p, mr);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float2 Ac = __fmul2_rn(mr3, d[c]);
        const float2 Jc = __ffma2_rn(c1, Ac, __fmul2_rn(mr3, w[c]));
        const float2 Sc = __ffma2_rn(c3, Ac, __ffma2_rn(c2, Jc, __fmul2_rn(mr3, b[c])));
        A.a[c] = __fadd2_rn(A.a[c], Ac);
        A.j[c] = __fadd2_rn(A.j[c], Jc);
        A.s[c] = __fadd2_rn(A.s[c], Sc);
    }
}

__global__ void __launch_bounds__(FORCE_THREADS, 2) force6_kernel(Force6Args P)
{
    pdl_wait();       // pdl.h
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* tiles = reinterpret_cast<float*>(smem_raw);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + STG6 * TILE6_BYTES);
    int* rel = reinterpret_cast<int*>(smem_raw + STG6 * TILE6_BYTES + STG6 * 8);
    double* sd = reinterpret_cast<double*>(smem_raw + STG6 * (TILE6_BYTES + 16)) + threadIdx.x;   // [u][c][thread]

    const int tid = threadIdx.x;
    const int it = blockIdx.x % P.n_itiles, sp = blockIdx.x / P.n_itiles;
    const int t0 = (int)(((int64_t)P.ntiles * sp) / P.splits);
    const int t1 = (int)(((int64_t)P.ntiles * (sp + 1)) / P.splits);

    if (tid == 0) {
        for (int s = 0; s < STG6; ++s) {
            mbar_init(smem_u32(&bars[s]), 1);
            rel[s] = 0;
        }
        mbar_fence_init();
        for (int s = 0; s < STG6 && t0 + s < t1; ++s) {
            mbar_expect_tx(smem_u32(&bars[s]), TILE6_BYTES);
            bulk_g2s(smem_u32(tiles + s * TILE6_FLOATS), P.pack6 + (int64_t)(t0 + s) * TILE6_FLOATS, TILE6_BYTES,
                     smem_u32(&bars[s]));
        }
    }

    I6 I[IPT];
    int idx[IPT];
    bool ifl[IPT];
    A6 A[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int ku = it * ITILE + u * FORCE_THREADS + tid;
        int q = ku < P.ni ? P.i_list[ku] : 0;
        const bool bad = q < 0 || q >= P.n;
        if (bad) {
            atomicOr(P.err, 1);
            q = 0;
        }
        idx[u] = (ku < P.ni && !bad) ? q : -1;
        const float* b = P.pack6 + (int64_t)(q / TJ) * TILE6_FLOATS + (q % TJ);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            I[u].xh[c] = -b[c * TJ];
            I[u].xl[c] = -b[(3 + c) * TJ];
            I[u].v[c] = -b[(6 + c) * TJ];
            I[u].a[c] = -b[(9 + c) * TJ];
        }
        ifl[u] = P.any_flagged && (P.flags[q] & 1);
#pragma unroll
        for (int c = 0; c < 3; ++c) A[u].a[c] = A[u].j[c] = A[u].s[c] = make_float2(0.f, 0.f);
        A[u].p = make_float2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < NOUT6; ++c) sd[(u * NOUT6 + c) * FORCE_THREADS] = 0.0;
    }
    const float2 eps2 = dup6(P.eps2);
    __syncthreads();

    for (int t = t0; t < t1; ++t) {
        const int st = (t - t0) % STG6;
        mbar_wait(smem_u32(&bars[st]), ((t - t0) / STG6) & 1);
        const float* T = tiles + st * TILE6_FLOATS;
        int self[IPT];
#pragma unroll
        for (int u = 0; u < IPT; ++u) self[u] = idx[u] - t * TJ;      // position of the own index in this tile
#pragma unroll 1
        for (int p = 0; p < TJ; p += 4) {
            float4 g[14];
#pragma unroll
            for (int c = 0; c < 14; ++c) g[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
            float2 lo[14], hi[14];
#pragma unroll
            for (int c = 0; c < 14; ++c) {
                lo[c] = make_float2(g[c].x, g[c].y);
                hi[c] = make_float2(g[c].z, g[c].w);
            }
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                pair6(I[u], A[u], lo, eps2, self[u], p, ifl[u]);
                pair6(I[u], A[u], hi, eps2, self[u], p + 2, ifl[u]);
            }
        }
        // fp32 sums over NB_FLUSH_TILES tiles (128 terms per lane), then fp64 (as force.cu's all-i kernel)
        if (((t - t0) & (NB_FLUSH_TILES - 1)) == NB_FLUSH_TILES - 1 || t == t1 - 1)
#pragma unroll
        for (int u = 0; u < IPT; ++u) {
            double* d = sd + u * NOUT6 * FORCE_THREADS;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                d[c * FORCE_THREADS] += (double)(A[u].a[c].x + A[u].a[c].y);
                d[(3 + c) * FORCE_THREADS] += (double)(A[u].j[c].x + A[u].j[c].y);
                d[(6 + c) * FORCE_THREADS] += (double)(A[u].s[c].x + A[u].s[c].y);
                A[u].a[c] = A[u].j[c] = A[u].s[c] = make_float2(0.f, 0.f);
            }
            d[9 * FORCE_THREADS] -= (double)(A[u].p.x + A[u].p.y);
            A[u].p = make_float2(0.f, 0.f);
        }
        __syncwarp();
        if ((tid & 31) == 0) {
            __threadfence_block();
            const int old = atomicAdd(&rel[st], 1);
            if ((old & (NWARPS - 1)) == NWARPS - 1 && t + STG6 < t1) {
                mbar_expect_tx(smem_u32(&bars[st]), TILE6_BYTES);
                bulk_g2s(smem_u32(tiles + st * TILE6_FLOATS), P.pack6 + (int64_t)(t + STG6) * TILE6_FLOATS,
                         TILE6_BYTES, smem_u32(&bars[st]));
            }
        }
    }
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int ku = it * ITILE + u * FORCE_THREADS + tid;
#pragma unroll
        for (int c = 0; c < NOUT6; ++c)
            P.part[((int64_t)c * P.ni_pad + ku) * P.splits + sp] = sd[(u * NOUT6 + c) * FORCE_THREADS];
    }
}

// Sum of the S partials of each i (fixed order), the unsoftened flagged-flagged pairs in fp64 from the
// j-store (predicted x, v by R1 and a by R22), NaN for a rejected index.
__global__ void __launch_bounds__(128) reduce6_kernel(Force6Args P, StorePtrs st, const int32_t* flag_list, int nflag,
                                                      double t_pred, double* acc, double* jrk, double* snp,
                                                      double* pot)
{
    pdl_wait();       // pdl.h
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= P.ni) return;
    double o[NOUT6];
#pragma unroll
    for (int c = 0; c < NOUT6; ++c) o[c] = 0.0;
    for (int s = 0; s < P.splits; ++s) {
#pragma unroll
        for (int c = 0; c < NOUT6; ++c) o[c] += P.part[((int64_t)c * P.ni_pad + k) * P.splits + s];
    }
    const int i = P.i_list[k];
    if (i < 0 || i >= P.n) {
#pragma unroll
        for (int c = 0; c < NOUT6; ++c) o[c] = __longlong_as_double(0x7ff8000000000000LL);
    } else if (nflag > 1 && (P.flags[i] & 1)) {
        double xi[3], vi[3], ai[3];
        const double dti = t_pred - st.f[F_T][i];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            predict1(st.f[F_X + c][i], st.f[F_VX + c][i], st.f[F_AX + c][i], st.f[F_JX + c][i], dti, xi[c], vi[c]);
            ai[c] = fma(st.f[F_JX + c][i], dti, st.f[F_AX + c][i]);
        }
        for (int q = 0; q < nflag; ++q) {
            const int j = flag_list[q];
            if (j == i) continue;
            double r[3], w[3], b[3];
            const double dtj = t_pred - st.f[F_T][j];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double xj, vj;
                predict1(st.f[F_X + c][j], st.f[F_VX + c][j], st.f[F_AX + c][j], st.f[F_JX + c][j], dtj, xj, vj);
                r[c] = xj - xi[c];
                w[c] = vj - vi[c];
                b[c] = fma(st.f[F_JX + c][j], dtj, st.f[F_AX + c][j]) - ai[c];
            }
            const double s2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
            if (s2 == 0.0) continue;
            const double rinv = 1.0 / sqrt(s2), rinv2 = rinv * rinv;
            const double mr = st.f[F_M][j] * rinv, mr3 = mr * rinv2;
            const double al = (r[0] * w[0] + r[1] * w[1] + r[2] * w[2]) * rinv2;
            const double be = (w[0] * w[0] + w[1] * w[1] + w[2] * w[2] + r[0] * b[0] + r[1] * b[1] + r[2] * b[2]) * rinv2 +
                              al * al;
            o[9] -= mr;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double Ac = mr3 * r[c];
                const double Jc = mr3 * w[c] - 3.0 * al * Ac;
                o[c] += Ac;
                o[3 + c] += Jc;
                o[6 + c] += mr3 * b[c] - 6.0 * al * Jc - 3.0 * be * Ac;
            }
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        acc[(int64_t)c * P.ni + k] = o[c];
        jrk[(int64_t)c * P.ni + k] = o[3 + c];
        snp[(int64_t)c * P.ni + k] = o[6 + c];
    }
    pot[k] = o[9];
}

constexpr int F6_SMEM = STG6 * (TILE6_BYTES + 16) + IPT * NOUT6 * FORCE_THREADS * 8;

}  // namespace

cudaError_t force6_kernel_setup(int* blocks_per_sm)
{
    cudaError_t e = cudaFuncSetAttribute(force6_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, F6_SMEM);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, force6_kernel, FORCE_THREADS, F6_SMEM);
}

cudaError_t launch_force6(const Force6Args& a, const StorePtrs& st, const int32_t* flag_list, int nflag, double t_pred,
                          double* acc, double* jrk, double* snp, double* pot, cudaStream_t s)
{
    if (a.ntiles > 0) {
        cudaError_t e = pdl_launch(force6_kernel, (unsigned)a.n_itiles * (unsigned)a.splits, FORCE_THREADS, F6_SMEM, s, a);
        if (e != cudaSuccess) return e;
    }
    Force6Args r = a;
    if (a.ntiles == 0) r.splits = 0;
    return pdl_launch(reduce6_kernel, (unsigned)((a.ni + 127) / 128), 128, 0, s, r, st, flag_list, nflag, t_pred, acc, jrk, snp, pot);
}

}  // namespace nb
