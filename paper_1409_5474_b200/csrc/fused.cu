// fused.cu -- forces on a handful of active particles in ONE pass over the j-store (SURVEY.md 8(f)
// NEXT-3, second half): the Hermite predictor runs inside the pair loop, so the two O(N) passes of a
// block step with very few active particles (predict: 112 B read + 44 B written per particle;
// force: 44 B read) become one pass of 112 B read.  PAPER.md:55 counts "the time required to
// execute the optional prediction step on the j particles" among the costs of a step, and
// PAPER.md:51 is about exactly this regime (N_i far below what fills the device).
//
// Mapping: the N j-particles are spread over a full grid of 256-thread CTAs, one thread takes two
// particles at a time (128-bit loads of the 14 fp64 fields, as predict_kernel), predicts them to t
// (R1, the same predict1 as everywhere), and evaluates them against the NI <= 8 active particles,
// whose predicted state sits in shared memory.  Everything is fp64 (pair64.h): with so few
// interactions per byte the kernel is HBM-bound and double precision is free.  Per-thread sums are
// reduced by shuffles and shared memory to one partial per CTA, [7][NI][grid], and summed by
// reduce_kernel like every other force call.  The self pair is masked by index, flagged pairs get
// eps2 = 0 in the loop (R5, R7).
#include "nb_internal.h"
#include "pair64.h"
#include "pdl.h"

namespace nb {

namespace {

constexpr int FUSED_THREADS = 256;

__device__ __forceinline__ double2 ldg2(const double* p, int64_t i)
{
    return __ldg(reinterpret_cast<const double2*>(p + i));
}

template <int NI>
__global__ void __launch_bounds__(FUSED_THREADS)
fused_kernel(StorePtrs st, const uint8_t* __restrict__ flags, const int32_t* __restrict__ i_list, int ni,
             int64_t n, int64_t n_pad, double t, double eps2, int any_flagged, double* __restrict__ part,
             int* err)
{
    __shared__ double si[NI][6];
    __shared__ int sidx[NI];
    __shared__ int sflag[NI];
    __shared__ double sred[FUSED_THREADS / 32][NI][NOUT];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_wait();       // pdl.h

    // the active particles, predicted to t (R8: i and j alike are taken at their predicted state)
    if (tid < NI) {
        int q = tid < ni ? i_list[tid] : -1;
        if (tid < ni && (q < 0 || q >= n)) {
            atomicOr(err, 1);
            q = -1;
        }
        sidx[tid] = q;
        sflag[tid] = (q >= 0 && any_flagged) ? (flags[q] & 1) : 0;
        const int64_t i = q >= 0 ? q : 0;
        const double dt = t - st.f[F_T][i];
#pragma unroll
        for (int c = 0; c < 3; ++c)
            predict1(st.f[F_X + c][i], st.f[F_VX + c][i], st.f[F_AX + c][i], st.f[F_JX + c][i], dt,
                     si[tid][c], si[tid][3 + c]);
    }
    __syncthreads();

    Acc64 A[NI];
#pragma unroll
    for (int k = 0; k < NI; ++k) A[k].ax = A[k].ay = A[k].az = A[k].jx = A[k].jy = A[k].jz = A[k].p = 0.0;

    const int64_t stride = 2 * (int64_t)gridDim.x * FUSED_THREADS;
    for (int64_t p = 2 * ((int64_t)blockIdx.x * FUSED_THREADS + tid); p < n_pad; p += stride) {
        const double2 tj = ldg2(st.f[F_T], p);
        const double dt0 = t - tj.x, dt1 = t - tj.y;
        double xj[2][6];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double2 x = ldg2(st.f[F_X + c], p), v = ldg2(st.f[F_VX + c], p);
            const double2 a = ldg2(st.f[F_AX + c], p), j = ldg2(st.f[F_JX + c], p);
            predict1(x.x, v.x, a.x, j.x, dt0, xj[0][c], xj[0][3 + c]);
            predict1(x.y, v.y, a.y, j.y, dt1, xj[1][c], xj[1][3 + c]);
        }
        double2 m = ldg2(st.f[F_M], p);
        if (p >= n) m.x = 0.0;                     // padding beyond n: exerts nothing
        if (p + 1 >= n) m.y = 0.0;
        int f0 = 0, f1 = 0;
        if (any_flagged) {
            const uchar2 fl = *reinterpret_cast<const uchar2*>(flags + p);
            f0 = fl.x & 1;
            f1 = fl.y & 1;
        }
#pragma unroll
        for (int k = 0; k < NI; ++k) {
            if (k < ni) {
                const double e0 = (sflag[k] && f0) ? 0.0 : eps2;
                const double e1 = (sflag[k] && f1) ? 0.0 : eps2;
                pair64<true>(si[k], A[k], xj[0][0], xj[0][1], xj[0][2], xj[0][3], xj[0][4], xj[0][5], m.x, e0,
                             sidx[k] == (int)p);
                pair64<true>(si[k], A[k], xj[1][0], xj[1][1], xj[1][2], xj[1][3], xj[1][4], xj[1][5], m.y, e1,
                             sidx[k] == (int)(p + 1));
            }
        }
    }

    // one partial per CTA: fixed shuffle butterfly, then the warps in order (deterministic, R9)
#pragma unroll
    for (int k = 0; k < NI; ++k) {
        double o[NOUT] = {A[k].ax, A[k].ay, A[k].az, A[k].jx, A[k].jy, A[k].jz, A[k].p};
#pragma unroll
        for (int c = 0; c < NOUT; ++c) {
#pragma unroll
            for (int w = 16; w >= 1; w >>= 1) o[c] += __shfl_xor_sync(0xffffffffu, o[c], w);
            if (lane == 0) sred[warp][k][c] = o[c];
        }
    }
    __syncthreads();
    if (tid < NI * NOUT) {
        const int k = tid / NOUT, c = tid % NOUT;
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < FUSED_THREADS / 32; ++w) s += sred[w][k][c];
        part[((int64_t)c * NI + k) * gridDim.x + blockIdx.x] = s;      // [c][i][subset]
    }
}

}  // namespace

// grid: as many CTAs as keep every SM busy, but no more than there are particle pairs
cudaError_t launch_fused(const StorePtrs& st, const uint8_t* flags, const int32_t* i_list, int ni, int64_t n,
                         double t, double eps2, int any_flagged, double* part, int* err, int sm_count,
                         int* grid_out, int* ni_pad_out, cudaStream_t s)
{
    const int64_t n_pad = (n + 1) / 2 * 2;
    int64_t want = (n_pad / 2 + FUSED_THREADS - 1) / FUSED_THREADS;
    int grid = sm_count * 4;
    if (want < grid) grid = (int)(want > 0 ? want : 1);
    *grid_out = grid;
    if (ni <= 1) {
        *ni_pad_out = 1;
        return pdl_launch(fused_kernel<1>, grid, FUSED_THREADS, 0, s, st, flags, i_list, ni, n, n_pad, t, eps2, any_flagged, part, err);
    } else if (ni <= 2) {
        *ni_pad_out = 2;
        return pdl_launch(fused_kernel<2>, grid, FUSED_THREADS, 0, s, st, flags, i_list, ni, n, n_pad, t, eps2, any_flagged, part, err);
    } else if (ni <= 4) {
        *ni_pad_out = 4;
        return pdl_launch(fused_kernel<4>, grid, FUSED_THREADS, 0, s, st, flags, i_list, ni, n, n_pad, t, eps2, any_flagged, part, err);
    } else {
        *ni_pad_out = 8;
        return pdl_launch(fused_kernel<8>, grid, FUSED_THREADS, 0, s, st, flags, i_list, ni, n, n_pad, t, eps2, any_flagged, part, err);
    }
    return cudaGetLastError();
}

}  // namespace nb
