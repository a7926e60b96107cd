// force64.cu -- the pair loop in IEEE double precision throughout.
//
// "The integration of the orbits of objects with an extreme mass ratio, like
// planetesimals around super-massive black holes, remains hard to achieve without IEEE-754 double
// precision arithmetic.  The latest GPUs support double precision and therefore enable such
// research."  nb_set_precision(ctx, 1) selects this kernel for nb_force / nb_force_ext.
//
// Same mapping as force.cu (CTA = 128 threads x 2 i-particles, one j-subset, j-tiles brought in by
// 1-D bulk copies into an mbarrier ring, partial sums for reduce_kernel), but: the tile holds the
// predicted state as doubles (8 arrays of TJ: x y z vx vy vz m flag = 8 KB), every difference,
// product and sum is fp64, and the reciprocal square root is MUFU.RSQ on the fp32-rounded s
// followed by two Newton steps in fp64 (error 2^-22 -> 1e-13 -> rounding).  The self pair is
// masked by index (no epilogue correction), s = 0 pairs contribute nothing (R6), flagged-flagged
// pairs use eps2 = 0 inside the loop (R7).  35 fp64 operations per interaction; the FP64 pipe
// issues 64 lanes/clk/SM, so the ceiling is 1.83 interactions/clk/SM = 43 % of the 60-flop FP32
// roofline.
#include "nb_internal.h"
#include "pair64.h"
#include "tma.h"
#include "pdl.h"

namespace nb {

namespace {

constexpr int STAGES64 = 4;
constexpr int F64_SMEM = STAGES64 * (TILE64_BYTES + 16);

// FLAGS: some particle carries the unsoftened flag (R7).  MODE as in force.cu: 0 = i by index,
// 1 = i by value, 2 = i by value and acc + pot only.
template <bool FLAGS, int MODE>
__global__ void __launch_bounds__(FORCE_THREADS, 3) force64_kernel(ForceArgs P)
{
    constexpr bool JERK = (MODE != 2);
    pdl_wait();       // pdl.h
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* tiles = reinterpret_cast<double*>(smem_raw);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + STAGES64 * TILE64_BYTES);
    int* rel = reinterpret_cast<int*>(smem_raw + STAGES64 * TILE64_BYTES + STAGES64 * 8);

    const int tid = threadIdx.x;
    const int it = blockIdx.x % P.n_itiles;
    const int sp = blockIdx.x / P.n_itiles;
    const int t0 = (int)(((int64_t)P.ntiles * sp) / P.splits);
    const int t1 = (int)(((int64_t)P.ntiles * (sp + 1)) / P.splits);

    if (tid == 0) {
        for (int s = 0; s < STAGES64; ++s) {
            mbar_init(smem_u32(&bars[s]), 1);
            rel[s] = 0;
        }
        mbar_fence_init();
        for (int s = 0; s < STAGES64 && t0 + s < t1; ++s) {
            mbar_expect_tx(smem_u32(&bars[s]), TILE64_BYTES);
            bulk_g2s(smem_u32(tiles + s * TILE64_DOUBLES), P.pack64 + (int64_t)(t0 + s) * TILE64_DOUBLES,
                      TILE64_BYTES, smem_u32(&bars[s]));
        }
    }

    // a2: i-gather, fp64
    double xi[IPT][6];
    int idx[IPT];
    bool ifl[IPT];
    Acc64 A[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int ku = it * ITILE + u * FORCE_THREADS + tid;
        const bool on = P.k0 + ku < P.ni;
        ifl[u] = false;
        if (MODE != 0) {
            const int64_t e = on ? P.k0 + ku : 0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                xi[u][c] = P.ext_x[(int64_t)c * P.ni + e];
                xi[u][3 + c] = (MODE == 1) ? P.ext_v[(int64_t)c * P.ni + e] : 0.0;
            }
            idx[u] = on ? -2 : -1;
        } else {
            int q = on ? P.i_list[P.k0 + ku] : 0;
            const bool bad = (q < 0) || (q >= P.n);
            if (bad) {
                atomicOr(P.err, 1);
                q = 0;
            }
            idx[u] = (on && !bad) ? q : -1;
            const double* b = P.pack64 + (int64_t)(q / TJ) * TILE64_DOUBLES + (q % TJ);
#pragma unroll
            for (int c = 0; c < 6; ++c) xi[u][c] = b[c * TJ];
            if (FLAGS) ifl[u] = (P.flags[q] & 1) != 0;
        }
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = 0.0;
    }
    __syncthreads();

    for (int t = t0; t < t1; ++t) {
        const int st = (t - t0) % STAGES64;
        mbar_wait(smem_u32(&bars[st]), ((t - t0) / STAGES64) & 1);
        const double* T = tiles + st * TILE64_DOUBLES;
        const int jbase = t * TJ;
#pragma unroll 2
        for (int p = 0; p < TJ; p += 2) {
            double2 g[8];
#pragma unroll
            for (int c = 0; c < 8; ++c)
                if ((JERK || c < 3 || c == 6) && (FLAGS || c < 7))
                    g[c] = *reinterpret_cast<const double2*>(T + c * TJ + p);
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                double e0 = P.eps2d, e1 = P.eps2d;
                if (FLAGS) {
                    e0 = (ifl[u] && g[7].x != 0.0) ? 0.0 : P.eps2d;
                    e1 = (ifl[u] && g[7].y != 0.0) ? 0.0 : P.eps2d;
                }
                pair64<JERK>(xi[u], A[u], g[0].x, g[1].x, g[2].x, g[3].x, g[4].x, g[5].x, g[6].x, e0,
                             idx[u] == jbase + p);
                pair64<JERK>(xi[u], A[u], g[0].y, g[1].y, g[2].y, g[3].y, g[4].y, g[5].y, g[6].y, e1,
                             idx[u] == jbase + p + 1);
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) {
            __threadfence_block();
            const int old = atomicAdd(&rel[st], 1);
            if ((old & (NWARPS - 1)) == NWARPS - 1 && t + STAGES64 < t1) {
                mbar_expect_tx(smem_u32(&bars[st]), TILE64_BYTES);
                bulk_g2s(smem_u32(tiles + st * TILE64_DOUBLES),
                          P.pack64 + (int64_t)(t + STAGES64) * TILE64_DOUBLES, TILE64_BYTES,
                          smem_u32(&bars[st]));
            }
        }
    }

#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int ku = it * ITILE + u * FORCE_THREADS + tid;
        const double o[NOUT] = {A[u].ax, A[u].ay, A[u].az, A[u].jx, A[u].jy, A[u].jz, A[u].p};
#pragma unroll
        for (int c = 0; c < NOUT; ++c) P.part[((int64_t)c * P.ni_pad + ku) * P.splits + sp] = o[c];
    }
}

template <bool FLAGS, int MODE>
cudaError_t setup64(int* blocks)
{
    cudaError_t e = cudaFuncSetAttribute(force64_kernel<FLAGS, MODE>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, F64_SMEM);
    if (e != cudaSuccess) return e;
    int b = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, force64_kernel<FLAGS, MODE>, FORCE_THREADS, F64_SMEM);
    if (e == cudaSuccess && (*blocks == 0 || b < *blocks)) *blocks = b;
    return e;
}

}  // namespace

cudaError_t force64_kernel_setup(int* blocks_per_sm)
{
    *blocks_per_sm = 0;
    cudaError_t e = setup64<false, 0>(blocks_per_sm);
    if (e == cudaSuccess) e = setup64<true, 0>(blocks_per_sm);
    if (e == cudaSuccess) e = setup64<false, 1>(blocks_per_sm);
    if (e == cudaSuccess) e = setup64<false, 2>(blocks_per_sm);
    return e;
}

cudaError_t launch_force64(const ForceArgs& a, int mode, cudaStream_t s)
{
    const unsigned grid = (unsigned)a.n_itiles * (unsigned)a.splits;
    if (mode == 1) return pdl_launch(force64_kernel<false, 1>, grid, FORCE_THREADS, F64_SMEM, s, a);
    if (mode == 2) return pdl_launch(force64_kernel<false, 2>, grid, FORCE_THREADS, F64_SMEM, s, a);
    if (a.any_flagged) return pdl_launch(force64_kernel<true, 0>, grid, FORCE_THREADS, F64_SMEM, s, a);
    return pdl_launch(force64_kernel<false, 0>, grid, FORCE_THREADS, F64_SMEM, s, a);
}

}  // namespace nb
