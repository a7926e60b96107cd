// steps.cu -- nb_steps: many block steps in ONE persistent cooperative kernel, no host round trip and
// no kernel launch per step (SURVEY.md 8(f) NEXT-1 "a whole ph4-style step never leaves the GPU").
//
// PAPER.md:83 calls the host link "the crucial bottleneck"; PAPER.md:41/:49 describe block time steps
// in which "only the particles are updated that require a force update at a certain time", and
// PAPER.md:51 says a handful of active particles cannot hide latencies.  With individual steps most
// blocks ARE a handful of particles (median 4 at N = 16384), so a block step done as five launches
// plus a synchronisation (nb_step) is all latency.  Here one grid of at most one 512-thread CTA per
// SM runs the whole loop and meets at three grid-wide barriers per step:
//   A  t1 = min_j (t_j + dt_j): each CTA scans its slice of the particles, one atomicMin per CTA  (R21)
//      -- barrier --
//   B  particles due at t1 append themselves to a scratch list (atomic counter)                  (R21)
//      -- barrier --   every CTA now knows N_i; a block that is too large for this kernel ends it
//   C  every CTA sorts the (short) list by rank in shared memory -- ascending, as R21 states, so the
//      result does not depend on the order of the atomics --, predicts the due particles (R1, R8),
//      then streams ITS slice of the j-store once: 512 particles at a time are predicted into shared
//      memory and the threads, arranged as (i-particle, j-stride), evaluate the pairs in IEEE
//      double (pair64.h: the same body as nb_force_fused; self pair by index, flagged pairs
//      unsoftened, R5..R7).  One partial sum per CTA and i-particle, [7][N_i][CTAs].
//      -- barrier --
//   D  the CTA that owns a due particle sums its partials (a warp per particle, fixed order:
//      deterministic, R9), stores the forces for nb_block_forces and runs the corrector and the
//      step criterion (correct_one: R12, R18..R20).  It then goes straight on to A of the next step:
//      A and B only read the CTA's own slice.
// The kernel stops when its budget of steps is used up, when the next block time exceeds t_end, or
// when the next block is larger than it handles (N_i > STEPS_NI_MAX or N_i x N above the caller's
// bound): the host then takes that one block through nb_step's launches, where the packed fp32 pair
// kernel is faster, and starts the kernel again.  (t1, N_i) of every step go to a device log.
#include <cooperative_groups.h>

#include "hermite_dev.h"
#include "nb_internal.h"
#include "pair64.h"

namespace cg = cooperative_groups;

namespace nb {

namespace {

constexpr int ST_THREADS = 512;
constexpr int ST_WARPS = ST_THREADS / 32;
constexpr int ST_TILE = ST_THREADS;           // j-particles predicted into shared memory at a time

__device__ __forceinline__ double ldcg(const double* p) { return __ldcg(p); }

__global__ void __launch_bounds__(ST_THREADS, 1) steps_kernel(StepsArgs P)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ double si[STEPS_NI_MAX][6];            // predicted state of the due particles
    __shared__ double tile[NOUT][ST_TILE];            // x y z vx vy vz m of 512 j; later: the slice sums
    __shared__ int sl_raw[STEPS_NI_MAX], sl[STEPS_NI_MAX];
    __shared__ unsigned char sfl[STEPS_NI_MAX], tfl[ST_TILE];
    __shared__ unsigned long long swmin[ST_WARPS];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = (int)gridDim.x, b = (int)blockIdx.x;
    const int64_t n = P.n;
    const int64_t chunk = (n + G - 1) / G;
    const int64_t lo = (int64_t)b * chunk < n ? (int64_t)b * chunk : n;
    const int64_t hi = lo + chunk < n ? lo + chunk : n;
    const double* __restrict__ T = P.st.f[F_T];
    volatile unsigned long long* meta = P.meta;

    long long last_ni = 0;                    // size of the last block this launch completed
    for (int64_t s = 0; s < P.budget; ++s) {
        const int par = (int)(s & 1);

        // ---- A: the next block time (R21) ----------------------------------------------------
        unsigned long long k = ~0ull;
        for (int64_t p = lo + tid; p < hi; p += ST_THREADS) {
            const unsigned long long q = key_of(ldcg(T + p) + ldcg(P.dts + p));
            k = q < k ? q : k;
        }
#pragma unroll
        for (int w = 16; w >= 1; w >>= 1) {
            const unsigned long long o = __shfl_xor_sync(0xffffffffu, k, w);
            k = o < k ? o : k;
        }
        if (lane == 0) swmin[warp] = k;
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < ST_WARPS; ++w) k = swmin[w] < k ? swmin[w] : k;
            atomicMin(P.meta + par, k);
        }
        grid.sync();
        const double t1 = of_key(meta[par]);
        if (b == 0 && tid == 0) {             // the other parity's slots, for the next step
            meta[par ^ 1] = ~0ull;
            meta[2 + (par ^ 1)] = 0ull;
        }

        // ---- B: who is due (R21) ---------------------------------------------------------------
        for (int64_t p = lo + tid; p < hi; p += ST_THREADS) {
            if (ldcg(T + p) + ldcg(P.dts + p) == t1) {
                const unsigned long long pos = atomicAdd(P.meta + 2 + par, 1ull);
                if (pos < (unsigned long long)STEPS_NI_MAX) P.scratch[pos] = (int32_t)p;
            }
        }
        grid.sync();
        const long long ni64 = (long long)meta[2 + par];
        int reason = STEPS_RUNNING;
        if (ni64 == 0) reason = STEPS_STUCK;                        // every t + dt is NaN
        else if (!(t1 <= P.t_end)) reason = STEPS_T_END;
        else if (ni64 > STEPS_NI_MAX || ni64 > P.cap || ni64 * n > P.max_pairs) reason = STEPS_BIG;
        if (reason != STEPS_RUNNING) {        // uniform over the grid: everybody leaves
            if (b == 0 && tid == 0) {
                meta[4] = (unsigned long long)s;
                meta[5] = (unsigned long long)reason;
                meta[6] = key_of(t1);
                meta[7] = (unsigned long long)(reason == STEPS_BIG ? ni64 : last_ni);
            }
            return;
        }
        const int ni = (int)ni64;
        if (b == 0 && tid == 0) {
            P.log_t[s] = t1;
            P.log_ni[s] = ni64;
        }

        // ---- C: sorted list, predicted i-particles, one pass over this CTA's j-slice -----------
        if (tid < ni) sl_raw[tid] = __ldcg(P.scratch + tid);
        __syncthreads();
        if (tid < ni) {
            const int me = sl_raw[tid];
            int rank = 0;
            for (int q = 0; q < ni; ++q) rank += sl_raw[q] < me ? 1 : 0;
            sl[rank] = me;
        }
        __syncthreads();
        if (tid < ni) {
            const int64_t i = sl[tid];
            const double dti = t1 - ldcg(T + i);
#pragma unroll
            for (int c = 0; c < 3; ++c)
                predict1(ldcg(P.st.f[F_X + c] + i), ldcg(P.st.f[F_VX + c] + i), ldcg(P.st.f[F_AX + c] + i),
                         ldcg(P.st.f[F_JX + c] + i), dti, si[tid][c], si[tid][3 + c]);
            sfl[tid] = P.any_flagged ? (P.flags[i] & 1) : 0;
            if (b == 0) P.list[tid] = (int32_t)i;
        }
        const int ii = tid % ni, slice = tid / ni, nsl = ST_THREADS / ni;
        Acc64 A;
        A.ax = A.ay = A.az = A.jx = A.jy = A.jz = A.p = 0.0;
        for (int64_t base = lo; base < hi; base += ST_TILE) {
            const int64_t p = base + tid;
            if (p < hi) {
                const double dtj = t1 - ldcg(T + p);
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    predict1(ldcg(P.st.f[F_X + c] + p), ldcg(P.st.f[F_VX + c] + p), ldcg(P.st.f[F_AX + c] + p),
                             ldcg(P.st.f[F_JX + c] + p), dtj, tile[c][tid], tile[3 + c][tid]);
                tile[6][tid] = ldcg(P.st.f[F_M] + p);
                tfl[tid] = P.any_flagged ? (P.flags[p] & 1) : 0;
            }
            __syncthreads();                  // tile (and, the first time, si / sfl / sl) complete
            const int cnt = (int)(hi - base < ST_TILE ? hi - base : ST_TILE);
            if (slice < nsl) {
                const int self = sl[ii] - (int)base;      // position of the own index in this tile, if any
#pragma unroll 2
                for (int q = slice; q < cnt; q += nsl) {
                    const double e2 = (sfl[ii] && tfl[q]) ? 0.0 : P.eps2;
                    pair64<true>(si[ii], A, tile[0][q], tile[1][q], tile[2][q], tile[3][q], tile[4][q], tile[5][q],
                                 tile[6][q], e2, q == self);
                }
            }
            __syncthreads();                  // everybody is done with the tile
        }
        // sums of the j-strides of one i-particle -> one partial per (CTA, i, component)
        tile[0][tid] = A.ax; tile[1][tid] = A.ay; tile[2][tid] = A.az;
        tile[3][tid] = A.jx; tile[4][tid] = A.jy; tile[5][tid] = A.jz; tile[6][tid] = A.p;
        __syncthreads();
        const int ntask = NOUT * ni;
        if (nsl <= 16) {
            for (int task = tid; task < ntask; task += ST_THREADS) {
                const int c = task / ni, i = task % ni;
                double sum = 0.0;
                for (int q = 0; q < nsl; ++q) sum += tile[c][q * ni + i];
                P.part[((int64_t)c * ni + i) * G + b] = sum;
            }
        } else {
            for (int task = warp; task < ntask; task += ST_WARPS) {
                const int c = task / ni, i = task % ni;
                double sum = 0.0;
                for (int q = lane; q < nsl; q += 32) sum += tile[c][q * ni + i];
#pragma unroll
                for (int w = 16; w >= 1; w >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, w);
                if (lane == 0) P.part[((int64_t)c * ni + i) * G + b] = sum;
            }
        }
        grid.sync();

        // ---- D: the owner of a due particle sums its partials and corrects it ------------------
        for (int q = warp; q < ni; q += ST_WARPS) {
            const int64_t i = sl[q];
            if (i < lo || i >= hi) continue;
            double o[NOUT];
#pragma unroll
            for (int c = 0; c < NOUT; ++c) {
                double sum = 0.0;
                const double* src = P.part + ((int64_t)c * ni + q) * G;
                for (int g = lane; g < G; g += 32) sum += ldcg(src + g);
#pragma unroll
                for (int w = 16; w >= 1; w >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, w);
                o[c] = sum;
            }
            if (lane == 0) {
#pragma unroll
                for (int c = 0; c < NOUT; ++c) P.out[(int64_t)c * ni + q] = o[c];
                correct_one(P.st, P.dts, i, t1, o, o + 3, P.eta, P.dt_min, P.dt_max, P.err);
            }
        }
        __syncthreads();                      // the new (t, dt) of my slice are visible to my next scan
        last_ni = ni64;
    }
    if (b == 0 && tid == 0) {
        meta[4] = (unsigned long long)P.budget;
        meta[5] = (unsigned long long)STEPS_DONE;
        meta[6] = 0ull;
        meta[7] = (unsigned long long)last_ni;
    }
}

}  // namespace

cudaError_t steps_kernel_setup(int* blocks_per_sm)
{
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, steps_kernel, ST_THREADS, 0);
}

// meta[0] (min key of step 0) and meta[2] (its counter) are preset here; the kernel resets the slots
// of the other parity itself.  Grid: one CTA per SM, fewer when the set is small.
cudaError_t launch_steps(const StepsArgs& a, int sm_count, cudaStream_t s)
{
    const unsigned long long init[4] = {~0ull, ~0ull, 0ull, 0ull};
    cudaError_t e = cudaMemcpyAsync(a.meta, init, sizeof(init), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return e;
    int64_t want = (a.n + 63) / 64;
    int grid = sm_count;
    if (want < grid) grid = (int)(want > 0 ? want : 1);
    StepsArgs copy = a;
    void* args[] = {(void*)&copy};
    return cudaLaunchCooperativeKernel((const void*)steps_kernel, dim3(grid), dim3(ST_THREADS), args, 0, s);
}

}  // namespace nb
