// direct.cu -- nb_force (and the by-value calls with jerk) for a HANDFUL of active particles
// (N_i <= DIRECT_NI_MAX): one launch that streams the packed predicted j-set once at HBM speed.
//
// with few active i "the thread-per-i mapping cannot hide latencies".  With a handful of
// them the call is not arithmetic at all: it is one pass over N x 44 B.  The tile-ring kernel of
// force.cu spends ~300 warp-instructions of control per 128-j tile on four warps, which is what its
// time then consists of.  Here the mapping is turned round: a thread owns j-QUADS (four consecutive
// j: ten coalesced 128-bit loads straight from global memory, no shared memory, no barriers) and
// carries ALL active i-particles in shared memory (broadcast reads) with their fp32 sums in
// registers.  A grid of one 256-thread CTA per SM gives every thread ~7 quads at N = 2^20, i.e. at
// most a few dozen terms per fp32 lane sum (the R17 bound is 64; the host falls back to the ring
// kernel beyond it).  Sums go to fp64 at the end of the thread's range, meet in a warp butterfly and
// a shared-memory pass (fixed order: deterministic, R9), one partial per CTA [7][NI][CTAs]; the CTA
// that draws the last ticket adds the partials, the unsoftened flagged pairs (R7) and stores.
//
// Pair rules: the self pair is excluded by index -- the quad that holds an i-particle's own index
// goes through the masked scalar pair for that particle (R5); so does a quad with a flagged j for a
// flagged i (R7, flagged-flagged pairs are left to the fp64 pass); eps2 below EPS2_GUARD uses the
// guarded packed pair (R6).
#include "nb_internal.h"
#include "pair32.h"
#include "xchg.h"
#include "pdl.h"

namespace nb {

namespace {

constexpr int DIRECT_THREADS = 256;

template <int NI, bool GUARD>
__global__ void __launch_bounds__(DIRECT_THREADS, 1)
direct_kernel(ForceArgs P, ReduceArgs R)
{
    __shared__ IPart sI[NI];
    __shared__ int sself[NI];
    __shared__ unsigned sflagged;
    __shared__ double sred[DIRECT_THREADS / 32][NI][NOUT];
    __shared__ int s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_wait();       // pdl.h

    // a3 starts here: the first UNR quads of this thread are requested before anything else -- they do
    // not depend on the i-particles, whose gather (two dependent loads) then runs under their latency
    constexpr int UNR = NI <= 2 ? 4 : (NI <= 4 ? 2 : 1);
    const int64_t nquads = (int64_t)P.ntiles * (TJ / 4);
    const int64_t stride = (int64_t)gridDim.x * DIRECT_THREADS;
    const int64_t qfirst = (int64_t)blockIdx.x * DIRECT_THREADS + threadIdx.x;
    float4 fa[UNR][10];
#pragma unroll
    for (int r = 0; r < UNR; ++r) {
        const int64_t qd = qfirst + r * stride;
        if (qd < nquads) {
            const float* T = P.pack + (qd / (TJ / 4)) * TILE_FLOATS + (int)(qd % (TJ / 4)) * 4;
#pragma unroll
            for (int c = 0; c < 10; ++c) fa[r][c] = __ldg(reinterpret_cast<const float4*>(T + c * TJ));
        }
    }

    // a2: the active particles, from the pack (two-float position, fp32 velocity; R8, R17)
    if (tid == 0) sflagged = 0u;
    __syncthreads();
    if (tid < NI && P.ext_x) {
        // by value (nb_force_ext / nb_force_ext_ids / nb_xforce): fp64 position split in two floats here
        // (PAPER.md:53), velocity rounded; the member of the j-set it is, if any, is excluded by index
        const int e = tid < P.ni ? tid : 0;
        float h[3], l[3], w[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double xc = P.ext_x[(int64_t)c * P.ni + e];
            h[c] = __double2float_rn(xc);
            l[c] = __double2float_rn(xc - (double)h[c]);
            w[c] = __double2float_rn(P.ext_v[(int64_t)c * P.ni + e]);
        }
        IPart I;
        I.nxh = dup(-h[0]); I.nyh = dup(-h[1]); I.nzh = dup(-h[2]);
        I.nxl = dup(-l[0]); I.nyl = dup(-l[1]); I.nzl = dup(-l[2]);
        I.nvx = dup(-w[0]); I.nvy = dup(-w[1]); I.nvz = dup(-w[2]);
        sI[tid] = I;
        int q = -1;
        if (tid < P.ni && P.ext_self) {
            const int s = P.ext_self[e];
            if (s >= 0 && s < P.n) q = s;
            if (P.any_flagged && P.ext_flags && (P.ext_flags[e] & 1)) atomicOr(&sflagged, 1u << tid);
        }
        sself[tid] = q;
    } else if (tid < NI) {
        int q = tid < P.ni ? P.i_list[tid] : -1;
        if (tid < P.ni && (q < 0 || q >= P.n)) {
            atomicOr(P.err, 1);
            q = -1;
        }
        sself[tid] = q;
        const int g = q >= 0 ? q : 0;
        const float* b = P.pack + (int64_t)(g / TJ) * TILE_FLOATS + (g % TJ);
        IPart I;
        I.nxh = dup(-b[P_XH * TJ]); I.nyh = dup(-b[P_YH * TJ]); I.nzh = dup(-b[P_ZH * TJ]);
        I.nxl = dup(-b[P_XL * TJ]); I.nyl = dup(-b[P_YL * TJ]); I.nzl = dup(-b[P_ZL * TJ]);
        I.nvx = dup(-b[P_VX * TJ]); I.nvy = dup(-b[P_VY * TJ]); I.nvz = dup(-b[P_VZ * TJ]);
        sI[tid] = I;
        if (q >= 0 && P.any_flagged && (P.flags[q] & 1)) atomicOr(&sflagged, 1u << tid);
    }
    __syncthreads();
    const unsigned iflagged = sflagged;

    Acc32 A[NI];
#pragma unroll
    for (int k = 0; k < NI; ++k)
        A[k].ax = A[k].ay = A[k].az = A[k].jx = A[k].jy = A[k].jz = A[k].p = make_float2(0.f, 0.f);
    const float2 eps2 = dup(P.eps2);
    const float2 m3 = dup(-3.0f);

    // a3: my j-quads, strided over the grid (a warp reads 512 contiguous bytes of each tile array).
    // UNR quads are fetched before the first is evaluated, so that a thread has 10 x UNR 128-bit
    // loads in flight: with a cold L2 the loop is DRAM latency otherwise.  (First round: see above.)
    for (int64_t qd0 = qfirst; qd0 < nquads; qd0 += UNR * stride) {
        if (qd0 != qfirst) {
#pragma unroll
            for (int r = 0; r < UNR; ++r) {
                const int64_t qd = qd0 + r * stride;
                if (qd < nquads) {
                    const float* T = P.pack + (qd / (TJ / 4)) * TILE_FLOATS + (int)(qd % (TJ / 4)) * 4;
#pragma unroll
                    for (int c = 0; c < 10; ++c) fa[r][c] = __ldg(reinterpret_cast<const float4*>(T + c * TJ));
                }
            }
        }
#pragma unroll
        for (int r = 0; r < UNR; ++r) {
            const int64_t qd = qd0 + r * stride;
            if (qd >= nquads) break;
            const float4* f = fa[r];
            const int64_t tile = qd / (TJ / 4);
            const int p = (int)(qd % (TJ / 4)) * 4;
            const int j0 = (int)(tile * TJ) + p;                      // index of the quad's first particle
            unsigned jfl = 0u;                                        // flag bits of the four j (only if needed)
            if (iflagged && ((P.tileflag[tile >> 5] >> (tile & 31)) & 1u)) {
                const float4 ff = __ldg(reinterpret_cast<const float4*>(P.pack + tile * TILE_FLOATS + p + P_FLAG * TJ));
                jfl = (__float_as_uint(ff.x) & 1u) | ((__float_as_uint(ff.y) & 1u) << 1) |
                      ((__float_as_uint(ff.z) & 1u) << 2) | ((__float_as_uint(ff.w) & 1u) << 3);
            }
#pragma unroll
            for (int k = 0; k < NI; ++k) {
                if (k < P.ni) {
                    const int self = sself[k] - j0;                   // 0..3: my own index is in this quad
                    const bool fl = ((iflagged >> k) & 1u) && jfl;
                    if ((unsigned)self < 4u || fl) {
                        const float xs[4][10] = {
                            {f[0].x, f[1].x, f[2].x, f[3].x, f[4].x, f[5].x, f[6].x, f[7].x, f[8].x, f[9].x},
                            {f[0].y, f[1].y, f[2].y, f[3].y, f[4].y, f[5].y, f[6].y, f[7].y, f[8].y, f[9].y},
                            {f[0].z, f[1].z, f[2].z, f[3].z, f[4].z, f[5].z, f[6].z, f[7].z, f[8].z, f[9].z},
                            {f[0].w, f[1].w, f[2].w, f[3].w, f[4].w, f[5].w, f[6].w, f[7].w, f[8].w, f[9].w}};
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            pair1_vals(sI[k], A[k], xs[e][0], xs[e][1], xs[e][2], xs[e][3], xs[e][4], xs[e][5],
                                       xs[e][6], xs[e][7], xs[e][8], xs[e][9],
                                       e == self || (fl && ((jfl >> e) & 1u)), P.eps2);
                    } else {
                        quad<true, GUARD>(sI[k], A[k], f, eps2, m3);
                    }
                }
            }
        }
    }

    // a4: per-thread sums to fp64, warp butterfly, then the warps in order: one partial per CTA
#pragma unroll
    for (int k = 0; k < NI; ++k) {
        double o[NOUT] = {(double)(A[k].ax.x + A[k].ax.y), (double)(A[k].ay.x + A[k].ay.y),
                          (double)(A[k].az.x + A[k].az.y), (double)(A[k].jx.x + A[k].jx.y),
                          (double)(A[k].jy.x + A[k].jy.y), (double)(A[k].jz.x + A[k].jz.y),
                          -(double)(A[k].p.x + A[k].p.y)};
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
        for (int w = 0; w < DIRECT_THREADS / 32; ++w) s += sred[w][k][c];
        P.part[((int64_t)c * P.ni_pad + k) * gridDim.x + blockIdx.x] = s;      // [c][i][CTA]
    }

    // a4/a5: the CTA that draws the last ticket sums the partials of all CTAs (one launch per call)
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(R.counter, 1u) == gridDim.x - 1;
    __syncthreads();
    if (s_last) {
        __threadfence();
        for (int k = warp; k < R.ni; k += DIRECT_THREADS / 32) reduce_row<true>(R, k, lane);
        if (tid == 0) *R.counter = 0u;
        // j-sharded call (nb_xforce): the same CTA exchanges with the peers (xchg.h)
        if (R.xchg) xchg_in_cta<DIRECT_THREADS>(R, P.err, tid);
    }
}

template <int NI>
cudaError_t launch_ni(const ForceArgs& a, const ReduceArgs& r, int grid, cudaStream_t s)
{
    if (a.eps2 < EPS2_GUARD) return pdl_launch(direct_kernel<NI, true>, grid, DIRECT_THREADS, 0, s, a, r);
    return pdl_launch(direct_kernel<NI, false>, grid, DIRECT_THREADS, 0, s, a, r);
}

}  // namespace

// Grid: one CTA per SM (fewer when there are fewer than two quads per thread).  The caller sets
// a.ni_pad and r.splits from *grid_out* BEFORE the launch: pass grid_out first with launch = false.
int direct_grid(int ntiles, int sm_count)
{
    const int64_t nquads = (int64_t)ntiles * (TJ / 4);
    int64_t want = (nquads + 2 * DIRECT_THREADS - 1) / (2 * DIRECT_THREADS);
    if (want < 1) want = 1;
    return (int)(want < sm_count ? want : sm_count);
}

// most fp32 terms one lane sum of one thread collects (the host checks it against R17's bound)
int64_t direct_terms_per_lane(int ntiles, int grid)
{
    const int64_t nquads = (int64_t)ntiles * (TJ / 4);
    const int64_t per_thread = (nquads + (int64_t)grid * DIRECT_THREADS - 1) / ((int64_t)grid * DIRECT_THREADS);
    return 2 * per_thread;
}

cudaError_t launch_direct(const ForceArgs& a, const ReduceArgs& r, int grid, cudaStream_t s)
{
    if (a.ni <= 1) return launch_ni<1>(a, r, grid, s);
    if (a.ni <= 2) return launch_ni<2>(a, r, grid, s);
    if (a.ni <= 4) return launch_ni<4>(a, r, grid, s);
    return launch_ni<8>(a, r, grid, s);
}

}  // namespace nb
