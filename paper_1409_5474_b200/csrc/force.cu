// force.cu -- a2..a5: i-gather, pair loop, j-split partials, reduction.
//
// Mapping.  A CTA of 128 threads owns ITILE = 256 active i-particles (two
// per thread, held in registers as negated, lane-duplicated f32x2 values) and one of S j-subsets
// (PAPER.md:51).  It streams its j-tiles (TJ = 128 particles, 5632 B, SoA inside the tile) from
// L2/HBM into a 4-deep shared-memory ring with 1-D bulk async copies (TMA unit, cp.async.bulk)
// completing on mbarriers; no thread spends issue slots on the copy.  Two consecutive j's form the
// two lanes of every packed FP32 instruction (fma/add/mul .f32x2), so one issue slot serves two
// pair interactions; per interaction the FP32 pipe executes 33 lane-ops (9 for the two-float
// position difference) plus one MUFU.RSQ.  fp32 partial sums run over one tile (64
// terms per lane) and are then flushed to fp64 registers.  The self pair and flagged-flagged pairs
// are masked only in the tiles that contain them (warp-uniform slow path), so the common tile pays
// nothing for R5/R7.  No tensor cores: the pair kernel with its reciprocal square root is not a
// contraction.
#include "nb_internal.h"
#include "pair32.h"
#include "tma.h"
#include "xchg.h"
#include "pdl.h"

namespace nb {

namespace {

// Threads per i-particle ("split the j-particles in subsets" when few i are active;
// here inside the CTA).  The all-i kernel (FEW = false) gives every thread two i-particles and all
// 128 j of a tile.  The few-i kernel (FEW = true) lets jl = 2, 4, .. 32 threads share one i-slot:
// the 256 slots of a CTA then hold 256 / jl particles, lane g of a slot takes the j-quads g, g + jl,
// g + 2 jl, .. of every tile (neighbouring lanes read neighbouring 16-byte pieces: no bank
// conflicts), and the jl partial sums meet in a shuffle butterfly before the CTA's partial is
// written.  Ring depth: the few-i kernel does little arithmetic per tile and lives on bytes in flight.
// few-i kernel: a ring stage holds KT consecutive tiles (one bulk copy, one wait, one release per KT
// tiles: with 8 j per thread and tile the per-tile ring work was as many instructions as the pairs)
__host__ __device__ constexpr int tiles_per_stage(bool few) { return few ? 4 : 1; }
__host__ __device__ constexpr int stages_for(bool few) { return few ? 2 : STAGES; }

// MODE 0: i-particles are members of the j-set, given by index (nb_force).  MODE 1: i-particles
// given by value, "a completely different set", acc + jerk + pot -- optionally with the
// index of the j-set member each one is and its flag (nb_force_ext_ids: the j-sharded scheme of
// PAPER.md:55); MODE 2: by value, acc + pot only (nb_force_ext).
// GUARD: the call's eps2 is below EPS2_GUARD (zero included): pairs with r = 0 are dropped inside the
// packed pair (R5, R6), so no tile needs the self-pair treatment.
// The few-i kernel also does the reduction (a4/a5): the last CTA to finish -- a ticket counter --
// sums the partials of all CTAs, so that such a call is ONE launch.
// The body takes the CTA's work item `work` (i-tile x j-subset) as an argument: force_kernel passes
// blockIdx.x, force_dyn_kernel (block steps queued without the host, nb_steps) loops over the items
// of a launch shape that was decided on the device.  DYN: the second form (the item is then carried
// in a register through the pair loop instead of being read from %ctaid again).
template <bool ATOMIC, bool FEW, int MODE, bool GUARD, bool DYN>
__device__ __forceinline__ void force_body(const ForceArgs& P, const ReduceArgs& R, const unsigned work,
                                           double* __restrict__ oacc, double* __restrict__ ojrk,
                                           double* __restrict__ opot)
{
    constexpr int STG = stages_for(FEW);
    constexpr int KT = tiles_per_stage(FEW);
    constexpr int STAGE_BYTES = KT * TILE_BYTES;
    constexpr bool JERK = (MODE != 2);
    constexpr int FT = (MODE == 2) ? 1 : NB_FLUSH_TILES;     // tiles per fp32 run of the all-i kernel (nb_internal.h)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* tiles = reinterpret_cast<float*>(smem_raw);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + STG * STAGE_BYTES);
    int* rel = reinterpret_cast<int*>(smem_raw + STG * STAGE_BYTES + STG * 8);
    // all-i kernel: the fp64 sums live in shared memory ([u][c][thread], touched once per tile)
    constexpr bool DSM = !FEW;
    double* sd = reinterpret_cast<double*>(smem_raw + STG * (STAGE_BYTES + 16)) + threadIdx.x;
    // index of each i (or -1), only needed in the masked path and in the tail: kept out of registers
    int* sidx = reinterpret_cast<int*>(smem_raw + STG * (STAGE_BYTES + 16) +
                                       (DSM ? IPT * NOUT * FORCE_THREADS * 8 : 0)) + threadIdx.x;

    const int tid = threadIdx.x;
    const int jsh = FEW ? P.jsh : 0;              // log2 of the threads per i-slot
    const int jl = 1 << jsh;
    const int jlane = tid & (jl - 1);
    const int it = work % P.n_itiles;             // neighbouring CTAs share the j-subset (L2 reuse)
    const int sp = work / P.n_itiles;
    const int t0 = (int)(((int64_t)P.ntiles * sp) / P.splits);
    const int t1 = (int)(((int64_t)P.ntiles * (sp + 1)) / P.splits);

    // a4: the j-subset of this CTA is tiles [t0, t1).  Thread 0 runs the copy ring.
    if (tid == 0) {
        for (int s = 0; s < STG; ++s) {
            mbar_init(smem_u32(&bars[s]), 1);
            rel[s] = 0;
        }
        mbar_fence_init();
        for (int s = 0; s < STG && t0 + s * KT < t1; ++s) {
            const int nt = t1 - (t0 + s * KT) < KT ? t1 - (t0 + s * KT) : KT;      // tiles are contiguous: one copy
            mbar_expect_tx(smem_u32(&bars[s]), nt * TILE_BYTES);
            bulk_g2s(smem_u32(tiles + s * KT * TILE_FLOATS), P.pack + (int64_t)(t0 + s * KT) * TILE_FLOATS,
                     nt * TILE_BYTES, smem_u32(&bars[s]));
        }
    }

    // a2: i-gather from the pack (two-float position = 48 bits, fp32 velocity; R8, R17)
    IPart I[IPT];
    unsigned iflags = 0;      // bit u: i-particle u carries the unsoftened flag (R7)
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int ku = it * (ITILE >> jsh) + ((u * FORCE_THREADS + tid) >> jsh);   // position inside the segment
        if (MODE != 0) {
            // by value: fp64 position split in two floats here, velocity rounded
            const bool on = P.k0 + ku < P.ni;
            const int64_t e = on ? P.k0 + ku : 0;
            float h[3], l[3], w[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double xc = P.ext_x[(int64_t)c * P.ni + e];
                h[c] = __double2float_rn(xc);
                l[c] = __double2float_rn(xc - (double)h[c]);
                w[c] = (MODE == 1) ? __double2float_rn(P.ext_v[(int64_t)c * P.ni + e]) : 0.0f;
            }
            I[u].nxh = dup(-h[0]); I[u].nyh = dup(-h[1]); I[u].nzh = dup(-h[2]);
            I[u].nxl = dup(-l[0]); I[u].nyl = dup(-l[1]); I[u].nzl = dup(-l[2]);
            I[u].nvx = dup(-w[0]); I[u].nvy = dup(-w[1]); I[u].nvz = dup(-w[2]);
            int self = -2;                               // -2: active, member of no tile
            if (MODE == 1 && on && P.ext_self) {
                const int q = P.ext_self[e];
                if (q >= 0 && q < P.n) self = q;
                if (P.any_flagged && P.ext_flags && (P.ext_flags[e] & 1)) iflags |= 1u << u;
            }
            sidx[u * FORCE_THREADS] = on ? self : -1;
            continue;
        }
        int q = (P.k0 + ku < P.ni) ? P.i_list[P.k0 + ku] : 0;
        const bool bad = (q < 0) || (q >= P.n);
        if (bad) {
            atomicOr(P.err, 1);
            q = 0;
        }
        sidx[u * FORCE_THREADS] = (P.k0 + ku < P.ni && !bad) ? q : -1;
        const float* b = P.pack + (int64_t)(q / TJ) * TILE_FLOATS + (q % TJ);
        I[u].nxh = dup(-b[P_XH * TJ]); I[u].nyh = dup(-b[P_YH * TJ]); I[u].nzh = dup(-b[P_ZH * TJ]);
        I[u].nxl = dup(-b[P_XL * TJ]); I[u].nyl = dup(-b[P_YL * TJ]); I[u].nzl = dup(-b[P_ZL * TJ]);
        I[u].nvx = dup(-b[P_VX * TJ]); I[u].nvy = dup(-b[P_VY * TJ]); I[u].nvz = dup(-b[P_VZ * TJ]);
        if (P.any_flagged && (P.flags[q] & 1)) iflags |= 1u << u;
    }

    const float2 eps2 = dup(P.eps2);
    const float2 m3 = dup(-3.0f);
    Acc32 A[IPT];
    double D[DSM ? 1 : IPT][NOUT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = make_float2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < NOUT; ++c) {
            if (DSM) sd[(u * NOUT + c) * FORCE_THREADS] = 0.0;
            else D[u][c] = 0.0;
        }
    }
    __syncthreads();   // barrier inits and the zeroed release counters visible to all warps

    // a3: pair loop over the tiles of the subset.  No CTA-wide barrier inside: a warp that is done
    // with a stage bumps the stage's release counter, and the warp that brings it to a multiple of
    // NWARPS (the last one out) refills the stage, so warps drift up to STG-1 tiles apart.
    for (int tg = t0; tg < t1; tg += KT) {
        const int st = ((tg - t0) / KT) % STG;
        mbar_wait(smem_u32(&bars[st]), (((tg - t0) / KT) / STG) & 1);
        const int tend = tg + KT < t1 ? tg + KT : t1;
        // does the stage hold the own index of one of my i-particles (R5)?  Once per stage, so that
        // the common tile pays nothing for it
        bool own = false;
        if (KT > 1 && (MODE == 1 || (MODE == 0 && !GUARD))) {
#pragma unroll
            for (int u = 0; u < IPT; ++u)
                own = own || (unsigned)(sidx[u * FORCE_THREADS] - tg * TJ) < (unsigned)((tend - tg) * TJ);
        }
#pragma unroll 1
        for (int t = tg; t < tend; ++t) {
        const float* T = tiles + (st * KT + (t - tg)) * TILE_FLOATS;

        // Flagged-flagged pairs (R7): the whole tile goes through the masked scalar pair, warp-uniform;
        // that path also excludes the self pair by index.  Every other tile is packed.
        constexpr int UNROLL_Q = NB_UNROLL;       // j-quads per trip of the pair loop
        const int nq = (TJ / 4) >> jsh;           // j-quads of a tile that are mine: jlane, jlane + jl, ..
        bool slow = false;
        if (iflags) slow = (P.tileflag[t >> 5] >> (t & 31)) & 1u;
        if (__any_sync(0xffffffffu, slow)) {
#pragma unroll 1
            for (int k = 0; k < nq; ++k) {
#pragma unroll 1
                for (int p = 4 * (jlane + (k << jsh)); p < 4 * (jlane + (k << jsh)) + 4; ++p) {
#pragma unroll
                    for (int u = 0; u < IPT; ++u)
                        pair1_masked(I[u], A[u], T, p, MODE != 2 && sidx[u * FORCE_THREADS] == t * TJ + p,
                                     (iflags >> u) & 1u, P.eps2);
                }
            }
        } else {
            // R5 (see pot_lane): when this tile holds the own index of one of my i-particles, in my
            // share of the tile, that particle's fp32 sums are moved to fp64 first, so that the pot
            // lane starts empty (the all-i kernel flushes after every tile anyway)
            if (FEW && own && (MODE == 1 || (MODE == 0 && !GUARD))) {
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    const int q = sidx[u * FORCE_THREADS] - t * TJ;
                    if ((unsigned)q < (unsigned)TJ && ((q >> 2) & (jl - 1)) == jlane) flush<1, JERK>(A[u], D[DSM ? 0 : u]);
                }
            }
            if (!FEW && FT > 1 && (MODE == 1 || (MODE == 0 && !GUARD))) {
                // sums run over FT tiles: the tile with the own index must start empty
#pragma unroll
                for (int u = 0; u < IPT; ++u)
                    if ((unsigned)(sidx[u * FORCE_THREADS] - t * TJ) < (unsigned)TJ)
                        flush<FORCE_THREADS, JERK>(A[u], sd + u * NOUT * FORCE_THREADS);
            }
            if (FEW) {
#pragma unroll 2
                for (int k = 0; k < nq; ++k) {
                    float4 f[10];
                    load_quad<JERK>(f, T, 4 * (jlane + (k << jsh)));
#pragma unroll
                    for (int u = 0; u < IPT; ++u) quad<JERK, GUARD>(I[u], A[u], f, eps2, m3);
                }
            } else {
#pragma unroll UNROLL_Q
                for (int p = 0; p < TJ; p += 4) {
                    float4 f[10];
                    load_quad<JERK>(f, T, p);
#pragma unroll
                    for (int u = 0; u < IPT; ++u) quad<JERK, GUARD>(I[u], A[u], f, eps2, m3);
                }
            }
            if ((KT == 1 || own) && (MODE == 1 || (MODE == 0 && !GUARD))) {
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    const int q = sidx[u * FORCE_THREADS] - t * TJ;
                    if ((unsigned)q < (unsigned)TJ && ((q >> 2) & (jl - 1)) == jlane) {
                        if (MODE == 1) {
                            // by value: the i-particle need not sit EXACTLY on the member it is (its
                            // state may come from another predictor), so r != 0 and the self pair
                            // would also leave m r eps^-3 in acc and jerk: this particle's share of
                            // the tile is summed again, pair by pair, without it
                            A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = make_float2(0.f, 0.f);
#pragma unroll 1
                            for (int k = 0; k < nq; ++k)
#pragma unroll 1
                                for (int e = 4 * (jlane + (k << jsh)); e < 4 * (jlane + (k << jsh)) + 4; ++e)
                                    pair1_masked(I[u], A[u], T, e, e == q, false, P.eps2);
                        } else {
                            const float ps = pot_lane(I[u], T, jlane, jsh, q, P.eps2);
                            if (q & 1) A[u].p.y = ps;
                            else A[u].p.x = ps;
                        }
                    }
                }
            }
        }
        // fp32 sums stay short before they move to fp64: a thread adds 64 / jl terms per lane and tile; the
        // all-i kernel flushes every FT tiles (128 terms), the few-i kernel every jl tiles (64)
        if ((!FEW && ((t - t0) & (FT - 1)) == FT - 1) || (FEW && ((t - t0) & (jl - 1)) == jl - 1) || t == t1 - 1) {
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                if (DSM) flush<FORCE_THREADS, JERK>(A[u], sd + u * NOUT * FORCE_THREADS);
                else flush<1, JERK>(A[u], D[DSM ? 0 : u]);
            }
        }

        }   // tiles of the stage

        // release the stage; the last warp out refills it with the tiles STG stages further on
        __syncwarp();
        if ((tid & 31) == 0) {
            __threadfence_block();     // this warp's reads of the stage are ordered before its release
            const int old = atomicAdd(&rel[st], 1);
            const int tn = tg + STG * KT;
            if ((old & (NWARPS - 1)) == NWARPS - 1 && tn < t1) {
                const int nt = t1 - tn < KT ? t1 - tn : KT;
                mbar_expect_tx(smem_u32(&bars[st]), nt * TILE_BYTES);
                bulk_g2s(smem_u32(tiles + st * KT * TILE_FLOATS), P.pack + (int64_t)tn * TILE_FLOATS, nt * TILE_BYTES,
                         smem_u32(&bars[st]));
            }
        }
    }

    // a4 inside the CTA: the jl lanes of one i add their sums (fixed butterfly: deterministic)
    if (FEW) {
        for (int w = 1; w < jl; w <<= 1) {
#pragma unroll
            for (int u = 0; u < IPT; ++u)
#pragma unroll
                for (int c = 0; c < NOUT; ++c) D[DSM ? 0 : u][c] += __shfl_xor_sync(0xffffffffu, D[DSM ? 0 : u][c], w);
        }
    }

    // the CTA's place in the grid is read again here, so that it does not hold registers through
    // the pair loop (the all-i kernel then fits 128 registers unspilled: 4 CTAs per SM)
    unsigned bid = work;
    if (!DYN) asm volatile("mov.u32 %0, %%ctaid.x;" : "=r"(bid));
    const int it2 = bid % P.n_itiles, sp2 = bid / P.n_itiles;

    // a4: partial sums of this j-subset (second kernel adds them), or atomics (:63)
    if (jlane == 0) {
#pragma unroll
        for (int u = 0; u < IPT; ++u) {
            double o[NOUT];
#pragma unroll
            for (int c = 0; c < NOUT; ++c) o[c] = DSM ? sd[(u * NOUT + c) * FORCE_THREADS] : D[DSM ? 0 : u][c];
            const int ku = it2 * (ITILE >> jsh) + ((u * FORCE_THREADS + tid) >> jsh);
            const int q = sidx[u * FORCE_THREADS];
            if (ATOMIC) {
                if (q != -1) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        atomicAdd(oacc + (int64_t)c * P.ni + P.k0 + ku, o[c]);
                        if (JERK) atomicAdd(ojrk + (int64_t)c * P.ni + P.k0 + ku, o[3 + c]);
                    }
                    atomicAdd(opot + P.k0 + ku, o[6]);
                }
            } else {
#pragma unroll
                for (int c = 0; c < NOUT; ++c)
                    P.part[P.part_i_fastest ? ((int64_t)c * P.splits + sp2) * P.ni_pad + ku      // [c][subset][i]
                                            : ((int64_t)c * P.ni_pad + ku) * P.splits + sp2] = o[c];    // [c][i][subset]
            }
        }
    }

    // a4/a5 in the same launch (few-i kernel): the CTA that draws the last ticket sums all partials
    if (FEW && !ATOMIC && P.reduce_here) {
        __shared__ int s_last;
        __threadfence();                      // my partials are visible before my ticket is drawn
        __syncthreads();
        if (tid == 0) {
            const unsigned ticket = atomicAdd(R.counter, 1u);
            s_last = ticket == gridDim.x - 1;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();                  // acquire: the other CTAs' partials
            for (int k = tid >> 5; k < R.ni; k += NWARPS) reduce_row<true>(R, k, tid & 31);
            if (tid == 0) *R.counter = 0u;    // ready for the next call on this stream
            // j-sharded call (nb_xforce): the same CTA exchanges with the peers (xchg.h)
            if (MODE == 1 && R.xchg) xchg_in_cta<FORCE_THREADS>(R, P.err, tid);
        }
    }
    if (DYN) {
        // the CTA goes on to its next work item, which sets the ring up again: every warp is done
        // with this one first, and a barrier is invalidated before it is initialised anew
        __syncthreads();
        if (tid == 0)
            for (int s = 0; s < STG; ++s) mbar_inval(smem_u32(&bars[s]));
    }
}

template <bool ATOMIC, bool FEW, int MODE, bool GUARD>
__global__ void __launch_bounds__(FORCE_THREADS, FEW ? NB_MINB_FEW : NB_MINB)
force_kernel(ForceArgs P, ReduceArgs R, double* __restrict__ oacc, double* __restrict__ ojrk,
             double* __restrict__ opot)
{
    pdl_wait();       // pdl.h: the pack and the partial buffers belong to earlier kernels until this returns
    force_body<ATOMIC, FEW, MODE, GUARD, false>(P, R, blockIdx.x, oacc, ojrk, opot);
}

// The pair kernel of a block whose size is only known on the device (nb_steps, steps.cu): the launch
// shape -- threads per i, i-tiles, j-subsets -- was written to *plan by plan_kernel; a fixed grid of
// resident CTAs loops over the work items.  Exits at once when no block is pending or when the plan
// asks for the other instantiation.
template <bool FEW, bool GUARD>
__global__ void __launch_bounds__(FORCE_THREADS, FEW ? NB_DYN_MINB : NB_DYN_MINB_ALL) force_dyn_kernel(DynPlan* __restrict__ plan)
{
    if (!plan->go) return;
    // the plan's segment for this instantiation: the block itself (fa), or -- few-i form only -- its tail (fb)
    const bool tail = FEW && plan->fa.jsh == 0 && plan->go_b;
    if ((plan->fa.jsh > 0) != FEW && !tail) return;
    __shared__ ForceArgs sP;
    __shared__ ReduceArgs sR;
    __shared__ unsigned s_w;
    if (threadIdx.x == 0) {
        sP = tail ? plan->fb : plan->fa;
        sR = plan->ra;
    }
    unsigned* const next = tail ? &plan->next_b : &plan->next;
    __syncthreads();
    // the first item of a CTA is its place in the grid; further items are drawn from a counter (the
    // plan kernel zeroed it), so that a CTA whose items ran long does not hold up the launch's tail
    const unsigned items = (unsigned)sP.n_itiles * (unsigned)sP.splits;
    unsigned w = blockIdx.x;
    while (w < items) {
        force_body<false, FEW, 0, GUARD, true>(sP, sR, w, nullptr, nullptr, nullptr);   // ends with a CTA barrier
        if (threadIdx.x == 0) s_w = gridDim.x + atomicAdd(next, 1u);
        __syncthreads();
        w = s_w;
        __syncthreads();
    }
}

// a4/a5 as a kernel of its own (all-i calls, atomics mode, fp64 and fused kernels)
template <bool WARP>
__global__ void __launch_bounds__(128) reduce_kernel(ReduceArgs R)
{
    pdl_wait();       // pdl.h
    if (!WARP && R.warp_rows > 0) {
        // the first CTAs take positions [0, ni - warp_rows) one per thread, the others the rest one per warp
        const int first = R.ni - R.warp_rows, ctas_a = (first + 127) / 128;
        if ((int)blockIdx.x >= ctas_a) {
            const int k = first + ((int)blockIdx.x - ctas_a) * 4 + (int)(threadIdx.x >> 5);
            if (k < R.ni) reduce_row<true, true>(R, k, threadIdx.x & 31);
        } else {
            const int k = blockIdx.x * blockDim.x + threadIdx.x;
            if (k < first) reduce_row<false>(R, k, threadIdx.x & 31);
        }
        return;
    }
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int k = WARP ? gt / 32 : gt;
    if (k >= R.ni) return;
    reduce_row<WARP>(R, k, threadIdx.x & 31);
}

// the reduction of a block planned on the device: one warp per i while the block is small and its
// j-subsets many, else one thread per i; the grid is sized for the largest block and exits early
__global__ void __launch_bounds__(128) reduce_dyn_kernel(const DynPlan* __restrict__ plan)
{
    if (!plan->go) return;
    __shared__ ReduceArgs sR;
    if (threadIdx.x == 0) sR = plan->ra;
    __syncthreads();
    // a grid of fixed, modest size strides over the block (it was launched before the block's size was known)
    const int64_t gt = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nthreads = (int64_t)gridDim.x * blockDim.x;
    const int most = sR.splits > sR.splits_b ? sR.splits : sR.splits_b;
    if (most > 8 && sR.ni <= 4096) {
        for (int64_t k = gt / 32; k < sR.ni; k += nthreads / 32) reduce_row<true>(sR, (int)k, threadIdx.x & 31);
    } else {
        // the positions of a tail segment (its hundreds of j-subsets) one warp each, the others one thread each
        const int64_t first = sR.ni - sR.warp_rows;
        for (int64_t k = gt; k < first; k += nthreads) reduce_row<false>(sR, (int)k, threadIdx.x & 31);
        for (int64_t k = first + gt / 32; k < sR.ni; k += nthreads / 32) reduce_row<true>(sR, (int)k, threadIdx.x & 31);
    }
}

__global__ void __launch_bounds__(256) zero_out_kernel(double* acc, double* jrk, double* pot, int64_t ni)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= ni) return;
    for (int c = 0; c < 3; ++c) {
        acc[c * ni + k] = 0.0;
        jrk[c * ni + k] = 0.0;
    }
    pot[k] = 0.0;
}

constexpr int NWARPS_CHECK = FORCE_THREADS / 32;
static_assert((NWARPS_CHECK & (NWARPS_CHECK - 1)) == 0, "warps per CTA must be a power of two");
__host__ __device__ constexpr int force_smem(bool few)
{
    return stages_for(few) * (tiles_per_stage(few) * TILE_BYTES + 16) + (few ? 0 : IPT * NOUT * FORCE_THREADS * 8) +
           IPT * FORCE_THREADS * 4;
}

}  // namespace

template <bool FEW>
cudaError_t setup_one(int* blocks, int* blocks_guard, int* blocks_dyn, int* blocks_dyn_guard)
{
    const void* k[8] = {(const void*)force_kernel<false, FEW, 0, false>, (const void*)force_kernel<true, FEW, 0, false>,
                        (const void*)force_kernel<false, FEW, 1, false>, (const void*)force_kernel<false, FEW, 2, false>,
                        (const void*)force_kernel<false, FEW, 0, true>,  (const void*)force_kernel<true, FEW, 0, true>,
                        (const void*)force_kernel<false, FEW, 1, true>,  (const void*)force_kernel<false, FEW, 2, true>};
    int least = 0;
    for (int q = 0; q < 8; ++q) {
        cudaError_t e = cudaFuncSetAttribute(k[q], cudaFuncAttributeMaxDynamicSharedMemorySize, force_smem(FEW));
        if (e != cudaSuccess) return e;
        int b = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k[q], FORCE_THREADS, force_smem(FEW));
        if (e != cudaSuccess) return e;
        if (q == 0 || b < least) least = b;
    }
    {
        const void* kd[2] = {(const void*)force_dyn_kernel<FEW, false>, (const void*)force_dyn_kernel<FEW, true>};
        int* out[2] = {blocks_dyn, blocks_dyn_guard};
        for (int q = 0; q < 2; ++q) {
            cudaError_t e = cudaFuncSetAttribute(kd[q], cudaFuncAttributeMaxDynamicSharedMemorySize, force_smem(FEW));
            if (e != cudaSuccess) return e;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(out[q], kd[q], FORCE_THREADS, force_smem(FEW));
            if (e != cudaSuccess) return e;
            if (*out[q] < least) least = *out[q];
        }
    }
    // the dispatcher sizes whole waves with the by-index kernels' residency; the others only need >= 1
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks, k[0], FORCE_THREADS, force_smem(FEW));
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_guard, k[4], FORCE_THREADS, force_smem(FEW));
    return (e == cudaSuccess && least < 1) ? cudaErrorLaunchOutOfResources : e;
}

// blocks_per_sm[0..3]: CTAs per SM of the all-i kernel, its guarded form, the few-i kernel, its guarded
// form; [4..7]: the same for the device-planned kernels of nb_steps (force_dyn_kernel)
cudaError_t force_kernel_setup(int* blocks_per_sm)
{
    cudaError_t e = setup_one<false>(blocks_per_sm + 0, blocks_per_sm + 1, blocks_per_sm + 4, blocks_per_sm + 5);
    if (e != cudaSuccess) return e;
    return setup_one<true>(blocks_per_sm + 2, blocks_per_sm + 3, blocks_per_sm + 6, blocks_per_sm + 7);
}

// mode: 0 = by index (nb_force), 1 = by value with jerk, 2 = by value, acc + pot only (nb_force_ext;
// no atomics variant there)
template <bool FEW, bool GUARD>
void launch_one(const ForceArgs& a, const ReduceArgs& r, int mode, int atomic_mode, double* acc, double* jrk,
                double* pot, cudaStream_t s)
{
    const unsigned grid = (unsigned)a.n_itiles * (unsigned)a.splits;
    if (mode == 1)
        pdl_launch(force_kernel<false, FEW, 1, GUARD>, grid, FORCE_THREADS, force_smem(FEW), s, a, r, acc, jrk, pot);
    else if (mode == 2)
        pdl_launch(force_kernel<false, FEW, 2, GUARD>, grid, FORCE_THREADS, force_smem(FEW), s, a, r, acc, jrk, pot);
    else if (atomic_mode)
        pdl_launch(force_kernel<true, FEW, 0, GUARD>, grid, FORCE_THREADS, force_smem(FEW), s, a, r, acc, jrk, pot);
    else
        pdl_launch(force_kernel<false, FEW, 0, GUARD>, grid, FORCE_THREADS, force_smem(FEW), s, a, r, acc, jrk, pot);
}

// a.jsh > 0 selects the few-i kernel, which also reduces (unless atomic_mode): r must then be complete
cudaError_t launch_force(const ForceArgs& a, const ReduceArgs& r, int mode, int atomic_mode, double* acc,
                         double* jrk, double* pot, cudaStream_t s)
{
    const bool guard = a.eps2 < EPS2_GUARD;
    if (a.jsh > 0) {
        if (guard) launch_one<true, true>(a, r, mode, atomic_mode, acc, jrk, pot, s);
        else launch_one<true, false>(a, r, mode, atomic_mode, acc, jrk, pot, s);
    } else {
        if (guard) launch_one<false, true>(a, r, mode, atomic_mode, acc, jrk, pot, s);
        else launch_one<false, false>(a, r, mode, atomic_mode, acc, jrk, pot, s);
    }
    return cudaGetLastError();
}

// both instantiations are queued; the plan decides on the device which one works
cudaError_t launch_force_dyn(DynPlan* plan, float eps2, int resident_all, int resident_few, cudaStream_t s)
{
    if (eps2 < EPS2_GUARD) {
        force_dyn_kernel<true, true><<<resident_few, FORCE_THREADS, force_smem(true), s>>>(plan);
        force_dyn_kernel<false, true><<<resident_all, FORCE_THREADS, force_smem(false), s>>>(plan);
    } else {
        force_dyn_kernel<true, false><<<resident_few, FORCE_THREADS, force_smem(true), s>>>(plan);
        force_dyn_kernel<false, false><<<resident_all, FORCE_THREADS, force_smem(false), s>>>(plan);
    }
    return cudaGetLastError();
}

cudaError_t launch_reduce_dyn(const DynPlan* plan, int64_t ni_max, cudaStream_t s)
{
    // one thread per i, or one warp per i up to 4096 particles: at most 1024 CTAs, which stride
    int64_t grid = ni_max <= 4096 ? (ni_max * 32 + 127) / 128 : 1024;
    if (grid < 1) grid = 1;
    if (grid > 1024) grid = 1024;
    reduce_dyn_kernel<<<(unsigned)grid, 128, 0, s>>>(plan);
    return cudaGetLastError();
}

cudaError_t launch_reduce(const ReduceArgs& a, cudaStream_t s)
{
    const int most = a.splits > a.splits_b ? a.splits : a.splits_b;
    const bool warp = !a.atomic_mode && most > 8 && a.ni <= 4096;
    const unsigned grid = warp ? (a.ni + 3) / 4
                               : (a.warp_rows > 0 ? (a.ni - a.warp_rows + 127) / 128 + (a.warp_rows + 3) / 4
                                                  : (a.ni + 127) / 128);
    return warp ? pdl_launch(reduce_kernel<true>, grid, 128, 0, s, a) : pdl_launch(reduce_kernel<false>, grid, 128, 0, s, a);
}

cudaError_t launch_zero_out(double* acc, double* jrk, double* pot, int64_t ni, cudaStream_t s)
{
    zero_out_kernel<<<(unsigned)((ni + 255) / 256), 256, 0, s>>>(acc, jrk, pot, ni);
    return cudaGetLastError();
}

}  // namespace nb
