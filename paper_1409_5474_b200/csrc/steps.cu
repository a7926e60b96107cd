// steps.cu -- nb_steps: many block steps in ONE persistent cooperative kernel, no host round trip and
// no kernel launch per step (SURVEY.md 8(f) NEXT-1 "a whole ph4-style step never leaves the GPU").
//
// PAPER.md:83 calls the host link "the crucial bottleneck"; PAPER.md:41/:49 describe block time steps
// in which "only the particles are updated that require a force update at a certain time", and
// PAPER.md:51 says a handful of active particles cannot hide latencies.  With individual steps most
// blocks ARE a handful of particles (median 4 at N = 16384), so a block step done as five launches
// plus a synchronisation (nb_step) is all latency.  Here one grid of at most one 512-thread CTA per
// SM runs the whole loop and meets at TWO grid-wide barriers per step:
//   A  each CTA scans its slice of the particles (their keys t_j + dt_j sit in shared memory) for
//      the slice's earliest time and publishes it with the particles due then, ascending   (R21)
//      -- barrier 1 --
//   B  every CTA reads the <= 148 published minima: the smallest is the block time t1, the slices
//      that attain it hold the due particles; concatenated in slice order the list is ascending,
//      as R21 states, without atomics.  A block that is too large for this kernel ends it here.
//   C  every CTA predicts the due particles (R1, R8), then streams ITS slice of the j-store once:
//      512 particles at a time are predicted into shared memory and the threads, arranged as
//      (i-particle, j-stride), evaluate the pairs in IEEE double (pair64.h: the same body as
//      nb_force_fused; self pair by index, flagged pairs unsoftened, R5..R7).  One partial sum per
//      CTA and i-particle, [7][N_i][CTAs].
//      -- barrier 2 --
//   D  the CTA that owns a due particle sums its partials (a warp per particle, fixed order:
//      deterministic, R9), stores the forces for nb_block_forces and runs the corrector and the
//      step criterion (correct_stored: R12, R18..R20; the particle's stored state was fetched while
//      waiting at barrier 2).  It then goes straight on to A of the next step, which only reads the
//      CTA's own slice.
// The kernel stops when its budget of steps is used up, when the next block time exceeds t_end, or
// when the next block is larger than it handles (N_i > STEPS_NI_MAX, N_i x N above the caller's
// bound, or more than STEPS_SLOT due particles in one slice): the host then takes that one block
// through nb_step's launches, where the packed fp32 pair kernel is faster, and starts the kernel
// again.  (t1, N_i) and a device time stamp of every step go to a device log.
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
constexpr int ST_KEYS = 2048;                 // keys of a slice kept in shared memory (else re-read)
constexpr int ST_GMAX = 256;                  // most CTAs (slices)

// dynamic shared memory: si [NI_MAX][6] | tile [7][512] | keys [ST_KEYS]
constexpr int ST_SMEM = STEPS_NI_MAX * 6 * 8 + NOUT * ST_TILE * 8 + ST_KEYS * 8;

// NB_STEPS_TRACE (development builds only): CTA 0 stamps %globaltimer at the phase boundaries of every
// step into the partial buffer's tail, 8 words per step
#ifdef NB_STEPS_TRACE
#define TRACE(k) do { if (P.trace && b == 0 && tid == 0) P.trace[s * 8 + (k)] = gtime(); } while (0)
#else
#define TRACE(k) do { } while (0)
#endif

__device__ __forceinline__ double ldcg(const double* p) { return __ldcg(p); }
__device__ __forceinline__ unsigned long long gtime()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// block-wide minimum of one key per thread (all threads get the result)
__device__ __forceinline__ unsigned long long block_min(unsigned long long k, unsigned long long* sw, int lane,
                                                        int warp)
{
#pragma unroll
    for (int w = 16; w >= 1; w >>= 1) {
        const unsigned long long o = __shfl_xor_sync(0xffffffffu, k, w);
        k = o < k ? o : k;
    }
    __syncthreads();                          // sw may still be read from the previous use
    if (lane == 0) sw[warp] = k;
    __syncthreads();
    k = sw[0];
#pragma unroll
    for (int w = 1; w < ST_WARPS; ++w) k = sw[w] < k ? sw[w] : k;
    return k;
}

// The particles of this CTA's slice whose key equals kmin, ascending, to dst[0 .. cap_dst): ordered
// compaction by ballots, 512 particles at a time.  Returns how many there are (may exceed cap_dst).
__device__ __forceinline__ int compact_due(const unsigned long long* keys, bool cached, const double* T,
                                           const double* dts, int64_t lo, int cnt_own, unsigned long long kmin,
                                           int32_t* dst, int cap_dst, int* swsum, int tid, int lane, int warp)
{
    int base = 0;
    for (int q0 = 0; q0 < cnt_own; q0 += ST_THREADS) {
        const int q = q0 + tid;
        bool due = false;
        if (q < cnt_own) due = (cached ? keys[q] : key_of(ldcg(T + lo + q) + ldcg(dts + lo + q))) == kmin;
        const unsigned bal = __ballot_sync(0xffffffffu, due);
        if (lane == 0) swsum[warp] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < ST_WARPS; ++w) {
            const int c = swsum[w];
            total += c;
            if (w < warp) before += c;
        }
        if (due) {
            const int pos = base + before + __popc(bal & ((1u << lane) - 1u));
            if (pos < cap_dst) dst[pos] = (int32_t)(lo + q);
        }
        base += total;
        __syncthreads();
    }
    return base;
}

__global__ void __launch_bounds__(ST_THREADS, 1) steps_kernel(StepsArgs P)
{
    cg::grid_group grid = cg::this_grid();
    extern __shared__ __align__(16) unsigned char dyn[];
    double (*si)[6] = reinterpret_cast<double (*)[6]>(dyn);
    double (*tile)[ST_TILE] = reinterpret_cast<double (*)[ST_TILE]>(dyn + STEPS_NI_MAX * 6 * 8);
    unsigned long long* keys = reinterpret_cast<unsigned long long*>(dyn + STEPS_NI_MAX * 6 * 8 + NOUT * ST_TILE * 8);
    __shared__ int sl[STEPS_NI_MAX];
    __shared__ unsigned char sfl[STEPS_NI_MAX], tfl[ST_TILE];
    __shared__ unsigned long long swmin[ST_WARPS];
    __shared__ int swsum[ST_WARPS];
    __shared__ int goff[ST_GMAX + 1];
    __shared__ __align__(16) int sfirst[ST_GMAX][4];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = (int)gridDim.x, b = (int)blockIdx.x;
    const int64_t n = P.n;
    const int64_t chunk = (n + G - 1) / G;
    const int64_t lo = (int64_t)b * chunk < n ? (int64_t)b * chunk : n;
    const int64_t hi = lo + chunk < n ? lo + chunk : n;
    const int cnt_own = (int)(hi - lo);
    const bool cached = chunk <= ST_KEYS;
    const double* __restrict__ T = P.st.f[F_T];
    volatile unsigned long long* meta = P.meta;
    StepsSlot* slots = P.slots;

    if (cached)
        for (int q = tid; q < cnt_own; q += ST_THREADS) keys[q] = key_of(ldcg(T + lo + q) + ldcg(P.dts + lo + q));
    __syncthreads();

    // queued batches (nb_steps): how many steps are left and where the log continues is read from
    // device memory, because the host queued this launch before it knew; every CTA reads the same
    // values (they were written before this launch)
    int64_t budget = P.budget;
    if (P.prog) {
        const long long done0 = P.prog->done;
        budget = P.prog->final ? 0 : P.prog->k - done0;
        if (budget <= 0) {                    // nothing left: close the last step's time stamp once
            if (b == 0 && tid == 0 && !P.prog->closed) {
                P.log_ns[done0] = gtime();
                P.prog->closed = 1;
            }
            return;
        }
        P.log_t += done0;
        P.log_ni += done0;
        P.log_ns += done0;
    }
    long long last_ni = 0;                    // size of the last block this launch completed
    for (int64_t s = 0; s <= budget; ++s) {
        if (b == 0 && tid == 0) P.log_ns[s] = gtime();
        if (s == budget) break;
        TRACE(0);

        // ---- A: earliest time of my slice and who is due then (R21) ----------------------------
        unsigned long long k = ~0ull;
        for (int q = tid; q < cnt_own; q += ST_THREADS) {
            const unsigned long long kq = cached ? keys[q] : key_of(ldcg(T + lo + q) + ldcg(P.dts + lo + q));
            k = kq < k ? kq : k;
        }
        const unsigned long long kmin = block_min(k, swmin, lane, warp);
        const int base = compact_due(keys, cached, T, P.dts, lo, cnt_own, kmin, slots[b].idx, STEPS_SLOT, swsum, tid,
                                     lane, warp);
        if (tid == 0) {
            slots[b].key = kmin;
            slots[b].count = base;
        }
        TRACE(1);
        grid.sync();                                                            // ---- barrier 1
        TRACE(2);

        // ---- B: the block time and the due list, from the published slices ---------------------
        unsigned long long kg = ~0ull;
        int cg_ = 0;
        if (tid < G) {
            // key, count and -- in the same round trip -- the first four published indices of the slice:
            // most blocks are a handful of particles, whose indices then need no second trip
            const int4 head = __ldcg(reinterpret_cast<const int4*>(&slots[tid].key));
            kg = ((unsigned long long)(unsigned)head.y << 32) | (unsigned)head.x;
            cg_ = head.z;
            *reinterpret_cast<int4*>(&sfirst[tid][0]) = __ldcg(reinterpret_cast<const int4*>(&slots[tid].idx[0]));
        }
        const unsigned long long kall = block_min(kg, swmin, lane, warp);
        const int mine = (tid < G && kg == kall && kall != ~0ull) ? cg_ : 0;
        int incl = mine;                      // inclusive scan over the block
#pragma unroll
        for (int w = 1; w < 32; w <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, incl, w);
            if (lane >= w) incl += o;
        }
        if (lane == 31) swsum[warp] = incl;
        const int trunc = __syncthreads_or(mine > STEPS_SLOT);
        int wbase = 0, ni_all = 0;
#pragma unroll
        for (int w = 0; w < ST_WARPS; ++w) {
            const int c = swsum[w];
            ni_all += c;
            if (w < warp) wbase += c;
        }
        if (tid < G) goff[tid] = wbase + incl - mine;
        if (tid == 0) goff[G] = ni_all;
        const double t1 = of_key(kall);
        const long long ni64 = ni_all;
        int reason = STEPS_RUNNING;
        if (ni64 == 0 || t1 != t1) reason = STEPS_STUCK;            // no particle, or every t + dt is NaN
        else if (!(t1 <= P.t_end)) reason = STEPS_T_END;
        else if (trunc || ni64 > STEPS_NI_MAX || ni64 > P.cap || ni64 * n > P.max_pairs) reason = STEPS_BIG;
        if (reason != STEPS_RUNNING) {        // uniform over the grid: everybody leaves
            if (reason == STEPS_BIG && ni64 <= P.cap) {
                // leave the whole ascending list for the host path: each slice that attains t1 writes
                // its due particles at its offset (the published lists stop at STEPS_SLOT entries)
                __syncthreads();              // goff complete
                if (__ldcg(&slots[b].key) == kall)
                    compact_due(keys, cached, T, P.dts, lo, cnt_own, kall, P.list + goff[b], (int)(P.cap - goff[b]),
                                swsum, tid, lane, warp);
            }
            if (b == 0 && tid == 0) {
                meta[4] = (unsigned long long)s;
                meta[5] = (unsigned long long)reason;
                meta[6] = kall;
                meta[7] = (unsigned long long)(reason == STEPS_BIG ? ni64 : last_ni);
                if (P.prog) {
                    P.prog->done += s;
                    P.prog->reason = reason;
                    if (reason != STEPS_BIG) {
                        P.prog->final = 1;
                        P.prog->closed = 1;   // log_ns[s] was stamped when this step began
                    }
                }
            }
            return;
        }
        const int ni = (int)ni64;
        if (b == 0 && tid == 0) {
            P.log_t[s] = t1;
            P.log_ni[s] = ni64;
        }
        // the stored state of my j-particle of the first tile is requested before anything else
        double rx[3], rv[3], ra[3], rj[3], rt = 0.0, rm = 0.0;
        int rfl = 0;
        if (lo + tid < hi) {
            const int64_t p = lo + tid;
            rt = ldcg(T + p);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                rx[c] = ldcg(P.st.f[F_X + c] + p);
                rv[c] = ldcg(P.st.f[F_VX + c] + p);
                ra[c] = ldcg(P.st.f[F_AX + c] + p);
                rj[c] = ldcg(P.st.f[F_JX + c] + p);
            }
            rm = ldcg(P.st.f[F_M] + p);
            rfl = P.any_flagged ? (P.flags[p] & 1) : 0;
        }
        __syncthreads();                      // goff complete
        if (tid < ni) {
            int g0 = 0, g1 = G;               // the last slice g with goff[g] <= tid holds entry tid
            while (g1 - g0 > 1) {
                const int gm = (g0 + g1) >> 1;
                if (goff[gm] <= tid) g0 = gm;
                else g1 = gm;
            }
            const int pos = tid - goff[g0];
            const int64_t i = pos < 4 ? sfirst[g0][pos] : __ldcg(&slots[g0].idx[pos]);
            sl[tid] = (int)i;
            // ---- C: predicted i-particles ...
            const double dti = t1 - ldcg(T + i);
#pragma unroll
            for (int c = 0; c < 3; ++c)
                predict1(ldcg(P.st.f[F_X + c] + i), ldcg(P.st.f[F_VX + c] + i), ldcg(P.st.f[F_AX + c] + i),
                         ldcg(P.st.f[F_JX + c] + i), dti, si[tid][c], si[tid][3 + c]);
            sfl[tid] = P.any_flagged ? (P.flags[i] & 1) : 0;
            if (b == 0) P.list[tid] = (int32_t)i;
        }
        TRACE(3);
        // ... and one pass over this CTA's j-slice
        const int ii = tid % ni, slice = tid / ni, nsl = ST_THREADS / ni;
        Acc64 A;
        A.ax = A.ay = A.az = A.jx = A.jy = A.jz = A.p = 0.0;
        for (int64_t base_j = lo; base_j < hi; base_j += ST_TILE) {
            const int64_t p = base_j + tid;
            if (p < hi) {
                if (base_j != lo) {           // later tiles: fetched here
                    rt = ldcg(T + p);
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        rx[c] = ldcg(P.st.f[F_X + c] + p);
                        rv[c] = ldcg(P.st.f[F_VX + c] + p);
                        ra[c] = ldcg(P.st.f[F_AX + c] + p);
                        rj[c] = ldcg(P.st.f[F_JX + c] + p);
                    }
                    rm = ldcg(P.st.f[F_M] + p);
                    rfl = P.any_flagged ? (P.flags[p] & 1) : 0;
                }
                const double dtj = t1 - rt;
#pragma unroll
                for (int c = 0; c < 3; ++c) predict1(rx[c], rv[c], ra[c], rj[c], dtj, tile[c][tid], tile[3 + c][tid]);
                tile[6][tid] = rm;
                tfl[tid] = (unsigned char)rfl;
            }
            __syncthreads();                  // tile (and, the first time, si / sfl / sl) complete
            const int cnt = (int)(hi - base_j < ST_TILE ? hi - base_j : ST_TILE);
            if (slice < nsl) {
                // my i-particle in registers: read from shared memory inside the loop its six doubles
                // (48-byte rows: bank conflicts) would make the pair loop shared-memory-bound
                double xi[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) xi[c] = si[ii][c];
                const bool ifl = sfl[ii] != 0;
                const int self = sl[ii] - (int)base_j;    // position of the own index in this tile, if any
#pragma unroll 2
                for (int q = slice; q < cnt; q += nsl) {
                    const double e2 = (ifl && tfl[q]) ? 0.0 : P.eps2;
                    pair64<true>(xi, A, tile[0][q], tile[1][q], tile[2][q], tile[3][q], tile[4][q], tile[5][q],
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

        // ---- D: the owner of a due particle sums its partials and corrects it ------------------
        // my due particles are entries [goff[b], goff[b+1]) of the list when my slice attains t1; a
        // warp takes one of them at a time and fetches its stored state BEFORE the barrier
        const int first = goff[b];
        const int mycnt = goff[b + 1] - first;
        Stored s0;
        if (warp < mycnt) s0 = load_stored(P.st, P.dts, sl[first + warp]);
        TRACE(4);
        grid.sync();                                                            // ---- barrier 2
        TRACE(5);
        for (int q = warp; q < mycnt; q += ST_WARPS) {
            const int64_t i = sl[first + q];
            if (q != warp) s0 = load_stored(P.st, P.dts, i);
            double o[NOUT];
#pragma unroll
            for (int c = 0; c < NOUT; ++c) o[c] = 0.0;
            // four partials per lane and component in flight (28 loads): the sum is all load latency
            for (int g0 = 0; g0 < G; g0 += 128) {
                double pv[4][NOUT];
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    const int g = g0 + 32 * w + lane;
#pragma unroll
                    for (int c = 0; c < NOUT; ++c)
                        pv[w][c] = g < G ? ldcg(P.part + ((int64_t)c * ni + first + q) * G + g) : 0.0;
                }
#pragma unroll
                for (int w = 0; w < 4; ++w)
#pragma unroll
                    for (int c = 0; c < NOUT; ++c) o[c] += pv[w][c];
            }
#pragma unroll
            for (int c = 0; c < NOUT; ++c)
#pragma unroll
                for (int w = 16; w >= 1; w >>= 1) o[c] += __shfl_xor_sync(0xffffffffu, o[c], w);
            if (lane == 0) {
#pragma unroll
                for (int c = 0; c < NOUT; ++c) P.out[(int64_t)c * ni + first + q] = o[c];
                const double d = correct_stored(P.st, P.dts, i, s0, t1, o, o + 3, P.eta, P.dt_min, P.dt_max, P.err);
                // the particle's new key; after a refused correction (zero step) the store is unchanged
                if (cached) keys[i - lo] = key_of((t1 - s0.t != 0.0 ? t1 : s0.t) + d);
            }
        }
        __syncthreads();                      // the new keys / (t, dt) of my slice are visible to my next scan
        TRACE(6);
        last_ni = ni64;
    }
    if (b == 0 && tid == 0) {
        meta[4] = (unsigned long long)budget;
        meta[5] = (unsigned long long)STEPS_DONE;
        meta[6] = 0ull;
        meta[7] = (unsigned long long)last_ni;
        if (P.prog) {
            P.prog->done += budget;
            P.prog->reason = STEPS_DONE;
            P.prog->closed = 1;
        }
    }
}

// After the persistent kernel: if it stopped at a block it does not take itself, plan that block's
// kernels -- threads per i, i-tiles, j-subsets, buffers -- in device memory, log it and count it as
// done (its kernels are queued right behind this one).  One thread.
__device__ __forceinline__ bool plan_block(const StepsArgs& P, DynPlan* plan, ForceArgs& fa, ReduceArgs& ra,
                                           int resident_all, int resident_few, size_t part_bytes);

// loop != 0: the kernel sits in the body of a graph's WHILE node and decides whether the body runs
// again (another round is needed while steps are left and nothing stopped the run)
__global__ void plan_kernel(StepsArgs P, DynPlan* plan, ForceArgs fa, ReduceArgs ra, int resident_all,
                            int resident_few, size_t part_bytes, cudaGraphConditionalHandle handle, int loop)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    P.prog->rounds += 1;
    plan_block(P, plan, fa, ra, resident_all, resident_few, part_bytes);
    if (loop) {
        const StepsProgress* g = P.prog;
        cudaGraphSetConditional(handle, (!g->final && g->done < g->k) ? 1u : 0u);
    }
}

__device__ __forceinline__ bool plan_block(const StepsArgs& P, DynPlan* plan, ForceArgs& fa, ReduceArgs& ra,
                                           int resident_all, int resident_few, size_t part_bytes)
{
    plan->go = 0;
    StepsProgress* g = P.prog;
    if (g->final || g->reason != STEPS_BIG || g->done >= g->k) return false;
    const long long ni = (long long)P.meta[7];
    if (ni > P.cap) {                         // the list was truncated: the host reports the error
        g->final = 1;
        g->pending_ni = ni;
        return false;
    }
    const double t1 = of_key(P.meta[6]);
    // launch shape (nb_api.cu force_impl does the same on the host for nb_force)
    int jsh = 0;
    while (jsh < JSH_MAX && (ITILE >> (jsh + 1)) >= ni) ++jsh;
    const int itile = ITILE >> jsh;
    const int n_itiles = (int)((ni + itile - 1) / itile);
    // a last i-tile that is at most half full becomes a segment of its own for the few-i instantiation
    // (the rule of nb_api.cu force_impl)
    int jsh_b = 0, itile_b = 0;
    if (NB_TAIL_SEGMENT && jsh == 0 && ni > ITILE && ni <= 16384) {
        const int rem = (int)(ni % ITILE);
        if (rem >= 1 && rem <= ITILE / 2) {
            int jb = 0;
            while (jb < JSH_MAX && (ITILE >> (jb + 1)) >= rem) ++jb;
            const int ib = ITILE >> jb;
            if ((double)fa.n * ((double)ITILE - 1.3 * ib) / 0.9e12 >= NB_TAIL_GAIN_NEEDED(ib, ni)) {
                jsh_b = jb;
                itile_b = ib;
            }
        }
    }
    const bool tail = itile_b > 0;
    const int tiles_a = tail ? n_itiles - 1 : n_itiles;
    const long long pad_a = (long long)tiles_a * itile;
    // j-subsets: the resident CTAs loop over tiles x S work items, so for every
    // number of waves w the best S is the largest one that still fits w waves; of those the one with
    // the best useful-tile fraction wins (each item also pays about half a tile of gather, pipeline fill
    // and partial store -- the model nb_api.cu choose_splits uses on the host)
    auto best_splits = [&](int tiles, int resident, size_t bytes, long long slots) -> long long {
        long long smax = (long long)(bytes / (NOUT * sizeof(double) * (size_t)slots));
        if (smax > fa.ntiles) smax = fa.ntiles;
        if (smax > 4096) smax = 4096;
        long long splits = 1;
        double best = -1.0;
        const long long w0 = (tiles + resident - 1) / resident;
        for (long long w = w0; w < w0 + 12; ++w) {
            long long sw = w * resident / tiles;
            if (sw > smax) sw = smax;
            if (sw < 1) sw = 1;
            const long long items = (long long)tiles * sw;
            const long long waves = (items + resident - 1) / resident;
            const long long per = (fa.ntiles + sw - 1) / sw;
            const double eff = (double)tiles * fa.ntiles / ((double)waves * resident * ((double)per + 0.5));
            // (no term for the number of waves here, unlike choose_splits: the resident CTAs of force_dyn_kernel
            // draw their items from a counter, which balances the SMs by itself)
            if (eff > best * 1.004) {
                best = eff;
                splits = sw;
            }
            if (sw == smax) break;
        }
        return splits;
    };
    // room for the tail's partials first: at most two waves of its CTAs
    size_t keep = 0;
    if (tail) {
        const long long sb_max = fa.ntiles < 2 * resident_few ? fa.ntiles : 2 * resident_few;
        keep = (size_t)NOUT * sizeof(double) * (size_t)itile_b * (size_t)sb_max;
    }
    const long long splits = best_splits(tiles_a, jsh > 0 ? resident_few : resident_all, part_bytes - keep, pad_a);
    fa.ni = (int)ni;
    fa.jsh = jsh;
    fa.k0 = 0;
    fa.n_itiles = tiles_a;
    fa.ni_pad = (int)pad_a;
    fa.splits = (int)splits;
    fa.reduce_here = 0;
    ra.kA = tail ? (int)pad_a : (int)ni;
    ra.ni = (int)ni;
    ra.ni_pad = fa.ni_pad;
    ra.splits = (int)splits;
    ra.jrk = ra.acc + 3 * ni;                 // the context's block forces: [7][ni]
    ra.pot = ra.acc + 6 * ni;
    ra.t_pred = t1;
    plan->go_b = 0;
    if (tail) {
        ForceArgs fb = fa;
        double* part_b = fa.part + (size_t)NOUT * (size_t)pad_a * (size_t)splits;
        const long long splits_b = best_splits(1, resident_few, part_bytes - (size_t)NOUT * sizeof(double) * (size_t)pad_a *
                                                                                  (size_t)splits, itile_b);
        fb.jsh = jsh_b;
        fb.k0 = (int)pad_a;
        fb.n_itiles = 1;
        fb.ni_pad = itile_b;
        fb.splits = (int)splits_b;
        fb.part = part_b;
        ra.part_b = part_b;
        ra.ni_pad_b = itile_b;
        ra.splits_b = (int)splits_b;
        const long long most = splits > splits_b ? splits : splits_b;
        ra.warp_rows = (most > 8 && ni <= 4096) ? 0 : (int)(ni - pad_a);      // force.cu reduce_dyn_kernel
        plan->fb = fb;
        plan->next_b = 0u;
        plan->go_b = 1;
    }
    plan->fa = fa;
    plan->ra = ra;
    plan->t1 = t1;
    plan->ni = ni;
    plan->next = 0u;
    plan->go = 1;
    P.log_t[g->done] = t1;
    P.log_ni[g->done] = ni;
    g->done += 1;
    g->closed = 0;                            // the step's closing time stamp is the next launch's first
    g->reason = STEPS_RUNNING;                // taken: a kernel that starts with nothing left must not see it again
    P.meta[7] = (unsigned long long)ni;       // for nb_block_forces after the batch
    return true;
}

// corrector of a device-planned block (hermite.cu correct_kernel with its arguments read from the plan)
__global__ void __launch_bounds__(128)
correct_dyn_kernel(StorePtrs st, double* __restrict__ dts, const DynPlan* __restrict__ plan, int64_t n, double eta,
                   double dt_min, double dt_max, int* err)
{
    if (!plan->go) return;
    const int64_t ni = plan->ni;
    // a grid of fixed, modest size strides over the block (launched before the block's size was known)
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < ni; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = plan->ra.i_list[k];
        if (i < 0 || i >= n) {
            atomicOr(err, 1);
            continue;
        }
        double a1[3], j1[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            a1[c] = plan->ra.acc[(int64_t)c * ni + k];
            j1[c] = plan->ra.jrk[(int64_t)c * ni + k];
        }
        correct_one(st, dts, i, plan->t1, a1, j1, eta, dt_min, dt_max, err);
    }
}

}  // namespace

cudaError_t steps_kernel_setup(int* blocks_per_sm)
{
    cudaError_t e = cudaFuncSetAttribute(steps_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ST_SMEM);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, steps_kernel, ST_THREADS, ST_SMEM);
}

// Grid: one CTA per SM, fewer when the set is small (at least 64 particles per slice).
cudaError_t launch_steps(const StepsArgs& a, int sm_count, cudaStream_t s)
{
    int64_t want = (a.n + 63) / 64;
    int grid = sm_count < ST_GMAX ? sm_count : ST_GMAX;
    if (want < grid) grid = (int)(want > 0 ? want : 1);
    StepsArgs copy = a;
    void* args[] = {(void*)&copy};
    return cudaLaunchCooperativeKernel((const void*)steps_kernel, dim3(grid), dim3(ST_THREADS), args, ST_SMEM, s);
}

cudaError_t launch_plan(const StepsArgs& a, DynPlan* plan, StepsProgress* prog, const ForceArgs& fa_base,
                        const ReduceArgs& ra_base, int resident_all, int resident_few, size_t part_bytes,
                        cudaStream_t s, unsigned long long cond_handle, int loop)
{
    StepsArgs copy = a;
    copy.prog = prog;
    plan_kernel<<<1, 32, 0, s>>>(copy, plan, fa_base, ra_base, resident_all, resident_few, part_bytes,
                                 (cudaGraphConditionalHandle)cond_handle, loop);
    return cudaGetLastError();
}

cudaError_t launch_correct_dyn(const StorePtrs& st, double* dts, const DynPlan* plan, int64_t n, int64_t ni_max,
                               double eta, double dt_min, double dt_max, int* err, cudaStream_t s)
{
    int64_t grid = (ni_max + 127) / 128;
    if (grid > 1184) grid = 1184;
    correct_dyn_kernel<<<(unsigned)grid, 128, 0, s>>>(st, dts, plan, n, eta, dt_min, dt_max, err);
    return cudaGetLastError();
}

}  // namespace nb
