// nb_api.cu -- the C-ABI of include/nb.h: context, argument checks, host dispatcher.
#include <math.h>
#include <new>
#include <stdio.h>
#include <string.h>
#include <vector>

#include <cstdlib>
#include "nb_internal.h"
#include "xchg.h"

using namespace nb;

struct nb_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int64_t n_max = 0, ni_max = 0, n_cap = 0, n = 0;

    // j-sharded calls (nb_xforce): this rank's exchange window and the peers' as mapped here (xchg.h)
    Xchg xchg_host{};                   // host copy of the descriptor; world == 0: no window
    Xchg* xchg_dev = nullptr;
    unsigned char* xchg_win = nullptr;
    unsigned* xchg_ticket = nullptr;
    bool xchg_ipc[XCHG_MAX_WORLD] = {}; // win[r] was opened from an IPC handle (closed by nb_xchg_destroy)
    unsigned xchg_epoch = 0;            // epoch of the last push
    int xchg_call = -1;                 // phase of the nb_xforce call in progress (-1: an ordinary force call)
    unsigned long long xchg_limit_ns = XCHG_LIMIT_NS;
    int sm_count = 148;
    int blocks_per_sm[8] = {1, 1, 1, 1, 1, 1, 1, 1};   // all-i kernel, its guarded form, few-i kernel, its guarded form; [4..7] the same for nb_steps' device-planned kernels

    // device memory: either one cudaMalloc'ed slab or the caller's workspace
    bool allocated = false, own_slab = false;
    unsigned char* slab = nullptr;
    size_t lent_bytes = 0;
    StorePtrs store{};
    float* pack = nullptr;
    uint8_t* flags = nullptr;
    uint32_t* tileflag = nullptr;
    int32_t* flag_list = nullptr;
    int32_t* flag_stage = nullptr;      // [2 x count] staging of nb_set_flags: indices, then values
    double* part = nullptr;
    size_t part_bytes = 0;
    int* err = nullptr;
    unsigned* ticket = nullptr;         // the few-i kernel's reduction ticket (zero between calls)
    int32_t* h_ilist = nullptr;   // device staging for the *_host force call
    double* h_out = nullptr;      // [7][ni_max]
    double* h_in = nullptr;       // [14][ni_pad] staging of nb_update_j_host
    int64_t ni_pad = 0;
    // block-step state (hermite.cu): per-particle step, the scheduler's list and meta words, and
    // the forces of the current block
    double* dts = nullptr;              // [n_cap]
    int32_t* blk_list = nullptr;        // [ni_pad]
    double* blk_out = nullptr;          // [7][ni_pad]
    unsigned long long* sel_meta = nullptr;   // [0] key of t1, [1] count
    int* sel_counts = nullptr;          // [SEL_MAX_BLOCKS]
    StepsSlot* steps_slots = nullptr;   // [256] (steps.cu)
    unsigned long long* steps_meta = nullptr;   // [8]
    double* steps_log_t = nullptr;      // device log of nb_steps, cudaMalloc'ed and grown on demand
    long long* steps_log_ni = nullptr;
    unsigned long long* steps_log_ns = nullptr;
    int64_t steps_log_cap = 0;
    int64_t steps_max_pairs = 15000000; // blocks with ni x n above this go through the packed fp32 pair kernel
    int steps_ok = -1;                  // -1 unknown, 0 the cooperative kernel cannot be resident, 1 fine
    DynPlan* steps_plan = nullptr;      // the device-planned launch shape of a handed-over block
    StepsProgress* steps_prog = nullptr;   // where a queued batch of nb_steps stands
    int steps_queue = -1;               // 0: host handover; 1: rounds queued ahead on the stream; 2: one graph with a WHILE node;
                                        // -1: by the size of the j-set (queue_mode)
    // the graph of mode 2 (built on first use, rebuilt when an argument baked into its kernels changes)
    cudaStream_t cap_stream = nullptr;
    cudaGraph_t steps_graph = nullptr;
    cudaGraphExec_t steps_exec = nullptr;
    int steps_graph_state = 0;          // 0 none yet, 1 usable, -1 cannot be built here (mode 1 is used)
    double steps_key[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const void* steps_key_ptr[3] = {nullptr, nullptr, nullptr};
    void* steps_pinned = nullptr;       // pinned: StepsProgress in / out, the exit words of the last kernel
    double blk_t = 0.0;                 // what the last nb_next_block returned
    int64_t blk_ni = -1;

    // full-double pair loop (force64.cu): fp64 tiles, allocated when the mode is first selected
    int precision = 0;
    double* pack64 = nullptr;
    int blocks_per_sm64 = 1;

    // 6th-order pair loop (force6.cu): tiles with the predicted acceleration, allocated when selected
    int order = 4;
    float* pack6 = nullptr;
    int blocks_per_sm6 = 1;

    int* err_pinned = nullptr;          // pinned, 256 B: [0] error latch copy; bytes 8..23: sel_meta copy; 32..63: nb_steps status;
                                        // 64..: StepsProgress sent, 128..: StepsProgress read back, 192..: exit words
    std::vector<int32_t> flagged;   // host copy of the flagged set (sorted)

    struct SplitMemo {
        int n_itiles = -1, ntiles = 0;
        int64_t ni_pad = 0;
        size_t part_bytes = 0;
        int64_t resident = 0;
        int tune = 0, splits = 1;
    };
    SplitMemo memo[8];
    int memo_next = 0;

    bool predicted = false;
    double t_pred = 0.0;
    int tune_splits = 0, tune_reduce = 0, tune_fused = 1;
    int64_t last[4] = {0, 0, 0, 0};
    int64_t launches = 0;

    // optional per-kernel timing (nb_set_profiling): a ring of event records on the context's
    // stream, drained into running sums by nb_kernel_times (or when the ring is full)
    bool prof = false;
    struct Rec {
        cudaEvent_t e[3] = {nullptr, nullptr, nullptr};   // kind 0: predict [0,1]; kind 1: pair [0,1], reduce [1,2]
        int kind = -1;
    };
    std::vector<Rec> ring;
    size_t ring_used = 0;
    double prof_ms[3] = {0, 0, 0};
    int64_t prof_n[3] = {0, 0, 0};
};

namespace {

constexpr size_t ALIGN = 256;
inline size_t up(size_t x, size_t a = ALIGN) { return (x + a - 1) / a * a; }

struct Layout {
    size_t store, pack, flags, tileflag, flag_list, flag_stage, part, err, ilist, out, in, dts, blk_list, blk_out,
        sel_meta, sel_counts, steps_slots, steps_meta, steps_plan, steps_prog, total;
    int64_t ni_pad;
    size_t part_bytes;
    int64_t n_cap;
};

Layout layout(int64_t n_max, int64_t ni_max)
{
    Layout L{};
    L.n_cap = (int64_t)up((size_t)(n_max > 0 ? n_max : 1), 2 * TJ);
    const int64_t ntiles = L.n_cap / TJ;
    const int64_t ni_pad = (int64_t)up((size_t)(ni_max > 0 ? ni_max : 1), ITILE);
    size_t off = 0;
    L.store = off; off += up((size_t)NFIELD * L.n_cap * sizeof(double));
    L.pack = off; off += up((size_t)ntiles * TILE_BYTES);
    L.flags = off; off += up((size_t)L.n_cap);
    L.tileflag = off; off += up((size_t)(ntiles + 31) / 32 * 4);
    L.flag_list = off; off += up((size_t)NB_MAX_FLAGGED * 4);
    L.flag_stage = off; off += up((size_t)4 * NB_MAX_FLAGGED * 4);    // (index, value) pairs of one nb_set_flags
    // partial sums: S * 7 * ni_pad doubles.  S = 1 needs 56 B per i; what is split is at most one wave
    // of i-tiles (the remainder segment, or a call that does not fill the chip once): room for 16
    // j-subsets of up to 640 i-tiles (160 SMs x 4 CTAs), so that such a call can fill whole waves
    // (with 4 x ni_pad an all-active call of 131072 particles was held to 4 subsets: 0.66 of the peak)
    {
        const size_t wave = (size_t)640 * ITILE;
        const size_t split_part = (size_t)ni_pad < wave ? (size_t)ni_pad : wave;
        L.part_bytes = (size_t)NOUT * sizeof(double) * ((size_t)2 * ni_pad + 15 * split_part);   // 2: the whole waves, two subsets
    }
    if (L.part_bytes < ((size_t)32 << 20)) L.part_bytes = (size_t)32 << 20;
    L.part = off; off += up(L.part_bytes);
    L.err = off; off += up(2 * sizeof(int));           // error latch, reduction ticket
    L.ilist = off; off += up((size_t)ni_pad * 4);
    L.out = off; off += up((size_t)NOUT * ni_pad * sizeof(double));
    L.in = off; off += up((size_t)NFIELD * ni_pad * sizeof(double));
    L.dts = off; off += up((size_t)L.n_cap * sizeof(double));
    L.blk_list = off; off += up((size_t)ni_pad * 4);
    L.blk_out = off; off += up((size_t)NOUT * ni_pad * sizeof(double));
    L.sel_meta = off; off += up(16);
    L.sel_counts = off; off += up((size_t)SEL_MAX_BLOCKS * 4);
    L.steps_slots = off; off += up((size_t)256 * sizeof(StepsSlot));
    L.steps_meta = off; off += up(8 * 8);
    L.steps_plan = off; off += up(sizeof(DynPlan));
    L.steps_prog = off; off += up(sizeof(StepsProgress));
    L.ni_pad = ni_pad;
    L.total = off;
    return L;
}

int ensure_alloc(nb_ctx* c)
{
    if (c->allocated) return NB_OK;
    const Layout L = layout(c->n_max, c->ni_max);
    if (c->slab) {
        if (c->lent_bytes < L.total) return NB_ERR_ALLOC;
    } else {
        if (cudaMalloc(&c->slab, L.total) != cudaSuccess) {
            cudaGetLastError();
            c->slab = nullptr;
            return NB_ERR_ALLOC;
        }
        c->own_slab = true;
    }
    // zero the store (never-written particles are m = 0 at the origin), flags and the latch
    if (cudaMemsetAsync(c->slab, 0, L.total, c->stream) != cudaSuccess) return NB_ERR_CUDA;
    c->n_cap = L.n_cap;
    for (int f = 0; f < NFIELD; ++f)
        c->store.f[f] = reinterpret_cast<double*>(c->slab + L.store) + (size_t)f * L.n_cap;
    c->pack = reinterpret_cast<float*>(c->slab + L.pack);
    c->flags = c->slab + L.flags;
    c->tileflag = reinterpret_cast<uint32_t*>(c->slab + L.tileflag);
    c->flag_list = reinterpret_cast<int32_t*>(c->slab + L.flag_list);
    c->flag_stage = reinterpret_cast<int32_t*>(c->slab + L.flag_stage);
    c->part = reinterpret_cast<double*>(c->slab + L.part);
    c->part_bytes = L.part_bytes;
    c->err = reinterpret_cast<int*>(c->slab + L.err);
    c->ticket = reinterpret_cast<unsigned*>(c->slab + L.err) + 1;
    c->h_ilist = reinterpret_cast<int32_t*>(c->slab + L.ilist);
    c->h_out = reinterpret_cast<double*>(c->slab + L.out);
    c->h_in = reinterpret_cast<double*>(c->slab + L.in);
    c->dts = reinterpret_cast<double*>(c->slab + L.dts);
    c->blk_list = reinterpret_cast<int32_t*>(c->slab + L.blk_list);
    c->blk_out = reinterpret_cast<double*>(c->slab + L.blk_out);
    c->sel_meta = reinterpret_cast<unsigned long long*>(c->slab + L.sel_meta);
    c->sel_counts = reinterpret_cast<int*>(c->slab + L.sel_counts);
    c->steps_slots = reinterpret_cast<StepsSlot*>(c->slab + L.steps_slots);
    c->steps_meta = reinterpret_cast<unsigned long long*>(c->slab + L.steps_meta);
    c->steps_plan = reinterpret_cast<DynPlan*>(c->slab + L.steps_plan);
    c->steps_prog = reinterpret_cast<StepsProgress*>(c->slab + L.steps_prog);
    c->ni_pad = L.ni_pad;
    c->allocated = true;
    return NB_OK;
}

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev)
    {
        cudaGetDevice(&prev);
        if (prev != dev) cudaSetDevice(dev);
        else prev = -1;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

constexpr size_t PROF_RING = 256;

// Sum the finished records into prof_ms / prof_n (synchronises the stream).
int prof_drain(nb_ctx* c)
{
    if (c->ring_used == 0) return NB_OK;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return NB_ERR_CUDA;
    for (size_t r = 0; r < c->ring_used; ++r) {
        nb_ctx::Rec& R = c->ring[r];
        float ms = 0.f;
        if (R.kind == 0) {
            if (cudaEventElapsedTime(&ms, R.e[0], R.e[1]) != cudaSuccess) return NB_ERR_CUDA;
            c->prof_ms[0] += ms; c->prof_n[0] += 1;
        } else if (R.kind == 1) {
            if (cudaEventElapsedTime(&ms, R.e[0], R.e[1]) != cudaSuccess) return NB_ERR_CUDA;
            c->prof_ms[1] += ms; c->prof_n[1] += 1;
            if (cudaEventElapsedTime(&ms, R.e[1], R.e[2]) != cudaSuccess) return NB_ERR_CUDA;
            c->prof_ms[2] += ms; c->prof_n[2] += 1;
        }
        R.kind = -1;
    }
    c->ring_used = 0;
    return NB_OK;
}

nb_ctx::Rec* prof_next(nb_ctx* c)
{
    if (!c->prof) return nullptr;
    if (c->ring_used == c->ring.size() && prof_drain(c) != NB_OK) return nullptr;
    return &c->ring[c->ring_used];
}

SrcPtrs make_src(const double* m, const double* x, const double* y, const double* z,
                 const double* vx, const double* vy, const double* vz, const double* ax,
                 const double* ay, const double* az, const double* jx, const double* jy,
                 const double* jz, const double* t)
{
    SrcPtrs s;
    const double* a[NFIELD] = {m, x, y, z, vx, vy, vz, ax, ay, az, jx, jy, jz, t};
    for (int f = 0; f < NFIELD; ++f) s.f[f] = a[f];
    return s;
}

// choose the number of j-subsets S so that (i-tiles x S) fills the chip.  Efficiency
// of a choice = useful tile-passes / (waves x resident CTAs x tiles per CTA).
int choose_splits_scan(const nb_ctx* c, int n_itiles, int ntiles, int64_t ni_pad, size_t part_bytes,
                       int64_t resident)
{
    int64_t smax = (int64_t)(part_bytes / (NOUT * sizeof(double) * (size_t)ni_pad));
    if (smax > ntiles) smax = ntiles;
    if (smax > 4096) smax = 4096;
    if (smax < 1) smax = 1;
    if (c->tune_splits > 0) return (int)(c->tune_splits < smax ? c->tune_splits : smax);
    int best = 1;
    double best_eff = -1.0;
    for (int64_t s = 1; s <= smax; ++s) {
        const int64_t ctas = (int64_t)n_itiles * s;
        const int64_t waves = (ctas + resident - 1) / resident;
        const int64_t per = (ntiles + s - 1) / s;
        // each CTA also pays a fixed cost of about half a tile (gather, pipeline fill, partial store; fitted:
        // with 2 tiles config 2 ran at 0.755, with 0.5 at 0.769, mean over a 114-point (N, N_i) sweep +0.5 %); and
        // the SMs do not all run at one speed, so a call of few waves ends with its slowest SM while many
        // short CTAs balance (measured at N = 2^20, N_i = 151552: 1 / 2 / 4 / 6 / 12 / 23 waves of equal
        // CTAs: 0.759 / 0.770 / 0.776 / 0.778 / 0.780 / 0.781 of the peak)
        const double eff = (double)n_itiles * ntiles / ((double)waves * resident * (per + 0.5)) *
                           (1.0 - 0.028 / pow((double)waves, 1.25));
        if (eff > best_eff * 1.004) {   // prefer fewer splits unless better by more than noise
            best_eff = eff;
            best = (int)s;
        }
    }
    return best;
}

int choose_splits(nb_ctx* c, int n_itiles, int ntiles, int64_t ni_pad, size_t part_bytes,
                  int64_t resident)
{
    // block steps call this with the same few shapes over and over: remember the last answers
    for (const nb_ctx::SplitMemo& q : c->memo)
        if (q.n_itiles == n_itiles && q.ntiles == ntiles && q.ni_pad == ni_pad && q.part_bytes == part_bytes &&
            q.resident == resident && q.tune == c->tune_splits)
            return q.splits;
    const int ans = choose_splits_scan(c, n_itiles, ntiles, ni_pad, part_bytes, resident);
    c->memo[c->memo_next] = {n_itiles, ntiles, ni_pad, part_bytes, resident, c->tune_splits, ans};
    c->memo_next = (c->memo_next + 1) % (int)(sizeof(c->memo) / sizeof(c->memo[0]));
    return ans;
}

// ext_x != NULL: i-particles by value (nb_force_ext); ext_v == NULL then means acc + pot only;
// ext_self / ext_flags: which member of the j-set each one is, and its flag (nb_force_ext_ids)
int force_impl(nb_ctx* c, const int32_t* i_list, int64_t ni, double eps2, double* acc, double* jrk,
               double* pot, const double* ext_x = nullptr, const double* ext_v = nullptr,
               const int32_t* ext_self = nullptr, const uint8_t* ext_flags = nullptr)
{
    const int kmode = ext_x ? (ext_v ? 1 : 2) : 0;
    const bool f64 = c->precision == 1;
    if (!c->predicted) return NB_ERR_STATE;
    c->last[0] = c->last[1] = c->last[2] = 0;
    if (ni == 0) return NB_OK;
    const int64_t n_launch = c->n > 0 ? c->n : 0;
    const bool ids = kmode == 1 && ext_self != nullptr;
    ForceArgs a{};
    a.pack = c->pack;
    a.i_list = i_list;
    a.ext_x = ext_x;
    a.ext_v = ext_v;
    a.ext_self = ext_self;
    a.ext_flags = ext_flags;
    a.flags = c->flags;
    a.tileflag = c->tileflag;
    a.err = c->err;
    a.ni = (int)ni;
    a.n = (int)n_launch;
    a.ntiles = (int)((n_launch + TJ - 1) / TJ);
    a.eps2 = (float)eps2;
    a.any_flagged = (c->flagged.empty() || !(kmode == 0 || ids)) ? 0 : 1;
    a.pack64 = c->pack64;
    a.eps2d = eps2;
    const int mode = (c->tune_reduce && kmode == 0 && !f64) ? 1 : 0;
    // few active i: 2, 4, .. 32 threads share one i-slot and split the j of a tile, so
    // that one CTA's 256 slots hold the smallest power of two >= ni particles (down to 8)
    int jsh = 0;
    if (!f64)
        while (jsh < JSH_MAX && (ITILE >> (jsh + 1)) >= ni) ++jsh;
    a.jsh = jsh;
    const int itile = ITILE >> jsh;
    const int n_itiles = (int)((ni + itile - 1) / itile);
    const bool guard = (float)eps2 < EPS2_GUARD;
    const int resident = c->sm_count * (f64 ? c->blocks_per_sm64 : c->blocks_per_sm[(jsh > 0 ? 2 : 0) + (guard ? 1 : 0)]);

    // the i-tiles are cut in two segments.  A = the largest multiple of the resident CTA
    // count, one j-subset each (whole waves of equal CTAs); B = the rest, whose j is split in S
    // subsets so that its CTAs fill the chip once more instead of leaving a ragged last wave.
    // (fewer than four whole waves are better cut finer as well: see choose_splits)
    int tiles_a = (c->tune_splits > 0 || n_itiles / resident < 4) ? 0 : (n_itiles / resident) * resident;
    int tiles_b = n_itiles - tiles_a;
    // Mid-size calls whose last i-tile is at most half full (N_i = 256 q + rem, rem <= 128): that tile would
    // cost a full pass over j for 256 slots.  It is taken out as a segment of its own for the few-i kernel
    // (2^jsh threads per i: 128 .. 8 slots per CTA), A = the q full tiles with j split by choose_splits --
    // when a 256-slot pass over j costs clearly more than the smaller one plus a launch (measured at
    // N = 131072: N_i = 288 / 320 went from 100 us to 74 / 82 us, at N = 2^20: N_i = 257 from 591 us to 325 us;
    // at N = 32768 a launch costs what the pass costs, so small j-sets keep one segment: the model's saving
    // must reach NB_TAIL_MIN_GAIN, nb_internal.h).  Above 4096
    // particles the reduction is one thread per i, which would add the tail's hundreds of j-subsets one
    // dependent load at a time (measured: +130 us at N_i = 4128): the tail's positions are then summed by
    // one warp each (ReduceArgs.warp_rows).  Beyond 16384 particles the tile is < 1.6 % of the call (measured at 16400 and 32800: -0.7 ... +2 %).
    int jsh_b = jsh, itile_b = itile, resident_b = resident;
    bool tail = false;
    if (!f64 && !mode && jsh == 0 && tiles_a == 0 && c->tune_splits == 0 && NB_TAIL_SEGMENT && ni > ITILE && ni <= 16384 &&
        a.ntiles > 0) {
        const int rem = (int)(ni % ITILE);
        if (rem >= 1 && rem <= ITILE / 2) {
            int jb = 0;
            while (jb < JSH_MAX && (ITILE >> (jb + 1)) >= rem) ++jb;
            const int ib = ITILE >> jb;
            const double saved_s = (double)n_launch * ((double)ITILE - 1.3 * ib) / 0.9e12;
            if (saved_s >= NB_TAIL_GAIN_NEEDED(ib, ni)) {
                tail = true;
                jsh_b = jb;
                itile_b = ib;
                tiles_a = n_itiles - 1;
                tiles_b = 1;
                resident_b = c->sm_count * c->blocks_per_sm[2 + (guard ? 1 : 0)];
            }
        }
    }
    const int64_t pad_a = (int64_t)tiles_a * itile, pad_b = (int64_t)tiles_b * itile_b;
    // A's whole waves run with two j-subsets when the partial-sum buffer has the room (it has, as nb_create
    // sizes it): twice as many, half as long CTAs balance the SMs better (measured on the headline call:
    // 1 / 2 / 4 subsets: 0.7880 / 0.7897 / 0.7904 of the peak)
    int splits_a = tiles_a > 0 ? 1 : 0, splits_b = 0;
    if (tiles_a > 0 && a.ntiles >= 64 &&
        (size_t)NOUT * sizeof(double) * ((size_t)2 * pad_a + (size_t)16 * pad_b) <= c->part_bytes)
        splits_a = 2;
    if (tail) {
        // room for the tail's partials first: at most two waves of its CTAs
        const int64_t sb_max = a.ntiles < 2 * resident_b ? a.ntiles : 2 * resident_b;
        const size_t keep = (size_t)NOUT * sizeof(double) * (size_t)pad_b * (size_t)sb_max;
        splits_a = choose_splits(c, tiles_a, a.ntiles, pad_a, c->part_bytes - keep, resident);
    }
    double* part_b = c->part + (size_t)NOUT * pad_a * splits_a;
    if (a.ntiles > 0 && tiles_b > 0) {
        const size_t left = c->part_bytes - (size_t)NOUT * sizeof(double) * (size_t)pad_a * splits_a;
        splits_b = choose_splits(c, tiles_b, a.ntiles, pad_b, left, resident_b);
    }
    if (a.ntiles == 0) splits_a = splits_b = 0;   // n == 0: the reduction of zero partials writes zeros

    ReduceArgs r{};
    r.part = c->part;
    r.part_b = part_b;
    r.kA = (int)pad_a;
    r.ni_pad_b = (int)pad_b;
    r.splits_b = splits_b;
    r.i_list = i_list;
    r.acc = acc;
    r.jrk = jrk;
    r.pot = pot;
    r.store = c->store;
    r.flags = c->flags;
    r.flag_list = c->flag_list;
    // the fp64 kernel handles flagged pairs itself; by-value calls have them only with ids
    r.nflag = (f64 || !(kmode == 0 || ids)) ? 0 : (int)c->flagged.size();
    r.ni = (int)ni;
    r.ni_pad = (int)pad_a;
    r.splits = splits_a;
    r.n = (int)n_launch;
    r.t_pred = c->t_pred;
    r.atomic_mode = (mode && a.ntiles > 0) ? 1 : 0;
    r.ext_x = ext_x;
    r.ext_v = ext_v;
    r.ext_self = ext_self;
    r.ext_flags = ext_flags;
    r.counter = c->ticket;
    // a handful of i: the few-i kernel's last CTA also reduces, the call is one launch
    const bool reduce_here = jsh > 0 && !mode && !f64 && a.ntiles > 0 && tiles_a == 0 && ni <= 16;
    a.reduce_here = reduce_here ? 1 : 0;
    // nb_xforce: the reducing CTA also exchanges with the peers (force.cu); otherwise two small kernels
    // after the reduction do (below)
    // the thread-per-i reduction (launch_reduce: few subsets or many particles) reads [c][subset][i],
    // which the pair kernel stores coalesced; the warp-per-i reduction strides over [c][i][subset]
    {
        const int most = splits_a > splits_b ? splits_a : splits_b;
        const bool warp_reduce = !r.atomic_mode && most > 8 && ni <= 4096;
        a.part_i_fastest = r.part_i_fastest = (!f64 && !reduce_here && !warp_reduce) ? 1 : 0;
        r.warp_rows = (tail && !warp_reduce && splits_b > 8) ? (int)(ni - pad_a) : 0;
    }
    const bool xchg = c->xchg_call >= 0;
    const bool direct = (kmode == 0 || kmode == 1) && !f64 && !mode && c->tune_splits == 0 && ni <= DIRECT_NI_MAX &&
                        a.ntiles > 0 &&
                        direct_terms_per_lane(a.ntiles, direct_grid(a.ntiles, c->sm_count)) <= 64;
    if (xchg && (reduce_here || direct)) {
        r.xchg = c->xchg_dev;
        r.xchg_epoch = c->xchg_epoch;
        r.xchg_phase = c->xchg_call;
        r.xchg_limit_ns = c->xchg_limit_ns;
    }

    int launched = 0;
    nb_ctx::Rec* rec = nullptr;
    // a handful of active particles (members of the j-set, or by value with jerk): the direct kernel
    // (direct.cu) streams the pack once, one launch; it keeps whole per-thread sums in fp32, so only
    // while they stay within R17's 64 terms
    if (direct) {
        const int grid = direct_grid(a.ntiles, c->sm_count);
        {
            const int nip = ni <= 1 ? 1 : (ni <= 2 ? 2 : (ni <= 4 ? 4 : 8));
            a.jsh = 0;
            a.k0 = 0;
            a.n_itiles = 1;
            a.ni_pad = nip;
            a.splits = grid;
            a.part = c->part;
            r.part = c->part;
            r.part_b = c->part;
            r.kA = (int)ni;
            r.ni_pad = nip;
            r.splits = grid;
            rec = prof_next(c);
            if (rec) cudaEventRecord(rec->e[0], c->stream);
            if (launch_direct(a, r, grid, c->stream) != cudaSuccess) return NB_ERR_CUDA;
            if (rec) {
                cudaEventRecord(rec->e[1], c->stream);
                cudaEventRecord(rec->e[2], c->stream);
                rec->kind = 1;
                c->ring_used += 1;
            }
            c->last[0] = grid;
            c->last[1] = grid;
            c->last[2] = 1;
            c->last[3] = 0;
            c->launches += 1;
            return NB_OK;
        }
    }
    if (a.ntiles > 0) {
        if (mode) {
            if (launch_zero_out(acc, jrk, pot, ni, c->stream) != cudaSuccess) return NB_ERR_CUDA;
            ++launched;
        }
        rec = prof_next(c);
        if (rec) cudaEventRecord(rec->e[0], c->stream);
        if (tiles_a > 0) {
            a.k0 = 0;
            a.jsh = jsh;
            a.n_itiles = tiles_a;
            a.ni_pad = (int)pad_a;
            a.splits = splits_a;
            a.part = c->part;
            if ((f64 ? launch_force64(a, kmode, c->stream)
                     : launch_force(a, r, kmode, mode, acc, jrk, pot, c->stream)) != cudaSuccess)
                return NB_ERR_CUDA;
            ++launched;
        }
        if (tiles_b > 0) {
            a.k0 = (int)pad_a;
            a.jsh = jsh_b;
            a.n_itiles = tiles_b;
            a.ni_pad = (int)pad_b;
            a.splits = splits_b;
            a.part = part_b;
            if ((f64 ? launch_force64(a, kmode, c->stream)
                     : launch_force(a, r, kmode, mode, acc, jrk, pot, c->stream)) != cudaSuccess)
                return NB_ERR_CUDA;
            ++launched;
        }
        if (rec) cudaEventRecord(rec->e[1], c->stream);
    }
    if (!reduce_here) {
        if (launch_reduce(r, c->stream) != cudaSuccess) return NB_ERR_CUDA;
        ++launched;
        if (xchg) {
            if (launch_xchg_push(c->xchg_dev, c->xchg_epoch, acc, jrk, pot, ni, c->xchg_ticket, c->stream) != cudaSuccess)
                return NB_ERR_CUDA;
            ++launched;
            if (c->xchg_call == 0) {
                if (launch_xchg_sum(c->xchg_dev, c->xchg_epoch, acc, jrk, pot, ni, c->err, c->xchg_limit_ns, c->stream) != cudaSuccess)
                    return NB_ERR_CUDA;
                ++launched;
            }
        }
    }
    if (rec) {
        cudaEventRecord(rec->e[2], c->stream);
        rec->kind = 1;
        c->ring_used += 1;
    }
    c->last[0] = tiles_b > 0 ? splits_b : splits_a;
    c->last[1] = (int64_t)tiles_a * splits_a + (int64_t)tiles_b * splits_b;
    c->last[2] = launched;
    c->last[3] = mode;
    c->launches += launched;
    return NB_OK;
}

void xchg_release(nb_ctx* c)
{
    for (int r = 0; r < XCHG_MAX_WORLD; ++r) {
        if (c->xchg_ipc[r] && c->xchg_host.win[r]) cudaIpcCloseMemHandle(c->xchg_host.win[r]);
        c->xchg_ipc[r] = false;
    }
    if (c->xchg_win) cudaFree(c->xchg_win);
    if (c->xchg_dev) cudaFree(c->xchg_dev);
    if (c->xchg_ticket) cudaFree(c->xchg_ticket);
    c->xchg_win = nullptr;
    c->xchg_dev = nullptr;
    c->xchg_ticket = nullptr;
    c->xchg_host = Xchg{};
    c->xchg_epoch = 0;
    cudaGetLastError();
}

}  // namespace

extern "C" {

const char* nb_version(void) { return "nb 0.1 (sm_100a)"; }

const char* nb_strerror(int status)
{
    switch (status) {
        case NB_OK: return "ok";
        case NB_ERR_ARG: return "invalid argument";
        case NB_ERR_ALLOC: return "allocation failed or workspace too small";
        case NB_ERR_CUDA: return "CUDA error";
        case NB_ERR_INDEX: return "particle index out of range";
        case NB_ERR_STATE: return "call out of order (predict before force; workspace before data)";
        case NB_ERR_ARCH: return "device is not compute capability 10.x";
        case NB_ERR_PEER: return "a peer rank did not answer the exchange in time";
        default: return "unknown status";
    }
}

size_t nb_workspace_bytes(int64_t n_max, int64_t ni_max)
{
    if (n_max < 0 || ni_max < 0) return 0;
    return layout(n_max, ni_max).total;
}

int nb_create(nb_ctx** out, int64_t n_max, int64_t ni_max, int device, void* stream)
{
    if (!out) return NB_ERR_ARG;
    *out = nullptr;
    if (n_max < 1 || ni_max < 1 || n_max >= ((int64_t)1 << 31) - 4 * TJ ||
        ni_max >= ((int64_t)1 << 31) - 4 * ITILE)
        return NB_ERR_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return NB_ERR_CUDA;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return NB_ERR_CUDA;
    if (prop.major != 10) return NB_ERR_ARCH;
    nb_ctx* c = new (std::nothrow) nb_ctx();
    if (!c) return NB_ERR_ALLOC;
    c->device = device;
    c->stream = (cudaStream_t)stream;
    c->n_max = n_max;
    c->ni_max = ni_max;
    c->sm_count = prop.multiProcessorCount;
    DeviceGuard g(device);
    if (force_kernel_setup(c->blocks_per_sm) != cudaSuccess || c->blocks_per_sm[0] < 1 || c->blocks_per_sm[1] < 1 ||
        c->blocks_per_sm[2] < 1 || c->blocks_per_sm[3] < 1) {
        cudaGetLastError();
        delete c;
        return NB_ERR_CUDA;
    }
    if (cudaMallocHost(&c->err_pinned, 256) != cudaSuccess) {
        cudaGetLastError();
        delete c;
        return NB_ERR_ALLOC;
    }
    *out = c;
    return NB_OK;
}

int nb_destroy(nb_ctx* c)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    cudaStreamSynchronize(c->stream);
    if (c->own_slab && c->slab) cudaFree(c->slab);
    if (c->pack64) cudaFree(c->pack64);
    if (c->pack6) cudaFree(c->pack6);
    if (c->steps_log_t) cudaFree(c->steps_log_t);
    if (c->steps_log_ni) cudaFree(c->steps_log_ni);
    if (c->steps_log_ns) cudaFree(c->steps_log_ns);
    if (c->steps_exec) cudaGraphExecDestroy(c->steps_exec);
    if (c->steps_graph) cudaGraphDestroy(c->steps_graph);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    xchg_release(c);
    if (c->err_pinned) cudaFreeHost(c->err_pinned);
    for (nb_ctx::Rec& R : c->ring)
        for (cudaEvent_t e : R.e)
            if (e) cudaEventDestroy(e);
    delete c;
    return NB_OK;
}

int nb_set_stream(nb_ctx* c, void* stream)
{
    if (!c) return NB_ERR_ARG;
    c->stream = (cudaStream_t)stream;
    return NB_OK;
}

int nb_set_workspace(nb_ctx* c, void* dev_ptr, size_t bytes)
{
    if (!c || !dev_ptr || ((uintptr_t)dev_ptr % ALIGN) != 0) return NB_ERR_ARG;
    if (c->allocated) return NB_ERR_STATE;
    if (bytes < layout(c->n_max, c->ni_max).total) return NB_ERR_ALLOC;
    c->slab = static_cast<unsigned char*>(dev_ptr);
    c->lent_bytes = bytes;
    c->own_slab = false;
    return NB_OK;
}

static int set_j_common(nb_ctx* c, int64_t first, int64_t count, const SrcPtrs& src, bool host)
{
    if (!c || first < 0 || count < 0 || first + count > c->n_max) return NB_ERR_ARG;
    for (int f = F_M; f <= F_VZ; ++f)
        if (!src.f[f] && count > 0) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (host) {
        for (int f = 0; f < NFIELD && count > 0; ++f) {
            cudaError_t e = src.f[f]
                ? cudaMemcpyAsync(c->store.f[f] + first, src.f[f], (size_t)count * sizeof(double),
                                  cudaMemcpyHostToDevice, c->stream)
                : cudaMemsetAsync(c->store.f[f] + first, 0, (size_t)count * sizeof(double), c->stream);
            if (e != cudaSuccess) return NB_ERR_CUDA;
        }
    } else {
        if (launch_set_j(c->store, src, first, count, c->stream) != cudaSuccess) return NB_ERR_CUDA;
        if (count > 0) c->launches += 1;
    }
    if (first + count > c->n) c->n = first + count;
    c->predicted = false;
    return NB_OK;
}

int nb_set_j(nb_ctx* c, int64_t first, int64_t count, const double* m, const double* x,
             const double* y, const double* z, const double* vx, const double* vy, const double* vz,
             const double* ax, const double* ay, const double* az, const double* jx,
             const double* jy, const double* jz, const double* t)
{
    return set_j_common(c, first, count, make_src(m, x, y, z, vx, vy, vz, ax, ay, az, jx, jy, jz, t),
                        false);
}

int nb_set_j_host(nb_ctx* c, int64_t first, int64_t count, const double* m, const double* x,
                  const double* y, const double* z, const double* vx, const double* vy,
                  const double* vz, const double* ax, const double* ay, const double* az,
                  const double* jx, const double* jy, const double* jz, const double* t)
{
    return set_j_common(c, first, count, make_src(m, x, y, z, vx, vy, vz, ax, ay, az, jx, jy, jz, t),
                        true);
}

int nb_update_j(nb_ctx* c, const int32_t* idx, int64_t count, const double* m, const double* x,
                const double* y, const double* z, const double* vx, const double* vy,
                const double* vz, const double* ax, const double* ay, const double* az,
                const double* jx, const double* jy, const double* jz, const double* t)
{
    if (!c || count < 0 || (count > 0 && !idx)) return NB_ERR_ARG;
    if (count == 0) return NB_OK;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    const SrcPtrs src = make_src(m, x, y, z, vx, vy, vz, ax, ay, az, jx, jy, jz, t);
    if (launch_update_j(c->store, src, idx, count, c->n, c->err, c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    c->launches += 1;
    c->predicted = false;
    return NB_OK;
}

int nb_update_j_host(nb_ctx* c, const int32_t* idx, int64_t count, const double* m, const double* x,
                     const double* y, const double* z, const double* vx, const double* vy,
                     const double* vz, const double* ax, const double* ay, const double* az,
                     const double* jx, const double* jy, const double* jz, const double* t)
{
    if (!c || count < 0 || count > c->ni_max || (count > 0 && !idx)) return NB_ERR_ARG;
    if (count == 0) return NB_OK;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    const SrcPtrs host = make_src(m, x, y, z, vx, vy, vz, ax, ay, az, jx, jy, jz, t);
    SrcPtrs dev{};
    if (cudaMemcpyAsync(c->h_ilist, idx, (size_t)count * 4, cudaMemcpyHostToDevice, c->stream) !=
        cudaSuccess)
        return NB_ERR_CUDA;
    for (int f = 0; f < NFIELD; ++f) {
        dev.f[f] = nullptr;
        if (!host.f[f]) continue;
        double* stage = c->h_in + (size_t)f * c->ni_pad;
        if (cudaMemcpyAsync(stage, host.f[f], (size_t)count * sizeof(double), cudaMemcpyHostToDevice,
                            c->stream) != cudaSuccess)
            return NB_ERR_CUDA;
        dev.f[f] = stage;
    }
    if (launch_update_j(c->store, dev, c->h_ilist, count, c->n, c->err, c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    c->launches += 1;
    c->predicted = false;
    return NB_OK;
}

int nb_clear(nb_ctx* c)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    if (c->allocated) {
        const Layout L = layout(c->n_max, c->ni_max);
        if (cudaMemsetAsync(c->slab, 0, L.part, c->stream) != cudaSuccess) return NB_ERR_CUDA;
        if (cudaMemsetAsync(c->dts, 0, (size_t)c->n_cap * sizeof(double), c->stream) != cudaSuccess)
            return NB_ERR_CUDA;
    }
    c->blk_ni = -1;
    c->n = 0;
    c->flagged.clear();
    c->predicted = false;
    return NB_OK;
}

int64_t nb_count(const nb_ctx* c) { return c ? c->n : (int64_t)NB_ERR_ARG; }

int nb_set_flags(nb_ctx* c, const int32_t* idx, const uint8_t* flags, int64_t count)
{
    if (!c || count < 0 || (count > 0 && (!idx || !flags))) return NB_ERR_ARG;
    if (count == 0) return NB_OK;
    std::vector<int32_t> next = c->flagged;
    for (int64_t k = 0; k < count; ++k) {
        if (idx[k] < 0 || idx[k] >= c->n_max) return NB_ERR_INDEX;
        size_t pos = 0;
        bool have = false;
        for (; pos < next.size(); ++pos)
            if (next[pos] == idx[k]) { have = true; break; }
        if ((flags[k] & 1) && !have) next.push_back(idx[k]);
        if (!(flags[k] & 1) && have) next.erase(next.begin() + pos);
    }
    if (next.size() > NB_MAX_FLAGGED) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    // one staged list of (index, value) for the old set (-> 0) and the new set (-> 1), scattered by a
    // small kernel; then the tile bitmap and the flagged list.  The sources are pageable host
    // vectors: cudaMemcpyAsync stages such a source before it returns, so they may die here.
    const int64_t ntiles = c->n_cap / TJ;
    std::vector<uint32_t> tf((size_t)(ntiles + 31) / 32, 0u);
    std::vector<int32_t> stage;
    for (int32_t i : c->flagged) stage.push_back(i);
    for (int32_t i : next) {
        stage.push_back(i);
        tf[(size_t)(i / TJ) >> 5] |= 1u << ((i / TJ) & 31);
    }
    const int cnt = (int)stage.size();
    for (int k = 0; k < cnt; ++k) stage.push_back(k < (int)c->flagged.size() ? 0 : 1);
    if (cnt > 0) {
        if (cudaMemcpyAsync(c->flag_stage, stage.data(), stage.size() * 4, cudaMemcpyHostToDevice,
                            c->stream) != cudaSuccess ||
            launch_set_flags(c->flags, c->flag_stage, cnt, c->stream) != cudaSuccess)
            return NB_ERR_CUDA;
        c->launches += 1;
    }
    if (cudaMemcpyAsync(c->tileflag, tf.data(), tf.size() * 4, cudaMemcpyHostToDevice, c->stream) !=
        cudaSuccess)
        return NB_ERR_CUDA;
    if (!next.empty() &&
        cudaMemcpyAsync(c->flag_list, next.data(), next.size() * 4, cudaMemcpyHostToDevice,
                        c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    c->flagged.swap(next);
    c->predicted = false;   // the pack carries the flag word
    return NB_OK;
}

int nb_predict(nb_ctx* c, double t)
{
    if (!c || !isfinite(t)) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    nb_ctx::Rec* rec = c->n > 0 ? prof_next(c) : nullptr;
    if (rec) cudaEventRecord(rec->e[0], c->stream);
    if (launch_predict(c->store, c->flags, c->pack, c->precision == 1 ? c->pack64 : nullptr,
                       c->order == 6 ? c->pack6 : nullptr, c->n, t, c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    if (rec) {
        cudaEventRecord(rec->e[1], c->stream);
        rec->kind = 0;
        c->ring_used += 1;
    }
    if (c->n > 0) c->launches += 1;
    c->predicted = true;
    c->t_pred = t;
    return NB_OK;
}

int nb_get_predicted(nb_ctx* c, int64_t first, int64_t count, double* out)
{
    if (!c || first < 0 || count < 0 || first + count > c->n || (count > 0 && !out)) return NB_ERR_ARG;
    if (!c->predicted) return NB_ERR_STATE;
    DeviceGuard g(c->device);
    if (launch_get_predicted(c->store, first, count, c->t_pred, out, c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    if (count > 0) c->launches += 1;
    return NB_OK;
}

int nb_force(nb_ctx* c, const int32_t* i_list, int64_t ni, double eps2, double* acc, double* jrk,
             double* pot)
{
    if (!c || ni < 0 || ni > c->ni_max || !isfinite(eps2) || eps2 < 0.0) return NB_ERR_ARG;
    if (ni > 0 && (!i_list || !acc || !jrk || !pot)) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    return force_impl(c, i_list, ni, eps2, acc, jrk, pot);
}

int nb_force_ext(nb_ctx* c, int64_t ni, const double* x, const double* v, double eps2, double* acc,
                 double* jrk, double* pot)
{
    if (!c || ni < 0 || ni > c->ni_max || !isfinite(eps2) || eps2 < 0.0) return NB_ERR_ARG;
    if (ni > 0 && (!x || !acc || !pot)) return NB_ERR_ARG;
    if ((v == nullptr) != (jrk == nullptr)) return NB_ERR_ARG;     // jerk needs velocities, and only then
    DeviceGuard g(c->device);
    return force_impl(c, nullptr, ni, eps2, acc, jrk, pot, x, v);
}

int nb_force_ext_ids(nb_ctx* c, int64_t ni, const double* x, const double* v, const int32_t* self_idx,
                     const uint8_t* iflags, double eps2, double* acc, double* jrk, double* pot)
{
    if (!c || ni < 0 || ni > c->ni_max || !isfinite(eps2) || eps2 < 0.0) return NB_ERR_ARG;
    if (ni > 0 && (!x || !v || !self_idx || !acc || !jrk || !pot)) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    return force_impl(c, nullptr, ni, eps2, acc, jrk, pot, x, v, self_idx, iflags);
}

int nb_xchg_create(nb_ctx* c, int rank, int world, int64_t ni_cap)
{
    if (!c || world < 1 || world > XCHG_MAX_WORLD || rank < 0 || rank >= world || ni_cap < 1 || ni_cap > c->ni_max)
        return NB_ERR_ARG;
    DeviceGuard g(c->device);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return NB_ERR_CUDA;
    xchg_release(c);
    const size_t bytes = (size_t)XCHG_HDR + (size_t)2 * world * NOUT * (size_t)ni_cap * sizeof(double);
    if (cudaMalloc(&c->xchg_win, bytes) != cudaSuccess || cudaMalloc(&c->xchg_dev, sizeof(Xchg)) != cudaSuccess ||
        cudaMalloc(&c->xchg_ticket, sizeof(unsigned)) != cudaSuccess) {
        xchg_release(c);
        return NB_ERR_ALLOC;
    }
    c->xchg_host.rank = rank;
    c->xchg_host.world = world;
    c->xchg_host.ni_cap = ni_cap;
    c->xchg_host.win[rank] = c->xchg_win;
    if (cudaMemset(c->xchg_win, 0, bytes) != cudaSuccess || cudaMemset(c->xchg_ticket, 0, sizeof(unsigned)) != cudaSuccess ||
        cudaMemcpy(c->xchg_dev, &c->xchg_host, sizeof(Xchg), cudaMemcpyHostToDevice) != cudaSuccess) {
        xchg_release(c);
        return NB_ERR_CUDA;
    }
    return NB_OK;
}

int nb_xchg_export(nb_ctx* c, unsigned char* handle, void** dev_ptr)
{
    if (!c || (!handle && !dev_ptr)) return NB_ERR_ARG;
    if (!c->xchg_win) return NB_ERR_STATE;
    DeviceGuard g(c->device);
    if (handle) {
        static_assert(sizeof(cudaIpcMemHandle_t) == NB_XCHG_HANDLE_BYTES, "IPC handle size");
        cudaIpcMemHandle_t h;
        if (cudaIpcGetMemHandle(&h, c->xchg_win) != cudaSuccess) {
            cudaGetLastError();
            return NB_ERR_CUDA;
        }
        memcpy(handle, &h, sizeof(h));
    }
    if (dev_ptr) *dev_ptr = c->xchg_win;
    return NB_OK;
}

int nb_xchg_attach(nb_ctx* c, int peer, const unsigned char* handle, void* same_process_ptr)
{
    if (!c) return NB_ERR_ARG;
    if (!c->xchg_win) return NB_ERR_STATE;
    if (peer < 0 || peer >= c->xchg_host.world || (!handle == !same_process_ptr)) return NB_ERR_ARG;
    if (peer == c->xchg_host.rank) return NB_OK;           // my own window is attached by nb_xchg_create
    DeviceGuard g(c->device);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return NB_ERR_CUDA;
    if (c->xchg_ipc[peer] && c->xchg_host.win[peer]) cudaIpcCloseMemHandle(c->xchg_host.win[peer]);
    c->xchg_ipc[peer] = false;
    c->xchg_host.win[peer] = nullptr;
    if (handle) {
        cudaIpcMemHandle_t h;
        memcpy(&h, handle, sizeof(h));
        void* p = nullptr;
        if (cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
            cudaGetLastError();
            return NB_ERR_CUDA;
        }
        c->xchg_host.win[peer] = static_cast<unsigned char*>(p);
        c->xchg_ipc[peer] = true;
    } else {
        // a window of another context of THIS process; on another device peer access is switched on
        cudaPointerAttributes at{};
        if (cudaPointerGetAttributes(&at, same_process_ptr) != cudaSuccess || at.type != cudaMemoryTypeDevice) {
            cudaGetLastError();
            return NB_ERR_ARG;
        }
        if (at.device != c->device) {
            const cudaError_t e = cudaDeviceEnablePeerAccess(at.device, 0);
            if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) {
                cudaGetLastError();
                return NB_ERR_CUDA;
            }
            cudaGetLastError();
        }
        c->xchg_host.win[peer] = static_cast<unsigned char*>(same_process_ptr);
    }
    if (cudaMemcpy(c->xchg_dev, &c->xchg_host, sizeof(Xchg), cudaMemcpyHostToDevice) != cudaSuccess) return NB_ERR_CUDA;
    return NB_OK;
}

int nb_xchg_set_timeout(nb_ctx* c, double seconds)
{
    if (!c || !(seconds > 0.0) || seconds > 3600.0) return NB_ERR_ARG;
    c->xchg_limit_ns = (unsigned long long)(seconds * 1e9);
    return NB_OK;
}

int nb_xchg_destroy(nb_ctx* c)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    cudaStreamSynchronize(c->stream);
    xchg_release(c);
    return NB_OK;
}

int nb_xforce(nb_ctx* c, int phase, int64_t ni, const double* x, const double* v, const int32_t* self_idx,
              const uint8_t* iflags, double eps2, double* acc, double* jrk, double* pot)
{
    if (!c || phase < 0 || phase > 2 || ni < 0 || !isfinite(eps2) || eps2 < 0.0) return NB_ERR_ARG;
    if (!c->xchg_win) return NB_ERR_STATE;
    for (int r = 0; r < c->xchg_host.world; ++r)
        if (!c->xchg_host.win[r]) return NB_ERR_STATE;   // a peer's window is not attached yet
    if (ni > c->xchg_host.ni_cap) return NB_ERR_ARG;
    if (ni > 0 && (!acc || !jrk || !pot || (phase != 2 && (!x || !v)))) return NB_ERR_ARG;
    if (c->precision != 0 || c->tune_reduce != 0) return NB_ERR_STATE;   // mixed precision, partial-sum reduction
    if (ni == 0) return NB_OK;
    DeviceGuard g(c->device);
    if (phase == 2) {
        // the other half of a phase-1 call: wait for the peers' pushes of that epoch, add in rank order
        if (c->xchg_epoch == 0) return NB_ERR_STATE;
        if (launch_xchg_sum(c->xchg_dev, c->xchg_epoch, acc, jrk, pot, ni, c->err, c->xchg_limit_ns, c->stream) != cudaSuccess)
            return NB_ERR_CUDA;
        c->launches += 1;
        return NB_OK;
    }
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (!c->predicted) return NB_ERR_STATE;
    c->xchg_epoch += 1;
    if (c->xchg_epoch == 0) c->xchg_epoch = 2;     // 0 is the windows' initial flag value; parity keeps alternating
    c->xchg_call = phase;
    rc = force_impl(c, nullptr, ni, eps2, acc, jrk, pot, x, v, self_idx, iflags);
    c->xchg_call = -1;
    return rc;
}

int nb_force_host(nb_ctx* c, const int32_t* i_list, int64_t ni, double eps2, double* acc,
                  double* jrk, double* pot)
{
    if (!c || ni < 0 || ni > c->ni_max || !isfinite(eps2) || eps2 < 0.0) return NB_ERR_ARG;
    if (ni > 0 && (!i_list || !acc || !jrk || !pot)) return NB_ERR_ARG;
    if (!c->predicted) return NB_ERR_STATE;
    if (ni == 0) return nb_sync(c);
    DeviceGuard g(c->device);
    if (cudaMemcpyAsync(c->h_ilist, i_list, (size_t)ni * 4, cudaMemcpyHostToDevice, c->stream) !=
        cudaSuccess)
        return NB_ERR_CUDA;
    double* d_acc = c->h_out;
    double* d_jrk = c->h_out + 3 * ni;
    double* d_pot = c->h_out + 6 * ni;
    int rc = force_impl(c, c->h_ilist, ni, eps2, d_acc, d_jrk, d_pot);
    if (rc != NB_OK) return rc;
    const size_t b = (size_t)ni * sizeof(double);
    if (cudaMemcpyAsync(acc, d_acc, 3 * b, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(jrk, d_jrk, 3 * b, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(pot, d_pot, b, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    return nb_sync(c);
}

int nb_set_precision(nb_ctx* c, int mode)
{
    if (!c || (mode != 0 && mode != 1)) return NB_ERR_ARG;
    if (mode == c->precision) return NB_OK;
    DeviceGuard g(c->device);
    if (mode == 1 && !c->pack64) {
        int rc = ensure_alloc(c);
        if (rc != NB_OK) return rc;
        if (force64_kernel_setup(&c->blocks_per_sm64) != cudaSuccess || c->blocks_per_sm64 < 1) {
            cudaGetLastError();
            return NB_ERR_CUDA;
        }
        const size_t bytes = (size_t)(c->n_cap / TJ) * TILE64_BYTES;
        if (cudaMalloc(&c->pack64, bytes) != cudaSuccess) {
            cudaGetLastError();
            c->pack64 = nullptr;
            return NB_ERR_ALLOC;
        }
    }
    c->precision = mode;
    c->predicted = false;      // the tiles of the new mode are written by the next nb_predict
    return NB_OK;
}

int nb_set_order(nb_ctx* c, int order)
{
    if (!c || (order != 4 && order != 6)) return NB_ERR_ARG;
    if (order == c->order) return NB_OK;
    DeviceGuard g(c->device);
    if (order == 6 && !c->pack6) {
        int rc = ensure_alloc(c);
        if (rc != NB_OK) return rc;
        if (force6_kernel_setup(&c->blocks_per_sm6) != cudaSuccess || c->blocks_per_sm6 < 1) {
            cudaGetLastError();
            return NB_ERR_CUDA;
        }
        if (cudaMalloc(&c->pack6, (size_t)(c->n_cap / TJ) * TILE6_BYTES) != cudaSuccess) {
            cudaGetLastError();
            c->pack6 = nullptr;
            return NB_ERR_ALLOC;
        }
    }
    c->order = order;
    c->predicted = false;      // the tiles of the new order are written by the next nb_predict
    return NB_OK;
}

int nb_force6(nb_ctx* c, const int32_t* i_list, int64_t ni, double eps2, double* acc, double* jrk, double* snp,
              double* pot)
{
    if (!c || ni < 0 || ni > c->ni_max || !isfinite(eps2) || eps2 < 0.0) return NB_ERR_ARG;
    if (ni > 0 && (!i_list || !acc || !jrk || !snp || !pot)) return NB_ERR_ARG;
    if (c->order != 6 || !c->predicted) return NB_ERR_STATE;
    if (ni == 0) return NB_OK;
    DeviceGuard g(c->device);
    const int64_t n_launch = c->n > 0 ? c->n : 0;
    Force6Args a{};
    a.pack6 = c->pack6;
    a.i_list = i_list;
    a.part = c->part;
    a.flags = c->flags;
    a.err = c->err;
    a.ni = (int)ni;
    a.n = (int)n_launch;
    a.ntiles = (int)((n_launch + TJ - 1) / TJ);
    a.n_itiles = (int)((ni + ITILE - 1) / ITILE);
    a.ni_pad = a.n_itiles * ITILE;
    a.eps2 = (float)eps2;
    a.any_flagged = c->flagged.empty() ? 0 : 1;
    // j split in subsets while the i-tiles alone do not fill the chip; 10 sums per i
    const int resident = c->sm_count * c->blocks_per_sm6;
    a.splits = 1;
    // (also for a few waves of i-tiles, whose ragged last wave and slowest SM would set the time: choose_splits)
    if (a.ntiles > 0 && a.n_itiles < 4 * resident)
        a.splits = choose_splits(c, a.n_itiles, a.ntiles, a.ni_pad, c->part_bytes * NOUT / 10, resident);
    nb_ctx::Rec* rec = prof_next(c);
    if (rec) cudaEventRecord(rec->e[0], c->stream);
    if (launch_force6(a, c->store, c->flag_list, (int)c->flagged.size(), c->t_pred, acc, jrk, snp, pot, c->stream) !=
        cudaSuccess)
        return NB_ERR_CUDA;
    if (rec) {                                // pair kernel and its reduction are timed together here
        cudaEventRecord(rec->e[1], c->stream);
        cudaEventRecord(rec->e[2], c->stream);
        rec->kind = 1;
        c->ring_used += 1;
    }
    c->last[0] = a.splits;
    c->last[1] = (int64_t)a.n_itiles * a.splits;
    c->last[2] = 2;
    c->last[3] = 0;
    c->launches += 2;
    return NB_OK;
}

int nb_set_tuning(nb_ctx* c, int j_splits, int reduce_mode)
{
    if (!c || j_splits < 0 || reduce_mode < 0 || reduce_mode > 1) return NB_ERR_ARG;
    c->tune_splits = j_splits;
    c->tune_reduce = reduce_mode;
    return NB_OK;
}

int nb_set_fused(nb_ctx* c, int on)
{
    if (!c) return NB_ERR_ARG;
    c->tune_fused = on ? 1 : 0;
    return NB_OK;
}

int nb_last_launch(const nb_ctx* c, int64_t* out)
{
    if (!c || !out) return NB_ERR_ARG;
    memcpy(out, c->last, sizeof(c->last));
    return NB_OK;
}

int64_t nb_launch_count(const nb_ctx* c) { return c ? c->launches : (int64_t)NB_ERR_ARG; }

int nb_set_profiling(nb_ctx* c, int on)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    if (c->prof) {
        int rc = prof_drain(c);
        if (rc != NB_OK) return rc;
    }
    if (on && c->ring.empty()) {
        c->ring.resize(PROF_RING);
        for (nb_ctx::Rec& R : c->ring)
            for (cudaEvent_t& e : R.e)
                if (cudaEventCreate(&e) != cudaSuccess) return NB_ERR_CUDA;
    }
    c->prof = on != 0;
    for (int k = 0; k < 3; ++k) {
        c->prof_ms[k] = 0.0;
        c->prof_n[k] = 0;
    }
    return NB_OK;
}

int nb_kernel_times(nb_ctx* c, double* out)
{
    if (!c || !out) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    for (int k = 0; k < 6; ++k) out[k] = 0.0;
    if (!c->prof) return NB_ERR_STATE;
    int rc = prof_drain(c);
    if (rc != NB_OK) return rc;
    for (int k = 0; k < 3; ++k) {
        out[k] = c->prof_ms[k];
        out[3 + k] = (double)c->prof_n[k];
    }
    return NB_OK;
}

// One pass over the j-store: predictor inside the pair loop (fused.cu), ni <= NB_FUSED_MAX
static int fused_impl(nb_ctx* c, double t, const int32_t* i_list, int64_t ni, double eps2, double* acc,
                      double* jrk, double* pot)
{
    int grid = 0, ni_pad = 0;
    if (launch_fused(c->store, c->flags, i_list, (int)ni, c->n, t, eps2, c->flagged.empty() ? 0 : 1, c->part,
                     c->err, c->sm_count, &grid, &ni_pad, c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    ReduceArgs r{};
    r.part = c->part;
    r.part_b = c->part;
    r.kA = (int)ni;                 // every position lies in the first (only) segment
    r.i_list = i_list;
    r.acc = acc;
    r.jrk = jrk;
    r.pot = pot;
    r.store = c->store;
    r.flags = c->flags;
    r.flag_list = c->flag_list;
    r.nflag = 0;                    // flagged pairs are handled inside the fused loop
    r.ni = (int)ni;
    r.ni_pad = ni_pad;
    r.splits = grid;
    r.n = (int)c->n;
    r.t_pred = t;
    if (launch_reduce(r, c->stream) != cudaSuccess) return NB_ERR_CUDA;
    c->last[0] = grid;
    c->last[1] = grid;
    c->last[2] = 2;
    c->last[3] = 0;
    c->launches += 2;
    return NB_OK;
}

int nb_force_fused(nb_ctx* c, double t, const int32_t* i_list, int64_t ni, double eps2, double* acc,
                   double* jrk, double* pot)
{
    if (!c || ni < 0 || ni > NB_FUSED_MAX || ni > c->ni_max || !isfinite(t) || !isfinite(eps2) || eps2 < 0.0)
        return NB_ERR_ARG;
    if (ni > 0 && (!i_list || !acc || !jrk || !pot)) return NB_ERR_ARG;
    if (ni == 0) return NB_OK;
    if (c->n < 1) return NB_ERR_STATE;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    return fused_impl(c, t, i_list, ni, eps2, acc, jrk, pot);
}

// ---- block-step layer (hermite.cu; R12, R18..R21) ---------------------------------

static bool steps_ok(double dt_min, double dt_max)
{
    // both must be powers of two (block grid), 0 < dt_min <= dt_max
    if (!(dt_min > 0.0) || !(dt_max >= dt_min) || !isfinite(dt_max)) return false;
    int e;
    return frexp(dt_min, &e) == 0.5 && frexp(dt_max, &e) == 0.5;
}

int nb_set_dt(nb_ctx* c, int64_t first, int64_t count, const double* dt)
{
    if (!c || first < 0 || count < 0 || first + count > c->n || (count > 0 && !dt)) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (count > 0 && cudaMemcpyAsync(c->dts + first, dt, (size_t)count * sizeof(double),
                                     cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    return NB_OK;
}

int nb_get_state(nb_ctx* c, int64_t first, int64_t count, double* out)
{
    if (!c || first < 0 || count < 0 || first + count > c->n || (count > 0 && !out)) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (launch_get_state(c->store, c->dts, first, count, out, c->stream) != cudaSuccess) return NB_ERR_CUDA;
    if (count > 0) c->launches += 1;
    return NB_OK;
}

int nb_init_steps(nb_ctx* c, const int32_t* i_list, int64_t ni, const double* acc, const double* jrk,
                  double eta_s, double dt_min, double dt_max)
{
    if (!c || ni < 0 || !(eta_s > 0.0) || !steps_ok(dt_min, dt_max)) return NB_ERR_ARG;
    if (ni > 0 && (!i_list || !acc || !jrk)) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (launch_init_steps(c->store, c->dts, i_list, ni, c->n, acc, jrk, eta_s, dt_min, dt_max, c->err,
                          c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    if (ni > 0) {
        c->launches += 1;
        c->predicted = false;      // stored (a, jerk) changed: the packed predicted state is stale
    }
    return NB_OK;
}

int nb_next_block(nb_ctx* c, double* t_next, int64_t* ni, const int32_t** i_list)
{
    if (!c || !t_next || !ni) return NB_ERR_ARG;
    if (c->n < 1) return NB_ERR_STATE;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (launch_select(c->store.f[F_T], c->dts, c->n, c->sel_meta, c->sel_counts, c->blk_list, c->ni_pad,
                      c->sm_count, c->stream) != cudaSuccess) {
        cudaGetLastError();
        return NB_ERR_CUDA;
    }
    c->launches += 1;
    unsigned long long* host = reinterpret_cast<unsigned long long*>(c->err_pinned) + 1;
    if (cudaMemcpyAsync(host, c->sel_meta, 16, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    // decode the order-preserving key (hermite.cu key_of)
    const long long b = (long long)host[0];
    const long long bits = b ^ ((~b >> 63) | (long long)0x8000000000000000ull);
    double t;
    memcpy(&t, &bits, 8);
    c->blk_t = t;
    c->blk_ni = (int64_t)host[1];
    *t_next = t;
    *ni = c->blk_ni;
    if (i_list) *i_list = c->blk_list;
    if (c->blk_ni > c->ni_max) return NB_ERR_ARG;     // the list was truncated to ni_max entries
    return NB_OK;
}

int nb_correct(nb_ctx* c, const int32_t* i_list, int64_t ni, double t1, const double* acc,
               const double* jrk, double eta, double dt_min, double dt_max)
{
    if (!c || ni < 0 || !isfinite(t1) || !(eta > 0.0) || !steps_ok(dt_min, dt_max)) return NB_ERR_ARG;
    if (ni > 0 && (!i_list || !acc || !jrk)) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (launch_correct(c->store, c->dts, i_list, ni, c->n, t1, acc, jrk, eta, dt_min, dt_max, c->err,
                       c->stream) != cudaSuccess)
        return NB_ERR_CUDA;
    if (ni > 0) {
        c->launches += 1;
        c->predicted = false;      // the j-store moved on: the packed predicted state is stale
    }
    return NB_OK;
}

// the part of a block step after the scheduler: forces on the k particles of the context's block list
// at time t, then corrector and new steps
static int step_body(nb_ctx* c, double t, int64_t k, double eps2, double eta, double dt_min, double dt_max)
{
    double* acc = c->blk_out;
    double* jrk = c->blk_out + 3 * k;
    double* pot = c->blk_out + 6 * k;
    // where the fused pass wins (one timing table): up to 4 particles at any N; 5..8
    // only while its fp64 arithmetic (35 ops x ni per j) stays below the cost of the saved pass
    const bool small = k <= 4 || (k <= NB_FUSED_MAX && c->n <= ((int64_t)1 << 18));
    int rc;
    if (small && c->tune_fused) {
        // a handful of particles: one fused pass over the j-store instead of predict + force
        rc = fused_impl(c, t, c->blk_list, k, eps2, acc, jrk, pot);
        c->predicted = false;
    } else {
        rc = nb_predict(c, t);
        if (rc != NB_OK) return rc;
        rc = force_impl(c, c->blk_list, k, eps2, acc, jrk, pot);
    }
    if (rc != NB_OK) return rc;
    return nb_correct(c, c->blk_list, k, t, acc, jrk, eta, dt_min, dt_max);
}

int nb_step(nb_ctx* c, double eps2, double eta, double dt_min, double dt_max, double* t, int64_t* ni)
{
    if (!c || !t || !ni || !isfinite(eps2) || eps2 < 0.0 || !(eta > 0.0) || !steps_ok(dt_min, dt_max))
        return NB_ERR_ARG;
    int rc = nb_next_block(c, t, ni, nullptr);
    if (rc != NB_OK) return rc;
    if (*ni == 0) return NB_ERR_STATE;       // every t + dt is NaN: nothing can be scheduled
    DeviceGuard g(c->device);
    return step_body(c, *t, *ni, eps2, eta, dt_min, dt_max);
}

int nb_set_steps_bound(nb_ctx* c, int64_t max_pairs)
{
    if (!c || max_pairs < 0) return NB_ERR_ARG;
    c->steps_max_pairs = max_pairs;
    return NB_OK;
}
int nb_set_steps_queue(nb_ctx* c, int on)
{
    if (!c) return NB_ERR_ARG;
    if (on < -1 || on > 2) return NB_ERR_ARG;
    c->steps_queue = on;
    return NB_OK;
}

// The mode in force.  Automatic: rounds planned on the device in one graph while the j-set is small (no
// host round trip per large block), the host's own launches from 262144 particles on, where the large
// blocks are most of the time and nb_step's pair kernel (4 CTAs per SM; the device-planned form has 3) is
// the faster one.  Measured per block step (bench.py --blockstep), mode 2 / mode 0, N = 131072: 130.9 /
// 134.3 us, 262144: 329.5 / 327.6, 524288: 490.5 / 478.4, 2^20: 1278 / 1248.
static int queue_mode(const nb_ctx* c)
{
    if (c->steps_queue >= 0) return c->steps_queue;
    return c->n >= 262144 ? 0 : 2;
}

// nb_steps with handed-over blocks planned ON THE DEVICE (steps.cu plan_kernel): the host queues
// rounds of [persistent kernel, plan, predictor, pair kernel (both mappings), reduction, corrector]
// without knowing how large the block of a round is, or whether there is one -- every kernel of a
// round reads the plan and exits at once when it has nothing to do -- and looks at the progress
// record once per batch of rounds.  No host round trip per large block.
static int steps_queued(nb_ctx* c, int64_t k, double eps2, double eta, double dt_min, double dt_max, double t_end,
                        bool want_us, int64_t* done)
{
    unsigned char* pin = reinterpret_cast<unsigned char*>(c->err_pinned);
    StepsProgress* p_in = reinterpret_cast<StepsProgress*>(pin + 64);
    StepsProgress* p_out = reinterpret_cast<StepsProgress*>(pin + 128);
    unsigned long long* meta_out = reinterpret_cast<unsigned long long*>(pin + 192);
    memset(p_in, 0, sizeof(StepsProgress));
    p_in->k = k;
    p_in->reason = STEPS_RUNNING;
    if (cudaMemcpyAsync(c->steps_prog, p_in, sizeof(StepsProgress), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemsetAsync(c->steps_plan, 0, sizeof(int), c->stream) != cudaSuccess)
        return NB_ERR_CUDA;

    StepsArgs a{};
    a.st = c->store;
    a.dts = c->dts;
    a.flags = c->flags;
    a.any_flagged = c->flagged.empty() ? 0 : 1;
    a.n = c->n;
    a.slots = c->steps_slots;
    a.list = c->blk_list;
    a.cap = c->ni_max;
    a.part = c->part;
    a.out = c->blk_out;
    a.meta = c->steps_meta;
    a.log_t = c->steps_log_t;
    a.log_ni = c->steps_log_ni;
    a.log_ns = c->steps_log_ns;
    a.budget = 0;
    a.eps2 = eps2;
    a.eta = eta;
    a.dt_min = dt_min;
    a.dt_max = dt_max;
    a.t_end = t_end;
    a.max_pairs = c->steps_max_pairs;
    a.err = c->err;
    a.trace = nullptr;
    a.prog = c->steps_prog;

    // what the plan cannot know: the fixed arguments of the pair kernel and of the reduction
    ForceArgs fa{};
    fa.pack = c->pack;
    fa.i_list = c->blk_list;
    fa.part = c->part;
    fa.flags = c->flags;
    fa.tileflag = c->tileflag;
    fa.err = c->err;
    fa.n = (int)c->n;
    fa.ntiles = (int)((c->n + TJ - 1) / TJ);
    fa.eps2 = (float)eps2;
    fa.any_flagged = a.any_flagged;
    fa.pack64 = nullptr;
    fa.eps2d = eps2;
    ReduceArgs ra{};
    ra.part = c->part;
    ra.part_b = c->part;
    ra.i_list = c->blk_list;
    ra.acc = c->blk_out;
    ra.store = c->store;
    ra.flags = c->flags;
    ra.flag_list = c->flag_list;
    ra.nflag = (int)c->flagged.size();
    ra.n = (int)c->n;
    ra.counter = c->ticket;
    const bool guard = (float)eps2 < EPS2_GUARD;
    const int resident_all = c->sm_count * c->blocks_per_sm[guard ? 5 : 4];
    const int resident_few = c->sm_count * c->blocks_per_sm[guard ? 7 : 6];

    // one round on stream st; cond/loop: the plan kernel also drives the WHILE node of the graph
    auto round = [&](cudaStream_t st, unsigned long long cond, int loop) -> bool {
        return launch_steps(a, c->sm_count, st) == cudaSuccess &&
               launch_plan(a, c->steps_plan, c->steps_prog, fa, ra, resident_all, resident_few, c->part_bytes, st, cond,
                           loop) == cudaSuccess &&
               launch_predict(c->store, c->flags, c->pack, nullptr, nullptr, c->n, 0.0, st, c->steps_plan) ==
                   cudaSuccess &&
               launch_force_dyn(c->steps_plan, (float)eps2, resident_all, resident_few, st) == cudaSuccess &&
               launch_reduce_dyn(c->steps_plan, c->ni_max, st) == cudaSuccess &&
               launch_correct_dyn(c->store, c->dts, c->steps_plan, c->n, c->ni_max, eta, dt_min, dt_max, c->err, st) ==
                   cudaSuccess;
    };

    // Mode 2: the rounds are the body of a WHILE node of ONE graph (the plan kernel sets the loop
    // condition on the device), followed by a launch that closes the last time stamp: one graph launch
    // per nb_steps call, no empty rounds, nothing for the host to do until the end.
    if (queue_mode(c) == 2 && c->steps_graph_state >= 0) {
        const double key[8] = {eps2, eta, dt_min, dt_max, t_end, (double)c->steps_max_pairs, (double)c->n,
                               (double)c->flagged.size()};
        const void* kp[3] = {c->steps_log_t, c->steps_log_ni, c->steps_log_ns};
        const bool same = c->steps_graph_state == 1 && memcmp(key, c->steps_key, sizeof(key)) == 0 &&
                          memcmp(kp, c->steps_key_ptr, sizeof(kp)) == 0;
        if (!same) {
            if (c->steps_exec) cudaGraphExecDestroy(c->steps_exec);
            if (c->steps_graph) cudaGraphDestroy(c->steps_graph);
            c->steps_exec = nullptr;
            c->steps_graph = nullptr;
            c->steps_graph_state = -1;
            bool ok = c->cap_stream || cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) == cudaSuccess;
            cudaGraphConditionalHandle handle = 0;
            cudaGraphNode_t wnode = nullptr;
            cudaGraph_t body = nullptr, tmp = nullptr;
            ok = ok && cudaGraphCreate(&c->steps_graph, 0) == cudaSuccess;
            ok = ok && cudaGraphConditionalHandleCreate(&handle, c->steps_graph, 1, cudaGraphCondAssignDefault) ==
                           cudaSuccess;
            if (ok) {
                cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
                memset(&np, 0, sizeof(np));
                np.type = cudaGraphNodeTypeConditional;
                np.conditional.handle = handle;
                np.conditional.type = cudaGraphCondTypeWhile;
                np.conditional.size = 1;
                ok = cudaGraphAddNode(&wnode, c->steps_graph, nullptr, 0, &np) == cudaSuccess;
                if (ok) body = np.conditional.phGraph_out[0];
            }
            if (ok && cudaStreamBeginCaptureToGraph(c->cap_stream, body, nullptr, nullptr, 0,
                                                     cudaStreamCaptureModeRelaxed) == cudaSuccess) {
                const bool queued_ok = round(c->cap_stream, (unsigned long long)handle, 1);
                ok = cudaStreamEndCapture(c->cap_stream, &tmp) == cudaSuccess && queued_ok;
            } else {
                ok = false;
            }
            if (ok && cudaStreamBeginCaptureToGraph(c->cap_stream, c->steps_graph, &wnode, nullptr, 1,
                                                     cudaStreamCaptureModeRelaxed) == cudaSuccess) {
                const bool queued_ok = launch_steps(a, c->sm_count, c->cap_stream) == cudaSuccess;
                ok = cudaStreamEndCapture(c->cap_stream, &tmp) == cudaSuccess && queued_ok;
            } else {
                ok = false;
            }
            ok = ok && cudaGraphInstantiate(&c->steps_exec, c->steps_graph, 0) == cudaSuccess;
            if (ok) {
                c->steps_graph_state = 1;
                memcpy(c->steps_key, key, sizeof(key));
                memcpy(c->steps_key_ptr, kp, sizeof(kp));
            } else {
                cudaGetLastError();               // this driver cannot build it: stream-queued rounds from now on
                if (c->steps_exec) cudaGraphExecDestroy(c->steps_exec);
                if (c->steps_graph) cudaGraphDestroy(c->steps_graph);
                c->steps_exec = nullptr;
                c->steps_graph = nullptr;
            }
        }
    }

    int result = NB_OK;
    if (queue_mode(c) == 2 && c->steps_graph_state == 1) {
        if (cudaGraphLaunch(c->steps_exec, c->stream) != cudaSuccess) {
            cudaGetLastError();
            return NB_ERR_CUDA;
        }
        c->launches += 1;                         // one graph launch; its kernels are counted from the log below
        c->predicted = false;
        if (cudaMemcpyAsync(p_out, c->steps_prog, sizeof(StepsProgress), cudaMemcpyDeviceToHost, c->stream) !=
                cudaSuccess ||
            cudaMemcpyAsync(meta_out, c->steps_meta + 4, 32, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess)
            return NB_ERR_CUDA;
        c->launches += 7 * (int64_t)p_out->rounds;
    } else {
    int64_t rounds = k < 4 ? k : 4;           // rounds in the first batch
    int64_t rounds_total = 0;
    for (;;) {
        for (int64_t r = 0; r < rounds; ++r) {
            if (!round(c->stream, 0ull, 0)) {
                cudaGetLastError();
                return NB_ERR_CUDA;
            }
            c->launches += 7;
        }
        c->predicted = false;
        if (cudaMemcpyAsync(p_out, c->steps_prog, sizeof(StepsProgress), cudaMemcpyDeviceToHost, c->stream) !=
                cudaSuccess ||
            cudaMemcpyAsync(meta_out, c->steps_meta + 4, 32, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess)
            return NB_ERR_CUDA;
        if (p_out->final || p_out->done >= k) break;
        // every round of the batch ended at a large block: size the next batch by the rate seen so far
        rounds_total += rounds;
        const double per_step = (double)rounds_total / (double)(p_out->done > 0 ? p_out->done : 1);
        int64_t want = (int64_t)(per_step * (double)(k - p_out->done) * 1.1) + 1;
        rounds = want < 2 ? 2 : (want > 64 ? 64 : want);
    }
    }
    *done = p_out->done;
    if (p_out->pending_ni > 0) result = NB_ERR_ARG;            // a block above ni_max: the list was truncated
    else if (p_out->final && p_out->reason == STEPS_STUCK) result = NB_ERR_STATE;
    if (p_out->done > 0) c->blk_ni = (int64_t)meta_out[3];     // for nb_block_forces
    if (want_us && !p_out->closed && p_out->pending_ni == 0 && !(queue_mode(c) == 2 && c->steps_graph_state == 1)) {
        // the batch ended with a device-planned block: one more (empty) launch stamps the closing time
        if (launch_steps(a, c->sm_count, c->stream) != cudaSuccess) {
            cudaGetLastError();
            return NB_ERR_CUDA;
        }
        c->launches += 1;
    }
    return result;
}

int nb_steps(nb_ctx* c, int64_t k, double eps2, double eta, double dt_min, double dt_max, double t_end,
             double* t_log, int64_t* ni_log, double* us_log, int64_t* done)
{
    if (!c || k < 0 || !done || !isfinite(eps2) || eps2 < 0.0 || !(eta > 0.0) || !steps_ok(dt_min, dt_max) ||
        t_end != t_end)
        return NB_ERR_ARG;
    *done = 0;
    if (k == 0) return NB_OK;
    if (c->n < 1) return NB_ERR_STATE;
    DeviceGuard g(c->device);
    int rc = ensure_alloc(c);
    if (rc != NB_OK) return rc;
    if (c->steps_ok < 0) {
        int b = 0;
        c->steps_ok = (steps_kernel_setup(&b) == cudaSuccess && b >= 1) ? 1 : 0;
        cudaGetLastError();
    }
    if (k > c->steps_log_cap) {               // the device log grows to the largest k asked for
        if (c->steps_log_t) cudaFree(c->steps_log_t);
        if (c->steps_log_ni) cudaFree(c->steps_log_ni);
        if (c->steps_log_ns) cudaFree(c->steps_log_ns);
        c->steps_log_t = nullptr;
        c->steps_log_ni = nullptr;
        c->steps_log_ns = nullptr;
        c->steps_log_cap = 0;
        // (re)allocation synchronises the device: at least 4096 entries, then doubling
        int64_t cap = c->steps_log_cap > 0 ? c->steps_log_cap : 4096;
        while (cap < k) cap *= 2;
        if (cudaMalloc(&c->steps_log_t, (size_t)cap * 8) != cudaSuccess ||
            cudaMalloc(&c->steps_log_ni, (size_t)cap * 8) != cudaSuccess ||
            cudaMalloc(&c->steps_log_ns, (size_t)(cap + 1) * 8) != cudaSuccess) {
            cudaGetLastError();
            return NB_ERR_ALLOC;
        }
        c->steps_log_cap = cap;
    }
    unsigned long long* status = reinterpret_cast<unsigned long long*>(c->err_pinned) + 4;
    // handed-over blocks are planned on the device and queued, unless the mode was switched off, the
    // pair loop is the IEEE-double one (its launch shapes are not planned on the device) or the
    // reduction runs by atomics
    const bool queued = c->steps_ok == 1 && queue_mode(c) != 0 && c->precision == 0 && c->tune_reduce == 0 &&
                        c->tune_splits == 0;
    std::vector<int64_t> host_idx;            // steps that went through the host path: (index, t, ni)
    std::vector<double> host_t;
    std::vector<int64_t> host_ni;
    int64_t s = 0;
    int result = NB_OK;
    bool last_was_host = false;
    auto launch = [&](int64_t budget) -> int {
        StepsArgs a{};
        a.st = c->store;
        a.dts = c->dts;
        a.flags = c->flags;
        a.any_flagged = c->flagged.empty() ? 0 : 1;
        a.n = c->n;
        a.slots = c->steps_slots;
        a.list = c->blk_list;
        a.cap = c->ni_max;
        a.part = c->part;
        a.out = c->blk_out;
        a.meta = c->steps_meta;
        a.log_t = c->steps_log_t + s;
        a.log_ni = c->steps_log_ni + s;
        a.log_ns = c->steps_log_ns + s;
        a.budget = budget;
        a.eps2 = eps2;
        a.eta = eta;
        a.dt_min = dt_min;
        a.dt_max = dt_max;
        a.t_end = t_end;
        a.max_pairs = c->steps_max_pairs;
        a.err = c->err;
        a.trace = reinterpret_cast<unsigned long long*>(c->part) + (c->part_bytes / 8 - (size_t)8 * 4096);
        if (launch_steps(a, c->sm_count, c->stream) != cudaSuccess) {
            cudaGetLastError();
            return NB_ERR_CUDA;
        }
        c->launches += 1;
        c->predicted = false;
        return NB_OK;
    };
    if (queued) {
        result = steps_queued(c, k, eps2, eta, dt_min, dt_max, t_end, us_log != nullptr, &s);
        if (result == NB_ERR_CUDA) return result;
    }
    while (!queued && s < k) {
        double t = 0.0;
        int64_t ni = 0;
        if (c->steps_ok == 1) {
            rc = launch(k - s);
            if (rc != NB_OK) return rc;
            if (cudaMemcpyAsync(status, c->steps_meta + 4, 32, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
                cudaStreamSynchronize(c->stream) != cudaSuccess)
                return NB_ERR_CUDA;
            const int64_t did = (int64_t)status[0];
            const int reason = (int)status[1];
#ifdef NB_STEPS_TRACE
            {   // development builds: dump CTA 0's phase stamps of this launch (ns since its first stamp)
                std::vector<unsigned long long> tr((size_t)8 * (did < 4096 ? did : 4096));
                cudaMemcpy(tr.data(), reinterpret_cast<unsigned long long*>(c->part) + (c->part_bytes / 8 - (size_t)8 * 4096),
                           tr.size() * 8, cudaMemcpyDeviceToHost);
                if (FILE* f = fopen("gpurun_out/steps_trace.txt", "a")) {
                    for (int64_t q = 0; q < (int64_t)tr.size() / 8; ++q) {
                        for (int w = 1; w < 7; ++w) fprintf(f, "%lld ", (long long)(tr[q * 8 + w] - tr[q * 8 + w - 1]));
                        fprintf(f, "\n");
                    }
                    fclose(f);
                }
            }
#endif
            if (did > 0) {
                last_was_host = false;
                if (reason != STEPS_BIG) c->blk_ni = (int64_t)status[3];   // for nb_block_forces
            }
            s += did;
            if (reason == STEPS_DONE || reason == STEPS_T_END) break;
            if (reason == STEPS_STUCK) {
                result = NB_ERR_STATE;
                break;
            }
            // one block the persistent kernel does not take.  It left the block's ascending list on
            // the device and its time and size are known, so nb_step's launches (predictor, packed
            // fp32 pair kernel, reduction, corrector) are queued without another synchronisation.
            const long long kb = (long long)status[2];
            const long long bits = kb ^ ((~kb >> 63) | (long long)0x8000000000000000ull);
            memcpy(&t, &bits, 8);
            ni = (int64_t)status[3];
            if (ni > c->ni_max) {
                result = NB_ERR_ARG;
                break;
            }
            c->blk_t = t;
            c->blk_ni = ni;
            rc = step_body(c, t, ni, eps2, eta, dt_min, dt_max);
        } else {                              // no persistent kernel on this device: nb_step does everything
            rc = nb_next_block(c, &t, &ni, nullptr);
            if (rc == NB_OK && ni == 0) rc = NB_ERR_STATE;
            if (rc != NB_OK) { result = rc; break; }
            if (!(t <= t_end)) break;
            rc = step_body(c, t, ni, eps2, eta, dt_min, dt_max);
        }
        if (rc != NB_OK) { result = rc; break; }
        host_idx.push_back(s);
        host_t.push_back(t);
        host_ni.push_back(ni);
        last_was_host = true;
        s += 1;
    }
    *done = s;
    if (s > 0 && (t_log || ni_log || us_log)) {
        std::vector<unsigned long long> ns;
        if (us_log && c->steps_ok == 1) {
            if (last_was_host && launch(0) != NB_OK) return NB_ERR_CUDA;   // closing time stamp after a host block
            ns.resize((size_t)s + 1);
            if (cudaMemcpyAsync(ns.data(), c->steps_log_ns, ns.size() * 8, cudaMemcpyDeviceToHost, c->stream) !=
                cudaSuccess)
                return NB_ERR_CUDA;
        }
        if (t_log && cudaMemcpyAsync(t_log, c->steps_log_t, (size_t)s * 8, cudaMemcpyDeviceToHost, c->stream) !=
                         cudaSuccess)
            return NB_ERR_CUDA;
        if (ni_log && cudaMemcpyAsync(ni_log, c->steps_log_ni, (size_t)s * 8, cudaMemcpyDeviceToHost,
                                      c->stream) != cudaSuccess)
            return NB_ERR_CUDA;
        if (cudaStreamSynchronize(c->stream) != cudaSuccess) return NB_ERR_CUDA;
        for (size_t q = 0; q < host_idx.size(); ++q) {
            if (t_log) t_log[host_idx[q]] = host_t[q];
            if (ni_log) ni_log[host_idx[q]] = host_ni[q];
        }
        if (us_log)
            for (int64_t q = 0; q < s; ++q)
                us_log[q] = ns.empty() ? 0.0 : (double)(long long)(ns[q + 1] - ns[q]) * 1e-3;
    }
    return result;
}

int nb_block_forces(nb_ctx* c, const double** acc, const double** jrk, const double** pot)
{
    if (!c || c->blk_ni < 0 || !c->allocated) return c ? NB_ERR_STATE : NB_ERR_ARG;
    if (acc) *acc = c->blk_out;
    if (jrk) *jrk = c->blk_out + 3 * c->blk_ni;
    if (pot) *pot = c->blk_out + 6 * c->blk_ni;
    return NB_OK;
}

int nb_sync(nb_ctx* c)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard g(c->device);
    if (c->allocated) {
        if (cudaMemcpyAsync(c->err_pinned, c->err, sizeof(int), cudaMemcpyDeviceToHost, c->stream) !=
            cudaSuccess)
            return NB_ERR_CUDA;
    } else {
        *c->err_pinned = 0;
    }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return NB_ERR_CUDA;
    if (*c->err_pinned) {
        // device latch: bit 0 = an index was out of range, bit 1 = a due particle had a zero step,
        // bit 2 = a peer did not answer an exchange (nb_xforce)
        const int bits = *c->err_pinned;
        *c->err_pinned = 0;
        if (cudaMemsetAsync(c->err, 0, sizeof(int), c->stream) != cudaSuccess) return NB_ERR_CUDA;
        return (bits & 1) ? NB_ERR_INDEX : ((bits & 4) ? NB_ERR_PEER : NB_ERR_STATE);
    }
    return NB_OK;
}

}  // extern "C"
