// nb_internal.h -- shared declarations of libnb.so (context, device layouts, kernel launchers).
// Product code: nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/nb.h"

namespace nb {

// ---- device data layout ------------------------------------------------
// j-store: 14 fp64 arrays of stride n_cap (SoA): m, x,y,z, vx,vy,vz, ax,ay,az, jx,jy,jz, t.
enum Field { F_M = 0, F_X, F_Y, F_Z, F_VX, F_VY, F_VZ, F_AX, F_AY, F_AZ, F_JX, F_JY, F_JZ, F_T, NFIELD };

// pack: the force-ready predicted j-set, written by the predictor, streamed by the pair kernel.
// Tiles of TJ particles, SoA inside a tile: NPF float arrays of TJ entries, so that one tile is one
// contiguous 1-D bulk copy and two consecutive j's form an f32x2 operand pair.
#ifndef NB_TJ
#define NB_TJ 128
#endif
#ifndef NB_STAGES
#define NB_STAGES 4
#endif
#ifndef NB_MINB
#define NB_MINB 3
#endif
#ifndef NB_FLUSH_TILES
#define NB_FLUSH_TILES 2           // all-i kernel: tiles per fp32 run before the sums move to fp64 (power of two):
                                   // 128 terms per lane sum.  Measured at config 3's headline call, 1 / 2 / 4 tiles: 0.778 /
                                   // 0.787 / 0.789 of the FP32 peak; worst errors over the five configs (tolerances 1e-5,
                                   // 1e-4, 1e-5): acc 9.8e-7 / 1.5e-6 / 3.0e-6, jerk 7.2e-6 / 8.4e-6 / 1.3e-5, pot
                                   // 7.7e-7 / 1.9e-6 / 4.0e-6
#endif
#ifndef NB_MINB_FEW
#define NB_MINB_FEW 3
#endif
#ifndef NB_PDL
#define NB_PDL 1                   // force_kernel and reduce_kernel are launched with programmatic stream serialization
                                   // and wait for the kernel before them with griddepcontrol.wait (force.cu pdl_launch)
#endif
#ifndef NB_TAIL_SEGMENT
#define NB_TAIL_SEGMENT 1          // nb_force: a last i-tile that is at most half full goes to the few-i kernel as a
                                   // segment of its own (nb_api.cu force_impl); 0 = one all-i segment as before
#endif
#ifndef NB_TAIL_MIN_GAIN
#define NB_TAIL_MIN_GAIN 9e-6      // ... when the model says it saves at least this many seconds (an extra launch costs ~5 us);
#define NB_TAIL_MIN_GAIN_HALF 13e-6   // a 128-slot tail saves 0.42 of a pass at best and needs more (measured at N = 98304,
                                      // N_i = 1152: 166 -> 180 us with 9e-6; at N = 131072: 207 -> 203 us)
#endif
// (and 20e-6 above 4096 particles, where the call's reduction is the thread-per-i one: N = 131072, N_i = 4224: 640 -> 652 us
// with 13e-6; N = 262144: 1256 -> 1210 us)
#define NB_TAIL_GAIN_NEEDED(slots, ni) ((slots) >= ITILE / 2 ? ((ni) > 4096 ? 20e-6 : NB_TAIL_MIN_GAIN_HALF) : NB_TAIL_MIN_GAIN)
#ifndef NB_DYN_MINB
#define NB_DYN_MINB 3
#endif
#ifndef NB_DYN_MINB_ALL
#define NB_DYN_MINB_ALL 3          // the all-i form of force_dyn_kernel: 135 registers, 3 CTAs per SM (4: 128 registers,
                                   // 4 CTAs; measured -1.2 % per block step at N = 2^20, +1.5 % at N = 131072)
#endif
#ifndef NB_UNROLL
#define NB_UNROLL 2
#endif
constexpr int TJ = NB_TJ;                     // j-particles per tile
enum PackField { P_XH = 0, P_YH, P_ZH, P_XL, P_YL, P_ZL, P_VX, P_VY, P_VZ, P_M, P_FLAG, NPF };
constexpr int TILE_FLOATS = TJ * NPF;         // 1408
constexpr int TILE_BYTES = TILE_FLOATS * 4;   // 5632 (multiple of 16: legal bulk-copy size)

// pair kernel shape
constexpr int FORCE_THREADS = 128;
constexpr int NWARPS = FORCE_THREADS / 32;
constexpr int IPT = 2;                        // i-particles per thread
constexpr int ITILE = FORCE_THREADS * IPT;    // i-slots per CTA (= i-particles when JL = 1)
constexpr int JSH_MAX = 5;                    // up to 2^5 = 32 threads per i-slot in the few-i kernel (force.cu)
constexpr int STAGES = NB_STAGES;             // j-tile ring depth
constexpr int NOUT = 7;                       // ax ay az jx jy jz pot

// pack64: the same tiles in fp64 for the full-double pair loop (force64.cu): 8 double arrays of TJ
enum Pack64Field { Q_X = 0, Q_Y, Q_Z, Q_VX, Q_VY, Q_VZ, Q_M, Q_FLAG, NQF };
constexpr int TILE64_DOUBLES = TJ * NQF;      // 1024
constexpr int TILE64_BYTES = TILE64_DOUBLES * 8;   // 8192

// pack6: the tiles of the 6th-order pair loop (force6.cu): 14 float arrays of TJ: two-float position,
// velocity, predicted acceleration, mass, flag
constexpr int NPF6 = 14;
constexpr int TILE6_FLOATS = TJ * NPF6;       // 1792
constexpr int TILE6_BYTES = TILE6_FLOATS * 4; // 7168

// calls with eps2 below this (zero included) drop r = 0 pairs inside the packed pair (force.cu GUARD):
// the self pair's m eps^-3 would leave the fp32 range (m up to ~1e8 is safe at the threshold)
constexpr float EPS2_GUARD = 1.0e-20f;
constexpr float PAD_POS = 1.0e10f;            // where the m = 0 padding records of the last tile sit

struct StorePtrs {
    double* f[NFIELD];
};

struct SrcPtrs {
    const double* f[NFIELD];
};

struct ForceArgs {
    const float* pack;        // [ntiles][NPF][TJ]
    const int32_t* i_list;    // [ni] (by-index calls, nb_force)
    const double* ext_x;      // [3][ni]: i-particles by value (nb_force_ext), else unused
    const double* ext_v;      // [3][ni], or NULL for acc + pot only
    const int32_t* ext_self;  // [ni] by value: index of the j-set member this i-particle is (or < 0), or NULL
    const uint8_t* ext_flags; // [ni] by value: bit 0 = it carries the unsoftened flag, or NULL
    int jsh;                  // few-i kernel: log2 of the threads per i-slot (0 = all-i kernel)
    int reduce_here;          // few-i kernel: the last CTA to finish also reduces (one launch per call)
    double* part;             // [S][NOUT][ni_pad] partial sums (reduce_mode 0)
    const uint8_t* flags;     // [n_cap] bit 0: unsoftened among flagged
    const uint32_t* tileflag; // bit t: tile t holds a flagged particle
    int* err;                 // device error latch
    int ni;                   // length of i_list (bounds, output stride)
    int k0;                   // first i_list position of this launch (segment), multiple of ITILE
    int ni_pad, n_itiles;     // padded length and i-tiles of the segment
    int n, ntiles, splits;
    float eps2;
    int any_flagged;
    const double* pack64;     // fp64 tiles (precision mode 1), else unused
    double eps2d;
    int part_i_fastest;       // partial sums as [c][subset][i] (coalesced stores; the thread-per-i reduction) instead of [c][i][subset]
};

struct ReduceArgs {
    const double* part;       // segment A: [NOUT][ni_pad][splits] (subset index fastest), positions [0, kA)
    const double* part_b;     // segment B: [NOUT][ni_pad_b][splits_b], positions [kA, ni)
    int kA, ni_pad_b, splits_b;
    const int32_t* i_list;
    double *acc, *jrk, *pot;
    StorePtrs store;          // for the fp64 flagged-pair terms
    const uint8_t* flags;
    const int32_t* flag_list; // indices of flagged particles
    int nflag;
    int ni, ni_pad, splits, n;
    double t_pred;
    int atomic_mode;          // 1: acc/jrk/pot already hold the sums (atomics); only fix-ups here
    const double *ext_x, *ext_v;      // by-value calls: the i-particles (for their flagged pairs)
    const int32_t* ext_self;
    const uint8_t* ext_flags;
    unsigned* counter;        // ticket counter of the few-i kernel's own reduction (zero between calls)
    const struct Xchg* xchg;  // j-sharded call (nb_xforce, xchg.h): the rank's exchange descriptor, else NULL
    unsigned xchg_epoch;      // ... the call's epoch
    int xchg_phase;           // ... 0: push, wait and sum inside the reducing CTA; 1: push only
    unsigned long long xchg_limit_ns;   // ... how long to wait for a peer
    int part_i_fastest;       // layout of part / part_b, as in ForceArgs
    int warp_rows;            // thread-per-i reduction only: the LAST warp_rows positions (a tail segment with hundreds
                              // of j-subsets) are summed by one warp each instead (0: none)
};

// kernel launchers (each returns the cudaError of the launch)
cudaError_t launch_set_j(const StorePtrs& dst, const SrcPtrs& src, int64_t first, int64_t count,
                         cudaStream_t s);
cudaError_t launch_update_j(const StorePtrs& dst, const SrcPtrs& src, const int32_t* idx,
                            int64_t count, int64_t n, int* err, cudaStream_t s);
cudaError_t launch_set_flags(uint8_t* flags, const int32_t* idx_then_val, int count, cudaStream_t s);
cudaError_t launch_predict(const StorePtrs& store, const uint8_t* flags, float* pack, double* pack64, float* pack6,
                           int64_t n, double t, cudaStream_t s, const struct DynPlan* plan = nullptr);
cudaError_t launch_get_predicted(const StorePtrs& store, int64_t first, int64_t count, double t,
                                 double* out, cudaStream_t s);
cudaError_t force_kernel_setup(int* blocks_per_sm /*[8]*/);
cudaError_t force64_kernel_setup(int* blocks_per_sm);
cudaError_t launch_force64(const ForceArgs& a, int mode, cudaStream_t s);
cudaError_t launch_force(const ForceArgs& a, const ReduceArgs& r, int mode, int atomic_mode, double* acc,
                         double* jrk, double* pot, cudaStream_t s);
cudaError_t launch_reduce(const ReduceArgs& a, cudaStream_t s);
// direct.cu: the one-launch force call for a handful of active particles
constexpr int DIRECT_NI_MAX = 8;
int direct_grid(int ntiles, int sm_count);
int64_t direct_terms_per_lane(int ntiles, int grid);
cudaError_t launch_direct(const ForceArgs& a, const ReduceArgs& r, int grid, cudaStream_t s);
constexpr int SEL_MAX_BLOCKS = 1024;          // most CTAs the cooperative scheduler kernel uses
cudaError_t launch_select(const double* t, const double* dt, int64_t n, unsigned long long* meta,
                          int* counts, int32_t* list, int64_t cap, int sm_count, cudaStream_t s);
cudaError_t launch_correct(const StorePtrs& st, double* dts, const int32_t* list, int64_t ni, int64_t n,
                           double t1, const double* acc, const double* jrk, double eta, double dt_min,
                           double dt_max, int* err, cudaStream_t s);
cudaError_t launch_init_steps(const StorePtrs& st, double* dts, const int32_t* list, int64_t ni, int64_t n,
                              const double* acc, const double* jrk, double eta_s, double dt_min,
                              double dt_max, int* err, cudaStream_t s);
cudaError_t launch_get_state(const StorePtrs& st, const double* dts, int64_t first, int64_t count,
                             double* out, cudaStream_t s);
cudaError_t launch_fused(const StorePtrs& st, const uint8_t* flags, const int32_t* i_list, int ni, int64_t n,
                         double t, double eps2, int any_flagged, double* part, int* err, int sm_count,
                         int* grid_out, int* ni_pad_out, cudaStream_t s);
cudaError_t launch_zero_out(double* acc, double* jrk, double* pot, int64_t ni, cudaStream_t s);

struct Force6Args {
    const float* pack6;       // [ntiles][NPF6][TJ]
    const int32_t* i_list;
    double* part;             // [10][ni_pad][splits]
    const uint8_t* flags;
    int* err;
    int ni, ni_pad, n_itiles, n, ntiles, splits;
    float eps2;
    int any_flagged;
};
cudaError_t force6_kernel_setup(int* blocks_per_sm);
cudaError_t launch_force6(const Force6Args& a, const StorePtrs& st, const int32_t* flag_list, int nflag, double t_pred,
                          double* acc, double* jrk, double* snp, double* pot, cudaStream_t s);

// ---- nb_steps (steps.cu): block steps in one persistent cooperative kernel ---------------------
constexpr int STEPS_NI_MAX = 512;             // largest block the persistent kernel takes itself
constexpr int STEPS_SLOT = 128;               // most due particles one slice can publish
enum StepsReason { STEPS_RUNNING = 0, STEPS_DONE, STEPS_BIG, STEPS_T_END, STEPS_STUCK };
struct StepsSlot {                            // what one CTA publishes about its slice of the particles
    unsigned long long key;                   // order-preserving key of its earliest t + dt
    int count, pad;                           // how many of its particles are due then
    int32_t idx[STEPS_SLOT];                  // their indices, ascending (the first STEPS_SLOT)
};
struct StepsArgs {
    StorePtrs st;
    double* dts;
    const uint8_t* flags;
    int any_flagged;
    int64_t n;
    StepsSlot* slots;             // [CTAs]
    int32_t* list;                // the context's block list (ascending), as nb_next_block leaves it
    int64_t cap;                  // ni_max
    double* part;                 // [NOUT][ni][CTAs]
    double* out;                  // the context's block forces [NOUT][ni]
    unsigned long long* meta;     // [4..7] exit status: steps done, StepsReason, key of the pending block
                                  // time, N_i of the pending block (STEPS_BIG) or of the last one completed
    double* log_t;                // [budget] block times, from this launch's first step
    long long* log_ni;            // [budget] block sizes
    unsigned long long* log_ns;   // [budget + 1] %globaltimer at the start of each step and at the exit
    int64_t budget;
    double eps2, eta, dt_min, dt_max, t_end;
    int64_t max_pairs;            // a block with ni x n above this is left to the host path
    int* err;
    unsigned long long* trace;    // NB_STEPS_TRACE builds only
    struct StepsProgress* prog;   // non-NULL: budget and log offset come from here (queued batches)
};
// A block that the persistent kernel hands over, planned ON THE DEVICE so that the host can queue its
// kernels without knowing its size (steps.cu plan_kernel -> predict / force_dyn / reduce_dyn /
// correct_dyn, all of which exit at once while go == 0).
struct DynPlan {
    int go;                       // 1: a block is pending and planned
    unsigned next;                // work items of the pair kernel handed out beyond the first one per CTA
    double t1;                    // its time
    long long ni;                 // its size
    ForceArgs fa;                 // launch shape and arguments of the pair kernel
    ReduceArgs ra;                // ... and of the reduction
    int go_b;                     // 1: the block's last, at most half full i-tile is a segment of its own (fb) for the
    unsigned next_b;              // few-i instantiation, with its own work counter (nb_api.cu force_impl: tail segment)
    ForceArgs fb;
};
struct StepsProgress {            // where a batch of queued kernels stands (device memory)
    long long done;               // block steps completed since nb_steps was called
    long long k;                  // steps asked for
    int final;                    // 1: stop (t_end reached, nothing schedulable, an error)
    int reason;                   // StepsReason of the last persistent-kernel exit
    long long pending_ni;         // size of a block that could not be planned (ni > ni_max)
    int closed;                   // 1: log_ns[done] holds the time stamp that closes the last step
    int rounds;                   // rounds (persistent kernel + plan + block kernels) run so far
};
cudaError_t steps_kernel_setup(int* blocks_per_sm);
// one round of the device-planned path for a handed-over block; every kernel is a no-op while no block
// is pending.  resident = CTAs of the pair kernel that fit the chip (grid of force_dyn_kernel).
cudaError_t launch_plan(const StepsArgs& a, DynPlan* plan, StepsProgress* prog, const ForceArgs& fa_base,
                        const ReduceArgs& ra_base, int resident_all, int resident_few, size_t part_bytes,
                        cudaStream_t s, unsigned long long cond_handle = 0, int loop = 0);
cudaError_t launch_force_dyn(DynPlan* plan, float eps2, int resident_all, int resident_few, cudaStream_t s);
cudaError_t launch_reduce_dyn(const DynPlan* plan, int64_t ni_max, cudaStream_t s);
cudaError_t launch_correct_dyn(const StorePtrs& st, double* dts, const DynPlan* plan, int64_t n, int64_t ni_max,
                               double eta, double dt_min, double dt_max, int* err, cudaStream_t s);
cudaError_t launch_steps(const StepsArgs& a, int sm_count, cudaStream_t s);

// Hermite predictor of one component (R1), shared by predict / get_predicted / the flagged-pair
// fix-up so that all three see the same fp64 state.
__device__ __forceinline__ void predict1(double x, double v, double a, double j, double dt,
                                         double& xp, double& vp)
{
    const double h = 0.5 * dt, s = dt * (1.0 / 3.0);
    // xp = x + dt (v + dt/2 (a + dt/3 j)) ; vp = v + dt (a + dt/2 j)
    xp = fma(dt, fma(h, fma(s, j, a), v), x);
    vp = fma(dt, fma(h, j, a), v);
}

}  // namespace nb
