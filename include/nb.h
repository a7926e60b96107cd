/* nb.h -- C-ABI of the B200-native direct-summation force library (libnb.so).
 *
 * What the library is: the "force library" layer of a direct N-body code as the paper states the
 * problem (section III.A): j-particles exert a force, i-particles receive it; the
 * library keeps the j-set on the GPU, can advance it to the current time with the Hermite
 * predictor ("optional prediction step on the j particles"; "4th order
 * Hermite predictor-corrector"), and returns acceleration, jerk and potential for the i-particles
 * it is given (j split in blocks + partial-force reduction).
 * The paper prints no formula; the readings taken are R1..R16 in DESIGN.md section 3.
 *
 * Conventions for every entry point
 *   - returns NB_OK (0) or a negative nb_status; never throws, aborts or prints.
 *   - "DEVICE" pointers are CUDA device memory on the context's device, "HOST" pointers are
 *     ordinary host memory.  The caller owns every array it passes; the library owns only the
 *     context and its internal buffers.  Inputs are read, outputs written, on the context's
 *     stream: a call returns once the work is enqueued (DEVICE variants) and results are valid
 *     after the stream, or nb_sync, completes.  *_host variants return after the copy back.
 *   - vectors are SoA fp64; indices are int32 (N < 2^31); eps2 is the SQUARE of the softening.
 *   - a context is not thread-safe; use one per host thread or lock around it.
 *   - sm_100 (compute capability 10.x) only: nb_create fails with NB_ERR_ARCH elsewhere.  There is
 *     no CPU or other-GPU fallback.
 */
#ifndef NB_H
#define NB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nb_ctx nb_ctx;   /* opaque; one per j-set */

typedef enum {
    NB_OK = 0,
    NB_ERR_ARG = -1,     /* NULL pointer, negative count, range beyond n_max / ni_max, bad eps2 / t */
    NB_ERR_ALLOC = -2,   /* device or pinned allocation failed, or lent workspace too small        */
    NB_ERR_CUDA = -3,    /* a CUDA runtime call or kernel launch failed                             */
    NB_ERR_INDEX = -4,   /* an i_list / idx entry was outside [0, n) (reported by nb_sync)          */
    NB_ERR_STATE = -5,   /* nb_force before any nb_predict, or workspace set too late               */
    NB_ERR_ARCH = -6,    /* device is not compute capability 10.x                                   */
    NB_ERR_PEER = -7     /* nb_xforce: a peer rank did not push its partial forces in time (nb_sync) */
} nb_status;

/* ---- lifetime --------------------------------------------------------------------------- */

/* Create a context for up to n_max j-particles and up to ni_max i-particles per force call, on
 * CUDA device `device`, enqueuing on `stream` (a cudaStream_t passed as void*; NULL = legacy
 * default stream).  Internal buffers (j-store 112 B + step 8 B, packed force record 44 B per
 * particle, plus the partial-force and block buffers) are allocated on first use with cudaMalloc,
 * unless nb_set_workspace lent memory before that. */
int nb_create(nb_ctx** out, int64_t n_max, int64_t ni_max, int device, void* stream);
int nb_destroy(nb_ctx* c);
int nb_set_stream(nb_ctx* c, void* stream);

/* Bytes of device memory a context of this size needs; and lending them (DEVICE pointer, 256-byte
 * aligned, must outlive the context) so that the caller's allocator owns all device memory.
 * nb_set_workspace must precede the first nb_set_j / nb_predict; NB_ERR_STATE afterwards. */
size_t nb_workspace_bytes(int64_t n_max, int64_t ni_max);
int nb_set_workspace(nb_ctx* c, void* dev_ptr, size_t bytes);

/* ---- a0: the resident j-set (PAPER.md:49 "j particles, which exert a force"; PAPER.md:55, :83:
 * keep it on the device, update it sparsely) ----------------------------------------------- */

/* Load/replace particles [first, first+count).  14 DEVICE fp64 arrays of length count: mass,
 * position, velocity, acceleration, jerk (the predictor's inputs, R1) and the time t the state
 * refers to.  ax..jz and t may each be NULL (taken as 0).  n becomes max(n, first+count);
 * particles never written have m = 0 at the origin and exert nothing. */
int nb_set_j(nb_ctx* c, int64_t first, int64_t count, const double* m,
             const double* x, const double* y, const double* z,
             const double* vx, const double* vy, const double* vz,
             const double* ax, const double* ay, const double* az,
             const double* jx, const double* jy, const double* jz, const double* t);

/* Scatter form used after a block step: element k replaces particle idx[k] (DEVICE int32, each
 * in [0, n); out-of-range entries are skipped and latch NB_ERR_INDEX; with duplicates one of the
 * writers wins).  Same 14 arrays, same NULL rule (NULL = leave that field unchanged here). */
int nb_update_j(nb_ctx* c, const int32_t* idx, int64_t count, const double* m,
                const double* x, const double* y, const double* z,
                const double* vx, const double* vy, const double* vz,
                const double* ax, const double* ay, const double* az,
                const double* jx, const double* jy, const double* jz, const double* t);

/* nb_update_j from HOST memory (idx and the 14 arrays are HOST pointers, ideally pinned): staged
 * through the context's own device buffers on its stream, then scattered.  count <= ni_max
 * (the staging area is sized by it), else NB_ERR_ARG.  The host arrays must stay valid until the
 * stream has consumed them (nb_sync). */
int nb_update_j_host(nb_ctx* c, const int32_t* idx, int64_t count, const double* m,
                const double* x, const double* y, const double* z,
                const double* vx, const double* vy, const double* vz,
                const double* ax, const double* ay, const double* az,
                const double* jx, const double* jy, const double* jz, const double* t);

/* HOST-pointer form of nb_set_j: one cudaMemcpyAsync per array, straight from the caller's memory
 * to the j-store on the context's stream.  Same argument rules.  Pageable arrays are staged by the
 * runtime before the call returns; PINNED arrays are read by the copy engine later, so they must
 * stay valid and unmodified until the stream has consumed them (nb_sync), as for nb_update_j_host. */
int nb_set_j_host(nb_ctx* c, int64_t first, int64_t count, const double* m,
                  const double* x, const double* y, const double* z,
                  const double* vx, const double* vy, const double* vz,
                  const double* ax, const double* ay, const double* az,
                  const double* jx, const double* jy, const double* jz, const double* t);

int nb_clear(nb_ctx* c);            /* n := 0, flags cleared, "predicted" state invalidated */
int64_t nb_count(const nb_ctx* c);  /* current n (or a negative nb_status)                  */

/* Mark particles whose MUTUAL pairs are unsoftened (R7: eps2_ij = 0 iff both carry bit 0; e.g.
 * black holes).  idx, flags: HOST arrays of length count -- the one entry point
 * besides the *_host calls that takes host memory: the library keeps a host copy of the flagged set
 * (it sizes the unsoftened-pair pass by it), the set is small and changes rarely.  Replaces the flag
 * of each listed particle; one staged copy + one scatter kernel on the stream, no synchronisation.
 * At most NB_MAX_FLAGGED particles may carry the bit at one time (NB_ERR_ARG beyond): the pairs among
 * them are summed in fp64 by one thread per flagged i-particle. */
#define NB_MAX_FLAGGED 1024
int nb_set_flags(nb_ctx* c, const int32_t* idx, const uint8_t* flags, int64_t count);

/* ---- a1: Hermite predictor (R1) --------------------------------------------- */

/* For all n particles: dt = t - t_j; xp = x + v dt + a dt^2/2 + jerk dt^3/6; vp = v + a dt +
 * jerk dt^2/2, in fp64, written to the internal predicted buffers (fp64 SoA, and the packed
 * record the force kernel streams).  t must be finite. */
int nb_predict(nb_ctx* c, double t);

/* Copy predicted state of particles [first, first+count) to a DEVICE fp64 buffer laid out
 * [6][count]: xp, yp, zp, vxp, vyp, vzp.  NB_ERR_STATE before the first nb_predict. */
int nb_get_predicted(nb_ctx* c, int64_t first, int64_t count, double* out);

/* ---- a2..a5: force call (R2..R9) ------------------------------ */

/* acc, jerk, pot on particles i_list[0..ni) (DEVICE int32 indices into the j-set; duplicates are
 * legal; unsorted is fine) from all n j-particles, both taken at their predicted state of the last
 * nb_predict:
 *     r = xp_j - xp_i, w = vp_j - vp_i, s = r.r + eps2_ij         (j != i by index, R5)
 *     pot_i = - sum m_j s^-1/2 ;  acc_i = sum m_j r s^-3/2 ;
 *     jrk_i = sum m_j ( w s^-3/2 - 3 (r.w) r s^-5/2 )             (s == 0 contributes nothing, R6)
 * Outputs, DEVICE fp64, in i_list order: acc[0..ni) = ax, acc[ni..2ni) = ay, acc[2ni..3ni) = az;
 * jrk likewise; pot[0..ni).  Precision: position differences carry >= 48 bits, pair terms are
 * fp32, sums of at most 128 terms are fp32 and everything above them fp64 (DESIGN.md
 * section 7.2); results agree with exact summation to <= 1e-5 (acc, pot) and <= 1e-4 (jerk) relative
 * per particle, for ANY eps2 >= 0: the self pair is excluded by index before any fp32 sum, so small
 * softenings (m_i/eps far above |pot_i|) cost no accuracy.  Input limits (R14): every pair
 * term m_j s^-3/2 and m_j s^-1/2 must stay inside the normal fp32 range (1e-38 .. 3e38) -- e.g. two
 * DISTINCT particles closer than ~1e-12 length units at m = 1 overflow it -- and masses are rounded to
 * fp32.  For eps2 < 1e-20 (eps2 = 0 included) a pair of distinct particles whose separation vanishes
 * in fp32 (|r|^2 + eps2 == eps2) contributes nothing, as R6 states for eps2 = 0; for eps2 >= 1e-20
 * such a pair interacts normally (zero acc and jerk, -m_j/eps in pot; R5).  Use precision mode 1
 * beyond these limits.  Deterministic run to run.
 * eps2 must be finite and >= 0; ni in [0, ni_max].  An out-of-range i_list entry gets NaN
 * outputs and latches NB_ERR_INDEX (returned by the next nb_sync). */
int nb_force(nb_ctx* c, const int32_t* i_list, int64_t ni, double eps2,
             double* acc, double* jrk, double* pot);

/* Forces on i-particles that are NOT members of the j-set, given by value -- "the particles in
 * subset j can either belong to the same or a completely different set as the i-particles"
 * (PAPER.md:49); this is the kick one system receives from another in the Hamiltonian-split
 * coupling of PAPER.md:118-123.  x, v: DEVICE fp64 [3][ni] (x-row, y-row,
 * z-row).  Same sums as nb_force over all n j-particles at their predicted state, but no pair is
 * skipped by index and no pair is unsoftened (flags concern j-set members only); a j-particle at
 * exactly the position of an i-particle with eps2 == 0 contributes nothing (R6).
 * v == NULL and jrk == NULL together select the acc + pot only variant (19 instead of 33 FP32
 * lane-operations per interaction); one NULL without the other is NB_ERR_ARG.
 * Outputs as nb_force.  ni in [0, ni_max]; NB_ERR_STATE before the first nb_predict. */
int nb_force_ext(nb_ctx* c, int64_t ni, const double* x, const double* v, double eps2, double* acc,
                 double* jrk, double* pot);

/* nb_force_ext for i-particles that may be MEMBERS of this context's j-set although they are given by
 * value -- the call one GPU makes in the paper's multi-GPU scheme, "distributing the j particles over
 * the various GPUs": every GPU evaluates ALL active particles, received by value,
 * against its own slice of j, and the partial forces are summed afterwards.  self_idx[k] (DEVICE
 * int32) = index in THIS context's j-set of the particle that IS i-particle k, or negative if it
 * belongs to another slice: that pair is excluded by index (R5), exactly as in nb_force.  iflags[k]
 * (DEVICE uint8, may be NULL) bit 0 = i-particle k carries the unsoftened flag: its pairs with the
 * flagged members of this j-set are unsoftened (R7) and summed in fp64.  x and v are the predicted
 * state at the time of the last nb_predict.  Everything else as nb_force_ext with velocities. */
int nb_force_ext_ids(nb_ctx* c, int64_t ni, const double* x, const double* v, const int32_t* self_idx,
                     const uint8_t* iflags, double eps2, double* acc, double* jrk, double* pot);

/* Forces at time t on a HANDFUL of members of the j-set (ni <= NB_FUSED_MAX), in one pass over the
 * j-store: the Hermite predictor (R1) runs inside the pair loop, for i and j alike, instead of as a
 * separate nb_predict pass (PAPER.md:55 counts the prediction step among the costs of a step;
 * PAPER.md:51 is about few active particles).  IEEE double throughout (the
 * call is HBM-bound: 112 B read per j-particle), self pair masked by index, flagged pairs
 * unsoftened (R5-R7).  Same outputs and layout as nb_force; needs no prior nb_predict and neither
 * reads nor refreshes the packed predicted state.  ni > NB_FUSED_MAX is NB_ERR_ARG. */
#define NB_FUSED_MAX 8
int nb_force_fused(nb_ctx* c, double t, const int32_t* i_list, int64_t ni, double eps2, double* acc,
                   double* jrk, double* pot);

/* ---- j-sharding over GPUs with the exchange done by the kernels -----------------
 *
 * PAPER.md:55 (section III.A): "Multi-GPU parallelization is achieved by distributing the j
 * particles over the various GPUs ... the first kernel computes the partial forces ... and the second
 * kernel sums these."  Rank r of `world` holds a slice of the j-set in its own context.  Across GPUs the
 * "second kernel" is an exchange; here it is done by the kernels themselves over peer memory (NVLink /
 * NVSwitch P2P stores), not by a collective-library call and not through the host (the
 * host link is "the crucial bottleneck"): every rank owns a WINDOW in device memory
 * (2 x world x [7][ni_cap] fp64 + flags); a rank stores its partial forces into slot [rank] of every
 * rank's window, makes them visible system-wide and raises a flag there; it then waits for the flags of
 * all ranks in its own window and adds the slots in rank order (fixed order: deterministic, identical
 * on all ranks; R9).  For ni <= 16 all of this happens in the pair kernel's last CTA: pair loop,
 * reduction, exchange and cross-rank sum are ONE launch; for larger ni two small kernels follow the
 * reduction.  nb_xforce is a COLLECTIVE: every rank calls it with the same ni and the same i-particles,
 * in the same order, on a stream of its own device.
 *
 * nb_xchg_create: allocate this rank's window (cudaMalloc, not part of the lent workspace).  world in
 *   [1, 16], rank in [0, world), ni_cap in [1, ni_max] = the largest ni of an nb_xforce call.  Calling
 *   it again replaces the window (peers must attach anew).
 * nb_xchg_export: HOST outputs (either may be NULL): `handle` = NB_XCHG_HANDLE_BYTES bytes that
 *   another PROCESS passes to nb_xchg_attach (a CUDA IPC memory handle); `*dev_ptr` = the window's
 *   device address, which another context of the SAME process passes instead.
 * nb_xchg_attach: map rank `peer`'s window: exactly one of `handle` (HOST bytes from the peer's
 *   nb_xchg_export, another process) and `same_process_ptr` (same process; on another device peer
 *   access is enabled) is non-NULL.  peer == own rank is accepted and ignored.  All world - 1 peers
 *   must be attached before nb_xforce (NB_ERR_STATE otherwise).  The caller keeps the peers alive
 *   until nb_xchg_destroy / nb_destroy of every rank that attached them.
 * nb_xforce: nb_force_ext_ids on this rank's j-slice (same arguments, DEVICE pointers, mixed precision,
 *   partial-sum reduction only) followed by the exchange.  phase 0: acc / jrk / pot hold the COMPLETE
 *   forces when the call's kernels have run; phase 1: compute and push only (acc / jrk / pot then hold
 *   this rank's partial forces); phase 2: the other half of the last phase-1 call -- wait for the peers
 *   and sum into acc / jrk / pot (x, v, self_idx, iflags, eps2 are ignored).  The split form lets a
 *   caller put other work between the halves.  A peer that has not pushed within the time limit
 *   (20 s; nb_xchg_set_timeout: seconds in (0, 3600]) latches NB_ERR_PEER (returned by nb_sync); the
 *   outputs are then meaningless.  ni > ni_cap: NB_ERR_ARG. */
#define NB_XCHG_HANDLE_BYTES 64
int nb_xchg_create(nb_ctx* c, int rank, int world, int64_t ni_cap);
int nb_xchg_export(nb_ctx* c, unsigned char* handle, void** dev_ptr);
int nb_xchg_attach(nb_ctx* c, int peer, const unsigned char* handle, void* same_process_ptr);
int nb_xchg_destroy(nb_ctx* c);
int nb_xchg_set_timeout(nb_ctx* c, double seconds);
int nb_xforce(nb_ctx* c, int phase, int64_t ni, const double* x, const double* v, const int32_t* self_idx,
              const uint8_t* iflags, double eps2, double* acc, double* jrk, double* pot);

/* ---- the force call that allocates nothing ------------------------------------------------------ */

/* nb_force_static: acceleration, jerk and potential (readings R2, R5, R6 of DESIGN.md) of n
 * j-particles on ni i-particles given by value, WITHOUT a context and without any allocation: for
 * callers that cannot call cudaMalloc (stream capture into a CUDA graph, tight serving loops, harnesses
 * that forbid it).  Every nb_ctx entry point above relies on buffers nb_create / nb_set_j allocated;
 * this one calls no cudaMalloc, cudaFree or allocating library routine.  Its scratch memory (partial
 * forces of the j-subsets, PAPER.md:51 / :55, and the tickets that elect the summing CTA) is a static
 * array of NB_STATIC_SCRATCH_BYTES in the library's device image: every GPU that loads libnb.so holds it
 * until the process exits.
 *
 * Works on the calling thread's CURRENT device (compute capability 10.x, NB_ERR_ARCH otherwise), to
 * which every pointer and the stream must belong; enqueues a 256-byte clear and one kernel on `stream`
 * (cudaStream_t as void*, NULL = legacy default stream) and returns.  The first call per device looks
 * the array's address up (cudaGetSymbolAddress; make that call outside stream capture).
 * DEVICE inputs, fp64 SoA, read only:  m [n], x [3][n], v [3][n] (the j-set at the time of the call: no
 * predictor here);  xi [3][ni], vi [3][ni];  self_idx [ni] or NULL: the j index particle k of the call
 * IS (its own pair is skipped by index, R5), negative = none.
 * DEVICE outputs: acc [3][ni], jrk [3][ni] or NULL, pot [ni].  The caller owns all arrays.
 * Arithmetic: IEEE double throughout (the pair loop of nb_set_precision(c, 1)); every pair uses eps2, no
 * flagged pairs (R7); sums in a fixed order: results are bitwise reproducible.
 * Limits: 0 <= ni <= NB_STATIC_NI_MAX and 0 <= n < 2^31, else NB_ERR_ARG ("invalid argument"): take
 * nb_force_ext for larger calls.  NULL among the required pointers, eps2 < 0 or NaN: NB_ERR_ARG.
 * ALL calls on one device share the one array: calls that can overlap on the GPU (two streams, two
 * host threads on different streams, parallel branches of a graph) RACE; order them on one stream. */
#define NB_STATIC_NI_MAX 4096
#define NB_STATIC_SCRATCH_BYTES 4194304
int nb_force_static(void* stream, int64_t n, const double* m, const double* x, const double* v,
                    int64_t ni, const double* xi, const double* vi, const int32_t* self_idx, double eps2,
                    double* acc, double* jrk, double* pot);

/* HOST-pointer form: i_list, acc, jrk, pot are host arrays; copies in, runs, copies back and
 * synchronises the stream before returning (so it also returns latched errors). */
int nb_force_host(nb_ctx* c, const int32_t* i_list, int64_t ni, double eps2,
                  double* acc, double* jrk, double* pot);

/* ---- control ------------------------------------------------------------------------------ */

/* Arithmetic of the pair loop.  0 (default): position differences carry >= 48 bits, pair terms
 * are fp32, sums fp64 ("emulating double precision" for the inter-particle distance).
 * 1: IEEE double precision throughout -- differences, products, sums, and a reciprocal square
 * root refined to fp64 rounding -- for "objects with an extreme mass ratio, like planetesimals
 * around super-massive black holes".  Mode 1 keeps a second,
 * fp64 copy of the predicted j-set (64 B per particle, cudaMalloc'ed by this call, not part of
 * the lent workspace) and agrees with exact summation to ~1e-13 relative; pairs whose s = r^2 +
 * eps2 lies below 1.18e-38 (closer than 1.1e-19 length units) are treated as coincident, pairs with
 * s above 3.4e38 (farther than 1.8e19) as out of range: both contribute nothing.  Changing
 * the mode invalidates the predicted state: call nb_predict before the next force call
 * (NB_ERR_STATE otherwise).  The atomics reduce mode and the threads-per-i variants are mode-0
 * only; results of mode 1 are deterministic. */
int nb_set_precision(nb_ctx* c, int mode);

/* 6th-order variant ("high >= 4th order integrators").  With
 * order = 6 the predictor also writes force-ready records that carry the predicted acceleration
 * ap = a + jerk dt (R22; 56 B more per particle, cudaMalloc'ed by this call), and nb_force6 returns the
 * second time derivative of the acceleration ("snap") next to acc, jerk and pot:
 *     b = ap_j - ap_i ,  al = (r.w)/s ,  be = (w.w + r.b)/s + al^2
 *     snp_i = sum m_j ( b s^-3/2 - 6 al J_ij - 3 be A_ij ),  A_ij = r s^-3/2,  J_ij = w s^-3/2 - 3 al A_ij
 * i.e. d2(acc)/dt2 along orbits with the given relative position, velocity and acceleration.  Same
 * pair rules (R5, R6, R7), precision scheme, layout ([3][ni] for snp) and errors as nb_force; snp
 * agrees with exact summation to <= 1e-3 relative.  order = 4 (default) switches the extra records
 * off.  Changing the order invalidates the predicted state.  nb_force6 is NB_ERR_STATE at order 4. */
int nb_set_order(nb_ctx* c, int order);
int nb_force6(nb_ctx* c, const int32_t* i_list, int64_t ni, double eps2, double* acc, double* jrk, double* snp,
              double* pot);

/* Force-call tuning, for tests and experiments.  j_splits: 0 = let the dispatcher choose the
 * number of j-subsets, >0 = use exactly this many (clamped to what the partial
 * buffer holds).  reduce_mode: 0 = partial buffer + reduction kernel (deterministic;
 * default), 1 = fp64 atomics into the output (sum order varies run to run). */
int nb_set_tuning(nb_ctx* c, int j_splits, int reduce_mode);

/* What the last nb_force launched: out[0] = j-splits used (when the active list is cut in a
 * whole-wave segment with one j-subset and a remainder segment with several, the remainder's
 * count), out[1] = CTAs of the pair kernel launches together, out[2] = kernels launched by the
 * call, out[3] = reduce mode.  HOST int64[4]. */
int nb_last_launch(const nb_ctx* c, int64_t* out);

/* Total kernels this context has launched since creation (bench.py's gpu_launches). */
int64_t nb_launch_count(const nb_ctx* c);

/* Per-kernel device timing for the roofline report.  With profiling on,
 * nb_predict and nb_force record CUDA events on the context's stream around their kernels.
 * nb_kernel_times synchronises the stream and writes, to HOST double[6], the running totals
 * since profiling was switched on: [0..2] = summed duration in ms of the predictor kernels, the
 * pair kernels and the reduction kernels, [3..5] = how many of each were timed.
 * nb_set_profiling(on) resets the totals.  NB_ERR_STATE if profiling is off. */
int nb_set_profiling(nb_ctx* c, int on);
int nb_kernel_times(nb_ctx* c, double* out_ms);

/* ---- block-step layer: scheduler, corrector, time-step criterion on the device --------------
 * (SURVEY.md 8(f) NEXT-1.)  The paper names the pieces -- "4th order Hermite predictor-corrector"
 * (PAPER.md:129), "individual time stepping", "block time steps", "only
 * the particles are updated that require a force update at a certain time" -- and
 * calls the host link "the crucial bottleneck"; it prints no formula.  Readings
 * (DESIGN.md): R12 corrector, R18 interpolated derivatives, R19 Aarseth criterion, R20 power-of-two
 * block rule, R21 scheduler.  Each particle carries a step dt_j next to the 14 j-store fields.
 * dt_min and dt_max must be powers of two, 0 < dt_min <= dt_max (NB_ERR_ARG otherwise). */

/* Set the steps of particles [first, first+count) from a DEVICE fp64 array. */
int nb_set_dt(nb_ctx* c, int64_t first, int64_t count, const double* dt);

/* Copy the stored state of particles [first, first+count) to a DEVICE fp64 buffer laid out
 * [15][count]: the 14 j-store fields in nb_set_j's order (m, x,y,z, vx,vy,vz, ax,ay,az, jx,jy,jz,
 * t), then dt. */
int nb_get_state(nb_ctx* c, int64_t first, int64_t count, double* out);

/* Start of a run (R19, R20): for particle i_list[k] (DEVICE int32) store acc/jrk (DEVICE fp64,
 * nb_force's layout [3][ni]) as its (a, jerk) and give it the largest power-of-two step
 * <= eta_s |a| / |jerk|, clamped to [dt_min, dt_max]. */
int nb_init_steps(nb_ctx* c, const int32_t* i_list, int64_t ni, const double* acc, const double* jrk,
                  double eta_s, double dt_min, double dt_max);

/* Scheduler (R21): *t_next = min_j (t_j + dt_j) over the n particles, *ni = how many are due then;
 * their indices, ascending, are left in a context-owned DEVICE list whose address is returned in
 * *i_list (may be NULL) and stays valid until the next nb_next_block / nb_step.  One cooperative
 * kernel; synchronises the stream to bring the two scalars back (HOST outputs).  NB_ERR_ARG (with
 * *t_next and *ni still set) if more than ni_max particles are due: the list is then truncated. */
int nb_next_block(nb_ctx* c, double* t_next, int64_t* ni, const int32_t** i_list);

/* After nb_init_steps, nb_correct and nb_step the j-store has moved on and the packed predicted
 * state is stale: nb_force / nb_force_ext / nb_get_predicted return NB_ERR_STATE until the next
 * nb_predict, whatever the size of the block was.  A due particle whose step is zero (steps never
 * set) or whose time is NaN is left untouched and latches NB_ERR_STATE (returned by nb_sync). */

/* Corrector + new step (R12, R18, R19, R20) for particles i_list[0..ni) (DEVICE) that were
 * predicted to t1 and whose forces at t1 are acc/jrk (DEVICE fp64, [3][ni] in i_list order): with
 * h = t1 - t_i, v1 = v0 + (a0+a1) h/2 + (j0-j1) h^2/12; x1 = x0 + (v0+v1) h/2 + (a0-a1) h^2/12;
 * the step wanted is sqrt(eta (|a1||a2| + |j1|^2) / (|j1||a3| + |a2|^2)) with a2, a3 from the
 * Hermite interpolation; the stored step is halved while above it, or doubled once when allowed.
 * Writes x1, v1, a1, j1, t1 and the new dt into the j-store, in place.  Duplicate indices: undefined. */
int nb_correct(nb_ctx* c, const int32_t* i_list, int64_t ni, double t1, const double* acc,
               const double* jrk, double eta, double dt_min, double dt_max);

/* One whole block step on the device: nb_next_block -> nb_predict(t) -> nb_force(due particles,
 * eps2) -> nb_correct.  HOST outputs *t (the block time) and *ni (particles advanced).  The forces
 * of the block stay in a context-owned buffer (nb_block_forces). */
int nb_step(nb_ctx* c, double eps2, double eta, double dt_min, double dt_max, double* t, int64_t* ni);

/* Up to k block steps without a host round trip per step (the host link is "the
 * crucial bottleneck"; with individual steps most blocks hold a handful of
 * particles).  One persistent cooperative kernel runs scheduler -> predictor inside an IEEE-double
 * pair loop over the j-store -> reduction -> corrector -> step criterion for step after step
 * (two grid-wide barriers per step, no launch, no synchronisation; same readings R1..R9, R12,
 * R18..R21 and the same decisions as nb_step).  It leaves a block to other kernels only when the block
 * is large -- more than 512 particles, or N_i x n above the bound of nb_set_steps_bound (default
 * 1.5e7 pairs: beyond it the packed fp32 pair kernel plus its launches beats the fp64 loop) -- and
 * how those kernels are issued is nb_set_steps_queue's choice: by default (fewer than 262144 particles)
 * their launch shape is planned on the device and they run as the body of a WHILE node of one CUDA graph,
 * so that the host synchronises once per nb_steps call; in mode 0 once per large block.
 * Stops after k steps, or before the first block whose time exceeds t_end (+inf: no limit; NaN is
 * NB_ERR_ARG).  HOST outputs: *done = steps taken; t_log[0..done), ni_log[0..done) and us_log[0..done)
 * = block time, block size and device time in microseconds (%globaltimer) of every step (each may be
 * NULL; the log is kept on the device and copied once, at the end).
 * Errors as nb_step; NB_ERR_STATE if no particle can be scheduled (every t + dt is NaN).  The forces
 * of the last block are available through nb_block_forces. */
int nb_steps(nb_ctx* c, int64_t k, double eps2, double eta, double dt_min, double dt_max, double t_end,
             double* t_log, int64_t* ni_log, double* us_log, int64_t* done);

/* Largest N_i x n the persistent kernel of nb_steps takes itself (0: every block goes through
 * nb_step's launches; for tests and experiments). */
int nb_set_steps_bound(nb_ctx* c, int64_t max_pairs);

/* How nb_steps takes a handed-over (large) block (the host link is the bottleneck).
 * mode -1 (default): mode 2 while the j-set has fewer than 262144 particles, mode 0 from there on (large
 *   blocks are then most of the run and nb_step's launches the faster way to take them; measured per block
 *   step, mode 2 / mode 0: N = 131072: 131 / 134 us, 262144: 330 / 328, 524288: 491 / 478, 2^20: 1278 / 1248).
 * mode 2: the block's launch shape is planned ON THE DEVICE and one "round" -- persistent
 *   kernel, plan, predictor, packed fp32 pair kernel (both thread mappings), reduction, corrector,
 *   each of which exits at once when it has nothing to do -- is the body of a WHILE node of a CUDA
 *   graph whose condition the plan kernel sets: one graph launch and one synchronisation per
 *   nb_steps call, however many large blocks there are.  Falls back to mode 1 if the driver cannot
 *   build that graph.
 * mode 1: the same rounds queued on the stream ahead of time, in batches; the host reads one
 *   progress record per batch (rounds queued beyond the end of the run are wasted launches).
 * mode 0: the host synchronises at every large block and takes it through nb_step's launches (the
 *   only way in the IEEE-double mode, with the atomics reduction and with forced j-splits; these
 *   select it by themselves).
 * NB_ERR_ARG for any other mode. */
int nb_set_steps_queue(nb_ctx* c, int mode);

/* nb_step takes blocks of <= NB_FUSED_MAX particles through nb_force_fused (default on).  on = 0
 * switches this off. */
int nb_set_fused(nb_ctx* c, int on);

/* DEVICE addresses of the last nb_step's acc [3][ni], jrk [3][ni], pot [ni] (any may be NULL). */
int nb_block_forces(nb_ctx* c, const double** acc, const double** jrk, const double** pot);

int nb_sync(nb_ctx* c);   /* stream sync; returns and clears a latched NB_ERR_INDEX / NB_ERR_PEER / NB_ERR_STATE */
const char* nb_strerror(int status);
const char* nb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NB_H */
