// xchg.h -- the exchange step of the j-sharded scheme ("distributing the j particles over
// the various GPUs ... the first kernel computes the partial forces ... the second kernel sums these")
// done by the kernels themselves over peer memory (NVLink / NVSwitch P2P stores), not by a collective
// library call: every rank owns a WINDOW in its device memory; a rank that has its partial forces
// stores them into slot [its rank] of every rank's window (its own included), makes them visible
// system-wide and raises its flag there; a rank sums the slots of its own window in rank order (fixed
// order: deterministic and identical on every rank, R9) once all flags carry the call's epoch.
//
// Window of one rank (device memory, cudaMalloc'ed, exported with cudaIpcGetMemHandle):
//   [0, XCHG_HDR)                    unsigned flag[2][XCHG_MAX_WORLD]: epoch of the last complete push
//                                    of rank s into buffer b
//   XCHG_HDR + ...                   double data[2][world][NOUT][ni_cap]
// Two buffers, taken in turn by the epoch's parity: a rank can be at most one call ahead of a peer (its
// call e + 1 cannot complete before the peer has pushed e + 1, which the peer does after it has summed
// call e), so a push of call e + 2 never lands in a buffer that a peer still reads for call e.
#pragma once
#include "nb_internal.h"

namespace nb {

constexpr int XCHG_MAX_WORLD = 16;
constexpr int XCHG_HDR = 1024;

struct Xchg {                     // lives in device memory; written by nb_xchg_create / nb_xchg_attach
    int rank, world;
    long long ni_cap;
    unsigned char* win[XCHG_MAX_WORLD];   // window of every rank, as mapped into THIS device's address space
};

__device__ __forceinline__ double* xchg_slot(unsigned char* win, int buf, int src, int world, long long ni_cap)
{
    return reinterpret_cast<double*>(win + XCHG_HDR) + ((long long)(buf * world + src) * NOUT) * ni_cap;
}
__device__ __forceinline__ unsigned* xchg_flag(unsigned char* win, int buf, int src)
{
    return reinterpret_cast<unsigned*>(win) + buf * XCHG_MAX_WORLD + src;
}
__device__ __forceinline__ void st_release_sys(unsigned* p, unsigned v)
{
    asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire_sys(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ double ld_sys(const double* p)
{
    double v;
    asm volatile("ld.relaxed.sys.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long xchg_now()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// component c of particle k in the caller's SoA outputs (acc [3][ni], jrk [3][ni] or NULL, pot [ni])
__device__ __forceinline__ double* out_ptr(double* acc, double* jrk, double* pot, int c, long long k, long long ni)
{
    return c < 3 ? acc + c * ni + k : (c < 6 ? (jrk ? jrk + (c - 3) * ni + k : nullptr) : pot + k);
}

// Raise my flag for this epoch in every rank's window.  Call with the whole CTA, after every thread's
// stores into the windows: __threadfence_system() by every storing thread, a CTA barrier, then one
// release store per destination.
__device__ __forceinline__ void xchg_raise(const Xchg* X, unsigned epoch, int tid)
{
    __threadfence_system();
    __syncthreads();
    if (tid < X->world) st_release_sys(xchg_flag(X->win[tid], epoch & 1u, X->rank), epoch);
}

// Wait until every rank's flag in MY window carries the epoch (threads 0 .. world-1 poll one flag
// each; the others wait at the barrier).  A peer that does not answer within limit_ns latches bit 2 of
// *err (NB_ERR_PEER) and the wait ends: the sums are then wrong and the caller is told so by nb_sync.
__device__ __forceinline__ void xchg_wait(const Xchg* X, unsigned epoch, int tid, int* err, unsigned long long limit_ns)
{
    if (tid < X->world) {
        const unsigned* f = xchg_flag(X->win[X->rank], epoch & 1u, tid);
        const unsigned long long t0 = xchg_now();
        while (ld_acquire_sys(f) != epoch) {
            if (xchg_now() - t0 > limit_ns) {
                atomicOr(err, 4);
                break;
            }
            __nanosleep(64);
        }
    }
    __syncthreads();
}

// sum of the world slots of my window for (c, k), rank 0 first
__device__ __forceinline__ double xchg_sum(const Xchg* X, unsigned epoch, int c, long long k)
{
    unsigned char* w = X->win[X->rank];
    double s = ld_sys(xchg_slot(w, epoch & 1u, 0, X->world, X->ni_cap) + c * X->ni_cap + k);
    for (int r = 1; r < X->world; ++r) s += ld_sys(xchg_slot(w, epoch & 1u, r, X->world, X->ni_cap) + c * X->ni_cap + k);
    return s;
}

constexpr unsigned long long XCHG_LIMIT_NS = 20ull * 1000ull * 1000ull * 1000ull;   // default: 20 s (nb_xchg_set_timeout)

// The exchange inside the CTA that has just reduced a j-sharded call (force.cu few-i kernel, direct.cu):
// what R.acc / R.jrk / R.pot hold is this rank's PARTIAL force.  The CTA (NT threads, all of them call
// this) stores it into slot [rank] of every rank's window over peer memory, raises its flags, and --
// phase 0 -- waits for the peers' flags and adds the slots in rank order into R.acc / R.jrk / R.pot:
// pair loop, reduction, exchange and cross-rank sum are one launch, no collective call, no host.
template <int NT>
__device__ __forceinline__ void xchg_in_cta(const ReduceArgs& R, int* err, int tid)
{
    __syncthreads();                  // the sums of all warps are in R.acc / R.jrk / R.pot
    const Xchg* X = R.xchg;
    const int world = X->world, total = NOUT * R.ni;
    for (int q = tid; q < total; q += NT) {
        const int c = q / R.ni, k = q % R.ni;
        const double v = *out_ptr(R.acc, R.jrk, R.pot, c, k, R.ni);
        for (int p = 0; p < world; ++p)
            xchg_slot(X->win[p], R.xchg_epoch & 1u, X->rank, world, X->ni_cap)[c * X->ni_cap + k] = v;
    }
    xchg_raise(X, R.xchg_epoch, tid);
    if (R.xchg_phase == 0) {
        xchg_wait(X, R.xchg_epoch, tid, err, R.xchg_limit_ns);
        for (int q = tid; q < total; q += NT) {
            const int c = q / R.ni, k = q % R.ni;
            *out_ptr(R.acc, R.jrk, R.pot, c, k, R.ni) = xchg_sum(X, R.xchg_epoch, c, k);
        }
    }
}

// launchers (xchg.cu): the two halves as kernels of their own, for calls whose reduction is not done by
// the pair kernel's last CTA (ni > 16) and for the split-phase form of nb_xforce
cudaError_t launch_xchg_push(const Xchg* X, unsigned epoch, double* acc, double* jrk, double* pot, long long ni,
                             unsigned* ticket, cudaStream_t s);
cudaError_t launch_xchg_sum(const Xchg* X, unsigned epoch, double* acc, double* jrk, double* pot, long long ni, int* err,
                            unsigned long long limit_ns, cudaStream_t s);

}  // namespace nb
