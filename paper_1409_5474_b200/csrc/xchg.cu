// xchg.cu -- the two halves of the peer-memory exchange (xchg.h) as kernels of their own: for j-sharded
// force calls whose reduction is a separate kernel (N_i > 16) and for the split-phase form of nb_xforce.
// For a handful of active particles the same steps run inside the pair kernel's last CTA (force.cu), so
// that pair loop, reduction, exchange and cross-rank sum are ONE launch.
#include "xchg.h"
#include "pdl.h"

namespace nb {

namespace {

constexpr int XT = 256;

// my partial forces [7][ni] -> slot [my rank] of every rank's window; the CTA that draws the last ticket
// raises my flags (every CTA fenced its stores system-wide before it drew)
__global__ void __launch_bounds__(XT) xchg_push_kernel(const Xchg* __restrict__ X, unsigned epoch, double* acc, double* jrk,
                                                        double* pot, long long ni, unsigned* ticket)
{
    __shared__ int s_last;
    pdl_wait();       // pdl.h: the reduction before this kernel has written acc / jrk / pot
    const int world = X->world, rank = X->rank;
    const long long total = (long long)NOUT * ni;
    for (long long q = (long long)blockIdx.x * XT + threadIdx.x; q < total; q += (long long)gridDim.x * XT) {
        const int c = (int)(q / ni);
        const long long k = q % ni;
        const double* src = out_ptr(acc, jrk, pot, c, k, ni);
        const double v = src ? *src : 0.0;
        for (int p = 0; p < world; ++p) xchg_slot(X->win[p], epoch & 1u, rank, world, X->ni_cap)[c * X->ni_cap + k] = v;
    }
    __threadfence_system();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (s_last) {
        __threadfence_system();
        if (threadIdx.x < world) st_release_sys(xchg_flag(X->win[threadIdx.x], epoch & 1u, rank), epoch);
        if (threadIdx.x == 0) *ticket = 0u;
    }
}

// every CTA waits for the flags by itself (it depends on the peers only, never on another CTA of this
// grid), then sums its share of the slots in rank order
__global__ void __launch_bounds__(XT) xchg_sum_kernel(const Xchg* __restrict__ X, unsigned epoch, double* acc, double* jrk,
                                                       double* pot, long long ni, int* err, unsigned long long limit_ns)
{
    pdl_wait();       // pdl.h: my own push (the kernel before this one) is complete
    xchg_wait(X, epoch, threadIdx.x, err, limit_ns);
    const long long total = (long long)NOUT * ni;
    for (long long q = (long long)blockIdx.x * XT + threadIdx.x; q < total; q += (long long)gridDim.x * XT) {
        const int c = (int)(q / ni);
        const long long k = q % ni;
        double* dst = out_ptr(acc, jrk, pot, c, k, ni);
        if (dst) *dst = xchg_sum(X, epoch, c, k);
    }
}

unsigned grid_for(long long ni)
{
    long long g = ((long long)NOUT * ni + XT - 1) / XT;
    return (unsigned)(g < 1 ? 1 : (g > 592 ? 592 : g));
}

}  // namespace

cudaError_t launch_xchg_push(const Xchg* X, unsigned epoch, double* acc, double* jrk, double* pot, long long ni,
                             unsigned* ticket, cudaStream_t s)
{
    return pdl_launch(xchg_push_kernel, grid_for(ni), XT, 0, s, X, epoch, acc, jrk, pot, ni, ticket);
}

cudaError_t launch_xchg_sum(const Xchg* X, unsigned epoch, double* acc, double* jrk, double* pot, long long ni, int* err,
                            unsigned long long limit_ns, cudaStream_t s)
{
    return pdl_launch(xchg_sum_kernel, grid_for(ni), XT, 0, s, X, epoch, acc, jrk, pot, ni, err, limit_ns);
}

}  // namespace nb
