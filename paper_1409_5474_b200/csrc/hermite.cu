// hermite.cu -- the steps on either side of the force call, kept on the device (SURVEY.md 8(f)
// NEXT-1): block scheduler ("block time steps", "only the particles are
// updated that require a force update at a certain time"), Hermite corrector and time-step
// criterion ("4th order Hermite predictor-corrector", "individual time
// stepping").  The paper prints none of the formulas: DESIGN.md R12, R18..R21.  All fp64; these
// kernels are O(N) or O(N_i) and bandwidth/latency-bound, they exist so that a block step never
// leaves the GPU (the host link is "the crucial bottleneck").
#include <cooperative_groups.h>

#include "nb_internal.h"
#include "hermite_dev.h"
#include "pdl.h"

namespace cg = cooperative_groups;

namespace nb {

namespace {

constexpr int SEL_THREADS = 256;

// R21 in one cooperative launch: (1) t1 = min_j (t_j + dt_j); (2) per-block counts of the particles
// due at t1; (3) their indices, ascending, into list[0..ni).  meta: [0] = key of t1 (preset to
// ~0), [1] = ni (written by block 0).  counts: one int per block.
__global__ void __launch_bounds__(SEL_THREADS)
select_kernel(const double* __restrict__ t, const double* __restrict__ dt, int64_t n,
              unsigned long long* meta, int* counts, int32_t* list, int64_t cap)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ unsigned long long smin[SEL_THREADS / 32];
    __shared__ int ssum[SEL_THREADS / 32];
    __shared__ int sbase;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t chunk = ((n + gridDim.x - 1) / gridDim.x + SEL_THREADS - 1) / SEL_THREADS * SEL_THREADS;
    const int64_t lo = (int64_t)blockIdx.x * chunk;
    const int64_t hi = lo + chunk < n ? lo + chunk : n;

    unsigned long long k = ~0ull;
    for (int64_t p = lo + tid; p < hi; p += SEL_THREADS) {
        const unsigned long long q = key_of(t[p] + dt[p]);
        k = q < k ? q : k;
    }
#pragma unroll
    for (int w = 16; w >= 1; w >>= 1) {
        const unsigned long long o = __shfl_xor_sync(0xffffffffu, k, w);
        k = o < k ? o : k;
    }
    if (lane == 0) smin[warp] = k;
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < SEL_THREADS / 32; ++w) k = smin[w] < k ? smin[w] : k;
        atomicMin(meta, k);
    }
    grid.sync();

    const double t1 = of_key(*reinterpret_cast<volatile unsigned long long*>(meta));
    int cnt = 0;
    for (int64_t p = lo + tid; p < hi; p += SEL_THREADS) cnt += (t[p] + dt[p] == t1) ? 1 : 0;
#pragma unroll
    for (int w = 16; w >= 1; w >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, w);
    if (lane == 0) ssum[warp] = cnt;
    __syncthreads();
    if (tid == 0) {
        int s = 0;
        for (int w = 0; w < SEL_THREADS / 32; ++w) s += ssum[w];
        counts[blockIdx.x] = s;
    }
    grid.sync();

    // exclusive offset of this block = counts of the blocks before it
    int part = 0, all = 0;
    for (int b = tid; b < (int)gridDim.x; b += SEL_THREADS) {
        const int cb = *reinterpret_cast<volatile int*>(counts + b);
        all += cb;
        if (b < (int)blockIdx.x) part += cb;
    }
#pragma unroll
    for (int w = 16; w >= 1; w >>= 1) {
        part += __shfl_xor_sync(0xffffffffu, part, w);
        all += __shfl_xor_sync(0xffffffffu, all, w);
    }
    __syncthreads();
    if (lane == 0) {
        ssum[warp] = part;
        smin[warp] = (unsigned long long)all;
    }
    __syncthreads();
    if (tid == 0) {
        int s = 0;
        unsigned long long a = 0;
        for (int w = 0; w < SEL_THREADS / 32; ++w) {
            s += ssum[w];
            a += smin[w];
        }
        sbase = s;
        if (blockIdx.x == 0) meta[1] = a;
    }
    __syncthreads();
    int base = sbase;

    // ordered scatter, one slab of SEL_THREADS particles at a time
    for (int64_t p0 = lo; p0 < hi; p0 += SEL_THREADS) {
        const int64_t p = p0 + tid;
        const bool due = p < hi && (t[p] + dt[p] == t1);
        const unsigned bal = __ballot_sync(0xffffffffu, due);
        __syncthreads();
        if (lane == 0) ssum[warp] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < SEL_THREADS / 32; ++w) {
            const int c = ssum[w];
            total += c;
            if (w < warp) before += c;
        }
        if (due) {
            const int64_t pos = (int64_t)base + before + __popc(bal & ((1u << lane) - 1u));
            if (pos < cap) list[pos] = (int32_t)p;
        }
        base += total;
    }
}

// R12 + R18 + R19 + R20 for the particles list[0..ni): forces (a1, j1) at t1 are acc/jrk[c*ni + k].
// In place on the j-store; writes t = t1 and the new step.
__global__ void __launch_bounds__(128)
correct_kernel(StorePtrs st, double* __restrict__ dts, const int32_t* __restrict__ list, int64_t ni,
               int64_t n, double t1, const double* __restrict__ acc, const double* __restrict__ jrk,
               double eta, double dt_min, double dt_max, int* err)
{
    pdl_wait();       // pdl.h
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= ni) return;
    const int64_t i = list[k];
    if (i < 0 || i >= n) {
        atomicOr(err, 1);
        return;
    }
    double a1[3], j1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a1[c] = acc[(int64_t)c * ni + k];
        j1[c] = jrk[(int64_t)c * ni + k];
    }
    correct_one(st, dts, i, t1, a1, j1, eta, dt_min, dt_max, err);
}

// Start (R19, R20): store (a, j) of the listed particles and give each its first step.
__global__ void __launch_bounds__(128)
init_steps_kernel(StorePtrs st, double* __restrict__ dts, const int32_t* __restrict__ list, int64_t ni,
                  int64_t n, const double* __restrict__ acc, const double* __restrict__ jrk,
                  double eta_s, double dt_min, double dt_max, int* err)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= ni) return;
    const int64_t i = list[k];
    if (i < 0 || i >= n) {
        atomicOr(err, 1);
        return;
    }
    double a[3], j[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a[c] = acc[(int64_t)c * ni + k];
        j[c] = jrk[(int64_t)c * ni + k];
        st.f[F_AX + c][i] = a[c];
        st.f[F_JX + c][i] = j[c];
    }
    const double na = norm3(a[0], a[1], a[2]), nj = norm3(j[0], j[1], j[2]);
    const double want = nj > 0.0 ? eta_s * na / nj : __longlong_as_double(0x7ff0000000000000ll);
    double d = dt_max;
    while (d > want && d * 0.5 >= dt_min) d *= 0.5;
    dts[i] = d;
}

__global__ void __launch_bounds__(256)
get_state_kernel(StorePtrs st, const double* __restrict__ dts, int64_t first, int64_t count, double* out)
{
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= count) return;
#pragma unroll
    for (int f = 0; f < NFIELD; ++f) out[(int64_t)f * count + q] = st.f[f][first + q];
    out[(int64_t)NFIELD * count + q] = dts[first + q];
}

}  // namespace

cudaError_t launch_select(const double* t, const double* dt, int64_t n, unsigned long long* meta,
                          int* counts, int32_t* list, int64_t cap, int sm_count, cudaStream_t s)
{
    // meta[0] = ~0 (identity of the min); meta[1] is plainly written by block 0
    cudaError_t e = cudaMemsetAsync(meta, 0xff, 8, s);
    if (e != cudaSuccess) return e;
    int64_t want = (n + SEL_THREADS - 1) / SEL_THREADS;
    int grid = sm_count * 4;                       // co-resident by a wide margin (256 threads, ~2 KB smem)
    if (grid > SEL_MAX_BLOCKS) grid = SEL_MAX_BLOCKS;
    if (want < grid) grid = (int)(want > 0 ? want : 1);
    void* args[] = {(void*)&t, (void*)&dt, (void*)&n, (void*)&meta, (void*)&counts, (void*)&list, (void*)&cap};
    return cudaLaunchCooperativeKernel((const void*)select_kernel, dim3(grid), dim3(SEL_THREADS), args, 0, s);
}

cudaError_t launch_correct(const StorePtrs& st, double* dts, const int32_t* list, int64_t ni, int64_t n,
                           double t1, const double* acc, const double* jrk, double eta, double dt_min,
                           double dt_max, int* err, cudaStream_t s)
{
    if (ni == 0) return cudaSuccess;
    return pdl_launch(correct_kernel, (unsigned)((ni + 127) / 128), 128, 0, s, st, dts, list, ni, n, t1, acc, jrk, eta, dt_min,
                      dt_max, err);
}

cudaError_t launch_init_steps(const StorePtrs& st, double* dts, const int32_t* list, int64_t ni, int64_t n,
                              const double* acc, const double* jrk, double eta_s, double dt_min,
                              double dt_max, int* err, cudaStream_t s)
{
    if (ni == 0) return cudaSuccess;
    init_steps_kernel<<<(unsigned)((ni + 127) / 128), 128, 0, s>>>(st, dts, list, ni, n, acc, jrk, eta_s,
                                                                   dt_min, dt_max, err);
    return cudaGetLastError();
}

cudaError_t launch_get_state(const StorePtrs& st, const double* dts, int64_t first, int64_t count,
                             double* out, cudaStream_t s)
{
    if (count == 0) return cudaSuccess;
    get_state_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(st, dts, first, count, out);
    return cudaGetLastError();
}

}  // namespace nb
