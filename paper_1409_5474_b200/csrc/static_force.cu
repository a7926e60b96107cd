// static_force.cu -- nb_force_static: the by-value force call (forces of the j-particles on
// the i-particles it is given; j split in blocks + partial-force sum) for callers that
// must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// Every other entry point works on an nb_ctx, whose buffers nb_create / the first nb_set_j allocate.  This
// one takes no context.  It is a variant of force64.cu's kernel (IEEE-double pair loop, i by value,
// thread per i, j split over CTAs): the j-set is read straight from the caller's SoA arrays instead of a
// predicted pack, and the scratch memory of the j-split -- the partial forces [split][7][ni_pad] and the
// per-i-tile tickets that elect the CTA which adds them -- is the file-scope array below, part of the
// library's image on every GPU that loads it (NB_STATIC_SCRATCH_BYTES, held until the process exits).
// The function calls no cudaMalloc / cudaFree / allocating library routine, ever.
//
// One array per device, shared by every call: two calls that overlap on the GPU (different streams, or
// graph branches) race on it.  It keeps the last call's contents: the partials are overwritten before
// they are read; the tickets must start at zero and are cleared on the stream before every launch.
#include <mutex>

#include "nb_internal.h"
#include "pair64.h"

// THE scratch memory (file scope).  In host code this name is a host-side stand-in, not a device address:
// the kernel is given what cudaGetSymbolAddress returns for it (scratch_of_current_device below).
static __device__ __align__(256) unsigned char nb_static_scratch[NB_STATIC_SCRATCH_BYTES];

namespace nb {

namespace {

constexpr int SF_THREADS = 128;
constexpr int SF_TJ = 128;                    // j per shared-memory tile (one per thread to load)
constexpr int SF_TICKET_BYTES = 256;          // unsigned ticket[64], one per i-tile
constexpr int SF_MAX_ITILES = SF_TICKET_BYTES / 4;
constexpr int SF_MAX_SPLITS = 64;
constexpr int SF_WANT_CTAS = 592;             // a constant, not SMs x occupancy: same split on every device
constexpr size_t SF_PART_BYTES = (size_t)NB_STATIC_SCRATCH_BYTES - SF_TICKET_BYTES;

static_assert(NB_STATIC_NI_MAX <= SF_MAX_ITILES * SF_THREADS, "a ticket per i-tile");
static_assert((size_t)NOUT * NB_STATIC_NI_MAX * sizeof(double) <= SF_PART_BYTES, "one split must fit");

struct StaticArgs {
    const double* m;                          // [n]
    const double* x;                          // [3][n]
    const double* v;                          // [3][n]
    const double* xi;                         // [3][ni]
    const double* vi;                         // [3][ni]
    const int32_t* self_idx;                  // [ni] or NULL
    double *acc, *jrk, *pot;                  // [3][ni], [3][ni] or NULL, [ni]
    unsigned char* scratch;                   // device address of nb_static_scratch
    int64_t n;
    double eps2;
    int ni, ni_pad, n_itiles, splits, ntiles;
};

// IPT i-particles per thread; CTA (it, sp) = i-tile it x j-subset sp of `splits`
template <int IPT>
__global__ void __launch_bounds__(SF_THREADS) static_force_kernel(StaticArgs P)
{
    constexpr int ITILE_S = IPT * SF_THREADS;
    __shared__ double sj[2][7][SF_TJ];        // x y z vx vy vz m of one j-tile, two buffers
    __shared__ int s_last;
    const int tid = threadIdx.x;
    const int it = blockIdx.x % P.n_itiles;
    const int sp = blockIdx.x / P.n_itiles;
    const int t0 = (int)(((int64_t)P.ntiles * sp) / P.splits);
    const int t1 = (int)(((int64_t)P.ntiles * (sp + 1)) / P.splits);

    double xi[IPT][6];
    int64_t self[IPT];
    Acc64 A[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int k = it * ITILE_S + u * SF_THREADS + tid;
        const bool on = k < P.ni;
        const int e = on ? k : 0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            xi[u][c] = P.xi[(int64_t)c * P.ni + e];
            xi[u][3 + c] = P.vi[(int64_t)c * P.ni + e];
        }
        self[u] = (on && P.self_idx) ? (int64_t)P.self_idx[e] : -1;     // never equals a j index when < 0
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = 0.0;
    }

    // my particle of a tile: the seven doubles, or a massless one beyond n (contributes nothing)
    auto fetch = [&](int t, double* r) {
        const int64_t j = (int64_t)t * SF_TJ + tid;
        if (j < P.n) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                r[c] = P.x[(int64_t)c * P.n + j];
                r[3 + c] = P.v[(int64_t)c * P.n + j];
            }
            r[6] = P.m[j];
        } else {
#pragma unroll
            for (int c = 0; c < 7; ++c) r[c] = 0.0;
        }
    };

    double r[7];
    if (t0 < t1) fetch(t0, r);
    for (int t = t0; t < t1; ++t) {
        const int b = (t - t0) & 1;
#pragma unroll
        for (int c = 0; c < 7; ++c) sj[b][c][tid] = r[c];
        __syncthreads();                      // tile t is in sj[b]; everybody is done with tile t - 1
        if (t + 1 < t1) fetch(t + 1, r);      // in flight under the pair loop
        const int64_t jbase = (int64_t)t * SF_TJ;
#pragma unroll 2
        for (int p = 0; p < SF_TJ; p += 2) {
            double2 g[7];
#pragma unroll
            for (int c = 0; c < 7; ++c) g[c] = *reinterpret_cast<const double2*>(&sj[b][c][p]);
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                pair64<true>(xi[u], A[u], g[0].x, g[1].x, g[2].x, g[3].x, g[4].x, g[5].x, g[6].x, P.eps2,
                             self[u] == jbase + p);
                pair64<true>(xi[u], A[u], g[0].y, g[1].y, g[2].y, g[3].y, g[4].y, g[5].y, g[6].y, P.eps2,
                             self[u] == jbase + p + 1);
            }
        }
    }

    // partial forces of this j-subset -> scratch [sp][c][k]
    unsigned* ticket = reinterpret_cast<unsigned*>(P.scratch);
    double* part = reinterpret_cast<double*>(P.scratch + SF_TICKET_BYTES);
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int k = it * ITILE_S + u * SF_THREADS + tid;
        const double o[NOUT] = {A[u].ax, A[u].ay, A[u].az, A[u].jx, A[u].jy, A[u].jz, A[u].p};
#pragma unroll
        for (int c = 0; c < NOUT; ++c) part[((int64_t)sp * NOUT + c) * P.ni_pad + k] = o[c];
    }

    // the CTA that draws the last ticket of this i-tile adds the subsets in order (deterministic)
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(&ticket[it], 1u) == (unsigned)P.splits - 1u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int q = tid; q < NOUT * ITILE_S; q += SF_THREADS) {
        const int c = q / ITILE_S, k = it * ITILE_S + q % ITILE_S;
        if (k >= P.ni) continue;
        double s = 0.0;
        for (int w = 0; w < P.splits; ++w) s += __ldcg(&part[((int64_t)w * NOUT + c) * P.ni_pad + k]);
        if (c < 3) P.acc[(int64_t)c * P.ni + k] = s;
        else if (c < 6) {
            if (P.jrk) P.jrk[(int64_t)(c - 3) * P.ni + k] = s;
        } else P.pot[k] = s;
    }
    if (tid == 0) ticket[it] = 0u;            // as the next call's clear would leave it
}

// Set-up, once per device, with that device current: the device address of the array on THIS device.
constexpr int SF_MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char* g_scratch[SF_MAX_DEVICES];
int g_state[SF_MAX_DEVICES];                  // 0 = not set up, 1 = ready, < 0 = the nb_status it failed with

int scratch_of_current_device(unsigned char** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return NB_ERR_CUDA;
    if (dev < 0 || dev >= SF_MAX_DEVICES) return NB_ERR_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_state[dev] == 0) {
        int major = 0;
        void* p = nullptr;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
            g_state[dev] = NB_ERR_CUDA;
        } else if (major != 10) {
            g_state[dev] = NB_ERR_ARCH;
        } else if (cudaGetSymbolAddress(&p, nb_static_scratch) != cudaSuccess || p == nullptr) {
            (void)cudaGetLastError();
            g_state[dev] = NB_ERR_CUDA;
        } else {
            g_scratch[dev] = static_cast<unsigned char*>(p);
            g_state[dev] = 1;
        }
    }
    if (g_state[dev] != 1) return g_state[dev];
    *out = g_scratch[dev];
    return NB_OK;
}

}  // namespace

}  // namespace nb

extern "C" int nb_force_static(void* stream, int64_t n, const double* m, const double* x, const double* v,
                               int64_t ni, const double* xi, const double* vi, const int32_t* self_idx,
                               double eps2, double* acc, double* jrk, double* pot)
{
    using namespace nb;
    if (n < 0 || ni < 0 || ni > NB_STATIC_NI_MAX || n > 2147483647ll) return NB_ERR_ARG;
    if (!(eps2 >= 0.0) || !(eps2 < 1e300)) return NB_ERR_ARG;
    if (ni == 0) return NB_OK;
    if (!xi || !vi || !acc || !pot || (n > 0 && (!m || !x || !v))) return NB_ERR_ARG;
    unsigned char* scratch = nullptr;
    const int st = scratch_of_current_device(&scratch);
    if (st != NB_OK) return st;

    StaticArgs a;
    a.m = m; a.x = x; a.v = v; a.xi = xi; a.vi = vi; a.self_idx = self_idx;
    a.acc = acc; a.jrk = jrk; a.pot = pot;
    a.scratch = scratch;
    a.n = n;
    a.eps2 = eps2;
    a.ni = (int)ni;
    const int ipt = ni > 1024 ? 2 : 1;
    const int itile = ipt * SF_THREADS;
    a.n_itiles = (int)((ni + itile - 1) / itile);
    a.ni_pad = a.n_itiles * itile;
    a.ntiles = (int)((n + SF_TJ - 1) / SF_TJ);
    int64_t splits = (SF_WANT_CTAS + a.n_itiles - 1) / a.n_itiles;
    const int64_t fit = (int64_t)(SF_PART_BYTES / ((size_t)NOUT * a.ni_pad * sizeof(double)));
    if (splits > fit) splits = fit;
    if (splits > SF_MAX_SPLITS) splits = SF_MAX_SPLITS;
    if (splits > a.ntiles) splits = a.ntiles;
    if (splits < 1) splits = 1;               // n = 0: one CTA per i-tile stores zeros
    a.splits = (int)splits;

    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (cudaMemsetAsync(scratch, 0, SF_TICKET_BYTES, s) != cudaSuccess) return NB_ERR_CUDA;
    const unsigned grid = (unsigned)a.n_itiles * (unsigned)a.splits;
    if (ipt == 2) static_force_kernel<2><<<grid, SF_THREADS, 0, s>>>(a);
    else static_force_kernel<1><<<grid, SF_THREADS, 0, s>>>(a);
    return cudaGetLastError() == cudaSuccess ? NB_OK : NB_ERR_CUDA;
}
