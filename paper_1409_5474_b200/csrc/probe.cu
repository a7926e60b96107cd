// probe.cu -- nb_probe_fp32: the attainable rate of the FP32 FMA pipe on this device, measured the
// way the pair kernel uses it: a full grid of 128-thread CTAs, 8 independent
// register chains per thread, scalar FFMA (kind 0) or packed FFMA2 (kind 1).  bench.py reports the
// pair kernel against the nominal peak AND against this measured rate.  Not on the hot path.
#include "nb_internal.h"

namespace nb {

namespace {

template <int KIND>
__global__ void __launch_bounds__(128) fma_rate_kernel(float* out, int iters, float a0)
{
    constexpr int NCH = 8;
    float2 f[NCH];
#pragma unroll
    for (int c = 0; c < NCH; ++c) f[c] = make_float2(a0 + c + threadIdx.x, a0 - c);
    const float2 m = make_float2(a0 * 0.999f, a0 * 1.001f);
    const float2 b = make_float2(a0 * 1e-3f, -a0 * 1e-3f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                if (KIND == 1) {
                    f[c] = __ffma2_rn(f[c], m, b);
                } else {
                    f[c].x = fmaf(f[c].x, m.x, b.x);
                    f[c].y = fmaf(f[c].y, m.y, b.y);
                }
            }
        }
    }
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < NCH; ++c) acc += f[c].x + f[c].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

}  // namespace

// FMA lane-operations per second (one fused multiply-add on one fp32 lane = 1) over the whole chip.
cudaError_t probe_fp32(int kind, int sm_count, float* scratch, cudaStream_t s, double* lane_ops_per_s)
{
    const int grid = sm_count * 8, iters = 2000;
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) {
        cudaEventDestroy(e0);
        return e;
    }
    float best = 0.f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, s);
        if (kind == 1) fma_rate_kernel<1><<<grid, 128, 0, s>>>(scratch, iters, 1.0f);
        else fma_rate_kernel<0><<<grid, 128, 0, s>>>(scratch, iters, 1.0f);
        cudaEventRecord(e1, s);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && (best == 0.f || ms < best)) best = ms;   // first launch is the warm-up
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return e;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    // per thread per iteration: 8 x 8 chain steps, each 2 lane-FMAs (both lanes of the pair)
    const double ops = (double)grid * 128.0 * iters * 64.0 * 2.0;
    *lane_ops_per_s = ops / ((double)best * 1e-3);
    return cudaSuccess;
}

}  // namespace nb
