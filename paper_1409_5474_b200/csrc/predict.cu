// predict.cu -- a0 (j-store load / scatter) and a1 (Hermite predictor) kernels.
//
// The predictor ("optional prediction step on the j particles"; reading
// R1 in DESIGN.md) is bandwidth-bound: per particle it reads the 14 fp64 fields of the j-store
// (112 B) and writes one 44-byte force-ready record (two-float position, fp32 velocity and mass,
// flag word) into the tiled pack the pair kernel streams.  All accesses are unit-stride across
// the warp; each thread handles two particles so that loads are 128-bit and stores 64-bit.
#include "nb_internal.h"
#include "pdl.h"

namespace nb {

namespace {

__global__ void __launch_bounds__(256) set_j_kernel(StorePtrs dst, SrcPtrs src, int64_t first,
                                                    int64_t count)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < count; p += stride) {
#pragma unroll
        for (int f = 0; f < NFIELD; ++f)
            dst.f[f][first + p] = src.f[f] ? src.f[f][p] : 0.0;
    }
}

__global__ void __launch_bounds__(256) update_j_kernel(StorePtrs dst, SrcPtrs src,
                                                       const int32_t* __restrict__ idx,
                                                       int64_t count, int64_t n, int* err)
{
    pdl_wait();       // pdl.h
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < count; p += stride) {
        const int64_t q = idx[p];
        if (q < 0 || q >= n) {
            atomicOr(err, 1);
            continue;
        }
#pragma unroll
        for (int f = 0; f < NFIELD; ++f)
            if (src.f[f]) dst.f[f][q] = src.f[f][p];
    }
}

// nb_set_flags: stage[0..count) = particle indices, stage[count..2 count) = new flag values, in
// order (a particle listed twice -- leaving the old set and entering the new one -- ends as 1
// because one thread walks the list)
__global__ void set_flags_kernel(uint8_t* flags, const int32_t* __restrict__ stage, int count)
{
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (int k = 0; k < count; ++k) flags[stage[k]] = (uint8_t)stage[count + k];
}

__device__ __forceinline__ double2 ld2(const double* p, int64_t i)
{
    return __ldg(reinterpret_cast<const double2*>(p + i));
}

// split a double into hi + lo floats (hi = nearest float, lo = nearest float of the remainder):
// hi + lo carries >= 48 bits of x (emulated double for the inter-particle distance).
__device__ __forceinline__ void split(double x, float& hi, float& lo)
{
    hi = __double2float_rn(x);
    lo = __double2float_rn(x - (double)hi);
}

// One thread = particles 2q, 2q+1.  n_pad = ntiles * TJ; particles in [n, n_pad) become m = 0
// padding records far away.  Store arrays are n_cap >= n_pad long, so loads never leave them.
// P64: also write the fp64 tiles of the full-double pair loop (force64.cu; 64 B more per particle).
// P6: also write the tiles of the 6th-order pair loop (force6.cu; 56 B more), which carry the
// predicted acceleration a + jerk dt (R22).
template <bool P64, bool P6>
__global__ void __launch_bounds__(128) predict_kernel(StorePtrs st, const uint8_t* __restrict__ flags,
                                                      float* __restrict__ pack,
                                                      double* __restrict__ pack64, float* __restrict__ pack6,
                                                      int64_t n, int64_t n_pad, double t,
                                                      const DynPlan* __restrict__ plan)
{
    pdl_wait();       // pdl.h (a no-op in the rounds nb_steps queues: those are launched without the attribute)
    if (plan) {                   // a block planned on the device (nb_steps): its time, or nothing to do
        if (!plan->go) return;
        t = plan->t1;
    }
    const int64_t p = 2 * ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
    if (p >= n_pad) return;
    const double2 tj = ld2(st.f[F_T], p);
    const double dt0 = t - tj.x, dt1 = t - tj.y;
    float2 out[NPF];
    double2 o64[NQF];
    float2 oa[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double2 x = ld2(st.f[F_X + c], p), v = ld2(st.f[F_VX + c], p);
        const double2 a = ld2(st.f[F_AX + c], p), j = ld2(st.f[F_JX + c], p);
        double xp0, vp0, xp1, vp1;
        predict1(x.x, v.x, a.x, j.x, dt0, xp0, vp0);
        predict1(x.y, v.y, a.y, j.y, dt1, xp1, vp1);
        split(xp0, out[P_XH + c].x, out[P_XL + c].x);
        split(xp1, out[P_XH + c].y, out[P_XL + c].y);
        out[P_VX + c] = make_float2(__double2float_rn(vp0), __double2float_rn(vp1));
        if (P6) oa[c] = make_float2(__double2float_rn(fma(j.x, dt0, a.x)), __double2float_rn(fma(j.y, dt1, a.y)));
        if (P64) {
            o64[Q_X + c] = make_double2(xp0, xp1);
            o64[Q_VX + c] = make_double2(vp0, vp1);
        }
    }
    const double2 m = ld2(st.f[F_M], p);
    out[P_M] = make_float2(__double2float_rn(m.x), __double2float_rn(m.y));
    const uchar2 fl = *reinterpret_cast<const uchar2*>(flags + p);
    out[P_FLAG] = make_float2(__uint_as_float(fl.x & 1u), __uint_as_float(fl.y & 1u));
    if (p >= n || p + 1 >= n) {
#pragma unroll
        for (int f = 0; f < NPF; ++f) {
            const float pad = (f <= P_ZH) ? PAD_POS : 0.0f;
            if (p >= n) out[f].x = pad;
            if (p + 1 >= n) out[f].y = pad;
        }
    }
    if (P64) {
        o64[Q_M] = m;
        o64[Q_FLAG] = make_double2((double)(fl.x & 1u), (double)(fl.y & 1u));
#pragma unroll
        for (int f = 0; f < NQF; ++f) {
            const double pad = (f <= Q_Z) ? (double)PAD_POS : 0.0;
            if (p >= n) o64[f].x = pad;
            if (p + 1 >= n) o64[f].y = pad;
        }
        double* b64 = pack64 + (p / TJ) * TILE64_DOUBLES + (p % TJ);
#pragma unroll
        for (int f = 0; f < NQF; ++f) *reinterpret_cast<double2*>(b64 + f * TJ) = o64[f];
    }
    float* base = pack + (p / TJ) * TILE_FLOATS + (p % TJ);
#pragma unroll
    for (int f = 0; f < NPF; ++f) *reinterpret_cast<float2*>(base + f * TJ) = out[f];
    if (P6) {
        // same records with the acceleration between velocity and mass: xh xl v | a | m flag
        float* b6 = pack6 + (p / TJ) * TILE6_FLOATS + (p % TJ);
#pragma unroll
        for (int f = 0; f < 9; ++f) *reinterpret_cast<float2*>(b6 + f * TJ) = out[f];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if (p >= n) oa[c].x = 0.0f;
            if (p + 1 >= n) oa[c].y = 0.0f;
            *reinterpret_cast<float2*>(b6 + (9 + c) * TJ) = oa[c];
        }
        *reinterpret_cast<float2*>(b6 + 12 * TJ) = out[P_M];
        *reinterpret_cast<float2*>(b6 + 13 * TJ) = out[P_FLAG];
    }
}

__global__ void __launch_bounds__(256) get_predicted_kernel(StorePtrs st, int64_t first,
                                                            int64_t count, double t, double* out)
{
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= count) return;
    const int64_t p = first + q;
    const double dt = t - st.f[F_T][p];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double xp, vp;
        predict1(st.f[F_X + c][p], st.f[F_VX + c][p], st.f[F_AX + c][p], st.f[F_JX + c][p], dt, xp, vp);
        out[(int64_t)c * count + q] = xp;
        out[(int64_t)(3 + c) * count + q] = vp;
    }
}

inline int grid_for(int64_t work, int block, int cap)
{
    int64_t g = (work + block - 1) / block;
    if (g < 1) g = 1;
    if (g > cap) g = cap;
    return (int)g;
}

}  // namespace

cudaError_t launch_set_j(const StorePtrs& dst, const SrcPtrs& src, int64_t first, int64_t count,
                         cudaStream_t s)
{
    if (count == 0) return cudaSuccess;
    set_j_kernel<<<grid_for(count, 256, 148 * 16), 256, 0, s>>>(dst, src, first, count);
    return cudaGetLastError();
}

cudaError_t launch_update_j(const StorePtrs& dst, const SrcPtrs& src, const int32_t* idx,
                            int64_t count, int64_t n, int* err, cudaStream_t s)
{
    if (count == 0) return cudaSuccess;
    return pdl_launch(update_j_kernel, grid_for(count, 256, 148 * 16), 256, 0, s, dst, src, idx, count, n, err);
}

cudaError_t launch_set_flags(uint8_t* flags, const int32_t* idx_then_val, int count, cudaStream_t s)
{
    set_flags_kernel<<<1, 32, 0, s>>>(flags, idx_then_val, count);
    return cudaGetLastError();
}

cudaError_t launch_predict(const StorePtrs& store, const uint8_t* flags, float* pack, double* pack64,
                           float* pack6, int64_t n, double t, cudaStream_t s, const DynPlan* plan)
{
    if (n == 0) return cudaSuccess;
    const int64_t n_pad = (n + TJ - 1) / TJ * TJ;
    const int64_t threads = n_pad / 2;
    const unsigned grid = (unsigned)((threads + 127) / 128);
    if (pack64 && pack6) predict_kernel<true, true><<<grid, 128, 0, s>>>(store, flags, pack, pack64, pack6, n, n_pad, t, plan);
    else if (pack64) predict_kernel<true, false><<<grid, 128, 0, s>>>(store, flags, pack, pack64, nullptr, n, n_pad, t, plan);
    else if (pack6) predict_kernel<false, true><<<grid, 128, 0, s>>>(store, flags, pack, nullptr, pack6, n, n_pad, t, plan);
    else if (plan) predict_kernel<false, false><<<grid, 128, 0, s>>>(store, flags, pack, nullptr, nullptr, n, n_pad, t, plan);
    else   // the default mode outside nb_steps' queued rounds: may be set up while the kernel before it drains
        return pdl_launch(predict_kernel<false, false>, grid, 128, 0, s, store, flags, pack, (double*)nullptr, (float*)nullptr, n,
                          n_pad, t, plan);
    return cudaGetLastError();
}

cudaError_t launch_get_predicted(const StorePtrs& store, int64_t first, int64_t count, double t,
                                 double* out, cudaStream_t s)
{
    if (count == 0) return cudaSuccess;
    get_predicted_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(store, first, count, t, out);
    return cudaGetLastError();
}

}  // namespace nb
