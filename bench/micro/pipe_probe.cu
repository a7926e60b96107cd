// pipe_probe.cu -- standalone probe of the SM pipes the pair kernels live on.
// Not part of libnb.so and not on any product path (micro-benchmarks
// that gate the design live in bench/micro/): it exists so that the rates DESIGN.md quotes (FFMA vs
// FFMA2, FP64 lanes per clock, MUFU, F2F, and whether the pipes overlap) can be re-measured:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pipe_probe bench/micro/pipe_probe.cu && ./pipe_probe [all|rates|bodies|hetero]
// Part 1 (rates): raw instruction rates (8 independent register chains per thread, full chip).
// Part 2 (bodies): candidate pair bodies of SURVEY.md section 7's encoding table, loop only (no
//         tile pipeline): C = two-float positions (what force_kernel runs), D = fp64 position
//         differences + F2F.F32.F64 (3 DADD + 3 F2F per interaction, 24 FP32 lane-ops), and mixes.
// Part 3 (hetero): fp32 warps and fp64 warps side by side in one CTA (round 1's experiment).
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cstring>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while (0)

__device__ __forceinline__ float rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// ---------------- raw pipe rates: NCH independent chains per thread ----------------
// kind 0 FFMA2, 1 FFMA, 2 FADD2, 3 DADD, 5 MUFU.RSQ, 6 FMUL2, 7 DFMA, 8 IADD3/LOP3 mix (alu),
// 9: FFMA2 + alu interleaved 1:1, 10: FFMA2 + DADD 4:1, 12: FFMA2 + MUFU 8:1, 13/14: FFMA2 + FFMA,
// 17: F2F.F32.F64 (one per step, fed by a DADD, consumed by an FADD), 11: FFMA2 + (DADD, F2F) 4:1,
// 18: body D's mix per interaction: 12 FFMA2 : 3 DADD : 3 F2F : 1 MUFU (scaled: 32 : 8 : 8 : ~2.7)
template <int KIND>
__global__ void __launch_bounds__(128) rate_kernel(float* out, int iters, float a0, double d0)
{
    constexpr int NCH = 8;
    float2 f[NCH], g[NCH];
    double d[NCH];
    unsigned u[NCH];
    float s[NCH];
    for (int c = 0; c < NCH; ++c) {
        f[c] = make_float2(a0 + c + threadIdx.x, a0 - c);
        g[c] = make_float2(a0 * 0.5f + c, a0 + 2 * c);
        d[c] = d0 + c + threadIdx.x;
        u[c] = threadIdx.x * 31 + c;
        s[c] = a0 + c * 0.5f + threadIdx.x;
    }
    const float2 m = make_float2(a0 * 0.999f, a0 * 1.001f);
    const float2 b = make_float2(a0 * 1e-3f, -a0 * 1e-3f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                if (KIND == 0) f[c] = __ffma2_rn(f[c], m, b);
                if (KIND == 1) s[c] = fmaf(s[c], m.x, b.x);
                if (KIND == 2) f[c] = __fadd2_rn(f[c], b);
                if (KIND == 3) d[c] = __dadd_rn(d[c], d0);
                if (KIND == 5) s[c] = rsq(s[c]);
                if (KIND == 6) f[c] = __fmul2_rn(f[c], m);
                if (KIND == 7) d[c] = fma(d[c], d0, d0);
                if (KIND == 8) { u[c] = (u[c] + 0x9e3779b9u) ^ (u[c] >> 3); }
                if (KIND == 9) { f[c] = __ffma2_rn(f[c], m, b); u[c] = (u[c] & 0x7fffffffu) + 0x38000001u; }
                if (KIND == 10) { f[c] = __ffma2_rn(f[c], m, b); if ((c & 3) == 0) d[c] = __dadd_rn(d[c], d0); }
                if (KIND == 13) { f[c] = __ffma2_rn(f[c], m, b); s[c] = fmaf(s[c], m.x, b.x); }
                if (KIND == 14) { f[c] = __ffma2_rn(f[c], m, b); if (c & 1) s[c] = fmaf(s[c], m.x, b.x); }
                if (KIND == 12) { f[c] = __ffma2_rn(f[c], m, b); if (c == 0) s[c] = rsq(s[c]); }
                // 4/11/17: one F2F.F32.F64 per step fed by a DADD and consumed by an FADD (different pipes)
                if (KIND == 17) { d[c] = __dadd_rn(d[c], d0); s[c] += __double2float_rn(d[c]); }
                if (KIND == 11) { f[c] = __ffma2_rn(f[c], m, b); if ((c & 3) == 0) { d[c] = __dadd_rn(d[c], d0); s[c] += __double2float_rn(d[c]); } }
                // 20/21: the pair body's own mix, 13 FADD2 : 6 FMUL2 : 14 FFMA2, on independent chains
                // (no MUFU, no loads): 20 = type changes at every instruction, 21 = runs of one type
                if (KIND == 20) {
                    f[c] = __ffma2_rn(f[c], m, b); f[c] = __fadd2_rn(f[c], b); f[c] = __ffma2_rn(f[c], m, b); f[c] = __fadd2_rn(f[c], m);
                    f[c] = __fmul2_rn(f[c], m); f[c] = __ffma2_rn(f[c], m, b); f[c] = __fadd2_rn(f[c], b); f[c] = __ffma2_rn(f[c], b, m);
                    if (r < 2) { f[c] = __fadd2_rn(f[c], b); f[c] = __fmul2_rn(f[c], m); }
                    else if (r < 4) { f[c] = __ffma2_rn(f[c], m, b); }
                    else if (r < 7) { f[c] = __fadd2_rn(f[c], m); }
                }
                if (KIND == 21) {
                    if (r < 3) { f[c] = __fadd2_rn(f[c], b); f[c] = __fadd2_rn(f[c], m); f[c] = __fadd2_rn(f[c], b); f[c] = __fadd2_rn(f[c], m); }
                    else if (r == 3) { f[c] = __fadd2_rn(f[c], b); f[c] = __fmul2_rn(f[c], m); f[c] = __fmul2_rn(f[c], m); f[c] = __fmul2_rn(f[c], m); }
                    else if (r == 4) { f[c] = __fmul2_rn(f[c], m); f[c] = __fmul2_rn(f[c], m); f[c] = __fmul2_rn(f[c], m); f[c] = __ffma2_rn(f[c], m, b); f[c] = __ffma2_rn(f[c], b, m); }
                    else { f[c] = __ffma2_rn(f[c], m, b); f[c] = __ffma2_rn(f[c], b, m); f[c] = __ffma2_rn(f[c], m, b); f[c] = __ffma2_rn(f[c], b, m); }
                }
                // 22..25: operands that are all live registers (no constant the reuse cache can hold)
                if (KIND == 22) f[c] = __ffma2_rn(f[(c + 1) & 7], f[(c + 2) & 7], f[c]);
                if (KIND == 23) f[c] = __fadd2_rn(f[(c + 1) & 7], f[c]);
                if (KIND == 24) f[c] = __ffma2_rn(f[(c + 1) & 7], f[(c + 1) & 7], f[c]);
                if (KIND == 25) f[c] = __ffma2_rn(f[(c + 1) & 7], m, f[c]);
                // 26: six-word FFMA2 alternating with a two-word FMUL2 (does the operand fetch average out?)
                if (KIND == 26) { f[c] = __ffma2_rn(f[(c + 1) & 7], f[(c + 2) & 7], f[c]); g[c] = __fmul2_rn(g[c], g[c]); }
                // 27: six-word FFMA2 x3 sharing the first operand (a reuse chain), then the next chain
                if (KIND == 27) {
                    const float2 a = f[(c + 3) & 7];
                    g[c] = __ffma2_rn(a, f[(c + 1) & 7], g[c]);
                    g[(c + 1) & 7] = __ffma2_rn(a, f[(c + 2) & 7], g[(c + 1) & 7]);
                    g[(c + 2) & 7] = __ffma2_rn(a, f[(c + 4) & 7], g[(c + 2) & 7]);
                }
                // 28: FFMA2 with one scalar (broadcast) operand: five words
                if (KIND == 28) f[c] = __ffma2_rn(f[(c + 1) & 7], make_float2(s[c], s[c]), f[c]);
                if (KIND == 18) { f[c] = __ffma2_rn(f[c], m, b); if ((c & 3) == 0) { d[c] = __dadd_rn(d[c], d0); s[c] += __double2float_rn(d[c]); } if (c == 7 && (r & 3) == 0) s[c] = rsq(s[c]); }
            }
        }
    }
    float acc = 0.f;
    for (int c = 0; c < NCH; ++c) acc += f[c].x + f[c].y + g[c].x + g[c].y + (float)d[c] + s[c] + (float)u[c];
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}


constexpr int TJ = 128;
struct Acc { float2 ax, ay, az, jx, jy, jz, p; };

__device__ __forceinline__ void body32(float2 dx, float2 dy, float2 dz, float2 wx, float2 wy, float2 wz,
                                       float2 m, float2 eps2, float2 m3, Acc& A)
{
    float2 r2 = __ffma2_rn(dx, dx, eps2);
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dz, dz, r2);
    float2 rinv;
    rinv.x = rsq(r2.x);
    rinv.y = rsq(r2.y);
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 mr = __fmul2_rn(m, rinv);
    const float2 mr3 = __fmul2_rn(mr, rinv2);
    float2 rv = __fmul2_rn(dx, wx);
    rv = __ffma2_rn(dy, wy, rv);
    rv = __ffma2_rn(dz, wz, rv);
    const float2 al = __fmul2_rn(__fmul2_rn(rinv2, m3), rv);
    A.p = __fadd2_rn(A.p, mr);
    A.ax = __ffma2_rn(mr3, dx, A.ax);
    A.ay = __ffma2_rn(mr3, dy, A.ay);
    A.az = __ffma2_rn(mr3, dz, A.az);
    A.jx = __ffma2_rn(mr3, __ffma2_rn(al, dx, wx), A.jx);
    A.jy = __ffma2_rn(mr3, __ffma2_rn(al, dy, wy), A.jy);
    A.jz = __ffma2_rn(mr3, __ffma2_rn(al, dz, wz), A.jz);
}
__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }

// fp64 -> fp32 (truncating) and fp32 -> fp64 through the integer pipe (normal numbers only)
__device__ __forceinline__ float d2f_bits(double d)
{
    const unsigned hi = (unsigned)__double2hiint(d), lo = (unsigned)__double2loint(d);
    const unsigned h2 = hi - 0x38000000u;
    return __uint_as_float(__funnelshift_l(lo, h2, 3));
}
__device__ __forceinline__ double f2d_bits(float f)
{
    const unsigned u = __float_as_uint(f);
    return __hiloint2double((int)((u >> 3) + 0x38000000u), (int)(u << 29));
}


// ---------------- candidate pair bodies (SURVEY.md section 7 encoding table), 2 i per thread -------------
// NDBL of the three position components are differenced in fp64 (DADD) and converted (F2F.F32.F64,
// or with CONV = 1 by integer-pipe bit operations, truncating; rate probe only: zero is not handled),
// the others as two-float sums (3 FADD2 lane-ops).  NDBL = 0 is encoding C (force_kernel today),
// NDBL = 3 is encoding D.  Same tile contents in both forms, 4 j per trip, loop only.
template <int NDBL, int CONV, int MINB>
__global__ void __launch_bounds__(128, MINB) body_kernel(float* out, int reps, float eps2f)
{
    __shared__ __align__(16) float T[10 * TJ];       // xh yh zh xl yl zl vx vy vz m
    __shared__ __align__(16) double TD[3 * TJ];      // x y z
    const int tid = threadIdx.x;
    for (int q = tid; q < TJ; q += 128) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.37 * ((q * 2654435761u + c * 40503u) % 1000) / 1000.0 - 0.18;
            TD[c * TJ + q] = x;
            const float h = (float)x;
            T[c * TJ + q] = h;
            T[(3 + c) * TJ + q] = (float)(x - (double)h);
            T[(6 + c) * TJ + q] = 0.01f * (float)((q * 7 + c * 13) % 17 - 8);
        }
        T[9 * TJ + q] = 1.0f / 1048576.0f;
    }
    __syncthreads();
    constexpr int IPT = 2;
    double xi[IPT][3];
    float2 nxh[IPT][3], nxl[IPT][3], nv[IPT][3];
    Acc A[IPT];
    for (int u = 0; u < IPT; ++u) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.001 * (tid + 128 * u) + 0.1 * c + 1e-9 * blockIdx.x;
            const float h = (float)x;
            xi[u][c] = x;
            nxh[u][c] = dup(-h);
            nxl[u][c] = dup(-(float)(x - (double)h));
            nv[u][c] = dup(0.003f * (tid % 7) - 0.01f * c + 0.002f * u);
        }
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = make_float2(0.f, 0.f);
    }
    const float2 eps2 = dup(eps2f), m3 = dup(-3.0f);
    for (int r = 0; r < reps; ++r) {
#pragma unroll 2
        for (int p = 0; p < TJ; p += 4) {
            float4 f[10];
            double2 g[3][2];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                if (c < NDBL) {
                    g[c][0] = *reinterpret_cast<const double2*>(TD + c * TJ + p);
                    g[c][1] = *reinterpret_cast<const double2*>(TD + c * TJ + p + 2);
                } else {
                    f[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
                    f[3 + c] = *reinterpret_cast<const float4*>(T + (3 + c) * TJ + p);
                }
            }
#pragma unroll
            for (int c = 6; c < 10; ++c) f[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    float2 d[3], w[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        if (c < NDBL) {
                            const double e0 = g[c][h].x - xi[u][c], e1 = g[c][h].y - xi[u][c];
                            d[c] = CONV ? make_float2(d2f_bits(e0), d2f_bits(e1))
                                        : make_float2(__double2float_rn(e0), __double2float_rn(e1));
                        } else {
                            const float2 xh = h ? make_float2(f[c].z, f[c].w) : make_float2(f[c].x, f[c].y);
                            const float2 xl = h ? make_float2(f[3 + c].z, f[3 + c].w) : make_float2(f[3 + c].x, f[3 + c].y);
                            d[c] = __fadd2_rn(__fadd2_rn(xh, nxh[u][c]), __fadd2_rn(xl, nxl[u][c]));
                        }
                        const float2 vv = h ? make_float2(f[6 + c].z, f[6 + c].w) : make_float2(f[6 + c].x, f[6 + c].y);
                        w[c] = __fadd2_rn(vv, nv[u][c]);
                    }
                    const float2 mm = h ? make_float2(f[9].z, f[9].w) : make_float2(f[9].x, f[9].y);
                    body32(d[0], d[1], d[2], w[0], w[1], w[2], mm, eps2, m3, A[u]);
                }
            }
        }
    }
    float res = 0.f;
    for (int u = 0; u < IPT; ++u)
        res += A[u].ax.x + A[u].ax.y + A[u].ay.x + A[u].ay.y + A[u].az.x + A[u].az.y + A[u].jx.x + A[u].jx.y +
               A[u].jy.x + A[u].jy.y + A[u].jz.x + A[u].jz.y + A[u].p.x + A[u].p.y;
    out[blockIdx.x * 128 + tid] = res;
}

// ---------------- the same pair (encoding C) with SCALAR FP32 instructions ----------------
// Packed f32x2 instructions halve the issue slots but run at 90 % (FFMA2) / 97 % (FADD2, FMUL2) of the
// lane rate; scalar FFMA sustains 95 %.  A scalar body needs an issue slot per lane-op, so everything
// else (MUFU, LDS, loop) competes with the FP32 pipe for issue: IPT i-particles per thread share the
// ten LDS.128 of a j-quad.  33 FFMA-class + 1 MUFU + 10/(4 IPT) LDS per interaction.
// ---------------- encoding C with the multiply-add CHAINS kept together ----------------
// Register-file bandwidth (rates 22..25): an FFMA2 whose three operands are three different live
// register pairs runs at 65 % of the packed rate, one with two different pairs at 96 %: the register
// file delivers two 32-bit words per lane and clock, an instruction with six operand words takes three
// clocks of a two-clock pipe slot unless an operand comes from the reuse cache (same register in the
// same operand slot of the previous instruction).  The pair body has eleven such FFMA2 per j-pair:
// three t = al*d + w (al shared), six sums += mr3 * (d | t) (mr3 shared), two of the r.w chain.  ptxas
// treats the sums as leaves and sprinkles them as fillers, which breaks the chains.  SEP != 0 puts the
// chains of a j-quad into a section of their own, after everything else of that quad.
__device__ __forceinline__ unsigned long long f2u(float2 v)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(v.x), "f"(v.y));
    return r;
}
__device__ __forceinline__ float2 u2f(unsigned long long r)
{
    float2 v;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(v.x), "=f"(v.y) : "l"(r));
    return v;
}

template <int SEP>
__device__ __forceinline__ void section()
{
    if (SEP == 1) __syncwarp();
    if (SEP == 2) asm volatile("bar.warp.sync 0xffffffff;" ::: "memory");
    if (SEP == 3) asm volatile("" ::: "memory");
}

template <int MINB, int SEP, int UNR>
__global__ void __launch_bounds__(128, MINB) body_chain_kernel(float* out, int reps, float eps2f, int opaque)
{
    __shared__ __align__(16) float T[10 * TJ];       // xh yh zh xl yl zl vx vy vz m
    const int tid = threadIdx.x;
    for (int q = tid; q < TJ; q += 128) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.37 * ((q * 2654435761u + c * 40503u) % 1000) / 1000.0 - 0.18;
            const float h = (float)x;
            T[c * TJ + q] = h;
            T[(3 + c) * TJ + q] = (float)(x - (double)h);
            T[(6 + c) * TJ + q] = 0.01f * (float)((q * 7 + c * 13) % 17 - 8);
        }
        T[9 * TJ + q] = 1.0f / 1048576.0f;
    }
    __syncthreads();
    constexpr int IPT = 2;
    float2 nxh[IPT][3], nxl[IPT][3], nv[IPT][3];
    Acc A[IPT];
    for (int u = 0; u < IPT; ++u) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.001 * (tid + 128 * u) + 0.1 * c + 1e-9 * blockIdx.x;
            const float h = (float)x;
            nxh[u][c] = dup(-h);
            nxl[u][c] = dup(-(float)(x - (double)h));
            nv[u][c] = dup(0.003f * (tid % 7) - 0.01f * c + 0.002f * u);
        }
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = make_float2(0.f, 0.f);
    }
    const float2 eps2 = dup(eps2f), m3 = dup(-3.0f);
    for (int r = 0; r < reps; ++r) {
#pragma unroll UNR
        for (int p = 0; p < TJ; p += 4) {
            float4 f[10];
#pragma unroll
            for (int c = 0; c < 10; ++c) f[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
            float2 d[4][3], w[4][3], mr[4], mr3[4], al[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int u = e >> 1, h = e & 1;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float2 xh = h ? make_float2(f[c].z, f[c].w) : make_float2(f[c].x, f[c].y);
                    const float2 xl = h ? make_float2(f[3 + c].z, f[3 + c].w) : make_float2(f[3 + c].x, f[3 + c].y);
                    d[e][c] = __fadd2_rn(__fadd2_rn(xh, nxh[u][c]), __fadd2_rn(xl, nxl[u][c]));
                    const float2 vv = h ? make_float2(f[6 + c].z, f[6 + c].w) : make_float2(f[6 + c].x, f[6 + c].y);
                    w[e][c] = __fadd2_rn(vv, nv[u][c]);
                }
                const float2 mm = h ? make_float2(f[9].z, f[9].w) : make_float2(f[9].x, f[9].y);
                float2 r2 = __ffma2_rn(d[e][0], d[e][0], eps2);
                r2 = __ffma2_rn(d[e][1], d[e][1], r2);
                r2 = __ffma2_rn(d[e][2], d[e][2], r2);
                float2 rinv;
                rinv.x = rsq(r2.x);
                rinv.y = rsq(r2.y);
                const float2 rinv2 = __fmul2_rn(rinv, rinv);
                mr[e] = __fmul2_rn(mm, rinv);
                mr3[e] = __fmul2_rn(mr[e], rinv2);
                float2 rv = __fmul2_rn(d[e][0], w[e][0]);
                rv = __ffma2_rn(d[e][1], w[e][1], rv);
                rv = __ffma2_rn(d[e][2], w[e][2], rv);
                al[e] = __fmul2_rn(__fmul2_rn(rinv2, m3), rv);
            }
            section<SEP>();
            if (SEP == 4 && opaque) out[0] = 0.f;
            if (SEP == 5) {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int u = e >> 1;
                    unsigned long long ax = f2u(A[u].ax), ay = f2u(A[u].ay), az = f2u(A[u].az), jx = f2u(A[u].jx),
                                       jy = f2u(A[u].jy), jz = f2u(A[u].jz), pp = f2u(A[u].p);
                    asm volatile(
                        "{\n\t.reg .b64 tx, ty, tz;\n\t"
                        "fma.rn.f32x2 tx, %7, %8, %11;\n\t"
                        "fma.rn.f32x2 ty, %7, %9, %12;\n\t"
                        "fma.rn.f32x2 tz, %7, %10, %13;\n\t"
                        "fma.rn.f32x2 %0, %14, %8, %0;\n\t"
                        "fma.rn.f32x2 %1, %14, %9, %1;\n\t"
                        "fma.rn.f32x2 %2, %14, %10, %2;\n\t"
                        "fma.rn.f32x2 %3, %14, tx, %3;\n\t"
                        "fma.rn.f32x2 %4, %14, ty, %4;\n\t"
                        "fma.rn.f32x2 %5, %14, tz, %5;\n\t"
                        "add.rn.f32x2 %6, %6, %15;\n\t}"
                        : "+l"(ax), "+l"(ay), "+l"(az), "+l"(jx), "+l"(jy), "+l"(jz), "+l"(pp)
                        : "l"(f2u(al[e])), "l"(f2u(d[e][0])), "l"(f2u(d[e][1])), "l"(f2u(d[e][2])), "l"(f2u(w[e][0])),
                          "l"(f2u(w[e][1])), "l"(f2u(w[e][2])), "l"(f2u(mr3[e])), "l"(f2u(mr[e])));
                    A[u].ax = u2f(ax); A[u].ay = u2f(ay); A[u].az = u2f(az); A[u].jx = u2f(jx);
                    A[u].jy = u2f(jy); A[u].jz = u2f(jz); A[u].p = u2f(pp);
                }
            } else
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int u = e >> 1;
                const float2 tx = __ffma2_rn(al[e], d[e][0], w[e][0]);
                const float2 ty = __ffma2_rn(al[e], d[e][1], w[e][1]);
                const float2 tz = __ffma2_rn(al[e], d[e][2], w[e][2]);
                A[u].ax = __ffma2_rn(mr3[e], d[e][0], A[u].ax);
                A[u].ay = __ffma2_rn(mr3[e], d[e][1], A[u].ay);
                A[u].az = __ffma2_rn(mr3[e], d[e][2], A[u].az);
                A[u].jx = __ffma2_rn(mr3[e], tx, A[u].jx);
                A[u].jy = __ffma2_rn(mr3[e], ty, A[u].jy);
                A[u].jz = __ffma2_rn(mr3[e], tz, A[u].jz);
                A[u].p = __fadd2_rn(A[u].p, mr[e]);
            }
            section<SEP>();
            if (SEP == 4 && opaque) out[1] = 0.f;
        }
    }
    float res = 0.f;
    for (int u = 0; u < IPT; ++u)
        res += A[u].ax.x + A[u].ax.y + A[u].ay.x + A[u].ay.y + A[u].az.x + A[u].az.y + A[u].jx.x + A[u].jx.y +
               A[u].jy.x + A[u].jy.y + A[u].jz.x + A[u].jz.y + A[u].p.x + A[u].p.y;
    out[blockIdx.x * 128 + tid] = res;
}

// ---------------- encoding C, thread-level instead of instruction-level parallelism ----------------
// One evaluation (one i against one j-pair) per loop trip and IPT i per thread: with a single
// evaluation in flight ptxas emits its instructions in dependency order, which keeps the chains
// t = al*d + w (x3, al shared) and sum += mr3*(d|t) (x6, mr3 shared) together, so that the reuse
// cache serves the shared operand; latency is hidden by the other warps (NT/32 x MINB per SM).
template <int IPT, int PAIRS, int MINB, int NT>
__global__ void __launch_bounds__(NT, MINB) body_tlp_kernel(float* out, int reps, float eps2f)
{
    __shared__ __align__(16) float T[10 * TJ];       // xh yh zh xl yl zl vx vy vz m
    const int tid = threadIdx.x;
    for (int q = tid; q < TJ; q += NT) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.37 * ((q * 2654435761u + c * 40503u) % 1000) / 1000.0 - 0.18;
            const float h = (float)x;
            T[c * TJ + q] = h;
            T[(3 + c) * TJ + q] = (float)(x - (double)h);
            T[(6 + c) * TJ + q] = 0.01f * (float)((q * 7 + c * 13) % 17 - 8);
        }
        T[9 * TJ + q] = 1.0f / 1048576.0f;
    }
    __syncthreads();
    float2 nxh[IPT][3], nxl[IPT][3], nv[IPT][3];
    Acc A[IPT];
    for (int u = 0; u < IPT; ++u) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.001 * (tid + NT * u) + 0.1 * c + 1e-9 * blockIdx.x;
            const float h = (float)x;
            nxh[u][c] = dup(-h);
            nxl[u][c] = dup(-(float)(x - (double)h));
            nv[u][c] = dup(0.003f * (tid % 7) - 0.01f * c + 0.002f * u);
        }
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = make_float2(0.f, 0.f);
    }
    const float2 eps2 = dup(eps2f), m3 = dup(-3.0f);
    for (int r = 0; r < reps; ++r) {
#pragma unroll 1
        for (int p = 0; p < TJ; p += 2 * PAIRS) {
            float2 f[PAIRS][10];
#pragma unroll
            for (int h = 0; h < PAIRS; ++h)
#pragma unroll
                for (int c = 0; c < 10; ++c) f[h][c] = *reinterpret_cast<const float2*>(T + c * TJ + p + 2 * h);
#pragma unroll
            for (int h = 0; h < PAIRS; ++h)
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    float2 d[3], w[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        d[c] = __fadd2_rn(__fadd2_rn(f[h][c], nxh[u][c]), __fadd2_rn(f[h][3 + c], nxl[u][c]));
                        w[c] = __fadd2_rn(f[h][6 + c], nv[u][c]);
                    }
                    body32(d[0], d[1], d[2], w[0], w[1], w[2], f[h][9], eps2, m3, A[u]);
                }
        }
    }
    float res = 0.f;
    for (int u = 0; u < IPT; ++u)
        res += A[u].ax.x + A[u].ax.y + A[u].ay.x + A[u].ay.y + A[u].az.x + A[u].az.y + A[u].jx.x + A[u].jx.y +
               A[u].jy.x + A[u].jy.y + A[u].jz.x + A[u].jz.y + A[u].p.x + A[u].p.y;
    out[blockIdx.x * NT + tid] = res;
}

struct Acc1 { float ax, ay, az, jx, jy, jz, p; };

__device__ __forceinline__ void body1(float dx, float dy, float dz, float wx, float wy, float wz, float m,
                                      float eps2, Acc1& A)
{
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
    const float rinv = rsq(r2);
    const float rinv2 = rinv * rinv;
    const float mr = m * rinv;
    const float mr3 = mr * rinv2;
    const float rv = fmaf(dz, wz, fmaf(dy, wy, dx * wx));
    const float al = (rinv2 * -3.0f) * rv;
    A.p += mr;
    A.ax = fmaf(mr3, dx, A.ax);
    A.ay = fmaf(mr3, dy, A.ay);
    A.az = fmaf(mr3, dz, A.az);
    A.jx = fmaf(mr3, fmaf(al, dx, wx), A.jx);
    A.jy = fmaf(mr3, fmaf(al, dy, wy), A.jy);
    A.jz = fmaf(mr3, fmaf(al, dz, wz), A.jz);
}

template <int IPT, int MINB, int UNR, int NT>
__global__ void __launch_bounds__(NT, MINB) scalar_body_kernel(float* out, int reps, float eps2)
{
    __shared__ __align__(16) float T[10 * TJ];       // xh yh zh xl yl zl vx vy vz m
    const int tid = threadIdx.x;
    for (int q = tid; q < TJ; q += NT) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.37 * ((q * 2654435761u + c * 40503u) % 1000) / 1000.0 - 0.18;
            const float h = (float)x;
            T[c * TJ + q] = h;
            T[(3 + c) * TJ + q] = (float)(x - (double)h);
            T[(6 + c) * TJ + q] = 0.01f * (float)((q * 7 + c * 13) % 17 - 8);
        }
        T[9 * TJ + q] = 1.0f / 1048576.0f;
    }
    __syncthreads();
    float nxh[IPT][3], nxl[IPT][3], nv[IPT][3];
    Acc1 A[IPT];
    for (int u = 0; u < IPT; ++u) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.001 * (tid + NT * u) + 0.1 * c + 1e-9 * blockIdx.x;
            const float h = (float)x;
            nxh[u][c] = -h;
            nxl[u][c] = -(float)(x - (double)h);
            nv[u][c] = 0.003f * (tid % 7) - 0.01f * c + 0.002f * u;
        }
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = 0.f;
    }
    for (int r = 0; r < reps; ++r) {
#pragma unroll UNR
        for (int p = 0; p < TJ; p += 4) {
            float4 f[10];
#pragma unroll
            for (int c = 0; c < 10; ++c) f[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float v[10];
#pragma unroll
                for (int c = 0; c < 10; ++c) v[c] = e == 0 ? f[c].x : (e == 1 ? f[c].y : (e == 2 ? f[c].z : f[c].w));
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    const float dx = (v[0] + nxh[u][0]) + (v[3] + nxl[u][0]);
                    const float dy = (v[1] + nxh[u][1]) + (v[4] + nxl[u][1]);
                    const float dz = (v[2] + nxh[u][2]) + (v[5] + nxl[u][2]);
                    body1(dx, dy, dz, v[6] + nv[u][0], v[7] + nv[u][1], v[8] + nv[u][2], v[9], eps2, A[u]);
                }
            }
        }
    }
    float res = 0.f;
    for (int u = 0; u < IPT; ++u) res += A[u].ax + A[u].ay + A[u].az + A[u].jx + A[u].jy + A[u].jz + A[u].p;
    out[blockIdx.x * NT + tid] = res;
}

struct Acc64 { double ax, ay, az, jx, jy, jz, p; };

// CONV: 0 = F2F conversions (XU pipe), 1 = integer-pipe bit conversions
template <int CONV>
__device__ __forceinline__ void body64(double xi, double yi, double zi, double vxi, double vyi, double vzi,
                                       double xj, double yj, double zj, double vxj, double vyj, double vzj,
                                       double m, double eps2, Acc64& A)
{
    const double dx = xj - xi, dy = yj - yi, dz = zj - zi;
    const double wx = vxj - vxi, wy = vyj - vyi, wz = vzj - vzi;
    const double r2 = fma(dz, dz, fma(dy, dy, fma(dx, dx, eps2)));
    const float r2f = CONV ? d2f_bits(r2) : __double2float_rn(r2);
    const float rf = rsq(r2f);
    const double rinv = CONV ? f2d_bits(rf) : (double)rf;
    const double rinv2 = rinv * rinv;
    const double mr = m * rinv;
    const double mr3 = mr * rinv2;
    const double rv = fma(dz, wz, fma(dy, wy, dx * wx));
    const double al = (rinv2 * -3.0) * rv;
    A.p += mr;
    A.ax = fma(mr3, dx, A.ax);
    A.ay = fma(mr3, dy, A.ay);
    A.az = fma(mr3, dz, A.az);
    A.jx = fma(mr3, fma(al, dx, wx), A.jx);
    A.jy = fma(mr3, fma(al, dy, wy), A.jy);
    A.jz = fma(mr3, fma(al, dz, wz), A.jz);
}

// NW32 warps run the fp32 two-float body (2 i per thread), NW64 warps the fp64 body (IPT64 i per
// thread); all read the same tile in shared memory, reps times.
template <int NW32, int NW64, int IPT64, int CONV, int MINB>
__global__ void __launch_bounds__((NW32 + NW64) * 32, MINB)
hetero_kernel(float* out, int reps, float eps2f, double eps2d)
{
    __shared__ __align__(16) float T[10 * TJ];       // xh yh zh xl yl zl vx vy vz m
    __shared__ __align__(16) double TD[7 * TJ];      // x y z vx vy vz m
    const int tid = threadIdx.x, nthr = (NW32 + NW64) * 32;
    for (int q = tid; q < TJ; q += nthr) {
        for (int c = 0; c < 3; ++c) {
            const double x = 0.37 * ((q * 2654435761u + c * 40503u) % 1000) / 1000.0 - 0.18;
            TD[c * TJ + q] = x;
            const float h = (float)x;
            T[c * TJ + q] = h;
            T[(3 + c) * TJ + q] = (float)(x - (double)h);
            T[(6 + c) * TJ + q] = 0.01f * (float)((q * 7 + c * 13) % 17 - 8);
            TD[(3 + c) * TJ + q] = 0.01 * ((q * 7 + c * 13) % 17 - 8);
        }
        T[9 * TJ + q] = 1.0f / 1048576.0f;
        TD[6 * TJ + q] = 1.0 / 1048576.0;
    }
    __syncthreads();
    const int warp = tid >> 5;
    float res = 0.f;
    if (warp < NW32) {
        constexpr int IPT = 2;
        float2 nxh[IPT][3], nxl[IPT][3], nv[IPT][3];
        Acc A[IPT];
        for (int u = 0; u < IPT; ++u) {
            for (int c = 0; c < 3; ++c) {
                const double x = 0.001 * (tid + 128 * u) + 0.1 * c + 1e-9 * blockIdx.x;
                const float h = (float)x;
                nxh[u][c] = dup(-h);
                nxl[u][c] = dup(-(float)(x - (double)h));
                nv[u][c] = dup(0.003f * (tid % 7) - 0.01f * c + 0.002f * u);
            }
            A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = make_float2(0.f, 0.f);
        }
        const float2 eps2 = dup(eps2f), m3 = dup(-3.0f);
        for (int r = 0; r < reps; ++r) {
#pragma unroll 2
            for (int p = 0; p < TJ; p += 4) {
                float4 f[10];
#pragma unroll
                for (int c = 0; c < 10; ++c) f[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        float2 d[3], w[3];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            const float2 xh = h ? make_float2(f[c].z, f[c].w) : make_float2(f[c].x, f[c].y);
                            const float2 xl = h ? make_float2(f[3 + c].z, f[3 + c].w) : make_float2(f[3 + c].x, f[3 + c].y);
                            const float2 vv = h ? make_float2(f[6 + c].z, f[6 + c].w) : make_float2(f[6 + c].x, f[6 + c].y);
                            d[c] = __fadd2_rn(__fadd2_rn(xh, nxh[u][c]), __fadd2_rn(xl, nxl[u][c]));
                            w[c] = __fadd2_rn(vv, nv[u][c]);
                        }
                        const float2 mm = h ? make_float2(f[9].z, f[9].w) : make_float2(f[9].x, f[9].y);
                        body32(d[0], d[1], d[2], w[0], w[1], w[2], mm, eps2, m3, A[u]);
                    }
                }
            }
        }
        for (int u = 0; u < IPT; ++u)
            res += A[u].ax.x + A[u].ax.y + A[u].ay.x + A[u].ay.y + A[u].az.x + A[u].az.y + A[u].jx.x + A[u].jx.y +
                   A[u].jy.x + A[u].jy.y + A[u].jz.x + A[u].jz.y + A[u].p.x + A[u].p.y;
    } else {
        double xi[IPT64][6];
        Acc64 A[IPT64];
        for (int u = 0; u < IPT64; ++u) {
            for (int c = 0; c < 3; ++c) {
                xi[u][c] = 0.001 * (tid + 128 * u) + 0.1 * c + 1e-9 * blockIdx.x;
                xi[u][3 + c] = 0.003 * (tid % 7) - 0.01 * c;
            }
            A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = 0.0;
        }
        for (int r = 0; r < reps; ++r) {
#pragma unroll 2
            for (int p = 0; p < TJ; p += 2) {
                double2 g[7];
#pragma unroll
                for (int c = 0; c < 7; ++c) g[c] = *reinterpret_cast<const double2*>(TD + c * TJ + p);
#pragma unroll
                for (int u = 0; u < IPT64; ++u) {
                    body64<CONV>(xi[u][0], xi[u][1], xi[u][2], xi[u][3], xi[u][4], xi[u][5], g[0].x, g[1].x,
                                 g[2].x, g[3].x, g[4].x, g[5].x, g[6].x, eps2d, A[u]);
                    body64<CONV>(xi[u][0], xi[u][1], xi[u][2], xi[u][3], xi[u][4], xi[u][5], g[0].y, g[1].y,
                                 g[2].y, g[3].y, g[4].y, g[5].y, g[6].y, eps2d, A[u]);
                }
            }
        }
        for (int u = 0; u < IPT64; ++u)
            res += (float)(A[u].ax + A[u].ay + A[u].az + A[u].jx + A[u].jy + A[u].jz + A[u].p);
    }
    out[blockIdx.x * nthr + tid] = res;
}

static float* d_out;
static int nsm;

template <typename F>
float time_ms(F launch)
{
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    launch(); launch();
    CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int r = 0; r < 3; ++r) {
        CK(cudaEventRecord(e0));
        launch();
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    CK(cudaGetLastError());
    return best;
}

template <int NW32, int NW64, int IPT64, int CONV, int MINB>
void run(int reps32_only = 0)
{
    const int reps = 300;
    const int grid = nsm * MINB * 5;
    int occ = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, hetero_kernel<NW32, NW64, IPT64, CONV, MINB>,
                                                     (NW32 + NW64) * 32, 0));
    cudaFuncAttributes fa;
    CK(cudaFuncGetAttributes(&fa, hetero_kernel<NW32, NW64, IPT64, CONV, MINB>));
    float ms = time_ms([&] { hetero_kernel<NW32, NW64, IPT64, CONV, MINB><<<grid, (NW32 + NW64) * 32>>>(d_out, reps, 1e-6f, 1e-6); });
    const double i32 = (double)grid * NW32 * 64 * (double)TJ * reps;
    const double i64 = (double)grid * NW64 * 32 * IPT64 * (double)TJ * reps;
    const double r = (i32 + i64) / (ms * 1e-3);
    printf("fp32 warps %d  fp64 warps %d (ipt %d, conv %d) minb %d regs %3d occ %d : %8.3f ms  %9.3e inter/s = %5.1f%% of 1.2408e12"
           "   (fp32 share %.2f)\n",
           NW32, NW64, IPT64, CONV, MINB, fa.numRegs, occ, ms, r, r / 1.2408e12 * 100, i32 / (i32 + i64));
}


template <int NDBL, int CONV, int MINB>
void run_body(const char* name)
{
    const int reps = 300;
    const int grid = nsm * MINB * 5;
    int occ = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, body_kernel<NDBL, CONV, MINB>, 128, 0));
    cudaFuncAttributes fa;
    CK(cudaFuncGetAttributes(&fa, body_kernel<NDBL, CONV, MINB>));
    float ms = time_ms([&] { body_kernel<NDBL, CONV, MINB><<<grid, 128>>>(d_out, reps, 1e-6f); });
    const double inter = (double)grid * 4 * 64 * (double)TJ * reps;
    const double r = inter / (ms * 1e-3);
    printf("body %-40s minb %d regs %3d occ %d : %8.3f ms  %9.3e inter/s = %5.1f%% of 1.2408e12\n", name, MINB,
           fa.numRegs, occ, ms, r, r / 1.2408e12 * 100);
}

template <int IPT, int MINB, int UNR, int NT>
void run_scalar()
{
    const int reps = 300;
    const int grid = nsm * MINB * 5;
    int occ = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, scalar_body_kernel<IPT, MINB, UNR, NT>, NT, 0));
    cudaFuncAttributes fa;
    CK(cudaFuncGetAttributes(&fa, scalar_body_kernel<IPT, MINB, UNR, NT>));
    float ms = time_ms([&] { scalar_body_kernel<IPT, MINB, UNR, NT><<<grid, NT>>>(d_out, reps, 1e-6f); });
    const double inter = (double)grid * NT * IPT * (double)TJ * reps;
    const double r = inter / (ms * 1e-3);
    printf("scalar body C: ipt %d threads %3d unroll %d minb %d regs %3d occ %d : %8.3f ms  %9.3e inter/s = %5.1f%% of 1.2408e12\n",
           IPT, NT, UNR, MINB, fa.numRegs, occ, ms, r, r / 1.2408e12 * 100);
}

template <int MINB, int SEP, int UNR>
void run_chain()
{
    const int reps = 300;
    const int grid = nsm * MINB * 5;
    int occ = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, body_chain_kernel<MINB, SEP, UNR>, 128, 0));
    cudaFuncAttributes fa;
    CK(cudaFuncGetAttributes(&fa, body_chain_kernel<MINB, SEP, UNR>));
    float ms = time_ms([&] { body_chain_kernel<MINB, SEP, UNR><<<grid, 128>>>(d_out, reps, 1e-6f, 0); });
    const double inter = (double)grid * 4 * 64 * (double)TJ * reps;
    const double r = inter / (ms * 1e-3);
    printf("chain body C: sep %d unroll %d minb %d regs %3d occ %d : %8.3f ms  %9.3e inter/s = %5.1f%% of 1.2408e12\n",
           SEP, UNR, MINB, fa.numRegs, occ, ms, r, r / 1.2408e12 * 100);
}

template <int IPT, int PAIRS, int MINB, int NT>
void run_tlp()
{
    const int reps = 300;
    const int grid = nsm * MINB * 5;
    int occ = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, body_tlp_kernel<IPT, PAIRS, MINB, NT>, NT, 0));
    cudaFuncAttributes fa;
    CK(cudaFuncGetAttributes(&fa, body_tlp_kernel<IPT, PAIRS, MINB, NT>));
    float ms = time_ms([&] { body_tlp_kernel<IPT, PAIRS, MINB, NT><<<grid, NT>>>(d_out, reps, 1e-6f); });
    const double inter = (double)grid * NT * IPT * (double)TJ * reps;
    const double r = inter / (ms * 1e-3);
    printf("tlp body C: ipt %d pairs/trip %d threads %3d minb %d regs %3d occ %2d (%2d warps/SM): %8.3f ms  %9.3e inter/s = %5.1f%% of 1.2408e12\n",
           IPT, PAIRS, NT, MINB, fa.numRegs, occ, occ * NT / 32, ms, r, r / 1.2408e12 * 100);
}

template <int KIND>
void run_rate(const char* name, double ops_per_iter_thread, int ctas_per_sm)
{
    const int iters = 4000;
    const int grid = nsm * ctas_per_sm;
    float ms = time_ms([&] { rate_kernel<KIND><<<grid, 128>>>(d_out, iters, 1.0f, 1.0); });
    // ops per thread per iter = 64 (8 x 8) of the primary kind
    const double ops = (double)grid * 128 * iters * ops_per_iter_thread;
    printf("rate %-28s ctas/SM %2d : %8.3f ms  %7.2f Gop/s/SM  (thread-ops; per-clk needs the clock)\n", name,
           ctas_per_sm, ms, ops / (ms * 1e-3) / nsm / 1e9);
}


int main(int argc, char** argv)
{
    const char* what = argc > 1 ? argv[1] : "all";
    const bool all = !strcmp(what, "all");
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    nsm = prop.multiProcessorCount;
    int clk = 0;
    CK(cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0));
    printf("device %s, %d SMs, max SM clock %d MHz\n", prop.name, nsm, clk / 1000);
    CK(cudaMalloc(&d_out, (size_t)nsm * 64 * 1024 * 4));
    if (all || !strcmp(what, "rates")) {
        printf("-- raw rates, thread-operations per second per SM (divide by the clock for lanes per clock)\n");
        run_rate<1>("FFMA", 64, 4);
        run_rate<0>("FFMA2", 64, 4);
        run_rate<2>("FADD2", 64, 4);
        run_rate<6>("FMUL2", 64, 4);
        run_rate<3>("DADD", 64, 4);
        run_rate<7>("DFMA", 64, 4);
        run_rate<5>("MUFU.RSQ", 64, 4);
        run_rate<8>("alu IADD+LOP/SHF", 64, 4);
        run_rate<9>("FFMA2 + alu(2 ops) 1:1 (count FFMA2)", 64, 4);
        run_rate<10>("FFMA2 + DADD 4:1 (count FFMA2)", 64, 4);
        run_rate<12>("FFMA2 + MUFU 8:1 (count FFMA2)", 64, 4);
        run_rate<13>("FFMA2 + FFMA 1:1 (count FFMA2)", 64, 4);
        run_rate<20>("body mix 13A:6M:14F alternating (count all)", 8 * (8 * 8 + 2 * 2 + 2 + 3), 4);
        run_rate<21>("body mix 13A:6M:14F in runs (count all)", 8 * (12 + 4 + 5 + 12), 4);
        run_rate<22>("FFMA2 d = a*b+d, a b d all live regs", 64, 4);
        run_rate<24>("FFMA2 d = a*a+d", 64, 4);
        run_rate<25>("FFMA2 d = a*const+d", 64, 4);
        run_rate<23>("FADD2 d = a+d, live regs", 64, 4);
        run_rate<26>("FFMA2 (6 words) + FMUL2 a*a (2 words) 1:1 (count both)", 128, 4);
        run_rate<27>("FFMA2 (6 words) in chains of 3 sharing operand a", 192, 4);
        run_rate<28>("FFMA2 d = a*scalar+d (5 words)", 64, 4);
        run_rate<17>("F2F.F32.F64 (+DADD feed, FADD use)", 64, 4);
        run_rate<11>("FFMA2 + (DADD,F2F) 4:1 (count FFMA2)", 64, 4);
        run_rate<18>("FFMA2:DADD:F2F:MUFU 12:3:3:1 (count FFMA2)", 64, 4);
    }
    if (all || !strcmp(what, "bodies")) {
        printf("-- pair bodies, loop only, 2 i per thread, 128 threads: NDBL components by fp64 DADD + conversion\n");
        run_body<0, 0, 4>("C: two-float x y z (force_kernel)");
        run_body<0, 0, 3>("C: two-float x y z (force_kernel)");
        run_body<3, 0, 4>("D: fp64 x y z + F2F");
        run_body<3, 0, 3>("D: fp64 x y z + F2F");
        run_body<2, 0, 4>("fp64 x y + F2F, two-float z");
        run_body<2, 0, 3>("fp64 x y + F2F, two-float z");
        run_body<1, 0, 4>("fp64 x + F2F, two-float y z");
        run_body<1, 0, 3>("fp64 x + F2F, two-float y z");
        run_body<3, 1, 4>("D': fp64 x y z + integer-pipe conversion");
        run_body<3, 1, 3>("D': fp64 x y z + integer-pipe conversion");
        run_body<2, 1, 4>("fp64 x y + int conversion, two-float z");
    }
    if (all || !strcmp(what, "scalar")) {
        printf("-- pair body C with scalar FP32 instructions, loop only\n");
        run_scalar<2, 4, 1, 128>();
        run_scalar<2, 4, 2, 128>();
        run_scalar<2, 3, 2, 128>();
        run_scalar<4, 4, 1, 128>();
        run_scalar<4, 3, 1, 128>();
        run_scalar<4, 4, 2, 128>();
        run_scalar<4, 2, 1, 256>();
        run_scalar<4, 1, 1, 512>();
        run_scalar<8, 2, 1, 128>();
        run_scalar<8, 3, 1, 128>();
        run_scalar<2, 5, 1, 128>();
        run_scalar<2, 2, 2, 256>();
        run_scalar<1, 4, 2, 256>();
    }
    if (all || !strcmp(what, "chain")) {
        printf("-- pair body C, chains of a j-quad in a section of their own (SEP: 0 none, 1 __syncwarp, 2 bar.warp.sync, 3 compiler fence, 4 opaque store)\n");
        run_chain<3, 0, 1>(); run_chain<3, 0, 2>(); run_chain<4, 0, 1>();
        run_chain<3, 1, 1>(); run_chain<3, 1, 2>(); run_chain<4, 1, 1>();
        run_chain<3, 2, 1>(); run_chain<3, 2, 2>();
        run_chain<3, 3, 1>(); run_chain<3, 3, 2>();
        run_chain<3, 4, 1>(); run_chain<3, 4, 2>(); run_chain<4, 4, 1>();
        run_chain<3, 5, 1>(); run_chain<3, 5, 2>(); run_chain<4, 5, 1>();
    }
    if (all || !strcmp(what, "tlp")) {
        printf("-- pair body C, one evaluation in flight per thread, latency hidden by warps\n");
        run_tlp<1, 1, 8, 128>(); run_tlp<1, 1, 6, 128>(); run_tlp<1, 1, 4, 128>(); run_tlp<1, 1, 4, 256>();
        run_tlp<1, 2, 8, 128>(); run_tlp<1, 2, 6, 128>(); run_tlp<1, 2, 4, 256>();
        run_tlp<2, 1, 6, 128>(); run_tlp<2, 1, 4, 128>(); run_tlp<2, 1, 3, 128>(); run_tlp<2, 1, 3, 256>();
        run_tlp<2, 2, 4, 128>(); run_tlp<2, 2, 3, 128>();
        run_tlp<4, 1, 3, 128>(); run_tlp<4, 1, 4, 128>();
        run_tlp<4, 2, 2, 128>(); run_tlp<3, 2, 3, 128>(); run_tlp<3, 2, 2, 128>(); run_tlp<3, 1, 3, 128>(); run_tlp<3, 1, 4, 128>();
    }
    if (all || !strcmp(what, "hetero")) {
        printf("-- fp32 two-float (2 i per thread) and fp64 (ipt i per thread) warps in one CTA\n");
        run<4, 0, 1, 0, 3>();
        run<0, 4, 1, 0, 3>();
        run<0, 4, 2, 0, 3>();
        run<4, 4, 1, 1, 1>();
        run<8, 4, 1, 1, 1>();
        run<12, 4, 2, 1, 1>();
    }
    return 0;
}
