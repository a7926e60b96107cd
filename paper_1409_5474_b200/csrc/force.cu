// force.cu -- a2..a5: i-gather, pair loop, j-split partials, reduction.
//
// Mapping.  A CTA of 128 threads owns ITILE = 256 active i-particles (two
// per thread, held in registers as negated, lane-duplicated f32x2 values) and one of S j-subsets
// (PAPER.md:51).  It streams its j-tiles (TJ = 128 particles, 5632 B, SoA inside the tile) from
// L2/HBM into a 4-deep shared-memory ring with 1-D bulk async copies (TMA unit, cp.async.bulk)
// completing on mbarriers; no thread spends issue slots on the copy.  Two consecutive j's form the
// two lanes of every packed FP32 instruction (fma/add/mul .f32x2), so one issue slot serves two
// pair interactions; per interaction the FP32 pipe executes 33 lane-ops (9 for the two-float
// position difference) plus one MUFU.RSQ.  fp32 partial sums run over one tile (64
// terms per lane) and are then flushed to fp64 registers.  The self pair and flagged-flagged pairs
// are masked only in the tiles that contain them (warp-uniform slow path), so the common tile pays
// nothing for R5/R7.  No tensor cores: the pair kernel with its reciprocal square root is not a
// contraction.
#include "nb_internal.h"
#include "tma.h"

namespace nb {

namespace {

struct IPart {            // one i-particle, negated and duplicated over both f32x2 lanes
    float2 nxh, nyh, nzh, nxl, nyl, nzl, nvx, nvy, nvz;
};
struct Acc32 {            // per-tile fp32 sums, lane 0 = even j, lane 1 = odd j
    float2 ax, ay, az, jx, jy, jz, p;
};

__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }

// One i against one pair of j's: 13 FADD2 + 14 FFMA2 + 6 FMUL2 + 2 MUFU (R2, R17).
// GUARD (calls with eps2 below EPS2_GUARD, eps2 == 0 among them): a pair whose s does not exceed
// eps2 -- r = 0 to fp32 precision: the self pair, or two particles at one place (R5, R6) -- gets
// rinv = 0 and so contributes nothing; the compare and select run on the ALU pipe, beside the FP32
// pipe the loop is bound by.
template <bool GUARD>
__device__ __forceinline__ void pair2(const IPart& I, Acc32& A, float2 xh, float2 yh, float2 zh,
                                      float2 xl, float2 yl, float2 zl, float2 vx, float2 vy,
                                      float2 vz, float2 m, float2 eps2, float2 m3)
{
    const float2 dx = __fadd2_rn(__fadd2_rn(xh, I.nxh), __fadd2_rn(xl, I.nxl));
    const float2 dy = __fadd2_rn(__fadd2_rn(yh, I.nyh), __fadd2_rn(yl, I.nyl));
    const float2 dz = __fadd2_rn(__fadd2_rn(zh, I.nzh), __fadd2_rn(zl, I.nzl));
    const float2 wx = __fadd2_rn(vx, I.nvx);
    const float2 wy = __fadd2_rn(vy, I.nvy);
    const float2 wz = __fadd2_rn(vz, I.nvz);
    float2 r2 = __ffma2_rn(dx, dx, eps2);
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dz, dz, r2);
    float2 rinv;
    rinv.x = rsqrt_fast(r2.x);
    rinv.y = rsqrt_fast(r2.y);
    if (GUARD) {
        rinv.x = r2.x > eps2.x ? rinv.x : 0.0f;
        rinv.y = r2.y > eps2.x ? rinv.y : 0.0f;
    }
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 mr = __fmul2_rn(m, rinv);
    const float2 mr3 = __fmul2_rn(mr, rinv2);
    float2 rv = __fmul2_rn(dx, wx);
    rv = __ffma2_rn(dy, wy, rv);
    rv = __ffma2_rn(dz, wz, rv);
    const float2 al = __fmul2_rn(__fmul2_rn(rinv2, m3), rv);      // -3 (r.w) / s
    A.p = __fadd2_rn(A.p, mr);
    A.ax = __ffma2_rn(mr3, dx, A.ax);
    A.ay = __ffma2_rn(mr3, dy, A.ay);
    A.az = __ffma2_rn(mr3, dz, A.az);
    A.jx = __ffma2_rn(mr3, __ffma2_rn(al, dx, wx), A.jx);
    A.jy = __ffma2_rn(mr3, __ffma2_rn(al, dy, wy), A.jy);
    A.jz = __ffma2_rn(mr3, __ffma2_rn(al, dz, wz), A.jz);
}

// acc + pot only (the kick of a bridge between two systems):
// 9 FADD2 + 6 FFMA2 + 3 FMUL2 + 1 FADD2 = 19 lane-ops per interaction, no velocities.
template <bool GUARD>
__device__ __forceinline__ void pair2_acc(const IPart& I, Acc32& A, float2 xh, float2 yh, float2 zh,
                                          float2 xl, float2 yl, float2 zl, float2 m, float2 eps2)
{
    const float2 dx = __fadd2_rn(__fadd2_rn(xh, I.nxh), __fadd2_rn(xl, I.nxl));
    const float2 dy = __fadd2_rn(__fadd2_rn(yh, I.nyh), __fadd2_rn(yl, I.nyl));
    const float2 dz = __fadd2_rn(__fadd2_rn(zh, I.nzh), __fadd2_rn(zl, I.nzl));
    float2 r2 = __ffma2_rn(dx, dx, eps2);
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dz, dz, r2);
    float2 rinv;
    rinv.x = rsqrt_fast(r2.x);
    rinv.y = rsqrt_fast(r2.y);
    if (GUARD) {
        rinv.x = r2.x > eps2.x ? rinv.x : 0.0f;
        rinv.y = r2.y > eps2.x ? rinv.y : 0.0f;
    }
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 mr = __fmul2_rn(m, rinv);
    const float2 mr3 = __fmul2_rn(mr, rinv2);
    A.p = __fadd2_rn(A.p, mr);
    A.ax = __ffma2_rn(mr3, dx, A.ax);
    A.ay = __ffma2_rn(mr3, dy, A.ay);
    A.az = __ffma2_rn(mr3, dz, A.az);
}

// One i against a quad of consecutive j (four floats of each tile array): two packed pairs.
template <bool JERK, bool GUARD>
__device__ __forceinline__ void quad(const IPart& I, Acc32& A, const float4* f, float2 eps2, float2 m3)
{
    if (!JERK) {
        pair2_acc<GUARD>(I, A, make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y),
                         make_float2(f[2].x, f[2].y), make_float2(f[3].x, f[3].y),
                         make_float2(f[4].x, f[4].y), make_float2(f[5].x, f[5].y),
                         make_float2(f[9].x, f[9].y), eps2);
        pair2_acc<GUARD>(I, A, make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w),
                         make_float2(f[2].z, f[2].w), make_float2(f[3].z, f[3].w),
                         make_float2(f[4].z, f[4].w), make_float2(f[5].z, f[5].w),
                         make_float2(f[9].z, f[9].w), eps2);
        return;
    }
    pair2<GUARD>(I, A, make_float2(f[0].x, f[0].y), make_float2(f[1].x, f[1].y),
                 make_float2(f[2].x, f[2].y), make_float2(f[3].x, f[3].y), make_float2(f[4].x, f[4].y),
                 make_float2(f[5].x, f[5].y), make_float2(f[6].x, f[6].y), make_float2(f[7].x, f[7].y),
                 make_float2(f[8].x, f[8].y), make_float2(f[9].x, f[9].y), eps2, m3);
    pair2<GUARD>(I, A, make_float2(f[0].z, f[0].w), make_float2(f[1].z, f[1].w),
                 make_float2(f[2].z, f[2].w), make_float2(f[3].z, f[3].w), make_float2(f[4].z, f[4].w),
                 make_float2(f[5].z, f[5].w), make_float2(f[6].z, f[6].w), make_float2(f[7].z, f[7].w),
                 make_float2(f[8].z, f[8].w), make_float2(f[9].z, f[9].w), eps2, m3);
}

template <bool JERK>
__device__ __forceinline__ void load_quad(float4* f, const float* T, int p)
{
#pragma unroll
    for (int c = 0; c < 10; ++c)
        if (JERK || c < 6 || c == 9) f[c] = *reinterpret_cast<const float4*>(T + c * TJ + p);
}

// Masked scalar pair for the rare tiles that hold the i-particle itself, a flagged partner of a
// flagged i, or when eps2 == 0 (R5, R6, R7): a skipped pair gets rinv = 0, i.e. contributes nothing.
__device__ __forceinline__ void pair1_masked(const IPart& I, Acc32& A, const float* T, int p,
                                             bool skip_self, bool iflag, float eps2)
{
    const float dx = (T[P_XH * TJ + p] + I.nxh.x) + (T[P_XL * TJ + p] + I.nxl.x);
    const float dy = (T[P_YH * TJ + p] + I.nyh.x) + (T[P_YL * TJ + p] + I.nyl.x);
    const float dz = (T[P_ZH * TJ + p] + I.nzh.x) + (T[P_ZL * TJ + p] + I.nzl.x);
    const float wx = T[P_VX * TJ + p] + I.nvx.x;
    const float wy = T[P_VY * TJ + p] + I.nvy.x;
    const float wz = T[P_VZ * TJ + p] + I.nvz.x;
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
    const bool jflag = (__float_as_uint(T[P_FLAG * TJ + p]) & 1u) != 0;
    const bool skip = skip_self || (iflag && jflag) || !(r2 > 0.0f);
    const float rinv = skip ? 0.0f : rsqrt_fast(r2);
    const float rinv2 = rinv * rinv;
    const float mr = T[P_M * TJ + p] * rinv;
    const float mr3 = mr * rinv2;
    const float rv = fmaf(dz, wz, fmaf(dy, wy, dx * wx));
    const float al = (rinv2 * -3.0f) * rv;
    A.p.x += mr;
    A.ax.x = fmaf(mr3, dx, A.ax.x);
    A.ay.x = fmaf(mr3, dy, A.ay.x);
    A.az.x = fmaf(mr3, dz, A.az.x);
    A.jx.x = fmaf(mr3, fmaf(al, dx, wx), A.jx.x);
    A.jy.x = fmaf(mr3, fmaf(al, dy, wy), A.jy.x);
    A.jz.x = fmaf(mr3, fmaf(al, dz, wz), A.jz.x);
}

// R5 in the packed path.  The packed loop runs over whole tiles, so in the one tile that holds the
// index of an i-particle it evaluates the self pair: r = w = 0 exactly, nothing for acc and jerk,
// but m_i/eps for pot -- a term that can be orders of magnitude above the real ones (|pot| ~ 1 at
// m_i/eps = 1e4), and an fp32 sum that holds it rounds them away.  So that tile's pot lane (the
// even or the odd j of the thread's share, whichever holds the self index) is summed again here
// without the self pair and replaces the polluted lane; the caller makes sure the lane held
// nothing else.  64 scalar terms, once per i-particle per call.
__device__ __forceinline__ float pot_lane(const IPart& I, const float* T, int k0, int k1, int self, float eps2)
{
    float ps = 0.0f;
#pragma unroll 1
    for (int k = k0 + (self & 1); k < k1; k += 2) {
        const float dx = (T[P_XH * TJ + k] + I.nxh.x) + (T[P_XL * TJ + k] + I.nxl.x);
        const float dy = (T[P_YH * TJ + k] + I.nyh.x) + (T[P_YL * TJ + k] + I.nyl.x);
        const float dz = (T[P_ZH * TJ + k] + I.nzh.x) + (T[P_ZL * TJ + k] + I.nzl.x);
        const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
        const float mr = T[P_M * TJ + k] * rsqrt_fast(r2);
        ps += (k == self) ? 0.0f : mr;
    }
    return ps;
}

// S = distance between the 7 sums of one i: 1 when they sit in registers, FORCE_THREADS when they
// sit in shared memory (the all-i kernel keeps them there: 28 registers fewer, 4 CTAs per SM)
template <int S, bool JERK>
__device__ __forceinline__ void flush(Acc32& A, double* d)
{
    d[0 * S] += (double)(A.ax.x + A.ax.y);
    d[1 * S] += (double)(A.ay.x + A.ay.y);
    d[2 * S] += (double)(A.az.x + A.az.y);
    if (JERK) {
        d[3 * S] += (double)(A.jx.x + A.jx.y);
        d[4 * S] += (double)(A.jy.x + A.jy.y);
        d[5 * S] += (double)(A.jz.x + A.jz.y);
    }
    d[6 * S] -= (double)(A.p.x + A.p.y);
    A.ax = A.ay = A.az = A.jx = A.jy = A.jz = A.p = make_float2(0.f, 0.f);
}

// JL = threads that share one i-particle ("split the j-particles in subsets" when few
// i are active; here inside the CTA).  The 256 i-slots of a CTA then hold ITILE / JL particles, lane
// jl of an i covers TJ / JL consecutive j of every tile, and the JL partial sums meet in a shuffle
// butterfly before the CTA's partial is written.  JL = 1 is the all-i kernel.
// ring depth: the few-i variants do little arithmetic per tile and live on bytes in flight
__host__ __device__ constexpr int stages_for(int jl) { return jl == 1 ? STAGES : 2 * STAGES; }

// MODE 0: i-particles are members of the j-set, given by index (nb_force).  MODE 1: i-particles
// given by value, "a completely different set", acc + jerk + pot; MODE 2: the same,
// acc + pot only (nb_force_ext).  No self pair and no flags in modes 1 and 2.
// GUARD: the call's eps2 is below EPS2_GUARD (zero included): pairs with r = 0 are dropped inside the
// packed pair (R5, R6), so no tile needs the self-pair treatment.
template <bool ATOMIC, int JL, int MODE, bool GUARD>
__global__ void __launch_bounds__(FORCE_THREADS, NB_MINB)
force_kernel(ForceArgs P, double* __restrict__ oacc, double* __restrict__ ojrk,
             double* __restrict__ opot)
{
    constexpr int STG = stages_for(JL);
    constexpr bool JERK = (MODE != 2);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* tiles = reinterpret_cast<float*>(smem_raw);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + STG * TILE_BYTES);
    int* rel = reinterpret_cast<int*>(smem_raw + STG * TILE_BYTES + STG * 8);
    // JL == 1: the fp64 sums live in shared memory ([u][c][thread], touched once per tile)
    constexpr bool DSM = (JL == 1);
    double* sd = reinterpret_cast<double*>(smem_raw + STG * (TILE_BYTES + 16)) + threadIdx.x;
    // index of each i (or -1), only needed in the masked path and in the tail: kept out of registers
    int* sidx = reinterpret_cast<int*>(smem_raw + STG * (TILE_BYTES + 16) +
                                       (DSM ? IPT * NOUT * FORCE_THREADS * 8 : 0)) + threadIdx.x;

    const int tid = threadIdx.x;
    const int it = blockIdx.x % P.n_itiles;       // neighbouring CTAs share the j-subset (L2 reuse)
    const int sp = blockIdx.x / P.n_itiles;
    const int t0 = (int)(((int64_t)P.ntiles * sp) / P.splits);
    const int t1 = (int)(((int64_t)P.ntiles * (sp + 1)) / P.splits);

    // a4: the j-subset of this CTA is tiles [t0, t1).  Thread 0 runs the copy ring.
    if (tid == 0) {
        for (int s = 0; s < STG; ++s) {
            mbar_init(smem_u32(&bars[s]), 1);
            rel[s] = 0;
        }
        mbar_fence_init();
        for (int s = 0; s < STG && t0 + s < t1; ++s) {
            mbar_expect_tx(smem_u32(&bars[s]), TILE_BYTES);
            bulk_g2s(smem_u32(tiles + s * TILE_FLOATS), P.pack + (int64_t)(t0 + s) * TILE_FLOATS,
                     TILE_BYTES, smem_u32(&bars[s]));
        }
    }

    // a2: i-gather from the pack (two-float position = 48 bits, fp32 velocity; R8, R17)
    IPart I[IPT];
    unsigned iflags = 0;      // bit u: i-particle u carries the unsoftened flag (R7)
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int ku = it * (ITILE / JL) + (u * FORCE_THREADS + tid) / JL;   // position inside the segment
        if (MODE != 0) {
            // by value: fp64 position split in two floats here, velocity rounded
            const bool on = P.k0 + ku < P.ni;
            const int64_t e = on ? P.k0 + ku : 0;
            float h[3], l[3], w[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double xc = P.ext_x[(int64_t)c * P.ni + e];
                h[c] = __double2float_rn(xc);
                l[c] = __double2float_rn(xc - (double)h[c]);
                w[c] = (MODE == 1) ? __double2float_rn(P.ext_v[(int64_t)c * P.ni + e]) : 0.0f;
            }
            I[u].nxh = dup(-h[0]); I[u].nyh = dup(-h[1]); I[u].nzh = dup(-h[2]);
            I[u].nxl = dup(-l[0]); I[u].nyl = dup(-l[1]); I[u].nzl = dup(-l[2]);
            I[u].nvx = dup(-w[0]); I[u].nvy = dup(-w[1]); I[u].nvz = dup(-w[2]);
            sidx[u * FORCE_THREADS] = on ? -2 : -1;      // -2: active, member of no tile
            continue;
        }
        int q = (P.k0 + ku < P.ni) ? P.i_list[P.k0 + ku] : 0;
        const bool bad = (q < 0) || (q >= P.n);
        if (bad) {
            atomicOr(P.err, 1);
            q = 0;
        }
        sidx[u * FORCE_THREADS] = (P.k0 + ku < P.ni && !bad) ? q : -1;
        const float* b = P.pack + (int64_t)(q / TJ) * TILE_FLOATS + (q % TJ);
        I[u].nxh = dup(-b[P_XH * TJ]); I[u].nyh = dup(-b[P_YH * TJ]); I[u].nzh = dup(-b[P_ZH * TJ]);
        I[u].nxl = dup(-b[P_XL * TJ]); I[u].nyl = dup(-b[P_YL * TJ]); I[u].nzl = dup(-b[P_ZL * TJ]);
        I[u].nvx = dup(-b[P_VX * TJ]); I[u].nvy = dup(-b[P_VY * TJ]); I[u].nvz = dup(-b[P_VZ * TJ]);
        if (P.any_flagged && (P.flags[q] & 1)) iflags |= 1u << u;
    }

    const float2 eps2 = dup(P.eps2);
    const float2 m3 = dup(-3.0f);
    Acc32 A[IPT];
    double D[DSM ? 1 : IPT][NOUT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        A[u].ax = A[u].ay = A[u].az = A[u].jx = A[u].jy = A[u].jz = A[u].p = make_float2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < NOUT; ++c) {
            if (DSM) sd[(u * NOUT + c) * FORCE_THREADS] = 0.0;
            else D[u][c] = 0.0;
        }
    }
    __syncthreads();   // barrier inits and the zeroed release counters visible to all warps

    // a3: pair loop over the tiles of the subset.  No CTA-wide barrier inside: a warp that is done
    // with a stage bumps the stage's release counter, and the warp that brings it to a multiple of
    // NWARPS (the last one out) refills the stage, so warps drift up to STG-1 tiles apart.
    for (int t = t0; t < t1; ++t) {
        const int st = (t - t0) % STG;
        mbar_wait(smem_u32(&bars[st]), ((t - t0) / STG) & 1);
        const float* T = tiles + st * TILE_FLOATS;

        // Flagged-flagged pairs (R7): the whole tile goes through the masked scalar pair, warp-uniform;
        // that path also excludes the self pair by index.  Every other tile is packed.
        constexpr int JPT = TJ / JL;              // j per thread per tile
        constexpr int UNROLL_Q = NB_UNROLL;       // j-quads per trip of the pair loop
        constexpr int FLUSH_EVERY = 2 * 64 / JPT > 1 ? 2 * 64 / JPT : 1;
        const int p0 = (tid % JL) * JPT;
        bool slow = false;
        if (iflags) slow = (P.tileflag[t >> 5] >> (t & 31)) & 1u;
        if (__any_sync(0xffffffffu, slow)) {
#pragma unroll 1
            for (int p = p0; p < p0 + JPT; ++p) {
#pragma unroll
                for (int u = 0; u < IPT; ++u)
                    pair1_masked(I[u], A[u], T, p, MODE == 0 && sidx[u * FORCE_THREADS] == t * TJ + p,
                                 (iflags >> u) & 1u, P.eps2);
            }
        } else {
            // R5 (see pot_lane): when this tile holds the own index of one of my i-particles, in my
            // share of the tile, that particle's fp32 sums are moved to fp64 first, so that the pot
            // lane starts empty (the all-i kernel flushes after every tile anyway)
            if (MODE == 0 && !GUARD && FLUSH_EVERY > 1) {
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    const int q = sidx[u * FORCE_THREADS] - t * TJ;
                    if (q >= p0 && q < p0 + JPT) flush<1, JERK>(A[u], D[DSM ? 0 : u]);
                }
            }
#pragma unroll UNROLL_Q
            for (int p = p0; p < p0 + JPT; p += 4) {
                float4 f[10];
                load_quad<JERK>(f, T, p);
#pragma unroll
                for (int u = 0; u < IPT; ++u) quad<JERK, GUARD>(I[u], A[u], f, eps2, m3);
            }
            if (MODE == 0 && !GUARD) {
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    const int q = sidx[u * FORCE_THREADS] - t * TJ;
                    if (q >= p0 && q < p0 + JPT) {
                        const float ps = pot_lane(I[u], T, p0, p0 + JPT, q, P.eps2);
                        if (q & 1) A[u].p.y = ps;
                        else A[u].p.x = ps;
                    }
                }
            }
        }
        // fp32 sums stay short (R17: 64 terms per lane) before they move to fp64
        if (FLUSH_EVERY == 1 || (t - t0) % FLUSH_EVERY == FLUSH_EVERY - 1 || t == t1 - 1) {
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                if (DSM) flush<FORCE_THREADS, JERK>(A[u], sd + u * NOUT * FORCE_THREADS);
                else flush<1, JERK>(A[u], D[DSM ? 0 : u]);
            }
        }

        // release the stage; the last warp out refills it with tile t + STG
        __syncwarp();
        if ((tid & 31) == 0) {
            __threadfence_block();     // this warp's reads of the stage are ordered before its release
            const int old = atomicAdd(&rel[st], 1);
            if ((old & (NWARPS - 1)) == NWARPS - 1 && t + STG < t1) {
                mbar_expect_tx(smem_u32(&bars[st]), TILE_BYTES);
                bulk_g2s(smem_u32(tiles + st * TILE_FLOATS),
                         P.pack + (int64_t)(t + STG) * TILE_FLOATS, TILE_BYTES, smem_u32(&bars[st]));
            }
        }
    }

    // a4 inside the CTA: the JL lanes of one i add their sums (fixed butterfly: deterministic)
    if (JL > 1) {
#pragma unroll
        for (int u = 0; u < IPT; ++u)
#pragma unroll
            for (int c = 0; c < NOUT; ++c)
#pragma unroll
                for (int w = 1; w < JL; w <<= 1)
                    D[DSM ? 0 : u][c] += __shfl_xor_sync(0xffffffffu, D[DSM ? 0 : u][c], w);
        if (tid % JL != 0) return;
    }

    // the CTA's place in the grid is read again here, so that it does not hold registers through
    // the pair loop (the all-i kernel then fits 128 registers unspilled: 4 CTAs per SM)
    unsigned bid;
    asm volatile("mov.u32 %0, %%ctaid.x;" : "=r"(bid));
    const int it2 = bid % P.n_itiles, sp2 = bid / P.n_itiles;

    // a4: partial sums of this j-subset (second kernel adds them), or atomics (:63)
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        double o[NOUT];
#pragma unroll
        for (int c = 0; c < NOUT; ++c) o[c] = DSM ? sd[(u * NOUT + c) * FORCE_THREADS] : D[DSM ? 0 : u][c];
        const int ku = it2 * (ITILE / JL) + (u * FORCE_THREADS + tid) / JL;
        const int q = sidx[u * FORCE_THREADS];
        if (ATOMIC) {
            if (q != -1) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    atomicAdd(oacc + (int64_t)c * P.ni + P.k0 + ku, o[c]);
                    if (JERK) atomicAdd(ojrk + (int64_t)c * P.ni + P.k0 + ku, o[3 + c]);
                }
                atomicAdd(opot + P.k0 + ku, o[6]);
            }
        } else {
#pragma unroll
            for (int c = 0; c < NOUT; ++c)
                P.part[((int64_t)c * P.ni_pad + ku) * P.splits + sp2] = o[c];   // [c][i][subset]
        }
    }
}

// a4/a5: sum the S partials in a fixed order (deterministic), add the unsoftened flagged-flagged
// pair terms in fp64 straight from the j-store (R7), NaN for rejected indices, store SoA.
// WARP = one warp per i (lanes stride over the partials, fixed butterfly) for the few-i calls whose
// many j-subsets would otherwise be summed by one thread; else one thread per i.
template <bool WARP>
__global__ void __launch_bounds__(128) reduce_kernel(ReduceArgs R)
{
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int k = WARP ? gt / 32 : gt;
    const int lane = threadIdx.x & 31;
    if (k >= R.ni) return;
    double o[NOUT];
    if (R.atomic_mode) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            o[c] = R.acc[(int64_t)c * R.ni + k];
            o[3 + c] = R.jrk[(int64_t)c * R.ni + k];
        }
        o[6] = R.pot[k];
    } else {
#pragma unroll
        for (int c = 0; c < NOUT; ++c) o[c] = 0.0;
        const bool in_b = k >= R.kA;
        const double* part = in_b ? R.part_b : R.part;
        const int64_t stride = in_b ? R.ni_pad_b : R.ni_pad;
        const int kl = in_b ? k - R.kA : k, ns = in_b ? R.splits_b : R.splits;
        for (int s = WARP ? lane : 0; s < ns; s += WARP ? 32 : 1) {
#pragma unroll
            for (int c = 0; c < NOUT; ++c) o[c] += part[((int64_t)c * stride + kl) * ns + s];
        }
        if (WARP) {
#pragma unroll
            for (int c = 0; c < NOUT; ++c)
#pragma unroll
                for (int w = 16; w >= 1; w >>= 1) o[c] += __shfl_xor_sync(0xffffffffu, o[c], w);
        }
    }
    if (WARP && lane != 0) return;
    const int i = R.i_list ? R.i_list[k] : 0;     // by-value calls (nb_force_ext) carry no index list
    if (R.i_list && (i < 0 || i >= R.n)) {
#pragma unroll
        for (int c = 0; c < NOUT; ++c) o[c] = __longlong_as_double(0x7ff8000000000000LL);
    } else if (R.i_list && R.nflag > 1 && (R.flags[i] & 1)) {
        double xi[3], vi[3];
        const double dti = R.t_pred - R.store.f[F_T][i];
#pragma unroll
        for (int c = 0; c < 3; ++c)
            predict1(R.store.f[F_X + c][i], R.store.f[F_VX + c][i], R.store.f[F_AX + c][i],
                     R.store.f[F_JX + c][i], dti, xi[c], vi[c]);
        for (int q = 0; q < R.nflag; ++q) {
            const int j = R.flag_list[q];
            if (j == i) continue;
            double r[3], w[3];
            const double dtj = R.t_pred - R.store.f[F_T][j];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double xj, vj;
                predict1(R.store.f[F_X + c][j], R.store.f[F_VX + c][j], R.store.f[F_AX + c][j],
                         R.store.f[F_JX + c][j], dtj, xj, vj);
                r[c] = xj - xi[c];
                w[c] = vj - vi[c];
            }
            const double s2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
            if (s2 == 0.0) continue;
            const double rinv = 1.0 / sqrt(s2), rinv2 = rinv * rinv;
            const double mr = R.store.f[F_M][j] * rinv, mr3 = mr * rinv2;
            const double b = 3.0 * (r[0] * w[0] + r[1] * w[1] + r[2] * w[2]) * rinv2;
            o[6] -= mr;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                o[c] += mr3 * r[c];
                o[3 + c] += mr3 * (w[c] - b * r[c]);
            }
        }
    } else if (R.atomic_mode) {
        return;   // sums are already in place
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        R.acc[(int64_t)c * R.ni + k] = o[c];
        if (R.jrk) R.jrk[(int64_t)c * R.ni + k] = o[3 + c];
    }
    R.pot[k] = o[6];
}

__global__ void __launch_bounds__(256) zero_out_kernel(double* acc, double* jrk, double* pot, int64_t ni)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= ni) return;
    for (int c = 0; c < 3; ++c) {
        acc[c * ni + k] = 0.0;
        jrk[c * ni + k] = 0.0;
    }
    pot[k] = 0.0;
}

constexpr int NWARPS_CHECK = FORCE_THREADS / 32;
static_assert((NWARPS_CHECK & (NWARPS_CHECK - 1)) == 0, "warps per CTA must be a power of two");
__host__ __device__ constexpr int force_smem(int jl)
{
    return stages_for(jl) * (TILE_BYTES + 16) + (jl == 1 ? IPT * NOUT * FORCE_THREADS * 8 : 0) +
           IPT * FORCE_THREADS * 4;
}

}  // namespace

template <int JL>
cudaError_t setup_one(int* blocks, int* blocks_guard)
{
    const void* k[8] = {(const void*)force_kernel<false, JL, 0, false>, (const void*)force_kernel<true, JL, 0, false>,
                        (const void*)force_kernel<false, JL, 1, false>, (const void*)force_kernel<false, JL, 2, false>,
                        (const void*)force_kernel<false, JL, 0, true>,  (const void*)force_kernel<true, JL, 0, true>,
                        (const void*)force_kernel<false, JL, 1, true>,  (const void*)force_kernel<false, JL, 2, true>};
    int least = 0;
    for (int q = 0; q < 8; ++q) {
        cudaError_t e = cudaFuncSetAttribute(k[q], cudaFuncAttributeMaxDynamicSharedMemorySize, force_smem(JL));
        if (e != cudaSuccess) return e;
        int b = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k[q], FORCE_THREADS, force_smem(JL));
        if (e != cudaSuccess) return e;
        if (q == 0 || b < least) least = b;
    }
    // the dispatcher sizes whole waves with the by-index kernels' residency; the others only need >= 1
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks, k[0], FORCE_THREADS, force_smem(JL));
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_guard, k[4], FORCE_THREADS, force_smem(JL));
    return (e == cudaSuccess && least < 1) ? cudaErrorLaunchOutOfResources : e;
}

cudaError_t force_kernel_setup(int* blocks_per_sm, int* blocks_per_sm_guard)
{
    int b = 0, g = 0;
    cudaError_t e = setup_one<JL_MID>(&b, &g);
    if (e != cudaSuccess) return e;
    e = setup_one<JL_MAX>(&b, &g);
    if (e != cudaSuccess) return e;
    return setup_one<1>(blocks_per_sm, blocks_per_sm_guard);
}

// mode: 0 = by index (nb_force), 1 = by value with jerk, 2 = by value, acc + pot only (nb_force_ext;
// no atomics variant there)
template <int JL, bool GUARD>
void launch_one(const ForceArgs& a, int mode, int atomic_mode, double* acc, double* jrk, double* pot,
                cudaStream_t s)
{
    const unsigned grid = (unsigned)a.n_itiles * (unsigned)a.splits;
    if (mode == 1)
        force_kernel<false, JL, 1, GUARD><<<grid, FORCE_THREADS, force_smem(JL), s>>>(a, acc, jrk, pot);
    else if (mode == 2)
        force_kernel<false, JL, 2, GUARD><<<grid, FORCE_THREADS, force_smem(JL), s>>>(a, acc, jrk, pot);
    else if (atomic_mode)
        force_kernel<true, JL, 0, GUARD><<<grid, FORCE_THREADS, force_smem(JL), s>>>(a, acc, jrk, pot);
    else
        force_kernel<false, JL, 0, GUARD><<<grid, FORCE_THREADS, force_smem(JL), s>>>(a, acc, jrk, pot);
}

cudaError_t launch_force(const ForceArgs& a, int jl, int mode, int atomic_mode, double* acc, double* jrk,
                         double* pot, cudaStream_t s)
{
    const bool guard = a.eps2 < EPS2_GUARD;
    if (jl == JL_MAX) {
        if (guard) launch_one<JL_MAX, true>(a, mode, atomic_mode, acc, jrk, pot, s);
        else launch_one<JL_MAX, false>(a, mode, atomic_mode, acc, jrk, pot, s);
    } else if (jl == JL_MID) {
        if (guard) launch_one<JL_MID, true>(a, mode, atomic_mode, acc, jrk, pot, s);
        else launch_one<JL_MID, false>(a, mode, atomic_mode, acc, jrk, pot, s);
    } else {
        if (guard) launch_one<1, true>(a, mode, atomic_mode, acc, jrk, pot, s);
        else launch_one<1, false>(a, mode, atomic_mode, acc, jrk, pot, s);
    }
    return cudaGetLastError();
}
cudaError_t launch_reduce(const ReduceArgs& a, cudaStream_t s)
{
    const int most = a.splits > a.splits_b ? a.splits : a.splits_b;
    if (!a.atomic_mode && most > 8 && a.ni <= 4096)
        reduce_kernel<true><<<(a.ni + 3) / 4, 128, 0, s>>>(a);
    else
        reduce_kernel<false><<<(a.ni + 127) / 128, 128, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_zero_out(double* acc, double* jrk, double* pot, int64_t ni, cudaStream_t s)
{
    zero_out_kernel<<<(unsigned)((ni + 255) / 256), 256, 0, s>>>(acc, jrk, pot, ni);
    return cudaGetLastError();
}

}  // namespace nb
