// rpy_pair.cuh -- the O(N^2) Rotne-Prager-Yamakawa pair kernel for sm_100a (B200).
//
// Computes, for every target i of its i-tile and every source j of its j-range (self term
// included), the sums of DESIGN.md sec. 3 (grand mobility eq. (7),
// PAPER.md:66-69; RPY pair tensors PAPER.md:173):
//
//   U_i = sum_j [ f_tt F_j + g_tt (rhat.F_j) rhat + g_c (T_j x rhat) ]
//   W_i = sum_j [ f_rr T_j + g_rr (rhat.T_j) rhat + g_c (F_j x rhat) ]
//
// Design (B200-first):
//   * one thread owns TPT targets; all 32 lanes of a warp walk the SAME sources, so every
//     shared-memory read is a broadcast LDS.128 (4 fp32 / 2 fp64 sources per instruction);
//   * sources are staged as structure-of-arrays tiles by 1-D TMA bulk copies
//     (cp.async.bulk.shared::cluster.global, SASS UBLKCP) completing on an mbarrier,
//     double/triple buffered -- no thread issues a global load in the main loop;
//   * fp32 arithmetic is packed two sources per instruction (FFMA2 / FMUL2 / FADD2, the
//     sm_100 f32x2 forms): the FMA pipe sees the same lane-ops, but the issue port is freed
//     for the MUFU, select and LDS instructions of the same pair;
//   * 1/r from MUFU.RSQ (fp32) or MUFU.RSQ64H + one cubically convergent correction (fp64);
//   * both branches are evaluated and selected per lane (FSEL) -- no divergence; r = 0 is
//     made safe by a tiny additive floor inside the r^2 FMA chain (no extra instruction);
//   * two-level accumulation: a packed per-tile accumulator is flushed into a per-thread
//     main accumulator at every tile end (keeps fp32 summation error ~ eps*sqrt(tile)).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "lm_common.cuh"

namespace lm {

// ---------------------------------------------------------------- packed two-lane arithmetic
template <typename T> struct P2;
template <> struct P2<float> { float2 v; };
template <> struct P2<double> { double x, y; };

__device__ __forceinline__ P2<float> splat(float s) { return {make_float2(s, s)}; }
__device__ __forceinline__ P2<double> splat(double s) { return {s, s}; }
__device__ __forceinline__ P2<float> mk2(float a, float b) { return {make_float2(a, b)}; }
__device__ __forceinline__ P2<double> mk2(double a, double b) { return {a, b}; }
__device__ __forceinline__ float lo(const P2<float>& a) { return a.v.x; }
__device__ __forceinline__ float hi(const P2<float>& a) { return a.v.y; }
__device__ __forceinline__ double lo(const P2<double>& a) { return a.x; }
__device__ __forceinline__ double hi(const P2<double>& a) { return a.y; }

__device__ __forceinline__ P2<float> fma2(P2<float> a, P2<float> b, P2<float> c) { return {__ffma2_rn(a.v, b.v, c.v)}; }
__device__ __forceinline__ P2<float> mul2(P2<float> a, P2<float> b) { return {__fmul2_rn(a.v, b.v)}; }
__device__ __forceinline__ P2<float> add2(P2<float> a, P2<float> b) { return {__fadd2_rn(a.v, b.v)}; }
__device__ __forceinline__ P2<double> fma2(P2<double> a, P2<double> b, P2<double> c) { return {fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)}; }
__device__ __forceinline__ P2<double> mul2(P2<double> a, P2<double> b) { return {a.x * b.x, a.y * b.y}; }
__device__ __forceinline__ P2<double> add2(P2<double> a, P2<double> b) { return {a.x + b.x, a.y + b.y}; }
template <typename T> __device__ __forceinline__ P2<T> neg2(P2<T> a) { return mk2(-lo(a), -hi(a)); }

// 1/sqrt(x): fp32 = one MUFU.RSQ per lane (rel. error ~2^-22, far inside the 2e-5 gate).
__device__ __forceinline__ float rsqrt1(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// fp64 = MUFU.RSQ64H seed (rel. error e0 ~ 2^-22) + ONE third-order (Halley-type) correction
//   e = 1 - x y0^2 ;  y1 = y0 (1 + e/2 + 3 e^2/8)   ->  rel. error ~ (5/16) e0^3 ~ 2^-68,
// i.e. below fp64 rounding: 5 DFMA-pipe operations instead of 8 for two Newton steps.
__device__ __forceinline__ double rsqrt1(double x)
{
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    double t = x * y0;
    double e = fma(-t, y0, 1.0);
    double p = fma(0.375, e, 0.5);
    double q = e * p;
    return fma(y0, q, y0);
}
template <typename T> __device__ __forceinline__ P2<T> rsqrt2(P2<T> a) { return mk2(rsqrt1(lo(a)), rsqrt1(hi(a))); }
template <typename T> __device__ __forceinline__ P2<T> sel2(bool pl, bool ph, P2<T> a, P2<T> b)
{
    return mk2(pl ? lo(a) : lo(b), ph ? hi(a) : hi(b));
}

// ---------------------------------------------------------------- constants of the pair tensors
// All derived on the host in fp64 from (eta, a) and rounded once to T.
// d := x_j - x_i = -r_vec is used un-normalised; every 1/r^n needed is folded into the scalars:
//   far  (r >= 2a): f_tt = invr (C1 + C2 u)          g_tt/r^2 = invr u (C1 - C3 u)       u = invr^2
//                   f_rr = -C7 invr^3                g_rr/r^2 = 3 C7 invr^5              h = g_c/r = C1 invr^3
//   near (r <  2a): f_tt = C4 - C5 r                 g_tt/r^2 = C6 invr
//                   f_rr = C8 + r (K1 + K2 r^2)      g_rr/r^2 = K3 invr + K4 r           h = K5 + K6 r
template <typename T> struct PairConsts {
    T tiny;    // additive floor of r^2: a^2 * 2^-80  (r = 0 -> finite 1/r, selected near branch)
    T four_a2; // (2a)^2
    T C1, C2, nC3, C4, nC5, C6;           // translation-translation
    T nC7, C7x3, C8, K1, K2, K3, K4, K5, K6; // rotation-rotation and coupling
};

template <typename T> struct PairParams {
    const T* __restrict__ pos;  // [3][npad]  x | y | z, ghosts (index >= N) are zeros
    const T* __restrict__ vec;  // [nrhs*NC][npad] packed right-hand sides, ghosts are zeros
    RhsOut<T> out;              // j_splits == 1: per right-hand side, 3N interleaved each
    T* __restrict__ partial;    // j_splits  > 1: [j_splits][nrhs*NC][npad]
    int64_t N;
    int64_t npad;               // multiple of TJ and of BLOCK*TPT
    int tiles_per_split;        // j-tiles handled by one CTA (last split may get fewer)
    int n_tiles;                // npad / TJ
    PairConsts<T> c;
};

// ---------------------------------------------------------------- TMA / mbarrier helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "LM_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra LM_DONE_%=;\n\t"
        "bra LM_WAIT_%=;\n\t"
        "LM_DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared, completion counted in bytes on `bar` (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------- one packed pair (2 sources) vs one target
template <typename T, int NRHS, bool ANG>
__device__ __forceinline__ void pair_eval(const PairConsts<T>& c, T nxi, T nyi, T nzi, P2<T> xj, P2<T> yj, P2<T> zj,
                                          const P2<T> (&V)[NRHS * (ANG ? 6 : 3)], P2<T> (&acc)[NRHS * (ANG ? 6 : 3)])
{
    constexpr int NC = ANG ? 6 : 3;
    const P2<T> dx = add2(xj, splat(nxi)), dy = add2(yj, splat(nyi)), dz = add2(zj, splat(nzi));
    const P2<T> r2 = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, splat(c.tiny))));
    const P2<T> invr = rsqrt2(r2);
    const P2<T> u = mul2(invr, invr);
    const P2<T> w3 = mul2(invr, u);
    const P2<T> r = mul2(r2, invr);
    const bool nl = lo(r2) < c.four_a2, nh = hi(r2) < c.four_a2;
    // translation-translation scalars
    const P2<T> f_far = mul2(invr, fma2(splat(c.C2), u, splat(c.C1)));
    const P2<T> g_far = mul2(w3, fma2(splat(c.nC3), u, splat(c.C1)));
    const P2<T> f_near = fma2(splat(c.nC5), r, splat(c.C4));
    const P2<T> g_near = mul2(splat(c.C6), invr);
    const P2<T> f = sel2(nl, nh, f_near, f_far);
    const P2<T> g = sel2(nl, nh, g_near, g_far);
    if constexpr (!ANG) {
#pragma unroll
        for (int q = 0; q < NRHS; ++q) {
            const P2<T> Fx = V[q * NC + 0], Fy = V[q * NC + 1], Fz = V[q * NC + 2];
            const P2<T> t = mul2(g, fma2(dz, Fz, fma2(dy, Fy, mul2(dx, Fx))));
            acc[q * NC + 0] = fma2(f, Fx, fma2(t, dx, acc[q * NC + 0]));
            acc[q * NC + 1] = fma2(f, Fy, fma2(t, dy, acc[q * NC + 1]));
            acc[q * NC + 2] = fma2(f, Fz, fma2(t, dz, acc[q * NC + 2]));
        }
    } else {
        // rotation-rotation and coupling scalars
        const P2<T> w5 = mul2(w3, u);
        const P2<T> frr_far = mul2(splat(c.nC7), w3);
        const P2<T> grr_far = mul2(splat(c.C7x3), w5);
        const P2<T> h_far = mul2(splat(c.C1), w3);
        const P2<T> frr_near = fma2(r, fma2(splat(c.K2), r2, splat(c.K1)), splat(c.C8));
        const P2<T> grr_near = fma2(splat(c.K3), invr, mul2(splat(c.K4), r));
        const P2<T> h_near = fma2(splat(c.K6), r, splat(c.K5));
        const P2<T> frr = sel2(nl, nh, frr_near, frr_far);
        const P2<T> grr = sel2(nl, nh, grr_near, grr_far);
        const P2<T> h = sel2(nl, nh, h_near, h_far);
        // with d = -r_vec:  g_c (T x rhat) = h (d x T),  g_c (F x rhat) = h (d x F)
        const P2<T> hx = mul2(h, dx), hy = mul2(h, dy), hz = mul2(h, dz);
        const P2<T> nhx = neg2(hx), nhy = neg2(hy), nhz = neg2(hz);
#pragma unroll
        for (int q = 0; q < NRHS; ++q) {
            const P2<T> Fx = V[q * NC + 0], Fy = V[q * NC + 1], Fz = V[q * NC + 2];
            const P2<T> Tx = V[q * NC + 3], Ty = V[q * NC + 4], Tz = V[q * NC + 5];
            const P2<T> t = mul2(g, fma2(dz, Fz, fma2(dy, Fy, mul2(dx, Fx))));
            const P2<T> s = mul2(grr, fma2(dz, Tz, fma2(dy, Ty, mul2(dx, Tx))));
            // U += f F + t d + (hd) x T
            acc[q * NC + 0] = fma2(nhz, Ty, fma2(hy, Tz, fma2(f, Fx, fma2(t, dx, acc[q * NC + 0]))));
            acc[q * NC + 1] = fma2(nhx, Tz, fma2(hz, Tx, fma2(f, Fy, fma2(t, dy, acc[q * NC + 1]))));
            acc[q * NC + 2] = fma2(nhy, Tx, fma2(hx, Ty, fma2(f, Fz, fma2(t, dz, acc[q * NC + 2]))));
            // W += f_rr T + s d + (hd) x F
            acc[q * NC + 3] = fma2(nhz, Fy, fma2(hy, Fz, fma2(frr, Tx, fma2(s, dx, acc[q * NC + 3]))));
            acc[q * NC + 4] = fma2(nhx, Fz, fma2(hz, Fx, fma2(frr, Ty, fma2(s, dy, acc[q * NC + 4]))));
            acc[q * NC + 5] = fma2(nhy, Fx, fma2(hx, Fy, fma2(frr, Tz, fma2(s, dz, acc[q * NC + 5]))));
        }
    }
}

// ---------------------------------------------------------------- kernel
template <typename T> struct Vec16;                   // 16-byte shared-memory load = 2 packed pairs (fp32) or 1 (fp64)
template <> struct Vec16<float> { static constexpr int N = 4; };
template <> struct Vec16<double> { static constexpr int N = 2; };

template <typename T, int NRHS, bool ANG, int TPT, int BLOCK, int TJ, int STAGES>
struct PairKernelTraits {
    static constexpr int NC = ANG ? 6 : 3;             // components per source per right-hand side
    static constexpr int NV = NRHS * NC;               // packed vector arrays
    static constexpr int ARRAYS = 3 + NV;              // x, y, z + vector components
    static constexpr int STAGE_BYTES = ARRAYS * TJ * (int)sizeof(T);
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + STAGES * 8;
    static constexpr int TARGETS = BLOCK * TPT;        // targets per CTA
};

template <typename T, int NRHS, bool ANG, int TPT, int BLOCK, int TJ, int STAGES, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) rpy_pair_kernel(const PairParams<T> p)
{
    using Tr = PairKernelTraits<T, NRHS, ANG, TPT, BLOCK, TJ, STAGES>;
    constexpr int NC = Tr::NC, NV = Tr::NV, ARRAYS = Tr::ARRAYS;
    constexpr int VN = Vec16<T>::N;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* tiles = reinterpret_cast<T*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + STAGES * Tr::STAGE_BYTES);

    const int tid = threadIdx.x;
    const int64_t i0 = (int64_t)blockIdx.x * Tr::TARGETS;
    const int jt_begin = blockIdx.y * p.tiles_per_split;
    const int jt_end = min(jt_begin + p.tiles_per_split, p.n_tiles);
    const int my_tiles = jt_end - jt_begin;

    auto issue = [&](int local_tile) {               // called by thread 0 only
        const int stage = local_tile % STAGES;
        const int64_t j0 = (int64_t)(jt_begin + local_tile) * TJ;
        T* dst = tiles + (size_t)stage * ARRAYS * TJ;
        mbar_expect_tx(&full[stage], (uint32_t)Tr::STAGE_BYTES);
#pragma unroll
        for (int a = 0; a < 3; ++a) bulk_g2s(dst + a * TJ, p.pos + a * p.npad + j0, TJ * sizeof(T), &full[stage]);
#pragma unroll
        for (int a = 0; a < NV; ++a) bulk_g2s(dst + (3 + a) * TJ, p.vec + a * p.npad + j0, TJ * sizeof(T), &full[stage]);
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int s = 0; s < STAGES && s < my_tiles; ++s) issue(s);
    }

    // targets: negated coordinates so that d = x_j + (-x_i) is one packed add
    T nxi[TPT], nyi[TPT], nzi[TPT];
#pragma unroll
    for (int t = 0; t < TPT; ++t) {
        const int64_t i = i0 + t * BLOCK + tid;      // < npad: ghost targets read zeros
        nxi[t] = -p.pos[i];
        nyi[t] = -p.pos[p.npad + i];
        nzi[t] = -p.pos[2 * p.npad + i];
    }
    T total[TPT][NV];
#pragma unroll
    for (int t = 0; t < TPT; ++t)
#pragma unroll
        for (int k = 0; k < NV; ++k) total[t][k] = T(0);

    for (int lt = 0; lt < my_tiles; ++lt) {
        const int stage = lt % STAGES;
        mbar_wait(&full[stage], (uint32_t)((lt / STAGES) & 1));
        const T* sx = tiles + (size_t)stage * ARRAYS * TJ;
        P2<T> acc[TPT][NV];
#pragma unroll
        for (int t = 0; t < TPT; ++t)
#pragma unroll
            for (int k = 0; k < NV; ++k) acc[t][k] = splat(T(0));

#pragma unroll 1
        for (int j = 0; j < TJ; j += VN) {
            if constexpr (VN == 4) {
                const float4 X = *reinterpret_cast<const float4*>(sx + j);
                const float4 Y = *reinterpret_cast<const float4*>(sx + TJ + j);
                const float4 Z = *reinterpret_cast<const float4*>(sx + 2 * TJ + j);
                P2<T> Va[NV], Vb[NV];
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    const float4 v = *reinterpret_cast<const float4*>(sx + (3 + k) * TJ + j);
                    Va[k] = mk2(v.x, v.y);
                    Vb[k] = mk2(v.z, v.w);
                }
#pragma unroll
                for (int t = 0; t < TPT; ++t) {
                    pair_eval<T, NRHS, ANG>(p.c, nxi[t], nyi[t], nzi[t], mk2(X.x, X.y), mk2(Y.x, Y.y), mk2(Z.x, Z.y), Va, acc[t]);
                    pair_eval<T, NRHS, ANG>(p.c, nxi[t], nyi[t], nzi[t], mk2(X.z, X.w), mk2(Y.z, Y.w), mk2(Z.z, Z.w), Vb, acc[t]);
                }
            } else {
                const double2 X = *reinterpret_cast<const double2*>(sx + j);
                const double2 Y = *reinterpret_cast<const double2*>(sx + TJ + j);
                const double2 Z = *reinterpret_cast<const double2*>(sx + 2 * TJ + j);
                P2<T> Va[NV];
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    const double2 v = *reinterpret_cast<const double2*>(sx + (3 + k) * TJ + j);
                    Va[k] = mk2(v.x, v.y);
                }
#pragma unroll
                for (int t = 0; t < TPT; ++t)
                    pair_eval<T, NRHS, ANG>(p.c, nxi[t], nyi[t], nzi[t], mk2(X.x, X.y), mk2(Y.x, Y.y), mk2(Z.x, Z.y), Va, acc[t]);
            }
        }
        // flush the per-tile packed accumulators (two-level summation)
#pragma unroll
        for (int t = 0; t < TPT; ++t)
#pragma unroll
            for (int k = 0; k < NV; ++k) total[t][k] += lo(acc[t][k]) + hi(acc[t][k]);

        __syncthreads();                               // every warp is done reading this stage
        if (tid == 0 && lt + STAGES < my_tiles) issue(lt + STAGES);
    }

    // ---- epilogue
    if (gridDim.y == 1) {
#pragma unroll
        for (int t = 0; t < TPT; ++t) {
            const int64_t i = i0 + t * BLOCK + tid;
            if (i < p.N) {
#pragma unroll
                for (int q = 0; q < NRHS; ++q) {
                    T* ul = p.out.lin[q] + 3 * i;
                    ul[0] = total[t][q * NC + 0];
                    ul[1] = total[t][q * NC + 1];
                    ul[2] = total[t][q * NC + 2];
                    if constexpr (ANG) {
                        T* ua = p.out.ang[q] + 3 * i;
                        ua[0] = total[t][q * NC + 3];
                        ua[1] = total[t][q * NC + 4];
                        ua[2] = total[t][q * NC + 5];
                    }
                }
            }
        }
    } else {
        T* part = p.partial + (size_t)blockIdx.y * NV * p.npad;
#pragma unroll
        for (int t = 0; t < TPT; ++t) {
            const int64_t i = i0 + t * BLOCK + tid;
#pragma unroll
            for (int k = 0; k < NV; ++k) part[(size_t)k * p.npad + i] = total[t][k];
        }
    }
}

}  // namespace lm
