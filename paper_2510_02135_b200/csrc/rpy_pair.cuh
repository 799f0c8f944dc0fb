// rpy_pair.cuh -- the O(N^2) Rotne-Prager-Yamakawa pair kernel for sm_100a (B200).
//
// Computes, for every target i of its i-tile and every source j of its j-range (self term
// included), the sums of DESIGN.md sec. 3 (grand mobility eq. (7),
// PAPER.md:66-69; RPY pair tensors PAPER.md:173):
//
//   U_i = sum_j [ f_tt F_j + g_tt (rhat.F_j) rhat + g_c (T_j x rhat) ]
//   W_i = sum_j [ f_rr T_j + g_rr (rhat.T_j) rhat + g_c (F_j x rhat) ]
//
// Design (B200-first, DESIGN.md sec. 5 and the machine model of sec. 7):
//   * one thread owns TPT targets held as TPT/2 PACKED TARGET PAIRS; all 32 lanes of a warp walk
//     the SAME sources, so every shared-memory read is a broadcast LDS.128 (4 fp32 / 2 fp64
//     sources per instruction) and every source value enters the arithmetic as a scalar-broadcast
//     operand (FFMA2 Rpair, R.F32, Rpair): at most two 64-bit register operands per packed
//     instruction, which is what the sm_100 register file can feed at the FMA pipe's rate;
//   * sources are staged as structure-of-arrays tiles by 1-D TMA bulk copies
//     (cp.async.bulk.shared::cluster.global, SASS UBLKCP) completing on an mbarrier,
//     double buffered -- no thread issues a global load in the main loop; a stage is released
//     without a CTA barrier: every warp arrives on the stage's `empty` mbarrier, the last one out issues the refill;
//   * fp32 arithmetic is packed two targets per instruction (FFMA2 / FMUL2 / FADD2, the
//     sm_100 f32x2 forms);  1/r from MUFU.RSQ (fp32) or MUFU.RSQ64H + one cubically convergent
//     correction (fp64);
//   * overlap (r < 2a) / far-field select without divergence, nothing evaluated twice, and the
//     near formulas paid for only where pairs overlap: sources are walked in groups of GS (2 or 4);
//     the geometry (d, r^2) of the whole group x all the thread's packed pairs comes first while a
//     running minimum collects min r^2; ONE warp vote per group then picks the FAR-FIELD body (no
//     near formulas, no selects) or the GENERAL body (both branches + per-lane FSEL) BEFORE
//     anything is accumulated;
//   * r = 0 is made safe by a tiny additive floor inside the r^2 FMA chain (no extra instruction);
//   * two-level accumulation: the per-tile packed accumulator is flushed into a per-thread total
//     at every tile end (keeps the fp32 summation error ~ eps*(sqrt(TJ)+sqrt(N/TJ)));
//   * the sources are dealt to the gridDim.y j-splits in units of SUB, the targets handled are the
//     rows [i_begin, i_end) (the whole problem, or one rank's block of a row-sharded apply).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

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
// scalar-broadcast forms (the scalar is a source quantity or a constant, identical for both targets)
template <typename T> __device__ __forceinline__ P2<T> fma2(P2<T> a, T s, P2<T> c) { return fma2(a, splat(s), c); }
template <typename T> __device__ __forceinline__ P2<T> fma2(P2<T> a, T s, T c) { return fma2(a, splat(s), splat(c)); }
template <typename T> __device__ __forceinline__ P2<T> fma2(P2<T> a, P2<T> b, T c) { return fma2(a, b, splat(c)); }
template <typename T> __device__ __forceinline__ P2<T> mul2(P2<T> a, T s) { return mul2(a, splat(s)); }
template <typename T> __device__ __forceinline__ P2<T> add2(P2<T> a, T s) { return add2(a, splat(s)); }

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
// d := x_j - x_i = -r_vec is used un-normalised, every 1/r^n needed is folded into the scalars, and
// the Oseen prefactor C1 = 1/(8 pi eta) is factored out of every scalar and applied once per target
// in the epilogue.  With s = 1/r, u = s^2, w3 = s^3, w5 = s^5 (all scalars below are "/ C1"):
//   far  (r >= 2a): f_tt = s + c2 w3                 g_tt/r^2 = w3 (1 - c3 u)            c2 = 2a^2/3, c3 = 2a^2
//                   f_rr = -w3/2                     g_rr/r^2 = 3 w5/2                   h = g_c/r = w3
//   near (r <  2a): f_tt = c4 - c5 r                 g_tt/r^2 = c6 s                     c4 = 4/(3a)
//                   f_rr = c8 + r (k1 + k2 r^2)      g_rr/r^2 = k3 s + k4 r              h = k5 + k6 r
template <typename T> struct PairConsts {
    T tiny;    // additive floor of r^2: a^2 * 2^-80  (r = 0 -> finite 1/r, selected near branch)
    T four_a2; // (2a)^2
    T c2, nc3, c4, nc5, c6;               // translation-translation
    T c8, k1, k2, k3, k4, k5, k6;         // rotation-rotation and coupling (near branch)
    T C1_lin, C1_ang;                     // 1/(8 pi eta) x the internal length unit (x its square): applied in the epilogue
    T wa2, wzz0, wzz1;                    // single-wall correction: a^2, -8 a^2/3, 20 a^2 (wall_apply)
};

// overlap detector of the far-field fast path: running minimum of r^2 over a group of pairs.
// fp32: one FMNMX3 per packed pair.  fp64: r^2 >= 0, so IEEE order = integer order of the bit
// pattern; the minimum is taken over the HIGH 32-bit words only (one VIMNMX3 on the integer pipe
// instead of two FP64 compares) and the test is "<=", a superset of the exact r^2 < 4a^2: a group
// flagged needlessly is evaluated by the general body, whose per-lane select is exact.
struct NearF32 { float m; };
struct NearF64 { int m; };
template <typename T> struct NearOf;
template <> struct NearOf<float> { using type = NearF32; };
template <> struct NearOf<double> { using type = NearF64; };
__device__ __forceinline__ void near_init(NearF32& n) { n.m = 3.0e38f; }
__device__ __forceinline__ void near_init(NearF64& n) { n.m = 0x7fffffff; }
__device__ __forceinline__ void near_update(NearF32& n, float a, float b)
{
    asm("min.f32 %0, %0, %1, %2;" : "+f"(n.m) : "f"(a), "f"(b));          // SASS: FMNMX3
}
__device__ __forceinline__ void near_update(NearF64& n, double a, double b) { n.m = min(n.m, min(__double2hiint(a), __double2hiint(b))); }
__device__ __forceinline__ bool near_test(const NearF32& n, float four_a2) { return n.m < four_a2; }
__device__ __forceinline__ bool near_test(const NearF64& n, double four_a2) { return n.m <= __double2hiint(four_a2); }

template <typename T> struct PairParams {
    const T* __restrict__ pos;  // [3][npad]  x | y | z, ghosts (index >= N) are zeros
    const T* __restrict__ vec;  // [nrhs*NC][npad] packed right-hand sides, ghosts are zeros
    RhsOut<T> out;              // j_splits == 1: per right-hand side, 3N interleaved each
    T* __restrict__ partial;    // j_splits  > 1: [j_splits][nrhs*NC][npad]
    const T* __restrict__ damp; // single wall: damping factors b_i [npad] (ghosts 0), applied to the targets in the epilogue
                                // (the packed right-hand sides already carry b_j); pos z = raised height above the wall
    int64_t N;
    int64_t i_begin, i_end;     // target rows handled by this launch: [i_begin, i_end) (whole problem: [0, N));
                                // i-tile b covers i_begin + b * TARGETS ...  (row-sharded applies)
    int64_t npad;               // multiple of NPAD_QUANTUM (hence of every SUB in use)
    int n_units;                // npad / SUB: the sources are dealt to the gridDim.y j-splits in units of
                                // SUB, as evenly as possible (split y gets units [y U / S, (y+1) U / S))
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
// Consumer release of a stage (the CUTLASS consumer_release / producer_acquire pattern without a dedicated
// producer): every warp arrives on the stage's `empty` mbarrier once it has read the tile for the last time
// (mbarrier.arrive has release semantics at CTA scope); the arrival that finds ONE arrival pending in the state it
// replaced completes the phase.  That warp then observes the completed phase (test_wait: acquire), which orders every
// warp's generic-proxy reads of the tile before the TMA (async-proxy) refill it goes on to issue.
__device__ __forceinline__ bool mbar_arrive_is_last(uint64_t* bar)
{
    uint64_t state;
    uint32_t pending;
    asm volatile("mbarrier.arrive.shared::cta.b64 %0, [%1];" : "=l"(state) : "r"(smem_u32(bar)) : "memory");
    asm("mbarrier.pending_count.b64 %0, %1;" : "=r"(pending) : "l"(state));
    return pending == 1u;
}
// One non-blocking look at a phase (acquire when it reports completion).  Used by the warp whose own arrival has
// just completed the phase -- no spin loop, so the compiler keeps the surrounding code convergent.
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0u;
}
// 1-D bulk copy global -> shared, completion counted in bytes on `bar` (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------- one source vs one packed target pair
// Split in two so that the far / general decision of a whole group of pairs is taken BEFORE anything
// is accumulated: pair_geom gives d = x_j - x_i and r^2 (and feeds the overlap detector); pair_apply
// builds the scalars and accumulates.
//   FAR == true : far-field formulas only (the caller has checked that no pair of the group overlaps).
//   FAR == false: both branches, selected per lane.
// (nx, ny, nz) = -x_i of the two targets; (xj, yj, zj), V[] = the source, warp-uniform scalars.
template <typename T> struct PairGeom { P2<T> dx, dy, dz, r2, invr; };

// EARLY_RSQRT: issue the MUFU before the vote, so that its latency overlaps the vote and the branch;
// pays off where the apply body is long (angular, 4 right-hand sides: measured +2 %), costs ~1 % in
// register pressure on the short translational bodies, which therefore take 1/r after the vote.
template <typename T, bool EARLY_RSQRT>
__device__ __forceinline__ PairGeom<T> pair_geom(const PairConsts<T>& c, P2<T> nx, P2<T> ny, P2<T> nz, T xj, T yj, T zj,
                                                 typename NearOf<T>::type& near)
{
    PairGeom<T> g;
    g.dx = add2(nx, xj);
    g.dy = add2(ny, yj);
    g.dz = add2(nz, zj);
    g.r2 = fma2(g.dz, g.dz, fma2(g.dy, g.dy, fma2(g.dx, g.dx, splat(c.tiny))));
    near_update(near, lo(g.r2), hi(g.r2));
    if constexpr (EARLY_RSQRT) g.invr = rsqrt2(g.r2);
    return g;
}

template <typename T, int NRHS, bool ANG, bool FAR, bool EARLY_RSQRT>
__device__ __forceinline__ void pair_apply(const PairConsts<T>& c, const PairGeom<T>& gm, const T (&V)[NRHS * (ANG ? 6 : 3)],
                                           P2<T> (&acc)[NRHS * (ANG ? 6 : 3)])
{
    constexpr int NC = ANG ? 6 : 3;
    const P2<T> dx = gm.dx, dy = gm.dy, dz = gm.dz, r2 = gm.r2;
    const P2<T> invr = EARLY_RSQRT ? gm.invr : rsqrt2(r2);
    const P2<T> u = mul2(invr, invr);
    const P2<T> w3 = mul2(invr, u);
    P2<T> w5, f, g, r;
    // translation-translation scalars
    f = fma2(w3, c.c2, invr);
    if constexpr (ANG) {
        w5 = mul2(w3, u);
        g = fma2(w5, c.nc3, w3);
    } else {
        g = mul2(w3, fma2(u, c.nc3, T(1)));
    }
    bool nl = false, nh = false;
    if constexpr (!FAR) {
        nl = lo(r2) < c.four_a2;
        nh = hi(r2) < c.four_a2;
        r = mul2(r2, invr);
        f = sel2(nl, nh, fma2(r, c.nc5, c.c4), f);
        g = sel2(nl, nh, mul2(invr, c.c6), g);
    }
    if constexpr (!ANG) {
#pragma unroll
        for (int q = 0; q < NRHS; ++q) {
            const T Fx = V[q * NC + 0], Fy = V[q * NC + 1], Fz = V[q * NC + 2];
            const P2<T> t = mul2(g, fma2(dz, Fz, fma2(dy, Fy, mul2(dx, Fx))));
            acc[q * NC + 0] = fma2(f, Fx, fma2(t, dx, acc[q * NC + 0]));
            acc[q * NC + 1] = fma2(f, Fy, fma2(t, dy, acc[q * NC + 1]));
            acc[q * NC + 2] = fma2(f, Fz, fma2(t, dz, acc[q * NC + 2]));
        }
    } else {
        // rotation-rotation and coupling scalars
        P2<T> frr = mul2(w3, T(-0.5));
        P2<T> grr = mul2(w5, T(1.5));
        P2<T> h = w3;
        if constexpr (!FAR) {
            frr = sel2(nl, nh, fma2(r, fma2(r2, c.k2, c.k1), splat(c.c8)), frr);
            grr = sel2(nl, nh, fma2(invr, c.k3, mul2(r, c.k4)), grr);
            h = sel2(nl, nh, fma2(r, c.k6, c.k5), h);
        }
        // with d = -r_vec:  g_c (T x rhat) = h (d x T),  g_c (F x rhat) = h (d x F)
        const P2<T> hx = mul2(h, dx), hy = mul2(h, dy), hz = mul2(h, dz);
#pragma unroll
        for (int q = 0; q < NRHS; ++q) {
            const T Fx = V[q * NC + 0], Fy = V[q * NC + 1], Fz = V[q * NC + 2];
            const T Tx = V[q * NC + 3], Ty = V[q * NC + 4], Tz = V[q * NC + 5];
            const P2<T> t = mul2(g, fma2(dz, Fz, fma2(dy, Fy, mul2(dx, Fx))));
            const P2<T> s = mul2(grr, fma2(dz, Tz, fma2(dy, Ty, mul2(dx, Tx))));
            // U += f F + t d + (hd) x T        ((hd) x T)_x = hy Tz - hz Ty
            acc[q * NC + 0] = fma2(hz, -Ty, fma2(hy, Tz, fma2(f, Fx, fma2(t, dx, acc[q * NC + 0]))));
            acc[q * NC + 1] = fma2(hx, -Tz, fma2(hz, Tx, fma2(f, Fy, fma2(t, dy, acc[q * NC + 1]))));
            acc[q * NC + 2] = fma2(hy, -Tx, fma2(hx, Ty, fma2(f, Fz, fma2(t, dz, acc[q * NC + 2]))));
            // W += f_rr T + s d + (hd) x F
            acc[q * NC + 3] = fma2(hz, -Fy, fma2(hy, Fz, fma2(frr, Tx, fma2(s, dx, acc[q * NC + 3]))));
            acc[q * NC + 4] = fma2(hx, -Fz, fma2(hz, Fx, fma2(frr, Ty, fma2(s, dy, acc[q * NC + 4]))));
            acc[q * NC + 5] = fma2(hy, -Fx, fma2(hx, Fy, fma2(frr, Tz, fma2(s, dz, acc[q * NC + 5]))));
        }
    }
}

// ---------------------------------------------------------------- single wall
// The correction by which a no-slip wall at height 0 changes the pair mobility (the "Swan-Brady kernel"
// of ref. [37]): the Faxen operators applied to the image part of the half-space Green's function, DESIGN.md
// appendix A (closed forms) and reading S18; heights are >= a (reading S19: raised before packing), so the image
// distance |R| >= 2a, the forms are smooth and there is no near/far select.  Notation: R = x_i - x_j*,
// D = -R = (dx, dy, nZ) with nZ = -(z_i + z_j), h = z_j, u = 1/|R|^2, i1 = 1/|R|, i3 = i1 u, t = Z^2 u, p = a^2 u,
// w = z_i z_j u; everything "/ C1" like the free-space scalars.  |R|^2 = r^2 + 4 z_i z_j.
//   translation:  U += tI F + D (tRR q - tRz F_z) + zhat (tzz F_z - tzR q),   q = D.F
//     tI  = i1 [-1 - 2w + p (-2/3 + 2t)  + p^2 (2/3 - 10/3 t)]      tRz = i3 [2h - nZ (-12w + p (-4 + 20t) + p^2 (40/3 - 140/3 t))]
//     tRR = i3 [-1 + 6w + p (2 - 10t)    + p^2 (-10/3 + 70/3 t)]    tzR = i3 [2h + 20/3 p^2 nZ]
//     tzz = i3 [-4h^2 + p (-4 Z^2 - 8/3 a^2 + 20 a^2 t)]
//   rotation:     W += rI T + D (rRR s - rRz T_z) + zhat (rzz T_z - rzR s),   s = D.T,  i5 = i3 u
//     rI = i3 (7/2 - 6t)   rRR = -9/2 i5   rRz = -3 nZ i5   rzR = -6 nZ i5   rzz = -3 i3
//   coupling w <- F:  W += B (zhat x F) + P S + zhat i3 (dy F_x - dx F_y),   P = (-dy, dx, 0),  S = -C q + Dc F_z
//     B = i3 [-dz - 2p nZ]     -C = i5 [6h + 10 p nZ]     Dc = i3 [1 - 12 h nZ u + p (2 - 20t)]
//   coupling u <- T (the transpose of the block of the swapped pair):  m = dy T_x - dx T_y
//     U += B' (T_y, -T_x, 0) + (dx, dy, -nZ) C' m + zhat D' m + i3 (-dy, dx, 0) T_z
//     B' = i3 [dz - 2p nZ]     C' = i5 [-6 z_i - 10 p nZ]     D' = i3 [1 + 12 z_i (-nZ) u ... ] = i3 [1 + 12 nz nZ u + p (2 - 20t)], nz = -z_i
// nz = -z_i and nz4 = 4 z_i are per-target registers; zj, V[] the warp-uniform source.
template <typename T, int NRHS, bool ANG>
__device__ __forceinline__ void wall_apply(const PairConsts<T>& c, const PairGeom<T>& gm, P2<T> nz, P2<T> z4, T zj, const T (&V)[NRHS * (ANG ? 6 : 3)],
                                           P2<T> (&acc)[NRHS * (ANG ? 6 : 3)])
{
    constexpr int NC = ANG ? 6 : 3;
    const P2<T> dx = gm.dx, dy = gm.dy;
    const T h = zj, h2 = zj + zj;
    const P2<T> nZ = add2(nz, -h);
    const P2<T> R2 = fma2(z4, h, gm.r2);
    const P2<T> i1 = rsqrt2(R2);
    const P2<T> u = mul2(i1, i1), i3 = mul2(i1, u);
    const P2<T> Z2 = mul2(nZ, nZ), t = mul2(Z2, u), p = mul2(u, c.wa2), p2 = mul2(p, p);
    const P2<T> w = mul2(mul2(nz, -h), u);
    const P2<T> tI = mul2(i1, fma2(p2, fma2(t, T(-10.0 / 3.0), T(2.0 / 3.0)), fma2(p, fma2(t, T(2), T(-2.0 / 3.0)), fma2(w, T(-2), T(-1)))));
    const P2<T> tRR = mul2(i3, fma2(p2, fma2(t, T(70.0 / 3.0), T(-10.0 / 3.0)), fma2(p, fma2(t, T(-10), T(2)), fma2(w, T(6), T(-1)))));
    const P2<T> inner = fma2(p2, fma2(t, T(-140.0 / 3.0), T(40.0 / 3.0)), fma2(p, fma2(t, T(20), T(-4)), mul2(w, T(-12))));
    const P2<T> ntRz = mul2(i3, fma2(nZ, inner, -h2));                              // -tRz
    const P2<T> ntzR = mul2(i3, fma2(mul2(p2, T(-20.0 / 3.0)), nZ, -h2));            // -tzR
    const P2<T> tzz = mul2(i3, fma2(p, fma2(Z2, T(-4), fma2(t, c.wzz1, c.wzz0)), T(-4) * h * h));
    if constexpr (!ANG) {
#pragma unroll
        for (int q = 0; q < NRHS; ++q) {
            const T Fx = V[q * NC + 0], Fy = V[q * NC + 1], Fz = V[q * NC + 2];
            const P2<T> qF = fma2(nZ, Fz, fma2(dy, Fy, mul2(dx, Fx)));
            const P2<T> A = fma2(tRR, qF, mul2(ntRz, Fz));
            const P2<T> B = fma2(tzz, Fz, mul2(ntzR, qF));
            acc[q * NC + 0] = fma2(tI, Fx, fma2(dx, A, acc[q * NC + 0]));
            acc[q * NC + 1] = fma2(tI, Fy, fma2(dy, A, acc[q * NC + 1]));
            acc[q * NC + 2] = fma2(tI, Fz, fma2(nZ, A, add2(B, acc[q * NC + 2])));
        }
    } else {
        const P2<T> dz = gm.dz;
        const P2<T> i5 = mul2(i3, u);
        const P2<T> pz = mul2(p, nZ);                                               // p nZ
        const P2<T> poly = fma2(t, T(-20), T(2));                                   // 2 - 20 t
        const P2<T> rI = mul2(i3, fma2(t, T(-6), T(3.5)));
        const P2<T> cB = mul2(i3, fma2(pz, T(-2), mul2(dz, T(-1))));                // B  = i3 (-dz - 2 p nZ)
        const P2<T> cBp = mul2(i3, fma2(pz, T(-2), dz));                            // B' = i3 ( dz - 2 p nZ)
        const P2<T> nC = mul2(i5, fma2(pz, T(10), T(6) * h));                       // -C = i5 (6h + 10 p nZ)
        const P2<T> cCp = mul2(i5, fma2(pz, T(-10), mul2(nz, T(6))));               // C' = i5 (6 nz - 10 p nZ)
        const P2<T> nzu = mul2(nZ, u);
        const P2<T> cD = mul2(i3, fma2(p, poly, fma2(nzu, T(-12) * h, T(1))));      // Dc = i3 (1 - 12 h nZ u + p (2 - 20t))
        const P2<T> cDp = mul2(i3, fma2(p, poly, fma2(mul2(nzu, nz), T(12), T(1))));// D' = i3 (1 + 12 nz nZ u + p (2 - 20t))
        const P2<T> zC = fma2(nZ, mul2(cCp, T(-1)), cDp);                           // Z C' + D' = -nZ C' + D'
#pragma unroll
        for (int q = 0; q < NRHS; ++q) {
            const T Fx = V[q * NC + 0], Fy = V[q * NC + 1], Fz = V[q * NC + 2];
            const T Tx = V[q * NC + 3], Ty = V[q * NC + 4], Tz = V[q * NC + 5];
            const P2<T> qF = fma2(nZ, Fz, fma2(dy, Fy, mul2(dx, Fx)));
            const P2<T> qT = fma2(nZ, Tz, fma2(dy, Ty, mul2(dx, Tx)));
            const P2<T> A = fma2(tRR, qF, mul2(ntRz, Fz));
            const P2<T> B = fma2(tzz, Fz, mul2(ntzR, qF));
            const P2<T> m = fma2(dy, Tx, mul2(dx, -Ty));                            // P'.T = dy T_x - dx T_y
            const P2<T> Cm = mul2(cCp, m);
            const P2<T> i3Tz = mul2(i3, Tz);
            // U += tI F + D A + zhat B + [B' T_y + dx C'm - dy i3 T_z,  -B' T_x + dy C'm + dx i3 T_z,  (Z C' + D') m]
            acc[q * NC + 0] = fma2(dy, mul2(i3Tz, T(-1)), fma2(dx, Cm, fma2(cBp, Ty, fma2(tI, Fx, fma2(dx, A, acc[q * NC + 0])))));
            acc[q * NC + 1] = fma2(dx, i3Tz, fma2(dy, Cm, fma2(cBp, -Tx, fma2(tI, Fy, fma2(dy, A, acc[q * NC + 1])))));
            acc[q * NC + 2] = fma2(zC, m, fma2(tI, Fz, fma2(nZ, A, add2(B, acc[q * NC + 2]))));
            // W += rI T + D AT + zhat BT + [-B F_y - dy S,  B F_x + dx S,  i3 (dy F_x - dx F_y)]
            const P2<T> AT = mul2(i5, fma2(mul2(nZ, T(3)), Tz, mul2(qT, T(-4.5))));  // rRR s - rRz T_z = i5 (-9/2 s + 3 nZ T_z)
            const P2<T> BT = fma2(mul2(mul2(nZ, T(6)), i5), qT, mul2(i3Tz, T(-3)));  // rzz T_z - rzR s = -3 i3 T_z + 6 nZ i5 s
            const P2<T> S = fma2(nC, qF, mul2(cD, Fz));
            acc[q * NC + 3] = fma2(dy, mul2(S, T(-1)), fma2(cB, -Fy, fma2(rI, Tx, fma2(dx, AT, acc[q * NC + 3]))));
            acc[q * NC + 4] = fma2(dx, S, fma2(cB, Fx, fma2(rI, Ty, fma2(dy, AT, acc[q * NC + 4]))));
            acc[q * NC + 5] = fma2(i3, fma2(dy, Fx, mul2(dx, -Fy)), fma2(rI, Tz, fma2(nZ, AT, add2(BT, acc[q * NC + 5]))));
        }
    }
}

// ---------------------------------------------------------------- kernel
template <typename T> struct Vec16;                   // 16-byte shared-memory load = 4 sources (fp32) or 2 (fp64)
template <> struct Vec16<float> { static constexpr int N = 4; using type = float4; };
template <> struct Vec16<double> { static constexpr int N = 2; using type = double2; };
__device__ __forceinline__ float vget(const float4& v, int k) { return k == 0 ? v.x : (k == 1 ? v.y : (k == 2 ? v.z : v.w)); }
__device__ __forceinline__ double vget(const double2& v, int k) { return k == 0 ? v.x : v.y; }

// ACC64 (fp32 kernels only; SURVEY.md sec. 8(f) NEXT-4 "mixed precision: fp32 pair math, fp64 accumulation"): the packed fp32
// accumulators are flushed every ACC64_RUN sources into per-thread fp64 totals kept in shared memory, the j-split
// partials are written in fp64 and the result is rounded to fp32 once.  The fp32 error of a sum is dominated by the
// LENGTH of the fp32 runs: runs of 32 instead of 512 + 7 + 37 take config 3 from 6.0e-7 to 1.4e-7.
constexpr int ACC64_RUN = 32;

template <typename T, int NRHS, bool ANG, int TPT, int BLOCK, int TJ, int STAGES, int SUB, bool ACC64 = false>
struct PairKernelTraits {
    static_assert(TPT % 2 == 0, "targets are held as packed pairs");
    static_assert(TJ % SUB == 0 && SUB % Vec16<T>::N == 0, "source units");
    // sources per far/general decision: the group's geometry (GS x NP packed d, r^2) stays in registers
    static constexpr int GS = ((TPT / 2 >= 2 || NRHS * (ANG ? 6 : 3) >= 12) && Vec16<T>::N > 2) ? 2 : Vec16<T>::N;
    static constexpr int NC = ANG ? 6 : 3;             // components per source per right-hand side
    static constexpr int NV = NRHS * NC;               // packed vector arrays
    static constexpr int NP = TPT / 2;                 // packed target pairs per thread
    static constexpr int ARRAYS = 3 + NV;              // x, y, z + vector components
    static constexpr int STAGE_BYTES = ARRAYS * TJ * (int)sizeof(T);
    static constexpr int BAR_BYTES = STAGES * 8 + STAGES * 8;                           // full mbarriers | empty mbarriers
    static constexpr int TOT64_BYTES = ACC64 ? TPT * NV * BLOCK * 8 : 0;               // fp64 totals [TPT * NV][BLOCK]
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + TOT64_BYTES;
    static constexpr int TARGETS = BLOCK * TPT;        // targets per CTA
    static_assert(!ACC64 || (std::is_same<T, float>::value && SUB % ACC64_RUN == 0 && ACC64_RUN % Vec16<T>::N == 0), "ACC64: fp32 kernels, runs aligned with the source units");
};

template <typename T, int NRHS, bool ANG, int TPT, int BLOCK, int TJ, int STAGES, int SUB, int MINB, bool WALL = false, bool ACC64 = false>
__global__ void __launch_bounds__(BLOCK, MINB) rpy_pair_kernel(const PairParams<T> p)
{
    using Tr = PairKernelTraits<T, NRHS, ANG, TPT, BLOCK, TJ, STAGES, SUB, ACC64>;
    constexpr int NC = Tr::NC, NV = Tr::NV, NP = Tr::NP, ARRAYS = Tr::ARRAYS;
    constexpr int VN = Vec16<T>::N, GS = Tr::GS;
    constexpr bool EARLY = ANG || NRHS >= 4;
    using V16 = typename Vec16<T>::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* tiles = reinterpret_cast<T*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + STAGES * Tr::STAGE_BYTES);
    uint64_t* empty = full + STAGES;                  // per stage: the BLOCK / 32 warps that have finished with it
    double* tot64 = reinterpret_cast<double*>(smem_raw + STAGES * Tr::STAGE_BYTES + Tr::BAR_BYTES);   // ACC64: [TPT * NV][BLOCK], thread-private columns
    constexpr unsigned int NWARPS = BLOCK / 32;

    const int tid = threadIdx.x;
    const int64_t i0 = p.i_begin + (int64_t)blockIdx.x * Tr::TARGETS;
    // this CTA's source range [j_begin, j_begin + j_count): a whole number of SUB-source units
    const int u_begin = (int)((int64_t)blockIdx.y * p.n_units / gridDim.y);
    const int u_end = (int)((int64_t)(blockIdx.y + 1) * p.n_units / gridDim.y);
    const int64_t j_begin = (int64_t)u_begin * SUB;
    const int j_count = (u_end - u_begin) * SUB;
    const int my_tiles = (j_count + TJ - 1) / TJ;     // the last tile may be short

    auto issue = [&](int local_tile) {               // called by thread 0 only
        const int stage = local_tile % STAGES;
        const int64_t j0 = j_begin + (int64_t)local_tile * TJ;
        const uint32_t nsrc = (uint32_t)min(TJ, j_count - local_tile * TJ);
        const uint32_t bytes = nsrc * (uint32_t)sizeof(T);     // multiple of 16: SUB * sizeof(T) is
        T* dst = tiles + (size_t)stage * ARRAYS * TJ;
        mbar_expect_tx(&full[stage], bytes * ARRAYS);
#pragma unroll
        for (int a = 0; a < 3; ++a) bulk_g2s(dst + a * TJ, p.pos + a * p.npad + j0, bytes, &full[stage]);
#pragma unroll
        for (int a = 0; a < NV; ++a) bulk_g2s(dst + (3 + a) * TJ, p.vec + a * p.npad + j0, bytes, &full[stage]);
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], NWARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int s = 0; s < STAGES && s < my_tiles; ++s) issue(s);
    }

    // targets: pair q holds targets i0 + (2q)*BLOCK + tid and i0 + (2q+1)*BLOCK + tid; negated
    // coordinates so that d = x_j + (-x_i) is one packed add.  Targets past npad (last i-tile)
    // re-read the last ghost; they are never stored.
    P2<T> nx[NP], ny[NP], nz[NP];
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        const int64_t ia = min(i0 + (2 * q) * BLOCK + tid, p.npad - 1), ib = min(i0 + (2 * q + 1) * BLOCK + tid, p.npad - 1);
        nx[q] = mk2(-p.pos[ia], -p.pos[ib]);
        ny[q] = mk2(-p.pos[p.npad + ia], -p.pos[p.npad + ib]);
        nz[q] = mk2(-p.pos[2 * p.npad + ia], -p.pos[2 * p.npad + ib]);
    }
    P2<T> z4[WALL ? NP : 1];                        // single wall: 4 z_i, so that |R|^2 = r^2 + (4 z_i) z_j is one FMA
    if constexpr (WALL) {
#pragma unroll
        for (int q = 0; q < NP; ++q) z4[q] = mul2(nz[q], T(-4));
    }
    P2<T> total[NP][NV];
#pragma unroll
    for (int q = 0; q < NP; ++q)
#pragma unroll
        for (int k = 0; k < NV; ++k) total[q][k] = splat(T(0));
    if constexpr (ACC64) {
#pragma unroll
        for (int s = 0; s < TPT * NV; ++s) tot64[s * BLOCK + tid] = 0.0;
    }

    using Near = typename NearOf<T>::type;

    for (int lt = 0; lt < my_tiles; ++lt) {
        const int stage = lt % STAGES;
        mbar_wait(&full[stage], (uint32_t)((lt / STAGES) & 1));
        const T* sx = tiles + (size_t)stage * ARRAYS * TJ;
        const int tile_count = min(TJ, j_count - lt * TJ);

        // per-tile packed accumulators (two-level summation: flushed into `total` at the tile end)
        P2<T> acc[NP][NV];
#pragma unroll
        for (int q = 0; q < NP; ++q)
#pragma unroll
            for (int k = 0; k < NV; ++k) acc[q][k] = splat(T(0));

        // sources are walked in groups of GS; the geometry of the whole group (GS x NP packed pairs)
        // comes first, one warp vote on its minimum r^2 picks the far-field or the general body
        auto walk = [&](int j) {                      // VN sources of the tile, from source j on
            const V16 X = *reinterpret_cast<const V16*>(sx + j);
            const V16 Y = *reinterpret_cast<const V16*>(sx + TJ + j);
            const V16 Z = *reinterpret_cast<const V16*>(sx + 2 * TJ + j);
            V16 Vv[NV];
#pragma unroll
            for (int k = 0; k < NV; ++k) Vv[k] = *reinterpret_cast<const V16*>(sx + (3 + k) * TJ + j);
#pragma unroll
            for (int e0 = 0; e0 < VN; e0 += GS) {
                PairGeom<T> gm[GS][NP];
                Near near;
                near_init(near);
#pragma unroll
                for (int e = 0; e < GS; ++e)
#pragma unroll
                    for (int q = 0; q < NP; ++q)
                        gm[e][q] = pair_geom<T, EARLY>(p.c, nx[q], ny[q], nz[q], vget(X, e0 + e), vget(Y, e0 + e), vget(Z, e0 + e), near);
                const bool hit = __any_sync(0xffffffffu, near_test(near, p.c.four_a2));
                auto body = [&](auto far_tag) {
                    constexpr bool FAR = decltype(far_tag)::value;
#pragma unroll
                    for (int e = 0; e < GS; ++e) {
                        T Vs[NV];
#pragma unroll
                        for (int k = 0; k < NV; ++k) Vs[k] = vget(Vv[k], e0 + e);
#pragma unroll
                        for (int q = 0; q < NP; ++q) {
                            pair_apply<T, NRHS, ANG, FAR, EARLY>(p.c, gm[e][q], Vs, acc[q]);
                            if constexpr (WALL) wall_apply<T, NRHS, ANG>(p.c, gm[e][q], nz[q], z4[q], vget(Z, e0 + e), Vs, acc[q]);
                        }
                    }
                };
                if (!hit) body(std::true_type{});
                else body(std::false_type{});
            }
        };
        if constexpr (!ACC64) {
#pragma unroll 1
            for (int j = 0; j < tile_count; j += VN) walk(j);
            // flush the per-tile packed accumulators
#pragma unroll
            for (int q = 0; q < NP; ++q)
#pragma unroll
                for (int k = 0; k < NV; ++k) total[q][k] = add2(total[q][k], acc[q][k]);
        } else {
            // fp32 runs of ACC64_RUN sources, each flushed into this thread's fp64 totals (tile_count is a multiple of SUB)
#pragma unroll 1
            for (int j0 = 0; j0 < tile_count; j0 += ACC64_RUN) {
#pragma unroll 1
                for (int j = j0; j < j0 + ACC64_RUN; j += VN) walk(j);
#pragma unroll
                for (int q = 0; q < NP; ++q)
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        double* t0 = tot64 + ((2 * q) * NV + k) * BLOCK + tid;
                        double* t1 = tot64 + ((2 * q + 1) * NV + k) * BLOCK + tid;
                        *t0 += (double)lo(acc[q][k]);
                        *t1 += (double)hi(acc[q][k]);
                        acc[q][k] = splat(T(0));
                    }
            }
        }

        // release the stage without a CTA-wide barrier: every warp arrives on the stage's `empty` mbarrier, the LAST
        // one to leave refills the stage (TMA) -- no warp ever waits for another except on the data it needs
        __syncwarp();
        if ((tid & 31) == 0 && mbar_arrive_is_last(&empty[stage]) && lt + STAGES < my_tiles) {
            // the phase was completed by this very arrival: observing it (acquire) orders the other warps' reads first
            // (a `__trap()` on the impossible "not complete" outcome was tried in round 3: +6 registers (122 -> 128) and
            // 3.4 % on the config-3 launch, 11.74 -> 12.15 ms; not kept)
            if (mbar_test(&empty[stage], (uint32_t)((lt / STAGES) & 1))) issue(lt + STAGES);
        }
    }

    // ---- epilogue: apply the factored-out Oseen prefactor once per target (single wall: times the damping factor b_i)
    if constexpr (ACC64) {
        // fp64 totals -> caller's arrays (rounded once) or fp64 j-split partials [split][NV][npad]
#pragma unroll
        for (int q = 0; q < NP; ++q) {
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                const int64_t i = i0 + (2 * q + half) * BLOCK + tid;
                double fl = (double)p.c.C1_lin, fa = (double)p.c.C1_ang;
                if constexpr (WALL) {
                    const double b = (double)p.damp[min(i, p.npad - 1)];
                    fl *= b;
                    fa *= b;
                }
                const double* mine = tot64 + ((2 * q + half) * NV) * BLOCK + tid;
                if (gridDim.y == 1) {
                    if (i < p.i_end) {
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) {
#pragma unroll
                            for (int k = 0; k < 3; ++k) p.out.lin[r][3 * i + k] = (T)(mine[(r * NC + k) * BLOCK] * fl);
                            if constexpr (ANG) {
#pragma unroll
                                for (int k = 0; k < 3; ++k) p.out.ang[r][3 * i + k] = (T)(mine[(r * NC + 3 + k) * BLOCK] * fa);
                            }
                        }
                    }
                } else if (i < p.npad) {
                    double* part = reinterpret_cast<double*>(p.partial) + (size_t)blockIdx.y * NV * p.npad;
#pragma unroll
                    for (int k = 0; k < NV; ++k) part[(size_t)k * p.npad + i] = mine[k * BLOCK] * ((k % NC) < 3 ? fl : fa);
                }
            }
        }
        return;
    }
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        P2<T> fl = splat(p.c.C1_lin), fa = splat(p.c.C1_ang);
        if constexpr (WALL) {
            const int64_t ia = min(i0 + (2 * q) * BLOCK + tid, p.npad - 1), ib = min(i0 + (2 * q + 1) * BLOCK + tid, p.npad - 1);
            const P2<T> b = mk2(p.damp[ia], p.damp[ib]);
            fl = mul2(fl, b);
            fa = mul2(fa, b);
        }
#pragma unroll
        for (int k = 0; k < NV; ++k) total[q][k] = mul2(total[q][k], (k % NC) < 3 ? fl : fa);
    }
#pragma unroll
    for (int q = 0; q < NP; ++q) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const int64_t i = i0 + (2 * q + half) * BLOCK + tid;
            if (gridDim.y == 1) {
                if (i < p.i_end) {
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) {
                        T* ul = p.out.lin[r] + 3 * i;
#pragma unroll
                        for (int k = 0; k < 3; ++k) ul[k] = half ? hi(total[q][r * NC + k]) : lo(total[q][r * NC + k]);
                        if constexpr (ANG) {
                            T* ua = p.out.ang[r] + 3 * i;
#pragma unroll
                            for (int k = 0; k < 3; ++k) ua[k] = half ? hi(total[q][r * NC + 3 + k]) : lo(total[q][r * NC + 3 + k]);
                        }
                    }
                }
            } else if (i < p.npad) {
                T* part = p.partial + (size_t)blockIdx.y * NV * p.npad;
#pragma unroll
                for (int k = 0; k < NV; ++k) part[(size_t)k * p.npad + i] = half ? hi(total[q][k]) : lo(total[q][k]);
            }
        }
    }
}

}  // namespace lm
