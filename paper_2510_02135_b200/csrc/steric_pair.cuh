// steric_pair.cuh -- all-pairs soft steric repulsion, eq. (13), and the stochastic
// Adams-Bashforth position update, eq. (14): the O(N^2) / O(N) kernels of the
// free-space Brownian-dynamics step built around the mobility hot path.
//
//   F_i = ext_i + sum_{j != i} m(r_ij) (x_i - x_j) / r_ij,   m(r) = -U'(r) = U0/b              (r <  d)
//                                                                        = U0/b exp((d - r)/b)  (r >= d),  d = 2a
//
// Same machine mapping as the RPY pair kernel (rpy_pair.cuh): one packed target pair per thread, all
// lanes of a warp walk the same sources from TMA-staged SoA tiles, broadcast LDS.128.  The
// interaction is short ranged (b << a): sources are walked in groups, the group's d and r^2 come
// first with a running minimum, and ONE warp vote skips the group when no pair is within the
// cut-off r_c = d + K b (K = 20 fp32, 40 fp64: exp(-K) is below the type's epsilon), so a far group
// costs 6 packed FP operations per pair and neither of the two MUFU ops.  Ghost sources (index >= N,
// stored at the origin) are masked by index; r = 0 (the self pair, coincident particles) adds nothing.
#pragma once
#include "rpy_pair.cuh"

namespace lm {

template <typename T> struct StericParams {
    const T* __restrict__ pos;   // [3][npad]  x | y | z   (single wall: [5][npad], the true height is array 3)
    int z_array;                 // which array holds z: 2, or 3 with a wall (array 2 is then the RAISED height of the mobility)
    T* __restrict__ partial;     // [j_splits][3][npad]
    int64_t N, npad;
    int64_t i_begin;             // first target row of this launch (row-sharded runs; 0 otherwise)
    int n_units;                 // npad / STERIC_SUB
    T tiny;                      // floor of r^2 (as in the RPY kernel)
    T d;                         // contact distance 2a
    T rc2;                       // cut-off radius squared
    T m0;                        // U0 / b
    T inv_b;                     // 1/b  (fp32: log2(e)/b, the exponential is taken as ex2)
};

constexpr int STERIC_BLOCK = 256, STERIC_TJ = 512, STERIC_STAGES = 2, STERIC_SUB = 32;
constexpr int STERIC_TARGETS = STERIC_BLOCK * 2;
template <typename T> constexpr int steric_smem_bytes() { return STERIC_STAGES * 3 * STERIC_TJ * (int)sizeof(T) + STERIC_STAGES * 16; }

__device__ __forceinline__ float steric_exp(float arg_log2) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(arg_log2)); return y; }
__device__ __forceinline__ double steric_exp(double arg) { return exp(arg); }

template <typename T>
__global__ void __launch_bounds__(STERIC_BLOCK, 2) steric_pair_kernel(const StericParams<T> p)
{
    constexpr int TJ = STERIC_TJ, STAGES = STERIC_STAGES, SUB = STERIC_SUB, BLOCK = STERIC_BLOCK;
    constexpr int VN = Vec16<T>::N;
    constexpr unsigned int NWARPS = BLOCK / 32;
    using V16 = typename Vec16<T>::type;
    using Near = typename NearOf<T>::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* tiles = reinterpret_cast<T*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + STAGES * 3 * TJ * sizeof(T));
    uint64_t* empty = full + STAGES;                  // per stage: the warps that have finished with it (rpy_pair.cuh mbar_arrive_is_last)

    const int tid = threadIdx.x;
    const int64_t i0 = p.i_begin + (int64_t)blockIdx.x * STERIC_TARGETS;
    const int u_begin = (int)((int64_t)blockIdx.y * p.n_units / gridDim.y);
    const int u_end = (int)((int64_t)(blockIdx.y + 1) * p.n_units / gridDim.y);
    const int64_t j_begin = (int64_t)u_begin * SUB;
    const int j_count = (u_end - u_begin) * SUB;
    const int my_tiles = (j_count + TJ - 1) / TJ;

    auto issue = [&](int local_tile) {
        const int stage = local_tile % STAGES;
        const int64_t j0 = j_begin + (int64_t)local_tile * TJ;
        const uint32_t bytes = (uint32_t)min(TJ, j_count - local_tile * TJ) * (uint32_t)sizeof(T);
        T* dst = tiles + (size_t)stage * 3 * TJ;
        mbar_expect_tx(&full[stage], bytes * 3);
#pragma unroll
        for (int a = 0; a < 3; ++a) bulk_g2s(dst + a * TJ, p.pos + (size_t)(a == 2 ? p.z_array : a) * p.npad + j0, bytes, &full[stage]);
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
    if (tid == 0)
        for (int s = 0; s < STAGES && s < my_tiles; ++s) issue(s);

    const int64_t ia = min(i0 + tid, p.npad - 1), ib = min(i0 + BLOCK + tid, p.npad - 1);
    const P2<T> nx = mk2(-p.pos[ia], -p.pos[ib]);
    const P2<T> ny = mk2(-p.pos[p.npad + ia], -p.pos[p.npad + ib]);
    const P2<T> nz = mk2(-p.pos[(size_t)p.z_array * p.npad + ia], -p.pos[(size_t)p.z_array * p.npad + ib]);
    P2<T> fx = splat(T(0)), fy = splat(T(0)), fz = splat(T(0));

    for (int lt = 0; lt < my_tiles; ++lt) {
        const int stage = lt % STAGES;
        mbar_wait(&full[stage], (uint32_t)((lt / STAGES) & 1));
        const T* sx = tiles + (size_t)stage * 3 * TJ;
        const int tile_count = min(TJ, j_count - lt * TJ);
        const int64_t jt0 = j_begin + (int64_t)lt * TJ;
#pragma unroll 1
        for (int j = 0; j < tile_count; j += VN) {
            const V16 X = *reinterpret_cast<const V16*>(sx + j);
            const V16 Y = *reinterpret_cast<const V16*>(sx + TJ + j);
            const V16 Z = *reinterpret_cast<const V16*>(sx + 2 * TJ + j);
            P2<T> dx[VN], dy[VN], dz[VN], r2[VN];
            Near near;
            near_init(near);
#pragma unroll
            for (int e = 0; e < VN; ++e) {
                dx[e] = add2(nx, vget(X, e));
                dy[e] = add2(ny, vget(Y, e));
                dz[e] = add2(nz, vget(Z, e));
                r2[e] = fma2(dz[e], dz[e], fma2(dy[e], dy[e], fma2(dx[e], dx[e], splat(p.tiny))));
                near_update(near, lo(r2[e]), hi(r2[e]));
            }
            if (!__any_sync(0xffffffffu, near_test(near, p.rc2))) continue;   // whole group beyond the cut-off
#pragma unroll
            for (int e = 0; e < VN; ++e) {
                const P2<T> invr = rsqrt2(r2[e]);
                const P2<T> r = mul2(r2[e], invr);
                const T valid = (jt0 + j + e) < p.N ? p.m0 : T(0);           // ghost sources exert nothing
                // m(r) = m0 min(1, exp((d - r)/b)): exp >= 1 exactly where r <= d
                const P2<T> arg = mul2(add2(mul2(r, T(-1)), p.d), p.inv_b);
                const T el = lo(arg) >= T(0) ? T(1) : steric_exp(lo(arg));
                const T eh = hi(arg) >= T(0) ? T(1) : steric_exp(hi(arg));
                // F_i += m (x_i - x_j)/r = -m invr d
                const P2<T> w = mul2(mul2(mk2(el, eh), invr), -valid);
                fx = fma2(w, dx[e], fx);
                fy = fma2(w, dy[e], fy);
                fz = fma2(w, dz[e], fz);
            }
        }
        __syncwarp();
        if ((tid & 31) == 0 && mbar_arrive_is_last(&empty[stage]) && lt + STAGES < my_tiles) {
            if (mbar_test(&empty[stage], (uint32_t)((lt / STAGES) & 1))) issue(lt + STAGES);   // completed by this arrival: acquire, then refill
        }
    }

    T* part = p.partial + (size_t)blockIdx.y * 3 * p.npad;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        const int64_t i = i0 + half * BLOCK + tid;
        if (i < p.npad) {
            part[i] = half ? hi(fx) : lo(fx);
            part[p.npad + i] = half ? hi(fy) : lo(fy);
            part[2 * p.npad + i] = half ? hi(fz) : lo(fz);
        }
    }
}

// F[3i+k] = ext[3i+k] + sum over splits of partial  (fixed order: deterministic).
// Single wall (`height` != null: the particles' heights above the wall, internal unit): plus the particle-wall repulsion
// of eq. (13) with r = height of the centre and d = a, F_z += U0/b (r < d), U0/b exp((d - r)/b) (r >= d).
template <typename T>
__global__ void __launch_bounds__(256) steric_reduce_kernel(const T* __restrict__ partial, int splits, int64_t i_begin, int64_t i_end, int64_t npad,
                                                            const T* __restrict__ ext, T* __restrict__ out, const T* __restrict__ height, T wall_d,
                                                            T wall_m0, T wall_inv_b)
{
    const int64_t i = i_begin + (int64_t)blockIdx.x * 256 + threadIdx.x;   // target rows [i_begin, i_end)
    if (i >= i_end) return;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        T s = ext ? ext[3 * i + k] : T(0);
        for (int q = 0; q < splits; ++q) s += partial[((size_t)q * 3 + k) * npad + i];
        if (height && k == 2) {
            const T r = height[i];
            s += r < wall_d ? wall_m0 : wall_m0 * exp((wall_d - r) * wall_inv_b);
        }
        out[3 * i + k] = s;
    }
}

// eq. (14): X += dt (c_n v_n - c_p v_prev) + pref y;  v_prev <- v_n.  (c_n, c_p) = (3/2, 1/2), or (1, 0)
// on the first step (forward Euler: no history).  y == nullptr: deterministic step.
template <typename T>
__global__ void __launch_bounds__(256) bd_update_kernel(T* __restrict__ pos, const T* __restrict__ v_n, T* __restrict__ v_prev,
                                                        const T* __restrict__ y, int64_t n3, T dt_cn, T dt_cp, T pref)
{
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n3) return;
    const T vn = v_n[i];
    T x = pos[i] + dt_cn * vn;
    if (dt_cp != T(0)) x -= dt_cp * v_prev[i];
    if (y) x += pref * y[i];
    pos[i] = x;
    v_prev[i] = vn;
}

}  // namespace lm
