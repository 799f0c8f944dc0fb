// vector_kernels.cuh -- the O(N) kernels around the pair kernel: packing to structure-of-arrays,
// split-j reduction, and the Lanczos vector operations.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "lm_common.cuh"

namespace lm {

constexpr int VEC_BLOCK = 256;       // threads per block of every kernel in this file
constexpr int RED_MAX_BLOCKS = 1024; // upper bound on the grid of the reduction kernels

// a1: interleaved positions (3N) -> x | y | z, each npad long, ghosts zero.  Lengths are stored multiplied by
// `len_scale`, the power of two nearest 1/a (exact): the pair kernel then works with a radius in [0.71, 1.41]
// whatever unit system the caller uses ("internal length unit").
//
// Single wall (`wall` != 0; reading S19, "damping matrix approach"): five arrays
// x | y | z~ | h | b  with h = (z - wall_z) the height of the centre above the wall, z~ = max(h, a) the RAISED height the
// pair kernel works with, and b = min(1, max(h, 0)/a) the damping factor (ghosts: z~ = a, b = 0).  All lengths x len_scale.
template <typename T> struct WallPack { int on; T wall_z, a_scaled; };   // wall_z in the caller's unit, a_scaled = a * len_scale

template <typename T> __device__ __forceinline__ void wall_raise(T h, T a_scaled, T& z_raised, T& b)
{
    z_raised = h > a_scaled ? h : a_scaled;
    b = h >= a_scaled ? T(1) : (h > T(0) ? h / a_scaled : T(0));
}

template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) pack_positions_kernel(const T* __restrict__ pos, int64_t N, int64_t npad, T len_scale, WallPack<T> wall,
                                                                   T* __restrict__ soa)
{
    const int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x;
    if (i >= npad) return;
    T x = T(0), y = T(0), z = T(0);
    if (i < N) { x = pos[3 * i] * len_scale; y = pos[3 * i + 1] * len_scale; z = (wall.on ? pos[3 * i + 2] - wall.wall_z : pos[3 * i + 2]) * len_scale; }
    soa[i] = x;
    soa[npad + i] = y;
    if (!wall.on) {
        soa[2 * npad + i] = z;
        return;
    }
    T zr = wall.a_scaled, b = T(0);
    if (i < N) wall_raise(z, wall.a_scaled, zr, b);
    soa[2 * npad + i] = zr;
    soa[3 * npad + i] = z;
    soa[4 * npad + i] = b;
}

// a2: right-hand sides -> [nrhs*NC][npad] component arrays (NC = 3: Fx Fy Fz; NC = 6: + Tx Ty Tz),
// ghosts zero; a null force / torque pointer means zeros.  Torques are stored multiplied by
// `len_scale` (the internal length unit: a torque is a force times a length).
// `damp` (single wall, else null): the sources' damping factors b_j, folded into the packed values (M~ = B M B).
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) pack_rhs_kernel(RhsIn<T> in, int nrhs, int nc, int64_t N, int64_t npad, T len_scale, const T* __restrict__ damp,
                                                             T* __restrict__ soa)
{
    const int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x;
    if (i >= npad) return;
    const T b = damp ? damp[i] : T(1);
    for (int q = 0; q < nrhs; ++q) {
        T v[6] = {T(0), T(0), T(0), T(0), T(0), T(0)};
        if (i < N) {
            if (in.f[q]) { v[0] = in.f[q][3 * i]; v[1] = in.f[q][3 * i + 1]; v[2] = in.f[q][3 * i + 2]; }
            if (nc == 6 && in.t[q]) { v[3] = in.t[q][3 * i] * len_scale; v[4] = in.t[q][3 * i + 1] * len_scale; v[5] = in.t[q][3 * i + 2] * len_scale; }
        }
        for (int k = 0; k < nc; ++k) soa[(size_t)(q * nc + k) * npad + i] = damp ? v[k] * b : v[k];
    }
}

// a6: sum the j-split partials in a fixed order (deterministic) and write interleaved outputs, for the right-hand
// sides [q_begin, nrhs) (the Lanczos driver reduces its own vectors inside its alpha kernel).
// One thread per (right-hand side, component, particle): consecutive threads read consecutive
// addresses of one partial array; the loads of the splits are independent and unrolled.
// TP = type of the partials: T, or double when the pair kernel accumulates in fp64 (LM_OPT_ACCUMULATE_F64): summed in TP,
// rounded to T once.
template <typename T, typename TP = T>
__global__ void __launch_bounds__(VEC_BLOCK) reduce_partials_kernel(const TP* __restrict__ partial, int splits, int nrhs, int nc, int q_begin,
                                                                    int64_t i_begin, int64_t i_end, int64_t npad, RhsOut<T> out)
{
    const int64_t i = i_begin + (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x;   // target rows [i_begin, i_end)
    if (i >= i_end) return;
    const int qk = q_begin * nc + blockIdx.y, q = qk / nc, k = qk % nc;          // right-hand sides [q_begin, nrhs): gridDim.y = (nrhs - q_begin) nc
    const size_t stride = (size_t)nrhs * nc * npad;
    const TP* p = partial + (size_t)qk * npad + i;
    TP s = TP(0);
    int sidx = 0;
    for (; sidx + 8 <= splits; sidx += 8) {
        TP v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = p[(size_t)(sidx + u) * stride];
#pragma unroll
        for (int u = 0; u < 8; ++u) s += v[u];
    }
    for (; sidx < splits; ++sidx) s += p[(size_t)sidx * stride];
    if (k < 3) out.lin[q][3 * i + k] = (T)s;
    else       out.ang[q][3 * i + (k - 3)] = (T)s;
}

// eq. (11) PAPER.md:151-155 (random finite difference): packed positions displaced along W,
// out[c][i] = soa[c][i] + s W[3i+c]  (s = +-delta/2); ghosts stay where they are.
// Single wall: the height h (array 3) is displaced and the raised height and damping factor are formed anew.
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) shift_positions_kernel(const T* __restrict__ soa, const T* __restrict__ W, int64_t N, int64_t npad, T s,
                                                                    WallPack<T> wall, T* __restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x;
    if (i >= npad) return;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        T v = soa[(size_t)((wall.on && c == 2) ? 3 : c) * npad + i];
        if (i < N) v += s * W[3 * i + c];
        if (wall.on && c == 2) {
            T zr = wall.a_scaled, b = T(0);
            if (i < N) wall_raise(v, wall.a_scaled, zr, b);
            out[(size_t)2 * npad + i] = zr;
            out[(size_t)3 * npad + i] = v;
            out[(size_t)4 * npad + i] = b;
        } else {
            out[(size_t)c * npad + i] = v;
        }
    }
}

// up = (up - um) * inv_delta   (the difference quotient of eq. (11))
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) rfd_difference_kernel(T* __restrict__ up, const T* __restrict__ um, int64_t n, T inv_delta)
{
    const int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x;
    if (i < n) up[i] = (up[i] - um[i]) * inv_delta;
}

// y += s x   (the drift term joining the deterministic velocity of eq. (14))
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) add_scaled_kernel(T* __restrict__ y, const T* __restrict__ x, T s, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x;
    if (i < n) y[i] = fma(s, x[i], y[i]);
}

// ---------------------------------------------------------------- Lanczos vector operations (a7)
// Reductions: warp shuffles -> one fp64 partial per block -> the last block to finish (ticket)
// adds the block partials in index order, so the result is deterministic for a given grid.
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ void block_reduce_to_scalar(double v, double* block_partials, unsigned int* ticket, double* result,
                                                       double* host_mirror = nullptr, int* advance = nullptr)
{
    __shared__ double warp_part[VEC_BLOCK / 32];
    __shared__ bool is_last;
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < VEC_BLOCK / 32; ++w) s += warp_part[w];
        block_partials[blockIdx.x] = s;
        __threadfence();
        const unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last && threadIdx.x < 32) {
        __threadfence();
        double s = 0.0;
        for (unsigned int b = threadIdx.x; b < gridDim.x; b += 32) s += ((volatile double*)block_partials)[b];
        s = warp_sum(s);
        if (threadIdx.x == 0) {
            *result = s;
            if (host_mirror) *host_mirror = s;
            if (advance) *advance += 1;       // every block has taken its ticket, hence read the old value: safe to move on
            *ticket = 0u;
        }
    }
}

// result = sum_i x_i^2          (|z|^2 of the noise vector)
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) sumsq_kernel(const T* __restrict__ x, int64_t n, double* block_partials, unsigned int* ticket,
                                                          double* result, double* host_mirror, int* advance)
{
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x; i < n; i += (int64_t)gridDim.x * VEC_BLOCK) {
        const double v = (double)x[i];
        s = fma(v, v, s);
    }
    block_reduce_to_scalar(s, block_partials, ticket, result, host_mirror, advance);
}

// The kernels of one Lanczos iteration read the index m of the NEWEST basis vector V[m] from device
// memory (`newest`), so that every iteration is the same sequence of launches with the same arguments:
// the driver captures it once in a CUDA graph and replays it (the loop is launch-bound at small N).
// Scalars the host needs for the stopping test are written straight into mapped pinned host memory.

// V[*newest] = x / sqrt(*sumsq)  (v_1 = z/|z|; v_{k+1} = w/beta_k: the reduction that produced *sumsq has
// already advanced *newest to the slot of the vector being written), and the same
// vector packed as the pair kernel's structure-of-arrays right-hand side (a2) for the next apply:
// soa[c][i], c < nc, ghosts zero.  x and V hold [3N linear | 3N angular].
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) lanczos_scale_pack_kernel(const T* __restrict__ x, int64_t N, int64_t npad, int nc, T len_scale,
                                                                       const double* sumsq, const int* __restrict__ newest,
                                                                       T* __restrict__ V, T* __restrict__ soa, const T* __restrict__ damp)
{
    const int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x;
    if (i >= npad) return;
    const double nrm = sqrt(*sumsq);
    const double inv = nrm > 0.0 ? 1.0 / nrm : 0.0;
    const int64_t n3 = 3 * N, dof = (int64_t)nc * N;
    T* v_out = V + (size_t)(*newest) * dof;
    for (int c = 0; c < nc; ++c) {
        T val = T(0);
        if (i < N) {
            const int64_t idx = (c < 3 ? 0 : n3) + 3 * i + (c % 3);
            val = (T)((double)x[idx] * inv);
            v_out[idx] = val;
        }
        T packed = c < 3 ? val : val * len_scale;                        // angular part: internal length unit, as in pack_rhs
        if (damp) packed *= damp[i];                                     // single wall: the source's damping factor
        soa[(size_t)c * npad + i] = packed;
    }
}

// v = V[*newest]:  w -= sqrt(*beta_prev_sq) * V[*newest - 1]  (skipped for *newest == 0);  *alpha = w . v.
// With `partial` != null the kernel is also the split-j reduce (a6) of the apply that precedes it: w is first
// formed as the sum over the splits of the pair kernel's partials [split][rhs * nc + c][npad] (fixed order,
// fp arithmetic in T exactly as reduce_partials_kernel), for right-hand side `rhs` of `nrhs`.
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) lanczos_alpha_kernel(T* __restrict__ w, const T* __restrict__ V, const int* __restrict__ newest,
                                                                  const double* beta_prev_sq, int64_t n, double* block_partials,
                                                                  unsigned int* ticket, double* alpha, const T* __restrict__ partial, int splits,
                                                                  int nrhs, int rhs, int nc, int64_t npad)
{
    const int m = *newest;
    const T* v = V + (size_t)m * n;
    const T* v_prev = m > 0 ? v - n : nullptr;
    const double bp = v_prev ? sqrt(*beta_prev_sq) : 0.0;
    const int64_t n3 = n / (nc / 3);
    const size_t stride = (size_t)nrhs * nc * npad;
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x; i < n; i += (int64_t)gridDim.x * VEC_BLOCK) {
        if (partial) {
            const int64_t rem = i < n3 ? i : i - n3;
            const T* p = partial + (size_t)(rhs * nc + (i < n3 ? 0 : 3) + (int)(rem % 3)) * npad + rem / 3;
            T acc = T(0);
            for (int sidx = 0; sidx < splits; ++sidx) acc += p[(size_t)sidx * stride];
            w[i] = acc;
        }
        double wi = (double)w[i];
        if (v_prev) {
            wi = fma(-bp, (double)v_prev[i], wi);
            w[i] = (T)wi;
            wi = (double)w[i];          // the dot product sees the stored (rounded) value
        }
        s = fma(wi, (double)v[i], s);
    }
    block_reduce_to_scalar(s, block_partials, ticket, alpha);
}

// w -= *alpha * V[*newest];  *beta_sq = |w|^2;  host_ab[2(m+1)] = alpha, host_ab[2(m+1)+1] = beta^2 (iteration k = m+1);
// then, if `advance` is given, *advance += 1 (the index moves to the slot of v_{k+1}; the last vector of a lockstep group does it)
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) lanczos_beta_kernel(T* __restrict__ w, const T* __restrict__ V, const int* newest,
                                                                 const double* alpha, int64_t n, double* block_partials, unsigned int* ticket,
                                                                 double* beta_sq, double* host_ab, int* advance)   // `advance` may alias `newest`: neither is __restrict__
{
    const int m = *newest;
    const T* v = V + (size_t)m * n;
    const double a = *alpha;
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x; i < n; i += (int64_t)gridDim.x * VEC_BLOCK) {
        const T wi = (T)fma(-a, (double)v[i], (double)w[i]);
        w[i] = wi;
        s = fma((double)wi, (double)wi, s);
    }
    block_reduce_to_scalar(s, block_partials, ticket, beta_sq, host_ab + 2 * (m + 1) + 1, advance);
    if (blockIdx.x == 0 && threadIdx.x == 0) host_ab[2 * (m + 1)] = a;
}

// Small N: the vector part of one Lanczos iteration -- lanczos_alpha_kernel, lanczos_beta_kernel and the scaling of
// lanczos_scale_pack_kernel -- in ONE launch of one CTA (the vectors are a few thousand elements; three launches and
// two grid-wide reductions cost more than the arithmetic; the Gram column is formed by the apply, rpy_small.cuh).  Same operations and rounding points as those kernels:
//   m = *newest;  w -= beta_{k-1} V[m-1] (m > 0);  alpha = w . V[m];  w -= alpha V[m];  beta^2 = |w|^2;  V[m+1] = w / beta;
//   host_ab[2(m+1)] = alpha, host_ab[2(m+1)+1] = beta^2;  scal[1] = alpha, scal[2] = beta^2;  `advance`: *newest = m + 1.
// No packed copy of V[m+1] is written: at these sizes the apply (rpy_small_kernel) reads V[*newest] itself.
// Reductions: fp64, warp shuffles, then the 32 warp sums added in warp order by every thread (deterministic).
constexpr int FUSED_BLOCK = 1024;
__device__ __forceinline__ double cta_sum_1024(double v, double* warp_part)
{
    v = warp_sum(v);
    __syncthreads();                                   // warp_part may still be read from the previous reduction
    if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < FUSED_BLOCK / 32; ++w) s += warp_part[w];
    return s;
}
// EPT = elements per thread (n <= EPT x 1024): every thread keeps its elements of w and V[m] in REGISTERS from the first load
// to the last store -- one global-memory round trip instead of three; w itself is not written back (nothing reads it
// before the next apply overwrites it).
template <typename T, int EPT>
__global__ void __launch_bounds__(FUSED_BLOCK) lanczos_fused_step_kernel(const T* __restrict__ w, T* __restrict__ V, int* newest, double* scal, int64_t n,
                                                                         double* host_ab, int advance)
{
    __shared__ double warp_part[FUSED_BLOCK / 32];
    const int m = *newest;
    const T* v = V + (size_t)m * n;
    const T* v_prev = m > 0 ? v - n : nullptr;
    T* v_next = V + (size_t)(m + 1) * n;
    const double bp = v_prev ? sqrt(scal[2]) : 0.0;
    T wr[EPT], vr[EPT];
    double s = 0.0;
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int64_t i = (int64_t)e * FUSED_BLOCK + threadIdx.x;
        wr[e] = T(0);
        vr[e] = T(0);
        if (i < n) {
            vr[e] = v[i];
            double wi = (double)w[i];
            if (v_prev) wi = (double)(T)fma(-bp, (double)v_prev[i], wi);     // rounded to T where the general kernel stores it
            wr[e] = (T)wi;
            s = fma((double)wr[e], (double)vr[e], s);
        }
    }
    const double alpha = cta_sum_1024(s, warp_part);
    s = 0.0;
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        wr[e] = (T)fma(-alpha, (double)vr[e], (double)wr[e]);                // elements past n stay zero
        s = fma((double)wr[e], (double)wr[e], s);
    }
    const double beta_sq = cta_sum_1024(s, warp_part);
    const double nrm = sqrt(beta_sq);
    const double inv = nrm > 0.0 ? 1.0 / nrm : 0.0;
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        const int64_t i = (int64_t)e * FUSED_BLOCK + threadIdx.x;
        if (i < n) v_next[i] = (T)((double)wr[e] * inv);
    }
    if (threadIdx.x == 0) {
        host_ab[2 * (m + 1)] = alpha;
        host_ab[2 * (m + 1) + 1] = beta_sq;
        scal[1] = alpha;
        scal[2] = beta_sq;
        if (advance) *newest = m + 1;
    }
}

// Gram column for the stopping test (a9): with c = *newest the column of the vector just written,
// g[j] = V[j] . V[c], j = 0..c, stored to host_gram[c * ld + j].  Lanczos without
// re-orthogonalisation loses orthogonality of V, so |y_k - y_{k-1}| = |z| |V_k delta| is evaluated as
// sqrt(delta^T G delta) with the true Gram matrix G = V^T V instead of assuming G = I.
// Grid (chunks, max columns): block (b, j) forms the part of V[j] . V[c] over [b*chunk, (b+1)*chunk) and
// exits at once for j > c; the last block to finish (ticket) adds the partials [j][b] in index order.
constexpr int GRAM_MAX_BLOCKS = 128;
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) gram_column_kernel(const T* __restrict__ V, int64_t dof, const int* __restrict__ newest, int64_t chunk, double* partials,
                                                                unsigned int* ticket, double* host_gram, int ld)
{
    __shared__ double warp_part[VEC_BLOCK / 32];
    __shared__ bool is_last;
    const int c = *newest;
    const int j = blockIdx.y;
    if (j > c) return;
    const int64_t lo_i = (int64_t)blockIdx.x * chunk, hi_i = min(lo_i + chunk, dof);
    const T* vc = V + (size_t)c * dof;
    const T* vj = V + (size_t)j * dof;
    double s = 0.0;
    for (int64_t i = lo_i + threadIdx.x; i < hi_i; i += VEC_BLOCK) s = fma((double)vj[i], (double)vc[i], s);
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < VEC_BLOCK / 32; ++w) t += warp_part[w];
        partials[(size_t)j * gridDim.x + blockIdx.x] = t;
        __threadfence();
        is_last = (atomicAdd(ticket, 1u) == gridDim.x * (unsigned int)(c + 1) - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        for (int jj = threadIdx.x; jj <= c; jj += VEC_BLOCK) {
            double t = 0.0;
            for (unsigned int b = 0; b < gridDim.x; ++b) t += ((volatile double*)partials)[(size_t)jj * gridDim.x + b];
            host_gram[(size_t)c * ld + jj] = t;
        }
        if (threadIdx.x == 0) *ticket = 0u;
    }
}

// a10: y = scale * sum_{m<k} coef[m] V[m]  split into the linear (first 3N) and angular (last 3N)
// outputs; accumulate != 0 adds to what is already there (lm_hydrodynamic_velocities).
template <typename T>
__global__ void __launch_bounds__(VEC_BLOCK) lanczos_combine_kernel(const T* __restrict__ V, int64_t dof, int k, const double* __restrict__ coef,
                                                                    double scale, int accumulate, int64_t n_lin, T* __restrict__ out_lin,
                                                                    T* __restrict__ out_ang)
{
    for (int64_t i = (int64_t)blockIdx.x * VEC_BLOCK + threadIdx.x; i < dof; i += (int64_t)gridDim.x * VEC_BLOCK) {
        double s = 0.0;
        for (int m = 0; m < k; ++m) s = fma(coef[m], (double)V[(size_t)m * dof + i], s);
        s *= scale;
        T* dst = i < n_lin ? out_lin + i : out_ang + (i - n_lin);
        *dst = accumulate ? (T)((double)*dst + s) : (T)s;
    }
}

}  // namespace lm
