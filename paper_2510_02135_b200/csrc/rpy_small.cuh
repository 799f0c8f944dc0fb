// rpy_small.cuh -- ONE-LAUNCH apply U = M.[F;T] for small N (SURVEY.md sec. 7 "Small N"; the regime the paper says the
// NBody solver is for, "< 50K particles", and where its own curves flatten).
//
// The general path (pack_rhs -> rpy_pair_kernel -> reduce_partials) needs three launches and a round trip of the j-split
// partial sums through global memory; below a few thousand particles those launches ARE the cost.  Here one kernel does
// all of it:
//   * it reads the caller's interleaved force / torque arrays directly into shared memory, kept interleaved (the whole
//     source range of a CTA fits many times over), so there is no packing launch;
//   * a CTA owns 64 targets (one packed target pair per lane, as in rpy_pair_kernel) and its WARPS split the CTA's
//     sources, so even N = 1024 spreads over every SM sub-partition;
//   * the sources are further split over the CTAs of a THREAD-BLOCK CLUSTER (cluster dims (1, S, 1)); every CTA adds
//     its warps' sums and pushes them through distributed shared memory (mapa + st.async ... mbarrier::complete_tx) to
//     the CTA that owns the output element, which waits on its own mbarrier for the bytes and adds the S contributions
//     in rank order (deterministic) -- no global partials, no reduce launch, no fence, no remote load;
//   * the pair arithmetic is rpy_pair.cuh's (pair_geom / pair_apply / wall_apply, far / general vote per source group).
#pragma once
#include "rpy_pair.cuh"

namespace lm {

constexpr int SM_TARGETS = 64;        // targets per CTA: 32 lanes x one packed pair
constexpr int SM_MAX_WARPS = 8;
constexpr int SM_MAX_CLUSTER = 8;     // portable cluster size

// Cluster barrier in two halves (PTX barrier.cluster): `arrive` is non-blocking, `wait` blocks until every thread of the
// cluster has arrived.  Used once, to know that every CTA of the cluster is running (and has initialised its mbarrier)
// before anybody writes into its shared memory.
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_acquire() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// shared::cluster address of `saddr` (a shared::cta address of this CTA) in the CTA of rank `rank`
__device__ __forceinline__ uint32_t map_to_rank(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// Asynchronous store into another CTA's shared memory that signals THAT CTA's mbarrier with the bytes written
// (st.async ... mbarrier::complete_tx::bytes): the receiver waits on its own barrier, nobody fences, nobody loads remotely.
__device__ __forceinline__ void st_async(uint32_t raddr, float v, uint32_t rbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f32 [%0], %1, [%2];" ::"r"(raddr), "f"(v), "r"(rbar) : "memory");
}
__device__ __forceinline__ void st_async(uint32_t raddr, double v, uint32_t rbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(raddr), "d"(v), "r"(rbar) : "memory");
}

template <typename T> struct SmallParams {
    const T* __restrict__ pos;   // the handle's packed positions x | y | z (| h | b), each npad long
    RhsIn<T> in;                 // caller's arrays, interleaved xyz, 3N each; null = zeros
    const int* in_index;         // null, or: every input array is read at in.f[q] + *in_index * in_stride (the Lanczos driver
    int64_t in_stride;           //   passes its basis and the device-side index of the newest vector: one launch fits every iteration)
    // Lanczos driver only: while applying M to V[c] (c = *in_index) the kernel also forms column c of the Gram matrix of
    // the basis, gram_out[q][c gram_ld + j] = V_q[j] . V_q[c], j <= c (one CTA per column) -- the stopping test needs it
    // one iteration later, so it rides along instead of being a launch of its own.  gram_out[0] == null: no Gram work.
    double* gram_out[MAX_RHS];
    int64_t gram_n;              // length of a basis vector (dof)
    int gram_ld;
    RhsOut<T> out;               // caller's outputs, interleaved xyz
    int64_t N, npad;
    int64_t i_begin, i_end;      // target rows [i_begin, i_end)
    int src_per_warp;            // sources walked by one warp: multiple of 4; warp g = blockIdx.y * W + w takes [g spw, (g+1) spw)
    T len_scale;                 // torques are multiplied by the internal length unit
    T ghost_z;                   // height given to sources past N (single wall: a; else 0); their forces are zero
    PairConsts<T> c;
};

// dynamic shared memory: the CTA's sources (positions x | y | z, then each right-hand-side array interleaved), the warps' sums [W][NV][64], and the
// contributions received from the cluster's CTAs for the elements this CTA owns (at most [8][NV 64 / S + 1] <= NV 64 + 8);
// the first 16 bytes hold the mbarrier those contributions are counted on
template <typename T, int NRHS, bool ANG> constexpr size_t small_smem_bytes(int warps, int src_per_warp)
{
    return 16 + ((size_t)(3 + NRHS * (ANG ? 6 : 3)) * warps * src_per_warp + (size_t)(warps + 1) * NRHS * (ANG ? 6 : 3) * SM_TARGETS + SM_MAX_CLUSTER) * sizeof(T);
}

template <typename T, int NRHS, bool ANG, bool WALL>
__global__ void __launch_bounds__(SM_MAX_WARPS * 32) rpy_small_kernel(const SmallParams<T> p)
{
    constexpr int NC = ANG ? 6 : 3, NV = NRHS * NC;
    constexpr int VN = Vec16<T>::N;
    constexpr int GS = (NV >= 12 && VN > 2) ? 2 : VN;
    constexpr bool EARLY = ANG || NRHS >= 4;
    using V16 = typename Vec16<T>::type;
    using Near = typename NearOf<T>::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int W = blockDim.x >> 5;
    const int S = gridDim.y;                                   // = cluster size: the cluster spans the whole y extent
    const int rank = blockIdx.y;
    const int spw = p.src_per_warp, cta_src = W * spw;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);     // counts the bytes pushed to this CTA by the cluster
    T* src = reinterpret_cast<T*>(smem_raw + 16);              // x | y | z, each cta_src long, then the right-hand sides
    T* red = src + (size_t)(3 + NV) * cta_src;                 // [W][NV][64]
    T* recv = red + (size_t)W * NV * SM_TARGETS;               // [S][elements owned by this CTA]
    const int64_t j0 = (int64_t)rank * cta_src;
    const int64_t i0 = p.i_begin + (int64_t)blockIdx.x * SM_TARGETS;
    // the output elements this CTA owns: [rank per, rank per + mine) of the E = NV x 64 of its i-tile
    constexpr int E = NV * SM_TARGETS;
    const int per = (E + S - 1) / S;
    const int mine = max(0, min(E, (rank + 1) * per) - rank * per);
    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        if (mine > 0) mbar_expect_tx(bar, (uint32_t)(mine * S * (int)sizeof(T)));   // every CTA of the cluster sends `mine` values
    }
    __syncwarp();
    cluster_arrive_relaxed();                                  // waited for just before the first remote store

    // ---- this lane's packed target pair: targets i0 + lane and i0 + 32 + lane (negated: d = x_j + (-x_i)); loaded first
    // so that their latency overlaps the staging below
    const int64_t ia = min(i0 + lane, p.npad - 1), ib = min(i0 + 32 + lane, p.npad - 1);
    const P2<T> nx = mk2(-p.pos[ia], -p.pos[ib]);
    const P2<T> ny = mk2(-p.pos[p.npad + ia], -p.pos[p.npad + ib]);
    const P2<T> nz = mk2(-p.pos[2 * p.npad + ia], -p.pos[2 * p.npad + ib]);

    // ---- stage this CTA's sources.  Positions: from the packed arrays (structure-of-arrays).  Right-hand sides: straight
    // from the caller, kept INTERLEAVED as they come (xyz xyz ...: one coalesced copy per array; the main loop reads the
    // 3 VN values of VN consecutive sources as three 16-byte loads).  Every load of a round (positions and right-hand
    // sides, STG_U elements of each per thread) is issued before anything is stored: one global-memory latency per round,
    // and a CTA of 8 warps stages its usual 128 sources in ONE round.
    constexpr int STG_U = 2;
    const int B = blockDim.x;
    const int n3_here = 3 * (int)max((int64_t)0, min((int64_t)cta_src, p.N - j0));   // real values of this CTA per array
    const int64_t in_off = (p.in_index ? (int64_t)(*p.in_index) * p.in_stride : 0) + 3 * j0;
    T* rhs = src + 3 * cta_src;                                // [NRHS][forces 3 cta_src (| torques 3 cta_src)]
    for (int base = tid; base < 3 * cta_src; base += STG_U * B) {        // positions need a third of the rounds
        T x[STG_U][3], f[NRHS][STG_U], t[ANG ? NRHS : 1][STG_U], b[STG_U];
#pragma unroll
        for (int u = 0; u < STG_U; ++u) {
            const int idx = base + u * B;
            const int64_t jg = j0 + idx;
            const bool in_pad = idx < cta_src && jg < p.npad;  // packed ghosts [N, npad) are already harmless
            x[u][0] = in_pad ? p.pos[jg] : T(0);
            x[u][1] = in_pad ? p.pos[p.npad + jg] : T(0);
            x[u][2] = in_pad ? p.pos[2 * p.npad + jg] : p.ghost_z;
            const bool real = idx < n3_here;
            b[u] = T(1);
            if constexpr (WALL) b[u] = real ? p.pos[4 * p.npad + j0 + idx / 3] : T(0);
#pragma unroll
            for (int q = 0; q < NRHS; ++q) {
                f[q][u] = (real && p.in.f[q]) ? p.in.f[q][in_off + idx] : T(0);
                if constexpr (ANG) t[q][u] = (real && p.in.t[q]) ? p.in.t[q][in_off + idx] : T(0);
            }
        }
#pragma unroll
        for (int u = 0; u < STG_U; ++u) {
            const int idx = base + u * B;
            if (idx < cta_src) { src[idx] = x[u][0]; src[cta_src + idx] = x[u][1]; src[2 * cta_src + idx] = x[u][2]; }
            if (idx < 3 * cta_src) {
#pragma unroll
                for (int q = 0; q < NRHS; ++q) {
                    rhs[(size_t)q * NC * cta_src + idx] = WALL ? f[q][u] * b[u] : f[q][u];
                    if constexpr (ANG) rhs[(size_t)(q * NC + 3) * cta_src + idx] = WALL ? t[q][u] * p.len_scale * b[u] : t[q][u] * p.len_scale;
                }
            }
        }
    }

    P2<T> z4 = splat(T(0));
    if constexpr (WALL) z4 = mul2(nz, T(-4));
    P2<T> acc[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) acc[k] = splat(T(0));
    __syncthreads();

    // ---- the warp's sources, in groups of GS with one far / general vote per group (rpy_pair.cuh)
    const T* sx = src + warp * spw;
#pragma unroll 1
    for (int j = 0; j < spw; j += VN) {
        const V16 X = *reinterpret_cast<const V16*>(sx + j);
        const V16 Y = *reinterpret_cast<const V16*>(sx + cta_src + j);
        const V16 Z = *reinterpret_cast<const V16*>(sx + 2 * cta_src + j);
        // right-hand side part m (forces of q: 2q or q; torques: 2q + 1): the 3 VN interleaved values of these VN sources
        V16 Vv[NV / 3][3];
#pragma unroll
        for (int m = 0; m < NV / 3; ++m)
#pragma unroll
            for (int c = 0; c < 3; ++c) Vv[m][c] = *reinterpret_cast<const V16*>(rhs + (size_t)m * 3 * cta_src + 3 * (warp * spw + j) + c * VN);
#pragma unroll
        for (int e0 = 0; e0 < VN; e0 += GS) {
            PairGeom<T> gm[GS];
            Near near;
            near_init(near);
#pragma unroll
            for (int e = 0; e < GS; ++e) gm[e] = pair_geom<T, EARLY>(p.c, nx, ny, nz, vget(X, e0 + e), vget(Y, e0 + e), vget(Z, e0 + e), near);
            const bool hit = __any_sync(0xffffffffu, near_test(near, p.c.four_a2));
            auto body = [&](auto far_tag) {
                constexpr bool FAR = decltype(far_tag)::value;
#pragma unroll
                for (int e = 0; e < GS; ++e) {
                    T Vs[NV];
#pragma unroll
                    for (int k = 0; k < NV; ++k) Vs[k] = vget(Vv[k / 3][(3 * (e0 + e) + k % 3) / VN], (3 * (e0 + e) + k % 3) % VN);
                    pair_apply<T, NRHS, ANG, FAR, EARLY>(p.c, gm[e], Vs, acc);
                    if constexpr (WALL) wall_apply<T, NRHS, ANG>(p.c, gm[e], nz, z4, vget(Z, e0 + e), Vs, acc);
                }
            };
            if (!hit) body(std::true_type{});
            else body(std::false_type{});
        }
    }

    // ---- reduction, deterministic: (1) the warp's sums -> shared memory; (2) every CTA adds its W warps in warp order and
    // PUSHES the result to the CTA of the cluster that owns the element (st.async: fire and forget, counted on the owner's
    // mbarrier); (3) the owner waits for its S x mine values, adds the S contributions in rank order, applies the
    // factored-out prefactor (single wall: times b_i) and writes the caller's array.
    // element e = ((q * PARTS + part) * 64 + t) * 3 + k3: consecutive e are consecutive addresses of one output array
    constexpr int PARTS = ANG ? 2 : 1;
    T* my = red + (size_t)warp * E;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        my[k * SM_TARGETS + lane] = lo(acc[k]);
        my[k * SM_TARGETS + 32 + lane] = hi(acc[k]);
    }
    __syncthreads();
    cluster_wait_acquire();                                    // every CTA of the cluster is running and its mbarrier is initialised
    const uint32_t recv_s = smem_u32(recv), bar_s = smem_u32(bar);
    for (int e = tid; e < E; e += blockDim.x) {
        const int k3 = e % 3, t = (e / 3) % SM_TARGETS, qp = e / (3 * SM_TARGETS), part = qp % PARTS, q = qp / PARTS;
        const int off = (q * NC + part * 3 + k3) * SM_TARGETS + t;
        T v[SM_MAX_WARPS];
#pragma unroll
        for (int w = 0; w < SM_MAX_WARPS; ++w) v[w] = w < W ? red[(size_t)w * E + off] : T(0);
        T s = v[0];
#pragma unroll
        for (int w = 1; w < SM_MAX_WARPS; ++w) s += v[w];     // adding the zeros of absent warps changes nothing
        const int owner = e / per;
        st_async(map_to_rank(recv_s + (uint32_t)((rank * per + (e - owner * per)) * (int)sizeof(T)), owner), s, map_to_rank(bar_s, owner));
    }
    if (mine > 0) mbar_wait(bar, 0u);                          // all S x mine values have landed (acquire)
    for (int el = tid; el < mine; el += blockDim.x) {
        const int e = rank * per + el;
        const int k3 = e % 3, t = (e / 3) % SM_TARGETS, qp = e / (3 * SM_TARGETS), part = qp % PARTS, q = qp / PARTS;
        const int64_t i = i0 + t;
        if (i >= p.i_end) continue;
        T v[SM_MAX_CLUSTER];
#pragma unroll
        for (int c = 0; c < SM_MAX_CLUSTER; ++c) v[c] = c < S ? recv[c * per + el] : T(0);
        T s = v[0];
#pragma unroll
        for (int c = 1; c < SM_MAX_CLUSTER; ++c) s += v[c];
        T fac = part ? p.c.C1_ang : p.c.C1_lin;
        if constexpr (WALL) fac *= p.pos[4 * p.npad + i];
        (part ? p.out.ang[q] : p.out.lin[q])[3 * i + k3] = s * fac;
    }

    // ---- Gram column of the vector being applied (Lanczos driver): CTA b takes the columns j = b, b + #CTAs, ...
    if (p.gram_out[0]) {
        __shared__ double gpart[SM_MAX_WARPS];
        const int c = *p.in_index;
        const int cta = blockIdx.y * gridDim.x + blockIdx.x, ncta = gridDim.x * gridDim.y;
#pragma unroll
        for (int q = 0; q < NRHS; ++q) {
            const T* Vq = p.in.f[q];                           // basis of vector q: V[j] = Vq + j gram_n  (in_stride == gram_n)
            const T* vc = Vq + (int64_t)c * p.gram_n;
            for (int j = cta; j <= c; j += ncta) {
                const T* vj = Vq + (int64_t)j * p.gram_n;
                double t = 0.0;
                for (int64_t i0 = tid; i0 < p.gram_n; i0 += 4 * blockDim.x) {      // 8 independent loads in flight per thread
                    T a[4], b[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int64_t i = i0 + (int64_t)u * blockDim.x;
                        a[u] = i < p.gram_n ? vj[i] : T(0);
                        b[u] = i < p.gram_n ? vc[i] : T(0);
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) t = fma((double)a[u], (double)b[u], t);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                __syncthreads();                               // gpart may still be read from the previous column
                if (lane == 0) gpart[warp] = t;
                __syncthreads();
                if (tid == 0) {
                    double sum = 0.0;
                    for (int w2 = 0; w2 < W; ++w2) sum += gpart[w2];
                    p.gram_out[q][(size_t)c * p.gram_ld + j] = sum;
                }
            }
        }
    }
}

}  // namespace lm
