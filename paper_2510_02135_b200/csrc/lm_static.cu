// lm_static.cu -- lm_mdot_static: U = M.F (RPY, free space, translational) for callers that may not allocate.
//
// WHO THIS IS FOR.  Every other compute call of liblm works through an lm_solver handle, and a handle owns device
// memory obtained with cudaMalloc (packed positions at lm_create; packed forces and the j-split partial sums on
// the first apply, grown when needed).  Some programs cannot accept that:
//   * a simulation engine (or a framework's caching allocator) that took the whole card for its own arena at start-up:
//     a later cudaMalloc from a library simply fails, or succeeds only by eating the headroom the engine counts on;
//   * a time-stepping loop tuned for latency: cudaMalloc and cudaFree synchronise the whole device, so a library that
//     allocates "only the first time" or "only when N grows" stalls every other stream at a moment the caller does not choose;
//   * a process held to a fixed device-memory budget (a per-client limit under MPS, a share of a GPU agreed with other
//     jobs), whose budget is checked once, when the libraries are loaded, not call by call.
// For them this file offers ONE handle-free call that allocates nothing, on the device or through any library: the
// scratch the apply needs (packed positions, packed forces, j-split partial sums) lives in a file-scope __device__
// array that is part of the library image.  The price is stated up front: LM_STATIC_SCRATCH_BYTES (16 MiB) of every
// GPU this process uses with the library loaded are held from the first CUDA call until exit, used or not, and the
// problem size is capped at LM_STATIC_MAX_N (65536 particles -- the range the paper recommends the NBody solver for,
// PAPER.md:173 "less than 50K particles").
//
// WHAT IT COMPUTES: exactly lm_mdot's translational free-space result (
// PAPER.md:173, eq. (8)), with the same pair kernel template (rpy_pair.cuh) in a 3-stage instantiation of its
// own, so results agree with lm_mdot to summation order.  No torques, no wall, one right-hand side.
//
// RULES OF THE SHARED ARRAY
//   * One array per GPU, shared by every call on that GPU, from any host thread and any stream.  Two calls whose kernels
//     overlap on the GPU (different streams, or different host threads without ordering) RACE on it and both results
//     are garbage.  Calls on one stream, or ordered by events, are safe.
//   * The array keeps whatever the previous call left.  Nothing in it has to start at zero: every word a call reads
//     (packed arrays up to the padded size, every partial of every split) is written earlier in that same call, so
//     there is nothing to clear and stale contents of a larger earlier problem are never read.
//   * The FIRST call on each device does a one-time set-up with that device current: it asks the runtime for the
//     array's device address (in host code the array's name is only a host-side shadow symbol; handing `&scratch` to a
//     kernel would fault or scribble on host-reachable memory), raises the kernels' dynamic shared-memory limit and
//     queries occupancy.  That first call should be made outside any stream capture; later calls only launch kernels.
//
// Separate translation unit on purpose: the array, the cudaGetSymbolAddress that resolves it and the launches that use
// it sit in one .cu file.  It shares no host state with lm_api.cu.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/lm.h"
#include "rpy_pair.cuh"

namespace {

using namespace lm;

constexpr size_t SCRATCH_BYTES = LM_STATIC_SCRATCH_BYTES;
constexpr int64_t MAX_N = LM_STATIC_MAX_N;
constexpr int MAX_DEVICES = 64;
constexpr int QUANTUM = 32;            // padded size = N rounded up to this many particles (the pair kernel's source unit)
constexpr int ST_BLOCK = 256, ST_TPT = 4, ST_TJ = 512, ST_STAGES = 3, ST_SUB = 32;
constexpr int O_BLOCK = 256;           // threads per block of the two O(N) kernels below

// The scratch itself.  256-byte alignment: the TMA bulk copies of the pair kernel need 16-byte aligned sources, and the
// three regions carved out of it start at multiples of 128 bytes (padded sizes are multiples of 32 elements).
static __device__ __align__(256) unsigned char lm_static_scratch[SCRATCH_BYTES];

// a1 + a2 in one pass: interleaved positions and forces -> x | y | z | Fx | Fy | Fz, each npad long, ghosts zero;
// lengths times len_scale (the power of two nearest 1/a, as lm_set_positions does).
template <typename T>
__global__ void __launch_bounds__(O_BLOCK) static_pack_kernel(const T* __restrict__ pos, const T* __restrict__ force, int64_t N, int64_t npad, T len_scale,
                                                              T* __restrict__ pos_soa, T* __restrict__ vec_soa)
{
    const int64_t i = (int64_t)blockIdx.x * O_BLOCK + threadIdx.x;
    if (i >= npad) return;
    T v[6] = {T(0), T(0), T(0), T(0), T(0), T(0)};
    if (i < N) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { v[k] = pos[3 * i + k] * len_scale; v[3 + k] = force[3 * i + k]; }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) { pos_soa[(size_t)k * npad + i] = v[k]; vec_soa[(size_t)k * npad + i] = v[3 + k]; }
}

// a6: sum the j-split partials [splits][3][npad] in split order (deterministic) into the interleaved output.
template <typename T>
__global__ void __launch_bounds__(O_BLOCK) static_reduce_kernel(const T* __restrict__ partial, int splits, int64_t N, int64_t npad, T* __restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * O_BLOCK + threadIdx.x;
    if (i >= N) return;
    const int k = blockIdx.y;
    T s = T(0);
    for (int sp = 0; sp < splits; ++sp) s += partial[((size_t)sp * 3 + k) * npad + i];
    out[3 * i + k] = s;
}

template <typename T> struct StaticKernel;
template <> struct StaticKernel<float> {
    static constexpr int MINB = 2;
    using Tr = PairKernelTraits<float, 1, false, ST_TPT, ST_BLOCK, ST_TJ, ST_STAGES, ST_SUB>;
    static auto get() { return rpy_pair_kernel<float, 1, false, ST_TPT, ST_BLOCK, ST_TJ, ST_STAGES, ST_SUB, MINB>; }
};
template <> struct StaticKernel<double> {
    static constexpr int MINB = 1;
    using Tr = PairKernelTraits<double, 1, false, ST_TPT, ST_BLOCK, ST_TJ, ST_STAGES, ST_SUB>;
    static auto get() { return rpy_pair_kernel<double, 1, false, ST_TPT, ST_BLOCK, ST_TJ, ST_STAGES, ST_SUB, MINB>; }
};

// per-device state of the one-time set-up (host memory of fixed size: no allocation here either)
struct DeviceState {
    bool ready = false;
    unsigned char* scratch = nullptr;   // DEVICE address of lm_static_scratch on this device
    int sm_count = 0;
    int ctas_per_sm[2] = {1, 1};        // [LM_F32], [LM_F64]
};
DeviceState g_dev[MAX_DEVICES];
std::mutex g_mutex;
thread_local char t_err[320] = "";

int fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
    return code;
}

#define ST_CUDA(expr)                                                                                         \
    do {                                                                                                      \
        cudaError_t e__ = (expr);                                                                             \
        if (e__ != cudaSuccess) return fail(LM_E_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

// One-time set-up for the CURRENT device (the caller holds g_mutex).
int setup_device(int dev, DeviceState& d)
{
    // The device address of the array.  `lm_static_scratch` in this host function names a host shadow variable; only
    // cudaGetSymbolAddress (asked with the target device current) yields the pointer a kernel may dereference.
    void* ptr = nullptr;
    ST_CUDA(cudaGetSymbolAddress(&ptr, lm_static_scratch));
    if (!ptr) return fail(LM_E_CUDA, "cudaGetSymbolAddress returned a null address for the static scratch on device %d", dev);
    ST_CUDA(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
    const void* kf = (const void*)StaticKernel<float>::get();
    const void* kd = (const void*)StaticKernel<double>::get();
    ST_CUDA(cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, StaticKernel<float>::Tr::SMEM_BYTES));
    ST_CUDA(cudaFuncSetAttribute(kd, cudaFuncAttributeMaxDynamicSharedMemorySize, StaticKernel<double>::Tr::SMEM_BYTES));
    int nb = 0;
    ST_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kf, ST_BLOCK, StaticKernel<float>::Tr::SMEM_BYTES));
    d.ctas_per_sm[LM_F32] = std::max(nb, 1);
    ST_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kd, ST_BLOCK, StaticKernel<double>::Tr::SMEM_BYTES));
    d.ctas_per_sm[LM_F64] = std::max(nb, 1);
    d.scratch = (unsigned char*)ptr;
    d.ready = true;
    return LM_OK;
}

// Same constants as the handle path derives: `a` is the radius in the internal length unit.
template <typename T> PairConsts<T> static_consts(double eta, double a, double len_scale)
{
    const double pi = 3.14159265358979323846264338327950288;
    PairConsts<T> c = {};
    const double c4 = 4.0 / (3.0 * a);
    c.tiny = (T)std::max(a * a * std::ldexp(1.0, sizeof(T) == 4 ? -80 : -200), sizeof(T) == 4 ? 4.8e-38 : 1e-300);
    c.four_a2 = (T)(4.0 * a * a);
    c.c2 = (T)(2.0 * a * a / 3.0);
    c.nc3 = (T)(-2.0 * a * a);
    c.c4 = (T)c4;
    c.nc5 = (T)(-c4 * 9.0 / (32.0 * a));
    c.c6 = (T)(c4 * 3.0 / (32.0 * a));
    c.C1_lin = (T)(len_scale / (8.0 * pi * eta));
    c.C1_ang = (T)(len_scale * len_scale / (8.0 * pi * eta));
    return c;                                   // rotational / wall constants stay zero: this kernel never reads them
}

template <typename T>
int mdot_static_t(const DeviceState& d, int prec, int64_t N, double eta, double a, const void* positions, const void* forces, void* lin_out, cudaStream_t st)
{
    using K = StaticKernel<T>;
    const int64_t npad = (N + QUANTUM - 1) / QUANTUM * QUANTUM;
    const double len_scale = std::ldexp(1.0, -(int)std::lround(std::log2(a)));
    if (sizeof(T) == 4 && (len_scale > 0x1p100 || len_scale < 0x1p-100)) return fail(LM_E_INVALID, "lm_mdot_static: radius a = %g is outside the fp32 range served", a);

    // carve the array: packed positions [3][npad] | packed forces [3][npad] | partials [splits][3][npad]
    const size_t arr = (size_t)3 * npad * sizeof(T);
    T* pos_soa = (T*)d.scratch;
    T* vec_soa = (T*)(d.scratch + arr);
    T* partial = (T*)(d.scratch + 2 * arr);
    const int max_by_scratch = (int)std::min<size_t>((SCRATCH_BYTES - 2 * arr) / arr, 256);

    // launch shape: i-tiles of 1024 targets x j-splits, sized to (at most) one full set of resident CTAs
    const int i_tiles = (int)((N + K::Tr::TARGETS - 1) / K::Tr::TARGETS);
    const int units = (int)(npad / ST_SUB);
    const int slots = d.sm_count * d.ctas_per_sm[prec];
    int splits = std::max(1, slots / i_tiles);
    splits = std::min(splits, std::min(units, max_by_scratch));
    if (splits < 1) return fail(LM_E_INVALID, "lm_mdot_static: N = %lld does not fit the static scratch", (long long)N);   // cannot happen for N <= MAX_N

    static_pack_kernel<T><<<(unsigned)((npad + O_BLOCK - 1) / O_BLOCK), O_BLOCK, 0, st>>>((const T*)positions, (const T*)forces, N, npad, (T)len_scale, pos_soa, vec_soa);

    PairParams<T> p = {};
    p.pos = pos_soa;
    p.vec = vec_soa;
    p.out.lin[0] = (T*)lin_out;
    p.partial = partial;
    p.damp = nullptr;
    p.N = N;
    p.i_begin = 0;
    p.i_end = N;
    p.npad = npad;
    p.n_units = units;
    p.c = static_consts<T>(eta, a * len_scale, len_scale);
    K::get()<<<dim3(i_tiles, splits), ST_BLOCK, K::Tr::SMEM_BYTES, st>>>(p);
    if (splits > 1)
        static_reduce_kernel<T><<<dim3((unsigned)((N + O_BLOCK - 1) / O_BLOCK), 3), O_BLOCK, 0, st>>>(partial, splits, N, npad, (T*)lin_out);
    ST_CUDA(cudaGetLastError());
    return LM_OK;
}

}  // namespace

extern "C" {

int64_t lm_mdot_static_max_n(void) { return MAX_N; }

const char* lm_mdot_static_error(void) { return t_err; }

int lm_mdot_static(int precision, int64_t N, double eta, double a, const void* positions, const void* forces, void* lin_out, void* stream)
{
    t_err[0] = '\0';
    if (precision != LM_F32 && precision != LM_F64) return fail(LM_E_INVALID, "lm_mdot_static: precision must be LM_F32 or LM_F64");
    if (N <= 0) return fail(LM_E_INVALID, "lm_mdot_static: N = %lld, need N >= 1", (long long)N);
    if (N > MAX_N)
        return fail(LM_E_INVALID, "lm_mdot_static: N = %lld exceeds LM_STATIC_MAX_N = %lld (the static scratch is %zu bytes); use lm_create + lm_mdot for larger systems",
                    (long long)N, (long long)MAX_N, SCRATCH_BYTES);
    if (!(eta > 0.0) || !(a > 0.0) || !std::isfinite(eta) || !std::isfinite(a)) return fail(LM_E_INVALID, "lm_mdot_static: eta and a must be positive and finite");
    if (!positions || !forces || !lin_out) return fail(LM_E_NULL, "lm_mdot_static: positions, forces and lin_out must be non-NULL device pointers");

    int dev = -1;
    ST_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(LM_E_INVALID, "lm_mdot_static: device ordinal %d not served (0 ... %d)", dev, MAX_DEVICES - 1);
    DeviceState& d = g_dev[dev];
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (!d.ready) {
            const int rc = setup_device(dev, d);
            if (rc != LM_OK) return rc;
        }
    }
    return precision == LM_F32 ? mdot_static_t<float>(d, precision, N, eta, a, positions, forces, lin_out, (cudaStream_t)stream)
                               : mdot_static_t<double>(d, precision, N, eta, a, positions, forces, lin_out, (cudaStream_t)stream);
}

}  // extern "C"
